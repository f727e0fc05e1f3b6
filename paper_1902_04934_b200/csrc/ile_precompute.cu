// ile_precompute.cu -- the overlap pre-computation of an intrinsic point (eq. 8a-c):
//
//   Q_{k,lm}[i] = <h_lm(. - tau_i) | d_k> = sum_n conj(x_{k,lm}[n]) d_k[n] exp(+2 pi i f_n tau_i),  tau_i = t0_Q + i / f_s
//   U_k[a][b]   = sum_n conj(x_a[n]) x_b[n]            V_k[a][b] = sum_n x_a[(-n) mod N] x_b[n]
//
// on the two-sided FFT grid f_n = n' f_s / N (n' the signed index of FFT order), whitened spectra in, complex128 throughout.
// "After the port it is what dominates for BNS" (L97, L175): one inverse FFT per (point, detector, mode) and M^2 dot
// products per (point, detector).
//
//   ile_overlap_tables_kernel      twiddles exp(2 pi i j / N) and start-time phases exp(2 pi i f_n t0_Q), once per (N, t0_Q)
//   ile_overlap_q_radix8_kernel    512 <= N <= 8192, N / 8 threads per series: register-resident radix-8 Stockham passes, first pass
//                                  from global memory (spectrum product, optional 1/S weight and band mask, start-time phase), last
//                                  pass to global memory, one padded shared buffer in between
//   ile_overlap_q_stockham_kernel  N < 512: radix-4 Stockham passes between two shared buffers (whitened spectra only)
//   ile_overlap_uv_small_kernel    M <= 5: one block per (detector, point), warp = (row a, frequency slice), pairs (a, b >= a) in registers
//   ile_overlap_uv_kernel          any M: register-blocked tiles of pairs (a, b), lanes over frequencies
// With S != NULL the inner products are eq. 2's (L30-L35): weight scale / S_k(|f_n|) inside f_min < |f_n| < f_max, 0 outside.
#include <mutex>

#include "ile_kernels.h"

#define PC_THREADS 256

__device__ __forceinline__ double2 pc_cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

// tab[0 .. N/2) = twiddles exp(+2 pi i j / N); tab[N/2 .. N/2 + N) = start-time phases exp(2 pi i f_n t0_Q), f_n = n' f_s / N
// (the same for every series of the call: computed once instead of 1.5 sincospi per point and series)
__global__ void __launch_bounds__(PC_THREADS) ile_overlap_tables_kernel(int32_t N, double fs_t0_over_n, double2 *__restrict__ tab)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    double s, c;
    if (j < N / 2) {
        sincospi(2.0 * (double)j / (double)N, &s, &c);
        tab[j] = make_double2(c, s);
    }
    if (j < N) {
        const int np = j < (N + 1) / 2 ? j : j - N;  // signed index
        sincospi(2.0 * (double)np * fs_t0_over_n, &s, &c);
        tab[N / 2 + j] = make_double2(c, s);
    }
}

// W_N^m = exp(+2 pi i m / N) for 0 <= m < N from the half-length table
__device__ __forceinline__ double2 pc_tw(const double2 *__restrict__ tab, int N, int m)
{
    const bool hi = m >= N / 2;
    const double2 w = __ldg(tab + (hi ? m - N / 2 : m));
    return hi ? make_double2(-w.x, -w.y) : w;
}

// Stockham autosort form (N <= 4096): natural order in and out through two ping-pong buffers, no bit reversal.  Stage with
// completed sub-transforms of length ns: u = in[j], v = W^(k N / 2ns) in[j + N/2], k = j mod ns;
// out[(j - k) 2 + k] = u + v, out[... + ns] = u - v.  EPT = N / PC_THREADS elements per thread, compile-time, so that the
// global loads of a thread are all in flight at once and the butterflies of a stage are independent instruction streams
// (EPT = 0: any N < 2 PC_THREADS, plain loops).  Twiddles come from the table through L1.
template <int EPT>
__global__ void __launch_bounds__(PC_THREADS)
    ile_overlap_q_stockham_kernel(int32_t M, int32_t N, int32_t log2n, const double2 *__restrict__ tab, const double2 *__restrict__ x,
                                  const double2 *__restrict__ d, double2 *__restrict__ Q)
{
    extern __shared__ double2 pc_sm[];
    double2 *in = pc_sm, *out = pc_sm + N;
    const size_t series = blockIdx.x;  // (point * K + k) * M + mode
    const double2 *xs = x + series * N;
    const double2 *ds = d + (series / M) * N;
    if (EPT > 0) {
        double2 xv[EPT > 0 ? EPT : 1], dv[EPT > 0 ? EPT : 1], pv[EPT > 0 ? EPT : 1];
#pragma unroll
        for (int e = 0; e < EPT; ++e) {
            const int n = e * PC_THREADS + threadIdx.x;
            xv[e] = __ldcs(xs + n), dv[e] = __ldg(ds + n), pv[e] = __ldg(tab + N / 2 + n);
        }
#pragma unroll
        for (int e = 0; e < EPT; ++e) {
            const double2 w = pc_cmul(dv[e], pv[e]);
            in[e * PC_THREADS + threadIdx.x] = make_double2(xv[e].x * w.x + xv[e].y * w.y, xv[e].x * w.y - xv[e].y * w.x);  // conj(x) d
        }
    } else {
        for (int n = threadIdx.x; n < N; n += PC_THREADS) {
            const double2 xv = xs[n], w = pc_cmul(ds[n], tab[N / 2 + n]);
            in[n] = make_double2(xv.x * w.x + xv.y * w.y, xv.x * w.y - xv.y * w.x);
        }
    }
    __syncthreads();
    // radix-4 passes (each element goes through shared memory once per pass: the transform is bound by the 16-byte shared
    // accesses, 4 wavefronts per warp instruction), then one radix-2 pass when log2 N is odd
    const int T4 = N >> 2;
    int ns = 1;
    for (; ns * 4 <= N; ns <<= 2) {
        const int tws = N / (4 * ns);  // W_N^(r k tws) = exp(2 pi i r k / (4 ns))
        auto pass4 = [&](int j) {
            const int k = j & (ns - 1), j0 = ((j - k) << 2) + k;
            double2 u0 = in[j], u1 = in[j + T4], u2 = in[j + 2 * T4], u3 = in[j + 3 * T4];
            if (ns > 1) {
                u1 = pc_cmul(pc_tw(tab, N, k * tws), u1);
                u2 = pc_cmul(pc_tw(tab, N, 2 * k * tws), u2);
                u3 = pc_cmul(pc_tw(tab, N, 3 * k * tws), u3);
            }
            const double2 v0 = make_double2(u0.x + u2.x, u0.y + u2.y), v1 = make_double2(u0.x - u2.x, u0.y - u2.y);
            const double2 v2 = make_double2(u1.x + u3.x, u1.y + u3.y);
            const double2 v3 = make_double2(-(u1.y - u3.y), u1.x - u3.x);  // (u1 - u3) * (+i): inverse transform
            out[j0] = make_double2(v0.x + v2.x, v0.y + v2.y);
            out[j0 + ns] = make_double2(v1.x + v3.x, v1.y + v3.y);
            out[j0 + 2 * ns] = make_double2(v0.x - v2.x, v0.y - v2.y);
            out[j0 + 3 * ns] = make_double2(v1.x - v3.x, v1.y - v3.y);
        };
        if (EPT >= 4) {
#pragma unroll
            for (int e = 0; e < EPT / 4; ++e) pass4(e * PC_THREADS + threadIdx.x);
        } else {
            for (int j = threadIdx.x; j < T4; j += PC_THREADS) pass4(j);
        }
        __syncthreads();
        double2 *t = in;
        in = out, out = t;
    }
    if (ns < N) {  // ns = N / 2
        for (int j = threadIdx.x; j < N / 2; j += PC_THREADS) {
            const double2 u = in[j], v = pc_cmul(__ldg(tab + j), in[j + N / 2]);  // k = j, W_N^k
            out[j] = make_double2(u.x + v.x, u.y + v.y);
            out[j + ns] = make_double2(u.x - v.x, u.y - v.y);
        }
        __syncthreads();
        double2 *t = in;
        in = out, out = t;
    }
    double2 *q = Q + series * N;
    for (int i = threadIdx.x; i < N; i += PC_THREADS) __stcs(q + i, in[i]);
}

// ------------------------------------------------------------------------------------------------------------
// Radix-8 Stockham transform, 512 <= N <= 8192, N / 8 threads per series: a thread owns one radix-8 butterfly per pass and keeps
// its eight points in registers.  The first pass takes its inputs straight from global memory (spectrum product, 1/S weight,
// band mask and start-time phase applied on the way), the last pass stores straight to Q; in between the points go through ONE
// shared buffer (read - barrier - write - barrier), padded by one element per eight so that every 16-byte access pattern of
// every pass is conflict free (quarter warps touch 128 consecutive bytes).  2048 points: passes 8, 8, 8, 4 -- three trips
// through shared memory instead of the six of the radix-4 form.
// ------------------------------------------------------------------------------------------------------------
#define PC_PAD(i) ((i) + ((i) >> 3))

__device__ __forceinline__ double2 pc_add(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 pc_sub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 pc_muli(double2 a) { return make_double2(-a.y, a.x); }  // a * (+i)

// inverse radix-4: v_q = sum_r a_r exp(+2 pi i q r / 4)
__device__ __forceinline__ void pc_bfly4(double2 a0, double2 a1, double2 a2, double2 a3, double2 &v0, double2 &v1, double2 &v2, double2 &v3)
{
    const double2 s02 = pc_add(a0, a2), d02 = pc_sub(a0, a2), s13 = pc_add(a1, a3), d13 = pc_muli(pc_sub(a1, a3));
    v0 = pc_add(s02, s13), v2 = pc_sub(s02, s13), v1 = pc_add(d02, d13), v3 = pc_sub(d02, d13);
}

// inverse radix-8 in place: u_q <- sum_r u_r exp(+2 pi i q r / 8)
__device__ __forceinline__ void pc_bfly8(double2 (&u)[8])
{
    double2 e0, e1, e2, e3, o0, o1, o2, o3;
    pc_bfly4(u[0], u[2], u[4], u[6], e0, e1, e2, e3);
    pc_bfly4(u[1], u[3], u[5], u[7], o0, o1, o2, o3);
    const double h = 0.70710678118654752440;
    o1 = make_double2(h * (o1.x - o1.y), h * (o1.x + o1.y));    // * (1 + i) / sqrt 2
    o2 = pc_muli(o2);                                           // * i
    o3 = make_double2(-h * (o3.x + o3.y), h * (o3.x - o3.y));   // * (-1 + i) / sqrt 2
    u[0] = pc_add(e0, o0), u[4] = pc_sub(e0, o0), u[1] = pc_add(e1, o1), u[5] = pc_sub(e1, o1);
    u[2] = pc_add(e2, o2), u[6] = pc_sub(e2, o2), u[3] = pc_add(e3, o3), u[7] = pc_sub(e3, o3);
}

// weight applied to the product conj(x[n]) d[n] on load: start-time phase, and for the un-whitened entry 1 / S_k(|f_n|) inside
// the band f_min < |f_n| < f_max, 0 outside (eq. 2)
struct PcWeight {
    const double *S;   // [P][K][N] one-sided PSD sampled on the FFT grid's |f_n| (FFT order), or NULL: spectra already whitened
    double df, fmin, fmax, scale;
};

// weight of frequency n: scale / S[n] inside the band f_min < |f_n| < f_max, 0 outside
__device__ __forceinline__ double pc_weight(const double *__restrict__ Ss, const PcWeight &wt, int N, int n)
{
    const int np = n < (N + 1) / 2 ? n : N - n;  // |n'|
    const double f = (double)np * wt.df;
    return (f > wt.fmin && f < wt.fmax) ? wt.scale / __ldg(Ss + n) : 0.0;
}

__device__ __forceinline__ double2 pc_input(const double2 *__restrict__ xs, const double2 *__restrict__ ds, const double2 *__restrict__ ph,
                                            const double *__restrict__ Ss, const PcWeight &wt, int N, int n)
{
    const double2 xv = __ldcs(xs + n);
    double2 w = pc_cmul(__ldg(ds + n), __ldg(ph + n));
    if (Ss) {
        const double g = pc_weight(Ss, wt, N, n);
        w.x *= g, w.y *= g;
    }
    return make_double2(xv.x * w.x + xv.y * w.y, xv.x * w.y - xv.y * w.x);  // conj(x) w
}

// STRIDE = 1: the whole transform of a series.  STRIDE = 8: the second level of a two-level transform of length 8 N -- block
// (series, i1) transforms row i1 of the first level's output (plain loads from `x`) and writes X[i1 + 8 i2]; `tab` is then the
// table of the LONG transform, whose every eighth twiddle is the short one's.
template <int T, int STRIDE>  // T = N / 8 threads
__global__ void __launch_bounds__(T)
    ile_overlap_q_radix8_kernel(int32_t M, int32_t N, const double2 *__restrict__ tab, const double2 *__restrict__ x,
                                const double2 *__restrict__ d, const PcWeight wt, double2 *__restrict__ Q)
{
    extern __shared__ double2 pc_sm[];
    const size_t series = blockIdx.x;  // (point * K + k) * M + mode; STRIDE = 8: that times 8 + i1
    const double2 *xs = x + series * N, *ds = d + (series / M) * N, *ph = tab + N / 2;
    const double *Ss = wt.S ? wt.S + (series / M) * N : nullptr;
    double2 *q = STRIDE == 1 ? Q + series * N : Q + (series / STRIDE) * ((size_t)N * STRIDE) + (series % STRIDE);
    const int NB = N * STRIDE;  // length the table was built for
    const int j = threadIdx.x;  // blockDim.x == T == N / 8: one radix-8 butterfly per thread and pass
    double2 u[8];
    // ---- pass 1 (sub-transform length 1, no twiddles): inputs from global memory
#pragma unroll
    for (int r = 0; r < 8; ++r) u[r] = STRIDE == 1 ? pc_input(xs, ds, ph, Ss, wt, N, j + r * T) : __ldcs(xs + j + r * T);
    pc_bfly8(u);
    int ns = 8;
    if (ns == N) {
#pragma unroll
        for (int r = 0; r < 8; ++r) q[(size_t)(j * 8 + r) * STRIDE] = u[r];
        return;
    }
#pragma unroll
    for (int r = 0; r < 8; ++r) pc_sm[PC_PAD(j * 8 + r)] = u[r];
    __syncthreads();
    // ---- radix-8 passes while they fit
    for (; ns * 8 <= N; ns <<= 3) {
        const int k = j & (ns - 1), j0 = ((j - k) << 3) + k;
#pragma unroll
        for (int r = 0; r < 8; ++r) u[r] = pc_sm[PC_PAD(j + r * T)];
        // twiddles exp(2 pi i r k / (8 ns)): the first from the table, the others by multiplication
        const double2 w1 = pc_tw(tab, NB, STRIDE * k * (N / (8 * ns)));
        double2 w = w1;
#pragma unroll
        for (int r = 1; r < 8; ++r) {
            u[r] = pc_cmul(w, u[r]);
            w = pc_cmul(w, w1);
        }
        pc_bfly8(u);
        if (ns * 8 == N) {  // last pass: natural order out, consecutive threads write consecutive addresses
#pragma unroll
            for (int r = 0; r < 8; ++r) __stcs(q + (size_t)(j0 + r * ns) * STRIDE, u[r]);
            return;
        }
        __syncthreads();  // everybody has read its inputs
#pragma unroll
        for (int r = 0; r < 8; ++r) pc_sm[PC_PAD(j0 + r * ns)] = u[r];
        __syncthreads();
    }
    // ---- final radix-4 or radix-2 pass (N / ns = 4 or 2), straight to global memory
    if (ns * 4 == N) {
        const int T4 = N >> 2;
        for (int jj = j; jj < T4; jj += T) {
            const int k = jj & (ns - 1), j0 = ((jj - k) << 2) + k;
            const double2 w1 = pc_tw(tab, NB, STRIDE * k), w2 = pc_cmul(w1, w1), w3 = pc_cmul(w2, w1);
            double2 v0, v1, v2, v3;
            pc_bfly4(pc_sm[PC_PAD(jj)], pc_cmul(w1, pc_sm[PC_PAD(jj + T4)]), pc_cmul(w2, pc_sm[PC_PAD(jj + 2 * T4)]),
                     pc_cmul(w3, pc_sm[PC_PAD(jj + 3 * T4)]), v0, v1, v2, v3);
            __stcs(q + (size_t)j0 * STRIDE, v0), __stcs(q + (size_t)(j0 + ns) * STRIDE, v1);
            __stcs(q + (size_t)(j0 + 2 * ns) * STRIDE, v2), __stcs(q + (size_t)(j0 + 3 * ns) * STRIDE, v3);
        }
    } else {
        const int T2 = N >> 1;
        for (int jj = j; jj < T2; jj += T) {  // ns = N / 2, k = jj
            const double2 a0 = pc_sm[PC_PAD(jj)], a1 = pc_cmul(pc_tw(tab, NB, STRIDE * jj), pc_sm[PC_PAD(jj + T2)]);
            __stcs(q + (size_t)jj * STRIDE, pc_add(a0, a1)), __stcs(q + (size_t)(jj + ns) * STRIDE, pc_sub(a0, a1));
        }
    }
}

// One block per (point, detector).  Work items = (tile of PC_TA rows a, tile of PC_TB columns b, slice of the frequency
// axis), dealt to the warps round robin.  A lane takes one frequency at a time: x_a[n] and x_a[-n] of the tile's rows and
// x_b[n] of its columns go to registers (coalesced 16-byte loads; the block's warps re-read the same 100-odd KB, which
// L1 serves) and all PC_TA x PC_TB pairs are updated from registers -- 8 FMA per pair and frequency, 9 loads per 72 FMA.
// The items' sums are reduced by shuffles and added to the pair's accumulator in shared memory.
#define PC_TA 3
#define PC_TB 3
__global__ void __launch_bounds__(PC_THREADS, 2)
    ile_overlap_uv_kernel(int32_t M, int32_t N, int32_t nsplit, const double2 *__restrict__ x, const PcWeight wt, double2 *__restrict__ U,
                          double2 *__restrict__ V)
{
    extern __shared__ double2 pc_sm[];
    double *acc = reinterpret_cast<double *>(pc_sm);  // [M*M][4]
    const size_t pk = blockIdx.x;                     // point * K + k
    const double2 *xk = x + pk * M * N;
    const double *Ss = wt.S ? wt.S + pk * N : nullptr;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, npairs = M * M;
    for (int i = threadIdx.x; i < 4 * npairs; i += PC_THREADS) acc[i] = 0.0;
    __syncthreads();
    const int ta = (M + PC_TA - 1) / PC_TA, tb = (M + PC_TB - 1) / PC_TB, items = ta * tb * nsplit;
    const int slice = ((N + nsplit - 1) / nsplit + 31) & ~31;
    for (int it = warp; it < items; it += PC_THREADS / 32) {
        const int sp = it % nsplit, tile = it / nsplit, a0 = (tile / tb) * PC_TA, b0 = (tile % tb) * PC_TB;
        const int lo = sp * slice, hi = min(lo + slice, N);
        double su[PC_TA][PC_TB][4];
#pragma unroll
        for (int i = 0; i < PC_TA; ++i)
#pragma unroll
            for (int j = 0; j < PC_TB; ++j) su[i][j][0] = su[i][j][1] = su[i][j][2] = su[i][j][3] = 0.0;
#pragma unroll 2
        for (int n = lo + lane; n < hi; n += 32) {
            const int nm = (N - n) & (N - 1);
            double2 p[PC_TA], m[PC_TA], q[PC_TB];
#pragma unroll
            for (int i = 0; i < PC_TA; ++i) {
                const int a = min(a0 + i, M - 1);  // rows past M repeat the last one; their sums are dropped
                p[i] = __ldg(xk + (size_t)a * N + n);
                m[i] = __ldg(xk + (size_t)a * N + nm);
            }
#pragma unroll
            for (int j = 0; j < PC_TB; ++j) q[j] = __ldg(xk + (size_t)min(b0 + j, M - 1) * N + n);
            if (Ss) {  // weight on the right factor
                const double g = pc_weight(Ss, wt, N, n);
#pragma unroll
                for (int j = 0; j < PC_TB; ++j) q[j].x *= g, q[j].y *= g;
            }
#pragma unroll
            for (int i = 0; i < PC_TA; ++i)
#pragma unroll
                for (int j = 0; j < PC_TB; ++j) {
                    su[i][j][0] += p[i].x * q[j].x + p[i].y * q[j].y;  // conj(x_a) x_b
                    su[i][j][1] += p[i].x * q[j].y - p[i].y * q[j].x;
                    su[i][j][2] += m[i].x * q[j].x - m[i].y * q[j].y;  // x_a(-f) x_b(f)
                    su[i][j][3] += m[i].x * q[j].y + m[i].y * q[j].x;
                }
        }
#pragma unroll
        for (int i = 0; i < PC_TA; ++i)
#pragma unroll
            for (int j = 0; j < PC_TB; ++j) {
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    double v = su[i][j][c];
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                    if (lane == 0 && a0 + i < M && b0 + j < M) atomicAdd(&acc[4 * ((a0 + i) * M + b0 + j) + c], v);
                }
            }
    }
    __syncthreads();
    for (int pr = threadIdx.x; pr < npairs; pr += PC_THREADS) {
        U[pk * npairs + pr] = make_double2(acc[4 * pr + 0], acc[4 * pr + 1]);
        V[pk * npairs + pr] = make_double2(acc[4 * pr + 2], acc[4 * pr + 3]);
    }
}

// First level of the two-level transform, N = 8 N2 (16384 ... 65536 points): with n = n2 + N2 n1 and i = i1 + 8 i2,
//   X[i1 + 8 i2] = sum_{n2} W_{N2}^{n2 i2} [ W_N^{n2 i1} sum_{n1} c[n2 + N2 n1] W_8^{n1 i1} ].
// Thread n2 does the bracket -- eight inputs at stride N2 (coalesced across threads), one radix-8 butterfly, the twiddles -- and
// writes row i1 of Z[series][8][N2]; the second level is the radix-8 kernel with STRIDE = 8 on every row.
__global__ void __launch_bounds__(PC_THREADS)
    ile_overlap_q_split8_kernel(int32_t M, int32_t N, const double2 *__restrict__ tab, const double2 *__restrict__ x,
                                const double2 *__restrict__ d, const PcWeight wt, double2 *__restrict__ Z)
{
    const size_t series = blockIdx.y;
    const int N2 = N >> 3, n2 = blockIdx.x * blockDim.x + threadIdx.x;
    if (n2 >= N2) return;
    const double2 *xs = x + series * N, *ds = d + (series / M) * N, *ph = tab + N / 2;
    const double *Ss = wt.S ? wt.S + (series / M) * N : nullptr;
    double2 u[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) u[r] = pc_input(xs, ds, ph, Ss, wt, N, n2 + r * N2);
    pc_bfly8(u);
    const double2 w1 = pc_tw(tab, N, n2);
    double2 w = w1;
    double2 *z = Z + series * N + n2;
    z[0] = u[0];
#pragma unroll
    for (int r = 1; r < 8; ++r) {
        z[(size_t)r * N2] = pc_cmul(w, u[r]);
        w = pc_cmul(w, w1);
    }
}

// Few modes (M <= PC_MS): one block per (point, detector); warp (a, slice) takes row a and one of PC_NS slices of the frequency
// axis, a lane one frequency at a time, and keeps the sums of the pairs (a, b >= a) in registers.  U is Hermitian and V symmetric
// by their definitions (U_ba = conj(U_ab); V_ba = sum_n x_b[-n] x_a[n] is the same set of products as V_ab), so only b >= a is
// accumulated and the mirror entries are filled from it.  The M row warps of a slice read the same spectra: once from L2 (the
// Q kernel of the batch has just brought them on chip), then from L1.
#define PC_MS 5
#define PC_NS 4
#define PC_UV_THREADS (32 * PC_MS * PC_NS)
template <bool WEIGHTED>
__global__ void __launch_bounds__(PC_UV_THREADS, 1)
    ile_overlap_uv_small_kernel(int32_t M, int32_t N, const double2 *__restrict__ x, const PcWeight wt, double2 *__restrict__ U,
                                double2 *__restrict__ V)
{
    __shared__ double acc[PC_MS * PC_MS * 4];
    const size_t pk = blockIdx.x;  // point * K + k
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, a = warp % PC_MS, slice = warp / PC_MS;
    const int nb = M - a;  // pairs (a, a + i), i < nb; warps with a >= M idle
    const double2 *xk = x + pk * M * N, *xa = xk + (size_t)a * N;
    const double *Ss = WEIGHTED ? wt.S + pk * N : nullptr;
    for (int i = threadIdx.x; i < PC_MS * PC_MS * 4; i += PC_UV_THREADS) acc[i] = 0.0;
    __syncthreads();
    if (nb > 0) {
        double su[PC_MS][4];
#pragma unroll
        for (int i = 0; i < PC_MS; ++i) su[i][0] = su[i][1] = su[i][2] = su[i][3] = 0.0;
        const int len = N / PC_NS, lo = slice * len, hi = slice == PC_NS - 1 ? N : lo + len;
#pragma unroll 2
        for (int n = lo + lane; n < hi; n += 32) {
            const int nm = (N - n) & (N - 1);
            double2 pa = __ldg(xa + n), ma = __ldg(xa + nm), q[PC_MS];
#pragma unroll
            for (int i = 0; i < PC_MS; ++i) q[i] = __ldg(xa + (size_t)(i < nb ? i : nb - 1) * N + n);  // columns past M repeat the last one
            if (WEIGHTED) {  // weight on the left factors: conj(x_a) g x_b and x_a(-f) g x_b(f)
                const double g = pc_weight(Ss, wt, N, n);
                pa.x *= g, pa.y *= g, ma.x *= g, ma.y *= g;
            }
#pragma unroll
            for (int i = 0; i < PC_MS; ++i) {
                su[i][0] += pa.x * q[i].x + pa.y * q[i].y;  // conj(x_a) x_b
                su[i][1] += pa.x * q[i].y - pa.y * q[i].x;
                su[i][2] += ma.x * q[i].x - ma.y * q[i].y;  // x_a(-f) x_b(f)
                su[i][3] += ma.x * q[i].y + ma.y * q[i].x;
            }
        }
#pragma unroll
        for (int i = 0; i < PC_MS; ++i)
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                double v = su[i][c];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                if (lane == 0 && i < nb) atomicAdd(&acc[(a * PC_MS + i) * 4 + c], v);
            }
    }
    __syncthreads();
    if (threadIdx.x < PC_MS * PC_MS) {
        const int ra = threadIdx.x / PC_MS, i = threadIdx.x % PC_MS, rb = ra + i;
        if (ra < M && rb < M) {
            const double *s4 = acc + (ra * PC_MS + i) * 4;
            const double2 u = make_double2(s4[0], i == 0 ? 0.0 : s4[1]), v = make_double2(s4[2], s4[3]);
            U[pk * M * M + ra * M + rb] = u, V[pk * M * M + ra * M + rb] = v;
            if (i) U[pk * M * M + rb * M + ra] = make_double2(u.x, -u.y), V[pk * M * M + rb * M + ra] = v;
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// U, V for few modes (M <= PC_MS) and N >= 512: persistent blocks fed by bulk copies (cp.async.bulk + mbarrier), so the bytes in
// flight do not depend on registers or occupancy -- round 2a's warp-per-row kernel was bound by the latency of its own loads
// (1.4 TB/s).  A work unit is (point-detector pk, chunk c): the PC_CH frequency pairs (n, N - n), n = c PC_CH + 1 + t, of all M
// modes, i.e. per mode one contiguous run x[n ..] and one contiguous run of mirrors x[N - (c + 1) PC_CH ..] -- 2 M bulk copies of 4 KB
// into one of PC_STG stage buffers.  Thread t owns pair t: both frequencies' terms of U_ab and V_ab, b >= a, are local (U Hermitian, V
// symmetric by their definitions), 16 FMA per pair (a, b), sums in registers across the chunks of a pk.  n = 0 and n = N / 2 pair
// with themselves and are added by the threads that flush.  Units are dealt to the blocks in contiguous
// ranges, so a pk is finished by one block or split between two neighbours: partial sums go to global memory with atomic adds onto
// zeros (two commuting addends: the result does not depend on their order).
// ------------------------------------------------------------------------------------------------------------
#define PC_CH 256
#define PC_STG 4

__device__ __forceinline__ void pc_mbar_init(uint32_t bar, uint32_t count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count)); }
__device__ __forceinline__ void pc_mbar_expect(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void pc_mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n.reg .pred p;\nPC_WAIT:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra PC_DONE;\nbra PC_WAIT;\nPC_DONE:\n}" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void pc_bulk_load(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}

// Sums of NV (a power of two <= 32) values over the 32 lanes of a warp by recursive halving: in a round a lane keeps half of its
// values and sends the other half across (lane ^ w), so 32 values cost 31 shuffles and not 160.  Returns the index of the value whose
// total ends up in v[0] of this lane (lanes that agree in the bits used hold the same total).
template <int NV>
__device__ __forceinline__ int pc_warp_sums(double (&v)[NV], int lane)
{
    int idx = 0, bit = 1, cnt = NV;
#pragma unroll
    for (int w = 16; w >= 1; w >>= 1) {
        if (cnt > 1) {
            const bool up = (lane & w) != 0;
#pragma unroll
            for (int i = 0; i < NV / 2; ++i)
                if (i < cnt / 2) {
                    const double keep = up ? v[2 * i + 1] : v[2 * i], send = up ? v[2 * i] : v[2 * i + 1];
                    v[i] = keep + __shfl_xor_sync(0xffffffffu, send, w);
                }
            if (up) idx |= bit;
            bit <<= 1, cnt >>= 1;
        } else {
            v[0] += __shfl_xor_sync(0xffffffffu, v[0], w);
        }
    }
    return idx;
}

// Threads 0 .. PC_CH-1 accumulate U, threads PC_CH .. 2 PC_CH-1 accumulate V of the same PC_CH frequency pairs (half the sums per
// thread: 16 warps of <= 128 registers per SM instead of 8 warps of 250).
template <int MM, bool WEIGHTED>
__global__ void __launch_bounds__(2 * PC_CH, 1)
    ile_overlap_uv_bulk_kernel(int32_t N, int32_t n_pk, const double2 *__restrict__ x, const PcWeight wt, double *__restrict__ U, double *__restrict__ V)
{
    constexpr int NPAIR = MM * (MM + 1) / 2;
    constexpr int NV = 2 * NPAIR <= 2 ? 2 : 2 * NPAIR <= 8 ? 8 : 2 * NPAIR <= 16 ? 16 : 32;
    constexpr uint32_t X_BYTES = PC_CH * 16, S_LEFT = (PC_CH + 2) * 8, S_MIRR = PC_CH * 8;
    constexpr uint32_t DC_OFF = MM * 2 * X_BYTES + (WEIGHTED ? S_LEFT + S_MIRR : 0);  // x_a[0] of the pk, with chunk 0 only
    constexpr uint32_t STAGE = DC_OFF + 128;
    extern __shared__ __align__(128) unsigned char pc_raw[];
    __shared__ __align__(8) uint64_t full[PC_STG];
    __shared__ double red[2][PC_CH / 32][NV];
    __shared__ double2 self0[MM], selfN[MM];  // x_a[0], x_a[N / 2] of the pk under way: the two frequencies that are their own mirrors
    __shared__ double wself[2];               // and their weights
    const uint32_t sm0 = (uint32_t)__cvta_generic_to_shared(pc_raw), bar0 = (uint32_t)__cvta_generic_to_shared(full);
    const int half = threadIdx.x / PC_CH, t = threadIdx.x % PC_CH, lane = t & 31, warp = t >> 5;
    const int nch = (N / 2) / PC_CH;
    const long long units = (long long)n_pk * nch;
    const long long u_lo = units * blockIdx.x / gridDim.x, u_hi = units * (blockIdx.x + 1) / gridDim.x;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < PC_STG; ++s) pc_mbar_init(bar0 + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    auto issue = [&](long long u) {  // thread 0: the copies of unit u into stage (u - u_lo) % PC_STG
        const int s = (int)((u - u_lo) % PC_STG);
        const size_t pk = (size_t)(u / nch);
        const int c = (int)(u % nch);
        const uint32_t bar = bar0 + 8 * s, dst = sm0 + s * STAGE;
        pc_mbar_expect(bar, DC_OFF + (c == 0 ? MM * 16 : 0));
#pragma unroll
        for (int a = 0; a < MM; ++a) {
            const double2 *xa = x + (pk * MM + a) * N;
            if (c == 0) pc_bulk_load(dst + DC_OFF + a * 16, xa, 16, bar);
            pc_bulk_load(dst + (2 * a) * X_BYTES, xa + c * PC_CH + 1, X_BYTES, bar);
            pc_bulk_load(dst + (2 * a + 1) * X_BYTES, xa + N - (c + 1) * PC_CH, X_BYTES, bar);
        }
        if (WEIGHTED) {
            const double *Ss = wt.S + pk * N;
            pc_bulk_load(dst + 2 * MM * X_BYTES, Ss + c * PC_CH, S_LEFT, bar);  // from the even index below n
            pc_bulk_load(dst + 2 * MM * X_BYTES + S_LEFT, Ss + N - (c + 1) * PC_CH, S_MIRR, bar);
        }
    };
    if (threadIdx.x == 0)
        for (long long u = u_lo; u < u_hi && u < u_lo + PC_STG; ++u) issue(u);

    bool dc_due = false, ny_due = false;
    double acc[NV];  // pair p: (re, im) at 2 p, 2 p + 1
#pragma unroll
    for (int i = 0; i < NV; ++i) acc[i] = 0.0;

    for (long long u = u_lo; u < u_hi; ++u) {
        const int s = (int)((u - u_lo) % PC_STG);
        const size_t pk = (size_t)(u / nch);
        const int c = (int)(u % nch);
        pc_mbar_wait(bar0 + 8 * s, (uint32_t)(((u - u_lo) / PC_STG) & 1));
        const unsigned char *st = pc_raw + (size_t)s * STAGE;
        const int n = c * PC_CH + 1 + t;  // n = N / 2 (its own mirror) is counted twice here: the flush takes one copy back
        double wl = 1.0, wm = 1.0;
        if (WEIGHTED) {
            const double f = (double)n * wt.df;
            const bool in = f > wt.fmin && f < wt.fmax;
            const double *sl = reinterpret_cast<const double *>(st + 2 * MM * X_BYTES);
            wl = in ? wt.scale / sl[t + 1] : 0.0;
            wm = in ? wt.scale / sl[PC_CH + 2 + PC_CH - 1 - t] : 0.0;
        }
        // left factors of the two terms of a pair: U_ab = conj(x_a[n]) g[n] x_b[n] + conj(x_a[-n]) g[-n] x_b[-n]  (threads of half 0),
        // V_ab = x_a[-n] g[n] x_b[n] + x_a[n] g[-n] x_b[-n]  (half 1); the right factors x_b[n], x_b[-n] carry the weights
        double2 X1[MM], X2[MM], L[MM], R[MM];
#pragma unroll
        for (int a = 0; a < MM; ++a) {
            L[a] = reinterpret_cast<const double2 *>(st + (2 * a) * X_BYTES)[t];
            R[a] = reinterpret_cast<const double2 *>(st + (2 * a + 1) * X_BYTES)[PC_CH - 1 - t];
            if (c == nch - 1 && threadIdx.x == PC_CH - 1) selfN[a] = L[a];  // n = N / 2: this thread counts it twice, the flush takes one back
            if (c == 0 && threadIdx.x == 0) self0[a] = reinterpret_cast<const double2 *>(st + DC_OFF)[a];
            X1[a] = half ? R[a] : make_double2(L[a].x, -L[a].y);
            X2[a] = half ? L[a] : make_double2(R[a].x, -R[a].y);
            if (WEIGHTED) L[a].x *= wl, L[a].y *= wl, R[a].x *= wm, R[a].y *= wm;
        }
        if (c == nch - 1 && threadIdx.x == PC_CH - 1) wself[1] = wl;
        if (c == 0 && threadIdx.x == 0) {
            double w0 = 1.0;
            if (WEIGHTED) w0 = (0.0 > wt.fmin && 0.0 < wt.fmax) ? wt.scale / reinterpret_cast<const double *>(st + 2 * MM * X_BYTES)[0] : 0.0;
            wself[0] = w0;
        }
        {
            int p = 0;
#pragma unroll
            for (int a = 0; a < MM; ++a)
#pragma unroll
                for (int b = a; b < MM; ++b, ++p) {
                    acc[2 * p] += X1[a].x * L[b].x - X1[a].y * L[b].y + X2[a].x * R[b].x - X2[a].y * R[b].y;
                    acc[2 * p + 1] += X1[a].x * L[b].y + X1[a].y * L[b].x + X2[a].x * R[b].y + X2[a].y * R[b].x;
                }
        }
        dc_due = dc_due || c == 0;
        ny_due = ny_due || c == nch - 1;
        const bool flush = u + 1 == u_hi || (u + 1) % nch == 0;  // the block's last unit, or the pk's
        __syncthreads();  // every thread has read stage s (an mbarrier per stage that lets the warps drift apart was measured: 64 vs 51 us)
        if (threadIdx.x == 0 && u + PC_STG < u_hi) issue(u + PC_STG);
        if (flush) {
            const int idx = pc_warp_sums<NV>(acc, lane);
            red[half][warp][idx] = acc[0];  // lanes that hold the same total write the same value
#pragma unroll
            for (int i = 0; i < NV; ++i) acc[i] = 0.0;
            __syncthreads();
            if (t < NPAIR) {
                int a = 0, b = t;  // pair index -> (a, b)
                while (b >= MM - a) b -= MM - a, ++a;
                b += a;
                double re = 0.0, im = 0.0;
#pragma unroll
                for (int w = 0; w < PC_CH / 32; ++w) re += red[half][w][2 * t], im += red[half][w][2 * t + 1];
                // the two frequencies that are their own mirrors: + n = 0 (came with chunk 0), - one of the two copies of n = N / 2 that
                // the last chunk's last thread has added
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    if (e == 0 ? dc_due : ny_due) {
                        const double2 xa = e == 0 ? self0[a] : selfN[a], xb = e == 0 ? self0[b] : selfN[b];
                        const double w0 = e == 0 ? wself[0] : -wself[1];
                        const double2 xw = make_double2(w0 * xb.x, w0 * xb.y);
                        if (half == 0) re += xa.x * xw.x + xa.y * xw.y, im += xa.x * xw.y - xa.y * xw.x;
                        else re += xa.x * xw.x - xa.y * xw.y, im += xa.x * xw.y + xa.y * xw.x;
                    }
                }
                double *Mk = (half == 0 ? U : V) + 2 * pk * MM * MM;
                const double ims = half == 0 ? -im : im;  // U_ba = conj(U_ab), V_ba = V_ab; the diagonal of U is real
                atomicAdd(Mk + 2 * (a * MM + b), re);
                if (a != b || half == 1) atomicAdd(Mk + 2 * (a * MM + b) + 1, im);
                if (a != b) atomicAdd(Mk + 2 * (b * MM + a), re), atomicAdd(Mk + 2 * (b * MM + a) + 1, ims);
            }
            __syncthreads();  // red is free again
            dc_due = ny_due = false;
        }
    }
}

__global__ void __launch_bounds__(256) ile_overlap_zero_kernel(double2 *__restrict__ U, double2 *__restrict__ V, long long n)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        U[i] = make_double2(0.0, 0.0), V[i] = make_double2(0.0, 0.0);
}

template <int MM>
static cudaError_t pc_launch_uv_bulk(int32_t N, int32_t n_pk, const double2 *x, const PcWeight &wt, double2 *U, double2 *V, int sm_count,
                                     cudaStream_t st)
{
    const long long n_uv = (long long)n_pk * MM * MM;
    ile_overlap_zero_kernel<<<(unsigned)((n_uv + 255) / 256 < 1024 ? (n_uv + 255) / 256 : 1024), 256, 0, st>>>(U, V, n_uv);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const long long units = (long long)n_pk * ((N / 2) / PC_CH);
    const unsigned grid = (unsigned)(units < sm_count ? units : sm_count);
    if (wt.S) {
        const size_t smem = (size_t)PC_STG * (MM * 2 * PC_CH * 16 + (PC_CH + 2) * 8 + PC_CH * 8 + 128);
        e = cudaFuncSetAttribute(ile_overlap_uv_bulk_kernel<MM, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        ile_overlap_uv_bulk_kernel<MM, true><<<grid, 2 * PC_CH, smem, st>>>(N, n_pk, x, wt, (double *)U, (double *)V);
    } else {
        const size_t smem = (size_t)PC_STG * (MM * 2 * PC_CH * 16 + 128);
        e = cudaFuncSetAttribute(ile_overlap_uv_bulk_kernel<MM, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        ile_overlap_uv_bulk_kernel<MM, false><<<grid, 2 * PC_CH, smem, st>>>(N, n_pk, x, wt, (double *)U, (double *)V);
    }
    return cudaGetLastError();
}

// Library-owned state of the pre-computation, one per device: the twiddle / start-time phase table (rebuilt in stream order when
// the grid or the start time changes) and the first-level output Z of the two-level transform (grown on demand).  Both are
// shared by every call on the device, so calls are serialised: g_pc_mutex covers the host side (the bookkeeping below and the
// launches of one call), and every call waits on the event recorded at the end of the previous one, so that a call on another
// stream neither reads a half-written table nor overwrites table / Z under kernels that still use them.  Never freed.
struct PcDevice {
    double2 *tab;
    int tab_n;
    double tab_alpha;
    double2 *z;
    size_t z_cap;
    cudaEvent_t done;  // end of the most recent call's work on this device
    bool have_done;
};
static PcDevice g_pc[64];
static std::mutex g_pc_mutex;

static cudaError_t pc_launch_locked(PcDevice &pd, int dev, int32_t n_points, int32_t K, int32_t M, int32_t N, double fs_hz, double t0_q_s,
                                    const double2 *x, const double2 *d, const double *S, double f_min_hz, double f_max_hz, double scale,
                                    double2 *Q, double2 *U, double2 *V, int32_t max_smem_optin, cudaStream_t st);

cudaError_t ile_launch_precompute(int32_t n_points, int32_t K, int32_t M, int32_t N, double fs_hz, double t0_q_s, const double2 *x,
                                  const double2 *d, const double *S, double f_min_hz, double f_max_hz, double scale, double2 *Q, double2 *U,
                                  double2 *V, int32_t max_smem_optin, cudaStream_t st)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_pc_mutex);
    PcDevice &pd = g_pc[dev];
    if (!pd.have_done) {
        e = cudaEventCreateWithFlags(&pd.done, cudaEventDisableTiming);
        if (e != cudaSuccess) return e;
        pd.have_done = true;
    } else {
        e = cudaStreamWaitEvent(st, pd.done, 0);  // no-op when the previous call was made on this stream
        if (e != cudaSuccess) return e;
    }
    e = pc_launch_locked(pd, dev, n_points, K, M, N, fs_hz, t0_q_s, x, d, S, f_min_hz, f_max_hz, scale, Q, U, V, max_smem_optin, st);
    const cudaError_t er = cudaEventRecord(pd.done, st);  // also after an error: part of the call may be in flight
    return e != cudaSuccess ? e : er;
}

static cudaError_t pc_launch_locked(PcDevice &pd, int dev, int32_t n_points, int32_t K, int32_t M, int32_t N, double fs_hz, double t0_q_s,
                                    const double2 *x, const double2 *d, const double *S, double f_min_hz, double f_max_hz, double scale,
                                    double2 *Q, double2 *U, double2 *V, int32_t max_smem_optin, cudaStream_t st)
{
    int log2n = 0;
    while ((1 << log2n) < N) ++log2n;
    if ((1 << log2n) != N || N < 2 || N > 65536) return cudaErrorInvalidValue;
    const bool radix8 = N >= 512, two_level = N > 8192;
    const int NS = two_level ? N / 8 : N;  // length of the shared-memory transform
    const size_t smem = radix8 ? (size_t)(NS + NS / 8) * 16 : (size_t)2 * N * 16;
    if (smem > (size_t)max_smem_optin) return cudaErrorInvalidValue;
    cudaError_t e = cudaSuccess;
    // U, V kernel for many modes: enough frequency slices that a block's 8 warps all have work items
    const int tiles = ((M + PC_TA - 1) / PC_TA) * ((M + PC_TB - 1) / PC_TB);
    int nsplit = (PC_THREADS / 32 + tiles - 1) / tiles;
    while (nsplit > 1 && N / nsplit < 32) --nsplit;
    const size_t smem_uv = (size_t)M * M * 32;
    if (!pd.tab) {
        double2 *t = nullptr;
        e = cudaMalloc(&t, (size_t)(32768 + 65536) * sizeof(double2));
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(ile_overlap_q_radix8_kernel<512, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(4608 * 16));
        if (e == cudaSuccess) e = cudaFuncSetAttribute(ile_overlap_q_radix8_kernel<1024, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(9216 * 16));
        if (e == cudaSuccess) e = cudaFuncSetAttribute(ile_overlap_q_radix8_kernel<512, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(4608 * 16));
        if (e == cudaSuccess) e = cudaFuncSetAttribute(ile_overlap_q_radix8_kernel<1024, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(9216 * 16));
        if (e != cudaSuccess) {
            cudaFree(t);
            return e;
        }
        pd.tab = t, pd.tab_n = 0;
    }
    double2 *tab = pd.tab;
    const double alpha = fs_hz * t0_q_s / (double)N;
    if (pd.tab_n != N || pd.tab_alpha != alpha) {
        pd.tab_n = 0;  // the table belongs to no grid until its kernel has been launched
        ile_overlap_tables_kernel<<<(N + PC_THREADS - 1) / PC_THREADS, PC_THREADS, 0, st>>>(N, alpha, tab);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        pd.tab_n = N, pd.tab_alpha = alpha;
    }
    PcWeight wt;
    wt.S = S, wt.df = fs_hz / (double)N, wt.fmin = f_min_hz, wt.fmax = f_max_hz, wt.scale = scale;
    // One launch per kernel over all points: cutting the call into L2-sized batches (so that the U, V kernel finds the spectra its
    // Q kernel has just read) was measured and lost -- 0.24 ms against 0.19 ms for 256 points of 3 x 5 x 2048: both kernels are
    // bound by the latency of a block's own load - compute - store chain, and batches serialise those chains.
    const unsigned n_series = (unsigned)((size_t)n_points * K * M);
    if (two_level) {
        const size_t need = (size_t)n_series * N;
        if (need > pd.z_cap) {
            e = cudaStreamSynchronize(st);  // st has waited for the previous call, whichever stream it ran on
            if (e != cudaSuccess) return e;
            cudaFree(pd.z);
            pd.z = nullptr, pd.z_cap = 0;
            e = cudaMalloc(&pd.z, need * sizeof(double2));
            if (e != cudaSuccess) return e;
            pd.z_cap = need;
        }
        double2 *Z = pd.z;
        ile_overlap_q_split8_kernel<<<dim3((unsigned)(NS / PC_THREADS), n_series), PC_THREADS, 0, st>>>(M, N, tab, x, d, wt, Z);
        switch (NS) {  // rows of the first level: plain loads, output stride 8, every eighth twiddle of the long table
            case 2048: ile_overlap_q_radix8_kernel<256, 8><<<n_series * 8, 256, smem, st>>>(M, NS, tab, Z, d, wt, Q); break;
            case 4096: ile_overlap_q_radix8_kernel<512, 8><<<n_series * 8, 512, smem, st>>>(M, NS, tab, Z, d, wt, Q); break;
            default: ile_overlap_q_radix8_kernel<1024, 8><<<n_series * 8, 1024, smem, st>>>(M, NS, tab, Z, d, wt, Q); break;
        }
    } else if (radix8) {
        switch (N) {
            case 512: ile_overlap_q_radix8_kernel<64, 1><<<n_series, 64, smem, st>>>(M, N, tab, x, d, wt, Q); break;
            case 1024: ile_overlap_q_radix8_kernel<128, 1><<<n_series, 128, smem, st>>>(M, N, tab, x, d, wt, Q); break;
            case 2048: ile_overlap_q_radix8_kernel<256, 1><<<n_series, 256, smem, st>>>(M, N, tab, x, d, wt, Q); break;
            case 4096: ile_overlap_q_radix8_kernel<512, 1><<<n_series, 512, smem, st>>>(M, N, tab, x, d, wt, Q); break;
            default: ile_overlap_q_radix8_kernel<1024, 1><<<n_series, 1024, smem, st>>>(M, N, tab, x, d, wt, Q); break;
        }
    } else {
        if (S) return cudaErrorInvalidValue;  // short transforms take whitened spectra only
        ile_overlap_q_stockham_kernel<0><<<n_series, PC_THREADS, smem, st>>>(M, N, log2n, tab, x, d, Q);
    }
    const unsigned n_pk = (unsigned)(n_points * K);
    if (M <= PC_MS && N >= 2 * PC_CH && ((uintptr_t)S & 15) == 0) {  // bulk copies need 16-byte aligned sources (x is double2)
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        switch (M) {
            case 1: return pc_launch_uv_bulk<1>(N, (int32_t)n_pk, x, wt, U, V, sms, st);
            case 2: return pc_launch_uv_bulk<2>(N, (int32_t)n_pk, x, wt, U, V, sms, st);
            case 3: return pc_launch_uv_bulk<3>(N, (int32_t)n_pk, x, wt, U, V, sms, st);
            case 4: return pc_launch_uv_bulk<4>(N, (int32_t)n_pk, x, wt, U, V, sms, st);
            default: return pc_launch_uv_bulk<5>(N, (int32_t)n_pk, x, wt, U, V, sms, st);
        }
    }
    if (M <= PC_MS && S) ile_overlap_uv_small_kernel<true><<<n_pk, PC_UV_THREADS, 0, st>>>(M, N, x, wt, U, V);
    else if (M <= PC_MS) ile_overlap_uv_small_kernel<false><<<n_pk, PC_UV_THREADS, 0, st>>>(M, N, x, wt, U, V);
    else ile_overlap_uv_kernel<<<n_pk, PC_THREADS, smem_uv, st>>>(M, N, nsplit, x, wt, U, V);
    return cudaGetLastError();
}
