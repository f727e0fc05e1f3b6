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
//   ile_overlap_q_stockham_kernel  N <= 4096, one block per series: spectrum product and start-time phase on load, Stockham
//                                  autosort radix-4 passes (+ one radix-2) between two shared-memory buffers, natural order in
//                                  and out; elements per thread known at compile time
//   ile_overlap_q_kernel           N = 8192: in-place radix-2 with a bit-reversed load (one buffer fits shared memory)
//   ile_overlap_uv_kernel          one block per (detector, point): register-blocked tiles of pairs (a, b), lanes over frequencies
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

__global__ void __launch_bounds__(PC_THREADS)
    ile_overlap_q_kernel(int32_t M, int32_t N, int32_t log2n, const double2 *__restrict__ tab, const double2 *__restrict__ x,
                         const double2 *__restrict__ d, double2 *__restrict__ Q)
{
    extern __shared__ double2 pc_sm[];
    double2 *a = pc_sm;       // N points
    double2 *W = pc_sm + N;   // N / 2 twiddles exp(+2 pi i j / N)
    const size_t series = blockIdx.x;             // (point * K + k) * M + mode
    const double2 *xs = x + series * N;
    const double2 *ds = d + (series / M) * N;
    for (int j = threadIdx.x; j < N / 2; j += PC_THREADS) W[j] = tab[j];
    for (int n = threadIdx.x; n < N; n += PC_THREADS) {
        const double2 xv = __ldcs(xs + n), dv = pc_cmul(ds[n], tab[N / 2 + n]);
        const double2 v = make_double2(xv.x * dv.x + xv.y * dv.y, xv.x * dv.y - xv.y * dv.x);  // conj(x) d
        a[__brev((unsigned)n) >> (32 - log2n)] = v;
    }
    __syncthreads();
    for (int st = 1; st <= log2n; ++st) {
        const int half = 1 << (st - 1), tw = N >> st;
        for (int j = threadIdx.x; j < N / 2; j += PC_THREADS) {
            const int pos = j & (half - 1), i0 = ((j >> (st - 1)) << st) + pos, i1 = i0 + half;
            const double2 t = pc_cmul(W[pos * tw], a[i1]), u = a[i0];
            a[i0] = make_double2(u.x + t.x, u.y + t.y);
            a[i1] = make_double2(u.x - t.x, u.y - t.y);
        }
        __syncthreads();
    }
    double2 *q = Q + series * N;
    for (int i = threadIdx.x; i < N; i += PC_THREADS) __stcs(q + i, a[i]);
}

// One block per (point, detector).  Work items = (tile of PC_TA rows a, tile of PC_TB columns b, slice of the frequency
// axis), dealt to the warps round robin.  A lane takes one frequency at a time: x_a[n] and x_a[-n] of the tile's rows and
// x_b[n] of its columns go to registers (coalesced 16-byte loads; the block's warps re-read the same 100-odd KB, which
// L1 serves) and all PC_TA x PC_TB pairs are updated from registers -- 8 FMA per pair and frequency, 9 loads per 72 FMA.
// The items' sums are reduced by shuffles and added to the pair's accumulator in shared memory.
#define PC_TA 3
#define PC_TB 3
__global__ void __launch_bounds__(PC_THREADS, 2)
    ile_overlap_uv_kernel(int32_t M, int32_t N, int32_t nsplit, const double2 *__restrict__ x, double2 *__restrict__ U, double2 *__restrict__ V)
{
    extern __shared__ double2 pc_sm[];
    double *acc = reinterpret_cast<double *>(pc_sm);  // [M*M][4]
    const size_t pk = blockIdx.x;                     // point * K + k
    const double2 *xk = x + pk * M * N;
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

cudaError_t ile_launch_precompute(int32_t n_points, int32_t K, int32_t M, int32_t N, double fs_hz, double t0_q_s, const double2 *x,
                                  const double2 *d, double2 *Q, double2 *U, double2 *V, int32_t max_smem_optin, cudaStream_t st)
{
    int log2n = 0;
    while ((1 << log2n) < N) ++log2n;
    if ((1 << log2n) != N || N < 2 || N > 8192) return cudaErrorInvalidValue;
    const bool stockham = N <= 4096;
    const size_t smem = stockham ? (size_t)2 * N * 16 : (size_t)N * 16 + (size_t)(N / 2) * 16;
    if (smem > (size_t)max_smem_optin) return cudaErrorInvalidValue;
    auto stock = [&](auto kern, unsigned grid, const double2 *tab) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        kern<<<grid, PC_THREADS, smem, st>>>(M, N, log2n, tab, x, d, Q);
        return cudaSuccess;
    };
    cudaError_t e = cudaSuccess;
    if (!stockham) e = cudaFuncSetAttribute(ile_overlap_q_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    // U, V kernel: enough frequency slices that a block's 8 warps all have work items
    const int tiles = ((M + PC_TA - 1) / PC_TA) * ((M + PC_TB - 1) / PC_TB);
    int nsplit = (PC_THREADS / 32 + tiles - 1) / tiles;
    while (nsplit > 1 && N / nsplit < 32) --nsplit;
    const size_t smem_uv = (size_t)M * M * 32;
    // twiddles and start-time phases: one table per device, recomputed (in stream order) when the grid or the start time
    // changes.  Calls for DIFFERENT (n_q, fs t0) must not run concurrently on two streams of one device.
    static double2 *g_tab[64] = {nullptr};
    static int g_tab_n[64] = {0};
    static double g_tab_alpha[64] = {0.0};
    int dev = 0;
    e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    if (!g_tab[dev]) {
        e = cudaMalloc(&g_tab[dev], (size_t)(4096 + 8192) * sizeof(double2));
        if (e != cudaSuccess) return e;
    }
    double2 *tab = g_tab[dev];
    const double alpha = fs_hz * t0_q_s / (double)N;
    if (g_tab_n[dev] != N || g_tab_alpha[dev] != alpha) {
        ile_overlap_tables_kernel<<<(N + PC_THREADS - 1) / PC_THREADS, PC_THREADS, 0, st>>>(N, alpha, tab);
        g_tab_n[dev] = N, g_tab_alpha[dev] = alpha;
    }
    const unsigned n_series = (unsigned)((size_t)n_points * K * M);
    if (!stockham) ile_overlap_q_kernel<<<n_series, PC_THREADS, smem, st>>>(M, N, log2n, tab, x, d, Q);
    else if (N == 16 * PC_THREADS) e = stock(ile_overlap_q_stockham_kernel<16>, n_series, tab);
    else if (N == 8 * PC_THREADS) e = stock(ile_overlap_q_stockham_kernel<8>, n_series, tab);
    else if (N == 4 * PC_THREADS) e = stock(ile_overlap_q_stockham_kernel<4>, n_series, tab);
    else if (N == 2 * PC_THREADS) e = stock(ile_overlap_q_stockham_kernel<2>, n_series, tab);
    else e = stock(ile_overlap_q_stockham_kernel<0>, n_series, tab);
    if (e != cudaSuccess) return e;
    ile_overlap_uv_kernel<<<(unsigned)(n_points * K), PC_THREADS, smem_uv, st>>>(M, N, nsplit, x, U, V);
    return cudaGetLastError();
}
