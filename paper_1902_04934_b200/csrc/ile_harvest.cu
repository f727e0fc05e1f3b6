// ile_harvest.cu -- extrinsic posterior harvesting (readings H1-H3).
//
// "The code also produces reliable extrinsic parameter distributions ... we harvest joint intrinsic and
// extrinsic information with a single final iteration."
//   H1  ile_resample_*   systematic resampling of the Monte Carlo draws by their posterior weight w L_margT (eq. 4's integrand):
//                        maximum, per-tile inclusive prefix sums of W = exp(e - max), tile offsets, one binary search per output
//   H2, H3  ile_harvest_kernel   for the (few) harvested samples: the lnL_j series of eq. 7 / eq. 10 over the window once more,
//                        one warp per sample -- first bin of the maximum and its lnL (H3), and the time bin drawn from the
//                        normalised exp(lnL_j) of eq. 9's integrand with a supplied uniform (H2)
// Nothing here is shared with oracle/harvest.py.
#include <math_constants.h>

#include "ile_kernels.h"

#define HV_WARPS 4
#define RS_THREADS 256
#define RS_PER 4
#define RS_TILE (RS_THREADS * RS_PER)

// ------------------------------------------------------------------------------------------------------------
// H2 + H3: one warp per harvested sample
// ------------------------------------------------------------------------------------------------------------
template <bool INTERP>
__global__ void __launch_bounds__(HV_WARPS * 32) ile_harvest_kernel(IleEvalArgs a, long long n_sel, const long long *__restrict__ ids,
                                                                    const double *__restrict__ v_uniform, int32_t *__restrict__ argmax_bin,
                                                                    double *__restrict__ lnL_max, int32_t *__restrict__ drawn_bin)
{
    extern __shared__ __align__(16) unsigned char hv_smem[];
    const IleDevParams *__restrict__ P = a.params;
    const int K = P->n_det, M = P->n_modes, KM = K * M, n_q = P->n_q, n_t = P->n_t;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const size_t per_warp = (((size_t)KM * sizeof(double2) + (size_t)K * (sizeof(double) + sizeof(int32_t))) + 15) & ~(size_t)15;
    double2 *A = reinterpret_cast<double2 *>(hv_smem + warp * per_warp);
    double *phiS = reinterpret_cast<double *>(A + KM);  // [K] fractional parts of the arrival times (INTERP; reading R8')
    int32_t *i0S = reinterpret_cast<int32_t *>(phiS + K);
    const size_t pglob = (size_t)a.point0;
    const double2 *__restrict__ Qp = a.Q + pglob * (size_t)KM * n_q;

    for (long long w = (long long)blockIdx.x * HV_WARPS + warp; w < n_sel; w += (long long)gridDim.x * HV_WARPS) {
        const long long s = ids ? ids[w] : w;
        double quad = 0.0;
        int bad = s < 0 || s >= a.n_per_point;
        if (lane == 0 && !bad)
            quad = ile_setup_sample(P, a.U + pglob * (size_t)KM * M, a.V + pglob * (size_t)KM * M, a.ra[s], a.dec[s], a.t_ref[s],
                                    a.phi_ref[s], a.psi[s], a.incl[s], a.dist[s], A, M, i0S, &bad, INTERP ? phiS : nullptr);
        __syncwarp();
        bad = __shfl_sync(0xffffffffu, bad, 0);
        quad = __shfl_sync(0xffffffffu, quad, 0);
        if (bad) {  // reading R9: no window, nothing to harvest
            if (lane == 0) {
                argmax_bin[w] = -1;
                lnL_max[w] = -CUDART_INF;
                if (drawn_bin) drawn_bin[w] = -1;
            }
            __syncwarp();
            continue;
        }
        auto lnl = [&](int j) {  // lnL_j = Re sum conj(A) Q[i0_k + j] - quad  (eq. 7), same summation order as the direct kernel
            double acc = 0.0;
            for (int k = 0; k < K; ++k) {
                const double2 *Qk = Qp + (size_t)k * M * n_q + i0S[k] + j;
                const double ph = INTERP ? phiS[k] : 0.0, om = 1.0 - ph;
                for (int m = 0; m < M; ++m) {
                    const double2 c = A[k * M + m];
                    double2 q = __ldg(Qk + (size_t)m * n_q);
                    if (INTERP) {  // (1 - phi) Q[i] + phi Q[i + 1], as the direct kernel forms it
                        const double2 q1 = __ldg(Qk + (size_t)m * n_q + 1);
                        q.x = om * q.x + ph * q1.x, q.y = om * q.y + ph * q1.y;
                    }
                    acc = fma(c.x, q.x, fma(c.y, q.y, acc));
                }
            }
            return acc - quad;
        };
        // pass 1: maximum, its first bin, and sum exp(lnL - max) by a lane-local online log-sum-exp
        double mx = -CUDART_INF, sm = 0.0;
        int jm = 0x7fffffff;
        for (int j = lane; j < n_t; j += 32) {
            const double x = lnl(j);
            if (x > mx) {
                sm = sm * exp(mx - x) + 1.0;  // exp(-inf) = 0 on the first element
                mx = x;
                jm = j;
            } else {
                sm += exp(x - mx);
            }
        }
        double Mx = mx;
        int J = jm;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double om = __shfl_xor_sync(0xffffffffu, Mx, o);
            const int oj = __shfl_xor_sync(0xffffffffu, J, o);
            if (om > Mx || (om == Mx && oj < J)) Mx = om, J = oj;
        }
        const double S = warp_sum(mx > -CUDART_INF ? sm * exp(mx - Mx) : 0.0);
        if (lane == 0) {
            argmax_bin[w] = J;
            lnL_max[w] = Mx;
        }
        if (drawn_bin) {
            // pass 2: inclusive cumulative in bin order, 32 bins at a time; the first bin whose cumulative reaches v S
            const double target = v_uniform[w] * S;
            double carry = 0.0;
            int found = -1;
            for (int j0 = 0; j0 < n_t && found < 0; j0 += 32) {
                const int j = j0 + lane;
                double p = j < n_t ? exp(lnl(j) - Mx) : 0.0;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const double t = __shfl_up_sync(0xffffffffu, p, o);
                    if (lane >= o) p += t;
                }
                p += carry;
                const unsigned hit = __ballot_sync(0xffffffffu, j < n_t && p >= target);
                if (hit) found = j0 + __ffs(hit) - 1;
                carry = __shfl_sync(0xffffffffu, p, 31);
            }
            if (lane == 0) drawn_bin[w] = found < 0 ? n_t - 1 : found;
        }
        __syncwarp();
    }
}

cudaError_t ile_launch_harvest(const IleSizes &sz, const IleEvalArgs &a, long long n_sel, const long long *ids, const double *v_uniform,
                               int32_t *argmax_bin, double *lnL_max, int32_t *drawn_bin, cudaStream_t st)
{
    if (n_sel <= 0) return cudaSuccess;
    const size_t per_warp =
        (((size_t)sz.n_det * sz.n_modes * sizeof(double2) + (size_t)sz.n_det * (sizeof(double) + sizeof(int32_t))) + 15) & ~(size_t)15;
    long long blocks = (n_sel + HV_WARPS - 1) / HV_WARPS;
    const long long cap = (long long)sz.sm_count * 16;
    if (blocks > cap) blocks = cap;
    if (sz.interp)
        ile_harvest_kernel<true><<<(unsigned)blocks, HV_WARPS * 32, per_warp * HV_WARPS, st>>>(a, n_sel, ids, v_uniform, argmax_bin, lnL_max, drawn_bin);
    else
        ile_harvest_kernel<false><<<(unsigned)blocks, HV_WARPS * 32, per_warp * HV_WARPS, st>>>(a, n_sel, ids, v_uniform, argmax_bin, lnL_max, drawn_bin);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------
// H1: systematic resampling.  scratch: prefix [n] (inclusive cumulative of W inside its tile), tsum [n_tiles + 1]
// (tile totals, then inclusive tile cumulatives), gmax [1] as an order-preserving integer
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ long long rs_key(double x)  // monotone map double -> signed 64-bit
{
    const long long b = __double_as_longlong(x);
    return b >= 0 ? b : b ^ 0x7fffffffffffffffLL;
}
__device__ __forceinline__ double rs_unkey(long long k) { return __longlong_as_double(k >= 0 ? k : k ^ 0x7fffffffffffffffLL); }

__global__ void __launch_bounds__(RS_THREADS) ile_resample_max_kernel(long long n, const double *__restrict__ lnL,
                                                                      const double *__restrict__ log_w, long long *__restrict__ gmax)
{
    double mx = -CUDART_INF;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const double e = lnL[i] + (log_w ? log_w[i] : 0.0);
        if (e == e) mx = fmax(mx, e);
    }
    mx = warp_max(mx);
    if ((threadIdx.x & 31) == 0) atomicMax(gmax, rs_key(mx));
}

// one block per tile of RS_TILE consecutive samples: W = exp(e - max), inclusive prefix inside the tile, tile total
__global__ void __launch_bounds__(RS_THREADS) ile_resample_scan_kernel(long long n, const double *__restrict__ lnL,
                                                                       const double *__restrict__ log_w, const long long *__restrict__ gmax,
                                                                       double *__restrict__ prefix, double *__restrict__ tsum)
{
    __shared__ double wtot[RS_THREADS / 32];
    const double M = rs_unkey(*gmax);
    const long long base = (long long)blockIdx.x * RS_TILE + (long long)threadIdx.x * RS_PER;
    double v[RS_PER];
    double run = 0.0;
#pragma unroll
    for (int u = 0; u < RS_PER; ++u) {
        const long long i = base + u;
        double W = 0.0;
        if (i < n && M > -CUDART_INF) {
            const double e = lnL[i] + (log_w ? log_w[i] : 0.0);
            W = e == e ? exp(e - M) : 0.0;
        }
        run += W;
        v[u] = run;
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double inc = run;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const double t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) wtot[warp] = inc;
    __syncthreads();
    double off = inc - run;
    for (int w = 0; w < warp; ++w) off += wtot[w];
#pragma unroll
    for (int u = 0; u < RS_PER; ++u)
        if (base + u < n) prefix[base + u] = off + v[u];
    if (threadIdx.x == RS_THREADS - 1) tsum[blockIdx.x] = off + run;
}

// inclusive cumulative of the tile totals, in place, one block (sequential per thread chunk + block scan)
__global__ void __launch_bounds__(1024) ile_resample_tiles_kernel(long long n_tiles, double *__restrict__ tsum)
{
    __shared__ double wtot[32];
    const long long per = (n_tiles + 1023) / 1024;
    const long long lo = min((long long)threadIdx.x * per, n_tiles), hi = min(lo + per, n_tiles);
    double loc = 0.0;
    for (long long i = lo; i < hi; ++i) loc += tsum[i];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double inc = loc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const double t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) wtot[warp] = inc;
    __syncthreads();
    double run = inc - loc;
    for (int w = 0; w < warp; ++w) run += wtot[w];
    for (long long i = lo; i < hi; ++i) {
        run += tsum[i];
        tsum[i] = run;
    }
}

// output i: the smallest sample a whose inclusive cumulative weight exceeds p_i = (i + v0) / n_out * total
__global__ void __launch_bounds__(RS_THREADS) ile_resample_pick_kernel(long long n, long long n_tiles, long long n_out, double v0,
                                                                       const double *__restrict__ prefix, const double *__restrict__ tsum,
                                                                       long long *__restrict__ ids)
{
    const double total = tsum[n_tiles - 1];
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_out; i += (long long)gridDim.x * blockDim.x) {
        if (!(total > 0.0)) {
            ids[i] = -1;  // no finite weight
            continue;
        }
        const double p = __dmul_rn(__ddiv_rn(__dadd_rn((double)i, v0), (double)n_out), total);
        long long lo = 0, hi = n_tiles - 1;  // smallest tile whose inclusive cumulative exceeds p
        while (lo < hi) {
            const long long mid = (lo + hi) >> 1;
            if (tsum[mid] > p) hi = mid;
            else lo = mid + 1;
        }
        const double off = lo ? tsum[lo - 1] : 0.0;
        long long a = lo * RS_TILE, b = min(a + RS_TILE, n) - 1;  // smallest sample in the tile with off + prefix > p
        while (a < b) {
            const long long mid = (a + b) >> 1;
            if (off + prefix[mid] > p) b = mid;
            else a = mid + 1;
        }
        ids[i] = a;
    }
}

size_t ile_resample_scratch_doubles(long long n) { return (size_t)n + (size_t)((n + RS_TILE - 1) / RS_TILE) + 2; }

cudaError_t ile_launch_resample(const IleSizes &sz, long long n, const double *lnL, const double *log_w, long long n_out, double v0,
                                double *scratch, long long *ids, cudaStream_t st, int *n_launches)
{
    if (n <= 0 || n_out <= 0) return cudaSuccess;
    const long long n_tiles = (n + RS_TILE - 1) / RS_TILE;
    double *prefix = scratch, *tsum = scratch + n;
    long long *gmax = reinterpret_cast<long long *>(tsum + n_tiles);
    const long long neg_inf_key = 0x800FFFFFFFFFFFFFLL;  // rs_key(-inf) = bits(-inf) ^ 0x7fff... 
    cudaError_t e = cudaMemcpyAsync(gmax, &neg_inf_key, sizeof(long long), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return e;
    long long mb = (n + RS_THREADS - 1) / RS_THREADS;
    if (mb > (long long)sz.sm_count * 8) mb = (long long)sz.sm_count * 8;
    ile_resample_max_kernel<<<(unsigned)mb, RS_THREADS, 0, st>>>(n, lnL, log_w, gmax);
    ile_resample_scan_kernel<<<(unsigned)n_tiles, RS_THREADS, 0, st>>>(n, lnL, log_w, gmax, prefix, tsum);
    ile_resample_tiles_kernel<<<1, 1024, 0, st>>>(n_tiles, tsum);
    long long pb = (n_out + RS_THREADS - 1) / RS_THREADS;
    if (pb > (long long)sz.sm_count * 8) pb = (long long)sz.sm_count * 8;
    ile_resample_pick_kernel<<<(unsigned)pb, RS_THREADS, 0, st>>>(n, n_tiles, n_out, v0, prefix, tsum, ids);
    if (n_launches) *n_launches += 4;
    return cudaGetLastError();
}
