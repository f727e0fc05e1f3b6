// ile_sampler.cu -- on-device Monte Carlo sampler (readings S1-S9).
//
// PAPER.md L47 (eq. 4: Monte Carlo over the extrinsic parameters with an adaptive sampler), L97 (blocks of samples per
// likelihood call), L119 / L125 (sampling prior in the two sky parameters and distance, regenerated from the most recent
// n_chunk points), L251 ("converting the Monte Carlo random number generation ... to GPU-based operations").
//   ile_sampler_uniform_kernel  S1: Philox4x32-10 uniforms of a range of sample indices (test entry)
//   ile_sampler_draw_kernel     S1-S5: one thread per sample -- uniforms, inverse CDF of the adaptive dimensions, the seven
//                               physical parameters, ln w = -sum ln h_d[bin_d], the bin indices
//   ile_sampler_refit_kernel    S6: one block -- chunk maximum, fixed-point weighted histograms in shared memory (integer
//                               atomics: the sums do not depend on the order), new densities and cumulatives
//   ile_sampler_tables_kernel   cumulatives of densities set from the host / reset to uniform
// Nothing here is shared with oracle/sampler.py.
#include <math_constants.h>

#include "ile_kernels.h"

#define SMP_THREADS 256
#define SMP_REFIT_THREADS 1024

struct uint4x {
    uint32_t v[4];
};

// Philox4x32-10 (Salmon et al., SC'11): ten rounds of two 32x32 -> 64 multiplications, key bumped by the Weyl constants
__device__ __forceinline__ uint4x smp_philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0, c1 = lo1, c2 = n2, c3 = lo0;
        k0 += 0x9E3779B9u, k1 += 0xBB67AE85u;
    }
    uint4x o;
    o.v[0] = c0, o.v[1] = c1, o.v[2] = c2, o.v[3] = c3;
    return o;
}

// S1: the seven uniforms of sample `idx`: ((w[2i] >> 5) 2^26 + (w[2i+1] >> 6) + 0.5) 2^-53, all exact in binary64
__device__ __forceinline__ void smp_uniforms(unsigned long long seed, unsigned long long idx, double u[7])
{
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32), a0 = (uint32_t)idx, a1 = (uint32_t)(idx >> 32);
    uint32_t w[16];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint4x o = smp_philox(a0, a1, (uint32_t)j, 0u, k0, k1);
#pragma unroll
        for (int e = 0; e < 4; ++e) w[4 * j + e] = o.v[e];
    }
#pragma unroll
    for (int i = 0; i < 7; ++i)
        u[i] = ((double)(w[2 * i] >> 5) * 67108864.0 + (double)(w[2 * i + 1] >> 6) + 0.5) * 1.1102230246251565e-16;
}

__global__ void __launch_bounds__(SMP_THREADS) ile_sampler_uniform_kernel(unsigned long long seed, long long first, long long n,
                                                                          double *__restrict__ out)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        double u[7];
        smp_uniforms(seed, (unsigned long long)(first + i), u);
#pragma unroll
        for (int d = 0; d < 7; ++d) out[i * 7 + d] = u[d];
    }
}

// tab: [3][n_bins] densities h, then [3][n_bins + 1] cumulatives C (S4: C[b+1] = C[b] + h[b] / n_bins, sequentially).
// The divisions are done by all threads into `w` (shared, 3 n_bins doubles); thread j < 3 then runs the additions of
// dimension j in bin order -- the same roundings as the plain loop.
__device__ __forceinline__ void smp_cumulatives(const double *__restrict__ h, double *__restrict__ C, double *w, int nb)
{
    const double dnb = (double)nb;
    for (int i = threadIdx.x; i < 3 * nb; i += blockDim.x) w[i] = __ddiv_rn(h[i], dnb);
    __syncthreads();
    if (threadIdx.x < 3) {
        const double *wj = w + threadIdx.x * nb;
        double *Cj = C + threadIdx.x * (nb + 1);
        double run = 0.0;
        Cj[0] = 0.0;
        for (int b = 0; b < nb; ++b) {
            run = __dadd_rn(run, wj[b]);
            Cj[b + 1] = run;
        }
    }
}

__global__ void __launch_bounds__(256) ile_sampler_tables_kernel(IleSamplerParams P, double *__restrict__ tab, int set_uniform)
{
    extern __shared__ double smp_w[];
    const int nb = P.n_bins;
    if (set_uniform)
        for (int i = threadIdx.x; i < 3 * nb; i += blockDim.x) tab[i] = 1.0;
    __syncthreads();
    smp_cumulatives(tab, tab + 3 * nb, smp_w, nb);
}

__global__ void __launch_bounds__(SMP_THREADS)
    ile_sampler_draw_kernel(const __grid_constant__ IleSamplerParams P, const double *__restrict__ tab, long long first, long long n,
                            double *__restrict__ ra, double *__restrict__ dec, double *__restrict__ t_ref, double *__restrict__ phi_ref,
                            double *__restrict__ psi, double *__restrict__ incl, double *__restrict__ dist, double *__restrict__ log_w,
                            int32_t *__restrict__ bins)
{
    extern __shared__ double smp_tab[];  // h [3][nb] | C [3][nb + 1]
    const int nb = P.n_bins;
    for (int i = threadIdx.x; i < 3 * nb + 3 * (nb + 1); i += blockDim.x) smp_tab[i] = tab[i];
    __syncthreads();
    const double dnb = (double)nb;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        double u[7];
        smp_uniforms(P.seed, (unsigned long long)(first + i), u);
        double lw = 0.0;
        const int dim[3] = {0, 1, 6};
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            int b = -1;
            if (P.adapt[j]) {
                const double *__restrict__ h = smp_tab + j * nb;
                const double *__restrict__ C = smp_tab + 3 * nb + j * (nb + 1);
                const double v = u[dim[j]];
                // S4: the largest b with C[b] <= v (C[0] = 0 <= v always), clamped to the last bin
                int lo = 0, hi = nb + 1;  // C[lo] <= v, C[hi] > v (hi = nb + 1: virtual +inf)
                while (hi - lo > 1) {
                    const int mid = (lo + hi) >> 1;
                    if (C[mid] <= v) lo = mid;
                    else hi = mid;
                }
                b = min(lo, nb - 1);
                const double width = __ddiv_rn(h[b], dnb);
                const double ud = __ddiv_rn(__dadd_rn((double)b, __ddiv_rn(__dsub_rn(v, C[b]), width)), dnb);
                u[dim[j]] = fmin(ud, 1.0 - 1.1102230246251565e-16);
                lw -= log(h[b]);
            }
            if (bins) bins[i * 3 + j] = b;
        }
        // S5 (every product and sum individually rounded: the same numbers wherever they are computed)
        ra[i] = __dmul_rn(6.283185307179586, u[0]);
        dec[i] = asin(__dsub_rn(__dmul_rn(2.0, u[1]), 1.0));
        t_ref[i] = __dadd_rn(P.t_lo, __dmul_rn(P.t_span, u[2]));
        phi_ref[i] = __dmul_rn(6.283185307179586, u[3]);
        psi[i] = __dmul_rn(3.141592653589793, u[4]);
        incl[i] = acos(__dsub_rn(__dmul_rn(2.0, u[5]), 1.0));
        dist[i] = cbrt(__dadd_rn(P.dmin3, __dmul_rn(u[6], P.d3_span)));
        if (log_w) log_w[i] = lw;
    }
}

// S6: refit from one chunk, two kernels.  (1) chunk maximum of e = lnL + ln w into an order-preserving integer key.
// (2) every block histograms its slice of the chunk: the fixed-point weights q < 2^42 are accumulated as three 14-bit pieces with
// native 32-bit shared-memory atomics (a block sees at most 2^18 samples, so the sums stay below 2^32), reassembled exactly and
// added to the 64-bit global histograms; the block that finishes last (ticket) turns them into the new densities and cumulatives
// and leaves the scratch (histograms, key, ticket) zeroed for the next call.
// work: [3 n_bins] 64-bit histograms | key | ticket
#define SMP_REFIT_SLICE 262144
__device__ __forceinline__ long long smp_key(double x)
{
    const long long b = __double_as_longlong(x);
    return b >= 0 ? b : b ^ 0x7fffffffffffffffLL;
}
__device__ __forceinline__ double smp_unkey(long long k) { return __longlong_as_double(k >= 0 ? k : k ^ 0x7fffffffffffffffLL); }
#define SMP_KEY_NEG_INF 0x800FFFFFFFFFFFFFLL /* smp_key(-inf) */

__global__ void __launch_bounds__(SMP_THREADS) ile_sampler_refit_max_kernel(long long n, const double *__restrict__ lnL,
                                                                            const double *__restrict__ log_w, long long *__restrict__ key)
{
    double mx = -CUDART_INF;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const double e = lnL[i] + (log_w ? log_w[i] : 0.0);
        if (e == e) mx = fmax(mx, e);
    }
    mx = warp_max(mx);
    if ((threadIdx.x & 31) == 0 && mx > -CUDART_INF) atomicMax(key, smp_key(mx));
}

__global__ void __launch_bounds__(SMP_REFIT_THREADS)
    ile_sampler_refit_kernel(const __grid_constant__ IleSamplerParams P, double *__restrict__ tab, long long n,
                             const int32_t *__restrict__ bins, const double *__restrict__ lnL, const double *__restrict__ log_w,
                             unsigned long long *__restrict__ work)
{
    extern __shared__ __align__(8) unsigned char smp_raw[];
    const int nb = P.n_bins, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double *w = reinterpret_cast<double *>(smp_raw);          // [3][nb] bin widths for the cumulatives (last block)
    uint32_t *H = reinterpret_cast<uint32_t *>(w + 3 * nb);   // [3 pieces][3][nb]
    __shared__ unsigned long long redq[3][SMP_REFIT_THREADS / 32];
    __shared__ unsigned long long tot_s[3];
    __shared__ bool last_s;
    long long *key = reinterpret_cast<long long *>(work + 3 * nb);
    unsigned int *ticket = reinterpret_cast<unsigned int *>(work + 3 * nb + 1);
    const double M = smp_unkey(*key);
    if (M > -CUDART_INF) {  // otherwise no finite sample: the densities are kept (the last block still cleans up)
        for (int i = threadIdx.x; i < 9 * nb; i += blockDim.x) H[i] = 0u;
        __syncthreads();
        const long long per = (n + gridDim.x - 1) / gridDim.x;  // <= SMP_REFIT_SLICE by the launcher's grid
        const long long lo = (long long)blockIdx.x * per, hi = lo + per < n ? lo + per : n;
        for (long long i = lo + threadIdx.x; i < hi; i += blockDim.x) {
            const double e = lnL[i] + (log_w ? log_w[i] : 0.0);
            const double W = exp(__dmul_rn(P.temper, __dsub_rn(e, M)));  // exp(-inf) = 0
            const unsigned long long q = (unsigned long long)__double2ll_rn(__dmul_rn(W, 1099511627776.0));
            if (q) {
                const uint32_t q0 = (uint32_t)(q & 0x3fffu), q1 = (uint32_t)((q >> 14) & 0x3fffu), q2 = (uint32_t)(q >> 28);
#pragma unroll
                for (int j = 0; j < 3; ++j)
                    if (P.adapt[j]) {
                        const int b = bins[i * 3 + j];
                        if (q0) atomicAdd(&H[j * nb + b], q0);
                        if (q1) atomicAdd(&H[(3 + j) * nb + b], q1);
                        if (q2) atomicAdd(&H[(6 + j) * nb + b], q2);
                    }
            }
        }
        __syncthreads();
        for (int i = threadIdx.x; i < 3 * nb; i += blockDim.x) {
            const unsigned long long v = (unsigned long long)H[i] + ((unsigned long long)H[3 * nb + i] << 14) + ((unsigned long long)H[6 * nb + i] << 28);
            if (v) atomicAdd(&work[i], v);
        }
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) last_s = atomicAdd(ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!last_s) return;
    __threadfence();
    // ---- the last block: totals, densities, cumulatives; scratch back to zero
    unsigned long long t[3] = {0ull, 0ull, 0ull};
    for (int b = threadIdx.x; b < nb; b += blockDim.x)
#pragma unroll
        for (int j = 0; j < 3; ++j) t[j] += __ldcg(&work[j * nb + b]);
#pragma unroll
    for (int j = 0; j < 3; ++j) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t[j] += __shfl_xor_sync(0xffffffffu, t[j], o);
        if (lane == 0) redq[j][warp] = t[j];
    }
    __syncthreads();
    if (threadIdx.x < 3) {
        unsigned long long s = 0ull;
        for (int ww = 0; ww < SMP_REFIT_THREADS / 32; ++ww) s += redq[threadIdx.x][ww];
        tot_s[threadIdx.x] = s;
    }
    __syncthreads();
    // h = (1 - floor) n_bins (H / total) + floor, one rounding per operation
    const double scale = __dmul_rn(__dsub_rn(1.0, P.floor_frac), (double)nb);
    for (int i = threadIdx.x; i < 3 * nb; i += blockDim.x) {
        const int j = i / nb;
        if (P.adapt[j] && tot_s[j])
            tab[i] = __dadd_rn(__dmul_rn(scale, __ddiv_rn((double)__ldcg(&work[i]), (double)tot_s[j])), P.floor_frac);
        work[i] = 0ull;
    }
    if (threadIdx.x == 0) {
        *key = SMP_KEY_NEG_INF;
        *ticket = 0u;
    }
    __syncthreads();
    smp_cumulatives(tab, tab + 3 * nb, w, nb);  // a dimension that was not refit gets the cumulative it already had
}

// ------------------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------------------
static unsigned smp_grid(long long n, int sm_count)
{
    long long b = (n + SMP_THREADS - 1) / SMP_THREADS;
    const long long cap = (long long)sm_count * 8;
    return (unsigned)(b > cap ? cap : b < 1 ? 1 : b);
}

size_t ile_sampler_table_doubles(int32_t n_bins) { return (size_t)3 * n_bins + (size_t)3 * (n_bins + 1); }

cudaError_t ile_launch_sampler_tables(const IleSamplerParams &P, double *tab, int set_uniform, cudaStream_t st)
{
    ile_sampler_tables_kernel<<<1, 256, (size_t)3 * P.n_bins * sizeof(double), st>>>(P, tab, set_uniform);
    return cudaGetLastError();
}

cudaError_t ile_launch_sampler_uniforms(const IleSamplerParams &P, int sm_count, long long first, long long n, double *u, cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    ile_sampler_uniform_kernel<<<smp_grid(n, sm_count), SMP_THREADS, 0, st>>>(P.seed, first, n, u);
    return cudaGetLastError();
}

cudaError_t ile_launch_sampler_draw(const IleSamplerParams &P, int sm_count, const double *tab, long long first, long long n, double *ra,
                                    double *dec, double *t_ref, double *phi_ref, double *psi, double *incl, double *dist, double *log_w,
                                    int32_t *bins, cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    const size_t smem = ile_sampler_table_doubles(P.n_bins) * sizeof(double);  // <= 49 KB for n_bins <= 1024
    ile_sampler_draw_kernel<<<smp_grid(n, sm_count), SMP_THREADS, smem, st>>>(P, tab, first, n, ra, dec, t_ref, phi_ref, psi, incl, dist,
                                                                             log_w, bins);
    return cudaGetLastError();
}

size_t ile_sampler_work_words(int32_t n_bins) { return (size_t)3 * n_bins + 2; }  // 64-bit words, zero + key = -inf before the first call

cudaError_t ile_sampler_work_init(const IleSamplerParams &P, unsigned long long *work, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(work, 0, ile_sampler_work_words(P.n_bins) * sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    const long long k = SMP_KEY_NEG_INF;
    return cudaMemcpyAsync(work + 3 * P.n_bins, &k, sizeof(k), cudaMemcpyHostToDevice, st);
}

cudaError_t ile_launch_sampler_refit(const IleSamplerParams &P, int sm_count, double *tab, long long n, const int32_t *bins, const double *lnL,
                                     const double *log_w, unsigned long long *work, cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    ile_sampler_refit_max_kernel<<<smp_grid(n, sm_count), SMP_THREADS, 0, st>>>(n, lnL, log_w, reinterpret_cast<long long *>(work + 3 * P.n_bins));
    long long g = (n + 8191) / 8192;  // 8 samples per thread and block while the grid allows
    if (g > sm_count) g = sm_count;
    const long long gmin = (n + SMP_REFIT_SLICE - 1) / SMP_REFIT_SLICE;  // a block's 32-bit piece sums must not overflow
    if (g < gmin) g = gmin;
    const size_t smem = (size_t)3 * P.n_bins * sizeof(double) + (size_t)9 * P.n_bins * sizeof(uint32_t);
    ile_sampler_refit_kernel<<<(unsigned)g, SMP_REFIT_THREADS, smem, st>>>(P, tab, n, bins, lnL, log_w, work);
    return cudaGetLastError();
}
