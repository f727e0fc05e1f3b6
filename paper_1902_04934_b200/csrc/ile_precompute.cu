// ile_precompute.cu -- the overlap pre-computation of an intrinsic point (eq. 8a-c):
//
//   Q_{k,lm}[i] = <h_lm(. - tau_i) | d_k> = sum_n conj(x_{k,lm}[n]) d_k[n] exp(+2 pi i f_n tau_i),  tau_i = t0_Q + i / f_s
//   U_k[a][b]   = sum_n conj(x_a[n]) x_b[n]            V_k[a][b] = sum_n x_a[(-n) mod N] x_b[n]
//
// on the two-sided FFT grid f_n = n' f_s / N (n' the signed index of FFT order), whitened spectra in, complex128 throughout.
// "After the port it is what dominates for BNS" (L97, L175): one inverse FFT per (point, detector, mode) and M^2 dot
// products per (point, detector).
//
//   ile_overlap_q_kernel   one block per series: spectrum product and the start-time phase on load (bit-reversed into shared
//                          memory), in-place radix-2 decimation-in-time butterflies with a twiddle table in shared memory,
//                          natural-order store.  N a power of two, 2 <= N <= 8192 (16 N + 8 N bytes of shared memory).
//   ile_overlap_uv_kernel  one block per (a, b, detector, point): both sums in one pass over n, warp-shuffle then block-level
//                          reduction.
#include "ile_kernels.h"

#define PC_THREADS 256

__device__ __forceinline__ double2 pc_cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

__global__ void __launch_bounds__(PC_THREADS)
    ile_overlap_q_kernel(int32_t M, int32_t N, int32_t log2n, double fs_t0_over_n, const double2 *__restrict__ x,
                         const double2 *__restrict__ d, double2 *__restrict__ Q)
{
    extern __shared__ double2 pc_sm[];
    double2 *a = pc_sm;       // N points
    double2 *W = pc_sm + N;   // N / 2 twiddles exp(+2 pi i j / N)
    const size_t series = blockIdx.x;             // (point * K + k) * M + mode
    const double2 *xs = x + series * N;
    const double2 *ds = d + (series / M) * N;
    for (int j = threadIdx.x; j < N / 2; j += PC_THREADS) {
        double s, c;
        sincospi(2.0 * (double)j / (double)N, &s, &c);
        W[j] = make_double2(c, s);
    }
    for (int n = threadIdx.x; n < N; n += PC_THREADS) {
        const int np = n < (N + 1) / 2 ? n : n - N;  // signed index
        double s, c;
        sincospi(2.0 * (double)np * fs_t0_over_n, &s, &c);  // exp(2 pi i f_n t0_Q), f_n = n' f_s / N
        const double2 xv = xs[n], dv = pc_cmul(ds[n], make_double2(c, s));
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
    for (int i = threadIdx.x; i < N; i += PC_THREADS) q[i] = a[i];
}

__global__ void __launch_bounds__(PC_THREADS)
    ile_overlap_uv_kernel(int32_t M, int32_t N, const double2 *__restrict__ x, double2 *__restrict__ U, double2 *__restrict__ V)
{
    __shared__ double red[4][PC_THREADS / 32];
    const int a = blockIdx.x / M, b = blockIdx.x % M;
    const size_t pk = blockIdx.y;  // point * K + k
    const double2 *xa = x + (pk * M + a) * N, *xb = x + (pk * M + b) * N;
    double ur = 0.0, ui = 0.0, vr = 0.0, vi = 0.0;
    for (int n = threadIdx.x; n < N; n += PC_THREADS) {
        const double2 p = xa[n], m = xa[(N - n) & (N - 1)], q = xb[n];
        ur += p.x * q.x + p.y * q.y;  // conj(x_a) x_b
        ui += p.x * q.y - p.y * q.x;
        vr += m.x * q.x - m.y * q.y;  // x_a(-f) x_b(f)
        vi += m.x * q.y + m.y * q.x;
    }
    double v[4] = {ur, ui, vr, vi};
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[c] += __shfl_xor_sync(0xffffffffu, v[c], o);
        if (lane == 0) red[c][warp] = v[c];
    }
    __syncthreads();
    if (threadIdx.x < 4) {
        double s = 0.0;
        for (int w = 0; w < PC_THREADS / 32; ++w) s += red[threadIdx.x][w];
        double *out = reinterpret_cast<double *>((threadIdx.x < 2 ? U : V) + (pk * M + a) * M + b);
        out[threadIdx.x & 1] = s;
    }
}

cudaError_t ile_launch_precompute(int32_t n_points, int32_t K, int32_t M, int32_t N, double fs_hz, double t0_q_s, const double2 *x,
                                  const double2 *d, double2 *Q, double2 *U, double2 *V, int32_t max_smem_optin, cudaStream_t st)
{
    int log2n = 0;
    while ((1 << log2n) < N) ++log2n;
    if ((1 << log2n) != N || N < 2 || N > 8192) return cudaErrorInvalidValue;
    const size_t smem = (size_t)N * 16 + (size_t)(N / 2) * 16;
    if (smem > (size_t)max_smem_optin) return cudaErrorInvalidValue;
    cudaError_t e = cudaFuncSetAttribute(ile_overlap_q_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    ile_overlap_q_kernel<<<(unsigned)((size_t)n_points * K * M), PC_THREADS, smem, st>>>(M, N, log2n, fs_hz * t0_q_s / (double)N, x, d, Q);
    dim3 grid((unsigned)(M * M), (unsigned)(n_points * K));
    ile_overlap_uv_kernel<<<grid, PC_THREADS, 0, st>>>(M, N, x, U, V);
    return cudaGetLastError();
}
