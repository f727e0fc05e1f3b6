// ile_quad_mma.cu -- step 4 (quadratic term) for many modes as an FP64-MMA contraction.
//
// The quadratic term of eq. 7 / eq. 10 needs, per sample and detector, Y^dagger U_k Y and Y^T V_k Y:
// O(K M^2) per sample, "cheap for 2-4 modes" but 10.6 k DFMA per sample for the 21 modes of l <= 4 -- more than the
// per-sample thread of the coefficient kernel can do without becoming the longest kernel of the call.  For a batch the
// two matrix-vector products W = U_k Y and Z = V_k Y are dense matrix-matrix products over the samples, so they run on
// DMMA.8x8x4 (mma.sync.m8n8k4.f64), one warp per 8 samples:
//   * real representation, padded to Mp = 8 ceil(M/8): y = [Re Y (Mp); Im Y (Mp)], X_real = [[Xr, -Xi], [Xi, Xr]]
//     (2Mp x 2Mp), so that  [Re W; Im W] = U_real y  and  [Re Z; Im Z] = V_real y.  Nothing is assumed about U or V
//     (reading R15).  The matrices are packed once per context in A-fragment order: [p][k][U|V][row block][k-step][32].
//   * B fragments: lane (r, cc) holds y[4s + cc] of sample r -- each lane evaluates its own 4 RBH entries of the
//     harmonics (Wigner-d finite sum, e^{-i m phi} by repeated multiplication).
//   * y in C-fragment layout (rows x samples), needed for the final dot products, is I y: two DMMAs per row block with
//     identity A fragments made in registers -- exact, and no shared memory.
//   * Re(Y^dagger W) = sum_rows y w;  Re(Y^T Z) = sum_{i<Mp} yr zr - yi zi;  Im(Y^T Z) = sum yr zi + yi zr: products in
//     the C layout (row i and row i + Mp sit in the same lane, RBH row blocks apart), then a sum over the 8 row lanes.
// Output: qform[sample][k][3] = (Re Y^dagger U_k Y, Re Y^T V_k Y, Im Y^T V_k Y), read by the coefficient kernel, which
// multiplies by |F_k|^2 and F_k^2 and adds up the detectors.
#include "ile_kernels.h"

#define QM_FULL 0xffffffffu
#define QM_THREADS 128

__device__ __forceinline__ void qm_dmma(double &c0, double &c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// RBH = Mp / 8 row blocks per half (real / imaginary part); RB = 2 RBH row blocks, KSQ = 4 RBH k-steps
template <int RBH>
__global__ void __launch_bounds__(QM_THREADS)
    ile_quad_mma_kernel(const __grid_constant__ IleDevParams P, const __grid_constant__ IleEvalArgs a,
                        const double *__restrict__ mats, double *__restrict__ qform)
{
    constexpr int RB = 2 * RBH, KSQ = 4 * RBH, MP = 8 * RBH;
    const int K = P.n_det, M = P.n_modes;
    const int lane = threadIdx.x & 31, r = lane >> 2, cc = lane & 3;
    const long long n_total = a.n_per_point * a.n_points;
    const long long n_groups = (n_total + 7) >> 3;
    const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_warps = ((long long)gridDim.x * blockDim.x) >> 5;
    const double aI0 = r == cc ? 1.0 : 0.0, aI1 = r == cc + 4 ? 1.0 : 0.0;  // identity A fragments of k-steps 2 rb, 2 rb + 1
    const size_t mat_stride = (size_t)RB * KSQ * 32;                          // one packed matrix

    for (long long g = warp0; g < n_groups; g += n_warps) {
        // a group never straddles two intrinsic points when n_per_point is a multiple of 8; otherwise the matrices of
        // the group's first sample would be wrong for its tail, so such groups are cut at the point boundary
        const long long s0 = g << 3;
        const int pt = (int)(s0 / a.n_per_point);
        const long long pt_end = (long long)(pt + 1) * a.n_per_point;
        const long long sidx = min(s0 + r, min(pt_end, n_total) - 1);  // lanes past the end repeat the last sample
        // ---- harmonics: this lane's entries y[4s + cc] of sample r
        double sh, ch, sphi, cphi;
        sincos(0.5 * a.incl[sidx], &sh, &ch);
        sincos(a.phi_ref[sidx], &sphi, &cphi);
        double bq[KSQ];
#pragma unroll
        for (int s = 0; s < KSQ; ++s) {
            const int i = 4 * s + cc, half = i >= MP, m = half ? i - MP : i;
            double y = 0.0;
            if (m < M) {
                double amp = 0.0;
                const int nt = P.mode_nterm[m];
                for (int t = 0; t < nt; ++t) amp += P.mode_coef[m][t] * ile_ipow(ch, P.mode_pc[m][t]) * ile_ipow(sh, P.mode_ps[m][t]);
                const int mm = P.mode_m[m], am = mm < 0 ? -mm : mm;
                double zx = 1.0, zy = 0.0;  // e^{-i |mm| phi} by repeated multiplication, conjugated for mm < 0
                for (int t = 0; t < am; ++t) {
                    const double nx = zx * cphi + zy * sphi, ny = zy * cphi - zx * sphi;
                    zx = nx, zy = ny;
                }
                if (mm < 0) zy = -zy;
                y = amp * (half ? zy : zx);
            }
            bq[s] = y;
        }
        // ---- y in C-fragment layout: yc[rb][c] = y[8 rb + r] of sample 2cc + c
        double yc[RB][2];
#pragma unroll
        for (int rb = 0; rb < RB; ++rb) {
            double c0 = 0.0, c1 = 0.0;
            qm_dmma(c0, c1, aI0, bq[2 * rb]);
            qm_dmma(c0, c1, aI1, bq[2 * rb + 1]);
            yc[rb][0] = c0, yc[rb][1] = c1;
        }
        const double *__restrict__ mp = mats + (size_t)(a.point0 + pt) * K * 2 * mat_stride + lane;
        for (int k = 0; k < K; ++k) {
            double uu[2] = {0.0, 0.0}, vr[2] = {0.0, 0.0}, vi[2] = {0.0, 0.0};
            const double *__restrict__ mu = mp + (size_t)(2 * k) * mat_stride, *__restrict__ mv = mu + mat_stride;
#pragma unroll
            for (int rb = 0; rb < RBH; ++rb) {
                // rows rb (real part) and rb + RBH (imaginary part) of W = U y and Z = V y: four independent chains
                double wr0 = 0.0, wr1 = 0.0, wi0 = 0.0, wi1 = 0.0, zr0 = 0.0, zr1 = 0.0, zi0 = 0.0, zi1 = 0.0;
#pragma unroll
                for (int s = 0; s < KSQ; ++s) {
                    qm_dmma(wr0, wr1, __ldg(mu + (size_t)(rb * KSQ + s) * 32), bq[s]);
                    qm_dmma(wi0, wi1, __ldg(mu + (size_t)((rb + RBH) * KSQ + s) * 32), bq[s]);
                    qm_dmma(zr0, zr1, __ldg(mv + (size_t)(rb * KSQ + s) * 32), bq[s]);
                    qm_dmma(zi0, zi1, __ldg(mv + (size_t)((rb + RBH) * KSQ + s) * 32), bq[s]);
                }
                const double yr0 = yc[rb][0], yr1 = yc[rb][1], yi0 = yc[rb + RBH][0], yi1 = yc[rb + RBH][1];
                uu[0] += yr0 * wr0 + yi0 * wi0;
                uu[1] += yr1 * wr1 + yi1 * wi1;
                vr[0] += yr0 * zr0 - yi0 * zi0;
                vr[1] += yr1 * zr1 - yi1 * zi1;
                vi[0] += yr0 * zi0 + yi0 * zr0;
                vi[1] += yr1 * zi1 + yi1 * zr1;
            }
#pragma unroll
            for (int o = 4; o < 32; o <<= 1) {
#pragma unroll
                for (int c = 0; c < 2; ++c) {
                    uu[c] += __shfl_xor_sync(QM_FULL, uu[c], o);
                    vr[c] += __shfl_xor_sync(QM_FULL, vr[c], o);
                    vi[c] += __shfl_xor_sync(QM_FULL, vi[c], o);
                }
            }
            if (r == 0) {
#pragma unroll
                for (int c = 0; c < 2; ++c) {
                    const long long sc = s0 + 2 * cc + c;
                    if (sc < min(pt_end, n_total)) {
                        double *q = qform + ((size_t)sc * K + k) * 3;
                        q[0] = uu[c], q[1] = vr[c], q[2] = vi[c];
                    }
                }
            }
        }
    }
}

// Host: real representation of U_k, V_k of every point in A-fragment order (see the header comment).
// U, V: host complex128 [P][K][M][M]; out: host doubles [P][K][2][RB][KSQ][32].
void ile_quad_pack_host(int32_t n_points, int32_t K, int32_t M, const double2 *U, const double2 *V, double *out)
{
    const int rbh = (M + 7) / 8, RB = 2 * rbh, KSQ = 4 * rbh, MP = 8 * rbh;
    size_t o = 0;
    for (int p = 0; p < n_points; ++p)
        for (int k = 0; k < K; ++k)
            for (int which = 0; which < 2; ++which) {
                const double2 *X = (which ? V : U) + ((size_t)p * K + k) * M * M;
                for (int rb = 0; rb < RB; ++rb)
                    for (int s = 0; s < KSQ; ++s)
                        for (int lane = 0; lane < 32; ++lane) {
                            const int row = 8 * rb + (lane >> 2), col = 4 * s + (lane & 3);
                            const int rh = row >= MP, ri = rh ? row - MP : row, chf = col >= MP, ci = chf ? col - MP : col;
                            double v = 0.0;
                            if (ri < M && ci < M) {
                                const double2 x = X[(size_t)ri * M + ci];
                                // [[Xr, -Xi], [Xi, Xr]]
                                v = rh == chf ? x.x : (rh ? x.y : -x.y);
                            }
                            out[o++] = v;
                        }
            }
}

size_t ile_quad_pack_doubles(int32_t n_points, int32_t K, int32_t M)
{
    const int rbh = (M + 7) / 8;
    return (size_t)n_points * K * 2 * (2 * rbh) * (4 * rbh) * 32;
}

cudaError_t ile_launch_quad_mma(const IleSizes &sz, const IleDevParams &hp, const IleEvalArgs &a, const double *mats, double *qform,
                                cudaStream_t st)
{
    const long long n_total = a.n_per_point * a.n_points;
    if (a.n_points > 1 && (a.n_per_point & 7)) return cudaErrorInvalidValue;  // groups of 8 must not straddle points
    const long long groups = (n_total + 7) / 8;
    long long blocks = (groups + QM_THREADS / 32 - 1) / (QM_THREADS / 32);
    const long long cap = (long long)sz.sm_count * 16;
    if (blocks > cap) blocks = cap;
    const int rbh = (sz.n_modes + 7) / 8;
    switch (rbh) {
        case 1: ile_quad_mma_kernel<1><<<(unsigned)blocks, QM_THREADS, 0, st>>>(hp, a, mats, qform); break;
        case 2: ile_quad_mma_kernel<2><<<(unsigned)blocks, QM_THREADS, 0, st>>>(hp, a, mats, qform); break;
        case 3: ile_quad_mma_kernel<3><<<(unsigned)blocks, QM_THREADS, 0, st>>>(hp, a, mats, qform); break;
        case 4: ile_quad_mma_kernel<4><<<(unsigned)blocks, QM_THREADS, 0, st>>>(hp, a, mats, qform); break;
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}
