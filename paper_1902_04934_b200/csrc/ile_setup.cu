// ile_setup.cu -- pre-pass of the sorted FP64-MMA evaluation path (variant 3): per-sample setup, cell keys, counting sort,
// and the one-off repacking of Q into MMA fragment order.
//
//   ile_pack_q_kernel   (ile_create) Q [P][K][M][n_q] complex128 -> Qp [P][K][nblk_q][ks][32] doubles, the A-fragment order
//                       of mma.m8n8k4.f64: lane = 4*(time % 8) + (channel % 4); channel 2m = Re, 2m+1 = Im
//   ile_setup_kernel    steps 1-4 of the hot path, one thread per sample: F_k, dt_k and the
//                       window start i0_k (L62, L88), Y_lm(iota, -phi_ref) (eq. 5-6), the quadratic term
//                       (eq. 7) and the coefficients a F_k Y_lm of the linear term, written as one record per
//                       sample; plus the out-of-range flag (reading R9), the cell id and the per-point histogram
//   ile_scan_kernel     exclusive scan of each point's histogram (one block per point), number of in-range samples
//   ile_scatter_kernel  perm[position] = sample
//
// Why sort: the contraction kernel keeps Q of one detector stationary in registers for a span of
// absolute time indices and lets groups of 8 samples share it.  A sample only uses the N_t indices starting at its
// own window start ("distinct time-of-flight-dependent time windows" per interferometer, L97), so samples that sit in
// one group must have nearly equal i0_k for every k.  Samples are independent (L97: blocks of samples, any order).
#include <math_constants.h>

#include "ile_kernels.h"

// ------------------------------------------------------------------------------------------------------------
// Q repacking (once per context)
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) ile_pack_q_kernel(int32_t n_points, int32_t K, int32_t M, int32_t n_q, int32_t ks,
                                                         int32_t nblk_q, const double2 *__restrict__ Q, double *__restrict__ Qp)
{
    const long long total = (long long)n_points * K * nblk_q * ks * 32;
    for (long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x; o < total; o += (long long)gridDim.x * blockDim.x) {
        const int lane = (int)(o & 31);
        long long q = o >> 5;
        const int s = (int)(q % ks);
        q /= ks;
        const int b = (int)(q % nblk_q);
        q /= nblk_q;  // = p * K + k
        const int r = lane >> 2, cc = lane & 3;
        const int ch = 4 * s + cc, m = ch >> 1, i = 8 * b + r;
        double v = 0.0;
        if (m < M && i < n_q) {
            const double2 z = Q[((size_t)q * M + m) * n_q + i];
            v = (ch & 1) ? z.y : z.x;
        }
        Qp[o] = v;
    }
}

cudaError_t ile_launch_pack_q(const IleSizes &sz, const IleMmaPlan &mp, int32_t n_points, const double2 *Q, double *Qp,
                              cudaStream_t st)
{
    const long long total = (long long)n_points * sz.n_det * mp.nblk_q * mp.ks * 32;
    long long blocks = (total + 255) / 256;
    if (blocks > (long long)sz.sm_count * 32) blocks = (long long)sz.sm_count * 32;
    ile_pack_q_kernel<<<(unsigned)blocks, 256, 0, st>>>(n_points, sz.n_det, sz.n_modes, sz.n_q, mp.ks, mp.nblk_q, Q, Qp);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------
// per-sample setup + cell key + histogram
// ------------------------------------------------------------------------------------------------------------
#define SETUP_THREADS 128
#ifndef SETUP_MINB
#define SETUP_MINB 6 /* <= 85 registers: 768 threads per SM, a 100,000-sample batch is one wave */
#endif

// SORT = false (variant 4): coefficients and quadratic term only -- window starts, cell keys and the histogram come
// from ile_index_kernel, which runs concurrently on the caller's stream.
template <int MMAX, bool SORT, bool QF>
__global__ void __launch_bounds__(SETUP_THREADS, (MMAX <= 5 ? SETUP_MINB : MMAX <= 12 ? 3 : 2))
    ile_setup_kernel(const __grid_constant__ IleDevParams P, const __grid_constant__ IleEvalArgs a, const int32_t cp,
                     const __grid_constant__ IleSortPlan sp, const __grid_constant__ IleMmaScratch sc)
{
    const long long n_total = a.n_per_point * a.n_points;
    const int K = P.n_det, M = P.n_modes;
    const int recg = K * cp;
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < n_total; s += (long long)gridDim.x * blockDim.x) {
        const int pt = (int)(s / a.n_per_point);
        const size_t pglob = (size_t)(a.point0 + pt);
        const double2 *__restrict__ U = a.U + pglob * (size_t)K * M * M;
        const double2 *__restrict__ V = a.V + pglob * (size_t)K * M * M;

        // ---- steps 1-2: sky geometry, antenna axes, source direction
        const IleSky g = ile_sky(a.ra[s], a.dec[s], a.psi[s], P.gmst);
        const double t_ref = a.t_ref[s];
        const double amp_a = P.d_ref / a.dist[s];

        // ---- step 3: Y_m = [sum_t coef_t c^pc_t s^ps_t] e^{-i m phi_ref}
        double sh, ch, sphi, cphi;
        sincos(0.5 * a.incl[s], &sh, &ch);
        sincos(a.phi_ref[s], &sphi, &cphi);
        double2 Y[MMAX];
#pragma unroll
        for (int m = 0; m < MMAX; ++m) {
            if (m < M) {
                double amp = 0.0;
                const int nt = P.mode_nterm[m];
                for (int t = 0; t < nt; ++t)
                    amp += P.mode_coef[m][t] * ile_ipow(ch, P.mode_pc[m][t]) * ile_ipow(sh, P.mode_ps[m][t]);
                // e^{-i |mm| phi} by repeated multiplication, conjugated for mm < 0
                const int mm = P.mode_m[m], am = mm < 0 ? -mm : mm;
                double2 z = make_double2(1.0, 0.0);
                for (int t = 0; t < am; ++t) z = make_double2(z.x * cphi + z.y * sphi, z.y * cphi - z.x * sphi);
                if (mm < 0) z.y = -z.y;
                Y[m] = make_double2(amp * z.x, amp * z.y);
            } else {
                Y[m] = make_double2(0.0, 0.0);
            }
        }

        // ---- steps 1, 2, 4 per detector; coefficients of the linear term
        double *__restrict__ rec = sc.rec + (size_t)s * recg;
        double tot = 0.0;
        int bad = 0;
        int32_t i0[3] = {0, 0, 0};
        for (int k = 0; k < K; ++k) {
            const double2 F = ile_antenna(P.det_tensor[k], g);
            double yuy = 0.0;
            double2 yvy = make_double2(0.0, 0.0);
            if (QF) {  // many modes: Y^dagger U_k Y and Y^T V_k Y come from the FP64-MMA kernel (ile_quad_mma.cu)
                const double *__restrict__ q = sc.qform + ((size_t)s * K + k) * 3;
                yuy = q[0];
                yvy = make_double2(q[1], q[2]);
            } else {
#pragma unroll
                for (int p = 0; p < MMAX; ++p) {
                    if (p < M) {
                        double2 tu = make_double2(0.0, 0.0), tv = make_double2(0.0, 0.0);
                        const double2 *Ur = U + ((size_t)k * M + p) * M;
                        const double2 *Vr = V + ((size_t)k * M + p) * M;
#pragma unroll
                        for (int q = 0; q < MMAX; ++q) {
                            if (q < M) {
                                const double2 Yq = Y[q], u = __ldg(Ur + q), v = __ldg(Vr + q);
                                tu.x += u.x * Yq.x - u.y * Yq.y;
                                tu.y += u.x * Yq.y + u.y * Yq.x;
                                tv.x += v.x * Yq.x - v.y * Yq.y;
                                tv.y += v.x * Yq.y + v.y * Yq.x;
                            }
                        }
                        const double2 Yp = Y[p];
                        yuy += Yp.x * tu.x + Yp.y * tu.y;  // Re(conj(Y_p) (U Y)_p): U not assumed Hermitian (reading R15)
                        const double2 t = ile_cmul(Yp, tv);
                        yvy.x += t.x;
                        yvy.y += t.y;
                    }
                }
            }
            const double F2 = F.x * F.x + F.y * F.y;
            const double2 FF = ile_cmul(F, F);
            tot += F2 * yuy + (FF.x * yvy.x - FF.y * yvy.y);

            if (SORT) {
                const int32_t idx = ile_window_index(P.vertex[k], g.s, t_ref, P.t0_q, P.fs, P.n_t);
                if (k < 3) i0[k] = idx;
                if (idx < 0 || (long long)idx + P.n_t > P.n_q) bad = 1;
                sc.i0[s * K + k] = idx;
                if (a.shift_idx) a.shift_idx[s * K + k] = idx;
            }

            const double2 aF = make_double2(amp_a * F.x, amp_a * F.y);
            double2 *__restrict__ rk = reinterpret_cast<double2 *>(rec + (size_t)k * cp);
#pragma unroll
            for (int m = 0; m < MMAX; ++m)
                if (m < M) rk[m] = ile_cmul(aF, Y[m]);
            for (int m = M; m < cp / 2; ++m) rk[m] = make_double2(0.0, 0.0);
        }
        sc.quad[s] = 0.25 * amp_a * amp_a * tot;
        if (!SORT) continue;

        // ---- cell of the counting sort (boustrophedon enumeration: consecutive cells are neighbours)
        int32_t c;
        if (bad) {
            c = sp.ncell - 1;
            atomicAdd(a.oob_counter, 1ULL);
            a.lnL[s] = -CUDART_INF;
        } else if (sp.mode == 1) {
            // variant 4: segment = (d1, d2) cell of width 2^g, then the exact i0_0 inside the segment
            int32_t seg = 0;
            if (sp.nd > 1) seg = min(max(i0[1] - i0[0] + sp.dmax[1], 0), 2 * sp.dmax[1]) >> sp.g;
            if (sp.nd > 2) seg = seg * sp.n2 + (min(max(i0[2] - i0[0] + sp.dmax[2], 0), 2 * sp.dmax[2]) >> sp.g);
            c = seg * sp.n0 + (i0[0] >> sp.g0);  // 0 <= i0_0 <= n_q - n_t here
        } else {
            c = i0[0] >> sp.g;  // 0 <= i0_0 <= n_q - n_t here
            if (sp.nd > 1) {
                int32_t c1 = min(max(i0[1] - i0[0] + sp.dmax[1], 0), 2 * sp.dmax[1]) >> sp.g;
                if (c & 1) c1 = sp.n1 - 1 - c1;
                c = c * sp.n1 + c1;
            }
            if (sp.nd > 2) {
                int32_t c2 = min(max(i0[2] - i0[0] + sp.dmax[2], 0), 2 * sp.dmax[2]) >> sp.g;
                if (c & 1) c2 = sp.n2 - 1 - c2;
                c = c * sp.n2 + c2;
            }
        }
        sc.cell[s] = c;
        atomicAdd(&sc.hist[(size_t)pt * sp.ncell + c], 1u);
    }
}

// ------------------------------------------------------------------------------------------------------------
// counting sort: scan and scatter
// ------------------------------------------------------------------------------------------------------------
#define SCAN_THREADS 1024
__global__ void __launch_bounds__(SCAN_THREADS) ile_scan_kernel(int32_t ncell, uint32_t *__restrict__ hist, int32_t *__restrict__ ngood)
{
    __shared__ uint32_t wsum[SCAN_THREADS / 32];
    uint32_t *h = hist + (size_t)blockIdx.x * ncell;
    const int per = (ncell + SCAN_THREADS - 1) / SCAN_THREADS;
    const int lo = min((int)threadIdx.x * per, ncell), hi = min(lo + per, ncell);
    uint32_t loc = 0;
    for (int i = lo; i < hi; ++i) loc += h[i];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t inc = loc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t v = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += v;
    }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        uint32_t w = wsum[lane], wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t v = __shfl_up_sync(0xffffffffu, wi, o);
            if (lane >= o) wi += v;
        }
        wsum[lane] = wi - w;
    }
    __syncthreads();
    uint32_t run = wsum[warp] + inc - loc;  // exclusive prefix of this thread's slice
    for (int i = lo; i < hi; ++i) {
        uint32_t v = h[i];
        h[i] = run;
        if (i == ncell - 1) ngood[blockIdx.x] = (int32_t)run;  // samples before the out-of-range cell
        run += v;
    }
}

__global__ void __launch_bounds__(256) ile_scatter_kernel(long long n_per_point, int32_t n_points, int32_t ncell,
                                                          const int32_t *__restrict__ cell, uint32_t *__restrict__ offs,
                                                          int32_t *__restrict__ perm)
{
    const long long n_total = n_per_point * n_points;
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < n_total; s += (long long)gridDim.x * blockDim.x) {
        const int pt = (int)(s / n_per_point);
        const uint32_t pos = atomicAdd(&offs[(size_t)pt * ncell + cell[s]], 1u);
        perm[(size_t)pt * n_per_point + pos] = (int32_t)(s - (long long)pt * n_per_point);
    }
}

// ------------------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------------------
// Cell grid for one launch.  dmax_d bounds |i0_d - i0_0| from the light travel time between the two sites.  The cell
// width trades the spread of window starts inside a tile (wasted MMA columns) against samples per cell (tiles that
// straddle two cells): a few hundred samples per occupied cell.
IleSortPlan ile_sort_plan(const IleSizes &sz, const IleDevParams &hp, long long n_per_point)
{
    IleSortPlan sp;
    sp.mode = 0;
    sp.g0 = 0;
    sp.nd = sz.n_det < 3 ? sz.n_det : 3;
    sp.g = n_per_point >= 200000 ? 4 : n_per_point >= 25000 ? 5 : n_per_point >= 3000 ? 6 : 7;
    sp.dmax[0] = 0;
    for (int d = 1; d < 3; ++d) {
        sp.dmax[d] = 0;
        if (d < sp.nd) {
            double dx = hp.vertex[d][0] - hp.vertex[0][0], dy = hp.vertex[d][1] - hp.vertex[0][1], dz = hp.vertex[d][2] - hp.vertex[0][2];
            double ds = sqrt(dx * dx + dy * dy + dz * dz) / ILE_C_SI * hp.fs;
            sp.dmax[d] = ds > 1.0e6 ? 1000000 : (int32_t)ceil(ds) + 2;
        }
    }
    for (;;) {
        sp.n0 = ((sz.n_q - sz.n_t) >> sp.g) + 1;
        sp.n1 = sp.nd > 1 ? ((2 * sp.dmax[1]) >> sp.g) + 1 : 1;
        sp.n2 = sp.nd > 2 ? ((2 * sp.dmax[2]) >> sp.g) + 1 : 1;
        long long nc = (long long)sp.n0 * sp.n1 * sp.n2 + 1;
        if (nc <= (1LL << 20) || sp.g >= 24) {
            sp.ncell = (int32_t)nc;
            break;
        }
        ++sp.g;  // keep the histogram small for exotic geometries
    }
    return sp;
}

template <int MMAX, bool SORT = true, bool QF = false>
static void setup_launch_t(unsigned blocks, const IleDevParams &hp, const IleEvalArgs &a, const IleMmaPlan &mp,
                           const IleSortPlan &sp, const IleMmaScratch &sc, cudaStream_t st)
{
    ile_setup_kernel<MMAX, SORT, QF><<<blocks, SETUP_THREADS, 0, st>>>(hp, a, mp.cp, sp, sc);
}

void ile_launch_setup_coef(const IleSizes &sz, const IleDevParams &hp, const IleEvalArgs &a, int32_t cp, const IleSortPlan &sp,
                           const IleMmaScratch &sc, cudaStream_t st)
{
    const long long n_total = a.n_per_point * a.n_points;
    long long blocks = (n_total + SETUP_THREADS - 1) / SETUP_THREADS;
    const long long cap = (long long)sz.sm_count * 16;
    if (blocks > cap) blocks = cap;
    IleMmaPlan mp;
    mp.cp = cp;
    const int M = sz.n_modes;
    if (sc.qform) {  // the quadratic forms were computed by ile_launch_quad_mma
        if (M <= 12) setup_launch_t<12, false, true>((unsigned)blocks, hp, a, mp, sp, sc, st);
        else if (M <= 21) setup_launch_t<21, false, true>((unsigned)blocks, hp, a, mp, sp, sc, st);
        else setup_launch_t<ILE_MAX_MODES, false, true>((unsigned)blocks, hp, a, mp, sp, sc, st);
    } else if (M <= 2) setup_launch_t<2, false>((unsigned)blocks, hp, a, mp, sp, sc, st);
    else if (M <= 5) setup_launch_t<5, false>((unsigned)blocks, hp, a, mp, sp, sc, st);
    else if (M <= 12) setup_launch_t<12, false>((unsigned)blocks, hp, a, mp, sp, sc, st);
    else if (M <= 21) setup_launch_t<21, false>((unsigned)blocks, hp, a, mp, sp, sc, st);
    else setup_launch_t<ILE_MAX_MODES, false>((unsigned)blocks, hp, a, mp, sp, sc, st);
}

cudaError_t ile_launch_setup_sort(const IleSizes &sz, const IleDevParams &hp, const IleEvalArgs &a, const IleMmaPlan &mp,
                                  const IleSortPlan &sp, const IleMmaScratch &sc, cudaStream_t st, int *n_launches)
{
    const long long n_total = a.n_per_point * a.n_points;
    cudaError_t e = cudaMemsetAsync(sc.hist, 0, (size_t)a.n_points * sp.ncell * sizeof(uint32_t), st);
    if (e != cudaSuccess) return e;
    long long blocks = (n_total + SETUP_THREADS - 1) / SETUP_THREADS;
    const long long cap = (long long)sz.sm_count * 16;
    if (blocks > cap) blocks = cap;
    const int M = sz.n_modes;
    if (M <= 2) setup_launch_t<2>((unsigned)blocks, hp, a, mp, sp, sc, st);
    else if (M <= 5) setup_launch_t<5>((unsigned)blocks, hp, a, mp, sp, sc, st);
    else if (M <= 12) setup_launch_t<12>((unsigned)blocks, hp, a, mp, sp, sc, st);
    else setup_launch_t<ILE_MAX_MODES>((unsigned)blocks, hp, a, mp, sp, sc, st);
    ile_scan_kernel<<<(unsigned)a.n_points, SCAN_THREADS, 0, st>>>(sp.ncell, sc.hist, sc.ngood);
    long long sblocks = (n_total + 255) / 256;
    if (sblocks > cap) sblocks = cap;
    ile_scatter_kernel<<<(unsigned)sblocks, 256, 0, st>>>(a.n_per_point, a.n_points, sp.ncell, sc.cell, sc.hist, sc.perm);
    if (n_launches) *n_launches += 3;
    return cudaGetLastError();
}
