// ile_setup.cu -- coefficient kernel of the streaming FP64-MMA evaluation path (variant 4): steps 1, 3, 4 of the hot path.
//
//   ile_setup_kernel    one thread per sample: F_k, Y_lm(iota, -phi_ref) (eq. 5-6), the
//                       quadratic term (eq. 7) and the coefficients a F_k Y_lm of the linear term, written as one
//                       record per sample.  Window starts, cell keys and the counting sort are the index kernel's job
//                       (ile_eval_stream.cu), which runs concurrently on the caller's stream.
#include <math_constants.h>
#include <string.h>

#include <type_traits>

#include "ile_kernels.h"

// ------------------------------------------------------------------------------------------------------------
// per-sample coefficients and quadratic term
// ------------------------------------------------------------------------------------------------------------
#define SETUP_THREADS 128
#ifndef SETUP_MINB
#define SETUP_MINB 6 /* <= 85 registers: 768 threads per SM, a 100,000-sample batch is one wave */
#endif

// U_k, V_k of ONE intrinsic point as a kernel parameter (constant bank): the 2 K M^2 entries are then operands of the multiply-adds
// instead of 2 K M^2 warp-uniform loads per thread (the long-scoreboard stalls on those loads were most of this kernel's time).
#define ILE_UVP_K 4
#define ILE_UVP_M 5
struct IleUVParams {
    double2 u[ILE_UVP_K][ILE_UVP_M][ILE_UVP_M], v[ILE_UVP_K][ILE_UVP_M][ILE_UVP_M];  // zero beyond (K, M, M)
};
struct IleUVNone {};

// One sample of the coefficient kernel.  QF: the quadratic forms Y^dagger U_k Y and Y^T V_k Y were computed by
// ile_launch_quad_mma (many modes).  UVP: U, V come from the parameter block uv (single-point launch, K <= ILE_UVP_K,
// M <= MMAX <= ILE_UVP_M; entries beyond (K, M, M) are zero, so no bounds are tested).
template <int MMAX, bool QF, bool UVP, class UV>
__device__ __forceinline__ void ile_setup_one(const IleDevParams &P, const IleEvalArgs &a, const int32_t cp, const IleSortScratch &sc,
                                              const UV &uv, const long long s)
{
    const int K = P.n_det, M = P.n_modes;
    const int recg = K * cp;
    const int pt = (int)(s / a.n_per_point);
    const size_t pglob = (size_t)(a.point0 + pt);
    const double2 *__restrict__ U = a.U + pglob * (size_t)K * M * M;
    const double2 *__restrict__ V = a.V + pglob * (size_t)K * M * M;

    // ---- step 1: sky geometry, antenna axes
    const IleSky g = ile_sky(a.ra[s], a.dec[s], a.psi[s], P.gmst);
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

    // ---- steps 1, 4 per detector; coefficients of the linear term
    double *__restrict__ rec = sc.rec + (size_t)s * recg;
    double tot = 0.0;
    auto detector = [&](const int k, auto KC) {
        constexpr int KP = decltype(KC)::value;  // UVP: k as a constant (index into the parameter block)
        const double2 F = ile_antenna(P.det_tensor[k], g);
        double yuy = 0.0;
        double2 yvy = make_double2(0.0, 0.0);
        if constexpr (QF) {  // many modes: Y^dagger U_k Y and Y^T V_k Y come from the FP64-MMA kernel (ile_quad_mma.cu)
            const double *__restrict__ q = sc.qform + ((size_t)s * K + k) * 3;
            yuy = q[0];
            yvy = make_double2(q[1], q[2]);
        } else {
#pragma unroll
            for (int p = 0; p < MMAX; ++p) {
                if (UVP || p < M) {
                    double2 tu = make_double2(0.0, 0.0), tv = make_double2(0.0, 0.0);
#pragma unroll
                    for (int q = 0; q < MMAX; ++q) {
                        if (UVP || q < M) {
                            double2 u, v;
                            if constexpr (UVP) {
                                u = uv.u[KP][p][q], v = uv.v[KP][p][q];
                            } else {
                                u = __ldg(U + ((size_t)k * M + p) * M + q), v = __ldg(V + ((size_t)k * M + p) * M + q);
                            }
                            const double2 Yq = Y[q];
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

        const double2 aF = make_double2(amp_a * F.x, amp_a * F.y);
        double2 *__restrict__ rk = reinterpret_cast<double2 *>(rec + (size_t)k * cp);
        if (P.interp) {  // reading R8': channels [0, 2M) weigh Q[i] by 1 - phi_k, channels [2M, 4M) weigh Q[i + 1] by phi_k
            double phi;
            ile_window_floor(P.vertex[k], g.s, a.t_ref[s], P.t0_q, P.fs, P.n_t, &phi);
            const double om = 1.0 - phi;
#pragma unroll
            for (int m = 0; m < MMAX; ++m)
                if (m < M) {
                    const double2 c = ile_cmul(aF, Y[m]);
                    rk[m] = make_double2(om * c.x, om * c.y);
                    rk[M + m] = make_double2(phi * c.x, phi * c.y);
                }
            for (int m = 2 * M; m < cp / 2; ++m) rk[m] = make_double2(0.0, 0.0);
        } else {
#pragma unroll
            for (int m = 0; m < MMAX; ++m)
                if (m < M) rk[m] = ile_cmul(aF, Y[m]);
            for (int m = M; m < cp / 2; ++m) rk[m] = make_double2(0.0, 0.0);
        }
    };
    if constexpr (UVP) {
        detector(0, std::integral_constant<int, 0>());
        if (K > 1) detector(1, std::integral_constant<int, 1>());
        if (K > 2) detector(2, std::integral_constant<int, 2>());
        if (K > 3) detector(3, std::integral_constant<int, 3>());
    } else {
        for (int k = 0; k < K; ++k) detector(k, std::integral_constant<int, 0>());
    }
    sc.quad[s] = 0.25 * amp_a * amp_a * tot;
}

template <int MMAX, bool QF>
__global__ void __launch_bounds__(SETUP_THREADS, (MMAX <= 5 ? SETUP_MINB : MMAX <= 12 ? 3 : 2))
    ile_setup_kernel(const __grid_constant__ IleDevParams P, const __grid_constant__ IleEvalArgs a, const int32_t cp,
                     const __grid_constant__ IleSortScratch sc)
{
    const long long n_total = a.n_per_point * a.n_points;
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < n_total; s += (long long)gridDim.x * blockDim.x)
        ile_setup_one<MMAX, QF, false>(P, a, cp, sc, IleUVNone(), s);
}

// single-point launches with few modes: U, V in the constant bank
template <int MMAX>
__global__ void __launch_bounds__(SETUP_THREADS, SETUP_MINB)
    ile_setup_uvp_kernel(const __grid_constant__ IleDevParams P, const __grid_constant__ IleEvalArgs a, const int32_t cp,
                         const __grid_constant__ IleSortScratch sc, const __grid_constant__ IleUVParams uv)
{
    const long long n_total = a.n_per_point;
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < n_total; s += (long long)gridDim.x * blockDim.x)
        ile_setup_one<MMAX, false, true>(P, a, cp, sc, uv, s);
}

// ------------------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------------------
template <int MMAX, bool QF = false>
static void setup_launch_t(unsigned blocks, const IleDevParams &hp, const IleEvalArgs &a, int32_t cp, const IleSortScratch &sc,
                           cudaStream_t st)
{
    ile_setup_kernel<MMAX, QF><<<blocks, SETUP_THREADS, 0, st>>>(hp, a, cp, sc);
}

// hU, hV: host mirrors of the context's U, V ([P][K][M][M]) or NULL.  Returns the number of kernels launched.
int ile_launch_setup_coef(const IleSizes &sz, const IleDevParams &hp, const IleEvalArgs &a, int32_t cp, const IleSortScratch &sc,
                          const double2 *hU, const double2 *hV, cudaStream_t st)
{
    const int M = sz.n_modes, K = sz.n_det;
    // few modes, one point per launch (a handful of launches for a handful of big points): U, V as kernel parameters
    if (!sc.qform && hU && hV && M <= ILE_UVP_M && K <= ILE_UVP_K && (a.n_points == 1 || (a.n_per_point >= 16384 && a.n_points <= 64))) {
        long long blocks = (a.n_per_point + SETUP_THREADS - 1) / SETUP_THREADS;
        const long long cap = (long long)sz.sm_count * 16;
        if (blocks > cap) blocks = cap;
        for (int32_t p = 0; p < a.n_points; ++p) {
            IleUVParams uv;
            memset(&uv, 0, sizeof(uv));
            const size_t base = (size_t)(a.point0 + p) * K * M * M;
            for (int k = 0; k < K; ++k)
                for (int i = 0; i < M; ++i)
                    for (int j = 0; j < M; ++j) {
                        uv.u[k][i][j] = hU[base + ((size_t)k * M + i) * M + j];
                        uv.v[k][i][j] = hV[base + ((size_t)k * M + i) * M + j];
                    }
            const long long off = (long long)p * a.n_per_point;
            IleEvalArgs g = a;
            g.point0 = a.point0 + p, g.n_points = 1;
            g.ra = a.ra + off, g.dec = a.dec + off, g.t_ref = a.t_ref + off, g.phi_ref = a.phi_ref + off, g.psi = a.psi + off;
            g.incl = a.incl + off, g.dist = a.dist + off;
            IleSortScratch scp = sc;
            scp.rec = sc.rec + (size_t)off * K * cp;
            scp.quad = sc.quad + off;
            if (M <= 2) ile_setup_uvp_kernel<2><<<(unsigned)blocks, SETUP_THREADS, 0, st>>>(hp, g, cp, scp, uv);
            else ile_setup_uvp_kernel<5><<<(unsigned)blocks, SETUP_THREADS, 0, st>>>(hp, g, cp, scp, uv);
        }
        return a.n_points;
    }
    const long long n_total = a.n_per_point * a.n_points;
    long long blocks = (n_total + SETUP_THREADS - 1) / SETUP_THREADS;
    const long long cap = (long long)sz.sm_count * 16;
    if (blocks > cap) blocks = cap;
    if (sc.qform) {  // the quadratic forms were computed by ile_launch_quad_mma
        if (M <= 12) setup_launch_t<12, true>((unsigned)blocks, hp, a, cp, sc, st);
        else if (M <= 21) setup_launch_t<21, true>((unsigned)blocks, hp, a, cp, sc, st);
        else setup_launch_t<ILE_MAX_MODES, true>((unsigned)blocks, hp, a, cp, sc, st);
    } else if (M <= 2) setup_launch_t<2>((unsigned)blocks, hp, a, cp, sc, st);
    else if (M <= 5) setup_launch_t<5>((unsigned)blocks, hp, a, cp, sc, st);
    else if (M <= 12) setup_launch_t<12>((unsigned)blocks, hp, a, cp, sc, st);
    else if (M <= 21) setup_launch_t<21>((unsigned)blocks, hp, a, cp, sc, st);
    else setup_launch_t<ILE_MAX_MODES>((unsigned)blocks, hp, a, cp, sc, st);
    return 1;
}
