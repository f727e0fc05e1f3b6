// ile_device.cuh -- device-side parameter block and the per-sample geometry shared by every evaluation kernel.
//
// Steps 1-4 of the hot path: antenna response F_k, arrival-time
// delay and window index (L62, L88), harmonics Y_lm(iota, -phi_ref) (eq. 5-6), quadratic term
// (eq. 7).  No code here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/ile.h"

#define ILE_MAX_TERMS 8 /* terms of the Wigner-d finite sum for l <= ILE_MAX_L and m' = 2: at most l - 1 */

struct IleDevParams {
    int32_t n_points, n_det, n_modes, n_q, n_t;
    int32_t interp;  // 1: linear interpolation of Q between samples (reading R8')
    double fs, t0_q, gmst, d_ref;
    double det_tensor[ILE_MAX_DET][6];  // D = (x x^T - y y^T)/2, symmetric: xx, xy, xz, yy, yz, zz
    double vertex[ILE_MAX_DET][3];      // metres
    int32_t mode_m[ILE_MAX_MODES];
    int32_t mode_nterm[ILE_MAX_MODES];
    // sqrt((2l+1)/4pi) d^l_{m,2}(iota) = sum_t coef[t] cos(iota/2)^pc[t] sin(iota/2)^ps[t]
    double mode_coef[ILE_MAX_MODES][ILE_MAX_TERMS];
    int8_t mode_pc[ILE_MAX_MODES][ILE_MAX_TERMS];
    int8_t mode_ps[ILE_MAX_MODES][ILE_MAX_TERMS];
};

#define ILE_C_SI 299792458.0

__device__ __forceinline__ double ile_ipow(double x, int n)
{
    double r = 1.0;
    while (n > 0) {
        if (n & 1) r *= x;
        x *= x;
        n >>= 1;
    }
    return r;
}

// Sky- and polarisation-dependent part of one sample: wave-frame axes X, Y and the source direction s.
struct IleSky {
    double X[3], Y[3], s[3];
};

// Unit vector Earth -> source from (RA, dec, GMST); also returns the sines and cosines it is built from.  Products are
// rounded one by one (no FMA) so that the window index derived from it is reproducible wherever it is computed.
__device__ __forceinline__ void ile_source_dir(double ra, double dec, double gmst, double s[3], double *sl, double *cl,
                                               double *sd, double *cd)
{
    double lon = ra - gmst;  // = -(Greenwich hour angle)
    sincos(lon, sl, cl);
    sincos(dec, sd, cd);
    s[0] = __dmul_rn(*cd, *cl);
    s[1] = __dmul_rn(*cd, *sl);
    s[2] = *sd;
}

__device__ __forceinline__ IleSky ile_sky(double ra, double dec, double psi, double gmst)
{
    IleSky g;
    double sl, cl, sd, cd, sp, cp;
    ile_source_dir(ra, dec, gmst, g.s, &sl, &cl, &sd, &cd);
    sincos(psi, &sp, &cp);
    // psi = 0: X local west, Y local north; X x Y = propagation direction; psi rotates X toward Y  (reading R6)
    double sg = -sl, cg = cl;  // sin, cos of gha = gmst - ra
    g.X[0] = -cp * sg - sp * cg * sd;
    g.X[1] = -cp * cg + sp * sg * sd;
    g.X[2] = sp * cd;
    g.Y[0] = sp * sg - cp * cg * sd;
    g.Y[1] = sp * cg + cp * sg * sd;
    g.Y[2] = cp * cd;
    return g;
}

// F_k = F+ + i Fx = D : (XX - YY) + i D : (XY + YX)   (reading R1: F = F+ + i Fx)
__device__ __forceinline__ double2 ile_antenna(const double *__restrict__ D, const IleSky &g)
{
    double DX0 = D[0] * g.X[0] + D[1] * g.X[1] + D[2] * g.X[2];
    double DX1 = D[1] * g.X[0] + D[3] * g.X[1] + D[4] * g.X[2];
    double DX2 = D[2] * g.X[0] + D[4] * g.X[1] + D[5] * g.X[2];
    double DY0 = D[0] * g.Y[0] + D[1] * g.Y[1] + D[2] * g.Y[2];
    double DY1 = D[1] * g.Y[0] + D[3] * g.Y[1] + D[4] * g.Y[2];
    double DY2 = D[2] * g.Y[0] + D[4] * g.Y[1] + D[5] * g.Y[2];
    double fp = (g.X[0] * DX0 + g.X[1] * DX1 + g.X[2] * DX2) - (g.Y[0] * DY0 + g.Y[1] * DY1 + g.Y[2] * DY2);
    double fc = 2.0 * (g.X[0] * DY0 + g.X[1] * DY1 + g.X[2] * DY2);
    return make_double2(fp, fc);
}

// Window start i0_k = rint(((t_ref + dt_k) - t0_Q) f_s) - floor(N_t/2), dt_k = -(x_k . s)/c  (readings R2, R8).
// Every operation is individually rounded, in a fixed order, so the integer is reproducible.
__device__ __forceinline__ int32_t ile_window_index(const double *__restrict__ v, const double *__restrict__ s,
                                                    double t_ref, double t0_q, double fs, int32_t n_t)
{
    double dot = __dadd_rn(__dadd_rn(__dmul_rn(v[0], s[0]), __dmul_rn(v[1], s[1])), __dmul_rn(v[2], s[2]));
    double dt = __ddiv_rn(-dot, ILE_C_SI);
    double x = __dmul_rn(__dsub_rn(__dadd_rn(t_ref, dt), t0_q), fs);
    return __double2int_rn(x) - n_t / 2;
}

// The same expression floored instead of rounded, with the fractional part (reading R8': linear interpolation between samples).
__device__ __forceinline__ int32_t ile_window_floor(const double *__restrict__ v, const double *__restrict__ s, double t_ref,
                                                    double t0_q, double fs, int32_t n_t, double *phi)
{
    double dot = __dadd_rn(__dadd_rn(__dmul_rn(v[0], s[0]), __dmul_rn(v[1], s[1])), __dmul_rn(v[2], s[2]));
    double dt = __ddiv_rn(-dot, ILE_C_SI);
    double x = __dmul_rn(__dsub_rn(__dadd_rn(t_ref, dt), t0_q), fs);
    double fl = floor(x);
    *phi = __dsub_rn(x, fl);
    return (int32_t)fl - n_t / 2;
}

// Y_lm(iota, -phi_ref) = [sum_t coef_t c^pc_t s^ps_t] e^{-i m phi_ref}, c = cos(iota/2), s = sin(iota/2)  (R4, R5)
__device__ __forceinline__ double2 ile_ylm(const IleDevParams *__restrict__ P, int mode, double ch, double sh,
                                           double phi_ref)
{
    double amp = 0.0;
    int nt = P->mode_nterm[mode];
    for (int t = 0; t < nt; ++t)
        amp += P->mode_coef[mode][t] * ile_ipow(ch, P->mode_pc[mode][t]) * ile_ipow(sh, P->mode_ps[mode][t]);
    double sm, cm;
    sincos((double)P->mode_m[mode] * phi_ref, &sm, &cm);
    return make_double2(amp * cm, -amp * sm);
}

__device__ __forceinline__ double2 ile_cmul(double2 a, double2 b)
{
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// ------------------------------------------------------------------------------------------------------------
// per-sample setup, one THREAD per sample (no redundant geometry across a warp): steps 1-4
// ------------------------------------------------------------------------------------------------------------
// On return: A[k*ldA + m] = (D_ref/D) F_k Y_m (so that lin_j = Re sum conj(A) Q), entries m in [M, ldA) zeroed,
// i0[k] = window start, returns quad = (a^2/4) sum_k [|F_k|^2 Re(Y^dagger U_k Y) + Re(F_k^2 Y^T V_k Y)]
// (eq. 7; U is not assumed Hermitian: reading R15).  *bad is set when a window leaves [0, n_q) (reading R9).
__device__ __forceinline__ double ile_setup_sample(const IleDevParams *__restrict__ P, const double2 *__restrict__ U,
                                                   const double2 *__restrict__ V, double ra, double dec, double t_ref,
                                                   double phi_ref, double psi, double incl, double dist, double2 *A,
                                                   int ldA, int32_t *i0, int *bad, double *phi = nullptr)
{
    const int K = P->n_det, M = P->n_modes;
    IleSky g = ile_sky(ra, dec, psi, P->gmst);
    double sh, ch;
    sincos(0.5 * incl, &sh, &ch);
    const double a = P->d_ref / dist;
    for (int m = 0; m < M; ++m) A[m] = ile_ylm(P, m, ch, sh, phi_ref);  // Y_m, parked in the k = 0 row

    double tot = 0.0;
    int oob = 0;
    for (int k = 0; k < K; ++k) {
        double2 F = ile_antenna(P->det_tensor[k], g);
        double yuy = 0.0;
        double2 yvy = make_double2(0.0, 0.0);
        for (int p = 0; p < M; ++p) {
            double2 tu = make_double2(0.0, 0.0), tv = make_double2(0.0, 0.0);
            const double2 *Ur = U + ((size_t)k * M + p) * M;
            const double2 *Vr = V + ((size_t)k * M + p) * M;
            for (int q = 0; q < M; ++q) {
                double2 Yq = A[q], u = __ldg(Ur + q), v = __ldg(Vr + q);
                tu.x += u.x * Yq.x - u.y * Yq.y;
                tu.y += u.x * Yq.y + u.y * Yq.x;
                tv.x += v.x * Yq.x - v.y * Yq.y;
                tv.y += v.x * Yq.y + v.y * Yq.x;
            }
            double2 Yp = A[p];
            yuy += Yp.x * tu.x + Yp.y * tu.y;  // Re(conj(Y_p) (U Y)_p)
            double2 t = ile_cmul(Yp, tv);
            yvy.x += t.x;
            yvy.y += t.y;
        }
        double F2 = F.x * F.x + F.y * F.y;
        double2 FF = ile_cmul(F, F);
        tot += F2 * yuy + (FF.x * yvy.x - FF.y * yvy.y);
        int32_t idx;
        if (phi) {  // interpolated shifts: one sample more is read
            idx = ile_window_floor(P->vertex[k], g.s, t_ref, P->t0_q, P->fs, P->n_t, phi + k);
            if (idx < 0 || (long long)idx + P->n_t + 1 > P->n_q) oob = 1;
        } else {
            idx = ile_window_index(P->vertex[k], g.s, t_ref, P->t0_q, P->fs, P->n_t);
            if (idx < 0 || (long long)idx + P->n_t > P->n_q) oob = 1;
        }
        i0[k] = idx;
    }
    for (int k = K - 1; k >= 0; --k) {  // k = 0 last: it overwrites the parked Y_m in place
        double2 F = ile_antenna(P->det_tensor[k], g);
        double2 aF = make_double2(a * F.x, a * F.y);
        for (int m = 0; m < M; ++m) A[k * ldA + m] = ile_cmul(aF, A[m]);
        for (int m = M; m < ldA; ++m) A[k * ldA + m] = make_double2(0.0, 0.0);
    }
    *bad = oob;
    return 0.25 * a * a * tot;
}

__device__ __forceinline__ double warp_max(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
