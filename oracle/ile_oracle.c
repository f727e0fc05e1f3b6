/*
 * ile_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU statement of what the ILE hot path computes
 * (arXiv 1902.04934; line numbers are /root/reference/PAPER.md), in IEEE binary64,
 * sample by sample and bin by bin, in the paper's order and notation.  It shares no
 * code with the CUDA path (paper_1902_04934_b200/csrc) and neither includes the other.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call it.  Build: gcc -O2 -ffp-contract=off [-fopenmp] (no FMA contraction,
 * no blocking, no reordering beyond the loops written here).
 *
 * Steps (DESIGN.md lists the readings R1-R16 taken where the
 * paper is silent or garbled):
 *   O1 antenna response F_k = F+ + i Fx          PAPER.md L62, L69 (sign: reading R1), L79
 *   O2 arrival-time shift and window index        PAPER.md L62, L88 (sign: reading R2; rounding: R8)
 *   O3 spin-weight -2 harmonics Y_lm(iota,-phi)   PAPER.md L55-L60 (eq. 5-6; convention: R4, R5)
 *   O4 quadratic term (U, V)                      PAPER.md L66 (eq. 7), L91 (eq. 10)
 *   O5 lnL over the time window                   PAPER.md L64 (eq. 7), L88-L93 (eq. 10)
 *   O6 time marginalisation                       PAPER.md L81-L86 (eq. 9; rule: R7)
 *   O7 evidence, O8 n_eff                         PAPER.md L42-L47 (eq. 4), L101 (R12)
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"): every function below is pinned to
 * something other than itself -- brute-force eq. 1+2, closed forms, invariants.  Nothing
 * here is "parity unpinned".
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#define ILE_ORACLE_C_SI 299792458.0 /* m/s */

typedef double complex cplx;

/* ---------------------------------------------------------------- O1 ------------------------ */
/* F_k = F+,k + i Fx,k for one detector and one sky position / polarisation angle.
 * h_k = F+ h+ + Fx hx;  L79: F is time-independent (one GMST per event).
 * D = (x x^T - y y^T)/2 with x, y the unit arm directions; F+ = X.D.X - Y.D.Y, Fx = X.D.Y + Y.D.X,
 * X, Y the wave-frame axes of SURVEY.md §8(c) O1 (reading R6). */
void ile_oracle_antenna(const double arm_x[3], const double arm_y[3], double gmst, double ra, double dec,
                        double psi, double out_F[2])
{
    double D[3][3];
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++)
            D[i][j] = 0.5 * (arm_x[i] * arm_x[j] - arm_y[i] * arm_y[j]);
    double gha = gmst - ra;
    double X[3], Y[3];
    X[0] = -cos(psi) * sin(gha) - sin(psi) * cos(gha) * sin(dec);
    X[1] = -cos(psi) * cos(gha) + sin(psi) * sin(gha) * sin(dec);
    X[2] = sin(psi) * cos(dec);
    Y[0] = sin(psi) * sin(gha) - cos(psi) * cos(gha) * sin(dec);
    Y[1] = sin(psi) * cos(gha) + cos(psi) * sin(gha) * sin(dec);
    Y[2] = cos(psi) * cos(dec);
    double fp = 0.0, fc = 0.0;
    for (int i = 0; i < 3; i++) {
        double DX = D[i][0] * X[0] + D[i][1] * X[1] + D[i][2] * X[2];
        double DY = D[i][0] * Y[0] + D[i][1] * Y[1] + D[i][2] * Y[2];
        fp += X[i] * DX - Y[i] * DY;
        fc += X[i] * DY + Y[i] * DX;
    }
    out_F[0] = fp;
    out_F[1] = fc;
}

/* ---------------------------------------------------------------- O2 ------------------------ */
/* Arrival-time offset of detector k relative to the geocentre, seconds.
 * PAPER.md L62 (t_k = t_c - x_k.n), L88 (Q(t + n.x_k)); reading R2: s points Earth -> source,
 * dt_k = -(x_k . s)/c, so a detector nearer the source sees the wave earlier. */
double ile_oracle_delay(const double vertex_m[3], double gmst, double ra, double dec)
{
    double s[3];
    s[0] = cos(dec) * cos(ra - gmst);
    s[1] = cos(dec) * sin(ra - gmst);
    s[2] = sin(dec);
    double dot = vertex_m[0] * s[0] + vertex_m[1] * s[1] + vertex_m[2] * s[2];
    return -dot / ILE_ORACLE_C_SI;
}

/* First Q index of the N_t-bin window: nearest sample (round-half-even) minus N_t/2 (readings R8, R10). */
int32_t ile_oracle_window_index(double t_ref, double delay, double t0_q, double fs, int32_t n_t)
{
    double x = ((t_ref + delay) - t0_q) * fs;
    return (int32_t)rint(x) - n_t / 2;
}

/* ---------------------------------------------------------------- O3 ------------------------ */
static double factorial(int n)
{
    double r = 1.0;
    for (int i = 2; i <= n; i++) r *= (double)i;
    return r;
}

/* Wigner small-d d^l_{mp,m}(beta) by its finite sum (terms with a negative factorial argument dropped). */
double ile_oracle_wigner_d(int l, int mp, int m, double beta)
{
    double c = cos(0.5 * beta), s = sin(0.5 * beta);
    double pref = sqrt(factorial(l + m) * factorial(l - m) * factorial(l + mp) * factorial(l - mp));
    double sum = 0.0;
    for (int k = 0; k <= 2 * l; k++) {
        int a = l + m - k, b = k, cc = l - k - mp, d = k - m + mp;
        if (a < 0 || b < 0 || cc < 0 || d < 0) continue;
        double sign = ((k - m + mp) % 2 == 0) ? 1.0 : -1.0;
        double term = sign * pref / (factorial(a) * factorial(b) * factorial(cc) * factorial(d));
        term *= pow(c, (double)(2 * l - 2 * k + m - mp)) * pow(s, (double)(2 * k - m + mp));
        sum += term;
    }
    return sum;
}

/* _{-2}Y_lm(theta, phi) = sqrt((2l+1)/4pi) d^l_{m,2}(theta) e^{i m phi}   (reading R5). */
void ile_oracle_sYlm(int l, int m, double theta, double phi, double out[2])
{
    double amp = sqrt((2.0 * l + 1.0) / (4.0 * M_PI)) * ile_oracle_wigner_d(l, m, 2, theta);
    out[0] = amp * cos(m * phi);
    out[1] = amp * sin(m * phi);
}

/* ---------------------------------------------------------------- O4 ------------------------ */
/* quad = (a^2/4) sum_k [ |F_k|^2 Re(Y^dagger U_k Y) + Re(F_k^2 Y^T V_k Y) ]  (eq. 7; L91, eq. 10).
 * U, V: [K][M][M] complex, row-major, U[k][a][b] = <h_a|h_b>_k, V[k][a][b] = <h_a^*|h_b>_k (eq. 8b, 8c). */
double ile_oracle_quad(int K, int M, const cplx *F, const cplx *Y, const cplx *U, const cplx *V, double a)
{
    double tot = 0.0;
    for (int k = 0; k < K; k++) {
        cplx yuy = 0.0, yvy = 0.0;
        for (int p = 0; p < M; p++)
            for (int q = 0; q < M; q++) {
                yuy += conj(Y[p]) * U[((size_t)k * M + p) * M + q] * Y[q];
                yvy += Y[p] * V[((size_t)k * M + p) * M + q] * Y[q];
            }
        double F2 = creal(F[k]) * creal(F[k]) + cimag(F[k]) * cimag(F[k]);
        tot += F2 * creal(yuy) + creal(F[k] * F[k] * yvy);
    }
    return 0.25 * a * a * tot;
}

/* ---------------------------------------------------------------- O6 ------------------------ */
/* ln of (1/N_t) sum_j exp(lnL_j), max-subtracted  (eq. 9; rectangle rule, T = N_t dt: R7). */
double ile_oracle_margT(const double *lnL, int32_t n_t)
{
    double mx = lnL[0];
    for (int32_t j = 1; j < n_t; j++)
        if (lnL[j] > mx) mx = lnL[j];
    if (!(mx > -INFINITY)) return -INFINITY;
    double s = 0.0;
    for (int32_t j = 0; j < n_t; j++) s += exp(lnL[j] - mx);
    return mx + log(s) - log((double)n_t);
}

/* ---------------------------------------------------------------- O1-O6, one sample --------- */
/* Writes lnL_j, j = 0..N_t-1 (O5) into lnL_series (caller's buffer) and returns lnL_margT (O6).
 * shift_idx receives i0_k (O2).  A window leaving [0, N_Q) gives -inf and *oob = 1 (reading R9). */
double ile_oracle_sample(int K, int M, const int32_t *l, const int32_t *m, int32_t n_q, int32_t n_t, double fs,
                         double t0_q, double gmst, double d_ref, const double *vertex_m, const double *arm_x,
                         const double *arm_y, const cplx *Q, const cplx *U, const cplx *V, double ra, double dec,
                         double t_ref, double phi_ref, double psi, double incl, double dist, double *lnL_series,
                         int32_t *shift_idx, int *oob)
{
    cplx *F = (cplx *)malloc(sizeof(cplx) * (size_t)K);
    cplx *Y = (cplx *)malloc(sizeof(cplx) * (size_t)M);
    int32_t *i0 = (int32_t *)malloc(sizeof(int32_t) * (size_t)K);
    int bad = 0;
    for (int k = 0; k < K; k++) {
        double f[2];
        ile_oracle_antenna(arm_x + 3 * k, arm_y + 3 * k, gmst, ra, dec, psi, f); /* O1 */
        F[k] = f[0] + I * f[1];                                                  /* R1: F = F+ + i Fx */
        double dtk = ile_oracle_delay(vertex_m + 3 * k, gmst, ra, dec);          /* O2 */
        i0[k] = ile_oracle_window_index(t_ref, dtk, t0_q, fs, n_t);
        if (shift_idx) shift_idx[k] = i0[k];
        if (i0[k] < 0 || (int64_t)i0[k] + n_t > n_q) bad = 1;
    }
    for (int j = 0; j < M; j++) {
        double y[2];
        ile_oracle_sYlm(l[j], m[j], incl, -phi_ref, y); /* O3: Y_lm(iota, -phi_ref) (R4) */
        Y[j] = y[0] + I * y[1];
    }
    double result;
    if (bad) {
        for (int32_t j = 0; j < n_t; j++) lnL_series[j] = -INFINITY;
        result = -INFINITY;
    } else {
        double a = d_ref / dist;
        double quad = ile_oracle_quad(K, M, F, Y, U, V, a); /* O4 */
        for (int32_t j = 0; j < n_t; j++) {                 /* O5 */
            cplx acc = 0.0;
            for (int k = 0; k < K; k++)
                for (int mm = 0; mm < M; mm++)
                    acc += conj(F[k] * Y[mm]) * Q[((size_t)k * M + mm) * n_q + (size_t)(i0[k] + j)];
            lnL_series[j] = a * creal(acc) - quad;
        }
        result = ile_oracle_margT(lnL_series, n_t); /* O6 */
    }
    if (oob) *oob = bad;
    free(F), free(Y), free(i0);
    return result;
}

/* ---------------------------------------------------------------- batch (O1-O6 for n samples) */
/* Q, U, V are those of ONE intrinsic point.  Returns the number of out-of-range samples.
 * n_threads > 1 splits the sample loop with OpenMP when compiled with -fopenmp (samples are independent). */
int64_t ile_oracle_eval(int K, int M, const int32_t *l, const int32_t *m, int32_t n_q, int32_t n_t, double fs,
                        double t0_q, double gmst, double d_ref, const double *vertex_m, const double *arm_x,
                        const double *arm_y, const cplx *Q, const cplx *U, const cplx *V, int64_t n,
                        const double *ra, const double *dec, const double *t_ref, const double *phi_ref,
                        const double *psi, const double *incl, const double *dist, double *lnL_margT,
                        int32_t *shift_idx, int n_threads)
{
    int64_t n_bad = 0;
    (void)n_threads;
#ifdef _OPENMP
#pragma omp parallel num_threads(n_threads > 0 ? n_threads : 1) reduction(+ : n_bad)
#endif
    {
        double *series = (double *)malloc(sizeof(double) * (size_t)n_t);
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
        for (int64_t s = 0; s < n; s++) {
            int bad = 0;
            lnL_margT[s] = ile_oracle_sample(K, M, l, m, n_q, n_t, fs, t0_q, gmst, d_ref, vertex_m, arm_x, arm_y, Q,
                                             U, V, ra[s], dec[s], t_ref[s], phi_ref[s], psi[s], incl[s], dist[s],
                                             series, shift_idx ? shift_idx + s * K : NULL, &bad);
            n_bad += bad;
        }
        free(series);
    }
    return n_bad;
}

/* ---------------------------------------------------------------- O7, O8 -------------------- */
/* lnZ = ln( (1/n) sum_a w_a L_margT,a ), max-subtracted; n_eff = sum_a (w L)_a / max_a (w L)_a.
 * PAPER.md L42-L47 (eq. 4: Monte Carlo integral over theta), L101 (n_eff); reading R12.  log_w may be NULL (= 0). */
void ile_oracle_evidence(int64_t n, const double *lnL_margT, const double *log_w, double *lnZ, double *n_eff)
{
    double mx = -INFINITY;
    for (int64_t a = 0; a < n; a++) {
        double e = lnL_margT[a] + (log_w ? log_w[a] : 0.0);
        if (e > mx) mx = e;
    }
    if (!(mx > -INFINITY)) {
        *lnZ = -INFINITY;
        *n_eff = 0.0;
        return;
    }
    double s = 0.0;
    for (int64_t a = 0; a < n; a++) {
        double e = lnL_margT[a] + (log_w ? log_w[a] : 0.0);
        s += exp(e - mx);
    }
    *lnZ = mx + log(s) - log((double)n);
    *n_eff = s;
}
