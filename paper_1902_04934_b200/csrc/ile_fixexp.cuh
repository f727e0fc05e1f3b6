// ile_fixexp.cuh -- constants of the fixed-point exp shared by the streaming kernel (ile_eval_stream.cu) and the tiled kernel
// (ile_eval_tiled.cu); the table is made once per context by ile_stream_tab_kernel.
#pragma once
#ifndef ST_TAB_LOG2
#define ST_TAB_LOG2 11
#endif
#define ST_TAB (1 << ST_TAB_LOG2)

// ---- exp for the time marginalisation (eq. 9), in fixed point.  For an element x and a column reference of n octaves
//   t = fma(x, ST_C1, mg),  mg = ST_MAGIC - n * ST_TAB,  ST_C1 = ST_TAB / ln 2,  ST_MAGIC = 1.5 * 2^20
// is ONE rounding of  ST_MAGIC + y,  y = (x / ln 2 - n) * ST_TAB  (x - n ln 2 in table steps), to ulp(t) = 2^-32 as long as
// |y| < 2^19: the low word of t is the fraction f of y (32 bits, floor semantics), the 20 mantissa bits of the high word are
// [k + ST_KOFF | i] with y = ST_TAB k + i + f 2^-32.  Then
//   exp(x - n ln 2) = 2^k * 2^(i / ST_TAB) * exp(ln 2 / ST_TAB * f 2^-32) = 2^(k + ST_KOFF) * tab[i] * p(g)
// with tab[i] = 2^(i / ST_TAB - ST_KOFF) in shared memory, g = 1 + f 2^-32 assembled from the bits of f, and p the minimax quadratic
// of exp(ln 2 / ST_TAB (g - 1)) on [1, 2) (error 2.0e-13 at 2048 entries; the rounding of y adds 4e-14): four FP64 instructions per
// element -- the fma above, two for p, one to accumulate -- and the bit work on the integer pipes.  An element more than
// ST_UP_OCT octaves above the reference (or NaN, +inf) shows as a high word above ST_HI_UP and takes the rare path, which moves
// the reference; elements below -ST_KOFF + 6 octaves are clamped there (2^-250 of an element the sum already holds).
#define ST_MAGIC 1572864.0                       /* 1.5 * 2^20 */
#define ST_C1 (1.4426950408889634 * ST_TAB)      /* ST_TAB / ln 2 */
#define ST_KOFF (1 << (19 - ST_TAB_LOG2))        /* offset of the octave field; the table carries 2^-ST_KOFF */
#define ST_IDX_MASK (ST_TAB - 1)
#define ST_K_MASK (0xFFFFF & ~ST_IDX_MASK)
#define ST_UP_OCT (3 * ST_KOFF / 4)
#define ST_HI_UP (0x41300000 + ((ST_KOFF + ST_UP_OCT) << ST_TAB_LOG2))
#define ST_HI_FLOOR (0x41300000 + (6 << ST_TAB_LOG2))
#if ST_TAB_LOG2 == 11
#define ST_A0 0x1.ffd3a5661bac7p-1
#define ST_A1 0x1.62c56e9ca3a21p-12
#define ST_A2 0x1.ec1130cd9fbd5p-25
#else
#error "ST_TAB_LOG2: 11 (the minimax coefficients below belong to the 2048-entry table)"
#endif

// exp(x) for x <= 0 (max-subtracted arguments) from the table in GLOBAL memory (L1-resident, 16 KB): 4 FP64 instructions and a load
// where a Cody-Waite reduction with a degree-11 polynomial takes 17.  x below -250 octaves comes out as 2^-250 e^0..1 (negligible
// next to the maximum's 1); NaN propagates.
__device__ __forceinline__ double ile_fixexp_nonpos(double x, const double *__restrict__ tab)
{
    const double t = fma(x, ST_C1, ST_MAGIC);
    const int lo = __double2loint(t);
    const int hi = max(__double2hiint(t), ST_HI_FLOOR);
    const double T = __ldg(tab + (hi & ST_IDX_MASK));
    const double S = __hiloint2double(__double2hiint(T) + ((hi & ST_K_MASK) << (20 - ST_TAB_LOG2)), __double2loint(T));
    const double g = __hiloint2double((int)__funnelshift_r((unsigned)lo, 0x3FFu, 12), lo << 20);
    const double r = fma(fma(ST_A2, g, ST_A1), g, ST_A0) * S;
    return x == x ? r : x;
}
