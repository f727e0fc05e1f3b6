// ile_eval_stream.cu -- variant 4: streaming FP64-MMA evaluation, one warp per group of 8 samples (steps 5-6 of the hot path).
//
// The linear term lin_j = Re sum_k sum_lm conj(A_k,lm) Q_k,lm[i0_k + j]  (eq. 7 / eq. 10; "the most
// costly part", L97) is, per detector, the dense contraction  T_k[i][alpha] = sum_c Qc_k[i][c] Ac_k[c][alpha]  over the 2M real
// channels c = (mode, re/im) -- "the necessary matrix multiplication" of L97 -- followed by a per-sample shift j = i - i0_k(alpha).
// It runs on the FP64 matrix instruction DMMA.8x8x4 (mma.sync.m8n8k4.f64): A = Q [8 time rows x 4 channels], B = coefficients
// [4 channels x 8 samples], C = lin [8 time rows x 8 samples].  On B200 DMMA and DFMA share the FP64 units (measured: their
// times add), so DMMA buys no arithmetic; it buys issue slots and operand delivery: one instruction does 8 DFMA per lane.
//
// Nothing of lin ever goes through shared memory and no block-level barrier exists.  A warp owns 8 samples for the whole window and streams over 8-row time blocks:
//   * rows are absolute time rows of detector 0 (row rho <-> Q_0 row G0 + rho, G0 = the group's smallest window start); a
//     sample's own window start inside the group, delta0 = i0_0 - G0, only decides WHICH rows enter its log-sum-exp;
//   * detector k >= 1 is evaluated on rows base_k + rho with base_k = G0 + min over the group of d_k = i0_k - i0_0; the
//     remaining per-sample offset eps_k = d_k - min d_k (0 <= eps_k < 8 NC, guaranteed by the sort: samples of a group come
//     from one (d_1, d_2) cell of width 8 NC) is applied to the C fragment in registers: the lane that holds row r' picks,
//     among the NC + 1 live blocks of that detector, the one its destination lane needs and one 64-bit warp shuffle moves
//     it to row (r' - eps) mod 8.  The shifted partial sums are the C input of detector 0's MMA, so the detector sum costs
//     K - 2 additions per element;
//   * the time marginalisation (eq. 9) is an online log-sum-exp per lane: a running reference of a whole number of
//     octaves and s = sum exp(lin) 2^-ref; an element more than 192 octaves above the reference moves it (rare: lin(t) is
//     smooth on the scale of a block).  exp runs in fixed point (see ST_MAGIC below): one FMA puts lin / ln 2 - ref into the
//     mantissa, a 2048-entry table of 2^(i/2048) in shared memory and a quadratic in the remaining 32 fraction bits do the rest --
//     4 FP64 instructions per element (round 1-2a: 9), relative error 2.4e-13.
// Per 8-row block and warp: K*KS DMMA (16 pipe cycles each), 2 x 4 FP64 operations of log-sum-exp, K*KS coalesced 256-byte
// fragment loads that hit L1 (consecutive groups use the same rows), 4 (K-1) SHFL.
//
// Q is repacked once per context as Qs[point][k][row / 8][s][row % 8][4]: the A fragment of (detector k, k-step s, rows
// base..base+7) is two contiguous runs of 32-byte rows (one if base is a multiple of 8) -- a 256-byte load per DMMA that touches
// 2-3 lines -- and the fragments of the other k-steps and of the following 8-row blocks lie at compile-time offsets from it, so
// a lane keeps ONE pointer per detector.  The series are zero padded in front and behind so that rows outside [0, N_Q), which only
// ever feed elements outside every window, read as zeros.
#include <cstdio>
#include <limits.h>
#include <math_constants.h>

#include <type_traits>

#include "ile_kernels.h"

#define ST_FULL 0xffffffffu
#ifndef ST_THREADS
#define ST_THREADS 128
#endif
#ifndef ST_MINB3
#define ST_MINB3 3
#endif
#ifndef ST_PIPE_MAXKS
#define ST_PIPE_MAXKS 4
#endif

__device__ __forceinline__ void st_dmma(double &c0, double &c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

#include "ile_fixexp.cuh"
#define ST_MG_UNSET (ST_MAGIC + 1073741824.0 * ST_TAB) /* reference at -2^30 octaves: the first valid element takes the rare path */

// 2^d for an integer-valued d <= 0; 0 below -1000
__device__ __forceinline__ double st_pow2_neg(double d)
{
    return d > -1000.0 ? __hiloint2double((1023 + (int)d) << 20, 0) : 0.0;
}

// octaves of the reference held in mg
__device__ __forceinline__ double st_ref_oct(double mg) { return (ST_MAGIC - mg) * (1.0 / ST_TAB); }

// rare path: element x becomes the reference of its column
__device__ __forceinline__ void st_reref(double x, double &mg, double &s)
{
    if (!(fabs(x) < 1.0e15)) {  // NaN, +inf: poison the sum (the reference stays, so every later element comes here too)
        s = CUDART_NAN;
        return;
    }
    const double n_new = rint(x * 1.4426950408889634);
    s *= st_pow2_neg(st_ref_oct(mg) - n_new);
    mg = ST_MAGIC - n_new * ST_TAB;
}

// Log-sum-exp of a pair of blocks (b = 0, 1) of the lane's two columns (c = 0, 1; column c carries (mg[c], s[c])), in two halves.
// First half: t for the lane's four elements; one branch for the four (rare: lin(t) is smooth on the scale of a block).  The
// elements of a column are taken in block order and all of them redone against the final reference (none has been added yet).
//   v : the element lies inside the sample's window (PRED only; otherwise every element does)
// Second half, branch free: s += 2^(k + ST_KOFF) tab[i] p(g).
template <bool PRED>
__device__ __forceinline__ void st_lse_pre2(const double (&x)[2][2], const bool (&v)[2][2], double (&mg)[2], double (&s)[2],
                                            double (&t)[2][2])
{
    bool any = false;
#pragma unroll
    for (int b = 0; b < 2; ++b)
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            t[b][c] = fma(x[b][c], ST_C1, mg[c]);
            bool g = __double2hiint(t[b][c]) > ST_HI_UP;
            if (PRED) g = g && v[b][c];
            any = any || g;
        }
    if (any) {
#pragma unroll
        for (int c = 0; c < 2; ++c) {
#pragma unroll
            for (int b = 0; b < 2; ++b) {
                bool g = __double2hiint(fma(x[b][c], ST_C1, mg[c])) > ST_HI_UP;
                if (PRED) g = g && v[b][c];
                if (g) st_reref(x[b][c], mg[c], s[c]);
            }
            t[0][c] = fma(x[0][c], ST_C1, mg[c]);
            t[1][c] = fma(x[1][c], ST_C1, mg[c]);
        }
    }
}

template <bool PRED>
__device__ __forceinline__ void st_lse_main2(const double (&t)[2][2], const bool (&v)[2][2], double (&s)[2], uint32_t tab)
{
    double e[2][2], S[2][2];
#pragma unroll
    for (int b = 0; b < 2; ++b)
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const int lo = __double2loint(t[b][c]);
            const int hi = max(__double2hiint(t[b][c]), ST_HI_FLOOR);
            double T;
            asm("ld.shared.f64 %0, [%1];" : "=d"(T) : "r"(tab + ((uint32_t)(hi & ST_IDX_MASK) << 3)));
            int Sh = __double2hiint(T) + ((hi & ST_K_MASK) << (20 - ST_TAB_LOG2));
            int Sl = __double2loint(T);
            if (PRED) {
                Sh = v[b][c] ? Sh : 0;
                Sl = v[b][c] ? Sl : 0;
            }
            S[b][c] = __hiloint2double(Sh, Sl);
            const double g = __hiloint2double((int)__funnelshift_r((unsigned)lo, 0x3FFu, 12), lo << 20);
            e[b][c] = fma(fma(ST_A2, g, ST_A1), g, ST_A0);
        }
#pragma unroll
    for (int c = 0; c < 2; ++c) s[c] = fma(e[1][c], S[1][c], fma(e[0][c], S[0][c], s[c]));
}

// loads of per-sample data that is used once: keep them from evicting the Q rows the SM's warps share in L1
#ifndef ST_STREAM_LD
#define ST_STREAM_LD(p) __ldcs(p)
#endif

__device__ __forceinline__ double st_shfl(double v, int src) { return __shfl_sync(ST_FULL, v, src); }


// m ? b : a for an all-ones / all-zeros mask m: two LOP3, no predicate
__device__ __forceinline__ double st_bsel(double a, double b, int m)
{
    const int al = __double2loint(a), ah = __double2hiint(a), bl = __double2loint(b), bh = __double2hiint(b);
    return __hiloint2double(ah ^ ((ah ^ bh) & m), al ^ ((al ^ bl) & m));
}

// ln S + n ln 2 for a finite S > 0 (else through log()): S = 2^e m, m in [1, 2); with c the table centre next to m,
// r = m / c - 1 (one rounding, |r| <= 2^-8) and ln m = ln c + (r - r^2/2 + ... - r^6/6), truncation 2e-18.  A dozen FP64
// instructions where log() issues several dozen -- behind the other warps' DMMAs each of them waits for the pipe.
__device__ __forceinline__ double st_log_plus(double S, double n, const double2 *__restrict__ ltab)
{
    const int hi = __double2hiint(S);
    if ((unsigned)(hi - 0x00100000) >= 0x7fe00000u) return fma(n, 0.6931471805599453, log(S));  // 0, subnormal, inf, NaN, negative
    const double m = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(S));
    const double2 t = ltab[(hi >> 13) & 127];
    const double r = fma(m, t.x, -1.0);
    double q = fma(r, -1.0 / 6.0, 0.2);
    q = fma(q, r, -0.25);
    q = fma(q, r, 1.0 / 3.0);
    q = fma(q, r, -0.5);
    q = fma(q * r, r, r);
    return fma(n + (double)((hi >> 20) - 1023), 0.6931471805599453, t.y + q);
}

struct IleStreamKArgs {
    int32_t n_t, point0, n_points, nqp, padf, recg, cp;
    int64_t n_per_point, slot_cap;
    const double *Qs;
    const double *rec;
    const double *quad;
    const int32_t *i0;
    const int32_t *slots;
    const int32_t *gcum;
    uint32_t *rcnt;         // [n_ranges] claim counters, zero at launch (the previous launch cleaned them: rcnt_next)
    uint32_t *rcnt_next;    // the claim counters of the NEXT launch, and
    uint32_t *zero_ptr;     // the sort's histograms and segment totals (not needed any more): zeroed here, so that no memset
    long long zero_n;       // stands in front of the next launch's index kernel
    int32_t n_ranges;
    double *lnL;
    const double *tabs;     // [ST_TAB] exp table, then [128][2] log table (ile_stream_tab_kernel, once per context)
};

template <int K, int KS, int NC, int MINB>
__global__ void __launch_bounds__(ST_THREADS, MINB) ile_eval_stream_kernel(const __grid_constant__ IleStreamKArgs a)
{
    __shared__ __align__(128) double tab[ST_TAB];
    __shared__ __align__(16) double2 ltab[128];  // (1 / c_i rounded, -ln of that) for c_i = 1 + (i + 1/2) / 128: st_log
    for (int i = threadIdx.x; i < ST_TAB; i += blockDim.x) tab[i] = a.tabs[i];
    for (int i = threadIdx.x; i < 128; i += blockDim.x) ltab[i] = make_double2(a.tabs[ST_TAB + 2 * i], a.tabs[ST_TAB + 2 * i + 1]);
    __syncthreads();
    const uint32_t tab_addr = (uint32_t)__cvta_generic_to_shared(tab);
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < a.zero_n; i += (long long)gridDim.x * blockDim.x) a.zero_ptr[i] = 0u;
    if (blockIdx.x == 0)
        for (int i = threadIdx.x; i < ILE_STREAM_MAX_RANGES; i += blockDim.x) a.rcnt_next[i] = 0u;

    const int lane = threadIdx.x & 31, r = lane >> 2, cc = lane & 3;
    const int n_t = a.n_t;
    const double log_nt = log((double)n_t);
    const int total = a.gcum[a.n_points];

    // Work distribution: the group list (all points, each in window-start order) is cut into n_ranges contiguous ranges of rq groups
    // and an SM works through the range of its own id, so that the warps of one SM stream the same few hundred rows of Q and the
    // fragments stay in its L1.  A warp whose range is used up moves on to another range for good (ranges only shrink).  Small
    // launches have ONE range (a plain global counter).
    unsigned smid;
    asm("mov.u32 %0, %%smid;" : "=r"(smid));
    const int nr = a.n_ranges;
    const int rq = (total + nr - 1) / nr;
    int rg = (int)(smid % (unsigned)nr);
    // the claim of a group is issued while the previous one is streamed (tn: lane 0's ticket in range rg)
    unsigned tn = 0;
    if (lane == 0) tn = atomicAdd(a.rcnt + rg, 1u);
    for (;;) {
        int w = -1;
        for (;;) {
            const int lo = rg * rq, hi = min(lo + rq, total);
            const unsigned t = __shfl_sync(ST_FULL, tn, 0);
            if (t < (unsigned)max(hi - lo, 0)) {
                w = lo + (int)t;
                break;
            }
            // own range used up: the lanes look at 32 other ranges at a time for one with groups left
            int found = -1;
            for (int base = 1; base < nr && found < 0; base += 32) {
                const int off = base + lane;
                int cand = rg + off;
                if (cand >= nr) cand -= nr;
                bool left = false;
                if (off < nr) {
                    const int clo = cand * rq, chi = min(clo + rq, total);
                    left = *((volatile uint32_t *)a.rcnt + cand) < (unsigned)max(chi - clo, 0);
                }
                const unsigned mk = __ballot_sync(ST_FULL, left);
                if (mk) {
                    found = rg + base + __ffs(mk) - 1;
                    if (found >= nr) found -= nr;
                }
            }
            if (found < 0) break;
            rg = found;
            if (lane == 0) tn = atomicAdd(a.rcnt + rg, 1u);
        }
        if (w < 0) break;
        if (lane == 0) tn = atomicAdd(a.rcnt + rg, 1u);  // the next group's ticket
        int pt = 0;
        if (a.n_points > 1) {
            int lo = 0, hi = a.n_points;
            while (hi - lo > 1) {
                const int mid = (lo + hi) >> 1;
                if (a.gcum[mid] <= w) lo = mid;
                else hi = mid;
            }
            pt = lo;
        }
        const int g = w - a.gcum[pt];  // groups in slot order: segment by segment, window starts ascending inside a segment
        const int32_t *__restrict__ slots = a.slots + (size_t)pt * a.slot_cap + 8 * (size_t)g;
        const long long sbase = (long long)pt * a.n_per_point;

        // ---- the group: window starts, bases, per-sample offsets.  Lane (r, cc) looks after (sample r, detector cc).
        const int sb = ST_STREAM_LD(slots + r);  // -1: empty slot (the group is the tail of its segment)
        const bool has = sb >= 0;
        const long long fb = sbase + (has ? sb : 0);
        const int my_i0 = (has && cc < K) ? ST_STREAM_LD(a.i0 + fb * K + cc) : 0;
        const int i00 = __shfl_sync(ST_FULL, my_i0, lane & ~3);
        const int G0 = __reduce_min_sync(ST_FULL, has ? i00 : INT_MAX);
        const int dspread = __reduce_max_sync(ST_FULL, has ? i00 - G0 : 0);
        const int dk = my_i0 - i00;
        int eps_mine = 0;
        int base[K];
        base[0] = G0;
#pragma unroll
        for (int k = 1; k < K; ++k) {
            const int mn = __reduce_min_sync(ST_FULL, (has && cc == k) ? dk : INT_MAX);
            base[k] = G0 + mn;
            if (has && cc == k) eps_mine = dk - mn;
        }
        const int del_mine = has ? i00 - G0 : (1 << 28);

        // ---- this lane's two C-fragment columns: samples 2cc and 2cc + 1
        const int lA = 8 * cc, lB = 8 * cc + 4;
        const int sA = __shfl_sync(ST_FULL, sb, lA), sB = __shfl_sync(ST_FULL, sb, lB);
        const int jA = r - __shfl_sync(ST_FULL, del_mine, lA), jB = r - __shfl_sync(ST_FULL, del_mine, lB);  // j of block 0
        // per shifted detector k and column c: src = the lane that holds my row; off = as a source, the block (relative to
        // the destination's) my destination lane wants
        int src[K][2], msk[K][2][NC];
#pragma unroll
        for (int k = 1; k < K; ++k) {
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                const int e = __shfl_sync(ST_FULL, eps_mine, 8 * cc + 4 * c + k);
                src[k][c] = (((r + e) & 7) << 2) | cc;
                const int off = (((r - e) & 7) + e) >> 3;
#pragma unroll
                for (int o = 0; o < NC; ++o) msk[k][c][o] = off == o + 1 ? -1 : 0;
            }
        }
        const int jc[2] = {jA, jB};

        const int nblk = ((dspread + n_t + 7) >> 3) + 1 & ~1;  // even: the stream advances two blocks per step
        const int t_lo = (dspread + 7) >> 3, t_hi = n_t >> 3;  // blocks [t_lo, t_hi) lie inside every window of the group

        // ---- B fragments: coefficients a F_k Y_lm of sample r, channels 4s + cc
        double bf[K][KS];
        {
            const double *__restrict__ rp = a.rec + (size_t)fb * a.recg + cc;
#pragma unroll
            for (int k = 0; k < K; ++k)
#pragma unroll
                for (int s = 0; s < KS; ++s) bf[k][s] = has ? ST_STREAM_LD(rp + k * a.cp + 4 * s) : 0.0;
        }
        // ---- A fragment pointers: pk[k] = this lane's element (row base_k + r, channel cc) of k-step 0 of detector k.  The packed
        // series is blocked by 8 rows with a block's KS k-steps side by side, so the other k-steps and the next 8-row blocks of the
        // lane are at compile-time offsets: (blocks * KS + s) * 32 doubles.
        const double *pk[K];
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const int row = a.padf + base[k] + r;
            pk[k] = a.Qs + (size_t)((a.point0 + pt) * K + k) * KS * a.nqp * 4 + (size_t)(row >> 3) * (KS * 32) + (row & 7) * 4 + cc;
        }

        // ---- prologue: blocks 0 .. NC-1 of the shifted detectors into the ring (slot of block b = b % 4); first fragments
        double ring[K > 1 ? K - 1 : 1][4][2];
#pragma unroll
        for (int k = 1; k < K; ++k) {
#pragma unroll
            for (int u = 0; u < NC; ++u) {
                double c0 = 0.0, c1 = 0.0;
#pragma unroll
                for (int s = 0; s < KS; ++s) st_dmma(c0, c1, __ldg(pk[k] + (u * KS + s) * 32), bf[k][s]);
                ring[k - 1][u][0] = c0;
                ring[k - 1][u][1] = c1;
            }
            pk[k] += NC * KS * 32;
        }
        // fragments in registers one step ahead while they fit (PIPE); otherwise loaded where they are used
        constexpr bool PIPE = KS <= ST_PIPE_MAXKS && K <= 3;  // four detectors: fragments per chain (register budget)
        double af[K][2][PIPE ? KS : 1];  // [k][block of the pair][k-step]; k = 0 is detector 0
        // too many k-steps for that: two chain-sized buffers, the fragments of chain i + 1 are loaded while chain i runs.
        // Chains of a step in order: (k = 1, bb = 0), (1, 1), ..., (K - 1, 1), (0, 0), (0, 1); 2K of them, so buffer parity
        // is the same in every step.
        double fa[2][PIPE ? 1 : KS];
        auto ldchain = [&](auto BUF, int k, int bb) {
            constexpr int B = decltype(BUF)::value;
#pragma unroll
            for (int s = 0; s < KS; ++s) fa[B][PIPE ? 0 : s] = __ldg(pk[k] + (bb * KS + s) * 32);
        };
        if (PIPE) {
#pragma unroll
            for (int k = 0; k < K; ++k) {
#pragma unroll
                for (int bb = 0; bb < 2; ++bb)
#pragma unroll
                    for (int s = 0; s < KS; ++s) af[k][bb][PIPE ? s : 0] = __ldg(pk[k] + (bb * KS + s) * 32);
                pk[k] += 64 * KS;
            }
        } else {
            ldchain(std::integral_constant<int, 0>(), K > 1 ? 1 : 0, 0);
        }

        // ---- the stream.  One step = two blocks (t0, t0 + 1): the shifted detectors' MMAs of blocks t0 + NC, t0 + NC + 1
        // (2 (K-1) independent chains), the log-sum-exp of the PREVIOUS pair (independent of everything else in the step),
        // the realignment, detector 0's MMAs (2 chains).  Fragments are loaded one step ahead into the registers the
        // chains have just released.
        double mg[2] = {ST_MG_UNSET, ST_MG_UNSET}, sm[2] = {0.0, 0.0}, lin[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
        auto step = [&](auto PC, auto PREDC, const int t0) {
            constexpr int P = decltype(PC)::value;  // t0 % 4 == 2 P
            constexpr bool PRED = decltype(PREDC)::value;
            bool v[2][2] = {{true, true}, {true, true}};
            if (PRED) {
#pragma unroll
                for (int bb = 0; bb < 2; ++bb)
#pragma unroll
                    for (int c = 0; c < 2; ++c) v[bb][c] = (unsigned)(jc[c] + 8 * (t0 - 2 + bb)) < (unsigned)n_t;
            }
            double d[2][2];
            st_lse_pre2<PRED>(lin, v, mg, sm, d);
            // shifted detectors: blocks t0 + NC + bb into ring slots (2 P + NC + bb) % 4
#pragma unroll
            for (int k = 1; k < K; ++k) {
#pragma unroll
                for (int bb = 0; bb < 2; ++bb) {
                    double c0 = 0.0, c1 = 0.0;
                    if (!PIPE) {  // next chain: (k, 1), (k + 1, 0) or detector 0's first
                        if (bb == 0) ldchain(std::integral_constant<int, 1>(), k, 1);
                        else ldchain(std::integral_constant<int, 0>(), k + 1 < K ? k + 1 : 0, 0);
                    }
#pragma unroll
                    for (int s = 0; s < KS; ++s) st_dmma(c0, c1, PIPE ? af[k][bb][PIPE ? s : 0] : fa[bb][PIPE ? 0 : s], bf[k][s]);
                    ring[k - 1][(2 * P + NC + bb) % 4][0] = c0;
                    ring[k - 1][(2 * P + NC + bb) % 4][1] = c1;
                }
            }
#pragma unroll
            for (int k = 1; k < K; ++k) {
                if (PIPE) {
#pragma unroll
                    for (int bb = 0; bb < 2; ++bb)
#pragma unroll
                        for (int s = 0; s < KS; ++s) af[k][bb][PIPE ? s : 0] = __ldg(pk[k] + (bb * KS + s) * 32);
                    pk[k] += 64 * KS;
                }
            }
            st_lse_main2<PRED>(d, v, sm, tab_addr);
            // realign: row rho of my column wants T_k[base_k + rho + eps]; I hold it for the lane (rho - eps) mod 8
            double z[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
#pragma unroll
            for (int k = 1; k < K; ++k) {
#pragma unroll
                for (int bb = 0; bb < 2; ++bb)
#pragma unroll
                    for (int c = 0; c < 2; ++c) {
                        double x = ring[k - 1][(2 * P + bb) % 4][c];
#pragma unroll
                        for (int o = 1; o <= NC; ++o) x = st_bsel(x, ring[k - 1][(2 * P + bb + o) % 4][c], msk[k][c][o - 1]);
                        const double y = st_shfl(x, src[k][c]);
                        z[bb][c] = k == 1 ? y : z[bb][c] + y;
                    }
            }
#pragma unroll
            for (int bb = 0; bb < 2; ++bb) {
                if (!PIPE) {
                    if (bb == 0) {
                        ldchain(std::integral_constant<int, 1>(), 0, 1);
                    } else {  // the step is over for the pointers: the next chain is the next step's first
#pragma unroll
                        for (int k = 0; k < K; ++k) pk[k] += 64 * KS;
                        ldchain(std::integral_constant<int, 0>(), K > 1 ? 1 : 0, 0);
                    }
                }
#pragma unroll
                for (int s = 0; s < KS; ++s) st_dmma(z[bb][0], z[bb][1], PIPE ? af[0][bb][PIPE ? s : 0] : fa[bb][PIPE ? 0 : s], bf[0][s]);
                lin[bb][0] = z[bb][0];
                lin[bb][1] = z[bb][1];
            }
            if (PIPE) {
#pragma unroll
                for (int bb = 0; bb < 2; ++bb)
#pragma unroll
                    for (int s = 0; s < KS; ++s) af[0][bb][PIPE ? s : 0] = __ldg(pk[0] + (bb * KS + s) * 32);
                pk[0] += 64 * KS;
            }
        };
#define ST_STEP(PP)                                                                                         \
    {                                                                                                       \
        const int t0 = tb + 2 * (PP);                                                                       \
        if (t0 < nblk) {                                                                                    \
            if (t0 - 2 >= t_lo && t0 <= t_hi) step(std::integral_constant<int, (PP)>(), std::false_type(), t0); \
            else step(std::integral_constant<int, (PP)>(), std::true_type(), t0);                          \
        }                                                                                                   \
    }
        for (int tb = 0; tb < nblk; tb += 4) {
            ST_STEP(0)
            ST_STEP(1)
        }
#undef ST_STEP
        // lanes of row 0 finish column A, lanes of row 1 column B: their sample's quad is fetched now, behind the last log-sum-exp
        const int s_fin = (r & 1) ? sB : sA;
        double quad_fin = 0.0;
        if (r < 2 && s_fin >= 0) quad_fin = ST_STREAM_LD(a.quad + sbase + s_fin);
        {  // the last pair's log-sum-exp
            bool v[2][2];
#pragma unroll
            for (int bb = 0; bb < 2; ++bb)
#pragma unroll
                for (int c = 0; c < 2; ++c) v[bb][c] = (unsigned)(jc[c] + 8 * (nblk - 2 + bb)) < (unsigned)n_t;
            double d[2][2];
            st_lse_pre2<true>(lin, v, mg, sm, d);
            st_lse_main2<true>(d, v, sm, tab_addr);
        }
        // ---- merge the 8 row lanes of each column, write lnL_margT = LSE - ln N_t - quad  (eq. 9 with the rectangle rule)
        const double nA = st_ref_oct(mg[0]), nB = st_ref_oct(mg[1]);  // references in octaves (-2^30: the lane saw no element)
        double NA = nA, NB = nB;
#pragma unroll
        for (int o = 4; o < 32; o <<= 1) {
            NA = fmax(NA, st_shfl(NA, lane ^ o));
            NB = fmax(NB, st_shfl(NB, lane ^ o));
        }
        double SA = sm[0] * st_pow2_neg(nA - NA), SB = sm[1] * st_pow2_neg(nB - NB);
#pragma unroll
        for (int o = 4; o < 32; o <<= 1) {
            SA += st_shfl(SA, lane ^ o);
            SB += st_shfl(SB, lane ^ o);
        }
        if (r < 2 && s_fin >= 0) a.lnL[sbase + s_fin] = st_log_plus((r & 1) ? SB : SA, (r & 1) ? NB : NA, ltab) - log_nt - quad_fin;
    }
}

// exp and log tables of the streaming kernel (once per context)
__global__ void ile_stream_tab_kernel(double *__restrict__ t)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < ST_TAB) t[i] = exp2((double)i * (1.0 / ST_TAB) - (double)ST_KOFF);
    if (i < 128) {
        const double rc = 1.0 / (1.0 + ((double)i + 0.5) * (1.0 / 128.0));
        t[ST_TAB + 2 * i] = rc;
        t[ST_TAB + 2 * i + 1] = -log(rc);
    }
}

cudaError_t ile_stream_alloc_tables(IleStreamScratch *ss)
{
    cudaError_t e = cudaMalloc(&ss->tabs, (ST_TAB + 256) * sizeof(double));
    if (e != cudaSuccess) return e;
    ile_stream_tab_kernel<<<(ST_TAB + 255) / 256, 256>>>(ss->tabs);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    return cudaSuccess;
}

// ------------------------------------------------------------------------------------------------------------
// Q repacking (once per context): Q [P][K][M][n_q] complex128 -> Qs [P][K][nqp / 8][ks][8][4] doubles, channel 2m = Re, 2m+1 = Im
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) ile_pack_q_stream_kernel(int32_t n_series, int32_t M, int32_t n_q, int32_t ks, int32_t nqp,
                                                                int32_t padf, int32_t interp, const double2 *__restrict__ Q,
                                                                double *__restrict__ Qs)
{
    const long long total = (long long)n_series * ks * nqp * 4;
    for (long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x; o < total; o += (long long)gridDim.x * blockDim.x) {
        // o = (((series * (nqp / 8) + block) * ks + s) * 8 + row in block) * 4 + channel in k-step
        const int c4 = (int)(o & 3), rr = (int)((o >> 2) & 7);
        long long q = o >> 5;
        const int s = (int)(q % ks);
        q /= ks;
        const int blk = (int)(q % (nqp >> 3));
        q /= (nqp >> 3);  // = p * K + k
        // interpolated shifts (reading R8'): channels [2M, 4M) are the series one sample later, so that
        // (1 - phi) Q[i] + phi Q[i + 1] is ONE contraction over 4M channels with coefficients (1 - phi) A and phi A
        int ch = 4 * s + c4, i = blk * 8 + rr - padf;
        if (interp && ch >= 2 * M) ch -= 2 * M, ++i;  // (channels from 4M on stay beyond the modes: zero)
        const int m = ch >> 1;
        double v = 0.0;
        if (m < M && i >= 0 && i < n_q) {
            const double2 z = Q[((size_t)q * M + m) * n_q + i];
            v = (ch & 1) ? z.y : z.x;
        }
        Qs[o] = v;
    }
}

cudaError_t ile_launch_pack_q_stream(const IleSizes &sz, const IleStreamPlan &pl, int32_t n_points, const double2 *Q, double *Qs,
                                     cudaStream_t st)
{
    const long long total = (long long)n_points * sz.n_det * pl.ks * pl.nqp * 4;
    long long blocks = (total + 255) / 256;
    if (blocks > (long long)sz.sm_count * 32) blocks = (long long)sz.sm_count * 32;
    ile_pack_q_stream_kernel<<<(unsigned)blocks, 256, 0, st>>>(n_points * sz.n_det, sz.n_modes, sz.n_q, pl.ks, pl.nqp, pl.padf, sz.interp, Q, Qs);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------
// counting sort of variant 4: cells = (segment, i0_0 >> g0); every segment's slots are padded to a multiple of 8 so that a
// group of 8 consecutive slots never mixes two (d1, d2) cells.  Three kernels: index (keys + histograms), scan (one block per
// segment: final slot position of every cell), scatter.
// ------------------------------------------------------------------------------------------------------------
#define SS_THREADS 256
#ifndef IX_THREADS
#define IX_THREADS 256
#endif

// Index pre-pass: step 2 of the hot path for every sample -- window starts i0_k (readings R2, R8, R9),
// the cell key and the cell histogram of the counting sort.
__global__ void __launch_bounds__(IX_THREADS)
    ile_stream_index_kernel(const __grid_constant__ IleDevParams P, const __grid_constant__ IleEvalArgs a,
                            const __grid_constant__ IleSortPlan sp, int32_t *__restrict__ i0_out, int32_t *__restrict__ cell,
                            uint32_t *__restrict__ hist)
{
    const long long n_total = a.n_per_point * a.n_points;
    const int K = P.n_det;
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < n_total; s += (long long)gridDim.x * blockDim.x) {
        const int pt = (int)(s / a.n_per_point);
        double dir[3], sl, cl, sd, cd;
        ile_source_dir(a.ra[s], a.dec[s], P.gmst, dir, &sl, &cl, &sd, &cd);
        const double t_ref = a.t_ref[s];
        int bad = 0;
        int32_t i0[4] = {0, 0, 0, 0};
        for (int k = 0; k < K; ++k) {
            double phi;
            const int32_t idx = P.interp ? ile_window_floor(P.vertex[k], dir, t_ref, P.t0_q, P.fs, P.n_t, &phi)
                                         : ile_window_index(P.vertex[k], dir, t_ref, P.t0_q, P.fs, P.n_t);
            if (k < 4) i0[k] = idx;
            if (idx < 0 || (long long)idx + P.n_t + (P.interp ? 1 : 0) > P.n_q) bad = 1;  // interpolation reads one sample more
            i0_out[s * K + k] = idx;
            if (a.shift_idx) a.shift_idx[s * K + k] = idx;
        }
        int32_t c;
        if (bad) {  // reading R9: -inf for the sample, sticky counter, never a wrapped or clamped window
            c = sp.ncell - 1;
            atomicAdd(a.oob_counter, 1ULL);
            a.lnL[s] = -CUDART_INF;
        } else {
            // segment = (d1, d2) cell of width 2^g, then the i0_0 bin inside the segment
            int32_t seg = 0;
            if (sp.nd > 1) seg = min(max(i0[1] - i0[0] + sp.dmax[1], 0), 2 * sp.dmax[1]) >> sp.g;
            if (sp.nd > 2) seg = seg * sp.n2 + (min(max(i0[2] - i0[0] + sp.dmax[2], 0), 2 * sp.dmax[2]) >> sp.g);
            if (sp.nd > 3) seg = seg * sp.n3 + (min(max(i0[3] - i0[0] + sp.dmax[3], 0), 2 * sp.dmax[3]) >> sp.g);
            c = seg * sp.n0 + (i0[0] >> sp.g0);  // 0 <= i0_0 <= n_q - n_t here
        }
        cell[s] = c;
        // warp-aggregated: lanes with the same counter send ONE atomic (late in a run the adaptive sampler's draws
        // crowd into a handful of cells, L47, L109, and one atomic per sample on the same address serialises in L2)
        const unsigned long long key = (unsigned long long)pt * sp.ncell + c;
        const unsigned peers = __match_any_sync(__activemask(), key);
        if ((int)(threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(&hist[key], (uint32_t)__popc(peers));
    }
}

// exclusive scan of v[0..n) held in shared memory by the NT threads of a block; returns the total
template <int NT>
__device__ uint32_t ss_block_scan(uint32_t *__restrict__ v, int n, uint32_t *wsum)
{
    const int per = ((n + NT - 1) / NT) | 1;  // odd: conflict-free
    const int lo = min((int)threadIdx.x * per, n), hi = min(lo + per, n);
    uint32_t loc = 0;
    for (int i = lo; i < hi; ++i) loc += v[i];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t inc = loc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t x = __shfl_up_sync(ST_FULL, inc, o);
        if (lane >= o) inc += x;
    }
    __syncthreads();  // wsum may still be read by a previous call
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        const uint32_t x = lane < NT / 32 ? wsum[lane] : 0u;
        uint32_t xi = x;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(ST_FULL, xi, o);
            if (lane >= o) xi += y;
        }
        wsum[lane] = xi - x;
        if (lane == 31) wsum[32] = xi;
    }
    __syncthreads();
    uint32_t run = wsum[warp] + inc - loc;
    for (int i = lo; i < hi; ++i) {
        const uint32_t x = v[i];
        v[i] = run;
        run += x;
    }
    __syncthreads();
    return wsum[32];
}

// Scan: block (seg, pt) turns the counts of the segment's i0_0 bins into exclusive positions inside the segment and
// records the segment's total.
__global__ void __launch_bounds__(SS_THREADS)
    ile_stream_scan_kernel(int32_t n0, int32_t nseg, int32_t ncell, uint32_t *__restrict__ hist, uint32_t *__restrict__ segtot)
{
    extern __shared__ uint32_t ss_v[];  // n0 words
    __shared__ uint32_t wsum[33];
    const int seg = blockIdx.x, pt = blockIdx.y;
    uint32_t *hg = hist + (size_t)pt * ncell + (size_t)seg * n0;
    for (int i = threadIdx.x; i < n0; i += SS_THREADS) ss_v[i] = hg[i];
    __syncthreads();
    const uint32_t tot = ss_block_scan<SS_THREADS>(ss_v, n0, wsum);
    for (int i = threadIdx.x; i < n0; i += SS_THREADS) hg[i] = ss_v[i];
    if (threadIdx.x == 0) segtot[(size_t)pt * nseg + seg] = tot;
}

// exclusive prefix of the points' group counts (multi-point launches)
__global__ void __launch_bounds__(1024) ile_stream_prefix_kernel(int32_t n_points, int32_t nseg, const uint32_t *__restrict__ segtot,
                                                                 int32_t *__restrict__ gcum)
{
    extern __shared__ uint32_t ss_v[];
    __shared__ uint32_t wsum[33];
    for (int p = threadIdx.x; p < n_points; p += 1024) {
        uint32_t g = 0;
        for (int sg = 0; sg < nseg; ++sg) g += (segtot[(size_t)p * nseg + sg] + 7u) >> 3;
        ss_v[p] = g;
    }
    __syncthreads();
    const uint32_t tot = ss_block_scan<1024>(ss_v, n_points, wsum);
    for (int p = threadIdx.x; p < n_points; p += 1024) gcum[p] = (int32_t)ss_v[p];
    if (threadIdx.x == 0) gcum[n_points] = (int32_t)tot;
}

// Scatter: blocks (b, pt).  Every block first builds the padded base of every segment of its point in shared memory (an
// exclusive scan of the segment totals rounded up to 8), then places its samples: slot = base[segment] + position of the
// cell inside the segment + rank inside the cell.  Block 0 of a point marks the padding at the end of every segment with -1
// and, for a single-point launch, records the number of groups.
__global__ void __launch_bounds__(IX_THREADS)
    ile_stream_scatter_kernel(long long n_per_point, int32_t n_points, int32_t ncell, int32_t n0, int32_t nseg, long long slot_cap,
                              const int32_t *__restrict__ cell, uint32_t *__restrict__ offs, const uint32_t *__restrict__ segtot,
                              int32_t *__restrict__ slots, int32_t *__restrict__ gcum)
{
    extern __shared__ uint32_t ss_v[];  // nseg words
    __shared__ uint32_t wsum[33];
    const int pt = blockIdx.y;
    const uint32_t *st = segtot + (size_t)pt * nseg;
    for (int i = threadIdx.x; i < nseg; i += IX_THREADS) ss_v[i] = (st[i] + 7u) & ~7u;
    __syncthreads();
    const uint32_t tot = ss_block_scan<IX_THREADS>(ss_v, nseg, wsum);
    int32_t *sl = slots + (size_t)pt * slot_cap;
    if (blockIdx.x == 0) {
        for (int sg = threadIdx.x; sg < nseg; sg += IX_THREADS) {
            const uint32_t cnt = st[sg];
            for (uint32_t i = cnt; i < ((cnt + 7u) & ~7u); ++i) sl[ss_v[sg] + i] = -1;
        }
        if (threadIdx.x == 0 && n_points == 1) gcum[0] = 0, gcum[1] = (int32_t)(tot >> 3);
    }
    const int32_t *cl = cell + (size_t)pt * n_per_point;
    uint32_t *of = offs + (size_t)pt * ncell;
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < n_per_point; s += (long long)gridDim.x * blockDim.x) {
        const int c = cl[s];
        if (c == ncell - 1) continue;  // out of range: lnL = -inf was written by the index kernel
        // warp-aggregated claim: the first lane of every set of lanes with the same counter takes the whole set's places
        const unsigned peers = __match_any_sync(__activemask(), c);
        const int lane = threadIdx.x & 31, leader = __ffs(peers) - 1;
        uint32_t first = 0;
        if (lane == leader) first = atomicAdd(&of[c], (uint32_t)__popc(peers));
        first = __shfl_sync(peers, first, leader);
        sl[ss_v[c / n0] + first + (uint32_t)__popc(peers & ((1u << lane) - 1u))] = (int32_t)s;
    }
}

// ------------------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------------------
static int st_round_ks(int ks)
{
    const int avail[] = {1, 2, 3, 4, 5, 6, 8, 11, 16};
    for (int v : avail)
        if (ks <= v) return v;
    return 0;
}

// Plan for one launch of n_per_point samples per point: cell widths and the padded Q geometry.  Returns false when the
// sizes do not fit this variant (more than 4 detectors, too many cells).
bool ile_stream_plan(const IleSizes &sz, const IleDevParams &hp, int nc, IleStreamPlan *out, IleSortPlan *spo)
{
    if (sz.n_det > 4) return false;  // a lane looks after one (sample, detector) pair of its group: 8 samples x 4 detectors
    IleStreamPlan pl;
    pl.ks = st_round_ks(((sz.interp ? 4 : 2) * sz.n_modes + 3) / 4);  // interpolated shifts: twice the channels
    if (!pl.ks) return false;
    pl.cp = 4 * pl.ks;
    pl.nc = nc;
    pl.padf = (sz.n_q - sz.n_t + 32 + 7) & ~7;                               // multiples of the 8-row blocking
    pl.nqp = (pl.padf + sz.n_q + (sz.n_q - sz.n_t) + 64 + 7) & ~7;
    IleSortPlan sp;
    sp.nd = sz.n_det;
    sp.g = pl.nc == 2 ? 4 : 3;
    sp.dmax[0] = 0;
    for (int d = 1; d < 4; ++d) {
        sp.dmax[d] = 0;
        if (d < sp.nd) {
            const double dx = hp.vertex[d][0] - hp.vertex[0][0], dy = hp.vertex[d][1] - hp.vertex[0][1], dz = hp.vertex[d][2] - hp.vertex[0][2];
            const double ds = sqrt(dx * dx + dy * dy + dz * dz) / ILE_C_SI * hp.fs;
            if (!(ds < 1.0e6)) return false;
            sp.dmax[d] = (int32_t)ceil(ds) + 2;
        }
    }
    sp.n1 = sp.nd > 1 ? ((2 * sp.dmax[1]) >> sp.g) + 1 : 1;
    sp.n2 = sp.nd > 2 ? ((2 * sp.dmax[2]) >> sp.g) + 1 : 1;
    sp.n3 = sp.nd > 3 ? ((2 * sp.dmax[3]) >> sp.g) + 1 : 1;
    if ((long long)sp.n1 * sp.n2 * sp.n3 > 12288) return false;  // the scatter kernel holds the per-segment bases in shared memory
    sp.nseg = sp.n1 * sp.n2 * sp.n3;
    int g0 = 3;
    for (;; ++g0) {  // i0_0 bins of 8 rows unless the series is so long that a segment's bins (shared memory) or the histogram get too big
        sp.n0 = ((sz.n_q - sz.n_t) >> g0) + 1;
        const long long nc = (long long)sp.n0 * sp.nseg + 1;
        if (sp.n0 <= 12288 && nc <= (1LL << 22)) {
            sp.ncell = (int32_t)nc;
            break;
        }
        if (g0 >= 30) return false;
    }
    sp.g0 = g0;
    *out = pl;
    *spo = sp;
    return true;
}

// Launch (ka != nullptr) or prepare (ka == nullptr: function attributes of the current device + resident CTAs per SM) the
// instantiation for (K, ks).  Function attributes are per device, so they are set by ile_stream_prepare for every context.
template <int K, int KS, int NC, int MINB>
static cudaError_t st_launch_t(const IleSizes &sz, const IleStreamKArgs *ka, long long max_groups, int *per_sm, cudaStream_t st)
{
    if (!ka) {
        cudaError_t e = cudaFuncSetAttribute(ile_eval_stream_kernel<K, KS, NC, MINB>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                             (MINB * (ST_TAB * 8 + 1024) * 100 + 228 * 1024 - 1) / (228 * 1024));
        if (e != cudaSuccess) return e;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm, ile_eval_stream_kernel<K, KS, NC, MINB>, ST_THREADS, 0);
        if (e != cudaSuccess) return e;
        return *per_sm < 1 ? cudaErrorInvalidConfiguration : cudaSuccess;
    }
    long long grid = (long long)sz.sm_count * *per_sm;
    const long long need = (max_groups + ST_THREADS / 32 - 1) / (ST_THREADS / 32);
    if (need < grid) grid = need < 1 ? 1 : need;
    ile_eval_stream_kernel<K, KS, NC, MINB><<<(unsigned)grid, ST_THREADS, 0, st>>>(*ka);
    return cudaGetLastError();
}

template <int K, int NC>
static cudaError_t st_launch_k(const IleSizes &sz, int ks, const IleStreamKArgs *ka, long long mg, int *per_sm, cudaStream_t st)
{
    switch (ks) {
        case 1: return st_launch_t<K, 1, NC, 4>(sz, ka, mg, per_sm, st);
        case 2: return st_launch_t<K, 2, NC, 4>(sz, ka, mg, per_sm, st);
        case 3: return st_launch_t<K, 3, NC, ST_MINB3>(sz, ka, mg, per_sm, st);
        case 4: return st_launch_t<K, 4, NC, 3>(sz, ka, mg, per_sm, st);
        case 5: return st_launch_t<K, 5, NC, 2>(sz, ka, mg, per_sm, st);
        case 6: return st_launch_t<K, 6, NC, 2>(sz, ka, mg, per_sm, st);
        case 8: return st_launch_t<K, 8, NC, 2>(sz, ka, mg, per_sm, st);
        case 11: return st_launch_t<K, 11, NC, 2>(sz, ka, mg, per_sm, st);
        case 16: return st_launch_t<K, 16, NC, 2>(sz, ka, mg, per_sm, st);
        default: return cudaErrorInvalidValue;
    }
}

static cudaError_t st_launch(const IleSizes &sz, int ks, int nc, const IleStreamKArgs *ka, long long mg, int *per_sm, cudaStream_t st)
{
    if (nc == 1) {
        if (sz.n_det == 1) return st_launch_k<1, 1>(sz, ks, ka, mg, per_sm, st);
        if (sz.n_det == 2) return st_launch_k<2, 1>(sz, ks, ka, mg, per_sm, st);
        if (sz.n_det == 3) return st_launch_k<3, 1>(sz, ks, ka, mg, per_sm, st);
        return st_launch_k<4, 1>(sz, ks, ka, mg, per_sm, st);
    }
    if (sz.n_det == 1) return st_launch_k<1, 2>(sz, ks, ka, mg, per_sm, st);
    if (sz.n_det == 2) return st_launch_k<2, 2>(sz, ks, ka, mg, per_sm, st);
    if (sz.n_det == 3) return st_launch_k<3, 2>(sz, ks, ka, mg, per_sm, st);
    return st_launch_k<4, 2>(sz, ks, ka, mg, per_sm, st);
}

// Once per context, on the context's device: carve-out and occupancy of the streaming kernel this context's sizes select.
cudaError_t ile_stream_prepare(const IleSizes &sz, IleStreamPlan *pl)
{
    int per_sm = 0;
    cudaError_t e = st_launch(sz, pl->ks, pl->nc, nullptr, 0, &per_sm, 0);
    pl->ctas_per_sm = per_sm;
    return e;
}

cudaError_t ile_launch_eval_stream(const IleSizes &sz, const IleDevParams &hp, const IleEvalArgs &a, const IleStreamPlan &pl,
                                   const IleSortPlan &sp, const IleSortScratch &sc, IleStreamScratch &ss, cudaStream_t st,
                                   int *n_launches)
{
    if (a.n_per_point <= 0 || a.n_points <= 0) return cudaSuccess;
    const long long n_total = a.n_per_point * a.n_points;
    const int nseg = sp.nseg;
    // sc.hist = [claim counters A][claim counters B][cell histograms][segment totals].  Everything in it is zero between launches: the
    // streaming kernel of a launch zeroes the histograms and totals (the sort is done with them by then) and the claim counters the NEXT
    // launch will use (A and B alternate), so no memset stands in front of the index kernel.  After a failed launch (hist_clean false)
    // the whole block is zeroed the plain way.
    const size_t n_hist = (size_t)a.n_points * sp.ncell, n_used = n_hist + (size_t)a.n_points * nseg;
    uint32_t *rcnt = sc.hist + ILE_STREAM_MAX_RANGES * (ss.launch_no & 1u), *rcnt_next = sc.hist + ILE_STREAM_MAX_RANGES * ((ss.launch_no + 1u) & 1u);
    uint32_t *hist = sc.hist + 2 * ILE_STREAM_MAX_RANGES, *segtot = hist + n_hist;
    cudaError_t e = cudaSuccess;
    if (!ss.hist_clean) {  // the failed launch may have been a larger one (more points or cells): clear everything that is allocated
        const size_t words = ss.hist_words > 2 * ILE_STREAM_MAX_RANGES + n_used ? ss.hist_words : 2 * ILE_STREAM_MAX_RANGES + n_used;
        e = cudaMemsetAsync(sc.hist, 0, words * sizeof(uint32_t), st);
        if (e != cudaSuccess) return e;
    }
    ss.hist_clean = false;
    long long iblocks = (n_total + IX_THREADS - 1) / IX_THREADS;
    const long long cap = (long long)sz.sm_count * 32;
    if (iblocks > cap) iblocks = cap;
    // fork: the side stream may start as soon as the caller's stream gets here; the index kernel is enqueued first so that
    // the short sorting kernels are not starved of SM resources by the coefficient kernel (steps 1, 3, 4)
    e = cudaEventRecord(ss.ev_fork, st);
    if (e != cudaSuccess) return e;
    int nl = 0;
    ile_stream_index_kernel<<<(unsigned)iblocks, IX_THREADS, 0, st>>>(hp, a, sp, sc.i0, sc.cell, hist);
    ++nl;
    e = cudaStreamWaitEvent(ss.aux, ss.ev_fork, 0);
    if (e != cudaSuccess) return e;
    // from here on work may sit on the side stream: an error return first makes the caller's stream wait for it, so that the caller
    // never frees or reuses buffers under a kernel it cannot see
    auto fail = [&](cudaError_t err) {
        if (cudaEventRecord(ss.ev_join, ss.aux) == cudaSuccess) cudaStreamWaitEvent(st, ss.ev_join, 0);
        return err;
    };
    if (ss.ev_late) {  // ile_run_host: those arrays are still being copied on the copy stream
        e = cudaStreamWaitEvent(ss.aux, ss.ev_late, 0);
        if (e != cudaSuccess) return fail(e);
    }
    if (ss.quad_mats && sc.qform) {
        e = ile_launch_quad_mma(sz, hp, a, ss.quad_mats, sc.qform, ss.aux);
        if (e != cudaSuccess) return fail(e);
        ++nl;
    }
    nl += ile_launch_setup_coef(sz, hp, a, pl.cp, sc, ss.hU, ss.hV, ss.aux);
    e = cudaEventRecord(ss.ev_join, ss.aux);
    if (e != cudaSuccess) return fail(e);
    ile_stream_scan_kernel<<<dim3((unsigned)nseg, (unsigned)a.n_points), SS_THREADS, (size_t)sp.n0 * sizeof(uint32_t), st>>>(sp.n0, nseg, sp.ncell,
                                                                                                                            hist, segtot);
    ++nl;
    if (a.n_points > 1) {
        ile_stream_prefix_kernel<<<1, 1024, (size_t)a.n_points * sizeof(uint32_t), st>>>(a.n_points, nseg, segtot, ss.gcum);
        ++nl;
    }
    long long sblocks = (a.n_per_point + IX_THREADS - 1) / IX_THREADS;
    const long long scap = ((long long)sz.sm_count * 8 + a.n_points - 1) / a.n_points;
    if (sblocks > scap) sblocks = scap;
    ile_stream_scatter_kernel<<<dim3((unsigned)sblocks, (unsigned)a.n_points), IX_THREADS, (size_t)nseg * sizeof(uint32_t), st>>>(
        a.n_per_point, a.n_points, sp.ncell, sp.n0, nseg, ss.slot_cap, sc.cell, hist, segtot, ss.slots, ss.gcum);
    ++nl;
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(e);

    e = cudaStreamWaitEvent(st, ss.ev_join, 0);  // join
    if (e != cudaSuccess) return e;

    IleStreamKArgs ka;
    ka.n_t = sz.n_t;
    ka.point0 = a.point0;
    ka.n_points = a.n_points;
    ka.nqp = pl.nqp;
    ka.padf = pl.padf;
    ka.recg = sz.n_det * pl.cp;
    ka.cp = pl.cp;
    ka.n_per_point = a.n_per_point;
    ka.slot_cap = ss.slot_cap;
    ka.Qs = ss.Qs;
    ka.rec = sc.rec;
    ka.quad = sc.quad;
    ka.i0 = sc.i0;
    ka.slots = ss.slots;
    ka.gcum = ss.gcum;
    ka.rcnt = rcnt;
    ka.rcnt_next = rcnt_next;
    ka.zero_ptr = hist;
    ka.zero_n = (long long)n_used;
    ka.lnL = a.lnL;
    ka.tabs = ss.tabs;
    const long long max_groups = (long long)a.n_points * (ss.slot_cap / 8);
    int per_sm = pl.ctas_per_sm;
    // per-SM ranges pay off from a few groups per SM (measured: 66 vs 72 us at 10,000 samples, 65 vs 59 us at 1,000); below
    // that one global counter
    const int nr_sm = sz.sm_count < ILE_STREAM_MAX_RANGES ? sz.sm_count : ILE_STREAM_MAX_RANGES;
    ka.n_ranges = max_groups < 4LL * nr_sm ? 1 : nr_sm;
    e = st_launch(sz, pl.ks, pl.nc, &ka, max_groups, &per_sm, st);
    ++nl;
    if (e == cudaSuccess) ss.hist_clean = true, ++ss.launch_no;
    if (e == cudaSuccess && n_launches) *n_launches += nl;
    return e;
}
