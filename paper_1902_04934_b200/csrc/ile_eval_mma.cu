// ile_eval_mma.cu -- variant 3: the sorted, Q-stationary FP64-MMA evaluation kernel for sm_100a (steps 5-6 of the hot path).
//
// The linear term lin_j = Re sum_k sum_lm conj(A_k,lm) Q_k,lm[i0_k + j]  (eq. 7 / eq. 10; "the most
// costly part", L97) is, per detector, a dense contraction  T_k[i][alpha] = sum_c Qc_k[i][c] * Ac_k[c][alpha]  over the
// 2M real channels c = (mode, re/im) -- "the necessary matrix multiplication" of L97 -- followed by a per-sample shift
// j = i - i0_k(alpha).  It runs here on the FP64 matrix instruction DMMA.8x8x4 (mma.sync.m8n8k4.f64):
//   A fragment = Q   [8 time indices x 4 channels]   stationary in registers for a chunk of 8*tb indices x 4*KS channels,
//                                                    loaded with coalesced 256-byte lines from the packed Q (ile_setup.cu)
//   B fragment = A   [4 channels x 8 samples]        one 8-byte shared-memory load per lane per 4 channels, no broadcast
//   C fragment = lin [8 time indices x 8 samples]    loaded from / stored to the samples' rows in shared memory
// On B200 DMMA has the same peak as DFMA (measured 36.9 vs 36.4 TFLOP/s, and they share the pipe), so nothing is gained
// in arithmetic; what is gained is operand delivery and issue slots (profiles/r01a_tiled_v3.md: the DFMA kernel spent
// 10 shared-memory wavefronts per (sample, detector, 64 indices) on warp-broadcast coefficient loads and 2534 warp
// instructions per sample).  One DMMA does the work of 8 DFMA per lane with two operand registers.
//
// Row layout.  A C fragment holds, per instruction, 4 samples x 8 consecutive time cells.  Rows of the two samples
// alpha and alpha^2 are interleaved in blocks of 8 cells (64 B):  cell (alpha, j) sits at 8-byte slot
//     pair(alpha) * 16 * NB + 16 * (j / 8) + 8 * ((alpha >> 1) & 1) + (j % 8),   pair(alpha) = 2 (alpha >> 2) + (alpha & 1)
// so 8 consecutive cells of one sample always cover the 8 slots of one half of a 128-byte line exactly once, whatever
// the window start i0_k(alpha) is, and the 4 samples of an instruction split 2 + 2 over the halves: every fragment
// load / store is conflict free (2 wavefronts for 256 B).
//
// Samples arrive sorted by window start (ile_setup.cu); a tile is S consecutive sorted samples of one intrinsic point.
// Per tile: the producer warp brings the records of the NEXT tile into shared memory with cp.async.bulk (TMA 1-D bulk
// copies completing on an mbarrier) while 8 consumer warps run one phase per detector.  In a phase a warp owns a chunk
// of 8*tb absolute time indices (tb chosen per tile so the union of the tile's windows splits evenly over the warps) and
// walks the tile's groups of 8 samples.  The LAST detector's phase does not store its C fragments: it reduces them
// to one (max, sum exp) pair per (sample, warp) -- the max-subtracted log-sum-exp of eq. 9 (L81-L86) -- and a final pass
// merges the 8 pairs of each sample.
#include <limits.h>
#include <math_constants.h>

#include "ile_kernels.h"

#define MMA_CWARPS 8
#define MMA_THREADS ((MMA_CWARPS + 1) * 32)
#define FULLMASK 0xffffffffu
#define BAR_EMPTY0 1 /* +b: setup buffer b no longer read (consumers arrive, producer waits) */
#define BAR_CONS 3   /* consumer warps only */

__device__ __forceinline__ void nbar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void nbar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }

// ---- mbarrier + bulk copy (TMA 1-D) ---------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
                 "r"(bytes), "r"(bar)
                 : "memory");
}

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ double lds64(uint32_t addr)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts64(uint32_t addr, double v) { asm volatile("st.shared.f64 [%0], %1;" ::"r"(addr), "d"(v) : "memory"); }

// exp(d) = p * scale for the max-subtracted arguments (d <= 0) of the log-sum-exp: Cody-Waite reduction d = k ln2 + r,
// |r| <= ln2/2, degree-10 polynomial (Chebyshev-node interpolant, relative error 3.4e-16 before rounding); scale = 2^k
// built from integer bits, 0 for k < -1022 and for d < -1024 (which also covers arguments too large for the rounding
// trick).  The caller folds the scale into its accumulation: sum = fma(p, scale, sum).  15 FP64-pipe operations.
__device__ __forceinline__ void ile_exp_split(double d, double &p, double &scale)
{
    const double MAGIC = 6755399441055744.0;  // 1.5 * 2^52: adding it rounds to the nearest integer
    const double t = fma(d, 1.4426950408889634, MAGIC);
    const double kf = t - MAGIC;
    double r = fma(kf, -6.93147180369123816490e-01, d);
    r = fma(kf, -1.90821492927058770002e-10, r);
    double q = 2.7626371065696354e-07;
    q = fma(q, r, 2.764019739169484e-06);
    q = fma(q, r, 2.480150431378554e-05);
    q = fma(q, r, 0.00019841170230570286);
    q = fma(q, r, 0.001388888893251478);
    q = fma(q, r, 0.008333333385699212);
    q = fma(q, r, 0.041666666666573066);
    q = fma(q, r, 0.16666666666554314);
    q = fma(q, r, 0.5000000000000006);
    q = fma(q, r, 1.0000000000000067);
    p = fma(q, r, 1.0);
    int e = max(__double2loint(t) + 1023, 0);
    if ((unsigned)__double2hiint(d) > 0xC0900000u) {  // d < -1024 (or a negative NaN): contributes nothing
        e = 0;
        p = 0.0;
    }
    scale = __hiloint2double(e << 20, 0);
}
__device__ __forceinline__ double ile_exp_le0(double d)
{
    double p, s;
    ile_exp_split(d, p, s);
    return p * s;
}

__device__ __forceinline__ double shfl_xor_d(double v, int m) { return __shfl_xor_sync(FULLMASK, v, m); }

// One group (8 samples) of one chunk: C = [old] + Q-fragment x A-fragment, then back to the rows, or (LAST) reduced to the
// group's (max, sum exp) pairs.
//   ad0, ad1 : shared-memory byte address of this lane's first cell (t = 0) for its two samples; cell t is 128*t further
//   j0, j1   : the j of that first cell (cell t has j + 8t); only used when PRED
//   part     : &part[a0][warp] (double2 = (max, sum)), part + MMA_CWARPS is sample a0 + 1; merge: a previous round of
//              this warp already wrote the pair
template <int KS, int TB, bool FIRST, bool LAST, bool PRED>
__device__ __forceinline__ void mma_group(const double (&qf)[TB][KS], const double (&bf)[KS], int tb, uint32_t ad0, uint32_t ad1,
                                          int j0, int j1, int n_t, double2 *part, bool merge, int r)
{
    double c[TB][2];
    bool v0[TB], v1[TB];
#pragma unroll
    for (int t = 0; t < TB; ++t) {
        v0[t] = t < tb && (!PRED || (unsigned)(j0 + 8 * t) < (unsigned)n_t);
        v1[t] = t < tb && (!PRED || (unsigned)(j1 + 8 * t) < (unsigned)n_t);
        c[t][0] = (!FIRST && v0[t]) ? lds64(ad0 + 128 * t) : 0.0;
        c[t][1] = (!FIRST && v1[t]) ? lds64(ad1 + 128 * t) : 0.0;
    }
#pragma unroll
    for (int s = 0; s < KS; ++s)
#pragma unroll
        for (int t = 0; t < TB; ++t)
            if (t < tb) dmma884(c[t][0], c[t][1], qf[t][s], bf[s]);
    if (!LAST) {
#pragma unroll
        for (int t = 0; t < TB; ++t) {
            if (v0[t]) sts64(ad0 + 128 * t, c[t][0]);
            if (v1[t]) sts64(ad1 + 128 * t, c[t][1]);
        }
    } else {
        double m0 = -CUDART_INF, m1 = -CUDART_INF;
#pragma unroll
        for (int t = 0; t < TB; ++t) {
            if (v0[t]) m0 = fmax(m0, c[t][0]);
            if (v1[t]) m1 = fmax(m1, c[t][1]);
        }
#pragma unroll
        for (int o = 4; o < 32; o <<= 1) {
            m0 = fmax(m0, shfl_xor_d(m0, o));
            m1 = fmax(m1, shfl_xor_d(m1, o));
        }
        const double ms0 = m0 > -CUDART_INF ? m0 : 0.0, ms1 = m1 > -CUDART_INF ? m1 : 0.0;
        double e0 = 0.0, e1 = 0.0;
#pragma unroll
        for (int t = 0; t < TB; ++t) {
            if (t < tb) {
                double p0, s0, p1, s1;
                ile_exp_split(c[t][0] - ms0, p0, s0);
                ile_exp_split(c[t][1] - ms1, p1, s1);
                if (v0[t]) e0 = fma(p0, s0, e0);
                if (v1[t]) e1 = fma(p1, s1, e1);
            }
        }
#pragma unroll
        for (int o = 4; o < 32; o <<= 1) {
            e0 += shfl_xor_d(e0, o);
            e1 += shfl_xor_d(e1, o);
        }
        if (r == 0) {
            if (merge) {  // rare: this warp already reduced another chunk of the same samples
                const double2 o0 = part[0], o1 = part[MMA_CWARPS];
                const double M0 = fmax(m0, o0.x), M1 = fmax(m1, o1.x);
                const double Ms0 = M0 > -CUDART_INF ? M0 : 0.0, Ms1 = M1 > -CUDART_INF ? M1 : 0.0;
                e0 = e0 * ile_exp_le0(ms0 - Ms0) * (m0 > -CUDART_INF ? 1.0 : 0.0) + (o0.x > -CUDART_INF ? o0.y * ile_exp_le0(o0.x - Ms0) : 0.0);
                e1 = e1 * ile_exp_le0(ms1 - Ms1) * (m1 > -CUDART_INF ? 1.0 : 0.0) + (o1.x > -CUDART_INF ? o1.y * ile_exp_le0(o1.x - Ms1) : 0.0);
                m0 = M0;
                m1 = M1;
            }
            part[0] = make_double2(m0, e0);
            part[MMA_CWARPS] = make_double2(m1, e1);
        }
    }
}

// One detector phase of one tile for one warp.
template <int KS, int TB, bool FIRST, bool LAST>
__device__ __forceinline__ void mma_phase(const double *__restrict__ Qk, const double *__restrict__ rec, const int32_t *__restrict__ i0S,
                                          int k, int K, int lo, int tb, int nchunk, int ngrp, int ldrec, int n_t, int NB,
                                          uint32_t rows_addr, double2 *part, int warp, int lane)
{
    constexpr int CP = 4 * KS;
    const int r = lane >> 2, cc = lane & 3;
    const int cht = 8 * tb;
    for (int c = warp; c < nchunk; c += MMA_CWARPS) {
        const int cb = lo + cht * c;
        double qf[TB][KS];
        {
            const double *q = Qk + (size_t)(cb >> 3) * (KS * 32);
#pragma unroll
            for (int t = 0; t < TB; ++t)
#pragma unroll
                for (int s = 0; s < KS; ++s) qf[t][s] = t < tb ? __ldg(q + (t * KS + s) * 32) : 0.0;
        }
        for (int g = 0; g < ngrp; ++g) {
            const int a0 = 8 * g + 2 * cc;  // this lane's C-fragment samples: a0, a0 + 1
            const int jb0 = cb - i0S[a0 * K + k], jb1 = cb - i0S[(a0 + 1) * K + k];
            const bool touch = (jb0 + cht > 0 && jb0 < n_t) || (jb1 + cht > 0 && jb1 < n_t);
            const bool full = jb0 >= 0 && jb0 + cht <= n_t && jb1 >= 0 && jb1 + cht <= n_t;
            if (!__any_sync(FULLMASK, touch)) continue;
            const bool allfull = __all_sync(FULLMASK, full);
            double bf[KS];
#pragma unroll
            for (int s = 0; s < KS; ++s) bf[s] = rec[(size_t)(8 * g + r) * ldrec + k * CP + 4 * s + cc];
            const int j0 = jb0 + r, j1 = jb1 + r;
            const int pair0 = 2 * (a0 >> 2), half = cc & 1;
            const uint32_t ad0 = rows_addr + 8u * (uint32_t)((pair0 * NB + (j0 >> 3)) * 16 + half * 8 + (j0 & 7));
            const uint32_t ad1 = rows_addr + 8u * (uint32_t)(((pair0 + 1) * NB + (j1 >> 3)) * 16 + half * 8 + (j1 & 7));
            double2 *pp = part + (size_t)a0 * MMA_CWARPS;
            const bool merge = c >= MMA_CWARPS;
            if (allfull) mma_group<KS, TB, FIRST, LAST, false>(qf, bf, tb, ad0, ad1, j0, j1, n_t, pp, merge, r);
            else mma_group<KS, TB, FIRST, LAST, true>(qf, bf, tb, ad0, ad1, j0, j1, n_t, pp, merge, r);
        }
    }
}

struct IleMmaKArgs {
    int32_t K, n_t, point0, n_points;
    int64_t n_per_point;
    double *lnL;
};

template <int KS, int TB>
__global__ void __launch_bounds__(MMA_THREADS, 2)
    ile_eval_mma_kernel(const __grid_constant__ IleMmaKArgs a, const __grid_constant__ IleMmaPlan L,
                        const __grid_constant__ IleMmaScratch sc)
{
    extern __shared__ __align__(128) unsigned char smem[];
    const int K = a.K, n_t = a.n_t, S = L.S, ldrec = L.ldrec, recg = L.recg;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long tiles_per_point = (a.n_per_point + S - 1) / S;
    const long long n_tiles = tiles_per_point * a.n_points;
    const uint32_t smem_addr = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t mbar_full = smem_addr + L.off_mbar, mbar_empty = mbar_full + 16;  // two 8-byte barriers each

    if (threadIdx.x == 0) {
        mbar_init(mbar_full, 1);
        mbar_init(mbar_full + 8, 1);
        mbar_init(mbar_empty, MMA_CWARPS);
        mbar_init(mbar_empty + 8, MMA_CWARPS);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == MMA_CWARPS) {
        // ================================================================ producer warp: records of the next tile
        int it = 0;
        for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            const int pt = (int)(tile / tiles_per_point);
            const long long s0 = (tile - (long long)pt * tiles_per_point) * S;
            const int cnt = (int)min((long long)S, (long long)sc.ngood[pt] - s0);
            if (cnt <= 0) continue;
            const int b = it & 1;
            unsigned char *sb = smem + (size_t)b * L.sb_bytes;
            double *rec = reinterpret_cast<double *>(sb);
            double *quadS = reinterpret_cast<double *>(sb + L.sb_quad);
            long long *flatS = reinterpret_cast<long long *>(sb + L.sb_flat);
            int32_t *i0S = reinterpret_cast<int32_t *>(sb + L.sb_i0);
            int32_t *miscS = reinterpret_cast<int32_t *>(sb + L.sb_misc);  // lo[K] | tb[K] | nchunk[K]

            if (it >= 2) mbar_wait(mbar_empty + 8 * b, ((it >> 1) + 1) & 1);
            const long long base = (long long)pt * a.n_per_point;
            long long flat = -1;
            if (lane < cnt) {
                flat = base + sc.perm[base + s0 + lane];
                bulk_g2s(smem_addr + (uint32_t)(b * L.sb_bytes) + (uint32_t)(lane * ldrec * 8), sc.rec + (size_t)flat * recg,
                         (uint32_t)(recg * 8), mbar_full + 8 * b);
                quadS[lane] = sc.quad[flat];
            } else if (lane < S) {  // padding sample: contributes nothing, sits on the first sample's windows
                for (int c = 0; c < recg; ++c) rec[(size_t)lane * ldrec + c] = 0.0;
            }
            if (lane < S) flatS[lane] = flat;
            for (int k = 0; k < K; ++k) {
                int v = lane < cnt ? sc.i0[flat * K + k] : 0;
                const int v0 = __shfl_sync(FULLMASK, v, 0);
                if (lane >= cnt) v = v0;
                if (lane < S) i0S[lane * K + k] = v;
                const int lo = __reduce_min_sync(FULLMASK, v) & ~7, hi = __reduce_max_sync(FULLMASK, v) + n_t;
                const int nblk = (hi - lo + 7) >> 3;
                int tb = (nblk + MMA_CWARPS - 1) / MMA_CWARPS;
                if (tb > TB) tb = TB;
                if (lane == 0) {
                    miscS[k] = lo;
                    miscS[K + k] = tb;
                    miscS[2 * K + k] = (nblk + tb - 1) / tb;
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive_expect_tx(mbar_full + 8 * b, (uint32_t)(cnt * recg * 8));
            ++it;
        }
        return;
    }

    // ==================================================================== consumer warps: steps 5-6
    const uint32_t rows_addr = smem_addr + L.off_rows;
    const int NB = L.nb;
    const double log_nt = log((double)n_t);
    int it = 0;
    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const int pt = (int)(tile / tiles_per_point);
        const long long s0 = (tile - (long long)pt * tiles_per_point) * S;
        const int cnt = (int)min((long long)S, (long long)sc.ngood[pt] - s0);
        if (cnt <= 0) continue;
        const int b = it & 1;
        const unsigned char *sb = smem + (size_t)b * L.sb_bytes;
        const double *rec = reinterpret_cast<const double *>(sb);
        const double *quadS = reinterpret_cast<const double *>(sb + L.sb_quad);
        const long long *flatS = reinterpret_cast<const long long *>(sb + L.sb_flat);
        const int32_t *i0S = reinterpret_cast<const int32_t *>(sb + L.sb_i0);
        const int32_t *miscS = reinterpret_cast<const int32_t *>(sb + L.sb_misc);
        double2 *part = reinterpret_cast<double2 *>(smem + L.off_part + (size_t)b * L.part_bytes);
        const size_t pglob = (size_t)(a.point0 + pt);
        const int ngrp = (cnt + 7) >> 3;

        mbar_wait(mbar_full + 8 * b, (it >> 1) & 1);
        if (lane < S) part[lane * MMA_CWARPS + warp] = make_double2(-CUDART_INF, 0.0);
        __syncwarp();

        // ---------------------------------------------------------------- step 5 (+ 6 in the last phase)
        for (int k = 0; k < K; ++k) {
            const double *Qk = sc.Qp + ((pglob * K + k) * (size_t)L.nblk_q) * (KS * 32) + lane;
            const int lo = miscS[k], tb = miscS[K + k], nchunk = miscS[2 * K + k];
            const bool first = k == 0, last = k == K - 1;
            if (first && last)
                mma_phase<KS, TB, true, true>(Qk, rec, i0S, k, K, lo, tb, nchunk, ngrp, ldrec, n_t, NB, rows_addr, part + warp, warp, lane);
            else if (first)
                mma_phase<KS, TB, true, false>(Qk, rec, i0S, k, K, lo, tb, nchunk, ngrp, ldrec, n_t, NB, rows_addr, part + warp, warp, lane);
            else if (last)
                mma_phase<KS, TB, false, true>(Qk, rec, i0S, k, K, lo, tb, nchunk, ngrp, ldrec, n_t, NB, rows_addr, part + warp, warp, lane);
            else
                mma_phase<KS, TB, false, false>(Qk, rec, i0S, k, K, lo, tb, nchunk, ngrp, ldrec, n_t, NB, rows_addr, part + warp, warp, lane);
            nbar_sync(BAR_CONS, MMA_CWARPS * 32);
        }

        // ---------------------------------------------------------------- step 6: merge the 8 pairs of each sample
        for (int al = warp; al < cnt; al += MMA_CWARPS) {
            double2 pr = make_double2(-CUDART_INF, 0.0);
            if (lane < MMA_CWARPS) pr = part[al * MMA_CWARPS + lane];
            double mx = pr.x;
            mx = fmax(mx, shfl_xor_d(mx, 1));
            mx = fmax(mx, shfl_xor_d(mx, 2));
            mx = fmax(mx, shfl_xor_d(mx, 4));
            double sm = pr.x > -CUDART_INF ? pr.y * ile_exp_le0(pr.x - mx) : 0.0;
            sm += shfl_xor_d(sm, 1);
            sm += shfl_xor_d(sm, 2);
            sm += shfl_xor_d(sm, 4);
            if (lane == 0) a.lnL[flatS[al]] = mx + log(sm) - log_nt - quadS[al];
        }
        __syncwarp();
        if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mbar_empty + 8 * b) : "memory");
        ++it;
    }
}

// ------------------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------------------
static int mma_tbmax(int KS) { return KS <= 3 ? 8 : KS <= 4 ? 6 : KS <= 6 ? 4 : KS <= 8 ? 3 : KS <= 12 ? 2 : 1; }

static IleMmaPlan mma_layout(const IleSizes &sz, int KS, int S)
{
    IleMmaPlan L;
    L.ks = KS;
    L.cp = 4 * KS;
    L.tbmax = mma_tbmax(KS);
    L.S = S;
    L.recg = sz.n_det * L.cp;
    int ld = L.recg;
    while (ld % 16 != 4) ++ld;  // 8 samples x 32 B of one B-fragment load land in distinct bank groups; rows stay 16-byte aligned
    L.ldrec = ld;
    L.nb = (sz.n_t + 7) / 8;
    L.nblk_q = (sz.n_q + 7) / 8 + L.tbmax + 2;
    uint32_t o = (uint32_t)(S * ld * sizeof(double));
    L.sb_quad = o;
    o += (uint32_t)(S * sizeof(double));
    L.sb_flat = o;
    o += (uint32_t)(S * sizeof(long long));
    L.sb_i0 = o;
    o += (uint32_t)(S * sz.n_det * sizeof(int32_t));
    L.sb_misc = o;
    o += (uint32_t)(3 * sz.n_det * sizeof(int32_t));
    L.sb_bytes = (o + 127u) & ~127u;
    L.off_part = 2 * L.sb_bytes;
    L.part_bytes = (uint32_t)(S * MMA_CWARPS * sizeof(double2));
    L.off_mbar = L.off_part + 2 * L.part_bytes;
    L.off_rows = (L.off_mbar + 32u + 127u) & ~127u;
    L.bytes = L.off_rows + (uint32_t)((S / 2) * L.nb * 16 * sizeof(double));
    return L;
}

bool ile_mma_plan(const IleSizes &sz, IleMmaPlan *out)
{
    const int KS = (2 * sz.n_modes + 3) / 4;
    if (KS > 16) return false;
    const size_t per_sm = (size_t)sz.smem_per_sm, reserve = 1024;
    for (int S = 32; S >= 8; S -= 8) {  // two resident blocks per SM
        IleMmaPlan L = mma_layout(sz, KS, S);
        if (2 * ((size_t)L.bytes + reserve) <= per_sm) {
            *out = L;
            return true;
        }
    }
    for (int S = 32; S >= 8; S -= 8) {  // one
        IleMmaPlan L = mma_layout(sz, KS, S);
        if ((size_t)L.bytes <= (size_t)sz.max_smem_optin) {
            *out = L;
            return true;
        }
    }
    return false;
}

template <int KS, int TB>
static cudaError_t mma_launch_t(const IleSizes &sz, const IleEvalArgs &a, const IleMmaPlan &L, const IleMmaScratch &sc, cudaStream_t st)
{
    static bool attr_set = false;
    static int per_sm = 0;
    static uint32_t attr_bytes = 0;
    cudaError_t e;
    if (!attr_set || attr_bytes != L.bytes) {
        e = cudaFuncSetAttribute(ile_eval_mma_kernel<KS, TB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.bytes);
        if (e != cudaSuccess) return e;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ile_eval_mma_kernel<KS, TB>, MMA_THREADS, L.bytes);
        if (e != cudaSuccess) return e;
        attr_set = true;
        attr_bytes = L.bytes;
    }
    if (per_sm < 1) return cudaErrorInvalidConfiguration;
    IleMmaKArgs ka;
    ka.K = sz.n_det;
    ka.n_t = sz.n_t;
    ka.point0 = a.point0;
    ka.n_points = a.n_points;
    ka.n_per_point = a.n_per_point;
    ka.lnL = a.lnL;
    const long long tiles = ((a.n_per_point + L.S - 1) / L.S) * a.n_points;
    long long grid = (long long)sz.sm_count * per_sm;
    if (tiles < grid) grid = tiles;
    ile_eval_mma_kernel<KS, TB><<<(unsigned)grid, MMA_THREADS, L.bytes, st>>>(ka, L, sc);
    return cudaGetLastError();
}

cudaError_t ile_launch_eval_mma(const IleSizes &sz, const IleDevParams &hp, const IleEvalArgs &a, const IleMmaPlan &L,
                                const IleMmaScratch &sc, cudaStream_t st, int *n_launches)
{
    (void)hp;
    if (a.n_per_point <= 0 || a.n_points <= 0) return cudaSuccess;
    cudaError_t e;
    switch (L.ks) {
        case 1: e = mma_launch_t<1, 8>(sz, a, L, sc, st); break;
        case 2: e = mma_launch_t<2, 8>(sz, a, L, sc, st); break;
        case 3: e = mma_launch_t<3, 8>(sz, a, L, sc, st); break;
        case 4: e = mma_launch_t<4, 6>(sz, a, L, sc, st); break;
        case 5: e = mma_launch_t<5, 4>(sz, a, L, sc, st); break;
        case 6: e = mma_launch_t<6, 4>(sz, a, L, sc, st); break;
        case 7: e = mma_launch_t<7, 3>(sz, a, L, sc, st); break;
        case 8: e = mma_launch_t<8, 3>(sz, a, L, sc, st); break;
        case 9: e = mma_launch_t<9, 2>(sz, a, L, sc, st); break;
        case 10: e = mma_launch_t<10, 2>(sz, a, L, sc, st); break;
        case 11: e = mma_launch_t<11, 2>(sz, a, L, sc, st); break;
        case 12: e = mma_launch_t<12, 2>(sz, a, L, sc, st); break;
        case 13: e = mma_launch_t<13, 1>(sz, a, L, sc, st); break;
        case 14: e = mma_launch_t<14, 1>(sz, a, L, sc, st); break;
        case 15: e = mma_launch_t<15, 1>(sz, a, L, sc, st); break;
        default: e = mma_launch_t<16, 1>(sz, a, L, sc, st); break;
    }
    if (e == cudaSuccess && n_launches) *n_launches += 1;
    return e;
}
