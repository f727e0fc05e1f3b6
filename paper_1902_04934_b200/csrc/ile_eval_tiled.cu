// ile_eval_tiled.cu -- variant 2: the tuned, Q-stationary evaluation kernel for sm_100a (steps 1-6 of the hot path).
//
// Why this shape: the linear term lin_j = Re sum_k sum_lm conj(A_k,lm) Q_k,lm[i0_k + j]
// (eq. 7 / eq. 10; "the most costly part", L97) needs 2 DFMA per 16-byte Q element.  Fed
// from shared memory per use that is 512 B/clk/SM for the 64 DFMA/clk/SM the B200 FP64 pipe can retire -- four
// times what shared memory delivers.  So Q is held in REGISTERS instead: a warp owns 64 absolute time indices of one
// detector (lane l: b + l and b + 32 + l, all modes of one mode group), walks the samples of the tile whose window
// touches them, fetches the sample's coefficients A = (D_ref/D) F_k Y_lm with warp-broadcast 16-byte loads and adds
// its per-detector partial sum into the sample's row lin[alpha][i - i0_k(alpha)] in shared memory (8-byte,
// lane-consecutive, conflict-free).  Detectors (and mode groups) are separate phases, so each row entry is touched
// by exactly one thread per phase.  A last pass does the max-subtracted log-sum-exp over each row (eq. 9),
// one warp per sample, row in registers, warp-shuffle reductions.
//
// Per tile of S <= 32 samples:  setup (lane = sample: steps 1-4)  ->  K*G accumulation phases  ->  LSE pass.
// The setup of tile t+1 runs in a ninth, producer warp while the eight consumer warps work on tile t; its outputs
// (A, i0, quad, flags, index ranges, chunk counters) are double-buffered and handed over with named barriers.
#include <limits.h>
#include <math_constants.h>

#include "ile_kernels.h"
#include "ile_fixexp.cuh"

#define TILED_CWARPS 8                         /* consumer warps: accumulation phases and the LSE pass */
#define TILED_THREADS ((TILED_CWARPS + 1) * 32) /* + one producer warp: per-sample setup of the next tile */
#define TILED_CHUNK 64


// ------------------------------------------------------------------------------------------------------------
// named barriers (PTX bar.sync / bar.arrive): producer warp <-> consumer warps hand-off of the per-tile setup
// ------------------------------------------------------------------------------------------------------------
#define BAR_FULL0 1  /* +b: setup buffer b written (producer arrives, consumers wait)   */
#define BAR_EMPTY0 3 /* +b: setup buffer b no longer read (consumers arrive, producer waits) */
#define BAR_CONS 5   /* consumer warps only */
#define FULLMASK 0xffffffffu

__device__ __forceinline__ void bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void bar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }

// One chunk of one accumulation phase: this warp holds Q[m][b + lane] (q0) and Q[m][b + 32 + lane] (q1) for the MG
// modes of the group; m_int / m_edge are the samples whose window covers the chunk completely / partly.
//   soff_l : (lane = sample) byte offset of lin[sample][b - i0_k(sample)] from the start of lin
//   rel_l  : (lane = sample) b - i0_k(sample)
//   Ab     : &A[sample 0][k][g * MG], a_stride = bytes between samples
//   linl   : (unsigned char*)lin + lane * 8
template <int MG, bool FIRST>
__device__ __forceinline__ void tiled_chunk(const double2 (&q0)[MG], const double2 (&q1)[MG], unsigned m_int,
                                            unsigned m_edge, int soff_l, int rel_l, const unsigned char *__restrict__ Ab,
                                            int a_stride, unsigned char *__restrict__ linl, int n_t, int lane)
{
    // ---- windows that cover all 64 indices: no per-lane predicates, two samples in flight
    while (m_int) {
        const int a0 = __ffs(m_int) - 1;
        m_int &= m_int - 1;
        if (m_int) {
            const int a1 = __ffs(m_int) - 1;
            m_int &= m_int - 1;
            const int so0 = __shfl_sync(FULLMASK, soff_l, a0), so1 = __shfl_sync(FULLMASK, soff_l, a1);
            const double2 *__restrict__ A0 = reinterpret_cast<const double2 *>(Ab + a0 * a_stride);
            const double2 *__restrict__ A1 = reinterpret_cast<const double2 *>(Ab + a1 * a_stride);
            double *__restrict__ r0 = reinterpret_cast<double *>(linl + so0);
            double *__restrict__ r1 = reinterpret_cast<double *>(linl + so1);
            double2 c0[MG], c1[MG];
#pragma unroll
            for (int mm = 0; mm < MG; ++mm) {
                c0[mm] = A0[mm];
                c1[mm] = A1[mm];
            }
            double o00 = 0.0, o01 = 0.0, o10 = 0.0, o11 = 0.0;
            if (!FIRST) {
                o00 = r0[0];
                o01 = r0[32];
                o10 = r1[0];
                o11 = r1[32];
            }
            double x00 = 0.0, y00 = 0.0, x01 = 0.0, y01 = 0.0, x10 = 0.0, y10 = 0.0, x11 = 0.0, y11 = 0.0;
#pragma unroll
            for (int mm = 0; mm < MG; ++mm) {
                x00 = fma(c0[mm].x, q0[mm].x, x00);
                y00 = fma(c0[mm].y, q0[mm].y, y00);
                x01 = fma(c0[mm].x, q1[mm].x, x01);
                y01 = fma(c0[mm].y, q1[mm].y, y01);
                x10 = fma(c1[mm].x, q0[mm].x, x10);
                y10 = fma(c1[mm].y, q0[mm].y, y10);
                x11 = fma(c1[mm].x, q1[mm].x, x11);
                y11 = fma(c1[mm].y, q1[mm].y, y11);
            }
            if (FIRST) {
                r0[0] = x00 + y00;
                r0[32] = x01 + y01;
                r1[0] = x10 + y10;
                r1[32] = x11 + y11;
            } else {
                r0[0] = o00 + (x00 + y00);
                r0[32] = o01 + (x01 + y01);
                r1[0] = o10 + (x10 + y10);
                r1[32] = o11 + (x11 + y11);
            }
        } else {
            const int so0 = __shfl_sync(FULLMASK, soff_l, a0);
            const double2 *__restrict__ A0 = reinterpret_cast<const double2 *>(Ab + a0 * a_stride);
            double *__restrict__ r0 = reinterpret_cast<double *>(linl + so0);
            double2 c0[MG];
#pragma unroll
            for (int mm = 0; mm < MG; ++mm) c0[mm] = A0[mm];
            double o00 = 0.0, o01 = 0.0;
            if (!FIRST) {
                o00 = r0[0];
                o01 = r0[32];
            }
            double x00 = 0.0, y00 = 0.0, x01 = 0.0, y01 = 0.0;
#pragma unroll
            for (int mm = 0; mm < MG; ++mm) {
                x00 = fma(c0[mm].x, q0[mm].x, x00);
                y00 = fma(c0[mm].y, q0[mm].y, y00);
                x01 = fma(c0[mm].x, q1[mm].x, x01);
                y01 = fma(c0[mm].y, q1[mm].y, y01);
            }
            if (FIRST) {
                r0[0] = x00 + y00;
                r0[32] = x01 + y01;
            } else {
                r0[0] = o00 + (x00 + y00);
                r0[32] = o01 + (x01 + y01);
            }
        }
    }
    // ---- windows that start or end inside the chunk: 32-index halves skipped when untouched, lanes predicated
    while (m_edge) {
        const int a0 = __ffs(m_edge) - 1;
        m_edge &= m_edge - 1;
        const int so0 = __shfl_sync(FULLMASK, soff_l, a0), rel = __shfl_sync(FULLMASK, rel_l, a0);
        const double2 *__restrict__ A0 = reinterpret_cast<const double2 *>(Ab + a0 * a_stride);
        double *__restrict__ r0 = reinterpret_cast<double *>(linl + so0);
        double2 c0[MG];
#pragma unroll
        for (int mm = 0; mm < MG; ++mm) c0[mm] = A0[mm];
        if (rel + 31 >= 0 && rel < n_t) {
            double x = 0.0, y = 0.0;
#pragma unroll
            for (int mm = 0; mm < MG; ++mm) {
                x = fma(c0[mm].x, q0[mm].x, x);
                y = fma(c0[mm].y, q0[mm].y, y);
            }
            if ((unsigned)(rel + lane) < (unsigned)n_t) r0[0] = FIRST ? (x + y) : (r0[0] + (x + y));
        }
        if (rel + 63 >= 0 && rel + 32 < n_t) {
            double x = 0.0, y = 0.0;
#pragma unroll
            for (int mm = 0; mm < MG; ++mm) {
                x = fma(c0[mm].x, q1[mm].x, x);
                y = fma(c0[mm].y, q1[mm].y, y);
            }
            if ((unsigned)(rel + 32 + lane) < (unsigned)n_t) r0[32] = FIRST ? (x + y) : (r0[32] + (x + y));
        }
    }
}

template <int MG>
__global__ void __launch_bounds__(TILED_THREADS, 2)
    ile_eval_tiled_kernel(const __grid_constant__ IleDevParams P, const __grid_constant__ IleEvalArgs a,
                          const __grid_constant__ IleTiledLayout L)
{
    extern __shared__ __align__(16) unsigned char smem[];
    double *__restrict__ lin = reinterpret_cast<double *>(smem + L.off_lin);

    const int K = P.n_det, M = P.n_modes, n_q = P.n_q, n_t = P.n_t;
    const int G = L.n_groups, ldA = G * MG, S = L.S, ldl = L.ldl, n_phase = K * G;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long tiles_per_point = (a.n_per_point + S - 1) / S;
    const long long n_tiles = tiles_per_point * a.n_points;

    if (warp == TILED_CWARPS) {
        // ================================================================ producer warp: steps 1-4, lane = sample
        int it = 0;
        for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
            const int b = it & 1;
            unsigned char *sb = smem + L.off_sb + (size_t)b * L.sb_bytes;
            double2 *A = reinterpret_cast<double2 *>(sb);
            double *quadS = reinterpret_cast<double *>(sb + L.sb_quad);
            int32_t *i0S = reinterpret_cast<int32_t *>(sb + L.sb_i0);
            int32_t *badS = reinterpret_cast<int32_t *>(sb + L.sb_bad);
            int32_t *rangeS = reinterpret_cast<int32_t *>(sb + L.sb_misc);
            int32_t *ctrS = rangeS + 2 * ILE_MAX_DET;

            const int pt = (int)(tile / tiles_per_point);
            const long long s0 = (tile - (long long)pt * tiles_per_point) * S;
            const int cnt = (int)min((long long)S, a.n_per_point - s0);
            const long long flat0 = (long long)pt * a.n_per_point + s0;
            const size_t pglob = (size_t)(a.point0 + pt);

            if (it >= 2) bar_sync(BAR_EMPTY0 + b, TILED_THREADS);
            int bad = 1;
            if (lane < cnt) {
                const long long s = flat0 + lane;
                double q = ile_setup_sample(&P, a.U + pglob * (size_t)K * M * M, a.V + pglob * (size_t)K * M * M, a.ra[s],
                                            a.dec[s], a.t_ref[s], a.phi_ref[s], a.psi[s], a.incl[s], a.dist[s],
                                            A + (size_t)lane * K * ldA, ldA, i0S + lane * K, &bad);
                quadS[lane] = q;
                if (a.shift_idx)
                    for (int k = 0; k < K; ++k) a.shift_idx[s * K + k] = i0S[lane * K + k];
                if (bad) {
                    atomicAdd(a.oob_counter, 1ULL);
                    a.lnL[s] = -CUDART_INF;
                }
            }
            badS[lane] = bad;
            for (int k = 0; k < K; ++k) {
                const int v = bad ? INT_MAX : i0S[lane * K + k];
                const int w = bad ? INT_MIN : i0S[lane * K + k];
                const int lo = __reduce_min_sync(FULLMASK, v), hi = __reduce_max_sync(FULLMASK, w);
                if (lane == 0) {
                    const bool any = hi != INT_MIN;
                    rangeS[k] = any ? lo : 0;
                    rangeS[ILE_MAX_DET + k] = any ? hi + n_t : 0;
                }
            }
            for (int p = lane; p < n_phase; p += 32) ctrS[p] = 0;
            __threadfence_block();
            bar_arrive(BAR_FULL0 + b, TILED_THREADS);
        }
        return;
    }

    // ==================================================================== consumer warps: steps 5-6
    const double log_nt = log((double)n_t);
    unsigned char *__restrict__ linl = reinterpret_cast<unsigned char *>(lin) + lane * 8;
    int it = 0;
    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
        const int b = it & 1;
        unsigned char *sb = smem + L.off_sb + (size_t)b * L.sb_bytes;
        const unsigned char *Abytes = sb;
        const double *quadS = reinterpret_cast<const double *>(sb + L.sb_quad);
        const int32_t *i0S = reinterpret_cast<const int32_t *>(sb + L.sb_i0);
        const int32_t *badS = reinterpret_cast<const int32_t *>(sb + L.sb_bad);
        const int32_t *rangeS = reinterpret_cast<const int32_t *>(sb + L.sb_misc);
        int32_t *ctrS = reinterpret_cast<int32_t *>(sb + L.sb_misc) + 2 * ILE_MAX_DET;

        const int pt = (int)(tile / tiles_per_point);
        const long long s0 = (tile - (long long)pt * tiles_per_point) * S;
        const int cnt = (int)min((long long)S, a.n_per_point - s0);
        const long long flat0 = (long long)pt * a.n_per_point + s0;
        const size_t pglob = (size_t)(a.point0 + pt);
        const double2 *__restrict__ Qp = a.Q + pglob * (size_t)K * M * n_q;
        const int a_stride = K * ldA * (int)sizeof(double2);

        bar_sync(BAR_FULL0 + b, TILED_THREADS);
        const bool good_l = lane < S && !badS[lane];

        // ---------------------------------------------------------------- step 5: accumulation phases
        for (int p = 0; p < n_phase; ++p) {
            const int k = p / G, g = p - k * G;
            const int lo = rangeS[k], hi = rangeS[ILE_MAX_DET + k];
            const int i0_l = good_l ? i0S[lane * K + k] : 0;
            const unsigned char *Ab = Abytes + (size_t)(k * ldA + g * MG) * sizeof(double2);
            for (;;) {
                int c = 0;
                if (lane == 0) c = atomicAdd(&ctrS[p], 1);
                c = __shfl_sync(FULLMASK, c, 0);
                const int bidx = lo + c * TILED_CHUNK;
                if (bidx >= hi) break;

                double2 q0[MG], q1[MG];
                {
                    const int ia = min(bidx + lane, n_q - 1), ib = min(bidx + 32 + lane, n_q - 1);
#pragma unroll
                    for (int mm = 0; mm < MG; ++mm) {
                        const int m = g * MG + mm;
                        if (m < M) {
                            const double2 *Qm = Qp + ((size_t)k * M + m) * n_q;
                            q0[mm] = __ldg(Qm + ia);
                            q1[mm] = __ldg(Qm + ib);
                        } else {
                            q0[mm] = make_double2(0.0, 0.0);
                            q1[mm] = make_double2(0.0, 0.0);
                        }
                    }
                }
                const int rel_l = bidx - i0_l;
                const bool touch = good_l && (rel_l + (TILED_CHUNK - 1) >= 0) && (rel_l < n_t);
                const bool inter = touch && rel_l >= 0 && rel_l + TILED_CHUNK <= n_t;
                const unsigned m_int = __ballot_sync(FULLMASK, inter);
                const unsigned m_edge = __ballot_sync(FULLMASK, touch && !inter);
                const int soff_l = (lane * ldl + rel_l) * 8;
                if (p == 0)
                    tiled_chunk<MG, true>(q0, q1, m_int, m_edge, soff_l, rel_l, Ab, a_stride, linl, n_t, lane);
                else
                    tiled_chunk<MG, false>(q0, q1, m_int, m_edge, soff_l, rel_l, Ab, a_stride, linl, n_t, lane);
            }
            bar_sync(BAR_CONS, TILED_CWARPS * 32);
        }

        // ---------------------------------------------------------------- step 6: log-sum-exp over each row
        for (int al = warp; al < cnt; al += TILED_CWARPS) {
            if (badS[al]) continue;
            const double *__restrict__ row = lin + (size_t)al * ldl + lane;
            const int nl = n_t - lane;  // this lane owns row[0], row[32], ... below nl
            double m0 = -CUDART_INF, m1 = -CUDART_INF;
            int j = 0;
            for (; j + 32 < nl; j += 64) {
                m0 = fmax(m0, row[j]);
                m1 = fmax(m1, row[j + 32]);
            }
            if (j < nl) m0 = fmax(m0, row[j]);
            const double mx = warp_max(fmax(m0, m1));
            double e0 = 0.0, e1 = 0.0, e2 = 0.0, e3 = 0.0;
            j = 0;
            for (; j + 96 < nl; j += 128) {
                const double x0 = row[j] - mx, x1 = row[j + 32] - mx, x2 = row[j + 64] - mx, x3 = row[j + 96] - mx;
                e0 += ile_fixexp_nonpos(x0, a.exp_tab);
                e1 += ile_fixexp_nonpos(x1, a.exp_tab);
                e2 += ile_fixexp_nonpos(x2, a.exp_tab);
                e3 += ile_fixexp_nonpos(x3, a.exp_tab);
            }
            for (; j < nl; j += 32) e0 += ile_fixexp_nonpos(row[j] - mx, a.exp_tab);
            const double sm = warp_sum((e0 + e1) + (e2 + e3));
            if (lane == 0) a.lnL[flat0 + al] = mx + log(sm) - log_nt - quadS[al];
        }
        if (tile + 2 * (long long)gridDim.x < n_tiles) bar_arrive(BAR_EMPTY0 + b, TILED_THREADS);
        bar_sync(BAR_CONS, TILED_CWARPS * 32);
    }
}

// ------------------------------------------------------------------------------------------------------------
// host side: shared-memory layout, tile size and launch
// ------------------------------------------------------------------------------------------------------------
static int tiled_pick_mg(int M)
{
    int best = 2, best_pad = INT_MAX;
    for (int mg = 2; mg <= 8; ++mg) {
        int pad = ((M + mg - 1) / mg) * mg - M;
        if (pad < best_pad || (pad == best_pad && mg > best)) {
            best = mg;
            best_pad = pad;
        }
    }
    return best;
}

static IleTiledLayout tiled_layout(const IleSizes &sz, int MG, int S)
{
    IleTiledLayout L;
    L.mg = MG;
    L.n_groups = (sz.n_modes + MG - 1) / MG;
    L.S = S;
    L.ldl = sz.n_t;
    // one setup buffer: A[S][K][G*MG] | quad[32] | i0[32][K] | bad[32] | lo[MAX_DET] hi[MAX_DET] ctr[K*G]
    uint32_t o = (uint32_t)(S * sz.n_det * L.n_groups * MG * sizeof(double2));
    L.sb_quad = o;
    o += (uint32_t)(32 * sizeof(double));
    L.sb_i0 = o;
    o += (uint32_t)(32 * sz.n_det * sizeof(int32_t));
    L.sb_bad = o;
    o += (uint32_t)(32 * sizeof(int32_t));
    L.sb_misc = o;
    o += (uint32_t)((2 * ILE_MAX_DET + sz.n_det * L.n_groups) * sizeof(int32_t));
    L.sb_bytes = (o + 15u) & ~15u;
    L.off_sb = 0;
    L.off_lin = 2 * L.sb_bytes;
    L.bytes = (L.off_lin + (uint32_t)(S * L.ldl * sizeof(double)) + 15u) & ~15u;
    return L;
}

bool ile_tiled_plan(const IleSizes &sz, long long n_total, IleTiledLayout *out)
{
    const int MG = tiled_pick_mg(sz.n_modes);
    const size_t per_sm = (size_t)sz.smem_per_sm, reserve = 1024;
    int S = 0;
    for (int s = 32; s >= 4; --s) {  // two resident blocks per SM if that leaves a tile of at least 16 samples
        if (2 * (tiled_layout(sz, MG, s).bytes + reserve) <= per_sm) {
            S = s;
            break;
        }
    }
    if (S < 16) {
        S = 0;
        for (int s = 32; s >= 4; --s) {
            if (tiled_layout(sz, MG, s).bytes <= (size_t)sz.max_smem_optin) {
                S = s;
                break;
            }
        }
    }
    if (S < 4) return false;
    // small batches: shrink the tile so that every SM gets work (latency-bound regime, SURVEY.md §7 hard part 5)
    long long want = (n_total + 2LL * sz.sm_count - 1) / (2LL * sz.sm_count);
    if (want < 8) want = 8;
    if (want < S) S = (int)want;
    *out = tiled_layout(sz, MG, S);
    return true;
}

template <int MG>
static cudaError_t tiled_launch_mg(const IleSizes &sz, const IleDevParams &hp, const IleEvalArgs &a, const IleTiledLayout &L,
                                   cudaStream_t st)
{
    cudaError_t e = cudaFuncSetAttribute(ile_eval_tiled_kernel<MG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.bytes);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ile_eval_tiled_kernel<MG>, TILED_THREADS, L.bytes);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorInvalidConfiguration;
    const long long tiles = ((a.n_per_point + L.S - 1) / L.S) * a.n_points;
    long long grid = (long long)sz.sm_count * per_sm;
    if (tiles < grid) grid = tiles;
    ile_eval_tiled_kernel<MG><<<(unsigned)grid, TILED_THREADS, L.bytes, st>>>(hp, a, L);
    return cudaGetLastError();
}

cudaError_t ile_launch_eval_tiled(const IleSizes &sz, const IleDevParams &hp, const IleEvalArgs &a, cudaStream_t st,
                                  int *n_launches)
{
    if (a.n_per_point <= 0 || a.n_points <= 0) return cudaSuccess;
    IleTiledLayout L;
    if (!ile_tiled_plan(sz, (long long)a.n_per_point * a.n_points, &L)) return cudaErrorInvalidConfiguration;
    cudaError_t e;
    switch (L.mg) {
        case 2: e = tiled_launch_mg<2>(sz, hp, a, L, st); break;
        case 3: e = tiled_launch_mg<3>(sz, hp, a, L, st); break;
        case 4: e = tiled_launch_mg<4>(sz, hp, a, L, st); break;
        case 5: e = tiled_launch_mg<5>(sz, hp, a, L, st); break;
        case 6: e = tiled_launch_mg<6>(sz, hp, a, L, st); break;
        case 7: e = tiled_launch_mg<7>(sz, hp, a, L, st); break;
        default: e = tiled_launch_mg<8>(sz, hp, a, L, st); break;
    }
    if (e == cudaSuccess && n_launches) *n_launches += 1;
    return e;
}
