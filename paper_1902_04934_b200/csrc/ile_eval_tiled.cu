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
// Per tile of S <= 32 samples:  setup (warp 0, lane = sample: steps 1-4)  ->  K*G accumulation phases  ->  LSE pass.
#include <limits.h>
#include <math_constants.h>

#include "ile_kernels.h"

#define TILED_WARPS 8
#define TILED_THREADS (TILED_WARPS * 32)
#define TILED_CHUNK 64
#define TILED_ROW_REGS 16 /* LSE pass keeps a row of up to 32 * 16 bins in registers */

// exp(x) for x <= 0 (max-subtracted arguments): Cody-Waite reduction x = k ln2 + r, |r| <= ln2/2, degree-11
// near-minimax polynomial (Chebyshev-node interpolant, relative error 1.7e-17 before rounding), exponent patched in
// as an integer add.  Arguments below -708 (result < 3.4e-308) return 0; NaN propagates.
__device__ __forceinline__ double ile_exp_nonpos(double x)
{
    const double MAGIC = 6755399441055744.0;  // 1.5 * 2^52: adding it rounds to the nearest integer
    const double t = fma(x, 1.4426950408889634, MAGIC);
    const double kf = t - MAGIC;
    double r = fma(kf, -6.93147180369123816490e-01, x);
    r = fma(kf, -1.90821492927058770002e-10, r);
    double p = 2.5110037605963777e-08;
    p = fma(p, r, 2.763263963904103e-07);
    p = fma(p, r, 2.755724091857897e-06);
    p = fma(p, r, 2.4801485482328494e-05);
    p = fma(p, r, 0.00019841269890047113);
    p = fma(p, r, 0.0013888888952314775);
    p = fma(p, r, 0.008333333333319601);
    p = fma(p, r, 0.0416666666664881);
    p = fma(p, r, 0.1666666666666668);
    p = fma(p, r, 0.5000000000000019);
    p = fma(p, r, 1.0);
    p = fma(p, r, 1.0);
    const int k = __double2loint(t);
    const double res = __hiloint2double(__double2hiint(p) + (k << 20), __double2loint(p));
    return x < -708.0 ? 0.0 : res;
}

template <int MG>
__global__ void __launch_bounds__(TILED_THREADS, 2) ile_eval_tiled_kernel(IleEvalArgs a, IleTiledLayout L)
{
    extern __shared__ __align__(16) unsigned char smem[];
    double *__restrict__ lin = reinterpret_cast<double *>(smem + L.off_lin);
    double2 *__restrict__ A = reinterpret_cast<double2 *>(smem + L.off_A);
    double *__restrict__ quadS = reinterpret_cast<double *>(smem + L.off_quad);
    int32_t *__restrict__ i0S = reinterpret_cast<int32_t *>(smem + L.off_i0);
    int32_t *__restrict__ badS = reinterpret_cast<int32_t *>(smem + L.off_bad);
    int32_t *__restrict__ rangeS = reinterpret_cast<int32_t *>(smem + L.off_misc);  // lo[K], hi[K]
    int32_t *__restrict__ ctrS = rangeS + 2 * ILE_MAX_DET;                          // one chunk counter per phase

    const IleDevParams *__restrict__ P = a.params;
    const int K = P->n_det, M = P->n_modes, n_q = P->n_q, n_t = P->n_t;
    const int G = L.n_groups, ldA = G * MG, S = L.S, ldl = L.ldl, n_phase = K * G;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long tiles_per_point = (a.n_per_point + S - 1) / S;
    const long long n_tiles = tiles_per_point * a.n_points;
    const double log_nt = log((double)n_t);

    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const int pt = (int)(tile / tiles_per_point);
        const long long s0 = (tile - (long long)pt * tiles_per_point) * S;
        const int cnt = (int)min((long long)S, a.n_per_point - s0);
        const long long flat0 = (long long)pt * a.n_per_point + s0;
        const size_t pglob = (size_t)(a.point0 + pt);
        const double2 *__restrict__ Qp = a.Q + pglob * (size_t)K * M * n_q;

        // ---------------------------------------------------------------- setup: steps 1-4, lane = sample
        if (warp == 0) {
            int bad = 1;
            if (lane < cnt) {
                const long long s = flat0 + lane;
                double q = ile_setup_sample(P, a.U + pglob * (size_t)K * M * M, a.V + pglob * (size_t)K * M * M, a.ra[s],
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
                int v = bad ? INT_MAX : i0S[lane * K + k];
                int w = bad ? INT_MIN : i0S[lane * K + k];
                int lo = __reduce_min_sync(0xffffffffu, v), hi = __reduce_max_sync(0xffffffffu, w);
                if (lane == 0) {
                    const bool any = hi != INT_MIN;
                    rangeS[k] = any ? lo : 0;
                    rangeS[ILE_MAX_DET + k] = any ? hi + n_t : 0;
                }
            }
            for (int p = lane; p < n_phase; p += 32) ctrS[p] = 0;
        }
        __syncthreads();

        // ---------------------------------------------------------------- step 5: accumulation phases
        for (int p = 0; p < n_phase; ++p) {
            const int k = p / G, g = p - k * G;
            const int lo = rangeS[k], hi = rangeS[ILE_MAX_DET + k];
            const bool first = (p == 0);
            for (;;) {
                int c = 0;
                if (lane == 0) c = atomicAdd(&ctrS[p], 1);
                c = __shfl_sync(0xffffffffu, c, 0);
                const int b = lo + c * TILED_CHUNK;
                if (b >= hi) break;

                double2 q0[MG], q1[MG];
                {
                    const int ia = min(b + lane, n_q - 1), ib = min(b + 32 + lane, n_q - 1);
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
                int rel_l = 0;
                bool act = false;
                if (lane < S && !badS[lane]) {
                    rel_l = b - i0S[lane * K + k];
                    act = (rel_l + (TILED_CHUNK - 1) >= 0) && (rel_l < n_t);
                }
                unsigned mask = __ballot_sync(0xffffffffu, act);
                while (mask) {
                    const int al = __ffs(mask) - 1;
                    mask &= mask - 1;
                    const int rel = __shfl_sync(0xffffffffu, rel_l, al);
                    const double2 *__restrict__ Aa = A + ((size_t)al * K + k) * ldA + g * MG;
                    double *__restrict__ row = lin + (size_t)al * ldl;
                    double2 cf[MG];
#pragma unroll
                    for (int mm = 0; mm < MG; ++mm) cf[mm] = Aa[mm];
                    if (rel + 31 >= 0 && rel < n_t) {
                        double tx = 0.0, ty = 0.0;
#pragma unroll
                        for (int mm = 0; mm < MG; ++mm) {
                            tx = fma(cf[mm].x, q0[mm].x, tx);
                            ty = fma(cf[mm].y, q0[mm].y, ty);
                        }
                        const int j = rel + lane;
                        if ((unsigned)j < (unsigned)n_t) row[j] = first ? (tx + ty) : (row[j] + (tx + ty));
                    }
                    if (rel + 63 >= 0 && rel + 32 < n_t) {
                        double tx = 0.0, ty = 0.0;
#pragma unroll
                        for (int mm = 0; mm < MG; ++mm) {
                            tx = fma(cf[mm].x, q1[mm].x, tx);
                            ty = fma(cf[mm].y, q1[mm].y, ty);
                        }
                        const int j = rel + 32 + lane;
                        if ((unsigned)j < (unsigned)n_t) row[j] = first ? (tx + ty) : (row[j] + (tx + ty));
                    }
                }
            }
            __syncthreads();
        }

        // ---------------------------------------------------------------- step 6: log-sum-exp over each row
        const int nt32 = (n_t + 31) >> 5;
        for (int al = warp; al < cnt; al += TILED_WARPS) {
            if (badS[al]) continue;
            const double *__restrict__ row = lin + (size_t)al * ldl;
            double mx = -CUDART_INF, sm = 0.0;
            if (nt32 <= TILED_ROW_REGS) {
                double v[TILED_ROW_REGS];
#pragma unroll
                for (int t = 0; t < TILED_ROW_REGS; ++t) {
                    v[t] = -CUDART_INF;
                    if (t < nt32) {
                        const int j = t * 32 + lane;
                        if (j < n_t) v[t] = row[j];
                        mx = fmax(mx, v[t]);
                    }
                }
                mx = warp_max(mx);
#pragma unroll
                for (int t = 0; t < TILED_ROW_REGS; ++t)
                    if (t < nt32) sm += ile_exp_nonpos(v[t] - mx);
            } else {
                for (int j = lane; j < n_t; j += 32) mx = fmax(mx, row[j]);
                mx = warp_max(mx);
                for (int j = lane; j < n_t; j += 32) sm += ile_exp_nonpos(row[j] - mx);
            }
            sm = warp_sum(sm);
            if (lane == 0) a.lnL[flat0 + al] = mx + log(sm) - log_nt - quadS[al];
        }
        __syncthreads();
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
    uint32_t off = 0;
    L.off_A = off;
    off += (uint32_t)(S * sz.n_det * L.n_groups * MG * sizeof(double2));
    L.off_lin = off;
    off += (uint32_t)(S * L.ldl * sizeof(double));
    L.off_quad = off;
    off += (uint32_t)(32 * sizeof(double));
    L.off_i0 = off;
    off += (uint32_t)(32 * sz.n_det * sizeof(int32_t));
    L.off_bad = off;
    off += (uint32_t)(32 * sizeof(int32_t));
    L.off_misc = off;
    off += (uint32_t)((2 * ILE_MAX_DET + sz.n_det * L.n_groups) * sizeof(int32_t));
    L.bytes = (off + 15u) & ~15u;
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
static cudaError_t tiled_launch_mg(const IleSizes &sz, const IleEvalArgs &a, const IleTiledLayout &L, cudaStream_t st)
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
    ile_eval_tiled_kernel<MG><<<(unsigned)grid, TILED_THREADS, L.bytes, st>>>(a, L);
    return cudaGetLastError();
}

cudaError_t ile_launch_eval_tiled(const IleSizes &sz, const IleEvalArgs &a, cudaStream_t st, int *n_launches)
{
    if (a.n_per_point <= 0 || a.n_points <= 0) return cudaSuccess;
    IleTiledLayout L;
    if (!ile_tiled_plan(sz, (long long)a.n_per_point * a.n_points, &L)) return cudaErrorInvalidConfiguration;
    cudaError_t e;
    switch (L.mg) {
        case 2: e = tiled_launch_mg<2>(sz, a, L, st); break;
        case 3: e = tiled_launch_mg<3>(sz, a, L, st); break;
        case 4: e = tiled_launch_mg<4>(sz, a, L, st); break;
        case 5: e = tiled_launch_mg<5>(sz, a, L, st); break;
        case 6: e = tiled_launch_mg<6>(sz, a, L, st); break;
        case 7: e = tiled_launch_mg<7>(sz, a, L, st); break;
        default: e = tiled_launch_mg<8>(sz, a, L, st); break;
    }
    if (e == cudaSuccess && n_launches) *n_launches += 1;
    return e;
}
