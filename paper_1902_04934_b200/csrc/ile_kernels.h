// ile_kernels.h -- host-side launchers of the CUDA kernels (internal; the public boundary is include/ile.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "ile_device.cuh"

struct IleEvalArgs {
    const IleDevParams *params;  // device
    const double2 *Q;            // device [P][K][M][n_q]
    const double2 *U, *V;        // device [P][K][M][M]
    int32_t point0;              // first intrinsic point of this launch
    int32_t n_points;            // points covered by this launch (1 for ile_eval, P for ile_eval_all)
    int64_t n_per_point;
    const double *ra, *dec, *t_ref, *phi_ref, *psi, *incl, *dist;
    double *lnL;
    int32_t *shift_idx;                 // may be NULL
    unsigned long long *oob_counter;    // device, sticky
    const double *exp_tab;              // device: 2^(i/2048 - 256), i < 2048 (ile_fixexp.cuh; made once per context)
};

// Host copy of the sizes every launcher needs.
struct IleSizes {
    int32_t n_det, n_modes, n_q, n_t;
    int32_t interp;          // 1: linear interpolation of Q between samples (direct kernel; streaming kernel with doubled channels)
    int32_t sm_count;
    int32_t max_smem_optin;  // largest dynamic shared memory one block may ask for
    int32_t smem_per_sm;     // shared memory of one SM
};

// Shared-memory carve-up of the tiled kernel (byte offsets), computed on the host and passed by value.
struct IleTiledLayout {
    int32_t mg;        // modes per group (template parameter of the kernel)
    int32_t n_groups;  // G = ceil(M / mg)
    int32_t S;         // samples per tile, <= 32
    int32_t ldl;       // row stride of lin in doubles
    uint32_t off_sb, sb_bytes;                  // two setup buffers of sb_bytes each, starting at off_sb
    uint32_t sb_quad, sb_i0, sb_bad, sb_misc;   // offsets inside a setup buffer (A sits at 0)
    uint32_t off_lin;                           // lin[S][ldl]
    uint32_t bytes;
};

// variant 1: direct kernel (one warp per sample, lanes over time bins, Q through L1/L2).  Any size.
cudaError_t ile_launch_eval_direct(const IleSizes &sz, const IleEvalArgs &a, cudaStream_t st, int *n_launches);

// variant 2: tiled, Q-stationary kernel (ile_eval_tiled.cu).  ile_tiled_plan returns false when the sizes do not fit.
bool ile_tiled_plan(const IleSizes &sz, long long n_total, IleTiledLayout *out);
cudaError_t ile_launch_eval_tiled(const IleSizes &sz, const IleDevParams &hp, const IleEvalArgs &a, cudaStream_t st,
                                  int *n_launches);

// ---- counting sort of the streaming path (variant 4) -----------------------------------------------------------------
// Cell grid: segments = (i0_1 - i0_0, i0_2 - i0_0[, i0_3 - i0_0]) cells of width 2^g, inside a segment bins of i0_0 of width 2^g0.
struct IleSortPlan {
    int32_t g;        // log2 of the (d1, d2) cell width in samples
    int32_t g0;       // log2 of the i0_0 bin width inside a segment
    int32_t nd;       // detectors that take part in the key (<= 4)
    int32_t n0, n1, n2, n3;
    int32_t nseg;     // n1*n2*n3 segments
    int32_t ncell;    // n0*nseg + 1; the last cell collects out-of-range samples
    int32_t dmax[4];  // bound on |i0_d - i0_0| from the light travel time between the sites
};

// Device scratch of the sorted path (owned by the context).
struct IleSortScratch {
    double *rec;       // [n][K * cp] coefficients a F_k Y_lm, (Re, Im) interleaved, zero padded to cp channels per detector
    double *quad;      // [n]
    int32_t *i0;       // [n][K]
    int32_t *cell;     // [n]
    uint32_t *hist;    // 2 x ILE_STREAM_MAX_RANGES claim counters, [n_points][ncell] cell counts -> positions inside the segment, [n_points][nseg] segment totals; zero between launches
    double *qform;     // [n][K][3] quadratic forms from the FP64-MMA kernel, or NULL (the coefficient kernel computes them)
};

// ---- variant 4: streaming FP64-MMA kernel, one warp per group of 8 samples (ile_eval_stream.cu) ------------------
struct IleStreamPlan {
    int32_t ks;       // k-steps of 4 real channels per detector: ceil(2M / 4), rounded up to an instantiated value
    int32_t cp;       // padded channels per detector = 4 * ks (= record stride per detector)
    int32_t nc;       // (d1, d2) cell width = 8 * nc rows; the shuffle realignment looks nc blocks ahead
    int32_t padf;     // zero rows in front of each packed series
    int32_t nqp;      // rows per packed series = padf + n_q + back padding
    int32_t ctas_per_sm;  // resident CTAs of the streaming kernel per SM on the context's device (ile_stream_prepare)
};

#define ILE_STREAM_MAX_RANGES 256 /* claim counters of the streaming kernel, kept right behind the histograms */

struct IleStreamScratch {
    const double *Qs;   // packed Q [P][K][ks][nqp][4]
    int32_t *slots;     // [n_points][slot_cap]: sample index or -1, groups of 8 consecutive slots
    int32_t *gcum;      // [n_points + 1]: exclusive prefix of the points' group counts
    int64_t slot_cap;   // slots per point (multiple of 8)
    cudaStream_t aux;   // side stream: the coefficient kernel runs there while the caller's stream sorts
    cudaEvent_t ev_fork, ev_join;
    const double *quad_mats;  // packed U, V for ile_launch_quad_mma, or NULL
    cudaEvent_t ev_late;  // if not NULL: the arrays the coefficient kernel reads (phi_ref, psi, incl, dist) arrive with this event
    const double2 *hU, *hV;  // host mirrors of U, V [P][K][M][M] (kernel-parameter path of the coefficient kernel), or NULL
    double *tabs;        // exp and log tables of the streaming kernel (ile_stream_alloc_tables)
    uint32_t launch_no;  // parity picks the claim counters of a launch
    bool hist_clean;     // sc.hist is all zero (set when it is allocated and by every successful launch)
    size_t hist_words;   // allocated words of sc.hist: what a launch after a failed one clears
};

cudaError_t ile_stream_alloc_tables(IleStreamScratch *ss);

// nc = 1, 2: (d1, d2) sort cells of 8 nc rows -- narrow cells need one select per realigned element instead of two but four times the
// segments (padding and shorter runs of equal rows); measured: nc = 1 wins by 2-6 % once a segment holds a thousand samples or more
// (three detectors: 280 segments, 1e6 samples; two: 21 segments, 1e5), nc = 2 below (6 % at 30,000 samples, three detectors)
bool ile_stream_plan(const IleSizes &sz, const IleDevParams &hp, int nc, IleStreamPlan *out, IleSortPlan *sp);
#define ILE_STREAM_NC1_MIN_PER_SEGMENT 1024
cudaError_t ile_stream_prepare(const IleSizes &sz, IleStreamPlan *pl);  // per context: function attributes + occupancy on its device
cudaError_t ile_launch_pack_q_stream(const IleSizes &sz, const IleStreamPlan &pl, int32_t n_points, const double2 *Q,
                                     double *Qs, cudaStream_t st);
// setup + sort of variant 4 (memsets + setup + scan + scatter), then the streaming kernel
cudaError_t ile_launch_eval_stream(const IleSizes &sz, const IleDevParams &hp, const IleEvalArgs &a, const IleStreamPlan &pl,
                                   const IleSortPlan &sp, const IleSortScratch &sc, IleStreamScratch &ss,
                                   cudaStream_t st, int *n_launches);
// variant 4: coefficients a F_k Y_lm and quadratic term of every sample (steps 1, 3, 4), no sorting work
// (hU, hV: host mirrors of the context's U, V, or NULL; returns the number of kernels launched)
int ile_launch_setup_coef(const IleSizes &sz, const IleDevParams &hp, const IleEvalArgs &a, int32_t cp, const IleSortScratch &sc,
                          const double2 *hU, const double2 *hV, cudaStream_t st);

// step 4 for many modes (ile_quad_mma.cu): packed real representations of U, V and the batched quadratic forms
size_t ile_quad_pack_doubles(int32_t n_points, int32_t K, int32_t M);
void ile_quad_pack_host(int32_t n_points, int32_t K, int32_t M, const double2 *U, const double2 *V, double *out);
cudaError_t ile_launch_quad_mma(const IleSizes &sz, const IleDevParams &hp, const IleEvalArgs &a, const double *mats, double *qform,
                                cudaStream_t st);

// ---- shared by the translation units of the C ABI (ile_api.cu, ile_sampler_api.cu) -----------------------------------------
int ile_cuda_fail(cudaError_t e);  // records the message for ile_strerror, returns ILE_ERR_CUDA
int ile_ctx_sm_count(const ile_ctx *c);
void ile_ctx_add_launches(ile_ctx *c, int n);

// ---- on-device Monte Carlo sampler (ile_sampler.cu; NEXT-2) ------------------------------------------------------------
struct IleSamplerParams {
    unsigned long long seed;
    int32_t n_bins;
    int32_t adapt[3];  // RA, dec, distance
    double floor_frac, temper;
    double t_lo, t_span;      // t_ref = t_lo + t_span u
    double dmin3, d3_span;    // D = cbrt(dmin3 + u d3_span), dmin3 = Dmin Dmin Dmin
};
size_t ile_sampler_table_doubles(int32_t n_bins);  // h [3][n_bins] followed by C [3][n_bins + 1]
cudaError_t ile_launch_sampler_tables(const IleSamplerParams &P, double *tab, int set_uniform, cudaStream_t st);
cudaError_t ile_launch_sampler_uniforms(const IleSamplerParams &P, int sm_count, long long first, long long n, double *u, cudaStream_t st);
cudaError_t ile_launch_sampler_draw(const IleSamplerParams &P, int sm_count, const double *tab, long long first, long long n, double *ra,
                                    double *dec, double *t_ref, double *phi_ref, double *psi, double *incl, double *dist, double *log_w,
                                    int32_t *bins, cudaStream_t st);
size_t ile_sampler_work_words(int32_t n_bins);  // 64-bit words of refit scratch
cudaError_t ile_sampler_work_init(const IleSamplerParams &P, unsigned long long *work, cudaStream_t st);
cudaError_t ile_launch_sampler_refit(const IleSamplerParams &P, int sm_count, double *tab, long long n, const int32_t *bins, const double *lnL,
                                     const double *log_w, unsigned long long *work, cudaStream_t st);  // 2 kernels

// ---- extrinsic posterior harvesting (ile_harvest.cu; NEXT-3) -------------------------------------------------------------
cudaError_t ile_launch_harvest(const IleSizes &sz, const IleEvalArgs &a, long long n_sel, const long long *ids, const double *v_uniform,
                               int32_t *argmax_bin, double *lnL_max, int32_t *drawn_bin, cudaStream_t st);
size_t ile_resample_scratch_doubles(long long n);
cudaError_t ile_launch_resample(const IleSizes &sz, long long n, const double *lnL, const double *log_w, long long n_out, double v0,
                                double *scratch, long long *ids, cudaStream_t st, int *n_launches);

// overlap pre-computation (ile_precompute.cu)
cudaError_t ile_launch_precompute(int32_t n_points, int32_t K, int32_t M, int32_t N, double fs_hz, double t0_q_s, const double2 *x,
                                  const double2 *d, const double *S /* NULL: whitened spectra */, double f_min_hz, double f_max_hz,
                                  double scale, double2 *Q, double2 *U, double2 *V, int32_t max_smem_optin, cudaStream_t st);

// evidence: one kernel (per-block partials; the block of a segment that finishes last folds them into the carried state).
// partials: n_segments * blocks_per_seg * 2 doubles; tickets: n_segments words, zero on entry, left zero on exit
cudaError_t ile_launch_evidence(int32_t n_segments, int64_t n_per_segment, const double *lnL, const double *log_w,
                                double *state, double *lnZ, double *n_eff, double *partials, unsigned int *tickets, int32_t blocks_per_seg,
                                cudaStream_t st, int *n_launches);
int32_t ile_evidence_blocks_per_segment(int32_t n_segments, int64_t n_per_segment, int32_t sm_count);
cudaError_t ile_launch_evidence_merge(int32_t n_segments, int32_t n_states, const double *states_in, double *state_out,
                                      double *lnZ, double *n_eff, cudaStream_t st, int *n_launches);
cudaError_t ile_launch_evidence_prefix(int32_t n_chunks, const double *states, double *run, double *hist, cudaStream_t st);
cudaError_t ile_launch_evidence_reset(int32_t n_segments, double *state, cudaStream_t st, int *n_launches);

// calibration kernels: dmma = 0 register-resident DFMA chains, 1 = DMMA.8x8x4 chains; 8 blocks of 256 threads per SM
cudaError_t ile_launch_fp64_peak(int32_t iters, int32_t sm_count, double *sink, int dmma, cudaStream_t st);
