/*
 * ile.h -- C ABI of the B200-native ILE hot path (libile_b200.so).
 *
 * What it computes (arXiv 1902.04934; line numbers are /root/reference/PAPER.md):
 * for one intrinsic point with precomputed mode overlap time series Q_{k,lm}(t) = <h_lm|d_k>(t) and mode-mode
 * matrices U_k, V_k (eq. 8a-c) and for each extrinsic sample (RA, dec, t_ref, phi_ref, psi, inclination,
 * distance), the time-marginalised log-likelihood
 *
 *     lnL_j     = (D_ref/D) Re sum_k sum_lm conj(F_k Y_lm) Q_{k,lm}[i0_k + j]                         eq. 7 / eq. 10 (L64-L67, L90-L91)
 *                 - (D_ref/D)^2/4 sum_k [ |F_k|^2 Y^dagger U_k Y + Re(F_k^2 Y^T V_k Y) ],  j = 0..N_t-1
 *     lnL_margT = ln( (1/N_t) sum_j exp(lnL_j) )                                                      eq. 9 (L81-L86)
 *
 * with F_k = F+,k + i Fx,k the antenna response (L62, L69, L79), Y_lm = _{-2}Y_lm(iota, -phi_ref) (eq. 5-6),
 * i0_k = rint((t_ref + dt_k - t0_Q) f_s) - floor(N_t/2) the per-detector window start from the arrival-time delay
 * dt_k = -(x_k . s)/c (L62, L88), and the Monte Carlo evidence lnZ = ln( (1/n) sum_a w_a L_margT,a ) (eq. 4)
 * with n_eff = sum_a (wL)_a / max_a (wL)_a (L101).  DESIGN.md lists the readings taken where the paper is silent.
 *
 * Conventions
 *  - Every function returns ILE_OK (0) or a negative ile_error; nothing throws across the ABI.
 *  - All floating point is IEEE binary64; complex128 is (re, im) pairs of doubles; indices are int32.
 *  - Angles in radians, times in seconds, distances in Mpc, positions in metres (Earth-fixed frame).
 *  - "device" pointers are CUDA device memory on the context's device; "host" pointers are ordinary host memory.
 *    The library copies Q, U, V and the geometry at ile_create; the caller may free them afterwards.  Sample and
 *    result buffers stay caller-owned.
 *  - Work is enqueued on the caller's CUDA stream (cudaStream_t passed as void*; NULL = default stream) and is
 *    asynchronous unless stated.  Errors detected on the device (a window leaving [0, N_Q)) write -inf for that
 *    sample, never read out of bounds, and bump a sticky counter readable with ile_status().
 *  - A context belongs to the device that was current at ile_create (calls made with another current device return
 *    ILE_ERR_BAD_ARGUMENT) and owns ONE set of scratch buffers: calls on one context must be issued in stream order
 *    (one stream at a time, or ordered by events).  Independent streams take independent contexts.
 *  - One GPU.  There is no CPU fallback and no backend dispatch: without a CUDA device every call fails.
 */
#ifndef ILE_H
#define ILE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    ILE_OK = 0,
    ILE_ERR_BAD_ARGUMENT = -1, /* NULL pointer, size out of the supported range, point index out of range */
    ILE_ERR_CUDA = -2,         /* a CUDA runtime call failed; ile_strerror() gives the CUDA message of the last one */
    ILE_ERR_NO_DEVICE = -3,    /* no CUDA device visible */
    ILE_ERR_UNSUPPORTED = -4,  /* valid but larger than this build's static limits (ILE_MAX_*) */
    ILE_ERR_OUT_OF_RANGE = -5  /* returned by ile_status(): at least one sample's window left the stored Q */
} ile_error;

#define ILE_MAX_DET 8    /* K.  The fast path (sorted streaming FP64-MMA kernel, variant 4) serves K <= 4; contexts with 5..8 detectors are
                            evaluated by the tiled DFMA kernel (variant 2: about twice the time per sample, 0.40 ms against 0.20 ms per
                            1e5 samples at K = 3) or, where its tile does not fit shared memory, by the direct kernel (variant 1, slower
                            still).  Results are the same within rounding.  The paper's own runs use two detectors (L109). */
#define ILE_MAX_MODES 32 /* M */
#define ILE_MAX_L 8      /* largest l of a mode */
#define ILE_SAMPLER_MAX_BINS 512 /* histogram bins per adaptive dimension */

typedef struct ile_ctx ile_ctx; /* opaque, owned by the library */

/* One interferometer: vertex position (m) and unit vectors along the two arms, Earth-fixed frame. */
typedef struct {
    double vertex_m[3];
    double arm_x[3];
    double arm_y[3];
} ile_detector;

typedef struct {
    int32_t n_points;  /* P >= 1 intrinsic points sharing every other field */
    int32_t n_det;     /* K, 1..ILE_MAX_DET */
    int32_t n_modes;   /* M, 1..ILE_MAX_MODES */
    const int32_t *l;  /* host, M entries, 2 <= l <= ILE_MAX_L */
    const int32_t *m;  /* host, M entries, |m| <= l */
    int32_t n_q;       /* N_Q samples per Q series */
    int32_t n_t;       /* N_t bins in the marginalisation window, 1..N_Q */
    double fs_hz;      /* sample rate of Q */
    double t0_q_s;     /* time of Q sample 0 relative to the geocentric reference epoch */
    double gmst_rad;   /* Greenwich mean sidereal time of the event: one value per event (L79) */
    double d_ref_mpc;  /* fiducial distance D_ref of eq. 6 */
    const ile_detector *det; /* host, K entries */
    int32_t shift_mode; /* 0: nearest-sample window shifts (reading R8, the hot path); 1: linear interpolation between the two
                           neighbouring samples of every detector's Q (NEXT-4, reading R8'): i0_k = floor(x_k) - floor(N_t/2),
                           lnL_j uses (1 - phi_k) Q[i0_k + j] + phi_k Q[i0_k + j + 1], phi_k = x_k - floor(x_k); the window then
                           needs i0_k + N_t + 1 <= N_Q; evaluated by the direct kernel (variant 1) and, with
                           twice the channels (Q[i] weighted 1 - phi, Q[i + 1] weighted phi), by the streaming kernel (variant 4) */
} ile_config;

/* Create a context on the current CUDA device: validates cfg, copies Q, U, V (host or device pointers) to the
 * device and builds the mode tables.  Synchronous.
 *   Q: complex128 [P][K][M][N_Q], C order   (eq. 8a; L86-L88: uniformly sampled, truncated to a coincidence window)
 *   U: complex128 [P][K][M][M], U[k][a][b] = <h_a|h_b>_k      (eq. 8b)
 *   V: complex128 [P][K][M][M], V[k][a][b] = <h_a^*|h_b>_k    (eq. 8c)                                            */
int ile_create(ile_ctx **out, const ile_config *cfg, const void *Q, const void *U, const void *V);

/* Time-marginalised lnL for n extrinsic samples of intrinsic point `point` (eq. 7, 9, 10; L97: blocks of samples).
 * All seven sample arrays are device, n doubles each (SoA).  lnL_margT: device, n doubles out.
 * shift_idx: device, n*K int32 out ([sample][detector], the window starts i0_k), or NULL.  n = 0 is a no-op.   */
int ile_eval(ile_ctx *ctx, int32_t point, int64_t n, const double *ra, const double *dec, const double *t_ref,
             const double *phi_ref, const double *psi, const double *incl, const double *dist_mpc,
             double *lnL_margT, int32_t *shift_idx, void *cuda_stream);

/* Every intrinsic point in one launch (BASELINE.json config 4): arrays are [P][n_per_point]; shift_idx
 * [P][n_per_point][K] or NULL. */
int ile_eval_all(ile_ctx *ctx, int64_t n_per_point, const double *ra, const double *dec, const double *t_ref,
                 const double *phi_ref, const double *psi, const double *incl, const double *dist_mpc,
                 double *lnL_margT, int32_t *shift_idx, void *cuda_stream);

/* Evidence (eq. 4; L101): for each of n_segments consecutive runs of n_per_segment samples,
 *   e_a = lnL_margT[a] + log_w[a],  lnZ = ln( (1/count) sum_a exp(e_a) ),  n_eff = sum_a exp(e_a - max_a e_a).
 * log_w: device, same shape as lnL_margT, or NULL (= 0).
 * state: device [n_segments][3] doubles = (running max, sum of exp(e - max), count), IN/OUT so that a long run can
 *        be fed in chunks from one stream (config 3); initialise with ile_evidence_reset or to (-inf, 0, 0).
 *        May be NULL: then the call is self-contained.
 * lnZ, n_eff: device, n_segments doubles out; n_eff may be NULL.  A segment with no finite sample gives
 * lnZ = -inf, n_eff = 0.  n_segments <= 65535 (else ILE_ERR_UNSUPPORTED). */
int ile_evidence(ile_ctx *ctx, int32_t n_segments, int64_t n_per_segment, const double *lnL_margT,
                 const double *log_w, double *state, double *lnZ, double *n_eff, void *cuda_stream);

/* Set n_segments evidence states (device [n_segments][3]) to (-inf, 0, 0). */
int ile_evidence_reset(ile_ctx *ctx, int32_t n_segments, double *state, void *cuda_stream);

/* Combine n_states evidence states of the same n_segments segments -- the sums of eq. 4 (L42-L47) taken over disjoint
 * parts of one sample set, e.g. by independent workers (L134-L141) or by several GPUs: states_in is device
 * [n_states][n_segments][3] doubles, each as ile_evidence leaves it.  Writes the merged state to state_out (device
 * [n_segments][3], may alias states_in[0], may be NULL) and lnZ / n_eff (device, n_segments doubles; n_eff may be NULL)
 * exactly as one ile_evidence call over the union would.  The only data a multi-GPU run of one intrinsic point has to
 * exchange is these 24 bytes per segment and rank. */
int ile_evidence_merge(ile_ctx *ctx, int32_t n_segments, int32_t n_states, const double *states_in, double *state_out,
                       double *lnZ, double *n_eff, void *cuda_stream);

/* ile_evidence without a context and without a single device allocation (eq. 4; n_eff L101): same inputs, same
 * outputs, same arithmetic as ile_evidence above.
 *
 * Why it exists: everything else in this library works out of an ile_ctx, and a context is built from cudaMalloc calls
 * (at ile_create, and later whenever its scratch has to grow).  That rules the library out for callers who may not
 * allocate on the device: code living inside a memory pool it does not own (a framework's caching allocator, a fixed
 * slab handed to a batch job -- a raw cudaMalloc goes around the pool, may fail while the pool still has room, and
 * stalls every stream of the device), real-time loops and plug-ins whose host forbids driver allocations after
 * start-up, or a worker that only wants to fold lnL_margT values it already has into lnZ.  Here the kernel's scratch
 * (per-block partial sums and one ticket word per segment) is a fixed array inside the library's device image, and the
 * call uses no cudaMalloc, cudaFree or allocating library routine.
 *
 * Limits and rules that come with that:
 *  - n_segments <= ILE_EVIDENCE_STATIC_MAX_SEGMENTS, else ILE_ERR_UNSUPPORTED ("size or variant not supported by this
 *    build") and nothing is launched; n_per_segment is not limited.  Devices with an ordinal >= 64 are refused likewise.
 *  - The array (ILE_EVIDENCE_STATIC_SCRATCH_BYTES) is held on every GPU that loads the library, until the process ends.
 *  - The first call made on a device looks up the array's device address (cudaGetSymbolAddress, once per device, with
 *    that device current) and the SM count.  Make that first call during start-up, before any stream capture begins.
 *  - One array per device, shared by all callers and threads, keeping whatever the last call left: each call clears the
 *    ticket words it needs on cuda_stream before its kernel.  Calls that can overlap on the GPU (two streams with no event
 *    between them) race on the array and give wrong results; calls on one stream, or ordered by events, are safe.
 *  - lnL_margT, log_w (may be NULL), state (IN/OUT, may be NULL), lnZ, n_eff (may be NULL): device memory of the current
 *    device, caller-owned, shapes as for ile_evidence.  Asynchronous on cuda_stream. */
#define ILE_EVIDENCE_STATIC_MAX_SEGMENTS 1024
#define ILE_EVIDENCE_STATIC_SCRATCH_BYTES 69632 /* 68 KiB: 1024 ticket words + 4096 (max, sum) pairs */
int ile_evidence_static(int32_t n_segments, int64_t n_per_segment, const double *lnL_margT, const double *log_w,
                        double *state, double *lnZ, double *n_eff, void *cuda_stream);

/* Overlap pre-computation of n_points intrinsic points (eq. 8a-c: Q_{k,lm}(t) = <h_lm|d_k>(t), U_k = <h_lm|h_l'm'>,
 * V_k = <h_lm^*|h_l'm'>) -- what ile_create takes as input, made on the GPU.  Discrete two-sided setting: n_q samples at
 * fs_hz, FFT-order frequency grid f_n = n' fs_hz / n_q (n' the signed index), whitened spectra, <a|b> = sum_n conj(a[n]) b[n]:
 *   Q[p][k][m][i] = sum_n conj(x[p][k][m][n]) d[p][k][n] exp(+2 pi i f_n (t0_q_s + i / fs_hz))   (one inverse FFT per series)
 *   U[p][k][a][b] = sum_n conj(x[p][k][a][n]) x[p][k][b][n],   V[p][k][a][b] = sum_n x[p][k][a][(-n) mod n_q] x[p][k][b][n]
 * x: device complex128 [P][K][M][n_q]; d: device complex128 [P][K][n_q]; Q, U, V: device outputs, caller-owned, shapes as
 * ile_create reads them.  n_q must be a power of two, 2..65536 (else ILE_ERR_UNSUPPORTED; above 8192 a two-level
 * transform through a library-owned scratch buffer).  Asynchronous on cuda_stream; needs no context.  The twiddle table and
 * that scratch buffer are library-owned, one set per device (never freed): calls are thread-safe, and calls on one device are
 * serialised on the GPU -- each waits for the kernels of the previous call, whichever stream that was issued on. */
int ile_precompute(int32_t n_points, int32_t n_det, int32_t n_modes, int32_t n_q, double fs_hz, double t0_q_s, const void *x,
                   const void *d, void *Q, void *U, void *V, void *cuda_stream);

/* The same from UN-whitened spectra with the inner product of eq. 2 (L30-L35), <a|b>_k = 2 int_{f_min < |f| < f_max} a~*(f) b~(f) /
 * S_k(|f|) df: every sum over n above carries the weight g_k[n] = scale / S[p][k][n] for f_min_hz < |f_n| < f_max_hz and 0
 * outside the band ("the inner products necessary to evaluate Q", L97, with the 1/S_n weighting and the band cut done on the
 * device):
 *   Q = sum_n g conj(h) d exp(...),   U = sum_n g conj(h_a) h_b,   V = sum_n g h_a[(-n) mod n_q] h_b[n]
 * h: device complex128 [P][K][M][n_q] mode spectra, d: device complex128 [P][K][n_q] data spectra, S: device double [P][K][n_q]
 * the one-sided noise power spectral density sampled at |f_n| in FFT order (> 0 inside the band), scale: the measure (2 df for
 * eq. 2 as printed, times the caller's Fourier-transform normalisation).  n_q a power of two, 512..65536. */
int ile_precompute_psd(int32_t n_points, int32_t n_det, int32_t n_modes, int32_t n_q, double fs_hz, double t0_q_s, const void *h,
                       const void *d, const double *S, double f_min_hz, double f_max_hz, double scale, void *Q, void *U, void *V,
                       void *cuda_stream);

/* Whole hot path from HOST buffers, for callers that keep samples on the host (the paper's workflow, L97: blocks
 * generated on the CPU and transferred to the board): H2D copy of the seven sample arrays (+ log_w), ile_eval,
 * ile_evidence, D2H of lnL_margT (if not NULL), lnZ and n_eff.  Host arrays of n doubles each; pinned memory makes
 * the copies asynchronous.  Synchronises the stream before returning.  Staging buffers are owned by the context
 * and grow on demand.  From 200,000 samples on (streaming kernel) the batch is cut into 2-4 slices, or one per launch group above 2^20 samples: slice i + 1
 * is uploaded and slice i - 1 downloaded on the context's own copy streams while slice i computes, the evidence state carried on
 * the device; results are those of the unsliced call within rounding. */
int ile_run_host(ile_ctx *ctx, int32_t point, int64_t n, const double *ra, const double *dec, const double *t_ref,
                 const double *phi_ref, const double *psi, const double *incl, const double *dist_mpc,
                 const double *log_w /* may be NULL */, double *lnL_margT /* host out, may be NULL */,
                 double *lnZ /* host out, 1 */, double *n_eff /* host out, 1, may be NULL */, void *cuda_stream);

/* The same for every intrinsic point in one call (BASELINE.json config 4): host arrays are [P][n_per_point] (log_w may be
 * NULL), lnL_margT host out [P][n_per_point] or NULL, lnZ / n_eff host out [P] (n_eff may be NULL).  One H2D per array,
 * one ile_eval_all, one ile_evidence over the P segments, one D2H per result. */
int ile_run_host_all(ile_ctx *ctx, int64_t n_per_point, const double *ra, const double *dec, const double *t_ref,
                     const double *phi_ref, const double *psi, const double *incl, const double *dist_mpc,
                     const double *log_w, double *lnL_margT, double *lnZ, double *n_eff, void *cuda_stream);

/* Sticky device-side status: synchronises the stream, writes the number of samples whose window left [0, N_Q)
 * since the context was created (or since the last reset) and returns ILE_OK or ILE_ERR_OUT_OF_RANGE.
 * reset != 0 clears the counter. */
int ile_status(ile_ctx *ctx, int64_t *n_out_of_range, int reset, void *cuda_stream);

/* Select the evaluation kernel: 0 = automatic (default), 1 = reference-shaped direct kernel (any size), 2 = tiled
 * Q-stationary DFMA kernel, 4 = sorted streaming FP64-MMA kernel (3 is retired).  Returns ILE_ERR_UNSUPPORTED if the variant cannot run this
 * context's sizes.  For tests and benchmarks; results are identical to within rounding. */
int ile_set_variant(ile_ctx *ctx, int32_t variant);

/* Number of kernels this library has launched on behalf of ctx since creation (for bench.py's gpu_launches). */
int64_t ile_launch_count(const ile_ctx *ctx);

/* Calibration: measured FP64 FMA throughput of the device's CUDA cores (register-resident DFMA chains, `iters`
 * dependent steps of 8 independent chains per thread, full grid), in TFLOP/s (2 flops per FMA), and the kernel time
 * in ms.  The roofline denominator for this ALU-bound path.  Synchronous. */
int ile_measure_fp64_peak(int32_t iters, double *tflops, double *ms);

/* The same for the FP64 matrix instruction (mma.sync.m8n8k4.f64, 256 FMA per warp instruction, 8 independent chains per
 * warp) -- the unit the streaming kernel's contraction runs on.  It shares the FP64 pipe with DFMA; bench.py takes the
 * larger of the two measurements as the roofline denominator. */
int ile_measure_dmma_peak(int32_t iters, double *tflops, double *ms);

/* ---------------------------------------------------------------------------------------------------------------------
 * Extrinsic posterior harvesting.  PAPER.md L265: "The code also produces reliable extrinsic parameter
 * distributions ... we harvest joint intrinsic and extrinsic information with a single final iteration."  Readings H1-H3 of
 * DESIGN.md "NEXT-3", restated in oracle/harvest.py.
 *
 * H1 ile_resample: equal-weight posterior samples of the Monte Carlo parameters by SYSTEMATIC resampling of n draws with weights
 * W_a = exp(lnL_margT[a] + log_w[a]) (eq. 4's integrand): output i (i = 0..n_out-1) is the smallest a whose inclusive cumulative
 * weight, accumulated in sample order and normalised, exceeds (i + v0) / n_out; v0 in [0, 1) is the caller's single uniform.
 * The cumulative is a parallel prefix sum in binary64: it equals the sequential sum to a few ulp, not bit for bit, so where a
 * threshold (i + v0) / n_out falls within that distance of a cumulative value the returned id may be the neighbouring sample
 * (both are valid draws; tests/test_gpu_harvest.py accepts either and checks the rest exactly).
 * lnL_margT, log_w (may be NULL): device, n doubles; ids_out: device int64 [n_out], non-decreasing; every entry -1 when no
 * sample has a finite weight. */
int ile_resample(ile_ctx *ctx, int64_t n, const double *lnL_margT, const double *log_w, int64_t n_out, double v0,
                 int64_t *ids_out, void *cuda_stream);

/* H2, H3 ile_harvest: for n_sel harvested samples of intrinsic point `point` -- sample ids[i] of the n-sample device arrays
 * (ids device int64 [n_sel], e.g. from ile_resample; NULL = samples 0..n_sel-1) -- the lnL_j series of eq. 7 over the sample's
 * window is evaluated once more and reduced to
 *   argmax_bin[i]  the first bin j* of the largest lnL_j and lnL_max[i] = lnL_{j*}   (maximised over time instead of eq. 9's average)
 *   drawn_bin[i]   (may be NULL) the smallest bin whose inclusive cumulative of exp(lnL_j) reaches v_uniform[i] times the total:
 *                  a draw of the arrival time from eq. 9's normalised integrand; v_uniform: device, n_sel doubles in (0, 1)
 * Bin j of a sample means the geocentric time t_ref + (j - floor(N_t/2)) / f_s.  A sample whose window leaves the stored Q
 * (reading R9) or an id outside [0, n) gives -1, -inf, -1.  All outputs device, n_sel entries.  With shift_mode = 1 the series is
 * the interpolated one of reading R8' (bin j then means t_ref + (j - floor(N_t/2)) / f_s exactly, not to the nearest sample). */
int ile_harvest(ile_ctx *ctx, int32_t point, int64_t n, const double *ra, const double *dec, const double *t_ref,
                const double *phi_ref, const double *psi, const double *incl, const double *dist_mpc, int64_t n_sel,
                const int64_t *ids, const double *v_uniform, int32_t *argmax_bin, double *lnL_max, int32_t *drawn_bin,
                void *cuda_stream);

void ile_destroy(ile_ctx *ctx);

/* ---------------------------------------------------------------------------------------------------------------------
 * On-device Monte Carlo sampler.  PAPER.md eq. 4: Monte Carlo over the extrinsic
 * parameters, prior uniform in volume and orientation, adaptive sampler of ref. [9]; L97: blocks of samples per likelihood
 * call; L119, L125: sampling prior in the two sky parameters and distance, regenerated every n_chunk draws from the most
 * recent chunk; L101: fixed threshold on n_eff; L251: random number generation on the GPU.  Ref. [9] is not part of the
 * paper: the algorithm is this build's reading (S1-S9), restated in oracle/sampler.py.
 *   S1 uniforms: Philox4x32-10, counters (index_lo, index_hi, j, 0), j = 0..3, key = seed; 53-bit uniforms in (0, 1)
 *   S2 unit-cube coordinates: RA/2pi, (sin dec + 1)/2, (t_ref - t_lo)/(t_hi - t_lo), phi_ref/2pi, psi/pi,
 *      (cos iota + 1)/2, (D^3 - Dmin^3)/(Dmax^3 - Dmin^3): the prior is uniform in them
 *   S3 sampling prior: piecewise-constant densities h_d on n_bins equal bins for d in {RA, dec, distance} (those enabled),
 *      every other dimension from the prior; ln w = -sum_d ln h_d[bin_d]
 *   S6 refit: W_a = exp(temper (lnL_a + ln w_a - max)), H_d[b] = sum rint(W_a 2^40) (integers),
 *      h_d[b] = (1 - floor) n_bins H_d[b] / sum_b H_d[b] + floor
 * All sample arrays are device memory; a sampler belongs to the device current at creation and, like a context, serialises
 * its own scratch (one stream at a time). */
typedef struct ile_sampler ile_sampler;

typedef struct {
    uint64_t seed;        /* Philox key */
    int32_t n_bins;       /* bins per adaptive dimension, 1..ILE_SAMPLER_MAX_BINS */
    int32_t adapt_ra;     /* != 0: RA is adaptive */
    int32_t adapt_dec;    /* != 0: declination is adaptive */
    int32_t adapt_dist;   /* != 0: distance is adaptive */
    double floor_frac;    /* share of the uniform density mixed into every refit density, [0, 1] */
    double temper;        /* exponent of the refit weights, > 0 */
    double dist_min_mpc;  /* prior range of the distance (uniform in volume) */
    double dist_max_mpc;
    double t_ref_lo_s;    /* prior range of t_ref (uniform); lo = hi fixes it */
    double t_ref_hi_s;
} ile_sampler_config;

/* Create a sampler on the current device with uniform densities (the prior).  Synchronous. */
int ile_sampler_create(ile_sampler **out, const ile_sampler_config *cfg);
void ile_sampler_destroy(ile_sampler *s);

/* Densities back to uniform (S9). */
int ile_sampler_reset(ile_sampler *s, void *cuda_stream);

/* Load densities: h host [3][n_bins] (RA, dec, distance; each should average 1), cumulatives rebuilt on the device.
 * Synchronises the stream. */
int ile_sampler_set_tables(ile_sampler *s, const double *h, void *cuda_stream);

/* Read the densities h (host [3][n_bins]) and, if C is not NULL, the cumulatives (host [3][n_bins + 1]).  Synchronises. */
int ile_sampler_get_tables(ile_sampler *s, double *h, double *C, void *cuda_stream);

/* S1 only: the seven Philox uniforms of samples first_index .. first_index + n - 1 -> u device [n][7]. */
int ile_sampler_uniforms(ile_sampler *s, int64_t first_index, int64_t n, double *u, void *cuda_stream);

/* S1-S5: draw samples first_index .. first_index + n - 1 from the current sampling prior.  Outputs are device arrays of n
 * doubles each, laid out as ile_eval reads them; log_w (may be NULL) = ln p - ln p_s, ready for ile_evidence;
 * bin_idx (may be NULL): device int32 [n][3], the bin of each adaptive dimension (-1 where not adaptive), input of the refit. */
int ile_sampler_draw(ile_sampler *s, int64_t first_index, int64_t n, double *ra, double *dec, double *t_ref, double *phi_ref,
                     double *psi, double *incl, double *dist_mpc, double *log_w, int32_t *bin_idx, void *cuda_stream);

/* S6: regenerate the sampling prior from one chunk: bin_idx as ile_sampler_draw wrote it, lnL_margT as ile_eval wrote it,
 * log_w may be NULL (= 0).  A chunk without a finite sample leaves the densities unchanged. */
int ile_sampler_refit(ile_sampler *s, int64_t n, const int32_t *bin_idx, const double *lnL_margT, const double *log_w,
                      void *cuda_stream);

/* Kernels launched on behalf of the sampler since creation. */
int64_t ile_sampler_launch_count(const ile_sampler *s);

/* S7-S8: the whole adaptive Monte Carlo integral of one intrinsic point on the device -- per chunk c: draw samples
 * c n_chunk .. (c+1) n_chunk - 1, ile_eval, ile_evidence with the carried state, refit while c < n_adapt_chunks; stop after
 * the first chunk with n_eff >= n_eff_min or after max_chunks.  Nothing but two doubles per chunk crosses the bus.
 * The sampler's densities are reset first.  Host outputs: lnZ, n_eff (may be NULL), n_samples (may be NULL) = samples used,
 * history (may be NULL): [max_chunks][2] running (lnZ, n_eff) after every chunk up to the stop.  Synchronous. */
int ile_integrate(ile_ctx *ctx, ile_sampler *s, int32_t point, int64_t n_chunk, int32_t max_chunks, int32_t n_adapt_chunks,
                  double n_eff_min, double *lnZ, double *n_eff, int64_t *n_samples, double *history, void *cuda_stream);

/* Static string for an ile_error; for ILE_ERR_CUDA the message of the most recent CUDA failure in this thread. */
const char *ile_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* ILE_H */
