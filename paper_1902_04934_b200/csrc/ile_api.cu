// ile_api.cu -- the C ABI of include/ile.h: context management, argument checking, kernel dispatch.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "ile_kernels.h"

#define ILE_PIPE_MAX_SLICES 16
#ifndef ILE_PIPE_MIN_SLICE
#define ILE_PIPE_MIN_SLICE 100000 /* samples per slice of a pipelined ile_run_host: at 50,000 the host needs as long to issue two slices as the copies take (measured: 0.369 against 0.374 ms at 1e5 samples), from 2 x 100,000 on the overlap wins (1e6 samples: 2.82 -> 2.16 ms) */
#endif

struct ile_ctx {
    int device;
    IleSizes sz;
    int32_t n_points;
    IleDevParams hparams;
    IleDevParams *dparams;
    double2 *dQ, *dU, *dV;
    double2 *hU, *hV;  // host mirrors of U, V (coefficient kernel: kernel-parameter path)
    unsigned long long *d_oob;
    double *d_partials;
    size_t partials_cap;  // doubles
    unsigned int *d_tickets;  // one word per evidence segment; zero between calls (the kernel's last block resets its own)
    size_t tickets_cap;
    double *d_stage;
    size_t stage_cap;  // doubles
    double *d_small;   // lnZ, n_eff (device)
    double *h_small;   // pinned mirror
    int32_t variant;
    long long launches;
    // variant 4 (sorted, streaming FP64-MMA path)
    int64_t chunk_samples;  // samples per launch group (bounds the scratch: <= 2 GiB of records, <= 2^20 samples)
    IleSortScratch sc;
    size_t sc_samples, sc_hist;  // capacities (samples, histogram words)
    int32_t sc_recg;             // doubles per record the scratch was sized for
    bool stream_ok;
    IleStreamPlan spl, spl1;  // sort cells of 16 rows (nc = 2) and of 8 rows (nc = 1, big batches)
    IleSortPlan ssp, ssp1;
    bool nc1_ok;
    double *dQs;
    IleStreamScratch ss;
    size_t ss_slots, ss_gcum;  // capacities in words
    double *d_quad_mats;  // packed real representations of U, V for the FP64-MMA quadratic forms (M >= ILE_QUAD_MMA_MIN_MODES)
    double *d_qform;      // [n][K][3]
    size_t qform_cap;     // samples
    double *d_resample;   // scratch of ile_resample
    size_t resample_cap;  // doubles
    cudaStream_t copy_stream;  // ile_run_host: second H2D queue
    cudaEvent_t ev_copy_go, ev_copy_done;
    // ile_run_host, sliced: uploads of slice i + 1 and the download of slice i - 1 run beside the kernels of slice i
    cudaStream_t d2h_stream;
    cudaEvent_t ev_pipe[3 * ILE_PIPE_MAX_SLICES];  // per slice: sort inputs arrived, other inputs arrived, lnL_margT ready
    cudaEvent_t ev_d2h_done;
    double *d_pipe_state;  // evidence state (max, sum, count) carried over the slices
};

static thread_local char g_cuda_msg[256] = "no CUDA error recorded";

static int cuda_fail(cudaError_t e)
{
    snprintf(g_cuda_msg, sizeof(g_cuda_msg), "CUDA error %d: %s", (int)e, cudaGetErrorString(e));
    return ILE_ERR_CUDA;
}
int ile_cuda_fail(cudaError_t e) { return cuda_fail(e); }  // for the other translation units of the C ABI
int ile_ctx_sm_count(const ile_ctx *c);
// Function attributes, streams and every buffer of a context belong to the device it was created on.
static int check_device(const ile_ctx *c)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return ILE_ERR_NO_DEVICE;
    return dev == c->device ? ILE_OK : ILE_ERR_BAD_ARGUMENT;
}
#ifndef ILE_CHUNK_BYTES
#define ILE_CHUNK_BYTES (2048u << 20) /* record scratch per launch group: bigger groups sort into tighter windows and pay one pre-pass */
#endif
#ifndef ILE_QUAD_MMA_MIN_MODES
#define ILE_QUAD_MMA_MIN_MODES 8
#endif
#ifndef ILE_STREAM_MIN_SAMPLES
#define ILE_STREAM_MIN_SAMPLES 10000 /* automatic choice: batches per point from this size on take the streaming variant */
#endif
#ifndef ILE_CHUNK_MAX
#define ILE_CHUNK_MAX 1048576
#endif
#define CK(call)                                  \
    do {                                          \
        cudaError_t e__ = (call);                 \
        if (e__ != cudaSuccess) return cuda_fail(e__); \
    } while (0)

static double factorial(int n)
{
    double r = 1.0;
    for (int i = 2; i <= n; ++i) r *= (double)i;
    return r;
}

// sqrt((2l+1)/4pi) d^l_{m,2}(beta) as sum_t coef_t cos(beta/2)^pc_t sin(beta/2)^ps_t  (Wigner's finite sum with m' = m, m = 2;
// _{-2}Y_lm = sqrt((2l+1)/4pi) d^l_{m,2}(theta) e^{i m phi}, reading R5)
static int build_mode_table(IleDevParams &P, int idx, int l, int m)
{
    const double norm = std::sqrt((2.0 * l + 1.0) / (4.0 * M_PI));
    const double pref = std::sqrt(factorial(l + 2) * factorial(l - 2) * factorial(l + m) * factorial(l - m));
    int nt = 0;
    for (int k = 0; k <= 2 * l; ++k) {
        int a = l + 2 - k, b = k, c = l - k - m, d = k - 2 + m;
        if (a < 0 || b < 0 || c < 0 || d < 0) continue;
        if (nt >= ILE_MAX_TERMS) return ILE_ERR_UNSUPPORTED;
        double sign = (d % 2 == 0) ? 1.0 : -1.0;
        P.mode_coef[idx][nt] = norm * sign * pref / (factorial(a) * factorial(b) * factorial(c) * factorial(d));
        P.mode_pc[idx][nt] = (int8_t)(2 * l - 2 * k + 2 - m);
        P.mode_ps[idx][nt] = (int8_t)(2 * k - 2 + m);
        ++nt;
    }
    P.mode_nterm[idx] = nt;
    P.mode_m[idx] = m;
    return ILE_OK;
}

extern "C" int ile_create(ile_ctx **out, const ile_config *cfg, const void *Q, const void *U, const void *V)
{
    if (!out || !cfg || !Q || !U || !V || !cfg->l || !cfg->m || !cfg->det) return ILE_ERR_BAD_ARGUMENT;
    *out = nullptr;
    if (cfg->n_points < 1 || cfg->n_det < 1 || cfg->n_modes < 1 || cfg->n_q < 1 || cfg->n_t < 1 || cfg->n_t > cfg->n_q)
        return ILE_ERR_BAD_ARGUMENT;
    if (!(cfg->fs_hz > 0.0) || !(cfg->d_ref_mpc > 0.0) || !std::isfinite(cfg->t0_q_s) || !std::isfinite(cfg->gmst_rad))
        return ILE_ERR_BAD_ARGUMENT;
    if (cfg->n_det > ILE_MAX_DET || cfg->n_modes > ILE_MAX_MODES) return ILE_ERR_UNSUPPORTED;
    if (cfg->shift_mode != 0 && cfg->shift_mode != 1) return ILE_ERR_BAD_ARGUMENT;
    for (int j = 0; j < cfg->n_modes; ++j) {
        if (cfg->l[j] < 2 || std::abs(cfg->m[j]) > cfg->l[j]) return ILE_ERR_BAD_ARGUMENT;
        if (cfg->l[j] > ILE_MAX_L) return ILE_ERR_UNSUPPORTED;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return ILE_ERR_NO_DEVICE;
    }
    int device = 0;
    cudaDeviceProp prop;
    CK(cudaGetDevice(&device));  // nothing is allocated yet: a failure here leaks nothing
    CK(cudaGetDeviceProperties(&prop, device));
    ile_ctx *c = new (std::nothrow) ile_ctx();
    if (!c) return ILE_ERR_BAD_ARGUMENT;
    std::memset(c, 0, sizeof(*c));
    c->device = device;
    c->sz.n_det = cfg->n_det;
    c->sz.n_modes = cfg->n_modes;
    c->sz.n_q = cfg->n_q;
    c->sz.n_t = cfg->n_t;
    c->sz.interp = cfg->shift_mode;
    c->sz.sm_count = prop.multiProcessorCount;
    c->sz.max_smem_optin = (int32_t)prop.sharedMemPerBlockOptin;
    c->sz.smem_per_sm = (int32_t)prop.sharedMemPerMultiprocessor;
    c->n_points = cfg->n_points;

    IleDevParams &P = c->hparams;
    P.n_points = cfg->n_points;
    P.n_det = cfg->n_det;
    P.n_modes = cfg->n_modes;
    P.n_q = cfg->n_q;
    P.n_t = cfg->n_t;
    P.interp = cfg->shift_mode;
    P.fs = cfg->fs_hz;
    P.t0_q = cfg->t0_q_s;
    P.gmst = cfg->gmst_rad;
    P.d_ref = cfg->d_ref_mpc;
    for (int k = 0; k < cfg->n_det; ++k) {
        const double *x = cfg->det[k].arm_x, *y = cfg->det[k].arm_y;
        const int ii[6] = {0, 0, 0, 1, 1, 2}, jj[6] = {0, 1, 2, 1, 2, 2};
        for (int e = 0; e < 6; ++e) P.det_tensor[k][e] = 0.5 * (x[ii[e]] * x[jj[e]] - y[ii[e]] * y[jj[e]]);
        for (int e = 0; e < 3; ++e) P.vertex[k][e] = cfg->det[k].vertex_m[e];
    }
    for (int j = 0; j < cfg->n_modes; ++j) {
        int r = build_mode_table(P, j, cfg->l[j], cfg->m[j]);
        if (r != ILE_OK) {
            delete c;
            return r;
        }
    }
    const size_t KM = (size_t)cfg->n_det * cfg->n_modes;
    const size_t nQ = (size_t)cfg->n_points * KM * cfg->n_q, nU = (size_t)cfg->n_points * KM * cfg->n_modes;
    cudaError_t e;
#define CKC(call)                 \
    do {                          \
        e = (call);               \
        if (e != cudaSuccess) {   \
            ile_destroy(c);       \
            return cuda_fail(e);  \
        }                         \
    } while (0)
    CKC(cudaMalloc(&c->dparams, sizeof(IleDevParams)));
    CKC(cudaMalloc(&c->dQ, nQ * sizeof(double2)));
    CKC(cudaMalloc(&c->dU, nU * sizeof(double2)));
    CKC(cudaMalloc(&c->dV, nU * sizeof(double2)));
    CKC(cudaMalloc(&c->d_oob, sizeof(unsigned long long)));
    CKC(cudaMalloc(&c->d_small, 2 * (size_t)cfg->n_points * sizeof(double)));  // lnZ[P], n_eff[P] of ile_run_host(_all)
    CKC(cudaMallocHost(&c->h_small, 2 * (size_t)cfg->n_points * sizeof(double)));
    CKC(cudaMemcpy(c->dparams, &P, sizeof(P), cudaMemcpyHostToDevice));
    CKC(cudaMemcpy(c->dQ, Q, nQ * sizeof(double2), cudaMemcpyDefault));
    CKC(cudaMemcpy(c->dU, U, nU * sizeof(double2), cudaMemcpyDefault));
    CKC(cudaMemcpy(c->dV, V, nU * sizeof(double2), cudaMemcpyDefault));
    CKC(cudaMemset(c->d_oob, 0, sizeof(unsigned long long)));
    c->hU = new (std::nothrow) double2[nU];
    c->hV = new (std::nothrow) double2[nU];
    if (!c->hU || !c->hV) {
        ile_destroy(c);
        return ILE_ERR_BAD_ARGUMENT;
    }
    CKC(cudaMemcpy(c->hU, c->dU, nU * sizeof(double2), cudaMemcpyDeviceToHost));
    CKC(cudaMemcpy(c->hV, c->dV, nU * sizeof(double2), cudaMemcpyDeviceToHost));
    CKC(ile_stream_alloc_tables(&c->ss));  // exp / log tables of the streaming and tiled kernels
    CKC(cudaStreamSynchronize(0));         // their kernel runs on the legacy default stream: done before ile_create returns, whatever follows
    c->stream_ok = ile_stream_plan(c->sz, c->hparams, 2, &c->spl, &c->ssp);
    // a streaming plan the device cannot host (no resident block) is a refused plan, not a failed create: variants 2 / 1 serve it
    if (c->stream_ok && ile_stream_prepare(c->sz, &c->spl) != cudaSuccess) {
        cudaGetLastError();
        c->stream_ok = false;
    }
    c->nc1_ok = c->stream_ok && ile_stream_plan(c->sz, c->hparams, 1, &c->spl1, &c->ssp1);
    if (c->nc1_ok && ile_stream_prepare(c->sz, &c->spl1) != cudaSuccess) {
        cudaGetLastError();
        c->nc1_ok = false;
    }
    if (c->stream_ok) {
        if (cfg->n_modes >= ILE_QUAD_MMA_MIN_MODES) {
            const size_t nd = ile_quad_pack_doubles(cfg->n_points, cfg->n_det, cfg->n_modes);
            double *hm = new (std::nothrow) double[nd];
            if (!hm) {
                ile_destroy(c);
                return ILE_ERR_CUDA;
            }
            cudaError_t e3 = cudaMalloc(&c->d_quad_mats, nd * sizeof(double));
            if (e3 == cudaSuccess) {
                ile_quad_pack_host(cfg->n_points, cfg->n_det, cfg->n_modes, c->hU, c->hV, hm);
                e3 = cudaMemcpy(c->d_quad_mats, hm, nd * sizeof(double), cudaMemcpyHostToDevice);
            }
            delete[] hm;
            CKC(e3);
        }
        CKC(cudaStreamCreateWithFlags(&c->ss.aux, cudaStreamNonBlocking));
        CKC(cudaEventCreateWithFlags(&c->ss.ev_fork, cudaEventDisableTiming));
        CKC(cudaEventCreateWithFlags(&c->ss.ev_join, cudaEventDisableTiming));
        CKC(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        CKC(cudaEventCreateWithFlags(&c->ev_copy_go, cudaEventDisableTiming));
        CKC(cudaEventCreateWithFlags(&c->ev_copy_done, cudaEventDisableTiming));
        CKC(cudaStreamCreateWithFlags(&c->d2h_stream, cudaStreamNonBlocking));
        for (int i = 0; i < 3 * ILE_PIPE_MAX_SLICES; ++i) CKC(cudaEventCreateWithFlags(&c->ev_pipe[i], cudaEventDisableTiming));
        CKC(cudaEventCreateWithFlags(&c->ev_d2h_done, cudaEventDisableTiming));
        CKC(cudaMalloc(&c->d_pipe_state, 3 * sizeof(double)));
        const size_t nQs = (size_t)cfg->n_points * cfg->n_det * c->spl.ks * c->spl.nqp * 4;
        CKC(cudaMalloc(&c->dQs, nQs * sizeof(double)));
        CKC(ile_launch_pack_q_stream(c->sz, c->spl, cfg->n_points, c->dQ, c->dQs, 0));
        CKC(cudaDeviceSynchronize());
        c->sc_recg = cfg->n_det * c->spl.cp;
        const int64_t cs = (int64_t)ILE_CHUNK_BYTES / ((int64_t)c->sc_recg * 8);
        c->chunk_samples = cs < 16384 ? 16384 : cs > ILE_CHUNK_MAX ? ILE_CHUNK_MAX : cs;
    }
#undef CKC
    *out = c;
    return ILE_OK;
}

extern "C" void ile_destroy(ile_ctx *c)
{
    if (!c) return;
    cudaFree(c->dparams);
    cudaFree(c->dQ);
    cudaFree(c->dU);
    cudaFree(c->dV);
    cudaFree(c->d_oob);
    cudaFree(c->d_partials);
    cudaFree(c->d_tickets);
    cudaFree(c->d_stage);
    cudaFree(c->d_small);
    cudaFree(c->sc.rec);
    cudaFree(c->sc.quad);
    cudaFree(c->sc.i0);
    cudaFree(c->sc.cell);
    cudaFree(c->sc.hist);
    cudaFree(c->dQs);
    cudaFree(c->ss.slots);
    cudaFree(c->ss.gcum);
    cudaFree(c->ss.tabs);
    cudaFree(c->d_quad_mats);
    cudaFree(c->d_qform);
    cudaFree(c->d_resample);
    if (c->ss.aux) cudaStreamDestroy(c->ss.aux);
    if (c->ss.ev_fork) cudaEventDestroy(c->ss.ev_fork);
    if (c->ss.ev_join) cudaEventDestroy(c->ss.ev_join);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    if (c->ev_copy_go) cudaEventDestroy(c->ev_copy_go);
    if (c->ev_copy_done) cudaEventDestroy(c->ev_copy_done);
    if (c->d2h_stream) cudaStreamDestroy(c->d2h_stream);
    for (int i = 0; i < 3 * ILE_PIPE_MAX_SLICES; ++i)
        if (c->ev_pipe[i]) cudaEventDestroy(c->ev_pipe[i]);
    if (c->ev_d2h_done) cudaEventDestroy(c->ev_d2h_done);
    cudaFree(c->d_pipe_state);
    if (c->h_small) cudaFreeHost(c->h_small);
    delete[] c->hU;
    delete[] c->hV;
    delete c;
}

// Scratch of the sorted path, grown on demand (never inside a launch sequence that still uses the old buffers: the
// stream is synchronised first).
static int ensure_scratch(ile_ctx *c, size_t samples, size_t hist_words, cudaStream_t st)
{
    if (samples > c->sc_samples) {
        CK(cudaStreamSynchronize(st));
        cudaFree(c->sc.rec), cudaFree(c->sc.quad), cudaFree(c->sc.i0), cudaFree(c->sc.cell);
        c->sc.rec = nullptr, c->sc.quad = nullptr, c->sc.i0 = nullptr, c->sc.cell = nullptr;
        c->sc_samples = 0;
        CK(cudaMalloc(&c->sc.rec, samples * c->sc_recg * sizeof(double)));
        CK(cudaMalloc(&c->sc.quad, samples * sizeof(double)));
        CK(cudaMalloc(&c->sc.i0, samples * c->sz.n_det * sizeof(int32_t)));
        CK(cudaMalloc(&c->sc.cell, samples * sizeof(int32_t)));
        c->sc_samples = samples;
    }
    if (hist_words > c->sc_hist) {
        CK(cudaStreamSynchronize(st));
        cudaFree(c->sc.hist);
        c->sc.hist = nullptr;
        c->sc_hist = 0;
        CK(cudaMalloc(&c->sc.hist, hist_words * sizeof(uint32_t)));
        CK(cudaMemsetAsync(c->sc.hist, 0, hist_words * sizeof(uint32_t), st));
        c->sc_hist = hist_words;
        c->ss.hist_words = hist_words;
        c->ss.hist_clean = true;
    }
    return ILE_OK;
}

// variant 4 for one launch group: setup + sort into padded segments + streaming kernel
static int eval_stream_group(ile_ctx *c, IleEvalArgs a, cudaStream_t st)
{
    const bool nc1 = c->nc1_ok && a.n_per_point >= (int64_t)ILE_STREAM_NC1_MIN_PER_SEGMENT * c->ssp1.nseg;
    const IleSortPlan &sp = nc1 ? c->ssp1 : c->ssp;
    const size_t nseg = (size_t)sp.nseg;
    const int64_t slot_cap = (((a.n_per_point + 7) & ~(int64_t)7) + 8 * (int64_t)nseg + 31) & ~(int64_t)31;  // groups per point: multiple of 4
    int r = ensure_scratch(c, (size_t)a.n_per_point * a.n_points, (size_t)a.n_points * (sp.ncell + nseg) + 2 * ILE_STREAM_MAX_RANGES, st);
    if (r != ILE_OK) return r;
    const size_t need_slots = (size_t)a.n_points * slot_cap, need_g = 2 * (size_t)a.n_points + 2;
    if (need_slots > c->ss_slots || need_g > c->ss_gcum) {
        CK(cudaStreamSynchronize(st));
        if (need_slots > c->ss_slots) {
            cudaFree(c->ss.slots);
            c->ss.slots = nullptr, c->ss_slots = 0;
            CK(cudaMalloc(&c->ss.slots, need_slots * sizeof(int32_t)));
            c->ss_slots = need_slots;
        }
        if (need_g > c->ss_gcum) {
            cudaFree(c->ss.gcum);
            c->ss.gcum = nullptr, c->ss_gcum = 0;
            CK(cudaMalloc(&c->ss.gcum, need_g * sizeof(int32_t)));
            c->ss_gcum = need_g;
        }
    }
    c->ss.Qs = c->dQs;
    c->ss.hU = c->hU, c->ss.hV = c->hV;
    c->ss.slot_cap = slot_cap;
    // many modes: the quadratic forms run as an FP64-MMA contraction in front of the coefficient kernel (side stream)
    const bool quad_mma = c->d_quad_mats && (a.n_points == 1 || (a.n_per_point & 7) == 0);
    if (quad_mma) {
        const size_t ns = (size_t)a.n_per_point * a.n_points;
        if (ns > c->qform_cap) {
            CK(cudaStreamSynchronize(st));
            cudaFree(c->d_qform);
            c->d_qform = nullptr, c->qform_cap = 0;
            CK(cudaMalloc(&c->d_qform, ns * c->sz.n_det * 3 * sizeof(double)));
            c->qform_cap = ns;
        }
    }
    c->sc.qform = quad_mma ? c->d_qform : nullptr;
    c->ss.quad_mats = quad_mma ? c->d_quad_mats : nullptr;
    int nl = 0;
    cudaError_t e = ile_launch_eval_stream(c->sz, c->hparams, a, nc1 ? c->spl1 : c->spl, sp, c->sc, c->ss, st, &nl);
    c->launches += nl;
    if (e != cudaSuccess) return cuda_fail(e);
    return ILE_OK;
}

static int eval_dispatch(ile_ctx *c, int32_t point0, int32_t n_points, int64_t n, const double *ra, const double *dec,
                         const double *t_ref, const double *phi_ref, const double *psi, const double *incl,
                         const double *dist, double *lnL, int32_t *shift_idx, cudaStream_t st)
{
    IleEvalArgs a;
    a.params = c->dparams;
    a.Q = c->dQ;
    a.U = c->dU;
    a.V = c->dV;
    a.point0 = point0;
    a.n_points = n_points;
    a.n_per_point = n;
    a.ra = ra, a.dec = dec, a.t_ref = t_ref, a.phi_ref = phi_ref, a.psi = psi, a.incl = incl, a.dist = dist;
    a.lnL = lnL;
    a.shift_idx = shift_idx;
    a.oob_counter = c->d_oob;
    a.exp_tab = c->ss.tabs;
    const bool use_stream = c->variant == 4 || (c->variant == 0 && c->stream_ok && n >= ILE_STREAM_MIN_SAMPLES);
    if (use_stream) {
        // launch groups of at most chunk_samples samples: whole points while they fit, else slices of one point
        const int64_t cs = c->chunk_samples;
        const int K = c->sz.n_det;
        auto shifted = [&](int64_t off, int32_t p0, int32_t np, int64_t cnt) {
            IleEvalArgs g = a;
            g.point0 = p0;
            g.n_points = np;
            g.n_per_point = cnt;
            g.ra = ra + off, g.dec = dec + off, g.t_ref = t_ref + off, g.phi_ref = phi_ref + off, g.psi = psi + off;
            g.incl = incl + off, g.dist = dist + off, g.lnL = lnL + off;
            g.shift_idx = shift_idx ? shift_idx + off * K : nullptr;
            return g;
        };
        if (n <= cs) {
            const int32_t per = (int32_t)(cs / n);
            for (int32_t p = 0; p < n_points; p += per) {
                const int32_t np = n_points - p < per ? n_points - p : per;
                const IleEvalArgs g = shifted((int64_t)p * n, point0 + p, np, n);
                int r = eval_stream_group(c, g, st);
                if (r != ILE_OK) return r;
            }
        } else {
            for (int32_t p = 0; p < n_points; ++p)
                for (int64_t off = 0; off < n; off += cs) {
                    const int64_t cnt = n - off < cs ? n - off : cs;
                    const IleEvalArgs g = shifted((int64_t)p * n + off, point0 + p, 1, cnt);
                    int r = eval_stream_group(c, g, st);
                    if (r != ILE_OK) return r;
                }
        }
        return ILE_OK;
    }
    int nl = 0;
    IleTiledLayout L;
    const bool tiled = !c->sz.interp && (c->variant == 2 || (c->variant == 0 && ile_tiled_plan(c->sz, (long long)n * n_points, &L)));
    cudaError_t e = tiled ? ile_launch_eval_tiled(c->sz, c->hparams, a, st, &nl) : ile_launch_eval_direct(c->sz, a, st, &nl);
    c->launches += nl;
    if (e != cudaSuccess) return cuda_fail(e);
    return ILE_OK;
}

extern "C" int ile_eval(ile_ctx *c, int32_t point, int64_t n, const double *ra, const double *dec, const double *t_ref,
                        const double *phi_ref, const double *psi, const double *incl, const double *dist_mpc,
                        double *lnL_margT, int32_t *shift_idx, void *cuda_stream)
{
    if (!c || n < 0 || point < 0 || point >= c->n_points) return ILE_ERR_BAD_ARGUMENT;
    if (n == 0) return ILE_OK;
    if (!ra || !dec || !t_ref || !phi_ref || !psi || !incl || !dist_mpc || !lnL_margT) return ILE_ERR_BAD_ARGUMENT;
    if (int r = check_device(c)) return r;
    return eval_dispatch(c, point, 1, n, ra, dec, t_ref, phi_ref, psi, incl, dist_mpc, lnL_margT, shift_idx,
                         (cudaStream_t)cuda_stream);
}

extern "C" int ile_eval_all(ile_ctx *c, int64_t n_per_point, const double *ra, const double *dec, const double *t_ref,
                            const double *phi_ref, const double *psi, const double *incl, const double *dist_mpc,
                            double *lnL_margT, int32_t *shift_idx, void *cuda_stream)
{
    if (!c || n_per_point < 0) return ILE_ERR_BAD_ARGUMENT;
    if (n_per_point == 0) return ILE_OK;
    if (!ra || !dec || !t_ref || !phi_ref || !psi || !incl || !dist_mpc || !lnL_margT) return ILE_ERR_BAD_ARGUMENT;
    if (int r = check_device(c)) return r;
    return eval_dispatch(c, 0, c->n_points, n_per_point, ra, dec, t_ref, phi_ref, psi, incl, dist_mpc, lnL_margT,
                         shift_idx, (cudaStream_t)cuda_stream);
}

static int ensure_evidence_scratch(ile_ctx *c, size_t doubles, size_t segments, cudaStream_t st)
{
    if (doubles > c->partials_cap || segments > c->tickets_cap) CK(cudaStreamSynchronize(st));  // an earlier call may still use them
    if (doubles > c->partials_cap) {
        cudaFree(c->d_partials);
        c->d_partials = nullptr;
        c->partials_cap = 0;
        CK(cudaMalloc(&c->d_partials, doubles * sizeof(double)));
        c->partials_cap = doubles;
    }
    if (segments > c->tickets_cap) {
        cudaFree(c->d_tickets);
        c->d_tickets = nullptr;
        c->tickets_cap = 0;
        const size_t cap = segments < 256 ? 256 : segments;
        CK(cudaMalloc(&c->d_tickets, cap * sizeof(unsigned int)));
        CK(cudaMemset(c->d_tickets, 0, cap * sizeof(unsigned int)));
        c->tickets_cap = cap;
    }
    return ILE_OK;
}

extern "C" int ile_evidence(ile_ctx *c, int32_t n_segments, int64_t n_per_segment, const double *lnL_margT,
                            const double *log_w, double *state, double *lnZ, double *n_eff, void *cuda_stream)
{
    if (!c || n_segments < 1 || n_per_segment < 0 || !lnZ) return ILE_ERR_BAD_ARGUMENT;
    if (n_per_segment > 0 && !lnL_margT) return ILE_ERR_BAD_ARGUMENT;
    if (n_segments > 65535) return ILE_ERR_UNSUPPORTED;  // segments are the y dimension of the grid
    int r = check_device(c);
    if (r != ILE_OK) return r;
    const int32_t B = ile_evidence_blocks_per_segment(n_segments, n_per_segment, c->sz.sm_count);
    // every segment has its own ticket word, zero between calls whatever layout the previous call used
    r = ensure_evidence_scratch(c, (size_t)n_segments * B * 2, (size_t)n_segments, (cudaStream_t)cuda_stream);
    if (r != ILE_OK) return r;
    int nl = 0;
    cudaError_t e = ile_launch_evidence(n_segments, n_per_segment, lnL_margT, log_w, state, lnZ, n_eff, c->d_partials,
                                        c->d_tickets, B, (cudaStream_t)cuda_stream, &nl);
    c->launches += nl;
    if (e != cudaSuccess) return cuda_fail(e);
    return ILE_OK;
}

static int precompute_any(int32_t n_points, int32_t n_det, int32_t n_modes, int32_t n_q, double fs_hz, double t0_q_s, const void *x,
                          const void *d, const double *S, double f_min_hz, double f_max_hz, double scale, void *Q, void *U, void *V,
                          void *cuda_stream)
{
    if (n_points < 1 || n_det < 1 || n_modes < 1 || n_q < 1 || !(fs_hz > 0.0) || !x || !d || !Q || !U || !V) return ILE_ERR_BAD_ARGUMENT;
    if (n_det > ILE_MAX_DET || n_modes > ILE_MAX_MODES || n_q < 2 || n_q > 65536 || (n_q & (n_q - 1))) return ILE_ERR_UNSUPPORTED;
    if (S && n_q < 512) return ILE_ERR_UNSUPPORTED;
    int dev = 0, optin = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return ILE_ERR_NO_DEVICE;
    CK(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    cudaError_t e = ile_launch_precompute(n_points, n_det, n_modes, n_q, fs_hz, t0_q_s, (const double2 *)x, (const double2 *)d, S, f_min_hz,
                                          f_max_hz, scale, (double2 *)Q, (double2 *)U, (double2 *)V, optin, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e);
    return ILE_OK;
}

extern "C" int ile_precompute(int32_t n_points, int32_t n_det, int32_t n_modes, int32_t n_q, double fs_hz, double t0_q_s,
                              const void *x, const void *d, void *Q, void *U, void *V, void *cuda_stream)
{
    return precompute_any(n_points, n_det, n_modes, n_q, fs_hz, t0_q_s, x, d, nullptr, 0.0, 0.0, 1.0, Q, U, V, cuda_stream);
}

extern "C" int ile_precompute_psd(int32_t n_points, int32_t n_det, int32_t n_modes, int32_t n_q, double fs_hz, double t0_q_s,
                                  const void *h, const void *d, const double *S, double f_min_hz, double f_max_hz, double scale, void *Q,
                                  void *U, void *V, void *cuda_stream)
{
    if (!S || !(f_max_hz > f_min_hz) || !(f_min_hz >= 0.0) || !std::isfinite(scale)) return ILE_ERR_BAD_ARGUMENT;
    return precompute_any(n_points, n_det, n_modes, n_q, fs_hz, t0_q_s, h, d, S, f_min_hz, f_max_hz, scale, Q, U, V, cuda_stream);
}

extern "C" int ile_evidence_merge(ile_ctx *c, int32_t n_segments, int32_t n_states, const double *states_in, double *state_out,
                                  double *lnZ, double *n_eff, void *cuda_stream)
{
    if (!c || n_segments < 1 || n_states < 1 || !states_in || !lnZ) return ILE_ERR_BAD_ARGUMENT;
    if (int r = check_device(c)) return r;
    int nl = 0;
    cudaError_t e = ile_launch_evidence_merge(n_segments, n_states, states_in, state_out, lnZ, n_eff, (cudaStream_t)cuda_stream, &nl);
    c->launches += nl;
    if (e != cudaSuccess) return cuda_fail(e);
    return ILE_OK;
}

extern "C" int ile_evidence_reset(ile_ctx *c, int32_t n_segments, double *state, void *cuda_stream)
{
    if (!c || n_segments < 1 || !state) return ILE_ERR_BAD_ARGUMENT;
    if (int r = check_device(c)) return r;
    int nl = 0;
    cudaError_t e = ile_launch_evidence_reset(n_segments, state, (cudaStream_t)cuda_stream, &nl);
    c->launches += nl;
    if (e != cudaSuccess) return cuda_fail(e);
    return ILE_OK;
}

// H2D of the sample arrays ([np][n] each), ile_eval / ile_eval_all, ile_evidence per point, D2H of the results.
static int run_host(ile_ctx *c, int32_t point0, int32_t np, int64_t n, const double *const src[8], double *lnL_margT, double *lnZ,
                    double *n_eff, cudaStream_t st)
{
    const size_t tot = (size_t)n * np;
    const size_t need = tot * 9;
    if (need > c->stage_cap) {
        CK(cudaStreamSynchronize(st));
        if (c->d_stage) CK(cudaFree(c->d_stage));
        c->d_stage = nullptr;
        c->stage_cap = 0;
        CK(cudaMalloc(&c->d_stage, need * sizeof(double)));
        c->stage_cap = need;
    }
    double *d = c->d_stage;
    // One point, streaming variant, one launch group, and enough samples for 2-4 efficient slices: pipeline the call (PAPER.md L97:
    // blocks "generated on the CPU and transferred to the board" -- the transfer of the next part hides behind the kernels of this one).
    const bool streaming = c->copy_stream && (c->variant == 4 || (c->variant == 0 && c->stream_ok));
    // slices: 2-4 while the batch is one launch group, else one per launch group (at most ILE_PIPE_MAX_SLICES: 1.6e7 samples)
    int64_t S = n / ILE_PIPE_MIN_SLICE < 4 ? n / ILE_PIPE_MIN_SLICE : 4;
    const int64_t groups = (n + c->chunk_samples - 1) / (c->chunk_samples > 0 ? c->chunk_samples : 1);
    if (S < groups) S = groups;
    const int64_t per = S > 0 ? (((n + S - 1) / S) + 1023) & ~(int64_t)1023 : 0;  // slice starts stay 8 KiB aligned
    if (np == 1 && streaming && S >= 2 && S <= ILE_PIPE_MAX_SLICES && per <= c->chunk_samples) {
        double *d_out = d + (size_t)8 * tot;
        CK(cudaEventRecord(c->ev_copy_go, st));  // the staging buffer is free once the caller's stream gets here
        CK(cudaStreamWaitEvent(c->copy_stream, c->ev_copy_go, 0));
        int n_sl = 0;
        for (int64_t lo = 0; lo < n; lo += per, ++n_sl) {  // every upload is queued up front, in the order the kernels want them
            const size_t cnt = (size_t)(n - lo < per ? n - lo : per);
            for (int i = 0; i < 8; ++i) {
                if (src[i]) CK(cudaMemcpyAsync(d + (size_t)i * tot + lo, src[i] + lo, cnt * sizeof(double), cudaMemcpyHostToDevice, c->copy_stream));
                if (i == 2) CK(cudaEventRecord(c->ev_pipe[3 * n_sl], c->copy_stream));  // ra, dec, t_ref: what the sort reads
            }
            CK(cudaEventRecord(c->ev_pipe[3 * n_sl + 1], c->copy_stream));
        }
        int nl = 0;
        cudaError_t e = ile_launch_evidence_reset(1, c->d_pipe_state, st, &nl);
        c->launches += nl;
        if (e != cudaSuccess) return cuda_fail(e);
        int sl = 0;
        for (int64_t lo = 0; lo < n; lo += per, ++sl) {
            const int64_t cnt = n - lo < per ? n - lo : per;
            CK(cudaStreamWaitEvent(st, c->ev_pipe[3 * sl], 0));
            c->ss.ev_late = c->ev_pipe[3 * sl + 1];  // the coefficient kernel (side stream) waits for the other five arrays
            int r = eval_dispatch(c, point0, 1, cnt, d + lo, d + tot + lo, d + 2 * tot + lo, d + 3 * tot + lo, d + 4 * tot + lo,
                                  d + 5 * tot + lo, d + 6 * tot + lo, d_out + lo, nullptr, st);
            c->ss.ev_late = nullptr;
            if (r != ILE_OK) return r;
            CK(cudaStreamWaitEvent(st, c->ev_pipe[3 * sl + 1], 0));  // log_w; a non-streaming slice (tiny tail) has not waited yet
            r = ile_evidence(c, 1, cnt, d_out + lo, src[7] ? d + 7 * tot + lo : nullptr, c->d_pipe_state, c->d_small, c->d_small + 1, st);
            if (r != ILE_OK) return r;
            if (lnL_margT) {
                CK(cudaEventRecord(c->ev_pipe[3 * sl + 2], st));
                CK(cudaStreamWaitEvent(c->d2h_stream, c->ev_pipe[3 * sl + 2], 0));
                CK(cudaMemcpyAsync(lnL_margT + lo, d_out + lo, (size_t)cnt * sizeof(double), cudaMemcpyDeviceToHost, c->d2h_stream));
            }
        }
        CK(cudaMemcpyAsync(c->h_small, c->d_small, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
        if (lnL_margT) {  // the downloads belong to the caller's stream order too
            CK(cudaEventRecord(c->ev_d2h_done, c->d2h_stream));
            CK(cudaStreamWaitEvent(st, c->ev_d2h_done, 0));
        }
        CK(cudaStreamSynchronize(st));
        lnZ[0] = c->h_small[0];
        if (n_eff) n_eff[0] = c->h_small[1];
        return ILE_OK;
    }
    // The sort needs ra, dec, t_ref only.  When the streaming variant will run as ONE launch group, the other arrays are
    // copied on a second queue and only the coefficient kernel (side stream) waits for them: their transfer overlaps the
    // index kernel, the scan and the scatter.
    const bool split = c->copy_stream && (c->variant == 4 || (c->variant == 0 && c->stream_ok && n >= ILE_STREAM_MIN_SAMPLES)) &&
                       (int64_t)tot <= c->chunk_samples;
    for (int i = 0; i < 3; ++i) CK(cudaMemcpyAsync(d + (size_t)i * tot, src[i], tot * sizeof(double), cudaMemcpyHostToDevice, st));
    cudaStream_t late = split ? c->copy_stream : st;
    if (split) {
        CK(cudaEventRecord(c->ev_copy_go, st));  // the staging buffer is free once the stream gets here
        CK(cudaStreamWaitEvent(late, c->ev_copy_go, 0));
    }
    for (int i = 3; i < 8; ++i)
        if (src[i]) CK(cudaMemcpyAsync(d + (size_t)i * tot, src[i], tot * sizeof(double), cudaMemcpyHostToDevice, late));
    if (split) CK(cudaEventRecord(c->ev_copy_done, late));
    double *d_out = d + (size_t)8 * tot;
    c->ss.ev_late = split ? c->ev_copy_done : nullptr;
    int r = eval_dispatch(c, point0, np, n, d, d + tot, d + 2 * tot, d + 3 * tot, d + 4 * tot, d + 5 * tot, d + 6 * tot, d_out, nullptr, st);
    c->ss.ev_late = nullptr;
    if (r != ILE_OK) return r;
    if (split) CK(cudaStreamWaitEvent(st, c->ev_copy_done, 0));  // log_w for the evidence (already implied by the join)
    r = ile_evidence(c, np, n, d_out, src[7] ? d + 7 * tot : nullptr, nullptr, c->d_small, c->d_small + np, st);
    if (r != ILE_OK) return r;
    if (lnL_margT) CK(cudaMemcpyAsync(lnL_margT, d_out, tot * sizeof(double), cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(c->h_small, c->d_small, 2 * (size_t)np * sizeof(double), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    for (int32_t p = 0; p < np; ++p) {
        lnZ[p] = c->h_small[p];
        if (n_eff) n_eff[p] = c->h_small[np + p];
    }
    return ILE_OK;
}

extern "C" int ile_run_host(ile_ctx *c, int32_t point, int64_t n, const double *ra, const double *dec,
                            const double *t_ref, const double *phi_ref, const double *psi, const double *incl,
                            const double *dist_mpc, const double *log_w, double *lnL_margT, double *lnZ, double *n_eff,
                            void *cuda_stream)
{
    if (!c || n < 1 || point < 0 || point >= c->n_points) return ILE_ERR_BAD_ARGUMENT;
    if (!ra || !dec || !t_ref || !phi_ref || !psi || !incl || !dist_mpc || !lnZ) return ILE_ERR_BAD_ARGUMENT;
    if (int r = check_device(c)) return r;
    const double *src[8] = {ra, dec, t_ref, phi_ref, psi, incl, dist_mpc, log_w};
    return run_host(c, point, 1, n, src, lnL_margT, lnZ, n_eff, (cudaStream_t)cuda_stream);
}

extern "C" int ile_run_host_all(ile_ctx *c, int64_t n_per_point, const double *ra, const double *dec, const double *t_ref,
                                const double *phi_ref, const double *psi, const double *incl, const double *dist_mpc,
                                const double *log_w, double *lnL_margT, double *lnZ, double *n_eff, void *cuda_stream)
{
    if (!c || n_per_point < 1) return ILE_ERR_BAD_ARGUMENT;
    if (!ra || !dec || !t_ref || !phi_ref || !psi || !incl || !dist_mpc || !lnZ) return ILE_ERR_BAD_ARGUMENT;
    if (int r = check_device(c)) return r;
    const double *src[8] = {ra, dec, t_ref, phi_ref, psi, incl, dist_mpc, log_w};
    return run_host(c, 0, c->n_points, n_per_point, src, lnL_margT, lnZ, n_eff, (cudaStream_t)cuda_stream);
}

extern "C" int ile_resample(ile_ctx *c, int64_t n, const double *lnL_margT, const double *log_w, int64_t n_out, double v0,
                            int64_t *ids_out, void *cuda_stream)
{
    if (!c || n < 0 || n_out < 0 || !(v0 >= 0.0) || !(v0 < 1.0)) return ILE_ERR_BAD_ARGUMENT;
    if (n_out == 0) return ILE_OK;
    if (n == 0 || !lnL_margT || !ids_out) return ILE_ERR_BAD_ARGUMENT;
    if (int r = check_device(c)) return r;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t need = ile_resample_scratch_doubles(n);
    if (need > c->resample_cap) {
        CK(cudaStreamSynchronize(st));
        cudaFree(c->d_resample);
        c->d_resample = nullptr, c->resample_cap = 0;
        CK(cudaMalloc(&c->d_resample, need * sizeof(double)));
        c->resample_cap = need;
    }
    int nl = 0;
    cudaError_t e = ile_launch_resample(c->sz, n, lnL_margT, log_w, n_out, v0, c->d_resample, reinterpret_cast<long long *>(ids_out), st, &nl);
    c->launches += nl;
    if (e != cudaSuccess) return cuda_fail(e);
    return ILE_OK;
}

extern "C" int ile_harvest(ile_ctx *c, int32_t point, int64_t n, const double *ra, const double *dec, const double *t_ref,
                           const double *phi_ref, const double *psi, const double *incl, const double *dist_mpc, int64_t n_sel,
                           const int64_t *ids, const double *v_uniform, int32_t *argmax_bin, double *lnL_max, int32_t *drawn_bin,
                           void *cuda_stream)
{
    if (!c || n < 0 || n_sel < 0 || point < 0 || point >= c->n_points) return ILE_ERR_BAD_ARGUMENT;
    if (n_sel == 0) return ILE_OK;
    if (!ra || !dec || !t_ref || !phi_ref || !psi || !incl || !dist_mpc || !argmax_bin || !lnL_max) return ILE_ERR_BAD_ARGUMENT;
    if (drawn_bin && !v_uniform) return ILE_ERR_BAD_ARGUMENT;
    if (!ids && n_sel > n) return ILE_ERR_BAD_ARGUMENT;
    if (int r = check_device(c)) return r;
    IleEvalArgs a;
    a.params = c->dparams;
    a.Q = c->dQ, a.U = c->dU, a.V = c->dV;
    a.point0 = point, a.n_points = 1, a.n_per_point = n;
    a.ra = ra, a.dec = dec, a.t_ref = t_ref, a.phi_ref = phi_ref, a.psi = psi, a.incl = incl, a.dist = dist_mpc;
    a.lnL = nullptr, a.shift_idx = nullptr, a.oob_counter = c->d_oob, a.exp_tab = c->ss.tabs;
    cudaError_t e = ile_launch_harvest(c->sz, a, n_sel, reinterpret_cast<const long long *>(ids), v_uniform, argmax_bin, lnL_max, drawn_bin,
                                       (cudaStream_t)cuda_stream);
    c->launches += 1;
    if (e != cudaSuccess) return cuda_fail(e);
    return ILE_OK;
}

extern "C" int ile_status(ile_ctx *c, int64_t *n_out_of_range, int reset, void *cuda_stream)
{
    if (!c) return ILE_ERR_BAD_ARGUMENT;
    if (int r = check_device(c)) return r;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    unsigned long long v = 0;
    CK(cudaMemcpyAsync(&v, c->d_oob, sizeof(v), cudaMemcpyDeviceToHost, st));
    if (reset) CK(cudaMemsetAsync(c->d_oob, 0, sizeof(v), st));
    CK(cudaStreamSynchronize(st));
    if (n_out_of_range) *n_out_of_range = (int64_t)v;
    return v ? ILE_ERR_OUT_OF_RANGE : ILE_OK;
}

extern "C" int ile_set_variant(ile_ctx *c, int32_t variant)
{
    if (!c || variant < 0) return ILE_ERR_BAD_ARGUMENT;
    if (variant > 4) return ILE_ERR_UNSUPPORTED;
    if (variant == 3) return ILE_ERR_UNSUPPORTED;  // retired (superseded by variant 4)
    if (variant == 4 && !c->stream_ok) return ILE_ERR_UNSUPPORTED;
    if (c->sz.interp && (variant == 2 || variant == 3)) return ILE_ERR_UNSUPPORTED;  // interpolated shifts: direct and streaming kernels
    if (variant == 2) {
        IleTiledLayout L;
        if (!ile_tiled_plan(c->sz, 1LL << 40, &L)) return ILE_ERR_UNSUPPORTED;
    }
    c->variant = variant;
    return ILE_OK;
}

extern "C" int64_t ile_launch_count(const ile_ctx *c) { return c ? (int64_t)c->launches : 0; }
int ile_ctx_sm_count(const ile_ctx *c) { return c->sz.sm_count; }
void ile_ctx_add_launches(ile_ctx *c, int n) { c->launches += n; }

static int measure_peak(int32_t iters, int dmma, double *tflops, double *ms)
{
    if (iters < 1 || !tflops) return ILE_ERR_BAD_ARGUMENT;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return ILE_ERR_NO_DEVICE;
    }
    int dev = 0;
    CK(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, dev));
    double *sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    float best = 1e30f;
    cudaError_t e = cudaMalloc(&sink, sizeof(double));
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {  // first repetition is the warm-up
        e = cudaEventRecord(e0, 0);
        if (e == cudaSuccess) e = ile_launch_fp64_peak(iters, prop.multiProcessorCount, sink, dmma, 0);
        if (e == cudaSuccess) e = cudaEventRecord(e1, 0);
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        float t = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&t, e0, e1);
        if (rep > 0 && t < best) best = t;
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(sink);
    if (e != cudaSuccess) return cuda_fail(e);
    // DFMA: 8 chains x 256 threads x 8 blocks per SM, 2 flops each; DMMA.8x8x4: 8 chains x 8 warps x 8 blocks, 512 flops each
    const double per_iter = dmma ? 8.0 * 8.0 * 8.0 * 512.0 : 8.0 * 256.0 * 8.0 * 2.0;
    *tflops = per_iter * (double)iters * prop.multiProcessorCount / (best * 1e-3) * 1e-12;
    if (ms) *ms = best;
    return ILE_OK;
}

extern "C" int ile_measure_fp64_peak(int32_t iters, double *tflops, double *ms) { return measure_peak(iters, 0, tflops, ms); }

extern "C" int ile_measure_dmma_peak(int32_t iters, double *tflops, double *ms) { return measure_peak(iters, 1, tflops, ms); }

extern "C" const char *ile_strerror(int code)
{
    switch (code) {
        case ILE_OK: return "ok";
        case ILE_ERR_BAD_ARGUMENT: return "bad argument";
        case ILE_ERR_CUDA: return g_cuda_msg;
        case ILE_ERR_NO_DEVICE: return "no CUDA device";
        case ILE_ERR_UNSUPPORTED: return "size or variant not supported by this build";
        case ILE_ERR_OUT_OF_RANGE: return "a sample's time window left the stored Q series";
        default: return "unknown error code";
    }
}
