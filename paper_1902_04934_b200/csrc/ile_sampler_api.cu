// ile_sampler_api.cu -- C ABI of the on-device Monte Carlo sampler and of the adaptive integration loop (include/ile.h,
// "NEXT-2"): argument checking, buffers, kernel dispatch.  The loop itself only strings public entries together:
// ile_sampler_draw -> ile_eval -> ile_evidence (carried state) -> ile_sampler_refit, with no host round trip of samples.
#include <cmath>
#include <cstring>
#include <new>

#include "ile_kernels.h"

struct ile_sampler {
    int device, sm_count;
    IleSamplerParams P;
    double *d_tab;        // h [3][nb] | C [3][nb + 1]
    unsigned long long *d_work;  // refit scratch: 64-bit histograms, maximum key, ticket (every refit leaves it clean)
    // scratch of ile_integrate (grown on demand): seven sample arrays, ln w, lnL ([9][cap] doubles), bins [cap][3]
    double *d_buf;
    int32_t *d_bins;
    int64_t cap;
    double *d_state;      // evidence state [3] + (lnZ, n_eff) per chunk slot [2][2]
    double *d_multi;      // frozen-density phase: per-chunk states [B][3], scratch lnZ / n_eff [2 B], history [B][2]
    int64_t multi_cap;    // B
    double *h_hist;       // pinned [max_chunks][2]
    int64_t hist_cap;
    cudaEvent_t ev[2];
    long long launches;
};

#define CK(call)                                           \
    do {                                                   \
        cudaError_t e__ = (call);                          \
        if (e__ != cudaSuccess) return ile_cuda_fail(e__); \
    } while (0)

static int smp_check_device(const ile_sampler *s)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return ILE_ERR_NO_DEVICE;
    return dev == s->device ? ILE_OK : ILE_ERR_BAD_ARGUMENT;
}

extern "C" int ile_sampler_create(ile_sampler **out, const ile_sampler_config *cfg)
{
    if (!out || !cfg) return ILE_ERR_BAD_ARGUMENT;
    *out = nullptr;
    if (cfg->n_bins < 1 || !(cfg->floor_frac >= 0.0) || !(cfg->floor_frac <= 1.0) || !(cfg->temper > 0.0)) return ILE_ERR_BAD_ARGUMENT;
    if (!(cfg->dist_min_mpc > 0.0) || !(cfg->dist_max_mpc > cfg->dist_min_mpc) || !(cfg->t_ref_hi_s >= cfg->t_ref_lo_s))
        return ILE_ERR_BAD_ARGUMENT;
    if (!std::isfinite(cfg->t_ref_lo_s) || !std::isfinite(cfg->t_ref_hi_s) || !std::isfinite(cfg->dist_max_mpc)) return ILE_ERR_BAD_ARGUMENT;
    if (cfg->n_bins > ILE_SAMPLER_MAX_BINS) return ILE_ERR_UNSUPPORTED;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return ILE_ERR_NO_DEVICE;
    }
    int device = 0, sms = 0;
    CK(cudaGetDevice(&device));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device));
    ile_sampler *s = new (std::nothrow) ile_sampler();
    if (!s) return ILE_ERR_BAD_ARGUMENT;
    std::memset(s, 0, sizeof(*s));
    s->device = device;
    s->sm_count = sms;
    IleSamplerParams &P = s->P;
    P.seed = cfg->seed;
    P.n_bins = cfg->n_bins;
    P.adapt[0] = cfg->adapt_ra != 0, P.adapt[1] = cfg->adapt_dec != 0, P.adapt[2] = cfg->adapt_dist != 0;
    P.floor_frac = cfg->floor_frac;
    P.temper = cfg->temper;
    P.t_lo = cfg->t_ref_lo_s;
    P.t_span = cfg->t_ref_hi_s - cfg->t_ref_lo_s;
    P.dmin3 = cfg->dist_min_mpc * cfg->dist_min_mpc * cfg->dist_min_mpc;
    P.d3_span = cfg->dist_max_mpc * cfg->dist_max_mpc * cfg->dist_max_mpc - P.dmin3;
    cudaError_t e = cudaMalloc(&s->d_tab, ile_sampler_table_doubles(P.n_bins) * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&s->d_state, 8 * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&s->d_work, ile_sampler_work_words(P.n_bins) * sizeof(unsigned long long));
    if (e == cudaSuccess) e = ile_sampler_work_init(P, s->d_work, 0);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->ev[0], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->ev[1], cudaEventDisableTiming);
    if (e == cudaSuccess) e = ile_launch_sampler_tables(P, s->d_tab, 1, 0);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e != cudaSuccess) {
        ile_sampler_destroy(s);
        return ile_cuda_fail(e);
    }
    s->launches = 1;
    *out = s;
    return ILE_OK;
}

extern "C" void ile_sampler_destroy(ile_sampler *s)
{
    if (!s) return;
    cudaFree(s->d_tab);
    cudaFree(s->d_work);
    cudaFree(s->d_buf);
    cudaFree(s->d_bins);
    cudaFree(s->d_state);
    cudaFree(s->d_multi);
    if (s->h_hist) cudaFreeHost(s->h_hist);
    if (s->ev[0]) cudaEventDestroy(s->ev[0]);
    if (s->ev[1]) cudaEventDestroy(s->ev[1]);
    delete s;
}

extern "C" int ile_sampler_reset(ile_sampler *s, void *cuda_stream)
{
    if (!s) return ILE_ERR_BAD_ARGUMENT;
    if (int r = smp_check_device(s)) return r;
    CK(ile_launch_sampler_tables(s->P, s->d_tab, 1, (cudaStream_t)cuda_stream));
    s->launches += 1;
    return ILE_OK;
}

extern "C" int ile_sampler_set_tables(ile_sampler *s, const double *h, void *cuda_stream)
{
    if (!s || !h) return ILE_ERR_BAD_ARGUMENT;
    if (int r = smp_check_device(s)) return r;
    for (int i = 0; i < 3 * s->P.n_bins; ++i)
        if (!(h[i] >= 0.0) || !std::isfinite(h[i])) return ILE_ERR_BAD_ARGUMENT;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CK(cudaMemcpyAsync(s->d_tab, h, (size_t)3 * s->P.n_bins * sizeof(double), cudaMemcpyHostToDevice, st));
    CK(ile_launch_sampler_tables(s->P, s->d_tab, 0, st));
    CK(cudaStreamSynchronize(st));  // h may be pageable and reused by the caller
    s->launches += 1;
    return ILE_OK;
}

extern "C" int ile_sampler_get_tables(ile_sampler *s, double *h, double *C, void *cuda_stream)
{
    if (!s || !h) return ILE_ERR_BAD_ARGUMENT;
    if (int r = smp_check_device(s)) return r;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int nb = s->P.n_bins;
    CK(cudaMemcpyAsync(h, s->d_tab, (size_t)3 * nb * sizeof(double), cudaMemcpyDeviceToHost, st));
    if (C) CK(cudaMemcpyAsync(C, s->d_tab + 3 * nb, (size_t)3 * (nb + 1) * sizeof(double), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return ILE_OK;
}

extern "C" int ile_sampler_uniforms(ile_sampler *s, int64_t first_index, int64_t n, double *u, void *cuda_stream)
{
    if (!s || n < 0 || first_index < 0 || (n > 0 && !u)) return ILE_ERR_BAD_ARGUMENT;
    if (int r = smp_check_device(s)) return r;
    CK(ile_launch_sampler_uniforms(s->P, s->sm_count, first_index, n, u, (cudaStream_t)cuda_stream));
    s->launches += n > 0;
    return ILE_OK;
}

extern "C" int ile_sampler_draw(ile_sampler *s, int64_t first_index, int64_t n, double *ra, double *dec, double *t_ref, double *phi_ref,
                                double *psi, double *incl, double *dist_mpc, double *log_w, int32_t *bin_idx, void *cuda_stream)
{
    if (!s || n < 0 || first_index < 0) return ILE_ERR_BAD_ARGUMENT;
    if (n == 0) return ILE_OK;
    if (!ra || !dec || !t_ref || !phi_ref || !psi || !incl || !dist_mpc) return ILE_ERR_BAD_ARGUMENT;
    if (int r = smp_check_device(s)) return r;
    CK(ile_launch_sampler_draw(s->P, s->sm_count, s->d_tab, first_index, n, ra, dec, t_ref, phi_ref, psi, incl, dist_mpc, log_w, bin_idx,
                               (cudaStream_t)cuda_stream));
    s->launches += 1;
    return ILE_OK;
}

extern "C" int ile_sampler_refit(ile_sampler *s, int64_t n, const int32_t *bin_idx, const double *lnL_margT, const double *log_w,
                                 void *cuda_stream)
{
    if (!s || n < 0) return ILE_ERR_BAD_ARGUMENT;
    if (n == 0) return ILE_OK;
    if (!bin_idx || !lnL_margT) return ILE_ERR_BAD_ARGUMENT;
    if (int r = smp_check_device(s)) return r;
    CK(ile_launch_sampler_refit(s->P, s->sm_count, s->d_tab, n, bin_idx, lnL_margT, log_w, s->d_work, (cudaStream_t)cuda_stream));
    s->launches += 2;
    return ILE_OK;
}

extern "C" int64_t ile_sampler_launch_count(const ile_sampler *s) { return s ? (int64_t)s->launches : 0; }

// ------------------------------------------------------------------------------------------------------------
// the adaptive Monte Carlo loop (S7-S8) with every array resident on the device
// ------------------------------------------------------------------------------------------------------------
static int smp_ensure(ile_sampler *s, int64_t n_samples, int32_t max_chunks, int64_t multi, cudaStream_t st)
{
    if (n_samples > s->cap) {
        CK(cudaStreamSynchronize(st));
        cudaFree(s->d_buf), cudaFree(s->d_bins);
        s->d_buf = nullptr, s->d_bins = nullptr, s->cap = 0;
        CK(cudaMalloc(&s->d_buf, (size_t)9 * n_samples * sizeof(double)));
        CK(cudaMalloc(&s->d_bins, (size_t)3 * n_samples * sizeof(int32_t)));
        s->cap = n_samples;
    }
    if (max_chunks > s->hist_cap) {
        CK(cudaStreamSynchronize(st));
        if (s->h_hist) cudaFreeHost(s->h_hist);
        s->h_hist = nullptr, s->hist_cap = 0;
        CK(cudaMallocHost(&s->h_hist, (size_t)2 * max_chunks * sizeof(double)));
        s->hist_cap = max_chunks;
    }
    if (multi > s->multi_cap) {
        CK(cudaStreamSynchronize(st));
        cudaFree(s->d_multi);
        s->d_multi = nullptr, s->multi_cap = 0;
        CK(cudaMalloc(&s->d_multi, (size_t)7 * multi * sizeof(double)));
        s->multi_cap = multi;
    }
    return ILE_OK;
}

extern "C" int ile_integrate(ile_ctx *ctx, ile_sampler *s, int32_t point, int64_t n_chunk, int32_t max_chunks, int32_t n_adapt_chunks,
                             double n_eff_min, double *lnZ, double *n_eff, int64_t *n_samples, double *history, void *cuda_stream)
{
    if (!ctx || !s || n_chunk < 1 || max_chunks < 1 || n_adapt_chunks < 0 || !lnZ) return ILE_ERR_BAD_ARGUMENT;
    if (int r = smp_check_device(s)) return r;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // Once the densities are frozen (c >= n_adapt_chunks) chunks no longer depend on one another: they are drawn and evaluated
    // `multi` at a time (about 2^20 samples per ile_eval) and only the evidence is still accumulated chunk by chunk.
    const int32_t frozen = max_chunks > n_adapt_chunks ? max_chunks - n_adapt_chunks : 0;
    int64_t multi = frozen ? ((int64_t)1 << 20) / n_chunk : 0;
    multi = multi < 1 ? (frozen ? 1 : 0) : multi > frozen ? frozen : multi;
    if (multi > 4096) multi = 4096;  // chunks of a batch are segments of one ile_evidence launch (grid.y) and steps of a one-thread prefix
    int r = smp_ensure(s, n_chunk * (multi > 1 ? multi : 1), max_chunks, multi, st);
    if (r != ILE_OK) return r;
    r = ile_sampler_reset(s, cuda_stream);  // S9: the first chunk is drawn from the prior
    if (r != ILE_OK) return r;
    double *b = s->d_buf;
    const int64_t n = n_chunk;
    double *ra = b, *dec = b + n, *t_ref = b + 2 * n, *phi = b + 3 * n, *psi = b + 4 * n, *incl = b + 5 * n, *dist = b + 6 * n;
    double *log_w = b + 7 * n, *lnL = b + 8 * n;
    double *state = s->d_state, *res = s->d_state + 4;  // res: [slot][lnZ, n_eff]
    r = ile_evidence_reset(ctx, 1, state, cuda_stream);
    if (r != ILE_OK) return r;
    // Chunk c's evidence is read back asynchronously; the host looks at it only after chunk c + 1 has been drawn, evaluated
    // and accumulated, so the GPU never idles on the stopping rule.  A chunk that turns out to lie beyond the stop is never
    // refit from and its numbers are never reported: results, densities and sample count are those of the strict rule S8.
    int32_t stop = -1, done = 0;
    const int32_t n_seq = multi > 1 ? (n_adapt_chunks < max_chunks ? n_adapt_chunks : max_chunks) : max_chunks;  // chunks taken one by one
    for (int32_t c = 0; c < n_seq && stop < 0; ++c) {
        r = ile_sampler_draw(s, (int64_t)c * n, n, ra, dec, t_ref, phi, psi, incl, dist, log_w, s->d_bins, cuda_stream);
        if (r == ILE_OK) r = ile_eval(ctx, point, n, ra, dec, t_ref, phi, psi, incl, dist, lnL, nullptr, cuda_stream);
        if (r == ILE_OK) r = ile_evidence(ctx, 1, n, lnL, log_w, state, res + 2 * (c & 1), res + 2 * (c & 1) + 1, cuda_stream);
        if (r != ILE_OK) return r;
        CK(cudaMemcpyAsync(s->h_hist + 2 * (size_t)c, res + 2 * (c & 1), 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
        CK(cudaEventRecord(s->ev[c & 1], st));
        done = c + 1;
        if (c >= 1) {
            CK(cudaEventSynchronize(s->ev[(c - 1) & 1]));
            if (s->h_hist[2 * (size_t)(c - 1) + 1] >= n_eff_min) stop = c - 1;
        }
        if (stop < 0 && c < n_adapt_chunks) {
            r = ile_sampler_refit(s, n, s->d_bins, lnL, log_w, cuda_stream);
            if (r != ILE_OK) return r;
        }
    }
    if (stop < 0 && done > 0 && done < max_chunks) {  // the last adaptive chunk decides whether the frozen phase starts at all
        CK(cudaEventSynchronize(s->ev[(done - 1) & 1]));
        if (s->h_hist[2 * (size_t)(done - 1) + 1] >= n_eff_min) stop = done - 1;
    }
    // ---- frozen densities: `cnt` chunks per draw / ile_eval, evidence per chunk (segmented reduction, then a running merge)
    while (stop < 0 && done < max_chunks) {
        const int32_t cnt = (int32_t)(max_chunks - done < multi ? max_chunks - done : multi);
        const int64_t tot = (int64_t)cnt * n;
        double *ra2 = b, *dec2 = b + tot, *t2 = b + 2 * tot, *phi2 = b + 3 * tot, *psi2 = b + 4 * tot, *incl2 = b + 5 * tot, *dist2 = b + 6 * tot;
        double *lw2 = b + 7 * tot, *lnL2 = b + 8 * tot;
        double *cst = s->d_multi, *ctmp = cst + 3 * (size_t)multi, *chist = ctmp + 2 * (size_t)multi;
        r = ile_sampler_draw(s, (int64_t)done * n, tot, ra2, dec2, t2, phi2, psi2, incl2, dist2, lw2, nullptr, cuda_stream);
        if (r == ILE_OK) r = ile_eval(ctx, point, tot, ra2, dec2, t2, phi2, psi2, incl2, dist2, lnL2, nullptr, cuda_stream);
        if (r == ILE_OK) r = ile_evidence_reset(ctx, cnt, cst, cuda_stream);
        if (r == ILE_OK) r = ile_evidence(ctx, cnt, n, lnL2, lw2, cst, ctmp, ctmp + cnt, cuda_stream);
        if (r != ILE_OK) return r;
        CK(ile_launch_evidence_prefix(cnt, cst, state, chist, st));
        ile_ctx_add_launches(ctx, 1);
        CK(cudaMemcpyAsync(s->h_hist + 2 * (size_t)done, chist, 2 * (size_t)cnt * sizeof(double), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        for (int32_t c = 0; c < cnt && stop < 0; ++c)
            if (s->h_hist[2 * (size_t)(done + c) + 1] >= n_eff_min) stop = done + c;
        done += cnt;
    }
    CK(cudaStreamSynchronize(st));
    if (stop < 0) stop = done - 1;  // the last chunk: threshold reached there, or max_chunks exhausted
    *lnZ = s->h_hist[2 * (size_t)stop];
    if (n_eff) *n_eff = s->h_hist[2 * (size_t)stop + 1];
    if (n_samples) *n_samples = (int64_t)(stop + 1) * n;
    if (history)
        for (int32_t c = 0; c <= stop; ++c) history[2 * c] = s->h_hist[2 * (size_t)c], history[2 * c + 1] = s->h_hist[2 * (size_t)c + 1];
    return ILE_OK;
}
