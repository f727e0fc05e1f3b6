// ile_evidence_static.cu -- ile_evidence_static(): the evidence reduction (step 7 of SURVEY.md 8(a); eq. 4,
// n_eff L101) for callers that must not, or cannot, allocate device memory.
//
// Who that is.  ile_evidence() works out of an ile_ctx, and a context is made of cudaMalloc calls (ile_create, and again
// whenever its scratch has to grow).  Some users of this library cannot afford that:
//   * code that runs inside a memory pool someone else owns (a PyTorch caching allocator, an RMM pool, a job that was
//     handed a fixed slab of HBM): a stray cudaMalloc bypasses the pool, can fail although the pool has room, and
//     synchronises the whole device when it succeeds;
//   * latency-critical loops and plug-ins loaded into a host application whose rules forbid driver allocations after start-up;
//   * a worker that only wants to fold per-sample lnL_margT values it already holds into lnZ and never builds a context.
// For them the block partials and ticket words the evidence kernel needs live in ONE fixed array in the library's own
// device image (below), so the call itself asks the driver for nothing.
//
// What that costs.  The array is part of the loaded module: every GPU that loads libile_b200.so keeps
// ILE_EVIDENCE_STATIC_SCRATCH_BYTES (68 KiB) until the process exits, used or not.  It is ONE array per device, shared by every call and
// every thread: two calls whose kernels can overlap on the GPU (different streams without an event between them) race on
// it.  Sizes are bounded (ILE_EVIDENCE_STATIC_MAX_SEGMENTS).  The existing ile_evidence() path is untouched and keeps
// its per-context, growable scratch.
#include <cuda_runtime.h>

#include <mutex>

#include "../../include/ile.h"
#include "ile_kernels.h"

// Layout: [0, 4 KiB) one ticket word per segment, then ILE_EVS_PARTIAL_PAIRS (max, sum) pairs of doubles shared out over the
// segments of a call.  Zero-initialised when the module is loaded; the ticket words are cleared again by every call.
#define ILE_EVS_TICKET_BYTES (ILE_EVIDENCE_STATIC_MAX_SEGMENTS * 4)
#define ILE_EVS_PARTIAL_PAIRS 4096
#define ILE_EVS_BYTES (ILE_EVS_TICKET_BYTES + ILE_EVS_PARTIAL_PAIRS * 16)
static_assert(ILE_EVS_BYTES == ILE_EVIDENCE_STATIC_SCRATCH_BYTES, "ile.h states the size of the static scratch");
static_assert(ILE_EVS_TICKET_BYTES % 256 == 0, "the partials keep the array's alignment");

static __device__ __align__(256) unsigned char g_evidence_static_scratch[ILE_EVS_BYTES];

// In host code the name g_evidence_static_scratch is only a handle for the runtime, NOT a device address: a kernel must
// be given what cudaGetSymbolAddress returns for it on the device that is current.  That is looked up once per device.
#define ILE_EVS_MAX_DEVICES 64
struct EvsDevice {
    bool ready;
    unsigned char *base;  // device address of g_evidence_static_scratch on this device
    int sm_count;
};
static EvsDevice g_evs_dev[ILE_EVS_MAX_DEVICES];
static std::mutex g_evs_mutex;

// First call on a device (with that device current): resolve the array's device address and read the SM count.
static int evs_setup(int dev, EvsDevice *out)
{
    std::lock_guard<std::mutex> lock(g_evs_mutex);
    EvsDevice &d = g_evs_dev[dev];
    if (!d.ready) {
        void *p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_evidence_static_scratch);
        if (e != cudaSuccess) return ile_cuda_fail(e);
        if (!p) return ile_cuda_fail(cudaErrorInvalidSymbol);
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return ile_cuda_fail(e);
        d.base = static_cast<unsigned char *>(p);
        d.sm_count = sms;
        d.ready = true;
    }
    *out = d;
    return ILE_OK;
}

extern "C" int ile_evidence_static(int32_t n_segments, int64_t n_per_segment, const double *lnL_margT, const double *log_w,
                                   double *state, double *lnZ, double *n_eff, void *cuda_stream)
{
    if (n_segments < 1 || n_per_segment < 0 || !lnZ) return ILE_ERR_BAD_ARGUMENT;
    if (n_per_segment > 0 && !lnL_margT) return ILE_ERR_BAD_ARGUMENT;
    if (n_segments > ILE_EVIDENCE_STATIC_MAX_SEGMENTS) return ILE_ERR_UNSUPPORTED;  // the fixed array has one ticket word per segment
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return ILE_ERR_NO_DEVICE;
    if (dev < 0 || dev >= ILE_EVS_MAX_DEVICES) return ILE_ERR_UNSUPPORTED;
    EvsDevice d;
    if (int r = evs_setup(dev, &d)) return r;

    cudaStream_t st = (cudaStream_t)cuda_stream;
    unsigned int *tickets = reinterpret_cast<unsigned int *>(d.base);
    double *partials = reinterpret_cast<double *>(d.base + ILE_EVS_TICKET_BYTES);
    // blocks per segment: what ile_evidence would take, cut down to the pairs the fixed array holds (>= 4 per segment)
    int32_t B = ile_evidence_blocks_per_segment(n_segments, n_per_segment, d.sm_count);
    const int32_t fit = ILE_EVS_PARTIAL_PAIRS / n_segments;
    if (B > fit) B = fit;
    // The tickets count the finished blocks of a segment and have to start at zero.  A completed call leaves them zero,
    // a call that died half-way (or raced with another) does not, and the array outlives both: clear them every time.
    // cudaMemsetAsync is stream-ordered and allocates nothing.  The partials need no clearing (written before they are read).
    cudaError_t e = cudaMemsetAsync(tickets, 0, (size_t)n_segments * sizeof(unsigned int), st);
    if (e != cudaSuccess) return ile_cuda_fail(e);
    e = ile_launch_evidence(n_segments, n_per_segment, lnL_margT, log_w, state, lnZ, n_eff, partials, tickets, B, st, nullptr);
    if (e != cudaSuccess) return ile_cuda_fail(e);
    return ILE_OK;
}
