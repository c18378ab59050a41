// noalloc.cu -- wcras_apply_D_noalloc: w = D v (step A1, BASELINE.json:north_star) for callers that may
// not allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// wcras_apply_D converts the canonical spinor to the internal SoA layout, applies the Dslash and converts back; its two
// internal-layout buffers are cudaMalloc'ed on the first call (api.cu: ensure_io).  Here the same three kernels run with
// those two buffers carved out of ONE file-scope device array of WCRAS_NOALLOC_SCRATCH_BYTES (16 MiB), which every GPU that
// loads the library holds until the process exits.  Nothing in this entry point calls cudaMalloc, cudaFree, an event or
// stream creation or any other allocating routine.
//
//   * In host code the array's name is a host-side stand-in, not a device address: its device address is obtained once per
//     device, with that device current, by cudaGetSymbolAddress below, and that pointer is what the kernels get.
//   * Every call (of every context, on every stream) of one device shares the array.  It keeps the last call's contents;
//     nothing has to start at zero (both buffers are written in full before they are read: to_internal writes all
//     12 V complex numbers, the Dslash all 12 V of its output), so nothing is cleared.  Calls that overlap on the GPU
//     (two streams, two host threads) race on it: the caller serialises them.
#include <mutex>

#include "wcras_internal.cuh"

using namespace wc;

static __device__ __align__(256) unsigned char g_noalloc_scratch[WCRAS_NOALLOC_SCRATCH_BYTES];

namespace {
constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
void* g_scratch_addr[MAX_DEVICES] = {};  // device address of g_noalloc_scratch on device d (nullptr: not asked yet)

// set-up, once per device, with that device current (it is: the library launches on the current device)
int scratch_address(wcras_ctx* ctx, unsigned char** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) {
        snprintf(ctx->err, sizeof ctx->err, "apply_D_noalloc: cudaGetDevice: %s", e != cudaSuccess ? cudaGetErrorString(e) : "device index out of range");
        return WCRAS_CUDA_ERROR;
    }
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) {
            snprintf(ctx->err, sizeof ctx->err, "apply_D_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
            return WCRAS_CUDA_ERROR;
        }
        g_scratch_addr[dev] = p;
    }
    *out = static_cast<unsigned char*>(g_scratch_addr[dev]);
    return WCRAS_OK;
}
}  // namespace

extern "C" int wcras_apply_D_noalloc(wcras_ctx* ctx, int prec, const void* in_dev, void* out_dev) {
    if (!ctx) return WCRAS_INVALID_ARG;
    if (!in_dev || !out_dev || in_dev == out_dev) {
        snprintf(ctx->err, sizeof ctx->err, "apply_D_noalloc: null or aliased buffers");
        return WCRAS_INVALID_ARG;
    }
    if (prec != 32 && prec != 64) {
        snprintf(ctx->err, sizeof ctx->err, "apply_D_noalloc: prec must be 32 or 64");
        return WCRAS_INVALID_ARG;
    }
    // two internal-layout spinors of 24 reals per site, each rounded up to the array's 256-byte alignment
    const size_t each = ((size_t)ctx->geom.V * 24 * (prec == 32 ? sizeof(float) : sizeof(double)) + 255) / 256 * 256;
    if (2 * each > (size_t)WCRAS_NOALLOC_SCRATCH_BYTES) {
        snprintf(ctx->err, sizeof ctx->err,
                 "apply_D_noalloc: %d sites at %d bits need %zu bytes of scratch, the static array holds %zu (at most %zu sites); use "
                 "wcras_apply_D",
                 ctx->geom.V, prec, 2 * each, (size_t)WCRAS_NOALLOC_SCRATCH_BYTES,
                 (size_t)WCRAS_NOALLOC_SCRATCH_BYTES / (2 * 24 * (prec == 32 ? sizeof(float) : sizeof(double))));
        return WCRAS_UNSUPPORTED;
    }
    unsigned char* base = nullptr;
    if (int rc = scratch_address(ctx, &base)) return rc;
    void* a = base;
    void* b = base + each;
    // the per-class event timers (wcras_set_timing) create events on demand: off for this call
    struct TimingOff {
        wcras_ctx* c;
        int saved;
        explicit TimingOff(wcras_ctx* cc) : c(cc), saved(cc->timing) { c->timing = 0; }
        ~TimingOff() { c->timing = saved; }
    } timing_off(ctx);
    if (int rc = to_internal(ctx, prec, in_dev, a)) return rc;
    const int rc = prec == 32 ? dslash<float>(ctx, (const float4*)a, (float4*)b) : dslash<double>(ctx, (const double2*)a, (double2*)b);
    if (rc) return rc;
    return from_internal(ctx, prec, b, out_dev);
}
