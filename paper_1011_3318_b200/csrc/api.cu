// api.cu -- the extern "C" boundary declared in include/wcras.h: argument checks and marshalling only.
#include <new>

#include "wcras_internal.cuh"

using namespace wc;

#define NEED(cond, msg)                                                  \
    do {                                                                 \
        if (!(cond)) {                                                   \
            if (ctx) snprintf(ctx->err, sizeof ctx->err, "%s", msg);     \
            return WCRAS_INVALID_ARG;                                    \
        }                                                                \
    } while (0)

static int ensure_io(wcras_ctx* ctx) {
    if (!ctx->io_a) {
        const size_t bytes = sizeof(double) * 24 * (size_t)ctx->geom.V;
        if (alloc_dev(ctx, &ctx->io_a, bytes)) return WCRAS_CUDA_ERROR;
        if (alloc_dev(ctx, &ctx->io_b, bytes)) return WCRAS_CUDA_ERROR;
    }
    return WCRAS_OK;
}

extern "C" {

int wcras_create(wcras_ctx** out, const int dims[4], double kappa, double csw, const double* gauge_dev, void* cuda_stream) {
    if (!out || !dims || !gauge_dev) return WCRAS_INVALID_ARG;
    *out = nullptr;
    long long V = 1;
    for (int mu = 0; mu < 4; mu++) {
        if (dims[mu] < 2) return WCRAS_INVALID_ARG;
        V *= dims[mu];
    }
    if (V * 36 >= (1LL << 31)) return WCRAS_INVALID_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return WCRAS_CUDA_ERROR;
    wcras_ctx* ctx = new (std::nothrow) wcras_ctx();
    if (!ctx) return WCRAS_CUDA_ERROR;
    for (int mu = 0; mu < 4; mu++) ctx->geom.L[mu] = dims[mu];
    ctx->geom.V = (int)V;
    ctx->kappa = kappa;
    ctx->csw = csw;
    ctx->stream = (cudaStream_t)cuda_stream;
    *out = ctx;  // returned even on failure so that wcras_last_error can be read; destroy it afterwards
    return setup_fields(ctx, gauge_dev);
}

int wcras_destroy(wcras_ctx* ctx) {
    if (!ctx) return WCRAS_INVALID_ARG;
    cudaStreamSynchronize(ctx->stream);
    for (void* p : ctx->owned) cudaFree(p);
    if (ctx->mr_rho) { cudaFree(ctx->mr_rho); cudaFree(ctx->mr_q); cudaFree(ctx->mr_v); cudaFree(ctx->mr_scal); }
    if (ctx->dm) cudaFree(ctx->dm);
    if (ctx->hb) cudaFree(ctx->hb);
    if (ctx->sc_host) cudaFreeHost(ctx->sc_host);
    for (cudaEvent_t e : ctx->ev_pool) cudaEventDestroy(e);
    delete ctx;
    return WCRAS_OK;
}

int wcras_apply_D(wcras_ctx* ctx, int prec, const void* in_dev, void* out_dev) {
    NEED(ctx, "null ctx");
    NEED(in_dev && out_dev && in_dev != out_dev, "apply_D: null or aliased buffers");
    NEED(prec == 32 || prec == 64, "apply_D: prec must be 32 or 64");
    if (int rc = ensure_io(ctx)) return rc;
    if (int rc = to_internal(ctx, prec, in_dev, ctx->io_a)) return rc;
    int rc = prec == 32 ? dslash<float>(ctx, (const float4*)ctx->io_a, (float4*)ctx->io_b)
                        : dslash<double>(ctx, (const double2*)ctx->io_a, (double2*)ctx->io_b);
    if (rc) return rc;
    return from_internal(ctx, prec, ctx->io_b, out_dev);
}

int wcras_ras_precondition(wcras_ctx* ctx, const int domain[4], int overlap_s, int block_iters, int nras) {
    NEED(ctx, "null ctx");
    NEED(domain, "ras_precondition: null domain");
    return ras_configure(ctx, domain, overlap_s, block_iters, nras);
}

int wcras_set_ras_tier(wcras_ctx* ctx, int tier) {
    NEED(ctx, "null ctx");
    NEED(tier >= 0 && tier <= 4, "set_ras_tier: tier must be 0..4");
    ctx->tier_request = tier == 4 ? 2 : tier;
    ctx->chain_cycles = tier != 4;
    return WCRAS_OK;
}

int wcras_apply_D_restricted(wcras_ctx* ctx, int prec, int domain_index, const void* in_dev, void* out_dev) {
    NEED(ctx, "null ctx");
    NEED(in_dev && out_dev && in_dev != out_dev, "apply_D_restricted: null or aliased buffers");
    NEED(prec == 32 || prec == 64, "apply_D_restricted: prec must be 32 or 64");
    NEED(ctx->ras.set, "apply_D_restricted: call wcras_ras_precondition first");
    NEED(domain_index >= -1 && domain_index < ctx->ras.nd, "apply_D_restricted: domain index out of range");
    NEED(domain_index >= 0 || ctx->ras.s == 0, "apply_D_restricted: domain_index -1 needs overlap 0");
    int start[4], ext[4];
    int d = domain_index < 0 ? 0 : domain_index;
    for (int mu = 0; mu < 4; mu++) {
        const int L = ctx->geom.L[mu], bc = d % ctx->ras.nblk[mu];
        d /= ctx->ras.nblk[mu];
        const bool split = ctx->ras.b[mu] < L;
        start[mu] = ((bc * ctx->ras.b[mu] - (split ? ctx->ras.s : 0)) % L + L) % L;
        ext[mu] = ctx->ras.ext[mu];
    }
    if (int rc = ensure_io(ctx)) return rc;
    if (int rc = to_internal(ctx, prec, in_dev, ctx->io_a)) return rc;
    int rc = prec == 32 ? dslash_box<float>(ctx, start, ext, domain_index < 0, (const float4*)ctx->io_a, (float4*)ctx->io_b)
                        : dslash_box<double>(ctx, start, ext, domain_index < 0, (const double2*)ctx->io_a, (double2*)ctx->io_b);
    if (rc) return rc;
    return from_internal(ctx, prec, ctx->io_b, out_dev);
}

int wcras_ras_apply(wcras_ctx* ctx, const float* r_dev, float* v_dev) {
    NEED(ctx, "null ctx");
    NEED(r_dev && v_dev && r_dev != v_dev, "ras_apply: null or aliased buffers");
    NEED(ctx->ras.set, "ras_apply: call wcras_ras_precondition first");
    if (int rc = ensure_io(ctx)) return rc;
    if (int rc = to_internal(ctx, 32, r_dev, ctx->io_a)) return rc;
    if (int rc = ras_apply(ctx, (const float4*)ctx->io_a, (float4*)ctx->io_b)) return rc;
    return from_internal(ctx, 32, ctx->io_b, v_dev);
}

int wcras_set_solver(wcras_ctx* ctx, double inner_tol, int inner_maxit, int outer_maxit, int use_ras) {
    NEED(ctx, "null ctx");
    NEED(inner_tol > 0 && inner_maxit >= 1 && outer_maxit >= 1, "set_solver: tolerances and caps must be positive");
    ctx->inner_tol = inner_tol;
    ctx->inner_maxit = inner_maxit;
    ctx->outer_maxit = outer_maxit;
    ctx->use_ras = use_ras ? 1 : 0;
    return WCRAS_OK;
}

int wcras_set_timing(wcras_ctx* ctx, int enable) {
    NEED(ctx, "null ctx");
    ctx->timing = enable ? 1 : 0;
    return WCRAS_OK;
}

int wcras_solve(wcras_ctx* ctx, const double* eta_dev, double* phi_dev, double tol, wcras_info* info) {
    NEED(ctx, "null ctx");
    NEED(eta_dev && phi_dev && eta_dev != phi_dev, "solve: null or aliased buffers");
    NEED(tol > 0, "solve: tol must be positive");
    NEED(!ctx->use_ras || ctx->ras.set, "solve: use_ras is set but wcras_ras_precondition was not called");
    return solve(ctx, eta_dev, phi_dev, tol, info);
}

int wcras_solve_host(wcras_ctx* ctx, const double* eta_host, double* phi_host, double tol, wcras_info* info) {
    NEED(ctx, "null ctx");
    NEED(eta_host && phi_host, "solve_host: null buffers");
    NEED(tol > 0, "solve_host: tol must be positive");
    NEED(!ctx->use_ras || ctx->ras.set, "solve_host: use_ras is set but wcras_ras_precondition was not called");
    if (int rc = ensure_io(ctx)) return rc;
    const size_t bytes = sizeof(double) * 24 * (size_t)ctx->geom.V;
    WC_CUDA(cudaMemcpyAsync(ctx->io_a, eta_host, bytes, cudaMemcpyHostToDevice, ctx->stream));
    int rc = solve(ctx, (const double*)ctx->io_a, (double*)ctx->io_b, tol, info);
    if (rc != WCRAS_OK && rc != WCRAS_NOT_CONVERGED && rc != WCRAS_BREAKDOWN) return rc;
    WC_CUDA(cudaMemcpyAsync(phi_host, ctx->io_b, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    WC_CUDA(cudaStreamSynchronize(ctx->stream));
    return rc;
}

int wcras_export_clover(wcras_ctx* ctx, double* out_dev) {
    NEED(ctx, "null ctx");
    NEED(out_dev, "export_clover: null buffer");
    return export_clover(ctx, out_dev);
}

int wcras_time_kernel(wcras_ctx* ctx, int which, int reps, double* ms_per_launch) {
    NEED(ctx, "null ctx");
    NEED(ms_per_launch && reps >= 1 && which >= 0 && which <= 3, "time_kernel: bad arguments");
    if (int rc = ensure_workspace(ctx)) return rc;
    if (which == 3) return time_blas(ctx, reps, ms_per_launch);
    NEED(which != 2 || ctx->ras.set, "time_kernel: call wcras_ras_precondition first");
    const size_t V = ctx->geom.V;
    // deterministic non-trivial scratch input: reuse the fp32 link array bytes as a spinor-sized pattern
    WC_CUDA(cudaMemcpyAsync(ctx->w32[0], ctx->g32a, sizeof(float4) * 6 * V, cudaMemcpyDeviceToDevice, ctx->stream));
    WC_CUDA(cudaMemcpyAsync(ctx->w64[0], ctx->g64, sizeof(double2) * 12 * V, cudaMemcpyDeviceToDevice, ctx->stream));
    cudaEvent_t e0, e1;
    WC_CUDA(cudaEventCreate(&e0));
    WC_CUDA(cudaEventCreate(&e1));
    int rc = WCRAS_OK;
    for (int pass = 0; pass < 2 && !rc; pass++) {  // pass 0 = warm-up
        const int n = pass == 0 ? 3 : reps;
        WC_CUDA(cudaEventRecord(e0, ctx->stream));
        for (int k = 0; k < n && !rc; k++) {
            if (which == 0) rc = dslash<float>(ctx, ctx->w32[0], ctx->w32[1]);
            else if (which == 1) rc = dslash<double>(ctx, ctx->w64[0], ctx->w64[1]);
            else rc = ras_block_solve(ctx, ctx->w32[0], ctx->w32[1]);
        }
        WC_CUDA(cudaEventRecord(e1, ctx->stream));
        WC_CUDA(cudaStreamSynchronize(ctx->stream));
    }
    float t = 0;
    WC_CUDA(cudaEventElapsedTime(&t, e0, e1));
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *ms_per_launch = t / reps;
    return rc;
}

long long wcras_launch_count(const wcras_ctx* ctx) { return ctx ? ctx->launches : 0; }

const char* wcras_last_error(const wcras_ctx* ctx) { return ctx ? ctx->err : "null ctx"; }

}  // extern "C"
