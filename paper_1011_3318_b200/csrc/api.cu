// api.cu -- the extern "C" boundary declared in include/wcras.h: argument checks and marshalling only.
#include <new>

#include <algorithm>
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
    drop_iter_graphs(ctx);
    if (ctx->cap_stream) cudaStreamDestroy(ctx->cap_stream);
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    if (ctx->ev_copy_ready) cudaEventDestroy(ctx->ev_copy_ready);
    if (ctx->ev_copy_done) cudaEventDestroy(ctx->ev_copy_done);
    for (void* p : ctx->owned) cudaFree(p);
    if (ctx->mr_rho) { cudaFree(ctx->mr_rho); cudaFree(ctx->mr_q); cudaFree(ctx->mr_v); cudaFree(ctx->mr_scal); }
    if (ctx->mr_q2) cudaFree(ctx->mr_q2);
    if (ctx->dm) cudaFree(ctx->dm);
    if (ctx->dm16) { cudaFree(ctx->dm16); cudaFree(ctx->rf_dm); }
    if (ctx->hb) cudaFree(ctx->hb);
    if (ctx->sc_host) cudaFreeHost(ctx->sc_host);
    if (ctx->sc_ring) cudaFreeHost(ctx->sc_ring);
    for (cudaEvent_t e : ctx->ev_ring) if (e) cudaEventDestroy(e);
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
    ctx->cfg_gen++;  // captured inner-iteration graphs are stale
    NEED(tier >= 0 && tier <= 6, "set_ras_tier: tier must be 0..6");
    ctx->tier_request = tier == 4 ? 2 : tier;
    ctx->chain_cycles = tier != 4;
    return WCRAS_OK;
}

int wcras_set_operand_precision(wcras_ctx* ctx, int bits) {
    NEED(ctx, "null ctx");
    ctx->cfg_gen++;  // captured inner-iteration graphs are stale
    NEED(bits == 32 || bits == 16, "set_operand_precision: bits must be 32 or 16");
    ctx->op_prec = bits;
    return WCRAS_OK;
}

int wcras_set_block_solver(wcras_ctx* ctx, int kind) {
    NEED(ctx, "null ctx");
    ctx->cfg_gen++;  // captured inner-iteration graphs are stale
    NEED(kind == 0 || kind == 1, "set_block_solver: kind must be 0 (MR) or 1 (two-dimensional minimal residual)");
    ctx->block_solver = kind;
    return WCRAS_OK;
}

int wcras_set_traversal(wcras_ctx* ctx, int ztile) {
    NEED(ctx, "null ctx");
    ctx->cfg_gen++;  // captured inner-iteration graphs are stale
    NEED(ztile >= -1 && ztile < ctx->geom.L[2] && (ztile <= 0 || ctx->geom.L[2] % ztile == 0),
         "set_traversal: ztile must be -1 (automatic), 0 (off) or a proper divisor of Lz");
    ctx->ztile_request = ztile;
    return WCRAS_OK;
}

int wcras_set_schwarz(wcras_ctx* ctx, int multiplicative) {
    NEED(ctx, "null ctx");
    ctx->cfg_gen++;  // captured inner-iteration graphs are stale
    NEED(multiplicative == 0 || multiplicative == 1, "set_schwarz: 0 (additive, RAS) or 1 (multiplicative, SAP)");
    ctx->schwarz = multiplicative;
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
    if (int rc = ensure_workspace(ctx)) return rc;  // the unchained cycles use work vectors (re-made after a failed growth)
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

int wcras_set_lookahead(wcras_ctx* ctx, int iterations) {
    NEED(ctx, "null ctx");
    NEED(iterations >= 0 && iterations <= 3, "set_lookahead: 0..3 iterations");
    ctx->lookahead = iterations;
    return WCRAS_OK;
}

int wcras_set_graphs(wcras_ctx* ctx, int enable) {
    NEED(ctx, "null ctx");
    ctx->use_graphs = enable ? 1 : 0;
    ctx->cfg_gen++;
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

int wcras_solve_multi(wcras_ctx* ctx, int nrhs, const double* eta_dev, double* phi_dev, double tol, wcras_info* info,
                      double* rel_resid_host) {
    NEED(ctx, "null ctx");
    NEED(eta_dev && phi_dev && eta_dev != phi_dev, "solve_multi: null or aliased buffers");
    NEED(nrhs >= 1 && nrhs <= 4, "solve_multi: nrhs must be 1..4");
    NEED(tol > 0, "solve_multi: tol must be positive");
    NEED(!ctx->use_ras || ctx->ras.set, "solve_multi: use_ras is set but wcras_ras_precondition was not called");
    if (nrhs != 1) ctx->cfg_gen++;  // the stack depth changes what an inner iteration launches
    ctx->nrhs = nrhs;
    const int rc = solve(ctx, eta_dev, phi_dev, tol, info, rel_resid_host);
    ctx->nrhs = 1;
    if (nrhs != 1) ctx->cfg_gen++;
    return rc;
}

int wcras_solve_host(wcras_ctx* ctx, const double* eta_host, double* phi_host, double tol, wcras_info* info) {
    NEED(ctx, "null ctx");
    NEED(eta_host && phi_host, "solve_host: null buffers");
    NEED(tol > 0, "solve_host: tol must be positive");
    NEED(!ctx->use_ras || ctx->ras.set, "solve_host: use_ras is set but wcras_ras_precondition was not called");
    if (int rc = ensure_io(ctx)) return rc;
    const size_t bytes = sizeof(double) * 24 * (size_t)ctx->geom.V;
    if (!ctx->copy_stream) {
        WC_CUDA(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
        WC_CUDA(cudaEventCreateWithFlags(&ctx->ev_copy_ready, cudaEventDisableTiming));
        WC_CUDA(cudaEventCreateWithFlags(&ctx->ev_copy_done, cudaEventDisableTiming));
    }
    WC_CUDA(cudaMemcpyAsync(ctx->io_a, eta_host, bytes, cudaMemcpyHostToDevice, ctx->stream));
    // solve() sends every candidate phi to phi_host on the copy stream while its fp64 true residual is still being checked;
    // the copy that belongs to the final phi is the last one, and solve() returns after it has completed
    ctx->host_out = phi_host;
    ctx->host_copied = false;
    int rc = solve(ctx, (const double*)ctx->io_a, (double*)ctx->io_b, tol, info);
    ctx->host_out = nullptr;
    if (rc != WCRAS_OK && rc != WCRAS_NOT_CONVERGED && rc != WCRAS_BREAKDOWN) {
        cudaStreamSynchronize(ctx->copy_stream);  // nothing may still write the caller's buffer after an error return
        return rc;
    }
    if (!ctx->host_copied) WC_CUDA(cudaMemcpyAsync(phi_host, ctx->io_b, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    WC_CUDA(cudaStreamSynchronize(ctx->stream));
    return rc;
}

int wcras_ras_autotune(wcras_ctx* ctx, const double* eta_dev, double tol, int max_rows, wcras_tune_row* best,
                       wcras_tune_row* table_host, int* nrows) {
    NEED(ctx, "null ctx");
    NEED(eta_dev && best && tol > 0 && max_rows >= 1, "ras_autotune: bad arguments");
    if (int rc = ensure_io(ctx)) return rc;
    const int* L = ctx->geom.L;
    // what the caller had configured, put back if the survey dies on a CUDA error
    const RasConfig prev = ctx->ras;
    const int prev_use = ctx->use_ras, prev_schwarz = ctx->schwarz, prev_bits = ctx->op_prec, prev_solver = ctx->block_solver;
    auto restore = [&]() {
        ctx->use_ras = prev_use; ctx->schwarz = prev_schwarz; ctx->op_prec = prev_bits; ctx->block_solver = prev_solver;
        if (prev.set) ras_configure(ctx, prev.b, prev.s, prev.niter, prev.nras);
    };
    std::vector<wcras_tune_row> rows;
    double* phi = (double*)ctx->io_b;
    int ibest = -1;
    int cur_solver = 0;  // block solver of the candidates being run (stages 0-2: MR, the block solver `configs` name)
    // run one candidate (untimed, then timed solve) and append its row; returns WCRAS_CUDA_ERROR or WCRAS_OK
    auto run = [&](const int b[4], int s, int it, int nras, int sap, int bits) -> int {
        if ((int)rows.size() >= max_rows) return WCRAS_OK;
        for (const wcras_tune_row& o : rows)  // already tried
            if (o.domain[0] == b[0] && o.domain[1] == b[1] && o.domain[2] == b[2] && o.domain[3] == b[3] && o.overlap_s == s &&
                o.block_iters == it && o.nras == nras && o.schwarz == sap && (it == 0 || (o.operand_bits == bits && o.block_solver == cur_solver)))
                return WCRAS_OK;
        wcras_tune_row r = {};
        for (int mu = 0; mu < 4; mu++) r.domain[mu] = b[mu];
        r.overlap_s = s; r.block_iters = it; r.nras = nras; r.schwarz = sap; r.operand_bits = it ? bits : 0;
        r.block_solver = it ? cur_solver : 0;
        if (it == 0) {
            ctx->use_ras = 0;
        } else {
            ctx->op_prec = bits;
            ctx->schwarz = sap;
            ctx->block_solver = cur_solver;
            const int rc = ras_configure(ctx, b, s, it, nras);
            if (rc == WCRAS_CUDA_ERROR) return rc;
            if (rc) { r.status = WCRAS_UNSUPPORTED; rows.push_back(r); return WCRAS_OK; }
            ctx->use_ras = 1;
        }
        wcras_info info = {};
        int rc = WCRAS_OK;
        for (int pass = 0; pass < 2; pass++) {  // pass 0 = warm-up
            rc = solve(ctx, eta_dev, phi, tol, &info);
            if (rc == WCRAS_CUDA_ERROR) return rc;
            if (rc == WCRAS_UNSUPPORTED) break;  // e.g. multiplicative Schwarz on a shape it cannot colour
        }
        r.status = rc; r.ms = info.ms_total; r.inner_iters = info.inner_iters; r.ras_applies = info.ras_applies;
        r.rel_resid_true = info.rel_resid_true;
        rows.push_back(r);
        if (rc == WCRAS_OK && (ibest < 0 || r.ms < rows[ibest].ms)) ibest = (int)rows.size() - 1;
        return WCRAS_OK;
    };
#define WC_RUN(...) do { if (run(__VA_ARGS__) == WCRAS_CUDA_ERROR) { restore(); return WCRAS_CUDA_ERROR; } } while (0)
    const int none[4] = {0, 0, 0, 0};
    const int bits0 = prev_bits;
    // ---- stage 0: no preconditioner; stage 1: block shapes x (N_dominv, NRAS) at overlap 0, additive ----
    WC_RUN(none, 0, 0, 0, 0, 0);
    static const int par[9][2] = {{2, 3}, {2, 2}, {2, 4}, {3, 2}, {3, 3}, {4, 1}, {4, 2}, {4, 3}, {5, 3}};
    std::vector<std::vector<int>> shapes;
    for (int b3 : {8, 4, 2}) for (int b2 : {8, 4, 2}) for (int b1 : {8, 4, 2}) for (int b0 : {8, 4, 2}) {
        const int b[4] = {b0, b1, b2, b3};
        long ns = 1;
        bool ok = true;
        for (int mu = 0; mu < 4; mu++) { ns *= b[mu]; ok = ok && L[mu] % b[mu] == 0; }
        // persistent tier (<= 256 sites, not tiny) with x >= y >= z >= t to skip permutations of the same cut,
        // and the cluster-tier shapes BASELINE.json:configs name
        const bool sorted = b0 >= b1 && b1 >= b2 && b2 >= b3;
        const bool named = (b0 == 8 && b1 == 4 && b2 == 4 && b3 == 4) || (b0 == 8 && b1 == 8 && b2 == 4 && b3 == 4) ||
                           (b0 == 8 && b1 == 8 && b2 == 8 && b3 == 8);
        if (ok && ((sorted && ns <= 256 && ns >= 64) || named)) shapes.push_back({b0, b1, b2, b3});
    }
    for (int p = 0; p < 9; p++)
        for (const auto& sh : shapes) WC_RUN(sh.data(), 0, par[p][0], par[p][1], 0, bits0);
    // ---- stage 2: around the best additive point: the paper's other axes (N_RAS = 1-10, N_dominv = 1-20,
    // d = 0, 2, 4).  The (N_dominv, NRAS) rectangle 1..8 x 1..5 on the best shape, overlap s = 1, 2 (d = 2s) on the best
    // three shapes, multiplicative Schwarz, and the other operand precision ----
    if (ibest > 0) {
        std::vector<int> order;  // converged additive rows, fastest first
        for (size_t k = 1; k < rows.size(); k++) if (rows[k].status == WCRAS_OK) order.push_back((int)k);
        std::sort(order.begin(), order.end(), [&](int a, int c) { return rows[a].ms < rows[c].ms; });
        const wcras_tune_row top = rows[order[0]];
        for (int it = 1; it <= 8; it++)
            for (int nras = 1; nras <= 5; nras++) WC_RUN(top.domain, 0, it, nras, 0, bits0);
        std::vector<std::vector<int>> seen;
        for (size_t k = 0; k < order.size() && seen.size() < 3; k++) {
            const wcras_tune_row& r = rows[order[k]];
            std::vector<int> sh(r.domain, r.domain + 4);
            if (std::find(seen.begin(), seen.end(), sh) != seen.end()) continue;
            seen.push_back(sh);
            const int it = r.block_iters, nras = r.nras;
            for (int s = 1; s <= 2; s++) {
                bool fits = true;
                for (int mu = 0; mu < 4; mu++) fits = fits && (sh[mu] == L[mu] || sh[mu] + 2 * s <= L[mu]);
                if (!fits) continue;
                WC_RUN(sh.data(), s, it, nras, 0, bits0);
                if (nras > 1) WC_RUN(sh.data(), s, it + 1, nras - 1, 0, bits0);
            }
            WC_RUN(sh.data(), 0, it, nras, 1, bits0);                      // SAP: nras = number of red-black cycles
            WC_RUN(sh.data(), 0, it + 1, nras > 1 ? nras - 1 : 1, 1, bits0);
        }
        const wcras_tune_row now = rows[ibest];
        if (now.block_iters) WC_RUN(now.domain, now.overlap_s, now.block_iters, now.nras, now.schwarz, bits0 == 16 ? 32 : 16);
        // ---- stage 3: the second block solver (wcras_set_block_solver(1), reading R2) where its kernel runs: 16-bit
        // operands, overlap 0, the fastest persistent-tier shape so far; N_dominv 2, 4, 6 x 2, 3 cycles, additive and
        // multiplicative (its best points are not MR's: fewer, longer cycles) ----
        const wcras_tune_row lead = rows[ibest];
        long lead_sites = 1;
        for (int mu = 0; mu < 4; mu++) lead_sites *= lead.domain[mu];
        if (lead.block_iters && lead.overlap_s == 0 && lead_sites <= 256) {
            cur_solver = 1;
            for (int sap = 1; sap >= 0; sap--)
                for (int it = 2; it <= 6; it += 2)
                    for (int nras = 2; nras <= 3; nras++) WC_RUN(lead.domain, 0, it, nras, sap, 16);
            cur_solver = 0;
        }
    }
#undef WC_RUN
    if (table_host) for (size_t k = 0; k < rows.size(); k++) table_host[k] = rows[k];
    if (nrows) *nrows = (int)rows.size();
    if (ibest < 0) {
        restore();
        snprintf(ctx->err, sizeof ctx->err, "ras_autotune: no candidate converged");
        return WCRAS_NOT_CONVERGED;
    }
    *best = rows[ibest];
    if (best->block_iters == 0) {
        ctx->use_ras = 0; ctx->schwarz = prev_schwarz; ctx->op_prec = prev_bits; ctx->block_solver = prev_solver;
        return WCRAS_OK;
    }
    ctx->use_ras = 1;
    ctx->schwarz = best->schwarz;
    ctx->op_prec = best->operand_bits;
    ctx->block_solver = best->block_solver;
    return ras_configure(ctx, best->domain, best->overlap_s, best->block_iters, best->nras);
}

int wcras_export_clover(wcras_ctx* ctx, double* out_dev) {
    NEED(ctx, "null ctx");
    NEED(out_dev, "export_clover: null buffer");
    return export_clover(ctx, out_dev);
}

int wcras_time_kernel(wcras_ctx* ctx, int which, int reps, double* ms_per_launch) {
    NEED(ctx, "null ctx");
    NEED(ms_per_launch && reps >= 1 && which >= 0 && which <= 4, "time_kernel: bad arguments");
    if (int rc = ensure_workspace(ctx)) return rc;
    if (which == 3) return time_blas(ctx, reps, ms_per_launch);
    NEED((which != 2 && which != 4) || ctx->ras.set, "time_kernel: call wcras_ras_precondition first");
    const size_t V = ctx->geom.V;
    // deterministic non-trivial scratch input: reuse the fp32 link array bytes as a spinor-sized pattern
    WC_CUDA(cudaMemcpyAsync(ctx->w32[0], ctx->g32a, sizeof(float4) * 6 * V, cudaMemcpyDeviceToDevice, ctx->stream));
    WC_CUDA(cudaMemcpyAsync(ctx->w64[0], ctx->g64, sizeof(double2) * 12 * V, cudaMemcpyDeviceToDevice, ctx->stream));
    EventPair ev;
    WC_CUDA(ev.create());
    const cudaEvent_t e0 = ev.a, e1 = ev.b;
    int rc = WCRAS_OK;
    for (int pass = 0; pass < 2 && !rc; pass++) {  // pass 0 = warm-up
        const int n = pass == 0 ? 3 : reps;
        WC_CUDA(cudaEventRecord(e0, ctx->stream));
        for (int k = 0; k < n && !rc; k++) {
            if (which == 0) rc = dslash<float>(ctx, ctx->w32[0], ctx->w32[1]);
            else if (which == 1) rc = dslash<double>(ctx, ctx->w64[0], ctx->w64[1]);
            else if (which == 2) rc = ras_block_solve(ctx, ctx->w32[0], ctx->w32[1]);
            else rc = ras_apply(ctx, ctx->w32[0], ctx->w32[1]);  // a whole K_RAS application: NRAS chained cycles
        }
        WC_CUDA(cudaEventRecord(e1, ctx->stream));
        WC_CUDA(cudaStreamSynchronize(ctx->stream));
    }
    float t = 0;
    WC_CUDA(cudaEventElapsedTime(&t, e0, e1));
    *ms_per_launch = t / reps;
    return rc;
}

long long wcras_launch_count(const wcras_ctx* ctx) { return ctx ? ctx->launches : 0; }

const char* wcras_last_error(const wcras_ctx* ctx) { return ctx ? ctx->err : "null ctx"; }

}  // extern "C"
