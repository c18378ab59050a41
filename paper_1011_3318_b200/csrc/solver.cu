// solver.cu -- steps A6 (inner fp32 BiCGStab on D K_RAS chi = b, Eq. 2.2) and A7 (outer fp64
// "flexible" BiCGStab whose preconditioner is the inner solve), with the fused BLAS-1 kernels
// of north_star (d).  Recurrences (reading Q13), identical for both precisions:
//   x=0, r=b, rt=r, rho=alpha=omega=1, v=p=0; loop:
//   rho'=<rt,r>; beta=(rho'/rho)(alpha/omega); p=r+beta(p-omega v); ph=K p; v=D ph; alpha=rho'/<rt,v>;
//   s=r-alpha v; [outer only: stop if |s|/|b|<tol with x+=alpha ph]; sh=K s; t=D sh; omega=<t,s>/<t,t>;
//   x+=alpha ph+omega sh; r=s-omega t; stop when |r|/|b|<tol.
#include <cmath>

#include "blas.cuh"

namespace wc {

template <typename T> struct cpx { T r, i; };

template <typename T> __device__ __forceinline__ void unpack(const float4& v, cpx<T>* c) { c[0] = {v.x, v.y}; c[1] = {v.z, v.w}; }
template <typename T> __device__ __forceinline__ void unpack(const double2& v, cpx<T>* c) { c[0] = {v.x, v.y}; }
__device__ __forceinline__ float4 pack(const cpx<float>* c, float4*) { return make_float4(c[0].r, c[0].i, c[1].r, c[1].i); }
__device__ __forceinline__ double2 pack(const cpx<double>* c, double2*) { return make_double2(c[0].r, c[0].i); }

template <typename T> __device__ __forceinline__ cpx<T> operator+(cpx<T> a, cpx<T> b) { return {a.r + b.r, a.i + b.i}; }
template <typename T> __device__ __forceinline__ cpx<T> operator-(cpx<T> a, cpx<T> b) { return {a.r - b.r, a.i - b.i}; }
template <typename T> __device__ __forceinline__ cpx<T> operator*(cpx<T> a, cpx<T> b) {
    return {a.r * b.r - a.i * b.i, a.r * b.i + a.i * b.r};
}
// acc += conj(a) * b in fp64
template <typename T> __device__ __forceinline__ void dot_acc(cpx<T> a, cpx<T> b, double& re, double& im) {
    re += (double)a.r * (double)b.r + (double)a.i * (double)b.i;
    im += (double)a.r * (double)b.i - (double)a.i * (double)b.r;
}
template <typename T> __device__ __forceinline__ cpx<T> ld_scalar(const double* s) { return {(T)s[0], (T)s[1]}; }

#define GRID_STRIDE(idx, n) for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < (n); idx += (size_t)gridDim.x * blockDim.x)

// bb = |b|^2; scalars reset.  No vector is written: the first iteration reads b in place of r (p = b, s = b - alpha v),
// writes x instead of updating it, and the shadow residual rt is b itself ("first iteration").
template <typename T, typename Vec>
__global__ void __launch_bounds__(RED_THREADS) k_init(size_t n, const Vec* __restrict__ b, Scalars* sc, double* partials,
                                                      unsigned* ticket, double tol, double tiny, int half) {
    constexpr int N = Cx<Vec>::N;
    double acc[1] = {0};
    GRID_STRIDE(k, n) {
        cpx<T> c[N];
        unpack<T>(b[k], c);
#pragma unroll
        for (int j = 0; j < N; j++) acc[0] += (double)c[j].r * c[j].r + (double)c[j].i * c[j].i;
    }
    double tot[1];
    if (grid_reduce<1>(acc, partials, ticket, tot)) {
        sc->bb = tot[0]; sc->rr = tot[0]; sc->ss = tot[0];
        sc->rho[0] = tot[0]; sc->rho[1] = 0; sc->rho_old[0] = 1; sc->rho_old[1] = 0;
        sc->alpha[0] = 1; sc->alpha[1] = 0; sc->omega[0] = 1; sc->omega[1] = 0;
        sc->thresh = tol * tol; sc->tiny = tiny; sc->half = half;
        sc->flag = tot[0] > 0 ? 0 : 1;  // zero right-hand side: x = 0 is the solution
        sc->it_done = 0; sc->half_exit = 0;
    }
}

// the same scalar reset when |b|^2 is already known (the outer solver: |eta|^2 and the true-residual norms are computed anyway)
__global__ void k_init_known(Scalars* sc, double bb, double tol, double tiny, int half) {
    sc->bb = bb; sc->rr = bb; sc->ss = bb;
    sc->rho[0] = bb; sc->rho[1] = 0; sc->rho_old[0] = 1; sc->rho_old[1] = 0;
    sc->alpha[0] = 1; sc->alpha[1] = 0; sc->omega[0] = 1; sc->omega[1] = 0;
    sc->thresh = tol * tol; sc->tiny = tiny; sc->half = half;
    sc->flag = bb > 0 ? 0 : 1;
    sc->it_done = 0; sc->half_exit = 0;
}

// restart: rt = r, p = v = 0, rho = <r,r>, rho_old = alpha = omega = 1
template <typename T, typename Vec>
__global__ void __launch_bounds__(RED_THREADS) k_restart(size_t n, const Vec* __restrict__ r, Vec* rt, Vec* p, Vec* v, Scalars* sc,
                                                         double* partials, unsigned* ticket) {
    constexpr int N = Cx<Vec>::N;
    double acc[1] = {0};
    Vec zero;
    memset(&zero, 0, sizeof zero);
    GRID_STRIDE(k, n) {
        const Vec rv = r[k];
        cpx<T> c[N];
        unpack<T>(rv, c);
#pragma unroll
        for (int j = 0; j < N; j++) acc[0] += (double)c[j].r * c[j].r + (double)c[j].i * c[j].i;
        rt[k] = rv; p[k] = zero; v[k] = zero;
    }
    double tot[1];
    if (grid_reduce<1>(acc, partials, ticket, tot)) {
        sc->rr = tot[0];
        sc->rho[0] = tot[0]; sc->rho[1] = 0; sc->rho_old[0] = 1; sc->rho_old[1] = 0;
        sc->alpha[0] = 1; sc->alpha[1] = 0; sc->omega[0] = 1; sc->omega[1] = 0;
        sc->flag = 0;
    }
}

// pout = r + beta (pin - omega v), beta = (rho/rho_old)(alpha/omega).  pin == pout in general; in the second iteration pin
// is b: the first iteration has p = r = b and works on b itself instead of on a copy.
template <typename T, typename Vec>
__global__ void __launch_bounds__(RED_THREADS) k_update_p(size_t n, const Vec* __restrict__ r, const Vec* pin, Vec* pout,
                                                          const Vec* __restrict__ v, const Scalars* __restrict__ sc) {
    constexpr int N = Cx<Vec>::N;
    if (sc->flag) return;
    const cd b = cmul(cdiv({sc->rho[0], sc->rho[1]}, {sc->rho_old[0], sc->rho_old[1]}),
                      cdiv({sc->alpha[0], sc->alpha[1]}, {sc->omega[0], sc->omega[1]}));
    const cpx<T> beta = {(T)b.r, (T)b.i}, omega = ld_scalar<T>(sc->omega);
    GRID_STRIDE(k, n) {
        cpx<T> rc[N], pc[N], vc[N];
        unpack<T>(r[k], rc); unpack<T>(pin[k], pc); unpack<T>(v[k], vc);
#pragma unroll
        for (int j = 0; j < N; j++) pc[j] = rc[j] + beta * (pc[j] - omega * vc[j]);
        pout[k] = pack(pc, (Vec*)nullptr);
    }
}

// <rt,v> (alpha) and <t,s>, <t,t> (omega) are fused into the Dslash that produces v and t (dslash.cu, DOT = 1 / 2)

// s = r - alpha v; ss = |s|^2
template <typename T, typename Vec>
__global__ void __launch_bounds__(RED_THREADS) k_update_s(size_t n, const Vec* __restrict__ r, const Vec* __restrict__ v,
                                                          Vec* __restrict__ s, Scalars* sc, double* partials, unsigned* ticket) {
    constexpr int N = Cx<Vec>::N;
    if (sc->flag) return;
    const cpx<T> alpha = ld_scalar<T>(sc->alpha);
    double acc[1] = {0};
    GRID_STRIDE(k, n) {
        cpx<T> rc[N], vc[N];
        unpack<T>(r[k], rc); unpack<T>(v[k], vc);
#pragma unroll
        for (int j = 0; j < N; j++) {
            rc[j] = rc[j] - alpha * vc[j];
            acc[0] += (double)rc[j].r * rc[j].r + (double)rc[j].i * rc[j].i;
        }
        s[k] = pack(rc, (Vec*)nullptr);
    }
    double tot[1];
    if (grid_reduce<1>(acc, partials, ticket, tot)) {
        sc->ss = tot[0];
        // half-step exit (van der Vorst): |s| already below the tolerance -> x += alpha ph finishes the solve; every kernel
        // up to k_update_xr of this iteration sees flag = 2 and returns, k_update_xr applies the half step
        if (sc->half && tot[0] < sc->thresh * sc->bb) sc->flag = 2;
    }
}

// x += alpha ph + omega sh; r = s - omega t; rho_old = rho; rho = <rt,r>; rr = |r|^2
template <typename T, typename Vec>
__global__ void __launch_bounds__(RED_THREADS) k_update_xr(size_t n, Vec* __restrict__ x, const Vec* __restrict__ ph,
                                                           const Vec* __restrict__ sh, const Vec* __restrict__ s,
                                                           const Vec* __restrict__ t, const Vec* __restrict__ rt, Vec* __restrict__ r,
                                                           Scalars* sc, double* partials, unsigned* ticket, int first) {
    constexpr int N = Cx<Vec>::N;
    const int fl = sc->flag;  // every block reads it before the last block (the only writer) can change it
    if (fl == 1 || fl == 3) return;
    const cpx<T> alpha = ld_scalar<T>(sc->alpha), omega = ld_scalar<T>(sc->omega);
    double acc[3] = {0, 0, 0};
    if (fl == 2) {  // half-step exit: x += alpha ph, the residual is s
        GRID_STRIDE(k, n) {
            cpx<T> xc[N], pc[N];
            if (first) {
#pragma unroll
                for (int j = 0; j < N; j++) xc[j] = {0, 0};
            } else {
                unpack<T>(x[k], xc);
            }
            unpack<T>(ph[k], pc);
#pragma unroll
            for (int j = 0; j < N; j++) xc[j] = xc[j] + alpha * pc[j];
            x[k] = pack(xc, (Vec*)nullptr);
        }
        double tot[3];
        if (grid_reduce<3>(acc, partials, ticket, tot)) {
            sc->rr = sc->ss; sc->it_done += 1; sc->half_exit = 1; sc->flag = 1;
        }
        return;
    }
    GRID_STRIDE(k, n) {
        cpx<T> xc[N], pc[N], hc[N], sc_[N], tc[N], rc[N];
        if (first) {  // x = 0 before the first iteration
#pragma unroll
            for (int j = 0; j < N; j++) xc[j] = {0, 0};
        } else {
            unpack<T>(x[k], xc);
        }
        unpack<T>(ph[k], pc); unpack<T>(sh[k], hc);
        unpack<T>(s[k], sc_); unpack<T>(t[k], tc); unpack<T>(rt[k], rc);
#pragma unroll
        for (int j = 0; j < N; j++) {
            xc[j] = xc[j] + alpha * pc[j] + omega * hc[j];
            sc_[j] = sc_[j] - omega * tc[j];
            dot_acc(rc[j], sc_[j], acc[0], acc[1]);
            acc[2] += (double)sc_[j].r * sc_[j].r + (double)sc_[j].i * sc_[j].i;
        }
        x[k] = pack(xc, (Vec*)nullptr);
        r[k] = pack(sc_, (Vec*)nullptr);
    }
    double tot[3];
    if (grid_reduce<3>(acc, partials, ticket, tot)) {
        sc->rho_old[0] = sc->rho[0]; sc->rho_old[1] = sc->rho[1];
        sc->rho[0] = tot[0]; sc->rho[1] = tot[1];
        sc->rr = tot[2];
        sc->it_done += 1;
        // convergence and breakdown are decided here, on the device: NaN or |rho|, |omega| underflow (reading Q13) stop the
        // iteration with flag 3 (the host restarts once), |r| below the tolerance with flag 1
        if (!(tot[2] == tot[2])) sc->flag = 3;
        else if (tot[2] < sc->thresh * sc->bb) sc->flag = 1;
        else if (hypot(tot[0], tot[1]) < sc->tiny * sc->bb || hypot(sc->omega[0], sc->omega[1]) < sc->tiny) sc->flag = 3;
    }
}

// nrm = |a|^2 (fp64 vectors)
__global__ void __launch_bounds__(RED_THREADS) k_norm2_d(size_t n, const double2* __restrict__ a, Scalars* sc, double* partials,
                                                         unsigned* ticket) {
    double acc[1] = {0};
    GRID_STRIDE(k, n) {
        const double2 v = a[k];
        acc[0] += v.x * v.x + v.y * v.y;
    }
    double tot[1];
    if (grid_reduce<1>(acc, partials, ticket, tot)) sc->nrm = tot[0];
}

// out32 = in64 / sqrt(nrm2), and the start of the inner solver on out32 in the same pass: bb = |out32|^2 from the rounded fp32
// values (what k_init would compute from them), scalars reset; the tolerance follows by k_set_tol once the host has it.
// fp32 SoA chunk c4 of site i (float4 [6][V]) holds the complex components 2*c4 and 2*c4+1, which live in fp64 SoA chunks
// 2*c4 and 2*c4+1 of the same site (double2 [12][V]).
__global__ void __launch_bounds__(RED_THREADS) k_d2f_init(size_t V, int nr, const double2* __restrict__ in, float4* __restrict__ out,
                                                          const double* __restrict__ nrm2, Scalars* sc, double* partials,
                                                          unsigned* ticket) {
    const double inv = *nrm2 > 0 ? rsqrt(*nrm2) : 0.0;
    double acc[1] = {0};
    GRID_STRIDE(k, 6 * V * nr) {
        const size_t r = k / (6 * V), kk = k - r * 6 * V, c4 = kk / V, i = kk - c4 * V;
        const double2* inr = in + r * 12 * V;
        const double2 a = inr[(2 * c4) * V + i], b = inr[(2 * c4 + 1) * V + i];
        const float4 o = make_float4((float)(a.x * inv), (float)(a.y * inv), (float)(b.x * inv), (float)(b.y * inv));
        out[k] = o;
        acc[0] += (double)o.x * o.x + (double)o.y * o.y + (double)o.z * o.z + (double)o.w * o.w;
    }
    double tot[1];
    if (grid_reduce<1>(acc, partials, ticket, tot)) {
        sc->bb = tot[0]; sc->rr = tot[0]; sc->ss = tot[0];
        sc->rho[0] = tot[0]; sc->rho[1] = 0; sc->rho_old[0] = 1; sc->rho_old[1] = 0;
        sc->alpha[0] = 1; sc->alpha[1] = 0; sc->omega[0] = 1; sc->omega[1] = 0;
        sc->flag = tot[0] > 0 ? 0 : 1;
        sc->it_done = 0; sc->half_exit = 0;
    }
}
__global__ void k_set_tol(Scalars* sc, double tol, double tiny, int half) {
    sc->thresh = tol * tol; sc->tiny = tiny; sc->half = half;
}
// out64 = in32 * sqrt(nrm)
__global__ void __launch_bounds__(RED_THREADS) k_f2d_scaled(size_t V, int nr, const float4* __restrict__ in,
                                                            double2* __restrict__ out, const double* __restrict__ nrm2) {
    const double sc_ = sqrt(*nrm2);
    GRID_STRIDE(k, 6 * V * nr) {
        const size_t r = k / (6 * V), kk = k - r * 6 * V, c4 = kk / V, i = kk - c4 * V;
        double2* outr = out + r * 12 * V;
        const float4 a = in[k];
        outr[(2 * c4) * V + i] = make_double2(a.x * sc_, a.y * sc_);
        outr[(2 * c4 + 1) * V + i] = make_double2(a.z * sc_, a.w * sc_);
    }
}
// a *= f (fp64)
__global__ void __launch_bounds__(RED_THREADS) k_scale_d(size_t n, double2* __restrict__ a, double f) {
    GRID_STRIDE(k, n) {
        double2 v = a[k];
        v.x *= f; v.y *= f;
        a[k] = v;
    }
}
// x += dx (fp64)
__global__ void __launch_bounds__(RED_THREADS) k_add_d(size_t n, double2* __restrict__ x, const double2* __restrict__ dx) {
    GRID_STRIDE(k, n) {
        double2 a = x[k];
        const double2 b = dx[k];
        a.x += b.x; a.y += b.y;
        x[k] = a;
    }
}

// ---------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------
static int read_scalars(wcras_ctx* ctx, const Scalars* sc) {
    WC_CUDA(cudaMemcpyAsync(ctx->sc_host, sc, sizeof(Scalars), cudaMemcpyDeviceToHost, ctx->stream));
    WC_CUDA(cudaStreamSynchronize(ctx->stream));
    return WCRAS_OK;
}

#define LAUNCH(kern, ...)                                                        \
    do {                                                                         \
        kern<<<RED_BLOCKS, RED_THREADS, 0, ctx->stream>>>(__VA_ARGS__);          \
        ctx->launches++;                                                         \
    } while (0)

template <typename T> struct Work {
    typedef typename VecOf<T>::type Vec;
    Vec *r, *rt, *p, *v, *s, *t, *ph, *sh;
    Scalars* sc;
    size_t n;
};

void drop_iter_graphs(wcras_ctx* ctx) {
    for (auto& row : ctx->iter_graph)
        for (auto& g : row) {
            if (g.exec) cudaGraphExecDestroy(g.exec);
            g = wcras_ctx::IterGraph();
        }
    ctx->graph_b = ctx->graph_x = nullptr;
}

// BiCGStab driver.  K(in,out) applies the preconditioner (ignored when k_identity).  status: 0 converged,
// WCRAS_NOT_CONVERGED, WCRAS_BREAKDOWN, or a CUDA error.
//
// Convergence, the half-step exit and breakdown are decided on the device (Scalars::flag, set by the last block of
// k_update_s / k_update_xr); every kernel of an iteration returns at once when the flag is set.  The host therefore
// does not wait for an iteration before it enqueues the next one: after every iteration it enqueues a copy of the scalars
// into a pinned ring slot and looks at the slot of `lookahead` iterations ago.  With lookahead 0 (the outer fp64 solver,
// whose preconditioner is a whole inner solve) every iteration is checked before the next one is enqueued, and the
// half-step flag is read before K(s).
template <typename T, typename KFunc>
static int bicgstab(wcras_ctx* ctx, Work<T>& w, const typename VecOf<T>::type* b, typename VecOf<T>::type* x, double tol, int maxit,
                    bool half_exit, bool k_identity, KFunc K, int* iters, double* relres, double bb_known = -1.0) {
    typedef typename VecOf<T>::type Vec;
    constexpr int RING = 4;
    const size_t n = w.n;
    double* part = ctx->partials;
    unsigned* tk = ctx->ticket;
    const int la = sizeof(T) == 4 ? (ctx->lookahead < RING - 1 ? ctx->lookahead : RING - 1) : 0;
    const double tiny = sizeof(T) == 4 ? 1e-30 : 1e-290;
    {
        TimedRegion tr(ctx, TC_BLAS);
        if (bb_known == -2.0) {  // scalars already reset by the kernel that produced b (k_d2f_init)
            k_set_tol<<<1, 1, 0, ctx->stream>>>(w.sc, tol, tiny, half_exit ? 1 : 0);
            ctx->launches++;
        } else if (bb_known >= 0) {
            k_init_known<<<1, 1, 0, ctx->stream>>>(w.sc, bb_known, tol, tiny, half_exit ? 1 : 0);
            ctx->launches++;
        } else {
            LAUNCH((k_init<T, Vec>), n, b, w.sc, part, tk, tol, tiny, half_exit ? 1 : 0);
        }
    }
    *iters = 0;
    *relres = 0;
    const Vec* sh = k_identity ? w.s : w.sh;
    const Vec* pprev = b;  // p of the previous iteration: b after the first one (p = r = b, never copied), then w.p
    const Vec* rt = b;    // shadow residual = initial residual = b (x0 = 0); a restart switches to the copy in w.rt
    const Vec* rcur = b;  // residual read by the first iteration; w.r from the first r = s - omega t on
    // the fp32 launches of this solver carry the device flag so that those enqueued past convergence are no-ops
    struct StopScope {
        wcras_ctx* c;
        bool on;
        StopScope(wcras_ctx* cc, const int* f, bool o) : c(cc), on(o) { if (on) { c->geom.stop = f; c->fused.stop = f; } }
        ~StopScope() { if (on) { c->geom.stop = nullptr; c->fused.stop = nullptr; } }
    } stop_scope(ctx, &w.sc->flag, sizeof(T) == 4);
    const int c0[4] = {ctx->dv32, ctx->dv64, ctx->block_dv, ctx->ras_applies};
    bool x_written = false, first = true;
    int enq = 0, restarts = 0, status = WCRAS_NOT_CONVERGED;
    double best = -1;
    int it_best = 0;
    for (;;) {
        bool stop = false;
        while (!stop && enq < maxit) {
            if (la > 0 && enq > la) {  // look at the iteration enqueued `la` iterations ago
                const int j = enq - la - 1;
                WC_CUDA(cudaEventSynchronize(ctx->ev_ring[j % RING]));
                const Scalars& h = ctx->sc_ring[j % RING];
                if (h.flag) break;
                // stagnation guard (fp32 inner solver at the end of its accuracy): no new minimum of |r| for 10 iterations
                if (best < 0 || h.rr < best) { best = h.rr; it_best = j; }
                else if (j - it_best >= 10) break;
            }
            // One iteration = 10-14 launches whose arguments depend only on its kind (0: first, p = r = b, x written; 1: second,
            // p of the previous iteration is b; 2: every later one).  The fp32 inner solver replays it as a CUDA graph from the
            // second time a kind runs with the same vectors and configuration (the first time runs eagerly, so that every
            // lazily allocated buffer exists before a capture): below 16^4 the solve is bound by the host's launch rate.
            const int kind = first ? 0 : (pprev == b ? 1 : 2);
            auto body = [&]() -> int {
                // K hints (outer solver): whose norm the device already holds -- 1: |p|^2 = |b|^2 (first iteration), 2: |s|^2, 0: none
                const Vec* pcur = w.p;
                if (kind == 0) {
                    pcur = rcur;  // p = r = b
                } else {
                    TimedRegion tr(ctx, TC_BLAS);
                    LAUNCH((k_update_p<T, Vec>), n, rcur, pprev, w.p, w.v, w.sc);
                }
                const Vec* ph = k_identity ? pcur : w.ph;
                if (!k_identity) if (int rc = K(pcur, w.ph, kind == 0 ? 1 : 0)) return rc;
                if (int rc = dslash<T>(ctx, ph, w.v, nullptr, 1, rt, w.sc)) return rc;  // v = D ph; <rt,v>, alpha fused
                {
                    TimedRegion tr(ctx, TC_BLAS);
                    LAUNCH((k_update_s<T, Vec>), n, rcur, w.v, w.s, w.sc, part, tk);
                }
                bool half_now = false;
                if (la == 0 && half_exit) {  // the second half costs a whole inner solve: read the flag first
                    if (int rc = read_scalars(ctx, w.sc)) return rc;
                    half_now = ctx->sc_host->flag == 2;
                }
                if (!half_now) {
                    if (!k_identity) if (int rc = K(w.s, w.sh, 2)) return rc;
                    if (int rc = dslash<T>(ctx, sh, w.t, nullptr, 2, w.s, w.sc)) return rc;  // t = D sh; <t,s>, <t,t>, omega fused
                }
                {
                    TimedRegion tr(ctx, TC_BLAS);
                    LAUNCH((k_update_xr<T, Vec>), n, x, ph, sh, w.s, w.t, rt, w.r, w.sc, part, tk, x_written ? 0 : 1);
                }
                return WCRAS_OK;
            };
            const bool graphable = sizeof(T) == 4 && la > 0 && ctx->use_graphs && !ctx->timing && restarts == 0 && rt == b &&
                                   (kind == 0) == !x_written;
            if (graphable) {
                if (ctx->graph_b != (const void*)b || ctx->graph_x != (const void*)x || ctx->graph_gen != ctx->cfg_gen) {
                    drop_iter_graphs(ctx);
                    ctx->graph_b = b; ctx->graph_x = x; ctx->graph_gen = ctx->cfg_gen;
                }
                wcras_ctx::IterGraph& g = ctx->iter_graph[k_identity ? 0 : 1][kind];
                if (g.exec) {
                    WC_CUDA(cudaGraphLaunch(g.exec, ctx->stream));
                    ctx->launches += g.d_launches; ctx->dv32 += g.d_dv32; ctx->block_dv += g.d_blk; ctx->ras_applies += g.d_ras;
                } else if (g.seen >= 1) {
                    const long long l0 = ctx->launches;
                    const int c1[3] = {ctx->dv32, ctx->block_dv, ctx->ras_applies};
                    if (!ctx->cap_stream) WC_CUDA(cudaStreamCreateWithFlags(&ctx->cap_stream, cudaStreamNonBlocking));
                    cudaStream_t user = ctx->stream;
                    WC_CUDA(cudaStreamBeginCapture(ctx->cap_stream, cudaStreamCaptureModeThreadLocal));
                    ctx->stream = ctx->cap_stream;  // every launch of the body goes to ctx->stream
                    const int rc = body();
                    ctx->stream = user;
                    cudaGraph_t graph = nullptr;
                    const cudaError_t ce = cudaStreamEndCapture(ctx->cap_stream, &graph);
                    if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
                    WC_CUDA(ce);
                    const cudaError_t ci = cudaGraphInstantiate(&g.exec, graph, 0);
                    cudaGraphDestroy(graph);
                    WC_CUDA(ci);
                    g.d_launches = ctx->launches - l0;
                    g.d_dv32 = ctx->dv32 - c1[0]; g.d_blk = ctx->block_dv - c1[1]; g.d_ras = ctx->ras_applies - c1[2];
                    WC_CUDA(cudaGraphLaunch(g.exec, ctx->stream));  // a capture records, it does not execute
                } else {
                    g.seen++;
                    if (int rc = body()) return rc;
                }
            } else {
                if (int rc = body()) return rc;
            }
            if (kind != 0) pprev = w.p;
            x_written = true;
            first = false;
            rcur = w.r;
            WC_CUDA(cudaMemcpyAsync(&ctx->sc_ring[enq % RING], w.sc, sizeof(Scalars), cudaMemcpyDeviceToHost, ctx->stream));
            WC_CUDA(cudaEventRecord(ctx->ev_ring[enq % RING], ctx->stream));
            enq++;
            if (la == 0) {
                WC_CUDA(cudaEventSynchronize(ctx->ev_ring[(enq - 1) % RING]));
                const Scalars& h = ctx->sc_ring[(enq - 1) % RING];
                if (h.flag) stop = true;
            }
        }
        if (int rc = read_scalars(ctx, w.sc)) return rc;  // drains the stream: the state is that of the last effective iteration
        const Scalars& h = *ctx->sc_host;
        if (h.flag == 1) { status = WCRAS_OK; break; }
        if (h.flag == 3 && restarts == 0 && h.rr == h.rr && enq < maxit) {  // breakdown: one restart with rt = r (reading Q13)
            restarts++;
            TimedRegion tr(ctx, TC_BLAS);
            LAUNCH((k_restart<T, Vec>), n, rcur, w.rt, w.p, w.v, w.sc, part, tk);
            rt = w.rt;
            first = false;  // p = v = 0 are stored now: the general p update applies
            pprev = w.p;
            enq = h.it_done;
            best = -1;
            continue;
        }
        status = h.flag == 3 ? WCRAS_BREAKDOWN : WCRAS_NOT_CONVERGED;
        break;
    }
    const Scalars& h = *ctx->sc_host;
    if (!x_written || h.it_done == 0) WC_CUDA(cudaMemsetAsync(x, 0, sizeof(Vec) * n, ctx->stream));  // no update of x happened
    if (la > 0 && enq > 0) {
        // iterations enqueued past convergence were no-ops: count the effective ones (every inner iteration adds the same
        // number of D and K applications, a half-step exit half of them)
        const long eff = 2L * h.it_done - (h.half_exit ? 1 : 0), all = 2L * enq;
        int* cnt[4] = {&ctx->dv32, &ctx->dv64, &ctx->block_dv, &ctx->ras_applies};
        for (int k = 0; k < 4; k++) *cnt[k] = c0[k] + (int)((long)(*cnt[k] - c0[k]) * eff / all);
    }
    WC_CHECK_LAUNCH();
    *iters = h.it_done;
    *relres = h.bb > 0 ? std::sqrt(h.rr / h.bb) : 0.0;
    return status;
}

static void free_owned(wcras_ctx* ctx, void* p) {
    if (!p) return;
    for (size_t k = 0; k < ctx->owned.size(); k++)
        if (ctx->owned[k] == p) { ctx->owned.erase(ctx->owned.begin() + k); break; }
    cudaFree(p);
}

// solver vectors, each a stack of ctx->nrhs lattice vectors; grown when a deeper stack arrives
int ensure_workspace(wcras_ctx* ctx) {
    const size_t V = ctx->geom.V;
    if (!ctx->sc32) {
        if (alloc_dev(ctx, (void**)&ctx->sc32, sizeof(Scalars))) return WCRAS_CUDA_ERROR;
        if (alloc_dev(ctx, (void**)&ctx->sc64, sizeof(Scalars))) return WCRAS_CUDA_ERROR;
        if (alloc_dev(ctx, (void**)&ctx->partials, sizeof(double) * RED_BLOCKS * 8)) return WCRAS_CUDA_ERROR;
        if (alloc_dev(ctx, (void**)&ctx->ticket, sizeof(unsigned))) return WCRAS_CUDA_ERROR;
        WC_CUDA(cudaMemsetAsync(ctx->ticket, 0, sizeof(unsigned), ctx->stream));
        WC_CUDA(cudaMallocHost((void**)&ctx->sc_host, sizeof(Scalars)));
        WC_CUDA(cudaMallocHost((void**)&ctx->sc_ring, sizeof(Scalars) * 4));
        for (int k = 0; k < 4; k++) WC_CUDA(cudaEventCreateWithFlags(&ctx->ev_ring[k], cudaEventDisableTiming));
    }
    if (ctx->ws_nrhs < ctx->nrhs) {
        // Grow for a deeper stack: the old vectors go first (two sets would not fit at the sizes this is for).  ws_nrhs is 0
        // while the set is incomplete, so that a failed growth (out of memory) leaves a context whose next solve allocates
        // afresh instead of running on missing vectors.
        WC_CUDA(cudaStreamSynchronize(ctx->stream));
        auto release = [&]() {
            for (int k = 0; k < 12; k++) { free_owned(ctx, ctx->w32[k]); free_owned(ctx, ctx->w64[k]); ctx->w32[k] = nullptr; ctx->w64[k] = nullptr; }
            for (int k = 0; k < 3; k++) { free_owned(ctx, ctx->ras32[k]); ctx->ras32[k] = nullptr; }
        };
        ctx->ws_nrhs = 0;
        ctx->cfg_gen++;  // the work vectors move: captured inner-iteration graphs are stale
        release();
        const size_t nr = ctx->nrhs;
        bool ok = true;
        for (int k = 0; k < 12 && ok; k++) ok = alloc_dev(ctx, (void**)&ctx->w32[k], sizeof(float4) * 6 * V * nr) == WCRAS_OK;
        for (int k = 0; k < 12 && ok; k++) ok = alloc_dev(ctx, (void**)&ctx->w64[k], sizeof(double2) * 12 * V * nr) == WCRAS_OK;
        for (int k = 0; k < 3 && ok; k++) ok = alloc_dev(ctx, (void**)&ctx->ras32[k], sizeof(float4) * 6 * V * nr) == WCRAS_OK;
        if (!ok) {
            release();          // ctx->err holds the cudaMalloc message
            cudaGetLastError();
            return WCRAS_CUDA_ERROR;
        }
        ctx->ws_nrhs = ctx->nrhs;
    }
    return WCRAS_OK;
}

static Work<float> work32(wcras_ctx* ctx) {
    Work<float> w;
    w.r = ctx->w32[0]; w.rt = ctx->w32[1]; w.p = ctx->w32[2]; w.v = ctx->w32[3]; w.s = ctx->w32[4];
    w.t = ctx->w32[5]; w.ph = ctx->w32[6]; w.sh = ctx->w32[7];
    w.sc = ctx->sc32; w.n = (size_t)6 * ctx->geom.V * ctx->nrhs;
    return w;
}
static Work<double> work64(wcras_ctx* ctx) {
    Work<double> w;
    w.r = ctx->w64[0]; w.rt = ctx->w64[1]; w.p = ctx->w64[2]; w.v = ctx->w64[3]; w.s = ctx->w64[4];
    w.t = ctx->w64[5]; w.ph = ctx->w64[6]; w.sh = ctx->w64[7];
    w.sc = ctx->sc64; w.n = (size_t)12 * ctx->geom.V * ctx->nrhs;
    return w;
}

// inner solve as the outer preconditioner: out64 ~= D^-1 in64
// hint: which scalar of the outer solver already holds |in64|^2 (1: bb, 2: ss), or 0: compute it (nrm)
static int inner_solve(wcras_ctx* ctx, const double2* in64, double2* out64, int hint, int* inner_iters, int* inner_solves) {
    const size_t V = ctx->geom.V;
    float4* b32 = ctx->w32[8];
    float4* x32 = ctx->w32[9];
    const double* nrm2 = hint == 1 ? &ctx->sc64->bb : hint == 2 ? &ctx->sc64->ss : &ctx->sc64->nrm;
    {
        TimedRegion tr(ctx, TC_BLAS);
        if (hint == 0) LAUNCH(k_norm2_d, (size_t)12 * V * ctx->nrhs, in64, ctx->sc64, ctx->partials, ctx->ticket);
        LAUNCH(k_d2f_init, V, ctx->nrhs, in64, b32, nrm2, ctx->sc32, ctx->partials, ctx->ticket);
    }
    // Tolerance of this inner solve (reading A2): the outer residual after this preconditioner call is
    // about (inner accuracy) x |in|, so the reduction still missing is R = target/|in|.  It is spread evenly over
    // the n = ceil(log R / log inner_tol) calls that are needed when no call may go deeper than inner_tol (the
    // accuracy fp32 can deliver), instead of solving every call to inner_tol and overshooting the target.
    if (int rc = read_scalars(ctx, ctx->sc64)) return rc;
    double itol = ctx->inner_tol;
    const double in_norm = std::sqrt(hint == 1 ? ctx->sc_host->bb : hint == 2 ? ctx->sc_host->ss : ctx->sc_host->nrm);
    if (ctx->outer_target > 0 && in_norm > 0) {
        const double R = 0.5 * ctx->outer_target / in_norm;
        if (R < 1.0) {
            const double n = std::ceil(std::log(R) / std::log(ctx->inner_tol) - 1e-9);
            itol = std::pow(R, 1.0 / (n < 1 ? 1 : n));
        } else {
            itol = 0.1;
        }
        if (itol < ctx->inner_tol) itol = ctx->inner_tol;
        if (itol > 0.1) itol = 0.1;
    }
    Work<float> w = work32(ctx);
    const bool use_ras = ctx->use_ras && ctx->ras.set;
    int it = 0;
    double rel = 0;
    auto K = [ctx](const float4* in, float4* out, int) { return ras_apply(ctx, in, out); };
    int rc = bicgstab<float>(ctx, w, b32, x32, itol, ctx->inner_maxit, true, !use_ras, K, &it, &rel, -2.0);
    *inner_iters += it;
    *inner_solves += 1;
    if (rc != WCRAS_OK && rc != WCRAS_NOT_CONVERGED && rc != WCRAS_BREAKDOWN) return rc;
    // an unconverged or broken-down inner solve is still a usable (flexible) preconditioner
    {
        TimedRegion tr(ctx, TC_BLAS);
        LAUNCH(k_f2d_scaled, V, ctx->nrhs, x32, out64, nrm2);
    }
    return WCRAS_OK;
}

// ctx->nrhs = 1: one system.  ctx->nrhs = N > 1 (wcras_solve_multi): the N systems D phi_k = eta_k
// are solved as ONE block-diagonal system diag(D,...,D) by the same nested BiCGStab on stacked vectors -- one set of
// Krylov scalars for the stack, links and clover loaded once per N spinors in the Dslash and in the block solver.
// Every eta_k is scaled to unit norm first so that all systems weigh equally, the stack is solved to tol/sqrt(N)
// (then |r_k| <= |r_stack| <= tol for every k), and the true residual of every system is checked on its own.
int solve(wcras_ctx* ctx, const double* eta_dev, double* phi_dev, double tol, wcras_info* info, double* resid_per_rhs) {
    if (int rc = ensure_workspace(ctx)) return rc;
    const int nr = ctx->nrhs;
    const size_t V = ctx->geom.V, n1 = 12 * V, n64 = n1 * nr;
    EventPair ev;
    WC_CUDA(ev.create());
    const cudaEvent_t e0 = ev.a, e1 = ev.b;
    WC_CUDA(cudaEventRecord(e0, ctx->stream));
    ctx->dv32 = ctx->dv64 = ctx->block_dv = ctx->ras_applies = 0;
    ctx->ev_used = 0;
    for (int k = 0; k < TC_COUNT; k++) ctx->ms_class[k] = 0;

    double2 *eta = ctx->w64[8], *phi = ctx->w64[9], *res = ctx->w64[10], *dx = ctx->w64[11];
    double norm_k[8], rel_k[8];
    double en2 = 0;
    for (int k = 0; k < nr; k++) {
        if (int rc = to_internal(ctx, 64, eta_dev + (size_t)k * 24 * V, eta + k * n1, ctx->sc64)) return rc;  // and |eta_k|^2
        if (int rc = read_scalars(ctx, ctx->sc64)) return rc;
        norm_k[k] = std::sqrt(ctx->sc_host->nrm);
        rel_k[k] = norm_k[k] > 0 ? 1.0 : 0.0;
        if (nr > 1 && norm_k[k] > 0) LAUNCH(k_scale_d, n1, eta + k * n1, 1.0 / norm_k[k]);
        en2 += nr > 1 ? (norm_k[k] > 0 ? 1.0 : 0.0) : ctx->sc_host->nrm;
    }
    const double tol_stack = nr > 1 ? tol / std::sqrt((double)nr) : tol;
    double rn2 = en2, recur = 1.0;
    int outer = 0, inner_iters = 0, inner_solves = 0, status = WCRAS_NOT_CONVERGED;
    if (en2 == 0.0) {  // zero source: phi = 0
        status = WCRAS_OK;
        WC_CUDA(cudaMemsetAsync(phi, 0, sizeof(double2) * n64, ctx->stream));
    }
    Work<double> w = work64(ctx);
    const bool spec = ctx->host_out != nullptr && nr == 1;  // see the pass loop
    bool spec_issued = false;
    auto K = [&](const double2* in, double2* out, int hint) { return inner_solve(ctx, in, out, hint, &inner_iters, &inner_solves); };
    for (int pass = 0; pass < 10 && status != WCRAS_OK && outer < ctx->outer_maxit; pass++) {
        int it = 0;
        double rel = 0;
        // solve D dx = res to relative accuracy tol*|eta|/|res| so that the total residual meets tol
        const double tol_pass = 0.7 * tol_stack * std::sqrt(en2 / rn2);
        ctx->outer_target = tol_pass * std::sqrt(rn2);  // absolute |r| this pass has to reach
        // pass 0: phi = 0 and res = eta, so the solver works on eta and writes phi directly; later passes solve
        // D dx = res for the correction and add it
        // |b|^2 is known (|eta|^2, then the norm of the true residual): no reduction pass to start the solver.  (Stacked
        // systems, pass 0: the unit norms of the scaled eta_k are exact only up to rounding, so it is computed.)
        const double bb = pass == 0 ? (nr == 1 ? en2 : -1.0) : rn2;
        int rc = pass == 0 ? bicgstab<double>(ctx, w, eta, phi, tol_pass, ctx->outer_maxit - outer, true, false, K, &it, &rel, bb)
                           : bicgstab<double>(ctx, w, res, dx, tol_pass, ctx->outer_maxit - outer, true, false, K, &it, &rel, bb);
        if (rc != WCRAS_OK && rc != WCRAS_NOT_CONVERGED && rc != WCRAS_BREAKDOWN) return rc;
        outer += it;
        recur = rel * std::sqrt(rn2 / en2);
        if (pass > 0) {
            TimedRegion tr(ctx, TC_BLAS);
            LAUNCH(k_add_d, n64, phi, dx);
        }
        if (spec) {
            // wcras_solve_host: this phi is final if its true residual passes the check below, so its way back to the host
            // (canonical layout, then the copy engine on the copy stream) starts now and runs beside the check.  A later
            // pass repeats this with the corrected phi, after the copy still in flight has finished reading phi_dev.
            if (spec_issued) WC_CUDA(cudaStreamWaitEvent(ctx->stream, ctx->ev_copy_done, 0));
            if (int r2 = from_internal(ctx, 64, phi, phi_dev)) return r2;
            WC_CUDA(cudaEventRecord(ctx->ev_copy_ready, ctx->stream));
        }
        // res = eta - D phi (true residual, fp64); one system: its norm comes out of the same kernel (DOT = 3)
        if (int r2 = dslash<double>(ctx, phi, res, eta, nr == 1 ? 3 : 0, nullptr, ctx->sc64)) return r2;
        if (spec) {  // (issued behind the launches of the check: a copy to pageable host memory may block the host)
            WC_CUDA(cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_copy_ready, 0));
            WC_CUDA(cudaMemcpyAsync(ctx->host_out, phi_dev, sizeof(double) * 24 * V, cudaMemcpyDeviceToHost, ctx->copy_stream));
            WC_CUDA(cudaEventRecord(ctx->ev_copy_done, ctx->copy_stream));
            spec_issued = true;
        }
        rn2 = 0;
        double worst = 0;
        bool nonfinite = false;
        for (int k = 0; k < nr; k++) {  // the true residual of every system on its own
            if (nr > 1) {
                TimedRegion tr(ctx, TC_BLAS);
                LAUNCH(k_norm2_d, n1, res + k * n1, ctx->sc64, ctx->partials, ctx->ticket);
            }
            if (int r3 = read_scalars(ctx, ctx->sc64)) return r3;
            const double nk = ctx->sc_host->nrm;
            rn2 += nk;
            const double ek = nr > 1 ? 1.0 : en2;  // |eta_k|^2 (unit after scaling)
            rel_k[k] = norm_k[k] > 0 ? std::sqrt(nk / ek) : 0.0;
            worst = rel_k[k] > worst ? rel_k[k] : worst;
            nonfinite = nonfinite || !std::isfinite(rel_k[k]);
        }
        if (nonfinite) { status = WCRAS_BREAKDOWN; break; }  // NaN / inf in the solution: never "converged" (a NaN compares false)
        if (worst <= tol) status = WCRAS_OK;
        else if (rc == WCRAS_BREAKDOWN) { status = WCRAS_BREAKDOWN; break; }
    }
    double worst = 0;
    for (int k = 0; k < nr; k++) {
        if (nr > 1 && norm_k[k] > 0) LAUNCH(k_scale_d, n1, phi + k * n1, norm_k[k]);
        if (!spec_issued) if (int rc = from_internal(ctx, 64, phi + k * n1, phi_dev + (size_t)k * 24 * V)) return rc;
        if (resid_per_rhs) resid_per_rhs[k] = rel_k[k];
        worst = rel_k[k] > worst || !std::isfinite(rel_k[k]) ? rel_k[k] : worst;
        if (!std::isfinite(rel_k[k])) break;  // reported as it is: a non-finite residual is never hidden behind a finite one
    }
    WC_CUDA(cudaEventRecord(e1, ctx->stream));
    if (spec_issued) {  // the caller's host buffer is receiving the final phi (ms_total does not include that copy, as before)
        WC_CUDA(cudaStreamWaitEvent(ctx->stream, ctx->ev_copy_done, 0));
        ctx->host_copied = true;
    }
    WC_CUDA(cudaStreamSynchronize(ctx->stream));
    float ms = 0;
    WC_CUDA(cudaEventElapsedTime(&ms, e0, e1));
    if (ctx->timing) {
        for (size_t k = 0; k + 1 < ctx->ev_used; k += 2) {
            float t = 0;
            cudaEventElapsedTime(&t, ctx->ev_pool[k], ctx->ev_pool[k + 1]);
            ctx->ms_class[ctx->ev_class[k]] += t;
        }
    }
    if (info) {
        info->outer_iters = outer; info->inner_iters = inner_iters; info->inner_solves = inner_solves;
        info->dv_fp32 = ctx->dv32; info->dv_fp64 = ctx->dv64; info->block_dv = ctx->block_dv;
        info->ras_applies = ctx->ras_applies; info->status = status;
        info->rel_resid_recur = recur; info->rel_resid_true = worst;
        info->ms_total = ms;
        info->ms_dslash = ctx->ms_class[TC_DSLASH]; info->ms_dslash64 = ctx->ms_class[TC_DSLASH64];
        info->ms_blocksolve = ctx->ms_class[TC_BLOCK]; info->ms_blas = ctx->ms_class[TC_BLAS];
    }
    if (status == WCRAS_NOT_CONVERGED) snprintf(ctx->err, sizeof ctx->err, "solve: not converged after %d outer iterations", outer);
    if (status == WCRAS_BREAKDOWN)
        snprintf(ctx->err, sizeof ctx->err, std::isfinite(worst) ? "solve: BiCGStab breakdown" : "solve: BiCGStab breakdown (non-finite residual)");
    return status;
}

int time_blas(wcras_ctx* ctx, int reps, double* ms) {
    if (int rc = ensure_workspace(ctx)) return rc;
    Work<float> w = work32(ctx);
    EventPair ev;
    WC_CUDA(ev.create());
    const cudaEvent_t e0 = ev.a, e1 = ev.b;
    WC_CUDA(cudaMemsetAsync(ctx->sc32, 0, sizeof(Scalars), ctx->stream));
    for (int k = 0; k < 8; k++) WC_CUDA(cudaMemsetAsync(ctx->w32[k], 0, sizeof(float4) * w.n, ctx->stream));
    WC_CUDA(cudaEventRecord(e0, ctx->stream));
    for (int k = 0; k < reps; k++)
        LAUNCH((k_update_xr<float, float4>), w.n, ctx->w32[9], w.ph, w.sh, w.s, w.t, w.rt, w.r, w.sc, ctx->partials, ctx->ticket, 0);
    WC_CUDA(cudaEventRecord(e1, ctx->stream));
    WC_CUDA(cudaStreamSynchronize(ctx->stream));
    float t = 0;
    WC_CUDA(cudaEventElapsedTime(&t, e0, e1));
    *ms = t / reps;
    return WCRAS_OK;
}

}  // namespace wc

TimedRegion::TimedRegion(wcras_ctx* c, int cls) : ctx(c), on(c->timing != 0) {
    if (!on) return;
    if (ctx->ev_used + 2 > ctx->ev_pool.size()) {
        for (int k = 0; k < 2; k++) {
            cudaEvent_t e;
            cudaEventCreate(&e);
            ctx->ev_pool.push_back(e);
            ctx->ev_class.push_back(cls);
        }
    }
    ctx->ev_class[ctx->ev_used] = cls;
    cudaEventRecord(ctx->ev_pool[ctx->ev_used], ctx->stream);
}
TimedRegion::~TimedRegion() {
    if (!on) return;
    cudaEventRecord(ctx->ev_pool[ctx->ev_used + 1], ctx->stream);
    ctx->ev_used += 2;
}
