// ras.cu -- steps A2-A5: the RAS preconditioner K_RAS (Alg. 1 :59-79, Eq. 2.1 :49-52).
//
// Domains (Q8): blocks of shape b tile the lattice, domain index lexicographic
// (x fastest); Omega'_i = block enlarged by s sites per side in every direction with b_mu < L_mu.
// Block solve (Q9): N_dominv MR iterations on D_Omega' v = P_Omega' r from v = 0, where
// D_Omega' is the principal sub-matrix of D on Omega' (hops leaving Omega' dropped; wrap-around hops that stay
// inside are kept, Q7).
//
// Tier 1 (this file, "generic"): domain-local vectors rho, q, v live in global memory as [domain][6][nloc]
// float4; one launch per MR half-step: (a) q = D_Omega' rho with the domain-local dots <q,rho>, <q,q>
// (block reduce + fp64 atomics per domain), (b) v += alpha rho, rho -= alpha q.  The projection P_Omega'
// (Alg.1 line 4) is fused into the first sweep (it reads the full-lattice r directly) and the restriction
// R_Omega (line 6) + sum (line 8) + phi += v (line 9) into the last update.  Works for every shape/overlap.
// Tier 2 (ras_fused.cu): one CTA per domain, everything on chip.
#include "blas.cuh"

namespace wc {

struct DomGeom {
    int b[4], ext[4], nblk[4], split[4];
    int s, nloc, nd;
};

__device__ __forceinline__ void domain_start(const Geom& g, const DomGeom& dg, int d, int start[4]) {
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        const int bc = d % dg.nblk[mu];
        d /= dg.nblk[mu];
        int st = bc * dg.b[mu] - (dg.split[mu] ? dg.s : 0);
        if (st < 0) st += g.L[mu];
        start[mu] = st;
    }
}

// q = D_Omega' rho for local site k of domain d; FIRST: rho is the full-lattice r (projection fused).
// Partial dots of CTA (d, chunk) go to scal[(d * nchunk + chunk) * sstride + 0..2] = <q,rho> (re, im), <q,q>.
// SECOND != 0 (second block solver, reading R2): the second application of a pair, q2 = D_Omega' q1 -- `rho` is
// then the q1 buffer, `q` the q2 buffer, and the partials go to slots 3..7 = <q2,q1> (re, im) = conj(a12), a22 = <q2,q2>,
// b2 = <q2,rho> (re, im) with the residual rho read from rho2 (SECOND = 1, domain-local) or from the full-lattice r
// (SECOND = 2, first pair: projection fused).
template <bool FIRST, int SECOND = 0>
__global__ void __launch_bounds__(128) mr_dslash_kernel(Geom g, DomGeom dg, Fields<float> f, float kappa, const float4* __restrict__ rglob,
                                                        const float4* __restrict__ rho, float4* __restrict__ q, double* __restrict__ scal,
                                                        int sstride, const float4* __restrict__ rho2) {
    static_assert(!(FIRST && SECOND), "the second application of a pair reads the domain-local q1");
    constexpr int NACC = SECOND ? 5 : 3;
    const int d = blockIdx.x;  // domain in gridDim.x (no 65535 limit), chunk of the domain in gridDim.y
    const int k = blockIdx.y * blockDim.x + threadIdx.x;
    double acc[NACC] = {};
    if (k < dg.nloc) {
        int start[4], c[4], x[4];
        domain_start(g, dg, d, start);
        {
            int kk = k;
            c[0] = kk % dg.ext[0]; kk /= dg.ext[0];
            c[1] = kk % dg.ext[1]; kk /= dg.ext[1];
            c[2] = kk % dg.ext[2];
            c[3] = kk / dg.ext[2];
        }
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            x[mu] = start[mu] + c[mu];
            if (x[mu] >= g.L[mu]) x[mu] -= g.L[mu];
        }
        const size_t V = g.V;
        const int i = x[0] + g.L[0] * (x[1] + g.L[1] * (x[2] + g.L[2] * x[3]));
        const int gs[4] = {1, g.L[0], g.L[0] * g.L[1], g.L[0] * g.L[1] * g.L[2]};
        const int ls[4] = {1, dg.ext[0], dg.ext[0] * dg.ext[1], dg.ext[0] * dg.ext[1] * dg.ext[2]};
        const float4* vin = FIRST ? rglob : rho + (size_t)d * 6 * dg.nloc;
        const size_t vstride = FIRST ? V : (size_t)dg.nloc;
        float hop[24];
#pragma unroll
        for (int n = 0; n < 24; n++) hop[n] = 0;
#define WC_MR_DIR(MU)                                                                                         \
    {                                                                                                         \
        const bool full = dg.ext[MU] == g.L[MU];                                                              \
        const bool kf = full || c[MU] + 1 < dg.ext[MU];                                                       \
        const bool kb = full || c[MU] > 0;                                                                    \
        const int gjb = x[MU] == 0 ? i + (g.L[MU] - 1) * gs[MU] : i - gs[MU];                                 \
        float u[18], sn[24];                                                                                  \
        if (kf) {                                                                                             \
            const int gjf = x[MU] + 1 == g.L[MU] ? i - (g.L[MU] - 1) * gs[MU] : i + gs[MU];                   \
            const int ljf = c[MU] + 1 == dg.ext[MU] ? k - (dg.ext[MU] - 1) * ls[MU] : k + ls[MU];             \
            load_link(f, V, i, MU, u);                                                                        \
            load_spinor(vin, vstride, FIRST ? gjf : ljf, sn);                                                 \
            hop_fwd<float, MU>(u, sn, hop);                                                                   \
        }                                                                                                     \
        if (kb) {                                                                                             \
            const int ljb = c[MU] == 0 ? k + (dg.ext[MU] - 1) * ls[MU] : k - ls[MU];                          \
            load_link(f, V, gjb, MU, u);                                                                      \
            load_spinor(vin, vstride, FIRST ? gjb : ljb, sn);                                                 \
            hop_bwd<float, MU>(u, sn, hop);                                                                   \
        }                                                                                                     \
    }
        WC_MR_DIR(0) WC_MR_DIR(1) WC_MR_DIR(2) WC_MR_DIR(3)
#undef WC_MR_DIR
        float sc[24], out[24];
        {
            float cl[72];
            load_spinor(vin, vstride, FIRST ? i : k, sc);
            load_clover(f, V, i, cl);
            clover_apply<float>(cl, sc, out);
        }
#pragma unroll
        for (int n = 0; n < 24; n++) out[n] -= kappa * hop[n];
        store_spinor(q + (size_t)d * 6 * dg.nloc, dg.nloc, k, out);
#pragma unroll
        for (int n = 0; n < 12; n++) {  // <q,rho> = sum conj(q) rho ; <q,q>
            const float qr = out[2 * n], qi = out[2 * n + 1], rr = sc[2 * n], ri = sc[2 * n + 1];
            acc[0] += (double)(qr * rr + qi * ri);
            acc[1] += (double)(qr * ri - qi * rr);
            acc[2] += (double)(qr * qr + qi * qi);
        }
        if (SECOND) {  // b2 = <q2,rho>
            float rt[24];
            if (SECOND == 2) load_spinor(rglob, V, i, rt);
            else load_spinor(rho2 + (size_t)d * 6 * dg.nloc, dg.nloc, k, rt);
#pragma unroll
            for (int n = 0; n < 12; n++) {
                const float qr = out[2 * n], qi = out[2 * n + 1], rr = rt[2 * n], ri = rt[2 * n + 1];
                acc[NACC - 2] += (double)(qr * rr + qi * ri);
                acc[NACC - 1] += (double)(qr * ri - qi * rr);
            }
        }
    }
    __shared__ double sm[NACC][4];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int n = 0; n < NACC; n++) {
        const double s = warp_sum(acc[n]);
        if (lane == 0) sm[n][w] = s;
    }
    __syncthreads();
    if (threadIdx.x < NACC) {  // one partial per CTA, summed in a fixed order by the update kernel (deterministic)
        double s = 0;
        for (int ww = 0; ww < (int)(blockDim.x >> 5); ww++) s += sm[threadIdx.x][ww];
        scal[((size_t)d * gridDim.y + blockIdx.y) * sstride + (SECOND ? 3 : 0) + threadIdx.x] = s;
    }
}

// v += alpha rho, rho -= alpha q; FIRST: rho_old = P r, v = alpha rho_old; LAST: no rho update and the
// restriction R_Omega: bulk sites go to the full-lattice vout (ACCUM: vout += v, Alg.1 line 9 phi += v)
template <bool FIRST, bool LAST, bool ACCUM>
__global__ void __launch_bounds__(128) mr_update_kernel(Geom g, DomGeom dg, const float4* __restrict__ rglob, float4* __restrict__ rho,
                                                        const float4* __restrict__ q, float4* __restrict__ v, float4* __restrict__ vout,
                                                        const double* __restrict__ scal) {
    const int d = blockIdx.x;
    const int k = blockIdx.y * blockDim.x + threadIdx.x;
    if (k >= dg.nloc) return;
    double qr = 0, qi = 0, qq = 0;
    for (unsigned c = 0; c < gridDim.y; c++) {  // the per-CTA partials of this domain, in order
        const double* p = scal + ((size_t)d * gridDim.y + c) * 4;
        qr += p[0]; qi += p[1]; qq += p[2];
    }
    // alpha = <q,rho>/<q,q>, 0 if <q,q> = 0 (Q9)
    const float ar = qq > 0 ? (float)(qr / qq) : 0.f, ai = qq > 0 ? (float)(qi / qq) : 0.f;
    int start[4], c[4], x[4];
    domain_start(g, dg, d, start);
    {
        int kk = k;
        c[0] = kk % dg.ext[0]; kk /= dg.ext[0];
        c[1] = kk % dg.ext[1]; kk /= dg.ext[1];
        c[2] = kk % dg.ext[2];
        c[3] = kk / dg.ext[2];
    }
    bool bulk = true;
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        x[mu] = start[mu] + c[mu];
        if (x[mu] >= g.L[mu]) x[mu] -= g.L[mu];
        if (dg.split[mu]) bulk = bulk && c[mu] >= dg.s && c[mu] < dg.s + dg.b[mu];
    }
    const size_t i = x[0] + g.L[0] * (x[1] + g.L[1] * (x[2] + (size_t)g.L[2] * x[3]));
    const size_t base = (size_t)d * 6 * dg.nloc + k;
#pragma unroll
    for (int ch = 0; ch < 6; ch++) {
        const size_t li = base + (size_t)ch * dg.nloc;
        const float4 rv = FIRST ? rglob[(size_t)ch * g.V + i] : rho[li];
        float4 vv = FIRST ? make_float4(0.f, 0.f, 0.f, 0.f) : v[li];
        vv.x += ar * rv.x - ai * rv.y; vv.y += ar * rv.y + ai * rv.x;
        vv.z += ar * rv.z - ai * rv.w; vv.w += ar * rv.w + ai * rv.z;
        if (!LAST) {
            const float4 qv = q[li];
            float4 rn;
            rn.x = rv.x - (ar * qv.x - ai * qv.y); rn.y = rv.y - (ar * qv.y + ai * qv.x);
            rn.z = rv.z - (ar * qv.z - ai * qv.w); rn.w = rv.w - (ar * qv.w + ai * qv.z);
            rho[li] = rn;
            v[li] = vv;
        } else if (bulk) {
            const size_t gi = (size_t)ch * g.V + i;
            if (ACCUM) {
                const float4 o = vout[gi];
                vv.x += o.x; vv.y += o.y; vv.z += o.z; vv.w += o.w;
            }
            vout[gi] = vv;
        }
    }
}

// Second block solver on the generic tier (reading R2; wcras_set_block_solver(1)): the update that closes a pair
// q1 = D_Omega' rho, q2 = D_Omega' q1.  (c1, c2) minimise |rho - c1 q1 - c2 q2| (2x2 normal equations in scale-free form:
// rows divided by a11 = <q1,q1> and a22 = <q2,q2>, g = |a12|^2 / (a11 a22); the plain MR step if 1 - g <= 1e-4 or a
// squared norm is 0); v += c1 rho + c2 q1, rho -= c1 q1 + c2 q2.  FIRST / LAST / ACCUM as in mr_update_kernel.  The dots
// arrive as per-CTA partials of 8 doubles: <q1,rho> (re, im), a11, <q2,q1> (re, im), a22, <q2,rho> (re, im).
template <bool FIRST, bool LAST, bool ACCUM>
__global__ void __launch_bounds__(128) mr2_update_kernel(Geom g, DomGeom dg, const float4* __restrict__ rglob, float4* __restrict__ rho,
                                                         const float4* __restrict__ q1, const float4* __restrict__ q2, float4* __restrict__ v,
                                                         float4* __restrict__ vout, const double* __restrict__ scal) {
    const int d = blockIdx.x;
    const int k = blockIdx.y * blockDim.x + threadIdx.x;
    if (k >= dg.nloc) return;
    double t[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (unsigned c = 0; c < gridDim.y; c++) {  // the per-CTA partials of this domain, in order
        const double* p = scal + ((size_t)d * gridDim.y + c) * 8;
#pragma unroll
        for (int n = 0; n < 8; n++) t[n] += p[n];
    }
    const double b1r = t[0], b1i = t[1], a11 = t[2], a12r = t[3], a12i = -t[4], a22 = t[5], b2r = t[6], b2i = t[7];  // a12 = conj(<q2,q1>)
    const double s1 = a11 > 0 ? 1.0 / a11 : 0.0, s2 = a22 > 0 ? 1.0 / a22 : 0.0;
    const double u1r = b1r * s1, u1i = b1i * s1, u2r = b2r * s2, u2i = b2i * s2;
    const double m1r = a12r * s1, m1i = a12i * s1, m2r = a12r * s2, m2i = -a12i * s2;  // a12 / a11, conj(a12) / a22
    const double gg = a11 > 0 && a22 > 0 ? m1r * m2r - m1i * m2i : 1.0;
    double c1r = u1r, c1i = u1i, c2r = 0, c2i = 0;  // q2 numerically parallel to q1, or rho = 0: the plain MR step
    if (1.0 - gg > 1e-4) {
        const double inv = 1.0 / (1.0 - gg);
        c1r = (u1r - (m1r * u2r - m1i * u2i)) * inv;
        c1i = (u1i - (m1r * u2i + m1i * u2r)) * inv;
        c2r = (u2r - (m2r * u1r - m2i * u1i)) * inv;
        c2i = (u2i - (m2r * u1i + m2i * u1r)) * inv;
    }
    const float ar = (float)c1r, ai = (float)c1i, br = (float)c2r, bi = (float)c2i;
    int start[4], c[4], x[4];
    domain_start(g, dg, d, start);
    {
        int kk = k;
        c[0] = kk % dg.ext[0]; kk /= dg.ext[0];
        c[1] = kk % dg.ext[1]; kk /= dg.ext[1];
        c[2] = kk % dg.ext[2];
        c[3] = kk / dg.ext[2];
    }
    bool bulk = true;
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        x[mu] = start[mu] + c[mu];
        if (x[mu] >= g.L[mu]) x[mu] -= g.L[mu];
        if (dg.split[mu]) bulk = bulk && c[mu] >= dg.s && c[mu] < dg.s + dg.b[mu];
    }
    const size_t i = x[0] + g.L[0] * (x[1] + g.L[1] * (x[2] + (size_t)g.L[2] * x[3]));
    const size_t base = (size_t)d * 6 * dg.nloc + k;
#pragma unroll
    for (int ch = 0; ch < 6; ch++) {
        const size_t li = base + (size_t)ch * dg.nloc;
        const float4 rv = FIRST ? rglob[(size_t)ch * g.V + i] : rho[li];
        const float4 xv = q1[li];
        float4 vv = FIRST ? make_float4(0.f, 0.f, 0.f, 0.f) : v[li];
        vv.x += ar * rv.x - ai * rv.y + br * xv.x - bi * xv.y; vv.y += ar * rv.y + ai * rv.x + br * xv.y + bi * xv.x;
        vv.z += ar * rv.z - ai * rv.w + br * xv.z - bi * xv.w; vv.w += ar * rv.w + ai * rv.z + br * xv.w + bi * xv.z;
        if (!LAST) {
            const float4 yv = q2[li];
            float4 rn;
            rn.x = rv.x - (ar * xv.x - ai * xv.y) - (br * yv.x - bi * yv.y); rn.y = rv.y - (ar * xv.y + ai * xv.x) - (br * yv.y + bi * yv.x);
            rn.z = rv.z - (ar * xv.z - ai * xv.w) - (br * yv.z - bi * yv.w); rn.w = rv.w - (ar * xv.w + ai * xv.z) - (br * yv.w + bi * yv.z);
            rho[li] = rn;
            v[li] = vv;
        } else if (bulk) {
            const size_t gi = (size_t)ch * g.V + i;
            if (ACCUM) {
                const float4 o = vout[gi];
                vv.x += o.x; vv.y += o.y; vv.z += o.z; vv.w += o.w;
            }
            vout[gi] = vv;
        }
    }
}

static DomGeom make_domgeom(const wcras_ctx* ctx) {
    DomGeom dg;
    for (int mu = 0; mu < 4; mu++) {
        dg.b[mu] = ctx->ras.b[mu]; dg.ext[mu] = ctx->ras.ext[mu]; dg.nblk[mu] = ctx->ras.nblk[mu];
        dg.split[mu] = ctx->ras.b[mu] < ctx->geom.L[mu];
    }
    dg.s = ctx->ras.s; dg.nloc = ctx->ras.nloc; dg.nd = ctx->ras.nd;
    return dg;
}

__global__ void __launch_bounds__(RED_THREADS) k_add_f(size_t n, float4* __restrict__ x, const float4* __restrict__ y) {
    for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (size_t)gridDim.x * blockDim.x) {
        float4 a = x[k];
        const float4 b = y[k];
        a.x += b.x; a.y += b.y; a.z += b.z; a.w += b.w;
        x[k] = a;
    }
}
int add_f(wcras_ctx* ctx, float4* x, const float4* y) {
    k_add_f<<<RED_BLOCKS, RED_THREADS, 0, ctx->stream>>>((size_t)6 * ctx->geom.V * ctx->nrhs, x, y);
    ctx->launches++;
    WC_CHECK_LAUNCH();
    return WCRAS_OK;
}

int ras_fused_prepare(const wcras_ctx* ctx, const int b[4], const int ext[4], int s, int niter, FusedGeom* out);
int ras_fused_block_solve(wcras_ctx* ctx, const float4* r, float4* vout, bool accum);
int ras_cta_prepare(wcras_ctx* ctx, const FusedGeom& fg, int nd);
int ras_cta_block_solve(wcras_ctx* ctx, const float4* r, float4* vout, bool accum);
int ras_cta_apply_chained(wcras_ctx* ctx, const float4* r, float4* v);
int ras_cta_apply_sap(wcras_ctx* ctx, const float4* r, float4* v);
int ras_fused_apply_chained(wcras_ctx* ctx, const float4* r, float4* v);
void ras_fused_pack(wcras_ctx* ctx, const FusedGeom& fg, int nd);
int ras_cta_sap_pdir(const FusedGeom& fg);
int ras_cta16_prepare(wcras_ctx* ctx, const FusedGeom& fg, int nd, const Fields<float>& f);
int ras_stream_prepare(wcras_ctx* ctx, const int b[4], const int ext[4], int s, int niter, FusedGeom* out);
int ras_stream_pack(wcras_ctx* ctx, const FusedGeom& fg, int nd, const Fields<float>& f);
int ras_stream_block_solve(wcras_ctx* ctx, const float4* r, float4* vout, bool accum);
int ras_round_fields(wcras_ctx* ctx);
int ras_cta16_block_solve(wcras_ctx* ctx, const float4* r, float4* vout, bool accum);
int ras_cta16_apply_chained(wcras_ctx* ctx, const float4* r, float4* v);
int ras_cta16_apply_sap(wcras_ctx* ctx, const float4* r, float4* v);
int ras_cl16_prepare(wcras_ctx* ctx, const FusedGeom& fg, int nd, const Fields<float>& f);
int ras_cl16_block_solve(wcras_ctx* ctx, const float4* r, float4* vout, bool accum);
int ras_cl16_apply_chained(wcras_ctx* ctx, const float4* r, float4* v);
int ras_pair_prepare(wcras_ctx* ctx, const FusedGeom& fg, int nd, const Fields<float>& f);
int ras_pair_block_solve(wcras_ctx* ctx, const float4* r, float4* vout, bool accum);
int ras_pair_apply_chained(wcras_ctx* ctx, const float4* r, float4* v);
int ras_pair_apply_sap(wcras_ctx* ctx, const float4* r, float4* v);

int ras_configure(wcras_ctx* ctx, const int domain[4], int s, int niter, int nras) {
    RasConfig rc;
    if (s < 0 || niter < 1 || nras < 1) { snprintf(ctx->err, sizeof ctx->err, "ras_precondition: need s>=0, block_iters>=1, nras>=1"); return WCRAS_INVALID_ARG; }
    rc.nd = 1; rc.nloc = 1;
    for (int mu = 0; mu < 4; mu++) {
        const int L = ctx->geom.L[mu], b = domain[mu];
        if (b < 1 || L % b) { snprintf(ctx->err, sizeof ctx->err, "ras_precondition: domain[%d]=%d does not divide %d", mu, b, L); return WCRAS_INVALID_ARG; }
        rc.b[mu] = b; rc.nblk[mu] = L / b;
        rc.ext[mu] = b < L ? b + 2 * s : L;
        if (rc.ext[mu] > L) { snprintf(ctx->err, sizeof ctx->err, "ras_precondition: domain[%d]+2*overlap=%d exceeds %d", mu, rc.ext[mu], L); return WCRAS_INVALID_ARG; }
        rc.nd *= rc.nblk[mu]; rc.nloc *= rc.ext[mu];
    }
    rc.s = s; rc.niter = niter; rc.nras = nras; rc.set = true;
    // from here on the buffers of the previous configuration are released: until the new one is complete the context has
    // no preconditioner (an allocation failure below leaves it that way, with the error message, instead of half of each)
    ctx->ras.set = false;
    ctx->cfg_gen++;  // captured inner-iteration graphs are stale
    FusedGeom fgeom;
    // tier request 5: force the streamed-operand cluster kernel (tier 2c); automatic: 2a/2b when Omega' fits on chip with
    // its operands, else 2c when the spinors fit a cluster, else the generic tier
    bool fused_ok = ctx->tier_request != 1 && ctx->tier_request != 5 && ras_fused_prepare(ctx, rc.b, rc.ext, s, niter, &fgeom) != 0;
    // The second block solver (reading R2) lives in the persistent one-CTA-per-domain kernel with 16-bit operand storage and
    // on the generic tier.  On the automatic tier a configuration the first cannot run (fp32 operands, an extended domain
    // above 256 sites) goes to the generic tier; a forced fused tier (requests 2..6) returns WCRAS_UNSUPPORTED below.
    if (ctx->block_solver == 1 && ctx->tier_request == 0 && !(fused_ok && ctx->op_prec == 16 && fgeom.C == 1 && fgeom.nsp <= FUSED_CTA_MAX_THREADS))
        fused_ok = false;
    const bool mr2_generic = ctx->block_solver == 1 && !fused_ok && ctx->tier_request <= 1;
    if (!fused_ok && !mr2_generic && (ctx->tier_request == 0 || ctx->tier_request == 5 || ctx->tier_request == 6) &&
        ras_stream_prepare(ctx, rc.b, rc.ext, s, niter, &fgeom) != 0) {
        fused_ok = true;
        rc.stream = true;
    }
    if (ctx->tier_request >= 2 && ctx->tier_request != 6 && !fused_ok) { snprintf(ctx->err, sizeof ctx->err, "ras_precondition: domain does not fit the fused tier"); return WCRAS_UNSUPPORTED; }
    rc.tier = (ctx->tier_request == 1 || !fused_ok) ? 1 : 2;
    if (int e = ensure_workspace(ctx)) return e;
    // 16-bit operand mode (reading R1): every path of the preconditioner sees the fp16-rounded links and clover blocks
    if (ctx->op_prec == 16) if (int e = ras_round_fields(ctx)) return e;
    // per-domain workspace of the generic tier (kept even when the fused tier is active: cheap to hold)
    if (ctx->mr_rho) {
        WC_CUDA(cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->mr_rho); cudaFree(ctx->mr_q); cudaFree(ctx->mr_v); cudaFree(ctx->mr_scal);
        if (ctx->mr_q2) cudaFree(ctx->mr_q2);
        ctx->mr_rho = ctx->mr_q = ctx->mr_v = ctx->mr_q2 = nullptr; ctx->mr_scal = nullptr;
    }
    if (rc.tier == 1) {
        const size_t nb = sizeof(float4) * 6 * (size_t)rc.nd * rc.nloc;
        WC_CUDA(cudaMalloc((void**)&ctx->mr_rho, nb));
        WC_CUDA(cudaMalloc((void**)&ctx->mr_q, nb));
        WC_CUDA(cudaMalloc((void**)&ctx->mr_v, nb));
        // [niter][nd][nchunk][4] per-CTA partial dots; the second block solver uses two iterations' worth per pair ([..][8])
        WC_CUDA(cudaMalloc((void**)&ctx->mr_scal, sizeof(double) * 4 * (size_t)rc.nd * ((rc.nloc + 127) / 128) * (niter + 1)));
        if (ctx->block_solver == 1) WC_CUDA(cudaMalloc((void**)&ctx->mr_q2, nb));
    }
    if (ctx->dm) {
        WC_CUDA(cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->dm);
        ctx->dm = nullptr;
    }
    if (ctx->dm16) {
        WC_CUDA(cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->dm16); cudaFree(ctx->rf_dm);
        ctx->dm16 = nullptr; ctx->rf_dm = nullptr;
    }
    if (rc.tier == 2 && rc.stream) {
        ctx->fused = fgeom;
        if (!ras_stream_pack(ctx, fgeom, rc.nd, ras_fields(ctx))) {
            snprintf(ctx->err, sizeof ctx->err, "ras_precondition: out of device memory for the streamed operand records");
            return WCRAS_CUDA_ERROR;
        }
    } else if (rc.tier == 2) {
        fgeom.pdir = ras_cta_sap_pdir(fgeom);
        ctx->fused = fgeom;
        rc.cta = ctx->tier_request != 3 && ras_cta_prepare(ctx, fgeom, rc.nd) != 0;  // tier request 3: force the cluster kernel
        // 16-bit operand mode: the staged fp16 kernel takes the single-right-hand-side work of this tier (its grid size
        // and halo geometry are those of ras_cta_prepare: same CTA shape, one CTA per SM)
        // (tier request 6: the two-threads-per-site variant ras_pair.cu instead -- measured slower, kept for comparison)
        rc.pair = rc.cta && ctx->op_prec == 16 && ctx->tier_request == 6 && ras_pair_prepare(ctx, fgeom, rc.nd, ras_fields(ctx)) != 0;
        fgeom.mr2 = ctx->block_solver == 1 ? 1 : 0;
        ctx->fused.mr2 = fgeom.mr2;
        rc.cta16 = rc.cta && ctx->op_prec == 16 && !rc.pair && ras_cta16_prepare(ctx, fgeom, rc.nd, ras_fields(ctx)) != 0;
        // 16-bit operand mode on the cluster tier: fp16 operands staged by TMA (ras_cl16.cu); otherwise ras_fused.cu
        rc.cl16 = !rc.cta && ctx->op_prec == 16 && fgeom.C > 1 && ras_cl16_prepare(ctx, fgeom, rc.nd, ras_fields(ctx)) != 0;
        if (!rc.cta && !rc.cl16) ras_fused_pack(ctx, ctx->fused, rc.nd);
        if (!rc.cta) {  // halo geometry of the chained cycles on the cluster tier (buffers allocated on first use)
            int nface = 1;
            for (int mu = 0; mu < 4; mu++) nface = rc.nloc / rc.ext[mu] > nface ? rc.nloc / rc.ext[mu] : nface;
            if (ctx->hb) { WC_CUDA(cudaStreamSynchronize(ctx->stream)); cudaFree(ctx->hb); ctx->hb = nullptr; }
            ctx->hb_nrhs = 0;
            ctx->nface = rc.cl16 ? fgeom.C * ctx->cl16_nfc : (nface + 7) / 8 * 8;  // ras_cl16: halo slots per CTA, [nd][C][8][3][nfc]
        }
    }
    if (ctx->block_solver == 1 && !rc.cta16 && rc.tier != 1) {
        // among the fused tiers the second block solver lives in the persistent one-CTA-per-domain kernel with 16-bit
        // operand storage only
        ctx->ras.set = false;
        snprintf(ctx->err, sizeof ctx->err,
                 "ras_precondition: on a forced fused tier block solver 1 (two-dimensional minimal residual) needs 16-bit operand "
                 "storage and an extended domain of at most 256 sites; the automatic and the generic tier take every shape");
        return WCRAS_UNSUPPORTED;
    }
    ctx->ras = rc;
    return WCRAS_OK;
}

// vout (+)= sum_i R_i MR_niter(D_Omega'_i, P_Omega'_i r)
static int generic_block_solve(wcras_ctx* ctx, const float4* r, float4* vout, bool accum) {
    const RasConfig& rc = ctx->ras;
    const DomGeom dg = make_domgeom(ctx);
    const int TH = 128;
    const int nchunk = (rc.nloc + TH - 1) / TH;
    const dim3 grid(rc.nd, nchunk);
    const Fields<float> f = ras_fields(ctx);
    const float kappa = (float)ctx->kappa;
    int it = 0;
    if (ctx->block_solver == 1) {
        // second block solver (reading R2): pairs of D_Omega' applications closed by the two-dimensional minimisation; an odd
        // N_dominv ends with one MR iteration (the loop below).  Partial dots: 8 doubles per (pair, domain, chunk).
        for (; it + 1 < rc.niter; it += 2) {
            double* scal = ctx->mr_scal + (size_t)it * rc.nd * nchunk * 4;  // [pair][nd][nchunk][8]
            const bool first = it == 0, last = it + 2 == rc.niter;
            if (first) {
                mr_dslash_kernel<true, 0><<<grid, TH, 0, ctx->stream>>>(ctx->geom, dg, f, kappa, r, ctx->mr_rho, ctx->mr_q, scal, 8, nullptr);
                mr_dslash_kernel<false, 2><<<grid, TH, 0, ctx->stream>>>(ctx->geom, dg, f, kappa, r, ctx->mr_q, ctx->mr_q2, scal, 8, nullptr);
            } else {
                mr_dslash_kernel<false, 0><<<grid, TH, 0, ctx->stream>>>(ctx->geom, dg, f, kappa, r, ctx->mr_rho, ctx->mr_q, scal, 8, nullptr);
                mr_dslash_kernel<false, 1><<<grid, TH, 0, ctx->stream>>>(ctx->geom, dg, f, kappa, r, ctx->mr_q, ctx->mr_q2, scal, 8, ctx->mr_rho);
            }
#define WC_UPD2(F, L, A) mr2_update_kernel<F, L, A><<<grid, TH, 0, ctx->stream>>>(ctx->geom, dg, r, ctx->mr_rho, ctx->mr_q, ctx->mr_q2, ctx->mr_v, vout, scal)
            if (first && last) { if (accum) WC_UPD2(true, true, true); else WC_UPD2(true, true, false); }
            else if (first) WC_UPD2(true, false, false);
            else if (last) { if (accum) WC_UPD2(false, true, true); else WC_UPD2(false, true, false); }
            else WC_UPD2(false, false, false);
#undef WC_UPD2
            ctx->launches += 3;
        }
    }
    for (; it < rc.niter; it++) {
        double* scal = ctx->mr_scal + (size_t)it * rc.nd * nchunk * 4;  // [niter][nd][nchunk][4] per-CTA partial dots
        const bool first = it == 0, last = it == rc.niter - 1;
        if (first) mr_dslash_kernel<true><<<grid, TH, 0, ctx->stream>>>(ctx->geom, dg, f, kappa, r, ctx->mr_rho, ctx->mr_q, scal, 4, nullptr);
        else mr_dslash_kernel<false><<<grid, TH, 0, ctx->stream>>>(ctx->geom, dg, f, kappa, r, ctx->mr_rho, ctx->mr_q, scal, 4, nullptr);
#define WC_UPD(F, L, A) mr_update_kernel<F, L, A><<<grid, TH, 0, ctx->stream>>>(ctx->geom, dg, r, ctx->mr_rho, ctx->mr_q, ctx->mr_v, vout, scal)
        if (first && last) { if (accum) WC_UPD(true, true, true); else WC_UPD(true, true, false); }
        else if (first) WC_UPD(true, false, false);
        else if (last) { if (accum) WC_UPD(false, true, true); else WC_UPD(false, true, false); }
        else WC_UPD(false, false, false);
#undef WC_UPD
        ctx->launches += 2;
    }
    WC_CHECK_LAUNCH();
    return WCRAS_OK;
}

static int block_solve(wcras_ctx* ctx, const float4* r, float4* vout, bool accum) {
    TimedRegion tr(ctx, TC_BLOCK);
    ctx->block_dv += ctx->ras.niter;
    const size_t rstride = (size_t)6 * ctx->geom.V;
    if (ctx->ras.tier == 2 && ctx->ras.pair && ctx->nrhs == 1) return ras_pair_block_solve(ctx, r, vout, accum);
    if (ctx->ras.tier == 2 && ctx->ras.cta16) {  // fp16 operand storage: the staged kernel, one right-hand side of the stack at a time
        for (int k = 0; k < ctx->nrhs; k++)
            if (int e = ras_cta16_block_solve(ctx, r + k * rstride, vout + k * rstride, accum)) return e;
        return WCRAS_OK;
    }
    if (ctx->ras.tier == 2 && ctx->ras.cta) return ras_cta_block_solve(ctx, r, vout, accum);  // handles the whole stack
    for (int k = 0; k < ctx->nrhs; k++) {  // cluster and generic tiers: one right-hand side of the stack at a time
        const int e = ctx->ras.tier == 2 ? (ctx->ras.stream ? ras_stream_block_solve(ctx, r + k * rstride, vout + k * rstride, accum)
                                            : ctx->ras.cl16 ? ras_cl16_block_solve(ctx, r + k * rstride, vout + k * rstride, accum)
                                                            : ras_fused_block_solve(ctx, r + k * rstride, vout + k * rstride, accum))
                                         : generic_block_solve(ctx, r + k * rstride, vout + k * rstride, accum);
        if (e) return e;
    }
    return WCRAS_OK;
}

int ras_block_solve(wcras_ctx* ctx, const float4* r, float4* v) { return block_solve(ctx, r, v, false); }

// v = K_RAS r  (Alg. 1).  phi = 0, r_0 = r; for j < NRAS: v_j = S r_j; phi += v_j; r_{j+1} = r_j - D v_j
// (the last residual update is dead and skipped, Q12).
int ras_apply(wcras_ctx* ctx, const float4* r, float4* v) {
    const RasConfig& rc = ctx->ras;
    if (!rc.set) { snprintf(ctx->err, sizeof ctx->err, "ras_apply: call wcras_ras_precondition first"); return WCRAS_INVALID_ARG; }
    ctx->ras_applies++;
    const size_t vstride = (size_t)6 * ctx->geom.V;  // stacked right-hand sides (wcras_solve_multi)
    if (ctx->schwarz == 1) {
        if (!(rc.tier == 2 && rc.cta && rc.s == 0 && ctx->fused.pdir >= 0)) {
            snprintf(ctx->err, sizeof ctx->err, "multiplicative Schwarz needs overlap 0, domains of <= 256 sites and an even number of blocks in every cut direction");
            return WCRAS_UNSUPPORTED;
        }
        if (rc.pair && ctx->nrhs == 1) return ras_pair_apply_sap(ctx, r, v);
        if (rc.cta16) {
            for (int k = 0; k < ctx->nrhs; k++)
                if (int e = ras_cta16_apply_sap(ctx, r + k * vstride, v + k * vstride)) return e;
            return WCRAS_OK;
        }
        return ras_cta_apply_sap(ctx, r, v);
    }
    if (rc.nras == 1) return block_solve(ctx, r, v, false);
    // overlap 0 on the persistent-CTA tier: chained cycles, the residual update is the boundary coupling only
    if (rc.tier == 2 && rc.pair && rc.s == 0 && ctx->chain_cycles && ctx->nrhs == 1) return ras_pair_apply_chained(ctx, r, v);
    if (rc.tier == 2 && rc.cta16 && rc.s == 0 && ctx->chain_cycles) {  // stacked right-hand sides: one after the other
        for (int k = 0; k < ctx->nrhs; k++)
            if (int e = ras_cta16_apply_chained(ctx, r + k * vstride, v + k * vstride)) return e;
        return WCRAS_OK;
    }
    if (rc.tier == 2 && rc.cta && rc.s == 0 && ctx->chain_cycles) return ras_cta_apply_chained(ctx, r, v);
    if (rc.tier == 2 && rc.cl16 && rc.s == 0 && ctx->chain_cycles) {
        for (int k = 0; k < ctx->nrhs; k++)
            if (int e = ras_cl16_apply_chained(ctx, r + k * vstride, v + k * vstride)) return e;
        return WCRAS_OK;
    }
    if (rc.tier == 2 && !rc.cta && !rc.stream && rc.s == 0 && ctx->chain_cycles && ctx->nrhs == 1) return ras_fused_apply_chained(ctx, r, v);
    float4* rw = ctx->ras32[0];
    float4* vj = ctx->ras32[1];
    const float4* rcur = r;
    // 16-bit operand mode: Alg.1 line 9 uses the same rounded operator as the block solves (reading R1)
    struct RoundedScope {
        wcras_ctx* c;
        explicit RoundedScope(wcras_ctx* cc) : c(cc) { c->dslash_rounded = c->op_prec == 16; }
        ~RoundedScope() { c->dslash_rounded = 0; }
    } rounded_scope(ctx);
    for (int j = 0; j < rc.nras; j++) {
        // v_j is needed on its own for r -= D v_j, so only the last cycle accumulates straight into phi
        const bool lastc = j == rc.nras - 1;
        if (j == 0) {
            if (int e = block_solve(ctx, rcur, v, false)) return e;
            if (!lastc) if (int e = dslash<float>(ctx, v, rw, rcur)) return e;  // rw = r - D v_0
        } else if (lastc) {
            if (int e = block_solve(ctx, rcur, v, true)) return e;  // phi += v_j fused
        } else {
            if (int e = block_solve(ctx, rcur, vj, false)) return e;
            if (int e = dslash<float>(ctx, vj, rw, rcur)) return e;  // in-place: rw = rw - D v_j
            TimedRegion tr(ctx, TC_BLAS);
            if (int e = add_f(ctx, v, vj)) return e;  // phi += v_j
        }
        rcur = rw;
    }
    return WCRAS_OK;
}

}  // namespace wc
