// ras_cta.cu -- tier 2a of the RAS block solver (north_star (c)): extended domains of at most 256 sites, one CTA
// per domain, PERSISTENT: each CTA walks over domains dom = blockIdx.x, blockIdx.x + gridDim.x, ... and, while it
// runs the MR sweeps of one domain on chip, the data of its next domain is pulled from HBM into L2
// (cp.async.bulk.prefetch.L2 on the contiguous domain-major block + prefetch.global.L2 on the residual rows), so
// HBM streams continuously behind the arithmetic.  Steps A2-A4 of SURVEY.md 8(a): projection P_Omega' r
// (Alg.1 line 4), N_dominv MR iterations on D_Omega' v = P r with Dirichlet boundaries (PAPER.md:68,
// :83; readings Q7, Q9), restriction R_Omega and the disjoint sum, optionally phi += v (line 9).
//
//   * Domain-major operand copy (built once in wcras_ras_precondition): dm = float4 [nd][36][nsp]; chunks 0..17 are
//     the 72 reals of the four forward links of the site PRE-SCALED by -kappa, chunks 18..35 the packed clover
//     blocks.  Thread k reads dm[(dom*36 + c)*nsp + k]: 4 KB contiguous per chunk, 147 KB contiguous per domain.
//     This is the paper's "overlapped region data is replicated per domain" applied to the operands.
//   * Per thread, in registers for the whole block solve: -kappa U_mu(x) (72), A(x) (72), rho(x), v(x) (24 + 24).
//   * Per MR iteration: scatter 8 projected half spinors (backward ones pre-multiplied by -kappa U^dag) into the
//     neighbour's slot in shared memory, q = A rho, barrier, gather the own 8 slots (forward ones multiplied by
//     -kappa U) straight onto q.  Slots of neighbours outside Omega' are never written and stay zero = Dirichlet.
//   * <q,rho>, <q,q>: warp shuffle -> one float4 per warp in shared memory -> fixed-order sum by every thread.
// Shared memory: 8 x 3 float4 x nsp half-spinor slots (96 KB at nsp = 256) + nwarps float4.
// Roofline: HBM, (96 + 576) B per extended site in + 96 B per bulk site out (768 B/site at s = 0); the sweeps
// cost ~1.4 k fp32 instructions per site each and must hide behind that stream.
// This kernel sits at the 255-register limit with fp32 operands (links in registers, 36-real clover blocks unpacked from
// shared memory): the aligned register pairs of the packed-fp32 arithmetic (site_math.cuh, WC_X2) make it spill
// (~500 B per thread, measured 12.3 -> 17.2 ms per solve), so this translation unit keeps the scalar FFMA forms.
#define WC_NO_F32X2
#include "ras_cta_common.cuh"

namespace wc {

// pack the domain-major operand copy: one thread per (domain, local site)
__global__ void pack_domain_major_kernel(FusedGeom fg, int nd, Fields<float> f, float mkappa, float4* __restrict__ dm) {
    const int dom = blockIdx.x, k = threadIdx.x;
    if (dom >= nd) return;
    float4* out = dm + (size_t)dom * 36 * fg.nsp + k;
    if (k >= fg.ns) {
        for (int c = 0; c < 36; c++) out[(size_t)c * fg.nsp] = make_float4(0.f, 0.f, 0.f, 0.f);
        return;
    }
    int lc[4], kk = k;
#pragma unroll
    for (int mu = 0; mu < 4; mu++) { lc[mu] = kk % fg.ext[mu]; kk /= fg.ext[mu]; }
    const size_t gi = cta_site(fg, dom, lc), V = fg.V;
    float u[72];
#pragma unroll
    for (int mu = 0; mu < 4; mu++) load_link(f, V, gi, mu, u + 18 * mu);
#pragma unroll
    for (int c = 0; c < 18; c++)
        out[(size_t)c * fg.nsp] = make_float4(mkappa * u[4 * c], mkappa * u[4 * c + 1], mkappa * u[4 * c + 2], mkappa * u[4 * c + 3]);
#pragma unroll
    for (int c = 0; c < 18; c++) out[(size_t)(18 + c) * fg.nsp] = f.cl[(size_t)c * V + gi];
}

// One K_RAS cycle (Alg.1 lines 3-9) for all domains.  Cycle 0: rho = P r.  Cycles j >= 1 (CHAIN, overlap 0 only):
// the MR recurrence of cycle j-1 left rho_fin = r_{j-1} - D_Omega v_{j-1} on every domain, so the residual update of
// Alg.1 line 9, r_j = r_{j-1} - D v_{j-1}, is rho_fin minus the hops of v_{j-1} that CROSS a domain boundary:
// no full-lattice D is applied between two cycles, only the boundary coupling, which is the data the paper
// exchanges between GPUs in T_Dv^comm.  The coupling travels as projected half spinors through a
// global halo buffer hb = float4 [nd][8 slots][3][nface], the continuation of the shared-memory slots across the
// domain boundary: a site on the lower mu-face sends P^-_mu v to slot 2mu of the domain at -mu, a site on the
// upper face sends (-kappa U_mu)^dag P^+_mu v to slot 2mu+1 of the domain at +mu (48 B per crossing hop).
//   r_src   residual source read at the own site: r (cycle 0) or rho_fin of the previous cycle
//   hb_in   CHAIN: halo slots of this domain, filled by its neighbours in the previous cycle
//   hb_out  halo buffer the final v of this cycle is scattered into (other parity), or nullptr
//   phi_in  own-site value added to v before the store (phi += v, Alg.1 line 9), or nullptr
//   phi_out where R_Omega (v [+ phi_in]) is stored
//   rho_out rho_fin of this cycle, or nullptr (then the last MR residual update is skipped, Q12)
template <bool CHAIN, bool MULTI>
__global__ void __launch_bounds__(FUSED_CTA_MAX_THREADS, 1)
ras_cta_kernel(FusedGeom fg, int ndl, int colour, int nface, const float4* __restrict__ dm, const float4* r_src,
               const float4* __restrict__ hb_in, float4* __restrict__ hb_out, const float4* phi_in, float4* phi_out,
               float4* rho_out, int nrhs, size_t rstride, size_t hstride) {
    // r_src and rho_out are the same buffer in the chained cycles (a thread reads its site before it writes it): no __restrict__
    // nrhs > 1 (wcras_solve_multi): every vector argument is a stack of nrhs vectors rstride apart (halo buffers:
    // hstride); the right-hand sides of a domain are solved one after the other with the operands loaded once
    if (fg.stop && __ldg(fg.stop)) return;  // the inner solver has converged (launch enqueued ahead of the host's check)
    extern __shared__ float4 smem[];
    const int nsp = fg.nsp;
    float4* hbuf = smem;            // [8][3][nsp]
    float4* As = smem + 24 * nsp;   // [18][nsp] clover blocks of the current domain (each thread reads back its own column)
    float4* red = smem + 42 * nsp;  // [nwarps]
    const int k = threadIdx.x, lane = k & 31, warp = k >> 5, nwarps = blockDim.x >> 5;
    const bool active = k < fg.ns;

    // ---- domain-independent geometry: local coordinates, bulk flag, destination slots ----
    int lc[4];
    bool bulk = active;
    {
        int kk = active ? k : 0;
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            lc[mu] = kk % fg.ext[mu]; kk /= fg.ext[mu];
            if (fg.split[mu]) bulk = bulk && lc[mu] >= fg.s && lc[mu] < fg.s + fg.b[mu];
        }
    }
    const unsigned chunk_bytes = (unsigned)nsp * 16u;
    unsigned dst[8];  // slot 2mu: receiver x-mu (its forward hop); slot 2mu+1: receiver x+mu (its backward hop)
    int fidx[4];      // index of the site within the mu-face (local index with coordinate mu removed)
    {
        const unsigned base = cta_smem_u32(hbuf);
        int lstride = 1;
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            const int e = fg.ext[mu];
            fidx[mu] = (k % lstride) + (k / (lstride * e)) * lstride;
            int kd = k - lstride;
            bool ok = active;
            if (lc[mu] == 0) { kd = k + (e - 1) * lstride; ok = ok && fg.wrap[mu]; }
            dst[2 * mu] = ok ? base + (unsigned)((2 * mu) * 3 * nsp + kd) * 16u : 0xffffffffu;
            kd = k + lstride;
            ok = active;
            if (lc[mu] + 1 == e) { kd = k - (e - 1) * lstride; ok = ok && fg.wrap[mu]; }
            dst[2 * mu + 1] = ok ? base + (unsigned)((2 * mu + 1) * 3 * nsp + kd) * 16u : 0xffffffffu;
            lstride *= e;
        }
    }
#pragma unroll
    for (int j = 0; j < 24; j++) hbuf[j * nsp + k] = make_float4(0.f, 0.f, 0.f, 0.f);
    __syncthreads();

    const size_t V = fg.V;
    const unsigned dm_bytes = 36u * (unsigned)nsp * 16u;
    // clover blocks: global -> shared with cp.async, into the thread's own column (only the owner reads it back, so
    // no barrier is involved); the copy for the NEXT domain is issued right after the last use in the current one
    const int dom0 = launch_dom(fg, blockIdx.x, colour);
    if ((int)blockIdx.x < ndl) {
        const float4* p0 = dm + ((size_t)dom0 * 36 + 18) * nsp + k;
#pragma unroll
        for (int c = 0; c < 18; c++) cp_async16(As + c * nsp + k, p0 + (size_t)c * nsp);
        cp_async_commit();
    }
    float U[72];
#define WC_LOAD_U(DOM)                                                                            \
    {                                                                                             \
        const float4* pu = dm + (size_t)(DOM) * 36 * nsp + k;                                     \
        for (int c = 0; c < 18; c++) {                                                            \
            const float4 t = __ldcs(pu + (size_t)c * nsp);                                        \
            U[4 * c] = t.x; U[4 * c + 1] = t.y; U[4 * c + 2] = t.z; U[4 * c + 3] = t.w;           \
        }                                                                                         \
    }
    if ((int)blockIdx.x < ndl) {
#pragma unroll
        WC_LOAD_U(dom0)
    }
    // Work items of this CTA: (domain, right-hand side) pairs, the nr right-hand sides of a domain one after the other
    // with the operands (links in registers, clover in shared memory) loaded once.  MULTI = false is the
    // single-right-hand-side instantiation: nr = 1 and the offsets fold away (the kernel sits at the 255-register limit).
    const int nr = MULTI ? nrhs : 1;
    for (int j = 0;; j++) {
        const int h = blockIdx.x + (j / nr) * gridDim.x;
        if (h >= ndl) break;
        const int rr = MULTI ? j % nr : 0;
        const bool last_rhs = rr + 1 == nr;                     // the next item is a new domain (or the end)
        const bool has_next = last_rhs ? h + (int)gridDim.x < ndl : true;
        const int dom = launch_dom(fg, h, colour);
        const int nxt = last_rhs ? launch_dom(fg, has_next ? h + gridDim.x : h, colour) : dom;  // domain of the next item
        const int rrn = last_rhs ? 0 : rr + 1;
        const size_t gi = cta_site(fg, dom, lc);
        bool u_early = false;  // links of the next domain already requested in the last sweep of this one
      {
        const size_t roff = MULTI ? rr * rstride : 0, hoff = MULTI ? rr * hstride : 0;
#define r_src_r (r_src + roff)
#define hb_in_r (hb_in + hoff)
#define hb_out_r (hb_out + hoff)
#define phi_out_r (phi_out + roff)
#define rho_out_r (rho_out + roff)
        float rho[24], v[24];
        if (active) {
#pragma unroll
            for (int c = 0; c < 6; c++) {
                const float4 t = r_src_r[(size_t)c * V + gi];
                rho[4 * c] = t.x; rho[4 * c + 1] = t.y; rho[4 * c + 2] = t.z; rho[4 * c + 3] = t.w;
            }
        } else {
#pragma unroll
            for (int n = 0; n < 24; n++) rho[n] = 0.f;
        }
        if (CHAIN) {
            // ---- boundary coupling: rho -= D-terms of v_{j-1} that cross the domain boundary.  A lane whose
            // in-domain slot 2mu+1 (2mu) has no receiver sits on the upper (lower) face and receives the
            // outside forward (backward) hop from halo slot 2mu (2mu+1).  All loads are issued first. ----
            const float4* hin = hb_in_r + (size_t)dom * 24 * nface;
            float hh[8][12];
#pragma unroll
            for (int sl = 0; sl < 8; sl++) {
                const bool rcv = active && dst[sl ^ 1] == 0xffffffffu;
                const float4* q4 = hin + (size_t)sl * 3 * nface + fidx[sl >> 1];
#pragma unroll
                for (int j = 0; j < 3; j++) {
                    float4 t = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (rcv) t = __ldcs(q4 + (size_t)j * nface);
                    hh[sl][4 * j] = t.x; hh[sl][4 * j + 1] = t.y; hh[sl][4 * j + 2] = t.z; hh[sl][4 * j + 3] = t.w;
                }
            }
            // a warp none of whose lanes sits on the face in question skips that hop (z and t faces are warp-uniform
            // for x-fastest local indices)
            float g[12];
#define WC_CROSS(MU)                                                                              \
    if (__any_sync(0xffffffffu, active && dst[2 * MU + 1] == 0xffffffffu)) {                      \
        su3_mul<float>(U + 18 * MU, hh[2 * MU], g);                                               \
        reconstruct_sub<float, MU, -1>(g, rho);                                                   \
    }                                                                                             \
    if (__any_sync(0xffffffffu, active && dst[2 * MU] == 0xffffffffu))                            \
        reconstruct_sub<float, MU, +1>(hh[2 * MU + 1], rho);
            WC_CROSS(0) WC_CROSS(1) WC_CROSS(2) WC_CROSS(3)
#undef WC_CROSS
        }
        // ---- pull the next domain of this CTA towards L2 while this one is solved ----
        {
            if (has_next) {
                const size_t roffn = MULTI ? rrn * rstride : 0, hoffn = MULTI ? rrn * hstride : 0;
                if (k == 0 && last_rhs) prefetch_l2_bulk(dm + (size_t)nxt * 36 * nsp, dm_bytes);
                if (CHAIN && k == 32) prefetch_l2_bulk(hb_in + hoffn + (size_t)nxt * 24 * nface, 24u * (unsigned)nface * 16u);
                if (active) {
                    const size_t gn = cta_site(fg, nxt, lc);
#pragma unroll
                    for (int c = 0; c < 6; c++) prefetch_l2(r_src + roffn + (size_t)c * V + gn);
                }
            }
        }
#pragma unroll
        for (int n = 0; n < 24; n++) v[n] = 0.f;

        for (int it = 0; it < fg.niter; it++) {
            {
                float h[12], g[12];
#define WC_SCATTER(MU)                                       \
    project<float, MU, -1>(rho, h);                          \
    st_half_pred(dst[2 * MU], chunk_bytes, h);               \
    project<float, MU, +1>(rho, h);                          \
    su3_adj_mul<float>(U + 18 * MU, h, g);                   \
    st_half_pred(dst[2 * MU + 1], chunk_bytes, g);
                WC_SCATTER(0) WC_SCATTER(1) WC_SCATTER(2) WC_SCATTER(3)
#undef WC_SCATTER
            }
            float q[24];
            if (it == 0) cp_async_wait();
#pragma unroll
            for (int ch = 0; ch < 2; ch++) {
                float Ab[36];
#pragma unroll
                for (int c = 0; c < 9; c++) {
                    const float4 t = As[(9 * ch + c) * nsp + k];
                    Ab[4 * c] = t.x; Ab[4 * c + 1] = t.y; Ab[4 * c + 2] = t.z; Ab[4 * c + 3] = t.w;
                }
                herm6_mul<float>(Ab, rho + 12 * ch, q + 12 * ch);
            }
            if (it + 1 == fg.niter && has_next && last_rhs) {
                const float4* pn = dm + ((size_t)nxt * 36 + 18) * nsp + k;
#pragma unroll
                for (int c = 0; c < 18; c++) cp_async16(As + c * nsp + k, pn + (size_t)c * nsp);
                cp_async_commit();
            }
            __syncthreads();
            {
                float h[12], g[12];
#define WC_GATHER(MU)                                        \
    ld_half_cta(hbuf + (2 * MU) * 3 * nsp + k, nsp, h);      \
    su3_mul<float>(U + 18 * MU, h, g);                       \
    reconstruct_add<float, MU, -1>(g, q);                    \
    ld_half_cta(hbuf + (2 * MU + 1) * 3 * nsp + k, nsp, g);  \
    reconstruct_add<float, MU, +1>(g, q);
                WC_GATHER(0) WC_GATHER(1) WC_GATHER(2) WC_GATHER(3)
#undef WC_GATHER
            }
            // the links are dead after the last gather unless the halo scatter still needs them: request those of
            // the next domain now, their latency hides behind the dots, the update and the stores
            if (it + 1 == fg.niter && hb_out == nullptr && has_next && last_rhs) {
#pragma unroll
                WC_LOAD_U(nxt)
                u_early = true;
            }
            float d0 = 0.f, d1 = 0.f, d2 = 0.f;
#pragma unroll
            for (int n = 0; n < 12; n++) {
                const float qr = q[2 * n], qi = q[2 * n + 1], rr = rho[2 * n], ri = rho[2 * n + 1];
                d0 = fmaf(qr, rr, d0); d0 = fmaf(qi, ri, d0);
                d1 = fmaf(qr, ri, d1); d1 = fmaf(-qi, rr, d1);
                d2 = fmaf(qr, qr, d2); d2 = fmaf(qi, qi, d2);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                d0 += __shfl_xor_sync(0xffffffffu, d0, o);
                d1 += __shfl_xor_sync(0xffffffffu, d1, o);
                d2 += __shfl_xor_sync(0xffffffffu, d2, o);
            }
            if (lane == 0) red[warp] = make_float4(d0, d1, d2, 0.f);
            __syncthreads();
            float s0 = 0.f, s1 = 0.f, s2 = 0.f;
            for (int n = 0; n < nwarps; n++) {
                const float4 p = red[n];
                s0 += p.x; s1 += p.y; s2 += p.z;
            }
            // alpha = <q,rho>/<q,q>, 0 if <q,q> = 0 (Q9); v += alpha rho; rho -= alpha q
            const float inv = s2 > 0.f ? 1.f / s2 : 0.f;
            const float ar = s0 * inv, ai = s1 * inv;
            const bool upd_rho = it + 1 < fg.niter || rho_out != nullptr;
#pragma unroll
            for (int n = 0; n < 12; n++) {
                const float rr = rho[2 * n], ri = rho[2 * n + 1];
                v[2 * n] = fmaf(ar, rr, v[2 * n]); v[2 * n] = fmaf(-ai, ri, v[2 * n]);
                v[2 * n + 1] = fmaf(ar, ri, v[2 * n + 1]); v[2 * n + 1] = fmaf(ai, rr, v[2 * n + 1]);
                if (upd_rho) {
                    rho[2 * n] = fmaf(-ar, q[2 * n], rr); rho[2 * n] = fmaf(ai, q[2 * n + 1], rho[2 * n]);
                    rho[2 * n + 1] = fmaf(-ar, q[2 * n + 1], ri); rho[2 * n + 1] = fmaf(-ai, q[2 * n], rho[2 * n + 1]);
                }
            }
        }
        // ---- halo scatter for the next cycle: the hops of v that leave the domain, as projected half spinors ----
        if (hb_out) {
            int dd = dom, dstride = 1;
            float h[12], g[12];
#define WC_HALO(MU)                                                                                              \
    {                                                                                                            \
        const int nb = fg.nblk[MU], bc = dd % nb;                                                                \
        dd /= nb;                                                                                                \
        if (active && dst[2 * MU] == 0xffffffffu) { /* lower face -> slot 2mu of the domain at -mu */            \
            const int nbd = bc == 0 ? dom + (nb - 1) * dstride : dom - dstride;                                  \
            float4* o = hb_out_r + ((size_t)nbd * 8 + 2 * MU) * 3 * nface + fidx[MU];                            \
            project<float, MU, -1>(v, h);                                                                        \
            for (int j = 0; j < 3; j++) o[(size_t)j * nface] = make_float4(h[4 * j], h[4 * j + 1], h[4 * j + 2], h[4 * j + 3]); \
        }                                                                                                        \
        if (active && dst[2 * MU + 1] == 0xffffffffu) { /* upper face -> slot 2mu+1 of the domain at +mu */      \
            const int nbd = bc + 1 == nb ? dom - (nb - 1) * dstride : dom + dstride;                             \
            float4* o = hb_out_r + ((size_t)nbd * 8 + 2 * MU + 1) * 3 * nface + fidx[MU];                        \
            project<float, MU, +1>(v, h);                                                                        \
            su3_adj_mul<float>(U + 18 * MU, h, g);                                                               \
            for (int j = 0; j < 3; j++) o[(size_t)j * nface] = make_float4(g[4 * j], g[4 * j + 1], g[4 * j + 2], g[4 * j + 3]); \
        }                                                                                                        \
        dstride *= nb;                                                                                           \
    }
            WC_HALO(0) WC_HALO(1) WC_HALO(2) WC_HALO(3)
#undef WC_HALO
        }
        // ---- restriction R_Omega: bulk sites only; disjoint over domains, so a plain store (or phi += v) ----
        if (bulk) {
            if (rho_out) {
#pragma unroll
                for (int c = 0; c < 6; c++)
                    __stcs(rho_out_r + (size_t)c * V + gi, make_float4(rho[4 * c], rho[4 * c + 1], rho[4 * c + 2], rho[4 * c + 3]));
            }
            if (phi_in) {
                // phi += v as a fire-and-forget vector reduction (phi_in == phi_out; one writer per site, so the
                // result is the same single rounding as load-add-store, without waiting for the load)
#pragma unroll
                for (int c = 0; c < 6; c++)
                    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(phi_out_r + (size_t)c * V + gi), "f"(v[4 * c]),
                                 "f"(v[4 * c + 1]), "f"(v[4 * c + 2]), "f"(v[4 * c + 3])
                                 : "memory");
            } else {
#pragma unroll
                for (int c = 0; c < 6; c++)
                    phi_out_r[(size_t)c * V + gi] = make_float4(v[4 * c], v[4 * c + 1], v[4 * c + 2], v[4 * c + 3]);
            }
        }
      }  // right-hand sides of this domain
#undef r_src_r
#undef hb_in_r
#undef hb_out_r
#undef phi_out_r
#undef rho_out_r
        if (!u_early && has_next && last_rhs) {
#pragma unroll
            WC_LOAD_U(nxt)
        }
    }
#undef WC_LOAD_U
}

// ---- host side ----
typedef void (*cta_kernel_t)(FusedGeom, int, int, int, const float4*, const float4*, const float4*, float4*, const float4*, float4*,
                             float4*, int, size_t, size_t);
static cta_kernel_t cta_kernel(bool chain, bool multi) {
    if (chain) return multi ? ras_cta_kernel<true, true> : ras_cta_kernel<true, false>;
    return multi ? ras_cta_kernel<false, true> : ras_cta_kernel<false, false>;
}
static size_t cta_smem_bytes(const FusedGeom& fg) { return sizeof(float4) * ((size_t)42 * fg.nsp + fg.nsp / 32); }

// allocate and fill the domain-major operand copy; sets ctx->dm and the persistent grid size
int ras_cta_prepare(wcras_ctx* ctx, const FusedGeom& fg, int nd) {
    if (fg.C != 1 || fg.nsp > FUSED_CTA_MAX_THREADS) return 0;
    const size_t smem = cta_smem_bytes(fg);
    if (cudaFuncSetAttribute(ras_cta_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
        cudaFuncSetAttribute(ras_cta_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
        cudaFuncSetAttribute(ras_cta_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
        cudaFuncSetAttribute(ras_cta_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    int per_sm = 0, per_sm_chain = 0, dev = 0, sms = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ras_cta_kernel<false, false>, fg.nsp, smem) != cudaSuccess || per_sm < 1 ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm_chain, ras_cta_kernel<true, true>, fg.nsp, smem) != cudaSuccess ||
        per_sm_chain < 1) {
        cudaGetLastError();
        return 0;
    }
    if (per_sm_chain < per_sm) per_sm = per_sm_chain;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (ctx->dm) { cudaStreamSynchronize(ctx->stream); cudaFree(ctx->dm); ctx->dm = nullptr; }
    const size_t bytes = sizeof(float4) * 36 * (size_t)fg.nsp * nd;
    if (cudaMalloc((void**)&ctx->dm, bytes) != cudaSuccess) { cudaGetLastError(); ctx->dm = nullptr; return 0; }
    // face size of the halo buffers of the chained cycles (allocated on first use, ensure_halo)
    int nface = 1;
    for (int mu = 0; mu < 4; mu++) nface = fg.ns / fg.ext[mu] > nface ? fg.ns / fg.ext[mu] : nface;
    nface = (nface + 7) / 8 * 8;
    if (ctx->hb) { cudaFree(ctx->hb); ctx->hb = nullptr; }
    ctx->hb_nrhs = 0;
    ctx->nface = nface;
    pack_domain_major_kernel<<<nd, fg.nsp, 0, ctx->stream>>>(fg, nd, ras_fields(ctx), -(float)ctx->kappa, ctx->dm);
    ctx->launches++;
    if (cudaGetLastError() != cudaSuccess) return 0;
    const long want = (long)per_sm * sms;
    ctx->cta_grid = (int)(nd < want ? nd : want);
    return 1;
}

// halo buffers: float4 [2 parities][nrhs][nd][8][3][nface], grown when a deeper stack of right-hand sides arrives
int ensure_halo(wcras_ctx* ctx, int nrhs) {
    if (ctx->hb && ctx->hb_nrhs >= nrhs) return WCRAS_OK;
    if (ctx->hb) { WC_CUDA(cudaStreamSynchronize(ctx->stream)); cudaFree(ctx->hb); ctx->hb = nullptr; }
    WC_CUDA(cudaMalloc((void**)&ctx->hb, sizeof(float4) * 2 * 24 * (size_t)ctx->nface * ctx->ras.nd * nrhs));
    ctx->hb_nrhs = nrhs;
    return WCRAS_OK;
}

int ras_cta_block_solve(wcras_ctx* ctx, const float4* r, float4* vout, bool accum) {
    const FusedGeom& fg = ctx->fused;
    const size_t rstride = (size_t)6 * fg.V;
    cta_kernel(false, ctx->nrhs > 1)<<<ctx->cta_grid, fg.nsp, cta_smem_bytes(fg), ctx->stream>>>(
        fg, ctx->ras.nd, -1, ctx->nface, ctx->dm, r, nullptr, nullptr, accum ? vout : nullptr, vout, nullptr, ctx->nrhs, rstride, 0);
    ctx->launches++;
    WC_CHECK_LAUNCH();
    return WCRAS_OK;
}

// v = K_RAS r with NRAS chained cycles (overlap 0): one launch per cycle, no full-lattice D in between.
// rf = rho_fin (updated in place, own sites only); the halo buffer alternates between its two parities.
int ras_cta_apply_chained(wcras_ctx* ctx, const float4* r, float4* v) {
    const FusedGeom& fg = ctx->fused;
    const int nras = ctx->ras.nras, nd = ctx->ras.nd, nface = ctx->nface, nr = ctx->nrhs;
    if (int rc = ensure_halo(ctx, nr)) return rc;
    float4* rf = ctx->ras32[0];
    const size_t rstride = (size_t)6 * fg.V, hstride = (size_t)24 * nface * nd;
    float4* hb[2] = {ctx->hb, ctx->hb + hstride * ctx->hb_nrhs};
    const size_t smem = cta_smem_bytes(fg);
    for (int j = 0; j < nras; j++) {
        const bool last = j == nras - 1;
        TimedRegion tr(ctx, TC_BLOCK);
        ctx->block_dv += ctx->ras.niter;
        if (j == 0)
            cta_kernel(false, ctx->nrhs > 1)<<<ctx->cta_grid, fg.nsp, smem, ctx->stream>>>(fg, nd, -1, nface, ctx->dm, r, nullptr, last ? nullptr : hb[0],
                                                                                nullptr, v, last ? nullptr : rf, nr, rstride, hstride);
        else
            cta_kernel(true, ctx->nrhs > 1)<<<ctx->cta_grid, fg.nsp, smem, ctx->stream>>>(fg, nd, -1, nface, ctx->dm, rf, hb[(j - 1) & 1],
                                                                               last ? nullptr : hb[j & 1], v, v, last ? nullptr : rf, nr,
                                                                               rstride, hstride);
        ctx->launches++;
    }
    WC_CHECK_LAUNCH();
    return WCRAS_OK;
}

// Can the decomposition be two-coloured (multiplicative Schwarz)?  Needs a cut direction and an even number of
// blocks in every cut direction; returns the pairing direction or -1.
int ras_cta_sap_pdir(const FusedGeom& fg) {
    int pdir = -1;
    for (int mu = 0; mu < 4; mu++) {
        if (fg.nblk[mu] > 1 && fg.nblk[mu] % 2) return -1;
        if (fg.nblk[mu] > 1 && pdir < 0) pdir = mu;
    }
    return pdir;
}

// v = K_SAP r: multiplicative Schwarz (SAP; PAPER.md:33 ref [5]), overlap 0, NRAS cycles of
// (black half step, red half step).  Each half step is one launch over the domains of one colour: rho = r_store -
// (hops of the other colour's latest v across the boundary, from the halo buffer), N_dominv MR sweeps, phi += v,
// r_store = rho_fin, halo out for the other colour.  One halo buffer suffices: a launch reads the slots of its own
// colour and writes those of the other.
int ras_cta_apply_sap(wcras_ctx* ctx, const float4* r, float4* v) {
    const FusedGeom& fg = ctx->fused;
    const int ncyc = ctx->ras.nras, ndl = ctx->ras.nd / 2, nface = ctx->nface, nr = ctx->nrhs;
    if (int rc = ensure_halo(ctx, nr)) return rc;
    float4* rf = ctx->ras32[0];
    float4* hb = ctx->hb;
    const size_t rstride = (size_t)6 * fg.V, hstride = (size_t)24 * nface * ctx->ras.nd;
    const size_t smem = cta_smem_bytes(fg);
    const int grid = ndl < ctx->cta_grid ? ndl : ctx->cta_grid;
    for (int step = 0; step < 2 * ncyc; step++) {
        const int colour = step & 1;
        const bool first_visit = step < 2, last_step = step == 2 * ncyc - 1, last_visit = step >= 2 * ncyc - 2;
        TimedRegion tr(ctx, TC_BLOCK);
        if (colour == 0) ctx->block_dv += ctx->ras.niter;  // one sweep count per full cycle over all domains
        const float4* src = first_visit ? r : rf;
        float4* rho_out = last_visit ? nullptr : rf;          // the residual of this colour is dead after its last visit
        float4* halo_out = last_step ? nullptr : hb;
        if (step == 0)
            cta_kernel(false, ctx->nrhs > 1)<<<grid, fg.nsp, smem, ctx->stream>>>(fg, ndl, colour, nface, ctx->dm, src, nullptr, halo_out, nullptr,
                                                                        v, rho_out, nr, rstride, hstride);
        else
            cta_kernel(true, ctx->nrhs > 1)<<<grid, fg.nsp, smem, ctx->stream>>>(fg, ndl, colour, nface, ctx->dm, src, hb, halo_out,
                                                                       first_visit ? nullptr : v, v, rho_out, nr, rstride, hstride);
        ctx->launches++;
    }
    WC_CHECK_LAUNCH();
    return WCRAS_OK;
}

}  // namespace wc
