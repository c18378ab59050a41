// ras_cl16.cu -- tier 2b of the RAS block solver with REDUCED-PRECISION OPERAND STORAGE and TMA STAGING: one
// thread-block CLUSTER per extended domain of more than 256 sites (the shapes BASELINE.json:configs[3] names:
// 8x8x4x4 = 4 CTAs, 8^4 = 16 CTAs; the 6^4 = 4^4 + overlap 1 of configs[1]/[2]).  The B200 replacement of the paper's
// "one domain per GPU" for domains that do not fit one SM.
//
// Same algorithm as ras_fused.cu / ras_cta16.cu -- steps A2-A5 of SURVEY.md 8(a): projection P_Omega' r (PAPER.md:66,
// Alg.1 line 4), N_dominv MR iterations on D_Omega' v = P r with Dirichlet boundaries (readings Q7,
// Q9), restriction R_Omega, the disjoint sum, phi += v (line 9), chained cycles (reading A3) -- with
// the data path of ras_cta16.cu carried over to the cluster:
//   * Omega' is cut into C <= 16 sub-blocks of <= 256 sites, one CTA per sub-block, one thread per site; the CTAs of a
//     domain form a cluster.  A half spinor whose receiver sits in the same CTA is a plain st.shared; one that crosses a
//     sub-block face travels by st.async (DSMEM store that completes bytes on an mbarrier of the RECEIVING CTA), and the
//     receiver waits on that mbarrier: no cluster barrier and no memory fence in the MR iteration.  (barrier.cluster
//     arrive.release / wait.acquire twice per iteration cost 14 % of the warp time in MEMBAR stalls alone, ncu
//     profiles/r2_kernels.md.)  The domain-local dots travel the same way: one float4 per warp to every CTA of the
//     cluster, completing on a second pair of mbarriers; the table is double-buffered by sweep parity.
//   * Operands: links and packed clover blocks ROUNDED TO fp16 (reading R1), domain-major per CTA,
//     dm16 = uint4 [nd][C][18][nsp].  Each CTA stages its 18*nsp*16 bytes with two cp.async.bulk (TMA) copies onto
//     mbarriers while the previous domain of its cluster is still being solved: the links half as soon as every thread
//     has converted the current links into registers, the clover half after its last use.  (ras_fused.cu loads its
//     fp32 operands synchronously at the start of every domain: 0.12-0.15 ms per launch at 32^4 against 0.04 here.)
//   * Links pre-scaled by -kappa at conversion, so q accumulates the hops directly; packed fp32 arithmetic
//     (site_math.cuh, FFMA2).
//   * Chained cycles keep rho_fin domain-major (float4 [nd][C][6][nsp], one bulk copy per CTA) and the halo slots
//     CTA-major ([nd][C][8][3][nfc], nfc = largest face of a sub-block), so that a CTA stages its own 24*nfc*16 bytes with
//     one bulk copy as well.
// Shared memory per CTA at nsp = 256: 96 KB half-spinor slots + 72 KB operands + 24 KB residual + 24 KB halo + 4 KB dot
// partials.
// Roofline: HBM; algorithmic bytes per extended site and launch 288 operands + 96 residual in, 96 per bulk site out
// (+ 96 rho_fin, + halo in the chained cycles).
#include <cuda_fp16.h>

#include "ras_cta_common.cuh"

namespace wc {

constexpr int CL16_MAX_CLUSTER = 16;

__device__ __forceinline__ unsigned cl16_rank() {
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ unsigned cl16_mapa(unsigned addr, unsigned rank) {
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
// 16-byte store to a half-spinor slot: plain st.shared when the receiver is a site of this CTA (loc), st.async with
// completion on the receiving CTA's mbarrier when it sits in another CTA of the cluster (rem); neither: no receiver
// (Dirichlet).  addr is a shared::cta address in the first case and a shared::cluster address in the second.
__device__ __forceinline__ void st_slot_f4(unsigned addr, unsigned mbar, bool loc, bool rem, float a, float b, float c, float d) {
    asm volatile(
        "{\n\t.reg .pred pl, pr;\n\tsetp.ne.u32 pl, %6, 0;\n\tsetp.ne.u32 pr, %7, 0;\n\t"
        "@pl st.shared.v4.f32 [%0], {%1, %2, %3, %4};\n\t"
        "@pr st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.f32 [%0], {%1, %2, %3, %4}, [%5];\n\t}" ::"r"(addr),
        "f"(a), "f"(b), "f"(c), "f"(d), "r"(mbar), "r"((unsigned)loc), "r"((unsigned)rem)
        : "memory");
}
__device__ __forceinline__ void st_slot_half(unsigned dst, unsigned mbar, bool remote, unsigned chunk_bytes, const float* h) {
    const bool ok = dst != 0xffffffffu, loc = ok && !remote, rem = ok && remote;
    st_slot_f4(dst, mbar, loc, rem, h[0], h[1], h[2], h[3]);
    st_slot_f4(dst + chunk_bytes, mbar, loc, rem, h[4], h[5], h[6], h[7]);
    st_slot_f4(dst + 2 * chunk_bytes, mbar, loc, rem, h[8], h[9], h[10], h[11]);
}
__device__ __forceinline__ void cl_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cl_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

// pack the fp16 domain-major operand copy: one CTA per (domain, cluster rank), one thread per site; zero for the padding
// lanes; also the per-domain tables dom_org / dom_bc (see ras_cta16.cu)
__global__ void pack_cl16_kernel(FusedGeom fg, int nd, Fields<float> f, uint4* __restrict__ dm16, int4* __restrict__ dom_org,
                                 unsigned* __restrict__ dom_bc) {
    const int dom = blockIdx.x / fg.C, rank = blockIdx.x % fg.C, k = threadIdx.x;
    if (dom >= nd) return;
    int org[4];
    {
        int d = dom;
        unsigned pk = 0;
        for (int mu = 0; mu < 4; mu++) {
            const int bc = d % fg.nblk[mu];
            d /= fg.nblk[mu];
            int st = bc * fg.b[mu] - (fg.split[mu] ? fg.s : 0);
            if (st < 0) st += fg.L[mu];
            org[mu] = st;
            pk |= (unsigned)bc << (8 * mu);
        }
        if (k == 0 && rank == 0) {
            dom_org[dom] = make_int4(org[0], org[1], org[2], org[3]);
            dom_bc[dom] = pk;
        }
    }
    uint4* out = dm16 + (size_t)blockIdx.x * 18 * fg.nsp + k;
    if (k >= fg.ns) {
        for (int c = 0; c < 18; c++) out[(size_t)c * fg.nsp] = make_uint4(0u, 0u, 0u, 0u);
        return;
    }
    int x[4], kk = k, rr = rank;
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        const int lc = kk % fg.sb[mu]; kk /= fg.sb[mu];
        const int sc = rr % fg.c[mu]; rr /= fg.c[mu];
        int st = org[mu] + sc * fg.sb[mu] + lc;
        if (st >= fg.L[mu]) st -= fg.L[mu];
        x[mu] = st;
    }
    const size_t gi = x[0] + fg.L[0] * (x[1] + fg.L[1] * (x[2] + (size_t)fg.L[2] * x[3])), V = fg.V;
    float u[144];
#pragma unroll
    for (int mu = 0; mu < 4; mu++) load_link(f, V, gi, mu, u + 18 * mu);
    load_clover(f, V, gi, u + 72);
#pragma unroll
    for (int c = 0; c < 18; c++) {
        uint4 t;
        __half2* h = reinterpret_cast<__half2*>(&t);
#pragma unroll
        for (int j = 0; j < 4; j++) h[j] = __floats2half2_rn(u[8 * c + 2 * j], u[8 * c + 2 * j + 1]);
        out[(size_t)c * fg.nsp] = t;
    }
}

struct Cl16Smem {  // offsets in float4 units
    int hbuf, opbuf, rstage, hstage, red, bars, org;
    size_t bytes;
};
__host__ __device__ inline Cl16Smem cl16_smem(int nsp, int C, int nfc) {
    Cl16Smem s;
    s.hbuf = 0;
    s.opbuf = 24 * nsp;
    s.rstage = s.opbuf + 18 * nsp;
    s.hstage = s.rstage + 6 * nsp;            // [8][3][nfc] halo slots of this CTA (chained cycles)
    s.red = s.hstage + 24 * nfc;              // [2][C][nwarps] dot partials of the whole cluster, by sweep parity
    s.bars = s.red + 2 * C * (nsp / 32);      // 6 mbarriers: links, clover, vectors, exchange, dots[2]
    s.org = s.bars + 3;
    s.bytes = (size_t)(s.org + 3) * 16;       // org[2] = {bytes expected on the exchange mbarrier per MR iteration, ...}
    return s;
}

// One K_RAS cycle (Alg.1 lines 3-9) for all domains; arguments as ras_cta16_kernel (no colouring); nfc = padded size of
// the largest face of a sub-block, halo buffers CTA-major [nd][C][8][3][nfc]
template <bool CHAIN>
__global__ void __launch_bounds__(FUSED_CTA_MAX_THREADS, 1)
ras_cl16_kernel(FusedGeom fg, int nd, int nfc, float mkappa, const uint4* __restrict__ dm16, const float4* __restrict__ r_lat,
                const float4* __restrict__ r_dm, const float4* __restrict__ hb_in, float4* __restrict__ hb_out, const float4* phi_in,
                float4* phi_out, float4* __restrict__ rho_dm, const int4* __restrict__ dom_org, const unsigned* __restrict__ dom_bc) {
    if (fg.stop && __ldg(fg.stop)) return;  // the inner solver has converged (launch enqueued ahead of the host's check)
    extern __shared__ float4 smem[];
    const int nsp = fg.nsp, C = fg.C;
    const Cl16Smem lay = cl16_smem(nsp, C, nfc);
    float4* hbuf = smem + lay.hbuf;                                        // [8][3][nsp] half-spinor slots
    const uint4* opbuf = reinterpret_cast<const uint4*>(smem + lay.opbuf);  // [18][nsp] fp16 operands of the current domain
    float4* rstage = smem + lay.rstage;                                    // [6][nsp] residual of the current / next domain
    const float4* hstage = smem + lay.hstage;                              // [8][3][nfc] halo slots of this CTA (chained cycles)
    float4* red = smem + lay.red;                                          // [2][C][nwarps] dot partials of the whole cluster
    int4* org_s = reinterpret_cast<int4*>(smem + lay.org);                 // [2] first site of the current / next domain (table dom_org)
    const unsigned bar_links = cta_smem_u32(smem + lay.bars), bar_clov = bar_links + 8, bar_vec = bar_links + 16;
    const unsigned bar_x = bar_links + 24, bar_d = bar_links + 32;  // exchange (remote half spinors), dots [2] (by sweep parity)
    const int k = threadIdx.x, lane = k & 31, warp = k >> 5, nwarps = blockDim.x >> 5;
    const unsigned rank = cl16_rank();
    const int cl = blockIdx.x / C, ncl = gridDim.x / C;
    const bool active = k < fg.ns;
    const bool src_dm = r_dm != nullptr;

    // ---- domain-independent geometry: coordinates in the sub-block (lc), of the sub-block (sc), in Omega' (ec) ----
    int ec[4];
    bool bulk = active;
    unsigned dst[8];  // slot 2mu: receiver x-mu (its forward hop); slot 2mu+1: receiver x+mu (its backward hop)
    int fidx[4];      // index of the site within the mu-face of its sub-block (local index with coordinate mu removed)
    unsigned remote = 0;          // bit n: the receiver of slot n sits in another CTA of the cluster
    unsigned rk_pk = 0;           // 4 bits per direction: the rank of that CTA
    const unsigned chunk_bytes = (unsigned)nsp * 16u;
    {
        int lc[4], sc[4];
        int kk = active ? k : 0, rr = (int)rank;
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            lc[mu] = kk % fg.sb[mu]; kk /= fg.sb[mu];
            sc[mu] = rr % fg.c[mu]; rr /= fg.c[mu];
            ec[mu] = sc[mu] * fg.sb[mu] + lc[mu];
            if (fg.split[mu]) bulk = bulk && ec[mu] >= fg.s && ec[mu] < fg.s + fg.b[mu];
        }
        const unsigned base = cta_smem_u32(hbuf);
        int lstride = 1, cstride = 1;
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            fidx[mu] = (k % lstride) + (k / (lstride * fg.sb[mu])) * lstride;
#pragma unroll
            for (int sg = 0; sg < 2; sg++) {  // sg 0: receiver x-mu, sg 1: receiver x+mu
                int kd = k, rk = (int)rank;
                bool ok = active;
                if (sg == 0) {
                    if (lc[mu] > 0) kd -= lstride;
                    else {
                        kd += (fg.sb[mu] - 1) * lstride;
                        if (sc[mu] > 0) rk -= cstride;
                        else if (fg.wrap[mu]) rk += (fg.c[mu] - 1) * cstride;
                        else ok = false;
                    }
                } else {
                    if (lc[mu] + 1 < fg.sb[mu]) kd += lstride;
                    else {
                        kd -= (fg.sb[mu] - 1) * lstride;
                        if (sc[mu] + 1 < fg.c[mu]) rk += cstride;
                        else if (fg.wrap[mu]) rk -= (fg.c[mu] - 1) * cstride;
                        else ok = false;
                    }
                }
                const unsigned a_loc = base + (unsigned)((2 * mu + sg) * 3 * nsp + kd) * 16u;
                const bool far = rk != (int)rank;
                dst[2 * mu + sg] = ok ? (far ? cl16_mapa(a_loc, (unsigned)rk) : a_loc) : 0xffffffffu;
                if (ok && far) {  // at most one remote receiver per direction (sub-blocks are at least two sites thick)
                    remote |= 1u << (2 * mu + sg);
                    rk_pk |= (unsigned)rk << (4 * mu);
                }
            }
            lstride *= fg.sb[mu];
            cstride *= fg.c[mu];
        }
    }
    // coordinates in Omega' and face indices travel through the block solve as one / two registers
    const unsigned ec_pk = (unsigned)ec[0] | (unsigned)ec[1] << 8 | (unsigned)ec[2] << 16 | (unsigned)ec[3] << 24;
    const unsigned fidx_lo = (unsigned)fidx[0] | (unsigned)fidx[1] << 16, fidx_hi = (unsigned)fidx[2] | (unsigned)fidx[3] << 16;
#define WC_FIDX(MU) ((int)((((MU) < 2 ? fidx_lo : fidx_hi) >> (16 * ((MU) & 1))) & 0xffffu))
#pragma unroll
    for (int j = 0; j < 24; j++) hbuf[j * nsp + k] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (k == 0) {
        mbar_init(bar_links, 1);
        mbar_init(bar_clov, 1);
        mbar_init(bar_vec, 1);
        mbar_init(bar_x, 1);
        mbar_init(bar_d, 1);
        mbar_init(bar_d + 8, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // bytes of half spinors that arrive from other CTAs per MR iteration: slot 2mu of a site is written by x+mu and slot
    // 2mu+1 by x-mu, so a slot is filled remotely exactly when this site's own store in the opposite sense is remote
    {
        unsigned xb = 0;
#pragma unroll
        for (int n = 0; n < 8; n++) xb += 48u * (unsigned)__syncthreads_count(0 != (remote & (1u << n)));
        if (k == 0) org_s[2].x = (int)xb;  // read back by thread 0 at the top of every MR iteration
    }
    cl_arrive();
    cl_wait();  // every CTA of the cluster has zeroed its slots and initialised its mbarriers before anybody stores into it

    const size_t V = fg.V;
    const unsigned half_bytes = 9u * chunk_bytes;  // links or clover part of one CTA's share of a domain
    const unsigned halo_bytes = CHAIN ? 24u * (unsigned)nfc * 16u : 0u;
    const unsigned vec_bytes = (src_dm ? 6u * chunk_bytes : 0u) + halo_bytes;
    const unsigned op_addr = cta_smem_u32(opbuf), rs_addr = cta_smem_u32(rstage), hs_addr = cta_smem_u32(hstage);

    auto request_links_vec = [&](int d) {
        if (k == 0) {
            const size_t chunk = (size_t)d * C + rank;
            mbar_expect_tx(bar_links, half_bytes);
            bulk_g2s(op_addr, dm16 + chunk * 18 * nsp, half_bytes, bar_links);
            if (vec_bytes) {
                mbar_expect_tx(bar_vec, vec_bytes);
                if (src_dm) bulk_g2s(rs_addr, r_dm + chunk * 6 * nsp, 6u * chunk_bytes, bar_vec);
                if (CHAIN) bulk_g2s(hs_addr, hb_in + chunk * 24 * nfc, halo_bytes, bar_vec);
            }
        }
    };
    auto request_clover = [&](int d) {
        if (k == 0) {
            mbar_expect_tx(bar_clov, half_bytes);
            bulk_g2s(op_addr + half_bytes, dm16 + (((size_t)d * C + rank) * 18 + 9) * nsp, half_bytes, bar_clov);
        }
    };
    auto site_of = [&](const int4& org) -> size_t {
        int x0 = org.x + (int)(ec_pk & 255u), x1 = org.y + (int)((ec_pk >> 8) & 255u), x2 = org.z + (int)((ec_pk >> 16) & 255u),
            x3 = org.w + (int)(ec_pk >> 24);
        if (x0 >= fg.L[0]) x0 -= fg.L[0];
        if (x1 >= fg.L[1]) x1 -= fg.L[1];
        if (x2 >= fg.L[2]) x2 -= fg.L[2];
        if (x3 >= fg.L[3]) x3 -= fg.L[3];
        return x0 + fg.L[0] * (x1 + fg.L[1] * (x2 + (size_t)fg.L[2] * x3));
    };
    auto request_r_lat = [&](const int4& org) {  // own column, LDGSTS; waited for by the issuing thread itself
        if (active) {
            const size_t gn = site_of(org);
#pragma unroll
            for (int c = 0; c < 6; c++) cp_async16(rstage + c * nsp + k, r_lat + (size_t)c * V + gn);
        }
        cp_async_commit();
    };

    if (cl < nd) {
        request_links_vec(cl);
        request_clover(cl);
        if (k == 0) cp_async16(org_s, dom_org + cl);  // committed with (or as) the first group below, waited for at the loop top
        if (!src_dm) request_r_lat(dom_org[cl]);
        else cp_async_commit();
    }

    float U[72];
    unsigned sw = 0;  // MR iterations done by this cluster so far: parity of the exchange mbarrier, index / parity of the dots pair
    // the domain index is carried and the exit test uses has_next from the top of the iteration: recomputed at the bottom
    // they cost constant-bank loads with every warp waiting on them (see ras_cta16.cu; K_RAS application at 8^4, N_dominv 2,
    // NRAS 4: 1.380 -> 1.341 ms).  The other two changes made there (small tables at fixed shared-memory offsets, per-launch
    // uniforms pinned in a register) were measured slower here (1.349 with them, 1.41 with all three) and are not made.
    for (int j = 0, dom = cl; dom < nd; j++) {
        const unsigned par = (unsigned)j & 1u;
        const int dn = dom + ncl;
        const bool has_next = dn < nd;
        const int nxt = has_next ? dn : dom;
        const unsigned dom_bc_here = hb_out ? __ldg(dom_bc + dom) : 0u;
        int4 org_nxt = make_int4(0, 0, 0, 0);
        if (!src_dm) org_nxt = __ldg(dom_org + nxt);  // lattice-layout source: the next residual column is requested below

        // ---- operands: links from the staged fp16 block into registers, scaled by -kappa ----
        mbar_wait(bar_links, par);
#pragma unroll
        for (int c = 0; c < 9; c++) {
            float f[8];
            half8_to_float(opbuf[c * nsp + k], f);
#pragma unroll
            for (int n = 0; n < 8; n++) U[8 * c + n] = mkappa * f[n];
        }
        // ---- projection P_Omega' r: the staged residual column of this thread ----
        float rho[24], v[24];
        cp_async_wait();  // own residual column (lattice-layout source); thread 0: the origin of this domain in org_s
        if (vec_bytes) mbar_wait(bar_vec, par);
#pragma unroll
        for (int c = 0; c < 6; c++) {
            float4 t = rstage[c * nsp + k];
            if (!active) t = make_float4(0.f, 0.f, 0.f, 0.f);
            rho[4 * c] = t.x; rho[4 * c + 1] = t.y; rho[4 * c + 2] = t.z; rho[4 * c + 3] = t.w;
        }
        if (!src_dm && has_next) request_r_lat(org_nxt);  // own column: free as soon as it has been read
        if (CHAIN) {
            // ---- boundary coupling: rho -= D-terms of v_{j-1} that cross the domain boundary (reading A3), from the
            // staged halo slots of this CTA ----
            const float4* hin = hstage;
            float g[12], hh[12];
#define WC_CROSS_LOAD(SL)                                                                         \
    {                                                                                             \
        const bool rcv = active && dst[(SL) ^ 1] == 0xffffffffu;                                  \
        const float4* q4 = hin + (SL) * 3 * nfc + WC_FIDX((SL) >> 1);                             \
        _Pragma("unroll") for (int jj = 0; jj < 3; jj++) {                                        \
            float4 t = make_float4(0.f, 0.f, 0.f, 0.f);                                           \
            if (rcv) t = q4[jj * nfc];                                                            \
            hh[4 * jj] = t.x; hh[4 * jj + 1] = t.y; hh[4 * jj + 2] = t.z; hh[4 * jj + 3] = t.w;   \
        }                                                                                         \
    }
#define WC_CROSS(MU)                                                                              \
    if (__any_sync(0xffffffffu, active && dst[2 * MU + 1] == 0xffffffffu)) {                      \
        WC_CROSS_LOAD(2 * MU)                                                                     \
        su3_mul<float>(U + 18 * MU, hh, g);                                                       \
        reconstruct_sub<float, MU, -1>(g, rho);                                                   \
    }                                                                                             \
    if (__any_sync(0xffffffffu, active && dst[2 * MU] == 0xffffffffu)) {                          \
        WC_CROSS_LOAD(2 * MU + 1)                                                                 \
        reconstruct_sub<float, MU, +1>(hh, rho);                                                  \
    }
            WC_CROSS(0) WC_CROSS(1) WC_CROSS(2) WC_CROSS(3)
#undef WC_CROSS
#undef WC_CROSS_LOAD
        }
#pragma unroll
        for (int n = 0; n < 24; n++) v[n] = 0.f;

        for (int it = 0; it < fg.niter; it++, sw++) {
            const unsigned bar_dk = bar_d + 8u * (sw & 1u);
            if (k == 0) {  // this iteration's arrivals: the remote half spinors and the C * nwarps dot partials
                mbar_expect_tx(bar_x, (unsigned)org_s[2].x);
                mbar_expect_tx(bar_dk, 16u * (unsigned)(C * nwarps));
            }
            {
                float hs[12], g[12];
#define WC_SCATTER(MU)                                                                                  \
    {                                                                                                   \
        const unsigned xb = cl16_mapa(bar_x, (rk_pk >> (4 * MU)) & 15u);                                \
        project<float, MU, -1>(rho, hs);                                                                \
        st_slot_half(dst[2 * MU], xb, (remote >> (2 * MU)) & 1u, chunk_bytes, hs);                      \
        project<float, MU, +1>(rho, hs);                                                                \
        su3_adj_mul<float>(U + 18 * MU, hs, g);                                                         \
        st_slot_half(dst[2 * MU + 1], xb, (remote >> (2 * MU + 1)) & 1u, chunk_bytes, g);               \
    }
                WC_SCATTER(0) WC_SCATTER(1) WC_SCATTER(2) WC_SCATTER(3)
#undef WC_SCATTER
            }
            float q[24];
            if (it == 0) mbar_wait(bar_clov, par);
            // q = A rho from the staged fp16 clover blocks (independent of the exchange: covers the flight of the stores)
#pragma unroll
            for (int ch = 0; ch < 2; ch++) {
                float Ab[40];
#pragma unroll
                for (int c = 0; c < 5; c++) half8_to_float(opbuf[(9 + 4 * ch + c) * nsp + k], Ab + 8 * c);
                herm6_mul<float>(Ab + 4 * ch, rho + 12 * ch, q + 12 * ch);
            }
            __syncthreads();                               // the half spinors stored by this CTA
            mbar_wait(bar_x, sw & 1u);                     // those stored into it by the other CTAs of the cluster
            // Every thread of this CTA is past its staging reads of this domain (links, residual, halo: before the first
            // barrier; clover: before this barrier of the last sweep): thread 0 requests the next domain's data.
            if (has_next && warp == 0) {
                if (it == 0) {
                    request_links_vec(nxt);
                    if (k == 1) prefetch_l2_bulk(dm16 + (((size_t)nxt * C + rank) * 18 + 9) * nsp, half_bytes);
                    if (k == 0) { cp_async16(org_s + ((j + 1) & 1), dom_org + nxt); cp_async_commit(); }
                }
                if (it + 1 == fg.niter) request_clover(nxt);
            }
            {
                float hs[12], g[12];
#define WC_GATHER(MU)                                        \
    ld_half_cta(hbuf + (2 * MU) * 3 * nsp + k, nsp, hs);     \
    su3_mul<float>(U + 18 * MU, hs, g);                      \
    reconstruct_add<float, MU, -1>(g, q);                    \
    ld_half_cta(hbuf + (2 * MU + 1) * 3 * nsp + k, nsp, g);  \
    reconstruct_add<float, MU, +1>(g, q);
                WC_GATHER(0) WC_GATHER(1) WC_GATHER(2) WC_GATHER(3)
#undef WC_GATHER
            }
            float d0 = 0.f, d1 = 0.f, d2 = 0.f;
#ifdef WC_X2
            x2::mr_dots(q, rho, d0, d1, d2);
#else
#pragma unroll
            for (int n = 0; n < 12; n++) {
                const float qr = q[2 * n], qi = q[2 * n + 1], rr = rho[2 * n], ri = rho[2 * n + 1];
                d0 = fmaf(qr, rr, d0); d0 = fmaf(qi, ri, d0);
                d1 = fmaf(qr, ri, d1); d1 = fmaf(-qi, rr, d1);
                d2 = fmaf(qr, qr, d2); d2 = fmaf(qi, qi, d2);
            }
#endif
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                d0 += __shfl_xor_sync(0xffffffffu, d0, o);
                d1 += __shfl_xor_sync(0xffffffffu, d1, o);
                d2 += __shfl_xor_sync(0xffffffffu, d2, o);
            }
            // one float4 per warp, pushed by lane c into the partial table of CTA c (its copy for this sweep parity) with
            // completion on that CTA's dots mbarrier: every CTA sums the same table in the same order
            float4* redk = red + (sw & 1u) * (unsigned)(C * nwarps);
            if (lane < C) {
                const unsigned slot = cl16_mapa(cta_smem_u32(redk + rank * nwarps + warp), (unsigned)lane);
                const unsigned db = cl16_mapa(bar_dk, (unsigned)lane);
                asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.f32 [%0], {%1, %2, %3, %4}, [%5];" ::"r"(slot),
                             "f"(d0), "f"(d1), "f"(d2), "f"(0.f), "r"(db)
                             : "memory");
            }
            mbar_wait(bar_dk, (sw >> 1) & 1u);
            float s0 = 0.f, s1 = 0.f, s2 = 0.f;
            for (int n = lane; n < C * nwarps; n += 32) {
                const float4 p = redk[n];
                s0 += p.x; s1 += p.y; s2 += p.z;
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                s0 += __shfl_xor_sync(0xffffffffu, s0, o);
                s1 += __shfl_xor_sync(0xffffffffu, s1, o);
                s2 += __shfl_xor_sync(0xffffffffu, s2, o);
            }
            // alpha = <q,rho>/<q,q>, 0 if <q,q> = 0 (Q9); v += alpha rho; rho -= alpha q
            const float inv = s2 > 0.f ? 1.f / s2 : 0.f;
            const float ar = s0 * inv, ai = s1 * inv;
            const bool upd_rho = it + 1 < fg.niter || rho_dm != nullptr;
#ifdef WC_X2
            if (upd_rho) x2::mr_update<true>(ar, ai, q, rho, v);
            else x2::mr_update<false>(ar, ai, q, rho, v);
#else
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
#endif
        }
        // ---- halo scatter for the next cycle: the hops of v that leave the domain, as projected half spinors ----
        if (hb_out) {
            unsigned dd = dom_bc_here;
            int dstride = 1, cstr = 1;
            float hs[12], g[12];
#define WC_HALO(MU)                                                                                              \
    {                                                                                                            \
        const int nb = fg.nblk[MU], bc = (int)(dd & 255u), cspan = (fg.c[MU] - 1) * cstr;                        \
        dd >>= 8;                                                                                                \
        if (active && dst[2 * MU] == 0xffffffffu) { /* lower face -> slot 2mu of the last sub-block of the domain at -mu */ \
            const int nbd = bc == 0 ? dom + (nb - 1) * dstride : dom - dstride;                                  \
            float4* o = hb_out + (((size_t)nbd * C + rank + cspan) * 8 + 2 * MU) * 3 * nfc + WC_FIDX(MU);        \
            project<float, MU, -1>(v, hs);                                                                       \
            for (int jj = 0; jj < 3; jj++) o[jj * nfc] = make_float4(hs[4 * jj], hs[4 * jj + 1], hs[4 * jj + 2], hs[4 * jj + 3]); \
        }                                                                                                        \
        if (active && dst[2 * MU + 1] == 0xffffffffu) { /* upper face -> slot 2mu+1 of the first sub-block of the domain at +mu */ \
            const int nbd = bc + 1 == nb ? dom - (nb - 1) * dstride : dom + dstride;                             \
            float4* o = hb_out + (((size_t)nbd * C + rank - cspan) * 8 + 2 * MU + 1) * 3 * nfc + WC_FIDX(MU);    \
            project<float, MU, +1>(v, hs);                                                                       \
            su3_adj_mul<float>(U + 18 * MU, hs, g);                                                              \
            for (int jj = 0; jj < 3; jj++) o[jj * nfc] = make_float4(g[4 * jj], g[4 * jj + 1], g[4 * jj + 2], g[4 * jj + 3]); \
        }                                                                                                        \
        dstride *= nb;                                                                                           \
        cstr *= fg.c[MU];                                                                                        \
    }
            WC_HALO(0) WC_HALO(1) WC_HALO(2) WC_HALO(3)
#undef WC_HALO
        }
        // ---- rho_fin (domain-major, every site of the domain) and the restriction R_Omega (bulk sites only) ----
        if (rho_dm && active) {
            float4* o = rho_dm + ((size_t)dom * C + rank) * 6 * nsp + k;
#pragma unroll
            for (int c = 0; c < 6; c++) o[(size_t)c * nsp] = make_float4(rho[4 * c], rho[4 * c + 1], rho[4 * c + 2], rho[4 * c + 3]);
        }
        if (bulk) {
            const size_t gi = site_of(org_s[j & 1]);  // visible since the first barrier of this domain
            if (phi_in) {
                // phi += v as a fire-and-forget vector reduction (phi_in == phi_out; one writer per site)
#pragma unroll
                for (int c = 0; c < 6; c++)
                    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(phi_out + (size_t)c * V + gi), "f"(v[4 * c]),
                                 "f"(v[4 * c + 1]), "f"(v[4 * c + 2]), "f"(v[4 * c + 3])
                                 : "memory");
            } else {
#pragma unroll
                for (int c = 0; c < 6; c++)
                    phi_out[(size_t)c * V + gi] = make_float4(v[4 * c], v[4 * c + 1], v[4 * c + 2], v[4 * c + 3]);
            }
        }
        if (!has_next) break;
        dom = dn;
    }
    // no CTA leaves while a store from (or a read of its partials by) another CTA of the cluster could still be under way
    cl_arrive();
    cl_wait();
}

// ---- host side ----
static cudaError_t cl16_config(const FusedGeom& fg, int nclus, size_t smem, cudaStream_t stream, cudaLaunchConfig_t* cfg,
                               cudaLaunchAttribute* at) {
    *cfg = cudaLaunchConfig_t{};
    cfg->gridDim = dim3((unsigned)nclus * fg.C);
    cfg->blockDim = dim3((unsigned)fg.nsp);
    cfg->dynamicSmemBytes = smem;
    cfg->stream = stream;
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)fg.C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg->attrs = at;
    cfg->numAttrs = 1;
    return cudaSuccess;
}

template <bool CHAIN>
static cudaError_t cl16_launch(wcras_ctx* ctx, const float4* r_lat, const float4* r_dm, const float4* hb_in, float4* hb_out,
                               const float4* phi_in, float4* phi_out, float4* rho_dm) {
    const FusedGeom& fg = ctx->fused;
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute at[1];
    const int nclus = ctx->ras.nd < ctx->cl16_nclus ? ctx->ras.nd : ctx->cl16_nclus;
    cl16_config(fg, nclus, ctx->cta16_smem, ctx->stream, &cfg, at);
    return cudaLaunchKernelEx(&cfg, ras_cl16_kernel<CHAIN>, fg, ctx->ras.nd, ctx->cl16_nfc, -(float)ctx->kappa, (const uint4*)ctx->dm16, r_lat, r_dm,
                              hb_in, hb_out, phi_in, phi_out, rho_dm, (const int4*)ctx->dom_org, (const unsigned*)ctx->dom_bc);
}

// Build the fp16 domain-major operand copy and the domain-major rho_fin buffer of the cluster tier; returns 1 if this
// kernel can run the configuration (2 <= C <= 16, the cluster is schedulable, memory), 0 otherwise (ras_fused.cu runs).
int ras_cl16_prepare(wcras_ctx* ctx, const FusedGeom& fg, int nd, const Fields<float>& f) {
    if (fg.C < 2 || fg.C > CL16_MAX_CLUSTER || fg.nsp > FUSED_CTA_MAX_THREADS) return 0;
    int nfc = 1;
    for (int mu = 0; mu < 4; mu++) {
        if (fg.nblk[mu] > 255) return 0;                // dom_bc packs the block coordinates into 8 bits each
        if (fg.c[mu] > 1 && fg.sb[mu] < 2) return 0;    // a site has at most one receiver in another CTA per direction
        nfc = fg.ns / fg.sb[mu] > nfc ? fg.ns / fg.sb[mu] : nfc;
    }
    nfc = (nfc + 7) / 8 * 8;
    int smem_max = 0, dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    const size_t smem = cl16_smem(fg.nsp, fg.C, nfc).bytes;
    if (smem > (size_t)smem_max) return 0;
    int nclus = 0;
    for (int chain = 0; chain < 2; chain++) {
        const void* kern = chain ? (const void*)ras_cl16_kernel<true> : (const void*)ras_cl16_kernel<false>;
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
            cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, fg.C > 8 ? 1 : 0) != cudaSuccess) {
            cudaGetLastError();
            return 0;
        }
        cudaLaunchConfig_t cfg;
        cudaLaunchAttribute at[1];
        cl16_config(fg, 1, smem, ctx->stream, &cfg, at);
        int n = 0;
        if (cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess || n < 1) { cudaGetLastError(); return 0; }
        nclus = chain == 0 || n < nclus ? n : nclus;
    }
    if (ctx->dm16) { cudaStreamSynchronize(ctx->stream); cudaFree(ctx->dm16); ctx->dm16 = nullptr; }
    if (ctx->rf_dm) { cudaStreamSynchronize(ctx->stream); cudaFree(ctx->rf_dm); ctx->rf_dm = nullptr; }
    const size_t nchunk = (size_t)nd * fg.C;
    const size_t rf_bytes = sizeof(float4) * 6 * (size_t)fg.nsp * nchunk;
    if (cudaMalloc((void**)&ctx->dm16, sizeof(uint4) * 18 * (size_t)fg.nsp * nchunk) != cudaSuccess) { cudaGetLastError(); ctx->dm16 = nullptr; return 0; }
    if (cudaMalloc((void**)&ctx->rf_dm, rf_bytes + (sizeof(int4) + sizeof(unsigned)) * (size_t)nd) != cudaSuccess) {
        cudaGetLastError();
        cudaFree(ctx->dm16);
        ctx->dm16 = nullptr; ctx->rf_dm = nullptr;
        return 0;
    }
    ctx->dom_org = reinterpret_cast<int4*>(reinterpret_cast<char*>(ctx->rf_dm) + rf_bytes);
    ctx->dom_bc = reinterpret_cast<unsigned*>(ctx->dom_org + nd);
    ctx->cta16_smem = smem;
    ctx->cl16_nclus = nclus;
    ctx->cl16_nfc = nfc;
    pack_cl16_kernel<<<(unsigned)nchunk, fg.nsp, 0, ctx->stream>>>(fg, nd, f, ctx->dm16, ctx->dom_org, ctx->dom_bc);
    ctx->launches++;
    if (cudaGetLastError() != cudaSuccess) return 0;
    return 1;
}

int ras_cl16_block_solve(wcras_ctx* ctx, const float4* r, float4* vout, bool accum) {
    WC_CUDA(cl16_launch<false>(ctx, r, nullptr, nullptr, nullptr, accum ? vout : nullptr, vout, nullptr));
    ctx->launches++;
    return WCRAS_OK;
}

int ensure_halo(wcras_ctx* ctx, int nrhs);  // ras_cta.cu

// v = K_RAS r with NRAS chained cycles (overlap 0): one launch per cycle, no full-lattice D in between (reading A3);
// rho_fin travels domain-major through ctx->rf_dm, the halo buffer alternates between its two parities
int ras_cl16_apply_chained(wcras_ctx* ctx, const float4* r, float4* v) {
    const int nras = ctx->ras.nras, nd = ctx->ras.nd, nface = ctx->nface;  // nface = C * nfc: CTA-major halo slots
    if (int rc = ensure_halo(ctx, 1)) return rc;
    float4* rf = ctx->rf_dm;
    const size_t hstride = (size_t)24 * nface * nd;
    float4* hb[2] = {ctx->hb, ctx->hb + hstride * ctx->hb_nrhs};
    for (int j = 0; j < nras; j++) {
        const bool last = j == nras - 1;
        TimedRegion tr(ctx, TC_BLOCK);
        ctx->block_dv += ctx->ras.niter;
        if (j == 0) WC_CUDA(cl16_launch<false>(ctx, r, nullptr, nullptr, last ? nullptr : hb[0], nullptr, v, last ? nullptr : rf));
        else WC_CUDA(cl16_launch<true>(ctx, nullptr, rf, hb[(j - 1) & 1], last ? nullptr : hb[j & 1], v, v, last ? nullptr : rf));
        ctx->launches++;
    }
    return WCRAS_OK;
}

}  // namespace wc
