// ras_cta16.cu -- tier 2a of the RAS block solver with REDUCED-PRECISION OPERAND STORAGE and TMA STAGING
// (north_star (c): "links, clover and spinor staged into shared memory ... via TMA, the block iterations run to
// completion on-chip"; SURVEY.md 8(f) NEXT-4 "reduced-precision (fp16) storage links+clover"; reading R1).
//
// Same algorithm as ras_cta.cu -- steps A2-A5 of SURVEY.md 8(a): projection P_Omega' r (Alg.1 line 4),
// N_dominv MR iterations on D_Omega' v = P r with Dirichlet boundaries (readings Q7, Q9), restriction
// R_Omega, the disjoint sum and phi += v (line 9), chained cycles (reading A3) -- for extended domains
// of at most 256 sites, one persistent CTA walking over its domains, one thread per site.  What differs:
//
//   * The operands of the block solver are the links and the packed clover blocks ROUNDED TO fp16 (reading R1: K_RAS
//     of the operator D~ whose operands are the fp16 roundings of the fp32 fields; all arithmetic stays fp32).
//     Domain-major copy dm16 = uint4 [nd][18][nsp]: chunks 0..8 hold the 72 link reals of the site as halfs
//     (unscaled; -kappa is applied after the conversion), chunks 9..17 the 72 clover reals.  288 B per site instead of
//     576 B: the per-cycle operand stream that dominates the HBM traffic of a K_RAS application is halved.
//   * Everything the NEXT domain of the CTA needs travels into shared memory while the current one is being solved,
//     so no thread ever waits on a global load:
//       - operands: two cp.async.bulk (TMA) copies of 9*nsp*16 bytes each, completing on mbarriers.  The link half is
//         requested as soon as every thread has converted the current links into registers, the clover half (read
//         from shared memory in every sweep) after its last use; the clover half is prefetched to L2 meanwhile.
//       - residual: chained cycles keep rho_fin DOMAIN-MAJOR (float4 [nd][6][nsp]), one bulk copy; a lattice-layout
//         source (cycle 0) is fetched by each thread into its own column with cp.async (LDGSTS).
//       - halo slots of the chained cycles: contiguous per domain, one bulk copy (when they fit beside the rest).
//   * Shared memory at nsp = 256: 96 KB half-spinor slots + 72 KB operands + 24 KB residual + 24 KB halo = 216 KB.
// Roofline: HBM; algorithmic bytes per site and launch 288 operands + 96 residual in + 96 out (+ 96 rho_fin, + halo).
#include <cuda_fp16.h>

#include "ras_cta_common.cuh"

namespace wc {

// pack the fp16 domain-major operand copy: one thread per (domain, local site); zero for the padding lanes
// also fills the per-domain tables dom_org (first site of Omega', coordinates mod L) and dom_bc (block coordinates packed
// 8 bits each), so that the block solver needs no integer division per domain
__global__ void pack_dm16_kernel(FusedGeom fg, int nd, Fields<float> f, uint4* __restrict__ dm16, int4* __restrict__ dom_org,
                                 unsigned* __restrict__ dom_bc) {
    const int dom = blockIdx.x, k = threadIdx.x;
    if (dom >= nd) return;
    if (k == 0) {
        int d = dom, o[4];
        unsigned pk = 0;
        for (int mu = 0; mu < 4; mu++) {
            const int bc = d % fg.nblk[mu];
            d /= fg.nblk[mu];
            int st = bc * fg.b[mu] - (fg.split[mu] ? fg.s : 0);
            if (st < 0) st += fg.L[mu];
            o[mu] = st;
            pk |= (unsigned)bc << (8 * mu);
        }
        dom_org[dom] = make_int4(o[0], o[1], o[2], o[3]);
        dom_bc[dom] = pk;
    }
    uint4* out = dm16 + (size_t)dom * 18 * fg.nsp + k;
    if (k >= fg.ns) {
        for (int c = 0; c < 18; c++) out[(size_t)c * fg.nsp] = make_uint4(0u, 0u, 0u, 0u);
        return;
    }
    int lc[4], kk = k;
#pragma unroll
    for (int mu = 0; mu < 4; mu++) { lc[mu] = kk % fg.ext[mu]; kk /= fg.ext[mu]; }
    const size_t gi = cta_site(fg, dom, lc), V = fg.V;
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

// x -> fp32(fp16(x)), elementwise: the rounded fp32 field copies every other K_RAS path uses in 16-bit operand mode
__global__ void round_half_kernel(size_t n, const float* __restrict__ in, float* __restrict__ out) {
    for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (size_t)gridDim.x * blockDim.x)
        out[k] = __half2float(__float2half_rn(in[k]));
}

// cycle-level phase profile of CTA 0 (debug builds only: -DWC_CTA16_PROFILE prints the totals of thread 0)
#ifdef WC_CTA16_PROFILE
#define WC_T(n) { const long long t_ = clock64(); if (k == 0) prof[n] += t_ - tlast; tlast = t_; }
// has the link half of the NEXT domain landed?  (non-blocking test of the next phase of bar_links, thread 0)
#define WC_LANDED(n)                                                                                                          \
    if (k == 0) {                                                                                                             \
        unsigned ok_;                                                                                                         \
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"  \
                     : "=r"(ok_) : "r"(bar_links), "r"(par ^ 1u) : "memory");                                                 \
        landed[n] += ok_;                                                                                                     \
    }
#else
#define WC_T(n)
#define WC_LANDED(n) {}
#endif

struct Cta16Smem {  // offsets in float4 units
    int hbuf, opbuf, rstage, hstage, red, bars, org;
    size_t bytes;
};
// The small tables come first, at offsets that do not depend on the launch parameters: an address that needs nface or
// stage_halo costs a constant-bank load wherever the compiler rematerialises it (measured ~300 cycles, once per domain).
__host__ __device__ inline Cta16Smem cta16_smem(int nsp, int nface, int stage_halo) {
    Cta16Smem s;
    s.red = 0;    // [2][8] warp partials (the second row for the five dots of the MR2 block solver)
    s.bars = 16;
    s.org = 18;
    s.hbuf = 24;  // 384-byte offset: bulk-copy destinations stay 128-byte aligned
    s.opbuf = s.hbuf + 24 * nsp;
    s.rstage = s.opbuf + 18 * nsp;
    s.hstage = s.rstage + 6 * nsp;
    s.bytes = (size_t)(s.hstage + (stage_halo ? 24 * nface : 0)) * 16;
    return s;
}

// One K_RAS cycle (Alg.1 lines 3-9) for all domains of the launch; arguments as ras_cta_kernel except
//   r_lat   residual source in the lattice layout (cycle 0 / first visit), or nullptr
//   r_dm    residual source domain-major [nd][6][nsp] (rho_fin of the previous cycle), or nullptr
//   rho_dm  rho_fin of this cycle, domain-major, or nullptr (then the last MR residual update is skipped, Q12)
//   MR2     block solver: restarted two-dimensional minimal residual (reading R2) instead of MR
//   NSP     threads per CTA = sites per domain as a compile-time constant (256, no padding lanes: every slot, operand and
//           staging offset becomes an immediate and every thread is active), or 0 = fg.nsp / fg.ns at run time
template <bool CHAIN, int NSP, bool MR2>
__global__ void __launch_bounds__(FUSED_CTA_MAX_THREADS, 1)
ras_cta16_kernel(FusedGeom fg, int ndl, int colour, int nface, int stage_halo, float mkappa, const uint4* __restrict__ dm16,
                 const float4* __restrict__ r_lat, const float4* __restrict__ r_dm, const float4* __restrict__ hb_in,
                 float4* __restrict__ hb_out, const float4* phi_in, float4* phi_out, float4* __restrict__ rho_dm,
                 const int4* __restrict__ dom_org, const unsigned* __restrict__ dom_bc) {
    if (fg.stop && __ldg(fg.stop)) return;  // the inner solver has converged (launch enqueued ahead of the host's check)
    // Programmatic dependent launch: the next cycle of this K_RAS application (launched with the programmatic-serialization
    // attribute) may be scheduled as SMs fall free while this grid is still running; its set-up and its first operand
    // copies overlap our tail, and its griddepcontrol.wait below holds it until this grid has completed.
    asm volatile("griddepcontrol.launch_dependents;");
    extern __shared__ float4 smem[];
    const int nsp = NSP ? NSP : fg.nsp;
    const Cta16Smem lay = cta16_smem(nsp, nface, stage_halo);
    float4* hbuf = smem + lay.hbuf;                                       // [8][3][nsp] half-spinor slots
    const uint4* opbuf = reinterpret_cast<const uint4*>(smem + lay.opbuf);  // [18][nsp] fp16 operands of the current domain
    float4* rstage = smem + lay.rstage;                                   // [6][nsp] residual of the current / next domain
    const float4* hstage = smem + lay.hstage;                             // [8][3][nface] halo slots (stage_halo)
    float4* red = smem + lay.red;                                         // [nwarps]
    int4* org_s = reinterpret_cast<int4*>(smem + lay.org);                // [2] first site of the current / next domain (table dom_org)
    const unsigned bar_links = cta_smem_u32(smem + lay.bars), bar_clov = bar_links + 8, bar_vec = bar_links + 16;
    const int k = threadIdx.x, lane = k & 31, warp = k >> 5;
    const bool active = NSP ? true : k < fg.ns;  // NSP = 256 is only launched for domains of exactly 256 sites
    const bool src_dm = r_dm != nullptr;

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
    // local coordinates and face indices (all < 256) travel through the block solve as one register each
    const unsigned lc_pk = (unsigned)lc[0] | (unsigned)lc[1] << 8 | (unsigned)lc[2] << 16 | (unsigned)lc[3] << 24;
    const unsigned fidx_pk = (unsigned)fidx[0] | (unsigned)fidx[1] << 8 | (unsigned)fidx[2] << 16 | (unsigned)fidx[3] << 24;
#define WC_FIDX(MU) ((int)((fidx_pk >> (8 * (MU))) & 255u))
#pragma unroll
    for (int j = 0; j < 24; j++) hbuf[j * nsp + k] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (k < 2 * (FUSED_CTA_MAX_THREADS / 32)) red[k] = make_float4(0.f, 0.f, 0.f, 0.f);  // warps that do not exist contribute zero
    if (k == 0) {
        mbar_init(bar_links, 1);
        mbar_init(bar_clov, 1);
        mbar_init(bar_vec, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const size_t V = fg.V;
    const unsigned half_bytes = 9u * chunk_bytes;                    // links or clover part of one domain
    const unsigned vec_bytes = (src_dm ? 6u * chunk_bytes : 0u) + (CHAIN && stage_halo ? 24u * (unsigned)nface * 16u : 0u);
    const unsigned op_addr = cta_smem_u32(opbuf), rs_addr = cta_smem_u32(rstage), hs_addr = cta_smem_u32(hstage);

    // staging requests for domain d (thread 0: bulk copies; every thread: its own residual column when the source is
    // in the lattice layout)
    auto request_links_vec = [&](int d) {
        if (k == 0) {
            mbar_expect_tx(bar_links, half_bytes);
            bulk_g2s(op_addr, dm16 + (size_t)d * 18 * nsp, half_bytes, bar_links);
            if (vec_bytes) {
                mbar_expect_tx(bar_vec, vec_bytes);
                if (src_dm) bulk_g2s(rs_addr, r_dm + (size_t)d * 6 * nsp, 6u * chunk_bytes, bar_vec);
                if (CHAIN && stage_halo) bulk_g2s(hs_addr, hb_in + (size_t)d * 24 * nface, 24u * (unsigned)nface * 16u, bar_vec);
            }
        }
    };
    auto request_clover = [&](int d) {
        if (k == 0) {
            mbar_expect_tx(bar_clov, half_bytes);
            bulk_g2s(op_addr + half_bytes, dm16 + ((size_t)d * 18 + 9) * nsp, half_bytes, bar_clov);
        }
    };
    // global site index of this thread's site in the domain whose Omega' starts at org (no division: table dom_org)
    auto site_of = [&](const int4& org) -> size_t {
        int x0 = org.x + (int)(lc_pk & 255u), x1 = org.y + (int)((lc_pk >> 8) & 255u), x2 = org.z + (int)((lc_pk >> 16) & 255u),
            x3 = org.w + (int)(lc_pk >> 24);
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

    // the operands do not depend on the previous kernel: their copies (and everything above) run ahead of it
    if ((int)blockIdx.x < ndl && k == 0) {
        const int dom0 = launch_dom(fg, blockIdx.x, colour);
        mbar_expect_tx(bar_links, half_bytes);
        bulk_g2s(op_addr, dm16 + (size_t)dom0 * 18 * nsp, half_bytes, bar_links);
        mbar_expect_tx(bar_clov, half_bytes);
        bulk_g2s(op_addr + half_bytes, dm16 + ((size_t)dom0 * 18 + 9) * nsp, half_bytes, bar_clov);
    }
    asm volatile("griddepcontrol.wait;" ::: "memory");  // residual, halo slots, phi: written by the kernels before this one
    if ((int)blockIdx.x < ndl) {
        const int dom0 = launch_dom(fg, blockIdx.x, colour);
        if (k == 0 && vec_bytes) {
            mbar_expect_tx(bar_vec, vec_bytes);
            if (src_dm) bulk_g2s(rs_addr, r_dm + (size_t)dom0 * 6 * nsp, 6u * chunk_bytes, bar_vec);
            if (CHAIN && stage_halo) bulk_g2s(hs_addr, hb_in + (size_t)dom0 * 24 * nface, 24u * (unsigned)nface * 16u, bar_vec);
        }
        if (k == 0) cp_async16(org_s, dom_org + dom0);  // committed with (or as) the first group below, waited for at the loop top
        if (!src_dm) request_r_lat(dom_org[dom0]);
        else cp_async_commit();
    }

#ifdef WC_CTA16_PROFILE
    long long prof[12] = {0}, tlast = clock64();
    int landed[3] = {0, 0, 0};
#endif
    // Per-launch uniforms the domain loop tests after its last stores, pinned in one register: rematerialised from the
    // constant bank there, each is a load of a few hundred cycles that the ncu source page shows as a long-scoreboard stall
    // of every warp at once (K_RAS application 0.769 -> 0.767 ms).  bit 0: halo out, bit 1: rho_fin out, bit 2: phi += v;
    // bits 8..: ndl.
    unsigned uni = (hb_out ? 1u : 0u) | (rho_dm ? 2u : 0u) | (phi_in ? 4u : 0u) | ((unsigned)ndl << 8);
    asm volatile("" : "+r"(uni));
#define WC_UNI_HALO (uni & 1u)
#define WC_UNI_RHO (uni & 2u)
#define WC_UNI_ACC (uni & 4u)
#define WC_UNI_NDL ((int)(uni >> 8))
    float U[72];
    // h (this domain) is carried and the exit test uses has_next from the top of the iteration: recomputed at the bottom, h
    // and the test cost an S2R and two constant-bank loads with nothing left to hide them behind (with the fixed offsets
    // of the small shared-memory tables: K_RAS application 0.784 -> 0.769 ms, plain launch 0.162 -> 0.158 ms)
    for (int j = 0, h = blockIdx.x; h < WC_UNI_NDL; j++) {
        WC_T(0)
        const unsigned par = (unsigned)j & 1u;
        const int hn = h + (int)gridDim.x;
        const bool has_next = hn < WC_UNI_NDL;
        const int dom = launch_dom(fg, h, colour);
        const int nxt = launch_dom(fg, has_next ? hn : h, colour);
        const unsigned dom_bc_here = WC_UNI_HALO ? __ldg(dom_bc + dom) : 0u;  // consumed by the halo scatter after the sweeps
        int4 org_nxt = make_int4(0, 0, 0, 0);
        if (!src_dm) org_nxt = __ldg(dom_org + nxt);  // lattice-layout source: the next residual column is requested below
        // ---- operands: links from the staged fp16 block into registers, scaled by -kappa ----
        mbar_wait(bar_links, par);
        WC_T(1)
#pragma unroll
        for (int c = 0; c < 9; c++) {
            float f[8];
            half8_to_float(opbuf[c * nsp + k], f);
#ifdef WC_X2
            const x2::c2 mk2 = x2::bc(mkappa);
#pragma unroll
            for (int n = 0; n < 4; n++) x2::st(U + 8 * c + 2 * n, x2::mul(x2::ld(f + 2 * n), mk2));
#else
#pragma unroll
            for (int n = 0; n < 8; n++) U[8 * c + n] = mkappa * f[n];
#endif
        }
        // ---- projection P_Omega' r: the staged residual column of this thread ----
        float rho[24], v[24];
        WC_T(2)
        cp_async_wait();  // own residual column (lattice-layout source); thread 0: the origin of this domain in org_s
        if (vec_bytes) mbar_wait(bar_vec, par);
        WC_T(3)
#pragma unroll
        for (int c = 0; c < 6; c++) {
            float4 t = rstage[c * nsp + k];
            if (!active) t = make_float4(0.f, 0.f, 0.f, 0.f);
            rho[4 * c] = t.x; rho[4 * c + 1] = t.y; rho[4 * c + 2] = t.z; rho[4 * c + 3] = t.w;
        }
        if (!src_dm && has_next) request_r_lat(org_nxt);  // own column: free as soon as it has been read
        WC_T(4)
        if (CHAIN) {
            // ---- boundary coupling: rho -= D-terms of v_{j-1} that cross the domain boundary (reading A3).  A lane
            // whose in-domain slot 2mu+1 (2mu) has no receiver sits on the upper (lower) face and receives the outside
            // forward (backward) hop from halo slot 2mu (2mu+1). ----
            const float4* hin = stage_halo ? hstage : hb_in + (size_t)dom * 24 * nface;
            float g[12], hh[12];
#define WC_CROSS_LOAD(SL)                                                                         \
    {                                                                                             \
        const bool rcv = active && dst[(SL) ^ 1] == 0xffffffffu;                                  \
        const float4* q4 = hin + (size_t)(SL) * 3 * nface + WC_FIDX((SL) >> 1);                      \
        _Pragma("unroll") for (int jj = 0; jj < 3; jj++) {                                        \
            float4 t = make_float4(0.f, 0.f, 0.f, 0.f);                                           \
            if (rcv) t = q4[(size_t)jj * nface];                                                  \
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
        WC_T(5)

        // q = D_Omega' in for sweep number it of this domain (the staging requests of the next domain hang on it): scatter
        // of the projected half spinors, clover term, barrier, gather
        auto apply_D = [&](const float (&in)[24], float (&q)[24], int it) {
            {
                float hs[12], g[12];
#define WC_SCATTER(MU)                                       \
    project<float, MU, -1>(in, hs);                          \
    st_half_pred(dst[2 * MU], chunk_bytes, hs);              \
    project<float, MU, +1>(in, hs);                          \
    su3_adj_mul<float>(U + 18 * MU, hs, g);                  \
    st_half_pred(dst[2 * MU + 1], chunk_bytes, g);
                WC_SCATTER(0) WC_SCATTER(1) WC_SCATTER(2) WC_SCATTER(3)
#undef WC_SCATTER
            }
            WC_T(6)
            if (it == 1) { WC_LANDED(0) }
            if (it == 0) mbar_wait(bar_clov, par);
            WC_T(7)
            // q = A in from the staged fp16 clover blocks: block 0 = halfs 0..35 (chunks 9..13), block 1 = halfs
            // 36..71 (chunks 13..17, chunk 13 read twice)
#pragma unroll
            for (int ch = 0; ch < 2; ch++) {
                float Ab[40];
#pragma unroll
                for (int c = 0; c < 5; c++) half8_to_float(opbuf[(9 + 4 * ch + c) * nsp + k], Ab + 8 * c);
                herm6_mul<float>(Ab + 4 * ch, in + 12 * ch, q + 12 * ch);
            }
            WC_T(8)
            __syncthreads();
            WC_T(9)
            // Every thread is past its staging reads of this domain (links, residual, halo: before the first barrier;
            // clover: before this barrier of the last sweep): thread 0 requests the next domain's data.
            if (has_next && warp == 0) {
                if (it == 0) {
                    request_links_vec(nxt);
                    if (k == 1) prefetch_l2_bulk(dm16 + ((size_t)nxt * 18 + 9) * nsp, half_bytes);
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
        };
        int it = 0;
        if (MR2) {
            // Restarted two-dimensional minimal residual (reading R2): per pair of sweeps q1 = D rho, q2 = D q1, then
            // (c1, c2) = argmin |rho - c1 q1 - c2 q2| from the 2x2 normal equations; v += c1 rho + c2 q1; rho -= c1 q1 + c2 q2
            for (; it + 1 < fg.niter; it += 2) {
                float q1[24], q2[24];
                apply_D(rho, q1, it);
                __syncthreads();  // every thread is past its gather: the slots may be rewritten
                apply_D(q1, q2, it + 1);
                float e[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};  // b1 (re, im), a11, b2 (re, im), a22, a12 (re, im)
#pragma unroll
                for (int n = 0; n < 12; n++) {
                    const float ar_ = q1[2 * n], ai_ = q1[2 * n + 1], br_ = q2[2 * n], bi_ = q2[2 * n + 1], rr = rho[2 * n], ri = rho[2 * n + 1];
                    e[0] = fmaf(ar_, rr, e[0]); e[0] = fmaf(ai_, ri, e[0]); e[1] = fmaf(ar_, ri, e[1]); e[1] = fmaf(-ai_, rr, e[1]);
                    e[2] = fmaf(ar_, ar_, e[2]); e[2] = fmaf(ai_, ai_, e[2]);
                    e[3] = fmaf(br_, rr, e[3]); e[3] = fmaf(bi_, ri, e[3]); e[4] = fmaf(br_, ri, e[4]); e[4] = fmaf(-bi_, rr, e[4]);
                    e[5] = fmaf(br_, br_, e[5]); e[5] = fmaf(bi_, bi_, e[5]);
                    e[6] = fmaf(ar_, br_, e[6]); e[6] = fmaf(ai_, bi_, e[6]); e[7] = fmaf(ar_, bi_, e[7]); e[7] = fmaf(-ai_, br_, e[7]);
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1)
#pragma unroll
                    for (int n = 0; n < 8; n++) e[n] += __shfl_xor_sync(0xffffffffu, e[n], o);
                if (lane == 0) {
                    red[warp] = make_float4(e[0], e[1], e[2], e[3]);
                    red[FUSED_CTA_MAX_THREADS / 32 + warp] = make_float4(e[4], e[5], e[6], e[7]);
                }
                __syncthreads();
                float t[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
                for (int n = 0; n < FUSED_CTA_MAX_THREADS / 32; n++) {
                    const float4 p = red[n], p2 = red[FUSED_CTA_MAX_THREADS / 32 + n];
                    t[0] += p.x; t[1] += p.y; t[2] += p.z; t[3] += p.w; t[4] += p2.x; t[5] += p2.y; t[6] += p2.z; t[7] += p2.w;
                }
                const float b1r = t[0], b1i = t[1], a11 = t[2], b2r = t[3], b2i = t[4], a22 = t[5], a12r = t[6], a12i = t[7];
                // scale-free 2x2 solve (reading R2): rows divided by a11 and a22, g = cos^2 of the angle between q1 and q2.  No
                // product of two squared norms: late in an inner solve they are ~1e-25 each and a11 a22 would underflow (a
                // denormal determinant turned into inf * 0 = NaN).  Squared norms below FLT_MIN count as zero.
                const float s1 = a11 >= 1.17549435e-38f ? 1.f / a11 : 0.f, s2 = a22 >= 1.17549435e-38f ? 1.f / a22 : 0.f;
                const float u1r = b1r * s1, u1i = b1i * s1, u2r = b2r * s2, u2i = b2i * s2;
                const float m1r = a12r * s1, m1i = a12i * s1, m2r = a12r * s2, m2i = -a12i * s2;  // a12 / a11, conj(a12) / a22
                const float g = s1 > 0.f && s2 > 0.f ? m1r * m2r - m1i * m2i : 1.f;              // m1 m2 = |a12|^2 / (a11 a22), real
                float c1r = u1r, c1i = u1i, c2r = 0.f, c2i = 0.f;  // q2 numerically parallel to q1, or rho = 0: the plain MR step
                if (1.f - g > 1e-4f) {
                    const float inv = 1.f / (1.f - g);
                    c1r = (u1r - (m1r * u2r - m1i * u2i)) * inv;  // c1 = (u1 - m1 u2) / (1 - g)
                    c1i = (u1i - (m1r * u2i + m1i * u2r)) * inv;
                    c2r = (u2r - (m2r * u1r - m2i * u1i)) * inv;  // c2 = (u2 - m2 u1) / (1 - g)
                    c2i = (u2i - (m2r * u1i + m2i * u1r)) * inv;
                }
                const bool upd_rho = it + 2 < fg.niter || WC_UNI_RHO;
#pragma unroll
                for (int n = 0; n < 12; n++) {
                    const float rr = rho[2 * n], ri = rho[2 * n + 1], xr = q1[2 * n], xi = q1[2 * n + 1];
                    float vr = v[2 * n], vi = v[2 * n + 1];
                    vr = fmaf(c1r, rr, vr); vr = fmaf(-c1i, ri, vr); vr = fmaf(c2r, xr, vr); vr = fmaf(-c2i, xi, vr);
                    vi = fmaf(c1r, ri, vi); vi = fmaf(c1i, rr, vi); vi = fmaf(c2r, xi, vi); vi = fmaf(c2i, xr, vi);
                    v[2 * n] = vr; v[2 * n + 1] = vi;
                    if (upd_rho) {
                        const float yr = q2[2 * n], yi = q2[2 * n + 1];
                        float nr = rr, ni = ri;
                        nr = fmaf(-c1r, xr, nr); nr = fmaf(c1i, xi, nr); nr = fmaf(-c2r, yr, nr); nr = fmaf(c2i, yi, nr);
                        ni = fmaf(-c1r, xi, ni); ni = fmaf(-c1i, xr, ni); ni = fmaf(-c2r, yi, ni); ni = fmaf(-c2i, yr, ni);
                        rho[2 * n] = nr; rho[2 * n + 1] = ni;
                    }
                }
                // (the barrier inside the next apply_D separates these reads of the partial table from its next writes)
            }
        }
        for (; it < fg.niter; it++) {
            float q[24];
            apply_D(rho, q, it);
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
            if (lane == 0) red[warp] = make_float4(d0, d1, d2, 0.f);
            WC_T(10)
            __syncthreads();
            WC_T(9)
            // fixed-order sum over the zero-padded table of FUSED_CTA_MAX_THREADS / 32 warp partials, independent loads
            float s0 = 0.f, s1 = 0.f, s2 = 0.f;
#pragma unroll
            for (int n = 0; n < FUSED_CTA_MAX_THREADS / 32; n++) {
                const float4 p = red[n];
                s0 += p.x; s1 += p.y; s2 += p.z;
            }
            // alpha = <q,rho>/<q,q>, 0 if <q,q> = 0 (Q9); v += alpha rho; rho -= alpha q
            const float inv = s2 > 0.f ? 1.f / s2 : 0.f;
            const float ar = s0 * inv, ai = s1 * inv;
            const bool upd_rho = it + 1 < fg.niter || WC_UNI_RHO;
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
        WC_T(11)
        WC_LANDED(1)
        // ---- halo scatter for the next cycle: the hops of v that leave the domain, as projected half spinors ----
        if (WC_UNI_HALO) {
            unsigned dd = dom_bc_here;
            int dstride = 1;
            float hs[12], g[12];
#define WC_HALO(MU)                                                                                              \
    {                                                                                                            \
        const int nb = fg.nblk[MU], bc = (int)(dd & 255u);                                                       \
        dd >>= 8;                                                                                                \
        if (active && dst[2 * MU] == 0xffffffffu) { /* lower face -> slot 2mu of the domain at -mu */            \
            const int nbd = bc == 0 ? dom + (nb - 1) * dstride : dom - dstride;                                  \
            float4* o = hb_out + ((size_t)nbd * 8 + 2 * MU) * 3 * nface + WC_FIDX(MU);                             \
            project<float, MU, -1>(v, hs);                                                                       \
            for (int jj = 0; jj < 3; jj++) o[(size_t)jj * nface] = make_float4(hs[4 * jj], hs[4 * jj + 1], hs[4 * jj + 2], hs[4 * jj + 3]); \
        }                                                                                                        \
        if (active && dst[2 * MU + 1] == 0xffffffffu) { /* upper face -> slot 2mu+1 of the domain at +mu */      \
            const int nbd = bc + 1 == nb ? dom - (nb - 1) * dstride : dom + dstride;                             \
            float4* o = hb_out + ((size_t)nbd * 8 + 2 * MU + 1) * 3 * nface + WC_FIDX(MU);                         \
            project<float, MU, +1>(v, hs);                                                                       \
            su3_adj_mul<float>(U + 18 * MU, hs, g);                                                              \
            for (int jj = 0; jj < 3; jj++) o[(size_t)jj * nface] = make_float4(g[4 * jj], g[4 * jj + 1], g[4 * jj + 2], g[4 * jj + 3]); \
        }                                                                                                        \
        dstride *= nb;                                                                                           \
    }
            WC_HALO(0) WC_HALO(1) WC_HALO(2) WC_HALO(3)
#undef WC_HALO
        }
        // ---- rho_fin (domain-major, every site of the domain) and the restriction R_Omega (bulk sites only) ----
        if (WC_UNI_RHO && active) {
            float4* o = rho_dm + (size_t)dom * 6 * nsp + k;
#pragma unroll
            for (int c = 0; c < 6; c++) o[(size_t)c * nsp] = make_float4(rho[4 * c], rho[4 * c + 1], rho[4 * c + 2], rho[4 * c + 3]);
        }
        if (bulk) {
            const size_t gi = site_of(org_s[j & 1]);  // visible since the first barrier of this domain
            if (WC_UNI_ACC) {
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
        WC_LANDED(2)
        if (!has_next) break;
        h = hn;
    }
#undef WC_UNI_HALO
#undef WC_UNI_RHO
#undef WC_UNI_ACC
#undef WC_UNI_NDL
#ifdef WC_CTA16_PROFILE
    if (k == 0 && blockIdx.x == 0)
        printf("cta16 prof chain %d niter %d: epi/loop %lld | links wait %lld cvt %lld | vec wait %lld rho %lld cross %lld | scatter %lld clov wait %lld "
               "clover %lld | barriers %lld gather+dots %lld update %lld\n", (int)CHAIN, fg.niter, prof[0], prof[1], prof[2], prof[3], prof[4], prof[5],
               prof[6], prof[7], prof[8], prof[9], prof[10], prof[11]);
    if (k == 0 && blockIdx.x == 0)
        printf("cta16 next links landed (of %d next domains) chain %d: after the scatter of sweep 1 %d, after the last update %d, after the epilogue %d\n",
               (ndl - 1 - (int)blockIdx.x) / (int)gridDim.x, (int)CHAIN, landed[0], landed[1], landed[2]);
#endif
}

// ---- host side ----
typedef void (*cta16_kernel_t)(FusedGeom, int, int, int, int, float, const uint4*, const float4*, const float4*, const float4*, float4*,
                               const float4*, float4*, float4*, const int4*, const unsigned*);
// the NSP = 256 instance: domains of exactly 256 sites (no padding lane: the kernel takes every thread as active)
static cta16_kernel_t cta16_kernel(bool chain, const FusedGeom& fg) {
    if (fg.mr2) {
        if (fg.nsp == 256 && fg.ns == 256) return chain ? ras_cta16_kernel<true, 256, true> : ras_cta16_kernel<false, 256, true>;
        return chain ? ras_cta16_kernel<true, 0, true> : ras_cta16_kernel<false, 0, true>;
    }
    if (fg.nsp == 256 && fg.ns == 256) return chain ? ras_cta16_kernel<true, 256, false> : ras_cta16_kernel<false, 256, false>;
    return chain ? ras_cta16_kernel<true, 0, false> : ras_cta16_kernel<false, 0, false>;
}

int ensure_halo(wcras_ctx* ctx, int nrhs);  // ras_cta.cu

// every launch carries the programmatic-stream-serialization attribute: behind another ras_cta16_kernel (which triggers its
// dependents at once) it starts as SMs fall free and waits in griddepcontrol.wait; behind any other kernel the attribute
// changes nothing
template <typename... Args>
static cudaError_t cta16_launch(wcras_ctx* ctx, bool chain, int grid, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3((unsigned)ctx->fused.nsp);
    cfg.dynamicSmemBytes = ctx->cta16_smem;
    cfg.stream = ctx->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, cta16_kernel(chain, ctx->fused), args...);
}

// Build the fp16 domain-major operand copy and the domain-major rho_fin buffer; returns 1 if this tier can run the
// configuration (single CTA per domain, shared memory fits), 0 otherwise (the caller falls back to ras_cta.cu).
int ras_cta16_prepare(wcras_ctx* ctx, const FusedGeom& fg, int nd, const Fields<float>& f) {
    if (fg.C != 1 || fg.nsp > FUSED_CTA_MAX_THREADS) return 0;
    for (int mu = 0; mu < 4; mu++) if (fg.nblk[mu] > 255) return 0;  // dom_bc packs the block coordinates into 8 bits each
    int nface = 1;
    for (int mu = 0; mu < 4; mu++) nface = fg.ns / fg.ext[mu] > nface ? fg.ns / fg.ext[mu] : nface;
    nface = (nface + 7) / 8 * 8;
    int dev = 0, sms = 0, smem_max = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    // Halo slots staged in shared memory by a bulk copy, unless leaving them in global memory lets one more CTA live on
    // an SM (128-site domains: 98 KB instead of 123 KB per CTA, two independent domains per SM hide each other's
    // barriers and memory phases)
    int stage_halo = 1, per_sm = 0;
    size_t smem = 0;
    {
        int best = 0;
        for (int sh = 1; sh >= 0; sh--) {
            const size_t b = cta16_smem(fg.nsp, nface, sh).bytes;
            if (b > (size_t)smem_max) continue;
            if (cudaFuncSetAttribute(cta16_kernel(false, fg), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)b) != cudaSuccess ||
                cudaFuncSetAttribute(cta16_kernel(true, fg), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)b) != cudaSuccess) {
                cudaGetLastError();
                continue;
            }
            int n = 0;
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, cta16_kernel(true, fg), fg.nsp, b) != cudaSuccess) { cudaGetLastError(); n = 0; }
            if (n > best) { best = n; stage_halo = sh; smem = b; }
        }
        per_sm = best;
        if (per_sm < 1) return 0;
        cudaFuncSetAttribute(cta16_kernel(false, fg), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        cudaFuncSetAttribute(cta16_kernel(true, fg), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    }
    if (ctx->dm16) { cudaStreamSynchronize(ctx->stream); cudaFree(ctx->dm16); ctx->dm16 = nullptr; }
    if (ctx->rf_dm) { cudaStreamSynchronize(ctx->stream); cudaFree(ctx->rf_dm); ctx->rf_dm = nullptr; }
    // one allocation for rho_fin [nd][6][nsp] float4, then the tables dom_org [nd] int4 and dom_bc [nd] unsigned
    const size_t rf_bytes = sizeof(float4) * 6 * (size_t)fg.nsp * nd;
    if (cudaMalloc((void**)&ctx->dm16, sizeof(uint4) * 18 * (size_t)fg.nsp * nd) != cudaSuccess) { cudaGetLastError(); ctx->dm16 = nullptr; return 0; }
    if (cudaMalloc((void**)&ctx->rf_dm, rf_bytes + (sizeof(int4) + sizeof(unsigned)) * (size_t)nd) != cudaSuccess) {
        cudaGetLastError();
        cudaFree(ctx->dm16);
        ctx->dm16 = nullptr; ctx->rf_dm = nullptr;
        return 0;
    }
    ctx->dom_org = reinterpret_cast<int4*>(reinterpret_cast<char*>(ctx->rf_dm) + rf_bytes);
    ctx->dom_bc = reinterpret_cast<unsigned*>(ctx->dom_org + nd);
    if (ctx->hb) { cudaFree(ctx->hb); ctx->hb = nullptr; }
    ctx->hb_nrhs = 0;
    ctx->nface = nface;
    ctx->stage_halo = stage_halo;
    ctx->cta16_smem = smem;
    pack_dm16_kernel<<<nd, fg.nsp, 0, ctx->stream>>>(fg, nd, f, ctx->dm16, ctx->dom_org, ctx->dom_bc);
    ctx->launches++;
    if (cudaGetLastError() != cudaSuccess) return 0;
    const long want = (long)per_sm * sms;
    ctx->cta_grid = (int)(nd < want ? nd : want);
    return 1;
}

// the rounded fp32 field copies (links, clover) used by every K_RAS path other than this file's in 16-bit operand mode
int ras_round_fields(wcras_ctx* ctx) {
    const size_t V = ctx->geom.V;
    if (!ctx->r16a) {
        if (alloc_dev(ctx, (void**)&ctx->r16a, sizeof(float4) * 16 * V)) return WCRAS_CUDA_ERROR;
        if (alloc_dev(ctx, (void**)&ctx->r16b, sizeof(float2) * 4 * V)) return WCRAS_CUDA_ERROR;
        if (alloc_dev(ctx, (void**)&ctx->r16c, sizeof(float4) * 18 * V)) return WCRAS_CUDA_ERROR;
        round_half_kernel<<<RED_BLOCKS, RED_THREADS, 0, ctx->stream>>>(64 * V, (const float*)ctx->g32a, (float*)ctx->r16a);
        round_half_kernel<<<RED_BLOCKS, RED_THREADS, 0, ctx->stream>>>(8 * V, (const float*)ctx->g32b, (float*)ctx->r16b);
        round_half_kernel<<<RED_BLOCKS, RED_THREADS, 0, ctx->stream>>>(72 * V, (const float*)ctx->c32, (float*)ctx->r16c);
        ctx->launches += 3;
        WC_CHECK_LAUNCH();
    }
    return WCRAS_OK;
}

int ras_cta16_block_solve(wcras_ctx* ctx, const float4* r, float4* vout, bool accum) {
    const FusedGeom& fg = ctx->fused;
    WC_CUDA(cta16_launch(ctx, false, ctx->cta_grid, fg, ctx->ras.nd, -1, ctx->nface, ctx->stage_halo, -(float)ctx->kappa, (const uint4*)ctx->dm16,
                         r, (const float4*)nullptr, (const float4*)nullptr, (float4*)nullptr, (const float4*)(accum ? vout : nullptr), vout,
                         (float4*)nullptr, (const int4*)ctx->dom_org, (const unsigned*)ctx->dom_bc));
    ctx->launches++;
    return WCRAS_OK;
}

// v = K_RAS r with NRAS chained cycles (overlap 0): one launch per cycle, no full-lattice D in between (reading A3).
// rho_fin travels domain-major through ctx->rf_dm (updated in place: a CTA reads and writes only its own domains);
// the halo buffer alternates between its two parities.
int ras_cta16_apply_chained(wcras_ctx* ctx, const float4* r, float4* v) {
    const FusedGeom& fg = ctx->fused;
    const int nras = ctx->ras.nras, nd = ctx->ras.nd, nface = ctx->nface;
    if (int rc = ensure_halo(ctx, 1)) return rc;
    float4* rf = ctx->rf_dm;
    const size_t hstride = (size_t)24 * nface * nd;
    float4* hb[2] = {ctx->hb, ctx->hb + hstride * ctx->hb_nrhs};
    const float mk = -(float)ctx->kappa;
    for (int j = 0; j < nras; j++) {
        const bool last = j == nras - 1;
        TimedRegion tr(ctx, TC_BLOCK);
        ctx->block_dv += ctx->ras.niter;
        if (j == 0)
            WC_CUDA(cta16_launch(ctx, false, ctx->cta_grid, fg, nd, -1, nface, ctx->stage_halo, mk, (const uint4*)ctx->dm16, r, (const float4*)nullptr,
                                 (const float4*)nullptr, last ? (float4*)nullptr : hb[0], (const float4*)nullptr, v, last ? (float4*)nullptr : rf,
                                 (const int4*)ctx->dom_org, (const unsigned*)ctx->dom_bc));
        else
            WC_CUDA(cta16_launch(ctx, true, ctx->cta_grid, fg, nd, -1, nface, ctx->stage_halo, mk, (const uint4*)ctx->dm16, (const float4*)nullptr,
                                 (const float4*)rf, (const float4*)hb[(j - 1) & 1], last ? (float4*)nullptr : hb[j & 1], (const float4*)v, v,
                                 last ? (float4*)nullptr : rf, (const int4*)ctx->dom_org, (const unsigned*)ctx->dom_bc));
        ctx->launches++;
    }
    WC_CHECK_LAUNCH();
    return WCRAS_OK;
}

// v = K_SAP r (multiplicative Schwarz, see ras_cta_apply_sap): red-black half steps, one launch per colour
int ras_cta16_apply_sap(wcras_ctx* ctx, const float4* r, float4* v) {
    const FusedGeom& fg = ctx->fused;
    const int ncyc = ctx->ras.nras, ndl = ctx->ras.nd / 2, nface = ctx->nface;
    if (int rc = ensure_halo(ctx, 1)) return rc;
    float4* rf = ctx->rf_dm;
    float4* hb = ctx->hb;
    const int grid = ndl < ctx->cta_grid ? ndl : ctx->cta_grid;
    const float mk = -(float)ctx->kappa;
    for (int step = 0; step < 2 * ncyc; step++) {
        const int colour = step & 1;
        const bool first_visit = step < 2, last_step = step == 2 * ncyc - 1, last_visit = step >= 2 * ncyc - 2;
        TimedRegion tr(ctx, TC_BLOCK);
        if (colour == 0) ctx->block_dv += ctx->ras.niter;
        const float4* r_lat = first_visit ? r : nullptr;
        const float4* r_dm = first_visit ? nullptr : rf;
        float4* rho_out = last_visit ? nullptr : rf;
        float4* halo_out = last_step ? nullptr : hb;
        if (step == 0)
            WC_CUDA(cta16_launch(ctx, false, grid, fg, ndl, colour, nface, ctx->stage_halo, mk, (const uint4*)ctx->dm16, r_lat, r_dm, (const float4*)nullptr,
                                 halo_out, (const float4*)nullptr, v, rho_out, (const int4*)ctx->dom_org, (const unsigned*)ctx->dom_bc));
        else
            WC_CUDA(cta16_launch(ctx, true, grid, fg, ndl, colour, nface, ctx->stage_halo, mk, (const uint4*)ctx->dm16, r_lat, r_dm, (const float4*)hb,
                                 halo_out, (const float4*)(first_visit ? nullptr : v), v, rho_out, (const int4*)ctx->dom_org,
                                 (const unsigned*)ctx->dom_bc));
        ctx->launches++;
    }
    WC_CHECK_LAUNCH();
    return WCRAS_OK;
}

}  // namespace wc
