// ras_fused.cu -- tier 2 of the RAS block solver (north_star (c)): the whole block solve of one domain runs on
// chip in ONE launch.  Steps A2-A4 of SURVEY.md 8(a): projection P_Omega' r (Alg.1 line 4), N_dominv
// MR iterations on D_Omega' v = P r with Dirichlet boundaries (readings Q7, Q9), restriction
// R_Omega and the disjoint sum, optionally fused with phi += v (Alg.1 line 9).
//
// Mapping (north_star: "domains map onto CTAs or thread-block clusters"):
//   * The extended domain Omega' (extents ext[mu]) is cut into c[0] x c[1] x c[2] x c[3] sub-blocks of shape
//     sb[mu] = ext[mu]/c[mu] with at most 256 sites each; one CTA per sub-block, one thread per site, and the
//     C = prod c[mu] <= 16 CTAs of a domain form one thread-block cluster (C = 1: a plain CTA).
//   * Per thread, for the whole solve, IN REGISTERS (clover: shared memory): its 4 forward links U_mu(x) (72 reals), its clover
//     blocks A(x) (72 reals), the MR residual rho(x) and the iterate v(x) (24 reals each).  Links and clover
//     are read from HBM exactly once per block solve.
//   * Only projected half spinors (12 reals) travel between sites, through shared memory: in every MR
//     iteration site x scatters P^-_mu rho(x) to x-mu and U_mu(x)^dag P^+_mu rho(x) to x+mu (8 x 48 B), then
//     gathers its own 8 slots, multiplies the forward ones by its own links and reconstructs.  A neighbour in
//     another CTA of the cluster is reached with st.shared::cluster (DSMEM); a neighbour outside Omega' is
//     never written and its slot stays zero = Dirichlet boundary.  Wrap-around inside Omega' (ext = L) is kept.
//   * The domain-local dots <q,rho>, <q,q> go warp shuffle -> one float4 per warp pushed to every CTA of the
//     cluster -> summed in a fixed order by every warp after the barrier (deterministic, no atomics).
//   * PERSISTENT: the grid holds as many clusters as fit on the chip (cudaOccupancyMaxActiveClusters); a cluster walks
//     over its domains and prefetches the operands and the residual of the next one into L2 while it solves one.
//   * Two barriers per MR iteration (barrier.cluster arrive/wait when C > 1, bar.sync when C = 1).
// Shared memory per CTA: 8 x 3 float4 x 256 = 96 KB of half-spinor slots + 72 KB of clover blocks (own column per
// thread, read back one chiral block at a time) + 2 KB of dot partials.
// Roofline: HBM floor = (96 + 576) B per extended site in + 96 B per bulk site out; the N_dominv sweeps are bound
// by fp32 issue (~1.3 k instructions per site-sweep) and shared-memory traffic (768 B per site-sweep).
#include "wcras_internal.cuh"

namespace wc {

constexpr int FUSED_MAX_THREADS = 256;
constexpr int FUSED_MAX_CLUSTER = 16;


__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ unsigned cluster_rank() {
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ unsigned map_to_rank(unsigned addr, unsigned rank) {
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_cluster_f4(unsigned addr, float a, float b, float c, float d) {
    asm volatile("st.shared::cluster.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
__device__ __forceinline__ void st_local_f4(unsigned addr, float a, float b, float c, float d) {
    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
template <bool CL> __device__ __forceinline__ void barrier_arrive() {
    if (CL) asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
}
template <bool CL> __device__ __forceinline__ void barrier_wait() {
    if (CL) asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
    else __syncthreads();
}

// 12 reals -> slot (3 float4 with a stride of nsp float4); NONE = no receiver (Dirichlet)
constexpr unsigned NO_DST = 0xffffffffu;
template <bool CL>
__device__ __forceinline__ void st_half(unsigned dst, unsigned chunk_bytes, const float* h) {
    if (dst == NO_DST) return;
#pragma unroll
    for (int j = 0; j < 3; j++) {
        if (CL) st_cluster_f4(dst + j * chunk_bytes, h[4 * j], h[4 * j + 1], h[4 * j + 2], h[4 * j + 3]);
        else st_local_f4(dst + j * chunk_bytes, h[4 * j], h[4 * j + 1], h[4 * j + 2], h[4 * j + 3]);
    }
}
__device__ __forceinline__ void ld_half(const float4* __restrict__ slot, int nsp, float* h) {
#pragma unroll
    for (int j = 0; j < 3; j++) {
        const float4 v = slot[j * nsp];
        h[4 * j] = v.x; h[4 * j + 1] = v.y; h[4 * j + 2] = v.z; h[4 * j + 3] = v.w;
    }
}

template <bool CL>
__global__ void __launch_bounds__(FUSED_MAX_THREADS, 1)
ras_fused_kernel(FusedGeom fg, int nd, Fields<float> f, float kappa, const float4* r, float4* __restrict__ vout, int accum,
                 int nface, const float4* __restrict__ hb_in, float4* __restrict__ hb_out, float4* rho_out,
                 const float4* __restrict__ dmc) {
    // r and rho_out are the same buffer in the chained cycles (a thread reads its site before it writes it): no __restrict__
    // dmc (overlap 0 only): domain-major operand copy float4 [nd][C][36][nsp] -- the 72 link reals, then the 72 clover
    // reals of the sites of one CTA contiguous (147 KB), as in ras_cta.cu but with the links unscaled
    // Chained cycles (overlap 0; same scheme as ras_cta.cu, reading A3): hb_in != nullptr: r is rho_fin of the
    // previous cycle and the hops of the previous v that cross the domain boundary are subtracted from it (halo slots
    // filled by the neighbouring domains); hb_out: halo scatter of this cycle's v; rho_out: rho_fin of this cycle.
    if (fg.stop && __ldg(fg.stop)) return;  // the inner solver has converged (launch enqueued ahead of the host's check)
    extern __shared__ float4 smem[];
    const int nsp = fg.nsp;                 // threads per CTA = slots per chunk
    float4* hbuf = smem;                    // [8][3][nsp]
    float4* As = smem + 24 * nsp;           // [18][nsp] clover blocks, each thread its own column (as in ras_cta.cu)
    float4* red = smem + 42 * nsp;          // [C * nwarps]
    const int k = threadIdx.x, lane = k & 31, warp = k >> 5, nwarps = blockDim.x >> 5;
    const unsigned rank = CL ? cluster_rank() : 0u;
    // PERSISTENT: a cluster (or CTA) walks over the domains dom0, dom0 + nclus, ...; while it solves one, the operands
    // and the residual of its next one are pulled from HBM into L2 (prefetch.global.L2)
    const int dom0 = CL ? blockIdx.x / fg.C : blockIdx.x, nclus = CL ? gridDim.x / fg.C : gridDim.x;
    const bool active = k < fg.ns;

    // ---- geometry of this thread's site ----
    int lc[4], sc[4], ec[4];                // coords in the sub-block, of the sub-block, in Omega'
    {
        int kk = active ? k : 0, rr = (int)rank;
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            lc[mu] = kk % fg.sb[mu]; kk /= fg.sb[mu];
            sc[mu] = rr % fg.c[mu]; rr /= fg.c[mu];
            ec[mu] = sc[mu] * fg.sb[mu] + lc[mu];
        }
    }
    bool bulk = active;
#pragma unroll
    for (int mu = 0; mu < 4; mu++)
        if (fg.split[mu]) bulk = bulk && ec[mu] >= fg.s && ec[mu] < fg.s + fg.b[mu];
    int fidx[4];  // index of the site within the mu-face of Omega' (coordinate mu removed), unique over the cluster
    {
        int E = 0, es = 1;
#pragma unroll
        for (int mu = 0; mu < 4; mu++) { E += ec[mu] * es; es *= fg.ext[mu]; }
        es = 1;
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            fidx[mu] = (E % es) + (E / (es * fg.ext[mu])) * es;
            es *= fg.ext[mu];
        }
    }
    auto site_of = [&](int d) -> size_t {  // global site index of this thread's site in domain d
        int x[4];
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            const int bc = d % fg.nblk[mu];
            d /= fg.nblk[mu];
            int st = bc * fg.b[mu] - (fg.split[mu] ? fg.s : 0) + ec[mu];
            if (st < 0) st += fg.L[mu];
            if (st >= fg.L[mu]) st -= fg.L[mu];
            x[mu] = st;
        }
        return x[0] + fg.L[0] * (x[1] + fg.L[1] * (x[2] + (size_t)fg.L[2] * x[3]));
    };
    // destination slot of the half spinor sent in direction (mu, -) [index 2mu: receiver x-mu uses it for its
    // forward hop] and (mu, +) [index 2mu+1: receiver x+mu, backward hop]
    const unsigned chunk_bytes = (unsigned)nsp * 16u;
    unsigned dst[8];
    {
        const unsigned base = smem_u32(hbuf);
        int lstride = 1, cstride = 1;
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
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
                unsigned a = base + (unsigned)((2 * mu + sg) * 3 * nsp + kd) * 16u;
                if (CL) a = map_to_rank(a, (unsigned)rk);
                dst[2 * mu + sg] = ok ? a : NO_DST;
            }
            lstride *= fg.sb[mu];
            cstride *= fg.c[mu];
        }
    }

    // ---- zero the slots (Dirichlet faces are never written), load the site data ----
#pragma unroll
    for (int j = 0; j < 24; j++) hbuf[j * nsp + k] = make_float4(0.f, 0.f, 0.f, 0.f);
    barrier_arrive<CL>();
    barrier_wait<CL>();  // every CTA of the cluster has zeroed its slots before anybody scatters into them
    for (int dom = dom0; dom < nd; dom += nclus) {
    const size_t gi = site_of(dom);
    float U[72], rho[24], v[24];
    if (dmc) {
        const float4* p = dmc + ((size_t)dom * fg.C + rank) * 36 * nsp + k;  // zero-filled for the inactive lanes
#pragma unroll
        for (int c = 0; c < 18; c++) {
            const float4 t = __ldcs(p + (size_t)c * nsp);
            U[4 * c] = t.x; U[4 * c + 1] = t.y; U[4 * c + 2] = t.z; U[4 * c + 3] = t.w;
        }
#pragma unroll
        for (int c = 0; c < 18; c++) As[c * nsp + k] = __ldcs(p + (size_t)(18 + c) * nsp);
        if (active) {
            load_spinor(r, (size_t)fg.V, gi, rho);
        } else {
#pragma unroll
            for (int n = 0; n < 24; n++) rho[n] = 0.f;
        }
    } else if (active) {
#pragma unroll
        for (int mu = 0; mu < 4; mu++) load_link(f, (size_t)fg.V, gi, mu, U + 18 * mu);
#pragma unroll
        for (int c = 0; c < 18; c++) As[c * nsp + k] = f.cl[(size_t)c * fg.V + gi];
        load_spinor(r, (size_t)fg.V, gi, rho);  // projection P_Omega' r
    } else {
#pragma unroll
        for (int n = 0; n < 72; n++) U[n] = 0.f;
#pragma unroll
        for (int c = 0; c < 18; c++) As[c * nsp + k] = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int n = 0; n < 24; n++) rho[n] = 0.f;
    }
    if (hb_in) {
        // boundary coupling: rho += kappa [ recon^-(U h_2mu) + recon^+(h_2mu+1) ] over the halo slots of this domain; a
        // lane whose in-domain slot 2mu+1 (2mu) has no receiver sits on the upper (lower) face and receives slot 2mu (2mu+1)
        const float4* hin = hb_in + (size_t)dom * 24 * nface;
        float g[12], hh[12];
#define WC_CROSS(MU)                                                                                   \
    {                                                                                                  \
        const bool up = active && dst[2 * MU + 1] == NO_DST, lo = active && dst[2 * MU] == NO_DST;     \
        if (__any_sync(0xffffffffu, up)) {                                                             \
            for (int j = 0; j < 3; j++) {                                                              \
                float4 t = make_float4(0.f, 0.f, 0.f, 0.f);                                            \
                if (up) t = hin[((size_t)(2 * MU) * 3 + j) * nface + fidx[MU]];                        \
                hh[4 * j] = kappa * t.x; hh[4 * j + 1] = kappa * t.y; hh[4 * j + 2] = kappa * t.z; hh[4 * j + 3] = kappa * t.w; \
            }                                                                                          \
            su3_mul<float>(U + 18 * MU, hh, g);                                                        \
            reconstruct_add<float, MU, -1>(g, rho);                                                    \
        }                                                                                              \
        if (__any_sync(0xffffffffu, lo)) {                                                             \
            for (int j = 0; j < 3; j++) {                                                              \
                float4 t = make_float4(0.f, 0.f, 0.f, 0.f);                                            \
                if (lo) t = hin[((size_t)(2 * MU + 1) * 3 + j) * nface + fidx[MU]];                    \
                hh[4 * j] = kappa * t.x; hh[4 * j + 1] = kappa * t.y; hh[4 * j + 2] = kappa * t.z; hh[4 * j + 3] = kappa * t.w; \
            }                                                                                          \
            reconstruct_add<float, MU, +1>(hh, rho);                                                   \
        }                                                                                              \
    }
        WC_CROSS(0) WC_CROSS(1) WC_CROSS(2) WC_CROSS(3)
#undef WC_CROSS
    }
#pragma unroll
    for (int n = 0; n < 24; n++) v[n] = 0.f;
    if (dom + nclus < nd && dmc && k == 0)
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(dmc + ((size_t)(dom + nclus) * fg.C + rank) * 36 * nsp),
                     "r"(36u * (unsigned)nsp * 16u) : "memory");
    if (dom + nclus < nd && active) {  // next domain of this cluster towards L2
        const size_t gn = site_of(dom + nclus), V = fg.V;
        if (!dmc) {
#pragma unroll
            for (int c = 0; c < 16; c++) asm volatile("prefetch.global.L2 [%0];" ::"l"(f.ga + (size_t)c * V + gn));
#pragma unroll
            for (int c = 0; c < 4; c++) asm volatile("prefetch.global.L2 [%0];" ::"l"(f.gb + (size_t)c * V + gn));
#pragma unroll
            for (int c = 0; c < 18; c++) asm volatile("prefetch.global.L2 [%0];" ::"l"(f.cl + (size_t)c * V + gn));
        }
#pragma unroll
        for (int c = 0; c < 6; c++) asm volatile("prefetch.global.L2 [%0];" ::"l"(r + (size_t)c * V + gn));
    }

    for (int it = 0; it < fg.niter; it++) {
        // ---- scatter: projected half spinors to the 8 neighbours ----
        {
            float h[12], g[12];
#define WC_SCATTER(MU)                                            \
    project<float, MU, -1>(rho, h);                               \
    st_half<CL>(dst[2 * MU], chunk_bytes, h);                     \
    project<float, MU, +1>(rho, h);                               \
    su3_adj_mul<float>(U + 18 * MU, h, g);                        \
    st_half<CL>(dst[2 * MU + 1], chunk_bytes, g);
            WC_SCATTER(0) WC_SCATTER(1) WC_SCATTER(2) WC_SCATTER(3)
#undef WC_SCATTER
        }
        barrier_arrive<CL>();
        float q[24];
        // q = A rho from the shared-memory copy, one chiral block at a time; independent of the exchange: overlaps the barrier
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
        barrier_wait<CL>();
        // ---- gather: q = A rho - kappa * hop ----
        {
            float hop[24];
#pragma unroll
            for (int n = 0; n < 24; n++) hop[n] = 0.f;
            float h[12], g[12];
#define WC_GATHER(MU)                                             \
    ld_half(hbuf + (2 * MU) * 3 * nsp + k, nsp, h);               \
    su3_mul<float>(U + 18 * MU, h, g);                            \
    reconstruct_add<float, MU, -1>(g, hop);                       \
    ld_half(hbuf + (2 * MU + 1) * 3 * nsp + k, nsp, g);           \
    reconstruct_add<float, MU, +1>(g, hop);
            WC_GATHER(0) WC_GATHER(1) WC_GATHER(2) WC_GATHER(3)
#undef WC_GATHER
#pragma unroll
            for (int n = 0; n < 24; n++) q[n] -= kappa * hop[n];
        }
        // ---- domain-local dots <q,rho>, <q,q> ----
        float d0 = 0.f, d1 = 0.f, d2 = 0.f;
#pragma unroll
        for (int n = 0; n < 12; n++) {
            const float qr = q[2 * n], qi = q[2 * n + 1], rr = rho[2 * n], ri = rho[2 * n + 1];
            d0 += qr * rr + qi * ri;
            d1 += qr * ri - qi * rr;
            d2 += qr * qr + qi * qi;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            d0 += __shfl_xor_sync(0xffffffffu, d0, o);
            d1 += __shfl_xor_sync(0xffffffffu, d1, o);
            d2 += __shfl_xor_sync(0xffffffffu, d2, o);
        }
        {
            const unsigned slot = smem_u32(red + rank * nwarps + warp);
            if (CL) {
                if (lane < fg.C) st_cluster_f4(map_to_rank(slot, (unsigned)lane), d0, d1, d2, 0.f);
            } else if (lane == 0) {
                st_local_f4(slot, d0, d1, d2, 0.f);
            }
        }
        barrier_arrive<CL>();
        barrier_wait<CL>();
        float s0 = 0.f, s1 = 0.f, s2 = 0.f;
        for (int n = lane; n < fg.C * nwarps; n += 32) {
            const float4 p = red[n];
            s0 += p.x; s1 += p.y; s2 += p.z;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            s0 += __shfl_xor_sync(0xffffffffu, s0, o);
            s1 += __shfl_xor_sync(0xffffffffu, s1, o);
            s2 += __shfl_xor_sync(0xffffffffu, s2, o);
        }
        // alpha = <q,rho>/<q,q>, 0 if <q,q> = 0 (Q9); v += alpha rho; rho -= alpha q
        const float ar = s2 > 0.f ? s0 / s2 : 0.f, ai = s2 > 0.f ? s1 / s2 : 0.f;
        const bool last = it + 1 == fg.niter && rho_out == nullptr;  // rho_fin is needed by the next chained cycle
#pragma unroll
        for (int n = 0; n < 12; n++) {
            const float rr = rho[2 * n], ri = rho[2 * n + 1];
            v[2 * n] += ar * rr - ai * ri;
            v[2 * n + 1] += ar * ri + ai * rr;
            if (!last) {
                rho[2 * n] = rr - (ar * q[2 * n] - ai * q[2 * n + 1]);
                rho[2 * n + 1] = ri - (ar * q[2 * n + 1] + ai * q[2 * n]);
            }
        }
    }
    if (hb_out) {
        // halo scatter for the next cycle: the hops of v that leave the domain, as projected half spinors
        int dd = dom, dstride = 1;
        float h[12], g[12];
#define WC_HALO(MU)                                                                                              \
    {                                                                                                            \
        const int nb = fg.nblk[MU], bc = dd % nb;                                                                \
        dd /= nb;                                                                                                \
        if (active && dst[2 * MU] == NO_DST) { /* lower face -> slot 2mu of the domain at -mu */                 \
            const int nbd = bc == 0 ? dom + (nb - 1) * dstride : dom - dstride;                                  \
            float4* o = hb_out + ((size_t)nbd * 8 + 2 * MU) * 3 * nface + fidx[MU];                              \
            project<float, MU, -1>(v, h);                                                                        \
            for (int j = 0; j < 3; j++) o[(size_t)j * nface] = make_float4(h[4 * j], h[4 * j + 1], h[4 * j + 2], h[4 * j + 3]); \
        }                                                                                                        \
        if (active && dst[2 * MU + 1] == NO_DST) { /* upper face -> slot 2mu+1 of the domain at +mu */           \
            const int nbd = bc + 1 == nb ? dom - (nb - 1) * dstride : dom + dstride;                             \
            float4* o = hb_out + ((size_t)nbd * 8 + 2 * MU + 1) * 3 * nface + fidx[MU];                          \
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
        if (rho_out) store_spinor(rho_out, (size_t)fg.V, gi, rho);
        if (accum) {
            float o[24];
            load_spinor(vout, (size_t)fg.V, gi, o);
#pragma unroll
            for (int n = 0; n < 24; n++) v[n] += o[n];
        }
        store_spinor(vout, (size_t)fg.V, gi, v);
    }
    }  // domains of this cluster
}

// pack the domain-major operand copy of the cluster tier: one CTA per (domain, cluster rank), one thread per site
__global__ void pack_cluster_dm_kernel(FusedGeom fg, Fields<float> f, float4* __restrict__ dmc) {
    const int dom = blockIdx.x / fg.C, rank = blockIdx.x % fg.C, k = threadIdx.x;
    float4* out = dmc + (size_t)blockIdx.x * 36 * fg.nsp + k;
    if (k >= fg.ns) {
        for (int c = 0; c < 36; c++) out[(size_t)c * fg.nsp] = make_float4(0.f, 0.f, 0.f, 0.f);
        return;
    }
    int kk = k, rr = rank, d = dom, x[4];
    for (int mu = 0; mu < 4; mu++) {
        const int lc = kk % fg.sb[mu]; kk /= fg.sb[mu];
        const int sc = rr % fg.c[mu]; rr /= fg.c[mu];
        const int bc = d % fg.nblk[mu]; d /= fg.nblk[mu];
        int st = bc * fg.b[mu] - (fg.split[mu] ? fg.s : 0) + sc * fg.sb[mu] + lc;
        if (st < 0) st += fg.L[mu];
        if (st >= fg.L[mu]) st -= fg.L[mu];
        x[mu] = st;
    }
    const size_t gi = x[0] + fg.L[0] * (x[1] + fg.L[1] * (x[2] + (size_t)fg.L[2] * x[3])), V = fg.V;
    float u[72];
    for (int mu = 0; mu < 4; mu++) load_link(f, V, gi, mu, u + 18 * mu);
    for (int c = 0; c < 18; c++) out[(size_t)c * fg.nsp] = make_float4(u[4 * c], u[4 * c + 1], u[4 * c + 2], u[4 * c + 3]);
    for (int c = 0; c < 18; c++) out[(size_t)(18 + c) * fg.nsp] = f.cl[(size_t)c * V + gi];
}

// ---- host side ----
// Choose the cut of Omega' into sub-blocks: minimal cluster size, then the most cubic sub-block.
static bool choose_cut(const int ext[4], int c[4], int sb[4]) {
    int best_C = 1 << 30, best_spread = 1 << 30;
    bool found = false;
    for (int c0 = 1; c0 <= ext[0]; c0++) if (ext[0] % c0 == 0)
    for (int c1 = 1; c1 <= ext[1]; c1++) if (ext[1] % c1 == 0)
    for (int c2 = 1; c2 <= ext[2]; c2++) if (ext[2] % c2 == 0)
    for (int c3 = 1; c3 <= ext[3]; c3++) if (ext[3] % c3 == 0) {
        const int cc[4] = {c0, c1, c2, c3};
        long C = (long)c0 * c1 * c2 * c3, ns = 1;
        int mx = 0, mn = 1 << 30;
        for (int mu = 0; mu < 4; mu++) {
            const int e = ext[mu] / cc[mu];
            ns *= e; mx = e > mx ? e : mx; mn = e < mn ? e : mn;
        }
        if (C > FUSED_MAX_CLUSTER || ns > FUSED_MAX_THREADS) continue;
        const int spread = mx - mn;
        if (C < best_C || (C == best_C && spread < best_spread)) {
            best_C = (int)C; best_spread = spread; found = true;
            for (int mu = 0; mu < 4; mu++) { c[mu] = cc[mu]; sb[mu] = ext[mu] / cc[mu]; }
        }
    }
    return found;
}

static FusedGeom make_fused_geom(const wcras_ctx* ctx, const int b[4], const int ext[4], int s, int niter, bool* ok) {
    FusedGeom fg;
    *ok = choose_cut(ext, fg.c, fg.sb);
    fg.ns = 1; fg.C = 1;
    for (int mu = 0; mu < 4; mu++) {
        fg.L[mu] = ctx->geom.L[mu]; fg.b[mu] = b[mu]; fg.nblk[mu] = ctx->geom.L[mu] / b[mu]; fg.ext[mu] = ext[mu];
        fg.split[mu] = b[mu] < ctx->geom.L[mu];
        fg.wrap[mu] = ext[mu] == ctx->geom.L[mu];
        if (*ok) { fg.ns *= fg.sb[mu]; fg.C *= fg.c[mu]; }
    }
    fg.V = ctx->geom.V; fg.s = s; fg.niter = niter; fg.stop = nullptr;
    fg.nsp = (fg.ns + 31) / 32 * 32;
    return fg;
}

static size_t fused_smem_bytes(const FusedGeom& fg) { return sizeof(float4) * ((size_t)42 * fg.nsp + (size_t)fg.C * (fg.nsp / 32)); }

template <bool CL>
static cudaError_t prepare_fused(const FusedGeom& fg, int* max_clusters) {
    auto kern = ras_fused_kernel<CL>;
    const size_t smem = fused_smem_bytes(fg);
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (!CL) {  // plain CTAs: resident CTAs per SM x SMs
        int per_sm = 0, dev = 0, sms = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, fg.nsp, smem);
        if (e != cudaSuccess) return e;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        *max_clusters = per_sm * sms;
        return cudaSuccess;
    }
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, fg.C > 8 ? 1 : 0);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)fg.C);
    cfg.blockDim = dim3((unsigned)fg.nsp);
    cfg.dynamicSmemBytes = smem;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)fg.C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaOccupancyMaxActiveClusters(max_clusters, kern, &cfg);
}

template <bool CL>
static cudaError_t launch_fused(const FusedGeom& fg, int nd, int nclus, cudaStream_t stream, const Fields<float>& f, float kappa,
                                const float4* r, float4* vout, int accum, int nface = 0, const float4* hb_in = nullptr,
                                float4* hb_out = nullptr, float4* rho_out = nullptr, const float4* dmc = nullptr) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)nclus * fg.C);
    cfg.blockDim = dim3((unsigned)fg.nsp);
    cfg.dynamicSmemBytes = fused_smem_bytes(fg);
    cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)fg.C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = CL ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, ras_fused_kernel<CL>, fg, nd, f, kappa, r, vout, accum, nface, hb_in, hb_out, rho_out, dmc);
}

// Fill *out and return 1 if the extended domain fits the fused tier on this device: a cut into <= 16 sub-blocks of
// <= 256 sites exists and the cluster can be scheduled (cudaOccupancyMaxActiveClusters > 0).
int ras_fused_prepare(const wcras_ctx* ctx, const int b[4], const int ext[4], int s, int niter, FusedGeom* out) {
    bool ok;
    const FusedGeom fg = make_fused_geom(ctx, b, ext, s, niter, &ok);
    if (!ok) return 0;
    int nclusters = 0;
    const cudaError_t e = fg.C > 1 ? prepare_fused<true>(fg, &nclusters) : prepare_fused<false>(fg, &nclusters);
    if (e != cudaSuccess) { cudaGetLastError(); return 0; }
    if (nclusters < 1) return 0;
    FusedGeom fgo = fg;
    fgo.nclus = nclusters;
    *out = fgo;
    return 1;
}

int ensure_halo(wcras_ctx* ctx, int nrhs);  // ras_cta.cu

// overlap 0: build the domain-major operand copy of the cluster tier in ctx->dm (shared slot with tier 2a); on failure
// (memory) the kernel falls back to the SoA fields
void ras_fused_pack(wcras_ctx* ctx, const FusedGeom& fg, int nd) {
    if (ctx->dm) { cudaStreamSynchronize(ctx->stream); cudaFree(ctx->dm); ctx->dm = nullptr; }
    if (fg.s != 0) return;
    const size_t bytes = sizeof(float4) * 36 * (size_t)fg.nsp * fg.C * nd;
    if (cudaMalloc((void**)&ctx->dm, bytes) != cudaSuccess) { cudaGetLastError(); ctx->dm = nullptr; return; }
    pack_cluster_dm_kernel<<<nd * fg.C, fg.nsp, 0, ctx->stream>>>(fg, ras_fields(ctx), ctx->dm);
    ctx->launches++;
    if (cudaGetLastError() != cudaSuccess) { cudaFree(ctx->dm); ctx->dm = nullptr; }
}

// v = K_RAS r with NRAS chained cycles on the cluster tier (overlap 0, one right-hand side): as ras_cta_apply_chained
int ras_fused_apply_chained(wcras_ctx* ctx, const float4* r, float4* v) {
    const FusedGeom& fg = ctx->fused;
    const Fields<float> f = ras_fields(ctx);
    const int nras = ctx->ras.nras, nd = ctx->ras.nd, nface = ctx->nface;
    const int nclus = nd < fg.nclus ? nd : fg.nclus;
    if (int rc = ensure_halo(ctx, 1)) return rc;
    float4* rf = ctx->ras32[0];
    const size_t hstride = (size_t)24 * nface * nd;
    float4* hb[2] = {ctx->hb, ctx->hb + hstride * ctx->hb_nrhs};
    for (int j = 0; j < nras; j++) {
        const bool last = j == nras - 1;
        TimedRegion tr(ctx, TC_BLOCK);
        ctx->block_dv += ctx->ras.niter;
        const float4* src = j == 0 ? r : rf;
        const float4* hin = j == 0 ? nullptr : hb[(j - 1) & 1];
        float4* hout = last ? nullptr : hb[j & 1];
        float4* rout = last ? nullptr : rf;
        if (fg.C > 1) WC_CUDA(launch_fused<true>(fg, nd, nclus, ctx->stream, f, (float)ctx->kappa, src, v, j > 0, nface, hin, hout, rout, ctx->dm));
        else WC_CUDA(launch_fused<false>(fg, nd, nclus, ctx->stream, f, (float)ctx->kappa, src, v, j > 0, nface, hin, hout, rout, ctx->dm));
        ctx->launches++;
    }
    return WCRAS_OK;
}

int ras_fused_block_solve(wcras_ctx* ctx, const float4* r, float4* vout, bool accum) {
    const FusedGeom& fg = ctx->fused;
    const Fields<float> f = ras_fields(ctx);
    const int nclus = ctx->ras.nd < fg.nclus ? ctx->ras.nd : fg.nclus;
    if (fg.C > 1) WC_CUDA(launch_fused<true>(fg, ctx->ras.nd, nclus, ctx->stream, f, (float)ctx->kappa, r, vout, accum ? 1 : 0, 0, nullptr, nullptr, nullptr, ctx->dm));
    else WC_CUDA(launch_fused<false>(fg, ctx->ras.nd, nclus, ctx->stream, f, (float)ctx->kappa, r, vout, accum ? 1 : 0, 0, nullptr, nullptr, nullptr, ctx->dm));
    ctx->launches++;
    return WCRAS_OK;
}

}  // namespace wc
