// ras_stream.cu -- tier 2c of the RAS block solver (SURVEY.md 8(a) residency table: "spinors in DSMEM (cluster 16),
// links+clover streamed via L2"): extended domains too large for links and clover to stay on chip, e.g. the
// 10^4-site Omega' of BASELINE.json:configs[4] (8^4 blocks, overlap 1) or 12 x 8^3 (configs[2], 8x4^3, overlap 2).
// Steps A2-A4: projection P_Omega' r (Alg.1 line 4), N_dominv MR iterations on D_Omega' v = P r with
// Dirichlet boundaries (readings Q7, Q9), restriction R_Omega and the disjoint sum,
// optionally phi += v (line 9).  The paper keeps one such domain per GPU; here it is one thread-block
// cluster.
//
//   * Omega' is cut into C = c0 c1 c2 c3 <= 16 sub-blocks of at most 640 sites; one CTA per sub-block, one thread per
//     site, the C CTAs of a domain form a cluster; the grid is persistent (as many clusters as the chip holds).
//   * On chip, for the whole block solve: the MR vectors rho and v of the sub-block in shared memory (192 B per site,
//     120 KB at 625 sites), q in registers.  q = D_Omega' rho is a GATHER: every site reads the full spinors of its (up to) 8
//     neighbours from shared memory through a precomputed address: a shared::cta address for a neighbour in the same
//     CTA, the mapa result (DSMEM) for one in another CTA of the cluster, both read by the same generic load; a
//     neighbour outside Omega' is skipped (Dirichlet), wrap-around inside Omega' (ext = L) is kept.
//   * Links and clover are NOT resident: every sweep streams a domain-major operand record per site from global memory
//     -- 4 forward links, the 4 backward links U_mu(x-mu) already gathered to the site, the clover blocks; fp32 (58
//     16-byte chunks) or, in 16-bit operand mode (reading R1), fp16 (33 chunks = 528 B).  The N_dominv sweeps of a
//     domain re-read the same record, which L2 serves (a cluster's record is 5.3 MB in fp16 at 10^4 sites).  Pulling
//     the NEXT domain's record into L2 meanwhile (cp.async.bulk.prefetch.L2) was measured 5 % slower: it halves the L2
//     room of the records in use (ncu: L2 hit rate 51 %), so it is not done.
//   * Domain-local dots: warp shuffle -> one float4 per warp pushed to every CTA of the cluster -> fixed-order sum.
//     Two cluster barriers per MR iteration (dots; rho updated before the neighbours read it again).  Measured and not
//     kept (8^4 + overlap 1 at 32^4, fp16, 1.57 ms per launch of 4 sweeps): the partials by st.async onto an mbarrier and
//     the "rho in place" sync as remote mbarrier arrivals, 1.66 ms (20 polling warps take issue slots from the ones still
//     working; the barrier time is the wait for the slowest of 16 CTAs, not the barrier itself); the records through a
//     3-slot cp.async ring in shared memory two links ahead, 1.75 ms; prefetch.global.L1 one link ahead, 1.80 ms.
// Roofline: L2 operand stream, 528 (fp16) or 928 (fp32) B per site and sweep, against ~1.7 k fp32 instructions per site
// and sweep; HBM floor per block solve: one record + 96 B in per extended site, 96 B out per bulk site.
#include <cuda_fp16.h>

#include "wcras_internal.cuh"

namespace wc {

constexpr int STREAM_MAX_SITES = 640;
constexpr int STREAM_MAX_CLUSTER = 16;
constexpr unsigned ST_NONE = 0xffffffffu;

template <typename OP> struct Rec;
template <> struct Rec<__half> { static constexpr int LINK = 3, CLOV = 9, ALL = 8 * 3 + 9; };   // 16-byte chunks
template <> struct Rec<float> { static constexpr int LINK = 5, CLOV = 18, ALL = 8 * 5 + 18; };

__device__ __forceinline__ unsigned st_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ unsigned st_cluster_rank() {
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ unsigned st_mapa(unsigned addr, unsigned rank) {
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_cluster_push(unsigned addr, float a, float b, float c, float d) {
    asm volatile("st.shared::cluster.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
template <bool CL> __device__ __forceinline__ void st_barrier() {
    if (CL) {
        asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
        asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
    } else {
        __syncthreads();
    }
}

// n reals of a record (chunk stride = stride uint4) into fp32 registers
template <int NCHUNK, int NREAL, int SKIP = 0>
__device__ __forceinline__ void load_rec(const uint4* __restrict__ p, size_t stride, const __half*, float* out) {
    float f[NCHUNK * 8];
#pragma unroll
    for (int c = 0; c < NCHUNK; c++) {
        const uint4 t = __ldg(p + c * stride);
        const __half2* h = reinterpret_cast<const __half2*>(&t);
#pragma unroll
        for (int j = 0; j < 4; j++) {
            const float2 v = __half22float2(h[j]);
            f[8 * c + 2 * j] = v.x; f[8 * c + 2 * j + 1] = v.y;
        }
    }
#pragma unroll
    for (int n = 0; n < NREAL; n++) out[n] = f[SKIP + n];
}
template <int NCHUNK, int NREAL, int SKIP = 0>
__device__ __forceinline__ void load_rec(const uint4* __restrict__ p, size_t stride, const float*, float* out) {
    float f[NCHUNK * 4];
#pragma unroll
    for (int c = 0; c < NCHUNK; c++) {
        const uint4 t = __ldg(p + c * stride);
        f[4 * c] = __uint_as_float(t.x); f[4 * c + 1] = __uint_as_float(t.y);
        f[4 * c + 2] = __uint_as_float(t.z); f[4 * c + 3] = __uint_as_float(t.w);
    }
#pragma unroll
    for (int n = 0; n < NREAL; n++) out[n] = f[SKIP + n];
}

// the 36 packed reals of chiral block ch from the clover part of a record (p = its first chunk)
template <int CH>
__device__ __forceinline__ void load_clover_block(const uint4* __restrict__ p, size_t stride, const __half* t, float* Ab) {
    load_rec<5, 36, 4 * CH>(p + (size_t)(4 * CH) * stride, stride, t, Ab);  // halfs 36 CH .. 36 CH + 35 start inside chunk 4 CH
}
template <int CH>
__device__ __forceinline__ void load_clover_block(const uint4* __restrict__ p, size_t stride, const float* t, float* Ab) {
    load_rec<9, 36, 0>(p + (size_t)(9 * CH) * stride, stride, t, Ab);
}
// One load for both kinds of neighbour: a generic address whose low word is a shared::cta address (own CTA) or the
// result of mapa (another CTA of the cluster), the high word the shared window of the generic space.  A per-lane choice
// between ld.shared and ld.shared::cluster instead costs two predicated loads per chunk and an S2R per cluster load.
__device__ __forceinline__ float4 ld_window_f4(unsigned long long addr) {
    float4 v;
    asm volatile("ld.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(addr));
    return v;
}
__device__ __forceinline__ float4 ld_shared_f4(unsigned addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}

__device__ __forceinline__ void store_rec(uint4* p, size_t stride, int nchunk, const float* in, int nreal, const __half*) {
    for (int c = 0; c < nchunk; c++) {
        uint4 t;
        __half2* h = reinterpret_cast<__half2*>(&t);
        for (int j = 0; j < 4; j++) {
            const int n = 8 * c + 2 * j;
            h[j] = __floats2half2_rn(n < nreal ? in[n] : 0.f, n + 1 < nreal ? in[n + 1] : 0.f);
        }
        p[c * stride] = t;
    }
}
__device__ __forceinline__ void store_rec(uint4* p, size_t stride, int nchunk, const float* in, int nreal, const float*) {
    for (int c = 0; c < nchunk; c++) {
        uint4 t;
        unsigned* w = reinterpret_cast<unsigned*>(&t);
        for (int j = 0; j < 4; j++) {
            const int n = 4 * c + j;
            w[j] = __float_as_uint(n < nreal ? in[n] : 0.f);
        }
        p[c * stride] = t;
    }
}

// coordinates of this thread's site: lc in the sub-block, sc of the sub-block, ec in Omega'
__device__ __forceinline__ void stream_coords(const FusedGeom& fg, int k, int rank, int lc[4], int sc[4], int ec[4]) {
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        lc[mu] = k % fg.sb[mu]; k /= fg.sb[mu];
        sc[mu] = rank % fg.c[mu]; rank /= fg.c[mu];
        ec[mu] = sc[mu] * fg.sb[mu] + lc[mu];
    }
}
__device__ __forceinline__ void stream_site(const FusedGeom& fg, int dom, const int ec[4], int x[4]) {
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        const int bc = dom % fg.nblk[mu];
        dom /= fg.nblk[mu];
        int st = bc * fg.b[mu] - (fg.split[mu] ? fg.s : 0) + ec[mu];
        if (st < 0) st += fg.L[mu];
        if (st >= fg.L[mu]) st -= fg.L[mu];
        x[mu] = st;
    }
}

// pack the operand records: one CTA per (domain, cluster rank), one thread per site
template <typename OP>
__global__ void pack_stream_kernel(FusedGeom fg, Fields<float> f, uint4* __restrict__ rec) {
    typedef Rec<OP> R;
    const int dom = blockIdx.x / fg.C, rank = blockIdx.x % fg.C, k = threadIdx.x;
    const size_t stride = fg.nsp;
    uint4* out = rec + (size_t)blockIdx.x * R::ALL * stride + k;
    if (k >= fg.ns) {
        for (int c = 0; c < R::ALL; c++) out[c * stride] = make_uint4(0u, 0u, 0u, 0u);
        return;
    }
    int lc[4], sc[4], ec[4], x[4];
    stream_coords(fg, k, rank, lc, sc, ec);
    stream_site(fg, dom, ec, x);
    const size_t V = fg.V;
    const size_t gi = x[0] + fg.L[0] * (x[1] + fg.L[1] * (x[2] + (size_t)fg.L[2] * x[3]));
    const size_t gs[4] = {1, (size_t)fg.L[0], (size_t)fg.L[0] * fg.L[1], (size_t)fg.L[0] * fg.L[1] * fg.L[2]};
    float u[72];
    for (int mu = 0; mu < 4; mu++) {
        load_link(f, V, gi, mu, u);
        store_rec(out + (size_t)(mu * R::LINK) * stride, stride, R::LINK, u, 18, (const OP*)nullptr);
        // backward link U_mu(x - mu), periodic on the lattice; unused (zero) when x - mu is outside Omega'
        const bool inside = ec[mu] > 0 || fg.wrap[mu];
        const size_t gj = x[mu] == 0 ? gi + (size_t)(fg.L[mu] - 1) * gs[mu] : gi - gs[mu];
        if (inside) load_link(f, V, gj, mu, u);
        else for (int n = 0; n < 18; n++) u[n] = 0.f;
        store_rec(out + (size_t)((4 + mu) * R::LINK) * stride, stride, R::LINK, u, 18, (const OP*)nullptr);
    }
    load_clover(f, V, gi, u);
    store_rec(out + (size_t)(8 * R::LINK) * stride, stride, R::CLOV, u, 72, (const OP*)nullptr);
}

template <typename OP, bool CL>
__global__ void __launch_bounds__(STREAM_MAX_SITES, 1)
ras_stream_kernel(FusedGeom fg, int nd, float kappa, const uint4* __restrict__ rec, const float4* __restrict__ r,
                  float4* __restrict__ vout, int accum) {
    typedef Rec<OP> R;
    if (fg.stop && __ldg(fg.stop)) return;  // the inner solver has converged (launch enqueued ahead of the host's check)
    extern __shared__ float4 smem[];
    const int nsp = fg.nsp;
    float4* rho = smem;             // [6][nsp] MR residual: read by the neighbours, also across the cluster
    float4* vv = smem + 6 * nsp;    // [6][nsp] MR iterate (private to the site; kept here to free registers)
    float4* red = smem + 12 * nsp;  // [C * nwarps]
    const int k = threadIdx.x, lane = k & 31, warp = k >> 5, nwarps = blockDim.x >> 5;
    const unsigned rank = CL ? st_cluster_rank() : 0u;
    const int dom0 = CL ? blockIdx.x / fg.C : blockIdx.x, nclus = CL ? gridDim.x / fg.C : gridDim.x;
    const bool active = k < fg.ns;
    const unsigned chunk_bytes = (unsigned)nsp * 16u;
    const size_t stride = nsp;

    int lc[4], sc[4], ec[4];
    stream_coords(fg, active ? k : 0, (int)rank, lc, sc, ec);
    bool bulk = active;
#pragma unroll
    for (int mu = 0; mu < 4; mu++)
        if (fg.split[mu]) bulk = bulk && ec[mu] >= fg.s && ec[mu] < fg.s + fg.b[mu];
    // cluster-space address of chunk 0 of rho at the neighbour in direction (mu, +) [index 2mu] and (mu, -) [2mu+1]
    unsigned nbr[8];
    const unsigned long long win = (unsigned long long)(size_t)rho & 0xffffffff00000000ull;  // shared window of the generic space
    {
        const unsigned base = st_smem_u32(rho);
        int lstride = 1, cstride = 1;
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
#pragma unroll
            for (int sg = 0; sg < 2; sg++) {  // sg 0: x + mu, sg 1: x - mu
                int kd = k, rk = (int)rank;
                bool ok = active;
                if (sg == 0) {
                    if (lc[mu] + 1 < fg.sb[mu]) kd += lstride;
                    else {
                        kd -= (fg.sb[mu] - 1) * lstride;
                        if (sc[mu] + 1 < fg.c[mu]) rk += cstride;
                        else if (fg.wrap[mu]) rk -= (fg.c[mu] - 1) * cstride;
                        else ok = false;
                    }
                } else {
                    if (lc[mu] > 0) kd -= lstride;
                    else {
                        kd += (fg.sb[mu] - 1) * lstride;
                        if (sc[mu] > 0) rk -= cstride;
                        else if (fg.wrap[mu]) rk += (fg.c[mu] - 1) * cstride;
                        else ok = false;
                    }
                }
                // a neighbour in this CTA keeps its shared::cta address (served by the local shared memory at full
                // bandwidth); only a neighbour in another CTA gets a cluster-window address (DSMEM, ~20 B/clk per SM)
                unsigned a = base + (unsigned)kd * 16u;
                if (CL && rk != (int)rank) a = st_mapa(a, (unsigned)rk);
                nbr[2 * mu + sg] = ok ? a : ST_NONE;
            }
            lstride *= fg.sb[mu];
            cstride *= fg.c[mu];
        }
    }
    for (int dom = dom0; dom < nd; dom += nclus) {
        const uint4* myrec = rec + ((size_t)dom * fg.C + rank) * R::ALL * stride + k;
        int x[4];
        stream_site(fg, dom, ec, x);
        const size_t V = fg.V;
        const size_t gi = x[0] + fg.L[0] * (x[1] + fg.L[1] * (x[2] + (size_t)fg.L[2] * x[3]));
        // ---- projection P_Omega' r -> rho, v = 0; the next domain's record towards L2 ----
#pragma unroll
        for (int c = 0; c < 6; c++) {
            rho[c * nsp + k] = active ? r[(size_t)c * V + gi] : make_float4(0.f, 0.f, 0.f, 0.f);
            vv[c * nsp + k] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        st_barrier<CL>();  // every CTA of the cluster has its rho in place

        for (int it = 0; it < fg.niter; it++) {
            // ---- q = D_Omega' rho at the own site: gather over the neighbours inside Omega' ----
            float hop[24];
#pragma unroll
            for (int n = 0; n < 24; n++) hop[n] = 0.f;
#define WC_ST_DIR(MU)                                                                                         \
    if (nbr[2 * MU] != ST_NONE) {                                                                             \
        float u[18], sn[24];                                                                                  \
        load_rec<R::LINK, 18>(myrec + (size_t)(MU * R::LINK) * stride, stride, (const OP*)nullptr, u);        \
        _Pragma("unroll") for (int c = 0; c < 6; c++) {                                                       \
            const float4 t = CL ? ld_window_f4(win | (nbr[2 * MU] + c * chunk_bytes)) : ld_shared_f4(nbr[2 * MU] + c * chunk_bytes); \
            sn[4 * c] = t.x; sn[4 * c + 1] = t.y; sn[4 * c + 2] = t.z; sn[4 * c + 3] = t.w;                   \
        }                                                                                                     \
        hop_fwd<float, MU>(u, sn, hop);                                                                       \
    }                                                                                                         \
    if (nbr[2 * MU + 1] != ST_NONE) {                                                                         \
        float u[18], sn[24];                                                                                  \
        load_rec<R::LINK, 18>(myrec + (size_t)((4 + MU) * R::LINK) * stride, stride, (const OP*)nullptr, u);  \
        _Pragma("unroll") for (int c = 0; c < 6; c++) {                                                       \
            const float4 t = CL ? ld_window_f4(win | (nbr[2 * MU + 1] + c * chunk_bytes)) : ld_shared_f4(nbr[2 * MU + 1] + c * chunk_bytes); \
            sn[4 * c] = t.x; sn[4 * c + 1] = t.y; sn[4 * c + 2] = t.z; sn[4 * c + 3] = t.w;                   \
        }                                                                                                     \
        hop_bwd<float, MU>(u, sn, hop);                                                                       \
    }
            WC_ST_DIR(0) WC_ST_DIR(1) WC_ST_DIR(2) WC_ST_DIR(3)
#undef WC_ST_DIR
            float rs[24], q[24];
#pragma unroll
            for (int c = 0; c < 6; c++) {
                const float4 t = rho[c * nsp + k];
                rs[4 * c] = t.x; rs[4 * c + 1] = t.y; rs[4 * c + 2] = t.z; rs[4 * c + 3] = t.w;
            }
            {
                float Ab[36];
                load_clover_block<0>(myrec + (size_t)(8 * R::LINK) * stride, stride, (const OP*)nullptr, Ab);
                herm6_mul<float>(Ab, rs, q);
                load_clover_block<1>(myrec + (size_t)(8 * R::LINK) * stride, stride, (const OP*)nullptr, Ab);
                herm6_mul<float>(Ab, rs + 12, q + 12);
            }
            float d0 = 0.f, d1 = 0.f, d2 = 0.f;
#ifdef WC_X2
            {
                const x2::c2 mk = x2::bc(-kappa);
#pragma unroll
                for (int n = 0; n < 12; n++) x2::st(q + 2 * n, x2::fma(mk, x2::ld(hop + 2 * n), x2::ld(q + 2 * n)));
            }
            x2::mr_dots(q, rs, d0, d1, d2);
#else
#pragma unroll
            for (int n = 0; n < 24; n++) q[n] = fmaf(-kappa, hop[n], q[n]);
#pragma unroll
            for (int n = 0; n < 12; n++) {
                const float qr = q[2 * n], qi = q[2 * n + 1], rr = rs[2 * n], ri = rs[2 * n + 1];
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
            {
                const unsigned slot = st_smem_u32(red + rank * nwarps + warp);
                if (CL) {
                    if (lane < fg.C) st_cluster_push(st_mapa(slot, (unsigned)lane), d0, d1, d2, 0.f);
                } else if (lane == 0) {
                    red[warp] = make_float4(d0, d1, d2, 0.f);
                }
            }
            st_barrier<CL>();  // dots complete; every CTA is past its neighbour reads of this sweep
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
            const float inv = s2 > 0.f ? 1.f / s2 : 0.f;
            const float ar = s0 * inv, ai = s1 * inv;
            const bool last = it + 1 == fg.niter;
#pragma unroll
            for (int c = 0; c < 6; c++) {
                float4 t = vv[c * nsp + k];
#ifdef WC_X2
                float va[4] = {t.x, t.y, t.z, t.w};
                if (!last) x2::mr_update<true, 2>(ar, ai, q + 4 * c, rs + 4 * c, va);
                else x2::mr_update<false, 2>(ar, ai, q + 4 * c, rs + 4 * c, va);
                vv[c * nsp + k] = make_float4(va[0], va[1], va[2], va[3]);
                if (!last) rho[c * nsp + k] = make_float4(rs[4 * c], rs[4 * c + 1], rs[4 * c + 2], rs[4 * c + 3]);
#else
                const float r0 = rs[4 * c], r1 = rs[4 * c + 1], r2 = rs[4 * c + 2], r3 = rs[4 * c + 3];
                t.x = fmaf(ar, r0, t.x); t.x = fmaf(-ai, r1, t.x);
                t.y = fmaf(ar, r1, t.y); t.y = fmaf(ai, r0, t.y);
                t.z = fmaf(ar, r2, t.z); t.z = fmaf(-ai, r3, t.z);
                t.w = fmaf(ar, r3, t.w); t.w = fmaf(ai, r2, t.w);
                vv[c * nsp + k] = t;
                if (!last) {
                    float4 n4;
                    n4.x = fmaf(-ar, q[4 * c], r0); n4.x = fmaf(ai, q[4 * c + 1], n4.x);
                    n4.y = fmaf(-ar, q[4 * c + 1], r1); n4.y = fmaf(-ai, q[4 * c], n4.y);
                    n4.z = fmaf(-ar, q[4 * c + 2], r2); n4.z = fmaf(ai, q[4 * c + 3], n4.z);
                    n4.w = fmaf(-ar, q[4 * c + 3], r3); n4.w = fmaf(-ai, q[4 * c + 2], n4.w);
                    rho[c * nsp + k] = n4;
                }
#endif
            }
            if (!last) st_barrier<CL>();  // the new rho of every CTA is in place before the next sweep reads it
        }
        // ---- restriction R_Omega: bulk sites only; disjoint over domains, so a plain store (or phi += v) ----
        if (bulk) {
#pragma unroll
            for (int c = 0; c < 6; c++) {
                float4 t = vv[c * nsp + k];
                if (accum) {
                    const float4 o = vout[(size_t)c * V + gi];
                    t.x += o.x; t.y += o.y; t.z += o.z; t.w += o.w;
                }
                vout[(size_t)c * V + gi] = t;
            }
        }
    }
}

// ---- host side ----
// Cut of Omega' into <= 16 sub-blocks of <= 640 sites: minimal cluster size, then the most cubic sub-block.
static bool stream_cut(const int ext[4], int c[4], int sb[4]) {
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
        if (C > STREAM_MAX_CLUSTER || ns > STREAM_MAX_SITES) continue;
        const int spread = mx - mn;
        if (C < best_C || (C == best_C && spread < best_spread)) {
            best_C = (int)C; best_spread = spread; found = true;
            for (int mu = 0; mu < 4; mu++) { c[mu] = cc[mu]; sb[mu] = ext[mu] / cc[mu]; }
        }
    }
    return found;
}

static size_t stream_smem_bytes(const FusedGeom& fg) { return sizeof(float4) * ((size_t)12 * fg.nsp + (size_t)fg.C * (fg.nsp / 32)); }

template <typename OP, bool CL>
static cudaError_t stream_launch_cfg(const FusedGeom& fg, int nclus, cudaStream_t stream, cudaLaunchConfig_t* cfg, cudaLaunchAttribute* at) {
    *cfg = cudaLaunchConfig_t{};
    cfg->gridDim = dim3((unsigned)nclus * fg.C);
    cfg->blockDim = dim3((unsigned)fg.nsp);
    cfg->dynamicSmemBytes = stream_smem_bytes(fg);
    cfg->stream = stream;
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)fg.C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg->attrs = at;
    cfg->numAttrs = CL ? 1 : 0;
    return cudaSuccess;
}

template <typename OP, bool CL>
static cudaError_t stream_prepare_kernel(const FusedGeom& fg, int* max_clusters) {
    auto kern = ras_stream_kernel<OP, CL>;
    const size_t smem = stream_smem_bytes(fg);
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (!CL) {
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
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute at[1];
    stream_launch_cfg<OP, CL>(fg, 1, nullptr, &cfg, at);
    return cudaOccupancyMaxActiveClusters(max_clusters, kern, &cfg);
}

// Fill *out and return 1 if the extended domain fits this tier on this device.
int ras_stream_prepare(wcras_ctx* ctx, const int b[4], const int ext[4], int s, int niter, FusedGeom* out) {
    FusedGeom fg;
    if (!stream_cut(ext, fg.c, fg.sb)) return 0;
    fg.ns = 1; fg.C = 1;
    for (int mu = 0; mu < 4; mu++) {
        fg.L[mu] = ctx->geom.L[mu]; fg.b[mu] = b[mu]; fg.nblk[mu] = ctx->geom.L[mu] / b[mu]; fg.ext[mu] = ext[mu];
        fg.split[mu] = b[mu] < ctx->geom.L[mu];
        fg.wrap[mu] = ext[mu] == ctx->geom.L[mu];
        fg.ns *= fg.sb[mu]; fg.C *= fg.c[mu];
    }
    fg.V = ctx->geom.V; fg.s = s; fg.niter = niter; fg.pdir = -1; fg.stop = nullptr;
    fg.nsp = (fg.ns + 31) / 32 * 32;
    int dev = 0, smem_max = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (stream_smem_bytes(fg) > (size_t)smem_max) return 0;
    int nclusters = 0;
    const bool half = ctx->op_prec == 16;
    cudaError_t e;
    if (fg.C > 1) e = half ? stream_prepare_kernel<__half, true>(fg, &nclusters) : stream_prepare_kernel<float, true>(fg, &nclusters);
    else e = half ? stream_prepare_kernel<__half, false>(fg, &nclusters) : stream_prepare_kernel<float, false>(fg, &nclusters);
    if (e != cudaSuccess || nclusters < 1) { cudaGetLastError(); return 0; }
    fg.nclus = nclusters;
    *out = fg;
    return 1;
}

// build the operand records in ctx->dm (shared slot with the other fused tiers); returns 0 when memory is short
int ras_stream_pack(wcras_ctx* ctx, const FusedGeom& fg, int nd, const Fields<float>& f) {
    const bool half = ctx->op_prec == 16;
    const size_t chunks = half ? Rec<__half>::ALL : Rec<float>::ALL;
    if (ctx->dm) { cudaStreamSynchronize(ctx->stream); cudaFree(ctx->dm); ctx->dm = nullptr; }
    if (cudaMalloc((void**)&ctx->dm, sizeof(uint4) * chunks * fg.nsp * (size_t)fg.C * nd) != cudaSuccess) { cudaGetLastError(); ctx->dm = nullptr; return 0; }
    if (half) pack_stream_kernel<__half><<<nd * fg.C, fg.nsp, 0, ctx->stream>>>(fg, f, reinterpret_cast<uint4*>(ctx->dm));
    else pack_stream_kernel<float><<<nd * fg.C, fg.nsp, 0, ctx->stream>>>(fg, f, reinterpret_cast<uint4*>(ctx->dm));
    ctx->launches++;
    if (cudaGetLastError() != cudaSuccess) { cudaFree(ctx->dm); ctx->dm = nullptr; return 0; }
    ctx->stream_half = half ? 1 : 0;
    return 1;
}

template <typename OP, bool CL>
static cudaError_t stream_launch(wcras_ctx* ctx, const FusedGeom& fg, int nd, const float4* r, float4* vout, int accum) {
    const int nclus = nd < fg.nclus ? nd : fg.nclus;
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute at[1];
    stream_launch_cfg<OP, CL>(fg, nclus, ctx->stream, &cfg, at);
    return cudaLaunchKernelEx(&cfg, ras_stream_kernel<OP, CL>, fg, nd, (float)ctx->kappa, reinterpret_cast<const uint4*>(ctx->dm), r, vout, accum);
}

int ras_stream_block_solve(wcras_ctx* ctx, const float4* r, float4* vout, bool accum) {
    const FusedGeom& fg = ctx->fused;
    const int nd = ctx->ras.nd, a = accum ? 1 : 0;
    cudaError_t e;
    if (fg.C > 1) e = ctx->stream_half ? stream_launch<__half, true>(ctx, fg, nd, r, vout, a) : stream_launch<float, true>(ctx, fg, nd, r, vout, a);
    else e = ctx->stream_half ? stream_launch<__half, false>(ctx, fg, nd, r, vout, a) : stream_launch<float, false>(ctx, fg, nd, r, vout, a);
    WC_CUDA(e);
    ctx->launches++;
    return WCRAS_OK;
}

}  // namespace wc
