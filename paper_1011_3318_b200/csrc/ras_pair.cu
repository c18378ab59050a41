// ras_pair.cu -- tier 2a of the RAS block solver, TWO THREADS PER SITE (fp16 operand storage, TMA staging as in
// ras_cta16.cu).  Steps A2-A5 of SURVEY.md 8(a): projection P_Omega' r (Alg.1 line 4), N_dominv MR
// iterations on D_Omega' v = P r with Dirichlet boundaries (readings Q7, Q9), restriction R_Omega, the
// disjoint sum, phi += v (line 9), chained cycles (reading A3); extended domains of <= 256 sites, one
// persistent CTA of 2 x nsp threads walking over its domains.
//
// Why: with one thread per site the solver needs 230+ registers per thread, i.e. 8 warps per SM = 2 per scheduler, and
// issues at ~55-65 % of the slots (ncu: stalls on fixed-latency dependencies and shared-memory loads).  Here a site is
// shared by the lanes l and l + 16 of one warp ("halves" p = 0, 1); each half owns two of the four directions and one of
// the two chiralities, needs <= 128 registers, and the SM holds 16 warps = 4 per scheduler.
// RESULT (profiles/r2_kernels.md): correct (same parity tests), but SLOWER than ras_cta16.cu -- 410 against 337 us for
// four sweeps at 32^4: the issue rate rises only from 64 % to 69 % of the slots (1.9 eligible warps per cycle, the rest
// are dispatch and math-pipe stalls: the fp32 pipe and its register-file ports are the limit, not latency) while the
// instruction count grows by 32 % (exchange shuffles, selections, FFMA with sign registers instead of FADD, replicated
// address arithmetic).  It is therefore NOT the default: wcras_set_ras_tier(ctx, 6) selects it.
//
//   half 0: directions x, y; owns the upper chirality (spins 0,1); stores a spinor as R = (psi_up, psi_low)
//   half 1: directions z, t; owns the lower chirality;             stores a spinor as R = (W psi_low, psi_up),
//           W = -i sigma_2 = [[0,-1],[1,0]] on the spin index of the chirality
// In the chiral basis gamma_mu = [[0, B_mu], [B_mu^dag, 0]] with B_x = -i s1, B_y = -i s2, B_z = -i s3, B_t = 1, and a hop
// is  h = psi_up + s B psi_low,  g = U h,  out_up += g,  out_low += s B^dag g  (s = -1 forward, +1 backward).  In the
// storage of half 1 the same hop reads  h~ = R_up + s (W B^dag) R_low,  acc_up += g~,  acc_low += s (W B^dag)^dag g~  with
// the exchanged half spinor h~ = s W B^dag h; and W B_z^dag = -B_x, W B_t^dag = B_y.  BOTH HALVES THEREFORE RUN THE SAME
// INSTRUCTIONS: "slot A" = the x projector with a per-thread sign (+1 for half 0, -1 for half 1), "slot B" = the y
// projector; the clover block of half 1 is stored as W A_low W^dag.  (Checked numerically before the kernel was written;
// parity tests against the oracle cover every direction and both signs.)
//   * the halves exchange their contributions to the other chirality with __shfl_xor(.., 16): 12 reals of q per MR
//     iteration and the 12 updated reals of rho (the W rotation is a register selection and a sign);
//   * half-spinor slots, TMA-staged operands / residual / halo and the persistent domain loop are those of ras_cta16.cu;
//     operand record per site: 20 chunks of 8 halfs = [links x,y | links z,t | clover up | W clover low W^dag], each
//     group 36 halfs padded to 40 (320 B per site).
#include "ras_cta_common.cuh"

namespace wc {

constexpr int PAIR_MAX_THREADS = 2 * FUSED_CTA_MAX_THREADS;
constexpr int PAIR_CHUNKS = 20;

// ---- slot A: x projector with a runtime sign c = s * e (e = +1 half 0, -1 half 1) ----
// h = R_up + c B_x R_low,  B_x = -i sigma_1:  h0 = R0 - i c R3,  h1 = R1 - i c R2
__device__ __forceinline__ void project_a(const float* __restrict__ R, float* __restrict__ h, float c) {
#pragma unroll
    for (int col = 0; col < 3; col++) {
        const float s0r = R[2 * col], s0i = R[2 * col + 1], s1r = R[6 + 2 * col], s1i = R[6 + 2 * col + 1];
        const float s2r = R[12 + 2 * col], s2i = R[12 + 2 * col + 1], s3r = R[18 + 2 * col], s3i = R[18 + 2 * col + 1];
        h[2 * col] = fmaf(c, s3i, s0r); h[2 * col + 1] = fmaf(-c, s3r, s0i);
        h[6 + 2 * col] = fmaf(c, s2i, s1r); h[6 + 2 * col + 1] = fmaf(-c, s2r, s1i);
    }
}
// acc_up += g,  acc_low += c B_x^dag g,  B_x^dag = i sigma_1:  low0 += i c g1,  low1 += i c g0
__device__ __forceinline__ void reconstruct_a(const float* __restrict__ g, float* __restrict__ acc, float c, float sg) {
#pragma unroll
    for (int col = 0; col < 3; col++) {
        const float g0r = g[2 * col], g0i = g[2 * col + 1], g1r = g[6 + 2 * col], g1i = g[6 + 2 * col + 1];
        acc[2 * col] = fmaf(sg, g0r, acc[2 * col]); acc[2 * col + 1] = fmaf(sg, g0i, acc[2 * col + 1]);
        acc[6 + 2 * col] = fmaf(sg, g1r, acc[6 + 2 * col]); acc[6 + 2 * col + 1] = fmaf(sg, g1i, acc[6 + 2 * col + 1]);
        const float cs = c * sg;
        acc[12 + 2 * col] = fmaf(-cs, g1i, acc[12 + 2 * col]); acc[12 + 2 * col + 1] = fmaf(cs, g1r, acc[12 + 2 * col + 1]);
        acc[18 + 2 * col] = fmaf(-cs, g0i, acc[18 + 2 * col]); acc[18 + 2 * col + 1] = fmaf(cs, g0r, acc[18 + 2 * col + 1]);
    }
}

// The 12 reals a half receives from its partner, rotated into its own storage.  The partner's reals arrive in the
// partner's storage of that chirality; for half 0 <- half 1 that is already psi_up; for half 1 <- half 0 it is psi_low and
// W applies: out[0..5] = -in[6..11], out[6..11] = in[0..5].  TO_LOW: the received chirality is the receiver's R_low
// (rho refresh, v for the halo) -- then half 1 receives psi_up unrotated and half 0 receives W psi_low and un-rotates it
// with W^dag: out[0..5] = in[6..11], out[6..11] = -in[0..5].  `rot` says whether this thread rotates, `neg` carries the sign.
template <bool TO_LOW>
__device__ __forceinline__ void rotate_recv(const float* __restrict__ in, float* __restrict__ out, bool rot, float neg) {
#pragma unroll
    for (int j = 0; j < 12; j++) {
        const float t = rot ? in[(j + 6) % 12] : in[j];
        const bool flip = TO_LOW ? j >= 6 : j < 6;
        out[j] = flip ? neg * t : t;
    }
}
__device__ __forceinline__ void exchange12(const float* __restrict__ mine, float* __restrict__ theirs) {
#pragma unroll
    for (int j = 0; j < 12; j++) theirs[j] = __shfl_xor_sync(0xffffffffu, mine[j], 16);
}

// pack the pair operand records; also the per-domain tables (as pack_dm16_kernel).  One thread per (domain, site).
__global__ void pack_pair_kernel(FusedGeom fg, int nd, Fields<float> f, uint4* __restrict__ dmp, int4* __restrict__ dom_org,
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
    uint4* out = dmp + (size_t)dom * PAIR_CHUNKS * fg.nsp + k;
    if (k >= fg.ns) {
        for (int c = 0; c < PAIR_CHUNKS; c++) out[(size_t)c * fg.nsp] = make_uint4(0u, 0u, 0u, 0u);
        return;
    }
    int lc[4], kk = k;
    for (int mu = 0; mu < 4; mu++) { lc[mu] = kk % fg.ext[mu]; kk /= fg.ext[mu]; }
    const size_t gi = cta_site(fg, dom, lc), V = fg.V;
    float rec[160];
    for (int n = 0; n < 160; n++) rec[n] = 0.f;
    for (int mu = 0; mu < 4; mu++) load_link(f, V, gi, mu, rec + 40 * (mu / 2) + 18 * (mu % 2));
    float cl[72];
    load_clover(f, V, gi, cl);
    for (int n = 0; n < 36; n++) rec[80 + n] = cl[n];
    // half 1: A' = (W x 1) A_low (W x 1)^dag, entrywise A'[3a+c][3b+d] = (a == b ? +1 : -1) A_low[3(1-a)+c][3(1-b)+d]
    {
        const float* b = cl + 36;
        float* o = rec + 120;
        for (int i = 0; i < 6; i++) o[i] = b[(i + 3) % 6];
        for (int i = 1; i < 6; i++)
            for (int j = 0; j < i; j++) {
                const int pi = (i + 3) % 6, pj = (j + 3) % 6;
                const float sg = (i / 3 == j / 3) ? 1.f : -1.f;
                float re, im;
                if (pi > pj) { const int kq = 6 + 2 * (pi * (pi - 1) / 2 + pj); re = b[kq]; im = b[kq + 1]; }
                else { const int kq = 6 + 2 * (pj * (pj - 1) / 2 + pi); re = b[kq]; im = -b[kq + 1]; }
                const int ko = 6 + 2 * (i * (i - 1) / 2 + j);
                o[ko] = sg * re; o[ko + 1] = sg * im;
            }
    }
    for (int c = 0; c < PAIR_CHUNKS; c++) {
        uint4 t;
        __half2* h = reinterpret_cast<__half2*>(&t);
        for (int j = 0; j < 4; j++) h[j] = __floats2half2_rn(rec[8 * c + 2 * j], rec[8 * c + 2 * j + 1]);
        out[(size_t)c * fg.nsp] = t;
    }
}

struct PairSmem {  // offsets in float4 units
    int hbuf, links, clov, rstage, hstage, red, bars;
    size_t bytes;
};
__host__ __device__ inline PairSmem pair_smem(int nsp, int nface, int stage_halo) {
    PairSmem s;
    s.hbuf = 0;
    s.links = 24 * nsp;
    s.clov = s.links + 10 * nsp;
    s.rstage = s.clov + 10 * nsp;
    s.hstage = s.rstage + 6 * nsp;
    s.red = s.hstage + (stage_halo ? 24 * nface : 0);
    s.bars = s.red + 16;
    s.bytes = (size_t)(s.bars + 2) * 16;
    return s;
}

// One K_RAS cycle for all domains of the launch; arguments as ras_cta16_kernel.  rho_dm holds rho_fin in the STORAGE OF
// THE OWNING HALF (chunks 3p..3p+2 of a site = R_up of half p); it is only ever read back by this kernel.
template <bool CHAIN>
__global__ void __launch_bounds__(PAIR_MAX_THREADS, 1)
ras_pair_kernel(FusedGeom fg, int ndl, int colour, int nface, int stage_halo, float mkappa, const uint4* __restrict__ dmp,
                const float4* __restrict__ r_lat, const float4* __restrict__ r_dm, const float4* __restrict__ hb_in,
                float4* __restrict__ hb_out, const float4* phi_in, float4* phi_out, float4* __restrict__ rho_dm,
                const int4* __restrict__ dom_org, const unsigned* __restrict__ dom_bc) {
    if (fg.stop && __ldg(fg.stop)) return;  // the inner solver has converged (launch enqueued ahead of the host's check)
    extern __shared__ float4 smem[];
    const int nsp = fg.nsp;
    const PairSmem lay = pair_smem(nsp, nface, stage_halo);
    float4* hbuf = smem + lay.hbuf;                                          // [8][3][nsp] half-spinor slots
    const uint4* lbuf = reinterpret_cast<const uint4*>(smem + lay.links);    // [10][nsp] staged links (consumed at domain start)
    const uint4* cbuf = reinterpret_cast<const uint4*>(smem + lay.clov);     // [10][nsp] clover blocks of the current domain
    float4* rstage = smem + lay.rstage;                                      // [6][nsp] residual of the current / next domain
    const float4* hstage = smem + lay.hstage;                                // [8][3][nface] halo slots (stage_halo)
    float4* red = smem + lay.red;                                            // [nwarps]
    const unsigned bar_links = cta_smem_u32(smem + lay.bars), bar_clov = bar_links + 8, bar_vec = bar_links + 16;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
    const int p = (lane >> 4) & 1;             // half: 0 = directions x,y + upper chirality, 1 = z,t + lower chirality
    const int k = warp * 16 + (lane & 15);     // site
    const bool active = k < fg.ns;
    const bool src_dm = r_dm != nullptr;
    const bool rot = p == 1;
    const float e_a = p ? -1.f : 1.f;          // sign of slot A's projector in this half's storage (see the file header)
    const float cm = -e_a, cp = e_a;           // c = s * e for the forward (s = -1) and backward (s = +1) hop of slot A
    const float negq = p ? -1.f : 1.f;         // W on receipt (half 1):    out[0..5] = -in[6..11]
    const float negl = p ? 1.f : -1.f;         // W^dag on receipt (half 0): out[6..11] = -in[0..5]

    // ---- domain-independent geometry ----
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
    // own directions: slot j = 0 (A), 1 (B) is direction mu = 2p + j; destination slots of the half spinors this thread sends
    // (dst[2j]: receiver x - mu, its forward hop; dst[2j+1]: receiver x + mu, its backward hop), face indices, and the
    // domain stride / block count of those directions
    unsigned dst[4];
    int fidx[2], nbk[2], dstr[2];
    {
        const unsigned base = cta_smem_u32(hbuf);
        int lstride = 1, dstride = 1;
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            const int e = fg.ext[mu];
            if ((mu >> 1) == p) {
                const int j = mu & 1;
                fidx[j] = (k % lstride) + (k / (lstride * e)) * lstride;
                nbk[j] = fg.nblk[mu];
                dstr[j] = dstride;
                int kd = k - lstride;
                bool ok = active;
                if (lc[mu] == 0) { kd = k + (e - 1) * lstride; ok = ok && fg.wrap[mu]; }
                dst[2 * j] = ok ? base + (unsigned)((2 * mu) * 3 * nsp + kd) * 16u : 0xffffffffu;
                kd = k + lstride;
                ok = active;
                if (lc[mu] + 1 == e) { kd = k - (e - 1) * lstride; ok = ok && fg.wrap[mu]; }
                dst[2 * j + 1] = ok ? base + (unsigned)((2 * mu + 1) * 3 * nsp + kd) * 16u : 0xffffffffu;
            }
            lstride *= e;
            dstride *= fg.nblk[mu];
        }
    }
    const float4* myslots = hbuf + (size_t)(4 * p) * 3 * nsp + k;   // own four slots: 2 mu_A, 2 mu_A + 1, 2 mu_B, 2 mu_B + 1
    if (tid < nsp) {
#pragma unroll
        for (int j = 0; j < 24; j++) hbuf[j * nsp + tid] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    if (tid == 0) {
        mbar_init(bar_links, 1);
        mbar_init(bar_clov, 1);
        mbar_init(bar_vec, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const size_t V = fg.V;
    const unsigned part_bytes = 10u * chunk_bytes;                   // links or clover part of one domain
    const unsigned vec_bytes = (src_dm ? 6u * chunk_bytes : 0u) + (CHAIN && stage_halo ? 24u * (unsigned)nface * 16u : 0u);
    const unsigned l_addr = cta_smem_u32(lbuf), c_addr = cta_smem_u32(cbuf), rs_addr = cta_smem_u32(rstage), hs_addr = cta_smem_u32(hstage);

    auto request_links_vec = [&](int d) {
        if (tid == 0) {
            mbar_expect_tx(bar_links, part_bytes);
            bulk_g2s(l_addr, dmp + (size_t)d * PAIR_CHUNKS * nsp, part_bytes, bar_links);
            if (vec_bytes) {
                mbar_expect_tx(bar_vec, vec_bytes);
                if (src_dm) bulk_g2s(rs_addr, r_dm + (size_t)d * 6 * nsp, 6u * chunk_bytes, bar_vec);
                if (CHAIN && stage_halo) bulk_g2s(hs_addr, hb_in + (size_t)d * 24 * nface, 24u * (unsigned)nface * 16u, bar_vec);
            }
        }
    };
    auto request_clover = [&](int d) {
        if (tid == 0) {
            mbar_expect_tx(bar_clov, part_bytes);
            bulk_g2s(c_addr, dmp + ((size_t)d * PAIR_CHUNKS + 10) * nsp, part_bytes, bar_clov);
        }
    };
    auto site_of = [&](const int4& org) -> size_t {
        int x0 = org.x + lc[0], x1 = org.y + lc[1], x2 = org.z + lc[2], x3 = org.w + lc[3];
        if (x0 >= fg.L[0]) x0 -= fg.L[0];
        if (x1 >= fg.L[1]) x1 -= fg.L[1];
        if (x2 >= fg.L[2]) x2 -= fg.L[2];
        if (x3 >= fg.L[3]) x3 -= fg.L[3];
        return x0 + fg.L[0] * (x1 + fg.L[1] * (x2 + (size_t)fg.L[2] * x3));
    };
    auto request_r_lat = [&](const int4& org) {  // the own chirality of the own site, own column, LDGSTS
        if (active) {
            const size_t gn = site_of(org);
#pragma unroll
            for (int c = 0; c < 3; c++) cp_async16(rstage + (3 * p + c) * nsp + k, r_lat + (size_t)(3 * p + c) * V + gn);
        }
        cp_async_commit();
    };

    int4 org = make_int4(0, 0, 0, 0);
    if ((int)blockIdx.x < ndl) {
        const int dom0 = launch_dom(fg, blockIdx.x, colour);
        org = dom_org[dom0];
        request_links_vec(dom0);
        request_clover(dom0);
        if (!src_dm) request_r_lat(org);
    }

    float U[36];  // -kappa U_A, -kappa U_B
    for (int jd = 0;; jd++) {
        const int h = blockIdx.x + jd * gridDim.x;
        if (h >= ndl) break;
        const unsigned par = (unsigned)jd & 1u;
        const bool has_next = h + (int)gridDim.x < ndl;
        const int dom = launch_dom(fg, h, colour);
        const int nxt = launch_dom(fg, has_next ? h + gridDim.x : h, colour);
        const int4 org_nxt = __ldg(dom_org + nxt);
        const size_t gi = site_of(org);

        // ---- operands: the own two links into registers, scaled by -kappa ----
        mbar_wait(bar_links, par);
        {
            float f[40];
#pragma unroll
            for (int c = 0; c < 5; c++) half8_to_float(lbuf[(5 * p + c) * nsp + k], f + 8 * c);
#pragma unroll
            for (int n = 0; n < 36; n++) U[n] = mkappa * f[n];
        }
        // ---- projection P_Omega' r: the own chirality in the own storage ----
        float R[24], v[12];
        if (src_dm) {
            if (vec_bytes) mbar_wait(bar_vec, par);
        } else {
            cp_async_wait();
            if (CHAIN && vec_bytes) mbar_wait(bar_vec, par);
        }
        {
            float t[12];
#pragma unroll
            for (int c = 0; c < 3; c++) {
                float4 q4 = rstage[(3 * p + c) * nsp + k];
                if (!active) q4 = make_float4(0.f, 0.f, 0.f, 0.f);
                t[4 * c] = q4.x; t[4 * c + 1] = q4.y; t[4 * c + 2] = q4.z; t[4 * c + 3] = q4.w;
            }
            // a lattice-layout source holds psi: half 1 rotates its chirality with W; rho_fin is already in the own storage
            if (src_dm) {
#pragma unroll
                for (int j = 0; j < 12; j++) R[j] = t[j];
            } else {
                rotate_recv<false>(t, R, rot, negq);
            }
        }
        if (!src_dm && has_next) request_r_lat(org_nxt);
        if (CHAIN) {
            // ---- boundary coupling (reading A3): rho -= the hops of v_{j-1} that cross the domain boundary, own two
            // directions; the part that lands in the partner's chirality is handed over ----
            const float4* hin = stage_halo ? hstage : hb_in + (size_t)dom * 24 * nface;
            float acc[24], g[12], hh[12];
#pragma unroll
            for (int n = 0; n < 24; n++) acc[n] = 0.f;
#define WC_PAIR_LOAD(SL, J)                                                                       \
    {                                                                                             \
        const bool rcv = active && dst[(SL) ^ 1] == 0xffffffffu;                                  \
        const float4* q4 = hin + (size_t)(4 * p + (SL)) * 3 * nface + fidx[J];                    \
        _Pragma("unroll") for (int jj = 0; jj < 3; jj++) {                                        \
            float4 t = make_float4(0.f, 0.f, 0.f, 0.f);                                           \
            if (rcv) t = q4[(size_t)jj * nface];                                                  \
            hh[4 * jj] = t.x; hh[4 * jj + 1] = t.y; hh[4 * jj + 2] = t.z; hh[4 * jj + 3] = t.w;   \
        }                                                                                         \
    }
            if (__any_sync(0xffffffffu, active && dst[1] == 0xffffffffu)) {  // upper face of slot A: forward hop from outside
                WC_PAIR_LOAD(0, 0)
                su3_mul<float>(U, hh, g);
                reconstruct_a(g, acc, cm, -1.f);
            }
            if (__any_sync(0xffffffffu, active && dst[0] == 0xffffffffu)) {  // lower face of slot A: backward hop from outside
                WC_PAIR_LOAD(1, 0)
                reconstruct_a(hh, acc, cp, -1.f);
            }
            if (__any_sync(0xffffffffu, active && dst[3] == 0xffffffffu)) {
                WC_PAIR_LOAD(2, 1)
                su3_mul<float>(U + 18, hh, g);
                reconstruct_sub<float, 1, -1>(g, acc);
            }
            if (__any_sync(0xffffffffu, active && dst[2] == 0xffffffffu)) {
                WC_PAIR_LOAD(3, 1)
                reconstruct_sub<float, 1, +1>(hh, acc);
            }
#undef WC_PAIR_LOAD
            float recv[12], rr[12];
            exchange12(acc + 12, recv);
            rotate_recv<false>(recv, rr, rot, negq);
#pragma unroll
            for (int j = 0; j < 12; j++) R[j] += acc[j] + rr[j];
        }
#pragma unroll
        for (int n = 0; n < 12; n++) v[n] = 0.f;

        for (int it = 0; it < fg.niter; it++) {
            // ---- the partner's chirality of rho, rotated into the own storage ----
            {
                float recv[12];
                exchange12(R, recv);
                rotate_recv<true>(recv, R + 12, !rot, negl);
            }
            {
                float hs[12], g[12];
                project_a(R, hs, cm);
                st_half_pred(dst[0], chunk_bytes, hs);
                project_a(R, hs, cp);
                su3_adj_mul<float>(U, hs, g);
                st_half_pred(dst[1], chunk_bytes, g);
                project<float, 1, -1>(R, hs);
                st_half_pred(dst[2], chunk_bytes, hs);
                project<float, 1, +1>(R, hs);
                su3_adj_mul<float>(U + 18, hs, g);
                st_half_pred(dst[3], chunk_bytes, g);
            }
            float qa[24];  // [0..11] q of the own chirality, [12..23] the hop contributions to the partner's
            if (it == 0) mbar_wait(bar_clov, par);
            {
                float Ab[40];
#pragma unroll
                for (int c = 0; c < 5; c++) half8_to_float(cbuf[(5 * p + c) * nsp + k], Ab + 8 * c);
                herm6_mul<float>(Ab, R, qa);
            }
#pragma unroll
            for (int n = 12; n < 24; n++) qa[n] = 0.f;
            __syncthreads();
            // every thread is past its staging reads of this domain: thread 0 requests the next domain's data
            if (has_next) {
                if (it == 0) request_links_vec(nxt);
                if (it + 1 == fg.niter) request_clover(nxt);
            }
            {
                float hs[12], g[12];
                ld_half_cta(myslots, nsp, hs);
                su3_mul<float>(U, hs, g);
                reconstruct_a(g, qa, cm, 1.f);
                ld_half_cta(myslots + 3 * nsp, nsp, g);
                reconstruct_a(g, qa, cp, 1.f);
                ld_half_cta(myslots + 6 * nsp, nsp, hs);
                su3_mul<float>(U + 18, hs, g);
                reconstruct_add<float, 1, -1>(g, qa);
                ld_half_cta(myslots + 9 * nsp, nsp, g);
                reconstruct_add<float, 1, +1>(g, qa);
            }
            {
                float recv[12], rr[12];
                exchange12(qa + 12, recv);
                rotate_recv<false>(recv, rr, rot, negq);
#pragma unroll
                for (int j = 0; j < 12; j++) qa[j] += rr[j];
            }
            float d0 = 0.f, d1 = 0.f, d2 = 0.f;
#pragma unroll
            for (int n = 0; n < 6; n++) {
                const float qr = qa[2 * n], qi = qa[2 * n + 1], rr = R[2 * n], ri = R[2 * n + 1];
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
                const float4 pp = red[n];
                s0 += pp.x; s1 += pp.y; s2 += pp.z;
            }
            // alpha = <q,rho>/<q,q>, 0 if <q,q> = 0 (Q9); v += alpha rho; rho -= alpha q  (own chirality)
            const float inv = s2 > 0.f ? 1.f / s2 : 0.f;
            const float ar = s0 * inv, ai = s1 * inv;
            const bool upd_rho = it + 1 < fg.niter || rho_dm != nullptr;
#pragma unroll
            for (int n = 0; n < 6; n++) {
                const float rr = R[2 * n], ri = R[2 * n + 1];
                v[2 * n] = fmaf(ar, rr, v[2 * n]); v[2 * n] = fmaf(-ai, ri, v[2 * n]);
                v[2 * n + 1] = fmaf(ar, ri, v[2 * n + 1]); v[2 * n + 1] = fmaf(ai, rr, v[2 * n + 1]);
                if (upd_rho) {
                    R[2 * n] = fmaf(-ar, qa[2 * n], rr); R[2 * n] = fmaf(ai, qa[2 * n + 1], R[2 * n]);
                    R[2 * n + 1] = fmaf(-ar, qa[2 * n + 1], ri); R[2 * n + 1] = fmaf(-ai, qa[2 * n], R[2 * n + 1]);
                }
            }
        }
        // ---- halo scatter for the next cycle: the hops of v that leave the domain through the own two directions ----
        if (hb_out) {
            float vf[24], hs[12], g[12];
#pragma unroll
            for (int j = 0; j < 12; j++) vf[j] = v[j];
            {
                float recv[12];
                exchange12(v, recv);
                rotate_recv<true>(recv, vf + 12, !rot, negl);
            }
            const unsigned pk = __ldg(dom_bc + dom);
#define WC_PAIR_HALO(J, PROJ_LO, PROJ_HI)                                                                        \
    {                                                                                                            \
        const int mu = 2 * p + J, nb = nbk[J], bc = (int)((pk >> (8 * mu)) & 255u);                              \
        if (active && dst[2 * J] == 0xffffffffu) { /* lower face -> slot 2mu of the domain at -mu */             \
            const int nbd = bc == 0 ? dom + (nb - 1) * dstr[J] : dom - dstr[J];                                  \
            float4* o = hb_out + ((size_t)nbd * 8 + 2 * mu) * 3 * nface + fidx[J];                               \
            PROJ_LO;                                                                                             \
            for (int jj = 0; jj < 3; jj++) o[(size_t)jj * nface] = make_float4(hs[4 * jj], hs[4 * jj + 1], hs[4 * jj + 2], hs[4 * jj + 3]); \
        }                                                                                                        \
        if (active && dst[2 * J + 1] == 0xffffffffu) { /* upper face -> slot 2mu+1 of the domain at +mu */       \
            const int nbd = bc + 1 == nb ? dom - (nb - 1) * dstr[J] : dom + dstr[J];                             \
            float4* o = hb_out + ((size_t)nbd * 8 + 2 * mu + 1) * 3 * nface + fidx[J];                           \
            PROJ_HI;                                                                                             \
            su3_adj_mul<float>(U + 18 * J, hs, g);                                                               \
            for (int jj = 0; jj < 3; jj++) o[(size_t)jj * nface] = make_float4(g[4 * jj], g[4 * jj + 1], g[4 * jj + 2], g[4 * jj + 3]); \
        }                                                                                                        \
    }
            WC_PAIR_HALO(0, project_a(vf, hs, cm), project_a(vf, hs, cp))
            WC_PAIR_HALO(1, (project<float, 1, -1>(vf, hs)), (project<float, 1, +1>(vf, hs)))
#undef WC_PAIR_HALO
        }
        // ---- rho_fin: the own chirality in the own storage, domain-major ----
        if (rho_dm && active) {
            float4* o = rho_dm + ((size_t)dom * 6 + 3 * p) * nsp + k;
#pragma unroll
            for (int c = 0; c < 3; c++) o[(size_t)c * nsp] = make_float4(R[4 * c], R[4 * c + 1], R[4 * c + 2], R[4 * c + 3]);
        }
        // ---- restriction R_Omega (bulk sites only): the own chirality back in the spin basis of the lattice vectors ----
        if (bulk) {
            float w[12];
            // half 0: psi_up = v; half 1: psi_low = W^dag v: out[0..5] = v[6..11], out[6..11] = -v[0..5]
#pragma unroll
            for (int j = 0; j < 12; j++) {
                const float t = rot ? v[(j + 6) % 12] : v[j];
                w[j] = (j >= 6 && rot) ? -t : t;
            }
            float4* o = phi_out + (size_t)(3 * p) * V + gi;
            if (phi_in) {
                // phi += v as a fire-and-forget vector reduction (phi_in == phi_out; one writer per site and component)
#pragma unroll
                for (int c = 0; c < 3; c++)
                    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(o + (size_t)c * V), "f"(w[4 * c]), "f"(w[4 * c + 1]),
                                 "f"(w[4 * c + 2]), "f"(w[4 * c + 3])
                                 : "memory");
            } else {
#pragma unroll
                for (int c = 0; c < 3; c++) o[(size_t)c * V] = make_float4(w[4 * c], w[4 * c + 1], w[4 * c + 2], w[4 * c + 3]);
            }
        }
        org = org_nxt;
    }
}

// ---- host side ----
typedef void (*pair_kernel_t)(FusedGeom, int, int, int, int, float, const uint4*, const float4*, const float4*, const float4*, float4*,
                              const float4*, float4*, float4*, const int4*, const unsigned*);
static pair_kernel_t pair_kernel(bool chain) { return chain ? ras_pair_kernel<true> : ras_pair_kernel<false>; }

int ensure_halo(wcras_ctx* ctx, int nrhs);  // ras_cta.cu

// Build the pair operand records and the domain-major rho_fin buffer (ctx->dm16 / ctx->rf_dm, shared with ras_cta16.cu:
// only one of the two kernels is configured at a time); returns 1 if this kernel can run the configuration.
int ras_pair_prepare(wcras_ctx* ctx, const FusedGeom& fg, int nd, const Fields<float>& f) {
    if (fg.C != 1 || fg.nsp > FUSED_CTA_MAX_THREADS) return 0;
    for (int mu = 0; mu < 4; mu++) if (fg.nblk[mu] > 255) return 0;
    int nface = 1;
    for (int mu = 0; mu < 4; mu++) nface = fg.ns / fg.ext[mu] > nface ? fg.ns / fg.ext[mu] : nface;
    nface = (nface + 7) / 8 * 8;
    int dev = 0, sms = 0, smem_max = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    int stage_halo = 1;
    if (pair_smem(fg.nsp, nface, 1).bytes > (size_t)smem_max) stage_halo = 0;
    const size_t smem = pair_smem(fg.nsp, nface, stage_halo).bytes;
    if (smem > (size_t)smem_max) return 0;
    if (cudaFuncSetAttribute(ras_pair_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
        cudaFuncSetAttribute(ras_pair_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ras_pair_kernel<true>, 2 * fg.nsp, smem) != cudaSuccess || per_sm < 1) {
        cudaGetLastError();
        return 0;
    }
    if (ctx->dm16) { cudaStreamSynchronize(ctx->stream); cudaFree(ctx->dm16); ctx->dm16 = nullptr; }
    if (ctx->rf_dm) { cudaStreamSynchronize(ctx->stream); cudaFree(ctx->rf_dm); ctx->rf_dm = nullptr; }
    const size_t rf_bytes = sizeof(float4) * 6 * (size_t)fg.nsp * nd;
    if (cudaMalloc((void**)&ctx->dm16, sizeof(uint4) * PAIR_CHUNKS * (size_t)fg.nsp * nd) != cudaSuccess) { cudaGetLastError(); ctx->dm16 = nullptr; return 0; }
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
    pack_pair_kernel<<<nd, fg.nsp, 0, ctx->stream>>>(fg, nd, f, ctx->dm16, ctx->dom_org, ctx->dom_bc);
    ctx->launches++;
    if (cudaGetLastError() != cudaSuccess) return 0;
    const long want = (long)per_sm * sms;
    ctx->cta_grid = (int)(nd < want ? nd : want);
    return 1;
}

#define WC_PAIR_LAUNCH(CHAINV, GRID, ...)                                                                                   \
    pair_kernel(CHAINV)<<<(GRID), 2 * fg.nsp, ctx->cta16_smem, ctx->stream>>>(fg, __VA_ARGS__, ctx->dom_org, ctx->dom_bc)

int ras_pair_block_solve(wcras_ctx* ctx, const float4* r, float4* vout, bool accum) {
    const FusedGeom& fg = ctx->fused;
    WC_PAIR_LAUNCH(false, ctx->cta_grid, ctx->ras.nd, -1, ctx->nface, ctx->stage_halo, -(float)ctx->kappa, ctx->dm16, r, nullptr, nullptr, nullptr,
                   accum ? vout : nullptr, vout, nullptr);
    ctx->launches++;
    WC_CHECK_LAUNCH();
    return WCRAS_OK;
}

// v = K_RAS r with NRAS chained cycles (overlap 0), as ras_cta16_apply_chained
int ras_pair_apply_chained(wcras_ctx* ctx, const float4* r, float4* v) {
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
            WC_PAIR_LAUNCH(false, ctx->cta_grid, nd, -1, nface, ctx->stage_halo, mk, ctx->dm16, r, nullptr, nullptr, last ? nullptr : hb[0], nullptr, v,
                           last ? nullptr : rf);
        else
            WC_PAIR_LAUNCH(true, ctx->cta_grid, nd, -1, nface, ctx->stage_halo, mk, ctx->dm16, nullptr, rf, hb[(j - 1) & 1], last ? nullptr : hb[j & 1], v,
                           v, last ? nullptr : rf);
        ctx->launches++;
    }
    WC_CHECK_LAUNCH();
    return WCRAS_OK;
}

// v = K_SAP r (multiplicative Schwarz, see ras_cta_apply_sap): red-black half steps, one launch per colour
int ras_pair_apply_sap(wcras_ctx* ctx, const float4* r, float4* v) {
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
            WC_PAIR_LAUNCH(false, grid, ndl, colour, nface, ctx->stage_halo, mk, ctx->dm16, r_lat, r_dm, nullptr, halo_out, nullptr, v, rho_out);
        else
            WC_PAIR_LAUNCH(true, grid, ndl, colour, nface, ctx->stage_halo, mk, ctx->dm16, r_lat, r_dm, hb, halo_out, first_visit ? nullptr : v, v,
                           rho_out);
        ctx->launches++;
    }
    WC_CHECK_LAUNCH();
    return WCRAS_OK;
}

}  // namespace wc
