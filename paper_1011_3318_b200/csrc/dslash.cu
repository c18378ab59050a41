// dslash.cu -- step A1: full-lattice clover Dslash w = D v (north_star (b)), fp32 and fp64,
// plus the box-restricted operator on full-lattice vectors used by wcras_apply_D_restricted.
//
// One thread per site, consecutive threads = consecutive x (coalesced 16-byte loads from the SoA fields).
// HBM-bound: algorithmic traffic per site (fp32) = 4 links 288 B + clover 288 B + spinor in 96 B + out 96 B
// = 768 B (fp64: 1536 B); neighbour spinors and backward links are re-reads that L1/L2 must serve.
#include "wcras_internal.cuh"

namespace wc {

template <typename T, int MU, bool MASKED>
__device__ __forceinline__ void hop_pair(const Fields<T>& f, size_t V, const Geom& g, const int x[4], int i, int stride_mu,
                                         const typename VecOf<T>::type* __restrict__ in, bool keep_f, bool keep_b, T* hop) {
    const int L = g.L[MU];
    const int jf = x[MU] + 1 == L ? i - (L - 1) * stride_mu : i + stride_mu;
    const int jb = x[MU] == 0 ? i + (L - 1) * stride_mu : i - stride_mu;
    T u[18], sn[24];
    if (!MASKED || keep_f) {
        load_link(f, V, i, MU, u);
        load_spinor(in, V, jf, sn);
        hop_fwd<T, MU>(u, sn, hop);
    }
    if (!MASKED || keep_b) {
        load_link(f, V, jb, MU, u);
        load_spinor(in, V, jb, sn);
        hop_bwd<T, MU>(u, sn, hop);
    }
}

template <typename T, bool XPAY, int TH, int MINB>
__global__ void __launch_bounds__(TH, MINB) dslash_kernel(Geom g, Fields<T> f, T kappa, const typename VecOf<T>::type* __restrict__ in,
                                                     typename VecOf<T>::type* __restrict__ out,
                                                     const typename VecOf<T>::type* bsrc) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.V) return;
    const size_t V = g.V;
    int x[4];
    site_coords(g, i, x);
    T hop[24];
#pragma unroll
    for (int k = 0; k < 24; k++) hop[k] = 0;
    hop_pair<T, 0, false>(f, V, g, x, i, 1, in, true, true, hop);
    hop_pair<T, 1, false>(f, V, g, x, i, g.L[0], in, true, true, hop);
    hop_pair<T, 2, false>(f, V, g, x, i, g.L[0] * g.L[1], in, true, true, hop);
    hop_pair<T, 3, false>(f, V, g, x, i, g.L[0] * g.L[1] * g.L[2], in, true, true, hop);
    T s[24], acc[24];
    {
        T cl[72];
        load_spinor(in, V, i, s);
        load_clover(f, V, i, cl);
        clover_apply<T>(cl, s, acc);
    }
    if (XPAY) {
        load_spinor(bsrc, V, i, s);
#pragma unroll
        for (int k = 0; k < 24; k++) acc[k] = s[k] - (acc[k] - kappa * hop[k]);
    } else {
#pragma unroll
        for (int k = 0; k < 24; k++) acc[k] -= kappa * hop[k];
    }
    store_spinor(out, V, i, acc);
}

struct Box {
    int start[4], ext[4], blk[4];
    int all;  // 1: every site belongs to the block of shape blk that contains it (overlap 0)
};

__device__ __forceinline__ bool in_box(const Geom& g, const Box& b, const int y[4]) {
    bool ok = true;
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        int c = y[mu] - b.start[mu];
        if (c < 0) c += g.L[mu];
        ok = ok && (c < b.ext[mu]);
    }
    return ok;
}

// out = P'^T D_Omega' P' in on full-lattice vectors (checking / ABI path, not performance critical)
template <typename T>
__global__ void __launch_bounds__(128) dslash_box_kernel(Geom g, Fields<T> f, T kappa, Box box,
                                                         const typename VecOf<T>::type* __restrict__ in,
                                                         typename VecOf<T>::type* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.V) return;
    const size_t V = g.V;
    int x[4];
    site_coords(g, i, x);
    Box b = box;
    if (box.all) {
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            b.start[mu] = (x[mu] / box.blk[mu]) * box.blk[mu];
            b.ext[mu] = box.blk[mu];
        }
    }
    T acc[24];
    if (!in_box(g, b, x)) {
#pragma unroll
        for (int k = 0; k < 24; k++) acc[k] = 0;
        store_spinor(out, V, i, acc);
        return;
    }
    bool kf[4], kb[4];
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        int y[4] = {x[0], x[1], x[2], x[3]};
        y[mu] = x[mu] + 1 == g.L[mu] ? 0 : x[mu] + 1;
        kf[mu] = in_box(g, b, y);
        y[mu] = x[mu] == 0 ? g.L[mu] - 1 : x[mu] - 1;
        kb[mu] = in_box(g, b, y);
    }
    T hop[24];
#pragma unroll
    for (int k = 0; k < 24; k++) hop[k] = 0;
    hop_pair<T, 0, true>(f, V, g, x, i, 1, in, kf[0], kb[0], hop);
    hop_pair<T, 1, true>(f, V, g, x, i, g.L[0], in, kf[1], kb[1], hop);
    hop_pair<T, 2, true>(f, V, g, x, i, g.L[0] * g.L[1], in, kf[2], kb[2], hop);
    hop_pair<T, 3, true>(f, V, g, x, i, g.L[0] * g.L[1] * g.L[2], in, kf[3], kb[3], hop);
    T s[24], cl[72];
    load_spinor(in, V, i, s);
    load_clover(f, V, i, cl);
    clover_apply<T>(cl, s, acc);
#pragma unroll
    for (int k = 0; k < 24; k++) acc[k] -= kappa * hop[k];
    store_spinor(out, V, i, acc);
}

template <typename T>
int dslash(wcras_ctx* ctx, const typename VecOf<T>::type* in, typename VecOf<T>::type* out,
           const typename VecOf<T>::type* b_minus) {
    TimedRegion tr(ctx, sizeof(T) == 4 ? TC_DSLASH : TC_DSLASH64);
    const int V = ctx->geom.V;
    // 64-thread CTAs with the full register budget (165 registers fp32, 252 fp64): the compiler then keeps all
    // loads of a site in flight at once, which is what an HBM latency-bound stencil needs -- measured on B200 at
    // 32^4: 130 us (fp32) / 292 us (fp64) against 147 / 330 us at 96 / 186 registers with 128-thread CTAs.
    constexpr int TH = 64;
    const unsigned grid = (V + TH - 1) / TH;
    if (b_minus)
        dslash_kernel<T, true, TH, 1><<<grid, TH, 0, ctx->stream>>>(ctx->geom, ctx->fields<T>(), (T)ctx->kappa, in, out, b_minus);
    else
        dslash_kernel<T, false, TH, 1><<<grid, TH, 0, ctx->stream>>>(ctx->geom, ctx->fields<T>(), (T)ctx->kappa, in, out, nullptr);
    ctx->launches++;
    if (sizeof(T) == 4) ctx->dv32++; else ctx->dv64++;
    WC_CHECK_LAUNCH();
    return WCRAS_OK;
}

template <typename T>
int dslash_box(wcras_ctx* ctx, const int start[4], const int ext[4], bool all_blocks,
               const typename VecOf<T>::type* in, typename VecOf<T>::type* out) {
    Box b;
    for (int mu = 0; mu < 4; mu++) {
        b.start[mu] = start ? start[mu] : 0;
        b.ext[mu] = ext ? ext[mu] : ctx->geom.L[mu];
        b.blk[mu] = ctx->ras.b[mu];
    }
    b.all = all_blocks ? 1 : 0;
    const int V = ctx->geom.V, TH = 128;
    dslash_box_kernel<T><<<(V + TH - 1) / TH, TH, 0, ctx->stream>>>(ctx->geom, ctx->fields<T>(), (T)ctx->kappa, b, in, out);
    ctx->launches++;
    WC_CHECK_LAUNCH();
    return WCRAS_OK;
}

template int dslash<float>(wcras_ctx*, const float4*, float4*, const float4*);
template int dslash<double>(wcras_ctx*, const double2*, double2*, const double2*);
template int dslash_box<float>(wcras_ctx*, const int*, const int*, bool, const float4*, float4*);
template int dslash_box<double>(wcras_ctx*, const int*, const int*, bool, const double2*, double2*);

}  // namespace wc
