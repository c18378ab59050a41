// dslash.cu -- step A1: full-lattice clover Dslash w = D v (north_star (b)), fp32 and fp64,
// plus the box-restricted operator on full-lattice vectors used by wcras_apply_D_restricted.
//
// One thread per site, consecutive threads = consecutive x (coalesced 16-byte loads from the SoA fields).
// HBM-bound: algorithmic traffic per site (fp32) = 4 links 288 B + clover 288 B + spinor in 96 B + out 96 B
// = 768 B (fp64: 1536 B); neighbour spinors and backward links are re-reads that L1/L2 must serve.
#include "blas.cuh"

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

// Dots fused into the Dslash (north_star (d)): every CTA reduces its 3 sums (warp shuffle -> shared memory) and
// stores one partial, with no fence or atomic on the way (a __threadfence per 64-thread CTA would wait for the
// CTA's output stores and cost ~15 % of the kernel).  dot_finish_kernel, 16 CTAs launched right behind it, sums
// the partials in a fixed order and finishes the scalar recurrence: deterministic.
template <int TH>
__device__ __forceinline__ void dslash_block_partial(double (&v)[3], double* __restrict__ part, unsigned pstride, unsigned poff) {
    constexpr int NW = TH / 32;
    __shared__ double sm[3][NW];
    const int tid = threadIdx.y * blockDim.x + threadIdx.x, lane = tid & 31, w = tid >> 5;
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const double t = warp_sum(v[k]);
        if (lane == 0) sm[k][w] = t;
    }
    __syncthreads();
    if (tid < 3) {
        double t = 0;
        for (int j = 0; j < NW; j++) t += sm[tid][j];
        part[(size_t)tid * pstride + poff + blockIdx.x] = t;  // [3][pstride]: coalesced for the finish kernel
    }
}

// what the totals of the fused dots mean for the solver's scalars (one thread)
template <int DOT>
__device__ __forceinline__ void dot_finish_scalars(const double (&tot)[3], Scalars* sc) {
    if (DOT == 3) {
        sc->nrm = tot[2];
    } else if (DOT == 1) {
        sc->rtv[0] = tot[0]; sc->rtv[1] = tot[1];
        const cd a = cdiv({sc->rho[0], sc->rho[1]}, {tot[0], tot[1]});
        sc->alpha[0] = a.r; sc->alpha[1] = a.i;
    } else {
        sc->ts[0] = tot[0]; sc->ts[1] = tot[1]; sc->tt = tot[2];
        sc->omega[0] = tot[2] > 0 ? tot[0] / tot[2] : 0.0;
        sc->omega[1] = tot[2] > 0 ? tot[1] / tot[2] : 0.0;
    }
}

// Small lattices (at most FIN_INLINE_MAX partials; one right-hand side): the Dslash finishes its dots itself -- the last
// CTA to arrive (fence + atomic ticket) sums the partials of all CTAs in a fixed order and applies dot_finish_scalars.
// One kernel node less per Dslash where a solve is bound by the latency of its dependent launches (reading A1);
// at 32^4 the fence per 64-thread CTA costs ~15 % of the kernel, so large lattices keep the separate finish kernel.
constexpr unsigned FIN_INLINE_MAX = 512;  // measured: -16..18 % per solve at 4^4 and 8^4 (64 CTAs), no gain at 16^4 (1024 CTAs)
template <int TH, int DOT>
__device__ __forceinline__ void dslash_finish_inline(const double* part, unsigned nblk, unsigned* ticket, Scalars* sc) {
    constexpr int NW = TH / 32;
    __shared__ bool last_s;
    __shared__ double fs[3][NW];
    const int tid = threadIdx.y * blockDim.x + threadIdx.x, lane = tid & 31, w = tid >> 5;
    __syncthreads();  // the partial of this CTA has been written (threads 0..2)
    if (tid == 0) {
        __threadfence();
        last_s = atomicInc(ticket, nblk - 1) == nblk - 1;  // wraps back to 0: ready for the next launch
    }
    __syncthreads();
    if (!last_s) return;
    __threadfence();
    double t[3] = {0, 0, 0};
    for (unsigned j = tid; j < nblk; j += TH)
#pragma unroll
        for (int k = 0; k < 3; k++) t[k] += __ldcg(&part[(size_t)k * nblk + j]);
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const double u = warp_sum(t[k]);
        if (lane == 0) fs[k][w] = u;
    }
    __syncthreads();
    if (tid == 0) {
        double tot[3] = {0, 0, 0};
        for (int j = 0; j < NW; j++)
#pragma unroll
            for (int k = 0; k < 3; k++) tot[k] += fs[k][j];
        dot_finish_scalars<DOT>(tot, sc);
    }
}

// FIN_CTAS CTAs each sum a contiguous slice of the partials in a fixed order; the last one to finish (atomic ticket)
// sums the FIN_CTAS slice sums in a fixed order and finishes the scalar recurrence.
constexpr int FIN_CTAS = 16;
template <int DOT>
__global__ void __launch_bounds__(512) dot_finish_kernel(const double* __restrict__ part, unsigned nblk, double* __restrict__ slice,
                                                         unsigned* ticket, Scalars* sc, const int* stop) {
    if (stop && __ldg(stop)) return;
    __shared__ double sm[3][16];
    __shared__ bool last;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const unsigned per = (nblk + FIN_CTAS - 1) / FIN_CTAS, lo = blockIdx.x * per, hi = min(nblk, lo + per);
    double t[3] = {0, 0, 0};
    for (unsigned j = lo + threadIdx.x; j < hi; j += 512)
#pragma unroll
        for (int k = 0; k < 3; k++) t[k] += part[(size_t)k * nblk + j];
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const double u = warp_sum(t[k]);
        if (lane == 0) sm[k][w] = u;
    }
    __syncthreads();
    if (w == 0) {
#pragma unroll
        for (int k = 0; k < 3; k++) {
            const double u = warp_sum(lane < 16 ? sm[k][lane] : 0.0);
            if (lane == 0) slice[blockIdx.x * 3 + k] = u;
        }
        if (lane == 0) {
            __threadfence();
            last = atomicInc(ticket, FIN_CTAS - 1) == FIN_CTAS - 1;
        }
    }
    __syncthreads();
    if (!last || threadIdx.x != 0) return;
    __threadfence();
    double tot[3] = {0, 0, 0};
    for (int j = 0; j < FIN_CTAS; j++)
#pragma unroll
        for (int k = 0; k < 3; k++) tot[k] += __ldcg(&slice[j * 3 + k]);
    dot_finish_scalars<DOT>(tot, sc);
}

// DOT = 0: out = D in (XPAY: out = bsrc - D in).
// DOT = 1: also rtv = <dotv, out> and alpha = rho / rtv          (BiCGStab: v = D ph, dotv = rt)
// DOT = 2: also ts = <out, dotv>, tt = <out, out>, omega = ts/tt (BiCGStab: t = D sh, dotv = s)
// DOT = 3: also nrm = <out, out>                                  (true residual: out = eta - D phi)
// FIN: the kernel finishes its dots itself (dslash_finish_inline; fticket, sc), no dot_finish_kernel behind it.
template <typename T, bool XPAY, int TH, int MINB, int DOT, bool FIN = false>
__global__ void __launch_bounds__(TH, MINB) dslash_kernel(Geom g, Fields<T> f, T kappa, const typename VecOf<T>::type* __restrict__ in,
                                                     typename VecOf<T>::type* out,  // may be bsrc (r = r - D v in place)
                                                     const typename VecOf<T>::type* bsrc,
                                                     const typename VecOf<T>::type* __restrict__ dotv, double* part,
                                                     unsigned pstride, unsigned poff, size_t rstride, int ztile,
                                                     unsigned* fticket = nullptr, Scalars* fsc = nullptr) {
    // blockDim = (sites, right-hand sides): the threads threadIdx.y = 0..nrhs-1 of a site work on the vectors of a
    // stack rstride apart and load the same links and clover term, which L1 serves after the first warp has
    // fetched them (576/nrhs + 192 bytes of DRAM traffic per site and right-hand side)
    // the inner solver has converged: this launch was enqueued ahead of the host's check.  Read-only path (L1 per SM):
    // a plain load by every warp of the grid would serialise on one L2 sector
    if (g.stop && __ldg(g.stop)) return;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (ztile > 0 && i < g.V) {
        // Large lattices: visit the sites in the order (x, y, z within a tile of ztile planes, t, z tile) instead of
        // (x, y, z, t), so that the operands of the slabs t-1, t, t+1 of one z tile (a few MB each) are still in L2 when
        // the t-neighbours are read; a whole t-slice (85 MB at 48^3) is not.  Only the traversal changes, not a layout.
        const int plane = g.L[0] * g.L[1], slab = plane * ztile, per_tile = slab * g.L[3];
        const int zt = i / per_tile, r = i - zt * per_tile, t = r / slab, r2 = r - t * slab, zi = r2 / plane, xy = r2 - zi * plane;
        i = xy + plane * (zt * ztile + zi + g.L[2] * t);
    }
    {
        const size_t ro = threadIdx.y * rstride;
        in += ro; out += ro;
        if (XPAY) bsrc += ro;
        if (DOT == 1 || DOT == 2) dotv += ro;
    }
    const bool valid = i < g.V;
    if (!DOT && !valid) return;
    double dsum[3] = {0, 0, 0};
    if (valid) {
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
        if (DOT == 3) {
            T d2 = 0;
#pragma unroll
            for (int k = 0; k < 24; k++) d2 = wc_fma(acc[k], acc[k], d2);
            dsum[2] = d2;
        } else if (DOT) {
            load_spinor(dotv, V, i, s);
            T d0 = 0, d1 = 0, d2 = 0;  // per-site sums in T, accumulated over sites in fp64
#pragma unroll
            for (int n = 0; n < 12; n++) {
                const T ar = DOT == 1 ? s[2 * n] : acc[2 * n], ai = DOT == 1 ? s[2 * n + 1] : acc[2 * n + 1];
                const T br = DOT == 1 ? acc[2 * n] : s[2 * n], bi = DOT == 1 ? acc[2 * n + 1] : s[2 * n + 1];
                d0 = wc_fma(ar, br, d0); d0 = wc_fma(ai, bi, d0);   // Re conj(a) b
                d1 = wc_fma(ar, bi, d1); d1 = wc_fma(-ai, br, d1);  // Im conj(a) b
                d2 = wc_fma(acc[2 * n], acc[2 * n], d2); d2 = wc_fma(acc[2 * n + 1], acc[2 * n + 1], d2);
            }
            dsum[0] = d0; dsum[1] = d1; dsum[2] = d2;
        }
    }
    if (DOT) dslash_block_partial<TH>(dsum, part, pstride, poff);
    if (DOT && FIN) dslash_finish_inline<TH, DOT>(part, pstride, fticket, fsc);
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

// in / out / b_minus / dotv are stacks of ctx->nrhs vectors (one vector when nrhs = 1)
template <typename T>
int dslash(wcras_ctx* ctx, const typename VecOf<T>::type* in, typename VecOf<T>::type* out,
           const typename VecOf<T>::type* b_minus, int dot, const typename VecOf<T>::type* dotv, Scalars* sc) {
    typedef typename VecOf<T>::type Vec;
    TimedRegion tr(ctx, sizeof(T) == 4 ? TC_DSLASH : TC_DSLASH64);
    const int V = ctx->geom.V, nr = ctx->nrhs;
    const size_t rstride = (size_t)VecOf<T>::CHUNKS * V;
    // 64-thread CTAs with the full register budget (fp32: __launch_bounds__(64, 6) = at most 168 registers so that six CTAs
    // stay resident per SM, 252 fp64): the compiler then keeps all
    // loads of a site in flight at once, which is what an HBM latency-bound stencil needs -- measured on B200 at
    // 32^4: 130 us (fp32) / 292 us (fp64) against 147 / 330 us at 96 / 186 registers with 128-thread CTAs.
    // fp32, nrhs 2..4: one launch covers the whole stack with CTAs of 32 sites x nrhs right-hand sides; otherwise
    // (nrhs = 1, fp64) one launch of 64-site CTAs per vector of the stack
    // z tiling of the traversal when a t-slice of operands (links + clover + spinors) outgrows what L2 keeps between the
    // visits of t-1 and t+1: the largest divisor of Lz whose slab stays under 30 MB.  Measured on B200 at 48^3 x 96
    // (t-slice 85 MB fp32): 1.49 -> 1.34 ms fp32 (tile 16), 3.30 -> 2.99 ms fp64 (tile 8); at 32^4 (25 / 50 MB) the
    // plain order is as fast or faster, so the tiling starts above 60 MB.
    int ztile = 0;
    {
        const double plane_bytes = (sizeof(T) == 4 ? 768.0 : 1536.0) * ctx->geom.L[0] * ctx->geom.L[1];
        if (ctx->ztile_request >= 0)
            ztile = ctx->ztile_request;  // wcras_set_traversal
        else if (plane_bytes * ctx->geom.L[2] > 60e6)
            for (int z = 1; z < ctx->geom.L[2]; z++)
                if (ctx->geom.L[2] % z == 0 && plane_bytes * z <= 30e6) ztile = z;
    }
    const bool stacked = sizeof(T) == 4 && nr >= 2 && nr <= 4;
    const unsigned grid = stacked ? (V + 31) / 32 : (V + 63) / 64;
    const unsigned nblk = stacked ? grid : grid * (unsigned)nr;  // partials of the fused dots
    double* slice = nullptr;
    unsigned* fticket = nullptr;
    if (dot) {
        if (!ctx->dpart || ctx->dpart_blocks < nblk) {  // [3][nblk] per-CTA partials, then [FIN_CTAS][3] slice sums and one ticket
            if (alloc_dev(ctx, (void**)&ctx->dpart, sizeof(double) * (3 * (size_t)nblk + 3 * FIN_CTAS + 1))) return WCRAS_CUDA_ERROR;
            ctx->dpart_blocks = nblk;
            WC_CUDA(cudaMemsetAsync(ctx->dpart + 3 * (size_t)nblk + 3 * FIN_CTAS, 0, sizeof(double), ctx->stream));
        }
        slice = ctx->dpart + 3 * (size_t)ctx->dpart_blocks;
        fticket = (unsigned*)(slice + 3 * FIN_CTAS);
    }
    // small lattices, one right-hand side: the Dslash finishes its dots itself (dslash_finish_inline)
    const bool fin = dot && nr == 1 && nblk <= FIN_INLINE_MAX;
#define WC_DSL(TH, BLOCK, INP, OUTP, BM, DV, POFF)                                                                                    \
    {                                                                                                                              \
        if (fin && dot == 1)                                                                                                       \
            dslash_kernel<T, false, 64, (sizeof(T) == 4 ? 6 : 1), 1, true><<<grid, BLOCK, 0, ctx->stream>>>(ctx->geom, ctx->dslash_fields<T>(), (T)ctx->kappa, INP, OUTP, \
                                                                               nullptr, DV, ctx->dpart, nblk, POFF, rstride, ztile, fticket, sc); \
        else if (fin && dot == 2)                                                                                                  \
            dslash_kernel<T, false, 64, (sizeof(T) == 4 ? 6 : 1), 2, true><<<grid, BLOCK, 0, ctx->stream>>>(ctx->geom, ctx->dslash_fields<T>(), (T)ctx->kappa, INP, OUTP, \
                                                                               nullptr, DV, ctx->dpart, nblk, POFF, rstride, ztile, fticket, sc); \
        else if (fin && dot == 3)                                                                                                  \
            dslash_kernel<T, true, 64, (sizeof(T) == 4 ? 6 : 1), 3, true><<<grid, BLOCK, 0, ctx->stream>>>(ctx->geom, ctx->dslash_fields<T>(), (T)ctx->kappa, INP, OUTP, \
                                                                              BM, nullptr, ctx->dpart, nblk, POFF, rstride, ztile, fticket, sc); \
        else if (dot == 1)                                                                                                              \
            dslash_kernel<T, false, TH, (sizeof(T) == 4 ? 384 / TH : 1), 1><<<grid, BLOCK, 0, ctx->stream>>>(ctx->geom, ctx->dslash_fields<T>(), (T)ctx->kappa, INP, OUTP, \
                                                                               nullptr, DV, ctx->dpart, nblk, POFF, rstride, ztile); \
        else if (dot == 2)                                                                                                         \
            dslash_kernel<T, false, TH, (sizeof(T) == 4 ? 384 / TH : 1), 2><<<grid, BLOCK, 0, ctx->stream>>>(ctx->geom, ctx->dslash_fields<T>(), (T)ctx->kappa, INP, OUTP, \
                                                                               nullptr, DV, ctx->dpart, nblk, POFF, rstride, ztile); \
        else if (dot == 3)                                                                                                         \
            dslash_kernel<T, true, TH, (sizeof(T) == 4 ? 384 / TH : 1), 3><<<grid, BLOCK, 0, ctx->stream>>>(ctx->geom, ctx->dslash_fields<T>(), (T)ctx->kappa, INP, OUTP,  \
                                                                              BM, nullptr, ctx->dpart, nblk, POFF, rstride, ztile);  \
        else if (b_minus)                                                                                                          \
            dslash_kernel<T, true, TH, (sizeof(T) == 4 ? 384 / TH : 1), 0><<<grid, BLOCK, 0, ctx->stream>>>(ctx->geom, ctx->dslash_fields<T>(), (T)ctx->kappa, INP, OUTP,  \
                                                                              BM, nullptr, nullptr, 0, 0, rstride, ztile);         \
        else                                                                                                                       \
            dslash_kernel<T, false, TH, (sizeof(T) == 4 ? 384 / TH : 1), 0><<<grid, BLOCK, 0, ctx->stream>>>(ctx->geom, ctx->dslash_fields<T>(), (T)ctx->kappa, INP, OUTP, \
                                                                               nullptr, nullptr, nullptr, 0, 0, rstride, ztile);   \
        ctx->launches++;                                                                                                           \
    }
    if (stacked) {
        if (nr == 2) WC_DSL(64, dim3(32, 2), in, out, b_minus, dotv, 0)
        else if (nr == 3) WC_DSL(96, dim3(32, 3), in, out, b_minus, dotv, 0)
        else WC_DSL(128, dim3(32, 4), in, out, b_minus, dotv, 0)
    } else {
        for (int r = 0; r < nr; r++)
            WC_DSL(64, dim3(64, 1), in + r * rstride, out + r * rstride, b_minus + r * rstride, dotv + r * rstride, r * grid)
    }
#undef WC_DSL
    if (!fin) {
        if (dot == 1) dot_finish_kernel<1><<<FIN_CTAS, 512, 0, ctx->stream>>>(ctx->dpart, nblk, slice, fticket, sc, ctx->geom.stop);
        if (dot == 2) dot_finish_kernel<2><<<FIN_CTAS, 512, 0, ctx->stream>>>(ctx->dpart, nblk, slice, fticket, sc, ctx->geom.stop);
        if (dot == 3) dot_finish_kernel<3><<<FIN_CTAS, 512, 0, ctx->stream>>>(ctx->dpart, nblk, slice, fticket, sc, nullptr);
        if (dot) ctx->launches++;
    }
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

template int dslash<float>(wcras_ctx*, const float4*, float4*, const float4*, int, const float4*, Scalars*);
template int dslash<double>(wcras_ctx*, const double2*, double2*, const double2*, int, const double2*, Scalars*);
template int dslash_box<float>(wcras_ctx*, const int*, const int*, bool, const float4*, float4*);
template int dslash_box<double>(wcras_ctx*, const int*, const int*, bool, const double2*, double2*);

}  // namespace wc
