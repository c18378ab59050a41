// ras_cta_common.cuh -- device helpers shared by the two one-CTA-per-domain block solvers (ras_cta.cu: fp32 operands,
// ras_cta16.cu: fp16 operand storage staged by TMA): shared-memory half-spinor slots, asynchronous copies, the
// domain -> site geometry of PAPER.md:45 (Omega_i, Omega'_i) and the red-black domain enumeration.
#pragma once
#include <cuda_fp16.h>

#include "wcras_internal.cuh"

namespace wc {

__device__ __forceinline__ unsigned cta_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
// predicated 16-byte shared store (no branch): dst == 0xffffffff means "no receiver" (Dirichlet)
__device__ __forceinline__ void st_pred_f4(unsigned addr, float a, float b, float c, float d) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %0, 0xffffffff;\n\t@p st.shared.v4.f32 [%0], {%1, %2, %3, %4};\n\t}" ::"r"(addr),
        "f"(a), "f"(b), "f"(c), "f"(d)
        : "memory");
}
__device__ __forceinline__ void st_half_pred(unsigned dst, unsigned chunk_bytes, const float* h) {
    const unsigned d1 = dst == 0xffffffffu ? dst : dst + chunk_bytes;
    const unsigned d2 = dst == 0xffffffffu ? dst : dst + 2 * chunk_bytes;
    st_pred_f4(dst, h[0], h[1], h[2], h[3]);
    st_pred_f4(d1, h[4], h[5], h[6], h[7]);
    st_pred_f4(d2, h[8], h[9], h[10], h[11]);
}
__device__ __forceinline__ void ld_half_cta(const float4* __restrict__ slot, int nsp, float* h) {
#pragma unroll
    for (int j = 0; j < 3; j++) {
        const float4 v = slot[j * nsp];
        h[4 * j] = v.x; h[4 * j + 1] = v.y; h[4 * j + 2] = v.z; h[4 * j + 3] = v.w;
    }
}
// 16-byte asynchronous global -> shared copy (LDGSTS); the issuing thread waits for its own copies with cp_async_wait
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(cta_smem_u32(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ void prefetch_l2_bulk(const void* p, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// global site index of local site (lc) of domain dom; bulk = belongs to the non-overlapping block
__device__ __forceinline__ size_t cta_site(const FusedGeom& fg, int dom, const int lc[4], int x[4]) {
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        const int bc = dom % fg.nblk[mu];
        dom /= fg.nblk[mu];
        int st = bc * fg.b[mu] - (fg.split[mu] ? fg.s : 0) + lc[mu];
        if (st < 0) st += fg.L[mu];
        if (st >= fg.L[mu]) st -= fg.L[mu];
        x[mu] = st;
    }
    return x[0] + fg.L[0] * (x[1] + fg.L[1] * (x[2] + (size_t)fg.L[2] * x[3]));
}

__device__ __forceinline__ size_t cta_site(const FusedGeom& fg, int dom, const int lc[4]) {
    int x[4];
    return cta_site(fg, dom, lc, x);
}

// domain handled as the h-th of a launch: all domains (colour < 0), or the domains of one colour of the red-black
// (checkerboard) colouring by the parity of the block coordinates (multiplicative Schwarz).  fg.pdir is a direction
// with an even number >= 2 of blocks; h enumerates the lattice of blocks with that direction halved.
__device__ __forceinline__ int launch_dom(const FusedGeom& fg, int h, int colour) {
    if (colour < 0) return h;
    int dom = 0, stride = 1, par = 0, cp = 0, sp = 1;
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        const int nb = fg.nblk[mu], n = mu == fg.pdir ? nb / 2 : nb;
        const int c = h % n;
        h /= n;
        if (mu == fg.pdir) { cp = c; sp = stride; }
        else { par += c; dom += c * stride; }
        stride *= nb;
    }
    return dom + (2 * cp + ((colour + par) & 1)) * sp;
}

// ---- mbarrier + bulk-copy (TMA) helpers ----
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tWC_WAIT:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t@p bra WC_DONE;\n\tbra WC_WAIT;\n\tWC_DONE:\n\t}" ::"r"(bar),
        "r"(parity)
        : "memory");
}
// global -> shared bulk copy (TMA unit, SASS UBLKCP), bytes a multiple of 16, completion counted on the mbarrier
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
                 "r"(bytes), "r"(bar)
                 : "memory");
}

__device__ __forceinline__ void half8_to_float(const uint4& t, float* f) {
    const __half2* h = reinterpret_cast<const __half2*>(&t);
#pragma unroll
    for (int j = 0; j < 4; j++) {
        const float2 p = __half22float2(h[j]);
        f[2 * j] = p.x; f[2 * j + 1] = p.y;
    }
}

}  // namespace wc
