// site_math.cuh -- per-site arithmetic of the Wilson-clover operator, in registers.
//
// Everything here works on small fixed-size arrays that the kernels keep in registers:
//   spinor      T s[24]   index (spin*3 + colour)*2 + {re,im}
//   half spinor T h[12]   index (hs*3   + colour)*2 + {re,im}, hs = 0,1
//   link        T u[18]   index (row*3  + col)*2    + {re,im}, (U psi)_a = sum_b U[a][b] psi_b
//   clover      T c[72]   two chiral 6x6 Hermitian blocks of 36 reals: 6 real diagonal entries, then the
//                         15 strictly-lower entries (i>j, k = i(i-1)/2 + j) as {re,im}; block 0 acts on
//                         spins 0,1 and block 1 on spins 2,3 (component index within a block = spin*3+colour)
//
// Operator (BASELINE.json:north_star; PAPER.md:27-31 only names it):
//   (D psi)(x) = A(x) psi(x) - kappa sum_mu [ (1-gamma_mu) U_mu(x) psi(x+mu) + (1+gamma_mu) U_mu(x-mu)^dag psi(x-mu) ]
// gamma matrices: Hermitian chiral basis, gamma_k = sigma_2 (x) sigma_k, gamma_t = sigma_1 (x) 1 (Q2).
// In this basis (1 -+ gamma_mu) has rank 2 and rows 2,3 are +-1 or +-i times rows 0,1 of the projected
// spinor, so only a half spinor (2 spin x 3 colour) is multiplied by the link ("projected-spinor hopping
// term", north_star (b)).
#pragma once

#if defined(__CUDACC__)
#define WC_HD __host__ __device__ __forceinline__
#else
#define WC_HD inline
#endif

namespace wc {

// ---- packed fp32 pairs (Blackwell FFMA2 / FADD2 / FMUL2, PTX fma/add/mul.rn.f32x2) ----
// A complex number (re, im) occupies one aligned 64-bit register pair; the SASS forms take a per-operand lane swap, a
// per-lane negation and a 32-bit broadcast for free, so a complex multiply-accumulate by a scalar pair (u_re, u_im) is
// exactly two FFMA2 (acc += x * bc(u_re); acc += (i x) * bc(u_im)) instead of four FFMA, with the same products and
// the same accumulation order per component: results are bit-identical to the scalar code below.  The block solvers
// are bound by instruction issue, not by the FMA pipe (profiles/r1j_kernels.md), which is what this halves.
// Device code, T = float only; compiled out with -DWC_NO_F32X2.
#if defined(__CUDA_ARCH__) && !defined(WC_NO_F32X2)
#define WC_X2 1
namespace x2 {
typedef unsigned long long c2;
__device__ __forceinline__ c2 pk(float a, float b) { c2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void up(c2 r, float& a, float& b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(r)); }
__device__ __forceinline__ float lo(c2 r) { float a, b; up(r, a, b); return a; }
__device__ __forceinline__ float hi(c2 r) { float a, b; up(r, a, b); return b; }
__device__ __forceinline__ c2 ld(const float* p) { return pk(p[0], p[1]); }
__device__ __forceinline__ void st(float* p, c2 r) { up(r, p[0], p[1]); }
__device__ __forceinline__ c2 bc(float a) { return pk(a, a); }
__device__ __forceinline__ c2 rot(c2 a) { return pk(-hi(a), lo(a)); }    //  i a
__device__ __forceinline__ c2 mrot(c2 a) { return pk(hi(a), -lo(a)); }   // -i a
__device__ __forceinline__ c2 add(c2 a, c2 b) { c2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ c2 sub(c2 a, c2 b) { c2 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ c2 mul(c2 a, c2 b) { c2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ c2 fma(c2 a, c2 b, c2 c) { c2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
template <int S> __device__ __forceinline__ c2 addsub(c2 a, c2 b) { return S > 0 ? add(a, b) : sub(a, b); }          // a + S b
template <int S> __device__ __forceinline__ c2 addrot(c2 a, c2 b) { return S > 0 ? add(a, rot(b)) : add(a, mrot(b)); }  // a + S i b

template <int MU, int SIGN>
__device__ __forceinline__ void project(const float* __restrict__ s, float* __restrict__ h) {
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const c2 s0 = ld(s + 2 * c), s1 = ld(s + 6 + 2 * c), s2 = ld(s + 12 + 2 * c), s3 = ld(s + 18 + 2 * c);
        c2 h0, h1;
        if (MU == 0) { h0 = addrot<-SIGN>(s0, s3); h1 = addrot<-SIGN>(s1, s2); }
        else if (MU == 1) { h0 = addsub<-SIGN>(s0, s3); h1 = addsub<SIGN>(s1, s2); }
        else if (MU == 2) { h0 = addrot<-SIGN>(s0, s2); h1 = addrot<SIGN>(s1, s3); }
        else { h0 = addsub<SIGN>(s0, s2); h1 = addsub<SIGN>(s1, s3); }
        st(h + 2 * c, h0);
        st(h + 6 + 2 * c, h1);
    }
}

template <int MU, int SIGN, int NEG>
__device__ __forceinline__ void reconstruct_acc(const float* __restrict__ g, float* __restrict__ acc) {
    constexpr int SG = NEG ? -1 : 1;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const c2 g0 = ld(g + 2 * c), g1 = ld(g + 6 + 2 * c);
        st(acc + 2 * c, addsub<SG>(ld(acc + 2 * c), g0));
        st(acc + 6 + 2 * c, addsub<SG>(ld(acc + 6 + 2 * c), g1));
        float* a2 = acc + 12 + 2 * c;
        float* a3 = acc + 18 + 2 * c;
        if (MU == 0) { st(a2, addrot<SG * SIGN>(ld(a2), g1)); st(a3, addrot<SG * SIGN>(ld(a3), g0)); }         // r2 = SIGN i g1, r3 = SIGN i g0
        else if (MU == 1) { st(a2, addsub<SG * SIGN>(ld(a2), g1)); st(a3, addsub<-SG * SIGN>(ld(a3), g0)); }    // r2 = SIGN g1, r3 = -SIGN g0
        else if (MU == 2) { st(a2, addrot<SG * SIGN>(ld(a2), g0)); st(a3, addrot<-SG * SIGN>(ld(a3), g1)); }    // r2 = SIGN i g0, r3 = -SIGN i g1
        else { st(a2, addsub<SG * SIGN>(ld(a2), g0)); st(a3, addsub<SG * SIGN>(ld(a3), g1)); }                 // r2 = SIGN g0, r3 = SIGN g1
    }
}

__device__ __forceinline__ void su3_mul(const float* __restrict__ u, const float* __restrict__ h, float* __restrict__ g) {
#pragma unroll
    for (int hs = 0; hs < 2; hs++) {
        const c2 x0 = ld(h + hs * 6), x1 = ld(h + hs * 6 + 2), x2 = ld(h + hs * 6 + 4);
#pragma unroll
        for (int a = 0; a < 3; a++) {
            const float* ua = u + a * 6;
            c2 acc = mul(x0, bc(ua[0]));
            acc = fma(rot(x0), bc(ua[1]), acc);
            acc = fma(x1, bc(ua[2]), acc);
            acc = fma(rot(x1), bc(ua[3]), acc);
            acc = fma(x2, bc(ua[4]), acc);
            acc = fma(rot(x2), bc(ua[5]), acc);
            st(g + (hs * 3 + a) * 2, acc);
        }
    }
}

__device__ __forceinline__ void su3_adj_mul(const float* __restrict__ u, const float* __restrict__ h, float* __restrict__ g) {
#pragma unroll
    for (int hs = 0; hs < 2; hs++) {
        const c2 x0 = ld(h + hs * 6), x1 = ld(h + hs * 6 + 2), x2 = ld(h + hs * 6 + 4);
#pragma unroll
        for (int a = 0; a < 3; a++) {
            c2 acc = mul(x0, bc(u[a * 2]));
            acc = fma(mrot(x0), bc(u[a * 2 + 1]), acc);
            acc = fma(x1, bc(u[(3 + a) * 2]), acc);
            acc = fma(mrot(x1), bc(u[(3 + a) * 2 + 1]), acc);
            acc = fma(x2, bc(u[(6 + a) * 2]), acc);
            acc = fma(mrot(x2), bc(u[(6 + a) * 2 + 1]), acc);
            st(g + (hs * 3 + a) * 2, acc);
        }
    }
}

__device__ __forceinline__ void herm6_mul(const float* __restrict__ b, const float* __restrict__ x, float* __restrict__ out) {
    c2 xv[6];
#pragma unroll
    for (int j = 0; j < 6; j++) xv[j] = ld(x + 2 * j);
#pragma unroll
    for (int i = 0; i < 6; i++) {
        c2 acc = mul(xv[i], bc(b[i]));
#pragma unroll
        for (int j = 0; j < 6; j++) {
            if (j < i) {
                const int k = 6 + 2 * (i * (i - 1) / 2 + j);
                acc = fma(xv[j], bc(b[k]), acc);
                acc = fma(rot(xv[j]), bc(b[k + 1]), acc);
            } else if (j > i) {
                const int k = 6 + 2 * (j * (j - 1) / 2 + i);
                acc = fma(xv[j], bc(b[k]), acc);
                acc = fma(mrot(xv[j]), bc(b[k + 1]), acc);
            }
        }
        st(out + 2 * i, acc);
    }
}

// the three domain-local sums of one MR iteration (reading Q9) over the 12 components of a site:
// d0 + i d1 += <q, rho> (conjugate on q), d2 += <q, q>
__device__ __forceinline__ void mr_dots(const float* __restrict__ q, const float* __restrict__ rho, float& d0, float& d1, float& d2) {
    c2 d = pk(d0, d1), n = pk(d2, 0.f);
#pragma unroll
    for (int k = 0; k < 12; k++) {
        const c2 r = ld(rho + 2 * k), qq = ld(q + 2 * k);
        d = fma(r, bc(q[2 * k]), d);
        d = fma(mrot(r), bc(q[2 * k + 1]), d);
        n = fma(qq, qq, n);
    }
    up(d, d0, d1);
    d2 = lo(n) + hi(n);
}

// v += alpha rho; rho -= alpha q (UPD_RHO), alpha = ar + i ai
template <bool UPD_RHO, int NC = 12>
__device__ __forceinline__ void mr_update(float ar, float ai, const float* __restrict__ q, float* __restrict__ rho, float* __restrict__ v) {
#pragma unroll
    for (int k = 0; k < NC; k++) {
        const c2 r = ld(rho + 2 * k);
        c2 vv = ld(v + 2 * k);
        vv = fma(r, bc(ar), vv);
        vv = fma(rot(r), bc(ai), vv);
        st(v + 2 * k, vv);
        if (UPD_RHO) {
            const c2 qq = ld(q + 2 * k);
            c2 rr = fma(qq, bc(-ar), r);
            rr = fma(mrot(qq), bc(ai), rr);
            st(rho + 2 * k, rr);
        }
    }
}
}  // namespace x2
#endif

// h = upper two rows of (1 + SIGN*gamma_MU) s
template <typename T, int MU, int SIGN>
WC_HD void project(const T* __restrict__ s, T* __restrict__ h) {
#ifdef WC_X2
    if constexpr (sizeof(T) == 4) {
        x2::project<MU, SIGN>(reinterpret_cast<const float*>(s), reinterpret_cast<float*>(h));
    } else
#endif
    {
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const T s0r = s[2 * c], s0i = s[2 * c + 1];
        const T s1r = s[6 + 2 * c], s1i = s[6 + 2 * c + 1];
        const T s2r = s[12 + 2 * c], s2i = s[12 + 2 * c + 1];
        const T s3r = s[18 + 2 * c], s3i = s[18 + 2 * c + 1];
        T h0r, h0i, h1r, h1i;
        if (MU == 0) {  // (gamma_x s)_0 = -i s3, (gamma_x s)_1 = -i s2
            if (SIGN < 0) { h0r = s0r - s3i; h0i = s0i + s3r; h1r = s1r - s2i; h1i = s1i + s2r; }   // s0 + i s3, s1 + i s2
            else          { h0r = s0r + s3i; h0i = s0i - s3r; h1r = s1r + s2i; h1i = s1i - s2r; }   // s0 - i s3, s1 - i s2
        } else if (MU == 1) {  // (gamma_y s)_0 = -s3, (gamma_y s)_1 = s2
            if (SIGN < 0) { h0r = s0r + s3r; h0i = s0i + s3i; h1r = s1r - s2r; h1i = s1i - s2i; }
            else          { h0r = s0r - s3r; h0i = s0i - s3i; h1r = s1r + s2r; h1i = s1i + s2i; }
        } else if (MU == 2) {  // (gamma_z s)_0 = -i s2, (gamma_z s)_1 = i s3
            if (SIGN < 0) { h0r = s0r - s2i; h0i = s0i + s2r; h1r = s1r + s3i; h1i = s1i - s3r; }   // s0 + i s2, s1 - i s3
            else          { h0r = s0r + s2i; h0i = s0i - s2r; h1r = s1r - s3i; h1i = s1i + s3r; }   // s0 - i s2, s1 + i s3
        } else {  // (gamma_t s)_0 = s2, (gamma_t s)_1 = s3
            if (SIGN < 0) { h0r = s0r - s2r; h0i = s0i - s2i; h1r = s1r - s3r; h1i = s1i - s3i; }
            else          { h0r = s0r + s2r; h0i = s0i + s2i; h1r = s1r + s3r; h1i = s1i + s3i; }
        }
        h[2 * c] = h0r; h[2 * c + 1] = h0i;
        h[6 + 2 * c] = h1r; h[6 + 2 * c + 1] = h1i;
    }
    }
}

// acc += sg * (full spinor whose upper rows are g and whose rows 2,3 follow from (1 + SIGN*gamma_MU)), sg = +1 or,
// with NEG, -1 (a compile-time sign: it folds into the operand negation of the adds)
template <typename T, int MU, int SIGN, int NEG>
WC_HD void reconstruct_acc(const T* __restrict__ g, T* __restrict__ acc) {
#ifdef WC_X2
    if constexpr (sizeof(T) == 4) {
        x2::reconstruct_acc<MU, SIGN, NEG>(reinterpret_cast<const float*>(g), reinterpret_cast<float*>(acc));
    } else
#endif
    {
    const T sg = NEG ? T(-1) : T(1);
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const T g0r = g[2 * c], g0i = g[2 * c + 1];
        const T g1r = g[6 + 2 * c], g1i = g[6 + 2 * c + 1];
        acc[2 * c] += sg * g0r; acc[2 * c + 1] += sg * g0i;
        acc[6 + 2 * c] += sg * g1r; acc[6 + 2 * c + 1] += sg * g1i;
        T* a2 = acc + 12 + 2 * c;
        T* a3 = acc + 18 + 2 * c;
        if (MU == 0) {
            if (SIGN < 0) { a2[0] += sg * g1i; a2[1] -= sg * g1r; a3[0] += sg * g0i; a3[1] -= sg * g0r; }   // r2 = -i g1, r3 = -i g0
            else          { a2[0] -= sg * g1i; a2[1] += sg * g1r; a3[0] -= sg * g0i; a3[1] += sg * g0r; }   // r2 =  i g1, r3 =  i g0
        } else if (MU == 1) {
            if (SIGN < 0) { a2[0] -= sg * g1r; a2[1] -= sg * g1i; a3[0] += sg * g0r; a3[1] += sg * g0i; }   // r2 = -g1, r3 = g0
            else          { a2[0] += sg * g1r; a2[1] += sg * g1i; a3[0] -= sg * g0r; a3[1] -= sg * g0i; }   // r2 = g1, r3 = -g0
        } else if (MU == 2) {
            if (SIGN < 0) { a2[0] += sg * g0i; a2[1] -= sg * g0r; a3[0] -= sg * g1i; a3[1] += sg * g1r; }   // r2 = -i g0, r3 = i g1
            else          { a2[0] -= sg * g0i; a2[1] += sg * g0r; a3[0] += sg * g1i; a3[1] -= sg * g1r; }   // r2 = i g0, r3 = -i g1
        } else {
            if (SIGN < 0) { a2[0] -= sg * g0r; a2[1] -= sg * g0i; a3[0] -= sg * g1r; a3[1] -= sg * g1i; }   // r2 = -g0, r3 = -g1
            else          { a2[0] += sg * g0r; a2[1] += sg * g0i; a3[0] += sg * g1r; a3[1] += sg * g1i; }
        }
    }
    }
}

template <typename T, int MU, int SIGN>
WC_HD void reconstruct_add(const T* __restrict__ g, T* __restrict__ acc) { reconstruct_acc<T, MU, SIGN, 0>(g, acc); }
template <typename T, int MU, int SIGN>
WC_HD void reconstruct_sub(const T* __restrict__ g, T* __restrict__ acc) { reconstruct_acc<T, MU, SIGN, 1>(g, acc); }

// Explicit fused multiply-add chains: written out because the compiler may not re-associate
// "re += ur*hr - ui*hi" into two FMAs on the accumulator (it emits FMUL + FFMA + FADD instead).
WC_HD float wc_fma(float a, float b, float c) { return fmaf(a, b, c); }
WC_HD double wc_fma(double a, double b, double c) { return fma(a, b, c); }

// g = U h  (both half-spin components)
template <typename T>
WC_HD void su3_mul(const T* __restrict__ u, const T* __restrict__ h, T* __restrict__ g) {
#ifdef WC_X2
    if constexpr (sizeof(T) == 4) {
        x2::su3_mul(reinterpret_cast<const float*>(u), reinterpret_cast<const float*>(h), reinterpret_cast<float*>(g));
    } else
#endif
    {
#pragma unroll
    for (int hs = 0; hs < 2; hs++)
#pragma unroll
        for (int a = 0; a < 3; a++) {
            const T* ua = u + a * 6;
            const T* hh = h + hs * 6;
            T re = ua[0] * hh[0];
            T im = ua[0] * hh[1];
            re = wc_fma(-ua[1], hh[1], re);
            im = wc_fma(ua[1], hh[0], im);
#pragma unroll
            for (int b = 1; b < 3; b++) {
                re = wc_fma(ua[2 * b], hh[2 * b], re);
                im = wc_fma(ua[2 * b], hh[2 * b + 1], im);
                re = wc_fma(-ua[2 * b + 1], hh[2 * b + 1], re);
                im = wc_fma(ua[2 * b + 1], hh[2 * b], im);
            }
            g[(hs * 3 + a) * 2] = re;
            g[(hs * 3 + a) * 2 + 1] = im;
        }
    }
}

// g = U^dagger h
template <typename T>
WC_HD void su3_adj_mul(const T* __restrict__ u, const T* __restrict__ h, T* __restrict__ g) {
#ifdef WC_X2
    if constexpr (sizeof(T) == 4) {
        x2::su3_adj_mul(reinterpret_cast<const float*>(u), reinterpret_cast<const float*>(h), reinterpret_cast<float*>(g));
    } else
#endif
    {
#pragma unroll
    for (int hs = 0; hs < 2; hs++)
#pragma unroll
        for (int a = 0; a < 3; a++) {
            const T* hh = h + hs * 6;
            // (U^dag)_ab = conj(U_ba): real part u[(b*3+a)*2], imaginary part -u[(b*3+a)*2+1]
            T re = u[a * 2] * hh[0];
            T im = u[a * 2] * hh[1];
            re = wc_fma(u[a * 2 + 1], hh[1], re);
            im = wc_fma(-u[a * 2 + 1], hh[0], im);
#pragma unroll
            for (int b = 1; b < 3; b++) {
                const T ur = u[(b * 3 + a) * 2], ui = u[(b * 3 + a) * 2 + 1];
                re = wc_fma(ur, hh[2 * b], re);
                im = wc_fma(ur, hh[2 * b + 1], im);
                re = wc_fma(ui, hh[2 * b + 1], re);
                im = wc_fma(-ui, hh[2 * b], im);
            }
            g[(hs * 3 + a) * 2] = re;
            g[(hs * 3 + a) * 2 + 1] = im;
        }
    }
}

// hop += (1 - gamma_MU) U psi_fwd      (forward hop; u = U_MU(x), sf = psi(x+MU))
template <typename T, int MU>
WC_HD void hop_fwd(const T* __restrict__ u, const T* __restrict__ sf, T* __restrict__ hop) {
    T h[12], g[12];
    project<T, MU, -1>(sf, h);
    su3_mul<T>(u, h, g);
    reconstruct_add<T, MU, -1>(g, hop);
}

// hop += (1 + gamma_MU) U^dag psi_bwd  (backward hop; u = U_MU(x-MU), sb = psi(x-MU))
template <typename T, int MU>
WC_HD void hop_bwd(const T* __restrict__ u, const T* __restrict__ sb, T* __restrict__ hop) {
    T h[12], g[12];
    project<T, MU, +1>(sb, h);
    su3_adj_mul<T>(u, h, g);
    reconstruct_add<T, MU, +1>(g, hop);
}

// out[12 reals of one chirality] = B x, B = packed Hermitian 6x6 (36 reals), x = 6 complex
template <typename T>
WC_HD void herm6_mul(const T* __restrict__ b, const T* __restrict__ x, T* __restrict__ out) {
#ifdef WC_X2
    if constexpr (sizeof(T) == 4) {
        x2::herm6_mul(reinterpret_cast<const float*>(b), reinterpret_cast<const float*>(x), reinterpret_cast<float*>(out));
    } else
#endif
    {
#pragma unroll
    for (int i = 0; i < 6; i++) {
        T re = b[i] * x[2 * i], im = b[i] * x[2 * i + 1];
#pragma unroll
        for (int j = 0; j < 6; j++) {
            if (j < i) {  // A_ij, stored
                const int k = 6 + 2 * (i * (i - 1) / 2 + j);
                re = wc_fma(b[k], x[2 * j], re);
                im = wc_fma(b[k], x[2 * j + 1], im);
                re = wc_fma(-b[k + 1], x[2 * j + 1], re);
                im = wc_fma(b[k + 1], x[2 * j], im);
            } else if (j > i) {  // A_ij = conj(A_ji)
                const int k = 6 + 2 * (j * (j - 1) / 2 + i);
                re = wc_fma(b[k], x[2 * j], re);
                im = wc_fma(b[k], x[2 * j + 1], im);
                re = wc_fma(b[k + 1], x[2 * j + 1], re);
                im = wc_fma(-b[k + 1], x[2 * j], im);
            }
        }
        out[2 * i] = re;
        out[2 * i + 1] = im;
    }
    }
}

// out = A(x) s
template <typename T>
WC_HD void clover_apply(const T* __restrict__ cl, const T* __restrict__ s, T* __restrict__ out) {
    herm6_mul<T>(cl, s, out);
    herm6_mul<T>(cl + 36, s + 12, out + 12);
}

}  // namespace wc
