// layout.cu -- setup step A0: canonical -> internal SoA reordering of links and spinors, and the fp64
// construction of the clover term (clover_build.cuh).  One-time cost in wcras_create, not on the timed path.
#include <stdlib.h>
#include "clover_build.cuh"
#include "wcras_internal.cuh"

namespace wc {

int alloc_dev(wcras_ctx* ctx, void** p, size_t bytes) {
    *p = nullptr;
    // fault injection for the out-of-memory paths (tests/test_gpu_parity.py::test_workspace_growth_failure): allocations of
    // at least WCRAS_FAIL_ALLOC_ABOVE bytes fail as cudaMalloc would
    if (const char* e = getenv("WCRAS_FAIL_ALLOC_ABOVE")) {
        if (*e && bytes >= (size_t)strtoull(e, nullptr, 10)) {
            snprintf(ctx->err, sizeof ctx->err, "alloc_dev: out of memory (%zu bytes; injected)", bytes);
            return WCRAS_CUDA_ERROR;
        }
    }
    WC_CUDA(cudaMalloc(p, bytes));
    ctx->owned.push_back(*p);
    return WCRAS_OK;
}

// one thread per (site, mu): canonical [V][4][18] fp64 -> g64 [4][9][V], g32a [4][4][V], g32b [4][V]
__global__ void reorder_gauge_kernel(int V, const double* __restrict__ canon, double2* g64, float4* g32a, float2* g32b) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= 4 * V) return;
    const int mu = t / V, i = t - mu * V;
    const double* u = canon + ((size_t)i * 4 + mu) * 18;
    double r[18];
#pragma unroll
    for (int k = 0; k < 18; k++) r[k] = u[k];
#pragma unroll
    for (int k = 0; k < 9; k++) g64[(size_t)(mu * 9 + k) * V + i] = make_double2(r[2 * k], r[2 * k + 1]);
#pragma unroll
    for (int k = 0; k < 4; k++)
        g32a[(size_t)(mu * 4 + k) * V + i] =
            make_float4((float)r[4 * k], (float)r[4 * k + 1], (float)r[4 * k + 2], (float)r[4 * k + 3]);
    g32b[(size_t)mu * V + i] = make_float2((float)r[16], (float)r[17]);
}

__device__ __forceinline__ void ld_link64(const double2* __restrict__ g, size_t V, size_t site, int mu, double* u) {
#pragma unroll
    for (int k = 0; k < 9; k++) {
        const double2 v = g[(size_t)(mu * 9 + k) * V + site];
        u[2 * k] = v.x; u[2 * k + 1] = v.y;
    }
}

__device__ __forceinline__ int shift1(const Geom& g, const int x[4], int mu, int d) {
    int y[4] = {x[0], x[1], x[2], x[3]};
    y[mu] = (y[mu] + d + g.L[mu]) % g.L[mu];
    return y[0] + g.L[0] * (y[1] + g.L[1] * (y[2] + g.L[2] * y[3]));
}
__device__ __forceinline__ int shift2(const Geom& g, const int x[4], int mu, int d, int nu, int e) {
    int y[4] = {x[0], x[1], x[2], x[3]};
    y[mu] = (y[mu] + d + g.L[mu]) % g.L[mu];
    y[nu] = (y[nu] + e + g.L[nu]) % g.L[nu];
    return y[0] + g.L[0] * (y[1] + g.L[1] * (y[2] + g.L[2] * y[3]));
}

// one thread per (plane, site): F_mu_nu(x) -> ftmp [6][9][V] double2
__global__ void field_strength_kernel(Geom g, const double2* __restrict__ g64, double2* __restrict__ ftmp) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= 6 * g.V) return;
    const int p = t / g.V, i = t - p * g.V;
    const int mu = p < 3 ? 0 : (p < 5 ? 1 : 2);
    const int nu = p < 3 ? p + 1 : (p < 5 ? p - 1 : 3);
    int x[4];
    site_coords(g, i, x);
    const size_t V = g.V;
    const int xpm = shift1(g, x, mu, 1), xpn = shift1(g, x, nu, 1), xmm = shift1(g, x, mu, -1),
              xmn = shift1(g, x, nu, -1), xmmpn = shift2(g, x, mu, -1, nu, 1),
              xmmmn = shift2(g, x, mu, -1, nu, -1), xpmmn = shift2(g, x, mu, 1, nu, -1);
    double q[18], a[18], b[18], c[18], d[18], f[18];
#pragma unroll
    for (int k = 0; k < 18; k++) q[k] = 0;
    // U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
    ld_link64(g64, V, i, mu, a); ld_link64(g64, V, xpm, nu, b); ld_link64(g64, V, xpn, mu, c); ld_link64(g64, V, i, nu, d);
    leaf_add<false, false, true, true>(a, b, c, d, q);
    // U_nu(x) U_mu(x-mu+nu)^dag U_nu(x-mu)^dag U_mu(x-mu)
    ld_link64(g64, V, xmmpn, mu, b); ld_link64(g64, V, xmm, nu, c); ld_link64(g64, V, xmm, mu, a);
    leaf_add<false, true, true, false>(d, b, c, a, q);
    // U_mu(x-mu)^dag U_nu(x-mu-nu)^dag U_mu(x-mu-nu) U_nu(x-nu)
    ld_link64(g64, V, xmmmn, nu, b); ld_link64(g64, V, xmmmn, mu, c); ld_link64(g64, V, xmn, nu, d);
    leaf_add<true, true, false, false>(a, b, c, d, q);
    // U_nu(x-nu)^dag U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^dag
    ld_link64(g64, V, xmn, mu, b); ld_link64(g64, V, xpmmn, nu, c); ld_link64(g64, V, i, mu, a);
    leaf_add<true, false, false, true>(d, b, c, a, q);
    antiherm_to_F(q, f);
#pragma unroll
    for (int k = 0; k < 9; k++) ftmp[(size_t)(p * 9 + k) * V + i] = make_double2(f[2 * k], f[2 * k + 1]);
}

// one thread per site: F[6] -> packed clover blocks, fp64 and fp32
__global__ void clover_assemble_kernel(int V, double coeff, const double2* __restrict__ ftmp, double2* __restrict__ c64,
                                       float4* __restrict__ c32) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= V) return;
    double F[6][18];
#pragma unroll
    for (int p = 0; p < 6; p++)
#pragma unroll
        for (int k = 0; k < 9; k++) {
            const double2 v = ftmp[(size_t)(p * 9 + k) * V + i];
            F[p][2 * k] = v.x; F[p][2 * k + 1] = v.y;
        }
    double o[72];
    clover_assemble(F, coeff, o);
#pragma unroll
    for (int k = 0; k < 36; k++) c64[(size_t)k * V + i] = make_double2(o[2 * k], o[2 * k + 1]);
#pragma unroll
    for (int k = 0; k < 18; k++)
        c32[(size_t)k * V + i] = make_float4((float)o[4 * k], (float)o[4 * k + 1], (float)o[4 * k + 2], (float)o[4 * k + 3]);
}

__global__ void export_clover_kernel(int V, const double2* __restrict__ c64, double* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= V) return;
    for (int k = 0; k < 36; k++) {
        const double2 v = c64[(size_t)k * V + i];
        out[(size_t)i * 72 + 2 * k] = v.x;
        out[(size_t)i * 72 + 2 * k + 1] = v.y;
    }
}

// canonical [V][24] <-> SoA [CH][V] through a shared-memory tile of LAYOUT_TS sites: both the canonical side (a site's 24
// reals contiguous) and the SoA side (a chunk's sites contiguous) are then read and written as whole 16-byte rows
constexpr int LAYOUT_TS = 64;
// npart != nullptr: the block's sum of squares goes to npart[blockIdx.x] (|eta|^2 at the start of a solve without a pass of
// its own); norm_finish_kernel sums the partials in a fixed order
template <typename T, typename Vec, int CH>
__global__ void __launch_bounds__(256) spinor_to_internal_kernel(int V, const T* __restrict__ canon, Vec* __restrict__ soa,
                                                                 double* __restrict__ npart) {
    __shared__ Vec tile[LAYOUT_TS * CH];
    __shared__ double wsum[8];
    const size_t i0 = (size_t)blockIdx.x * LAYOUT_TS;
    const int ns = (int)((size_t)V - i0 < (size_t)LAYOUT_TS ? (size_t)V - i0 : (size_t)LAYOUT_TS);
    const Vec* src = reinterpret_cast<const Vec*>(canon) + i0 * CH;  // element e = local site * CH + chunk
    double acc = 0;
    for (int e = threadIdx.x; e < ns * CH; e += blockDim.x) {
        const Vec t = src[e];
        tile[e] = t;
        if (npart) {
            const T* c = reinterpret_cast<const T*>(&t);
#pragma unroll
            for (int j = 0; j < (int)(sizeof(Vec) / sizeof(T)); j++) acc = fma((double)c[j], (double)c[j], acc);
        }
    }
    if (npart) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = acc;
    }
    __syncthreads();
    if (npart && threadIdx.x == 0) {
        double t = 0;
        for (int w = 0; w < 8; w++) t += wsum[w];
        npart[blockIdx.x] = t;
    }
    for (int e = threadIdx.x; e < LAYOUT_TS * CH; e += blockDim.x) {
        const int c = e / LAYOUT_TS, sl = e % LAYOUT_TS;
        if (sl < ns) soa[(size_t)c * V + i0 + sl] = tile[sl * CH + c];
    }
}
__global__ void __launch_bounds__(1024) norm_finish_kernel(unsigned n, const double* __restrict__ npart, Scalars* sc) {
    __shared__ double wsum[32];
    double acc = 0;
    for (unsigned j = threadIdx.x; j < n; j += 1024) acc += npart[j];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0;
        for (int w = 0; w < 32; w++) t += wsum[w];
        sc->nrm = t;
    }
}
template <typename T, typename Vec, int CH>
__global__ void __launch_bounds__(256) spinor_from_internal_kernel(int V, const Vec* __restrict__ soa, T* __restrict__ canon) {
    __shared__ Vec tile[LAYOUT_TS * CH];
    const size_t i0 = (size_t)blockIdx.x * LAYOUT_TS;
    const int ns = (int)((size_t)V - i0 < (size_t)LAYOUT_TS ? (size_t)V - i0 : (size_t)LAYOUT_TS);
    for (int e = threadIdx.x; e < LAYOUT_TS * CH; e += blockDim.x) {
        const int c = e / LAYOUT_TS, sl = e % LAYOUT_TS;
        if (sl < ns) tile[sl * CH + c] = soa[(size_t)c * V + i0 + sl];
    }
    __syncthreads();
    Vec* dst = reinterpret_cast<Vec*>(canon) + i0 * CH;
    for (int e = threadIdx.x; e < ns * CH; e += blockDim.x) dst[e] = tile[e];
}

int setup_fields(wcras_ctx* ctx, const double* gauge_dev) {
    const size_t V = ctx->geom.V;
    if (alloc_dev(ctx, (void**)&ctx->g64, sizeof(double2) * 36 * V)) return WCRAS_CUDA_ERROR;
    if (alloc_dev(ctx, (void**)&ctx->g32a, sizeof(float4) * 16 * V)) return WCRAS_CUDA_ERROR;
    if (alloc_dev(ctx, (void**)&ctx->g32b, sizeof(float2) * 4 * V)) return WCRAS_CUDA_ERROR;
    if (alloc_dev(ctx, (void**)&ctx->c64, sizeof(double2) * 36 * V)) return WCRAS_CUDA_ERROR;
    if (alloc_dev(ctx, (void**)&ctx->c32, sizeof(float4) * 18 * V)) return WCRAS_CUDA_ERROR;
    double2* ftmp = nullptr;
    WC_CUDA(cudaMalloc((void**)&ftmp, sizeof(double2) * 54 * V));
    const int T = 128;
    reorder_gauge_kernel<<<(unsigned)((4 * V + T - 1) / T), T, 0, ctx->stream>>>((int)V, gauge_dev, ctx->g64, ctx->g32a, ctx->g32b);
    field_strength_kernel<<<(unsigned)((6 * V + T - 1) / T), T, 0, ctx->stream>>>(ctx->geom, ctx->g64, ftmp);
    // the literal north_star coefficient c_sw * kappa / 2 (reading Q5) -- the one place it is set
    const double clover_coeff = ctx->csw * ctx->kappa / 2.0;
    clover_assemble_kernel<<<(unsigned)((V + T - 1) / T), T, 0, ctx->stream>>>((int)V, clover_coeff, ftmp, ctx->c64, ctx->c32);
    ctx->launches += 3;
    cudaError_t e = cudaStreamSynchronize(ctx->stream);
    cudaFree(ftmp);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(ctx->err, sizeof ctx->err, "setup_fields: %s", cudaGetErrorString(e));
        return WCRAS_CUDA_ERROR;
    }
    return WCRAS_OK;
}

// norm_sc != nullptr: norm_sc->nrm = |canonical|^2 as well (one small kernel behind the conversion, no extra vector pass)
int to_internal(wcras_ctx* ctx, int prec, const void* canonical, void* internal, Scalars* norm_sc) {
    const int V = ctx->geom.V, T = 256;
    const unsigned nblk = (unsigned)((V + LAYOUT_TS - 1) / LAYOUT_TS);
    if ((uintptr_t)canonical & 15) { snprintf(ctx->err, sizeof ctx->err, "spinor buffers must be 16-byte aligned"); return WCRAS_INVALID_ARG; }
    double* npart = nullptr;
    if (norm_sc) {
        if (!ctx->npart || ctx->npart_blocks < nblk) {
            if (alloc_dev(ctx, (void**)&ctx->npart, sizeof(double) * nblk)) return WCRAS_CUDA_ERROR;
            ctx->npart_blocks = nblk;
        }
        npart = ctx->npart;
    }
    if (prec == 32)
        spinor_to_internal_kernel<float, float4, 6><<<nblk, T, 0, ctx->stream>>>(V, (const float*)canonical, (float4*)internal, npart);
    else
        spinor_to_internal_kernel<double, double2, 12><<<nblk, T, 0, ctx->stream>>>(V, (const double*)canonical, (double2*)internal, npart);
    ctx->launches++;
    if (norm_sc) {
        norm_finish_kernel<<<1, 1024, 0, ctx->stream>>>(nblk, npart, norm_sc);
        ctx->launches++;
    }
    WC_CHECK_LAUNCH();
    return WCRAS_OK;
}

int from_internal(wcras_ctx* ctx, int prec, const void* internal, void* canonical) {
    const int V = ctx->geom.V, T = 256;
    if ((uintptr_t)canonical & 15) { snprintf(ctx->err, sizeof ctx->err, "spinor buffers must be 16-byte aligned"); return WCRAS_INVALID_ARG; }
    if (prec == 32)
        spinor_from_internal_kernel<float, float4, 6><<<(unsigned)((V + LAYOUT_TS - 1) / LAYOUT_TS), T, 0, ctx->stream>>>(
            V, (const float4*)internal, (float*)canonical);
    else
        spinor_from_internal_kernel<double, double2, 12><<<(unsigned)((V + LAYOUT_TS - 1) / LAYOUT_TS), T, 0, ctx->stream>>>(
            V, (const double2*)internal, (double*)canonical);
    ctx->launches++;
    WC_CHECK_LAUNCH();
    return WCRAS_OK;
}

int export_clover(wcras_ctx* ctx, double* out_dev) {
    const int V = ctx->geom.V, T = 128;
    export_clover_kernel<<<(V + T - 1) / T, T, 0, ctx->stream>>>(V, ctx->c64, out_dev);
    ctx->launches++;
    WC_CHECK_LAUNCH();
    return WCRAS_OK;
}

}  // namespace wc
