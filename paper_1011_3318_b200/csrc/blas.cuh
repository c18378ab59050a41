// blas.cuh -- steps A6/A7: fused BLAS-1 kernels of BiCGStab (north_star (d)): axpy/xpay updates fused with
// the dot products and norms they feed, warp-shuffle reductions, results and the scalar recurrences
// (alpha, beta, omega) kept in device memory so that an iteration needs no host round trip for arithmetic.
//
// Vectors are the flat SoA arrays (fp32: float4 = 2 complex; fp64: double2 = 1 complex); every kernel is
// a grid-stride loop over RED_BLOCKS x RED_THREADS threads.  Reductions: per-thread fp64 accumulation ->
// warp shuffle -> shared memory -> one partial per block -> the last block to finish (atomic ticket) sums
// the partials in a fixed order and applies the scalar update ("post-op").  HBM-bound: 16 B per complex
// pair per pass (fp32), roofline = bytes moved / HBM bandwidth.
#pragma once
#include "wcras_internal.cuh"

namespace wc {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Block-reduce N values, write the block's partial, and let the last block produce the grid total.
// Returns true (in thread 0 of the last block only) with tot[] filled.
template <int N>
__device__ __forceinline__ bool grid_reduce(double (&v)[N], double* __restrict__ partials, unsigned* ticket, double (&tot)[N]) {
    __shared__ double sm[N][RED_THREADS / 32];
    __shared__ bool last;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < N; k++) {
        const double s = warp_sum(v[k]);
        if (lane == 0) sm[k][w] = s;
    }
    __syncthreads();
    if (w == 0) {
#pragma unroll
        for (int k = 0; k < N; k++) {
            double s = lane < RED_THREADS / 32 ? sm[k][lane] : 0.0;
            s = warp_sum(s);
            if (lane == 0) partials[(size_t)blockIdx.x * N + k] = s;
        }
        if (lane == 0) {
            __threadfence();
            const unsigned t = atomicInc(ticket, gridDim.x - 1);
            last = (t == gridDim.x - 1);
        }
    }
    __syncthreads();
    if (!last) return false;
    __threadfence();
    if (w == 0) {
#pragma unroll
        for (int k = 0; k < N; k++) {
            double s = 0;
            for (unsigned b = lane; b < gridDim.x; b += 32) s += __ldcg(&partials[(size_t)b * N + k]);
            tot[k] = warp_sum(s);
        }
        return lane == 0;
    }
    return false;
}

struct cd {  // complex double helper for the scalar recurrences
    double r, i;
};
__device__ __forceinline__ cd cmul(cd a, cd b) { return {a.r * b.r - a.i * b.i, a.r * b.i + a.i * b.r}; }
__device__ __forceinline__ cd cdiv(cd a, cd b) {
    const double d = b.r * b.r + b.i * b.i;
    if (d == 0.0) return {0.0, 0.0};
    return {(a.r * b.r + a.i * b.i) / d, (a.i * b.r - a.r * b.i) / d};
}

// complex element access on the vector types
template <typename Vec> struct Cx;
template <> struct Cx<float4> {
    static constexpr int N = 2;
    __device__ static __forceinline__ void get(const float4& v, int k, double& re, double& im) {
        re = k ? v.z : v.x; im = k ? v.w : v.y;
    }
    __device__ static __forceinline__ float4 make(const double* re, const double* im) {
        return make_float4((float)re[0], (float)im[0], (float)re[1], (float)im[1]);
    }
};
template <> struct Cx<double2> {
    static constexpr int N = 1;
    __device__ static __forceinline__ void get(const double2& v, int, double& re, double& im) { re = v.x; im = v.y; }
    __device__ static __forceinline__ double2 make(const double* re, const double* im) { return make_double2(re[0], im[0]); }
};

}  // namespace wc
