// microbench_f32x2.cu -- standalone measurement behind the packed-fp32 arithmetic of site_math.cuh (namespace x2):
// issue rate and dependent latency of FFMA / FFMA2 / FADD2 on sm_100a, the cost of the operand modifiers (lane swap,
// per-lane negation), and the FP32-pipe utilisation of the per-site building blocks (SU(3) x half spinor, projection +
// multiplication + reconstruction, packed Hermitian 6x6 x 6-vector) when they run from registers with 1, 2 or 4 warps per
// scheduler.  Not part of libwcras.so; built by `python paper_1011_3318_b200/build.py --microbench`, results in
// profiles/r2_microbench.md.
#include <cstdio>
#include <cuda_runtime.h>

#include "site_math.cuh"

using namespace wc;
typedef unsigned long long u64;

__device__ __forceinline__ u64 pk(float a, float b) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void up(u64 r, float& a, float& b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(r)); }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ u64 add2(u64 a, u64 b) { u64 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }

// MODE 0: FFMA2, 1: FFMA, 2: FADD2; NACC independent accumulators (NACC = 1: dependent latency)
template <int NACC, int MODE>
__global__ void k_rate(float* out, float a, float b, int iters, long long* cyc) {
    u64 acc[NACC];
    float sacc[NACC];
    for (int i = 0; i < NACC; i++) { acc[i] = pk(threadIdx.x * 0.001f + i, 1.f); sacc[i] = threadIdx.x * 0.001f + i; }
    const u64 bb = pk(b, b + 1.f);
    const long long t0 = clock64();
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int r = 0; r < 8; r++)
#pragma unroll
            for (int i = 0; i < NACC; i++) {
                if (MODE == 0) { const u64 aa = pk(a, a); asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc[i]) : "l"(aa), "l"(bb)); }
                else if (MODE == 1) { asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(sacc[i]) : "f"(a), "f"(b)); }
                else { asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(acc[i]) : "l"(bb)); }
            }
    }
    const long long t1 = clock64();
    float s = 0;
    for (int i = 0; i < NACC; i++) { float x, y; up(acc[i], x, y); s += x + y + sacc[i]; }
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

// operand modifiers: every second instruction takes the vector operand plain, the others swapped (MODE 1), swapped and
// negated in one lane (= i x, MODE 2, FFMA2) or the same through FADD2 (MODE 3); MODE 0 / 4: all plain FFMA2 / FADD2
template <int MODE>
__global__ void k_mod(float* out, const float* in, int iters, long long* cyc) {
    u64 acc[8];
    float xr = in[threadIdx.x], xi = in[threadIdx.x + 1024];
    const float s0 = in[threadIdx.x + 2048];
    for (int i = 0; i < 8; i++) acc[i] = pk(threadIdx.x * 0.001f + i, 1.f);
    const long long t0 = clock64();
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int r = 0; r < 8; r++)
#pragma unroll
            for (int i = 0; i < 8; i++) {
                u64 x;
                if (MODE == 0 || MODE == 4 || (i & 1) == 0) x = pk(xr, xi);
                else if (MODE == 1) x = pk(xi, xr);
                else x = pk(-xi, xr);
                if (MODE < 3) acc[i] = fma2(x, pk(s0, s0), acc[i]);
                else acc[i] = add2(acc[i], x);
            }
        xr += 1e-30f;
    }
    const long long t1 = clock64();
    float s = 0;
    for (int i = 0; i < 8; i++) { float x, y; up(acc[i], x, y); s += x + y; }
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

// the per-site building blocks of site_math.cuh from registers.  MODE 0: 8 SU(3) x half-spinor products in a dependent
// chain; 1: 8 x (projection, product, reconstruction) = the hopping part of one Dslash; 2: the two 6x6 clover blocks
template <int MODE>
__global__ void k_site(float* out, const float* in, int iters, long long* cyc) {
    float U[72], h[12], g[12], s[24], q[24], A[72];
    for (int i = 0; i < 72; i++) { U[i] = in[threadIdx.x + 32 * i]; A[i] = in[threadIdx.x + 32 * i + 7]; }
    for (int i = 0; i < 12; i++) h[i] = in[threadIdx.x + i * 64 + 3];
    for (int i = 0; i < 24; i++) { s[i] = in[threadIdx.x + i * 64 + 5]; q[i] = 0.f; }
    for (int i = 0; i < 12; i++) g[i] = 0.f;
    const long long t0 = clock64();
    for (int it = 0; it < iters; it++) {
        if (MODE == 0) {
#pragma unroll
            for (int mu = 0; mu < 4; mu++) { su3_mul<float>(U + 18 * mu, h, g); su3_adj_mul<float>(U + 18 * mu, g, h); }
        } else if (MODE == 1) {
#define HOP(MU)                                                                                        \
    project<float, MU, -1>(s, h); su3_mul<float>(U + 18 * MU, h, g); reconstruct_add<float, MU, -1>(g, q); \
    project<float, MU, +1>(s, h); su3_adj_mul<float>(U + 18 * MU, h, g); reconstruct_add<float, MU, +1>(g, q);
            HOP(0) HOP(1) HOP(2) HOP(3)
#undef HOP
#pragma unroll
            for (int i = 0; i < 24; i++) s[i] = q[i] * 0.1f;
        } else {
            herm6_mul<float>(A, s, q);
            herm6_mul<float>(A + 36, s + 12, q + 12);
#pragma unroll
            for (int i = 0; i < 24; i++) s[i] = q[i];
        }
    }
    const long long t1 = clock64();
    float r = 0;
    for (int i = 0; i < 12; i++) r += h[i] + g[i];
    for (int i = 0; i < 24; i++) r += q[i] + s[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = r;
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

static float* g_out;
static float* g_in;
static long long* g_cyc;

template <typename F> static double cycles(F launch) {
    long long h[148];
    launch();
    cudaDeviceSynchronize();
    launch();
    cudaMemcpy(h, g_cyc, sizeof h, cudaMemcpyDeviceToHost);
    return (double)h[0];
}

int main() {
    cudaMalloc(&g_out, 148 * 1024 * 4);
    cudaMalloc(&g_in, 65536 * 4);
    cudaMemset(g_in, 0, 65536 * 4);
    cudaMalloc(&g_cyc, 148 * 8);
    const int it = 1024;
    printf("== issue interval per warp (cycles per instruction; 148 CTAs, warps per scheduler = threads / 128) ==\n");
#define RATE(NAME, NACC, MODE, THR) \
    printf("%-6s %d accumulators, %4d threads: %.2f\n", NAME, NACC, THR, cycles([&] { k_rate<NACC, MODE><<<148, THR>>>(g_out, 1.0001f, 0.5f, it, g_cyc); }) / (it * 8.0 * NACC));
    RATE("FFMA2", 1, 0, 128) RATE("FFMA2", 2, 0, 128) RATE("FFMA2", 4, 0, 128) RATE("FFMA2", 8, 0, 128) RATE("FFMA2", 8, 0, 256) RATE("FFMA2", 8, 0, 512)
    RATE("FFMA", 1, 1, 128) RATE("FFMA", 2, 1, 128) RATE("FFMA", 4, 1, 128) RATE("FFMA", 8, 1, 128) RATE("FFMA", 8, 1, 256)
    RATE("FADD2", 1, 2, 128) RATE("FADD2", 4, 2, 128)
    printf("== operand modifiers (8 accumulators, 128 threads; cycles per instruction) ==\n");
#define MOD(NAME, MODE) printf("%-28s %.2f\n", NAME, cycles([&] { k_mod<MODE><<<148, 128>>>(g_out, g_in, it, g_cyc); }) / (it * 64.0));
    MOD("FFMA2 plain", 0) MOD("FFMA2 half swapped", 1) MOD("FFMA2 half swapped+negated", 2) MOD("FADD2 half swapped+negated", 3) MOD("FADD2 plain", 4)
    printf("== site_math.cuh building blocks from registers (FP32-pipe cycles needed = 2 per packed instruction) ==\n");
#define SITE(NAME, MODE, PACKED, THR)                                                                                   \
    {                                                                                                                   \
        const double c = cycles([&] { k_site<MODE><<<148, THR>>>(g_out, g_in, 512, g_cyc); }) / 512.0;                   \
        printf("%-30s %4d threads: %7.1f cycles per pass per warp, pipe need %4d -> %3.0f %% of the FP32 pipe\n", NAME, THR, c, 2 * (PACKED), \
               100.0 * 2 * (PACKED) * (THR / 128) / c);                                                                    \
    }
    SITE("8 SU(3) x half spinor", 0, 8 * 36, 128) SITE("8 SU(3) x half spinor", 0, 8 * 36, 256) SITE("8 SU(3) x half spinor", 0, 8 * 36, 512)
    SITE("8 x (project, U, reconstruct)", 1, 8 * (6 + 36 + 12) + 12, 128) SITE("8 x (project, U, reconstruct)", 1, 8 * (6 + 36 + 12) + 12, 256)
    SITE("2 clover blocks", 2, 2 * 66, 128) SITE("2 clover blocks", 2, 2 * 66, 256)
    printf("%s\n", cudaGetErrorString(cudaGetLastError()));
    return 0;
}
