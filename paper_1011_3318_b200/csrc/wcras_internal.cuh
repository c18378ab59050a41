// wcras_internal.cuh -- context, internal SoA layouts and loaders shared by the kernels of libwcras.
//
// Internal layouts (north_star (a): "coalesced, vectorised SoA"); V = sites, site index x fastest:
//   fp32 spinor  float4  [6][V]      chunk c holds reals 4c..4c+3 of the 24 (spin,colour,{re,im})
//   fp64 spinor  double2 [12][V]     one complex per chunk
//   fp32 links   float4  [4][4][V]   (mu, k<4: reals 4k..4k+3 of the 18) + float2 [4][V] (reals 16,17)
//   fp64 links   double2 [4][9][V]
//   fp32 clover  float4  [18][V]     72 packed reals (site_math.cuh)
//   fp64 clover  double2 [36][V]
// Consecutive threads handle consecutive sites, so every load is a full-width coalesced 16-byte access.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <vector>

#include "../../include/wcras.h"
#include "site_math.cuh"

namespace wc {

struct Geom {
    int L[4];
    int V;  // number of sites (<= 2^31 / 36)
    const int* stop = nullptr;  // device flag of the running inner solver: non-zero = converged, the launch is a no-op
};

template <typename T> struct VecOf;
template <> struct VecOf<float> { typedef float4 type; static constexpr int CHUNKS = 6; };
template <> struct VecOf<double> { typedef double2 type; static constexpr int CHUNKS = 12; };

template <typename T> struct Fields;
template <> struct Fields<float> {
    const float4* ga;
    const float2* gb;
    const float4* cl;
};
template <> struct Fields<double> {
    const double2* g;
    const double2* cl;
};

// ---- loaders (device) ----
__device__ __forceinline__ void load_spinor(const float4* __restrict__ p, size_t stride, size_t i, float* s) {
#pragma unroll
    for (int c = 0; c < 6; c++) {
        const float4 v = p[c * stride + i];
        s[4 * c] = v.x; s[4 * c + 1] = v.y; s[4 * c + 2] = v.z; s[4 * c + 3] = v.w;
    }
}
__device__ __forceinline__ void load_spinor(const double2* __restrict__ p, size_t stride, size_t i, double* s) {
#pragma unroll
    for (int c = 0; c < 12; c++) {
        const double2 v = p[c * stride + i];
        s[2 * c] = v.x; s[2 * c + 1] = v.y;
    }
}
__device__ __forceinline__ void store_spinor(float4* __restrict__ p, size_t stride, size_t i, const float* s) {
#pragma unroll
    for (int c = 0; c < 6; c++) p[c * stride + i] = make_float4(s[4 * c], s[4 * c + 1], s[4 * c + 2], s[4 * c + 3]);
}
__device__ __forceinline__ void store_spinor(double2* __restrict__ p, size_t stride, size_t i, const double* s) {
#pragma unroll
    for (int c = 0; c < 12; c++) p[c * stride + i] = make_double2(s[2 * c], s[2 * c + 1]);
}
__device__ __forceinline__ void load_link(const Fields<float>& f, size_t V, size_t site, int mu, float* u) {
#pragma unroll
    for (int k = 0; k < 4; k++) {
        const float4 v = f.ga[(mu * 4 + k) * V + site];
        u[4 * k] = v.x; u[4 * k + 1] = v.y; u[4 * k + 2] = v.z; u[4 * k + 3] = v.w;
    }
    const float2 w = f.gb[mu * V + site];
    u[16] = w.x; u[17] = w.y;
}
__device__ __forceinline__ void load_link(const Fields<double>& f, size_t V, size_t site, int mu, double* u) {
#pragma unroll
    for (int k = 0; k < 9; k++) {
        const double2 v = f.g[(mu * 9 + k) * V + site];
        u[2 * k] = v.x; u[2 * k + 1] = v.y;
    }
}
__device__ __forceinline__ void load_clover(const Fields<float>& f, size_t V, size_t site, float* c) {
#pragma unroll
    for (int k = 0; k < 18; k++) {
        const float4 v = f.cl[k * V + site];
        c[4 * k] = v.x; c[4 * k + 1] = v.y; c[4 * k + 2] = v.z; c[4 * k + 3] = v.w;
    }
}
__device__ __forceinline__ void load_clover(const Fields<double>& f, size_t V, size_t site, double* c) {
#pragma unroll
    for (int k = 0; k < 36; k++) {
        const double2 v = f.cl[k * V + site];
        c[2 * k] = v.x; c[2 * k + 1] = v.y;
    }
}

__device__ __forceinline__ void site_coords(const Geom& g, int i, int x[4]) {
    x[0] = i % g.L[0]; i /= g.L[0];
    x[1] = i % g.L[1]; i /= g.L[1];
    x[2] = i % g.L[2];
    x[3] = i / g.L[2];
}

// ---- device-resident solver scalars (all fp64) ----
struct Scalars {
    double rho[2];      // <rt, r> of the current residual
    double rho_old[2];  // value used in the previous iteration
    double alpha[2], omega[2], beta[2];
    double rtv[2];      // <rt, v>
    double ts[2];       // <t, s>
    double tt;          // <t, t>
    double rr;          // |r|^2
    double ss;          // |s|^2
    double bb;          // |b|^2
    double nrm;         // scratch norm^2 (conversion / true residual)
    double scale;       // scratch
    // device-side convergence control (no host round trip per iteration: the inner solver does "most of
    // arithmetics" on the GPU): every kernel of an iteration returns at once when flag != 0
    double thresh;      // tol^2: converged when |r|^2 < thresh * |b|^2
    double tiny;        // breakdown threshold on |rho| / |b|^2 and |omega|
    int flag;           // 0 running, 1 converged, 2 converged at the half step (x += alpha ph pending), 3 breakdown / NaN
    int it_done;        // completed iterations (a half-step exit counts as one)
    int half;           // test |s| after the first half step
    int half_exit;      // the solve ended at a half step
};

}  // namespace wc

// ---- RAS configuration ----
// geometry of the fused on-chip block solver (ras_fused.cu)
struct FusedGeom {
    int L[4], b[4], nblk[4], ext[4], sb[4], c[4];
    int split[4];  // b < L: direction is cut, Omega' extended by s per side, Dirichlet unless ext == L
    int wrap[4];   // ext == L: hops across the domain edge stay inside Omega' (Q7)
    int V, s, ns, nsp, C, niter;
    int nclus;       // tier 2b: clusters (or CTAs) resident at once = persistent grid size in clusters
    int pdir;        // multiplicative Schwarz: pairing direction of the red-black domain enumeration, -1 = not colourable
    int mr2 = 0;     // block solver: 1 = restarted two-dimensional minimal residual (reading R2; ras_cta16.cu; the generic tier reads ctx->block_solver)
    const int* stop; // device flag of the running inner solver (see wc::Geom::stop), or nullptr
};

struct RasConfig {
    bool set = false;
    int b[4] = {0, 0, 0, 0};      // block shape
    int ext[4] = {0, 0, 0, 0};    // extended-domain extents
    int nblk[4] = {0, 0, 0, 0};   // blocks per direction
    int s = 0, niter = 0, nras = 1;
    int nd = 0;                   // number of domains
    int nloc = 0;                 // sites per extended domain
    int tier = 1;                 // 1 generic, 2 fused
    bool cta = false;             // fused tier, single persistent CTA per domain (ras_cta.cu)
    bool cta16 = false;           // the same with fp16 operand storage staged by TMA (ras_cta16.cu)
    bool pair = false;            // the same with two threads per site, 16 warps per SM (ras_pair.cu)
    bool cl16 = false;            // cluster tier with fp16 operand storage staged by TMA (ras_cl16.cu)
    bool stream = false;          // fused tier 2c: rho, v in (distributed) shared memory, operands streamed (ras_stream.cu)
};
constexpr int FUSED_CTA_MAX_THREADS = 256;

enum TimeClass { TC_DSLASH = 0, TC_BLOCK = 1, TC_BLAS = 2, TC_DSLASH64 = 3, TC_COUNT = 4 };

struct wcras_ctx {
    wc::Geom geom;
    double kappa, csw;
    cudaStream_t stream;
    // fields
    double2* g64 = nullptr;
    float4* g32a = nullptr;
    float2* g32b = nullptr;
    double2* c64 = nullptr;
    float4* c32 = nullptr;
    // RAS
    RasConfig ras;
    int tier_request = 0;
    int ztile_request = -1;        // z-tile size of the Dslash traversal: -1 automatic, 0 off (wcras_set_traversal)
    int schwarz = 0;               // 0 additive (RAS, the paper's method), 1 multiplicative (SAP, red-black domains)
    int chain_cycles = 1;          // overlap 0, persistent-CTA tier: NRAS cycles chained through rho_fin (ras_cta.cu)
    FusedGeom fused;               // valid when ras.tier == 2
    float4* dm = nullptr;          // domain-major operand copy of the persistent-CTA tier: [nd][36][nsp]
    int op_prec = 32;              // operand storage of the block solver: 32, or 16 (reading R1: K_RAS of the operator with
                                   // fp16-rounded links and clover blocks), wcras_set_operand_precision
    uint4* dm16 = nullptr;         // fp16 domain-major operand copy (ras_cta16.cu): [nd][18][nsp]
    float4* rf_dm = nullptr;       // rho_fin of the chained cycles, domain-major: [nd][6][nsp]
    int4* dom_org = nullptr;       // ras_cta16: first site of every extended domain (inside the rf_dm allocation)
    unsigned* dom_bc = nullptr;    //            block coordinates of every domain, 8 bits each
    int stage_halo = 0;            // ras_cta16: halo slots staged in shared memory
    int stream_half = 0;           // ras_stream: operand records packed as fp16
    int block_solver = 0;          // wcras_set_block_solver: 0 = MR, 1 = two-dimensional minimal residual (reading R2)
    size_t cta16_smem = 0;         // its dynamic shared memory
    float4* r16a = nullptr;        // fp32 copies of the fp16-rounded links and clover blocks (16-bit operand mode):
    float2* r16b = nullptr;        //   operands of every K_RAS path that does not read dm16
    float4* r16c = nullptr;
    int dslash_rounded = 0;        // the next fp32 dslash applies the rounded operator (r -= D~ v inside K_RAS)
    int cta_grid = 0;              // its persistent grid size
    int cl16_nclus = 0;            // ras_cl16: clusters resident at once
    int cl16_nfc = 0;              //           padded size of the largest face of a sub-block (halo slots are CTA-major)
    float4* hb = nullptr;          // halo buffers of the chained K_RAS cycles: [2][nd][8][3][nface]
    int nface = 0;
    int hb_nrhs = 0;               // stack depth the halo buffers are allocated for
    float4 *mr_rho = nullptr, *mr_q = nullptr, *mr_v = nullptr;  // [nd][6][nloc]
    float4* mr_q2 = nullptr;                                        // second block solver on the generic tier: q2 = D q1
    double* mr_scal = nullptr;                                     // [niter][nd][nchunk][4] per-CTA partial dots
    // solver parameters
    double inner_tol = 5e-7;       // deepest relative accuracy asked of one fp32 inner solve (reading A2)
    double outer_target = 0;       // absolute residual norm the running outer pass has to reach
    int inner_maxit = 1000, outer_maxit = 50, use_ras = 1;
    // workspace (allocated lazily)
    std::vector<void*> owned;
    float4* w32[12] = {nullptr};   // fp32 vectors, 6V float4 each
    double2* w64[12] = {nullptr};  // fp64 vectors, 12V double2 each
    float4* ras32[3] = {nullptr};  // r, v, phi scratch inside K_RAS
    void* io_a = nullptr;          // canonical-layout staging for the ABI calls
    void* io_b = nullptr;
    wc::Scalars* sc32 = nullptr;   // device scalars of the inner solver
    wc::Scalars* sc64 = nullptr;   // device scalars of the outer solver
    wc::Scalars* sc_host = nullptr;  // pinned
    wc::Scalars* sc_ring = nullptr;  // pinned [SC_RING]: per-iteration snapshots the host polls a few iterations late
    cudaEvent_t ev_ring[4] = {nullptr, nullptr, nullptr, nullptr};
    int lookahead = 1;             // inner iterations enqueued ahead of the host's convergence check (0 = check every one)
    // CUDA graphs of one inner fp32 BiCGStab iteration (solver.cu): kind 0 = first iteration, 1 = second, 2 = every later
    // one; captured the second time a kind runs with the same vectors and configuration, replayed afterwards
    struct IterGraph {
        cudaGraphExec_t exec = nullptr;
        int seen = 0;
        long long d_launches = 0;
        int d_dv32 = 0, d_blk = 0, d_ras = 0;
    } iter_graph[2][3];             // [no preconditioner / preconditioner][kind]
    const void* graph_b = nullptr;  // key of the captured graphs: right-hand side and solution vectors, configuration generation
    const void* graph_x = nullptr;
    unsigned graph_gen = 0;
    unsigned cfg_gen = 1;          // bumped by every call that changes what an inner iteration launches
    int use_graphs = 1;
    // wcras_solve_host: the device->host copy of phi starts before the fp64 true-residual check of the same phi and runs beside
    // it on this stream (solve() in solver.cu); host_out != nullptr only while wcras_solve_host is inside solve()
    double* host_out = nullptr;
    bool host_copied = false;           // solve() has delivered the final phi to host_out
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_copy_ready = nullptr, ev_copy_done = nullptr;
    cudaStream_t cap_stream = nullptr;  // captures run on this internal stream (the caller's may be the legacy default stream, which cannot capture)
    double* partials = nullptr;    // reduction scratch [RED_BLOCKS][8]
    unsigned* ticket = nullptr;
    double* dpart = nullptr;       // per-CTA partials of the dots fused into the Dslash: [3][blocks], slice sums, ticket
    unsigned dpart_blocks = 0;
    double* npart = nullptr;       // per-CTA partials of the norm fused into the layout conversion
    unsigned npart_blocks = 0;
    int nrhs = 1;                  // right-hand sides stacked in every solver vector (wcras_solve_multi)
    int ws_nrhs = 0;               // stack depth the workspace is allocated for
    // timing
    int timing = 0;
    std::vector<cudaEvent_t> ev_pool;
    std::vector<int> ev_class;
    size_t ev_used = 0;
    double ms_class[TC_COUNT] = {0, 0, 0, 0};
    long long launches = 0;
    // counters of the running solve
    int dv32 = 0, dv64 = 0, block_dv = 0, ras_applies = 0;
    char err[512] = {0};

    template <typename T> wc::Fields<T> fields() const;
    template <typename T> wc::Fields<T> dslash_fields() const;  // fields<T>(), or the rounded copies while dslash_rounded
};
template <> inline wc::Fields<float> wcras_ctx::fields<float>() const { return wc::Fields<float>{g32a, g32b, c32}; }
template <> inline wc::Fields<double> wcras_ctx::fields<double>() const { return wc::Fields<double>{g64, c64}; }
template <> inline wc::Fields<double> wcras_ctx::dslash_fields<double>() const { return fields<double>(); }
template <> inline wc::Fields<float> wcras_ctx::dslash_fields<float>() const {
    return dslash_rounded && r16a ? wc::Fields<float>{r16a, r16b, r16c} : fields<float>();
}
// operands of the preconditioner: the fp32 fields, or their fp16-rounded copies in 16-bit operand mode (reading R1)
inline wc::Fields<float> ras_fields(const wcras_ctx* ctx) {
    return ctx->op_prec == 16 && ctx->r16a ? wc::Fields<float>{ctx->r16a, ctx->r16b, ctx->r16c} : ctx->fields<float>();
}

// two timing events, destroyed on every exit path of the function that owns them
struct EventPair {
    cudaEvent_t a = nullptr, b = nullptr;
    cudaError_t create() {
        cudaError_t e = cudaEventCreate(&a);
        return e != cudaSuccess ? e : cudaEventCreate(&b);
    }
    ~EventPair() {
        if (a) cudaEventDestroy(a);
        if (b) cudaEventDestroy(b);
    }
};

#define WC_CUDA(call)                                                                                   \
    do {                                                                                                \
        cudaError_t e_ = (call);                                                                        \
        if (e_ != cudaSuccess) {                                                                        \
            snprintf(ctx->err, sizeof ctx->err, "%s:%d: %s: %s", __FILE__, __LINE__, #call,             \
                     cudaGetErrorString(e_));                                                           \
            return WCRAS_CUDA_ERROR;                                                                    \
        }                                                                                               \
    } while (0)

#define WC_CHECK_LAUNCH() WC_CUDA(cudaGetLastError())

// scoped per-class timing (events only when ctx->timing)
struct TimedRegion {
    wcras_ctx* ctx;
    bool on;
    TimedRegion(wcras_ctx* c, int cls);
    ~TimedRegion();
};

// ---- host entry points implemented across the .cu files ----
namespace wc {
// BLAS-1 grid: ONE 1024-thread CTA per SM.  Measured on B200 at 32^4 (k_update_xr, 8 vector passes): 148 x 1024
// 125 us = 6.4 TB/s, 296 x 1024 127 us, 592 x 256 150 us, 1184 x 256 155 us, 296 x 256 221 us -- with several
// smaller CTAs per SM the block scheduler leaves the SMs unevenly loaded and the slowest SM sets the time.
#ifndef WC_RED_BLOCKS
#define WC_RED_BLOCKS 148
#endif
#ifndef WC_RED_THREADS
#define WC_RED_THREADS 1024
#endif
constexpr int RED_BLOCKS = WC_RED_BLOCKS;
constexpr int RED_THREADS = WC_RED_THREADS;

int alloc_dev(wcras_ctx* ctx, void** p, size_t bytes);
int ensure_workspace(wcras_ctx* ctx);
void drop_iter_graphs(wcras_ctx* ctx);  // solver.cu

// layout.cu
int setup_fields(wcras_ctx* ctx, const double* gauge_dev);
int to_internal(wcras_ctx* ctx, int prec, const void* canonical, void* internal, Scalars* norm_sc = nullptr);
int from_internal(wcras_ctx* ctx, int prec, const void* internal, void* canonical);
int export_clover(wcras_ctx* ctx, double* out_dev);

// dslash.cu : out = D in   or   out = b - D in (b may alias out)
// dot = 1: also rtv = <dotv, out>, alpha = rho/rtv; dot = 2: also ts = <out, dotv>, tt = |out|^2, omega = ts/tt (sc)
template <typename T>
int dslash(wcras_ctx* ctx, const typename VecOf<T>::type* in, typename VecOf<T>::type* out,
           const typename VecOf<T>::type* b_minus = nullptr, int dot = 0, const typename VecOf<T>::type* dotv = nullptr,
           Scalars* sc = nullptr);
template <typename T>
int dslash_box(wcras_ctx* ctx, const int start[4], const int ext[4], bool all_blocks,
               const typename VecOf<T>::type* in, typename VecOf<T>::type* out);

// ras.cu
int ras_configure(wcras_ctx* ctx, const int domain[4], int s, int niter, int nras);
int ras_apply(wcras_ctx* ctx, const float4* r, float4* v);  // v = K_RAS r, internal layout; r is preserved
int ras_block_solve(wcras_ctx* ctx, const float4* r, float4* v);

// solver.cu
int solve(wcras_ctx* ctx, const double* eta_dev, double* phi_dev, double tol, wcras_info* info, double* resid_per_rhs = nullptr);
int time_blas(wcras_ctx* ctx, int reps, double* ms);
}  // namespace wc
