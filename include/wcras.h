/*
 * wcras.h -- C ABI of libwcras: RAS-preconditioned mixed-precision nested BiCGStab for the
 * Wilson-clover Dirac equation D phi = eta on one NVIDIA B200 (sm_100a).
 *
 * Method: arXiv:1011.3318 (Osaki & Ishikawa, "Domain Decomposition method on GPU cluster").  Citations
 * below are PAPER.md:<line> (section / equation / algorithm) or BASELINE.json:north_star where the paper
 * gives no formula.  The readings Q1..Q20 are listed in DESIGN.md.
 *
 * Conventions common to every call
 *   - "dev" pointers are CUDA device pointers, "host" pointers are ordinary host memory.  The caller
 *     owns every buffer it passes; the library never frees or keeps a caller pointer after the call
 *     returns (wcras_create copies the gauge field into its own layouts, so it may be freed afterwards).
 *   - Canonical layouts at the boundary: site index i = x + Lx*(y + Ly*(z + Lz*t)), mu = 0..3 = x,y,z,t.
 *       gauge  [V][4][3][3][2]  fp64, (U psi)_a = sum_b U[a][b] psi_b, {re,im} innermost
 *       spinor [V][4][3][2]     spin, colour, {re,im}; fp32 or fp64 as stated per call; 16-byte aligned
 *                               (WCRAS_INVALID_ARG otherwise)
 *     The internal coalesced SoA layouts (north_star (a)) are private to the library.
 *   - All work is enqueued on the CUDA stream given to wcras_create.  wcras_solve* and wcras_time_kernel
 *     synchronise that stream before returning; the apply_* calls do not.
 *   - in/out buffers of one call must not alias.
 *   - Return value: WCRAS_OK (0) or a negative code; wcras_last_error gives a message.  No exceptions,
 *     no exit(), nothing is printed.  There is no CPU fallback: without a CUDA device every call that
 *     computes returns WCRAS_CUDA_ERROR.
 */
#ifndef WCRAS_H
#define WCRAS_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct wcras_ctx wcras_ctx; /* opaque; owns all internal device copies and workspace */

enum {
    WCRAS_OK = 0,
    WCRAS_INVALID_ARG = -1,   /* null pointer, dims < 2, b does not divide L, b+2s > L in a split direction, prec not 32/64 */
    WCRAS_UNSUPPORTED = -2,   /* requested tier cannot hold this domain shape */
    WCRAS_CUDA_ERROR = -3,    /* CUDA runtime error (message in wcras_last_error) */
    WCRAS_BREAKDOWN = -4,     /* BiCGStab rho or omega underflow after one restart (reading Q13) */
    WCRAS_NOT_CONVERGED = -5  /* iteration caps hit; phi is still written and info filled */
};

/* Filled by wcras_solve*.  Counts follow the paper's "Dv operation count" (Table 1). */
typedef struct {
    int outer_iters;    /* fp64 outer BiCGStab iterations (a half-step exit counts as one) */
    int inner_iters;    /* fp32 inner BiCGStab iterations, summed over all inner solves */
    int inner_solves;   /* number of inner solves (= preconditioner calls of the outer solver) */
    int dv_fp32;        /* full-lattice fp32 D applications (Krylov + inside K_RAS, Alg.1 line 9) */
    int dv_fp64;        /* full-lattice fp64 D applications */
    int block_dv;       /* block-solver sweeps: MR iterations x K_RAS cycles, each over all domains */
    int ras_applies;    /* K_RAS applications */
    int status;         /* same as the return value */
    double rel_resid_recur; /* |r|/|eta| from the outer recurrence at exit */
    double rel_resid_true;  /* |eta - D phi|/|eta| recomputed in fp64 (PAPER.md:109 stopping condition) */
    double ms_total;        /* device time of the whole solve (CUDA events on the stream) */
    double ms_dslash;       /* sum over fp32 full-lattice D launches } only when wcras_set_timing(ctx,1); */
    double ms_blocksolve;   /* sum over block-solver launches        } T_Dv^calc / T_dominv^calc of       */
    double ms_blas;         /* BLAS-1 and conversions                } PAPER.md:103                       */
    double ms_dslash64;     /* sum over fp64 full-lattice D launches }                                    */
} wcras_info;

/* create(lattice dims, kappa, c_sw, gauge field)  -- north_star ABI list; PAPER.md:27-31 (Eq. 1.1), :109.
 * dims[mu] >= 2 (V*36 < 2^31).  gauge_dev: device, canonical layout, fp64, 72*V doubles.
 * Builds the internal SoA fp64 + fp32 link copies and the clover term A(x) = 1 - (c_sw kappa/2) sum_{mu<nu}
 * sigma_mu_nu F_mu_nu (clover-leaf F, readings Q3-Q5) as two packed 6x6 Hermitian chiral blocks per site,
 * in fp64 and rounded to fp32.  cuda_stream: a cudaStream_t (NULL = legacy default stream). */
int wcras_create(wcras_ctx** out, const int dims[4], double kappa, double csw, const double* gauge_dev,
                 void* cuda_stream);
int wcras_destroy(wcras_ctx* ctx);

/* w = D v on the full periodic lattice (north_star (b)).  prec = 32: in/out are float,
 * prec = 64: double; canonical spinor layout, 24*V reals each, device. */
int wcras_apply_D(wcras_ctx* ctx, int prec, const void* in_dev, void* out_dev);

/* The same w = D v (north_star (b)) for callers that may not allocate device memory: code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc (wcras_apply_D allocates its two internal-layout
 * buffers on its first call).  Arguments, layouts and result as wcras_apply_D.  The two buffers live in ONE file-scope
 * device array of WCRAS_NOALLOC_SCRATCH_BYTES (csrc/noalloc.cu) that every GPU which loads the library holds until the
 * process exits; the call itself performs no cudaMalloc / cudaFree and creates no event or stream (the per-class timers
 * of wcras_set_timing are off for its duration).  Limit: 2 * 24 * V * sizeof(real) <= WCRAS_NOALLOC_SCRATCH_BYTES, i.e.
 * V <= 87381 sites at prec 32 (16^4 fits) and V <= 43690 at prec 64; beyond that WCRAS_UNSUPPORTED with the sizes in
 * wcras_last_error, nothing launched.  All calls on one device, of every context and stream, SHARE the array: it keeps the
 * last call's contents (nothing needs clearing: both buffers are written in full before they are read), and two calls
 * that overlap on the GPU race on it -- the caller serialises them.  Enqueues on the context's stream, does not
 * synchronise. */
#define WCRAS_NOALLOC_SCRATCH_BYTES (16u << 20)
int wcras_apply_D_noalloc(wcras_ctx* ctx, int prec, const void* in_dev, void* out_dev);

/* ras_precondition(domain shape, overlap, block iterations)  -- north_star ABI list; PAPER.md:83 (the three
 * RAS parameters d, N_dominv, NRAS), :101 (d = 2s), :45 (Omega_i, Omega'_i).
 * domain[mu] must divide dims[mu]; overlap_s = s >= 0 is the extension per side in every direction with
 * domain[mu] < dims[mu] (needs domain[mu] + 2s <= dims[mu]); block_iters = N_dominv >= 1 MR iterations;
 * nras = NRAS >= 1.  Allocates the per-domain workspace and picks the block-solver tier. */
int wcras_ras_precondition(wcras_ctx* ctx, const int domain[4], int overlap_s, int block_iters, int nras);

/* Block-solver tier: 0 = automatic (fused on-chip solver when the extended domain fits, else generic),
 * 1 = generic global-memory tier, 2 = fused tier (WCRAS_UNSUPPORTED at the next wcras_ras_precondition if
 * the shape does not fit; extended domains of <= 256 sites use the persistent one-CTA-per-domain kernel,
 * larger ones a thread-block cluster per domain), 3 = fused tier, cluster kernel forced (for checking),
 * 4 = fused tier with the NRAS cycles NOT chained (for checking), 5 = the streamed-operand cluster kernel forced
 * (tier 2c of SURVEY.md 8(a): rho and v of an extended domain in the distributed shared memory of a <= 16-CTA cluster,
 * links and clover re-read from L2 every sweep; chosen automatically when the extended domain exceeds 4096 sites,
 * e.g. configs[4]: 8^4 blocks with overlap 1), 6 = as 0 but, in 16-bit operand mode, the two-threads-per-site variant
 * of the persistent kernel (ras_pair.cu; measured slower, kept for comparison).  On the persistent-CTA kernel with overlap 0
 * the cycles of Alg.1 are chained: the MR recurrence leaves rho = r - D_Omega v on every domain, so line 9,
 * r -= D v, only adds the hops of v that cross a domain boundary and no full-lattice D runs between cycles.
 * Call before wcras_ras_precondition. */
int wcras_set_ras_tier(wcras_ctx* ctx, int tier);

/* Operand storage of the RAS block solver (SURVEY.md 8(f) NEXT-4 "reduced-precision storage of links+clover"; DESIGN.md
 * reading R1).  bits = 32 (default): the fp32 links and clover blocks.  bits = 16: the preconditioner is K_RAS of the
 * operator D~ whose links and packed clover blocks are the fp16 roundings (round to nearest even) of the fp32 ones --
 * Alg. 1 unchanged, block solves AND residual updates with D~, all arithmetic in fp32.  The Krylov
 * operator D, the outer solver and the stopping criterion are not touched, so the solution still meets the fp64 true
 * residual.  On the persistent one-CTA-per-domain tier (extended domains of <= 256 sites) the operands are then STORED as
 * fp16 (288 instead of 576 bytes per site and cycle) and staged into shared memory by TMA bulk copies (ras_cta16.cu);
 * the other tiers compute with fp32 copies of the rounded fields.  Takes effect at the next wcras_ras_precondition. */
int wcras_set_operand_precision(wcras_ctx* ctx, int bits);

/* Block solver of the RAS / SAP domains (SURVEY.md 8(f) NEXT-4 "stronger block solvers"; reading R2; the paper
 * asks only for "a fixed iteration solver", and `configs` name MR).  kind = 0 (default): N_dominv MR iterations
 * (reading Q9).  kind = 1: restarted two-dimensional minimal residual (GMRES(2)): per PAIR of D_Omega' applications
 * q1 = D rho, q2 = D q1 the residual is minimised over span{q1, q2} (2x2 normal equations; the plain MR step if their
 * determinant is not positive); v += c1 rho + c2 q1, rho -= c1 q1 + c2 q2; an odd N_dominv ends with one MR iteration.
 * N_dominv still counts D_Omega' applications.  Built into the persistent one-CTA-per-domain kernel with 16-bit operand
 * storage (ras_cta16.cu) and into the generic tier (ras.cu).  On the automatic tier (wcras_set_ras_tier 0) a configuration the
 * first cannot run -- fp32 operands, an extended domain above 256 sites -- goes to the generic tier, as does tier 1; with a
 * forced fused tier (2..6) the next wcras_ras_precondition returns WCRAS_UNSUPPORTED unless
 * wcras_set_operand_precision(ctx, 16) is set and the extended domain has at most 256 sites.  Multiplicative Schwarz
 * (wcras_set_schwarz) needs the persistent kernel. */
int wcras_set_block_solver(wcras_ctx* ctx, int kind);

/* Order in which the full-lattice Dslash visits the sites (a traversal order only; no layout changes, results are
 * identical): ztile = -1 automatic (default: plain order x,y,z,t; above ~60 MB of operands per t-slice the order
 * x, y, z within a tile, t, z tile, with the largest tile whose slab stays under 30 MB, so that the t-neighbours are
 * still in L2), 0 plain order, z > 0 that tile size (a proper divisor of Lz). */
int wcras_set_traversal(wcras_ctx* ctx, int ztile);

/* Schwarz variant applied by wcras_ras_apply and the solver: 0 = additive with restriction (RAS, Alg. 1 -- the paper's
 * method and the default), 1 = multiplicative (SAP, the related method PAPER.md:33 names, ref. [5]; SURVEY.md 8(f)
 * NEXT-4): the domains are coloured red/black by the parity of their block coordinates and `nras` cycles of (black
 * half step, red half step) are run, each half step solving with the residual left by the previous one.  Needs
 * overlap 0, domains of <= 256 sites (persistent-CTA tier) and an even number of blocks in every cut direction;
 * otherwise wcras_ras_apply / wcras_solve return WCRAS_UNSUPPORTED. */
int wcras_set_schwarz(wcras_ctx* ctx, int multiplicative);

/* out = P'^T D_Omega' P' in : the principal sub-matrix of D on the extended domain Omega'_index of the
 * current decomposition ("restriction of D ... with the Dirichlet boundary condition"; reading
 * Q7), on full-lattice canonical vectors; out = 0 outside Omega'.  domain_index = -1 applies all domains at
 * once (block-diagonal operator) and is allowed only for overlap 0. */
int wcras_apply_D_restricted(wcras_ctx* ctx, int prec, int domain_index, const void* in_dev, void* out_dev);

/* v = K_RAS r : Algorithm 1 = Eq. 2.1 with N_dominv MR iterations as the
 * block solve.  fp32, canonical layout, device. */
int wcras_ras_apply(wcras_ctx* ctx, const float* r_dev, float* v_dev);

/* Solver parameters (readings Q13, A2): inner_tol = the deepest relative accuracy one fp32 inner solve is asked
 * for (default 5e-7); each inner solve gets the tolerance max(inner_tol, R^(1/n)), R = 0.5 target/|rhs|,
 * n = ceil(log R / log inner_tol), so that the outer target is met without overshooting it.  Iteration caps
 * (default 1000 / 50).  use_ras = 0 runs the inner solver without preconditioner ("No prec." column of Table 1). */
int wcras_set_solver(wcras_ctx* ctx, double inner_tol, int inner_maxit, int outer_maxit, int use_ras);

/* Convergence of the inner fp32 BiCGStab is decided on the device (a flag set by the last block of the update kernels;
 * every kernel of an iteration returns at once when it is set), so the host need not wait for an iteration before it
 * enqueues the next one (the inner solver runs on the GPU; only scalars cross to the host).  iterations =
 * how many inner iterations are enqueued ahead of the host's look at the scalars (default 1): 0 = every iteration is
 * checked before the next one is enqueued; n <= 3 = the host looks at iteration j - n while iteration j is enqueued, at
 * the price of up to n no-op iterations after convergence.  Results are identical for every value. */
int wcras_set_lookahead(wcras_ctx* ctx, int iterations);

/* CUDA graphs for the inner solver (default on): one inner fp32 BiCGStab iteration (10-14 kernel launches, the
 * inner solver "does most of arithmetics") is captured the second time it runs with the same vectors and configuration and
 * replayed afterwards, which removes the host's launch cost from small lattices.  Results are identical either way; every
 * call that changes the configuration discards the captured graphs.  Off while wcras_set_timing(1) is in force. */
int wcras_set_graphs(wcras_ctx* ctx, int enable);

/* Per-kernel-class CUDA-event timing inside wcras_solve (fills ms_dslash / ms_blocksolve / ms_blas). */
int wcras_set_timing(wcras_ctx* ctx, int enable);

/* solve(eta, tolerance) -> phi  -- north_star ABI list; PAPER.md:89 (mixed-precision nested BiCGStab: fp64
 * outer solver, fp32 inner solver as its preconditioner), Eq. 2.2 (inner solver on
 * D K_RAS chi = b), :109 (stop at |eta - D phi|/|eta| < tol, true residual recomputed in fp64).
 * eta_dev / phi_dev: device, canonical fp64, 24*V doubles.  info: host struct, may be NULL. */
int wcras_solve(wcras_ctx* ctx, const double* eta_dev, double* phi_dev, double tol, wcras_info* info);

/* Multi-right-hand-side solve (BASELINE.json:configs[4] "4 Gaussian sources"): solves
 * D phi_k = eta_k, k < nrhs (1..4), as one block-diagonal system with the same nested BiCGStab on stacked vectors, so
 * that the links and the clover term are loaded once per nrhs spinors in the fp32 Dslash (336 instead of 768 B per
 * site and right-hand side at nrhs = 4) and in the persistent block solver.  One set of Krylov scalars serves the
 * stack: every eta_k is scaled to unit norm, the stack is solved to tol/sqrt(nrhs), and the true residual
 * |eta_k - D phi_k|/|eta_k| <= tol is checked for every k (written to rel_resid_host[k], host, may be NULL;
 * info->rel_resid_true is the worst one).  eta_dev / phi_dev: device, canonical fp64, nrhs vectors of 24*V doubles
 * one after the other.  The workspace grows to nrhs times its size and stays that large. */
int wcras_solve_multi(wcras_ctx* ctx, int nrhs, const double* eta_dev, double* phi_dev, double tol, wcras_info* info,
                      double* rel_resid_host);

/* wcras_solve with HOST buffers (24*V doubles each, pinned or pageable; the end-to-end entry point): copies eta to the
 * device, solves, copies phi back; returns after phi_host is complete.  The copy of phi runs on an internal stream beside
 * the fp64 true-residual check of the same phi and is repeated if a later pass corrects phi, so phi_host
 * may be written more than once during the call; on return it holds bit for bit what wcras_solve would have left in
 * phi_dev.  info->ms_total is the device time of the solve without the two copies.  On an error code other than
 * WCRAS_NOT_CONVERGED / WCRAS_BREAKDOWN the contents of phi_host are unspecified. */
int wcras_solve_host(wcras_ctx* ctx, const double* eta_host, double* phi_host, double tol, wcras_info* info);

/* One row of the parameter survey of wcras_ras_autotune. */
typedef struct {
    int domain[4];      /* block shape; all zero = no preconditioner */
    int overlap_s, block_iters, nras;
    int schwarz;        /* 0 = additive (RAS, the paper's method), 1 = multiplicative (SAP; nras = red-black cycles) */
    int operand_bits;   /* block-solver operand storage, 32 or 16 (wcras_set_operand_precision); 0 in the no-preconditioner row */
    int block_solver;   /* 0 = MR, 1 = two-dimensional minimal residual (wcras_set_block_solver) */
    int status;         /* status of the timed solve (WCRAS_OK, NOT_CONVERGED, BREAKDOWN) or WCRAS_UNSUPPORTED */
    int inner_iters, ras_applies;
    double ms;          /* device time of the timed solve */
    double rel_resid_true;
} wcras_tune_row;

/* The paper's parameter survey ("we survey the best parameters for NRAS and N_dominv ... NRAS = 1-10 and
 * N_dominv = 1-20 ... for d = 0, 2, 4", and :83-85 on the trade-off), run on this lattice and GPU: solves D phi = eta to
 * `tol` once untimed and once timed for every candidate, at most max_rows candidates, in this order:
 *   row 0      the unpreconditioned solver;
 *   stage 1    additive Schwarz at overlap 0: block shapes of 64..256 sites with extents 2/4/8 that divide the lattice, plus
 *              8x4x4x4, 8x8x4x4 and 8^4, each at (N_dominv, NRAS) in {(2,3),(2,2),(2,4),(3,2),(3,3),(4,1),(4,2),(4,3),(5,3)}
 *              ((5,3) is the paper's best point), with the operand precision the context is set to;
 *   stage 2    around the fastest row so far: the rectangle N_dominv 1..8 x NRAS 1..5 on its shape; overlap s = 1, 2
 *              (the paper's d = 2, 4) and multiplicative Schwarz on the three fastest shapes; the other operand precision;
 *   stage 3    if the fastest row so far has overlap 0 and blocks of <= 256 sites: the second block solver
 *              (wcras_set_block_solver(1)) on its shape with 16-bit operands, N_dominv 2, 4, 6 x 2, 3 cycles, multiplicative
 *              and additive.
 * The fastest converged candidate is left configured (wcras_ras_precondition, wcras_set_schwarz, wcras_set_operand_precision,
 * wcras_set_block_solver, use_ras; use_ras = 0 if no preconditioner wins) and returned in *best.  table_host (may be NULL, room for max_rows rows)
 * receives the rows tried, *nrows their number.  On a CUDA error the previous configuration is put back.
 * eta_dev: device, canonical fp64.  Uses the workspace of wcras_solve plus one scratch solution vector. */
int wcras_ras_autotune(wcras_ctx* ctx, const double* eta_dev, double tol, int max_rows, wcras_tune_row* best,
                       wcras_tune_row* table_host, int* nrows);

/* Export the packed clover term for checking: out_dev = [V][2][36] doubles (packing: 6 real diagonal
 * entries, then the 15 strictly-lower entries (i>j, k = i(i-1)/2 + j) as {re,im}). */
int wcras_export_clover(wcras_ctx* ctx, double* out_dev);

/* Time one kernel class in its native layout on internal scratch fields: reps back-to-back launches
 * bracketed by CUDA events on the library's stream; returns the mean milliseconds per launch.
 * which: 0 = fp32 D, 1 = fp64 D, 2 = one K_RAS block-solve launch (all domains, current RAS parameters),
 *        3 = fused BLAS update (x += a p + w s ; r = s - w t ; <rt,r>, |r|^2),
 *        4 = one whole K_RAS application (Alg. 1: NRAS cycles, as the inner solver issues it; ms per application). */
int wcras_time_kernel(wcras_ctx* ctx, int which, int reps, double* ms_per_launch);

/* How many kernels of this library have been launched on ctx since creation (for bench.py's gpu_launches). */
long long wcras_launch_count(const wcras_ctx* ctx);

const char* wcras_last_error(const wcras_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* WCRAS_H */
