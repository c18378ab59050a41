/*
 * wcoracle.c -- the ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, fp64 CPU statement of what the hot path of arXiv:1011.3318
 * (Osaki & Ishikawa, "Domain Decomposition method on GPU cluster") computes.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call it.  It shares no code, header, table or
 * helper with the CUDA path under paper_1011_3318_b200/csrc/.
 *
 * Style: naive loops over site, direction, spin, colour with the full 4x4
 * gamma matrices (no half-spinor projection, no chiral-block shortcut for the
 * clover term, no blocking, no fusion).  The only parallelism is an OpenMP
 * "parallel for" over sites (or over domains in the RAS block loop).
 *
 * Citations are PAPER.md:<line> (section / equation / algorithm) or
 * BASELINE.json:north_star where the paper gives no formula; the readings
 * Q1..Q20 are those listed in DESIGN.md ("Readings of the paper").
 *
 * Pins (tests/test_oracle_*.py, "-m 'not gpu'"): gamma algebra, free-field
 * plane-wave spectrum, F=0 at U=1, F_xy = sin(phi) on a constant abelian
 * field, the clover matrix of that field in closed form, gamma5-hermiticity,
 * gauge covariance, dense-matrix LU on 2^4, D_Omega' == dense sub-matrix,
 * MR orthogonality/monotonicity/convergence to the dense block inverse,
 * Alg.1 == Eq.(2.1) with dense exact block inverses, single-domain RAS ==
 * D^-1, Neumann-polynomial reduction, partition of unity.
 * Parity unpinned: only the *reading* Q5 (factor 1/2 in the clover
 * coefficient, taken literally from north_star) -- the implementation of the
 * literal formula is pinned by the closed-form clover matrix test.
 *
 * Stronger block solver (reading R2):
 * wco_mr2_block = restarted two-dimensional minimal residual (GMRES(2)): per
 * pair of D applications the residual is minimised over span{rho, D rho}.
 * wco_set_block_solver(1) makes wco_ras_apply / wco_sap_apply / the solvers use
 * it in place of MR.  Pins (tests/test_oracle_mr2.py): dense least squares on a
 * 2^4 box, exact solution in one cycle for a free-field plane wave (minimal
 * polynomial of degree 2), never worse than two MR steps.
 *
 * Reduced-precision operand storage (DESIGN.md reading
 * R1): the same algorithms applied to an operator whose links and site-diagonal
 * matrices A(x) were rounded entry by entry (fp64 -> fp32 -> fp16, round to
 * nearest even).  wco_clover_matrix writes A(x) out as a dense 12x12 matrix,
 * wco_round_half rounds, wco_set_explicit_clover makes every routine below use
 * the given A(x) instead of forming it from F.  Pins: the explicit path with
 * unrounded A reproduces the formula path; A(x) against the test's Kronecker
 * construction; the rounding against numpy's IEEE binary16 and closed-form ties.
 *
 * Layouts (row-major C arrays of double complex):
 *   site index i = x + Lx*(y + Ly*(z + Lz*t)); mu = 0..3 = x,y,z,t
 *   U   [V][4][3][3]   (U psi)_a = sum_b U[a][b] psi_b
 *   psi [V][4][3]      spin, colour
 *   F   [V][6][3][3]   planes (mu,nu) in the order (0,1)(0,2)(0,3)(1,2)(1,3)(2,3)
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

/* ------------------------------------------------------------------ */
/* gamma matrices: Hermitian chiral basis (reading Q2; paper is silent) */
/* ------------------------------------------------------------------ */
static const cplx GAMMA[4][4][4] = {
    /* gamma_x */ {{0, 0, 0, -I}, {0, 0, -I, 0}, {0, I, 0, 0}, {I, 0, 0, 0}},
    /* gamma_y */ {{0, 0, 0, -1}, {0, 0, 1, 0}, {0, 1, 0, 0}, {-1, 0, 0, 0}},
    /* gamma_z */ {{0, 0, -I, 0}, {0, 0, 0, I}, {I, 0, 0, 0}, {0, -I, 0, 0}},
    /* gamma_t */ {{0, 0, 1, 0}, {0, 0, 0, 1}, {1, 0, 0, 0}, {0, 1, 0, 0}},
};

/* out = gamma_mu for mu = 0..3, gamma_5 = gamma_x gamma_y gamma_z gamma_t for mu = 4 */
void wco_gamma(int mu, cplx out[16]) {
    if (mu < 4) {
        for (int a = 0; a < 4; a++)
            for (int b = 0; b < 4; b++) out[4 * a + b] = GAMMA[mu][a][b];
        return;
    }
    cplx p[4][4], q[4][4];
    for (int a = 0; a < 4; a++)
        for (int b = 0; b < 4; b++) p[a][b] = GAMMA[0][a][b];
    for (int m = 1; m < 4; m++) {
        for (int a = 0; a < 4; a++)
            for (int b = 0; b < 4; b++) {
                q[a][b] = 0;
                for (int c = 0; c < 4; c++) q[a][b] += p[a][c] * GAMMA[m][c][b];
            }
        memcpy(p, q, sizeof p);
    }
    for (int a = 0; a < 4; a++)
        for (int b = 0; b < 4; b++) out[4 * a + b] = p[a][b];
}

/* sigma_mu_nu = (i/2) [gamma_mu, gamma_nu]   (reading Q3) */
void wco_sigma(int mu, int nu, cplx out[16]) {
    for (int a = 0; a < 4; a++)
        for (int b = 0; b < 4; b++) {
            cplx s = 0;
            for (int c = 0; c < 4; c++)
                s += GAMMA[mu][a][c] * GAMMA[nu][c][b] - GAMMA[nu][a][c] * GAMMA[mu][c][b];
            out[4 * a + b] = 0.5 * I * s;
        }
}

/* The clover coefficient of BASELINE.json:north_star, taken literally (reading Q5):
 *   A(x) = 1 - (c_sw * kappa / 2) * sum_{mu<nu} sigma_mu_nu F_mu_nu(x).            */
static double clover_coeff(double kappa, double csw) { return csw * kappa / 2.0; }

/* ------------------------------------------------------------------ */
/* lattice geometry                                                    */
/* ------------------------------------------------------------------ */
static long volume(const int L[4]) { return (long)L[0] * L[1] * L[2] * L[3]; }

static long site_index(const int L[4], const int x[4]) {
    return x[0] + (long)L[0] * (x[1] + (long)L[1] * (x[2] + (long)L[2] * x[3]));
}

static void site_coords(const int L[4], long i, int x[4]) {
    x[0] = (int)(i % L[0]); i /= L[0];
    x[1] = (int)(i % L[1]); i /= L[1];
    x[2] = (int)(i % L[2]); i /= L[2];
    x[3] = (int)i;
}

/* y = x + d*mu_hat with periodic wrap (reading Q6: periodic in all four directions) */
static void shifted(const int L[4], const int x[4], int mu, int d, int y[4]) {
    for (int k = 0; k < 4; k++) y[k] = x[k];
    y[mu] = ((x[mu] + d) % L[mu] + L[mu]) % L[mu];
}

/* ------------------------------------------------------------------ */
/* 3x3 helpers                                                         */
/* ------------------------------------------------------------------ */
static void mat_mul(const cplx* a, const cplx* b, cplx* c) { /* c = a b */
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            cplx s = 0;
            for (int k = 0; k < 3; k++) s += a[3 * i + k] * b[3 * k + j];
            c[3 * i + j] = s;
        }
}
static void mat_dag(const cplx* a, cplx* c) { /* c = a^dagger */
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) c[3 * i + j] = conj(a[3 * j + i]);
}
/* q += m1 m2 m3 m4, each factor optionally daggered */
static void add_leaf(cplx* q, const cplx* m1, int d1, const cplx* m2, int d2, const cplx* m3, int d3,
                     const cplx* m4, int d4) {
    cplx f[4][9], t1[9], t2[9], t3[9];
    const cplx* m[4] = {m1, m2, m3, m4};
    int d[4] = {d1, d2, d3, d4};
    for (int k = 0; k < 4; k++) {
        if (d[k]) mat_dag(m[k], f[k]);
        else memcpy(f[k], m[k], sizeof t1);
    }
    mat_mul(f[0], f[1], t1);
    mat_mul(t1, f[2], t2);
    mat_mul(t2, f[3], t3);
    for (int k = 0; k < 9; k++) q[k] += t3[k];
}

/* ------------------------------------------------------------------ */
/* field strength  (reading Q4; the paper never writes the clover term) */
/*   Q_mu_nu(x) = sum of the four plaquette leaves in the (mu,nu) plane  */
/*   touching x, all traversed in the same orientation;                 */
/*   F_mu_nu = (Q - Q^dagger) / (8 i)  (Hermitian, trace not removed)   */
/* ------------------------------------------------------------------ */
static const int PLANE[6][2] = {{0, 1}, {0, 2}, {0, 3}, {1, 2}, {1, 3}, {2, 3}};

#define LINK(U, site, mu) ((U) + ((site) * 4 + (mu)) * 9)

void wco_field_strength(const int L[4], const cplx* U, cplx* F) {
    long V = volume(L);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < V; i++) {
        int x[4];
        site_coords(L, i, x);
        for (int p = 0; p < 6; p++) {
            int mu = PLANE[p][0], nu = PLANE[p][1];
            int xpm[4], xpn[4], xmm[4], xmn[4], xmmpn[4], xmmmn[4], xpmmn[4];
            shifted(L, x, mu, +1, xpm);
            shifted(L, x, nu, +1, xpn);
            shifted(L, x, mu, -1, xmm);
            shifted(L, x, nu, -1, xmn);
            shifted(L, xmm, nu, +1, xmmpn);
            shifted(L, xmm, nu, -1, xmmmn);
            shifted(L, xpm, nu, -1, xpmmn);
            long s = i, spm = site_index(L, xpm), spn = site_index(L, xpn), smm = site_index(L, xmm),
                 smn = site_index(L, xmn), smmpn = site_index(L, xmmpn), smmmn = site_index(L, xmmmn),
                 spmmn = site_index(L, xpmmn);
            cplx q[9] = {0}, qd[9];
            /* U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag */
            add_leaf(q, LINK(U, s, mu), 0, LINK(U, spm, nu), 0, LINK(U, spn, mu), 1, LINK(U, s, nu), 1);
            /* U_nu(x) U_mu(x-mu+nu)^dag U_nu(x-mu)^dag U_mu(x-mu) */
            add_leaf(q, LINK(U, s, nu), 0, LINK(U, smmpn, mu), 1, LINK(U, smm, nu), 1, LINK(U, smm, mu), 0);
            /* U_mu(x-mu)^dag U_nu(x-mu-nu)^dag U_mu(x-mu-nu) U_nu(x-nu) */
            add_leaf(q, LINK(U, smm, mu), 1, LINK(U, smmmn, nu), 1, LINK(U, smmmn, mu), 0, LINK(U, smn, nu), 0);
            /* U_nu(x-nu)^dag U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^dag */
            add_leaf(q, LINK(U, smn, nu), 1, LINK(U, smn, mu), 0, LINK(U, spmmn, nu), 0, LINK(U, s, mu), 1);
            mat_dag(q, qd);
            cplx* f = F + (i * 6 + p) * 9;
            for (int k = 0; k < 9; k++) f[k] = (q[k] - qd[k]) / (8.0 * I);
        }
    }
}

/* ------------------------------------------------------------------ */
/* the operator at one site                                            */
/*                                                                     */
/* (D psi)(x) = A(x) psi(x)                                            */
/*    - kappa sum_mu [ (1-gamma_mu) U_mu(x) psi(x+mu)                  */
/*                   + (1+gamma_mu) U_mu(x-mu)^dag psi(x-mu) ]         */
/* A(x) = 1 - (c_sw kappa/2) sum_{mu<nu} sigma_mu_nu (x) F_mu_nu(x)    */
/*                                                                     */
/* BASELINE.json:north_star (reading Q1); the paper only names D:      */
/* PAPER.md:27-31 (Sec.1, Eq. 1.1), :107-109 (Sec.5: kappa, c_SW).     */
/*                                                                     */
/* psi_fwd[mu] / psi_bwd[mu] point at psi(x+mu) / psi(x-mu), or are    */
/* NULL when that hop is dropped (Dirichlet boundary of a restricted   */
/* operator).  link_bwd[mu] = U_mu(x-mu).                 */
/* ------------------------------------------------------------------ */
/* Explicit site-diagonal matrices A(x), [V][12][12] with row/column index spin*3+colour, or NULL.
 * When set (reduced-precision operand variant, reading R1) A(x) psi(x) is the plain
 * matrix-vector product with the stored matrix and F, c_sw are not used. */
static const cplx* g_Aexp = NULL;
void wco_set_explicit_clover(const cplx* A) { g_Aexp = A; }
#define AEXP(site) (g_Aexp ? g_Aexp + (site) * 144 : NULL)

static void site_D(const cplx* link_fwd[4], const cplx* link_bwd[4], const cplx* Fx, const cplx* Ax, double kappa,
                   double csw, const cplx* psi_x, const cplx* psi_fwd[4], const cplx* psi_bwd[4],
                   cplx out[12]) {
    /* site-diagonal clover term A(x) psi(x) */
    double c = clover_coeff(kappa, csw);
    if (Ax) {
        for (int i = 0; i < 12; i++) {
            cplx s = 0;
            for (int j = 0; j < 12; j++) s += Ax[12 * i + j] * psi_x[j];
            out[i] = s;
        }
        c = 0.0;
    } else {
        for (int al = 0; al < 4; al++)
            for (int a = 0; a < 3; a++) out[3 * al + a] = psi_x[3 * al + a];
    }
    if (c != 0.0) {
        for (int p = 0; p < 6; p++) {
            cplx sig[16], fpsi[12];
            wco_sigma(PLANE[p][0], PLANE[p][1], sig);
            const cplx* f = Fx + p * 9;
            for (int be = 0; be < 4; be++)
                for (int a = 0; a < 3; a++) {
                    cplx s = 0;
                    for (int b = 0; b < 3; b++) s += f[3 * a + b] * psi_x[3 * be + b];
                    fpsi[3 * be + a] = s;
                }
            for (int al = 0; al < 4; al++)
                for (int a = 0; a < 3; a++) {
                    cplx s = 0;
                    for (int be = 0; be < 4; be++) s += sig[4 * al + be] * fpsi[3 * be + a];
                    out[3 * al + a] -= c * s;
                }
        }
    }
    /* hopping term */
    for (int mu = 0; mu < 4; mu++) {
        if (psi_fwd[mu]) {
            const cplx* u = link_fwd[mu];
            const cplx* ps = psi_fwd[mu];
            for (int al = 0; al < 4; al++)
                for (int a = 0; a < 3; a++) {
                    cplx s = 0;
                    for (int be = 0; be < 4; be++) {
                        cplx proj = (al == be ? 1.0 : 0.0) - GAMMA[mu][al][be]; /* (1 - gamma_mu) */
                        for (int b = 0; b < 3; b++) s += proj * u[3 * a + b] * ps[3 * be + b];
                    }
                    out[3 * al + a] -= kappa * s;
                }
        }
        if (psi_bwd[mu]) {
            const cplx* u = link_bwd[mu];
            const cplx* ps = psi_bwd[mu];
            for (int al = 0; al < 4; al++)
                for (int a = 0; a < 3; a++) {
                    cplx s = 0;
                    for (int be = 0; be < 4; be++) {
                        cplx proj = (al == be ? 1.0 : 0.0) + GAMMA[mu][al][be]; /* (1 + gamma_mu) */
                        for (int b = 0; b < 3; b++) s += proj * conj(u[3 * b + a]) * ps[3 * be + b];
                    }
                    out[3 * al + a] -= kappa * s;
                }
        }
    }
}

/* Is global site y inside the box Omega' = {start + c (mod L), 0 <= c_mu < ext_mu} ?  If so return
 * its local lexicographic index (x fastest), else -1.  ext_mu <= L_mu.                              */
static long box_local_index(const int L[4], const int start[4], const int ext[4], const int y[4]) {
    long idx = 0, stride = 1;
    for (int mu = 0; mu < 4; mu++) {
        int c = ((y[mu] - start[mu]) % L[mu] + L[mu]) % L[mu];
        if (c >= ext[mu]) return -1;
        idx += stride * c;
        stride *= ext[mu];
    }
    return idx;
}

/* w = D v on the full periodic lattice.  PAPER.md:31 ("w = Dv"). */
void wco_apply_D(const int L[4], const cplx* U, const cplx* F, double kappa, double csw, const cplx* in,
                 cplx* out) {
    long V = volume(L);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < V; i++) {
        int x[4], y[4];
        site_coords(L, i, x);
        const cplx *lf[4], *lb[4], *pf[4], *pb[4];
        for (int mu = 0; mu < 4; mu++) {
            shifted(L, x, mu, +1, y);
            pf[mu] = in + site_index(L, y) * 12;
            lf[mu] = LINK(U, i, mu);
            shifted(L, x, mu, -1, y);
            long j = site_index(L, y);
            pb[mu] = in + j * 12;
            lb[mu] = LINK(U, j, mu);
        }
        site_D(lf, lb, F + i * 54, AEXP(i), kappa, csw, in + i * 12, pf, pb, out + i * 12);
    }
}

/* out = P'^T D_Omega' P' in, on full-lattice vectors: D_Omega' is the principal sub-matrix of D on
 * the site set Omega' (box start/ext): a hop x -> x +- mu (mod L) contributes only if the neighbour
 * is in Omega'; A(x) unchanged; out = 0 outside Omega'.
 * PAPER.md:47 ("restriction of D to Omega_i with the Dirichlet boundary condition"), :68 (Alg.1
 * line 5); readings Q7 (sub-matrix reading: wrap-around hops that stay inside Omega' are kept). */
void wco_apply_D_box(const int L[4], const cplx* U, const cplx* F, double kappa, double csw,
                     const int start[4], const int ext[4], const cplx* in, cplx* out) {
    long V = volume(L);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < V; i++) {
        int x[4], y[4];
        site_coords(L, i, x);
        if (box_local_index(L, start, ext, x) < 0) {
            for (int k = 0; k < 12; k++) out[i * 12 + k] = 0;
            continue;
        }
        const cplx *lf[4], *lb[4], *pf[4], *pb[4];
        for (int mu = 0; mu < 4; mu++) {
            shifted(L, x, mu, +1, y);
            pf[mu] = box_local_index(L, start, ext, y) >= 0 ? in + site_index(L, y) * 12 : NULL;
            lf[mu] = LINK(U, i, mu);
            shifted(L, x, mu, -1, y);
            long j = site_index(L, y);
            pb[mu] = box_local_index(L, start, ext, y) >= 0 ? in + j * 12 : NULL;
            lb[mu] = LINK(U, j, mu);
        }
        site_D(lf, lb, F + i * 54, AEXP(i), kappa, csw, in + i * 12, pf, pb, out + i * 12);
    }
}

/* ------------------------------------------------------------------ */
/* domain decomposition  (readings Q3(domains), Q8) */
/*   blocks of shape b tile the lattice, domain index lexicographic     */
/*   with x fastest; Omega'_i = block enlarged by s sites on both sides */
/*   in every direction with b_mu < L_mu ("split" directions).          */
/* returns 0 on success, -1 if b does not divide L or b+2s > L.         */
/* ------------------------------------------------------------------ */
int wco_domain_count(const int L[4], const int b[4]) {
    int n = 1;
    for (int mu = 0; mu < 4; mu++) {
        if (b[mu] < 1 || L[mu] % b[mu]) return -1;
        n *= L[mu] / b[mu];
    }
    return n;
}

int wco_domain_box(const int L[4], const int b[4], int s, int idx, int origin[4], int start[4],
                   int ext[4]) {
    if (wco_domain_count(L, b) < 0 || s < 0) return -1;
    for (int mu = 0; mu < 4; mu++) {
        int nb = L[mu] / b[mu];
        origin[mu] = (idx % nb) * b[mu];
        idx /= nb;
        if (b[mu] < L[mu]) {
            if (b[mu] + 2 * s > L[mu]) return -1;
            start[mu] = ((origin[mu] - s) % L[mu] + L[mu]) % L[mu];
            ext[mu] = b[mu] + 2 * s;
        } else {
            start[mu] = 0;
            ext[mu] = L[mu];
        }
    }
    return 0;
}

/* ------------------------------------------------------------------ */
/* vectors: <a,b> = sum_k conj(a_k) b_k  (reading Q15)                 */
/* ------------------------------------------------------------------ */
static cplx vdot(long n, const cplx* a, const cplx* b) {
    double re = 0, im = 0;
#pragma omp parallel for reduction(+ : re, im) schedule(static)
    for (long k = 0; k < n; k++) {
        cplx t = conj(a[k]) * b[k];
        re += creal(t);
        im += cimag(t);
    }
    return re + I * im;
}
static double vnorm(long n, const cplx* a) { return sqrt(creal(vdot(n, a, a))); }

cplx wco_dot(long n, const cplx* a, const cplx* b) { return vdot(n, a, b); }

/* ------------------------------------------------------------------ */
/* block solve: N_dominv iterations of MR on D_Omega' v = r_Omega'      */
/* from v = 0   (PAPER.md:68 Alg.1 line 5; :83 "a fixed iteration      */
/* solver with the iteration number N_dominv"; the solver is named MR  */
/* only by BASELINE.json:configs -> reading Q9: plain MR, relaxation 1,*/
/* zero initial guess, exactly N_dominv iterations, alpha := 0 when    */
/* <q,q> = 0).                                                         */
/*   rho = r;  repeat: q = D_Omega' rho; alpha = <q,rho>/<q,q>;        */
/*                     v += alpha rho; rho -= alpha q                  */
/* Vectors are local to the box: local index lexicographic in the box  */
/* coordinates c (x fastest), global site = (start + c) mod L.         */
/* r_full is the full-lattice residual; the gather is the projection   */
/* P_Omega' of Alg.1 line 4.                             */
/* ------------------------------------------------------------------ */
static long box_volume(const int ext[4]) { return (long)ext[0] * ext[1] * ext[2] * ext[3]; }

static void box_global_coords(const int L[4], const int start[4], const int ext[4], long k, int x[4]) {
    for (int mu = 0; mu < 4; mu++) {
        int c = (int)(k % ext[mu]);
        k /= ext[mu];
        x[mu] = (start[mu] + c) % L[mu];
    }
}

/* q_local = D_Omega' rho_local */
static void box_apply_D_local(const int L[4], const cplx* U, const cplx* F, double kappa, double csw,
                              const int start[4], const int ext[4], const cplx* in, cplx* out) {
    long n = box_volume(ext);
    for (long k = 0; k < n; k++) {
        int x[4], y[4];
        box_global_coords(L, start, ext, k, x);
        long i = site_index(L, x);
        const cplx *lf[4], *lb[4], *pf[4], *pb[4];
        for (int mu = 0; mu < 4; mu++) {
            shifted(L, x, mu, +1, y);
            long kk = box_local_index(L, start, ext, y);
            pf[mu] = kk >= 0 ? in + kk * 12 : NULL;
            lf[mu] = LINK(U, i, mu);
            shifted(L, x, mu, -1, y);
            kk = box_local_index(L, start, ext, y);
            pb[mu] = kk >= 0 ? in + kk * 12 : NULL;
            lb[mu] = LINK(U, site_index(L, y), mu);
        }
        site_D(lf, lb, F + i * 54, AEXP(i), kappa, csw, in + k * 12, pf, pb, out + k * 12);
    }
}

static cplx sdot(long n, const cplx* a, const cplx* b) { /* serial <a,b> */
    cplx s = 0;
    for (long k = 0; k < n; k++) s += conj(a[k]) * b[k];
    return s;
}

/* v_local (box_volume*12) = MR_niter(D_Omega', P_Omega' r_full); rho_local (optional) = final residual */
void wco_mr_block(const int L[4], const cplx* U, const cplx* F, double kappa, double csw,
                  const int start[4], const int ext[4], int niter, const cplx* r_full, cplx* v_local,
                  cplx* rho_out) {
    long n = box_volume(ext), n12 = n * 12;
    cplx* rho = malloc(sizeof(cplx) * n12);
    cplx* q = malloc(sizeof(cplx) * n12);
    for (long k = 0; k < n; k++) { /* projection P_Omega' */
        int x[4];
        box_global_coords(L, start, ext, k, x);
        long i = site_index(L, x);
        for (int c = 0; c < 12; c++) rho[k * 12 + c] = r_full[i * 12 + c];
    }
    for (long k = 0; k < n12; k++) v_local[k] = 0;
    for (int it = 0; it < niter; it++) {
        box_apply_D_local(L, U, F, kappa, csw, start, ext, rho, q);
        cplx qr = sdot(n12, q, rho);
        double qq = creal(sdot(n12, q, q));
        cplx alpha = qq > 0 ? qr / qq : 0;
        for (long k = 0; k < n12; k++) v_local[k] += alpha * rho[k];
        for (long k = 0; k < n12; k++) rho[k] -= alpha * q[k];
    }
    if (rho_out) memcpy(rho_out, rho, sizeof(cplx) * n12);
    free(rho);
    free(q);
}

/* ------------------------------------------------------------------ */
/* Stronger block solver (SURVEY.md 8(f) NEXT-4 "stronger block        */
/* solvers"; reading R2; the paper only asks for "a fixed    */
/* iteration solver"): restarted two-dimensional minimal  */
/* residual = GMRES(2).  niter still counts D applications.            */
/*   v = 0, rho = P r                                                  */
/*   for every pair of D applications:                                 */
/*     q1 = D rho ; q2 = D q1                                          */
/*     (c1, c2) = argmin | rho - c1 q1 - c2 q2 | :                     */
/*        a11 c1 + a12 c2 = b1 ; conj(a12) c1 + a22 c2 = b2,           */
/*        a_ij = <q_i, q_j>, b_i = <q_i, rho>                          */
/*        g = (a12/a11)(conj(a12)/a22) (cos^2 of the angle of q1, q2;  */
/*        1 if a11 or a22 is 0).  If 1 - g <= 1e-4 (q2 numerically par. */
/*        to q1, or rho = 0): the plain MR step c1 = b1 / a11 (0 if    */
/*        a11 = 0), c2 = 0.  Otherwise, with the rows divided by a11   */
/*        and a22 (no product of two squared norms: a tiny rho must    */
/*        not underflow), u_i = b_i / a_ii, m1 = a12 / a11,            */
/*        m2 = conj(a12) / a22: c1 = (u1 - m1 u2) / (1 - g),           */
/*        c2 = (u2 - m2 u1) / (1 - g)                                  */
/*     v += c1 rho + c2 q1 ; rho -= c1 q1 + c2 q2                      */
/*   odd niter: one plain MR iteration at the end                      */
/* ------------------------------------------------------------------ */
#define WCO_MR2_DELTA 1e-4
void wco_mr2_block(const int L[4], const cplx* U, const cplx* F, double kappa, double csw,
                   const int start[4], const int ext[4], int niter, const cplx* r_full, cplx* v_local,
                   cplx* rho_out) {
    long n = box_volume(ext), n12 = n * 12;
    cplx* rho = malloc(sizeof(cplx) * n12);
    cplx* q1 = malloc(sizeof(cplx) * n12);
    cplx* q2 = malloc(sizeof(cplx) * n12);
    for (long k = 0; k < n; k++) { /* projection P_Omega' */
        int x[4];
        box_global_coords(L, start, ext, k, x);
        long i = site_index(L, x);
        for (int c = 0; c < 12; c++) rho[k * 12 + c] = r_full[i * 12 + c];
    }
    for (long k = 0; k < n12; k++) v_local[k] = 0;
    int it = 0;
    for (; it + 1 < niter; it += 2) {
        box_apply_D_local(L, U, F, kappa, csw, start, ext, rho, q1);
        box_apply_D_local(L, U, F, kappa, csw, start, ext, q1, q2);
        double a11 = creal(sdot(n12, q1, q1)), a22 = creal(sdot(n12, q2, q2));
        cplx a12 = sdot(n12, q1, q2), b1 = sdot(n12, q1, rho), b2 = sdot(n12, q2, rho);
        /* scale-free form of the 2x2 solve: rows divided by a11 and a22; g = cos^2 of the angle between q1 and q2 */
        double g = (a11 > 0 && a22 > 0) ? creal((a12 / a11) * (conj(a12) / a22)) : 1.0; /* no product a11 a22: it may underflow */
        cplx c1, c2;
        if (1.0 - g > WCO_MR2_DELTA) {
            cplx u1 = b1 / a11, u2 = b2 / a22, m1 = a12 / a11, m2 = conj(a12) / a22;
            c1 = (u1 - m1 * u2) / (1.0 - g);
            c2 = (u2 - m2 * u1) / (1.0 - g);
        } else {
            c1 = a11 > 0 ? b1 / a11 : 0;
            c2 = 0;
        }
        for (long k = 0; k < n12; k++) v_local[k] += c1 * rho[k] + c2 * q1[k];
        for (long k = 0; k < n12; k++) rho[k] -= c1 * q1[k] + c2 * q2[k];
    }
    if (it < niter) { /* odd count: a last MR iteration */
        box_apply_D_local(L, U, F, kappa, csw, start, ext, rho, q1);
        cplx qr = sdot(n12, q1, rho);
        double qq = creal(sdot(n12, q1, q1));
        cplx alpha = qq > 0 ? qr / qq : 0;
        for (long k = 0; k < n12; k++) v_local[k] += alpha * rho[k];
        for (long k = 0; k < n12; k++) rho[k] -= alpha * q1[k];
    }
    if (rho_out) memcpy(rho_out, rho, sizeof(cplx) * n12);
    free(rho);
    free(q1);
    free(q2);
}

/* which block solver Alg. 1, SAP and the solvers use: 0 = MR (the configs' "MR block iterations"), 1 = wco_mr2_block */
static int g_block_solver = 0;
void wco_set_block_solver(int kind) { g_block_solver = kind; }
static void block_solve(const int L[4], const cplx* U, const cplx* F, double kappa, double csw, const int start[4],
                        const int ext[4], int niter, const cplx* r_full, cplx* v_local) {
    if (g_block_solver == 1) wco_mr2_block(L, U, F, kappa, csw, start, ext, niter, r_full, v_local, NULL);
    else wco_mr_block(L, U, F, kappa, csw, start, ext, niter, r_full, v_local, NULL);
}

/* ------------------------------------------------------------------ */
/* RAS iteration, Algorithm 1 (line numbering as read  */
/* in Q11).  phi = K_RAS eta.                                          */
/*  1: phi = 0, r = eta                                                */
/*  2: for j = 0..NRAS-1                                               */
/*  3:   for every domain i                                            */
/*  4:     r_Omega'i = P_Omega'i r                                     */
/*  5:     solve D_Omega'i v_Omega'i = r_Omega'i  (N_dominv MR its)    */
/*  6:     v_Omegai = R_Omegai v_Omega'i   (keep bulk sites only)      */
/*  8:   v = sum_i v_Omegai                                            */
/*  9:   phi += v ; r -= D v   (the last r update is dead, reading Q12)*/
/* returns 0, or -1 for an invalid decomposition.                      */
/* ------------------------------------------------------------------ */
int wco_ras_apply(const int L[4], const cplx* U, const cplx* F, double kappa, double csw, const int b[4],
                  int s, int niter, int nras, const cplx* eta, cplx* phi) {
    int nd = wco_domain_count(L, b);
    if (nd < 0 || nras < 1) return -1;
    {
        int o[4], st[4], ex[4];
        if (wco_domain_box(L, b, s, 0, o, st, ex)) return -1;
    }
    long V = volume(L), n12 = V * 12;
    cplx* r = malloc(sizeof(cplx) * n12);
    cplx* v = malloc(sizeof(cplx) * n12);
    cplx* dv = malloc(sizeof(cplx) * n12);
    memcpy(r, eta, sizeof(cplx) * n12);
    for (long k = 0; k < n12; k++) phi[k] = 0;
    for (int j = 0; j < nras; j++) {
        for (long k = 0; k < n12; k++) v[k] = 0;
#pragma omp parallel for schedule(dynamic)
        for (int i = 0; i < nd; i++) {
            int origin[4], start[4], ext[4];
            wco_domain_box(L, b, s, i, origin, start, ext);
            long n = box_volume(ext);
            cplx* vl = malloc(sizeof(cplx) * n * 12);
            block_solve(L, U, F, kappa, csw, start, ext, niter, r, vl);
            for (long k = 0; k < n; k++) { /* restriction R_Omega_i: bulk sites only */
                int x[4], bulk = 1;
                box_global_coords(L, start, ext, k, x);
                for (int mu = 0; mu < 4; mu++) {
                    int c = ((x[mu] - origin[mu]) % L[mu] + L[mu]) % L[mu];
                    if (c >= b[mu]) bulk = 0;
                }
                if (!bulk) continue;
                long g = site_index(L, x);
                for (int c = 0; c < 12; c++) v[g * 12 + c] += vl[k * 12 + c]; /* disjoint sum, line 8 */
            }
            free(vl);
        }
        for (long k = 0; k < n12; k++) phi[k] += v[k];
        if (j < nras - 1) {
            wco_apply_D(L, U, F, kappa, csw, v, dv);
            for (long k = 0; k < n12; k++) r[k] -= dv[k];
        }
    }
    free(r);
    free(v);
    free(dv);
    return 0;
}

/* ------------------------------------------------------------------ */
/* Multiplicative Schwarz (SAP, Luescher; named as the related method  */
/* in PAPER.md:33, ref [5]), overlap 0.         */
/* Domains are coloured by the parity of the sum of their block        */
/* coordinates; the number of blocks must be even in every direction   */
/* that is cut, so that neighbouring domains have opposite colours.    */
/*  phi = 0, r = eta                                                   */
/*  for cycle = 0..ncycle-1, for colour = 0, 1:                        */
/*     for every domain i of that colour: v_Omegai = MR_niter(P_i r)   */
/*     v = sum_i v_Omegai ; phi += v ; r -= D v                        */
/*  (the last r update is dead and skipped, as in reading Q12)         */
/* returns 0, -1 for an invalid decomposition, -2 if it cannot be      */
/* two-coloured.                                                       */
/* ------------------------------------------------------------------ */
int wco_sap_apply(const int L[4], const cplx* U, const cplx* F, double kappa, double csw, const int b[4],
                  int niter, int ncycle, const cplx* eta, cplx* phi) {
    int nd = wco_domain_count(L, b);
    if (nd < 0 || ncycle < 1) return -1;
    int nblk[4], cut = 0;
    for (int mu = 0; mu < 4; mu++) {
        nblk[mu] = L[mu] / b[mu];
        if (nblk[mu] > 1) { cut = 1; if (nblk[mu] % 2) return -2; }
    }
    if (!cut) return -2;
    long V = volume(L), n12 = V * 12;
    cplx* r = malloc(sizeof(cplx) * n12);
    cplx* v = malloc(sizeof(cplx) * n12);
    cplx* dv = malloc(sizeof(cplx) * n12);
    memcpy(r, eta, sizeof(cplx) * n12);
    for (long k = 0; k < n12; k++) phi[k] = 0;
    for (int cyc = 0; cyc < ncycle; cyc++) {
        for (int colour = 0; colour < 2; colour++) {
            for (long k = 0; k < n12; k++) v[k] = 0;
#pragma omp parallel for schedule(dynamic)
            for (int i = 0; i < nd; i++) {
                int bc = i, par = 0;
                for (int mu = 0; mu < 4; mu++) { par += bc % nblk[mu]; bc /= nblk[mu]; }
                if ((par & 1) != colour) continue;
                int origin[4], start[4], ext[4];
                wco_domain_box(L, b, 0, i, origin, start, ext);
                long n = box_volume(ext);
                cplx* vl = malloc(sizeof(cplx) * n * 12);
                block_solve(L, U, F, kappa, csw, start, ext, niter, r, vl);
                for (long k = 0; k < n; k++) {
                    int x[4];
                    box_global_coords(L, start, ext, k, x);
                    long g = site_index(L, x);
                    for (int c = 0; c < 12; c++) v[g * 12 + c] = vl[k * 12 + c];
                }
                free(vl);
            }
            for (long k = 0; k < n12; k++) phi[k] += v[k];
            if (!(cyc == ncycle - 1 && colour == 1)) {
                wco_apply_D(L, U, F, kappa, csw, v, dv);
                for (long k = 0; k < n12; k++) r[k] -= dv[k];
            }
        }
    }
    free(r);
    free(v);
    free(dv);
    return 0;
}

/* ------------------------------------------------------------------ */
/* BiCGStab, right-preconditioned: solves D K chi = b, x = K chi       */
/* (PAPER.md:54-57 Eq. 2.2; :49 "We employ BiCGStab"; the recurrences  */
/* are the textbook ones, written out in DESIGN.md reading Q13):       */
/*   x=0, r=b, rt=r, rho=alpha=omega=1, v=p=0; loop:                   */
/*   rho'=<rt,r>; beta=(rho'/rho)(alpha/omega); p=r+beta(p-omega v);   */
/*   ph=K p; v=D ph; alpha=rho'/<rt,v>; s=r-alpha v; sh=K s; t=D sh;   */
/*   omega=<t,s>/<t,t>; x+=alpha ph+omega sh; r=s-omega t; rho=rho';   */
/*   stop when |r|/|b| < tol; also stop after the first half step when */
/*   |s|/|b| < tol (x += alpha ph), as in van der Vorst's statement.   */
/* K = identity, K_RAS (Alg.1), or (nested scheme) an inner BiCGStab.  */
/* Breakdown (reading Q13): |rho'| or |omega| below tiny -> one restart*/
/* with rt = r, a second one returns status -2.                        */
/* ------------------------------------------------------------------ */
typedef struct {
    const int* L;
    const cplx* U;
    const cplx* F;
    double kappa, csw;
    int use_ras, b[4], s, niter, nras;
    /* nested: inner solve as the preconditioner */
    int nested;
    double inner_tol;
    int inner_maxit;
    /* counters */
    long dv, ras_applies, inner_iters;
} wco_op;

static int bicgstab_core(wco_op* op, int level, const cplx* b, cplx* x, double tol, int maxit, int* iters,
                         double* relres);

static void apply_K(wco_op* op, int level, const cplx* in, cplx* out) {
    long n12 = volume(op->L) * 12;
    if (level == 1 && op->nested) {
        /* nested scheme: K(y) = |y| * inner BiCGStab(y/|y|, inner_tol)  (reading Q13) */
        double ny = vnorm(n12, in);
        if (ny == 0) {
            for (long k = 0; k < n12; k++) out[k] = 0;
            return;
        }
        cplx* y = malloc(sizeof(cplx) * n12);
        for (long k = 0; k < n12; k++) y[k] = in[k] / ny;
        int it;
        double rr;
        bicgstab_core(op, 0, y, out, op->inner_tol, op->inner_maxit, &it, &rr);
        op->inner_iters += it;
        for (long k = 0; k < n12; k++) out[k] *= ny;
        free(y);
        return;
    }
    if (op->use_ras) {
        wco_ras_apply(op->L, op->U, op->F, op->kappa, op->csw, op->b, op->s, op->niter, op->nras, in, out);
        op->ras_applies++;
        op->dv += op->nras - 1;
        return;
    }
    memcpy(out, in, sizeof(cplx) * n12);
}

static int bicgstab_core(wco_op* op, int level, const cplx* b, cplx* x, double tol, int maxit, int* iters,
                         double* relres) {
    long n12 = volume(op->L) * 12;
    const double tiny = 1e-300;
    cplx *r = malloc(sizeof(cplx) * n12), *rt = malloc(sizeof(cplx) * n12), *p = calloc(n12, sizeof(cplx)),
         *v = calloc(n12, sizeof(cplx)), *ph = malloc(sizeof(cplx) * n12), *s = malloc(sizeof(cplx) * n12),
         *sh = malloc(sizeof(cplx) * n12), *t = malloc(sizeof(cplx) * n12);
    for (long k = 0; k < n12; k++) x[k] = 0;
    memcpy(r, b, sizeof(cplx) * n12);
    memcpy(rt, r, sizeof(cplx) * n12);
    double bnorm = vnorm(n12, b);
    cplx rho = 1, alpha = 1, omega = 1;
    int it = 0, status = -1, restarts = 0;
    double rn = bnorm;
    if (bnorm == 0) { status = 0; rn = 0; bnorm = 1; }
    while (status != 0 && it < maxit) {
        cplx rho1 = vdot(n12, rt, r);
        if (cabs(rho1) < tiny || cabs(omega) < tiny) {
            if (restarts++) { status = -2; break; }
            memcpy(rt, r, sizeof(cplx) * n12);
            for (long k = 0; k < n12; k++) p[k] = v[k] = 0;
            rho = alpha = omega = 1;
            continue;
        }
        cplx beta = (rho1 / rho) * (alpha / omega);
        for (long k = 0; k < n12; k++) p[k] = r[k] + beta * (p[k] - omega * v[k]);
        apply_K(op, level, p, ph);
        wco_apply_D(op->L, op->U, op->F, op->kappa, op->csw, ph, v);
        op->dv++;
        alpha = rho1 / vdot(n12, rt, v);
        for (long k = 0; k < n12; k++) s[k] = r[k] - alpha * v[k];
        if (vnorm(n12, s) / bnorm < tol) { /* half-step exit: x += alpha ph, r = s (reading Q13) */
            for (long k = 0; k < n12; k++) x[k] += alpha * ph[k];
            memcpy(r, s, sizeof(cplx) * n12);
            it++;
            rn = vnorm(n12, r);
            status = 0;
            break;
        }
        apply_K(op, level, s, sh);
        wco_apply_D(op->L, op->U, op->F, op->kappa, op->csw, sh, t);
        op->dv++;
        double tt = creal(vdot(n12, t, t));
        omega = tt > 0 ? vdot(n12, t, s) / tt : 0;
        for (long k = 0; k < n12; k++) x[k] += alpha * ph[k] + omega * sh[k];
        for (long k = 0; k < n12; k++) r[k] = s[k] - omega * t[k];
        rho = rho1;
        it++;
        rn = vnorm(n12, r);
        if (rn / bnorm < tol) status = 0;
    }
    *iters = it;
    *relres = rn / bnorm;
    free(r); free(rt); free(p); free(v); free(ph); free(s); free(sh); free(t);
    return status;
}

/* Flat fp64 BiCGStab with K = identity (use_ras = 0) or K = K_RAS.  This is the timed CPU baseline.
 * counts[0] = iterations, counts[1] = full-lattice Dv count, counts[2] = K_RAS applications.
 * resid[0] = recurrence |r|/|eta|, resid[1] = true |eta - D x|/|eta|.  returns 0 / -1 (not converged)
 * / -2 (breakdown). */
int wco_bicgstab(const int L[4], const cplx* U, const cplx* F, double kappa, double csw, int use_ras,
                 const int b[4], int s, int niter, int nras, const cplx* eta, cplx* x, double tol, int maxit,
                 long counts[3], double resid[2]) {
    wco_op op = {L, U, F, kappa, csw, use_ras, {0, 0, 0, 0}, s, niter, nras, 0, 0, 0, 0, 0, 0};
    if (use_ras)
        for (int mu = 0; mu < 4; mu++) op.b[mu] = b[mu];
    int it;
    double rr;
    int st = bicgstab_core(&op, 0, eta, x, tol, maxit, &it, &rr);
    long n12 = volume(L) * 12;
    cplx* w = malloc(sizeof(cplx) * n12);
    wco_apply_D(L, U, F, kappa, csw, x, w);
    for (long k = 0; k < n12; k++) w[k] = eta[k] - w[k];
    double en = vnorm(n12, eta);
    counts[0] = it; counts[1] = op.dv; counts[2] = op.ras_applies;
    resid[0] = rr; resid[1] = en > 0 ? vnorm(n12, w) / en : 0;
    free(w);
    return st;
}

/* Nested ("flexible") BiCGStab, all in fp64 here: the oracle is the reference, not a
 * model of rounding (reading Q13).  Outer = bicgstab_core with K = inner solve;
 * on apparent convergence the true residual r = eta - D x is recomputed; accepted if <= tol, else the
 * outer solver is restarted on that r (x accumulates).
 * counts[0] = outer iterations, [1] = inner iterations, [2] = Dv count, [3] = K_RAS applications. */
int wco_nested_bicgstab(const int L[4], const cplx* U, const cplx* F, double kappa, double csw, int use_ras,
                        const int b[4], int s, int niter, int nras, const cplx* eta, cplx* x, double tol,
                        double inner_tol, int inner_maxit, int outer_maxit, long counts[4], double resid[2]) {
    wco_op op = {L, U, F, kappa, csw, use_ras, {0, 0, 0, 0}, s, niter, nras, 1, inner_tol, inner_maxit, 0, 0, 0};
    if (use_ras)
        for (int mu = 0; mu < 4; mu++) op.b[mu] = b[mu];
    long n12 = volume(L) * 12;
    cplx *r = malloc(sizeof(cplx) * n12), *dx = malloc(sizeof(cplx) * n12), *w = malloc(sizeof(cplx) * n12);
    for (long k = 0; k < n12; k++) x[k] = 0;
    memcpy(r, eta, sizeof(cplx) * n12);
    double en = vnorm(n12, eta), rn = en, rr = 1;
    int outer = 0, status = -1;
    if (en == 0) { status = 0; en = 1; }
    for (int pass = 0; pass < 10 && status != 0 && outer < outer_maxit; pass++) {
        int it;
        /* solve D dx = r to relative tol*|eta|/|r| so that the total residual meets tol */
        int st = bicgstab_core(&op, 1, r, dx, tol * en / rn, outer_maxit - outer, &it, &rr);
        outer += it;
        for (long k = 0; k < n12; k++) x[k] += dx[k];
        wco_apply_D(L, U, F, kappa, csw, x, w);
        op.dv++;
        for (long k = 0; k < n12; k++) r[k] = eta[k] - w[k];
        rn = vnorm(n12, r);
        if (rn / en <= tol) status = 0;
        else if (st == -2) { status = -2; break; }
    }
    counts[0] = outer; counts[1] = op.inner_iters; counts[2] = op.dv; counts[3] = op.ras_applies;
    resid[0] = rr; resid[1] = rn / en;
    free(r); free(dx); free(w);
    return status;
}

/* |eta - D phi| / |eta| in fp64: the final check used for grading (BASELINE.json:north_star;
 * PAPER.md:109 stopping condition). */
double wco_true_residual(const int L[4], const cplx* U, const cplx* F, double kappa, double csw,
                         const cplx* eta, const cplx* phi) {
    long n12 = volume(L) * 12;
    cplx* w = malloc(sizeof(cplx) * n12);
    wco_apply_D(L, U, F, kappa, csw, phi, w);
    for (long k = 0; k < n12; k++) w[k] = eta[k] - w[k];
    double rn = vnorm(n12, w), en = vnorm(n12, eta);
    free(w);
    return en > 0 ? rn / en : rn;
}

/* (D psi)(x) at a list of sites only -- same site routine as wco_apply_D; used to check sampled
 * outputs at sizes where a full oracle pass is too slow. */
void wco_apply_D_sites(const int L[4], const cplx* U, const cplx* F, double kappa, double csw, const cplx* in,
                       long nsites, const long* sites, cplx* out) {
#pragma omp parallel for schedule(static)
    for (long n = 0; n < nsites; n++) {
        long i = sites[n];
        int x[4], y[4];
        site_coords(L, i, x);
        const cplx *lf[4], *lb[4], *pf[4], *pb[4];
        for (int mu = 0; mu < 4; mu++) {
            shifted(L, x, mu, +1, y);
            pf[mu] = in + site_index(L, y) * 12;
            lf[mu] = LINK(U, i, mu);
            shifted(L, x, mu, -1, y);
            long j = site_index(L, y);
            pb[mu] = in + j * 12;
            lb[mu] = LINK(U, j, mu);
        }
        site_D(lf, lb, F + i * 54, AEXP(i), kappa, csw, in + i * 12, pf, pb, out + n * 12);
    }
}

/* ------------------------------------------------------------------ */
/* Reduced-precision operand variant (reading R1) */
/* ------------------------------------------------------------------ */
/* A(x) = 1 - (c_sw kappa/2) sum_{mu<nu} sigma_mu_nu (x) F_mu_nu(x) written out as a dense 12x12 matrix
 * per site, index spin*3+colour (BASELINE.json:north_star formula, reading Q5): A[V][12][12]. */
void wco_clover_matrix(const int L[4], const cplx* F, double kappa, double csw, cplx* A) {
    long V = volume(L);
    double c = clover_coeff(kappa, csw);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < V; i++) {
        cplx* a = A + i * 144;
        for (int k = 0; k < 144; k++) a[k] = 0;
        for (int k = 0; k < 12; k++) a[13 * k] = 1;
        for (int p = 0; p < 6; p++) {
            cplx sig[16];
            wco_sigma(PLANE[p][0], PLANE[p][1], sig);
            const cplx* f = F + (i * 6 + p) * 9;
            for (int al = 0; al < 4; al++)
                for (int be = 0; be < 4; be++)
                    for (int ca = 0; ca < 3; ca++)
                        for (int cb = 0; cb < 3; cb++)
                            a[12 * (3 * al + ca) + 3 * be + cb] -= c * sig[4 * al + be] * f[3 * ca + cb];
        }
    }
}

/* One real number rounded to IEEE binary16 (11-bit significand, exponents -14..15, gradual underflow),
 * round to nearest, ties to even, after a first rounding to binary32 (the CUDA path's reduced-precision
 * operands are roundings of its fp32 fields, reading Q16).  x = m 2^e with 0.5 <= m < 1 lies in the
 * binade whose spacing is 2^(e-11), or 2^-24 below the smallest normal; rint() rounds to nearest even in
 * the default rounding mode.  Values beyond the largest finite half (65504) do not occur (|U_ab| <= 1,
 * A(x) = 1 + small) and are returned as +-infinity. */
static double round_half_1(double x) {
    x = (double)(float)x;
    if (x == 0.0 || isnan(x) || isinf(x)) return x;
    int e;
    frexp(fabs(x), &e);
    int eq = e - 11;
    if (eq < -24) eq = -24;
    double q = ldexp(1.0, eq);
    double y = rint(x / q) * q;
    if (fabs(y) > 65504.0) y = copysign(INFINITY, x);
    return y;
}
/* out[k] = real and imaginary parts of in[k] rounded separately */
void wco_round_half(long n, const cplx* in, cplx* out) {
#pragma omp parallel for schedule(static)
    for (long k = 0; k < n; k++) out[k] = round_half_1(creal(in[k])) + I * round_half_1(cimag(in[k]));
}

int wco_num_threads(void) {
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp single
        n = omp_get_num_threads();
    }
#endif
    return n;
}
