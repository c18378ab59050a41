// clover_build.cuh -- fp64 construction of the clover term (setup step A0, not on the timed path).
//
// Not in the paper (PAPER.md:107-109 gives only kappa and c_SW); formula from BASELINE.json:north_star,
// readings Q3-Q5 of DESIGN.md:
//   Q_mu_nu(x) = sum of the four plaquette leaves in the (mu,nu) plane that touch x, same orientation
//   F_mu_nu    = (Q - Q^dag) / (8 i)
//   A(x)       = 1 - (c_sw kappa / 2) sum_{mu<nu} sigma_mu_nu (x) F_mu_nu
// In the chiral basis sigma_mu_nu is block diagonal, so A = diag(A_+, A_-) with
//   A_pm = 1 - c [ sigma_1 (x) (+-F_xt - F_yz) + sigma_2 (x) (F_xz +- F_yt) + sigma_3 (x) (+-F_zt - F_xy) ]
// which is stored packed (see site_math.cuh).
#pragma once
#include "site_math.cuh"

namespace wc {

// c = a b (3x3 complex, 18 reals each); DA / DB: use the adjoint of a / b
template <bool DA, bool DB>
WC_HD void m3_mul(const double* __restrict__ a, const double* __restrict__ b, double* __restrict__ c) {
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            double re = 0, im = 0;
#pragma unroll
            for (int k = 0; k < 3; k++) {
                const int ia = DA ? (k * 3 + i) * 2 : (i * 3 + k) * 2;
                const int ib = DB ? (j * 3 + k) * 2 : (k * 3 + j) * 2;
                const double ar = a[ia], ai = DA ? -a[ia + 1] : a[ia + 1];
                const double br = b[ib], bi = DB ? -b[ib + 1] : b[ib + 1];
                re += ar * br - ai * bi;
                im += ar * bi + ai * br;
            }
            c[(i * 3 + j) * 2] = re;
            c[(i * 3 + j) * 2 + 1] = im;
        }
}

// q += m1 m2 m3 m4 with the adjoint pattern D1..D4
template <bool D1, bool D2, bool D3, bool D4>
WC_HD void leaf_add(const double* m1, const double* m2, const double* m3, const double* m4, double* q) {
    double t1[18], t2[18];
    m3_mul<D1, D2>(m1, m2, t1);
    m3_mul<false, D3>(t1, m3, t2);
    m3_mul<false, D4>(t2, m4, t1);
#pragma unroll
    for (int k = 0; k < 18; k++) q[k] += t1[k];
}

// f = (q - q^dag) / (8 i):  f_ij = -i (q_ij - conj(q_ji)) / 8
WC_HD void antiherm_to_F(const double* __restrict__ q, double* __restrict__ f) {
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            const double dr = q[(i * 3 + j) * 2] - q[(j * 3 + i) * 2];
            const double di = q[(i * 3 + j) * 2 + 1] + q[(j * 3 + i) * 2 + 1];
            f[(i * 3 + j) * 2] = di * 0.125;       // -i (dr + i di) = di - i dr
            f[(i * 3 + j) * 2 + 1] = -dr * 0.125;
        }
}

// F[p] for the six planes (0,1)(0,2)(0,3)(1,2)(1,3)(2,3) -> packed clover blocks, coefficient c
WC_HD void clover_assemble(const double F[6][18], double c, double* __restrict__ out) {
#pragma unroll
    for (int blk = 0; blk < 2; blk++) {
        const double sg = blk == 0 ? 1.0 : -1.0;
        double* o = out + 36 * blk;
#pragma unroll
        for (int i = 0; i < 6; i++)
#pragma unroll
            for (int j = 0; j <= i; j++) {
                const int a = i % 3, b = j % 3, e = (a * 3 + b) * 2;
                double mr, mi;
                if ((i < 3) == (j < 3)) {  // +-B3 = +-(sg F_zt - F_xy)
                    const double s3 = i < 3 ? 1.0 : -1.0;
                    mr = s3 * (sg * F[5][e] - F[0][e]);
                    mi = s3 * (sg * F[5][e + 1] - F[0][e + 1]);
                } else {  // i >= 3 > j: B1 + i B2, B1 = sg F_xt - F_yz, B2 = F_xz + sg F_yt
                    const double b1r = sg * F[2][e] - F[3][e], b1i = sg * F[2][e + 1] - F[3][e + 1];
                    const double b2r = F[1][e] + sg * F[4][e], b2i = F[1][e + 1] + sg * F[4][e + 1];
                    mr = b1r - b2i;
                    mi = b1i + b2r;
                }
                if (i == j) o[i] = 1.0 - c * mr;
                else {
                    const int k = 6 + 2 * (i * (i - 1) / 2 + j);
                    o[k] = -c * mr;
                    o[k + 1] = -c * mi;
                }
            }
    }
}

}  // namespace wc
