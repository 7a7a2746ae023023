/*
 * blip_oracle.c — CPU fp64 ORACLE for the blip (periodic tricubic B-spline) orbital
 * evaluation of arxiv/paper_1204_1121 (Uejima & Maezono).
 *
 * THIS FILE IS TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, link or call it.  It
 * shares no code, header, table or helper with the CUDA path under
 * paper_1204_1121_b200/csrc/ and neither side includes the other.
 *
 * What it computes (Eq. 6-8): for every position r_j and orbital l
 *
 *      psi_l(r_j) = sum_{s=1..64} a_{l,s(r_j)} * Theta_s(r_j)                    (Eq. 6)
 *      Theta_s(r) = phi((x-X_s)/b_x) phi((y-Y_s)/b_y) phi((z-Z_s)/b_z)           (Eq. 7)
 *
 * with s(r_j) the 4x4x4 block of grid sites around r_j picked out of the whole periodic
 * grid (Eq. 8), plus the Cartesian gradient and Laplacian of psi_l (north_star; the paper
 * implies them through the local-energy call).  The steps below are the
 * paper's, in the paper's order: (1) locate the block s(r_j); (2) evaluate the 1-D basis
 * factors phi; (3) the 64-term multiply-add; (4) [not in paper] map the derivatives taken
 * in grid coordinates to Cartesian ones with the inverse lattice.  Plain loops, fp64,
 * no blocking or fusion.  Readings of the paper:
 *   R1 phi is the CUBIC cardinal B-spline (4-point support <=> degree 3; PAPER.md:98 says
 *      "second order" but 4 sites per axis);
 *   R2 normalisation sum_m phi = 1 (B(0) = 2/3, B(+-1) = 1/6);
 *   R3 the 4 sites along axis a are i_a-1 .. i_a+2 with i_a = floor(t_a);
 *   R4 coefficient c[k] sits at grid point k, no storage offset, periodic in k;
 *   R5 table order [k1][k2][k3][l], l innermost ("l ... sequential");
 *   R6 general lattice A (rows = lattice vectors), fractional u = r.A^-1, t_a = n_a u_a;
 *   R9 any finite r is wrapped into the cell by u - floor(u).
 *
 * Pins (tests/test_oracle_*.py, all "-m not gpu"): brute-force sum over ALL grid sites
 * (oracle/blip_brute.py, separate code: no cell search, no weight polynomials), partition
 * of unity, linear / quadratic / cubic closed forms, knot values 8/27, 2/27, 1/54, 1/216,
 * discrete cosine eigenfunction, lattice periodicity, central finite differences of oracle
 * VALUES for gradient and Laplacian (orthorhombic and triclinic), continuity across cell
 * faces, separable case against scipy.interpolate.BSpline, adversarial cell-index inputs.
 * blip_oracle_eval_hess (full Cartesian Hessian, added in round 2) has its own pins, listed at
 * the function.  No function here is "parity unpinned".
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -fPIC -shared (oracle/build.py).  The
 * -ffp-contract=off matters only for the index map (step 1), whose IEEE sequence is pinned
 * so that the GPU can reproduce the integer cell indices bit for bit.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define BLIP_ORACLE_VALUE 0
#define BLIP_ORACLE_VGL   1

/* ---------------------------------------------------------------------------------------
 * Inverse lattice G = A^-1 (so that u = r.G for a row vector r), by cofactors.
 * Pinned IEEE sequence: every cofactor is p*q - r*s, the
 * determinant is (A00*C00 + A01*C01) + A02*C02, and G[i][j] = C[j][i] / det (a true
 * division, no reciprocal-multiply).  Returns 0 on success, -1 if det is 0 or not finite.
 * ------------------------------------------------------------------------------------- */
int blip_oracle_inverse_lattice(const double A[9], double G[9])
{
    double C[9];
    C[0] = A[4] * A[8] - A[5] * A[7];
    C[1] = A[5] * A[6] - A[3] * A[8];
    C[2] = A[3] * A[7] - A[4] * A[6];
    C[3] = A[2] * A[7] - A[1] * A[8];
    C[4] = A[0] * A[8] - A[2] * A[6];
    C[5] = A[1] * A[6] - A[0] * A[7];
    C[6] = A[1] * A[5] - A[2] * A[4];
    C[7] = A[2] * A[3] - A[0] * A[5];
    C[8] = A[0] * A[4] - A[1] * A[3];
    double det = (A[0] * C[0] + A[1] * C[1]) + A[2] * C[2];
    if (!(det != 0.0) || !isfinite(det)) return -1;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
            G[3 * i + j] = C[3 * j + i] / det;
    return 0;
}

/* ---------------------------------------------------------------------------------------
 * Step 1 — which block of sites: s(r_j) of Eq. 8 (Fig. 1).
 * For one position r: fractional u_a = (x*G[0][a] + y*G[1][a]) + z*G[2][a]; wrap
 * u_a <- u_a - floor(u_a); grid coordinate t_a = u_a * n_a; i_a = floor(t_a); if the
 * wrap rounded up to the cell edge (i_a >= n_a) fold it back (i_a -= n_a, t_a -= n_a);
 * f_a = t_a - i_a in [0,1).  Returns 0, or -1 for a non-finite position (cell = -1).
 * ------------------------------------------------------------------------------------- */
static int cell_of(const double G[9], const int n[3], const double r[3], int i[3], double f[3])
{
    for (int a = 0; a < 3; ++a) {
        double u = (r[0] * G[0 + a] + r[1] * G[3 + a]) + r[2] * G[6 + a];
        if (!isfinite(u)) { i[0] = i[1] = i[2] = -1; f[0] = f[1] = f[2] = NAN; return -1; }
        u = u - floor(u);
        double t = u * (double)n[a];
        int ia = (int)floor(t);
        if (ia >= n[a]) { ia -= n[a]; t -= (double)n[a]; }
        i[a] = ia;
        f[a] = t - (double)ia;
    }
    return 0;
}

int blip_oracle_cellmap(const double A[9], const int n[3], const double *pos, long long M,
                        int *cell /* [M][3] */, double *frac /* [M][3] or NULL */)
{
    double G[9];
    if (blip_oracle_inverse_lattice(A, G)) return -1;
    for (long long e = 0; e < M; ++e) {
        int i[3]; double f[3];
        cell_of(G, n, pos + 3 * e, i, f);
        for (int a = 0; a < 3; ++a) {
            cell[3 * e + a] = i[a];
            if (frac) frac[3 * e + a] = f[a];
        }
    }
    return 0;
}

/* ---------------------------------------------------------------------------------------
 * Step 2 — the 1-D basis factor phi of Eq. 7 at the 4 sites i-1, i, i+1, i+2, as a
 * function of the offset f = t - i in [0,1): the uniform cubic B-spline pieces
 * [not printed in the paper; textbook, reading R1/R2], and their first and second
 * derivatives with respect to the grid coordinate t.
 * ------------------------------------------------------------------------------------- */
static void phi_weights(double f, double w[4], double d1[4], double d2[4])
{
    double g = 1.0 - f;
    w[0] = g * g * g / 6.0;
    w[1] = (3.0 * f * f * f - 6.0 * f * f + 4.0) / 6.0;
    w[2] = (-3.0 * f * f * f + 3.0 * f * f + 3.0 * f + 1.0) / 6.0;
    w[3] = f * f * f / 6.0;
    d1[0] = -g * g / 2.0;
    d1[1] = (3.0 * f * f - 4.0 * f) / 2.0;
    d1[2] = (-3.0 * f * f + 2.0 * f + 1.0) / 2.0;
    d1[3] = f * f / 2.0;
    d2[0] = g;
    d2[1] = 3.0 * f - 2.0;
    d2[2] = 1.0 - 3.0 * f;
    d2[3] = f;
}

/* ---------------------------------------------------------------------------------------
 * The evaluation: steps 1-4 for M positions and all L orbitals.
 *   A      [9]            lattice, row-major, row a = lattice vector a
 *   n      [3]            grid points per axis (each >= 4)
 *   L                     number of real orbitals
 *   c      [n1][n2][n3][L] fp32 coefficients (widened exactly to fp64 here)
 *   pos    [M][3]         Cartesian positions
 *   mode                  0 value only, 1 value + gradient + Laplacian
 *   val    [M][L]         fp64 out
 *   grad   [M][3][L]      fp64 out (mode 1), Cartesian components x,y,z
 *   lap    [M][L]         fp64 out (mode 1)
 *   cell   [M][3]         int out, optional (NULL ok)
 * Returns 0; -1 bad lattice; -2 bad arguments; -3 out of memory.
 * ------------------------------------------------------------------------------------- */
int blip_oracle_eval(const double A[9], const int n[3], int L, const float *c,
                     const double *pos, long long M, int mode,
                     double *val, double *grad, double *lap, int *cell)
{
    if (L < 1 || M < 0 || n[0] < 4 || n[1] < 4 || n[2] < 4 || !c || !val) return -2;
    if (mode != BLIP_ORACLE_VALUE && mode != BLIP_ORACLE_VGL) return -2;
    if (mode == BLIP_ORACLE_VGL && (!grad || !lap)) return -2;
    double G[9];
    if (blip_oracle_inverse_lattice(A, G)) return -1;

    /* Step 4 constants: t_a = n_a * sum_i r_i G[i][a]  =>  J[a][i] = dt_a/dr_i = n_a G[i][a];
     * Q = J J^T so that the Cartesian Laplacian is sum_ab Q[a][b] d2S/dt_a dt_b. */
    double J[3][3], Q[3][3];
    for (int a = 0; a < 3; ++a)
        for (int i = 0; i < 3; ++i)
            J[a][i] = (double)n[a] * G[3 * i + a];
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b)
            Q[a][b] = J[a][0] * J[b][0] + J[a][1] * J[b][1] + J[a][2] * J[b][2];

    int failed = 0;
#pragma omp parallel
    {
        /* per-thread accumulators in grid coordinates: S, dS/dt_a (3), d2S/dt_a dt_b (6) */
        double *acc = (double *)malloc(sizeof(double) * 10 * (size_t)L);
        if (!acc) {
#pragma omp atomic write
            failed = 1;
        }
#pragma omp for schedule(dynamic, 16)
        for (long long e = 0; e < M; ++e) {
            if (!acc) continue;
            int i[3]; double f[3];
            int bad = cell_of(G, n, pos + 3 * e, i, f);
            if (cell) { cell[3 * e] = i[0]; cell[3 * e + 1] = i[1]; cell[3 * e + 2] = i[2]; }
            if (bad) {
                for (int l = 0; l < L; ++l) {
                    val[e * L + l] = NAN;
                    if (mode == BLIP_ORACLE_VGL) {
                        grad[(e * 3 + 0) * L + l] = NAN;
                        grad[(e * 3 + 1) * L + l] = NAN;
                        grad[(e * 3 + 2) * L + l] = NAN;
                        lap[e * L + l] = NAN;
                    }
                }
                continue;
            }
            double w[3][4], d1[3][4], d2[3][4];
            for (int a = 0; a < 3; ++a) phi_weights(f[a], w[a], d1[a], d2[a]);

            double *S = acc, *T0 = acc + L, *T1 = acc + 2 * L, *T2 = acc + 3 * L;
            double *H00 = acc + 4 * L, *H11 = acc + 5 * L, *H22 = acc + 6 * L;
            double *H01 = acc + 7 * L, *H02 = acc + 8 * L, *H12 = acc + 9 * L;
            memset(acc, 0, sizeof(double) * 10 * (size_t)L);

            /* Step 3 — Eq. 6: the 64-term multiply-add over s = (m0,m1,m2). */
            for (int m0 = 0; m0 < 4; ++m0) {
                int k0 = ((i[0] - 1 + m0) % n[0] + n[0]) % n[0];
                for (int m1 = 0; m1 < 4; ++m1) {
                    int k1 = ((i[1] - 1 + m1) % n[1] + n[1]) % n[1];
                    for (int m2 = 0; m2 < 4; ++m2) {
                        int k2 = ((i[2] - 1 + m2) % n[2] + n[2]) % n[2];
                        const float *row = c + (((size_t)k0 * n[1] + k1) * n[2] + k2) * (size_t)L;
                        double th = w[0][m0] * w[1][m1] * w[2][m2]; /* Theta_s(r), Eq. 7 */
                        if (mode == BLIP_ORACLE_VALUE) {
                            for (int l = 0; l < L; ++l) S[l] += th * (double)row[l];
                        } else {
                            double t0 = d1[0][m0] * w[1][m1] * w[2][m2];
                            double t1 = w[0][m0] * d1[1][m1] * w[2][m2];
                            double t2 = w[0][m0] * w[1][m1] * d1[2][m2];
                            double h00 = d2[0][m0] * w[1][m1] * w[2][m2];
                            double h11 = w[0][m0] * d2[1][m1] * w[2][m2];
                            double h22 = w[0][m0] * w[1][m1] * d2[2][m2];
                            double h01 = d1[0][m0] * d1[1][m1] * w[2][m2];
                            double h02 = d1[0][m0] * w[1][m1] * d1[2][m2];
                            double h12 = w[0][m0] * d1[1][m1] * d1[2][m2];
                            for (int l = 0; l < L; ++l) {
                                double a = (double)row[l];
                                S[l] += th * a;
                                T0[l] += t0 * a; T1[l] += t1 * a; T2[l] += t2 * a;
                                H00[l] += h00 * a; H11[l] += h11 * a; H22[l] += h22 * a;
                                H01[l] += h01 * a; H02[l] += h02 * a; H12[l] += h12 * a;
                            }
                        }
                    }
                }
            }
            /* Step 4 — to Cartesian: grad_i = sum_a J[a][i] dS/dt_a,
             * lap = sum_ab Q[a][b] d2S/dt_a dt_b. */
            for (int l = 0; l < L; ++l) {
                val[e * L + l] = S[l];
                if (mode == BLIP_ORACLE_VGL) {
                    for (int x = 0; x < 3; ++x)
                        grad[(e * 3 + x) * L + l] =
                            J[0][x] * T0[l] + J[1][x] * T1[l] + J[2][x] * T2[l];
                    lap[e * L + l] = Q[0][0] * H00[l] + Q[1][1] * H11[l] + Q[2][2] * H22[l]
                                   + 2.0 * (Q[0][1] * H01[l] + Q[0][2] * H02[l] + Q[1][2] * H12[l]);
                }
            }
        }
        free(acc);
    }
    return failed ? -3 : 0;
}

/* ---------------------------------------------------------------------------------------
 * Value, Cartesian gradient and the full Cartesian HESSIAN (the paper's
 * local-energy call needs second derivatives).  Same steps 1-3 as
 * blip_oracle_eval — the 64-term sum of Eq. 6 for S, dS/dt_a and d2S/dt_a dt_b in grid
 * coordinates — and in step 4 the chain rule for second derivatives of a function of
 * t(r) = J r (J constant, so no first-derivative term appears):
 *      Hc[i][j] = d2S/dr_i dr_j = sum_ab J[a][i] Ht[a][b] J[b][j]
 *   hess   [M][6][L]  fp64 out, components in the order xx, yy, zz, xy, xz, yz
 * Returns as blip_oracle_eval.  Pins (tests/test_oracle_pins.py): trace = the Laplacian of
 * blip_oracle_eval; bilinear / quadratic tables (Hc = J_a^T J_b + J_b^T J_a); central
 * differences of oracle GRADIENTS; the brute-force definition (oracle/blip_brute.py).
 * ------------------------------------------------------------------------------------- */
int blip_oracle_eval_hess(const double A[9], const int n[3], int L, const float *c,
                          const double *pos, long long M,
                          double *val, double *grad, double *hess, int *cell)
{
    if (L < 1 || M < 0 || n[0] < 4 || n[1] < 4 || n[2] < 4 || !c || !val || !grad || !hess) return -2;
    double G[9];
    if (blip_oracle_inverse_lattice(A, G)) return -1;
    double J[3][3];
    for (int a = 0; a < 3; ++a)
        for (int i = 0; i < 3; ++i)
            J[a][i] = (double)n[a] * G[3 * i + a];
    static const int ci[6] = {0, 1, 2, 0, 0, 1}, cj[6] = {0, 1, 2, 1, 2, 2};   /* xx yy zz xy xz yz */

    int failed = 0;
#pragma omp parallel
    {
        double *acc = (double *)malloc(sizeof(double) * 10 * (size_t)L);
        if (!acc) {
#pragma omp atomic write
            failed = 1;
        }
#pragma omp for schedule(dynamic, 16)
        for (long long e = 0; e < M; ++e) {
            if (!acc) continue;
            int i[3]; double f[3];
            int bad = cell_of(G, n, pos + 3 * e, i, f);
            if (cell) { cell[3 * e] = i[0]; cell[3 * e + 1] = i[1]; cell[3 * e + 2] = i[2]; }
            if (bad) {
                for (int l = 0; l < L; ++l) {
                    val[e * L + l] = NAN;
                    for (int x = 0; x < 3; ++x) grad[(e * 3 + x) * L + l] = NAN;
                    for (int q = 0; q < 6; ++q) hess[(e * 6 + q) * L + l] = NAN;
                }
                continue;
            }
            double w[3][4], d1[3][4], d2[3][4];
            for (int a = 0; a < 3; ++a) phi_weights(f[a], w[a], d1[a], d2[a]);
            double *S = acc;
            double *T[3] = {acc + L, acc + 2 * L, acc + 3 * L};
            double *H[3][3];
            H[0][0] = acc + 4 * L; H[1][1] = acc + 5 * L; H[2][2] = acc + 6 * L;
            H[0][1] = H[1][0] = acc + 7 * L; H[0][2] = H[2][0] = acc + 8 * L; H[1][2] = H[2][1] = acc + 9 * L;
            memset(acc, 0, sizeof(double) * 10 * (size_t)L);
            for (int m0 = 0; m0 < 4; ++m0) {
                int k0 = ((i[0] - 1 + m0) % n[0] + n[0]) % n[0];
                for (int m1 = 0; m1 < 4; ++m1) {
                    int k1 = ((i[1] - 1 + m1) % n[1] + n[1]) % n[1];
                    for (int m2 = 0; m2 < 4; ++m2) {
                        int k2 = ((i[2] - 1 + m2) % n[2] + n[2]) % n[2];
                        const float *row = c + (((size_t)k0 * n[1] + k1) * n[2] + k2) * (size_t)L;
                        double th = w[0][m0] * w[1][m1] * w[2][m2];
                        double t0 = d1[0][m0] * w[1][m1] * w[2][m2];
                        double t1 = w[0][m0] * d1[1][m1] * w[2][m2];
                        double t2 = w[0][m0] * w[1][m1] * d1[2][m2];
                        double h00 = d2[0][m0] * w[1][m1] * w[2][m2];
                        double h11 = w[0][m0] * d2[1][m1] * w[2][m2];
                        double h22 = w[0][m0] * w[1][m1] * d2[2][m2];
                        double h01 = d1[0][m0] * d1[1][m1] * w[2][m2];
                        double h02 = d1[0][m0] * w[1][m1] * d1[2][m2];
                        double h12 = w[0][m0] * d1[1][m1] * d1[2][m2];
                        for (int l = 0; l < L; ++l) {
                            double a = (double)row[l];
                            S[l] += th * a;
                            T[0][l] += t0 * a; T[1][l] += t1 * a; T[2][l] += t2 * a;
                            H[0][0][l] += h00 * a; H[1][1][l] += h11 * a; H[2][2][l] += h22 * a;
                            H[0][1][l] += h01 * a; H[0][2][l] += h02 * a; H[1][2][l] += h12 * a;
                        }
                    }
                }
            }
            for (int l = 0; l < L; ++l) {
                val[e * L + l] = S[l];
                for (int x = 0; x < 3; ++x)
                    grad[(e * 3 + x) * L + l] = J[0][x] * T[0][l] + J[1][x] * T[1][l] + J[2][x] * T[2][l];
                for (int q = 0; q < 6; ++q) {
                    double s = 0.0;
                    for (int a = 0; a < 3; ++a)
                        for (int b = 0; b < 3; ++b)
                            s += J[a][ci[q]] * H[a][b][l] * J[b][cj[q]];
                    hess[(e * 6 + q) * L + l] = s;
                }
            }
        }
        free(acc);
    }
    return failed ? -3 : 0;
}

/* Perpendicular spacing of the grid planes along each axis, h_a = 1 / (n_a |column a of G|)
 * (reading R13: the "h" of the stated tolerances is max_a h_a). */
int blip_oracle_spacing(const double A[9], const int n[3], double h[3])
{
    double G[9];
    if (blip_oracle_inverse_lattice(A, G)) return -1;
    for (int a = 0; a < 3; ++a) {
        double s = sqrt(G[a] * G[a] + G[3 + a] * G[3 + a] + G[6 + a] * G[6 + a]);
        h[a] = 1.0 / ((double)n[a] * s);
    }
    return 0;
}

int blip_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void blip_oracle_set_num_threads(int t)
{
#ifdef _OPENMP
    if (t > 0) omp_set_num_threads(t);
#else
    (void)t;
#endif
}
