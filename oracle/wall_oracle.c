/*
 * wall_oracle.c -- CPU fp64 ORACLE for the single-wall ("Swan-Brady") Rotne-Prager-Yamakawa mobility.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and the cpu_baseline /
 * --impl reference legs of bench.py may build, load or call this file.  It shares no code, header, table
 * or constant with the CUDA path under paper_2510_02135_b200/csrc/.  It is compiled together with
 * rpy_oracle.c (the free-space pair scalars, pinned in tests/test_oracle_pins.py) into libwall_oracle.so.
 *
 * What it computes: U = M.[F;T] for libMobility's NBody solver with the geometry ("open","open",
 * "single_wall") -- PAPER.md:173: "single_wall, in which case the Swan-Brady kernel [37] is used. ... the
 * Swan-Brady kernel does not produce a symmetric positive definite (SPD) mobility matrix when particles
 * overlap the wall.  To address this, we have included the damping matrix approach ... that ensures the
 * mobility of a particle smoothly goes to zero as a particle approaches the wall in a way that maintains
 * the SPD property".  The paper prints neither the tensors nor the damping matrix (DESIGN.md readings
 * S18-S20).  Taken here:
 *
 *   S18  The pair blocks are eq. (8) / eq. (4) with delta_F = delta_T = the
 *        surface delta of a sphere of radius a and L = the Green's function of a half space bounded by a
 *        no-slip plane (Blake's image system) = Oseen tensor + image part G_im.  The free-space (Oseen)
 *        part gives the free-space RPY blocks of rpy_oracle.c, overlap forms included.  For spheres that
 *        do not cut the wall the double surface average of the image part is EXACTLY the Faxen form
 *            M^w_uF = (1 + a^2/6 lap_x)(1 + a^2/6 lap_y) G_im(x, y)
 *            M^w_wF = 1/2 curl_x (1 + a^2/6 lap_y) G_im          M^w_uT(i<-j) = [M^w_wF(j<-i)]^T
 *            M^w_wT = 1/4 curl_x curl_y G_im
 *        (the sphere average of a biharmonic field is its centre value + a^2/6 of its Laplacian; the curl
 *        of a Stokes velocity is harmonic), which is how ref. [37] obtains its kernel.  Carrying out the
 *        derivatives (DESIGN.md appendix A) gives the closed forms in wall_pair_correction() below.
 *   S19  Damping matrix: M~ = B M(x~) B with x~_i = x_i with its height raised to max(h_i, a) and
 *        B = diag(b_i) acting on all six components of particle i, b_i = min(1, max(h_i, 0) / a); h_i is the
 *        height of the centre above the wall.  M(x~) is then a double surface average for every pair (SPD), a
 *        diagonal congruence keeps it SPD (semi-definite when some b_i = 0), and a particle's mobility goes to
 *        zero continuously as h_i -> 0.
 *   S20  The wall is the plane z = wall_z (the paper's setParameters(wallHeight)); the
 *        fluid occupies z > wall_z.
 *
 * Plain double loop, j ascending, fp64 "+=", no blocking, no reordering.
 *
 * Parity pins (tests/test_oracle_wall.py): every block of wall_pair_correction against eq. (8)/(4) evaluated
 * by quadrature over the two spheres with an independent implementation of Blake's tensor (itself pinned:
 * no slip on the wall, incompressible, Stokes, Oseen singularity); against finite-difference Faxen operators;
 * the single-sphere wall mobilities against their known series in a/h (translation parallel / perpendicular,
 * rotation, coupling); free-space limit far from the wall; symmetric positive (semi-)definite dense M with
 * particles overlapping each other and the wall; invariances; row-sampled = full; dense M @ [F;T].
 * No function in this file is "parity unpinned".
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o libwall_oracle.so wall_oracle.c rpy_oracle.c -lm   (no fast-math)
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_PI 3.14159265358979323846264338327950288

void rpy_pair_scalars(double r, double a, double eta, double s[5]);   /* rpy_oracle.c */

/* The four 3x3 blocks (row-major, [k][l]) by which the wall CORRECTS the free-space pair mobility of
 * particle i (velocity side) <- particle j (force side), heights zi, zj >= a above the wall:
 *     uF: u_i <- F_j      uT: u_i <- T_j      wF: omega_i <- F_j      wT: omega_i <- T_j
 * Notation: R = x_i - x_j* with x_j* the mirror image of x_j, i.e. R = (x_i - x_j, y_i - y_j, zi + zj),
 * Rn = |R|, Z = R_z, h = zj (height of the force side), zhat = (0,0,1), P = R x zhat = (R_y, -R_x, 0),
 * [zhat]_x v = zhat x v.  All in units of 1/(8 pi eta); i == j is the same formula with R = (0,0,2h). */
void wall_pair_correction(const double xi[3], const double xj[3], double a, double eta,
                          double uF[9], double uT[9], double wF[9], double wT[9])
{
    const double pref = 1.0 / (8.0 * ORACLE_PI * eta);
    const double a2 = a * a, a4 = a2 * a2;
    for (int swap = 0; swap < 2; ++swap) {
        /* swap == 0: (i <- j) gives uF, wF, wT.  swap == 1: (j <- i) gives wF(j<-i), whose transpose is uT(i<-j). */
        const double *p = swap ? xj : xi, *q = swap ? xi : xj;
        const double R[3] = {p[0] - q[0], p[1] - q[1], p[2] + q[2]};
        const double h = q[2], Z = R[2];
        const double R2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2];
        const double Rn = sqrt(R2);
        const double i1 = 1.0 / Rn, i3 = i1 / R2, i5 = i3 / R2, i7 = i5 / R2, i9 = i7 / R2;
        const double zh[3] = {0.0, 0.0, 1.0};
        const double P[3] = {R[1], -R[0], 0.0};
        const double zx[9] = {0.0, -1.0, 0.0, 1.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        /* coupling  M^w_wF = B [zhat]_x + C P R^T + D P zhat^T + F zhat P^T */
        const double cB = (Z - 2.0 * h) * i3 + 2.0 * a2 * Z * i5;
        const double cC = -6.0 * h * i5 + 10.0 * a2 * Z * i7;
        const double cD = i3 + 12.0 * h * Z * i5 + a2 * (2.0 * i5 - 20.0 * Z * Z * i7);
        const double cF = -i3;
        double *dst = swap ? uT : wF;
        for (int k = 0; k < 3; ++k)
            for (int l = 0; l < 3; ++l) {
                const double v = pref * (cB * zx[3 * k + l] + cC * P[k] * R[l] + cD * P[k] * zh[l] + cF * zh[k] * P[l]);
                if (swap) dst[3 * l + k] = v;      /* transpose */
                else dst[3 * k + l] = v;
            }
        if (swap) break;
        /* translation-translation  M^w_uF = tI I + tRR R R^T + tRz R zhat^T + tzR zhat R^T + tzz zhat zhat^T */
        const double tI = -i1 - 2.0 * h * (Z - h) * i3 + a2 * (-2.0 / 3.0 * i3 + 2.0 * Z * Z * i5) + a4 * (2.0 / 3.0 * i5 - 10.0 / 3.0 * Z * Z * i7);
        const double tRR = -i3 + 6.0 * h * (Z - h) * i5 + a2 * (2.0 * i5 - 10.0 * Z * Z * i7) + a4 * (-10.0 / 3.0 * i7 + 70.0 / 3.0 * Z * Z * i9);
        const double tRz = 2.0 * h * i3 - 12.0 * h * Z * (Z - h) * i5 + a2 * (-4.0 * Z * i5 + 20.0 * Z * Z * Z * i7)
                           + a4 * (40.0 / 3.0 * Z * i7 - 140.0 / 3.0 * Z * Z * Z * i9);
        const double tzR = 2.0 * h * i3 - 20.0 / 3.0 * a4 * Z * i7;
        const double tzz = -4.0 * h * h * i3 - 4.0 * a2 * Z * Z * i5 + a4 * (-8.0 / 3.0 * i5 + 20.0 * Z * Z * i7);
        /* rotation-rotation  M^w_wT, same tensor basis */
        const double rI = 3.5 * i3 - 6.0 * Z * Z * i5, rRR = -4.5 * i5, rRz = 3.0 * Z * i5, rzR = 6.0 * Z * i5, rzz = -3.0 * i3;
        for (int k = 0; k < 3; ++k)
            for (int l = 0; l < 3; ++l) {
                const double dkl = (k == l) ? 1.0 : 0.0;
                uF[3 * k + l] = pref * (tI * dkl + tRR * R[k] * R[l] + tRz * R[k] * zh[l] + tzR * zh[k] * R[l] + tzz * zh[k] * zh[l]);
                wT[3 * k + l] = pref * (rI * dkl + rRR * R[k] * R[l] + rRz * R[k] * zh[l] + rzR * zh[k] * R[l] + rzz * zh[k] * zh[l]);
            }
    }
}

/* S19: height above the wall raised to at least a, and the damping factor b = min(1, max(h, 0)/a). */
static void damp(const double *x, double wall_z, double a, double xe[3], double *b)
{
    const double h = x[2] - wall_z;
    xe[0] = x[0];
    xe[1] = x[1];
    xe[2] = h > a ? h : a;
    *b = h >= a ? 1.0 : (h > 0.0 ? h / a : 0.0);
}

/* The four full pair blocks of M(x~) for (i <- j): free-space RPY blocks (rpy_oracle.c, SURVEY.md sec. 8(c) O1/O2,
 * evaluated at the raised positions) + the wall correction.  xi, xj: raised positions, heights above the wall. */
static void pair_blocks(const double xi[3], const double xj[3], double a, double eta, double uF[9], double uT[9], double wF[9], double wT[9])
{
    wall_pair_correction(xi, xj, a, eta, uF, uT, wF, wT);
    const double d[3] = {xi[0] - xj[0], xi[1] - xj[1], xi[2] - xj[2]};
    const double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    double s[5], e[3] = {0.0, 0.0, 0.0};
    rpy_pair_scalars(r, a, eta, s);
    if (r > 0.0) { e[0] = d[0] / r; e[1] = d[1] / r; e[2] = d[2] / r; }
    const double ex[9] = {0.0, -e[2], e[1], e[2], 0.0, -e[0], -e[1], e[0], 0.0};   /* [e]_x */
    for (int k = 0; k < 3; ++k)
        for (int l = 0; l < 3; ++l) {
            const double dkl = (k == l) ? 1.0 : 0.0;
            uF[3 * k + l] += s[0] * dkl + s[1] * e[k] * e[l];
            wT[3 * k + l] += s[2] * dkl + s[3] * e[k] * e[l];
            uT[3 * k + l] += -s[4] * ex[3 * k + l];            /* g_c (T x e) = -g_c [e]_x T */
            wF[3 * k + l] += -s[4] * ex[3 * k + l];
        }
}

/* One target row:  U_i = b_i sum_j [ uF b_j F_j + uT b_j T_j ],  W_i = b_i sum_j [ wF b_j F_j + wT b_j T_j ]  (S19). */
static void wall_row_apply(int64_t i, int64_t N, double a, double eta, double wall_z, const double *x,
                           const double *F, const double *T, double *Ui, double *Wi)
{
    double u[3] = {0.0, 0.0, 0.0}, w[3] = {0.0, 0.0, 0.0}, xi[3], bi;
    damp(x + 3 * i, wall_z, a, xi, &bi);
    for (int64_t j = 0; j < N; ++j) {
        double xj[3], bj, uF[9], uT[9], wF[9], wT[9];
        damp(x + 3 * j, wall_z, a, xj, &bj);
        pair_blocks(xi, xj, a, eta, uF, uT, wF, wT);
        double Fj[3] = {0.0, 0.0, 0.0}, Tj[3] = {0.0, 0.0, 0.0};
        if (F) { Fj[0] = bj * F[3 * j]; Fj[1] = bj * F[3 * j + 1]; Fj[2] = bj * F[3 * j + 2]; }
        if (T) { Tj[0] = bj * T[3 * j]; Tj[1] = bj * T[3 * j + 1]; Tj[2] = bj * T[3 * j + 2]; }
        for (int k = 0; k < 3; ++k)
            for (int l = 0; l < 3; ++l) {
                u[k] += uF[3 * k + l] * Fj[l] + uT[3 * k + l] * Tj[l];
                w[k] += wF[3 * k + l] * Fj[l] + wT[3 * k + l] * Tj[l];
            }
    }
    for (int k = 0; k < 3; ++k) {
        Ui[k] = bi * u[k];
        if (Wi) Wi[k] = bi * w[k];
    }
}

/* Chosen target rows against all N sources (rows == NULL: all rows, nrows = N).  Interleaved xyz arrays.
 * OpenMP over rows only.  Returns the number of threads used. */
int wall_mdot_rows(int64_t N, double a, double eta, double wall_z, const double *x, const double *F, const double *T,
                   int64_t nrows, const int64_t *rows, double *U, double *W)
{
    int nthreads = 1;
#ifdef _OPENMP
    const int par = (double)nrows * (double)N >= 65536.0;      /* tiny problems run on one thread */
#pragma omp parallel if (par)
    {
#pragma omp single
        nthreads = omp_get_num_threads();
    }
#pragma omp parallel for schedule(static) if (par)
#endif
    for (int64_t k = 0; k < nrows; ++k)
        wall_row_apply(rows ? rows[k] : k, N, a, eta, wall_z, x, F, T, U + 3 * k, W ? W + 3 * k : NULL);
    return nthreads;
}

/* Dense M~ = B M(x~) B, row-major dof x dof, dof = 3N (angular == 0) or 6N: [0,3N) linear, [3N,6N) angular. */
void wall_dense(int64_t N, double a, double eta, double wall_z, const double *x, int angular, double *M)
{
    const int64_t dof = angular ? 6 * N : 3 * N;
    for (int64_t i = 0; i < N; ++i) {
        double xi[3], bi;
        damp(x + 3 * i, wall_z, a, xi, &bi);
        for (int64_t j = 0; j < N; ++j) {
            double xj[3], bj, uF[9], uT[9], wF[9], wT[9];
            damp(x + 3 * j, wall_z, a, xj, &bj);
            pair_blocks(xi, xj, a, eta, uF, uT, wF, wT);
            for (int k = 0; k < 3; ++k)
                for (int l = 0; l < 3; ++l) {
                    M[(3 * i + k) * dof + (3 * j + l)] = bi * bj * uF[3 * k + l];
                    if (angular) {
                        M[(3 * i + k) * dof + (3 * N + 3 * j + l)] = bi * bj * uT[3 * k + l];
                        M[(3 * N + 3 * i + k) * dof + (3 * j + l)] = bi * bj * wF[3 * k + l];
                        M[(3 * N + 3 * i + k) * dof + (3 * N + 3 * j + l)] = bi * bj * wT[3 * k + l];
                    }
                }
        }
    }
}
