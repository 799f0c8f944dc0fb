/*
 * rpy_oracle.c -- CPU fp64 ORACLE for the free-space Rotne-Prager-Yamakawa (RPY) mobility.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call this file.  It shares
 * no code, header, table or constant with the CUDA path under paper_2510_02135_b200/csrc/.
 *
 * What it computes: the plain definition of U = M.[F;T] for libMobility's open-boundary NBody
 * solver ("a brute-force O(N^2) evaluation of pairwise RPY mobilities", sec. 3.5),
 * with the 6N x 6N grand mobility of eq. (7) whose blocks are eq. (8)
 * evaluated for equal spheres of radius a in an unbounded fluid of viscosity eta.
 * The paper names the pair tensors but does not print them; the closed
 * forms below are the textbook RPY tensors (DESIGN.md "Readings" S1):
 * Rotne-Prager / Yamakawa for translation, and their equal-radius extension to rotation and
 * translation-rotation coupling, each with the overlap (r < 2a) form that keeps M positive
 * definite.  Plain double loop, j ascending, fp64 "+=", no blocking, no reordering.
 *
 * Parity pins (tests/test_oracle_pins.py): self mobility 1/(6 pi eta a) and
 * 1/(8 pi eta a^3); continuity of all five scalars at r = 2a; Oseen limit; two-sphere
 * sedimentation closed forms; symmetric positive-definite dense M; divergence-free
 * (PAPER.md:87); the integral definition eq. (8)/(4) evaluated by quadrature over the two
 * spheres for the tt, rt and rr blocks in BOTH branches; handedness of the coupling; brute-force
 * numpy double loop.  No function in this file is "parity unpinned".
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o librpy_oracle.so rpy_oracle.c -lm   (no fast-math)
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_PI 3.14159265358979323846264338327950288

/* SURVEY.md sec. 8(c) O1 / DESIGN.md S1, S2: the five pair scalars at centre distance r >= 0.
 *   M_uF^{ij} = f_tt I + g_tt rhat rhat^T          (translation-translation)
 *   M_wT^{ij} = f_rr I + g_rr rhat rhat^T          (rotation-rotation)
 *   M_uT^{ij} = M_wF^{ij} = -g_c [rhat]_x          (coupling; [v]_x w = v x w)
 * Far branch for r >= 2a (S2), overlap branch for r < 2a.  s[0..4] = f_tt, g_tt, f_rr, g_rr, g_c. */
void rpy_pair_scalars(double r, double a, double eta, double s[5])
{
    if (r >= 2.0 * a) {
        double c = 1.0 / (8.0 * ORACLE_PI * eta * r);
        s[0] = c * (1.0 + 2.0 * a * a / (3.0 * r * r));
        s[1] = c * (1.0 - 2.0 * a * a / (r * r));
        s[2] = -1.0 / (16.0 * ORACLE_PI * eta * r * r * r);
        s[3] = 3.0 / (16.0 * ORACLE_PI * eta * r * r * r);
        s[4] = 1.0 / (8.0 * ORACLE_PI * eta * r * r);
    } else {
        double ct = 1.0 / (6.0 * ORACLE_PI * eta * a);
        double cr = 1.0 / (8.0 * ORACLE_PI * eta * a * a * a);
        double q = r / a;
        s[0] = ct * (1.0 - 9.0 * q / 32.0);
        s[1] = ct * (3.0 * q / 32.0);
        s[2] = cr * (1.0 - 27.0 * q / 32.0 + 5.0 * q * q * q / 64.0);
        s[3] = cr * (9.0 * q / 32.0 - 3.0 * q * q * q / 64.0);
        s[4] = 1.0 / (16.0 * ORACLE_PI * eta * a * a) * (q - 3.0 * q * q / 8.0);
    }
}

/* One target row i of SURVEY.md sec. 8(c) O2 (eq. (7) applied to [F;T]):
 *   U_i = sum_j [ f_tt F_j + g_tt (rhat.F_j) rhat + g_c (T_j x rhat) ]
 *   W_i = sum_j [ f_rr T_j + g_rr (rhat.T_j) rhat + g_c (F_j x rhat) ]
 * over ALL j including j = i, rhat = (x_i - x_j)/r and rhat := 0 when r = 0 (S5: the self term
 * is the r -> 0 limit of the overlap branch).  T == NULL means torques are zero; W may be NULL. */
static void row_apply(int64_t i, int64_t N, double a, double eta, const double *x,
                      const double *F, const double *T, double *Ui, double *Wi)
{
    double u[3] = {0.0, 0.0, 0.0}, w[3] = {0.0, 0.0, 0.0};
    for (int64_t j = 0; j < N; ++j) {
        double d[3] = {x[3 * i] - x[3 * j], x[3 * i + 1] - x[3 * j + 1], x[3 * i + 2] - x[3 * j + 2]};
        double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        double s[5];
        rpy_pair_scalars(r, a, eta, s);
        double e[3] = {0.0, 0.0, 0.0};
        if (r > 0.0) { e[0] = d[0] / r; e[1] = d[1] / r; e[2] = d[2] / r; }
        double Fj[3] = {0.0, 0.0, 0.0}, Tj[3] = {0.0, 0.0, 0.0};
        if (F) { Fj[0] = F[3 * j]; Fj[1] = F[3 * j + 1]; Fj[2] = F[3 * j + 2]; }
        if (T) { Tj[0] = T[3 * j]; Tj[1] = T[3 * j + 1]; Tj[2] = T[3 * j + 2]; }
        double eF = e[0] * Fj[0] + e[1] * Fj[1] + e[2] * Fj[2];
        double eT = e[0] * Tj[0] + e[1] * Tj[1] + e[2] * Tj[2];
        /* T_j x rhat and F_j x rhat */
        double Txe[3] = {Tj[1] * e[2] - Tj[2] * e[1], Tj[2] * e[0] - Tj[0] * e[2], Tj[0] * e[1] - Tj[1] * e[0]};
        double Fxe[3] = {Fj[1] * e[2] - Fj[2] * e[1], Fj[2] * e[0] - Fj[0] * e[2], Fj[0] * e[1] - Fj[1] * e[0]};
        for (int k = 0; k < 3; ++k) {
            u[k] += s[0] * Fj[k] + s[1] * eF * e[k] + s[4] * Txe[k];
            w[k] += s[2] * Tj[k] + s[3] * eT * e[k] + s[4] * Fxe[k];
        }
    }
    Ui[0] = u[0]; Ui[1] = u[1]; Ui[2] = u[2];
    if (Wi) { Wi[0] = w[0]; Wi[1] = w[1]; Wi[2] = w[2]; }
}

/* U (3N) and, if W != NULL, W (3N) for all target rows.  Arrays are interleaved xyz, length 3N
 * (the (N,3) row-major arrays of PAPER.md:128-138).  OpenMP over rows only (rows are independent;
 * the arithmetic of each row is untouched).  Returns the number of threads used. */
int rpy_mdot(int64_t N, double a, double eta, const double *x, const double *F, const double *T,
             double *U, double *W)
{
    int nthreads = 1;
#ifdef _OPENMP
    /* tiny problems run on one thread (the pins call this thousands of times with N ~ 5: thread wake-ups would be the cost) */
    const int par = (double)N * (double)N >= 65536.0;
#pragma omp parallel if (par)
    {
#pragma omp single
        nthreads = omp_get_num_threads();
    }
#pragma omp parallel for schedule(static) if (par)
#endif
    for (int64_t i = 0; i < N; ++i)
        row_apply(i, N, a, eta, x, F, T, U + 3 * i, W ? W + 3 * i : NULL);
    return nthreads;
}

/* The same sum for a chosen subset of target rows against all N sources ("row-sampled oracle",
 * SURVEY.md sec. 8(d)): rows are independent, so these rows are exact.  U, W are 3*nrows. */
int rpy_mdot_rows(int64_t N, double a, double eta, const double *x, const double *F, const double *T,
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
        row_apply(rows[k], N, a, eta, x, F, T, U + 3 * k, W ? W + 3 * k : NULL);
    return nthreads;
}

/* Dense grand mobility, row-major dof x dof with dof = 3N (angular == 0) or 6N (eq. (7),
 * PAPER.md:66-69): rows/cols [0,3N) linear (u / F), [3N,6N) angular (omega / T).  For tiny N. */
void rpy_dense(int64_t N, double a, double eta, const double *x, int angular, double *M)
{
    int64_t dof = angular ? 6 * N : 3 * N;
    for (int64_t i = 0; i < N; ++i) {
        for (int64_t j = 0; j < N; ++j) {
            double d[3] = {x[3 * i] - x[3 * j], x[3 * i + 1] - x[3 * j + 1], x[3 * i + 2] - x[3 * j + 2]};
            double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            double s[5];
            rpy_pair_scalars(r, a, eta, s);
            double e[3] = {0.0, 0.0, 0.0};
            if (r > 0.0) { e[0] = d[0] / r; e[1] = d[1] / r; e[2] = d[2] / r; }
            /* [e]_x : ([e]_x v)_k = (e x v)_k */
            double ex[3][3] = {{0.0, -e[2], e[1]}, {e[2], 0.0, -e[0]}, {-e[1], e[0], 0.0}};
            for (int k = 0; k < 3; ++k) {
                for (int l = 0; l < 3; ++l) {
                    double dkl = (k == l) ? 1.0 : 0.0;
                    M[(3 * i + k) * dof + (3 * j + l)] = s[0] * dkl + s[1] * e[k] * e[l];
                    if (angular) {
                        /* T_j x e = -(e x T_j) = -[e]_x T_j */
                        M[(3 * i + k) * dof + (3 * N + 3 * j + l)] = -s[4] * ex[k][l];
                        M[(3 * N + 3 * i + k) * dof + (3 * j + l)] = -s[4] * ex[k][l];
                        M[(3 * N + 3 * i + k) * dof + (3 * N + 3 * j + l)] = s[2] * dkl + s[3] * e[k] * e[l];
                    }
                }
            }
        }
    }
}
