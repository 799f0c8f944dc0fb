/* lm_client.c -- a plain C client of liblm.so (include/lm.h): no Python, no torch, only the CUDA runtime for device memory.
 * Built and run by tests/test_gpu_c_client.py.  Checks what the paper fixes in closed form:
 *   (1) N = 1: U = F / (6 pi eta a), Omega = T / (8 pi eta a^3);
 *   (2) two spheres, equal forces along / across the line of centres (textbook RPY):
 *       U = F/(6 pi eta a) (1 + 3a/(2r) - a^3/r^3)  and  (1 + 3a/(4r) + a^3/(2r^3)),  r >= 2a;
 *   (3) lm_sqrt_mdot_w on one sphere: M^{1/2} W = W / sqrt(6 pi eta a);
 *   (4) the host-buffer twins give the same numbers; error codes for misuse.
 * Exit code 0 on success; prints the first failure otherwise. */
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "../../include/lm.h"

#define PI 3.14159265358979323846
#define CHECK(cond, ...) do { if (!(cond)) { fprintf(stderr, "FAIL %s:%d: ", __FILE__, __LINE__); fprintf(stderr, __VA_ARGS__); fprintf(stderr, "\n"); return 1; } } while (0)

static int close_to(double got, double want, double tol) { return fabs(got - want) <= tol * fmax(fabs(want), 1e-300); }

/* --time: microseconds per lm_mdot called back to back from C (no Python marshalling), fp32 and fp64, a few sizes */
static int time_applies(void)
{
    const int sizes[] = {64, 256, 1024, 2048, 4096};
    for (int prec = 0; prec < 2; ++prec)
        for (unsigned si = 0; si < sizeof sizes / sizeof sizes[0]; ++si) {
            const int N = sizes[si];
            const size_t es = prec ? 8 : 4, bytes = (size_t)3 * N * es;
            void *pos = malloc(bytes), *d_pos, *d_f, *d_u;
            const double side = cbrt(N * 4.0 * PI / 3.0 / 0.05);
            srand(7);
            for (int i = 0; i < 3 * N; ++i) {
                const double v = side * rand() / (double)RAND_MAX;
                if (prec) ((double*)pos)[i] = v; else ((float*)pos)[i] = (float)v;
            }
            cudaMalloc(&d_pos, bytes); cudaMalloc(&d_f, bytes); cudaMalloc(&d_u, bytes);
            cudaMemcpy(d_pos, pos, bytes, cudaMemcpyHostToDevice);
            cudaMemcpy(d_f, pos, bytes, cudaMemcpyHostToDevice);          /* any finite values serve as forces */
            lm_solver* s = NULL;
            CHECK(lm_create(&s, prec ? LM_F64 : LM_F32, N, 1.0, 1.0, 0) == LM_OK, "lm_create");
            CHECK(lm_set_positions(s, d_pos, NULL) == LM_OK, "%s", lm_last_error(s));
            cudaEvent_t e0, e1;
            cudaEventCreate(&e0); cudaEventCreate(&e1);
            float best = 1e30f;
            for (int rep = 0; rep < 4; ++rep) {
                const int n = 500;
                cudaEventRecord(e0, 0);
                for (int i = 0; i < n; ++i) CHECK(lm_mdot(s, d_f, NULL, d_u, NULL, NULL) == LM_OK, "%s", lm_last_error(s));
                cudaEventRecord(e1, 0);
                cudaEventSynchronize(e1);
                float ms; cudaEventElapsedTime(&ms, e0, e1);
                if (rep && ms / n < best) best = ms / n;
            }
            printf("{\"precision\": \"%s\", \"N\": %d, \"us_per_mdot_from_c\": %.3f, \"kernel\": \"%s\"}\n", prec ? "f64" : "f32", N, best * 1e3, lm_pair_kernel_name(s, 1));
            lm_destroy(s);
            cudaFree(d_pos); cudaFree(d_f); cudaFree(d_u); free(pos);
        }
    return 0;
}

int main(int argc, char** argv)
{
    if (argc > 1 && strcmp(argv[1], "--time") == 0) return time_applies();
    const double eta = 1.3, a = 0.7;
    const double mu_t = 1.0 / (6.0 * PI * eta * a), mu_r = 1.0 / (8.0 * PI * eta * a * a * a);
    double *d_pos, *d_f, *d_t, *d_u, *d_w;
    CHECK(cudaMalloc((void**)&d_pos, 6 * sizeof(double)) == cudaSuccess, "cudaMalloc");
    cudaMalloc((void**)&d_f, 6 * sizeof(double));
    cudaMalloc((void**)&d_t, 6 * sizeof(double));
    cudaMalloc((void**)&d_u, 6 * sizeof(double));
    cudaMalloc((void**)&d_w, 6 * sizeof(double));

    /* (1) one sphere, fp64, with the angular blocks */
    lm_solver* s = NULL;
    CHECK(lm_create(&s, LM_F64, 1, eta, a, 1) == LM_OK, "lm_create");
    const double pos1[3] = {0.3, -1.0, 2.0}, f1[3] = {1.0, -2.0, 0.5}, t1[3] = {0.25, 0.5, -1.5};
    double u[6], w[6];
    CHECK(lm_mdot(s, d_f, d_t, d_u, d_w, NULL) == LM_E_NOPOS, "mdot before set_positions must be LM_E_NOPOS");
    cudaMemcpy(d_pos, pos1, sizeof pos1, cudaMemcpyHostToDevice);
    cudaMemcpy(d_f, f1, sizeof f1, cudaMemcpyHostToDevice);
    cudaMemcpy(d_t, t1, sizeof t1, cudaMemcpyHostToDevice);
    CHECK(lm_set_positions(s, d_pos, NULL) == LM_OK, "%s", lm_last_error(s));
    CHECK(lm_mdot(s, d_f, d_t, d_u, d_w, NULL) == LM_OK, "%s", lm_last_error(s));
    cudaDeviceSynchronize();
    cudaMemcpy(u, d_u, 3 * sizeof(double), cudaMemcpyDeviceToHost);
    cudaMemcpy(w, d_w, 3 * sizeof(double), cudaMemcpyDeviceToHost);
    for (int k = 0; k < 3; ++k) {
        CHECK(close_to(u[k], mu_t * f1[k], 1e-13), "self mobility: U[%d] = %.17g, want %.17g", k, u[k], mu_t * f1[k]);
        CHECK(close_to(w[k], mu_r * t1[k], 1e-13), "rotational self mobility: W[%d] = %.17g, want %.17g", k, w[k], mu_r * t1[k]);
    }
    /* (3) M^{1/2} W of one sphere: block diagonal, sqrt of the two self mobilities */
    const double z[6] = {0.5, -1.0, 2.0, 1.5, 0.25, -0.75};
    cudaMemcpy(d_f, z, sizeof z, cudaMemcpyHostToDevice);
    int iters = -1;
    CHECK(lm_sqrt_mdot_w(s, d_f, 1e-10, d_u, d_w, &iters, NULL) == LM_OK, "%s", lm_last_error(s));
    cudaMemcpy(u, d_u, 3 * sizeof(double), cudaMemcpyDeviceToHost);
    cudaMemcpy(w, d_w, 3 * sizeof(double), cudaMemcpyDeviceToHost);
    for (int k = 0; k < 3; ++k) {
        CHECK(close_to(u[k], sqrt(mu_t) * z[k], 1e-9), "sqrt: U[%d] = %.17g, want %.17g", k, u[k], sqrt(mu_t) * z[k]);
        CHECK(close_to(w[k], sqrt(mu_r) * z[3 + k], 1e-9), "sqrt: W[%d] = %.17g, want %.17g", k, w[k], sqrt(mu_r) * z[3 + k]);
    }
    CHECK(iters >= 1 && iters <= 6, "Lanczos iterations on a 6-dof problem: %d", iters);
    lm_destroy(s);

    /* (2) two spheres, fp32 and fp64, through the host-buffer twins */
    for (int prec = 0; prec < 2; ++prec) {
        const double r = 3.1 * a;
        CHECK(lm_create(&s, prec ? LM_F64 : LM_F32, 2, eta, a, 0) == LM_OK, "lm_create");
        const double tol = prec ? 1e-13 : 2e-6;
        const double want_par = mu_t * (1.0 + 1.5 * a / r - a * a * a / (r * r * r));
        const double want_perp = mu_t * (1.0 + 0.75 * a / r + 0.5 * a * a * a / (r * r * r));
        if (prec) {
            const double pos2[6] = {0, 0, 0, r, 0, 0}, f2[6] = {1, 1, 0, 1, 1, 0};
            double out[6];
            CHECK(lm_set_positions_host(s, pos2, NULL) == LM_OK && lm_mdot_host(s, f2, NULL, out, NULL, NULL) == LM_OK, "%s", lm_last_error(s));
            CHECK(close_to(out[0], want_par, tol) && close_to(out[3], want_par, tol), "sedimentation along the line of centres: %.17g want %.17g", out[0], want_par);
            CHECK(close_to(out[1], want_perp, tol) && close_to(out[4], want_perp, tol), "sedimentation across: %.17g want %.17g", out[1], want_perp);
            CHECK(lm_mdot_host(s, f2, f2, out, NULL, NULL) == LM_E_ANGULAR, "torques on a translational handle must be LM_E_ANGULAR");
        } else {
            const float pos2[6] = {0, 0, 0, (float)r, 0, 0}, f2[6] = {1, 1, 0, 1, 1, 0};
            float out[6];
            const double rr = (double)pos2[3];
            const double wp = mu_t * (1.0 + 1.5 * a / rr - a * a * a / (rr * rr * rr)), wq = mu_t * (1.0 + 0.75 * a / rr + 0.5 * a * a * a / (rr * rr * rr));
            CHECK(lm_set_positions_host(s, pos2, NULL) == LM_OK && lm_mdot_host(s, f2, NULL, out, NULL, NULL) == LM_OK, "%s", lm_last_error(s));
            CHECK(close_to(out[0], wp, tol) && close_to(out[4], wq, tol), "fp32 sedimentation: %.9g want %.9g, %.9g want %.9g", out[0], wp, out[4], wq);
        }
        lm_destroy(s);
    }
    CHECK(lm_create(&s, LM_F32, 0, eta, a, 0) == LM_E_INVALID && s == NULL, "N = 0 must be refused");
    printf("lm_client: OK (%s)\n", lm_version());
    return 0;
}
