// tridiag_host.h -- host side of the Lanczos driver:
// symmetric tridiagonal eigensolve (implicit-shift QL with accumulated rotations) and
// c = T^{1/2} e_1 in fp64.  Plain C++; no CUDA; k <= max_iter (<= 1000).
#pragma once
#include <cmath>
#include <vector>

namespace lm {

// Eigen-decomposition of T = tridiag(e; d; e): on return d holds the eigenvalues and Z
// (row-major n x n) the eigenvectors as COLUMNS.  e has n entries, e[n-1] unused.
// Returns false if an eigenvalue needs more than 60 QL sweeps.
inline bool tridiag_eigh(int n, std::vector<double>& d, std::vector<double>& e, std::vector<double>& Z)
{
    Z.assign((size_t)n * n, 0.0);
    for (int i = 0; i < n; ++i) Z[(size_t)i * n + i] = 1.0;
    if (n == 1) return true;
    e[n - 1] = 0.0;
    for (int l = 0; l < n; ++l) {
        int iter = 0, m;
        do {
            for (m = l; m < n - 1; ++m) {
                const double dd = std::fabs(d[m]) + std::fabs(d[m + 1]);
                if (std::fabs(e[m]) <= 2.3e-16 * dd) break;
            }
            if (m != l) {
                if (iter++ == 60) return false;
                double g = (d[l + 1] - d[l]) / (2.0 * e[l]);
                double r = std::hypot(g, 1.0);
                g = d[m] - d[l] + e[l] / (g + std::copysign(r, g));
                double s = 1.0, c = 1.0, p = 0.0;
                int i;
                for (i = m - 1; i >= l; --i) {
                    double f = s * e[i];
                    const double b = c * e[i];
                    r = std::hypot(f, g);
                    e[i + 1] = r;
                    if (r == 0.0) {
                        d[i + 1] -= p;
                        e[m] = 0.0;
                        break;
                    }
                    s = f / r;
                    c = g / r;
                    g = d[i + 1] - p;
                    r = (d[i] - g) * s + 2.0 * c * b;
                    p = s * r;
                    d[i + 1] = g + p;
                    g = c * r - b;
                    for (int k = 0; k < n; ++k) {
                        f = Z[(size_t)k * n + i + 1];
                        Z[(size_t)k * n + i + 1] = s * Z[(size_t)k * n + i] + c * f;
                        Z[(size_t)k * n + i] = c * Z[(size_t)k * n + i] - s * f;
                    }
                }
                if (r == 0.0 && i >= l) continue;
                d[l] -= p;
                e[l] = g;
                e[m] = 0.0;
            }
        } while (m != l);
    }
    return true;
}

// c = T_k^{1/2} e_1 with negative eigenvalues clamped to zero (O4).
inline bool tridiag_sqrt_e1(int k, const double* alpha, const double* beta, double* c_out)
{
    std::vector<double> d(alpha, alpha + k), e(k, 0.0), Z;
    for (int i = 0; i + 1 < k; ++i) e[i] = beta[i];
    if (!tridiag_eigh(k, d, e, Z)) return false;
    for (int i = 0; i < k; ++i) c_out[i] = 0.0;
    for (int m = 0; m < k; ++m) {
        const double lam = d[m] > 0.0 ? d[m] : 0.0;
        const double wgt = std::sqrt(lam) * Z[m];      // Z[0][m]: first component of eigenvector m
        for (int i = 0; i < k; ++i) c_out[i] += Z[(size_t)i * k + m] * wgt;
    }
    return true;
}

}  // namespace lm
