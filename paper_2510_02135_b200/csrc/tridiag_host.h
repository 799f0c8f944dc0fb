// tridiag_host.h -- host side of the Lanczos driver:
// c = T^{1/2} e_1 in fp64 from a symmetric tridiagonal eigensolve (implicit-shift QL, rotations recorded
// rather than accumulated).  Plain C++; no CUDA; k <= max_iter (<= 1000).
#pragma once
#include <cmath>
#include <vector>

namespace lm {

// sqrt(a^2 + b^2) without std::hypot's over/underflow handling (several times slower, and called O(k^2) times):
// the entries are Lanczos coefficients of a mobility matrix, far from the limits of fp64 even squared.
inline double pythag(double a, double b) { return std::sqrt(a * a + b * b); }

// c = T_k^{1/2} e_1 for T = tridiag(beta; alpha; beta), negative eigenvalues clamped to zero (O4),
// in O(k^2): with T = Z L Z^T,  c = Z (sqrt(L) (Z^T e_1)).  Z is the product G_1 G_2 ... G_r of the plane
// rotations of the implicit-shift QL sweeps, so instead of accumulating the k x k matrix (O(k^3), the old
// bottleneck of a short Lanczos iteration: 89 us at k = 30, 2.3 ms at k = 100) the solve
//   (i)  tracks only the FIRST ROW of Z through the rotations  (= Z^T e_1, two entries per rotation),
//   (ii) records every rotation (i, c, s),
//   (iii) forms v = sqrt(L) . (Z^T e_1) and applies the rotations to it in reverse order:  c = G_1 (... (G_r v)).
// A rotation on columns (i, i+1) maps  z_i <- c z_i - s z_{i+1},  z_{i+1} <- s z_i + c z_{i+1};  as a matrix on a
// column vector:  (G v)_i = c v_i + s v_{i+1},  (G v)_{i+1} = -s v_i + c v_{i+1}.
// Returns false if an eigenvalue needs more than 60 QL sweeps.
inline bool tridiag_sqrt_e1(int n, const double* alpha, const double* beta, double* c_out)
{
    struct Rot { int i; double c, s; };
    static thread_local std::vector<double> d, e, row0;   // reused across calls: no allocation on the per-iteration path
    static thread_local std::vector<Rot> rots;
    d.assign(alpha, alpha + n);
    e.assign((size_t)n, 0.0);
    row0.assign((size_t)n, 0.0);
    for (int i = 0; i + 1 < n; ++i) e[i] = beta[i];
    row0[0] = 1.0;
    rots.clear();
    rots.reserve((size_t)3 * n * n / 2 + 16);
    for (int l = 0; l < n && n > 1; ++l) {
        int iter = 0, m;
        do {
            for (m = l; m < n - 1; ++m) {
                const double dd = std::fabs(d[m]) + std::fabs(d[m + 1]);
                if (std::fabs(e[m]) <= 2.3e-16 * dd) break;
            }
            if (m != l) {
                if (iter++ == 60) return false;
                double g = (d[l + 1] - d[l]) / (2.0 * e[l]);
                double r = pythag(g, 1.0);
                g = d[m] - d[l] + e[l] / (g + std::copysign(r, g));
                double s = 1.0, c = 1.0, p = 0.0;
                int i;
                for (i = m - 1; i >= l; --i) {
                    double f = s * e[i];
                    const double b = c * e[i];
                    r = pythag(f, g);
                    e[i + 1] = r;
                    if (r == 0.0) {
                        d[i + 1] -= p;
                        e[m] = 0.0;
                        break;
                    }
                    const double inv_r = 1.0 / r;
                    s = f * inv_r;
                    c = g * inv_r;
                    g = d[i + 1] - p;
                    r = (d[i] - g) * s + 2.0 * c * b;
                    p = s * r;
                    d[i + 1] = g + p;
                    g = c * r - b;
                    const double zi = row0[i], zj = row0[i + 1];
                    row0[i + 1] = s * zi + c * zj;
                    row0[i] = c * zi - s * zj;
                    rots.push_back({i, c, s});
                }
                if (r == 0.0 && i >= l) continue;
                d[l] -= p;
                e[l] = g;
                e[m] = 0.0;
            }
        } while (m != l);
    }
    for (int m = 0; m < n; ++m) c_out[m] = std::sqrt(d[m] > 0.0 ? d[m] : 0.0) * row0[m];
    for (size_t t = rots.size(); t-- > 0;) {
        const Rot& R = rots[t];
        const double vi = c_out[R.i], vj = c_out[R.i + 1];
        c_out[R.i] = R.c * vi + R.s * vj;
        c_out[R.i + 1] = -R.s * vi + R.c * vj;
    }
    return true;
}

}  // namespace lm
