// lanczos_host.h -- host side of the Lanczos driver that is NOT the eigensolve: the stopping test
// (readings S3 / S15) and the cross-rank agreement on it.
// Plain C++; no CUDA.  Included by lm_api.cu; tests/hooks/lm_host_hooks.cpp compiles the same header for the CPU tests.
#pragma once
#include <algorithm>
#include <cmath>
#include <cstddef>
#include <vector>

#include "tridiag_host.h"

namespace lm {

enum { RULE_ESTIMATE = 0, RULE_STEP = 1 };   // = LM_RULE_* of include/lm.h

// Error estimate of the newest iterate y_k from the relative steps s_2 .. s_k (reading S3; PAPER.md:147 fixes no
// rule).  The rule of ref. [35] takes the step s_k as the error; an iterate whose steps shrink by a ratio rho per
// iteration still has s_k (rho + rho^2 + ...) to travel, and single steps dip whenever a new Ritz value shows up:
//     e_k = max(s_k, s_{k-1}) * max(1, rho / (1 - rho)),
//     rho = min( (sum of the last m steps / sum of the m steps before)^(1/m), 0.98 ),  m = max(1, min(10, (k-1)/2)).
// `steps` holds s_2 .. s_k (k - 1 >= 2 values).
inline double lanczos_error_estimate(const std::vector<double>& steps)
{
    const int have = (int)steps.size();
    const int m = std::max(1, std::min(10, have / 2));
    double tail = 0.0, head = 0.0;
    for (int i = 0; i < m; ++i) {
        tail += steps[have - 1 - i];
        head += steps[have - 1 - m - i];
    }
    double amplify = 1.0;
    if (head > 0.0) {
        const double rho = std::min(std::pow(tail / head, 1.0 / m), 0.98);
        amplify = std::max(1.0, rho / (1.0 - rho));
    }
    return std::max(steps[have - 1], steps[have - 2]) * amplify;
}

// One noise vector's host state: T_k, c_k = T_k^{1/2} e_1 (a8), the Gram matrix of the basis and the stopping
// test (a9).  |y_k - y_{k-1}|^2 / |z|^2 = d^T G d with d = c_k - [c_{k-1}; 0] and G = V^T V the TRUE Gram matrix
// (S15: no re-orthogonalisation, so G != I in fp32 after ~20 steps); |y_{k-1}|^2 / |z|^2 = c_{k-1}^T G c_{k-1}.
struct LanczosStopper {
    enum Verdict { CONTINUE = 0, CONVERGED = 1, EIGENSOLVE_FAILED = -1 };
    int rule = RULE_ESTIMATE;
    double tol = 0.0, breakdown = 0.0;
    int ldg = 0;                                  // leading dimension of gram: max_iter + 1
    std::vector<double> gram;                     // gram[i * ldg + j] = V_i . V_j, filled one column per new basis vector
    std::vector<double> alphas, betas, c_prev, c_cur, steps, estimates;
    std::vector<double> dvec, gvec;               // scratch of feed(): d = c_k - [c_{k-1}; 0] and G d
    double pending_beta = 0.0;
    double den_cur = 0.0;                         // c_cur^T G c_cur = |y_k|^2 / |z|^2 of the newest iterate

    void reset(int rule_, double tol_, double breakdown_, int max_iter)
    {
        rule = rule_;
        tol = tol_;
        breakdown = breakdown_;
        ldg = max_iter + 1;
        gram.assign((size_t)ldg * ldg, 0.0);
        alphas.clear(); betas.clear(); c_prev.clear(); c_cur.clear(); steps.clear(); estimates.clear();
    }
    // column m of the Gram matrix: col[j] = V_j . V_m, j <= m  (V_m = v_{m+1}, the vector created by iteration m)
    template <typename Ptr> void set_gram_column(int m, Ptr col)
    {
        for (int j = 0; j <= m; ++j) gram[(size_t)j * ldg + m] = gram[(size_t)m * ldg + j] = (double)col[j];
    }
    double quad(const std::vector<double>& v, int n) const
    {
        double q = 0.0;
        for (int i = 0; i < n; ++i)
            for (int j = 0; j < n; ++j) q += v[i] * gram[(size_t)i * ldg + j] * v[j];
        return q;
    }
    // iteration k's scalars (k = 1, 2, ...; the Gram columns 0 .. k-1 are already set): the verdict of THIS rank.
    // c_cur holds c_k afterwards.  The recurrence only moves on when the caller says so (advance): in a row-sharded
    // run the verdict acted upon is rank 0's (agree_on_stops), which may differ from the local one.
    Verdict feed(int k, double alpha, double beta)
    {
        alphas.push_back(alpha);
        c_cur.assign((size_t)k, 0.0);
        if (!tridiag_sqrt_e1(k, alphas.data(), betas.data(), c_cur.data())) return EIGENSOLVE_FAILED;
        bool stop = false;
        if (k == 1) den_cur = quad(c_cur, 1);
        if (k >= 2) {
            // ONE product g = G d per iteration (the loop at small N waits for this host code): |y_k - y_{k-1}|^2 = d.g, and
            // |y_k|^2 = |y_{k-1}|^2 + 2 c_{k-1}.g + d.g carries the denominator forward (it only normalises: its
            // rounding, ~k eps, is immaterial; the numerator is formed directly, without cancellation)
            dvec.assign(c_cur.begin(), c_cur.end());
            for (int i = 0; i < k - 1; ++i) dvec[i] -= c_prev[i];
            gvec.assign((size_t)k, 0.0);
            for (int i = 0; i < k; ++i) {
                const double* gi = &gram[(size_t)i * ldg];
                double acc = 0.0;
                for (int j = 0; j < k; ++j) acc += gi[j] * dvec[j];
                gvec[i] = acc;
            }
            double dg = 0.0, cg = 0.0;
            for (int i = 0; i < k; ++i) dg += dvec[i] * gvec[i];
            for (int i = 0; i < k - 1; ++i) cg += c_prev[i] * gvec[i];
            const double num = std::max(dg, 0.0), den = std::max(den_cur, 0.0);
            den_cur = den_cur + 2.0 * cg + dg;
            // a zero previous iterate cannot happen for an SPD matrix (c_1 = sqrt(alpha_1) > 0); keep the ratio finite anyway
            steps.push_back(den > 0.0 ? std::sqrt(num / den) : (num > 0.0 ? HUGE_VAL : 0.0));
            if (rule == RULE_STEP) {
                stop = steps.back() <= tol;
            } else if (k >= 3) {
                estimates.push_back(lanczos_error_estimate(steps));
                stop = estimates.back() <= tol;
            }
        }
        if (beta <= breakdown * std::fabs(alpha)) stop = true;          // invariant subspace: the iterate is exact
        pending_beta = beta;
        return stop ? CONVERGED : CONTINUE;
    }
    // go on to iteration k + 1; the caller then sets Gram column k (the vector v_{k+1} just created)
    void advance()
    {
        betas.push_back(pending_beta);
        c_prev = c_cur;
    }
    // what the rule measured at the last iteration fed (NaN before it has anything to measure)
    double last_measure() const
    {
        if (rule == RULE_STEP) return steps.empty() ? NAN : steps.back();
        return estimates.empty() ? NAN : estimates.back();
    }
};

// Cross-rank agreement on the stopping decision (row-sharded runs).  Every rank evaluates the
// test on its own copy of the scalars; if the copies ever differed in the last bit (another driver, GPU bin,
// reduction grid), one rank would enqueue an all-gather the others never post.  So the verdicts of one iteration
// are packed into a word (bit q = vector q stops now, bit 31 = this rank hit a failure) and the ranks agree on
//   * the STOP bits of rank 0 (a broadcast), and
//   * the OR of everybody's FAILURE bit (a max-reduction): a failure seen on any rank -- not only on rank 0 -- makes all
//     ranks leave the loop together instead of one returning while the others post the next collective.
// `exchange(words)` is the transport (ncclBroadcast + ncclAllReduce in the library, gloo in the CPU test):
//   in:  words[0] = this rank's stop bits, words[1] = this rank's failure flag (0 / 1)
//   out: words[0] = rank 0's stop bits,    words[1] = max over ranks of the failure flags.
// Returns the agreed word; with one rank (distributed == false) it is the local word.
template <typename Exchange> inline unsigned agree_on_stops(unsigned local_word, Exchange&& exchange, bool distributed)
{
    if (!distributed) return local_word;
    unsigned words[2] = {local_word & 0x7fffffffu, local_word >> 31};
    exchange(words);
    return (words[0] & 0x7fffffffu) | (words[1] ? 0x80000000u : 0u);
}

}  // namespace lm
