// lm_host_hooks.cpp -- TEST HOOKS, not product code: exposes the host-only pieces of the Lanczos driver
// (paper_2510_02135_b200/csrc/tridiag_host.h, lanczos_host.h -- the very headers lm_api.cu compiles) through a C
// ABI so that the `-m "not gpu"` tests can drive them without a GPU.  Built by tests/hooks/__init__.py with g++.
#include <cstring>

#include "../../paper_2510_02135_b200/csrc/lanczos_host.h"

extern "C" {

int hook_tridiag_sqrt_e1(int k, const double* alpha, const double* beta, double* c_out)
{
    if (k < 1) return -1;
    if (!alpha || !c_out || (k > 1 && !beta)) return -4;
    return lm::tridiag_sqrt_e1(k, alpha, beta, c_out) ? 0 : -6;
}

double hook_error_estimate(const double* steps, int n)
{
    return lm::lanczos_error_estimate(std::vector<double>(steps, steps + n));
}

void* hook_stopper_new(int rule, double tol, double breakdown, int max_iter)
{
    auto* s = new lm::LanczosStopper();
    s->reset(rule, tol, breakdown, max_iter);
    return s;
}
void hook_stopper_free(void* p) { delete (lm::LanczosStopper*)p; }
void hook_stopper_gram_column(void* p, int m, const double* col) { ((lm::LanczosStopper*)p)->set_gram_column(m, col); }
int hook_stopper_feed(void* p, int k, double alpha, double beta) { return (int)((lm::LanczosStopper*)p)->feed(k, alpha, beta); }
void hook_stopper_advance(void* p) { ((lm::LanczosStopper*)p)->advance(); }
double hook_stopper_last_measure(void* p) { return ((lm::LanczosStopper*)p)->last_measure(); }
int hook_stopper_coefficients(void* p, double* c, int cap)
{
    auto& v = ((lm::LanczosStopper*)p)->c_cur;
    for (int i = 0; i < (int)v.size() && i < cap; ++i) c[i] = v[i];
    return (int)v.size();
}

// agree_on_stops with the transport supplied by the test (gloo: broadcast of words[0] from rank 0, max-reduction of words[1])
typedef void (*hook_exchange_fn)(unsigned* words);
unsigned hook_agree_on_stops(unsigned local_word, hook_exchange_fn exchange, int distributed)
{
    return lm::agree_on_stops(local_word, [&](unsigned* w) { exchange(w); }, distributed != 0);
}

}  // extern "C"
