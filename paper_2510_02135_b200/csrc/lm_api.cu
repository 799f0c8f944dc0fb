// lm_api.cu -- C ABI of liblm (include/lm.h).  One translation unit: the device kernels (rpy_pair.cuh,
// steric_pair.cuh, vector_kernels.cuh), then the host side in include order: lm_handle.cuh (state, launch
// chooser), lm_apply.cuh (one M.F apply), lm_lanczos.cuh (M^{1/2} W driver), lm_bd.cuh (eqs. 11, 13, 14),
// and below the typed front ends and the extern "C" entry points.
//
// Everything numerical runs in the kernels of rpy_pair.cuh / vector_kernels.cuh; the only host
// arithmetic is the k x k tridiagonal problem of the Lanczos stopping test (tridiag_host.h).
// There is no CPU fallback: without a CUDA device every compute call returns LM_E_CUDA.
#include <cuda_runtime.h>
#include <dlfcn.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <type_traits>
#include <vector>

#include "../../include/lm.h"
#include "rpy_pair.cuh"
#include "rpy_small.cuh"
#include "steric_pair.cuh"
#include "lanczos_host.h"
#include "tridiag_host.h"
#include "vector_kernels.cuh"

#include "lm_handle.cuh"
#include "lm_apply.cuh"
#include "lm_lanczos.cuh"
#include "lm_bd.cuh"

namespace {

// ---------------------------------------------------------------- typed front ends
template <typename T> int set_positions_t(lm_solver* h, const void* pos, cudaStream_t st)
{
    pack_positions_kernel<T><<<grid_1d(h->npad), VEC_BLOCK, 0, st>>>((const T*)pos, h->N, h->npad, (T)h->len_scale, wall_pack<T>(h), (T*)h->pos_soa);
    h->n_aux++;
    LM_CUDA(h, cudaGetLastError());
    h->have_pos = true;
    return LM_OK;
}

int check_io(lm_solver* h, const void* forces, const void* torques, const void* lin_out, const void* ang_out, bool need_input)
{
    if (!h) return LM_E_NULL;
    h->err.clear();
    if (!h->have_pos) return fail(h, LM_E_NOPOS, "positions not set: call lm_set_positions first");
    if (!lin_out) return fail(h, LM_E_NULL, "lin_out is NULL");
    if (!h->angular && (torques || ang_out)) return fail(h, LM_E_ANGULAR, "torques / ang_out given but the solver was created with include_angular = 0");
    if (h->angular && !ang_out) return fail(h, LM_E_ANGULAR, "include_angular = 1 requires ang_out");
    if (need_input && !forces && !torques) return fail(h, LM_E_NULL, "forces and torques are both NULL");
    return LM_OK;
}

int stage_in(lm_solver* h, int slot, const void* host, size_t bytes, cudaStream_t st, void** dev)
{
    *dev = nullptr;
    if (!host) return LM_OK;
    int rc = ensure(h, &h->st[slot], &h->st_bytes[slot], bytes);
    if (rc != LM_OK) return rc;
    LM_CUDA(h, cudaMemcpyAsync(h->st[slot], host, bytes, cudaMemcpyHostToDevice, st));
    *dev = h->st[slot];
    return LM_OK;
}
int stage_out_alloc(lm_solver* h, int slot, const void* host, size_t bytes, void** dev)
{
    *dev = nullptr;
    if (!host) return LM_OK;
    int rc = ensure(h, &h->st[slot], &h->st_bytes[slot], bytes);
    if (rc != LM_OK) return rc;
    *dev = h->st[slot];
    return LM_OK;
}

}  // namespace

// ================================================================ C ABI
extern "C" {

const char* lm_version(void) { return "liblm 0.2 (sm_100a)"; }

int lm_create(lm_solver** out, int precision, int64_t N, double eta, double a, int include_angular)
{
    if (!out) return LM_E_NULL;
    *out = nullptr;
    if ((precision != LM_F32 && precision != LM_F64) || N <= 0 || !(eta > 0.0) || !(a > 0.0) || !std::isfinite(eta) || !std::isfinite(a))
        return LM_E_INVALID;
    if (N > (int64_t)1 << 28) return LM_E_INVALID;
    lm_solver* h = new lm_solver();
    h->precision = precision;
    h->N = N;
    h->eta = eta;
    h->a = a;
    h->angular = include_angular ? 1 : 0;
    h->len_scale = std::ldexp(1.0, -(int)std::lround(std::log2(a)));      // power of two nearest 1/a
    if (precision == LM_F32 && (h->len_scale > 0x1p100 || h->len_scale < 0x1p-100)) { delete h; return LM_E_INVALID; }   // a outside fp32's comfortable range
    h->npad = (N + NPAD_QUANTUM - 1) / NPAD_QUANTUM * NPAD_QUANTUM;
    h->row_begin = 0;
    h->row_end = N;
    auto bail = [&](int code) { lm_destroy(h); return code; };
    if (cudaGetDevice(&h->device) != cudaSuccess) return bail(LM_E_CUDA);
    if (cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, h->device) != cudaSuccess) return bail(LM_E_CUDA);
    if (cudaMalloc(&h->pos_soa, (size_t)POS_ARRAYS * h->npad * esize(h)) != cudaSuccess) return bail(LM_E_CUDA);
    const int rc = precision == LM_F32 ? init_variants<float>(h) : init_variants<double>(h);
    if (rc != LM_OK) return bail(rc);
    *out = h;
    return LM_OK;
}

int lm_destroy(lm_solver* h)
{
    if (!h) return LM_OK;
    cudaFree(h->pos_soa);
    cudaFree(h->vec_soa);
    cudaFree(h->partial);
    cudaFree(h->V);
    cudaFree(h->w);
    cudaFree(h->d_scal);
    cudaFree(h->d_block);
    cudaFree(h->d_ticket);
    cudaFree(h->d_coef);
    cudaFree(h->d_gram_part);
    cudaFree(h->d_newest);
    cudaFree(h->d_word);
    if (h->h_word) cudaFreeHost(h->h_word);
    if (h->h_gram) cudaFreeHost(h->h_gram);
    if (h->h_ab) cudaFreeHost(h->h_ab);
    if (h->lz_graph) cudaGraphExecDestroy(h->lz_graph);
    for (auto& g : h->apply_graph) if (g.exec) cudaGraphExecDestroy(g.exec);
    if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
    for (void* p : h->st) cudaFree(p);
    for (void* p : h->bd) cudaFree(p);
    for (void* p : h->rfd) cudaFree(p);
    for (void* p : h->gath) cudaFree(p);
    if (h->nccl_comm && nccl_api().ok) nccl_api().CommDestroy((NcclApi::Comm)h->nccl_comm);
    for (auto e : h->lz_ev) if (e) cudaEventDestroy(e);
    for (auto& pr : h->pending) { cudaEventDestroy(pr.first); cudaEventDestroy(pr.second); }
    for (auto e : h->event_pool) cudaEventDestroy(e);
    cudaGetLastError();
    delete h;
    return LM_OK;
}

const char* lm_last_error(const lm_solver* h) { return h ? h->err.c_str() : "null handle"; }

int lm_set_max_iter(lm_solver* h, int max_iter)
{
    if (!h) return LM_E_NULL;
    if (max_iter < 1 || max_iter > 1000) return fail(h, LM_E_INVALID, "max_iter must be in [1, 1000]");
    h->max_iter = max_iter;
    return LM_OK;
}

int lm_last_iterations(const lm_solver* h) { return h ? h->last_iters : -1; }

int lm_set_wall(lm_solver* h, int enabled, double wall_height)
{
    if (!h) return LM_E_NULL;
    h->err.clear();
    if (!std::isfinite(wall_height)) return fail(h, LM_E_INVALID, "wall_height must be finite");
    h->wall = enabled ? 1 : 0;
    h->wall_z = wall_height;
    h->have_pos = false;                              // the packed copy (raised heights, damping factors) depends on the wall
    h->bd_have_prev = false;
    for (auto& slot : h->plan_cache) slot.valid = false;
    for (auto& slot : h->small_cache) slot.valid = false;
    return LM_OK;
}

int lm_set_option(lm_solver* h, int option, int value)
{
    if (!h) return LM_E_NULL;
    h->err.clear();
    switch (option) {
    case LM_OPT_LANCZOS_RULE:
        if (value != LM_RULE_ESTIMATE && value != LM_RULE_STEP) return fail(h, LM_E_INVALID, "LM_OPT_LANCZOS_RULE: LM_RULE_ESTIMATE or LM_RULE_STEP");
        h->lz_rule = value;
        return LM_OK;
    case LM_OPT_GRAPH_REPLAY: h->graph_replay = value != 0; return LM_OK;
    case LM_OPT_SHARE_FIRST_APPLY: h->share_first_apply = value != 0; return LM_OK;
    case LM_OPT_ACCUMULATE_F64:
        if (h->precision != LM_F32 && value != 0) return fail(h, LM_E_INVALID, "LM_OPT_ACCUMULATE_F64 is for fp32 handles (an fp64 handle accumulates in fp64 anyway)");
        h->acc64 = value != 0;
        for (auto& slot : h->plan_cache) slot.valid = false;
        for (auto& slot : h->small_cache) slot.valid = false;
        return LM_OK;
    case LM_OPT_GATHER_IN_PLACE: h->gather_in_caller = value != 0; return LM_OK;
    case LM_OPT_J_SPLITS:
        if (value < 0) return fail(h, LM_E_INVALID, "LM_OPT_J_SPLITS: 0 (chosen by the library) or the number of j-splits");
        h->force_splits = value;
        for (auto& slot : h->plan_cache) slot.valid = false;
        return LM_OK;
    case LM_OPT_SMALL_KERNEL: {
        const int S = value >> 8, W = value & 255;
        const bool shape = value > 1 && (S == 1 || S == 2 || S == 4 || S == 8) && (W == 1 || W == 2 || W == 4 || W == 8);
        if (value != 0 && value != 1 && !shape) return fail(h, LM_E_INVALID, "LM_OPT_SMALL_KERNEL: 0, 1 or (cluster << 8 | warps) with cluster, warps in {1, 2, 4, 8}");
        h->small_kernel = value;
        return LM_OK;
    }
    default: return fail(h, LM_E_INVALID, "unknown option");
    }
}

int lm_lanczos_history(const lm_solver* h, int vec, int cap, double* alpha, double* beta, double* step, double* estimate)
{
    if (!h) return LM_E_NULL;
    if (vec < 0 || vec >= (int)h->lz_stop.size()) return 0;
    const LanczosStopper& s = h->lz_stop[vec];
    const int k = (int)s.alphas.size();
    for (int i = 0; i < k && i < cap; ++i) {
        // iteration i + 1: alpha and beta; the relative step exists from k = 2, the estimate from k = 3
        if (alpha) alpha[i] = s.alphas[i];
        if (beta) beta[i] = i < (int)s.betas.size() ? s.betas[i] : s.pending_beta;
        if (step) step[i] = i >= 1 && i - 1 < (int)s.steps.size() ? s.steps[i - 1] : NAN;
        if (estimate) estimate[i] = i >= 2 && i - 2 < (int)s.estimates.size() ? s.estimates[i - 2] : NAN;
    }
    return k;
}

int lm_set_positions(lm_solver* h, const void* pos, void* stream)
{
    if (!h) return LM_E_NULL;
    h->err.clear();
    if (!pos) return fail(h, LM_E_NULL, "pos is NULL");
    cudaStream_t st = (cudaStream_t)stream;
    return h->precision == LM_F32 ? set_positions_t<float>(h, pos, st) : set_positions_t<double>(h, pos, st);
}

int lm_mdot_batch(lm_solver* h, int nrhs, const void* forces, const void* torques, void* lin_out, void* ang_out, void* stream)
{
    int rc = check_io(h, forces, torques, lin_out, ang_out, true);
    if (rc != LM_OK) return rc;
    if (nrhs < 1) return fail(h, LM_E_INVALID, "nrhs must be >= 1");
    cudaStream_t st = (cudaStream_t)stream;
    if (h->precision == LM_F32) return apply_batch<float>(h, nrhs, (const float*)forces, (const float*)torques, (float*)lin_out, (float*)ang_out, st);
    return apply_batch<double>(h, nrhs, (const double*)forces, (const double*)torques, (double*)lin_out, (double*)ang_out, st);
}

int lm_mdot(lm_solver* h, const void* forces, const void* torques, void* lin_out, void* ang_out, void* stream)
{
    return lm_mdot_batch(h, 1, forces, torques, lin_out, ang_out, stream);
}

int lm_sqrt_mdot_w(lm_solver* h, const void* noise, double tol, void* lin_out, void* ang_out, int* iters_out, void* stream)
{
    int rc = check_io(h, noise, nullptr, lin_out, ang_out, false);
    if (rc != LM_OK) return rc;
    if (!noise) return fail(h, LM_E_NULL, "noise is NULL");
    if (!(tol > 0.0) || !std::isfinite(tol)) return fail(h, LM_E_INVALID, "tol must be > 0");
    cudaStream_t st = (cudaStream_t)stream;
    rc = h->precision == LM_F32 ? lanczos_device<float>(h, 1, (const float*)noise, tol, (float*)lin_out, (float*)ang_out, 1.0, 0, nullptr, st)
                                : lanczos_device<double>(h, 1, (const double*)noise, tol, (double*)lin_out, (double*)ang_out, 1.0, 0, nullptr, st);
    if (iters_out) *iters_out = h->last_iters;
    return rc;
}

int lm_sqrt_mdot_w_batch(lm_solver* h, int nvec, const void* noise, double tol, void* lin_out, void* ang_out, int* iters_out, void* stream)
{
    int rc = check_io(h, noise, nullptr, lin_out, ang_out, false);
    if (rc != LM_OK) return rc;
    if (!noise) return fail(h, LM_E_NULL, "noise is NULL");
    if (nvec < 1) return fail(h, LM_E_INVALID, "nvec must be >= 1");
    if (!(tol > 0.0) || !std::isfinite(tol)) return fail(h, LM_E_INVALID, "tol must be > 0");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t es = esize(h);
    const int64_t dof = dof_of(h), n3 = 3 * h->N;
    int worst = LM_OK, max_iters = 0;
    std::string noconv;
    // groups of 4, 2, 1 vectors (angular or single wall: 2, 1): the right-hand-side counts the pair kernel is built for
    for (int q = 0; q < nvec;) {
        int g = nvec - q >= 4 ? 4 : (nvec - q >= 2 ? 2 : 1);
        if ((h->angular || h->wall) && g > 2) g = 2;
        const char* nz = (const char*)noise + (size_t)q * dof * es;
        char* lo = (char*)lin_out + (size_t)q * n3 * es;
        char* ao = ang_out ? (char*)ang_out + (size_t)q * n3 * es : nullptr;
        int* it = iters_out ? iters_out + q : nullptr;
        rc = h->precision == LM_F32 ? lanczos_device<float>(h, g, (const float*)nz, tol, (float*)lo, (float*)ao, 1.0, 0, it, st)
                                    : lanczos_device<double>(h, g, (const double*)nz, tol, (double*)lo, (double*)ao, 1.0, 0, it, st);
        if (rc == LM_E_NOCONV) { worst = rc; noconv = h->err; }
        else if (rc != LM_OK) return rc;
        max_iters = std::max(max_iters, h->last_iters);
        q += g;
    }
    h->last_iters = max_iters;
    if (worst != LM_OK) h->err = noconv;
    return worst;
}

}  // extern "C"

namespace {

// out = M.[F;T] + prefactor M^{1/2} W: the deterministic right-hand side rides along with the first Lanczos apply
// (one 2-right-hand-side launch) where a variant for it exists; otherwise M.[F;T] is a launch of its own
template <typename T>
int hydrodynamic_velocities_t(lm_solver* h, const T* forces, const T* torques, const T* noise, double noise_prefactor, double tol, T* lin_out, T* ang_out,
                              cudaStream_t st)
{
    const bool have_det = forces || torques;
    if (!noise) return apply_batch<T>(h, 1, forces, torques, lin_out, ang_out, st);
    if (!have_det) return lanczos_device<T>(h, 1, noise, tol, lin_out, ang_out, noise_prefactor, 0, nullptr, st);
    DetShare<T> det;
    det.f = forces;
    det.t = torques;
    det.lin = lin_out;
    det.ang = ang_out;
    if (!h->share_first_apply) {
        const int rc = apply_batch<T>(h, 1, forces, torques, lin_out, ang_out, st);
        if (rc != LM_OK) return rc;
        return lanczos_device<T>(h, 1, noise, tol, lin_out, ang_out, noise_prefactor, 1, nullptr, st);
    }
    // the Lanczos result is accumulated onto lin_out / ang_out at the end, after the shared launch has written M.[F;T] there
    return lanczos_device<T>(h, 1, noise, tol, lin_out, ang_out, noise_prefactor, 1, nullptr, st, &det);
}

}  // namespace

extern "C" {

int lm_hydrodynamic_velocities(lm_solver* h, const void* forces, const void* torques, const void* noise, double noise_prefactor, double tol,
                               void* lin_out, void* ang_out, void* stream)
{
    int rc = check_io(h, forces, torques, lin_out, ang_out, noise == nullptr);
    if (rc != LM_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if (noise && (!(tol > 0.0) || !std::isfinite(tol))) return fail(h, LM_E_INVALID, "tol must be > 0");
    return h->precision == LM_F32
               ? hydrodynamic_velocities_t<float>(h, (const float*)forces, (const float*)torques, (const float*)noise, noise_prefactor, tol, (float*)lin_out,
                                                  (float*)ang_out, st)
               : hydrodynamic_velocities_t<double>(h, (const double*)forces, (const double*)torques, (const double*)noise, noise_prefactor, tol,
                                                   (double*)lin_out, (double*)ang_out, st);
}

// ---------------------------------------------------------------- host-pointer variants
int lm_set_positions_host(lm_solver* h, const void* pos, void* stream)
{
    if (!h) return LM_E_NULL;
    h->err.clear();
    if (!pos) return fail(h, LM_E_NULL, "pos is NULL");
    cudaStream_t st = (cudaStream_t)stream;
    void* d = nullptr;
    int rc = stage_in(h, 0, pos, (size_t)3 * h->N * esize(h), st, &d);
    if (rc != LM_OK) return rc;
    rc = lm_set_positions(h, d, stream);
    if (rc != LM_OK) return rc;
    LM_CUDA(h, cudaStreamSynchronize(st));
    return LM_OK;
}

int lm_mdot_batch_host(lm_solver* h, int nrhs, const void* forces, const void* torques, void* lin_out, void* ang_out, void* stream)
{
    int rc = check_io(h, forces, torques, lin_out, ang_out, true);
    if (rc != LM_OK) return rc;
    if (nrhs < 1) return fail(h, LM_E_INVALID, "nrhs must be >= 1");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = (size_t)nrhs * 3 * h->N * esize(h);
    void *df, *dt, *dl, *da;
    if ((rc = stage_in(h, 1, forces, bytes, st, &df)) != LM_OK) return rc;
    if ((rc = stage_in(h, 2, torques, bytes, st, &dt)) != LM_OK) return rc;
    if ((rc = stage_out_alloc(h, 4, lin_out, bytes, &dl)) != LM_OK) return rc;
    if ((rc = stage_out_alloc(h, 5, ang_out, bytes, &da)) != LM_OK) return rc;
    if ((rc = lm_mdot_batch(h, nrhs, df, dt, dl, da, stream)) != LM_OK) return rc;
    LM_CUDA(h, cudaMemcpyAsync(lin_out, dl, bytes, cudaMemcpyDeviceToHost, st));
    if (ang_out) LM_CUDA(h, cudaMemcpyAsync(ang_out, da, bytes, cudaMemcpyDeviceToHost, st));
    LM_CUDA(h, cudaStreamSynchronize(st));
    return LM_OK;
}

int lm_mdot_host(lm_solver* h, const void* forces, const void* torques, void* lin_out, void* ang_out, void* stream)
{
    return lm_mdot_batch_host(h, 1, forces, torques, lin_out, ang_out, stream);
}

int lm_hydrodynamic_velocities_host(lm_solver* h, const void* forces, const void* torques, const void* noise, double noise_prefactor,
                                    double tol, void* lin_out, void* ang_out, void* stream)
{
    int rc = check_io(h, forces, torques, lin_out, ang_out, noise == nullptr);
    if (rc != LM_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = (size_t)3 * h->N * esize(h);
    void *df, *dt, *dn, *dl, *da;
    if ((rc = stage_in(h, 1, forces, bytes, st, &df)) != LM_OK) return rc;
    if ((rc = stage_in(h, 2, torques, bytes, st, &dt)) != LM_OK) return rc;
    if ((rc = stage_in(h, 3, noise, (size_t)dof_of(h) * esize(h), st, &dn)) != LM_OK) return rc;
    if ((rc = stage_out_alloc(h, 4, lin_out, bytes, &dl)) != LM_OK) return rc;
    if ((rc = stage_out_alloc(h, 5, ang_out, bytes, &da)) != LM_OK) return rc;
    rc = lm_hydrodynamic_velocities(h, df, dt, dn, noise_prefactor, tol, dl, da, stream);
    if (rc != LM_OK && rc != LM_E_NOCONV) return rc;
    LM_CUDA(h, cudaMemcpyAsync(lin_out, dl, bytes, cudaMemcpyDeviceToHost, st));
    if (ang_out) LM_CUDA(h, cudaMemcpyAsync(ang_out, da, bytes, cudaMemcpyDeviceToHost, st));
    LM_CUDA(h, cudaStreamSynchronize(st));
    return rc;
}

int lm_sqrt_mdot_w_host(lm_solver* h, const void* noise, double tol, void* lin_out, void* ang_out, int* iters_out, void* stream)
{
    if (h && !noise) { h->err.clear(); return fail(h, LM_E_NULL, "noise is NULL"); }
    const int rc = lm_hydrodynamic_velocities_host(h, nullptr, nullptr, noise, 1.0, tol, lin_out, ang_out, stream);
    if (iters_out && h) *iters_out = h->last_iters;
    return rc;
}

// ---------------------------------------------------------------- Brownian-dynamics step (eqs. (13), (14))
int lm_steric_forces(lm_solver* h, double U0, double b, const void* ext_forces, void* forces_out, void* stream)
{
    if (!h) return LM_E_NULL;
    h->err.clear();
    if (!h->have_pos) return fail(h, LM_E_NOPOS, "positions not set: call lm_set_positions first");
    if (!forces_out) return fail(h, LM_E_NULL, "forces_out is NULL");
    if (!(b > 0.0) || !std::isfinite(b) || !std::isfinite(U0)) return fail(h, LM_E_INVALID, "steric potential needs b > 0 and finite U0");
    cudaStream_t st = (cudaStream_t)stream;
    return h->precision == LM_F32 ? steric_device<float>(h, U0, b, (const float*)ext_forces, (float*)forces_out, st)
                                  : steric_device<double>(h, U0, b, (const double*)ext_forces, (double*)forces_out, st);
}

int lm_bd_reset(lm_solver* h)
{
    if (!h) return LM_E_NULL;
    h->bd_have_prev = false;
    return LM_OK;
}

int lm_bd_step_rfd(lm_solver* h, void* pos, const void* ext_forces, const void* ext_torques, const void* noise, const void* rfd_noise,
                   double rfd_delta, double dt, double kT, double U0, double b, double tol, void* stream)
{
    if (!h) return LM_E_NULL;
    h->err.clear();
    if (!pos) return fail(h, LM_E_NULL, "pos is NULL");
    if (!h->angular && ext_torques) return fail(h, LM_E_ANGULAR, "torques given but the solver was created with include_angular = 0");
    if (!(dt > 0.0) || !std::isfinite(dt) || !(kT >= 0.0) || !std::isfinite(kT)) return fail(h, LM_E_INVALID, "dt must be > 0 and kT >= 0");
    if (U0 != 0.0 && (!(b > 0.0) || !std::isfinite(b) || !std::isfinite(U0))) return fail(h, LM_E_INVALID, "steric potential needs b > 0 and finite U0");
    if (noise && kT > 0.0 && (!(tol > 0.0) || !std::isfinite(tol))) return fail(h, LM_E_INVALID, "tol must be > 0");
    if (rfd_noise && kT > 0.0 && (!(rfd_delta > 0.0) || !std::isfinite(rfd_delta))) return fail(h, LM_E_INVALID, "rfd_delta must be > 0");
    cudaStream_t st = (cudaStream_t)stream;
    return h->precision == LM_F32
               ? bd_step_device<float>(h, (float*)pos, (const float*)ext_forces, (const float*)ext_torques, (const float*)noise, (const float*)rfd_noise,
                                       rfd_delta, dt, kT, U0, b, tol, st)
               : bd_step_device<double>(h, (double*)pos, (const double*)ext_forces, (const double*)ext_torques, (const double*)noise,
                                        (const double*)rfd_noise, rfd_delta, dt, kT, U0, b, tol, st);
}

int lm_bd_step(lm_solver* h, void* pos, const void* ext_forces, const void* ext_torques, const void* noise, double dt, double kT, double U0,
               double b, double tol, void* stream)
{
    return lm_bd_step_rfd(h, pos, ext_forces, ext_torques, noise, nullptr, 0.0, dt, kT, U0, b, tol, stream);
}

int lm_bd_step_rfd_host(lm_solver* h, void* pos, const void* ext_forces, const void* ext_torques, const void* noise, const void* rfd_noise,
                        double rfd_delta, double dt, double kT, double U0, double b, double tol, void* stream)
{
    if (!h) return LM_E_NULL;
    h->err.clear();
    if (!pos) return fail(h, LM_E_NULL, "pos is NULL");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = (size_t)3 * h->N * esize(h);
    void *dp = nullptr, *df, *dt_, *dn, *dr;
    int rc = ensure(h, &h->bd[6], &h->bd_bytes[6], bytes);
    if (rc != LM_OK) return rc;
    dp = h->bd[6];
    LM_CUDA(h, cudaMemcpyAsync(dp, pos, bytes, cudaMemcpyHostToDevice, st));
    if ((rc = stage_in(h, 1, ext_forces, bytes, st, &df)) != LM_OK) return rc;
    if ((rc = stage_in(h, 2, ext_torques, bytes, st, &dt_)) != LM_OK) return rc;
    if ((rc = stage_in(h, 3, noise, (size_t)dof_of(h) * esize(h), st, &dn)) != LM_OK) return rc;
    if ((rc = stage_in(h, 4, rfd_noise, bytes, st, &dr)) != LM_OK) return rc;      // slot 4 (lin staging) is free in this call
    rc = lm_bd_step_rfd(h, dp, df, dt_, dn, dr, rfd_delta, dt, kT, U0, b, tol, stream);
    if (rc != LM_OK && rc != LM_E_NOCONV) return rc;
    LM_CUDA(h, cudaMemcpyAsync(pos, dp, bytes, cudaMemcpyDeviceToHost, st));
    LM_CUDA(h, cudaStreamSynchronize(st));
    return rc;
}

int lm_bd_step_host(lm_solver* h, void* pos, const void* ext_forces, const void* ext_torques, const void* noise, double dt, double kT,
                    double U0, double b, double tol, void* stream)
{
    return lm_bd_step_rfd_host(h, pos, ext_forces, ext_torques, noise, nullptr, 0.0, dt, kT, U0, b, tol, stream);
}

// ---------------------------------------------------------------- thermal drift
int lm_thermal_drift(lm_solver* h, void* lin_out, void* ang_out, void* stream)
{
    int rc = check_io(h, nullptr, nullptr, lin_out, ang_out, false);
    if (rc != LM_OK) return rc;
    // above a wall the divergence of the mobility is NOT zero: zeros would be silently wrong physics
    if (h->wall)
        return fail(h, LM_E_INVALID, "lm_thermal_drift is the zero default of open boundaries; with lm_set_wall use lm_thermal_drift_rfd or lm_bd_step_rfd (eq. 11)");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = (size_t)3 * h->N * esize(h);
    LM_CUDA(h, cudaMemsetAsync(lin_out, 0, bytes, st));
    if (h->angular) LM_CUDA(h, cudaMemsetAsync(ang_out, 0, bytes, st));
    return LM_OK;
}

int lm_thermal_drift_rfd(lm_solver* h, const void* noise, double delta, void* lin_out, void* ang_out, void* stream)
{
    int rc = check_io(h, noise, nullptr, lin_out, ang_out, false);
    if (rc != LM_OK) return rc;
    if (!noise) return fail(h, LM_E_NULL, "noise is NULL");
    if (!(delta > 0.0) || !std::isfinite(delta)) return fail(h, LM_E_INVALID, "delta must be > 0");
    cudaStream_t st = (cudaStream_t)stream;
    return h->precision == LM_F32 ? rfd_device<float>(h, (const float*)noise, delta, (float*)lin_out, (float*)ang_out, st)
                                  : rfd_device<double>(h, (const double*)noise, delta, (double*)lin_out, (double*)ang_out, st);
}

// ---------------------------------------------------------------- row-sharded applies
int lm_dist_row_block(int64_t N, int nranks, int rank, int64_t* row_begin, int64_t* row_end)
{
    if (N <= 0 || nranks < 1 || rank < 0 || rank >= nranks) return LM_E_INVALID;
    const int64_t B = (N + nranks - 1) / nranks;
    if (row_begin) *row_begin = std::min<int64_t>(N, (int64_t)rank * B);
    if (row_end) *row_end = std::min<int64_t>(N, (int64_t)(rank + 1) * B);
    return LM_OK;
}

int lm_dist_unique_id(void* out128)
{
    if (!out128) return LM_E_NULL;
    NcclApi& nccl = nccl_api();
    if (!nccl.ok) return LM_E_CUDA;
    NcclApi::UniqueId id;
    if (nccl.GetUniqueId(&id) != 0) return LM_E_CUDA;
    std::memcpy(out128, id.internal, sizeof id.internal);
    return LM_OK;
}

int lm_dist_init(lm_solver* h, int nranks, int rank, const void* unique_id128)
{
    if (!h) return LM_E_NULL;
    h->err.clear();
    if (!unique_id128) return fail(h, LM_E_NULL, "unique id is NULL");
    if (h->dist_ranks > 0) return fail(h, LM_E_INVALID, "lm_dist_init was already called on this handle");
    int64_t b = 0, e = 0;
    if (lm_dist_row_block(h->N, nranks, rank, &b, &e) != LM_OK) return fail(h, LM_E_INVALID, "need 0 <= rank < nranks");
    NcclApi& nccl = nccl_api();
    if (!nccl.ok) return fail(h, LM_E_CUDA, "NCCL unavailable: " + nccl.why);
    NcclApi::UniqueId id;
    std::memcpy(id.internal, unique_id128, sizeof id.internal);
    NcclApi::Comm comm = nullptr;
    const int nrc = nccl.CommInitRank(&comm, nranks, id, rank);
    if (nrc != 0) return fail(h, LM_E_CUDA, std::string("ncclCommInitRank failed: ") + nccl.GetErrorString(nrc));
    h->nccl_comm = comm;
    h->dist_ranks = nranks;
    h->dist_rank = rank;
    h->rows_per_rank = (h->N + nranks - 1) / nranks;
    h->row_begin = b;
    h->row_end = e;
    return LM_OK;
}

int lm_mdot_rows(lm_solver* h, int64_t row_begin, int64_t row_count, const void* forces, const void* torques, void* lin_out, void* ang_out,
                 void* stream)
{
    if (!h) return LM_E_NULL;
    h->err.clear();
    if (h->dist_ranks > 0) return fail(h, LM_E_INVALID, "lm_mdot_rows is for handles without a communicator (lm_dist_init shards by itself)");
    if (row_begin < 0 || row_count < 0 || row_begin + row_count > h->N) return fail(h, LM_E_INVALID, "row range outside [0, N)");
    h->row_begin = row_begin;
    h->row_end = row_begin + row_count;
    const int rc = lm_mdot_batch(h, 1, forces, torques, lin_out, ang_out, stream);
    h->row_begin = 0;
    h->row_end = h->N;
    return rc;
}

// ---------------------------------------------------------------- stats / introspection
int lm_set_profiling(lm_solver* h, int on)
{
    if (!h) return LM_E_NULL;
    h->profiling = on != 0;
    return LM_OK;
}

static int drain_events(lm_solver* h)
{
    for (auto& pr : h->pending) {
        LM_CUDA(h, cudaEventSynchronize(pr.second));
        float ms = 0.f;
        LM_CUDA(h, cudaEventElapsedTime(&ms, pr.first, pr.second));
        h->pair_ms += ms;
        h->event_pool.push_back(pr.first);
        h->event_pool.push_back(pr.second);
    }
    h->pending.clear();
    return LM_OK;
}

int lm_reset_stats(lm_solver* h)
{
    if (!h) return LM_E_NULL;
    const int rc = drain_events(h);
    h->n_pair = h->n_aux = 0;
    h->pairs = h->pair_ms = 0.0;
    return rc;
}

int lm_get_stats(lm_solver* h, int64_t* pair_kernel_launches, int64_t* aux_launches, double* pair_kernel_ms, double* pairs)
{
    if (!h) return LM_E_NULL;
    const int rc = drain_events(h);
    if (pair_kernel_launches) *pair_kernel_launches = h->n_pair;
    if (aux_launches) *aux_launches = h->n_aux;
    if (pair_kernel_ms) *pair_kernel_ms = h->pair_ms;
    if (pairs) *pairs = h->pairs;
    return rc;
}

const char* lm_pair_kernel_name(lm_solver* h, int nrhs)
{
    if (!h) return "";
    const SmallPlan sp = h->precision == LM_F32 ? choose_small<float>(h, nrhs) : choose_small<double>(h, nrhs);
    if (sp.variant >= 0) return "rpy_small_kernel";
    const LaunchPlan plan = h->precision == LM_F32 ? choose_plan<float>(h, nrhs) : choose_plan<double>(h, nrhs);
    return plan.variant >= 0 ? "rpy_pair_kernel" : "";
}

int lm_pair_launch_config(lm_solver* h, int nrhs, int* i_tiles, int* j_splits, int* block, int* targets_per_thread, int* smem_bytes)
{
    if (!h) return LM_E_NULL;
    const SmallPlan sp = h->precision == LM_F32 ? choose_small<float>(h, nrhs) : choose_small<double>(h, nrhs);
    if (sp.variant >= 0) {            // the one-launch kernel: j is split over the `cluster` CTAs of a cluster (and over each CTA's warps)
        if (i_tiles) *i_tiles = sp.i_tiles;
        if (j_splits) *j_splits = sp.cluster;
        if (block) *block = sp.warps * 32;
        if (targets_per_thread) *targets_per_thread = 2;
        if (smem_bytes) *smem_bytes = (int)sp.smem;
        return LM_OK;
    }
    LaunchPlan plan;
    int blk = 0, tpt = 0, smem = 0;
    if (h->precision == LM_F32) {
        plan = choose_plan<float>(h, nrhs);
        if (plan.variant >= 0) { blk = h->vf[plan.variant].block; tpt = h->vf[plan.variant].tpt; smem = h->vf[plan.variant].smem; }
    } else {
        plan = choose_plan<double>(h, nrhs);
        if (plan.variant >= 0) { blk = h->vd[plan.variant].block; tpt = h->vd[plan.variant].tpt; smem = h->vd[plan.variant].smem; }
    }
    if (plan.variant < 0) return fail(h, LM_E_INVALID, "no pair-kernel variant for this nrhs (use 1, 2 or 4; angular: 1 or 2)");
    if (i_tiles) *i_tiles = plan.i_tiles;
    if (j_splits) *j_splits = plan.j_splits;
    if (block) *block = blk;
    if (targets_per_thread) *targets_per_thread = tpt;
    if (smem_bytes) *smem_bytes = smem;
    return LM_OK;
}

}  // extern "C"
