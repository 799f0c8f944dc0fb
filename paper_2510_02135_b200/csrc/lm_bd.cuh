// lm_bd.cuh -- steric forces (eq. 13), random finite difference (eq. 11) and the Adams-Bashforth step (eq. 14) on the device.
// Included by lm_api.cu only, after lm_lanczos.cuh.
#pragma once

namespace {

// ---------------------------------------------------------------- steric forces and the BD step
template <typename T> int set_positions_t(lm_solver* h, const void* pos, cudaStream_t st);

template <typename T>
int steric_device(lm_solver* h, double U0, double b, const T* ext, T* out, cudaStream_t st)
{
    if (!h->steric_attr_set) {
        LM_CUDA(h, cudaFuncSetAttribute((const void*)steric_pair_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, steric_smem_bytes<T>()));
        h->steric_attr_set = true;
    }
    const int units = (int)(h->npad / STERIC_SUB);
    const int64_t rows = std::max<int64_t>(h->row_end - h->row_begin, 0);      // this rank's target rows (all rows unless sharded)
    const int i_tiles = (int)((rows + STERIC_TARGETS - 1) / STERIC_TARGETS);
    // about four resident sets of CTAs (2 per SM): the work per CTA depends on how many groups are within the cut-off
    const int splits = (int)std::max<int64_t>(1, std::min<int64_t>(units, ((int64_t)8 * h->sm_count + std::max(i_tiles, 1) - 1) / std::max(i_tiles, 1)));
    int rc = ensure(h, &h->partial, &h->partial_bytes, (size_t)splits * 3 * h->npad * sizeof(T));
    if (rc != LM_OK) return rc;
    const bool dist = h->dist_ranks > 0;
    const size_t seg = (size_t)3 * h->rows_per_rank;
    T* kout = out;
    if (dist) {
        if ((rc = ensure(h, &h->gath[0], &h->gath_bytes[0], seg * h->dist_ranks * sizeof(T))) != LM_OK) return rc;
        kout = (T*)h->gath[0];
    }
    const double K = sizeof(T) == 4 ? 20.0 : 40.0;           // exp(-K) below the type's epsilon
    StericParams<T> p;
    p.pos = (const T*)h->pos_soa;
    p.z_array = h->wall ? 3 : 2;                             // the forces act at the true heights, not the raised ones
    p.partial = (T*)h->partial;
    p.N = h->N;
    p.npad = h->npad;
    p.i_begin = h->row_begin;
    p.n_units = units;
    // lengths in the internal unit (x len_scale); the force magnitude U0 / b stays in the caller's units
    const double ls = h->len_scale, as = h->a * ls, bs = b * ls;
    p.tiny = make_consts<T>(h->eta, as, ls).tiny;
    p.d = (T)(2.0 * as);
    p.rc2 = (T)((2.0 * as + K * bs) * (2.0 * as + K * bs));
    p.m0 = (T)(U0 / b);
    p.inv_b = (T)(sizeof(T) == 4 ? 1.4426950408889634 / bs : 1.0 / bs);
    if (i_tiles > 0) {
        steric_pair_kernel<T><<<dim3(i_tiles, splits), STERIC_BLOCK, steric_smem_bytes<T>(), st>>>(p);
        // particle-wall repulsion: eq. (13) with d = a, heights in the internal unit
        steric_reduce_kernel<T><<<grid_1d(rows), VEC_BLOCK, 0, st>>>((const T*)h->partial, splits, h->row_begin, h->row_end, h->npad, ext, kout,
                                                                     h->wall ? (const T*)h->pos_soa + (size_t)3 * h->npad : nullptr, (T)as, (T)(U0 / b), (T)(1.0 / bs));
        h->n_aux += 2;
    }
    LM_CUDA(h, cudaGetLastError());
    if (dist) {                                              // row blocks -> every rank (as in launch_pair)
        NcclApi& nccl = nccl_api();
        const int nrc = nccl.AllGather(kout + seg * h->dist_rank, kout, seg, sizeof(T) == 4 ? NCCL_FLOAT32 : NCCL_FLOAT64, (NcclApi::Comm)h->nccl_comm, st);
        if (nrc != 0) return fail(h, LM_E_CUDA, std::string("ncclAllGather failed: ") + nccl.GetErrorString(nrc));
        LM_CUDA(h, cudaMemcpyAsync(out, kout, (size_t)3 * h->N * sizeof(T), cudaMemcpyDeviceToDevice, st));
    }
    return LM_OK;
}

// eq. (11): (1/delta) [ M(X + delta W/2) W - M(X - delta W/2) W ], one realisation
template <typename T>
int rfd_device(lm_solver* h, const T* W, double delta, T* lin_out, T* ang_out, cudaStream_t st)
{
    const int64_t n3 = 3 * h->N;
    int rc;
    if ((rc = ensure(h, &h->rfd[0], &h->rfd_bytes[0], (size_t)POS_ARRAYS * h->npad * sizeof(T))) != LM_OK) return rc;
    if ((rc = ensure(h, &h->rfd[1], &h->rfd_bytes[1], (size_t)n3 * sizeof(T))) != LM_OK) return rc;
    if (h->angular && (rc = ensure(h, &h->rfd[2], &h->rfd_bytes[2], (size_t)n3 * sizeof(T))) != LM_OK) return rc;
    void* const home = h->pos_soa;
    T* outs[2][2] = {{lin_out, ang_out}, {(T*)h->rfd[1], (T*)h->rfd[2]}};
    for (int side = 0; side < 2; ++side) {
        shift_positions_kernel<T><<<grid_1d(h->npad), VEC_BLOCK, 0, st>>>((const T*)home, W, h->N, h->npad, (T)((side ? -0.5 : 0.5) * delta * h->len_scale), wall_pack<T>(h), (T*)h->rfd[0]);
        h->n_aux++;
        h->pos_soa = h->rfd[0];                       // the apply reads the displaced copy; the handle's positions are untouched
        rc = apply_batch<T>(h, 1, W, nullptr, outs[side][0], h->angular ? outs[side][1] : nullptr, st);
        h->pos_soa = home;
        if (rc != LM_OK) return rc;
    }
    rfd_difference_kernel<T><<<grid_1d(n3), VEC_BLOCK, 0, st>>>(lin_out, (const T*)h->rfd[1], n3, (T)(1.0 / delta));
    if (h->angular) rfd_difference_kernel<T><<<grid_1d(n3), VEC_BLOCK, 0, st>>>(ang_out, (const T*)h->rfd[2], n3, (T)(1.0 / delta));
    h->n_aux += h->angular ? 2 : 1;
    LM_CUDA(h, cudaGetLastError());
    return LM_OK;
}

// rfd_noise != null (and kT > 0): the thermal-drift term of eq. (14), kT (d/dX).M^n, joins v_n as ONE random-finite-
// difference sample of eq. (11) with W~ = rfd_noise (zero mean for open boundaries, non-zero above a wall).
template <typename T>
int bd_step_device(lm_solver* h, T* pos, const T* ext_f, const T* ext_t, const T* noise, const T* rfd_noise, double rfd_delta, double dt, double kT,
                   double U0, double b, double tol, cudaStream_t st)
{
    const int64_t n3 = 3 * h->N;
    const size_t bytes = (size_t)n3 * sizeof(T);
    int rc;
    for (int k = 0; k < 6; ++k)
        if ((rc = ensure(h, &h->bd[k], &h->bd_bytes[k], bytes)) != LM_OK) return rc;
    const bool drift = rfd_noise && kT > 0.0;
    if (drift)
        for (int k = 7; k < 9; ++k)
            if ((rc = ensure(h, &h->bd[k], &h->bd_bytes[k], bytes)) != LM_OK) return rc;
    T *F = (T*)h->bd[0], *vn = (T*)h->bd[1], *vprev = (T*)h->bd[2], *y = (T*)h->bd[3], *ang = (T*)h->bd[4], *yang = (T*)h->bd[5];
    if ((rc = set_positions_t<T>(h, pos, st)) != LM_OK) return rc;
    // F^n = steric(X^n) + external;  v_n = M^n [F^n; T]
    const bool have_force = U0 != 0.0 || ext_f;
    if (U0 != 0.0) {
        if ((rc = steric_device<T>(h, U0, b, ext_f, F, st)) != LM_OK) return rc;
    }
    const T* Fin = U0 != 0.0 ? F : ext_f;
    const bool have_det = have_force || ext_t;
    int rc_noise = LM_OK;
    const bool noisy = noise && kT > 0.0;
    if (noisy && have_det && h->share_first_apply) {
        // v_n = M^n [F^n; T] rides along with the first Lanczos apply (one 2-right-hand-side launch)
        DetShare<T> det;
        det.f = Fin;
        det.t = ext_t;
        det.lin = vn;
        det.ang = h->angular ? ang : nullptr;
        rc_noise = lanczos_device<T>(h, 1, noise, tol, y, h->angular ? yang : nullptr, 1.0, 0, nullptr, st, &det);
        if (rc_noise != LM_OK && rc_noise != LM_E_NOCONV) return rc_noise;
    } else {
        if (have_det) {
            if ((rc = apply_batch<T>(h, 1, Fin, ext_t, vn, h->angular ? ang : nullptr, st)) != LM_OK) return rc;
        } else {
            LM_CUDA(h, cudaMemsetAsync(vn, 0, bytes, st));
        }
        if (noisy) {
            rc_noise = lanczos_device<T>(h, 1, noise, tol, y, h->angular ? yang : nullptr, 1.0, 0, nullptr, st);
            if (rc_noise != LM_OK && rc_noise != LM_E_NOCONV) return rc_noise;
        }
    }
    if (drift) {                                                     // v_n += kT * (one RFD sample of the divergence)
        T *dl = (T*)h->bd[7], *da = (T*)h->bd[8];
        if ((rc = rfd_device<T>(h, rfd_noise, rfd_delta, dl, h->angular ? da : nullptr, st)) != LM_OK) return rc;
        add_scaled_kernel<T><<<grid_1d(n3), VEC_BLOCK, 0, st>>>(vn, dl, (T)kT, n3);
        h->n_aux++;
    }
    const double cn = h->bd_have_prev ? 1.5 : 1.0, cp = h->bd_have_prev ? 0.5 : 0.0;
    bd_update_kernel<T><<<grid_1d(n3), VEC_BLOCK, 0, st>>>(pos, vn, vprev, noisy ? y : nullptr, n3, (T)(dt * cn), (T)(dt * cp),
                                                           (T)std::sqrt(2.0 * kT * dt));
    h->n_aux++;
    LM_CUDA(h, cudaGetLastError());
    h->bd_have_prev = true;
    if ((rc = set_positions_t<T>(h, pos, st)) != LM_OK) return rc;      // the handle follows the particles: packed copy = X^{n+1}
    return rc_noise;
}


}  // namespace
