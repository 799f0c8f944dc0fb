// lm_lanczos.cuh -- host driver of the Lanczos iteration for M^{1/2} W.
// Included by lm_api.cu only, after lm_apply.cuh.  The stopping test itself lives in lanczos_host.h.
#pragma once

namespace {

// One deterministic right-hand side [F;T] whose product M.[F;T] rides along with the FIRST Lanczos apply in one
// multi-right-hand-side launch (eq. (9) PAPER.md:78 / the sum of PAPER.md:137-138 needs both; SURVEY.md sec. 7
// step 7): the pair geometry of that launch is evaluated once for the two vectors.
template <typename T> struct DetShare {
    const T* f = nullptr;      // 3N forces or null
    const T* t = nullptr;      // 3N torques or null
    T* lin = nullptr;          // 3N: receives M.[F;T] (linear rows)
    T* ang = nullptr;          // 3N (angular handles)
};

// the transport of agree_on_stops (lanczos_host.h) in a row-sharded run: words[0] <- rank 0's stop bits (ncclBroadcast),
// words[1] <- max over ranks of the failure flags (ncclAllReduce), both in one NCCL group
int exchange_words(lm_solver* h, unsigned* words, cudaStream_t st)
{
    if (!h->d_word) {
        LM_CUDA(h, cudaMalloc((void**)&h->d_word, 2 * sizeof(unsigned)));
        LM_CUDA(h, cudaHostAlloc((void**)&h->h_word, 2 * sizeof(unsigned), cudaHostAllocDefault));
    }
    NcclApi& nccl = nccl_api();
    h->h_word[0] = words[0];
    h->h_word[1] = words[1];
    LM_CUDA(h, cudaMemcpyAsync(h->d_word, h->h_word, 2 * sizeof(unsigned), cudaMemcpyHostToDevice, st));
    int nrc = nccl.GroupStart();
    if (nrc == 0) nrc = nccl.Broadcast(h->d_word, h->d_word, 1, NCCL_INT32, 0, (NcclApi::Comm)h->nccl_comm, st);
    if (nrc == 0) nrc = nccl.AllReduce(h->d_word + 1, h->d_word + 1, 1, NCCL_INT32, NCCL_MAX, (NcclApi::Comm)h->nccl_comm, st);
    const int nrc_end = nccl.GroupEnd();
    if (nrc == 0) nrc = nrc_end;
    if (nrc != 0) return fail(h, LM_E_CUDA, std::string("ncclBroadcast / ncclAllReduce of the stopping word failed: ") + nccl.GetErrorString(nrc));
    LM_CUDA(h, cudaMemcpyAsync(h->h_word, h->d_word, 2 * sizeof(unsigned), cudaMemcpyDeviceToHost, st));
    LM_CUDA(h, cudaStreamSynchronize(st));
    words[0] = h->h_word[0];
    words[1] = h->h_word[1];
    return LM_OK;
}

// ---------------------------------------------------------------- Lanczos driver (a7-a10)
// nv <= MAX_RHS (angular: 2) independent Lanczos recurrences advanced in lockstep: one multi-right-hand-side
// pair-kernel launch per iteration serves all of them, every other kernel runs
// once per vector.  nv = 1 is lm_sqrt_mdot_w.  noise / outputs: [nv][dof] / [nv][3N].  iters_out: nv ints.
template <typename T>
int lanczos_device(lm_solver* h, int nv, const T* noise, double tol, T* lin_out, T* ang_out, double scale, int accumulate, int* iters_out,
                   cudaStream_t st, DetShare<T>* det = nullptr)
{
    const int64_t dof = dof_of(h), n3 = 3 * h->N;
    const int nc = h->angular ? 6 : 3;
    const int kmax = h->max_iter;
    const int ld = kmax + 2;
    int rc;
    if ((rc = ensure(h, &h->V, &h->V_bytes, (size_t)nv * (kmax + 1) * dof * sizeof(T))) != LM_OK) return rc;
    if ((rc = ensure(h, &h->w, &h->w_bytes, (size_t)nv * dof * sizeof(T))) != LM_OK) return rc;
    if (!h->d_scal) {
        LM_CUDA(h, cudaMalloc((void**)&h->d_scal, MAX_RHS * 4 * sizeof(double)));
        LM_CUDA(h, cudaMalloc((void**)&h->d_block, RED_MAX_BLOCKS * sizeof(double)));
        LM_CUDA(h, cudaMalloc((void**)&h->d_ticket, sizeof(unsigned int)));
        LM_CUDA(h, cudaMalloc((void**)&h->d_newest, sizeof(int)));
        LM_CUDA(h, cudaMemsetAsync(h->d_ticket, 0, sizeof(unsigned int), st));
        for (auto& e : h->lz_ev) LM_CUDA(h, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    }
    if ((rc = ensure_capture_stream(h)) != LM_OK) return rc;
    if (h->coef_cap < (size_t)(kmax + 2)) {
        if (h->d_coef) { LM_CUDA(h, cudaFree(h->d_coef)); LM_CUDA(h, cudaFree(h->d_gram_part)); LM_CUDA(h, cudaFreeHost(h->h_gram)); LM_CUDA(h, cudaFreeHost(h->h_ab)); }
        h->d_coef = nullptr;
        h->coef_cap = 0;
        LM_CUDA(h, cudaMalloc((void**)&h->d_coef, (size_t)MAX_RHS * (kmax + 2) * sizeof(double)));
        LM_CUDA(h, cudaMalloc((void**)&h->d_gram_part, (size_t)(kmax + 2) * GRAM_MAX_BLOCKS * sizeof(double)));
        LM_CUDA(h, cudaHostAlloc((void**)&h->h_gram, (size_t)MAX_RHS * ld * ld * sizeof(double), cudaHostAllocMapped));
        LM_CUDA(h, cudaHostAlloc((void**)&h->h_ab, (size_t)MAX_RHS * 2 * ld * sizeof(double), cudaHostAllocMapped));
        h->coef_cap = (size_t)(kmax + 2);
    }
    // per-vector views
    auto Vq = [&](int q) { return (T*)h->V + (size_t)q * (kmax + 1) * dof; };
    auto wq = [&](int q) { return (T*)h->w + (size_t)q * dof; };
    auto scal = [&](int q) { return h->d_scal + 4 * q; };                       // [0] |z|^2  [1] alpha  [2] beta^2
    auto ab = [&](int q) { return (volatile const double*)(h->h_ab + (size_t)q * 2 * ld); };
    auto hg = [&](int q) { return (volatile const double*)(h->h_gram + (size_t)q * ld * ld); };
    const int gr = grid_red(dof);
    const int gg = (int)std::min<int64_t>(GRAM_MAX_BLOCKS, std::max<int64_t>(1, dof / (4 * VEC_BLOCK)));
    const int64_t gchunk = (dof + gg - 1) / gg;
    // launch plans: `plan` for the nv Lanczos vectors; `plan_det` for the first apply when a deterministic right-hand
    // side rides along (one more vector; only where a variant for nv + 1 exists).  Both sized before any launch.
    LaunchPlan plan, plan_det;
    // Small N: the apply is ONE launch of rpy_small_kernel reading V[*newest] directly (no packed copy, no partials),
    // and the vector part of an iteration ONE launch of lanczos_fused_step_kernel: 3 launches per
    // iteration instead of 5-6.  M.[F;T] is then a (one-launch) apply of its own.
    const SmallPlan sp = dof <= (int64_t)FUSED_BLOCK * 32 ? choose_small<T>(h, nv) : SmallPlan();
    const bool small = sp.variant >= 0;
    const bool share = det && !small && choose_plan<T>(h, nv + 1).variant >= 0;
    // no variant for nv + 1 vectors: M.[F;T] is a launch of its own, before the packed array holds v_1
    if (det && !share && (rc = apply_batch<T>(h, 1, det->f, det->t, det->lin, det->ang, st)) != LM_OK) return rc;
    if (share && (rc = prepare_apply<T>(h, nv + 1, plan_det)) != LM_OK) return rc;
    if ((rc = prepare_apply<T>(h, nv, plan)) != LM_OK) return rc;
    auto soa = [&](int q) { return (T*)h->vec_soa + (size_t)q * nc * h->npad; };
    std::vector<LanczosStopper>& stop = h->lz_stop;
    stop.resize(nv);
    const double breakdown = (h->precision == LM_F32) ? 1e-6 : 1e-14;
    for (int q = 0; q < nv; ++q) stop[q].reset(h->lz_rule, tol, breakdown, kmax);
    // new basis vectors V_q[*newest + 1] = x_q / sqrt(sumsq_q) (+ packed copies for the next apply), their Gram
    // columns; *newest was advanced to their slot by the reduction that produced the norms (sumsq / beta kernel of
    // the LAST vector: the recurrences move in lockstep)
    auto new_vectors = [&](const T* x, int which_scal, cudaStream_t s2) {
        for (int q = 0; q < nv; ++q) {
            lanczos_scale_pack_kernel<T><<<grid_1d(h->npad), VEC_BLOCK, 0, s2>>>(x + (size_t)q * dof, h->N, h->npad, nc, (T)h->len_scale, scal(q) + which_scal, h->d_newest,
                                                                              Vq(q), soa(q), damp_of<T>(h));
            gram_column_kernel<T><<<dim3(gg, kmax + 1), VEC_BLOCK, 0, s2>>>(Vq(q), dof, h->d_newest, gchunk, h->d_gram_part, h->d_ticket,
                                                                             h->h_gram + (size_t)q * ld * ld, ld);
        }
    };

    // v_1 = z / |z|
    LM_CUDA(h, cudaMemsetAsync(h->d_newest, 0xff, sizeof(int), st));            // *newest = -1
    for (int q = 0; q < nv; ++q)
        sumsq_kernel<T><<<gr, VEC_BLOCK, 0, st>>>(noise + (size_t)q * dof, dof, h->d_block, h->d_ticket, scal(q), h->h_ab + (size_t)q * 2 * ld + 1,
                                                  q == nv - 1 ? h->d_newest : nullptr);
    new_vectors(noise, 0, st);
    if (share) {                                       // the deterministic right-hand side goes into slot nv of the packed array
        RhsIn<T> din{};
        din.f[0] = det->f;
        din.t[0] = det->t;
        pack_rhs_kernel<T><<<grid_1d(h->npad), VEC_BLOCK, 0, st>>>(din, 1, nc, h->N, h->npad, (T)h->len_scale, damp_of<T>(h), soa(nv));
        h->n_aux++;
    }
    h->n_aux += 3 * nv;
    LM_CUDA(h, cudaGetLastError());
    LM_CUDA(h, cudaStreamSynchronize(st));
    std::vector<double> znorm(nv);
    std::vector<char> done(nv, 0), conv(nv, 0);
    std::vector<int> kfin(nv, 0);
    std::vector<std::vector<double>> c_fin(nv);
    int remaining = nv;
    for (int q = 0; q < nv; ++q) {
        stop[q].set_gram_column(0, hg(q));
        if (!std::isfinite((double)ab(q)[1])) return fail(h, LM_E_INVALID, "Lanczos: the noise vector holds a non-finite value");
        znorm[q] = std::sqrt(ab(q)[1]);
        if (!(znorm[q] > 0.0)) { done[q] = conv[q] = 1; --remaining; }            // zero noise: M^{1/2} 0 = 0
    }
    h->last_iters = 0;
    // zero noise: no first apply to ride along with, M.[F;T] is a launch of its own (no iteration follows)
    if (share && remaining == 0 && (rc = apply_batch<T>(h, 1, det->f, det->t, det->lin, det->ang, st)) != LM_OK) return rc;
    const bool ride = share && remaining > 0;

    // Iteration k on the device, with m = k - 1 = *newest, for every vector:  w = M v_k;  w -= beta_{k-1} v_{k-1};
    // alpha_k;  w -= alpha_k v_k;  beta_k^2;  v_{k+1} = w / beta_k (+ packed for the next apply);  Gram column k.
    // Everything the device needs stays on the device; the host only READS (alpha_k, beta_k^2, Gram column)
    // from mapped pinned memory for the stopping test.  The launch sequence and its arguments are the
    // same for every k, so it is captured once as a CUDA graph.
    RhsOut<T> out{};
    for (int q = 0; q < nv; ++q) {
        out.lin[q] = wq(q);
        out.ang[q] = h->angular ? wq(q) + n3 : nullptr;
    }
    // the alpha kernel doubles as the split-j reduce of the apply (one launch less per vector and iteration),
    // except for row-sharded runs, where w must be all-gathered before any rank can use it
    auto fused = [&](const LaunchPlan& pl) { return pl.j_splits > 1 && pl.i_tiles > 0 && h->dist_ranks == 0 && !h->acc64; };
    auto body_small = [&](cudaStream_t s2, bool timed) -> int {
        RhsIn<T> in{};
        for (int q = 0; q < nv; ++q) {
            in.f[q] = Vq(q);
            in.t[q] = h->angular ? Vq(q) + n3 : nullptr;
        }
        // the apply of V[c] also forms Gram column c (needed by the stopping test of the NEXT iteration): no Gram launch
        double* gout[MAX_RHS] = {nullptr, nullptr, nullptr, nullptr};
        for (int q = 0; q < nv; ++q) gout[q] = h->h_gram + (size_t)q * ld * ld;
        const int rc2 = launch_small<T>(h, nv, sp, in, out, s2, timed, h->d_newest, dof, false, gout, ld);
        if (rc2 != LM_OK) return rc2;
        const int ept = (int)((dof + FUSED_BLOCK - 1) / FUSED_BLOCK);
        for (int q = 0; q < nv; ++q) {
            double* habq = h->h_ab + (size_t)q * 2 * ld;
            const int adv = q == nv - 1;
            if (ept <= 4)       lanczos_fused_step_kernel<T, 4><<<1, FUSED_BLOCK, 0, s2>>>(wq(q), Vq(q), h->d_newest, scal(q), dof, habq, adv);
            else if (ept <= 8)  lanczos_fused_step_kernel<T, 8><<<1, FUSED_BLOCK, 0, s2>>>(wq(q), Vq(q), h->d_newest, scal(q), dof, habq, adv);
            else if (ept <= 16) lanczos_fused_step_kernel<T, 16><<<1, FUSED_BLOCK, 0, s2>>>(wq(q), Vq(q), h->d_newest, scal(q), dof, habq, adv);
            else                lanczos_fused_step_kernel<T, 32><<<1, FUSED_BLOCK, 0, s2>>>(wq(q), Vq(q), h->d_newest, scal(q), dof, habq, adv);
        }
        LM_CUDA(h, cudaGetLastError());
        return LM_OK;
    };
    auto body = [&](cudaStream_t s2, bool timed, bool with_det) -> int {
        if (small) return body_small(s2, timed);
        int rc2;
        const LaunchPlan& pl = with_det ? plan_det : plan;
        const int nr = with_det ? nv + 1 : nv;
        RhsOut<T> o = out;
        if (with_det) {
            o.lin[nv] = det->lin;
            o.ang[nv] = h->angular ? det->ang : nullptr;
        }
        const bool fuse = fused(pl);
        // w_q = M v_k,q (and M.[F;T]); with a fused reduce only the deterministic vector is reduced here
        if ((rc2 = launch_pair<T>(h, nr, pl, o, s2, timed, fuse ? nv : 0)) != LM_OK) return rc2;
        for (int q = 0; q < nv; ++q) {
            lanczos_alpha_kernel<T><<<gr, VEC_BLOCK, 0, s2>>>(wq(q), Vq(q), h->d_newest, scal(q) + 2, dof, h->d_block, h->d_ticket, scal(q) + 1,
                                                              fuse ? (const T*)h->partial : nullptr, pl.j_splits, nr, q, nc, h->npad);
            lanczos_beta_kernel<T><<<gr, VEC_BLOCK, 0, s2>>>(wq(q), Vq(q), h->d_newest, scal(q) + 1, dof, h->d_block, h->d_ticket, scal(q) + 2,
                                                             h->h_ab + (size_t)q * 2 * ld, q == nv - 1 ? h->d_newest : nullptr);
        }
        new_vectors((const T*)h->w, 2, s2);
        LM_CUDA(h, cudaGetLastError());
        return LM_OK;
    };
    // One iteration of look-ahead when an apply is short: iteration k+1 is enqueued BEFORE the host waits
    // for iteration k's scalars, so the device never idles on the host round trip.  The price is one
    // wasted apply at convergence, so it is used only where an apply costs less than the round trips it
    // saves (~25 iterations x 50 us); the same regime is launch-bound, so there the body runs as a graph.
    // Row-sharded runs agree on the verdict through the stream after every iteration: no look-ahead there.
    const double apply_cost = (double)h->N * (double)h->N * (h->angular ? 2.3 : 1.0) * (h->precision == LM_F64 ? 2.5 : 1.0) * (0.6 + 0.4 * nv) * (h->wall ? 3.4 : 1.0);
    const bool dist = h->dist_ranks > 0;
    const bool lookahead = apply_cost < 2.0e9 && !dist;
    const bool use_graph = lookahead && !h->profiling && h->graph_replay;
    if (use_graph && remaining > 0) {
        const lm_solver::GraphKey key = {h->V, h->w, h->vec_soa, h->partial, h->pos_soa, kmax, small ? 1000 + sp.variant : plan.variant,
                                         small ? sp.cluster * 16 + sp.warps : plan.j_splits, h->precision * 8 + nv};
        if (!h->lz_graph || std::memcmp(&key, &h->lz_key, sizeof key) != 0) {
            if (h->lz_graph) { LM_CUDA(h, cudaGraphExecDestroy(h->lz_graph)); h->lz_graph = nullptr; }
            cudaGraph_t graph = nullptr;
            LM_CUDA(h, cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeRelaxed));
            const int rc_body = body(h->cap_stream, false, false);
            const cudaError_t ce = cudaStreamEndCapture(h->cap_stream, &graph);
            if (rc_body != LM_OK) { if (graph) cudaGraphDestroy(graph); return rc_body; }
            LM_CUDA(h, ce);
            const cudaError_t ci = cudaGraphInstantiate(&h->lz_graph, graph, 0);
            cudaGraphDestroy(graph);
            LM_CUDA(h, ci);
            h->lz_key = key;
        }
    }
    int enqueued = 0;
    auto enqueue = [&](int k) -> int {
        const bool with_det = ride && k == 1;           // the first apply carries the deterministic right-hand side
        if (use_graph && !with_det) {
            LM_CUDA(h, cudaGraphLaunch(h->lz_graph, st));
        } else {
            const int rc2 = body(st, h->profiling, with_det);
            if (rc2 != LM_OK) return rc2;
        }
        if (small) {
            h->n_pair++;
            h->pairs += (double)std::max<int64_t>(h->row_end - h->row_begin, 0) * (double)h->N;
            h->n_aux += nv;
        } else {
            if (with_det && plan_det.j_splits > 1 && fused(plan_det)) h->n_aux++;    // the deterministic vector's own reduce
            count_apply(h, with_det ? plan_det : plan);
            h->n_aux += 4 * nv;
        }
        ++enqueued;
        LM_CUDA(h, cudaEventRecord(h->lz_ev[k & 1], st));
        return LM_OK;
    };

    int k = 0, consumed = 0;
    if (remaining > 0 && (rc = enqueue(1)) != LM_OK) return rc;
    for (k = 1; k <= kmax && remaining > 0; ++k) {
        if (lookahead && k < kmax && (rc = enqueue(k + 1)) != LM_OK) return rc;
        LM_CUDA(h, cudaEventSynchronize(h->lz_ev[k & 1]));
        ++consumed;
        if (small && k >= 2)                                    // the apply of this iteration wrote the Gram column of the vector it applied
            for (int q = 0; q < nv; ++q)
                if (!done[q]) stop[q].set_gram_column(k - 1, hg(q) + (size_t)(k - 1) * ld);
        // this rank's verdicts: bit q = vector q stops at this k (converged, or k == kmax); bit 31 = a failure
        unsigned word = 0u;
        int local_fail = LM_OK;
        std::vector<char> verdict(nv, 0);
        for (int q = 0; q < nv; ++q) {
            if (done[q]) continue;
            const double alpha = ab(q)[2 * k], beta = std::sqrt(std::max((double)ab(q)[2 * k + 1], 0.0));
            if (!std::isfinite(alpha) || !std::isfinite(beta)) { local_fail = LM_E_INVALID; word |= 0x80000000u; break; }
            const LanczosStopper::Verdict v = stop[q].feed(k, alpha, beta);
            if (v == LanczosStopper::EIGENSOLVE_FAILED) { local_fail = LM_E_NOCONV; word |= 0x80000000u; break; }
            verdict[q] = v == LanczosStopper::CONVERGED;
            if (verdict[q]) word |= 1u << q;
        }
        const unsigned local_word = word;
        int rc_x = LM_OK;
        word = agree_on_stops(local_word, [&](unsigned* wd) { rc_x = exchange_words(h, wd, st); }, dist && h->dist_ranks > 1);
        if (rc_x != LM_OK) return rc_x;
        if ((word | local_word) & 0x80000000u) {
            cudaStreamSynchronize(st);
            if (local_fail == LM_E_NOCONV) return fail(h, LM_E_NOCONV, "Lanczos: tridiagonal eigensolve did not converge");
            if (local_fail == LM_E_INVALID) return fail(h, LM_E_INVALID, "Lanczos: non-finite alpha/beta -- the positions (or the noise) hold a non-finite value");
            return fail(h, LM_E_CUDA, "Lanczos: another rank reported a failure (its lm_last_error has the reason); all ranks left the loop together");
        }
        for (int q = 0; q < nv; ++q) {
            if (done[q]) continue;
            const bool stops = (word >> q) & 1u;
            if (stops || k == kmax) {
                done[q] = 1;
                conv[q] = stops;
                kfin[q] = k;
                c_fin[q] = stop[q].c_cur;
                --remaining;
                continue;
            }
            stop[q].advance();
            if (!small) stop[q].set_gram_column(k, hg(q) + (size_t)k * ld);      // small N: column k is written by the NEXT apply
        }
        if (!lookahead && remaining > 0 && k < kmax && (rc = enqueue(k + 1)) != LM_OK) return rc;
    }
    // a look-ahead iteration enqueued but never consumed did no useful pair evaluations
    if (enqueued > consumed) h->pairs -= (double)(enqueued - consumed) * (double)std::max<int64_t>(h->row_end - h->row_begin, 0) * (double)h->N;
    // results: y_q = scale |z_q| V_q c_q  (a10)
    bool all_converged = true;
    std::vector<double> coef((size_t)nv * (kmax + 2), 0.0);
    for (int q = 0; q < nv; ++q) {
        all_converged = all_converged && conv[q];
        for (int i = 0; i < kfin[q]; ++i) coef[(size_t)q * (kmax + 2) + i] = c_fin[q][i];
        if (iters_out) iters_out[q] = kfin[q];
        h->last_iters = std::max(h->last_iters, kfin[q]);
    }
    LM_CUDA(h, cudaMemcpyAsync(h->d_coef, coef.data(), coef.size() * sizeof(double), cudaMemcpyHostToDevice, st));
    for (int q = 0; q < nv; ++q) {
        T* lo = lin_out + (size_t)q * n3;
        T* ao = h->angular ? ang_out + (size_t)q * n3 : nullptr;
        if (kfin[q] == 0) {               // zero noise vector
            if (!accumulate) {
                LM_CUDA(h, cudaMemsetAsync(lo, 0, (size_t)n3 * sizeof(T), st));
                if (h->angular) LM_CUDA(h, cudaMemsetAsync(ao, 0, (size_t)n3 * sizeof(T), st));
            }
            continue;
        }
        lanczos_combine_kernel<T><<<grid_1d(dof), VEC_BLOCK, 0, st>>>(Vq(q), dof, kfin[q], h->d_coef + (size_t)q * (kmax + 2), scale * znorm[q], accumulate,
                                                                       n3, lo, ao);
        h->n_aux++;
    }
    LM_CUDA(h, cudaGetLastError());
    LM_CUDA(h, cudaStreamSynchronize(st));      // coef (pageable) must outlive the copy; drains a look-ahead iteration
    if (!all_converged) return fail(h, LM_E_NOCONV, "Lanczos: max_iter reached before the tolerance was met (last iterate written)");
    return LM_OK;
}


}  // namespace
