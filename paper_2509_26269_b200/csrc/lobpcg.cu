// lobpcg.cu -- device-resident block LOBPCG driver ("HVP-driven Krylov eigensolvers
// (Lanczos or LOBPCG) in operator mode"; :160; Knyazev ref [27] PAPER.md:221).
//
// One iteration = [block HVP on W] -> [Gram of S=[X,W,P] against [S,AS]] -> [single-CTA Rayleigh-Ritz]
// -> [X,P,AX,AP update] -> [residual R = AX - X Theta, W = Proj(R), convergence flag].  Every decision
// (convergence, breakdown, basis truncation) is taken on the device: kernels read SolverState::done and
// return at once when it is set, so the host enqueues iterations in batches without waiting on any of
// them; it only looks at a pinned copy of the status after each batch, one batch behind the GPU.
#include "common.cuh"

static int apply_operator(moto_ctx* c, const double* d_state, const double* V, int kb, double* AV) {
    if (c->kind == MOTO_KIND_TRI2D) return spin_hvp(c, d_state, c->c, V, kb, AV, /*project_input=*/0, &c->st->done);
    return cart_hvp(c, V, kb, AV, &c->st->done);
}

static int project_block(moto_ctx* c, const double* d_state, double* V, int kb) {
    if (c->kind == MOTO_KIND_TRI2D) return spin_project(c, d_state, V, kb);
    return cart_mask(c, V, kb);
}

// lobpcg_fast.cu / rayleigh_ritz.cu
int fast_gram_full(moto_ctx*, int kb, int* nblk_out);
int fast_dot_waw(moto_ctx*, int kb, double* partialsK, int* nblk_out);
int fast_update(moto_ctx*, const double* m_or_null, int kb, int* nblk_out);
int rr_solve_fast(moto_ctx*, int kb, int nblkU, const double* partialsK, int nblkK, int check, int k, double tol);

static moto_status finish(moto_ctx* c, int k, int kb, int enq, const HostStatus& last, moto_solve_info* info) {
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    int iters = last.iter < enq ? last.iter : enq;
    if (info) {
        info->iters = iters;
        info->converged = (last.done && !last.bad) ? 1 : 0;
        for (int a = 0; a < MOTO_KMAX; ++a) info->resid[a] = a < k ? last.resid[a] : 0.0;
        info->hvp_count = (int64_t)kb * (1 + iters);
    }
    if (last.bad) return moto_fail(c, MOTO_ECUDA, "moto_lowest_modes: numerical breakdown (NaN or rank loss) in Rayleigh-Ritz");
    if (!last.done) return moto_fail(c, MOTO_ENOTCONV, "moto_lowest_modes: max_iter reached; outputs hold the best iterate");
    return MOTO_OK;
}

// Fused path for kb <= 2 (lobpcg_fast.cu): per iteration  K1 -> k_rr (check + Rayleigh-Ritz) -> k_update_fused.
static moto_status lobpcg_solve_fast(moto_ctx* c, const double* d_state, int k, int kb, double tol, int max_iter, int warm_start,
                                     moto_solve_info* info) {
    const size_t bs = (size_t)3 * c->N;
    const int check_every = c->opts.check_every > 0 ? c->opts.check_every : 8;
    double* partialsK = c->partials + (size_t)MOTO_RED_BLOCKS * 64;   // after the [<=296][<=44] tri partials
    const double* m_proj = (c->kind == MOTO_KIND_TRI2D) ? d_state : nullptr;
    int n = 0, nblkU = 0, nblkK = 0;

    if (c->kind == MOTO_KIND_TRI2D) n += spin_curvature(c, d_state, c->c);
    else n += cart_build_lists(c, d_state);
    MOTO_CUDA_CHECK(c, cudaMemsetAsync(c->st, 0, sizeof(SolverState), c->stream));
    if (!warm_start) n += block_random(c, c->X, kb, c->opts.seed);
    else if (kb > k) n += block_random(c, c->X + (size_t)k * bs, kb - k, c->opts.seed ^ 0x5bd1e995u);
    n += project_block(c, d_state, c->X, kb);
    n += apply_operator(c, d_state, c->X, kb, c->AX);
    n += block_zero(c, c->W, (long long)kb * bs);
    n += block_zero(c, c->AW, (long long)kb * bs);
    n += block_zero(c, c->P, (long long)kb * bs);
    n += block_zero(c, c->AP, (long long)kb * bs);
    // start-up: Rayleigh-Ritz on span(X) alone, then the first fused update produces W = R and the Gram partials
    n += fast_gram_full(c, kb, &nblkU);
    n += rr_solve_fast(c, kb, nblkU, nullptr, 0, /*check=*/0, k, tol);
    n += fast_update(c, m_proj, kb, &nblkU);

    int enq = 0, slot = 0, pending = 0;
    bool finished = false;
    HostStatus last; memset(&last, 0, sizeof(last));
    while (!finished) {
        int batch = max_iter - enq < check_every ? max_iter - enq : check_every;
        for (int b = 0; b < batch; ++b) {
            // AW = Hess[W] with the W^T AW partials fused into the TMA kernel's epilogue when that path applies
            int nk = (c->kind == MOTO_KIND_TRI2D) ? spin_hvp_tma_ex(c, d_state, c->c, c->W, kb, c->AW, &c->st->done, partialsK, 0, 0.0, 0.0, 0.0, nullptr) : 0;
            if (nk > 0) { n += nk; nblkK = spin_tma_grid(c); }
            else {
                n += apply_operator(c, d_state, c->W, kb, c->AW);
                n += fast_dot_waw(c, kb, partialsK, &nblkK);
            }
            n += rr_solve_fast(c, kb, nblkU, partialsK, nblkK, /*check=*/1, k, tol);
            n += fast_update(c, m_proj, kb, &nblkU);
        }
        enq += batch;
        if (enq >= max_iter)   // final look at the residuals of the last update (no solve follows: done or not, X stays)
            n += rr_solve_fast(c, kb, nblkU, nullptr, 0, /*check=*/2, k, tol);
        MOTO_CUDA_CHECK(c, cudaMemcpyAsync(&c->hstat[slot], &c->st->theta, sizeof(HostStatus), cudaMemcpyDeviceToHost, c->stream));
        MOTO_CUDA_CHECK(c, cudaEventRecord(c->ev[slot], c->stream));
        if (pending) {
            MOTO_CUDA_CHECK(c, cudaEventSynchronize(c->ev[slot ^ 1]));
            last = c->hstat[slot ^ 1];
            if (last.done) finished = true;
        }
        pending = 1;
        slot ^= 1;
        if (enq >= max_iter) finished = true;
    }
    MOTO_CUDA_CHECK(c, cudaEventSynchronize(c->ev[slot ^ 1]));
    last = c->hstat[slot ^ 1];
    // keep the returned block exactly tangent / masked (rounding drift of the recurrences)
    n += project_block(c, d_state, c->X, k);
    c->launches += n;
    return finish(c, k, kb, enq, last, info);
}

moto_status lobpcg_solve(moto_ctx* c, const double* d_state, int k, double tol, int max_iter, int warm_start,
                         moto_solve_info* info) {
    int kb = k + (c->opts.guard > 0 ? c->opts.guard : 0);
    if (kb > c->kmax) kb = c->kmax;
    const long long dof = (c->kind == MOTO_KIND_TRI2D) ? 2ll * c->N : 3ll * c->N;
    if (3ll * kb > dof) kb = (int)(dof / 3 > 0 ? dof / 3 : 1);
    if (kb < k) return moto_fail(c, MOTO_EINVAL, "moto_lowest_modes: k too large for this system (need 3k <= dof)");
    if (kb <= 2 && max_iter > 0) return lobpcg_solve_fast(c, d_state, k, kb, tol, max_iter, warm_start, info);
    const size_t bs = (size_t)3 * c->N;
    const int check_every = c->opts.check_every > 0 ? c->opts.check_every : 8;
    const double* m_proj = (c->kind == MOTO_KIND_TRI2D) ? d_state : nullptr;
    int n = 0;

    // operator set-up: c_i = m_i . g_i (fixed during the solve) / neighbour table
    if (c->kind == MOTO_KIND_TRI2D) n += spin_curvature(c, d_state, c->c);
    else n += cart_build_lists(c, d_state);
    MOTO_CUDA_CHECK(c, cudaMemsetAsync(c->st, 0, sizeof(SolverState), c->stream));

    // start block
    if (!warm_start) n += block_random(c, c->X, kb, c->opts.seed);
    else if (kb > k) {  // guard columns are always fresh
        n += block_random(c, c->X + (size_t)k * bs, kb - k, c->opts.seed ^ 0x5bd1e995u);
    }
    n += project_block(c, d_state, c->X, kb);
    n += apply_operator(c, d_state, c->X, kb, c->AX);
    n += block_zero(c, c->W, (long long)kb * bs);
    n += block_zero(c, c->AW, (long long)kb * bs);
    n += block_zero(c, c->P, (long long)kb * bs);
    n += block_zero(c, c->AP, (long long)kb * bs);
    const int nblk = gram_blocks(c);
    n += block_gram_lobpcg(c, kb);
    n += rr_solve_lobpcg(c, kb, nblk);
    n += block_update(c, kb);
    n += block_residual(c, m_proj, kb, k, tol);

    int enq = 0, slot = 0, pending = 0;
    bool finished = false;
    HostStatus last; memset(&last, 0, sizeof(last));
    while (!finished) {
        int batch = max_iter - enq < check_every ? max_iter - enq : check_every;
        for (int b = 0; b < batch; ++b) {
            n += apply_operator(c, d_state, c->W, kb, c->AW);
            n += block_gram_lobpcg(c, kb);
            n += rr_solve_lobpcg(c, kb, nblk);
            n += block_update(c, kb);
            n += block_residual(c, m_proj, kb, k, tol);
        }
        enq += batch;
        MOTO_CUDA_CHECK(c, cudaMemcpyAsync(&c->hstat[slot], &c->st->theta, sizeof(HostStatus), cudaMemcpyDeviceToHost, c->stream));
        MOTO_CUDA_CHECK(c, cudaEventRecord(c->ev[slot], c->stream));
        if (pending) {  // look at the previous batch while this one runs
            MOTO_CUDA_CHECK(c, cudaEventSynchronize(c->ev[slot ^ 1]));
            last = c->hstat[slot ^ 1];
            if (last.done) finished = true;
        }
        pending = 1;
        slot ^= 1;
        if (enq >= max_iter) finished = true;
    }
    MOTO_CUDA_CHECK(c, cudaEventSynchronize(c->ev[slot ^ 1]));
    last = c->hstat[slot ^ 1];
    c->launches += n;
    MOTO_CUDA_CHECK(c, cudaGetLastError());

    int iters = last.iter < enq ? last.iter : enq;
    if (info) {
        info->iters = iters;
        info->converged = (last.done && !last.bad) ? 1 : 0;
        for (int a = 0; a < MOTO_KMAX; ++a) info->resid[a] = a < k ? last.resid[a] : 0.0;
        info->hvp_count = (int64_t)kb * (1 + iters);
    }
    if (last.bad) return moto_fail(c, MOTO_ECUDA, "moto_lowest_modes: numerical breakdown (NaN or rank loss) in Rayleigh-Ritz");
    if (!last.done) return moto_fail(c, MOTO_ENOTCONV, "moto_lowest_modes: max_iter reached; outputs hold the best iterate");
    return MOTO_OK;
}
