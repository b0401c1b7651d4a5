// lobpcg.cu -- device-resident block LOBPCG driver ("HVP-driven Krylov eigensolvers
// (Lanczos or LOBPCG) in operator mode"; :160; Knyazev ref [27] PAPER.md:221).
//
// One iteration = [block HVP on W] -> [Gram of S=[X,W,P] against [S,AS]] -> [single-CTA Rayleigh-Ritz]
// -> [X,P,AX,AP update] -> [residual R = AX - X Theta, W = Proj(R), convergence flag].  Every decision
// (convergence, breakdown, basis truncation) is taken on the device: kernels read SolverState::done and
// return at once when it is set, so the host enqueues iterations in batches without waiting on any of
// them; it only looks at a pinned copy of the status after each batch, one batch behind the GPU.
#include <stdlib.h>
#include "common.cuh"

constexpr int ATOMS_AUTO_DEGREE = 24;   // Cartesian atoms (launch-latency bound at 10^3 atoms)
constexpr int SHELL_AUTO_DEGREE = 16;   // precond_degree = 0 on general shells (HVP-bound: a lower degree than the stencil's 40)

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
int fast_dot_waw(moto_ctx*, int kb, const double* W, const double* AW, double* partialsK, int* nblk_out);
int fast_negc_max(moto_ctx*, double* partial_max, int* nmax_out);
int fast_acheck(moto_ctx*, int kb, int k, double tol, const double* d_T, double* partials, int store = 0);
int fast_cheb_coef(moto_ctx*, int k, int d, double margin, double lnorm, double hi_user, const double* partial_max, int nmax);
int fast_update(moto_ctx*, const double* m_or_null, int kb, int* nblk_out);
int rr_solve_fast(moto_ctx*, int kb, int nblkU, const double* partialsK, int nblkK, int check, int k, double tol, int hvp_inc);

static moto_status finish(moto_ctx* c, int k, int kb, int enq, const HostStatus& last, moto_solve_info* info) {
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    int iters = last.iter < enq ? last.iter : enq;
    if (info) {
        info->iters = iters;
        info->converged = (last.done && !last.bad) ? 1 : 0;
        for (int a = 0; a < MOTO_KMAX; ++a) info->resid[a] = a < k ? last.resid[a] : 0.0;
        info->hvp_count = last.nhvp > 0 ? (int64_t)last.nhvp : (int64_t)kb * (1 + iters);
    }
    if (last.bad) return moto_fail(c, MOTO_ECUDA, "moto_lowest_modes: numerical breakdown (NaN or rank loss) in Rayleigh-Ritz");
    if (!last.done) return moto_fail(c, MOTO_ENOTCONV, "moto_lowest_modes: max_iter reached; outputs hold the best iterate");
    return MOTO_OK;
}

// ------------------------------------------------------------------------------------------------------------
// Fused path for kb <= 2 (lobpcg_fast.cu): per iteration  op(W) -> k_rr (check + Rayleigh-Ritz) -> k_update_fused.
//
// op is either the Hessian itself (one K1 launch with the W^T AW partials fused in) or, on spin lattices with the
// TMA K1 path (or, on general shells, the dense shell kernel), the Chebyshev spectral transformation -p_d(A): d steps of
// its product form alpha_s (A - r_s) over the Leja-ordered roots, coefficients on the device (k_cheb_coef), two steps
// per pass of one persistent launch -- 64 B/site per Hessian application at k = 2 instead of the ~700 B/site of a full
// LOBPCG iteration.  The transformation is fixed for a phase of `phase_len` iterations;
// between phases the true A-Ritz values and A-residuals are recomputed (that is also the only convergence test
// while transformed), the interval [a, b] is re-centred on them and LOBPCG restarts from the current X.
// The host never waits per iteration: it enqueues whole phases and looks at a pinned status copy one batch behind.
struct FastCtx {
    moto_ctx* c; const double* state; const double* m_proj; int k, kb; double tol;
    double* partialsK; int nblkU, nblkK; int n;   // n: kernels enqueued
    int degree;      // 0: op = A
    bool failed;     // a recurrence launch failed: the blocks hold nothing usable
};

// OV = op(V), with the V^T OV partials left in partialsK.  V = X goes to AX, V = W goes to AW.
static void fast_apply(FastCtx& f, const double* V, double* OV) {
    moto_ctx* c = f.c;
    if (f.degree == 0) {
        int nk = (c->kind == MOTO_KIND_TRI2D) ? spin_hvp_tma_ex(c, f.state, c->c, V, f.kb, OV, &c->st->done, f.partialsK, 0, 0.0, 0.0, 0.0, nullptr, nullptr) : 0;
        if (nk > 0) { f.n += nk; f.nblkK = spin_tma_grid(c); return; }
        f.n += apply_operator(c, f.state, V, f.kb, OV);
        f.n += fast_dot_waw(c, f.kb, V, OV, f.partialsK, &f.nblkK);
        return;
    }
    // the whole recurrence: two steps per pass in one persistent cooperative launch when it fits (spin_cheb2_tma.cu), else one
    // step per pass, else one launch per step (moto_solver_opts.cheb_mode)
    const int nk = c->kind == MOTO_KIND_TRI2D ? spin_cheb_recurrence(c, f.state, c->c, V, f.kb, f.degree, OV, &c->st->cheb[0][0], &c->st->done)
                                              : cart_cheb_recurrence(c, V, f.kb, f.degree, OV, &c->st->cheb[0][0], &c->st->done);
    if (nk <= 0) { f.failed = true; return; }
    f.n += nk;
    f.n += fast_dot_waw(c, f.kb, V, OV, f.partialsK, &f.nblkK);
}

// (re)start LOBPCG on span(X) for the current op: OX = op(X), Rayleigh-Ritz on X alone, first fused update (W = R)
static void fast_phase_start(FastCtx& f) {
    moto_ctx* c = f.c;
    const size_t bs = (size_t)3 * c->N;
    fast_apply(f, c->X, c->AX);
    f.n += block_zero(c, c->W, (long long)f.kb * bs);
    f.n += block_zero(c, c->AW, (long long)f.kb * bs);
    f.n += block_zero(c, c->P, (long long)f.kb * bs);
    f.n += block_zero(c, c->AP, (long long)f.kb * bs);
    f.n += fast_gram_full(c, f.kb, &f.nblkU);
    f.n += rr_solve_fast(c, f.kb, f.nblkU, nullptr, 0, /*check=*/0, f.k, f.tol, f.kb * (f.degree ? f.degree : 1));
    f.n += fast_update(c, f.m_proj, f.kb, &f.nblkU);
}

static void fast_iterate(FastCtx& f, int check_mode) {
    moto_ctx* c = f.c;
    fast_apply(f, c->W, c->AW);
    f.n += rr_solve_fast(c, f.kb, f.nblkU, f.partialsK, f.nblkK, check_mode, f.k, f.tol, f.kb * (f.degree ? f.degree : 1));
    f.n += fast_update(c, f.m_proj, f.kb, &f.nblkU);
}

static moto_status lobpcg_solve_fast(moto_ctx* c, const double* d_state, int k, int kb, double tol, int max_iter, int warm_start,
                                     moto_solve_info* info) {
    const size_t bs = (size_t)3 * c->N;
    FastCtx f;
    f.c = c; f.state = d_state; f.k = k; f.kb = kb; f.tol = tol; f.n = 0; f.nblkU = f.nblkK = 0; f.degree = 0; f.failed = false;
    f.partialsK = c->partials + (size_t)MOTO_RED_BLOCKS * 64;   // after the [<=296][<=44] tri partials
    f.m_proj = (c->kind == MOTO_KIND_TRI2D) ? d_state : nullptr;
    double* pmax = c->partials + (size_t)MOTO_RED_BLOCKS * 128;

    // spectral transformation: precond_degree 0 = auto (40 where the TMA K1 applies), < 0 = off
    int degree = c->opts.precond_degree;
    const bool shells = shell_dense_applicable(c, kb);   // general shells: the recurrence runs on k_shell_dense, one launch per step
    const bool atoms = c->kind == MOTO_KIND_CARTESIAN && c->N <= 8192;   // (block maxima of the Gershgorin bound: <= 1024 CTAs)
    const bool can_filter = (atoms || (c->kind == MOTO_KIND_TRI2D && (spin_tma_applicable(c) || shells))) && c->T1 && c->T2 &&
                            3ll * kb * 8 <= 2ll * c->N;
    // (atoms, warm start: the re-solves of the MMF loop are ~35 launch-bound plain iterations = 6 ms per outer step at cfg 4, 9 ms transformed)
    if (degree == 0) degree = can_filter ? (shells ? SHELL_AUTO_DEGREE : (atoms ? (warm_start ? 0 : ATOMS_AUTO_DEGREE) : 40)) : 0;
    if (degree < 0 || !can_filter) degree = 0;
    if (degree > MOTO_CHEB_MAX) degree = MOTO_CHEB_MAX;
    const double margin = c->opts.precond_lo > 0 ? c->opts.precond_lo : 0.01;
    // cold start: 20 plain iterations first so that theta_k (hence a) means something; a warm start already has it
    // tuned on cfg 3 (two seeds) and its 316^2 instance; shells (degree 16, 12 plain iterations) on the 366-neighbour table at
    // 36^2, 64^2 and 100^2
    const int phase_len = 20, plain_start = warm_start ? 0 : ((shells || atoms) ? 12 : 20);
    // cheap A-residual test inside transformed phases: every 4 iterations; every 2 on a warm start below 2^18 sites, where a re-solve
    // is a handful of iterations and the test (one HVP + four streaming kernels) is short beside them (256^2, k = 2: MMF re-solve
    // 3.6 -> 3.2 ms; at 10^6 sites the test costs what it saves: 19.5 vs 19.9 ms)
    const int acheck_every = (warm_start && c->N <= (1 << 18)) ? 2 : 4;
    // b = max_i(-c_i) + lambda_max(L) >= lambda_max(Hess); atoms: the block Gershgorin bound of the stored pair coefficients
    const double lnorm = atoms ? 0.0 : c->lmax_L;

    if (c->kind == MOTO_KIND_TRI2D) f.n += spin_curvature(c, d_state, c->c);
    else f.n += cart_build_lists(c, d_state);
    MOTO_CUDA_CHECK(c, cudaMemsetAsync(c->st, 0, sizeof(SolverState), c->stream));
    int nmax = 0;
    // soft locking, as in the generic transformed solver: a column whose A-residual is within tol / 10 (k_rr where the residuals are
    // A's, k_acheck_final inside transformed phases) gets no new W_j / P_j from k_update_fused.  Without it a column that is done
    // keeps iterating at the rounding floor of -p_d(A) and its noise decides when the other one converges: 10^6 random spins took 32
    // or 36 iterations depending on the last bits of c_i (1090 vs 1412 HVPs).
    if (degree > 0) MOTO_CUDA_CHECK(c, cudaMemsetAsync(&c->st->lock_on, 1, 1, c->stream));
    if (degree > 0) {
        if (atoms) { const int nb = cart_rowbound(c, pmax, &nmax); if (nb > 0) f.n += nb; else degree = 0; }
        else f.n += fast_negc_max(c, pmax, &nmax);
    }
    if (!warm_start) f.n += block_random(c, c->X, kb, c->opts.seed);
    else if (kb > k && !c->keep_guard) f.n += block_random(c, c->X + (size_t)k * bs, kb - k, c->opts.seed ^ 0x5bd1e995u);
    f.n += project_block(c, d_state, c->X, kb);
    fast_phase_start(f);

    int enq = 0, slot = 0, pending = 0, in_phase = 0;
    bool finished = false, transformed = false;
    HostStatus last; memset(&last, 0, sizeof(last));
    while (!finished) {
        // iterations enqueued between host looks: 8 plain ones (a few short launches each), 2 transformed ones (each d operator
        // applications long, so the look hides behind them, and every iteration enqueued past convergence is d + 3 early-exit
        // launches: Cartesian atoms, cold start, 5.5 -> 4.8 ms; 366-neighbour shells 9.8 -> 9.0 ms; no change at 10^6 spins)
        const int check_every = c->opts.check_every > 0 ? c->opts.check_every : ((degree > 0 && enq >= plain_start) ? 2 : 8);
        int batch = max_iter - enq < check_every ? max_iter - enq : check_every;
        for (int b = 0; b < batch; ++b) {
            if (degree > 0 && ((!transformed && enq + b >= plain_start) || (transformed && in_phase >= phase_len))) {
                // phase boundary: true A-Ritz pairs and residuals of the current X, convergence test, new interval
                f.degree = 0;
                fast_phase_start(f);
                f.n += rr_solve_fast(c, kb, f.nblkU, nullptr, 0, /*check=*/2, k, tol, 0);
                f.n += fast_cheb_coef(c, k, degree, margin, lnorm, c->opts.precond_hi, pmax, nmax);
                f.degree = degree;
                fast_phase_start(f);
                transformed = true; in_phase = 0;
            }
            fast_iterate(f, transformed ? 3 : 1);
            ++in_phase;
            if (transformed && in_phase < phase_len && in_phase % acheck_every == 0) {
                // cheap convergence test between restarts: T1 = A X, |A x_j - (x_j.A x_j) x_j| (T1/T2 are free between applies)
                if (shells || atoms) f.n += apply_operator(c, d_state, c->X, kb, c->T1);
                else f.n += spin_hvp_tma_ex(c, d_state, c->c, c->X, kb, c->T1, &c->st->done, nullptr, 0, 0.0, 0.0, 0.0, nullptr, nullptr);
                f.n += fast_acheck(c, kb, k, tol, c->T1, pmax + 1024);
            }
        }
        enq += batch;
        if (f.failed) { c->launches += f.n; return moto_fail(c, MOTO_ECUDA, "moto_lowest_modes: a launch of the Chebyshev recurrence failed"); }
        if (enq >= max_iter) {   // final look: residuals of the last update if op = A, else a last A-phase start
            if (transformed) { f.degree = 0; fast_phase_start(f); }
            f.n += rr_solve_fast(c, kb, f.nblkU, nullptr, 0, /*check=*/2, k, tol, 0);
        }
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
    f.n += project_block(c, d_state, c->X, k);
    c->launches += f.n;
    return finish(c, k, kb, enq, last, info);
}

// ------------------------------------------------------------------------------------------------------------
// Block sizes kb > 2 on spin lattices that take the TMA K1 path: the generic block algebra (k_gram, k_update,
// k_residual) run on the same Chebyshev-transformed operator -p_d(A) as the fused path, two columns per persistent
// multi-step K1 launch.  Same phase structure: A-Ritz pairs + A-residual test + new interval at every boundary.
static int gen_apply(moto_ctx* c, const double* d_state, const double* V, int kb, double* OV, int degree) {
    if (degree == 0) return apply_operator(c, d_state, V, kb, OV);
    const size_t bs = (size_t)3 * c->N;
    int n = 0, a0 = 0;
    // all column pairs in ONE two-steps-per-pass launch, each pair on its own share of the SMs (spin_cheb2_multistep, ngroups): at
    // cfg 2 a pair's 32-step launch is bound by its neighbour synchronisation (72 us for 443 sites per CTA), three of them in one
    // launch cost about the same (solve 7.5 -> 6.3 ms, MMF re-solve 8.3 -> 5.8 ms); still ahead at 10^6 sites (k = 4: 244 -> 221 ms).
    // Bit-identical to pair-by-pair launches (a column's arithmetic does not depend on which CTA owns its rows).
    if (kb >= 4 && (c->opts.cheb_mode == 0 || c->opts.cheb_mode == 3) && degree >= 2 && !(degree & 1) && c->nsh == 0) {
        const int nk = spin_cheb2_multistep(c, d_state, c->c, V, 2, degree, OV, &c->st->cheb[0][0], &c->st->done, 1, kb / 2);
        if (nk > 0) { n += nk; a0 = 2 * (kb / 2); }
    }
    for (; a0 < kb; a0 += 2) {
        const int kk = kb - a0 >= 2 ? 2 : 1;
        const int nk = spin_cheb_recurrence(c, d_state, c->c, V + a0 * bs, kk, degree, OV + a0 * bs, &c->st->cheb[0][0], &c->st->done);
        if (nk <= 0) return -1000000;   // reported by the caller as a failed solve
        n += nk;
    }
    return n;
}

static int gen_phase_start(moto_ctx* c, const double* d_state, int kb, int k, double tol, int degree, int nblk) {
    const size_t bs = (size_t)3 * c->N;
    int n = gen_apply(c, d_state, c->X, kb, c->AX, degree);
    n += block_zero(c, c->W, (long long)kb * bs);
    n += block_zero(c, c->AW, (long long)kb * bs);
    n += block_zero(c, c->P, (long long)kb * bs);
    n += block_zero(c, c->AP, (long long)kb * bs);
    n += block_gram_lobpcg(c, kb);
    n += rr_solve_lobpcg(c, kb, nblk);
    n += block_update(c, kb);
    n += block_residual(c, d_state, kb, k, degree ? -1.0 : tol);   // transformed residuals never decide convergence
    return n;
}

static moto_status lobpcg_solve_generic_filtered(moto_ctx* c, const double* d_state, int k, int kb, double tol, int max_iter,
                                                 int warm_start, int degree, moto_solve_info* info) {
    const size_t bs = (size_t)3 * c->N;
    const double margin = c->opts.precond_lo > 0 ? c->opts.precond_lo : 0.01;
    // A-residual test: every iteration on a warm start (a re-solve of the MMF loop is a handful of iterations, each worth kb * degree
    // HVPs, the test kb), every second one on a cold start
    // 12 plain iterations before the first transformed phase (swept 4 .. 20 over 27 lattices / block sizes / guard counts: 12 and 16
    // are ahead of 20 on two thirds of them by 5-15 %, behind on the 256^2 and 10^6 random-spin states by as much; all converge)
    const int phase_len = 20, plain_start = warm_start ? 0 : 12, acheck_every = warm_start ? 1 : 2;
    double* pmax = c->g;   // [<= 296] block maxima of -c_i (the gradient scratch is free during a solve; the Gram partials fill c->partials)
    int n = 0, nmax = 0;
    n += spin_curvature(c, d_state, c->c);
    MOTO_CUDA_CHECK(c, cudaMemsetAsync(c->st, 0, sizeof(SolverState), c->stream));
    // soft locking (k_check / k_acheck_final set st->locked[j] once the A-residual of column j is within tol / 10, k_residual and
    // k_update then give that column no new W_j / P_j; it stays in the Rayleigh-Ritz basis).  Without it converged columns keep
    // iterating at the rounding floor of -p_d(A), where their normalised residuals are noise that the Rayleigh-Ritz step mixes
    // back into the block: 70 x 40 random spins, k = 3 + 2 guards, degree 32 bounced between 1e-9 and 1e-2 for 4000 iterations.
    MOTO_CUDA_CHECK(c, cudaMemsetAsync(&c->st->lock_on, 1, 1, c->stream));
    n += fast_negc_max(c, pmax, &nmax);
    if (!warm_start) n += block_random(c, c->X, kb, c->opts.seed);
    else if (kb > k && !c->keep_guard) n += block_random(c, c->X + (size_t)k * bs, kb - k, c->opts.seed ^ 0x5bd1e995u);
    n += project_block(c, d_state, c->X, kb);
    const int nblk = gram_blocks(c);
    n += gen_phase_start(c, d_state, kb, k, tol, 0, nblk);

    int enq = 0, slot = 0, pending = 0, in_phase = 0, cur_degree = 0;
    long long hv = kb;
    bool finished = false;
    HostStatus last; memset(&last, 0, sizeof(last));
    while (!finished) {
        const int check_every = c->opts.check_every > 0 ? c->opts.check_every : (enq >= plain_start ? 2 : 8);   // as on the fused path
        int batch = max_iter - enq < check_every ? max_iter - enq : check_every;
        for (int b = 0; b < batch; ++b) {
            if ((cur_degree == 0 && enq + b >= plain_start) || (cur_degree > 0 && in_phase >= phase_len)) {
                if (cur_degree > 0) { n += gen_phase_start(c, d_state, kb, k, tol, 0, nblk); hv += kb; }   // A-Ritz pairs, A-residual test
                // the damped interval starts above the whole block, theta_kb + margin: guard columns are amplified like the wanted ones
                // (with a = theta_k + margin they sat inside [a, b], where -p_d(A) is a cluster at 0 they could never resolve)
                n += fast_cheb_coef(c, kb, degree, margin, c->lmax_L, c->opts.precond_hi, pmax, nmax);
                n += gen_phase_start(c, d_state, kb, k, tol, degree, nblk);
                hv += (long long)kb * degree;
                cur_degree = degree; in_phase = 0;
            }
            n += gen_apply(c, d_state, c->W, kb, c->AW, cur_degree);
            n += block_gram_lobpcg(c, kb);
            n += rr_solve_lobpcg(c, kb, nblk);
            n += block_update(c, kb);
            n += block_residual(c, d_state, kb, k, cur_degree ? -1.0 : tol);
            hv += (long long)kb * (cur_degree ? cur_degree : 1);
            ++in_phase;
            if (cur_degree > 0 && in_phase < phase_len && in_phase % acheck_every == 0) {
                // cheap convergence test between boundaries, as on the fused path: T1 = A X, |A x_j - (x_j.A x_j) x_j|.  Without
                // it a block that converges inside a phase is iterated past convergence until the boundary, where the residuals
                // of the columns that were done first have drifted up again -- the solve then hovers at the tolerance
                n += apply_operator(c, d_state, c->X, kb, c->T1);
                n += fast_acheck(c, kb, k, tol, c->T1, c->g + 4096);
                hv += kb;
            }
        }
        enq += batch;
        if (n < 0) return moto_fail(c, MOTO_ECUDA, "moto_lowest_modes: a launch of the Chebyshev recurrence failed");
        if (enq >= max_iter && cur_degree > 0) { n += gen_phase_start(c, d_state, kb, k, tol, 0, nblk); hv += kb; }
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
    c->launches += n;
    last.nhvp = hv;   // enqueued applications (an upper bound when the device stopped early inside the last batch)
    return finish(c, k, kb, enq, last, info);
}

moto_status lobpcg_solve(moto_ctx* c, const double* d_state, int k, double tol, int max_iter, int warm_start,
                         moto_solve_info* info) {
    if (c->opts.method == 1) return lanczos_solve(c, d_state, k, tol, max_iter, warm_start, info);
    int kb = k + (c->opts.guard > 0 ? c->opts.guard : 0);
    if (kb > c->kmax) kb = c->kmax;
    const long long dof = (c->kind == MOTO_KIND_TRI2D) ? 2ll * c->N : 3ll * c->N;
    if (3ll * kb > dof) kb = (int)(dof / 3 > 0 ? dof / 3 : 1);
    if (kb < k) return moto_fail(c, MOTO_EINVAL, "moto_lowest_modes: k too large for this system (need 3k <= dof)");
    if (kb <= 2 && max_iter > 0) return lobpcg_solve_fast(c, d_state, k, kb, tol, max_iter, warm_start, info);
    // kb > 2 where the TMA K1 applies: the generic block algebra on -p_d(A) (degree 32 unless precond_degree says otherwise,
    // precond_degree < 0 = plain LOBPCG), cold and warm starts alike: cfg 2 k = 6 30 -> 7.3 ms, its warm-started MMF re-solves
    // 14.4 -> 8.3 ms per outer step (moto_mmf_run: 12.5 -> 4.5), cfg 3 k = 4 2184 -> 243 ms; converges where the plain iteration
    // runs into its cap (128 x 128 skyrmion, k = 6; 316 x 316 cfg-3 recipe, k = 6).
    constexpr int GENERIC_AUTO_DEGREE = 32;
    // Lattices below the 16 384 sites from which hvp_path = auto takes the TMA K1: a single HVP is faster on the generic kernel there,
    // but a block size above 2 is 3-6x faster on the transformed operator (40 x 40 skyrmion, k = 6: 55 -> 8.8 ms; 64 x 50 random spins,
    // k = 4: 17 -> 4.4 ms), so from 512 sites on such a solve runs with the TMA path switched on for its duration
    // (40 x 20 random spins, k = 3: 395 plain iterations, 31 ms).
    const int path0 = c->opts.hvp_path;
    if (max_iter > 0 && c->kind == MOTO_KIND_TRI2D && c->nsh == 0 && path0 == 0 && c->T1 && c->opts.precond_degree >= 0 && c->N >= 512 &&
        !(c->lat.Lx & 1) && c->lat.Lx >= 8)
        c->opts.hvp_path = 2;
    if (max_iter > 0 && c->kind == MOTO_KIND_TRI2D && spin_tma_applicable(c) && c->T1 && c->opts.precond_degree >= 0 &&
        (c->opts.precond_degree > 0 || 3ll * kb * 8 <= 2ll * c->N)) {
        int degree = c->opts.precond_degree > 0 ? c->opts.precond_degree : GENERIC_AUTO_DEGREE;
        if (degree > MOTO_CHEB_MAX) degree = MOTO_CHEB_MAX;
        const moto_status fs = lobpcg_solve_generic_filtered(c, d_state, k, kb, tol, max_iter, warm_start, degree, info);
        c->opts.hvp_path = path0;
        return fs;
    }
    c->opts.hvp_path = path0;
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
    else if (kb > k && !c->keep_guard) {  // guard columns are fresh unless the caller warm-starts them too (moto_mmf_run)
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
