// lanczos.cu -- device-resident thick-restart Lanczos behind moto_lowest_modes (moto_solver_opts.method = 1):
// the paper's second inner solver ("HVP-driven Krylov eigensolvers (Lanczos or LOBPCG) in operator mode", PAPER.md:54-60;
// "Lanczos performs better at larger sizes, so we use it for the remaining experiments"; ref. [26]
// PAPER.md:220).  The paper calls a library routine; the method is thick-restart Lanczos with full
// re-orthogonalisation (Wu and Simon 2000), restated in oracle/lanczos_oracle.py from the same source.
//
// One Lanczos step j is SIX launches and three passes over the basis V = [v_0 .. v_j] plus the new vector u:
//   K1            u = Hess[v_j]  (input re-projected, so rounding-level radial parts of v_j are not fed back)
//   k_lz_dots     h = V^T u                                   (CTA partials)
//   k_lz_fin(1)   h summed; T[j][j] = h_j
//   k_lz_upd(1)   u <- u - V h,  partials of h' = V^T u and of ||u||^2 in the same pass
//   k_lz_fin(2)   h' summed; beta_j^2 = ||u||^2 - ||h'||^2 (V orthonormal); T[j][j+1] = beta_j
//   k_lz_upd(2)   v_{j+1} = (u - V h') / beta_j
// i.e. classical Gram-Schmidt applied twice, with the second pass's dot products and the norm fused into the first
// update.  After step m - 1:  k_lz_ritz (one CTA: Jacobi on the m x m matrix T, residual estimates |beta s_{m-1,i}|,
// stop test, bordered-diagonal T of the restart) and k_lz_restart (V <- [V S_k, v_m], one pass, in place).
// Every decision is taken on the device; the host enqueues cycles in batches and looks at a pinned status copy one
// batch behind, exactly like the LOBPCG driver.  The basis lives in the LOBPCG blocks of the workspace (no extra
// memory): m = min(24, slots - 1) with slots = (8 or 6) * kmax.
#include "common.cuh"

namespace {

constexpr int LZ_THREADS = 256;

struct LzBasis {
    double* base; size_t block_stride; int kmax; long long n3;
    __host__ __device__ double* vec(int i) const { return base + (size_t)(i / kmax) * block_stride + (size_t)(i % kmax) * (size_t)n3; }
};

constexpr int LZ_U = 4;          // flat elements per thread per trip (independent loads in flight)

// acc[i] += v_i[e] * ue for the LZ_U elements of this trip (i <= j); the i-loop is unrolled so acc stays in registers
__device__ __forceinline__ void lz_dot_trip(const LzBasis& B, int j, long long e0, long long stride, const double (&ue)[LZ_U],
                                            double (&acc)[MOTO_LZ_MAX]) {
#pragma unroll
    for (int i = 0; i < MOTO_LZ_MAX; ++i) {
        if (i <= j) {
            const double* p = B.vec(i);
            double v[LZ_U];
#pragma unroll
            for (int u = 0; u < LZ_U; ++u) { const long long e = e0 + u * stride; v[u] = (e < B.n3) ? p[e] : 0.0; }
#pragma unroll
            for (int u = 0; u < LZ_U; ++u) acc[i] = fma(v[u], ue[u], acc[i]);
        }
    }
}

// CTA sums of acc[0..j] and an -> partials[blk][0..j], partials[blk][MOTO_LZ_MAX]
__device__ __forceinline__ void lz_block_sums(int j, const double (&acc)[MOTO_LZ_MAX], double an, double* __restrict__ partials) {
    __shared__ double red[LZ_THREADS / 32][MOTO_LZ_MAX + 1];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int i = 0; i < MOTO_LZ_MAX; ++i) {
        if (i <= j) {
            double s = acc[i];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (lane == 0) red[warp][i] = s;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) an += __shfl_xor_sync(0xffffffffu, an, o);
    if (lane == 0) red[warp][MOTO_LZ_MAX] = an;
    __syncthreads();
    const int t = threadIdx.x;
    if (t <= j || t == MOTO_LZ_MAX) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < LZ_THREADS / 32; ++w) s += red[w][t];
        partials[(size_t)blockIdx.x * (MOTO_LZ_MAX + 1) + t] = s;
    }
}

// partials[blk][i] = sum over this CTA's elements of v_i[e] u[e] (i <= j), partials[blk][MOTO_LZ_MAX] = sum u[e]^2;  u = v_{j+1}
__global__ void __launch_bounds__(LZ_THREADS) k_lz_dots(LzBasis B, int j, double* __restrict__ partials, const int* __restrict__ stop) {
    if (*stop) return;
    const double* u = B.vec(j + 1);
    double acc[MOTO_LZ_MAX], an = 0.0;
#pragma unroll
    for (int i = 0; i < MOTO_LZ_MAX; ++i) acc[i] = 0.0;
    const long long stride = (long long)gridDim.x * LZ_THREADS;
    for (long long e0 = blockIdx.x * (long long)LZ_THREADS + threadIdx.x; e0 < B.n3; e0 += LZ_U * stride) {
        double ue[LZ_U];
#pragma unroll
        for (int t = 0; t < LZ_U; ++t) { const long long e = e0 + t * stride; ue[t] = (e < B.n3) ? u[e] : 0.0; an = fma(ue[t], ue[t], an); }
        lz_dot_trip(B, j, e0, stride, ue, acc);
    }
    lz_block_sums(j, acc, an, partials);
}

// pass 1: u <- u - V h and partials of V^T u, ||u||^2 of the updated u;   pass 2: v_{j+1} = (u - V h) * (1 / beta)
template <int PASS>
__global__ void __launch_bounds__(LZ_THREADS) k_lz_upd(LzBasis B, int j, SolverState* st, double* __restrict__ partials) {
    if (st->done) return;
    __shared__ double h[MOTO_LZ_MAX];
    if (threadIdx.x < MOTO_LZ_MAX) h[threadIdx.x] = (threadIdx.x <= j) ? st->lz_h[threadIdx.x] : 0.0;
    __syncthreads();
    double* u = B.vec(j + 1);
    const double scale = (PASS == 2) ? st->lz_rbeta : 1.0;
    double acc[MOTO_LZ_MAX], an = 0.0;
#pragma unroll
    for (int i = 0; i < MOTO_LZ_MAX; ++i) acc[i] = 0.0;
    const long long stride = (long long)gridDim.x * LZ_THREADS;
    for (long long e0 = blockIdx.x * (long long)LZ_THREADS + threadIdx.x; e0 < B.n3; e0 += LZ_U * stride) {
        double ue[LZ_U];
#pragma unroll
        for (int t = 0; t < LZ_U; ++t) { const long long e = e0 + t * stride; ue[t] = (e < B.n3) ? u[e] : 0.0; }
        for (int i = 0; i <= j; ++i) {          // runtime loop: LZ_U independent loads per basis vector
            const double* p = B.vec(i);
            const double hi = h[i];
            double v[LZ_U];
#pragma unroll
            for (int t = 0; t < LZ_U; ++t) { const long long e = e0 + t * stride; v[t] = (e < B.n3) ? p[e] : 0.0; }
#pragma unroll
            for (int t = 0; t < LZ_U; ++t) ue[t] = fma(-hi, v[t], ue[t]);
        }
#pragma unroll
        for (int t = 0; t < LZ_U; ++t) { const long long e = e0 + t * stride; if (e < B.n3) u[e] = ue[t] * scale; }
        if (PASS == 1) {
#pragma unroll
            for (int t = 0; t < LZ_U; ++t) an = fma(ue[t], ue[t], an);
            lz_dot_trip(B, j, e0, stride, ue, acc);      // second read of the basis at these elements (cache-resident)
        }
    }
    if (PASS == 1) lz_block_sums(j, acc, an, partials);
}

// One CTA, one warp per entry: sums the CTA partials in a fixed order and does the scalar bookkeeping of the step.
// pass 0: normalisation of the start vector (beta = ||u||);  pass 1, 2: see the file header.
__global__ void __launch_bounds__(32 * (MOTO_LZ_MAX + 1)) k_lz_fin(const double* __restrict__ partials, int nblk, int j, int m, int pass,
                                                                    SolverState* st) {
    if (st->done) return;
    __shared__ double h[MOTO_LZ_MAX + 1];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (w <= j || w == MOTO_LZ_MAX) {
        double s = 0.0;
        for (int b = lane; b < nblk; b += 32) s += partials[(size_t)b * (MOTO_LZ_MAX + 1) + w];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) h[w] = s;
    }
    __syncthreads();
    if (threadIdx.x <= j && j >= 0) st->lz_h[threadIdx.x] = h[threadIdx.x];
    if (threadIdx.x == 0) {
        if (pass == 1) st->lz_T[j * MOTO_LZ_MAX + j] = h[j];
        else {
            double nrm2 = h[MOTO_LZ_MAX];
            if (pass == 2) for (int i = 0; i <= j; ++i) nrm2 -= h[i] * h[i];
            const double beta = sqrt(nrm2 > 0.0 ? nrm2 : 0.0);
            st->lz_beta = beta;
            st->lz_rbeta = 1.0 / beta;
            if (pass == 2) {
                if (j + 1 < m) { st->lz_T[j * MOTO_LZ_MAX + j + 1] = beta; st->lz_T[(j + 1) * MOTO_LZ_MAX + j] = beta; }
                st->iter += 1;
                st->nhvp += 1;
            }
            if (!(beta > 1e-290) || !(beta == beta) || !(beta < 1e290)) { st->bad = 1; st->done = 1; }   // breakdown / NaN
        }
    }
}

// V <- [V S_k, v_m]: each thread owns flat elements, reads v_0..v_m there and writes slots 0..k (in place)
__global__ void __launch_bounds__(LZ_THREADS) k_lz_restart(LzBasis B, int m, int k, int cycle, const SolverState* __restrict__ st) {
    if (st->lz_cycle != cycle) return;     // runs exactly when this cycle's k_lz_ritz ran
    __shared__ double Y[MOTO_LZ_MAX * MOTO_KMAX];
    for (int t = threadIdx.x; t < m * k; t += LZ_THREADS) Y[t] = st->lz_Y[t];   // [m][k]
    __syncthreads();
    double* vp[MOTO_LZ_MAX + 1];
#pragma unroll
    for (int i = 0; i <= MOTO_LZ_MAX; ++i) vp[i] = (i <= m) ? B.vec(i) : nullptr;
    for (long long e = blockIdx.x * (long long)LZ_THREADS + threadIdx.x; e < B.n3; e += (long long)gridDim.x * LZ_THREADS) {
        double v[MOTO_LZ_MAX];
#pragma unroll
        for (int i = 0; i < MOTO_LZ_MAX; ++i) v[i] = (i < m) ? vp[i][e] : 0.0;
        double vm = 0.0;
#pragma unroll
        for (int i = 0; i <= MOTO_LZ_MAX; ++i) if (i == m) vm = vp[i][e];
#pragma unroll
        for (int a = 0; a < MOTO_KMAX; ++a) {
            if (a < k) {
                double s = 0.0;
#pragma unroll
                for (int i = 0; i < MOTO_LZ_MAX; ++i) if (i < m) s = fma(Y[i * k + a], v[i], s);
                vp[a][e] = s;
            }
        }
#pragma unroll
        for (int i = 0; i <= MOTO_KMAX; ++i) if (i == k) vp[i][e] = vm;
    }
}

// v_0 = sum of the first k slots (warm start from a block of directions; reading A25)
__global__ void __launch_bounds__(LZ_THREADS) k_lz_sum_cols(LzBasis B, int k, const int* __restrict__ done = nullptr) {
    if (done && *done) return;
    for (long long e = blockIdx.x * (long long)LZ_THREADS + threadIdx.x; e < B.n3; e += (long long)gridDim.x * LZ_THREADS) {
        double s = 0.0;
        for (int a = 0; a < k; ++a) s += B.vec(a)[e];
        B.vec(0)[e] = s;
    }
}

}  // namespace

int lz_ritz(moto_ctx* c, int m, int k, double tol, int cycle);   // rayleigh_ritz.cu
int fast_negc_max(moto_ctx*, double* partial_max, int* nmax_out);   // lobpcg_fast.cu
int fast_acheck(moto_ctx*, int kb, int k, double tol, const double* d_T, double* partials, int store);
int fast_cheb_coef(moto_ctx*, int k, int d, double margin, double lnorm, double hi_user, const double* partial_max, int nmax);

moto_status lanczos_solve(moto_ctx* c, const double* d_state, int k, double tol, int max_iter, int warm_start,
                          moto_solve_info* info) {
    const long long n3 = 3ll * c->N;
    const long long dof = (c->kind == MOTO_KIND_TRI2D) ? 2ll * c->N : 3ll * c->N;
    // Lanczos on the Chebyshev-transformed operator -p_d(A) (the transformation of the LOBPCG path, lobpcg.cu): where the TMA K1
    // applies and k <= 2, unless precond_degree = -1.  Plain Lanczos stalls on clustered spectra at 10^6 spins (cfg 3: lambda_1..3
    // within 4e-4 at the bottom of a spectrum 18 wide); on -p_d(A) the wanted end is stretched by ~d^2.  One start cycle on A gives
    // Ritz values for the first interval; then phases of LZ_PHASE restart cycles on -p_d(A), each phase opened by the true
    // A-Rayleigh quotients and A-residuals of the current Ritz vectors (the only convergence test) and a new interval from them.
    int degree = c->opts.precond_degree;
    const bool shells = shell_dense_applicable(c, k <= 2 ? k : 1);   // general shells: the recurrence as d launches of k_shell_dense
    const bool can_filter = c->kind == MOTO_KIND_TRI2D && (spin_tma_applicable(c) || shells) && c->T1 && k <= 2;
    if (degree == 0) degree = can_filter ? (shells ? 16 : 40) : 0;
    if (degree < 0 || !can_filter) degree = 0;
    if (degree > MOTO_CHEB_MAX) degree = MOTO_CHEB_MAX;
    // the recurrence uses T1..T4 as scratch, so the basis then lives in the six solver blocks only
    int m = (degree > 0 ? 6 : (c->nblocks > 8 ? 8 : c->nblocks)) * c->kmax - 1;
    if (m > MOTO_LZ_MAX) m = MOTO_LZ_MAX;
    if (c->opts.ncv > 0 && c->opts.ncv < m) m = c->opts.ncv;
    if (m > dof - 1) m = (int)(dof - 1);
    if (m < k + 2) {
        snprintf(c->err, sizeof(c->err), "moto_lowest_modes (Lanczos): basis too small, need k + 2 <= ncv <= min(24, %d kmax - 1, dof - 1)",
                 c->nblocks > 8 ? 8 : c->nblocks);
        return MOTO_EINVAL;
    }
    if (max_iter < 1) return moto_fail(c, MOTO_EINVAL, "moto_lowest_modes (Lanczos): max_iter must be >= 1");
    LzBasis B = {c->X, c->block_bytes / sizeof(double), c->kmax, n3};
    const int check_every = c->opts.check_every > 0 ? c->opts.check_every : 8;
    int grid = (int)((n3 + LZ_THREADS - 1) / LZ_THREADS);
    if (grid > MOTO_RED_BLOCKS) grid = MOTO_RED_BLOCKS;
    int n = 0;

    if (c->kind == MOTO_KIND_TRI2D) n += spin_curvature(c, d_state, c->c);
    else n += cart_build_lists(c, d_state);
    MOTO_CUDA_CHECK(c, cudaMemsetAsync(c->st, 0, sizeof(SolverState), c->stream));
    // start vector: seeded random, or the sum of the caller's block; projected / masked, normalised
    if (!warm_start) n += block_random(c, c->X, 1, c->opts.seed);
    else if (k > 1) { k_lz_sum_cols<<<grid, LZ_THREADS, 0, c->stream>>>(B, k); ++n; }
    if (c->kind == MOTO_KIND_TRI2D) n += spin_project(c, d_state, c->X, 1); else n += cart_mask(c, c->X, 1);
    k_lz_dots<<<grid, LZ_THREADS, 0, c->stream>>>(B, -1, c->partials, &c->st->done);
    k_lz_fin<<<1, 32 * (MOTO_LZ_MAX + 1), 0, c->stream>>>(c->partials, grid, -1, m, 0, c->st);
    k_lz_upd<2><<<grid, LZ_THREADS, 0, c->stream>>>(B, -1, c->st, c->partials);
    n += 3;

    bool filtered = false, op_failed = false;   // which operator the steps apply: A, or -p_d(A) once an interval exists
    long long hv = 0;                           // single-vector HVPs enqueued (host count; the device counts steps)
    auto step = [&](int j) {
        if (filtered) {
            const int nk = spin_cheb_recurrence(c, d_state, c->c, B.vec(j), 1, degree, B.vec(j + 1), &c->st->cheb[0][0], &c->st->done);
            if (nk <= 0) op_failed = true; else n += nk;
            n += spin_project(c, d_state, B.vec(j + 1), 1);   // the recurrence does not re-project (reading A24): keep the basis tangent
            hv += degree;
        } else {
            if (c->kind == MOTO_KIND_TRI2D) n += spin_hvp(c, d_state, c->c, B.vec(j), 1, B.vec(j + 1), /*project_input=*/1, &c->st->done);
            else n += cart_hvp(c, B.vec(j), 1, B.vec(j + 1), &c->st->done);
            hv += 1;
        }
        k_lz_dots<<<grid, LZ_THREADS, 0, c->stream>>>(B, j, c->partials, &c->st->done);
        k_lz_fin<<<1, 32 * (MOTO_LZ_MAX + 1), 0, c->stream>>>(c->partials, grid, j, m, 1, c->st);
        k_lz_upd<1><<<grid, LZ_THREADS, 0, c->stream>>>(B, j, c->st, c->partials);
        k_lz_fin<<<1, 32 * (MOTO_LZ_MAX + 1), 0, c->stream>>>(c->partials, grid, j, m, 2, c->st);
        k_lz_upd<2><<<grid, LZ_THREADS, 0, c->stream>>>(B, j, c->st, c->partials);
        n += 5;
    };

    int steps = 0, cycle = 0, k0 = 0, slot = 0, pending = 0, since = 0;
    bool finished = false;
    HostStatus last; memset(&last, 0, sizeof(last));
    const int LZ_PHASE = 3;                     // restart cycles per interval
    const double margin = c->opts.precond_lo > 0 ? c->opts.precond_lo : 0.01;
    double* pmax = c->partials + (size_t)MOTO_RED_BLOCKS * 128;
    int nmax = 0, in_phase = 0;
    if (degree > 0) n += fast_negc_max(c, pmax, &nmax);
    while (!finished) {
        for (int j = k0; j < m; ++j) step(j);
        steps += m - k0; since += m - k0;
        ++cycle;
        n += lz_ritz(c, m, k, degree > 0 ? -1.0 : tol, cycle);   // filtered: the Lanczos estimates are those of -p_d(A), never the stop test
        k_lz_restart<<<grid, LZ_THREADS, 0, c->stream>>>(B, m, k, cycle, c->st); ++n;
        k0 = k;
        if (degree > 0) {
            // after every restart: T1 = A X of the k Ritz vectors, A-Rayleigh quotients and A-residuals -- the convergence test
            if (shells) n += spin_hvp(c, d_state, c->c, c->X, k, c->T1, /*project_input=*/0, &c->st->done);
            else n += spin_hvp_tma_ex(c, d_state, c->c, c->X, k, c->T1, &c->st->done, nullptr, 0, 0.0, 0.0, 0.0, nullptr, nullptr);
            n += fast_acheck(c, k, k, tol, c->T1, pmax + 1024, /*store=*/1);
            hv += k;
        }
        if (degree > 0 && (!filtered || ++in_phase >= LZ_PHASE)) {
            // phase boundary: next interval from the A-Rayleigh quotients, and a fresh Lanczos run on the new operator from the
            // sum of the Ritz vectors
            n += fast_cheb_coef(c, k, degree, margin, c->lmax_L, c->opts.precond_hi, pmax, nmax);
            if (k > 1) { k_lz_sum_cols<<<grid, LZ_THREADS, 0, c->stream>>>(B, k, &c->st->done); ++n; }
            MOTO_CUDA_CHECK(c, cudaMemsetAsync(c->st->lz_T, 0, sizeof(c->st->lz_T), c->stream));   // no bordered rows of the old run
            k_lz_dots<<<grid, LZ_THREADS, 0, c->stream>>>(B, -1, c->partials, &c->st->done);
            k_lz_fin<<<1, 32 * (MOTO_LZ_MAX + 1), 0, c->stream>>>(c->partials, grid, -1, m, 0, c->st);
            k_lz_upd<2><<<grid, LZ_THREADS, 0, c->stream>>>(B, -1, c->st, c->partials);
            n += 3;
            filtered = true; in_phase = 0; k0 = 0;
        }
        const bool cap = steps >= max_iter;
        // host look: every 8 steps on A, every 2 on the transformed operator (a step is then d applications long; as in lobpcg.cu)
        if (since >= (c->opts.check_every > 0 ? check_every : (filtered ? 2 : 8)) || cap) {
            since = 0;
            MOTO_CUDA_CHECK(c, cudaMemcpyAsync(&c->hstat[slot], &c->st->theta, sizeof(HostStatus), cudaMemcpyDeviceToHost, c->stream));
            MOTO_CUDA_CHECK(c, cudaEventRecord(c->ev[slot], c->stream));
            if (pending) {
                MOTO_CUDA_CHECK(c, cudaEventSynchronize(c->ev[slot ^ 1]));
                last = c->hstat[slot ^ 1];
                if (last.done) finished = true;
            }
            pending = 1;
            slot ^= 1;
        }
        if (cap || op_failed) finished = true;
    }
    if (op_failed) { c->launches += n; return moto_fail(c, MOTO_ECUDA, "moto_lowest_modes (Lanczos): a launch of the Chebyshev recurrence failed"); }
    MOTO_CUDA_CHECK(c, cudaEventSynchronize(c->ev[slot ^ 1]));
    last = c->hstat[slot ^ 1];
    // true residuals of the returned pairs: AX = Hess[X], r_j = AX_j - theta_j X_j (the stop test used the Lanczos estimates)
    const int conv = last.done && !last.bad;
    if (!last.bad) {
        MOTO_CUDA_CHECK(c, cudaMemsetAsync(&c->st->done, 0, sizeof(int), c->stream));
        if (c->kind == MOTO_KIND_TRI2D) n += spin_hvp(c, d_state, c->c, c->X, k, c->AX, 1, nullptr);
        else n += cart_hvp(c, c->X, k, c->AX, nullptr);
        n += block_residual(c, c->kind == MOTO_KIND_TRI2D ? d_state : nullptr, k, k, -1.0);
        MOTO_CUDA_CHECK(c, cudaMemcpyAsync(&c->hstat[0], &c->st->theta, sizeof(HostStatus), cudaMemcpyDeviceToHost, c->stream));
        MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
        for (int a = 0; a < MOTO_KMAX; ++a) last.resid[a] = c->hstat[0].resid[a];
    }
    c->launches += n;
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    if (info) {
        info->iters = last.iter;
        info->converged = conv;
        for (int a = 0; a < MOTO_KMAX; ++a) info->resid[a] = a < k ? last.resid[a] : 0.0;
        info->hvp_count = degree > 0 ? (int64_t)hv + (last.bad ? 0 : k) : (int64_t)last.nhvp + (last.bad ? 0 : k);
    }
    if (last.bad) return moto_fail(c, MOTO_ECUDA, "moto_lowest_modes (Lanczos): numerical breakdown (NaN or an invariant Krylov space)");
    if (!conv) return moto_fail(c, MOTO_ENOTCONV, "moto_lowest_modes (Lanczos): max_iter reached; outputs hold the best iterate");
    return MOTO_OK;
}
