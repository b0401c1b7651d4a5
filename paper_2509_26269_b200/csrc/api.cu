// api.cu -- the C ABI of libmoto.so (include/moto.h): argument checks, workspace carving, dispatch.
#include <atomic>
#include <thread>
#include <vector>
#include <math.h>
#include <new>
#include "common.cuh"

static size_t al256(size_t x) { return (x + 255) & ~(size_t)255; }

static int lattice_sites(const moto_lattice* lat) {
    return lat->kind == MOTO_KIND_TRI2D ? lat->Lx * lat->Ly : lat->n_atoms;
}

static bool lattice_ok(const moto_lattice* lat) {
    if (!lat) return false;
    if (lat->kind == MOTO_KIND_TRI2D) return lat->Lx >= 1 && lat->Ly >= 1 && (long long)lat->Lx * lat->Ly < (1ll << 30);
    if (lat->kind == MOTO_KIND_CARTESIAN) return lat->n_atoms >= 1;
    return false;
}

// Upper bound on lambda_max of the constant Euclidean Hessian L of Eq. 4 on the infinite
// triangular lattice (a finite open or periodic lattice is a compression / sub-sampling of it, so the bound holds).
// Fourier symbol: L(q) = a(q) I3 + i [w(q)]x - 2 K z z^T with a(q) = -4 J sum_p cos(q.r_p), w(q) = 4 sum_p sin(q.r_p) D_p
// over the three bond pairs; eigenvalues of i[w]x are {0, +-|w|}, so lambda_max(L) <= max_q (a + |w|) + 2|K|.
// Used for the upper end b = max_i(-c_i) + lambda_max(L) of the Chebyshev interval (Weyl + compression to the
// tangent space).  The symbol is smooth; a 512 x 512 grid plus a second-derivative allowance is a safe maximum.
static double stencil_lmax_bound(const moto_spin_params& sp) {
    const double rx[3] = {1.0, 0.5, -0.5}, ry[3] = {0.0, 0.86602540378443864676, 0.86602540378443864676};
    const int G = 512;
    const double two_pi = 6.283185307179586476925;
    double best = -1e300;
    for (int i = 0; i < G; ++i)
        for (int j = 0; j < G; ++j) {
            // q = q1 b1 + q2 b2 with q.a1 = 2 pi i/G, q.a2 = 2 pi j/G  => phases of the three bonds
            const double t1 = two_pi * i / G, t2 = two_pi * j / G;
            const double ph[3] = {t1, t2, t2 - t1};
            double a = 0.0, wx = 0.0, wy = 0.0;
            for (int p = 0; p < 3; ++p) {
                a += -4.0 * sp.J * cos(ph[p]);
                // D_p = D (z x r_p) = D (-ry, rx, 0)
                wx += 4.0 * sin(ph[p]) * sp.D * (-ry[p]);
                wy += 4.0 * sin(ph[p]) * sp.D * (rx[p]);
            }
            const double v = a + sqrt(wx * wx + wy * wy);
            if (v > best) best = v;
        }
    const double h = two_pi / G;   // grid spacing in each phase; |second derivatives| <= 12 (|J| + |D|)
    return best + 0.25 * h * h * 12.0 * (fabs(sp.J) + fabs(sp.D)) * 2.0 + 2.0 * fabs(sp.K);
}

struct WsLayout { size_t block, c, g, stage, partials, st, flags, shell, cart, total; int nblocks; };

static WsLayout ws_layout(const moto_lattice* lat, int kmax) {
    WsLayout w;
    size_t N = (size_t)lattice_sites(lat);
    w.block = al256((size_t)kmax * N * 3 * sizeof(double));
    w.c = al256(N * sizeof(double));
    w.g = al256(N * 3 * sizeof(double));
    w.stage = al256(N * 3 * sizeof(double));
    w.partials = al256((size_t)MOTO_RED_BLOCKS * 2 * MOTO_NS * MOTO_NS * sizeof(double));
    w.st = al256(sizeof(SolverState));
    w.cart = lat->kind == MOTO_KIND_CARTESIAN ? cart_lists_bytes(lat) : 0;
    w.nblocks = lat->kind == MOTO_KIND_TRI2D ? 10 : 8;   // + blocks of the filter recurrence: four on spin lattices (T1..T4), two for atoms (T1, T2)
    w.flags = 4096;
    w.shell = lat->kind == MOTO_KIND_TRI2D ? al256((size_t)MOTO_MAX_SHELLS * (2 * sizeof(int) + 4 * sizeof(double))) +
                                                 al256((size_t)MOTO_SH_DENSE * 4 * sizeof(double)) + al256((size_t)MOTO_SH_SEGS * 4 * sizeof(int)) : 0;
    w.total = w.nblocks * w.block + w.c + w.g + w.stage + w.partials + w.st + w.flags + w.shell + w.cart;
    return w;
}

extern "C" {

const char* moto_version(void) { return "moto-b200 0.1 (sm_100a, fp64)"; }

size_t moto_workspace_bytes(const moto_lattice* lat, int kmax) {
    if (!lattice_ok(lat) || kmax < 1 || kmax > MOTO_KMAX) return 0;
    return ws_layout(lat, kmax).total;
}

moto_status moto_create(const moto_lattice* lat, const void* params, void* d_workspace, size_t ws_bytes, void* cuda_stream,
                        int kmax, moto_ctx** out) {
    if (!out) return MOTO_EINVAL;
    *out = nullptr;
    if (!lattice_ok(lat) || !params || !d_workspace || kmax < 1 || kmax > MOTO_KMAX) return MOTO_EINVAL;
    if (((uintptr_t)d_workspace & 255) != 0) return MOTO_EINVAL;
    WsLayout w = ws_layout(lat, kmax);
    if (ws_bytes < w.total) return MOTO_EINVAL;
    moto_ctx* c = new (std::nothrow) moto_ctx;
    if (!c) return MOTO_ENOMEM;
    memset(c, 0, sizeof(*c));
    c->lat = *lat;
    c->kind = lat->kind;
    c->N = lattice_sites(lat);
    c->kmax = kmax;
    c->stream = (cudaStream_t)cuda_stream;
    c->ws = (char*)d_workspace;
    c->ws_bytes = ws_bytes;
    c->opts.check_every = 0;   // auto
    c->opts.seed = 0x9E3779B97F4A7C15ull;
    if (c->kind == MOTO_KIND_TRI2D) {
        c->sp = *(const moto_spin_params*)params;
        c->lmax_L = stencil_lmax_bound(c->sp);
        c->lat.d_fixed = nullptr;
    } else {
        c->mp = *(const moto_morse_params*)params;
        if (!(c->mp.rc > 0) || !cart_geometry_ok(lat, c->mp.rc)) { delete c; return MOTO_EINVAL; }
    }
    char* p = c->ws;
    c->block_bytes = w.block; c->nblocks = w.nblocks;
    c->X = (double*)p; p += w.block;  c->AX = (double*)p; p += w.block;
    c->W = (double*)p; p += w.block;  c->AW = (double*)p; p += w.block;
    c->P = (double*)p; p += w.block;  c->AP = (double*)p; p += w.block;
    if (w.nblocks >= 8) { c->T1 = (double*)p; p += w.block; c->T2 = (double*)p; p += w.block; }
    if (w.nblocks == 10) { c->T3 = (double*)p; p += w.block; c->T4 = (double*)p; p += w.block; }
    c->c = (double*)p; p += w.c;
    c->g = (double*)p; p += w.g;
    c->stage_m = (double*)p; p += w.stage;
    c->partials = (double*)p; p += w.partials;
    c->st = (SolverState*)p; p += w.st;
    c->flags = (unsigned long long*)p; p += w.flags;
    if (w.shell) {
        c->sh_jd = (double*)p; c->sh_off = (int*)(p + (size_t)MOTO_MAX_SHELLS * 4 * sizeof(double));
        char* p2 = p + al256((size_t)MOTO_MAX_SHELLS * (2 * sizeof(int) + 4 * sizeof(double)));
        c->sh_jd2 = (double*)p2; c->sh_seg = (int*)(p2 + al256((size_t)MOTO_SH_DENSE * 4 * sizeof(double)));
        p += w.shell;
    }
    if (c->kind == MOTO_KIND_CARTESIAN) cart_lists_carve(c, p);
    cudaError_t e = cudaHostAlloc((void**)&c->hstat, 2 * sizeof(HostStatus), cudaHostAllocDefault);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->flags, 0, w.flags, c->stream);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev[0], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev[1], cudaEventDisableTiming);
    if (e != cudaSuccess) {
        if (c->hstat) cudaFreeHost(c->hstat);
        delete c;
        return MOTO_ECUDA;
    }
    *out = c;
    return MOTO_OK;
}

void moto_destroy(moto_ctx* c) {
    if (!c) return;
    if (c->ev[0]) cudaEventDestroy(c->ev[0]);
    if (c->ev[1]) cudaEventDestroy(c->ev[1]);
    if (c->hstat) cudaFreeHost(c->hstat);
    delete c;
}

moto_status moto_set_solver(moto_ctx* c, const moto_solver_opts* o) {
    if (!c || !o) return MOTO_EINVAL;
    if (o->guard < 0 || o->check_every < 0 || o->precond_degree < -1 || o->hvp_path < 0 || o->hvp_path > 2) return moto_fail(c, MOTO_EINVAL, "moto_set_solver: negative option");
    if (o->method < 0 || o->method > 1 || o->ncv < 0 || o->ncv > MOTO_LZ_MAX) return moto_fail(c, MOTO_EINVAL, "moto_set_solver: method must be 0 or 1, ncv in 0..24");
    if (o->persistent < 0 || o->persistent > 2) return moto_fail(c, MOTO_EINVAL, "moto_set_solver: persistent must be 0, 1 or 2");
    if (o->cheb_mode < 0 || o->cheb_mode > 3) return moto_fail(c, MOTO_EINVAL, "moto_set_solver: cheb_mode must be 0..3");
    moto_solver_opts n = *o;
    if (n.seed == 0) n.seed = 0x9E3779B97F4A7C15ull;
    c->opts = n;
    return MOTO_OK;
}

moto_status moto_set_shells(moto_ctx* c, int n, const int32_t* h_offsets, const double* h_J, const double* h_D) {
    if (!c) return MOTO_EINVAL;
    if (c->kind != MOTO_KIND_TRI2D) return moto_fail(c, MOTO_ESTATE, "moto_set_shells: spin lattices only");
    if (n < 0 || n > MOTO_MAX_SHELLS || (n > 0 && (!h_offsets || !h_J || !h_D))) return moto_fail(c, MOTO_EINVAL, "moto_set_shells: need 0 <= n <= 512 and non-null tables");
    const moto_status s = shell_set(c, n, h_offsets, h_J, h_D);
    if (s == MOTO_OK && n == 0) c->lmax_L = stencil_lmax_bound(c->sp);
    return s;
}

const char* moto_last_error(const moto_ctx* c) { return c ? c->err : "null context"; }
int64_t moto_launch_count(const moto_ctx* c) { return c ? c->launches : 0; }

moto_status moto_energy_grad(moto_ctx* c, const double* d_spins, double* d_E, double* d_g) {
    if (!c || !d_spins || (!d_E && !d_g)) return c ? moto_fail(c, MOTO_EINVAL, "moto_energy_grad: null argument") : MOTO_EINVAL;
    if (c->kind == MOTO_KIND_TRI2D) c->launches += spin_energy_grad(c, d_spins, d_E, d_g, nullptr);
    else { c->launches += cart_build_lists(c, d_spins); c->launches += cart_energy_grad(c, d_spins, d_E, d_g); }
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    return MOTO_OK;
}

moto_status moto_check_overflow(moto_ctx* c) {
    if (!c) return MOTO_EINVAL;
    if (c->kind != MOTO_KIND_CARTESIAN) return MOTO_OK;
    int ov = 0;
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(&ov, c->cl.overflow, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    if (ov) return moto_fail(c, MOTO_ENOMEM, "neighbour capacity MOTO_MAX_NEIGH exceeded: pair sums are truncated");
    return MOTO_OK;
}

moto_status moto_hvp(moto_ctx* c, const double* d_spins, const double* d_V, int k, double* d_HV) {
    if (!c) return MOTO_EINVAL;
    if (!d_spins || !d_V || !d_HV || d_V == d_HV) return moto_fail(c, MOTO_EINVAL, "moto_hvp: null or aliased argument");
    if (k < 1 || k > MOTO_KMAX) return moto_fail(c, MOTO_EINVAL, "moto_hvp: k out of range [1, MOTO_KMAX]");
    if (c->kind == MOTO_KIND_TRI2D) c->launches += spin_hvp(c, d_spins, nullptr, d_V, k, d_HV, 1, nullptr);
    else { c->launches += cart_build_lists(c, d_spins); c->launches += cart_hvp(c, d_V, k, d_HV, nullptr); }
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    return MOTO_OK;
}

// solve with the start block already in ctx->X (if warm_start); results left in ctx->X / st->theta
static moto_status solve_internal(moto_ctx* c, const double* d_spins, int k, double tol, int max_iter, int warm_start,
                                  moto_solve_info* info) {
    moto_status s = lobpcg_solve(c, d_spins, k, tol, max_iter, warm_start, info);
    if (s != MOTO_OK && s != MOTO_ENOTCONV) return s;
    moto_status s2 = moto_check_overflow(c);
    if (s2 != MOTO_OK) return s2;
    c->launches += block_sign_normalise(c, c->X, k);
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    return s;
}

moto_status moto_lowest_modes(moto_ctx* c, const double* d_spins, int k, double tol, int max_iter, int warm_start,
                              double* d_lambda, double* d_V, moto_solve_info* info) {
    if (!c) return MOTO_EINVAL;
    if (!d_spins || !d_lambda || !d_V) return moto_fail(c, MOTO_EINVAL, "moto_lowest_modes: null argument");
    if (k < 1 || k > c->kmax) return moto_fail(c, MOTO_EINVAL, "moto_lowest_modes: k out of range [1, kmax]");
    if (!(tol > 0) || max_iter < 0) return moto_fail(c, MOTO_EINVAL, "moto_lowest_modes: tol must be > 0, max_iter >= 0");
    if (persistent_applicable(c, k, max_iter)) {   // small lattice: the whole solve in one persistent kernel (same code as the batch)
        moto_ctx* one[1] = {c};
        const double* sp[1] = {d_spins};
        double* lam[1] = {d_lambda};
        double* vv[1] = {d_V};
        return persistent_solve(one, 1, sp, k, tol, max_iter, warm_start, lam, vv, info, nullptr);
    }
    const size_t bytes = (size_t)k * c->N * 3 * sizeof(double);
    if (warm_start) MOTO_CUDA_CHECK(c, cudaMemcpyAsync(c->X, d_V, bytes, cudaMemcpyDeviceToDevice, c->stream));
    moto_status s = solve_internal(c, d_spins, k, tol, max_iter, warm_start, info);
    if (s != MOTO_OK && s != MOTO_ENOTCONV) return s;
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(d_V, c->X, bytes, cudaMemcpyDeviceToDevice, c->stream));
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(d_lambda, c->st->theta, k * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
    MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    return s;
}

// Population solve: P independent problems, one host thread per context (at most 32 at a time) so that their launch-latency-bound
// kernel sequences overlap on the GPU through the contexts' own streams.
moto_status moto_lowest_modes_batch(moto_ctx* const* ctxs, int P, const double* const* d_spins, int k, double tol, int max_iter,
                                    int warm_start, double* const* d_lambda, double* const* d_V, moto_solve_info* infos,
                                    int32_t* statuses) {
    if (!ctxs || !d_spins || !d_lambda || !d_V || P < 1 || P > 4096) return MOTO_EINVAL;
    for (int p = 0; p < P; ++p) {
        if (!ctxs[p]) return MOTO_EINVAL;
        for (int q = 0; q < p; ++q)
            if (ctxs[q] == ctxs[p]) return moto_fail(ctxs[p], MOTO_EINVAL, "moto_lowest_modes_batch: the same context appears twice");
    }
    // batched path: every problem on the same small nearest-neighbour lattice -> one persistent kernel for all of them
    bool same = tol > 0 && max_iter >= 1 && k >= 1;
    for (int p = 0; p < P && same; ++p) {
        const moto_ctx* a = ctxs[0]; const moto_ctx* b = ctxs[p];
        same = d_spins[p] && d_lambda[p] && d_V[p] && persistent_applicable(b, k, max_iter) && b->lat.Lx == a->lat.Lx && b->lat.Ly == a->lat.Ly &&
               b->lat.pbc_x == a->lat.pbc_x && b->lat.pbc_y == a->lat.pbc_y && memcmp(&b->sp, &a->sp, sizeof(moto_spin_params)) == 0 &&
               b->opts.seed == a->opts.seed;
    }
    if (same) return persistent_solve(ctxs, P, d_spins, k, tol, max_iter, warm_start, d_lambda, d_V, infos, statuses);
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return MOTO_ECUDA;
    std::vector<int32_t> st(P, (int32_t)MOTO_OK);
    std::atomic<int> next(0);
    auto worker = [&]() {
        cudaSetDevice(dev);
        for (int p = next.fetch_add(1); p < P; p = next.fetch_add(1))
            st[p] = (int32_t)moto_lowest_modes(ctxs[p], d_spins[p], k, tol, max_iter, warm_start, d_lambda[p], d_V[p], infos ? infos + p : nullptr);
    };
    const int nthreads = P < 32 ? P : 32;
    std::vector<std::thread> pool;
    pool.reserve(nthreads);
    for (int t = 0; t < nthreads; ++t) pool.emplace_back(worker);
    for (auto& t : pool) t.join();
    moto_status worst = MOTO_OK;
    for (int p = 0; p < P; ++p) {
        if (statuses) statuses[p] = st[p];
        if (st[p] != MOTO_OK && (worst == MOTO_OK || worst == MOTO_ENOTCONV)) worst = (moto_status)st[p];
    }
    return worst;
}

moto_status moto_mmf_step(moto_ctx* c, const double* d_spins, const double* d_v, int kr, double dt, double* d_out, double* d_fnorm) {
    if (!c) return MOTO_EINVAL;
    if (!d_spins || !d_v || !d_out) return moto_fail(c, MOTO_EINVAL, "moto_mmf_step: null argument");
    if (kr < 1 || kr > MOTO_KMAX) return moto_fail(c, MOTO_EINVAL, "moto_mmf_step: kr out of range");
    if (c->kind == MOTO_KIND_TRI2D) c->launches += spin_mmf_step(c, d_spins, d_v, kr, dt, d_out, d_fnorm);
    else { c->launches += cart_build_lists(c, d_spins); c->launches += cart_mmf_step(c, d_spins, d_v, kr, dt, d_out, d_fnorm); }
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    return MOTO_OK;
}

// Re-solve for moto_mmf_run: a block of kb columns is iterated and warm-started as a whole, but only the first one has to
// meet tol (the reflected force needs v_1 alone, Eq. 2; lambda_2 is only needed for the sign test at the very end).  The other
// columns ride along as guard columns: they speed up v_1 (its convergence then depends on the gap to lambda_{kb+1}) and leave
// Ritz values theta_2.. >= lambda_2.. in d_lambda.  Block LOBPCG only.
static moto_status solve_first_column_impl(moto_ctx* c, const double* d_state, int kb, double tol, int max_iter, int warm, double* d_lambda,
                                      double* d_V, moto_solve_info* info) {
    const size_t bytes = (size_t)kb * c->N * 3 * sizeof(double);
    if (warm) MOTO_CUDA_CHECK(c, cudaMemcpyAsync(c->X, d_V, bytes, cudaMemcpyDeviceToDevice, c->stream));
    const int guard0 = c->opts.guard;
    c->opts.guard = kb - 1;
    c->keep_guard = warm;
    moto_status s = solve_internal(c, d_state, 1, tol, max_iter, warm, info);
    c->opts.guard = guard0;
    c->keep_guard = 0;
    if (s != MOTO_OK && s != MOTO_ENOTCONV) return s;
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(d_V, c->X, bytes, cudaMemcpyDeviceToDevice, c->stream));
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(d_lambda, c->st->theta, kb * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
    MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    return s;
}

moto_status moto_mmf_run(moto_ctx* c, double* d_state, int k, double dt, int max_steps, double tau_F, double tol, int max_iter,
                         int warm_start, double* d_V, moto_mmf_info* info) {
    if (!c) return MOTO_EINVAL;
    if (!d_state || !d_V) return moto_fail(c, MOTO_EINVAL, "moto_mmf_run: null argument");
    if (k < 2 || k > c->kmax) return moto_fail(c, MOTO_EINVAL, "moto_mmf_run: k out of range [2, kmax] (the saddle test needs lambda_2)");
    if (!(tol > 0) || max_iter < 0 || max_steps < 0 || !(tau_F >= 0)) return moto_fail(c, MOTO_EINVAL, "moto_mmf_run: bad tolerance or cap");
    const size_t vb = (size_t)c->N * 3 * sizeof(double);
    double* d_lam = c->st->scal;          // [k] device scratch (k <= 8)
    double* d_fn = c->st->cheb_ab;        // scalar scratch (rewritten by the next solve)
    double h_lam[MOTO_KMAX], h_fn = 0.0;
    moto_mmf_info out; memset(&out, 0, sizeof(out));
    moto_status st = MOTO_OK;
    int warm = warm_start;
    // block LOBPCG: per step only v_1 is converged (solve_first_column); all k columns are converged where lambda_2 decides
    const bool first_only = c->opts.method == 0 && max_iter > 0;
    for (int step = 0;; ++step) {
        moto_solve_info si = {};
        bool full = !first_only;
        st = first_only ? solve_first_column_impl(c, d_state, k, tol, max_iter, warm, d_lam, d_V, &si)
                        : moto_lowest_modes(c, d_state, k, tol, max_iter, warm, d_lam, d_V, &si);
        for (;;) {
            if (st != MOTO_OK && st != MOTO_ENOTCONV) break;
            out.hvp_count += si.hvp_count; out.solver_iters += si.iters;
            MOTO_CUDA_CHECK(c, cudaMemcpyAsync(h_lam, d_lam, k * sizeof(double), cudaMemcpyDeviceToHost, c->stream));   // before the step reuses scal
            // candidate update into the staging vector; ||F_mmf|| of the CURRENT state comes with it
            st = moto_mmf_step(c, d_state, d_V, 1, dt, c->stage_m, d_fn);
            if (st != MOTO_OK) break;
            MOTO_CUDA_CHECK(c, cudaMemcpyAsync(&h_fn, d_fn, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
            MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
            if ((st = moto_check_overflow(c)) != MOTO_OK) break;
            // the cheap solve left theta_2 >= lambda_2: the saddle test can only hold if theta_2 > 0; then (and on the last
            // step, so that the returned eigenvalues are the converged ones) all k columns are converged and the test redone
            const bool need_full = !full && ((h_fn <= tau_F && h_lam[0] < 0.0 && h_lam[1] > 0.0) || step >= max_steps);
            if (!need_full) break;
            st = moto_lowest_modes(c, d_state, k, tol, max_iter, 1, d_lam, d_V, &si);
            full = true;
        }
        if (st != MOTO_OK && st != MOTO_ENOTCONV) break;
        out.fnorm = h_fn;
        for (int a = 0; a < k; ++a) out.lambda[a] = h_lam[a];
        out.steps = step;
        if (full && h_fn <= tau_F && h_lam[0] < 0.0 && h_lam[1] > 0.0) { out.converged = 1; st = MOTO_OK; break; }
        if (step >= max_steps) { st = moto_fail(c, MOTO_ENOTCONV, "moto_mmf_run: max_steps reached before the saddle test held"); break; }
        MOTO_CUDA_CHECK(c, cudaMemcpyAsync(d_state, c->stage_m, vb, cudaMemcpyDeviceToDevice, c->stream));
        moto_status t = moto_transport(c, d_state, d_V, k);
        if (t != MOTO_OK) { st = t; break; }
        warm = 1;
    }
    if (info) *info = out;
    return st;
}

moto_status moto_mmf_run_cg(moto_ctx* c, double* d_state, int k, double delta, double smax, int max_steps, double tau_F, double tol,
                            int max_iter, int warm_start, double* d_V, double* d_scratch, moto_mmf_info* info) {
    if (!c) return MOTO_EINVAL;
    if (!d_state || !d_V || !d_scratch) return moto_fail(c, MOTO_EINVAL, "moto_mmf_run_cg: null argument");
    if (k < 2 || k > c->kmax) return moto_fail(c, MOTO_EINVAL, "moto_mmf_run_cg: k out of range [2, kmax] (the saddle test needs lambda_2)");
    if (!(tol > 0) || max_iter < 0 || max_steps < 0 || !(tau_F >= 0) || !(delta > 0) || !(smax > 0))
        return moto_fail(c, MOTO_EINVAL, "moto_mmf_run_cg: bad tolerance, cap or step length");
    return mmf_cg_run(c, d_state, k, delta, smax, max_steps, tau_F, tol, max_iter, warm_start, d_V, d_scratch, info);
}

moto_status moto_relax(moto_ctx* c, double* d_state, int max_steps, double tau_F, double alpha0, moto_relax_info* info) {
    if (!c) return MOTO_EINVAL;
    if (!d_state) return moto_fail(c, MOTO_EINVAL, "moto_relax: null argument");
    if (max_steps < 0 || !(tau_F >= 0) || !(alpha0 > 0)) return moto_fail(c, MOTO_EINVAL, "moto_relax: need max_steps >= 0, tau_F >= 0, alpha0 > 0");
    return relax_run(c, d_state, max_steps, tau_F, alpha0, info);
}

moto_status moto_relax_lbfgs(moto_ctx* c, double* d_state, int max_steps, double tau_F, double alpha0, int m, double* d_scratch,
                             moto_relax_info* info) {
    if (!c) return MOTO_EINVAL;
    if (!d_state || !d_scratch) return moto_fail(c, MOTO_EINVAL, "moto_relax_lbfgs: null argument");
    if (max_steps < 0 || !(tau_F >= 0) || !(alpha0 > 0) || m < 1 || m > 8)
        return moto_fail(c, MOTO_EINVAL, "moto_relax_lbfgs: need max_steps >= 0, tau_F >= 0, alpha0 > 0, 1 <= m <= 8");
    return relax_lbfgs_run(c, d_state, max_steps, tau_F, alpha0, m, d_scratch, info);
}

moto_status moto_mmf_run_lbfgs(moto_ctx* c, double* d_state, int k, double alpha0, double smax, int max_steps, double tau_F, double tol,
                               int max_iter, int warm_start, int m, double* d_V, double* d_scratch, moto_mmf_info* info) {
    if (!c) return MOTO_EINVAL;
    if (!d_state || !d_V || !d_scratch) return moto_fail(c, MOTO_EINVAL, "moto_mmf_run_lbfgs: null argument");
    if (k < 2 || k > c->kmax) return moto_fail(c, MOTO_EINVAL, "moto_mmf_run_lbfgs: k out of range [2, kmax] (the saddle test needs lambda_2)");
    if (!(tol > 0) || max_iter < 0 || max_steps < 0 || !(tau_F >= 0) || !(alpha0 > 0) || !(smax > 0) || m < 1 || m > 8)
        return moto_fail(c, MOTO_EINVAL, "moto_mmf_run_lbfgs: bad tolerance, cap, step length or history size (1 <= m <= 8)");
    return mmf_lbfgs_run(c, d_state, k, alpha0, smax, max_steps, tau_F, tol, max_iter, warm_start, m, d_V, d_scratch, info);
}

moto_status moto_two_sided_descent(moto_ctx* c, const double* d_saddle, const double* d_vmin, double eta, int max_steps, double tau_F,
                                   double alpha0, double* d_min_plus, double* d_min_minus, moto_relax_info* info) {
    if (!c) return MOTO_EINVAL;
    if (!d_saddle || !d_vmin || !d_min_plus || !d_min_minus) return moto_fail(c, MOTO_EINVAL, "moto_two_sided_descent: null argument");
    if (d_min_plus == d_min_minus || d_min_plus == d_saddle || d_min_minus == d_saddle || d_min_plus == d_vmin || d_min_minus == d_vmin)
        return moto_fail(c, MOTO_EINVAL, "moto_two_sided_descent: outputs must not alias the inputs or each other");
    if (max_steps < 0 || !(tau_F >= 0) || !(alpha0 > 0) || !(eta == eta)) return moto_fail(c, MOTO_EINVAL, "moto_two_sided_descent: need max_steps >= 0, tau_F >= 0, alpha0 > 0");
    moto_status worst = MOTO_OK;
    for (int b = 0; b < 2; ++b) {
        double* out = b == 0 ? d_min_plus : d_min_minus;
        moto_status s = relax_seed(c, d_saddle, d_vmin, b == 0 ? eta : -eta, out);   // Alg. 1 l.16
        if (s != MOTO_OK) return s;
        s = relax_run(c, out, max_steps, tau_F, alpha0, info ? info + b : nullptr);   // Alg. 1 l.17
        if (s != MOTO_OK && s != MOTO_ENOTCONV) return s;
        if (s == MOTO_ENOTCONV) worst = s;
    }
    return worst;
}

moto_status moto_transport(moto_ctx* c, const double* d_spins_new, double* d_V, int k) {
    if (!c) return MOTO_EINVAL;
    if (!d_spins_new || !d_V || k < 1 || k > MOTO_KMAX) return moto_fail(c, MOTO_EINVAL, "moto_transport: bad argument");
    const size_t bs = (size_t)3 * c->N;
    int n = 0;
    if (c->kind == MOTO_KIND_TRI2D) n += spin_project(c, d_spins_new, d_V, k);
    else n += cart_mask(c, d_V, k);
    const double* S[MOTO_KMAX];
    for (int a = 0; a < k; ++a) S[a] = d_V + a * bs;
    n += block_gram(c, S, k, S, k, c->st->GB, nullptr);
    n += rr_solve(c, nullptr, c->st->GB, k, k, c->st->theta, c->st->C, /*mode=*/1, nullptr);
    n += block_apply_coeffs(c, d_V, k, c->st->C, nullptr);
    c->launches += n;
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    return MOTO_OK;
}

moto_status moto_hvp_three_term(moto_ctx* c, const double* d_spins, const double* d_V, int k, double alpha, double c0, double beta,
                                const double* d_U, double* d_out, int refresh_c) {
    if (!c) return MOTO_EINVAL;
    if (c->kind != MOTO_KIND_TRI2D) return moto_fail(c, MOTO_ESTATE, "moto_hvp_three_term: spin lattices only");
    if (!d_spins || !d_V || !d_out || d_V == d_out) return moto_fail(c, MOTO_EINVAL, "moto_hvp_three_term: null or aliased argument");
    if (k < 1 || k > MOTO_KMAX) return moto_fail(c, MOTO_EINVAL, "moto_hvp_three_term: k out of range [1, MOTO_KMAX]");
    if (refresh_c) c->launches += spin_curvature(c, d_spins, c->c);
    int n = spin_hvp_tma_ex(c, d_spins, c->c, d_V, k, d_out, nullptr, nullptr, 1, alpha, c0, beta, d_U, nullptr);
    if (n <= 0) n = spin_hvp_three_term_generic(c, d_spins, c->c, d_V, k, alpha, c0, beta, d_U, d_out);
    c->launches += n;
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    return MOTO_OK;
}

moto_status moto_cheb_apply(moto_ctx* c, const double* d_spins, const double* d_V, int k, int d, double a, double b, double a_L,
                            double* d_out, int refresh_c) {
    if (!c) return MOTO_EINVAL;
    if (c->kind != MOTO_KIND_TRI2D) return moto_fail(c, MOTO_ESTATE, "moto_cheb_apply: spin lattices only");
    if (!d_spins || !d_V || !d_out || d_V == d_out) return moto_fail(c, MOTO_EINVAL, "moto_cheb_apply: null or aliased argument");
    if (k < 1 || k > 2 || k > c->kmax || d < 1 || d > MOTO_CHEB_MAX || !(a_L < a) || !(a < b))
        return moto_fail(c, MOTO_EINVAL, "moto_cheb_apply: need 1 <= k <= min(2, kmax), 1 <= d <= 256, a_L < a < b");
    int n = refresh_c ? spin_curvature(c, d_spins, c->c) : 0;
    MOTO_CUDA_CHECK(c, cudaMemsetAsync(&c->st->done, 0, 4 * sizeof(int), c->stream));
    n += fast_cheb_coef_explicit(c, d, a, b, a_L);
    const int nk = spin_cheb_recurrence(c, d_spins, c->c, d_V, k, d, d_out, &c->st->cheb[0][0], nullptr);
    if (nk <= 0) return moto_fail(c, MOTO_ESTATE, "moto_cheb_apply: needs the TMA K1 path (even Lx >= 8; hvp_path != 1) or, on general shells, the dense kernel (Lx >= 32)");
    n += nk;
    c->launches += n;
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    return MOTO_OK;
}

moto_status moto_gram(moto_ctx* c, const double* d_S, int ns, const double* d_T, int nt, double* d_G) {
    if (!c) return MOTO_EINVAL;
    if (!d_S || !d_T || !d_G || ns < 1 || nt < 1 || ns > MOTO_NS || nt > 2 * MOTO_NS) return moto_fail(c, MOTO_EINVAL, "moto_gram: bad argument");
    const size_t bs = (size_t)3 * c->N;
    const double* S[MOTO_NS]; const double* T[2 * MOTO_NS];
    for (int i = 0; i < ns; ++i) S[i] = d_S + i * bs;
    for (int j = 0; j < nt; ++j) T[j] = d_T + j * bs;
    c->launches += block_gram(c, S, ns, T, nt, d_G, nullptr);
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    return MOTO_OK;
}

moto_status moto_rayleigh_ritz(moto_ctx* c, const double* d_GA, const double* d_GB, int n, int nev, double* d_theta, double* d_C) {
    if (!c) return MOTO_EINVAL;
    if (!d_GA || !d_GB || !d_theta || !d_C || n < 1 || n > MOTO_NS || nev < 1 || nev > n)
        return moto_fail(c, MOTO_EINVAL, "moto_rayleigh_ritz: bad argument");
    c->launches += rr_solve(c, d_GA, d_GB, n, nev, d_theta, d_C, 0, nullptr);
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    return MOTO_OK;
}

// ------------------------------------------------------------------ host-buffer variants
moto_status moto_energy_grad_host(moto_ctx* c, const double* h_spins, double* h_E, double* h_g) {
    if (!c) return MOTO_EINVAL;
    if (!h_spins || (!h_E && !h_g)) return moto_fail(c, MOTO_EINVAL, "moto_energy_grad_host: null argument");
    const size_t vb = (size_t)c->N * 3 * sizeof(double);
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(c->stage_m, h_spins, vb, cudaMemcpyHostToDevice, c->stream));
    double* dE = c->st->scal + 7;
    moto_status s = moto_energy_grad(c, c->stage_m, h_E ? dE : nullptr, h_g ? c->AP : nullptr);
    if (s != MOTO_OK) return s;
    if (h_E) MOTO_CUDA_CHECK(c, cudaMemcpyAsync(h_E, dE, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    if (h_g) MOTO_CUDA_CHECK(c, cudaMemcpyAsync(h_g, c->AP, vb, cudaMemcpyDeviceToHost, c->stream));
    MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    return moto_check_overflow(c);
}

moto_status moto_hvp_host(moto_ctx* c, const double* h_spins, const double* h_V, int k, double* h_HV) {
    if (!c) return MOTO_EINVAL;
    if (!h_spins || !h_V || !h_HV) return moto_fail(c, MOTO_EINVAL, "moto_hvp_host: null argument");
    if (k < 1 || k > c->kmax) return moto_fail(c, MOTO_EINVAL, "moto_hvp_host: k out of range [1, kmax]");
    const size_t vb = (size_t)c->N * 3 * sizeof(double);
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(c->stage_m, h_spins, vb, cudaMemcpyHostToDevice, c->stream));
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(c->P, h_V, k * vb, cudaMemcpyHostToDevice, c->stream));
    moto_status s = moto_hvp(c, c->stage_m, c->P, k, c->AP);
    if (s != MOTO_OK) return s;
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(h_HV, c->AP, k * vb, cudaMemcpyDeviceToHost, c->stream));
    MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    return moto_check_overflow(c);
}

moto_status moto_lowest_modes_host(moto_ctx* c, const double* h_spins, int k, double tol, int max_iter, int warm_start,
                                   double* h_lambda, double* h_V, moto_solve_info* info) {
    if (!c) return MOTO_EINVAL;
    if (!h_spins || !h_lambda || !h_V) return moto_fail(c, MOTO_EINVAL, "moto_lowest_modes_host: null argument");
    if (k < 1 || k > c->kmax) return moto_fail(c, MOTO_EINVAL, "moto_lowest_modes_host: k out of range [1, kmax]");
    if (!(tol > 0) || max_iter < 0) return moto_fail(c, MOTO_EINVAL, "moto_lowest_modes_host: tol must be > 0, max_iter >= 0");
    const size_t vb = (size_t)c->N * 3 * sizeof(double);
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(c->stage_m, h_spins, vb, cudaMemcpyHostToDevice, c->stream));
    if (warm_start) MOTO_CUDA_CHECK(c, cudaMemcpyAsync(c->X, h_V, k * vb, cudaMemcpyHostToDevice, c->stream));
    moto_status s = solve_internal(c, c->stage_m, k, tol, max_iter, warm_start, info);
    if (s != MOTO_OK && s != MOTO_ENOTCONV) return s;
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(h_V, c->X, k * vb, cudaMemcpyDeviceToHost, c->stream));
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(h_lambda, c->st->theta, k * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    return s;
}

moto_status moto_mmf_step_host(moto_ctx* c, const double* h_spins, const double* h_v, int kr, double dt, double* h_out, double* h_fnorm) {
    if (!c) return MOTO_EINVAL;
    if (!h_spins || !h_v || !h_out) return moto_fail(c, MOTO_EINVAL, "moto_mmf_step_host: null argument");
    if (kr < 1 || kr > c->kmax) return moto_fail(c, MOTO_EINVAL, "moto_mmf_step_host: kr out of range [1, kmax]");
    const size_t vb = (size_t)c->N * 3 * sizeof(double);
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(c->stage_m, h_spins, vb, cudaMemcpyHostToDevice, c->stream));
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(c->P, h_v, kr * vb, cudaMemcpyHostToDevice, c->stream));
    double* dF = c->st->scal + 7;
    moto_status s = moto_mmf_step(c, c->stage_m, c->P, kr, dt, c->stage_m, dF);
    if (s != MOTO_OK) return s;
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(h_out, c->stage_m, vb, cudaMemcpyDeviceToHost, c->stream));
    if (h_fnorm) MOTO_CUDA_CHECK(c, cudaMemcpyAsync(h_fnorm, dF, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    return moto_check_overflow(c);
}

}  // extern "C"

// C++-linkage entry for relax.cu (moto_mmf_run_cg)
moto_status solve_first_column(moto_ctx* c, const double* d_state, int kb, double tol, int max_iter, int warm, double* d_lambda, double* d_V,
                               moto_solve_info* info) {
    return solve_first_column_impl(c, d_state, kb, tol, max_iter, warm, d_lambda, d_V, info);
}
