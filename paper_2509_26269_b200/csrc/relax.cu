// relax.cu -- two-sided minimum-mode descent (Alg. 1 l.15-18; Suppl. Note 1 b(iii), PAPER.md:307;
// SURVEY 8(f) f2): seeds x_saddle +- eta v_min, each relaxed downhill "using a deterministic optimizer (e.g., L-BFGS/CG)".
// The paper gives no more than that; the optimiser is reading A26 of DESIGN.md: Riemannian Polak-Ribiere+ conjugate
// gradients with backtracking,
//   trial x_t = R(x + a d), a = alpha, alpha/2, ...;  accept if g_t.d <= SIGMA |g.d| and (Armijo or E_t <= E + EPS_E |E|)
//   beta = max(0, (g_t.g_t - g_t.g)/(g.g));  d <- -g_t + beta T(d)  (T = tangent projection at x_t / identity for atoms)
//   alpha <- 2a if the first trial was accepted else a;  stop at |g| <= tau_F.
// Every vector operation runs on the device.  Spins: a trial is ONE fused pass (k_relax_eval in spin_stencil.cu: retraction
// recomputed at the site and its neighbours, stencil gradient, projection and the four sums E_t, g_t.g_t, g_t.g, g_t.d;
// 120 B/site) plus the direction update (96 B/site) once a step is accepted.  Atoms: trial kernel, neighbour lists + K7
// gradient, one Gram launch, and the host reads four scalars per trial and decides.  On spin lattices the decision is taken
// on the device as well (k_relax_decide, same arithmetic): eval -> decide -> direction update are enqueued eight trials at a
// time and the host only looks at the state between batches (relax_run_device).
#include "common.cuh"
#include "device_utils.cuh"

#define RELAX_C1 1e-4
#define RELAX_EPS_E 1e-10
#define RELAX_SIGMA 0.5
#define RELAX_MAX_BACKTRACKS 40

namespace {

// x_t = R(x + a d): per-site renormalisation for spins (A7), identity for atoms (d is zero on fixed atoms)
// (x and xt may be the same array -- moto_mmf_run_cg updates the state in place -- so neither is __restrict__)
__global__ void __launch_bounds__(256) k_relax_trial(long long N, const double* x, const double* __restrict__ d, double a,
                                                     double* xt, int retract) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        d3 y = axpy3(a, ld3(d, i), ld3(x, i));
        if (retract) y = scale3(1.0 / sqrt(dot3(y, y)), y);
        st3(xt, i, y);
    }
}

// d <- sg g_t + beta T(d)   (sg = -1: descent on the gradient, moto_relax;  sg = +1: g_t is a force, moto_mmf_run_cg)
__global__ void __launch_bounds__(256) k_relax_dir(long long N, const double* __restrict__ xt, const double* __restrict__ gt, double beta,
                                                   double* __restrict__ d, int project, double sg = -1.0) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        d3 di = mk3(0.0, 0.0, 0.0);
        if (beta != 0.0) {                       // beta == 0: d may be uninitialised, never read it
            di = ld3(d, i);
            if (project) di = proj3(ld3(xt, i), di);
        }
        d3 g = ld3(gt, i);
        st3(d, i, mk3(fma(beta, di.x, sg * g.x), fma(beta, di.y, sg * g.y), fma(beta, di.z, sg * g.z)));
    }
}

int grid_for(long long N) {
    long long b = (N + 255) / 256;
    return (int)(b < 4 * MOTO_NUM_SMS ? (b > 0 ? b : 1) : 4 * MOTO_NUM_SMS);
}

// One evaluation: trial point x_t = R(x + a d) (d != nullptr) or x itself (d == nullptr); leaves g_new = gradient there and
// brings {E, g_new.g_new, g_new.g_old, g_new.d} to the host with one synchronisation.
// Spins: one fused pass (k_relax_eval, spin_stencil.cu).  Atoms: trial kernel, neighbour lists + K7 gradient, one Gram launch.
moto_status eval_point(moto_ctx* c, const double* x, const double* d, double a, const double* g_old, double* xt, double* g_new,
                       double* h4) {
    double* dE = c->st->scal;          // [0] E, [1..3] dots
    int fused = c->kind == MOTO_KIND_TRI2D ? spin_relax_eval(c, x, d, a, g_old, xt, g_new, dE) : 0;
    c->launches += fused;
    if (!fused) {
        if (d) { k_relax_trial<<<grid_for(c->N), 256, 0, c->stream>>>((long long)c->N, x, d, a, xt, c->kind == MOTO_KIND_TRI2D); c->launches += 1; }
        moto_status s = moto_energy_grad(c, d ? xt : x, dE, g_new);
        if (s != MOTO_OK) return s;
        const double* S[1] = {g_new};
        const double* T[3] = {g_new, g_old ? g_old : g_new, d ? d : g_new};
        c->launches += block_gram(c, S, 1, T, 3, dE + 1, nullptr);
    }
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(h4, dE, 4 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    if (c->kind == MOTO_KIND_CARTESIAN) {
        int ov = 0;
        MOTO_CUDA_CHECK(c, cudaMemcpy(&ov, c->cl.overflow, sizeof(int), cudaMemcpyDeviceToHost));
        if (ov) return moto_fail(c, MOTO_ENOMEM, "neighbour capacity MOTO_MAX_NEIGH exceeded");
    }
    return MOTO_OK;
}

}  // namespace

// ---------------------------------------------------------------- device-resident line search (spin lattices, fused trial kernel)
namespace {

// sums the four partial columns of the last evaluation, then ONE thread takes the decision the host loop of relax_run_host
// takes (same arithmetic, same order), and leaves the next trial's description in *rs
__global__ void __launch_bounds__(1024) k_relax_decide(const double* __restrict__ partials, int nblk, RelaxDev* rs, int init) {
    __shared__ double sm[1024];
    if (rs->status) return;
    const int j = threadIdx.x & 3, r = threadIdx.x >> 2;
    double s = 0.0;
    for (int b = r; b < nblk; b += 256) s += partials[(size_t)b * 4 + j];
    sm[threadIdx.x] = s;
    __syncthreads();
    for (int off = 512; off >= 4; off >>= 1) {
        if (threadIdx.x < off) sm[threadIdx.x] += sm[threadIdx.x + off];
        __syncthreads();
    }
    if (threadIdx.x != 0) return;
    if (init) {
        rs->E = sm[0]; rs->gg = sm[1]; rs->slope = -sm[1];
        rs->a = rs->alpha; rs->steepest = 1; rs->first = 1; rs->bt = 0; rs->evals = 1; rs->steps = 0;
        rs->dir_mode = 2;
    } else {
        rs->evals += 1;
        const double Et = sm[0], gtgt = sm[1], gtg = sm[2], gtd = sm[3], a = rs->a, E = rs->E, slope = rs->slope;
        const bool acc = gtd <= RELAX_SIGMA * fabs(slope) && (Et <= E + RELAX_C1 * a * slope || Et <= E + RELAX_EPS_E * fabs(E));
        if (acc) {
            double beta = (gtgt - gtg) / rs->gg;
            if (!(beta > 0.0)) beta = 0.0;
            double new_slope = -gtgt + beta * gtd;
            if (new_slope >= 0.0) { beta = 0.0; new_slope = -gtgt; }
            rs->beta = beta; rs->steepest = beta == 0.0;
            rs->cur = rs->cur == 1 ? 2 : 1; rs->gcur ^= 1;
            rs->E = Et; rs->gg = gtgt; rs->slope = new_slope;
            rs->alpha = rs->first ? 2.0 * a : a;
            rs->steps += 1;
            rs->a = rs->alpha; rs->first = 1; rs->bt = 0;
            rs->dir_mode = 1;
        } else {
            rs->a = 0.5 * a; rs->first = 0; rs->bt += 1; rs->dir_mode = 0;
            if (rs->bt >= RELAX_MAX_BACKTRACKS) {
                if (rs->steepest) { rs->status = 3; return; }
                rs->dir_mode = 2; rs->slope = -rs->gg; rs->steepest = 1; rs->a = rs->alpha; rs->first = 1; rs->bt = 0;
            }
            return;
        }
    }
    const double gg = rs->gg;
    if (!(gg == gg)) rs->status = 4;
    else if (sqrt(gg) <= rs->tau) rs->status = 1;
    else if (rs->steps >= rs->max_steps) rs->status = 2;
}

__global__ void __launch_bounds__(256) k_relax_dir_dev(long long N, const RelaxDev* __restrict__ rs) {
    const int mode = rs->dir_mode;
    if (mode == 0 || rs->status) return;
    const double* __restrict__ xt = rs->x[rs->cur];
    const double* __restrict__ gt = rs->g[rs->gcur];
    double* __restrict__ d = rs->d;
    const double beta = mode == 1 ? rs->beta : 0.0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        d3 di = mk3(0.0, 0.0, 0.0);
        if (beta != 0.0) di = proj3(ld3(xt, i), ld3(d, i));
        const d3 g = ld3(gt, i);
        st3(d, i, mk3(fma(beta, di.x, -g.x), fma(beta, di.y, -g.y), fma(beta, di.z, -g.z)));
    }
}

}  // namespace

// Spin lattices with the fused trial kernel: a trial is eval -> decide -> (direction update) with nothing coming back to the
// host; the host enqueues eight trials at a time and then looks at the state once.
static moto_status relax_run_device(moto_ctx* c, double* d_state, int max_steps, double tau_F, double alpha0, moto_relax_info* info, int nblk) {
    const long long N = c->N;
    const size_t vb = (size_t)N * 3 * sizeof(double);
    const int grid = grid_for(N);
    RelaxDev* rs = reinterpret_cast<RelaxDev*>(c->st->lz_T);   // solver scratch: no solve runs during a relaxation
    static_assert(sizeof(RelaxDev) <= sizeof(double) * MOTO_LZ_MAX * MOTO_LZ_MAX, "RelaxDev does not fit its scratch");
    RelaxDev h; memset(&h, 0, sizeof(h));
    h.alpha = alpha0; h.tau = tau_F; h.max_steps = max_steps;
    h.x[0] = d_state; h.x[1] = c->stage_m; h.x[2] = c->P; h.g[0] = c->g; h.g[1] = c->W; h.d = c->AW;
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(rs, &h, sizeof(h), cudaMemcpyHostToDevice, c->stream));
    c->launches += spin_relax_eval(c, d_state, nullptr, 0.0, nullptr, nullptr, c->g, c->st->scal);
    k_relax_decide<<<1, 1024, 0, c->stream>>>(c->partials, nblk, rs, 1);
    k_relax_dir_dev<<<grid, 256, 0, c->stream>>>(N, rs);
    c->launches += 2;
    for (;;) {
        MOTO_CUDA_CHECK(c, cudaMemcpyAsync(&h, rs, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
        MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
        if (h.status) break;
        for (int b = 0; b < 8; ++b) {
            int nb = 0;
            c->launches += spin_relax_eval_dev(c, rs, &nb);
            k_relax_decide<<<1, 1024, 0, c->stream>>>(c->partials, nb, rs, 0);
            k_relax_dir_dev<<<grid, 256, 0, c->stream>>>(N, rs);
            c->launches += 2;
        }
        MOTO_CUDA_CHECK(c, cudaGetLastError());
    }
    if (h.cur != 0) MOTO_CUDA_CHECK(c, cudaMemcpyAsync(d_state, h.x[h.cur], vb, cudaMemcpyDeviceToDevice, c->stream));
    MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    if (info) {
        memset(info, 0, sizeof(*info));
        info->steps = h.steps; info->converged = h.status == 1; info->evals = h.evals;
        info->energy = h.E; info->gnorm = sqrt(h.gg); info->alpha = h.alpha;
    }
    if (h.status == 1) return MOTO_OK;
    if (h.status == 2) return moto_fail(c, MOTO_ENOTCONV, "moto_relax: max_steps reached");
    if (h.status == 3) return moto_fail(c, MOTO_ENOTCONV, "moto_relax: stalled (no acceptable step along -g)");
    return moto_fail(c, MOTO_ESTATE, "moto_relax: NaN gradient");
}

// d_state in/out.  Scratch (no solver is running): g, g_t = ctx->g / W (swapped on acceptance), d = AW, and the current and
// trial states ping-pong between stage_m and P, so an accepted step costs no copy; d_state is written once at the end.
moto_status relax_run(moto_ctx* c, double* d_state, int max_steps, double tau_F, double alpha0, moto_relax_info* info) {
    if (const int nblk = spin_relax_nblk(c)) return relax_run_device(c, d_state, max_steps, tau_F, alpha0, info, nblk);
    const long long N = c->N;
    const size_t vb = (size_t)N * 3 * sizeof(double);
    const int spin = c->kind == MOTO_KIND_TRI2D;
    const int grid = grid_for(N);
    double *g = c->g, *gt = c->W, *d = c->AW;
    double* bufs[2] = {c->stage_m, c->P};
    int which = 0;
    const double* x = d_state;
    moto_relax_info out; memset(&out, 0, sizeof(out));
    double h[4];
    moto_status s = eval_point(c, x, nullptr, 0.0, nullptr, nullptr, g, h);
    if (s != MOTO_OK) return s;
    out.evals = 1;
    double E = h[0], gg = h[1], slope = -gg, alpha = alpha0;
    k_relax_dir<<<grid, 256, 0, c->stream>>>(N, x, g, 0.0, d, 0);   // d = -g (beta = 0: the old d is never read)
    c->launches += 1;
    bool steepest = true;
    moto_status ret = MOTO_OK;
    for (;;) {
        if (!(gg == gg)) { ret = moto_fail(c, MOTO_ESTATE, "moto_relax: NaN gradient"); break; }
        if (sqrt(gg) <= tau_F) { out.converged = 1; break; }
        if (out.steps >= max_steps) { ret = moto_fail(c, MOTO_ENOTCONV, "moto_relax: max_steps reached"); break; }
        double* xt = bufs[which];
        double a = alpha;
        bool accepted = false, first = true;
        for (int bt = 0; bt < RELAX_MAX_BACKTRACKS; ++bt) {
            s = eval_point(c, x, d, a, g, xt, gt, h);
            if (s != MOTO_OK) return s;
            out.evals += 1;
            const double Et = h[0], gtd = h[3];
            if (gtd <= RELAX_SIGMA * fabs(slope) && (Et <= E + RELAX_C1 * a * slope || Et <= E + RELAX_EPS_E * fabs(E))) { accepted = true; break; }
            a *= 0.5;
            first = false;
        }
        if (!accepted) {
            if (steepest) { ret = moto_fail(c, MOTO_ENOTCONV, "moto_relax: stalled (no acceptable step along -g)"); break; }
            k_relax_dir<<<grid, 256, 0, c->stream>>>(N, x, g, 0.0, d, 0);
            c->launches += 1;
            slope = -gg; steepest = true;
            continue;
        }
        const double Et = h[0], gtgt = h[1], gtg = h[2], gtd = h[3];
        double beta = (gtgt - gtg) / gg;
        if (!(beta > 0.0)) beta = 0.0;
        double new_slope = -gtgt + beta * gtd;
        if (new_slope >= 0.0) { beta = 0.0; new_slope = -gtgt; }
        k_relax_dir<<<grid, 256, 0, c->stream>>>(N, xt, gt, beta, d, spin);
        c->launches += 1;
        steepest = beta == 0.0;
        x = xt; which ^= 1;
        double* t = g; g = gt; gt = t;
        E = Et; gg = gtgt; slope = new_slope;
        alpha = first ? 2.0 * a : a;
        out.steps += 1;
    }
    if (x != d_state) MOTO_CUDA_CHECK(c, cudaMemcpyAsync(d_state, x, vb, cudaMemcpyDeviceToDevice, c->stream));
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    out.energy = E; out.gnorm = sqrt(gg); out.alpha = alpha;
    if (info) *info = out;
    return ret;
}

moto_status relax_seed(moto_ctx* c, const double* d_saddle, const double* d_v, double s_eta, double* d_out) {
    k_relax_trial<<<grid_for(c->N), 256, 0, c->stream>>>((long long)c->N, d_saddle, d_v, s_eta, d_out, c->kind == MOTO_KIND_TRI2D);
    c->launches += 1;
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    return MOTO_OK;
}

// ================================================================ outer MMF loop with a conjugate-gradient step rule
// (Alg. 1 l.12 "Lbfgs/CG"; reading A28): PR+ conjugate directions on the reflected force, one-trial secant line
// search on the force component along the direction (the translation step of the dimer method).  Two MinMode solves per
// iteration (trial point, new point), v_1-only re-solves with warm-started guard columns as in moto_mmf_run.
namespace {

struct ForceEval { double lam[MOTO_KMAX]; double fn; };

// F_mmf at y into F_out; V (k columns, modes at the previously evaluated point) is transported to y and re-solved
moto_status eval_force(moto_ctx* c, const double* y, int k, double tol, int max_iter, int warm, int transport, double* d_V, double* F_out,
                       bool full, ForceEval* fe, moto_mmf_info* acc) {
    double* d_lam = c->st->scal;
    double* d_fn = c->st->cheb_ab;
    if (transport) { moto_status t = moto_transport(c, y, d_V, k); if (t != MOTO_OK) return t; }
    moto_solve_info si = {};
    moto_status s = (c->opts.method == 0 && !full && max_iter > 0) ? solve_first_column(c, y, k, tol, max_iter, warm, d_lam, d_V, &si)
                                                                   : moto_lowest_modes(c, y, k, tol, max_iter, warm, d_lam, d_V, &si);
    if (s != MOTO_OK && s != MOTO_ENOTCONV) return s;
    acc->hvp_count += si.hvp_count; acc->solver_iters += si.iters;
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(fe->lam, d_lam, k * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    c->fmmf_out = F_out;
    s = moto_mmf_step(c, y, d_V, 1, 0.0, c->stage_m, d_fn);      // dt = 0: only the force and its norm are wanted
    c->fmmf_out = nullptr;
    if (s != MOTO_OK) return s;
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(&fe->fn, d_fn, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    return moto_check_overflow(c);   // atoms: a truncated neighbour table would give a silently wrong force
}

moto_status dots(moto_ctx* c, const double* a, const double* b0, const double* b1, const double* b2, int nb, double* h) {
    const double* S[1] = {a};
    const double* T[3] = {b0, b1 ? b1 : b0, b2 ? b2 : b0};
    c->launches += block_gram(c, S, 1, T, nb, c->st->scal, nullptr);
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(h, c->st->scal, nb * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    return MOTO_OK;
}

}  // namespace

moto_status mmf_cg_run(moto_ctx* c, double* d_state, int k, double delta, double smax, int max_steps, double tau_F, double tol, int max_iter,
                       int warm_start, double* d_V, double* d_scratch, moto_mmf_info* info) {
    const long long N = c->N;
    const size_t n3 = (size_t)3 * N, vb = n3 * sizeof(double);
    const int spin = c->kind == MOTO_KIND_TRI2D;
    const int grid = grid_for(N);
    double *F = d_scratch, *d = d_scratch + n3, *Fn = d_scratch + 2 * n3, *xt = d_scratch + 3 * n3;
    moto_mmf_info out; memset(&out, 0, sizeof(out));
    ForceEval fe;
    auto fail = [&](moto_status e) { if (info) *info = out; return e; };   // the caller always gets the counters so far
    moto_status st = eval_force(c, d_state, k, tol, max_iter, warm_start, 0, d_V, F, false, &fe, &out);
    if (st != MOTO_OK) return fail(st);
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(d, F, vb, cudaMemcpyDeviceToDevice, c->stream));
    bool full = c->opts.method != 0;
    moto_status ret = MOTO_OK;
    double h[3];
    for (int step = 0;; ++step) {
        // saddle test; lambda_2 decides only on converged pairs (see moto_mmf_run)
        if (!full && ((fe.fn <= tau_F && fe.lam[0] < 0.0 && fe.lam[1] > 0.0) || step >= max_steps)) {
            st = eval_force(c, d_state, k, tol, max_iter, 1, 0, d_V, F, true, &fe, &out);
            if (st != MOTO_OK) return fail(st);
            full = true;
        }
        out.steps = step; out.fnorm = fe.fn;
        for (int a = 0; a < k; ++a) out.lambda[a] = fe.lam[a];
        if (full && fe.fn <= tau_F && fe.lam[0] < 0.0 && fe.lam[1] > 0.0) { out.converged = 1; break; }
        if (step >= max_steps) { ret = moto_fail(c, MOTO_ENOTCONV, "moto_mmf_run_cg: max_steps reached before the saddle test held"); break; }
        full = c->opts.method != 0;
        st = dots(c, F, F, d, nullptr, 2, h);                         // F.F, F.d
        if (st != MOTO_OK) return fail(st);
        const double FF = h[0], Fd = h[1];
        st = dots(c, d, d, nullptr, nullptr, 1, h);                   // d.d
        if (st != MOTO_OK) return fail(st);
        const double dn = sqrt(h[0]);
        if (!(dn > 0.0) || !(FF > 0.0)) { ret = moto_fail(c, MOTO_ESTATE, "moto_mmf_run_cg: zero force"); break; }
        const double f0 = Fd / dn;
        k_relax_trial<<<grid, 256, 0, c->stream>>>(N, d_state, d, delta / dn, xt, spin);
        c->launches += 1;
        ForceEval ft;
        st = eval_force(c, xt, k, tol, max_iter, 1, 1, d_V, Fn, false, &ft, &out);
        if (st != MOTO_OK) return fail(st);
        st = dots(c, Fn, d, nullptr, nullptr, 1, h);                  // F_t.d  (F_t is tangent at x_t: transporting d changes nothing)
        if (st != MOTO_OK) return fail(st);
        const double f1 = h[0] / dn;
        const double Cv = (f0 - f1) / delta;
        double s = Cv > 0.0 ? f0 / Cv : smax;
        s = s > smax ? smax : (s < -smax ? -smax : s);
        k_relax_trial<<<grid, 256, 0, c->stream>>>(N, d_state, d, s / dn, d_state, spin);   // in place: element-wise
        c->launches += 1;
        st = eval_force(c, d_state, k, tol, max_iter, 1, 1, d_V, Fn, false, &fe, &out);
        if (st != MOTO_OK) return fail(st);
        st = dots(c, Fn, Fn, F, nullptr, 2, h);                       // F_new.F_new, F_new.F
        if (st != MOTO_OK) return fail(st);
        double beta = (h[0] - h[1]) / FF;
        if (!(beta > 0.0)) beta = 0.0;
        k_relax_dir<<<grid, 256, 0, c->stream>>>(N, d_state, Fn, beta, d, spin, 1.0);
        c->launches += 1;
        double* t = F; F = Fn; Fn = t;
    }
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    if (info) *info = out;
    return ret;
}

// ================================================================ L-BFGS variants (readings A29, A30; "We employ a
// GPU implementation of LBFGS ... and a nonlinear conjugate-gradient (CG) variant for comparison", :262, :275)
// The inverse-Hessian product is evaluated in the span of {q, s_1..s_n, y_1..y_n}: ONE Gram launch gives every inner
// product the two-loop recursion needs (the pairs are re-transported at every step, so their inner products change and are
// recomputed anyway), the recursion itself then runs on coefficient vectors on the host (it synchronises once per trial
// already), and ONE pass forms the direction as a linear combination.  Per accepted step: transport of the history (one
// projection pass over 2n vectors), new pair (one pass), Gram (one pass), combination (one pass).
namespace {

constexpr int LB_MAX = 8;                       // largest history M
constexpr int LB_NV = 2 * LB_MAX + 1;
constexpr double LB_CURV_EPS = 1e-10;

struct LinComb { const double* v[LB_NV]; double coef[LB_NV]; int n; };

__global__ void __launch_bounds__(256) k_lincomb(long long n3, LinComb lc, double* __restrict__ out) {
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n3; e += (long long)gridDim.x * blockDim.x) {
        double s = 0.0;
        for (int b = 0; b < lc.n; ++b) s = fma(lc.coef[b], lc.v[b][e], s);
        out[e] = s;
    }
}

// new pair at the accepted point xt:  s = a T(d),  y = sy (g_t - T(g))   (T = tangent projection at xt for spins, identity for atoms)
__global__ void __launch_bounds__(256) k_lbfgs_pair(long long N, const double* __restrict__ xt, const double* __restrict__ d, double a,
                                                    const double* __restrict__ gt, const double* __restrict__ g, double sy, int project,
                                                    double* __restrict__ s_out, double* __restrict__ y_out) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        d3 di = ld3(d, i), gi = ld3(g, i);
        if (project) { const d3 x = ld3(xt, i); di = proj3(x, di); gi = proj3(x, gi); }
        const d3 gn = ld3(gt, i);
        st3(s_out, i, scale3(a, di));
        st3(y_out, i, scale3(sy, sub3(gn, gi)));
    }
}

struct LbfgsHist {
    double* S[LB_MAX]; double* Y[LB_MAX];   // slot storage
    int order[LB_MAX + 1];                  // slots in use, oldest first
    int n, M;
};

// r = H q in coefficients over {q, S[order[0..n)], Y[order[0..n)]}; G: Gram of that basis, row-major (2n+1)^2, index 0 = q,
// 1 + i = s_i, 1 + n + i = y_i (i in history order).  gamma0: H_0 = gamma0 I when the history is empty.
void lbfgs_coeffs(const double* G, int n, double gamma0, double* r /*[2n+1]*/) {
    const int nb = 2 * n + 1;
    double q[LB_NV], al[LB_MAX];
    for (int b = 0; b < nb; ++b) q[b] = 0.0;
    q[0] = 1.0;
    if (n == 0) { r[0] = gamma0; return; }
    auto dot = [&](int row, const double* cf) { double s = 0.0; for (int b = 0; b < nb; ++b) s += cf[b] * G[row * nb + b]; return s; };
    for (int i = n - 1; i >= 0; --i) {
        const double rho = 1.0 / G[(1 + i) * nb + (1 + n + i)];
        al[i] = rho * dot(1 + i, q);
        q[1 + n + i] -= al[i];
    }
    const double gamma = G[(1 + n - 1) * nb + (1 + n + n - 1)] / G[(1 + n + n - 1) * nb + (1 + n + n - 1)];
    for (int b = 0; b < nb; ++b) r[b] = gamma * q[b];
    for (int i = 0; i < n; ++i) {
        const double rho = 1.0 / G[(1 + i) * nb + (1 + n + i)];
        const double be = rho * dot(1 + n + i, r);
        r[1 + i] += al[i] - be;
    }
}

// Gram of {q, S, Y} to the host (one launch pair + one synchronisation)
moto_status lbfgs_gram(moto_ctx* c, const LbfgsHist& h, const double* q, double* G_host, double* d_G) {
    const int nb = 2 * h.n + 1;
    const double* B[LB_NV];
    B[0] = q;
    for (int i = 0; i < h.n; ++i) { B[1 + i] = h.S[h.order[i]]; B[1 + h.n + i] = h.Y[h.order[i]]; }
    c->launches += block_gram(c, B, nb, B, nb, d_G, nullptr);
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(G_host, d_G, (size_t)nb * nb * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    return MOTO_OK;
}

// drop pairs whose curvature s.y is not safely positive (they would break positive definiteness); newest pair last.
// Returns true if the basis changed (the caller then rebuilds G by deleting rows / columns -- done here in place).
bool lbfgs_prune_newest(LbfgsHist& h, double* G) {
    if (h.n == 0) return false;
    const int n = h.n, nb = 2 * n + 1, i = n - 1;
    const double sy = G[(1 + i) * nb + (1 + n + i)], ss = G[(1 + i) * nb + (1 + i)], yy = G[(1 + n + i) * nb + (1 + n + i)];
    if (sy > LB_CURV_EPS * sqrt(ss) * sqrt(yy)) return false;
    // delete rows / columns (1 + i) and (1 + n + i)
    double T[LB_NV * LB_NV];
    int keep[LB_NV], nk = 0;
    for (int b = 0; b < nb; ++b) if (b != 1 + i && b != 1 + n + i) keep[nk++] = b;
    for (int a = 0; a < nk; ++a) for (int b = 0; b < nk; ++b) T[a * nk + b] = G[keep[a] * nb + keep[b]];
    memcpy(G, T, sizeof(double) * nk * nk);
    h.n = n - 1;
    return true;
}

void lbfgs_push_slot(LbfgsHist& h, int* slot_out) {
    // slot for a new pair: a free one, or the oldest (which is dropped)
    bool used[LB_MAX] = {false};
    for (int i = 0; i < h.n; ++i) used[h.order[i]] = true;
    if (h.n == h.M) { *slot_out = h.order[0]; for (int i = 1; i < h.n; ++i) h.order[i - 1] = h.order[i]; h.n -= 1; }
    else { int s = 0; while (used[s]) ++s; *slot_out = s; }
    h.order[h.n] = *slot_out;
    h.n += 1;
}

moto_status lbfgs_direction(moto_ctx* c, const LbfgsHist& h, const double* q, const double* r, double sign, double* out) {
    LinComb lc;
    lc.n = 2 * h.n + 1;
    lc.v[0] = q; lc.coef[0] = sign * r[0];
    for (int i = 0; i < h.n; ++i) {
        lc.v[1 + i] = h.S[h.order[i]]; lc.coef[1 + i] = sign * r[1 + i];
        lc.v[1 + h.n + i] = h.Y[h.order[i]]; lc.coef[1 + h.n + i] = sign * r[1 + h.n + i];
    }
    k_lincomb<<<grid_for(c->N), 256, 0, c->stream>>>(3ll * c->N, lc, out);
    c->launches += 1;
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    return MOTO_OK;
}

}  // namespace

// RelaxDownHill with L-BFGS (reading A29).  d_scratch: [2 M + 5][N][3].
moto_status relax_lbfgs_run(moto_ctx* c, double* d_state, int max_steps, double tau_F, double alpha0, int M, double* d_scratch,
                            moto_relax_info* info) {
    const long long N = c->N;
    const size_t n3 = (size_t)3 * N, vb = n3 * sizeof(double);
    const int spin = c->kind == MOTO_KIND_TRI2D;
    LbfgsHist h; memset(&h, 0, sizeof(h));
    h.M = M;
    for (int i = 0; i < M; ++i) { h.S[i] = d_scratch + (size_t)i * n3; h.Y[i] = d_scratch + (size_t)(M + i) * n3; }
    double* bufs[2] = {d_scratch + (size_t)(2 * M) * n3, d_scratch + (size_t)(2 * M + 1) * n3};
    double *g = d_scratch + (size_t)(2 * M + 2) * n3, *gt = d_scratch + (size_t)(2 * M + 3) * n3, *d = d_scratch + (size_t)(2 * M + 4) * n3;
    double* d_G = c->partials + 150000;           // device scratch for the Gram matrix (beyond the reduction partials in use)
    int which = 0;
    const double* x = d_state;
    moto_relax_info out; memset(&out, 0, sizeof(out));
    double hv[4], G[LB_NV * LB_NV], r[LB_NV];
    moto_status s = eval_point(c, x, nullptr, 0.0, nullptr, nullptr, g, hv);
    if (s != MOTO_OK) return s;
    out.evals = 1;
    double E = hv[0], gg = hv[1], alpha = alpha0;
    moto_status ret = MOTO_OK;
    for (;;) {
        if (!(gg == gg)) { ret = moto_fail(c, MOTO_ESTATE, "moto_relax_lbfgs: NaN gradient"); break; }
        if (sqrt(gg) <= tau_F) { out.converged = 1; break; }
        if (out.steps >= max_steps) { ret = moto_fail(c, MOTO_ENOTCONV, "moto_relax_lbfgs: max_steps reached"); break; }
        double* xt = bufs[which];
        bool accepted = false, first = true;
        double a = 0.0;
        int npairs = 0;
        for (;;) {
            npairs = h.n;
            double slope;
            if (npairs) {
                s = lbfgs_gram(c, h, g, G, d_G);
                if (s != MOTO_OK) return s;
                while (lbfgs_prune_newest(h, G)) {}
                npairs = h.n;
            }
            if (npairs) {
                lbfgs_coeffs(G, npairs, 1.0, r);
                const int nb = 2 * npairs + 1;
                slope = 0.0;
                for (int b = 0; b < nb; ++b) slope -= r[b] * G[b];          // g.d = -sum_b r_b <g, basis_b>
                if (!(slope < 0.0)) { h.n = 0; continue; }                   // not a descent direction: drop the history
                s = lbfgs_direction(c, h, g, r, -1.0, d);
                if (s != MOTO_OK) return s;
            } else {
                k_relax_dir<<<grid_for(N), 256, 0, c->stream>>>(N, x, g, 0.0, d, 0);   // d = -g
                c->launches += 1;
                slope = -gg;
            }
            a = npairs ? 1.0 : alpha;
            first = true;
            for (int bt = 0; bt < RELAX_MAX_BACKTRACKS; ++bt) {
                s = eval_point(c, x, d, a, g, xt, gt, hv);
                if (s != MOTO_OK) return s;
                out.evals += 1;
                const double Et = hv[0], gtd = hv[3];
                if (gtd <= RELAX_SIGMA * fabs(slope) && (Et <= E + RELAX_C1 * a * slope || Et <= E + RELAX_EPS_E * fabs(E))) { accepted = true; break; }
                a *= 0.5;
                first = false;
            }
            if (accepted || !npairs) break;
            h.n = 0;                                                          // every trial along the quasi-Newton direction rejected
        }
        if (!accepted) { ret = moto_fail(c, MOTO_ENOTCONV, "moto_relax_lbfgs: stalled (no acceptable step along -g)"); break; }
        if (!npairs) alpha = first ? 2.0 * a : a;
        // history to the new tangent space, then the new pair (its curvature is tested with the next Gram)
        if (spin && h.n > 0)
            for (int i = 0; i < h.n; ++i) { c->launches += spin_project(c, xt, h.S[h.order[i]], 1); c->launches += spin_project(c, xt, h.Y[h.order[i]], 1); }
        int slot;
        lbfgs_push_slot(h, &slot);
        k_lbfgs_pair<<<grid_for(N), 256, 0, c->stream>>>(N, xt, d, a, gt, g, 1.0, spin, h.S[slot], h.Y[slot]);
        c->launches += 1;
        x = xt; which ^= 1;
        double* t = g; g = gt; gt = t;
        E = hv[0]; gg = hv[1];
        out.steps += 1;
    }
    if (x != d_state) MOTO_CUDA_CHECK(c, cudaMemcpyAsync(d_state, x, vb, cudaMemcpyDeviceToDevice, c->stream));
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    out.energy = E; out.gnorm = sqrt(gg); out.alpha = alpha;
    if (info) *info = out;
    return ret;
}

// Outer climb with the L-BFGS step rule (reading A30).  d_scratch: [2 M + 4][N][3].
moto_status mmf_lbfgs_run(moto_ctx* c, double* d_state, int k, double alpha0, double smax, int max_steps, double tau_F, double tol,
                          int max_iter, int warm_start, int M, double* d_V, double* d_scratch, moto_mmf_info* info) {
    const long long N = c->N;
    const size_t n3 = (size_t)3 * N;
    const int spin = c->kind == MOTO_KIND_TRI2D;
    LbfgsHist h; memset(&h, 0, sizeof(h));
    h.M = M;
    for (int i = 0; i < M; ++i) { h.S[i] = d_scratch + (size_t)i * n3; h.Y[i] = d_scratch + (size_t)(M + i) * n3; }
    double *F = d_scratch + (size_t)(2 * M) * n3, *Fn = d_scratch + (size_t)(2 * M + 1) * n3, *p = d_scratch + (size_t)(2 * M + 2) * n3,
           *xn = d_scratch + (size_t)(2 * M + 3) * n3;
    double* d_G = c->partials + 150000;
    moto_mmf_info out; memset(&out, 0, sizeof(out));
    auto fail = [&](moto_status e) { if (info) *info = out; return e; };
    ForceEval fe;
    moto_status st = eval_force(c, d_state, k, tol, max_iter, warm_start, 0, d_V, F, false, &fe, &out);
    if (st != MOTO_OK) return fail(st);
    bool full = c->opts.method != 0;
    moto_status ret = MOTO_OK;
    double G[LB_NV * LB_NV], r[LB_NV];
    for (int step = 0;; ++step) {
        if (!full && ((fe.fn <= tau_F && fe.lam[0] < 0.0 && fe.lam[1] > 0.0) || step >= max_steps)) {
            st = eval_force(c, d_state, k, tol, max_iter, 1, 0, d_V, F, true, &fe, &out);
            if (st != MOTO_OK) return fail(st);
            full = true;
        }
        out.steps = step; out.fnorm = fe.fn;
        for (int a = 0; a < k; ++a) out.lambda[a] = fe.lam[a];
        if (full && fe.fn <= tau_F && fe.lam[0] < 0.0 && fe.lam[1] > 0.0) { out.converged = 1; break; }
        if (step >= max_steps) { ret = moto_fail(c, MOTO_ENOTCONV, "moto_mmf_run_lbfgs: max_steps reached before the saddle test held"); break; }
        full = c->opts.method != 0;
        // p = H F, capped at smax
        double pn2;
        for (;;) {
            st = lbfgs_gram(c, h, F, G, d_G);
            if (st != MOTO_OK) return fail(st);
            while (lbfgs_prune_newest(h, G)) {}
            const int nb = 2 * h.n + 1;
            lbfgs_coeffs(G, h.n, alpha0, r);
            double Fp = 0.0;
            for (int b = 0; b < nb; ++b) Fp += r[b] * G[b];
            if (h.n > 0 && !(Fp > 0.0)) { h.n = 0; continue; }
            pn2 = 0.0;
            for (int a = 0; a < nb; ++a) for (int b = 0; b < nb; ++b) pn2 += r[a] * r[b] * G[a * nb + b];
            break;
        }
        const double pn = sqrt(pn2 > 0.0 ? pn2 : 0.0);
        if (!(pn > 0.0)) { ret = moto_fail(c, MOTO_ESTATE, "moto_mmf_run_lbfgs: zero force"); break; }
        const double scale = pn > smax ? smax / pn : 1.0;
        st = lbfgs_direction(c, h, F, r, scale, p);
        if (st != MOTO_OK) return fail(st);
        k_relax_trial<<<grid_for(N), 256, 0, c->stream>>>(N, d_state, p, 1.0, xn, spin);
        c->launches += 1;
        st = eval_force(c, xn, k, tol, max_iter, 1, 1, d_V, Fn, false, &fe, &out);
        if (st != MOTO_OK) return fail(st);
        if (spin && h.n > 0)
            for (int i = 0; i < h.n; ++i) { c->launches += spin_project(c, xn, h.S[h.order[i]], 1); c->launches += spin_project(c, xn, h.Y[h.order[i]], 1); }
        int slot;
        lbfgs_push_slot(h, &slot);
        k_lbfgs_pair<<<grid_for(N), 256, 0, c->stream>>>(N, xn, p, 1.0, Fn, F, -1.0, spin, h.S[slot], h.Y[slot]);   // s = T(p), y = -(F_new - T(F))
        c->launches += 1;
        MOTO_CUDA_CHECK(c, cudaMemcpyAsync(d_state, xn, n3 * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
        double* t = F; F = Fn; Fn = t;
    }
    MOTO_CUDA_CHECK(c, cudaGetLastError());
    MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    if (info) *info = out;
    return ret;
}
