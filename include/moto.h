/* moto.h -- C ABI of libmoto.so: the B200-native (sm_100a, fp64) hot path of the bilayer
 * minimum-mode kernel of arxiv 2509.26269 ("MOTO").  Citations are PAPER.md:<line> of the paper
 * text and BASELINE.json:north_star; readings A1..A23 are listed in DESIGN.md.
 *
 * Conventions (all entry points)
 *   - Pointers named d_* are DEVICE pointers, h_* are HOST pointers; sizes are element counts.
 *   - Layouts: configuration  m or x : [N][3]   fp64, site/atom-major (Eq. 3)
 *              block of directions V : [k][N][3] fp64 (V_min = [v_1..v_k])
 *   - Ownership: the caller owns every array including the workspace; the library allocates no
 *     device memory (it keeps one small pinned host status buffer per context).
 *   - All work is enqueued on the CUDA stream given to moto_create.  Calls return after
 *     enqueueing, except moto_lowest_modes and the *_host variants, which synchronise the stream.
 *   - Errors: every call returns a moto_status; nothing aborts or throws.  moto_last_error gives
 *     a message.  MOTO_ENOTCONV still leaves the best iterate and its residuals in the outputs.
 *   - There is no CPU fallback: without a CUDA device every compute call returns MOTO_ECUDA.
 */
#ifndef MOTO_H
#define MOTO_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MOTO_KMAX 8            /* largest block size k accepted by moto_hvp / moto_lowest_modes */
#define MOTO_NSMAX (3 * MOTO_KMAX) /* largest Rayleigh-Ritz basis [X,W,P] */

typedef struct moto_ctx moto_ctx; /* opaque */

typedef enum {
    MOTO_OK = 0,
    MOTO_EINVAL = 1,   /* bad argument (k out of range, NULL pointer, bad lattice, workspace too small) */
    MOTO_ENOMEM = 2,   /* host allocation failed / neighbour capacity exceeded */
    MOTO_ECUDA = 3,    /* a CUDA runtime call failed (message in moto_last_error) */
    MOTO_ENOTCONV = 4, /* eigen-solver hit max_iter; outputs hold the best iterate */
    MOTO_ESTATE = 5    /* call not valid for this context kind */
} moto_status;

enum { MOTO_KIND_TRI2D = 0, MOTO_KIND_CARTESIAN = 1 };

/* Lattice / atom container.
 * kind 0: 2-D triangular spin lattice, site i = iy*Lx + ix at r_i = ix*a1 + iy*a2, a1=(1,0),
 *         a2=(1/2,sqrt3/2); six neighbours at offsets (+-1,0),(0,+-1),(-1,+1),(+1,-1); pbc_x/pbc_y
 *         select periodic (1) or open (0) boundaries (open: the missing neighbour contributes 0).
 * kind 1: n_atoms Cartesian atoms, periodic in the in-plane cell spanned by the rows of cell
 *         (Angstrom), open in z.  d_fixed: optional device mask [N], 1 = frozen (the paper's mask
 *         Omega); NULL = all free.  Ignored for kind 0. */
typedef struct {
    int32_t kind;
    int32_t Lx, Ly;
    int32_t pbc_x, pbc_y;
    int32_t n_atoms;
    double cell[2][2];
    const uint8_t* d_fixed;
} moto_lattice;

/* Eq. 4, nearest neighbours only: exchange J, interfacial DMI
 * D_ij = D (z x rhat_ij) with rhat_ij = r_j - r_i, easy axis z with strength K, field B, moment mu.
 * The pair sums run over ORDERED pairs i != j exactly as printed (reading A1). */
typedef struct { double J, D, K, B[3], mu; } moto_spin_params;

/* Morse pair potential phi(r) = De[exp(-2 alpha (r-r0)) - 2 exp(-alpha (r-r0))], r < rc
 * (BASELINE.json configs[4]); energy shifted by -phi(rc) per pair (reading A21). */
typedef struct { double De, alpha, r0, rc; } moto_morse_params;

/* Eigen-solver knobs (PAPER.md:120 names Krylov depth / reorthogonalisation as the sensitive ones).
 * Zero-initialise and pass to moto_set_solver to change the defaults given in brackets. */
typedef struct {
    int32_t guard;          /* extra block columns iterated but not returned            [0]  */
    int32_t check_every;    /* iterations enqueued between host looks at the status; 0 = auto: 8 plain LOBPCG iterations,
                               2 iterations on the transformed operator (each is d operator applications long)  [0]  */
    int32_t precond_degree; /* degree d of the Chebyshev spectral transformation -p_d(A) LOBPCG runs on:
                               0 = auto (40 on spin lattices that take the TMA K1 path with kb <= 2; 32 with kb > 2 (soft locking) on every nearest-neighbour
                               lattice with even Lx >= 8 and at least 512 sites, the TMA path switched on for the solve; 16 inside the
                               persistent small-lattice kernel and on general shells with the dense kernel, 24 for Cartesian atoms
                               with kb <= 2 and at most 8192 atoms, else off),
                               -1 = off (plain LOBPCG on A, the paper's solver), 1..256 = degree          [0]  */
    int32_t hvp_path;       /* K1 kernel choice: 0 auto, 1 generic (any lattice), 2 TMA-staged (even Lx >= 8) [0] */
    double precond_lo;      /* margin: the damped interval starts at theta_k + margin           [0 -> 0.01] */
    double precond_hi;      /* upper end b >= lambda_max of the damped interval    [0 -> max(-c_i) + ||L||] */
    uint64_t seed;          /* seed of the counter-based start block when warm_start=0  [0x9E3779B97F4A7C15] */
    int32_t method;         /* 0 = block LOBPCG, 1 = thick-restart Lanczos with full re-orthogonalisation
                               (single start vector, guard / precond_* ignored)          [0]  */
    int32_t ncv;            /* Lanczos basis size m, k + 2 <= m <= min(24, S kmax - 1, dof - 1) with S = 8 blocks
                               (spin lattices) or 6 (Cartesian) of the workspace; 0 = the largest that fits   [0]  */
    int32_t cheb_mode;      /* how the degree-d recurrence of -p_d(A) (product form: d steps alpha_s (A - r_s), k_cheb_coef) is launched
                               on the TMA K1 path: 0 = auto (= 3, the fastest as measured at 10^6 spins), 1 = one step per pass in one
                               persistent cooperative launch, 2 = d dependent launches, 3 = two steps per pass in one cooperative
                               launch with the intermediate step kept in shared memory (spin_cheb2_tma.cu; odd d: + one single
                               step; block sizes above 2: all column pairs side by side in that one launch, each pair on its
                               own share of the SMs).  All give bit-identical results.                                  [0]  */
    int32_t persistent;     /* the whole solve as ONE persistent cooperative kernel (nearest-neighbour spin lattices up to 37 888
                               sites = 148 SMs x 256, k <= 2, no guard columns, method 0): 0 = where it applies, unless an explicit
                               precond_degree > 0 asks for the multi-launch transformed solver; 1 = also with an explicit
                               precond_degree <= 32; 2 = never (the multi-launch solver).  Inside the kernel precond_degree 0 = auto
                               means degree 16 from 128 sites on (plain LOBPCG below), -1 = plain.                  [0]  */
} moto_solver_opts;

typedef struct {
    int32_t iters;              /* LOBPCG iterations executed */
    int32_t converged;          /* 1 if every returned column met tol */
    double resid[MOTO_KMAX];    /* ||Hess v_j - lambda_j v_j||_2 of the returned columns */
    int64_t hvp_count;          /* single-vector HVP applications (k per block HVP) */
} moto_solve_info;

/* Bytes of device workspace moto_create needs for block sizes up to kmax (<= MOTO_KMAX, guard included). */
size_t moto_workspace_bytes(const moto_lattice* lat, int kmax);

/* Build a context.  params: moto_spin_params* (kind 0) or moto_morse_params* (kind 1), copied.
 * d_workspace: device buffer of >= moto_workspace_bytes bytes, 256-byte aligned, owned by the
 * caller and alive until moto_destroy.  cuda_stream: a cudaStream_t (NULL = default stream). */
moto_status moto_create(const moto_lattice* lat, const void* params, void* d_workspace, size_t ws_bytes,
                        void* cuda_stream, int kmax, moto_ctx** out);
void moto_destroy(moto_ctx* ctx);
moto_status moto_set_solver(moto_ctx* ctx, const moto_solver_opts* opts);
const char* moto_last_error(const moto_ctx* ctx);

/* General neighbour shells (Eq. 4, is written for arbitrary pairs and the paper's
 * Pd/Fe/Ir(111) workload tabulates J_ij and three-component D_ij over ~340 neighbours per site):
 * replace the nearest-neighbour J, D of moto_spin_params by a translation-invariant table over lattice offsets,
 *   J_ij = h_J[t], D_ij = h_D[t][0..2]  for  j = i + (h_offsets[t][0], h_offsets[t][1])   (K, B, mu stay as created).
 * All three arrays are HOST pointers, copied (n <= 512).  The table must hold distinct non-zero offsets and be inversion
 * symmetric, J(-d) = J(d), D(-d) = -D(d) (the same bond seen from its other end, reading A2), else MOTO_EINVAL.  Ordered
 * pairs are counted as printed (reading A1).  n = 0 returns to the nearest-neighbour model.  Kind 0 only.  Every call
 * (energy_grad, hvp, lowest_modes, mmf_step, mmf_run, relax, ...) then runs on the table.  Energy / gradient and block HVPs of k <= 2 directions on
 * lattices with Lx >= 32 take the register-blocked kernel of spin_shells_dense.cu (table as dense column segments, fields staged
 * in shared memory, at most 1024 dense entries incl. zero-filled holes); there moto_cheb_apply works (d launches) and
 * moto_lowest_modes runs LOBPCG on the Chebyshev transformation -p_16(A) by default (precond_degree 0; -1 = plain).  Everything
 * else (k > 2, Lx < 32) runs on the warp-per-site kernels of spin_shells.cu, without the transformation.
 * The TMA path and the persistent small-lattice kernel are nearest-neighbour only. */
moto_status moto_set_shells(moto_ctx* ctx, int n, const int32_t* h_offsets, const double* h_J, const double* h_D);

/* E(m) and its gradient.  d_E: [1] device.  d_g: [N][3] device, may be NULL.
 * kind 0: d_g = tangent-projected gradient P g = g - (m.g) m ("forces ... understood as
 *         tangent-projected").   kind 1: Euclidean gradient, rows of fixed atoms zero. */
moto_status moto_energy_grad(moto_ctx* ctx, const double* d_spins, double* d_E, double* d_g);

/* Block Hessian-vector product (north_star): for each column a,
 * kind 0: HV_a = P (L Pv_a) - (m.g) Pv_a   (input projected, output tangent, reading A5)
 * kind 1: HV_a = M H M v_a, M = mask of free atoms.   d_V, d_HV: [k][N][3]; must not alias.
 * The call is stateless: on Cartesian atoms moto_hvp and moto_energy_grad rebuild the cell list and the neighbour table from
 * d_spins (= positions) on every call (three small launches, most of the ~55 us of a call at 1607 atoms); the solvers
 * (moto_lowest_modes, moto_mmf_run*, moto_relax*) build them once per state and apply the operator on the stored table. */
moto_status moto_hvp(moto_ctx* ctx, const double* d_spins, const double* d_V, int k, double* d_HV);

/* Smallest-k eigenpairs of the (masked) tangent Hessian by device-resident block LOBPCG
 * (ref [27]).  Stops when every ||Hess v_j - lambda_j v_j||_2 <= tol
 * (absolute, ||v_j|| = 1; reading A9) or after max_iter iterations (paper's cap: 200).
 * warm_start = 1: d_V holds a start block (any full-rank block; it is projected and orthonormalised).
 * Outputs: d_lambda [k] ascending; d_V [k][N][3] tangent, orthonormal, sign-normalised so the
 * largest-|component| entry of each column is positive; info (host) may be NULL. */
moto_status moto_lowest_modes(moto_ctx* ctx, const double* d_spins, int k, double tol, int max_iter,
                              int warm_start, double* d_lambda, double* d_V, moto_solve_info* info);

/* Population solve (Alg. 1 l.3-5: the explorer evaluates (lambda_1, lambda_2) once per candidate per
 * generation, P = 24 in the paper): moto_lowest_modes on P independent problems at once.
 * ctxs[p] are P DISTINCT contexts; every array argument is a HOST array of P device pointers / P structs, entry p with the
 * meaning it has in moto_lowest_modes.
 * Batched path: when all contexts describe the same nearest-neighbour spin lattice (size, boundaries, parameters) small enough
 * for the persistent solver (moto_solver_opts.persistent; k <= 2), the P solves run inside ONE cooperative kernel launch per 24
 * problems on ctxs[0]'s stream: problem index = a grid dimension, a barrier among the CTAs of one problem only, one
 * Rayleigh-Ritz per problem and iteration on the device, problems finish at their own iteration counts.
 * Otherwise (different lattices, atoms, general shells, larger lattices): one host thread per context (at most 32 at a time),
 * each driving the multi-launch solver on its context's own stream, so that the P launch chains overlap -- create the
 * contexts on their OWN streams for that; in
 * moto_lowest_modes.  Inputs must be complete on the device before the call (the contexts' streams are not ordered against
 * the stream that produced them).  statuses [P] (host, may be NULL) receives each problem's status; the return value is MOTO_OK,
 * MOTO_ENOTCONV if some problem hit max_iter (and none failed), else the first failure.  Results are bit-identical to P
 * separate moto_lowest_modes calls. */
moto_status moto_lowest_modes_batch(moto_ctx* const* ctxs, int P, const double* const* d_spins, int k, double tol, int max_iter,
                                    int warm_start, double* const* d_lambda, double* const* d_V, moto_solve_info* infos,
                                    int32_t* statuses);

/* One reflected-force step (Eq. 2; Alg. 1 l.11-12):
 * F = -grad (tangent-projected / masked), F_mmf = F - 2 sum_a (F.v_a) v_a over the kr columns given,
 * kind 0: m' = normalize(m + dt F_mmf) per site (retraction);  kind 1: x' = x + dt F_mmf.
 * d_spins_out may alias d_spins.  d_fnorm: optional [1] device, receives ||F_mmf||_2. */
moto_status moto_mmf_step(moto_ctx* ctx, const double* d_spins, const double* d_v, int kr, double dt,
                          double* d_spins_out, double* d_fnorm);

/* Outer minimum-mode-following loop with the paper's termination test (Alg. 1 l.9-14; SURVEY 8(f) f2,
 * fixed step instead of a line search):
 *   repeat:  (lambda, V) <- lowest k modes at x (warm-started from the transported V of the previous step)
 *            F_mmf = F - 2 (F.v_1) v_1                                  (Eq. 2; v_1 only)
 *            if ||F_mmf||_2 <= tau_F and lambda_1 < 0 < lambda_2: stop, x is an index-1 saddle
 *            x <- R(x + dt F_mmf)                                        (retraction for spins)
 * d_state [N][3] in/out; d_V [k][N][3]: start block if warm_start, holds the modes at the final x on return; k >= 2
 * (the test needs lambda_2).  info->steps = updates applied, info->converged = the test held at the returned x.
 * With the block LOBPCG solver the per-step re-solve converges v_1 only (the reflected force needs nothing else); the other
 * k-1 columns are iterated and warm-started with it as guard columns, which leaves a Ritz value theta_2 >= lambda_2.  All k
 * columns are converged to tol where lambda_2 decides -- when ||F_mmf|| <= tau_F with lambda_1 < 0 < theta_2, and at the last
 * step -- so the test and the returned eigenvalues always use converged pairs.  (Lanczos: all k columns every step.)
 * Returns MOTO_ENOTCONV if max_steps was reached without the test holding (outputs valid), or the solver's status if an
 * inner solve failed.  Synchronises the stream once per step (two scalars and k eigenvalues come back). */
typedef struct {
    int32_t steps;              /* updates applied */
    int32_t converged;          /* 1: ||F_mmf|| <= tau_F and lambda_1 < 0 < lambda_2 at the returned state */
    double fnorm;               /* ||F_mmf||_2 at the returned state */
    double lambda[MOTO_KMAX];   /* lowest eigenvalues at the returned state */
    int64_t hvp_count;          /* single-vector HVPs over all inner solves */
    int64_t solver_iters;       /* LOBPCG iterations over all inner solves */
} moto_mmf_info;
moto_status moto_mmf_run(moto_ctx* ctx, double* d_state, int k, double dt, int max_steps, double tau_F, double tol, int max_iter,
                         int warm_start, double* d_V, moto_mmf_info* info);

/* The same outer loop with a conjugate-gradient step rule (Alg. 1 l.12: "x <- R_x(x + alpha F_mmf)  > Lbfgs/CG", PAPER.md:262;
 * SURVEY 8(f) f2).  F_mmf is not the gradient of a function, so there is no energy line search; reading A28 is the
 * translation step of the dimer method: Polak-Ribiere+ conjugate directions on the reflected force with a one-trial secant
 * line search on the force component along the direction,
 *   dh = d/|d|, f0 = F_mmf(x).dh;  trial x_t = R(x + delta dh), f1 = F_mmf(x_t).dh;  C = (f0 - f1)/delta;
 *   s = f0/C if C > 0 else smax, clipped to [-smax, smax];  x <- R(x + s dh);
 *   beta = max(0, F_new.(F_new - F)/(F.F));  d <- F_new + beta T(d)      (T: tangent projection for spins, identity for atoms)
 * i.e. two minimum-mode solves per iteration (v_1-only re-solves as in moto_mmf_run) instead of one, and an order of
 * magnitude fewer iterations.  delta: trial displacement, smax: largest displacement per iteration, both in the 2-norm of
 * the whole configuration.  d_scratch: caller-owned device scratch [4][N][3].  Other arguments, outputs, termination test
 * and return values as moto_mmf_run; info->steps counts iterations. */
moto_status moto_mmf_run_cg(moto_ctx* ctx, double* d_state, int k, double delta, double smax, int max_steps, double tau_F, double tol,
                            int max_iter, int warm_start, double* d_V, double* d_scratch, moto_mmf_info* info);

/* Two-sided minimum-mode descent (Alg. 1 l.15-18; Suppl. Note 1 b(iii)).
 * moto_relax: "RelaxDownHill" with a deterministic optimiser.  The paper names the class ("L-BFGS/CG") and nothing else;
 *   this is Riemannian Polak-Ribiere+ conjugate gradients with backtracking (reading A26):
 *     trial x_t = R(x + a d), a = alpha, alpha/2, ... (<= 40);  accepted when g_t.d <= 0.5 |g.d| and
 *     (E_t <= E + 1e-4 a g.d  or  E_t <= E + 1e-10 |E|);  beta = max(0, (g_t.g_t - g_t.g)/(g.g));
 *     d <- -g_t + beta T(d) (T = tangent projection at x_t for spins, identity for atoms; reset to -g_t if not a descent
 *     direction);  alpha <- 2a if the first trial was accepted, else a.  g = tangent-projected / masked gradient.
 *   d_state [N][3] in/out (unit spins / positions).  Stops when ||g||_2 <= tau_F (MOTO_OK, converged = 1), after
 *   max_steps accepted steps or when no step along -g is acceptable (MOTO_ENOTCONV; d_state = best iterate, info valid).
 *   alpha0 > 0: first trial step.  Spin lattices: the accept/reject decisions are taken on the device, the host looks at the
 *   state once per eight trials; atoms (and general shells): one synchronisation per trial (four scalars come back).  Uses the solver
 *   blocks of the workspace as scratch: modes left there by an earlier solve are overwritten (user arrays are not).
 * moto_two_sided_descent: seeds x_saddle + s eta v_min, s = +1 then -1 (retracted for spins), each relaxed as above into
 *   d_min_plus / d_min_minus [N][3] (must not alias the inputs or each other); info[2] (host, may be NULL) in that order.
 *   Returns MOTO_ENOTCONV if either branch did not converge (both outputs valid). */
typedef struct {
    int32_t steps;       /* accepted steps */
    int32_t converged;   /* 1: ||g|| <= tau_F at the returned state */
    int32_t evals;       /* energy + gradient evaluations (one per trial, plus the first) */
    int32_t pad_;
    double energy;       /* E at the returned state */
    double gnorm;        /* ||g||_2 at the returned state */
    double alpha;        /* trial step the next iteration would start from */
} moto_relax_info;
moto_status moto_relax(moto_ctx* ctx, double* d_state, int max_steps, double tau_F, double alpha0, moto_relax_info* info);
moto_status moto_two_sided_descent(moto_ctx* ctx, const double* d_saddle, const double* d_vmin, double eta, int max_steps,
                                   double tau_F, double alpha0, double* d_min_plus, double* d_min_minus, moto_relax_info* info);

/* The L-BFGS variants of the two loops above -- the paper's primary optimiser ("We employ a GPU implementation of
 * LBFGS ... and a nonlinear conjugate-gradient (CG) variant for comparison"; Alg. 1 l.12, l.17).  The paper calls
 * a library routine and prints no algorithm; readings A29, A30:
 * moto_relax_lbfgs: RelaxDownHill.  History of at most m pairs s = T(a d), y = g_new - T(g_old), all transported to the current
 *   tangent space at every accepted step (projection for spins, identity for atoms); d = -H g by the two-loop recursion with
 *   H_0 = (s.y / y.y) I of the newest pair, d = -g while the history is empty; a pair is kept only if s.y > 1e-10 |s| |y|;
 *   acceptance test of moto_relax (reading A26) on trial steps a = a_0, a_0/2, ... with a_0 = 1 (alpha0-scaled first-step
 *   length while the history is empty); a direction that is not downhill or along which every trial fails drops the history.
 *   d_scratch: caller-owned device scratch [2 m + 5][N][3].  info / return values as moto_relax.  One synchronisation per trial.
 * moto_mmf_run_lbfgs: the outer climb, x <- R(x + p), p = H F_mmf with pairs s = T(p), y = -(F_new - T(F_old)), H_0 = alpha0 I
 *   while the history is empty, |p|_2 capped at smax, history dropped if F.p <= 0.  ONE minimum-mode solve per iteration
 *   (moto_mmf_run_cg spends two).  d_scratch: [2 m + 4][N][3].  Other arguments, termination test, info and return values as
 *   moto_mmf_run.  1 <= m <= 8. */
moto_status moto_relax_lbfgs(moto_ctx* ctx, double* d_state, int max_steps, double tau_F, double alpha0, int m, double* d_scratch,
                             moto_relax_info* info);
moto_status moto_mmf_run_lbfgs(moto_ctx* ctx, double* d_state, int k, double alpha0, double smax, int max_steps, double tau_F, double tol,
                               int max_iter, int warm_start, int m, double* d_V, double* d_scratch, moto_mmf_info* info);

/* Vector transport for warm starts after m -> m' (reading A17): V <- orthonormalise(P_{m'} V), in place. */
moto_status moto_transport(moto_ctx* ctx, const double* d_spins_new, double* d_V, int k);

/* Building blocks of the LOBPCG iteration, exported so they can be tested alone.
 * moto_gram: G[i][j] = S_i . T_j for block vectors S [ns][N][3], T [nt][N][3]; d_G [ns][nt] row-major.
 * moto_rayleigh_ritz: lowest nev pairs of G_A c = theta G_B c (n <= MOTO_NSMAX, row-major symmetric,
 *   G_B positive semi-definite: near-null directions are dropped); d_theta [nev], d_C [n][nev] with
 *   C^T G_B C = I.  Single CTA, Jacobi; nothing leaves the GPU. */
moto_status moto_gram(moto_ctx* ctx, const double* d_S, int ns, const double* d_T, int nt, double* d_G);
moto_status moto_rayleigh_ritz(moto_ctx* ctx, const double* d_GA, const double* d_GB, int n, int nev,
                               double* d_theta, double* d_C);

/* One step of the three-term recurrence the transformed solver is made of (the kernel that dominates
 * moto_lowest_modes), exported so it can be tested and timed alone:
 *   d_out = alpha (Hess[V] - c0 V) + beta U      (U may be NULL: beta ignored; d_out may alias d_U, not d_V)
 * kind 0 only.  V must be tangent (it is NOT re-projected: solver mode, reading A24); c_i = m_i.g_i is recomputed
 * from d_spins when refresh_c != 0, else the values cached in the workspace by the previous call are used. */
moto_status moto_hvp_three_term(moto_ctx* ctx, const double* d_spins, const double* d_V, int k, double alpha, double c0,
                                double beta, const double* d_U, double* d_out, int refresh_c);

/* The operator the transformed solver runs LOBPCG on, exported so it can be tested and timed alone:
 *   d_out = -p_d(Hess) V ,  p_d = Chebyshev polynomial of degree d scaled so that p_d(a_L) = 1, |p_d| <= 1 on [a, b]
 * (Zhou-Saad three-term form: sigma_1 = e/(a_L - c0), e = (b-a)/2, c0 = (b+a)/2;  Y_1 = (sigma_1/e)(A - c0) V,
 *  Y_{i+1} = (2 sigma_{i+1}/e)(A - c0) Y_i - sigma_i sigma_{i+1} Y_{i-1}, sigma_{i+1} = 1/(2/sigma_1 - sigma_i)).
 * kind 0 only, k <= 2, 1 <= d <= 256, V tangent (solver mode), a_L < a < b.  On lattices that take the TMA K1 path
 * the whole recurrence is ONE persistent cooperative launch; otherwise d launches.  d_out must not alias d_V.
 * refresh_c as in moto_hvp_three_term. */
moto_status moto_cheb_apply(moto_ctx* ctx, const double* d_spins, const double* d_V, int k, int d, double a, double b,
                            double a_L, double* d_out, int refresh_c);

/* Host-buffer variants (end-to-end path): same semantics, all array arguments are HOST pointers
 * (pinned or pageable); the library stages them through its workspace (host->device, compute,
 * device->host) and synchronises the stream before returning. */
moto_status moto_energy_grad_host(moto_ctx* ctx, const double* h_spins, double* h_E, double* h_g);
moto_status moto_hvp_host(moto_ctx* ctx, const double* h_spins, const double* h_V, int k, double* h_HV);
moto_status moto_lowest_modes_host(moto_ctx* ctx, const double* h_spins, int k, double tol, int max_iter,
                                   int warm_start, double* h_lambda, double* h_V, moto_solve_info* info);
moto_status moto_mmf_step_host(moto_ctx* ctx, const double* h_spins, const double* h_v, int kr, double dt,
                               double* h_spins_out, double* h_fnorm);

/* Cartesian atoms: the neighbour table holds at most 160 neighbours per atom.  moto_lowest_modes, moto_mmf_run*, moto_relax and the
 * *_host variants check the overflow flag themselves (MOTO_ENOMEM); the asynchronous device-pointer calls moto_energy_grad,
 * moto_hvp and moto_mmf_step do not wait for it -- call this after them (it synchronises the stream) when the density of the
 * configuration is not known to be safe.  MOTO_OK for spin lattices. */
moto_status moto_check_overflow(moto_ctx* ctx);

/* moto_gram_static: moto_gram for callers that cannot allocate (CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc).  No context and no workspace: G[i][j] = S_i . T_j (the reduced pencil of LOBPCG) for
 *   d_S [ns][n3], d_T [nt][n3] device, fp64, rows of n3 contiguous elements (n3 = 3 N for a block vector); d_G [ns][nt]
 *   device, row-major, written by the kernel; stream: a cudaStream_t passed as a plain pointer (NULL = the default stream).
 * Limit: ns <= 6 and nt <= 12 (the [X W P] x [S, A S] pencil at block size 2); anything larger returns MOTO_EINVAL and
 * launches nothing -- use moto_gram.  The per-CTA partial sums live in a file-scope __device__ array (170 752 bytes on every
 * GPU that loads the library, held until the process exits); the call performs no cudaMalloc / cudaFree and calls no
 * allocating library routine: one 256-byte cudaMemsetAsync (the ticket of the reduction) and one kernel, asynchronous on
 * `stream`; the caller owns all buffers.  ALL calls on a device share that array: calls that overlap on the GPU (two streams,
 * no dependency between them) race; order them.  Sums are formed in a fixed order (bit-identical reruns).
 * moto_gram_static_last_error: message of this host thread's last failed moto_gram_static call ("" after a success). */
moto_status moto_gram_static(const double* d_S, int ns, const double* d_T, int nt, int64_t n3, double* d_G, void* stream);
const char* moto_gram_static_last_error(void);

/* Number of kernels this context has launched so far (bench.py's gpu_launches). */
int64_t moto_launch_count(const moto_ctx* ctx);
const char* moto_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MOTO_H */
