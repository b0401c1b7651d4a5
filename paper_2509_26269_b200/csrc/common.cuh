// common.cuh -- context, device-side solver state and launch prototypes shared by the libmoto
// translation units.  Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
#include "../../include/moto.h"

#define MOTO_NS MOTO_NSMAX   // 24
#define MOTO_NUM_SMS 148     // B200
#define MOTO_LZ_MAX 24       // largest Lanczos basis (the single-CTA Jacobi solves up to MOTO_NS = 24)
#define MOTO_RED_BLOCKS 296  // CTAs of every grid-reduction kernel (2 per SM): fixed => deterministic sums
#define MOTO_MAX_NEIGH 160   // Cartesian: neighbour capacity per atom
#define MOTO_MAX_SHELLS 512 // largest neighbour table of moto_set_shells
#define MOTO_SH_DENSE 1024  // dense column-segment form of the table: entries (zero-filled holes included) ...
#define MOTO_SH_SEGS 128    // ... segments of <= 12 taps of one dx column ...
#define MOTO_SH_GROUPS 16   // ... and tap groups (warps of a CTA)
#define MOTO_CHEB_MAX 256    // largest degree of the Chebyshev spectral transformation

// Device-resident LOBPCG state: Gram matrices, Ritz coefficients, residuals, control flags.
// Lives in the workspace; the host only ever reads the tail (ctl) through a pinned copy.
struct SolverState {
    double GA[MOTO_NS * MOTO_NS];
    double GB[MOTO_NS * MOTO_NS];
    double C[MOTO_NS * MOTO_KMAX];   // [ns][kb] coefficients of the new X in the basis [X,W,P]
    double scal[8];                  // scratch scalars: F.v dots, signs ...
    double ack[2 * MOTO_KMAX];       // A-residual check (lobpcg_fast.cu): theta_j = x_j.A x_j / x_j.x_j at [j], x_j.x_j at [KMAX + j]
    double cheb[MOTO_CHEB_MAX][4];   // per-step {alpha, c0, beta, -} of the Chebyshev recurrence (k_cheb_coef)
    double cheb_ab[4];               // a, b, a_L, scale of the current transformation
    int leja_d, leja_pad;            // degree whose Leja root order is in leja[] (0: none)
    unsigned char leja[MOTO_CHEB_MAX];   // Leja order of the Chebyshev roots (product form of the filter, k_cheb_coef)
    // ---- thick-restart Lanczos (lanczos.cu)
    double lz_T[MOTO_LZ_MAX * MOTO_LZ_MAX];   // projected matrix V^T A V: tridiagonal, bordered-diagonal after a restart
    double lz_Y[MOTO_LZ_MAX * MOTO_KMAX];     // [m][k] Ritz coefficients of the restart
    double lz_h[MOTO_LZ_MAX + 1];             // Gram-Schmidt coefficients of the current pass
    double lz_beta, lz_rbeta;                 // ||u|| of the current step and its reciprocal
    int lz_cycle, lz_pad;                     // index of the last restart cycle whose Rayleigh-Ritz ran
    unsigned long long pbar;                  // barrier counter of the persistent small-lattice solver (lobpcg_persistent.cu)
    int lock_on, lock_pad;                    // soft locking (generic transformed LOBPCG): columns with locked[j] get no new W_j / P_j
    int locked[MOTO_KMAX];
    // ---- tail mirrored to the host (layout == HostStatus)
    double theta[MOTO_KMAX];
    double resid[MOTO_KMAX];
    int done;      // 1 once all wanted residuals <= tol (kernels early-exit)
    int iter;      // iterations completed
    int nkeep;     // basis directions kept by the last Rayleigh-Ritz
    int bad;       // 1 if a NaN/breakdown was seen
    long long nhvp;  // single-vector HVP applications so far
};

// Device-resident line-search state of moto_relax on spin lattices (relax.cu): the accept/reject decision of a trial is taken by
// k_relax_decide, the next trial reads its step, buffers and direction mode from here -- no host look per trial.
struct RelaxDev {
    double E, gg, slope, alpha, a, beta, tau;
    int cur, gcur;        // current state buffer (0 = the caller's array, 1, 2 = workspace), current gradient buffer (0, 1)
    int steepest, first, bt, steps, evals, max_steps;
    int status;           // 0 running, 1 converged, 2 max_steps, 3 stalled, 4 NaN
    int dir_mode;         // what k_relax_dir does next: 0 nothing, 1 d <- -g + beta T(d), 2 d <- -g
    double* x[3];
    double* g[2];
    double* d;
};

struct HostStatus {  // pinned mirror of the control block + residuals
    double theta[MOTO_KMAX];
    double resid[MOTO_KMAX];
    int done, iter, nkeep, bad;
    long long nhvp;
};

struct CartLists {
    int ncx, ncy, ncell;
    int* cell_of;      // [Na]
    int* cell_count;   // [ncell]
    int* cell_start;   // [ncell+1]
    int* cell_atoms;   // [Na] sorted by (cell, atom id)
    int* nb_count;     // [Na]
    int* nb_idx;       // [Na][MOTO_MAX_NEIGH] neighbour ids, ascending
    double* nb_coef;   // [Na][MOTO_MAX_NEIGH][5]: nx, ny, nz, phi'', phi'/r
    int* overflow;     // [1] set if an atom exceeded MOTO_MAX_NEIGH
};

struct moto_ctx {
    moto_lattice lat;
    int kind;
    int N;       // sites or atoms
    int kmax;
    moto_spin_params sp;
    double lmax_L;     // upper bound on the top eigenvalue of the constant stencil operator L (spin lattices)
    moto_morse_params mp;
    moto_solver_opts opts;
    cudaStream_t stream;
    char* ws;
    size_t ws_bytes;
    size_t block_bytes;   // stride between the [kmax][N][3] blocks X, AX, W, AW, P, AP(, T1, T2)
    int nblocks;
    // workspace views
    double *X, *AX, *W, *AW, *P, *AP;  // [kmax][N][3] each
    double *T1, *T2, *T3, *T4;   // [kmax][N][3] rotating blocks of the Chebyshev recurrence (spin lattices; the one-step-per-pass
                                 // kernel ping-pongs between T1 and T2, the two-step kernel rotates through all four)
    unsigned long long* flags;   // [MOTO_NUM_SMS] per-CTA step flags of the multi-step K1 (zeroed at create)
    unsigned long long epoch;    // flag base of the latest multi-step launch
    int coop_max_ctas;           // co-resident CTAs of the multi-step K1 (cooperative launch limit)
    int coop2_max_ctas;          // the same for the two-steps-per-pass K1 (spin_cheb2_tma.cu)
    double* c;         // [N]   m_i . g_i
    double* g;         // [N][3] gradient scratch
    double* stage_m;   // [N][3] host-variant staging
    double* partials;  // [MOTO_RED_BLOCKS][2*NS*NS] grid-reduction partials
    SolverState* st;
    CartLists cl;
    double* fmmf_out;  // internal: when set, moto_mmf_step also writes the reflected force F_mmf [N][3] there (moto_mmf_run_cg)
    int keep_guard;    // internal: a warm start also carries the guard columns (moto_mmf_run's v_1-only re-solves)
    int nsh;           // > 0: general neighbour shells (moto_set_shells) replace the nearest-neighbour J, D of sp
    int* sh_off;       // [MOTO_MAX_SHELLS][2] device
    double* sh_jd;     // [MOTO_MAX_SHELLS][4] device: J, Dx, Dy, Dz
    // the same table as dense column segments for the register-blocked kernel (spin_shells_dense.cu); sh_nseg == 0: not available
    int sh_nseg, sh_nd;              // segments, dense entries (holes zero-filled)
    int sh_Hx, sh_Hy;                // halo: largest |dx|, |dy| of the table
    int sh_grp[3][MOTO_SH_GROUPS + 1];   // tap groups for S = 8, 12, 16 warps per staged field: group s owns segments [grp[s], grp[s + 1])
    int* sh_seg;       // [MOTO_SH_SEGS][4] device: dx, dy0, n, first entry
    double* sh_jd2;    // [MOTO_SH_DENSE][4] device
    HostStatus* hstat;  // pinned
    cudaEvent_t ev[2];
    int64_t launches;
    char err[256];
};

#define MOTO_CUDA_CHECK(ctx, call)                                                              \
    do {                                                                                        \
        cudaError_t e__ = (call);                                                               \
        if (e__ != cudaSuccess) {                                                               \
            snprintf((ctx)->err, sizeof((ctx)->err), "%s:%d %s: %s", __FILE__, __LINE__, #call, \
                     cudaGetErrorString(e__));                                                  \
            return MOTO_ECUDA;                                                                  \
        }                                                                                       \
    } while (0)

static inline moto_status moto_fail(moto_ctx* ctx, moto_status s, const char* msg) {
    if (ctx) snprintf(ctx->err, sizeof(ctx->err), "%s", msg);
    return s;
}

moto_status moto_check_overflow(moto_ctx* ctx);   // api.cu (also exported, include/moto.h)

// ---- launch wrappers (each returns the number of kernels it enqueued; errors via cudaGetLastError)
// spin_stencil.cu
int spin_energy_grad(moto_ctx*, const double* m, double* d_E, double* d_g, double* d_c);
int spin_energy_grad_tma(moto_ctx*, const double* m, double* d_E, double* d_g, double* d_c);   // 0: not applicable
int spin_mmf_pass1_tma(moto_ctx*, const double* m, const double* v, double* Fbuf, double* d_alpha);   // 0: not applicable
void launch_final_sum(moto_ctx* c, const double* partials, int nblk, int stride, int nval, double* out, int take_sqrt);
int spin_curvature(moto_ctx*, const double* m, double* d_c);
int spin_hvp(moto_ctx*, const double* m, const double* c_or_null, const double* V, int k, double* HV,
             int project_input, const int* d_done);
int spin_mmf_step(moto_ctx*, const double* m, const double* v, int kr, double dt, double* m_out, double* d_fnorm);
int spin_project(moto_ctx*, const double* m, double* V, int k);
int spin_relax_eval(moto_ctx*, const double* x, const double* d, double a, const double* g_old, double* xt, double* gt, double* d_out4);
int spin_relax_nblk(const moto_ctx*);
int spin_relax_eval_dev(moto_ctx*, const RelaxDev* rs, int* nblk_out);   // trial described by the device state; partials left in ctx->partials
int spin_hvp_three_term_generic(moto_ctx*, const double* m, const double* cvec, const double* V, int k, double alpha, double c0,
                                double beta, const double* U, double* out);
// spin_stencil_tma.cu
bool spin_tma_applicable(const moto_ctx*);
int spin_tma_grid(const moto_ctx*);
int spin_tma_coop_limit(int k);
int spin_cheb_multistep(moto_ctx*, const double* m, const double* cvec, const double* V, int k, int d, double* OUT,
                        const double* d_coef, const int* d_done);
// spin_cheb2_tma.cu
int spin_cheb2_multistep(moto_ctx*, const double* m, const double* cvec, const double* V, int k, int d, double* OUT,
                         const double* d_coef, const int* d_done, int product_form, int ngroups);
int spin_cheb_recurrence(moto_ctx*, const double* m, const double* cvec, const double* V, int k, int d, double* OUT,
                         const double* d_coef, const int* d_done);
int spin_hvp_tma_ex(moto_ctx*, const double* m, const double* cvec, const double* V, int k, double* HV, const int* d_done,
                    double* waw_partials, int cheb, double alpha, double c0, double beta, const double* U, const double* d_coef);
// spin_shells.cu
int shell_energy_grad(moto_ctx*, const double* m, double* d_E, double* d_g, double* d_c);
int shell_hvp(moto_ctx*, const double* m, const double* cvec, const double* V, int k, double* HV, int project_input, const int* d_done);
int shell_three_term(moto_ctx*, const double* m, const double* cvec, const double* V, int k, double alpha, double c0, double beta,
                     const double* U, double* out);
int shell_mmf_pass1(moto_ctx*, const double* m, const double* v, int kr);
moto_status shell_set(moto_ctx*, int n, const int32_t* h_off, const double* h_J, const double* h_D);
// spin_shells_dense.cu: register-blocked direct convolution (k <= 2); 0 launches = not applicable, the caller falls back
moto_status shell_dense_build(moto_ctx*, int n, const int32_t* h_off, const double* h_jd);
int shell_dense_hvp(moto_ctx*, const double* m, const double* cvec, const double* V, int k, double* HV, int project_input, const int* d_done,
                    int cheb, double alpha, double c0, double beta, const double* U, const double* d_coef);
bool shell_dense_applicable(const moto_ctx*, int k);
int shell_dense_energy_grad(moto_ctx*, const double* m, double* d_g, double* d_c, double* e_part, int* grid_out);
int shell_cheb_recurrence(moto_ctx*, const double* m, const double* cvec, const double* V, int k, int d, double* OUT, const double* d_coef,
                          const int* d_done);
// cart_morse.cu
int cart_build_lists(moto_ctx*, const double* x);
int cart_energy_grad(moto_ctx*, const double* x, double* d_E, double* d_g);
int cart_hvp(moto_ctx*, const double* V, int k, double* HV, const int* d_done);
int cart_cheb_recurrence(moto_ctx*, const double* V, int k, int d, double* OUT, const double* d_coef, const int* d_done);
int cart_rowbound(moto_ctx*, double* partial_max, int* nmax_out);
int cart_mmf_step(moto_ctx*, const double* x, const double* v, int kr, double dt, double* x_out, double* d_fnorm);
int cart_mask(moto_ctx*, double* V, int k);
size_t cart_lists_bytes(const moto_lattice* lat);
int cart_lists_carve(moto_ctx*, char* base);
// block_algebra.cu
int block_gram(moto_ctx*, const double* const* S, int ns, const double* const* T, int nt, double* d_G,
               const int* d_done);
int block_gram_lobpcg(moto_ctx*, int kb);
int block_update(moto_ctx*, int kb);
int block_residual(moto_ctx*, const double* m_or_null, int kb, int k, double tol);
int block_random(moto_ctx*, double* X, int kb, uint64_t seed);
int block_zero(moto_ctx*, double* X, long long n);
int gram_blocks(const moto_ctx*);
double* gram_reduced(const moto_ctx*);   // [G_B upper triangle | G_A upper triangle] left by block_gram_lobpcg
int rr_solve_lobpcg(moto_ctx*, int kb, int nblk);
bool cart_geometry_ok(const moto_lattice* lat, double rc);
int block_apply_coeffs(moto_ctx*, double* V, int k, const double* d_C, double* scratch);
int block_sign_normalise(moto_ctx*, double* V, int k);
// lobpcg_fast.cu
int fast_cheb_coef_explicit(moto_ctx* c, int d, double a, double b, double aL);
// rayleigh_ritz.cu
int rr_solve(moto_ctx*, const double* d_GA, const double* d_GB, int n, int nev, double* d_theta, double* d_C,
             int mode, SolverState* st_or_null);
// lanczos.cu
moto_status lanczos_solve(moto_ctx*, const double* d_state, int k, double tol, int max_iter, int warm_start,
                          moto_solve_info* info);
// relax.cu
moto_status relax_run(moto_ctx*, double* d_state, int max_steps, double tau_F, double alpha0, moto_relax_info* info);
moto_status mmf_cg_run(moto_ctx*, double* d_state, int k, double delta, double smax, int max_steps, double tau_F, double tol, int max_iter,
                       int warm_start, double* d_V, double* d_scratch, moto_mmf_info* info);
moto_status relax_lbfgs_run(moto_ctx*, double* d_state, int max_steps, double tau_F, double alpha0, int M, double* d_scratch, moto_relax_info* info);
moto_status mmf_lbfgs_run(moto_ctx*, double* d_state, int k, double alpha0, double smax, int max_steps, double tau_F, double tol, int max_iter,
                          int warm_start, int M, double* d_V, double* d_scratch, moto_mmf_info* info);
moto_status solve_first_column(moto_ctx*, const double* d_state, int kb, double tol, int max_iter, int warm, double* d_lambda, double* d_V,
                               moto_solve_info* info);   // api.cu
moto_status relax_seed(moto_ctx*, const double* d_saddle, const double* d_v, double s_eta, double* d_out);
// lobpcg_persistent.cu
bool persistent_applicable(const moto_ctx*, int k, int max_iter);
moto_status persistent_solve(moto_ctx* const* ctxs, int P, const double* const* d_spins, int k, double tol, int max_iter, int warm_start,
                             double* const* d_lambda, double* const* d_V, moto_solve_info* infos, int32_t* statuses);
// lobpcg.cu
moto_status lobpcg_solve(moto_ctx*, const double* d_state, int k, double tol, int max_iter, int warm_start,
                         moto_solve_info* info);

// ---- programmatic dependent launch for the small kernels of a solver iteration: a kernel that starts with MOTO_PDL_PROLOGUE() and is
// launched through launch_pdl becomes resident while its predecessor in the stream still runs and waits at griddepcontrol.wait until that
// one has completed and flushed -- stream order as before, minus the launch latency (~2 us per launch of a launch-bound iteration).
#ifdef __CUDACC__
#define MOTO_PDL_PROLOGUE()                                                 \
    do {                                                                    \
        asm volatile("griddepcontrol.launch_dependents;" ::: "memory");    \
        asm volatile("griddepcontrol.wait;" ::: "memory");                 \
    } while (0)
template <typename... KArgs, typename... Args>
static inline void launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    if (cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...) != cudaSuccess) {
        (void)cudaGetLastError();
        kern<<<grid, block, smem, st>>>(static_cast<KArgs>(args)...);
    }
}
#endif
