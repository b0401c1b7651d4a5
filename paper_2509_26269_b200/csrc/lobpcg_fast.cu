// lobpcg_fast.cu -- fused block-vector algebra of the device-resident LOBPCG for block sizes kb <= 2
// (the headline case: two lowest modes; Knyazev ref [27] PAPER.md:221).
//
// One iteration is TWO streaming kernels and one single-CTA kernel:
//   K1            AW = Hess[W]                       (+ per-CTA partials of W^T AW)
//   k_rr          reduce partials -> residual check -> Rayleigh-Ritz on the 3kb x 3kb pencil
//   k_update_fused  one pass over [X,W,P,AX,AW,AP]:  X' = S C, P' = [W,P] C_wp, AX', AP' by the same
//                 coefficients, W' = R = AX' - X' Theta, partials of |r_j|^2 AND of every Gram entry the
//                 next Rayleigh-Ritz needs except W'^T A W' (which needs the next HVP)
// so no separate Gram pass exists: per iteration the block vectors are read once and written once.
// W' is re-projected onto the tangent space inside the same pass (see k_update_fused); masked (fixed-atom)
// rows stay exactly zero because every block is a combination of masked vectors.
//
// Reductions are two-stage with
// a fixed CTA count and fixed order (bit-reproducible, no float atomics).
#include "common.cuh"
#include "device_utils.cuh"
#include "lobpcg_blocks.cuh"

namespace {

using namespace lob;   // Tri, Blk6, gram_accum, block_reduce_store, update_site (lobpcg_blocks.cuh)

// ---------------------------------------------------------------- full Gram of the six blocks (start-up only)
template <int KB>
__global__ void __launch_bounds__(256) k_gram_tri(long long n3, Blk6 b, double* __restrict__ partials, const int* __restrict__ done) {
    if (*done) return;
    using T = Tri<KB>;
    double acc[T::NEU];
#pragma unroll
    for (int i = 0; i < T::NEU; ++i) acc[i] = 0.0;
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n3; e += (long long)gridDim.x * blockDim.x) {
        double s[T::NS], a[T::NS];
#pragma unroll
        for (int i = 0; i < KB; ++i) {
            s[i] = b.X[i * n3 + e]; s[KB + i] = b.W[i * n3 + e]; s[2 * KB + i] = b.P[i * n3 + e];
            a[i] = b.AX[i * n3 + e]; a[KB + i] = b.AW[i * n3 + e]; a[2 * KB + i] = b.AP[i * n3 + e];
        }
        gram_accum<KB, false>(s, a, acc);
    }
    block_reduce_store<T::NEU>(acc, partials + (size_t)blockIdx.x * T::NEU);
}

// ---------------------------------------------------------------- W^T A W partials (generic-K1 path; the TMA K1 fuses this)
template <int KB>
__global__ void __launch_bounds__(256) k_dot_waw(long long n3, const double* __restrict__ W, const double* __restrict__ AW,
                                                 double* __restrict__ partials, const int* __restrict__ done) {
    MOTO_PDL_PROLOGUE();
    if (*done) return;
    constexpr int NK = Tri<KB>::NK;
    double acc[NK];
#pragma unroll
    for (int i = 0; i < NK; ++i) acc[i] = 0.0;
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n3; e += (long long)gridDim.x * blockDim.x) {
        double w[KB], a[KB];
#pragma unroll
        for (int i = 0; i < KB; ++i) { w[i] = W[i * n3 + e]; a[i] = AW[i * n3 + e]; }
        int t = 0;
#pragma unroll
        for (int i = 0; i < KB; ++i)
#pragma unroll
            for (int j = i; j < KB; ++j) { acc[t] = fma(w[i], a[j], acc[t]); ++t; }
    }
    block_reduce_store<NK>(acc, partials + (size_t)blockIdx.x * NK);
}

// ---------------------------------------------------------------- fused update + residual + next Gram
// C: [3KB][KB] row-major (rows: X, W, P), theta[KB].  In place on all six blocks.  One thread per site
// (the three components of a site stay together because W' = P_m R needs m_i . r_i).
//
// Why W' must be projected every iteration: a radial component rho of X is mapped by the solver-mode
// operator to -c_i rho (c_i ~ -12 J), so R carries -(c_i + theta) rho and X'' = C_x X' + C_w W' would
// multiply rho by (1 + 12 C_w) per iteration -- exponential growth from 1e-16 (seen as a residual that
// stalls at 1e-9 and then creeps up).  With rad(W') = 0 the radial part of X can only shrink.
//
// Gram entries that pair W' with a tangent vector (X', P', AX', AP') use R in place of W' = P_m R
// (t . P_m r = t . r for tangent t); only W'^T W' needs the correction  r_i.r_j - (m.r_i)(m.r_j).
template <int KB, bool PROJECT>
__global__ void __launch_bounds__(256) k_update_fused(long long N, Blk6 b, const double* __restrict__ m,
                                                      const SolverState* __restrict__ st, double* __restrict__ partials) {
    MOTO_PDL_PROLOGUE();
    if (st->done) return;
    using T = Tri<KB>;
    __shared__ double sC[3 * KB * KB + KB];
    for (int t = threadIdx.x; t < 3 * KB * KB + KB; t += blockDim.x) sC[t] = t < 3 * KB * KB ? st->C[t] : st->theta[t - 3 * KB * KB];
    bool lk[KB];   // soft locking (transformed solves): see lobpcg_solve_fast
#pragma unroll
    for (int j = 0; j < KB; ++j) lk[j] = st->lock_on && st->locked[j];
    __syncthreads();
    double acc[T::NEU];
#pragma unroll
    for (int i = 0; i < T::NEU; ++i) acc[i] = 0.0;
    const long long n3 = 3 * N;
    for (long long site = blockIdx.x * (long long)blockDim.x + threadIdx.x; site < N; site += (long long)gridDim.x * blockDim.x)
        update_site<KB, PROJECT>(b, m, sC, 3 * site, n3, acc, lk);
    block_reduce_store<T::NEU>(acc, partials + (size_t)blockIdx.x * T::NEU);
}

// ---------------------------------------------------------------- Chebyshev spectral transformation (coefficients)
// p(lambda) = scaled Chebyshev polynomial of degree d that is <= 1 in magnitude on [a, b] and grows below a
// (Zhou & Saad's scaled three-term form, p(a_L) = 1).  LOBPCG is run on -p(A): same eigenvectors, lowest
// eigenvalues of A <-> lowest of -p(A), relative gaps d^2 times wider as long as d^2 (a - lambda) <~ (b - a)/4.
// a = theta_k + margin from the current A-Ritz values (theta_k >= lambda_k, so the wanted pairs stay below a),
// b = max_i(-c_i) + ||L||  >= lambda_max (Gershgorin-type bound), a_L = theta_1.  All on the device.
__global__ void k_negc_max(long long N, const double* __restrict__ c, double* __restrict__ partial_max) {
    __shared__ double sm[8];
    double v = -1e300;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) v = fmax(v, -c[i]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) v = fmax(v, sm[w]);
        partial_max[blockIdx.x] = v;
    }
}

// The filter p_d(x) = T_d(l(x)) / T_d(l(a_L)), l(x) = (2x - a - b)/(b - a), is applied in PRODUCT form over its roots
//   p_d(A) = prod_s (A - r_s) / (a_L - r_s),   r_s = c0 + e cos((2 j_s - 1) pi / (2 d)),  c0 = (a + b)/2, e = (b - a)/2
// (same polynomial: same roots, same value 1 at a_L), i.e. as d TWO-term steps  Y_s = alpha_s (A - r_s) Y_{s-1}  with
// alpha_s = 1 / (a_L - r_s): a step reads m, c, Y_{s-1} and writes Y_s -- 128 B/site at k = 2 -- where the three-term Chebyshev
// recurrence also reads Y_{s-2} (176 B/site).  The product form is only stable if the roots are taken in a LEJA order (each
// next root maximises the product of its distances to the ones already used): prefix and suffix products then stay within
// ~3e2 of the end result, and the rounding error equals the three-term recurrence's (3e-14 relative at d = 40 and 128 on a
// spectrum [-0.16, 18]; the natural orders lose every digit from d = 40 on).  The order depends on d only and is kept in the
// solver state.  The coefficient rows stay {alpha, shift, beta = 0, -}: every kernel that runs the recurrence reads them
// as a three-term step and skips the Y_{s-2} operand when beta == 0.
//
// explicit == 1: interval given (a = margin, b = hi_user, a_L = lnorm): the moto_cheb_apply building block
__global__ void k_cheb_coef(SolverState* st, int k, int d, double margin, double lnorm, double hi_user,
                            const double* __restrict__ partial_max, int nmax, int explicit_ab) {
    if (st->done) return;
    const int lane = threadIdx.x;   // one warp
    __shared__ unsigned char order[MOTO_CHEB_MAX];
    if (st->leja_d != d) {
        // Leja order of the d normalised roots x_j = cos((2j - 1) pi / (2d)): lane l owns candidates l, l + 32, ...; products of
        // distances as sums of logs (fp32 is enough to rank them; ties go to the lower index, so the order is deterministic)
        float lp[MOTO_CHEB_MAX / 32];
        bool used[MOTO_CHEB_MAX / 32];
#pragma unroll
        for (int q = 0; q < MOTO_CHEB_MAX / 32; ++q) { lp[q] = 0.0f; used[q] = false; }
        int pick = 0;                                  // x_1: the root nearest b
        for (int s = 0; s < d; ++s) {
            if (lane == 0) order[s] = (unsigned char)pick;
            const double xp = cospi((2.0 * pick + 1.0) / (2.0 * d));
            float best = -3.0e38f; int bj = 1 << 20;
#pragma unroll
            for (int q = 0; q < MOTO_CHEB_MAX / 32; ++q) {
                const int j = lane + 32 * q;
                if (j == pick) used[q] = true;
                if (j < d && !used[q]) {
                    lp[q] += __logf((float)fabs(cospi((2.0 * j + 1.0) / (2.0 * d)) - xp));
                    if (lp[q] > best) { best = lp[q]; bj = j; }
                }
            }
            for (int o = 16; o > 0; o >>= 1) {
                const float ob = __shfl_xor_sync(0xffffffffu, best, o);
                const int oj = __shfl_xor_sync(0xffffffffu, bj, o);
                if (ob > best || (ob == best && oj < bj)) { best = ob; bj = oj; }
            }
            pick = bj;
        }
        __syncwarp();
        for (int s = lane; s < d; s += 32) st->leja[s] = order[s];
        __syncwarp();
        if (lane == 0) st->leja_d = d;
    } else {
        for (int s = lane; s < d; s += 32) order[s] = st->leja[s];
    }
    __syncwarp();
    double b = hi_user;
    if (!explicit_ab && !(b > 0.0)) {
        double mx = -1e300;
        for (int i = 0; i < nmax; ++i) mx = fmax(mx, partial_max[i]);
        b = mx + lnorm;
    }
    const double aL = explicit_ab ? lnorm : st->theta[0];
    double a = explicit_ab ? margin : st->theta[k - 1] + margin;
    if (!explicit_ab && a > 0.5 * (aL + b)) a = 0.5 * (aL + b);   // crude early Ritz values: keep the interval sane
    const double e = 0.5 * (b - a), c0 = 0.5 * (b + a);
    if (lane == 0) { st->cheb_ab[0] = a; st->cheb_ab[1] = b; st->cheb_ab[2] = aL; st->cheb_ab[3] = (double)d; }
    for (int s = lane; s < d; s += 32) {
        const double r = c0 + e * cospi((2.0 * order[s] + 1.0) / (2.0 * d));
        double alpha = 1.0 / (aL - r);
        if (s == d - 1) alpha = -alpha;                            // the transformed operator is -p(A)
        st->cheb[s][0] = alpha; st->cheb[s][1] = r; st->cheb[s][2] = 0.0; st->cheb[s][3] = 0.0;
    }
}

// ---------------------------------------------------------------- A-residual check while LOBPCG runs on -p(A)
// T = A X is given.  Two streaming passes, because the residual must not be formed from the expanded expression
// tt - 2 theta xt + theta^2 xx: with tt ~ 1e-2 its rounding floor is ~ 1e-8 in |r|, so below tol ~ 1e-8 that test would
// decide on noise.  Pass 1: partials of x_j.x_j and x_j.t_j  ->  theta_j = xt / xx (k_acheck_theta, into st->ack).
// Pass 2: partials of |t_j - theta_j x_j|^2, formed element by element  ->  |A x_j - theta_j x_j| / |x_j|, decision.
template <int KB>
__global__ void __launch_bounds__(256) k_acheck_dots(long long n3, const double* __restrict__ X, const double* __restrict__ T,
                                                     double* __restrict__ partials, const int* __restrict__ done) {
    MOTO_PDL_PROLOGUE();
    if (*done) return;
    double acc[2 * KB];
#pragma unroll
    for (int i = 0; i < 2 * KB; ++i) acc[i] = 0.0;
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n3; e += (long long)gridDim.x * blockDim.x) {
#pragma unroll
        for (int j = 0; j < KB; ++j) {
            const double x = X[j * n3 + e], t = T[j * n3 + e];
            acc[2 * j] = fma(x, x, acc[2 * j]); acc[2 * j + 1] = fma(x, t, acc[2 * j + 1]);
        }
    }
    block_reduce_store<2 * KB>(acc, partials + (size_t)blockIdx.x * 2 * KB);
}

// theta_j = (x_j.t_j) / (x_j.x_j) into st->ack[j], x_j.x_j into st->ack[KMAX + j]
__global__ void k_acheck_theta(const double* __restrict__ partials, int nblk, int kb, SolverState* st) {
    MOTO_PDL_PROLOGUE();
    if (st->done) return;
    __shared__ double v[2 * MOTO_KMAX];
    const int e = threadIdx.x >> 5, lane = threadIdx.x & 31;   // one warp per entry
    if (e < 2 * kb) {
        double s = 0.0;
        for (int b = lane; b < nblk; b += 32) s += partials[(size_t)b * 2 * kb + e];
        s = warp_sum(s);
        if (lane == 0) v[e] = s;
    }
    __syncthreads();
    if (threadIdx.x < kb) { st->ack[threadIdx.x] = v[2 * threadIdx.x + 1] / v[2 * threadIdx.x]; st->ack[MOTO_KMAX + threadIdx.x] = v[2 * threadIdx.x]; }
}

template <int KB>
__global__ void __launch_bounds__(256) k_acheck_resid(long long n3, const double* __restrict__ X, const double* __restrict__ T,
                                                      const SolverState* __restrict__ st, double* __restrict__ partials) {
    MOTO_PDL_PROLOGUE();
    if (st->done) return;
    double th[KB], acc[KB];
#pragma unroll
    for (int j = 0; j < KB; ++j) { th[j] = st->ack[j]; acc[j] = 0.0; }
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n3; e += (long long)gridDim.x * blockDim.x) {
#pragma unroll
        for (int j = 0; j < KB; ++j) {
            const double r = fma(-th[j], X[j * n3 + e], T[j * n3 + e]);
            acc[j] = fma(r, r, acc[j]);
        }
    }
    block_reduce_store<KB>(acc, partials + (size_t)blockIdx.x * KB);
}

// store: also leave theta / resid in the state when the test fails (the Lanczos variant sets its next interval from them)
__global__ void k_acheck_final(const double* __restrict__ partials, int nblk, int kb, int k, double tol, SolverState* st, int store) {
    MOTO_PDL_PROLOGUE();
    // (soft locking, st->lock_on: every column whose A-residual is within tol is locked, and unlocked should it drift out again)
    if (st->done) return;
    __shared__ double v[MOTO_KMAX];
    const int e = threadIdx.x >> 5, lane = threadIdx.x & 31;   // one warp per column
    if (e < kb) {
        double s = 0.0;
        for (int b = lane; b < nblk; b += 32) s += partials[(size_t)b * kb + e];
        s = warp_sum(s);
        if (lane == 0) v[e] = s;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        bool ok = true;
        double rs[MOTO_KMAX];
        for (int j = 0; j < kb; ++j) {
            const double r2 = v[j] / st->ack[MOTO_KMAX + j];
            rs[j] = sqrt(r2);
            if (j < k) ok = ok && (rs[j] <= tol) && (r2 == r2);
            if (st->lock_on) st->locked[j] = rs[j] <= 0.1 * tol;
        }
        st->nhvp += kb;
        if (ok || store)
            for (int j = 0; j < kb; ++j) { st->theta[j] = st->ack[j]; st->resid[j] = rs[j]; }
        if (ok) st->done = 1;
    }
}

int fast_grid(long long work_items) {
    long long b = (work_items + 255) / 256;
    return (int)(b < 1 ? 1 : (b > MOTO_RED_BLOCKS ? MOTO_RED_BLOCKS : b));
}

Blk6 blocks_of(moto_ctx* c) { Blk6 b; b.X = c->X; b.W = c->W; b.P = c->P; b.AX = c->AX; b.AW = c->AW; b.AP = c->AP; return b; }

}  // namespace

// ================================================================ host side
int fast_gram_full(moto_ctx* c, int kb, int* nblk_out) {
    const long long n3 = 3ll * c->N;
    const int g = fast_grid(n3);
    *nblk_out = g;
    if (kb == 1) k_gram_tri<1><<<g, 256, 0, c->stream>>>(n3, blocks_of(c), c->partials, &c->st->done);
    else k_gram_tri<2><<<g, 256, 0, c->stream>>>(n3, blocks_of(c), c->partials, &c->st->done);
    return 1;
}

int fast_dot_waw(moto_ctx* c, int kb, const double* W, const double* AW, double* partialsK, int* nblk_out) {
    const long long n3 = 3ll * c->N;
    const int g = fast_grid(n3);
    *nblk_out = g;
    if (kb == 1) launch_pdl(k_dot_waw<1>, dim3(g), dim3(256), 0, c->stream, n3, W, AW, partialsK, &c->st->done);
    else launch_pdl(k_dot_waw<2>, dim3(g), dim3(256), 0, c->stream, n3, W, AW, partialsK, &c->st->done);
    return 1;
}

int fast_update(moto_ctx* c, const double* m_or_null, int kb, int* nblk_out) {
    const long long N = c->N;
    const int g = fast_grid(N);
    *nblk_out = g;
    Blk6 b = blocks_of(c);
    if (kb == 1) {
        if (m_or_null) launch_pdl(k_update_fused<1, true>, dim3(g), dim3(256), 0, c->stream, N, b, m_or_null, c->st, c->partials);
        else launch_pdl(k_update_fused<1, false>, dim3(g), dim3(256), 0, c->stream, N, b, m_or_null, c->st, c->partials);
    } else {
        if (m_or_null) launch_pdl(k_update_fused<2, true>, dim3(g), dim3(256), 0, c->stream, N, b, m_or_null, c->st, c->partials);
        else launch_pdl(k_update_fused<2, false>, dim3(g), dim3(256), 0, c->stream, N, b, m_or_null, c->st, c->partials);
    }
    return 1;
}

int fast_negc_max(moto_ctx* c, double* partial_max, int* nmax_out) {
    const int g = fast_grid(c->N);
    *nmax_out = g;
    k_negc_max<<<g, 256, 0, c->stream>>>((long long)c->N, c->c, partial_max);
    return 1;
}

int fast_cheb_coef(moto_ctx* c, int k, int d, double margin, double lnorm, double hi_user, const double* partial_max, int nmax) {
    k_cheb_coef<<<1, 32, 0, c->stream>>>(c->st, k, d, margin, lnorm, hi_user, partial_max, nmax, 0);
    return 1;
}

int fast_cheb_coef_explicit(moto_ctx* c, int d, double a, double b, double aL) {
    k_cheb_coef<<<1, 32, 0, c->stream>>>(c->st, 1, d, a, aL, b, nullptr, 0, 1);
    return 1;
}

// T = A X must already be in d_T.  Sets done (and theta, resid) when every wanted A-residual is below tol.
int fast_acheck(moto_ctx* c, int kb, int k, double tol, const double* d_T, double* partials, int store) {
    const long long n3 = 3ll * c->N;
    const int g = fast_grid(n3);
#define ACK_DOTS(KB) launch_pdl(k_acheck_dots<KB>, dim3(g), dim3(256), 0, c->stream, n3, c->X, d_T, partials, &c->st->done)
#define ACK_RESID(KB) launch_pdl(k_acheck_resid<KB>, dim3(g), dim3(256), 0, c->stream, n3, c->X, d_T, c->st, partials)
#define ACK_SWITCH(M) switch (kb) { case 1: M(1); break; case 2: M(2); break; case 3: M(3); break; case 4: M(4); break; \
                                    case 5: M(5); break; case 6: M(6); break; case 7: M(7); break; default: M(8); break; }
    ACK_SWITCH(ACK_DOTS);
    launch_pdl(k_acheck_theta, dim3(1), dim3(32 * 2 * kb), 0, c->stream, partials, g, kb, c->st);
    ACK_SWITCH(ACK_RESID);
#undef ACK_SWITCH
#undef ACK_RESID
#undef ACK_DOTS
    launch_pdl(k_acheck_final, dim3(1), dim3(32 * kb), 0, c->stream, partials, g, kb, k, tol, c->st, store);
    return 4;
}
