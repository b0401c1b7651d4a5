// rayleigh_ritz.cu -- K4: single-CTA generalized symmetric eigen-solve  G_A c = theta G_B c  for the
// LOBPCG basis [X,W,P] (n = 3 kb <= 24), kept on the GPU (BASELINE.json north_star (3); the paper does
// this host-side inside CuPy).
//
// Numerics: G_B is scaled to unit diagonal, diagonalised by cyclic Jacobi (parallel round-robin
// ordering), directions with eigenvalue <= tau * max are dropped (canonical orthogonalisation: this is
// what makes the un-orthogonalised basis [X,W,P] safe, incl. P = 0 on the first iteration), the
// reduced standard problem M^T G_A M is diagonalised by the same Jacobi routine, eigenvalues sorted.
#include "common.cuh"

namespace {

constexpr int NMAX = MOTO_NS;       // 24
constexpr int LD = NMAX + 1;        // smem leading dimension
constexpr int RR_THREADS = 256;     // gather phase; the dense phase runs on warp 0 alone (warp-level syncs only)
// dense phase: one warp (warp-level syncs) for n <= 8, the whole CTA for larger pencils (more rotations per round)
#define RR_SYNC() do { if (wide) __syncthreads(); else __syncwarp(); } while (0)

struct JacobiScratch { int p[NMAX / 2], q[NMAX / 2]; double c[NMAX / 2], s[NMAX / 2]; double off, diag; };

// Symmetric eigen-decomposition in shared memory: A (n x n, LD) -> diag(A) = eigenvalues, V = eigenvectors (cols).
__device__ void jacobi_eig(double* A, double* V, int n, JacobiScratch* js, bool wide) {
    const int tid = threadIdx.x, nt = wide ? blockDim.x : 32;
    for (int t = tid; t < n * n; t += nt) { int i = t / n, j = t - i * n; V[i * LD + j] = (i == j) ? 1.0 : 0.0; }
    RR_SYNC();
    if (n == 1) return;
    const int np = (n + 1) & ~1, half = np / 2;
    for (int sweep = 0; sweep < 30; ++sweep) {
        double off = 0.0, dg = 0.0;
        if (tid < 32) {   // warp 0 sums (n*n <= 576 entries), everyone reads the verdict
            for (int t = tid; t < n * n; t += 32) {
                int i = t / n, j = t - i * n;
                double a = A[i * LD + j];
                if (i == j) dg += a * a; else if (j > i) off += a * a;
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) { off += __shfl_xor_sync(0xffffffffu, off, o); dg += __shfl_xor_sync(0xffffffffu, dg, o); }
            if (tid == 0) { js->off = off; js->diag = dg; }
        }
        RR_SYNC();
        off = js->off; dg = js->diag;
        RR_SYNC();
        if (off <= 1e-30 * dg || off == 0.0) break;   // off-diagonals below 1e-15 of the diagonal scale: rounding level   // off-diagonals below 1e-15 of the diagonal scale: rounding level
        for (int r = 0; r < np - 1; ++r) {
            if (tid < half) {
                int p, q;
                if (tid == 0) { p = np - 1; q = r; }
                else { p = (r + tid) % (np - 1); q = (r - tid + (np - 1)) % (np - 1); }
                if (p > q) { int t = p; p = q; q = t; }
                double c = 1.0, s = 0.0;
                if (q < n) {
                    double apq = A[p * LD + q];
                    if (apq != 0.0) {
                        double app = A[p * LD + p], aqq = A[q * LD + q];
                        double tau = (aqq - app) / (2.0 * apq);
                        double t = (tau >= 0.0 ? 1.0 : -1.0) / (fabs(tau) + sqrt(1.0 + tau * tau));
                        c = 1.0 / sqrt(1.0 + t * t);
                        s = t * c;
                    }
                } else { p = -1; }
                js->p[tid] = p; js->q[tid] = q; js->c[tid] = c; js->s[tid] = s;
            }
            RR_SYNC();
            // columns: A <- A J, V <- V J
            for (int w = tid; w < half * n; w += nt) {
                int t = w / n, i = w - t * n, p = js->p[t], q = js->q[t];
                if (p < 0) continue;
                double c = js->c[t], s = js->s[t];
                double aip = A[i * LD + p], aiq = A[i * LD + q];
                A[i * LD + p] = c * aip - s * aiq; A[i * LD + q] = s * aip + c * aiq;
                double vip = V[i * LD + p], viq = V[i * LD + q];
                V[i * LD + p] = c * vip - s * viq; V[i * LD + q] = s * vip + c * viq;
            }
            RR_SYNC();
            // rows: A <- J^T A
            for (int w = tid; w < half * n; w += nt) {
                int t = w / n, j = w - t * n, p = js->p[t], q = js->q[t];
                if (p < 0) continue;
                double c = js->c[t], s = js->s[t];
                double apj = A[p * LD + j], aqj = A[q * LD + j];
                A[p * LD + j] = c * apj - s * aqj; A[q * LD + j] = s * apj + c * aqj;
            }
            RR_SYNC();
            if (tid < half && js->p[tid] >= 0) { int p = js->p[tid], q = js->q[tid]; A[p * LD + q] = 0.0; A[q * LD + p] = 0.0; }
            RR_SYNC();
        }
    }
    RR_SYNC();
}

// vals[e] = sum_b partials[b * stride + e] in a fixed order with every load independent (the serial version of
// this loop was latency-bound on ~300 dependent L2 reads).  Thread (g, e) sums the CTAs b = g, g+G, ... with four
// interleaved accumulators; the G group sums are then added in order.  scratch: >= G * ne doubles of smem.
__device__ void reduce_partials(const double* __restrict__ partials, int nblk, int stride, int ne, double* vals, double* scratch) {
    const int tid = threadIdx.x, nt = blockDim.x;
    const int G = (ne <= 64) ? nt / 64 : 1, ne_g = (G > 1) ? 64 : ne;
    for (int idx = tid; idx < ne_g * G; idx += nt) {
        const int g = idx / ne_g, e = idx - g * ne_g;
        if (e >= ne) continue;
        double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
        int b = g;
        for (; b + 3 * G < nblk; b += 4 * G) {
            a0 += partials[(size_t)b * stride + e];
            a1 += partials[(size_t)(b + G) * stride + e];
            a2 += partials[(size_t)(b + 2 * G) * stride + e];
            a3 += partials[(size_t)(b + 3 * G) * stride + e];
        }
        for (; b < nblk; b += G) a0 += partials[(size_t)b * stride + e];
        const double sum = (a0 + a1) + (a2 + a3);
        if (G > 1) scratch[g * ne + e] = sum; else vals[e] = sum;
    }
    if (G > 1) {
        __syncthreads();
        for (int e = tid; e < ne; e += nt) {
            double sum = 0.0;
            for (int g = 0; g < G; ++g) sum += scratch[g * ne + e];
            vals[e] = sum;
        }
    }
}

struct RRFast {            // inputs of the fused kb <= 2 path (lobpcg_fast.cu); kb == 0: not used
    const double* partialsK;   // [nblkK][kb(kb+1)/2]  W^T A W from K1 (NULL: already inside the tri partials)
    int nblkK;
    int kb;
    int check;             // 1: finish the residual norms of the last update and decide convergence first; 2: only that;
                           // 3: count the iteration without testing (transformed operator: its residuals are not A's)
    int hvp_inc;           // single-vector HVPs the caller spent since the previous Rayleigh-Ritz
    int k;                 // wanted columns
    double tol;
};

// mode 0: Rayleigh-Ritz (theta[nev], C[n][nev]);  mode 1: Loewdin orthonormalisation from G_B only (C[n][n])
__global__ void __launch_bounds__(RR_THREADS) k_rr(const double* __restrict__ partials, int nblk, const double* __restrict__ GA_in,
                                                   const double* __restrict__ GB_in, int n, int nev, double* __restrict__ theta_out,
                                                   double* __restrict__ C_out, int mode, SolverState* st, double tau, RRFast fz) {
    if (st && st->done) return;
    __shared__ double A[NMAX * LD], B[NMAX * LD], U[NMAX * LD], M[NMAX * LD], T[NMAX * LD], Z[NMAX * LD];
    __shared__ double vals[NMAX * 2 * NMAX];
    __shared__ double d[NMAX], sig[NMAX], th[NMAX];
    __shared__ int keep[NMAX], ord[NMAX], na_s, bad_s, stop_s;
    __shared__ JacobiScratch js;
    const int tid = threadIdx.x;
    int nt = blockDim.x;

    // 1. gather G_A, G_B (from grid-reduction partials, fixed order, or from given matrices); symmetrise
    if (partials && fz.kb > 0) {
        // upper triangles [G_B | G_A | |r_j|^2] from k_update_fused / k_gram_tri, W^T A W from K1
        const int kb = fz.kb, nT = n * (n + 1) / 2, nK = kb * (kb + 1) / 2, neu = 2 * nT + kb;
        reduce_partials(partials, nblk, neu, neu, vals, Z);
        if (fz.partialsK) { __syncthreads(); reduce_partials(fz.partialsK, fz.nblkK, nK, nK, vals + neu, Z); }
        if (tid == 0) stop_s = 0;
        __syncthreads();
        if (fz.check == 3 && tid == 0) st->iter += 1;
        if ((fz.check == 1 || fz.check == 2) && tid == 0) {
            bool ok = true, bad = false;
            for (int a = 0; a < kb; ++a) {
                double r = sqrt(vals[2 * nT + a]);
                st->resid[a] = r;
                if (a < fz.k) { ok = ok && (r <= fz.tol); bad = bad || !(r == r); }
            }
            if (bad) { st->bad = 1; st->done = 1; stop_s = 1; }
            else if (ok) { st->done = 1; stop_s = 1; }
            else if (fz.check == 1) st->iter += 1;
        }
        __syncthreads();
        if (stop_s || fz.check == 2) return;
        if (tid == 0) st->nhvp += fz.hvp_inc;
        for (int t = tid; t < n * n; t += nt) {
            int i = t / n, j = t - i * n;
            int a = i < j ? i : j, b = i < j ? j : i;
            int e = a * n - a * (a - 1) / 2 + (b - a);
            double ga = vals[nT + e];
            if (fz.partialsK && a >= kb && b < 2 * kb) {   // (W_a', W_b') block
                int wa = a - kb, wb = b - kb;
                ga = vals[neu + wa * kb - wa * (wa - 1) / 2 + (wb - wa)];
            }
            U[i * LD + j] = vals[e];
            T[i * LD + j] = ga;
        }
    } else if (partials) {
        const int ntc = 2 * n, ne = n * ntc;
        reduce_partials(partials, nblk, ne, ne, vals, Z);
        __syncthreads();
        for (int t = tid; t < 2 * n * n; t += nt) {
            int which = t / (n * n), e = t - which * n * n, i = e / n, j = e - i * n;
            double s = vals[i * ntc + which * n + j];
            if (which) T[i * LD + j] = s; else U[i * LD + j] = s;  // U <- raw G_B, T <- raw G_A
        }
    } else {
        for (int t = tid; t < n * n; t += nt) {
            int i = t / n, j = t - i * n;
            U[i * LD + j] = GB_in[t];
            T[i * LD + j] = GA_in ? GA_in[t] : 0.0;
        }
    }
    __syncthreads();
    for (int t = tid; t < n * n; t += nt) {
        int i = t / n, j = t - i * n;
        B[i * LD + j] = 0.5 * (U[i * LD + j] + U[j * LD + i]);
        A[i * LD + j] = 0.5 * (T[i * LD + j] + T[j * LD + i]);
    }
    __syncthreads();
    // ---- dense phase: warp 0 alone for small pencils (warp-level synchronisation only), the whole CTA otherwise
    const bool wide = n > 8;
    if (!wide) { if (tid >= 32) return; nt = 32; }
    if (st && partials) {  // keep a copy for diagnostics
        for (int t = tid; t < n * n; t += nt) { int i = t / n, j = t - i * n; st->GA[t] = A[i * LD + j]; st->GB[t] = B[i * LD + j]; }
    }
    // 2. scale to unit diagonal; non-positive / NaN diagonal => inactive column
    if (tid < n) {
        double bii = B[tid * LD + tid];
        d[tid] = (bii > 1e-300) ? rsqrt(bii) : 0.0;
    }
    if (tid == 0) bad_s = 0;
    RR_SYNC();
    for (int t = tid; t < n * n; t += nt) { int i = t / n, j = t - i * n; B[i * LD + j] *= d[i] * d[j]; }
    RR_SYNC();
    // 3. eigen-decomposition of the scaled G_B
    jacobi_eig(B, U, n, &js, wide);
    if (tid == 0) {
        double smax = 0.0;
        for (int j = 0; j < n; ++j) { sig[j] = B[j * LD + j]; if (sig[j] > smax) smax = sig[j]; }
        int na = 0;
        for (int j = 0; j < n; ++j) if (sig[j] > tau * smax && sig[j] > 0.0) keep[na++] = j;
        na_s = na;
        if (!(smax == smax)) bad_s = 1;
    }
    RR_SYNC();
    const int na = na_s;
    // M = D U_keep Sigma^{-1/2}   (n x na)
    for (int t = tid; t < n * na; t += nt) {
        int i = t / na, l = t - i * na, j = keep[l];
        M[i * LD + l] = d[i] * U[i * LD + j] * rsqrt(sig[j]);
    }
    RR_SYNC();
    if (mode == 1) {
        // Loewdin: C = M (U_keep)^T D^{-1}... applied to the ORIGINAL vectors: C = D U S^{-1/2} U^T  (n x n)
        for (int t = tid; t < n * n; t += nt) {
            int i = t / n, j = t - i * n;
            double s = 0.0;
            for (int l = 0; l < na; ++l) s += M[i * LD + l] * U[j * LD + keep[l]];
            C_out[i * n + j] = s;
        }
        if (st && tid == 0) { st->nkeep = na; if (na < n || bad_s) st->bad = 1; }
        return;
    }
    // 4. reduced standard problem  At = M^T A M
    for (int t = tid; t < n * na; t += nt) {
        int i = t / na, l = t - i * na;
        double s = 0.0;
        for (int j = 0; j < n; ++j) s += A[i * LD + j] * M[j * LD + l];
        T[i * LD + l] = s;
    }
    RR_SYNC();
    for (int t = tid; t < na * na; t += nt) {
        int a = t / na, b = t - a * na;
        double s = 0.0;
        for (int i = 0; i < n; ++i) s += M[i * LD + a] * T[i * LD + b];
        B[a * LD + b] = s;
    }
    RR_SYNC();
    for (int t = tid; t < na * na; t += nt) { int a = t / na, b = t - a * na; A[a * LD + b] = 0.5 * (B[a * LD + b] + B[b * LD + a]); }
    RR_SYNC();
    jacobi_eig(A, Z, na, &js, wide);
    // 5. sort ascending
    if (tid == 0) {
        for (int j = 0; j < na; ++j) { th[j] = A[j * LD + j]; ord[j] = j; }
        for (int a = 0; a < na; ++a) {
            int best = a;
            for (int b = a + 1; b < na; ++b) if (th[ord[b]] < th[ord[best]]) best = b;
            int t = ord[a]; ord[a] = ord[best]; ord[best] = t;
        }
        if (na < nev) bad_s = 1;
        for (int a = 0; a < nev && a < na; ++a) if (!(th[ord[a]] == th[ord[a]])) bad_s = 1;
    }
    RR_SYNC();
    // 6. C = M Z[:, lowest nev]
    for (int t = tid; t < n * nev; t += nt) {
        int i = t / nev, j = t - i * nev;
        double s = 0.0;
        if (j < na) { int zj = ord[j]; for (int l = 0; l < na; ++l) s += M[i * LD + l] * Z[l * LD + zj]; }
        C_out[i * nev + j] = s;
    }
    if (tid < nev) theta_out[tid] = (tid < na) ? th[ord[tid]] : 0.0;
    if (st && tid == 0) { st->nkeep = na; if (bad_s) { st->bad = 1; st->done = 1; } }
}

}  // namespace

int rr_solve(moto_ctx* c, const double* d_GA, const double* d_GB, int n, int nev, double* d_theta, double* d_C, int mode,
             SolverState* st) {
    const double tau = 1e-10;
    RRFast fz = {nullptr, 0, 0, 0, 0, 0, 0.0};
    k_rr<<<1, RR_THREADS, 0, c->stream>>>(nullptr, 0, d_GA, d_GB, n, nev, d_theta, d_C, mode, st, tau, fz);
    return 1;
}

// LOBPCG flavour: inputs are the Gram partials left in ctx->partials by block_gram_lobpcg
int rr_solve_lobpcg(moto_ctx* c, int kb, int nblk) {
    const double tau = 1e-10;
    RRFast fz = {nullptr, 0, 0, 0, 0, 0, 0.0};
    k_rr<<<1, RR_THREADS, 0, c->stream>>>(c->partials, nblk, nullptr, nullptr, 3 * kb, kb, c->st->theta, c->st->C, 0, c->st, tau, fz);
    return 1;
}

// fused kb <= 2 path: tri partials [nblkU][2 nT + kb] in ctx->partials, optional W^T A W partials, optional check
int rr_solve_fast(moto_ctx* c, int kb, int nblkU, const double* partialsK, int nblkK, int check, int k, double tol, int hvp_inc) {
    const double tau = 1e-10;
    RRFast fz = {partialsK, nblkK, kb, check, hvp_inc, k, tol};
    k_rr<<<1, RR_THREADS, 0, c->stream>>>(c->partials, nblkU, nullptr, nullptr, 3 * kb, kb, c->st->theta, c->st->C, 0, c->st, tau, fz);
    return 1;
}
