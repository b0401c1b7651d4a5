// block_algebra.cu -- K2 (tall-skinny Gram products), K3/K5 (block update, residual + projection),
// start-block generation and sign normalisation for the device-resident LOBPCG (
// Knyazev, ref [27] PAPER.md:221).  Generic path: any block size kb <= MOTO_KMAX, both lattice kinds.
// All reductions are two-stage with a fixed block count and fixed summation order (no float atomics),
// so reruns are bit-identical.
#include "common.cuh"
#include "device_utils.cuh"
#include "tma_utils.cuh"   // ensure_smem_attr

namespace {

struct PtrList { const double* p[3 * MOTO_NS]; };

constexpr int GRAM_CH = 64;       // flat elements staged per chunk
constexpr int GRAM_LD = GRAM_CH + 1;
constexpr int GRAM_THREADS = 256;
constexpr int GRAM_MAXE = (MOTO_NS * 2 * MOTO_NS + GRAM_THREADS - 1) / GRAM_THREADS;  // entries per thread

// partials[blk][i*nt + j] = sum over this CTA's chunks of S_i . T_j
__global__ void __launch_bounds__(GRAM_THREADS) k_gram(PtrList S, int ns, PtrList T, int nt, long long n3,
                                                       double* __restrict__ partials, const int* __restrict__ done) {
    if (done && *done) return;
    extern __shared__ double sm[];
    double* sS = sm;
    double* sT = sm + (size_t)ns * GRAM_LD;
    const int ne = ns * nt;
    double acc[GRAM_MAXE];
#pragma unroll
    for (int r = 0; r < GRAM_MAXE; ++r) acc[r] = 0.0;
    const long long nchunk = (n3 + GRAM_CH - 1) / GRAM_CH;
    for (long long ch = blockIdx.x; ch < nchunk; ch += gridDim.x) {
        const long long base = ch * GRAM_CH;
        for (int t = threadIdx.x; t < (ns + nt) * GRAM_CH; t += GRAM_THREADS) {
            int row = t / GRAM_CH, q = t - row * GRAM_CH;
            long long e = base + q;
            double val = 0.0;
            if (e < n3) val = (row < ns) ? S.p[row][e] : T.p[row - ns][e];
            if (row < ns) sS[row * GRAM_LD + q] = val; else sT[(row - ns) * GRAM_LD + q] = val;
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < GRAM_MAXE; ++r) {
            int e = threadIdx.x + r * GRAM_THREADS;
            if (e < ne) {
                int i = e / nt, j = e - i * nt;
                const double* a = sS + i * GRAM_LD;
                const double* b = sT + j * GRAM_LD;
                double s = 0.0;
#pragma unroll 8
                for (int q = 0; q < GRAM_CH; ++q) s = fma(a[q], b[q], s);
                acc[r] += s;
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < GRAM_MAXE; ++r) {
        int e = threadIdx.x + r * GRAM_THREADS;
        if (e < ne) partials[(size_t)blockIdx.x * ne + e] = acc[r];
    }
}

__global__ void k_gram_final(const double* __restrict__ partials, int nblk, int ne, double* __restrict__ G) {
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= ne) return;
    double s = 0.0;
    for (int b = 0; b < nblk; ++b) s += partials[(size_t)b * ne + e];
    G[e] = s;
}

// ---------------------------------------------------------------- K3 for the LOBPCG basis: symmetric, register-tiled
// Upper triangles of G_B = S^T S and G_A = S^T (A S) for S = [X,W,P] (n = 3 kb columns).  k_gram above spends two
// shared-memory loads per multiply-add and forms all n x 2n products; here a thread owns one 3 x 3 tile (I <= J) of
// both matrices for a slice of the staged chunk: nine loads feed eighteen multiply-adds, and only the nb (nb + 1) / 2
// upper tiles exist.  Threads = tiles x slices; slices are summed in a fixed order at the end.
// Output per CTA: [G_B upper triangle (nT) | G_A upper triangle (nT)], entry (a <= b) at a n - a (a - 1) / 2 + (b - a).
struct GramPtrs { const double* s[MOTO_NS]; const double* as[MOTO_NS]; };
constexpr int GS_THREADS = 256;
constexpr int GS_QPER = 4;        // flat elements per slice per staged chunk
constexpr int GS_LMAX = 10;       // staged values per thread per chunk: 2 n Q / 256 <= 9.4 for every kb <= 8

__global__ void __launch_bounds__(GS_THREADS) k_gram_sym(GramPtrs P, int n, int nslice, long long n3,
                                                         double* __restrict__ partials, const int* __restrict__ done) {
    MOTO_PDL_PROLOGUE();
    if (done && *done) return;
    extern __shared__ double sm[];
    const int nb = n / 3, ntile = nb * (nb + 1) / 2, NR = 2 * n + 1, Q = nslice * GS_QPER;
    const int t = threadIdx.x;
    const int tile = t % ntile, slice = t / ntile;
    const bool act = slice < nslice;
    int I = 0, rem = tile;
    while (rem >= nb - I) { rem -= nb - I; ++I; }
    const int J = I + rem;
    double gb[9], ga[9];
#pragma unroll
    for (int x = 0; x < 9; ++x) { gb[x] = 0.0; ga[x] = 0.0; }
    const long long nchunk = (n3 + Q - 1) / Q;
    const int tot = 2 * n * Q;                 // staged values per chunk (<= GS_LMAX per thread)
    // chunk ch + gridDim.x is fetched into registers (all loads in flight at once) while chunk ch is multiplied
    // per-thread staging slots (chunk-invariant): source pointer at q = 0 of the chunk, flat offset q, smem offset
    double v[GS_LMAX];
    const double* gp[GS_LMAX];
    int qo[GS_LMAX];       // (q << 16) | smem offset; -1: no slot
#pragma unroll
    for (int u = 0; u < GS_LMAX; ++u) {
        const int idx = t + u * GS_THREADS;
        qo[u] = -1; gp[u] = nullptr;
        if (idx < tot) {
            const int row = idx / Q, q = idx - row * Q;
            gp[u] = ((row < n) ? P.s[row] : P.as[row - n]) + q;
            qo[u] = (q << 16) | (q * NR + row);
        }
    }
    auto fetch = [&](long long ch) {
        const long long base = ch * Q;
        const bool full = base + Q <= n3;
#pragma unroll
        for (int u = 0; u < GS_LMAX; ++u) {
            v[u] = 0.0;
            if (qo[u] >= 0 && (full || base + (qo[u] >> 16) < n3)) v[u] = gp[u][base];
        }
    };
    if (blockIdx.x < nchunk) fetch(blockIdx.x);
    for (long long ch = blockIdx.x; ch < nchunk; ch += gridDim.x) {
#pragma unroll
        for (int u = 0; u < GS_LMAX; ++u)
            if (qo[u] >= 0) sm[qo[u] & 0xffff] = v[u];
        __syncthreads();
        if (ch + gridDim.x < nchunk) fetch(ch + gridDim.x);
        if (act) {
#pragma unroll
            for (int u = 0; u < GS_QPER; ++u) {
                const double* r = sm + (slice + u * nslice) * NR;
                double si[3], sj[3], aj[3];
#pragma unroll
                for (int a = 0; a < 3; ++a) { si[a] = r[3 * I + a]; sj[a] = r[3 * J + a]; aj[a] = r[n + 3 * J + a]; }
#pragma unroll
                for (int a = 0; a < 3; ++a)
#pragma unroll
                    for (int b = 0; b < 3; ++b) { gb[a * 3 + b] = fma(si[a], sj[b], gb[a * 3 + b]); ga[a * 3 + b] = fma(si[a], aj[b], ga[a * 3 + b]); }
            }
        }
        __syncthreads();
    }
    // slices -> one partial per CTA, fixed order
    double* red = sm;    // [GS_THREADS][18]
#pragma unroll
    for (int x = 0; x < 9; ++x) { red[t * 18 + x] = act ? gb[x] : 0.0; red[t * 18 + 9 + x] = act ? ga[x] : 0.0; }
    __syncthreads();
    const int nT = n * (n + 1) / 2;
    for (int o = t; o < ntile * 18; o += GS_THREADS) {
        const int tl = o / 18, x = o - tl * 18, which = x / 9, ab = x - which * 9, a = ab / 3, b = ab - a * 3;
        int I2 = 0, rem2 = tl;
        while (rem2 >= nb - I2) { rem2 -= nb - I2; ++I2; }
        const int i = 3 * I2 + a, j = 3 * (I2 + rem2) + b;
        if (i > j) continue;    // lower half of a diagonal tile
        double sum = 0.0;
        for (int sl = 0; sl < nslice; ++sl) sum += red[(sl * ntile + tl) * 18 + x];
        partials[(size_t)blockIdx.x * (2 * nT) + which * nT + i * n - i * (i - 1) / 2 + (j - i)] = sum;
    }
}

// out[e] = sum_b partials[b][e]: one warp per entry, lanes stride over the CTAs, fixed shuffle tree
__global__ void __launch_bounds__(256) k_reduce_partials(const double* __restrict__ partials, int nblk, int ne, double* __restrict__ out,
                                                         const int* __restrict__ done) {
    MOTO_PDL_PROLOGUE();
    if (done && *done) return;
    const int e = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (e >= ne) return;
    double s = 0.0;
    for (int b = lane; b < nblk; b += 32) s += partials[(size_t)b * ne + e];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) out[e] = s;
}

// ---------------------------------------------------------------- K5 block update, element-wise, in place
//   X' = [X,W,P] C ; P' = [W,P] C_{W,P rows} ; same coefficients on AX, AW, AP (PAPER.md ref [27])
template <int KB>
__global__ void __launch_bounds__(256) k_update(long long n3, double* __restrict__ X, double* __restrict__ W,
                                                double* __restrict__ P, double* __restrict__ AX, double* __restrict__ AW,
                                                double* __restrict__ AP, const SolverState* __restrict__ st) {
    MOTO_PDL_PROLOGUE();
    if (st->done) return;
    __shared__ double sC[3 * KB * KB];
    for (int t = threadIdx.x; t < 3 * KB * KB; t += blockDim.x) sC[t] = st->C[t];  // [3KB][KB] row-major
    bool lk[KB];          // soft locking: P_j of a locked column is dropped
#pragma unroll
    for (int j = 0; j < KB; ++j) lk[j] = st->lock_on && st->locked[j];
    __syncthreads();
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n3; e += (long long)gridDim.x * blockDim.x) {
#pragma unroll
        for (int pass = 0; pass < 2; ++pass) {
            double* x = pass ? AX : X; double* w = pass ? AW : W; double* p = pass ? AP : P;
            double s[3 * KB];
#pragma unroll
            for (int i = 0; i < KB; ++i) {
                s[i] = x[(size_t)i * n3 + e];
                s[KB + i] = w[(size_t)i * n3 + e];
                s[2 * KB + i] = p[(size_t)i * n3 + e];
            }
#pragma unroll
            for (int j = 0; j < KB; ++j) {
                double pn = 0.0;
#pragma unroll
                for (int i = KB; i < 3 * KB; ++i) pn = fma(sC[i * KB + j], s[i], pn);
                double xn = pn;
#pragma unroll
                for (int i = 0; i < KB; ++i) xn = fma(sC[i * KB + j], s[i], xn);
                x[(size_t)j * n3 + e] = xn;
                p[(size_t)j * n3 + e] = lk[j] ? 0.0 : pn;
            }
        }
    }
}

// ---------------------------------------------------------------- residual  W = Proj(AX - X theta), |r_j|^2 partials
__global__ void __launch_bounds__(256) k_residual(long long N, int kb, const double* __restrict__ m,
                                                  const uint8_t* __restrict__ fixed, const double* __restrict__ X,
                                                  const double* __restrict__ AX, double* __restrict__ W,
                                                  const SolverState* __restrict__ st, double* __restrict__ partials) {
    MOTO_PDL_PROLOGUE();
    if (st->done) return;
    __shared__ double red[32 * MOTO_KMAX];
    double acc[MOTO_KMAX];
    double th[MOTO_KMAX];
#pragma unroll
    for (int a = 0; a < MOTO_KMAX; ++a) { acc[a] = 0.0; th[a] = (a < kb) ? st->theta[a] : 0.0; }
    bool lk[MOTO_KMAX];   // soft locking: a locked column contributes no search direction
#pragma unroll
    for (int a = 0; a < MOTO_KMAX; ++a) lk[a] = st->lock_on && a < kb && st->locked[a];
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        d3 mi = m ? ld3(m, i) : mk3(0, 0, 0);
        const bool fx = fixed && fixed[i];
#pragma unroll
        for (int a = 0; a < MOTO_KMAX; ++a) {
            if (a < kb) {
                d3 r = axpy3(-th[a], ld3(X + (size_t)a * 3 * N, i), ld3(AX + (size_t)a * 3 * N, i));
                acc[a] += dot3(r, r);
                if (m) r = proj3(mi, r);
                if (fx || lk[a]) r = mk3(0, 0, 0);
                st3(W + (size_t)a * 3 * N, i, r);
            }
        }
    }
    block_sum<MOTO_KMAX>(acc, red);
    if (threadIdx.x == 0)
        for (int a = 0; a < MOTO_KMAX; ++a) partials[blockIdx.x * MOTO_KMAX + a] = acc[a];
}

// single thread block: finish the residual norms, convergence decision, iteration counter
__global__ void k_check(const double* __restrict__ partials, int nblk, int kb, int k, double tol, SolverState* st) {
    MOTO_PDL_PROLOGUE();
    if (st->done) return;
    __shared__ double r[MOTO_KMAX];
    const int j = threadIdx.x >> 5, lane = threadIdx.x & 31;   // one warp per column, lanes over CTAs, fixed order
    if (j < kb) {
        double s = 0.0;
        for (int b = lane; b < nblk; b += 32) s += partials[b * MOTO_KMAX + j];
        s = warp_sum(s);
        if (lane == 0) {   // tol < 0: residuals of the transformed operator, never reported
            r[j] = sqrt(s);
            if (tol >= 0.0) { st->resid[j] = r[j]; if (st->lock_on) st->locked[j] = r[j] <= 0.1 * tol; }
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        bool ok = true, bad = false;
        for (int a = 0; a < k; ++a) { ok = ok && (r[a] <= tol); bad = bad || !(r[a] == r[a]); }
        if (bad) { st->bad = 1; st->done = 1; }
        else if (ok) st->done = 1;
        else st->iter += 1;
    }
}

// ---------------------------------------------------------------- start block: counter-based uniform(-1/2,1/2)
__device__ __forceinline__ uint64_t splitmix64(uint64_t x) {
    x += 0x9E3779B97F4A7C15ull;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    return x ^ (x >> 31);
}
__global__ void k_random(long long n, double* __restrict__ X, uint64_t seed) {
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
        uint64_t h = splitmix64(seed ^ splitmix64((uint64_t)e));
        X[e] = (double)(h >> 11) * (1.0 / 9007199254740992.0) - 0.5;
    }
}

__global__ void k_zero(long long n, double* __restrict__ X) {
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) X[e] = 0.0;
}

// V <- V C  (k x k, row-major C[i][j]: new column j = sum_i C[i][j] V_i), element-wise in place
__global__ void k_apply_coeffs(long long n3, int k, double* __restrict__ V, const double* __restrict__ C) {
    __shared__ double sC[MOTO_KMAX * MOTO_KMAX];
    for (int t = threadIdx.x; t < k * k; t += blockDim.x) sC[t] = C[t];
    __syncthreads();
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n3; e += (long long)gridDim.x * blockDim.x) {
        double s[MOTO_KMAX], o[MOTO_KMAX];
#pragma unroll
        for (int i = 0; i < MOTO_KMAX; ++i) s[i] = (i < k) ? V[(size_t)i * n3 + e] : 0.0;
#pragma unroll
        for (int j = 0; j < MOTO_KMAX; ++j) {
            o[j] = 0.0;
#pragma unroll
            for (int i = 0; i < MOTO_KMAX; ++i)
                if (i < k && j < k) o[j] = fma(sC[i * k + j], s[i], o[j]);
        }
#pragma unroll
        for (int j = 0; j < MOTO_KMAX; ++j)
            if (j < k) V[(size_t)j * n3 + e] = o[j];
    }
}

// ---------------------------------------------------------------- sign normalisation (largest |component| positive)
__global__ void __launch_bounds__(256) k_absmax_partial(long long n3, int k, const double* __restrict__ V,
                                                        double* __restrict__ pval, long long* __restrict__ pidx) {
    __shared__ double sv[256];
    __shared__ long long si[256];
    for (int a = 0; a < k; ++a) {
        const double* v = V + (size_t)a * n3;
        double best = -1.0; long long bi = -1;
        for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n3; e += (long long)gridDim.x * blockDim.x) {
            double x = fabs(v[e]);
            if (x > best) { best = x; bi = e; }
        }
        sv[threadIdx.x] = best; si[threadIdx.x] = bi;
        __syncthreads();
        for (int s = 128; s > 0; s >>= 1) {
            if (threadIdx.x < s) {
                double o = sv[threadIdx.x + s]; long long oi = si[threadIdx.x + s];
                if (o > sv[threadIdx.x] || (o == sv[threadIdx.x] && oi >= 0 && (si[threadIdx.x] < 0 || oi < si[threadIdx.x]))) {
                    sv[threadIdx.x] = o; si[threadIdx.x] = oi;
                }
            }
            __syncthreads();
        }
        if (threadIdx.x == 0) { pval[blockIdx.x * MOTO_KMAX + a] = sv[0]; pidx[blockIdx.x * MOTO_KMAX + a] = si[0]; }
        __syncthreads();
    }
}
__global__ void k_absmax_final(int nblk, int k, const double* __restrict__ V, long long n3, const double* __restrict__ pval,
                               const long long* __restrict__ pidx, double* __restrict__ sign) {
    int a = threadIdx.x;
    if (a >= k) return;
    double best = -1.0; long long bi = -1;
    for (int b = 0; b < nblk; ++b) {
        double o = pval[b * MOTO_KMAX + a]; long long oi = pidx[b * MOTO_KMAX + a];
        if (oi >= 0 && (o > best || (o == best && oi < bi))) { best = o; bi = oi; }
    }
    sign[a] = (bi >= 0 && V[(size_t)a * n3 + bi] < 0.0) ? -1.0 : 1.0;
}
__global__ void k_scale_cols(long long n3, int k, double* __restrict__ V, const double* __restrict__ sign) {
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n3; e += (long long)gridDim.x * blockDim.x)
        for (int a = 0; a < k; ++a)
            if (sign[a] < 0.0) V[(size_t)a * n3 + e] = -V[(size_t)a * n3 + e];
}

int grid_for(long long n, int threads) {
    long long b = (n + threads - 1) / threads;
    long long cap = MOTO_NUM_SMS * 8;
    return (int)(b < 1 ? 1 : (b > cap ? cap : b));
}

}  // namespace

// ================================================================ host wrappers
int block_gram(moto_ctx* c, const double* const* S, int ns, const double* const* T, int nt, double* d_G, const int* d_done) {
    PtrList ps, pt;
    for (int i = 0; i < ns; ++i) ps.p[i] = S[i];
    for (int j = 0; j < nt; ++j) pt.p[j] = T[j];
    const long long n3 = 3ll * c->N;
    const long long nchunk = (n3 + GRAM_CH - 1) / GRAM_CH;
    int blocks = (int)(nchunk < MOTO_RED_BLOCKS ? nchunk : MOTO_RED_BLOCKS);
    size_t smem = (size_t)(ns + nt) * GRAM_LD * sizeof(double);
    static std::atomic<unsigned long long> attr_seen{0};   // per device, safe against the host threads of the batch call
    if (!tma::ensure_smem_attr(k_gram, (size_t)3 * MOTO_NS * GRAM_LD * 8, attr_seen)) return 0;
    k_gram<<<blocks, GRAM_THREADS, smem, c->stream>>>(ps, ns, pt, nt, n3, c->partials, d_done);
    if (d_G) {
        k_gram_final<<<(ns * nt + 127) / 128, 128, 0, c->stream>>>(c->partials, blocks, ns * nt, d_G);
        return 2;
    }
    return 1;
}

// Gram of the LOBPCG basis S = [X,W,P] (n = 3 kb): upper triangles of S^T S and S^T (A S), summed over the CTAs into
// gram_reduced(c) = [G_B tri | G_A tri] for rr_solve_lobpcg.
double* gram_reduced(const moto_ctx* c) { return c->partials + (size_t)(MOTO_RED_BLOCKS - 1) * 2 * MOTO_NS * MOTO_NS; }

int block_gram_lobpcg(moto_ctx* c, int kb) {
    const size_t bs = (size_t)3 * c->N;
    GramPtrs P;
    for (int j = 0; j < kb; ++j) {
        P.s[j] = c->X + j * bs; P.s[kb + j] = c->W + j * bs; P.s[2 * kb + j] = c->P + j * bs;
        P.as[j] = c->AX + j * bs; P.as[kb + j] = c->AW + j * bs; P.as[2 * kb + j] = c->AP + j * bs;
    }
    const int n = 3 * kb, ntile = kb * (kb + 1) / 2, nT = n * (n + 1) / 2;
    int nslice = GS_THREADS / ntile;
    if (nslice > 32) nslice = 32;
    const long long n3 = 3ll * c->N;
    const int Q = nslice * GS_QPER;
    const long long nchunk = (n3 + Q - 1) / Q;
    const int blocks = (int)(nchunk < MOTO_RED_BLOCKS ? nchunk : MOTO_RED_BLOCKS);
    size_t smem = (size_t)Q * (2 * n + 1) * sizeof(double), smem_red = (size_t)GS_THREADS * 18 * sizeof(double);
    if (smem < smem_red) smem = smem_red;
    launch_pdl(k_gram_sym, dim3(blocks), dim3(GS_THREADS), smem, c->stream, P, n, nslice, n3, c->partials, &c->st->done);
    launch_pdl(k_reduce_partials, dim3((2 * nT * 32 + 255) / 256), dim3(256), 0, c->stream, c->partials, blocks, 2 * nT, gram_reduced(c), &c->st->done);
    return 2;
}

int gram_blocks(const moto_ctx* c) {
    const long long n3 = 3ll * c->N;
    const long long nchunk = (n3 + GRAM_CH - 1) / GRAM_CH;
    return (int)(nchunk < MOTO_RED_BLOCKS ? nchunk : MOTO_RED_BLOCKS);
}

int block_update(moto_ctx* c, int kb) {
    const long long n3 = 3ll * c->N;
    int g = grid_for(n3, 256);
#define UPD(KB) case KB: launch_pdl(k_update<KB>, dim3(g), dim3(256), 0, c->stream, n3, c->X, c->W, c->P, c->AX, c->AW, c->AP, c->st); break;
    switch (kb) { UPD(1) UPD(2) UPD(3) UPD(4) UPD(5) UPD(6) UPD(7) UPD(8) }
#undef UPD
    return 1;
}

int block_residual(moto_ctx* c, const double* m_or_null, int kb, int k, double tol) {
    launch_pdl(k_residual, dim3(MOTO_RED_BLOCKS), dim3(256), 0, c->stream, (long long)c->N, kb, m_or_null, c->kind == MOTO_KIND_CARTESIAN ? c->lat.d_fixed : nullptr,
                                                       c->X, c->AX, c->W, c->st, c->partials);
    launch_pdl(k_check, dim3(1), dim3(32 * kb), 0, c->stream, c->partials, MOTO_RED_BLOCKS, kb, k, tol, c->st);
    return 2;
}

int block_random(moto_ctx* c, double* X, int kb, uint64_t seed) {
    const long long n = 3ll * c->N * kb;
    k_random<<<grid_for(n, 256), 256, 0, c->stream>>>(n, X, seed);
    return 1;
}

int block_zero(moto_ctx* c, double* X, long long n) {
    k_zero<<<grid_for(n, 256), 256, 0, c->stream>>>(n, X);
    return 1;
}

int block_apply_coeffs(moto_ctx* c, double* V, int k, const double* d_C, double*) {
    const long long n3 = 3ll * c->N;
    k_apply_coeffs<<<grid_for(n3, 256), 256, 0, c->stream>>>(n3, k, V, d_C);
    return 1;
}

int block_sign_normalise(moto_ctx* c, double* V, int k) {
    const long long n3 = 3ll * c->N;
    double* pval = c->partials;
    long long* pidx = (long long*)(c->partials + MOTO_RED_BLOCKS * MOTO_KMAX);
    double* sign = c->st->scal;
    int blocks = (int)((n3 + 255) / 256 < MOTO_RED_BLOCKS ? (n3 + 255) / 256 : MOTO_RED_BLOCKS);
    k_absmax_partial<<<blocks, 256, 0, c->stream>>>(n3, k, V, pval, pidx);
    k_absmax_final<<<1, 32, 0, c->stream>>>(blocks, k, V, n3, pval, pidx, sign);
    k_scale_cols<<<grid_for(n3, 256), 256, 0, c->stream>>>(n3, k, V, sign);
    return 3;
}
