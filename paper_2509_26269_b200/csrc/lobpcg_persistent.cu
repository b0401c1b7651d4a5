// lobpcg_persistent.cu -- the small-lattice regime of the inner solve and the population solve of the explorer as ONE
// persistent cooperative kernel (Alg. 1 l.3-5 "(lambda_1, lambda_2) <- HVPOptimization(x)" once per
// candidate, P = 24 per generation; BASELINE.json north_star (3) "no host round-trip per iteration").
//
// On a 70x70 lattice a block vector is 118 KB: the multi-launch LOBPCG of lobpcg.cu spends its 46 us per iteration on launch
// latency and on a 37 us single-CTA Rayleigh-Ritz, and a population of such solves cannot fill the GPU one launch chain at a
// time.  Here the whole block LOBPCG (block size kb <= 2, same algebra as lobpcg_fast.cu) of P independent problems runs
// inside one launch, for every lattice up to 148 x 256 = 37 888 sites (one 256-site chunk per CTA of a full grid):
//   grid = P x cpp CTAs, problem index = blockIdx.x / cpp; a problem's cpp CTAs own its 256-site chunks round-robin;
//   an iteration is  [H: AW = op(W), W^T (op W) partials]  barrier  [R: reduce partials, residual test, Rayleigh-Ritz]
//                    [U: fused update of the six blocks + Gram partials]  barrier
//   with a barrier among the cpp CTAs of ONE problem only (a counter in that problem's solver state) -- problems never wait
//   for each other and finish at their own iteration counts;
//   R is done redundantly by every CTA of the problem from the same partials in the same order (no broadcast step), by one
//   warp: Cholesky whitening of the unit-diagonal Gram matrix (rank-revealing Jacobi when a pivot is small) and a
//   round-robin parallel Jacobi on the reduced 3kb x 3kb pencil; nothing leaves the GPU until the kernel ends.
// op is the Hessian or, from N >= 128 sites on, the Chebyshev transformation -p_d(A) of lobpcg.cu (d = 16 steps of its product
// form per application, each one pass over the CTA's chunks + the problem barrier): the Rayleigh-Ritz (~35 us, the dominant cost
// of a plain iteration here) is then paid once per 16 Hessian applications, and the clustered spectra that stall the plain
// operator (cfg 3 at 100 x 100: 2155 plain iterations) converge in ~50.  8 plain iterations (cold start) fix the interval,
// phases of 20 transformed iterations follow, each closed by a restart on A that yields the A-Ritz pairs and true
// A-residuals (the only convergence test while transformed, together with a cheap |A x - theta x| test every 2 iterations).
// Partial sums are formed per 256-site chunk and combined in chunk order, so the result does not depend on cpp or P: a
// problem solved alone (moto_lowest_modes) and inside a batch (moto_lowest_modes_batch) give bit-identical results.
#include "common.cuh"
#include "device_utils.cuh"
#include "lobpcg_blocks.cuh"
#include "stencil_math.cuh"

namespace {

using namespace lob;

constexpr int PT = 256;        // threads per CTA = sites per chunk
constexpr int PMAXP = 24;      // problems per launch (they travel as kernel parameters)
constexpr int NM = 6;          // largest pencil (3 kb, kb <= 2)
constexpr int PDEG = 32;       // largest degree of the Chebyshev transformation inside the kernel
// precond_degree = 0 (auto): degree, smallest lattice that takes it, plain iterations of a cold start, phase length, iterations
// between cheap A-residual tests -- swept on cfg 1, its 40x40 instance, random spins 64x64, cfg 3 at 100x100 and the P = 24 batch
constexpr int PAUTO_DEGREE = 16, PAUTO_MIN_N = 128, PAUTO_PLAIN = 8, PAUTO_PHASE = 20, PAUTO_ACHECK = 2;
constexpr double RR_TAU = 1e-10, RR_CHOL = 1e-2;   // rank truncation / Cholesky admission, as on the fused path of rayleigh_ritz.cu

struct PProb {
    const double* m;            // [N][3] configuration
    double* V;                  // [k][N][3] in (warm start) / out
    double* lambda;             // [k] out
    Blk6 b;                     // the six solver blocks of this problem's workspace
    double* c;                  // [N]
    double *T1, *T2;            // [kb][N][3] each: intermediate steps of the Chebyshev recurrence
    double* part;               // chunk partials
    SolverState* st;
};
struct PBatch { PProb p[PMAXP]; };
struct PParams {
    Lat l;
    int N, nchunk, cpp, k, max_iter, warm;
    double tol;
    unsigned long long seed;
    // Chebyshev transformation -p_d(A) (same construction as lobpcg.cu / k_cheb_coef): degree 0 = plain operator throughout
    int degree, plain_start, phase_len, acheck_every;
    double margin, lnorm, hi_user;
    HostStatus* out;            // [P] device: what the host reads back (one copy for the whole batch)
};

__device__ __forceinline__ uint64_t splitmix64(uint64_t x) {
    x += 0x9E3779B97F4A7C15ull;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    return x ^ (x >> 31);
}

// neighbour site index or -1 (open boundary)
__device__ __forceinline__ int nbi(const Lat& l, int ix, int iy, int dx, int dy) {
    int jx = ix + dx, jy = iy + dy;
    if (jx < 0) { if (!l.px) return -1; jx += l.Lx; }
    if (jx >= l.Lx) { if (!l.px) return -1; jx -= l.Lx; }
    if (jy < 0) { if (!l.py) return -1; jy += l.Ly; }
    if (jy >= l.Ly) { if (!l.py) return -1; jy -= l.Ly; }
    return jy * l.Lx + jx;
}
// values written by other CTAs since the last barrier: read through L2
__device__ __forceinline__ d3 ldn_cg(const double* u, int j) {
    return j >= 0 ? mk3(__ldcg(u + 3 * j), __ldcg(u + 3 * j + 1), __ldcg(u + 3 * j + 2)) : mk3(0.0, 0.0, 0.0);
}
__device__ __forceinline__ d3 stencil_at(const Lat& l, const double* u, const int (&nb)[6], double uz) {
    return stencil_apply(l, ldn_cg(u, nb[0]), ldn_cg(u, nb[1]), ldn_cg(u, nb[2]), ldn_cg(u, nb[3]), ldn_cg(u, nb[4]), ldn_cg(u, nb[5]), uz);
}

// barrier among the cpp CTAs of one problem: monotone counter, release / acquire at gpu scope (bounded spin)
__device__ __forceinline__ void prob_barrier(unsigned long long* bar, int cpp, unsigned long long& round, int* err) {
    __syncthreads();
    ++round;
    if (cpp > 1 && threadIdx.x == 0) {
        __threadfence();
        atomicAdd(bar, 1ull);
        const unsigned long long want = round * (unsigned long long)cpp;
        unsigned long long v; int spins = 0;
        do {
            asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(bar) : "memory");
        } while (v < want && ++spins < (1 << 26));
        if (v < want) *err = 1;
    }
    __syncthreads();
}

// ---------------------------------------------------------------- dense 3kb x 3kb work, one warp, matrices in shared memory
struct RRs {
    double A[NM * NM], B[NM * NM], U[NM * NM], M[NM * NM], T[NM * NM], Z[NM * NM];
    double d[NM], sig[NM], cs[NM], sn[NM];
    int keep[NM], ord[NM], partner[NM], na, bad, chol;
    double off;
};

// eigen-decomposition of the symmetric n x n matrix A (n <= 6) by round-robin parallel Jacobi: A -> diagonal, V = eigenvectors
// (columns).  All 32 lanes of one warp call it; T is scratch.
__device__ void warp_jacobi(double* A, double* V, double* T, double* cs, double* sn, int* partner, int n, int lane) {
    // lane owns the matrix entries e = lane and lane + 32 of the NM x NM array (row e / NM, column e % NM: constant divisors)
    const int e0 = lane, e1 = lane + 32;
    const int i0 = e0 / NM, j0 = e0 % NM, i1 = e1 / NM, j1 = e1 % NM;
    const bool in0 = i0 < n && j0 < n, in1 = e1 < NM * NM && i1 < n && j1 < n;
    V[e0] = (i0 == j0) ? 1.0 : 0.0;
    if (e1 < NM * NM) V[e1] = (i1 == j1) ? 1.0 : 0.0;
    __syncwarp();
    const int np = (n + 1) & ~1;
    for (int sweep = 0; sweep < 10 && np >= 2; ++sweep) {
        double off = 0.0, dg = 0.0;
        if (in0) { const double v = A[e0] * A[e0]; if (i0 == j0) dg += v; else off += v; }
        if (in1) { const double v = A[e1] * A[e1]; if (i1 == j1) dg += v; else off += v; }
        off = warp_sum(off); dg = warp_sum(dg);
        if (!(off > 1e-30 * dg)) break;
        // off-diagonal part at rounding level of the diagonal (or NaN: the caller flags it)
        for (int r = 0; r < np - 1; ++r) {
            // pairs of round r: (np - 1, r) and ((r + i) mod (np - 1), (r - i) mod (np - 1)), i = 1 .. np/2 - 1
            if (lane < np / 2) {
                int p, q;
                if (lane == 0) { p = np - 1; q = r; }
                else { p = (r + lane) % (np - 1); q = (r - lane + (np - 1)) % (np - 1); }
                if (p > q) { const int t = p; p = q; q = t; }
                if (q < n) {
                    const double apq = A[p * NM + q], dd = A[q * NM + q] - A[p * NM + p];
                    double c = 1.0, s = 0.0;
                    if (fabs(apq) > 1e-300) {
                        // tan of the rotation angle: the smaller root of t^2 + (dd / apq) t - 1 = 0, cancellation-free form
                        const double t = (dd >= 0.0 ? 2.0 : -2.0) * apq / (fabs(dd) + sqrt(fma(dd, dd, 4.0 * apq * apq)));
                        c = rsqrt(fma(t, t, 1.0)); s = t * c;
                    }
                    // column p of J: (c at p, -s at q); column q: (s at p, c at q)
                    cs[p] = c; sn[p] = -s; partner[p] = q;
                    cs[q] = c; sn[q] = s; partner[q] = p;
                } else if (p < n) { cs[p] = 1.0; sn[p] = 0.0; partner[p] = p; }
            }
            __syncwarp();
            // T = J^T A : T(i, l) = cs_i A(i, l) + sn_i A(partner_i, l)
            if (in0) T[e0] = cs[i0] * A[e0] + sn[i0] * A[partner[i0] * NM + j0];
            if (in1) T[e1] = cs[i1] * A[e1] + sn[i1] * A[partner[i1] * NM + j1];
            __syncwarp();
            // A = T J : A(i, j) = T(i, j) cs_j + T(i, partner_j) sn_j ;  V = V J likewise
            double v0 = 0.0, v1 = 0.0;
            if (in0) { A[e0] = T[e0] * cs[j0] + T[i0 * NM + partner[j0]] * sn[j0]; v0 = V[e0] * cs[j0] + V[i0 * NM + partner[j0]] * sn[j0]; }
            if (in1) { A[e1] = T[e1] * cs[j1] + T[i1 * NM + partner[j1]] * sn[j1]; v1 = V[e1] * cs[j1] + V[i1 * NM + partner[j1]] * sn[j1]; }
            __syncwarp();
            if (in0) V[e0] = v0;
            if (in1) V[e1] = v1;
            __syncwarp();
        }
    }
    __syncwarp();
}

// Rayleigh-Ritz on the pencil (A, B) of size n (both symmetric, in s.A / s.B): lowest nev pairs -> theta[nev], C[n][nev]
// (row-major, C^T B C = I).  Directions of B below RR_TAU of its largest eigenvalue are dropped.  One warp.
__device__ void warp_rr(RRs& s, int n, int nev, double* theta, double* C, int lane) {
    // unit-diagonal scaling
    if (lane < n) { const double bii = s.B[lane * NM + lane]; s.d[lane] = bii > 1e-300 ? rsqrt(bii) : 0.0; }
    if (lane == 0) { s.bad = 0; s.chol = 1; }
    __syncwarp();
    for (int t = lane; t < n * n; t += 32) { const int i = t / n, j = t - i * n; s.B[i * NM + j] *= s.d[i] * s.d[j]; s.Z[i * NM + j] = 0.0; }
    __syncwarp();
    // Cholesky of the scaled B (lane 0; 6 x 6): B = L L^T, admitted while every pivot >= RR_CHOL
    if (lane == 0) {
        for (int j = 0; j < n && s.chol; ++j) {
            double dj = s.B[j * NM + j];
            for (int l = 0; l < j; ++l) dj -= s.Z[j * NM + l] * s.Z[j * NM + l];
            if (!(dj >= RR_CHOL)) { s.chol = 0; break; }
            const double ljj = sqrt(dj);
            s.Z[j * NM + j] = ljj;
            for (int i = j + 1; i < n; ++i) {
                double v = s.B[i * NM + j];
                for (int l = 0; l < j; ++l) v -= s.Z[i * NM + l] * s.Z[j * NM + l];
                s.Z[i * NM + j] = v / ljj;
            }
        }
        if (s.chol) {   // U = L^{-1} (lower triangular), then M = D L^{-T}: M(i, l) = d_i U(l, i)
            for (int jc = 0; jc < n; ++jc)
                for (int i = 0; i < n; ++i) {
                    double v = (i == jc) ? 1.0 : 0.0;
                    if (i < jc) { s.U[i * NM + jc] = 0.0; continue; }
                    for (int l = jc; l < i; ++l) v -= s.Z[i * NM + l] * s.U[l * NM + jc];
                    s.U[i * NM + jc] = v / s.Z[i * NM + i];
                }
            s.na = n;
        }
    }
    __syncwarp();
    if (s.chol) {
        for (int t = lane; t < n * n; t += 32) { const int i = t / n, l = t - i * n; s.M[i * NM + l] = s.d[i] * s.U[l * NM + i]; }
    } else {
        warp_jacobi(s.B, s.U, s.T, s.cs, s.sn, s.partner, n, lane);
        if (lane == 0) {
            double smax = 0.0;
            for (int j = 0; j < n; ++j) { s.sig[j] = s.B[j * NM + j]; if (s.sig[j] > smax) smax = s.sig[j]; }
            int na = 0;
            for (int j = 0; j < n; ++j) if (s.sig[j] > RR_TAU * smax && s.sig[j] > 0.0) s.keep[na++] = j;
            s.na = na;
            if (!(smax == smax)) s.bad = 1;
        }
        __syncwarp();
        for (int t = lane; t < n * s.na; t += 32) {
            const int i = t / s.na, l = t - i * s.na, j = s.keep[l];
            s.M[i * NM + l] = s.d[i] * s.U[i * NM + j] * rsqrt(s.sig[j]);
        }
    }
    __syncwarp();
    const int na = s.na;
    // reduced standard problem  At = M^T A M
    for (int t = lane; t < n * na; t += 32) {
        const int i = t / na, l = t - i * na;
        double v = 0.0;
        for (int j = 0; j < n; ++j) v += s.A[i * NM + j] * s.M[j * NM + l];
        s.T[i * NM + l] = v;
    }
    __syncwarp();
    for (int t = lane; t < na * na; t += 32) {
        const int a = t / na, b = t - a * na;
        double v = 0.0;
        for (int i = 0; i < n; ++i) v += s.M[i * NM + a] * s.T[i * NM + b];
        s.B[a * NM + b] = v;
    }
    __syncwarp();
    for (int t = lane; t < na * na; t += 32) { const int a = t / na, b = t - a * na; s.A[a * NM + b] = 0.5 * (s.B[a * NM + b] + s.B[b * NM + a]); }
    __syncwarp();
    warp_jacobi(s.A, s.Z, s.T, s.cs, s.sn, s.partner, na, lane);
    // sort ascending (ties by index; NaNs rank last and flag the solve)
    if (lane < na) {
        const double x = s.A[lane * NM + lane];
        int rank = 0;
        for (int b = 0; b < na; ++b) {
            const double y = s.A[b * NM + b];
            if (y < x || (y == x && b < lane) || (!(x == x) && (y == y || b < lane))) ++rank;
        }
        s.ord[rank] = lane;
        if (rank < nev && !(x == x)) s.bad = 1;
    }
    if (lane == 0 && na < nev) s.bad = 1;
    __syncwarp();
    for (int t = lane; t < n * nev; t += 32) {
        const int i = t / nev, j = t - i * nev;
        double v = 0.0;
        if (j < na) { const int zj = s.ord[j]; for (int l = 0; l < na; ++l) v += s.M[i * NM + l] * s.Z[l * NM + zj]; }
        C[i * nev + j] = v;
    }
    if (lane < nev) theta[lane] = lane < na ? s.A[s.ord[lane] * NM + s.ord[lane]] : 0.0;
    __syncwarp();
}

// Sum of nv (<= 64) values over the chunks of one problem in a fixed order that depends on nchunk only (so it is the same
// for every CTA of the problem and for every cpp): thread (v, g) adds the chunks g, g + G, ... (all loads of the CTA in
// flight together), then thread v combines the G group sums in order.  out[v] valid after the trailing __syncthreads.
__device__ void reduce_chunks(const double* part, int nchunk, int nv, double* out, double* scratch /*[PT]*/) {
    const int G = PT / nv, v = threadIdx.x % nv, g = threadIdx.x / nv;
    if (g < G) {
        double s = 0.0;
        for (int ch = g; ch < nchunk; ch += G) s += __ldcg(part + (size_t)ch * nv + v);
        scratch[g * nv + v] = s;
    }
    __syncthreads();
    if (threadIdx.x < nv) {
        double s = 0.0;
        for (int gg = 0; gg < G; ++gg) s += scratch[gg * nv + threadIdx.x];
        out[threadIdx.x] = s;
    }
    __syncthreads();
}

template <int KB>
__global__ void __launch_bounds__(PT, 1) k_lobpcg_persistent(const __grid_constant__ PBatch batch, const PParams q) {
    using T = Tri<KB>;
    constexpr int NS = T::NS, NT = T::NT, NK = T::NK, NEU = T::NEU;
    __shared__ double sC[3 * KB * KB + KB];
    __shared__ double sval[NEU + NK];
    __shared__ double ssign[KB];
    __shared__ double sscr[PT];
    __shared__ RRs rr;
    __shared__ int s_stop;
    __shared__ double scoef[3 * PDEG];
    __shared__ double s_hi;
    __shared__ int sord[PDEG];
    __shared__ double sack[3 * KB];
    const int prob = blockIdx.x / q.cpp, jc = blockIdx.x - prob * q.cpp;
    const PProb& pr = batch.p[prob];
    const Lat& l = q.l;
    const int N = q.N, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const long long n3 = 3ll * N;
    SolverState* st = pr.st;
    unsigned long long* bar = &st->pbar;
    unsigned long long round = 0;
    const Blk6 b = pr.b;
    double* partU[2] = {pr.part, pr.part + (size_t)q.nchunk * NEU};
    double* partK = pr.part + (size_t)2 * q.nchunk * NEU;
    double* partMv = partK + (size_t)q.nchunk * NK;
    long long* partMi = reinterpret_cast<long long*>(partMv + (size_t)q.nchunk * KB);
    const d3 muB = mk3(l.mu * l.Bx, l.mu * l.By, l.mu * l.Bz);
    const bool lead = jc == 0 && tid == 0;       // the one thread that writes this problem's solver state

    auto neighbours6 = [&](int i, int (&nb)[6]) {
        const int iy = i / l.Lx, ix = i - iy * l.Lx;
        nb[0] = nbi(l, ix, iy, 1, 0);  nb[1] = nbi(l, ix, iy, -1, 0);
        nb[2] = nbi(l, ix, iy, 0, 1);  nb[3] = nbi(l, ix, iy, 0, -1);
        nb[4] = nbi(l, ix, iy, -1, 1); nb[5] = nbi(l, ix, iy, 1, -1);
    };

    // ---------------------------------------------------------------- phase 0: c_i = m_i . g_i, start block, max(-c_i)
    for (int ch = jc; ch < q.nchunk; ch += q.cpp) {
        const int i = ch * PT + tid;
        double negc = -1e300;
        if (i < N) {
            int nb[6];
            neighbours6(i, nb);
            const d3 mi = ld3(pr.m, i);
            const d3 Lm = stencil_apply(l, ldn_cg(pr.m, nb[0]), ldn_cg(pr.m, nb[1]), ldn_cg(pr.m, nb[2]), ldn_cg(pr.m, nb[3]),
                                        ldn_cg(pr.m, nb[4]), ldn_cg(pr.m, nb[5]), mi.z);
            const double ci = dot3(mi, Lm) - dot3(mi, muB);
            pr.c[i] = ci;
            negc = -ci;
#pragma unroll
            for (int a = 0; a < KB; ++a) {
                d3 x;
                if (q.warm) x = ld3(pr.V + (size_t)a * n3, i);
                else {
                    const unsigned long long e = (unsigned long long)a * n3 + 3ull * i;
                    x.x = (double)(splitmix64(q.seed ^ splitmix64(e)) >> 11) * (1.0 / 9007199254740992.0) - 0.5;
                    x.y = (double)(splitmix64(q.seed ^ splitmix64(e + 1)) >> 11) * (1.0 / 9007199254740992.0) - 0.5;
                    x.z = (double)(splitmix64(q.seed ^ splitmix64(e + 2)) >> 11) * (1.0 / 9007199254740992.0) - 0.5;
                }
                st3(b.X + (size_t)a * n3, i, proj3(mi, x));
            }
        }
        if (q.degree > 0) {   // chunk maximum of -c_i: the upper end of the filter interval is max_i(-c_i) + lambda_max(L)
            sscr[tid] = negc;
            __syncthreads();
            for (int s = PT / 2; s > 0; s >>= 1) {
                if (tid < s) sscr[tid] = fmax(sscr[tid], sscr[tid + s]);
                __syncthreads();
            }
            if (tid == 0) partMv[ch] = sscr[0];
            __syncthreads();
        }
    }
    prob_barrier(bar, q.cpp, round, &st->bad);
    if (q.degree > 0) {
        if (tid == 0) {
            double mx = -1e300;
            for (int ch = 0; ch < q.nchunk; ++ch) mx = fmax(mx, __ldcg(partMv + ch));
            s_hi = q.hi_user > 0.0 ? q.hi_user : mx + q.lnorm;
        }
        if (tid == 32) {   // Leja order of the normalised Chebyshev roots cos((2j + 1) pi / (2d)) (depends on d only), as k_cheb_coef
            float lp[PDEG]; bool used[PDEG];
            for (int j = 0; j < PDEG; ++j) { lp[j] = 0.0f; used[j] = false; }
            int pick = 0;
            for (int sI = 0; sI < q.degree; ++sI) {
                sord[sI] = pick; used[pick] = true;
                const double xp = cospi((2.0 * pick + 1.0) / (2.0 * q.degree));
                float best = -3.0e38f; int bj = 0;
                for (int j = 0; j < q.degree; ++j) {
                    if (used[j]) continue;
                    lp[j] += __logf((float)fabs(cospi((2.0 * j + 1.0) / (2.0 * q.degree)) - xp));
                    if (lp[j] > best) { best = lp[j]; bj = j; }
                }
                pick = bj;
            }
        }
        __syncthreads();
    }

    int parity = 0, deg = 0;
    long long nhvp = 0;
    // One step over this CTA's chunks:  dst = al (Hess[src] - c0 src) + be u   (plain: dst = Hess[src]); u, dst are touched at
    // the thread's own site only, so dst may be u.  wd: also leave the partials of wd^T dst in partK.  Ends with the barrier.
    auto op_step = [&](const double* src, const double* u, double* dst, bool plain, double al, double c0, double be, const double* wd) {
        for (int ch = jc; ch < q.nchunk; ch += q.cpp) {
            const int i = ch * PT + tid;
            double acc[NK];
#pragma unroll
            for (int t = 0; t < NK; ++t) acc[t] = 0.0;
            if (i < N) {
                int nb[6];
                neighbours6(i, nb);
                const d3 mi = ld3(pr.m, i);
                const double ci = pr.c[i];
                d3 w[KB], y[KB];
#pragma unroll
                for (int a = 0; a < KB; ++a) {
                    const d3 s = ld3(src + (size_t)a * n3, i);
                    d3 v = axpy3(-ci, s, proj3(mi, stencil_at(l, src + (size_t)a * n3, nb, s.z)));
                    if (!plain) {
                        v = scale3(al, axpy3(-c0, s, v));
                        if (u) v = axpy3(be, ld3(u + (size_t)a * n3, i), v);
                    }
                    st3(dst + (size_t)a * n3, i, v);
                    y[a] = v;
                    if (wd) w[a] = (wd == src) ? s : ld3(wd + (size_t)a * n3, i);
                }
                if (wd) {
                    int t = 0;
#pragma unroll
                    for (int a = 0; a < KB; ++a)
#pragma unroll
                        for (int c2 = a; c2 < KB; ++c2) { acc[t] = dot3(w[a], y[c2]); ++t; }
                }
            }
            if (wd) {
                block_reduce_store<NK>(acc, partK + (size_t)ch * NK);
                __syncthreads();
            }
        }
        prob_barrier(bar, q.cpp, round, &st->bad);
    };
    // DST = op(SRC): the Hessian (deg == 0) or -p_deg(Hess) as deg product-form steps, Y_i alternating between T1 and T2
    auto apply_op = [&](const double* SRC, double* DST, bool dots) {
        if (deg == 0) { op_step(SRC, nullptr, DST, true, 1.0, 0.0, 0.0, dots ? SRC : nullptr); nhvp += KB; return; }
        double* buf[2] = {pr.T1, pr.T2};
        const double* ym1 = SRC;       // Y_{i-1}
        for (int i = 1; i <= deg; ++i) {
            double* dst = (i == deg) ? DST : buf[i & 1];
            op_step(ym1, nullptr, dst, false, scoef[3 * i - 3], scoef[3 * i - 2], 0.0, (dots && i == deg) ? SRC : nullptr);
            ym1 = dst;
        }
        nhvp += (long long)KB * deg;
    };
    // (re)start LOBPCG on span(X) for the current operator: AX = op(X), W = AW = P = AP = 0, Gram partials of the X block
    auto restart = [&]() {
        apply_op(b.X, b.AX, false);
        parity ^= 1;
        for (int ch = jc; ch < q.nchunk; ch += q.cpp) {
            const int i = ch * PT + tid;
            double acc[NEU];
#pragma unroll
            for (int t = 0; t < NEU; ++t) acc[t] = 0.0;
            if (i < N) {
                d3 x[KB], ax[KB];
                const d3 z = mk3(0.0, 0.0, 0.0);
#pragma unroll
                for (int a = 0; a < KB; ++a) {
                    x[a] = ld3(b.X + (size_t)a * n3, i); ax[a] = ld3(b.AX + (size_t)a * n3, i);
                    st3(b.W + (size_t)a * n3, i, z); st3(b.AW + (size_t)a * n3, i, z);
                    st3(b.P + (size_t)a * n3, i, z); st3(b.AP + (size_t)a * n3, i, z);
                }
#pragma unroll
                for (int a = 0; a < KB; ++a)
#pragma unroll
                    for (int c2 = a; c2 < KB; ++c2) {
                        acc[T::idx(a, c2)] = x[a].x * x[c2].x + x[a].y * x[c2].y + x[a].z * x[c2].z;
                        acc[NT + T::idx(a, c2)] = x[a].x * ax[c2].x + x[a].y * ax[c2].y + x[a].z * ax[c2].z;
                    }
            }
            block_reduce_store<NEU>(acc, partU[parity] + (size_t)ch * NEU);
            __syncthreads();
        }
        prob_barrier(bar, q.cpp, round, &st->bad);
    };

    // Phases (as lobpcg.cu): plain_start iterations on A, then phases of phase_len iterations on -p_d(A) with the interval
    // re-centred on the A-Ritz values at every boundary.  While transformed, convergence is decided on true A-residuals only:
    // at a boundary the solver restarts on A (probing), one Rayleigh-Ritz on span(X) + update gives the A-Ritz pairs and
    // W = A X - X Theta, and the next pass tests |W_j|.  Every decision below is taken by all CTAs of the problem from the
    // same numbers, so they stay in step without a broadcast.
    int iter = 0, in_phase = 0, nupd = 0;
    bool done = false, bad = false, fresh = true, probing = false;
    restart();
    for (;;) {
        // ------------------------------------------------------------ R: partial sums, residual test, Rayleigh-Ritz
        reduce_chunks(partU[parity], q.nchunk, NEU, sval, sscr);
        if (!fresh && !probing) reduce_chunks(partK, q.nchunk, NK, sval + NEU, sscr);
        if (tid == 0) {
            int stop = 0;
            if (!fresh) {
                bool ok = true, nan = false;
                for (int a = 0; a < KB; ++a) {
                    const double r = sqrt(sval[2 * NT + a]);
                    if (lead && deg == 0) st->resid[a] = r;
                    if (a < q.k) { ok = ok && (r <= q.tol); nan = nan || !(r == r); }
                }
                if (nan) stop = 3; else if (deg == 0 && ok) stop = 1; else if (deg == 0 && iter >= q.max_iter) stop = 2;
            }
            s_stop = stop;
        }
        __syncthreads();
        if (s_stop) { done = s_stop == 1; bad = s_stop == 3; break; }
        if (!fresh && !probing) { ++iter; if (deg > 0) ++in_phase; }
        if (q.degree > 0 && !fresh) {
            if (deg == 0 && (probing || iter >= q.plain_start)) {
                // interval [a, b] from the A-Ritz values of the last Rayleigh-Ritz (sC), coefficients as k_cheb_coef
                if (tid < q.degree) {
                    // product form over the Leja-ordered roots (see k_cheb_coef): step s is alpha_s (A - r_s), alpha_s = 1 / (a_L - r_s)
                    const double bb = s_hi, aL = sC[3 * KB * KB];
                    double aa = sC[3 * KB * KB + q.k - 1] + q.margin;
                    if (aa > 0.5 * (aL + bb)) aa = 0.5 * (aL + bb);
                    const double e = 0.5 * (bb - aa), c0 = 0.5 * (bb + aa);
                    const double r = c0 + e * cospi((2.0 * sord[tid] + 1.0) / (2.0 * q.degree));
                    double alpha = 1.0 / (aL - r);
                    if (tid == q.degree - 1) alpha = -alpha;                   // the transformed operator is -p(A)
                    scoef[3 * tid] = alpha; scoef[3 * tid + 1] = r; scoef[3 * tid + 2] = 0.0;
                }
                __syncthreads();
                deg = q.degree; in_phase = 0; nupd = 0; probing = false; fresh = true;
                restart();
                continue;
            }
            if (deg > 0 && (in_phase >= q.phase_len || iter >= q.max_iter)) {
                deg = 0; nupd = 0; probing = true; fresh = true;
                restart();
                continue;
            }
        }
        if (warp == 0) {
            for (int t = lane; t < NS * NS; t += 32) {
                const int i = t / NS, j = t - i * NS;
                const int a = i < j ? i : j, c2 = i < j ? j : i;
                const int e = T::idx(a, c2);
                double ga = sval[NT + e];
                if (!fresh && a >= KB && c2 < 2 * KB) ga = sval[NEU + (a - KB) * KB - (a - KB) * (a - KB - 1) / 2 + (c2 - a)];   // (W, W) block from H
                rr.B[i * NM + j] = sval[e];
                rr.A[i * NM + j] = ga;
            }
            __syncwarp();
            warp_rr(rr, NS, KB, sC + 3 * KB * KB, sC, lane);
        }
        __syncthreads();
        if (rr.bad) { bad = true; break; }
        if (lead) {
            if (deg == 0) for (int a = 0; a < KB; ++a) st->theta[a] = sC[3 * KB * KB + a];
            st->nkeep = rr.na; st->iter = iter; st->nhvp = nhvp;
        }
        // ------------------------------------------------------------ U: fused update of the six blocks + Gram partials
        parity ^= 1;
        for (int ch = jc; ch < q.nchunk; ch += q.cpp) {
            const int i = ch * PT + tid;
            double acc[NEU];
#pragma unroll
            for (int t = 0; t < NEU; ++t) acc[t] = 0.0;
            if (i < N) update_site<KB, true>(b, pr.m, sC, 3ll * i, n3, acc);
            block_reduce_store<NEU>(acc, partU[parity] + (size_t)ch * NEU);
            __syncthreads();
        }
        prob_barrier(bar, q.cpp, round, &st->bad);
        fresh = false;
        // ------------------------------------------------------------ cheap convergence test between boundaries (transformed only):
        // T1 = A X, theta_j = x_j.t_j / x_j.x_j, |t_j - theta_j x_j| / |x_j| formed element by element (as fast_acheck, lobpcg_fast.cu)
        ++nupd;
        if (deg > 0 && q.acheck_every > 0 && nupd > 1 && (nupd - 1) % q.acheck_every == 0) {
            for (int ch = jc; ch < q.nchunk; ch += q.cpp) {
                const int i = ch * PT + tid;
                double acc[2 * KB];
#pragma unroll
                for (int t = 0; t < 2 * KB; ++t) acc[t] = 0.0;
                if (i < N) {
                    int nb[6];
                    neighbours6(i, nb);
                    const d3 mi = ld3(pr.m, i);
                    const double ci = pr.c[i];
#pragma unroll
                    for (int a = 0; a < KB; ++a) {
                        const d3 x = ld3(b.X + (size_t)a * n3, i);
                        const d3 t = axpy3(-ci, x, proj3(mi, stencil_at(l, b.X + (size_t)a * n3, nb, x.z)));
                        st3(pr.T1 + (size_t)a * n3, i, t);
                        acc[2 * a] = dot3(x, x); acc[2 * a + 1] = dot3(x, t);
                    }
                }
                block_reduce_store<2 * KB>(acc, partK + (size_t)ch * 2 * KB);   // 2 KB <= NK + KB: partK and partMv are free here
                __syncthreads();
            }
            nhvp += KB;
            prob_barrier(bar, q.cpp, round, &st->bad);
            reduce_chunks(partK, q.nchunk, 2 * KB, sack, sscr);
            for (int ch = jc; ch < q.nchunk; ch += q.cpp) {
                const int i = ch * PT + tid;
                double acc[KB];
#pragma unroll
                for (int a = 0; a < KB; ++a) {
                    acc[a] = 0.0;
                    if (i < N) {
                        const double th = sack[2 * a + 1] / sack[2 * a];
                        const d3 x = ld3(b.X + (size_t)a * n3, i), t = ld3(pr.T1 + (size_t)a * n3, i);
                        const d3 r = axpy3(-th, x, t);
                        acc[a] = dot3(r, r);
                    }
                }
                block_reduce_store<KB>(acc, partU[parity ^ 1] + (size_t)ch * KB);   // the other parity's partials were consumed by R
                __syncthreads();
            }
            prob_barrier(bar, q.cpp, round, &st->bad);
            reduce_chunks(partU[parity ^ 1], q.nchunk, KB, sack + 2 * KB, sscr);
            bool ok = true;
            for (int a = 0; a < q.k; ++a) ok = ok && (sqrt(sack[2 * KB + a] / sack[2 * a]) <= q.tol);
            if (ok) {
                if (lead) for (int a = 0; a < KB; ++a) { st->theta[a] = sack[2 * a + 1] / sack[2 * a]; st->resid[a] = sqrt(sack[2 * KB + a] / sack[2 * a]); }
                ++iter;
                done = true;
                break;
            }
        }
        // ------------------------------------------------------------ H: AW = op(W), W^T (op W) partials (not needed for a probe)
        if (!(probing && q.degree > 0)) apply_op(b.W, b.AW, true);
    }

    // ---------------------------------------------------------------- finish: exactly tangent, sign-normalised block out
    for (int ch = jc; ch < q.nchunk; ch += q.cpp) {
        const int i = ch * PT + tid;
        __shared__ double sv[PT];
        __shared__ long long si[PT];
        for (int a = 0; a < KB; ++a) {
            double best = -1.0; long long bi = -1;
            if (i < N) {
                const d3 x = proj3(ld3(pr.m, i), ld3(b.X + (size_t)a * n3, i));
                st3(b.X + (size_t)a * n3, i, x);
                const double cx[3] = {fabs(x.x), fabs(x.y), fabs(x.z)};
                for (int c2 = 0; c2 < 3; ++c2) if (cx[c2] > best) { best = cx[c2]; bi = 3ll * i + c2; }
            }
            sv[tid] = best; si[tid] = bi;
            __syncthreads();
            for (int s = PT / 2; s > 0; s >>= 1) {
                if (tid < s) {
                    const double o = sv[tid + s]; const long long oi = si[tid + s];
                    if (o > sv[tid] || (o == sv[tid] && oi >= 0 && (si[tid] < 0 || oi < si[tid]))) { sv[tid] = o; si[tid] = oi; }
                }
                __syncthreads();
            }
            if (tid == 0) { partMv[(size_t)ch * KB + a] = sv[0]; partMi[(size_t)ch * KB + a] = si[0]; }
            __syncthreads();
        }
    }
    prob_barrier(bar, q.cpp, round, &st->bad);
    if (tid < KB) {
        double best = -1.0; long long bi = -1;
        for (int ch = 0; ch < q.nchunk; ++ch) {
            const double o = __ldcg(partMv + (size_t)ch * KB + tid); const long long oi = __ldcg(partMi + (size_t)ch * KB + tid);
            if (oi >= 0 && (o > best || (o == best && oi < bi))) { best = o; bi = oi; }
        }
        ssign[tid] = (bi >= 0 && __ldcg(b.X + (size_t)tid * n3 + bi) < 0.0) ? -1.0 : 1.0;
    }
    __syncthreads();
    for (int ch = jc; ch < q.nchunk; ch += q.cpp) {
        const int i = ch * PT + tid;
        if (i >= N) continue;
        for (int a = 0; a < q.k; ++a) {
            d3 x = ld3(b.X + (size_t)a * n3, i);
            if (ssign[a] < 0.0) { x = scale3(-1.0, x); st3(b.X + (size_t)a * n3, i, x); }
            st3(pr.V + (size_t)a * n3, i, x);
        }
    }
    if (lead) {
        HostStatus hs;
        for (int a = 0; a < MOTO_KMAX; ++a) { hs.theta[a] = a < KB ? st->theta[a] : 0.0; hs.resid[a] = a < KB ? st->resid[a] : 0.0; }
        hs.done = done ? 1 : 0; hs.iter = iter; hs.nkeep = st->nkeep; hs.bad = (bad || st->bad) ? 1 : 0; hs.nhvp = nhvp;
        st->done = hs.done; st->iter = iter; st->bad = hs.bad; st->nhvp = nhvp;
        q.out[prob] = hs;
        for (int a = 0; a < q.k; ++a) pr.lambda[a] = hs.theta[a];
    }
}

}  // namespace

// May this context's solve run in the persistent kernel?  Nearest-neighbour spin lattice, block size <= 2 without guard
// columns, LOBPCG, small enough that a solve is latency bound (one chunk per CTA of a full cooperative grid).
bool persistent_applicable(const moto_ctx* c, int k, int max_iter) {
    if (c->kind != MOTO_KIND_TRI2D || c->nsh > 0 || c->opts.method != 0 || c->opts.guard > 0 || c->keep_guard) return false;
    if (k < 1 || k > 2 || k > c->kmax || max_iter < 1) return false;
    if (c->opts.hvp_path == 2 || c->opts.persistent == 2) return false;                                 // forced TMA path / opt-out
    // an explicit degree asks for the multi-launch transformation of lobpcg.cu unless the persistent kernel is asked for too
    if (c->opts.precond_degree > 0 && (c->opts.persistent != 1 || c->opts.precond_degree > PDEG || !c->T1 || !c->T2)) return false;
    if (2ll * c->N < 3ll * k) return false;
    return c->N <= PT * MOTO_NUM_SMS;   // 37 888 sites: one 256-site chunk per CTA of a full cooperative grid
}

// Solve P problems (ctxs[p], d_spins[p]) in one launch chain on ctxs[0]'s stream; all contexts share lattice and parameters
// (the caller checked).  Results to d_V[p], d_lambda[p], infos[p]; statuses[p] per problem.
moto_status persistent_solve(moto_ctx* const* ctxs, int P, const double* const* d_spins, int k, double tol, int max_iter, int warm_start,
                             double* const* d_lambda, double* const* d_V, moto_solve_info* infos, int32_t* statuses) {
    moto_ctx* c0 = ctxs[0];
    const int N = c0->N, nchunk = (N + PT - 1) / PT;
    int dev = 0, sms = 0;
    MOTO_CUDA_CHECK(c0, cudaGetDevice(&dev));
    MOTO_CUDA_CHECK(c0, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    HostStatus* d_out = reinterpret_cast<HostStatus*>(c0->partials + 200000);          // [P] beyond every chunk partial
    static_assert(sizeof(HostStatus) * PMAXP <= 8 * 100000, "status array does not fit");
    moto_status worst = MOTO_OK;
    for (int p0 = 0; p0 < P; p0 += PMAXP) {
        const int Pn = P - p0 < PMAXP ? P - p0 : PMAXP;
        int cpp = sms / Pn;
        if (cpp > nchunk) cpp = nchunk;
        if (cpp < 1) cpp = 1;
        PBatch batch;
        memset(&batch, 0, sizeof(batch));
        for (int p = 0; p < Pn; ++p) {
            moto_ctx* c = ctxs[p0 + p];
            PProb& pr = batch.p[p];
            pr.m = d_spins[p0 + p]; pr.V = d_V[p0 + p]; pr.lambda = d_lambda[p0 + p];
            pr.b.X = c->X; pr.b.W = c->W; pr.b.P = c->P; pr.b.AX = c->AX; pr.b.AW = c->AW; pr.b.AP = c->AP;
            pr.c = c->c; pr.T1 = c->T1; pr.T2 = c->T2; pr.part = c->partials; pr.st = c->st;
            MOTO_CUDA_CHECK(c0, cudaMemsetAsync(c->st, 0, sizeof(SolverState), c0->stream));
        }
        PParams q;
        q.l = make_lat(c0); q.N = N; q.nchunk = nchunk; q.cpp = cpp; q.k = k; q.max_iter = max_iter; q.warm = warm_start;
        q.tol = tol; q.seed = c0->opts.seed; q.out = d_out;
        // transformation: precond_degree 0 = auto, < 0 = off; every context of the batch needs the two recurrence blocks
        q.degree = c0->opts.precond_degree > 0 ? c0->opts.precond_degree : (c0->opts.precond_degree == 0 && N >= PAUTO_MIN_N ? PAUTO_DEGREE : 0);
        for (int p = 0; p < Pn; ++p) if (!batch.p[p].T1 || !batch.p[p].T2) q.degree = 0;
        if (3ll * k * 8 > 2ll * N) q.degree = 0;
        q.plain_start = warm_start ? 0 : PAUTO_PLAIN; q.phase_len = PAUTO_PHASE; q.acheck_every = PAUTO_ACHECK;
        q.margin = c0->opts.precond_lo > 0 ? c0->opts.precond_lo : 0.01; q.lnorm = c0->lmax_L; q.hi_user = c0->opts.precond_hi;
        void* args[2] = {(void*)&batch, (void*)&q};
        const void* fn = k == 1 ? (const void*)k_lobpcg_persistent<1> : (const void*)k_lobpcg_persistent<2>;
        MOTO_CUDA_CHECK(c0, cudaLaunchCooperativeKernel(fn, dim3(Pn * cpp), dim3(PT), args, 0, c0->stream));
        c0->launches += 1;
        HostStatus hs[PMAXP];
        MOTO_CUDA_CHECK(c0, cudaMemcpyAsync(hs, d_out, Pn * sizeof(HostStatus), cudaMemcpyDeviceToHost, c0->stream));
        MOTO_CUDA_CHECK(c0, cudaStreamSynchronize(c0->stream));
        for (int p = 0; p < Pn; ++p) {
            moto_ctx* c = ctxs[p0 + p];
            moto_status s = MOTO_OK;
            if (hs[p].bad) s = moto_fail(c, MOTO_ECUDA, "moto_lowest_modes: numerical breakdown (NaN or rank loss) in Rayleigh-Ritz");
            else if (!hs[p].done) s = moto_fail(c, MOTO_ENOTCONV, "moto_lowest_modes: max_iter reached; outputs hold the best iterate");
            if (infos) {
                moto_solve_info& in = infos[p0 + p];
                in.iters = hs[p].iter; in.converged = (hs[p].done && !hs[p].bad) ? 1 : 0; in.hvp_count = hs[p].nhvp;
                for (int a = 0; a < MOTO_KMAX; ++a) in.resid[a] = a < k ? hs[p].resid[a] : 0.0;
            }
            if (statuses) statuses[p0 + p] = (int32_t)s;
            if (s != MOTO_OK && (worst == MOTO_OK || worst == MOTO_ENOTCONV)) worst = s;
        }
    }
    return worst;
}
