// spin_shells.cu -- K1 for GENERAL neighbour shells: Eq. 4 with a translation-invariant
// table of couplings J_delta and three-component D_delta over lattice offsets delta = (dx, dy) -- the paper's real
// Pd/Fe/Ir(111) workload class (Tables I/II PAPER.md:328-616: ~340 neighbours per site, 100x100 periodic).
//   (L u)_i = -2 sum_delta [ J_delta u_{i+delta} + u_{i+delta} x D_delta ] - 2 K u_iz z      (ordered pairs, reading A1)
//   g = L m - mu B,  c_i = m_i.g_i,  Hess[v]_i = P_i (L Pv)_i - c_i (Pv)_i                  (reading A5)
// With hundreds of neighbours per site the step is no longer HBM-bound (10^4 sites x 24 B fit in L1/L2 many times over)
// but bound by the fp64 pipe and by load issue: 9 flops per neighbour per field.  One WARP per site: the lanes stride over
// the table (entries are sorted by (dy, dx), so consecutive lanes read consecutive sites: coalesced), every lane
// accumulates J u + u x D for m and the k directions from ONE read of each neighbour, a shuffle tree sums the lanes, and
// lanes 0..k-1 finish one direction each.  10^4 sites x 32 lanes = 1250 CTAs: fills the 148 SMs where a thread per site
// would occupy 40.
#include "common.cuh"
#include "device_utils.cuh"
#include "stencil_math.cuh"

namespace {

struct ShellTab { int n; const int* off; const double* jd; };   // off [n][2] = (dx, dy); jd [n][4] = J, Dx, Dy, Dz

__device__ __forceinline__ d3 cross3(d3 u, d3 D) { return mk3(u.y * D.z - u.z * D.y, u.z * D.x - u.x * D.z, u.x * D.y - u.y * D.x); }

// neighbour site of (ix, iy) at table entry t, or -1 (open boundary)
__device__ __forceinline__ long long shell_nb(const Lat& l, const ShellTab& tb, int t, int ix, int iy) {
    int jx = ix + tb.off[2 * t], jy = iy + tb.off[2 * t + 1];
    if (jx < 0 || jx >= l.Lx) {      // one conditional add covers |dx| <= Lx; the division only runs for longer offsets
        if (!l.px) return -1;
        jx += jx < 0 ? l.Lx : -l.Lx;
        if (jx < 0 || jx >= l.Lx) { jx %= l.Lx; if (jx < 0) jx += l.Lx; }
    }
    if (jy < 0 || jy >= l.Ly) {
        if (!l.py) return -1;
        jy += jy < 0 ? l.Ly : -l.Ly;
        if (jy < 0 || jy >= l.Ly) { jy %= l.Ly; if (jy < 0) jy += l.Ly; }
    }
    return (long long)jy * l.Lx + jx;
}

// the CTA's copy of the table in shared memory (20 KB at 512 entries): no dependent global loads in the neighbour loop
struct ShellSmem { double jd[MOTO_MAX_SHELLS * 4]; int off[MOTO_MAX_SHELLS * 2]; };
__device__ __forceinline__ ShellTab stage_table(const ShellTab& tb, ShellSmem& sm) {
    for (int t = threadIdx.x; t < 4 * tb.n; t += blockDim.x) sm.jd[t] = tb.jd[t];
    for (int t = threadIdx.x; t < 2 * tb.n; t += blockDim.x) sm.off[t] = tb.off[t];
    __syncthreads();
    ShellTab r; r.n = tb.n; r.off = sm.off; r.jd = sm.jd;
    return r;
}

__device__ __forceinline__ d3 warp_sum3(d3 v) { return mk3(warp_sum(v.x), warp_sum(v.y), warp_sum(v.z)); }

// energy partials + tangent-projected gradient (+ c)
__global__ void __launch_bounds__(256) k_shell_energy_grad(Lat l, ShellTab tbg, const double* __restrict__ m, double* __restrict__ g_out,
                                                           double* __restrict__ c_out, double* __restrict__ partials) {
    __shared__ double red[32];
    __shared__ ShellSmem ssm;
    const ShellTab tb = stage_table(tbg, ssm);
    const long long N = (long long)l.Lx * l.Ly;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double e[1] = {0.0};
    const d3 B = mk3(l.mu * l.Bx, l.mu * l.By, l.mu * l.Bz);
    for (long long i = (long long)blockIdx.x * 8 + warp; i < N; i += (long long)gridDim.x * 8) {
        const int iy = (int)(i / l.Lx), ix = (int)(i - (long long)iy * l.Lx);
        d3 acc = mk3(0.0, 0.0, 0.0);
        for (int t = lane; t < tb.n; t += 32) {
            const long long j = shell_nb(l, tb, t, ix, iy);
            if (j < 0) continue;
            const d3 mj = ld3(m, j);
            const d3 D = mk3(tb.jd[4 * t + 1], tb.jd[4 * t + 2], tb.jd[4 * t + 3]);
            acc = add3(acc, axpy3(tb.jd[4 * t], mj, cross3(mj, D)));
        }
        acc = warp_sum3(acc);
        if (lane == 0) {
            const d3 mi = ld3(m, i);
            const d3 Lm = mk3(-2.0 * acc.x, -2.0 * acc.y, -2.0 * acc.z - 2.0 * l.K * mi.z);
            const d3 g = sub3(Lm, B);
            const double c = dot3(mi, g);
            e[0] += 0.5 * dot3(mi, Lm) - dot3(mi, B);
            if (g_out) st3(g_out, i, axpy3(-c, mi, g));
            if (c_out) c_out[i] = c;
        }
    }
    block_sum<1>(e, red);
    if (threadIdx.x == 0) partials[blockIdx.x] = e[0];
}

__global__ void __launch_bounds__(1024) k_shell_final_sum(const double* __restrict__ partials, int nblk, double* __restrict__ out) {
    __shared__ double sm[1024];
    double s = 0.0;
    for (int b = threadIdx.x; b < nblk; b += 1024) s += partials[b];
    sm[threadIdx.x] = s;
    __syncthreads();
    for (int off = 512; off >= 1; off >>= 1) {
        if (threadIdx.x < off) sm[threadIdx.x] += sm[threadIdx.x + off];
        __syncthreads();
    }
    if (threadIdx.x == 0) out[0] = sm[0];
}

// block HVP.  PROJECT: API mode (neighbours projected, P_j v_j).  cvec == nullptr: c from the same pass over m.
// CHEB: three-term epilogue out = alpha (Hess[v] - c0 v) + beta u (solver mode).
template <bool PROJECT, bool CHEB, int KT>   // KT: compile-time bound on k (1, 2 or MOTO_KMAX): accumulators and unrolling
__global__ void __launch_bounds__(256) k_shell_hvp(Lat l, ShellTab tbg, const double* __restrict__ m, const double* __restrict__ cvec,
                                                   const double* __restrict__ V, int k, double* __restrict__ HV,
                                                   const int* __restrict__ done, double alpha, double c0, double beta,
                                                   const double* U) {
    if (done && *done) return;
    __shared__ ShellSmem ssm;
    const ShellTab tb = stage_table(tbg, ssm);
    const long long N = (long long)l.Lx * l.Ly;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const bool need_c = cvec == nullptr;
    const d3 B = mk3(l.mu * l.Bx, l.mu * l.By, l.mu * l.Bz);
    for (long long i = (long long)blockIdx.x * 8 + warp; i < N; i += (long long)gridDim.x * 8) {
        const int iy = (int)(i / l.Lx), ix = (int)(i - (long long)iy * l.Lx);
        d3 accm = mk3(0.0, 0.0, 0.0);
        d3 acc[KT];
#pragma unroll
        for (int a = 0; a < KT; ++a) acc[a] = mk3(0.0, 0.0, 0.0);
        // (unrolling this loop by four with the absent neighbours predicated instead of skipped was slower, 46 -> 62 us at
        //  k = 2: more registers, fewer resident warps)
        for (int t = lane; t < tb.n; t += 32) {
            const long long j = shell_nb(l, tb, t, ix, iy);
            if (j < 0) continue;
            const double J = tb.jd[4 * t];
            const d3 D = mk3(tb.jd[4 * t + 1], tb.jd[4 * t + 2], tb.jd[4 * t + 3]);
            d3 mj = mk3(0.0, 0.0, 0.0);
            if (PROJECT || need_c) mj = ld3(m, j);
            if (need_c) accm = add3(accm, axpy3(J, mj, cross3(mj, D)));
#pragma unroll
            for (int a = 0; a < KT; ++a) {
                if (a < k) {
                    d3 vj = ld3(V + (size_t)a * 3 * N, j);
                    if (PROJECT) vj = proj3(mj, vj);
                    acc[a] = add3(acc[a], axpy3(J, vj, cross3(vj, D)));
                }
            }
        }
        if (need_c) accm = warp_sum3(accm);
#pragma unroll
        for (int a = 0; a < KT; ++a)
            if (a < k) acc[a] = warp_sum3(acc[a]);
        // lanes 0..k-1 finish one direction each (the sums are in every lane after the xor tree)
        d3 mine = mk3(0.0, 0.0, 0.0);
#pragma unroll
        for (int a = 0; a < KT; ++a)
            if (a == lane) mine = acc[a];
        if (lane < k) {
            const d3 mi = ld3(m, i);
            double c;
            if (need_c) {
                const d3 Lm = mk3(-2.0 * accm.x, -2.0 * accm.y, -2.0 * accm.z - 2.0 * l.K * mi.z);
                c = dot3(mi, Lm) - dot3(mi, B);
            } else {
                c = cvec[i];
            }
            const size_t o = (size_t)lane * 3 * N;
            d3 vi = ld3(V + o, i);
            if (PROJECT) vi = proj3(mi, vi);
            const d3 Lv = mk3(-2.0 * mine.x, -2.0 * mine.y, -2.0 * mine.z - 2.0 * l.K * vi.z);
            d3 h = axpy3(-c, vi, proj3(mi, Lv));
            if (CHEB) {
                h = scale3(alpha, axpy3(-c0, vi, h));
                if (U) h = axpy3(beta, ld3(U + o, i), h);
            }
            st3(HV + o, i, h);
        }
    }
}

// F = -g in place, partial dots alpha_a = F . v_a  (pass 1 of the reflected-force step when g came from k_shell_energy_grad)
__global__ void __launch_bounds__(256) k_shell_negdots(long long N, double* __restrict__ F, const double* __restrict__ v, int kr,
                                                       double* __restrict__ partials) {
    __shared__ double red[32 * MOTO_KMAX];
    double acc[MOTO_KMAX];
#pragma unroll
    for (int a = 0; a < MOTO_KMAX; ++a) acc[a] = 0.0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        const d3 f = scale3(-1.0, ld3(F, i));
        st3(F, i, f);
#pragma unroll
        for (int a = 0; a < MOTO_KMAX; ++a)
            if (a < kr) acc[a] += dot3(f, ld3(v + (size_t)a * 3 * N, i));
    }
    block_sum<MOTO_KMAX>(acc, red);
    if (threadIdx.x == 0)
        for (int a = 0; a < MOTO_KMAX; ++a) partials[blockIdx.x * MOTO_KMAX + a] = acc[a];
}

ShellTab tab_of(const moto_ctx* c) { ShellTab t; t.n = c->nsh; t.off = c->sh_off; t.jd = c->sh_jd; return t; }

int shell_grid(const moto_ctx* c) {
    long long b = ((long long)c->N + 7) / 8;
    return (int)(b < 4096 ? (b > 0 ? b : 1) : 4096);
}

}  // namespace

int shell_energy_grad(moto_ctx* c, const double* m, double* d_E, double* d_g, double* d_c) {
    int gd = 0;
    if (shell_dense_energy_grad(c, m, d_g, d_c, c->partials, &gd)) {   // register-blocked kernel, m the only staged field
        if (d_E) { k_shell_final_sum<<<1, 1024, 0, c->stream>>>(c->partials, gd, d_E); return 2; }
        return 1;
    }
    const int grid = shell_grid(c);
    k_shell_energy_grad<<<grid, 256, 0, c->stream>>>(make_lat(c), tab_of(c), m, d_g, d_c, c->partials);
    int n = 1;
    if (d_E) { k_shell_final_sum<<<1, 1024, 0, c->stream>>>(c->partials, grid, d_E); ++n; }
    return n;
}

int shell_hvp(moto_ctx* c, const double* m, const double* cvec, const double* V, int k, double* HV, int project_input, const int* d_done) {
    if (const int nd = shell_dense_hvp(c, m, cvec, V, k, HV, project_input, d_done, 0, 0.0, 0.0, 0.0, nullptr, nullptr)) return nd;
    const int grid = shell_grid(c);
#define SHELL_HVP(P, KT) k_shell_hvp<P, false, KT><<<grid, 256, 0, c->stream>>>(make_lat(c), tab_of(c), m, cvec, V, k, HV, d_done, 0.0, 0.0, 0.0, nullptr)
    if (project_input) { if (k == 1) SHELL_HVP(true, 1); else if (k == 2) SHELL_HVP(true, 2); else SHELL_HVP(true, MOTO_KMAX); }
    else { if (k == 1) SHELL_HVP(false, 1); else if (k == 2) SHELL_HVP(false, 2); else SHELL_HVP(false, MOTO_KMAX); }
#undef SHELL_HVP
    return 1;
}

int shell_three_term(moto_ctx* c, const double* m, const double* cvec, const double* V, int k, double alpha, double c0, double beta,
                     const double* U, double* out) {
    if (cvec)
        if (const int nd = shell_dense_hvp(c, m, cvec, V, k, out, 0, nullptr, 1, alpha, c0, beta, U, nullptr)) return nd;
    if (k <= 2) k_shell_hvp<false, true, 2><<<shell_grid(c), 256, 0, c->stream>>>(make_lat(c), tab_of(c), m, cvec, V, k, out, nullptr, alpha, c0, beta, U);
    else k_shell_hvp<false, true, MOTO_KMAX><<<shell_grid(c), 256, 0, c->stream>>>(make_lat(c), tab_of(c), m, cvec, V, k, out, nullptr, alpha, c0, beta, U);
    return 1;
}

// pass 1 of the reflected-force step: F = -P g into ctx->g, partial dots F.v_a into ctx->partials [MOTO_RED_BLOCKS][KMAX]
int shell_mmf_pass1(moto_ctx* c, const double* m, const double* v, int kr) {
    int n = shell_energy_grad(c, m, nullptr, c->g, nullptr);
    k_shell_negdots<<<MOTO_RED_BLOCKS, 256, 0, c->stream>>>((long long)c->N, c->g, v, kr, c->partials);
    return n + 1;
}

// host side of moto_set_shells: validate (distinct, non-zero, inversion symmetric), copy the table into the workspace
moto_status shell_set(moto_ctx* c, int n, const int32_t* h_off, const double* h_J, const double* h_D) {
    if (n == 0) { c->nsh = 0; c->sh_nseg = 0; return MOTO_OK; }   // (moto_set_shells restores the stencil's lmax_L)
    for (int t = 0; t < n; ++t) {
        const int dx = h_off[2 * t], dy = h_off[2 * t + 1];
        if (dx == 0 && dy == 0) return moto_fail(c, MOTO_EINVAL, "moto_set_shells: zero offset");
        int partner = -1;
        for (int u = 0; u < n; ++u) {
            if (u != t && h_off[2 * u] == dx && h_off[2 * u + 1] == dy) return moto_fail(c, MOTO_EINVAL, "moto_set_shells: duplicate offset");
            if (h_off[2 * u] == -dx && h_off[2 * u + 1] == -dy) partner = u;
        }
        if (partner < 0 || h_J[partner] != h_J[t] || h_D[3 * partner] != -h_D[3 * t] || h_D[3 * partner + 1] != -h_D[3 * t + 1] ||
            h_D[3 * partner + 2] != -h_D[3 * t + 2])
            return moto_fail(c, MOTO_EINVAL, "moto_set_shells: table must be inversion symmetric, J(-d) = J(d), D(-d) = -D(d)");
    }
    double jd[MOTO_MAX_SHELLS * 4];
    for (int t = 0; t < n; ++t) { jd[4 * t] = h_J[t]; jd[4 * t + 1] = h_D[3 * t]; jd[4 * t + 2] = h_D[3 * t + 1]; jd[4 * t + 3] = h_D[3 * t + 2]; }
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(c->sh_off, h_off, (size_t)n * 2 * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(c->sh_jd, jd, (size_t)n * 4 * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    c->nsh = n;
    // ||L|| <= 2 sum_delta (|J_delta| + |D_delta|) + 2 |K|: the upper end of the Chebyshev interval is max_i(-c_i) + this
    double bound = 2.0 * fabs(c->sp.K);
    for (int t = 0; t < n; ++t) bound += 2.0 * (fabs(h_J[t]) + sqrt(h_D[3 * t] * h_D[3 * t] + h_D[3 * t + 1] * h_D[3 * t + 1] + h_D[3 * t + 2] * h_D[3 * t + 2]));
    c->lmax_L = bound;
    return shell_dense_build(c, n, h_off, jd);
}
