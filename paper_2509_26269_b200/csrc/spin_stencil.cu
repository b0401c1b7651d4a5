// spin_stencil.cu -- K1 (fused gradient + block Riemannian HVP stencil), K6 (reflected-force step +
// retraction) and the tangent projector for the 2-D triangular spin lattice.
//
// The Euclidean Hessian of Eq. 4 is constant: with ordered-pair counting (A1)
//   (L u)_i = -2 sum_{j in nn(i)} [ J u_j + u_j x D_ij ] - 2 K u_iz z ,   D_ij = D (z x rhat_ij)
// so  g_i = (L m)_i - mu B,  c_i = m_i . g_i,  and on a tangent vector v (A5)
//   Hess[v]_i = P_i (L v)_i - c_i v_i ,  P_i = I - m_i m_i^T.
// For a +- bond pair with unit vector (rx, ry):  u+ x D+ + u- x D-  =  D ( -rx dz, -ry dz, rx dx + ry dy ),
// d = u+ - u-, which is all the DMI costs.
//
// This file holds the generic path (any Lx, Ly, boundary): one thread per site, neighbours through
// L1/L2.  The TMA-staged fast path lives in spin_stencil_tma.cu.
#include "common.cuh"
#include "device_utils.cuh"
#include "stencil_math.cuh"

namespace {

// neighbour site index or -1 (open boundary)
__device__ __forceinline__ long long nb(const Lat& l, int ix, int iy, int dx, int dy) {
    int jx = ix + dx, jy = iy + dy;
    if (jx < 0) { if (!l.px) return -1; jx += l.Lx; }
    if (jx >= l.Lx) { if (!l.px) return -1; jx -= l.Lx; }
    if (jy < 0) { if (!l.py) return -1; jy += l.Ly; }
    if (jy >= l.Ly) { if (!l.py) return -1; jy -= l.Ly; }
    return (long long)jy * l.Lx + jx;
}

struct Nbrs { long long p1, m1, p2, m2, p3, m3; };  // +-a1, +-a2, +-(a2-a1)

__device__ __forceinline__ Nbrs neighbours(const Lat& l, int ix, int iy) {
    Nbrs n;
    n.p1 = nb(l, ix, iy, 1, 0);  n.m1 = nb(l, ix, iy, -1, 0);
    n.p2 = nb(l, ix, iy, 0, 1);  n.m2 = nb(l, ix, iy, 0, -1);
    n.p3 = nb(l, ix, iy, -1, 1); n.m3 = nb(l, ix, iy, 1, -1);
    return n;
}

__device__ __forceinline__ d3 ldn(const double* __restrict__ u, long long j) {
    return j >= 0 ? ld3(u, j) : mk3(0.0, 0.0, 0.0);
}

__device__ __forceinline__ d3 stencil_field(const Lat& l, const double* __restrict__ u, const Nbrs& n, double uz) {
    return stencil_apply(l, ldn(u, n.p1), ldn(u, n.m1), ldn(u, n.p2), ldn(u, n.m2), ldn(u, n.p3), ldn(u, n.m3), uz);
}

// projected neighbour value  P_j v_j
__device__ __forceinline__ d3 ldnp(const double* __restrict__ m, const double* __restrict__ v, long long j) {
    if (j < 0) return mk3(0.0, 0.0, 0.0);
    return proj3(ld3(m, j), ld3(v, j));
}

// ---------------------------------------------------------------- energy + gradient (+ c)
__global__ void __launch_bounds__(256) k_energy_grad(Lat l, const double* __restrict__ m, double* __restrict__ g_out,
                                                     double* __restrict__ c_out, double* __restrict__ partials,
                                                     double* __restrict__ e_out, unsigned* counter) {
    __shared__ double red[32];
    const long long N = (long long)l.Lx * l.Ly;
    double e[1] = {0.0};
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        int iy = (int)(i / l.Lx), ix = (int)(i - (long long)iy * l.Lx);
        Nbrs n = neighbours(l, ix, iy);
        d3 mi = ld3(m, i);
        d3 Lm = stencil_field(l, m, n, mi.z);
        d3 B = mk3(l.mu * l.Bx, l.mu * l.By, l.mu * l.Bz);
        d3 g = sub3(Lm, B);
        double c = dot3(mi, g);
        e[0] += 0.5 * dot3(mi, Lm) - dot3(mi, B);
        if (g_out) st3(g_out, i, axpy3(-c, mi, g));
        if (c_out) c_out[i] = c;
    }
    block_sum<1>(e, red);
    if (threadIdx.x == 0) partials[blockIdx.x] = e[0];
    last_cta_sum(partials, 1, 1, e_out, 0, counter);   // E itself, by the CTA that finishes last
}

// ---------------------------------------------------------------- fused line-search trial of moto_relax (relax.cu)
// One pass per trial: a CTA stages the 32 x 8 site tile plus its one-site halo of the TRIAL state x_t = R(x + a d) in shared
// memory (retraction computed once per staged site: 340 for 256 sites), applies the stencil from there, and emits x_t,
// g_t = P_t (L x_t - mu B) and the partial sums of E_t, g_t.g_t, g_t.g, g_t.d: 120 B/site, the trial state never makes a round
// trip through HBM before the stencil.  (Recomputing x_t at the seven sites per thread straight from global memory was
// 3x slower than the plain gradient: 14 strided site loads per thread.)
// TRIAL = false: plain evaluation at x (d, g ignored, nothing retracted, x_t not written).
#define RT_W 32
#define RT_H 8
template <bool TRIAL>
__global__ void __launch_bounds__(RT_W * RT_H) k_relax_eval(Lat l, const double* __restrict__ x, const double* __restrict__ d, double a,
                                                            const double* __restrict__ g_old, double* __restrict__ xt_out,
                                                            double* __restrict__ gt_out, double* __restrict__ partials,
                                                            const RelaxDev* __restrict__ rs = nullptr) {
    __shared__ double tile[RT_H + 2][RT_W + 2][3];
    __shared__ double red[32 * 4];
    if (rs) {   // device-resident line search: the trial is described by the state k_relax_decide left
        if (rs->status) return;
        x = rs->x[rs->cur]; xt_out = rs->x[rs->cur == 1 ? 2 : 1]; d = rs->d; a = rs->a;
        g_old = rs->g[rs->gcur]; gt_out = rs->g[rs->gcur ^ 1];
    }
    const int tx0 = blockIdx.x * RT_W, ty0 = blockIdx.y * RT_H;
    for (int cell = threadIdx.x; cell < (RT_W + 2) * (RT_H + 2); cell += RT_W * RT_H) {
        const int ly = cell / (RT_W + 2), lx = cell - ly * (RT_W + 2);
        int gx = tx0 + lx - 1, gy = ty0 + ly - 1;
        bool ok = true;
        if (gx < 0 || gx >= l.Lx) { if (l.px) gx = ((gx % l.Lx) + l.Lx) % l.Lx; else ok = false; }
        if (gy < 0 || gy >= l.Ly) { if (l.py) gy = ((gy % l.Ly) + l.Ly) % l.Ly; else ok = false; }
        d3 y = mk3(0.0, 0.0, 0.0);                     // absent neighbour (open boundary) contributes 0
        if (ok) {
            const long long j = (long long)gy * l.Lx + gx;
            y = ld3(x, j);
            if (TRIAL) {
                y = axpy3(a, ld3(d, j), y);
                y = scale3(1.0 / sqrt(dot3(y, y)), y);
            }
        }
        tile[ly][lx][0] = y.x; tile[ly][lx][1] = y.y; tile[ly][lx][2] = y.z;
    }
    __syncthreads();
    const int lx = threadIdx.x % RT_W, ly = threadIdx.x / RT_W;
    const int gx = tx0 + lx, gy = ty0 + ly;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    if (gx < l.Lx && gy < l.Ly) {
        const long long i = (long long)gy * l.Lx + gx;
        auto T = [&](int yy, int xx) { return mk3(tile[yy][xx][0], tile[yy][xx][1], tile[yy][xx][2]); };
        const d3 mi = T(ly + 1, lx + 1);
        // +-a1 = (+-1, 0), +-a2 = (0, +-1), +-(a2 - a1) = (-+1, +-1)
        const d3 Lm = stencil_apply(l, T(ly + 1, lx + 2), T(ly + 1, lx), T(ly + 2, lx + 1), T(ly, lx + 1), T(ly + 2, lx), T(ly, lx + 2), mi.z);
        const d3 B = mk3(l.mu * l.Bx, l.mu * l.By, l.mu * l.Bz);
        const d3 g = sub3(Lm, B);
        const d3 pg = axpy3(-dot3(mi, g), mi, g);
        acc[0] = 0.5 * dot3(mi, Lm) - dot3(mi, B);
        acc[1] = dot3(pg, pg);
        if (TRIAL) {
            acc[2] = dot3(pg, ld3(g_old, i));
            acc[3] = dot3(pg, ld3(d, i));
            st3(xt_out, i, mi);
        }
        st3(gt_out, i, pg);
    }
    block_sum<4>(acc, red);
    if (threadIdx.x == 0) {
        const size_t b = (size_t)blockIdx.y * gridDim.x + blockIdx.x;
        for (int j = 0; j < 4; ++j) partials[b * 4 + j] = acc[j];
    }
}

// out[j] = sum_b partials[b*4 + j], j < 4: 256 strided rows per value (coalesced), then a shared-memory tree; fixed order
__global__ void __launch_bounds__(1024) k_final_sum4(const double* __restrict__ partials, int nblk, double* __restrict__ out) {
    __shared__ double sm[1024];
    const int j = threadIdx.x & 3, r = threadIdx.x >> 2;
    double s = 0.0;
    for (int b = r; b < nblk; b += 256) s += partials[(size_t)b * 4 + j];
    sm[threadIdx.x] = s;
    __syncthreads();
    for (int off = 512; off >= 4; off >>= 1) {
        if (threadIdx.x < off) sm[threadIdx.x] += sm[threadIdx.x + off];
        __syncthreads();
    }
    if (threadIdx.x < 4) out[threadIdx.x] = sm[threadIdx.x];
}

// out[j] = sum_b partials[b*stride + j]  (optionally sqrt): one WARP per j (lanes stride over b, then a shuffle tree); fixed order.
// Launch with FS_GRID(nval) blocks of 256 threads.  (One thread per j took 17 us for 296 partials, 40 us for the 1607
// per-atom energies of the Cartesian path.)
#define FS_GRID(nval) (((nval) + 7) / 8)
__global__ void __launch_bounds__(256) k_final_sum(const double* __restrict__ partials, int nblk, int stride, int nval,
                                                   double* __restrict__ out, int take_sqrt) {
    const int j = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (j >= nval) return;
    double s = 0.0;
    for (int b = lane; b < nblk; b += 32) s += partials[(size_t)b * stride + j];
    s = warp_sum(s);
    if (lane == 0) out[j] = take_sqrt ? sqrt(s) : s;
}

// ---------------------------------------------------------------- block HVP, generic path
template <bool HAVE_C, bool PROJECT>
__global__ void __launch_bounds__(256) k_hvp_generic(Lat l, const double* __restrict__ m, const double* __restrict__ cvec,
                                                     const double* __restrict__ V, int k, double* __restrict__ HV,
                                                     const int* __restrict__ done) {
    if (done && *done) return;
    const long long N = (long long)l.Lx * l.Ly;
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= N) return;
    int iy = (int)(i / l.Lx), ix = (int)(i - (long long)iy * l.Lx);
    Nbrs n = neighbours(l, ix, iy);
    d3 mi = ld3(m, i);
    double c;
    if (HAVE_C) {
        c = cvec[i];
    } else {
        d3 Lm = stencil_field(l, m, n, mi.z);
        c = dot3(mi, Lm) - l.mu * (mi.x * l.Bx + mi.y * l.By + mi.z * l.Bz);
    }
    for (int a = 0; a < k; ++a) {
        const double* __restrict__ v = V + (size_t)a * 3 * N;
        d3 vi = ld3(v, i);
        d3 Lv;
        if (PROJECT) {
            vi = proj3(mi, vi);
            Lv = stencil_apply(l, ldnp(m, v, n.p1), ldnp(m, v, n.m1), ldnp(m, v, n.p2), ldnp(m, v, n.m2),
                               ldnp(m, v, n.p3), ldnp(m, v, n.m3), vi.z);
        } else {
            Lv = stencil_field(l, v, n, vi.z);
        }
        d3 h = axpy3(-c, vi, proj3(mi, Lv));
        st3(HV + (size_t)a * 3 * N, i, h);
    }
}

// three-term step on the generic path: out = alpha (Hess[v] - c0 v) + beta u, solver mode (c given, v tangent)
__global__ void __launch_bounds__(256) k_three_term_generic(Lat l, const double* __restrict__ m, const double* __restrict__ cvec,
                                                            const double* __restrict__ V, int k, double alpha, double c0, double beta,
                                                            const double* U, double* out) {
    const long long N = (long long)l.Lx * l.Ly;
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= N) return;
    int iy = (int)(i / l.Lx), ix = (int)(i - (long long)iy * l.Lx);
    Nbrs n = neighbours(l, ix, iy);
    d3 mi = ld3(m, i);
    const double c = cvec[i];
    for (int a = 0; a < k; ++a) {
        const double* __restrict__ v = V + (size_t)a * 3 * N;
        d3 vi = ld3(v, i);
        d3 h = axpy3(-c, vi, proj3(mi, stencil_field(l, v, n, vi.z)));
        d3 o = scale3(alpha, axpy3(-c0, vi, h));
        if (U) o = axpy3(beta, ld3(U + (size_t)a * 3 * N, i), o);
        st3(out + (size_t)a * 3 * N, i, o);
    }
}

// ---------------------------------------------------------------- tangent projection of a block, in place
__global__ void k_project(long long N, const double* __restrict__ m, double* __restrict__ V, int k) {
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= N) return;
    d3 mi = ld3(m, i);
    for (int a = 0; a < k; ++a) {
        double* v = V + (size_t)a * 3 * N;
        st3(v, i, proj3(mi, ld3(v, i)));
    }
}

// ---------------------------------------------------------------- K6 reflected-force step
// pass 1: F = -P g  -> gbuf ; partial dots alpha_a = F . v_a
__global__ void __launch_bounds__(256) k_mmf_pass1(Lat l, const double* __restrict__ m, const double* __restrict__ v, int kr,
                                                   double* __restrict__ Fbuf, double* __restrict__ partials,
                                                   double* __restrict__ alpha_out, unsigned* counter) {
    __shared__ double red[32 * MOTO_KMAX];
    const long long N = (long long)l.Lx * l.Ly;
    double acc[MOTO_KMAX];
#pragma unroll
    for (int a = 0; a < MOTO_KMAX; ++a) acc[a] = 0.0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        int iy = (int)(i / l.Lx), ix = (int)(i - (long long)iy * l.Lx);
        Nbrs n = neighbours(l, ix, iy);
        d3 mi = ld3(m, i);
        d3 Lm = stencil_field(l, m, n, mi.z);
        d3 g = sub3(Lm, mk3(l.mu * l.Bx, l.mu * l.By, l.mu * l.Bz));
        d3 F = scale3(-1.0, proj3(mi, g));
        st3(Fbuf, i, F);
#pragma unroll
        for (int a = 0; a < MOTO_KMAX; ++a)
            if (a < kr) acc[a] += dot3(F, ld3(v + (size_t)a * 3 * N, i));
    }
    block_sum<MOTO_KMAX>(acc, red);
    if (threadIdx.x == 0)
        for (int a = 0; a < MOTO_KMAX; ++a) partials[blockIdx.x * MOTO_KMAX + a] = acc[a];
    last_cta_sum(partials, MOTO_KMAX, MOTO_KMAX, alpha_out, 0, counter);   // alpha_a = F . v_a
}

// pass 2: F_mmf = F - 2 sum_a alpha_a v_a ; m' = normalize(m + dt F_mmf) ; partial |F_mmf|^2
// (m_out may alias m -- moto_mmf_step allows it -- so neither is __restrict__)
__global__ void __launch_bounds__(256) k_mmf_pass2(long long N, const double* m, const double* __restrict__ v, int kr,
                                                   const double* __restrict__ Fbuf, const double* __restrict__ alpha, double dt,
                                                   double* m_out, double* __restrict__ partials, int retract,
                                                   const uint8_t* __restrict__ fixed, double* __restrict__ F_out,
                                                   double* __restrict__ fnorm_out = nullptr, unsigned* counter = nullptr) {
    __shared__ double red[32];
    double al[MOTO_KMAX];
#pragma unroll
    for (int a = 0; a < MOTO_KMAX; ++a) al[a] = (a < kr) ? alpha[a] : 0.0;
    double f2[1] = {0.0};
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        d3 F = ld3(Fbuf, i);
#pragma unroll
        for (int a = 0; a < MOTO_KMAX; ++a)
            if (a < kr) F = axpy3(-2.0 * al[a], ld3(v + (size_t)a * 3 * N, i), F);
        if (fixed && fixed[i]) F = mk3(0.0, 0.0, 0.0);
        f2[0] += dot3(F, F);
        if (F_out) st3(F_out, i, F);          // the reflected force itself (moto_mmf_run_cg)
        d3 x = axpy3(dt, F, ld3(m, i));
        if (retract) x = scale3(1.0 / sqrt(dot3(x, x)), x);
        st3(m_out, i, x);
    }
    block_sum<1>(f2, red);
    if (threadIdx.x == 0) partials[blockIdx.x] = f2[0];
    last_cta_sum(partials, 1, 1, fnorm_out, 1, counter);   // |F_mmf|
}

}  // namespace

// ================================================================ host wrappers
// arrival counters of last_cta_sum: words 500.. of the flag block (512 words, zeroed at create; the K1 launches use < 148)
static unsigned* sum_counter(moto_ctx* c, int which) { return reinterpret_cast<unsigned*>(c->flags + 500 + which); }
int spin_energy_grad(moto_ctx* c, const double* m, double* d_E, double* d_g, double* d_c) {
    if (c->nsh > 0) return shell_energy_grad(c, m, d_E, d_g, d_c);
    const int nt = spin_energy_grad_tma(c, m, d_E, d_g, d_c);   // spin_stencil_tma.cu: where the TMA-staged kernel applies   // spin_stencil_tma.cu: where the TMA-staged kernel applies
    if (nt > 0) return nt;
    Lat l = make_lat(c);
    k_energy_grad<<<MOTO_RED_BLOCKS, 256, 0, c->stream>>>(l, m, d_g, d_c, c->partials, d_E, sum_counter(c, 1));
    return 1;
}

// d_out4 = {E_t, g_t.g_t, g_t.g, g_t.d} (device); d == nullptr: plain evaluation at x (out4[2], [3] = 0)
int spin_relax_eval(moto_ctx* c, const double* x, const double* d, double a, const double* g_old, double* xt, double* gt, double* d_out4) {
    if (c->nsh > 0) return 0;   // general shells: the one-site halo tile does not apply, caller takes the three-pass route
    Lat l = make_lat(c);
    dim3 grid((l.Lx + RT_W - 1) / RT_W, (l.Ly + RT_H - 1) / RT_H);
    if ((size_t)grid.x * grid.y * 4 > (size_t)MOTO_RED_BLOCKS * 2 * MOTO_NS * MOTO_NS || grid.y > 65535) return 0;   // partials capacity: caller takes the three-pass route
    if (d) k_relax_eval<true><<<grid, RT_W * RT_H, 0, c->stream>>>(l, x, d, a, g_old, xt, gt, c->partials);
    else k_relax_eval<false><<<grid, RT_W * RT_H, 0, c->stream>>>(l, x, nullptr, 0.0, nullptr, nullptr, gt, c->partials);
    k_final_sum4<<<1, 1024, 0, c->stream>>>(c->partials, (int)(grid.x * grid.y), d_out4);
    return 2;
}

// number of CTAs (= rows of partials) of the fused trial kernel, 0 if it does not apply to this context
int spin_relax_nblk(const moto_ctx* c) {
    if (c->kind != MOTO_KIND_TRI2D || c->nsh > 0) return 0;
    const long long gx = (c->lat.Lx + RT_W - 1) / RT_W, gy = (c->lat.Ly + RT_H - 1) / RT_H;
    if ((size_t)gx * gy * 4 > (size_t)MOTO_RED_BLOCKS * 2 * MOTO_NS * MOTO_NS || gy > 65535) return 0;
    return (int)(gx * gy);
}

int spin_relax_eval_dev(moto_ctx* c, const RelaxDev* rs, int* nblk_out) {
    if (c->nsh > 0) return 0;
    Lat l = make_lat(c);
    dim3 grid((l.Lx + RT_W - 1) / RT_W, (l.Ly + RT_H - 1) / RT_H);
    if ((size_t)grid.x * grid.y * 4 > (size_t)MOTO_RED_BLOCKS * 2 * MOTO_NS * MOTO_NS || grid.y > 65535) return 0;
    k_relax_eval<true><<<grid, RT_W * RT_H, 0, c->stream>>>(l, nullptr, nullptr, 0.0, nullptr, nullptr, nullptr, c->partials, rs);
    *nblk_out = (int)(grid.x * grid.y);
    return 1;
}

int spin_curvature(moto_ctx* c, const double* m, double* d_c) { return spin_energy_grad(c, m, nullptr, nullptr, d_c); }

int spin_hvp_tma(moto_ctx* c, const double* m, const double* cvec, const double* V, int k, double* HV,
                 int project_input, const int* d_done);  // spin_stencil_tma.cu; returns 0 if not applicable

int spin_hvp(moto_ctx* c, const double* m, const double* cvec, const double* V, int k, double* HV, int project_input,
             const int* d_done) {
    if (c->nsh > 0) return shell_hvp(c, m, cvec, V, k, HV, project_input, d_done);
    int n = spin_hvp_tma(c, m, cvec, V, k, HV, project_input, d_done);
    if (n > 0) return n;
    Lat l = make_lat(c);
    const long long N = c->N;
    const int blocks = (int)((N + 255) / 256);
    if (cvec) {
        if (project_input) k_hvp_generic<true, true><<<blocks, 256, 0, c->stream>>>(l, m, cvec, V, k, HV, d_done);
        else k_hvp_generic<true, false><<<blocks, 256, 0, c->stream>>>(l, m, cvec, V, k, HV, d_done);
    } else {
        if (project_input) k_hvp_generic<false, true><<<blocks, 256, 0, c->stream>>>(l, m, cvec, V, k, HV, d_done);
        else k_hvp_generic<false, false><<<blocks, 256, 0, c->stream>>>(l, m, cvec, V, k, HV, d_done);
    }
    return 1;
}

int spin_hvp_three_term_generic(moto_ctx* c, const double* m, const double* cvec, const double* V, int k, double alpha, double c0,
                                double beta, const double* U, double* out) {
    if (c->nsh > 0) return shell_three_term(c, m, cvec, V, k, alpha, c0, beta, U, out);
    Lat l = make_lat(c);
    const long long N = c->N;
    k_three_term_generic<<<(int)((N + 255) / 256), 256, 0, c->stream>>>(l, m, cvec, V, k, alpha, c0, beta, U, out);
    return 1;
}

int spin_project(moto_ctx* c, const double* m, double* V, int k) {
    const long long N = c->N;
    k_project<<<(int)((N + 255) / 256), 256, 0, c->stream>>>(N, m, V, k);
    return 1;
}

int spin_mmf_step(moto_ctx* c, const double* m, const double* v, int kr, double dt, double* m_out, double* d_fnorm) {
    Lat l = make_lat(c);
    double* alpha = c->st->scal;  // [KMAX] would overflow scal[8]? KMAX == 8: exactly fits
    int n = 0;
    if (c->nsh > 0) {
        n += shell_mmf_pass1(c, m, v, kr);
        k_final_sum<<<FS_GRID(MOTO_KMAX), 256, 0, c->stream>>>(c->partials, MOTO_RED_BLOCKS, MOTO_KMAX, MOTO_KMAX, alpha, 0); ++n;
    } else if (kr == 1 && spin_mmf_pass1_tma(c, m, v, c->g, alpha) > 0) {
        ++n;   // large lattices: F = -P g and alpha_1 = F . v_1 from the TMA-staged kernel
    } else {
        k_mmf_pass1<<<MOTO_RED_BLOCKS, 256, 0, c->stream>>>(l, m, v, kr, c->g, c->partials, alpha, sum_counter(c, 2)); ++n;
    }
    // |F_mmf| of the current state comes out of pass 2 itself (the CTA that finishes last takes the square root of the sum)
    // (four CTAs per SM: 10^6 spins 51.7 -> 46.6 us per moto_mmf_step; 8 or 16 per SM are slower again)
    k_mmf_pass2<<<2 * MOTO_RED_BLOCKS, 256, 0, c->stream>>>((long long)c->N, m, v, kr, c->g, alpha, dt, m_out, c->partials, 1, nullptr, c->fmmf_out,
                                                      d_fnorm, sum_counter(c, 3));
    return n + 1;
}

// shared with cart_morse.cu (declared there as extern)
void launch_mmf_pass2(moto_ctx* c, const double* x, const double* v, int kr, const double* Fbuf, const double* alpha,
                      double dt, double* x_out, int retract) {
    k_mmf_pass2<<<MOTO_RED_BLOCKS, 256, 0, c->stream>>>((long long)c->N, x, v, kr, Fbuf, alpha, dt, x_out, c->partials, retract,
                                                      c->lat.d_fixed, c->fmmf_out);
}
void launch_final_sum(moto_ctx* c, const double* partials, int nblk, int stride, int nval, double* out, int take_sqrt) {
    k_final_sum<<<FS_GRID(nval), 256, 0, c->stream>>>(partials, nblk, stride, nval, out, take_sqrt);
}
