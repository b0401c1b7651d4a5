// spin_shells_dense.cu -- K1 for general neighbour shells as a register-blocked direct convolution (Eq. 4,
// PAPER.md:136-138; the paper's ~340-neighbour Pd/Fe/Ir(111) workload class, Tables I/II PAPER.md:328-616).
//   (L u)_i = -2 sum_delta [ J_delta u_{i+delta} + u_{i+delta} x D_delta ] - 2 K u_iz z,   Hess[v]_i = P_i (L Pv)_i - c_i (Pv)_i
// With 366 taps per site the step is bound by the fp64 pipe, not by HBM: 9 DFMA per tap and field, 3.6 us of DFMA issue for
// a block of two on 10^4 sites.  k_shell_hvp (spin_shells.cu: a warp per site, a lane per tap) pays for every tap with its
// own neighbour load, its own index arithmetic and its own table read -- 46 us.  Here
//   * the table is stored as dense SEGMENTS of one dx column each (<= 12 consecutive dy, holes zero-filled, two zero entries
//     after each segment so that the tap loop needs no bound test);
//   * a thread owns R = 2 or 3 output sites (x, y .. y + R - 1) and walks a segment down its column: the value read at row r
//     serves tap (dx, r - y - o) of output row o -- 9 R DFMA per 24 bytes read, the last R table entries stay in registers;
//   * a CTA owns 32 consecutive columns-of-R in flattened (row group, x) order (every lane works whatever Lx is) and first
//     STAGES the fields it needs (its rows and columns + the halo of the table) in shared memory, boundary conditions and,
//     in API mode, the projection of the neighbours applied there once per site: the staging loads are independent and all
//     in flight at once, the tap loop has no index arithmetic, no branch and no global load, lanes read consecutive
//     24-byte sites (conflict-free), the table entry is a broadcast read;
//   * warp (g, f) of a CTA accumulates tap group g (balanced on the host) of staged field f; the partial sums meet in shared
//     memory in a fixed order (bit-identical reruns) and the first R warps apply the epilogue (projection, -c v, optional
//     three-term recurrence);
//   * R is picked per lattice so that the fullest SM gets the least work (100 x 100: R = 3, 107 CTAs, one per SM).
// Measured at 100 x 100 / 366 taps (B200): moto_hvp k = 2 46 -> 22.6-24.6 us, solver mode 18.5 us; at 316 x 316 90 us
// (solver mode, k = 2: 40 % of the fp64 peak).  The DFMA pipe is 42 % busy over the kernel (ncu, solver mode): 107 of 148
// SMs have a CTA, ~8 us of the 18.5 are launch, staging, reduction and epilogue.
// Tensor cores are not used: the contraction has 3 output columns per site (fp64 DMMA would run at 3/8 fill at best and has
// no rate advantage over DFMA on this part).  Falls back to spin_shells.cu for k > 2, Lx < 32 or tables that do not fit.
#include <algorithm>
#include <vector>
#include <string.h>
#include "common.cuh"
#include "device_utils.cuh"
#include "stencil_math.cuh"
#include "tma_utils.cuh"   // ensure_smem_attr

namespace {

constexpr int SEGMAX = 12;      // taps per segment

struct DenseTab { int nseg, nd; const int* seg; const double* jd; int grp[MOTO_SH_GROUPS + 1]; };

struct T4 { double J, Dx, Dy, Dz; };

// acc += J v + v x D
__device__ __forceinline__ void tap_accum(d3& acc, const T4& t, const d3& v) {
    acc.x = fma(t.J, v.x, acc.x); acc.x = fma(v.y, t.Dz, acc.x); acc.x = fma(-v.z, t.Dy, acc.x);
    acc.y = fma(t.J, v.y, acc.y); acc.y = fma(v.z, t.Dx, acc.y); acc.y = fma(-v.x, t.Dz, acc.y);
    acc.z = fma(t.J, v.z, acc.z); acc.z = fma(v.x, t.Dy, acc.z); acc.z = fma(-v.y, t.Dx, acc.z);
}

__device__ __forceinline__ int wrap(int j, int L) {   // j mod L for any int
    if (j >= 0 && j < L) return j;
    j %= L;
    return j < 0 ? j + L : j;
}

// PROJECT: API mode (neighbours projected).  NEEDC: c from the same pass over m.  CHEB: out = alpha (Hess[v] - c0 v) + beta u.
// R: output rows per thread (2 or 3; the host picks the one that leaves the fullest SM with the least work).
//
// A CTA owns 32 consecutive output COLUMNS-OF-R of the flattened (row group, x) order -- at most two runs, A in row group ygA
// and B at the start of row group ygA + 1 -- and first stages, for each run, the fields over rows [R yg - Hy, R yg + R - 1 + Hy]
// and columns [x0 - Hx, x0 + cnt - 1 + Hx] into shared memory with the boundary handled there (periodic wrap, zeros beyond an
// open edge, neighbours projected once per site in API mode): every load of the staging loop is independent and in flight
// at once, and the tap loop that follows has no index arithmetic, no branch and no global load.
// Warp (g, f) of the S x NF warps accumulates tap group g of field f (the k directions, and m when c is wanted).
// GRAD (KT = 0, NEEDC): the only staged field is m; the epilogue writes the tangent-projected gradient to HV (if given), c_i to
// c_out (if given) and the CTA's energy partial sum_i (m_i.(Lm)_i / 2 - m_i.muB) to e_part[blockIdx.x].
template <bool PROJECT, bool NEEDC, bool CHEB, int KT, int R, bool GRAD = false>
__global__ void __launch_bounds__(768) k_shell_dense(Lat l, DenseTab tb, int Hx, int Hy, const double* __restrict__ m,
                                                     const double* __restrict__ cvec, const double* __restrict__ V,
                                                     double* __restrict__ HV, const int* __restrict__ done,
                                                     double alpha, double c0, double beta, const double* U, const double* __restrict__ d_coef,
                                                     double* __restrict__ c_out, double* __restrict__ e_part) {
    static_assert(!GRAD || (KT == 0 && NEEDC && !PROJECT && !CHEB), "GRAD: m only");
    constexpr int NF = KT + (NEEDC ? 1 : 0);     // staged / accumulated fields: the KT directions (+ m)
    constexpr int NV = NF * R * 3;               // sums per lane
    extern __shared__ double smem[];
    // programmatic dependent launch: the next launch of the recurrence may start on free SMs right away and stage its copy of the
    // coupling table (constant since moto_set_shells) while this one still runs; it reads nothing this launch writes -- the done flag,
    // the fields, the coefficients -- before its own griddepcontrol.wait below
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, S = (blockDim.x >> 5) / NF;
    const int grp = warp / NF, fld = warp - grp * NF;
    const int nent = tb.nd + 2 * tb.nseg;                            // the host puts two zero entries after every segment
    double* sjd = smem;                                              // [nent][4]
    int* sseg = reinterpret_cast<int*>(sjd + 4 * nent);              // [nseg][4]
    int* sgrp = sseg + 4 * tb.nseg;                                  // [MOTO_SH_GROUPS + 2]
    double* sreg = sjd + 4 * nent + 2 * tb.nseg + (MOTO_SH_GROUPS + 2) / 2;   // staged fields [NF][sites][3]; later the partial sums
    for (int t = threadIdx.x; t < 4 * nent; t += blockDim.x) sjd[t] = tb.jd[t];
    for (int t = threadIdx.x; t < 4 * tb.nseg; t += blockDim.x) sseg[t] = tb.seg[t];
    if (threadIdx.x <= MOTO_SH_GROUPS) sgrp[threadIdx.x] = tb.grp[threadIdx.x];   // (the table of this launch's S)
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (done && *done) return;

    const int Lx = l.Lx, Ly = l.Ly;
    const long long N = (long long)Lx * Ly;
    const int nyg = (Ly + R - 1) / R;                                // row groups
    const long long ncols = (long long)nyg * Lx;
    const long long p0 = (long long)blockIdx.x * 32;
    const int ygA = (int)(p0 / Lx), xA = (int)(p0 - (long long)ygA * Lx);
    const int nA = Lx - xA < 32 ? Lx - xA : 32;                      // run A: x = xA .. xA + nA - 1 of row group ygA
    int nB = 32 - nA;                                                // run B: x = 0 .. nB - 1 of row group ygA + 1
    if (ygA + 1 >= nyg) nB = 0;
    const int RH = R + 2 * Hy, wA = nA + 2 * Hx, wB = nB > 0 ? nB + 2 * Hx : 0;
    const int sitesA = wA * RH, sites = sitesA + wB * RH;
    const size_t fstr = (size_t)sites * 3;                           // field stride in doubles

    // ------------------------------------------------------------ staging
    for (int s = threadIdx.x; s < sites; s += blockDim.x) {
        const bool inB = s >= sitesA;
        const int q = inB ? s - sitesA : s, w = inB ? wB : wA;
        const int r = q / w, cx = q - r * w;
        int gx = (inB ? 0 : xA) - Hx + cx, gy = R * (inB ? ygA + 1 : ygA) - Hy + r;
        bool ok = true;
        if (gx < 0 || gx >= Lx) { if (l.px) gx = wrap(gx, Lx); else ok = false; }
        if (gy < 0 || gy >= Ly) { if (l.py) gy = wrap(gy, Ly); else ok = false; }
        d3 mj = mk3(0.0, 0.0, 0.0), vj[KT > 0 ? KT : 1];
#pragma unroll
        for (int a = 0; a < KT; ++a) vj[a] = mk3(0.0, 0.0, 0.0);
        if (ok) {
            const long long j = (long long)gy * Lx + gx;
            if (PROJECT || NEEDC) mj = ld3(m, j);
#pragma unroll
            for (int a = 0; a < KT; ++a) {
                vj[a] = ld3(V + (size_t)a * 3 * N, j);
                if (PROJECT) vj[a] = proj3(mj, vj[a]);
            }
        }
#pragma unroll
        for (int a = 0; a < KT; ++a) { double* d = sreg + a * fstr + 3 * (size_t)s; d[0] = vj[a].x; d[1] = vj[a].y; d[2] = vj[a].z; }
        if (NEEDC) { double* d = sreg + KT * fstr + 3 * (size_t)s; d[0] = mj.x; d[1] = mj.y; d[2] = mj.z; }
    }
    __syncthreads();

    // ------------------------------------------------------------ taps
    const bool active = p0 + lane < ncols && lane < nA + nB;
    const bool laneB = lane >= nA;
    const int pitch = 3 * (laneB ? wB : wA);                                          // doubles per staged row of this lane's run
    const int origin = 3 * ((laneB ? sitesA + (lane - nA) : lane) + Hx) + Hy * pitch;  // this lane's first output site
    d3 acc[R];
#pragma unroll
    for (int o = 0; o < R; ++o) acc[o] = mk3(0.0, 0.0, 0.0);
    if (active && grp < S) {
        for (int sg = sgrp[grp]; sg < sgrp[grp + 1]; ++sg) {
            const int dx = sseg[4 * sg], dy0 = sseg[4 * sg + 1], n = sseg[4 * sg + 2];
            const double* te = sjd + 4 * (sseg[4 * sg + 3] + 2 * sg);                 // + 2 sg: the zero entries of the segments before
            const double* pv = sreg + fld * fstr + origin + dy0 * pitch + 3 * dx;
            // the value at row y0 + dy0 + t serves tap dy0 + t - o of output row o: a window of the last R table entries
            // (zero before the segment's first and after its last tap)
            T4 win[R];
#pragma unroll
            for (int o = 0; o < R; ++o) win[o] = T4{0.0, 0.0, 0.0, 0.0};
#pragma unroll 4
            for (int t = 0; t < n + R - 1; ++t) {
#pragma unroll
                for (int o = R - 1; o > 0; --o) win[o] = win[o - 1];
                win[0] = T4{te[4 * t], te[4 * t + 1], te[4 * t + 2], te[4 * t + 3]};   // t >= n: the zero entries after the segment
                const d3 v = mk3(pv[0], pv[1], pv[2]);
#pragma unroll
                for (int o = 0; o < R; ++o) { acc[o].x = fma(win[o].J, v.x, acc[o].x); acc[o].y = fma(win[o].J, v.y, acc[o].y); acc[o].z = fma(win[o].J, v.z, acc[o].z); }
#pragma unroll
                for (int o = 0; o < R; ++o) { acc[o].x = fma(v.y, win[o].Dz, acc[o].x); acc[o].y = fma(v.z, win[o].Dx, acc[o].y); acc[o].z = fma(v.x, win[o].Dy, acc[o].z); }
#pragma unroll
                for (int o = 0; o < R; ++o) { acc[o].x = fma(-v.z, win[o].Dy, acc[o].x); acc[o].y = fma(-v.x, win[o].Dz, acc[o].y); acc[o].z = fma(-v.y, win[o].Dx, acc[o].z); }
                pv += pitch;
            }
        }
    }
    __syncthreads();                             // every warp is done with the staged fields: the partial sums take their place

    // partial sums [S][NV][32] -> shared memory, summed in group order
    double* spart = sreg;
    if (grp < S) {
        double* mine = spart + ((size_t)grp * NV + (size_t)fld * R * 3) * 32;
#pragma unroll
        for (int o = 0; o < R; ++o) { mine[(o * 3 + 0) * 32 + lane] = acc[o].x; mine[(o * 3 + 1) * 32 + lane] = acc[o].y; mine[(o * 3 + 2) * 32 + lane] = acc[o].z; }
    }
    __syncthreads();
    for (int e = threadIdx.x; e < NV * 32; e += blockDim.x) {
        double s = 0.0;
        for (int w = 0; w < S; ++w) s += spart[(size_t)w * NV * 32 + e];
        spart[e] = s;                            // entry e of group 0 is read by this thread only
    }
    __syncthreads();
    if (GRAD) {   // energy / gradient epilogue: warp o finishes output row o, the CTA's energy partial in warp order
        double e = 0.0;
        const int yg = laneB ? ygA + 1 : ygA, x = laneB ? lane - nA : xA + lane, y = R * yg + warp;
        if (warp < R && active && y < Ly) {
            const d3 B = mk3(l.mu * l.Bx, l.mu * l.By, l.mu * l.Bz);
            const long long i = (long long)y * Lx + x;
            const d3 mi = ld3(m, i);
            const double* sm = spart + (warp * 3) * 32 + lane;
            const d3 Lm = mk3(-2.0 * sm[0], -2.0 * sm[32], -2.0 * sm[64] - 2.0 * l.K * mi.z);
            const d3 g = sub3(Lm, B);
            const double c = dot3(mi, g);
            e = 0.5 * dot3(mi, Lm) - dot3(mi, B);
            if (HV) st3(HV, i, axpy3(-c, mi, g));
            if (c_out) c_out[i] = c;
        }
        double* sred = spart + NV * 32;          // beyond the summed entries (the region holds S NV 32 >= NV 32 + R doubles)
        if (warp < R) { e = warp_sum(e); if (lane == 0) sred[warp] = e; }
        __syncthreads();
        if (threadIdx.x == 0 && e_part) { double t = 0.0; for (int o = 0; o < R; ++o) t += sred[o]; e_part[blockIdx.x] = t; }
        return;
    }
    // epilogue: warp o finishes output row o of the 32 columns
    if (warp >= R || !active) return;
    const int yg = laneB ? ygA + 1 : ygA, x = laneB ? lane - nA : xA + lane, y = R * yg + warp;
    if (y >= Ly) return;
    const d3 B = mk3(l.mu * l.Bx, l.mu * l.By, l.mu * l.Bz);
    const long long i = (long long)y * Lx + x;
    const d3 mi = ld3(m, i);
    double c;
    if (NEEDC) {
        const double* sm = spart + ((KT * R + warp) * 3) * 32 + lane;
        const d3 Lm = mk3(-2.0 * sm[0], -2.0 * sm[32], -2.0 * sm[64] - 2.0 * l.K * mi.z);
        c = dot3(mi, Lm) - dot3(mi, B);
    } else {
        c = cvec[i];
    }
#pragma unroll
    for (int a = 0; a < KT; ++a) {
        const size_t ofs = (size_t)a * 3 * N;
        d3 vi = ld3(V + ofs, i);
        if (PROJECT) vi = proj3(mi, vi);
        const double* sa = spart + ((a * R + warp) * 3) * 32 + lane;
        const d3 Lv = mk3(-2.0 * sa[0], -2.0 * sa[32], -2.0 * sa[64] - 2.0 * l.K * vi.z);
        d3 h = axpy3(-c, vi, proj3(mi, Lv));
        if (CHEB) {
            if (d_coef) { alpha = d_coef[0]; c0 = d_coef[1]; beta = d_coef[2]; }   // coefficients computed on the device (k_cheb_coef)
            h = scale3(alpha, axpy3(-c0, vi, h));
            if (U) h = axpy3(beta, ld3(U + ofs, i), h);
        }
        st3(HV + ofs, i, h);
    }
}

DenseTab dense_of(const moto_ctx* c, int variant) {
    DenseTab t; t.nseg = c->sh_nseg; t.nd = c->sh_nd; t.seg = c->sh_seg; t.jd = c->sh_jd2;
    for (int s = 0; s <= MOTO_SH_GROUPS; ++s) t.grp[s] = c->sh_grp[variant][s];
    return t;
}

}  // namespace

// host side of moto_set_shells for this kernel: the table as dense column segments + balanced tap groups.
// h_jd [n][4] = J, Dx, Dy, Dz per offset.  Leaves sh_nseg = 0 (kernel not available) when the dense form does not fit.
moto_status shell_dense_build(moto_ctx* c, int n, const int32_t* h_off, const double* h_jd) {
    c->sh_nseg = 0; c->sh_nd = 0;
    if (n <= 0) return MOTO_OK;
    std::vector<int> order(n);
    for (int t = 0; t < n; ++t) order[t] = t;
    std::sort(order.begin(), order.end(), [&](int a, int b) {
        return h_off[2 * a] != h_off[2 * b] ? h_off[2 * a] < h_off[2 * b] : h_off[2 * a + 1] < h_off[2 * b + 1];
    });
    std::vector<int> seg;          // dx, dy0, n, first entry
    std::vector<double> jd;        // dense entries
    for (int b = 0; b < n;) {
        int e = b;
        while (e < n && h_off[2 * order[e]] == h_off[2 * order[b]]) ++e;
        const int dx = h_off[2 * order[b]], lo = h_off[2 * order[b] + 1], hi = h_off[2 * order[e - 1] + 1];
        const long long len = (long long)hi - lo + 1;
        if ((long long)jd.size() / 4 + len > MOTO_SH_DENSE) return MOTO_OK;      // too sparse / too large for the dense form
        const size_t first = jd.size() / 4;
        jd.resize(jd.size() + 4 * (size_t)len, 0.0);
        for (int q = b; q < e; ++q) {
            const int t = order[q], r = h_off[2 * t + 1] - lo;
            for (int z = 0; z < 4; ++z) jd[4 * (first + r) + z] = h_jd[4 * t + z];
        }
        const int parts = (int)((len + SEGMAX - 1) / SEGMAX);
        for (int q = 0; q < parts; ++q) {
            const int s0 = (int)(len * q / parts), s1 = (int)(len * (q + 1) / parts);
            seg.push_back(dx); seg.push_back(lo + s0); seg.push_back(s1 - s0); seg.push_back((int)first + s0);
        }
        b = e;
    }
    const int nseg = (int)seg.size() / 4;
    if (nseg > MOTO_SH_SEGS) return MOTO_OK;
    // tap groups: contiguous runs of segments, cost of a segment = its n + 2 row loads; one table per group count (the launch
    // takes 16 groups for one staged field, 12 for two, 8 for three: at most 24 warps per CTA).  Segment q goes to group
    // floor((cost before q + half its own) S / total): contiguous, balanced to within one segment
    long long total = 0;
    for (int q = 0; q < nseg; ++q) total += seg[4 * q + 2] + 2;
    const int Ss[3] = {8, 12, 16};
    for (int v = 0; v < 3; ++v) {
        const int S = Ss[v];
        int* grp = c->sh_grp[v];
        for (int s2 = 0; s2 <= MOTO_SH_GROUPS; ++s2) grp[s2] = nseg;
        long long cum = 0;
        for (int q = 0; q < nseg; ++q) {
            const long long w = seg[4 * q + 2] + 2;
            int g = (int)((2 * cum + w) * S / (2 * total));
            if (g > S - 1) g = S - 1;
            for (int s2 = 0; s2 <= g; ++s2) if (grp[s2] > q) grp[s2] = q;
            cum += w;
        }
    }
    // device table: the entries of segment q followed by two zero entries (the R - 1 <= 2 rows below the segment's last tap serve
    // the later output rows only), so that the tap loop needs no bound test
    const int nd = (int)(jd.size() / 4);
    if (nd + 2 * nseg > MOTO_SH_DENSE) return MOTO_OK;
    std::vector<double> jd2;
    jd2.reserve(4 * (size_t)(nd + 2 * nseg));
    int Hx = 0, Hy = 0;
    for (int q = 0; q < nseg; ++q) {
        const int first = seg[4 * q + 3], len = seg[4 * q + 2];
        jd2.insert(jd2.end(), jd.begin() + 4 * (size_t)first, jd.begin() + 4 * (size_t)(first + len));
        jd2.insert(jd2.end(), 8, 0.0);
        Hx = std::max(Hx, std::abs(seg[4 * q]));
        Hy = std::max(Hy, std::max(std::abs(seg[4 * q + 1]), std::abs(seg[4 * q + 1] + len - 1)));
    }
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(c->sh_seg, seg.data(), seg.size() * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    MOTO_CUDA_CHECK(c, cudaMemcpyAsync(c->sh_jd2, jd2.data(), jd2.size() * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    MOTO_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));    // seg / jd2 are host temporaries
    c->sh_nseg = nseg; c->sh_nd = nd; c->sh_Hx = Hx; c->sh_Hy = Hy;
    return MOTO_OK;
}

// 1 launch, or 0 when this kernel does not apply (k > 2, no dense table): the caller falls back to k_shell_hvp
int shell_dense_hvp(moto_ctx* c, const double* m, const double* cvec, const double* V, int k, double* HV, int project_input, const int* d_done,
                    int cheb, double alpha, double c0, double beta, const double* U, const double* d_coef) {
    if (c->sh_nseg <= 0 || k < 1 || k > 2 || c->lat.Lx < 32) return 0;
    const int Hx = c->sh_Hx, Hy = c->sh_Hy;
    const bool needc = cvec == nullptr;
    const int nf = k + (needc ? 1 : 0);
    const int variant = nf == 1 ? 2 : (nf == 2 ? 1 : 0), S = nf == 1 ? 16 : (nf == 2 ? 12 : 8);
    int sms = MOTO_NUM_SMS;
    // rows per thread: the fullest SM gets ceil(CTAs / SMs) CTAs of R rows each -- take the R with the least of that
    auto ctas = [&](int R) { return (long long)(((long long)((c->lat.Ly + R - 1) / R) * c->lat.Lx + 31) / 32); };
    const long long w2 = ((ctas(2) + sms - 1) / sms) * 2, w3 = ((ctas(3) + sms - 1) / sms) * 3;
    const int R = w3 < w2 ? 3 : 2;
    const int grid = (int)ctas(R);
    const size_t region = (size_t)nf * (32 + 4 * Hx) * (R + 2 * Hy) * 3, part = (size_t)S * nf * R * 3 * 32;   // doubles
    const size_t smem = ((size_t)4 * (c->sh_nd + 2 * c->sh_nseg) + 2 * c->sh_nseg + (MOTO_SH_GROUPS + 2) / 2 + std::max(region, part)) * sizeof(double);
    if (smem > 200 * 1024) return 0;
    const Lat l = make_lat(c);
    const DenseTab tb = dense_of(c, variant);
#define DENSE_R(P, NC, CH, KT, RR)                                                                                        \
    do {                                                                                                                   \
        static std::atomic<unsigned long long> seen{0};                                                                    \
        if (smem > 48 * 1024 && !tma::ensure_smem_attr(k_shell_dense<P, NC, CH, KT, RR>, 200 * 1024, seen)) return 0;      \
        cudaLaunchConfig_t cfg;                                                                                            \
        memset(&cfg, 0, sizeof(cfg));                                                                                      \
        cfg.gridDim = dim3(grid); cfg.blockDim = dim3(32 * S * nf); cfg.dynamicSmemBytes = smem; cfg.stream = c->stream;   \
        cudaLaunchAttribute attr[1];                                                                                       \
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;                                                   \
        attr[0].val.programmaticStreamSerializationAllowed = 1;                                                            \
        cfg.attrs = attr; cfg.numAttrs = 1;                                                                                \
        double* const np_ = nullptr;                                                                                       \
        if (cudaLaunchKernelEx(&cfg, k_shell_dense<P, NC, CH, KT, RR>, l, tb, Hx, Hy, m, cvec, V, HV, d_done, alpha, c0, beta, U, d_coef, np_, np_) != cudaSuccess) { \
            (void)cudaGetLastError();                                                                                      \
            k_shell_dense<P, NC, CH, KT, RR><<<grid, 32 * S * nf, smem, c->stream>>>(l, tb, Hx, Hy, m, cvec, V, HV, d_done, alpha, c0, beta, U, d_coef, nullptr, nullptr); \
        }                                                                                                                  \
    } while (0)
#define DENSE(P, NC, CH, KT) do { if (R == 3) DENSE_R(P, NC, CH, KT, 3); else DENSE_R(P, NC, CH, KT, 2); } while (0)
    if (cheb) { if (k == 1) DENSE(false, false, true, 1); else DENSE(false, false, true, 2); }
    else if (project_input && needc) { if (k == 1) DENSE(true, true, false, 1); else DENSE(true, true, false, 2); }
    else if (project_input) { if (k == 1) DENSE(true, false, false, 1); else DENSE(true, false, false, 2); }
    else if (needc) { if (k == 1) DENSE(false, true, false, 1); else DENSE(false, true, false, 2); }
    else { if (k == 1) DENSE(false, false, false, 1); else DENSE(false, false, false, 2); }
#undef DENSE
#undef DENSE_R
    return 1;
}

bool shell_dense_applicable(const moto_ctx* c, int k) { return c->nsh > 0 && c->sh_nseg > 0 && k >= 1 && k <= 2 && c->lat.Lx >= 32; }

// OUT = Y_d of the three-term recurrence Y_i = alpha_i (Hess[Y_{i-1}] - c0 Y_{i-1}) + beta_i Y_{i-2}, Y_0 = V (tangent), with the
// coefficients d_coef [d][4] on the device: d launches of k_shell_dense, Y_i alternating between T1 and T2 (a step writes over
// its own three-term operand, which it touches at the thread's own site only).  -1: not applicable.
int shell_cheb_recurrence(moto_ctx* c, const double* m, const double* cvec, const double* V, int k, int d, double* OUT,
                          const double* d_coef, const int* d_done) {
    if (!shell_dense_applicable(c, k) || !cvec || !c->T1 || !c->T2) return -1;
    int n = 0;
    const double* in = V; const double* prev = nullptr;
    for (int i = 1; i <= d; ++i) {
        double* out = (i == d) ? OUT : ((i & 1) ? c->T1 : c->T2);
        const int n1 = shell_dense_hvp(c, m, cvec, in, k, out, 0, d_done, 1, 0.0, 0.0, 0.0, prev, d_coef + 4 * (i - 1));
        if (n1 <= 0) return -1;
        n += n1;
        prev = in; in = out;
    }
    return n;
}

// energy partials (one per CTA, to e_part; *grid_out = their number), tangent-projected gradient (d_g, may be NULL) and c (d_c,
// may be NULL) in one launch of the dense kernel with m as the only staged field.  0: not applicable, the caller falls back.
int shell_dense_energy_grad(moto_ctx* c, const double* m, double* d_g, double* d_c, double* e_part, int* grid_out) {
    if (c->nsh <= 0 || c->sh_nseg <= 0 || c->lat.Lx < 32) return 0;
    const int Hx = c->sh_Hx, Hy = c->sh_Hy, S = 16, sms = MOTO_NUM_SMS;
    auto ctas = [&](int R) { return (long long)(((long long)((c->lat.Ly + R - 1) / R) * c->lat.Lx + 31) / 32); };
    const long long w2 = ((ctas(2) + sms - 1) / sms) * 2, w3 = ((ctas(3) + sms - 1) / sms) * 3;
    const int R = w3 < w2 ? 3 : 2;
    const int grid = (int)ctas(R);
    if (grid > MOTO_RED_BLOCKS * 2 * MOTO_NS * MOTO_NS) return 0;   // e_part is the context's partials array
    const size_t region = (size_t)(32 + 4 * Hx) * (R + 2 * Hy) * 3, part = (size_t)S * R * 3 * 32 + 8;   // doubles
    const size_t smem = ((size_t)4 * (c->sh_nd + 2 * c->sh_nseg) + 2 * c->sh_nseg + (MOTO_SH_GROUPS + 2) / 2 + std::max(region, part)) * sizeof(double);
    if (smem > 200 * 1024) return 0;
    const Lat l = make_lat(c);
    const DenseTab tb = dense_of(c, 2);
    static std::atomic<unsigned long long> seen2{0}, seen3{0};
    if (R == 3) {
        if (smem > 48 * 1024 && !tma::ensure_smem_attr(k_shell_dense<false, true, false, 0, 3, true>, 200 * 1024, seen3)) return 0;
        k_shell_dense<false, true, false, 0, 3, true><<<grid, 32 * S, smem, c->stream>>>(l, tb, Hx, Hy, m, nullptr, nullptr, d_g, nullptr, 0.0, 0.0, 0.0,
                                                                                         nullptr, nullptr, d_c, e_part);
    } else {
        if (smem > 48 * 1024 && !tma::ensure_smem_attr(k_shell_dense<false, true, false, 0, 2, true>, 200 * 1024, seen2)) return 0;
        k_shell_dense<false, true, false, 0, 2, true><<<grid, 32 * S, smem, c->stream>>>(l, tb, Hx, Hy, m, nullptr, nullptr, d_g, nullptr, 0.0, 0.0, 0.0,
                                                                                         nullptr, nullptr, d_c, e_part);
    }
    *grid_out = grid;
    return 1;
}
