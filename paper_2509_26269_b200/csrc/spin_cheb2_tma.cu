// spin_cheb2_tma.cu -- K1 with temporal blocking: TWO steps of the filter recurrence per pass over the lattice (the operator
// application of the transformed solver, lobpcg.cu; Eq. 4, Hv PAPER.md:156, :162).  The default launch of the
// recurrence (moto_solver_opts.cheb_mode 0 = 3).
//
//   Y_i = alpha_i (Hess[Y_{i-1}] - r_i Y_{i-1}) [+ beta_i Y_{i-2}],   Hess[v]_i = P_i (L v)_i - c_i v_i   (solver mode, v tangent)
//
// The library applies the filter in product form over its Leja-ordered roots (k_cheb_coef, lobpcg_fast.cu): beta_i = 0, so a
// step needs Y_{i-1} only.  spin_stencil_tma.cu runs one such step per pass: 128 B/site/step at k = 2 (m, c, Y_{i-1} in, Y_i out)
// and one neighbour synchronisation per step.  Here a pass stages m, c and Y_{i-1} with a TWO-site halo (the 64-site TMA row
// box of a <= 60-site strip already holds it), computes
//   phase A   Z = Y_i      on the strip plus a one-site halo ring   (written to the Z ring in shared memory only)
//   phase B   Y_{i+1}      on the strip from Z (shared memory)
// so that m, c and Y_{i-1} cross the memory system once per two steps and Y_i never leaves the SM: (24 + 8 + 48 k) in + 48 k out
// = 128 B/site per TWO steps at k = 2, and the CTAs synchronise with their halo partners once per pass.  The halo ring is
// computed redundantly by both neighbours with the same arithmetic on the same inputs (bit-identical values), so the result
// equals the step-by-step recurrence bit for bit.  The template flag PF = false keeps the general three-term step (beta != 0:
// Y_{i-2} read from global memory as flat row segments and transposed through shared memory, Y_i also written out because the
// next pass needs it as its third operand, four rotating blocks: 224 B/site per two steps) -- the launch the library used
// before the product form; nothing in the library requests it any more.
// Measured at 10^6 spins, k = 2 (B200): 22.2 us/step (one step per pass: 24.1); bound by the ten consumer warps, not by DRAM.
//
// Same skeleton as spin_stencil_tma.cu: persistent grid (one CTA per SM), column strips, one producer warp issuing
// cp.async.bulk.tensor boxes into a ring of row slots guarded by full/empty mbarriers, ten consumer warps (2 column
// halves x 5 row pairs, two rows per thread), even passes swept bottom-up on the point-reflected lattice for L2 reuse,
// release/acquire flags between halo partners.  Tensor cores are not used: a 7-point fp64 stencil, HBM/L2-bound.
#include "common.cuh"
#include "device_utils.cuh"
#include "stencil_math.cuh"
#include "tma_utils.cuh"

namespace {

using namespace tma;

constexpr int RC = 10;             // rows per ring stage = 2 rows per consumer row-pair x 5
constexpr int NCW = 10;            // consumer warps (+ 1 producer = 11 warps, 168 registers/thread)
constexpr int NTHREADS = (NCW + 1) * 32;
constexpr int ZS = RC + 2;         // rows of the Z ring: phase B of a block reads Z rows [first - 1, last + 1]
constexpr int SMEM_BUDGET = 227 * 1024 - 1024;

template <int K> struct Cfg2 {
    static constexpr int F = K + 1;                                        // 3-vector fields in the ring: m, Y_1..Y_K
    static constexpr int ROW_BYTES = (F * (ROWD + 2 * SIDED) + CROWD + 2 * SIDED) * 8;   // one row of everything
    static constexpr int Z_D = K * ZS * ROWD;
    static constexpr int S_FIT = (SMEM_BUDGET - Z_D * 8) / (ROW_BYTES * RC);
    static constexpr int S = S_FIT > 4 ? 4 : S_FIT;                        // ring stages
    static constexpr int NSLOT = S * RC;
    static constexpr int MAIN_D = F * NSLOT * ROWD;                        // [F][NSLOT][ROWD]
    static constexpr int SIDE_D = F * NSLOT * SIDED;                       // [F][NSLOT][SIDED], one each for the left and right wrap
    static constexpr int CM_D = NSLOT * CROWD;                             // [NSLOT][CROWD]
    static constexpr int CS_D = NSLOT * SIDED;                             // [NSLOT][SIDED], left / right
    static constexpr int UX_D = NCW * 96;                                  // per-warp transpose scratch of the three-term operand (32 sites x 3)
    static constexpr size_t SMEM = (size_t)(MAIN_D + 2 * SIDE_D + CM_D + 2 * CS_D + Z_D + UX_D) * 8 + 2 * S * 8 + 64 * 4;
    static_assert(S >= 3, "ring too shallow");
    static_assert(SMEM <= 232448, "over the 227 KB per-CTA limit");
};

struct FSet { CUtensorMap chunk, row, schunk, srow; };   // RC-row / 1-row boxes: main (64 sites) and side (16 doubles)
struct Maps2 {
    FSet m, c;      // c: [Ly][Lx] scalars, main box 64 wide, side box 16 wide
    FSet y[3];      // Y_{i-1} sources: [0] the input block (pass 1), [1] B1 (even passes), [2] B3 (odd passes >= 3)
};

struct KParams2 {
    Lat l;
    int nsx;                     // number of strips
    long long total;             // nsx * Ly strip-rows
    int npass;                   // passes = degree / 2
    const double* coef;          // [2 npass][4]: {alpha_i, c0, beta_i, -}
    const double* B[4];          // rotating blocks: Y_j lives in B[(j - 1) & 3], j >= 1
    double* Bw[4];
    double* out;                 // Y_{2 npass}
    const int* done;
    unsigned long long* flags;   // [grid] last pass finished by each CTA, as epoch + pass
    unsigned long long epoch;
    int* err;
    int gpair;                   // CTAs per column group: CTA b works on columns K (b / gpair) .. of every block with the
                                 // strip-rows of local CTA b % gpair (one launch for all column pairs of a block size above 2)
};

__device__ __forceinline__ d3 lds3(const double* p) { return mk3(p[0], p[1], p[2]); }
__device__ __forceinline__ void sts3(double* p, d3 v) { p[0] = v.x; p[1] = v.y; p[2] = v.z; }
// halo sites of the three-term operand were written by other SMs: read them through L2, never from a stale L1 line
__device__ __forceinline__ d3 ldcg3(const double* p, long long i) { return mk3(__ldcg(p + 3 * i), __ldcg(p + 3 * i + 1), __ldcg(p + 3 * i + 2)); }

// where stencil operand "box site index i" of a row lives: the main row box, or a wrap side box on the edge strips
struct Role { int off, pitch, fstr; };   // doubles: offset of field 0 / slot 0, row-slot pitch, field stride

// PF: every step of the launch is a product-form step (beta = 0): the third-operand path is compiled out.
template <int K, bool PF>
__global__ void __launch_bounds__(NTHREADS, 1) k_cheb2_tma(const __grid_constant__ Maps2 maps, const KParams2 p) {
    using C = Cfg2<K>;
    constexpr int F = C::F, S = C::S, NSLOT = C::NSLOT;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* smain = reinterpret_cast<double*>(smem_raw);          // [F][NSLOT][ROWD]
    double* sL = smain + C::MAIN_D;                               // [F][NSLOT][SIDED]   sites Lx-2, Lx-1 at doubles 10..15
    double* sR = sL + C::SIDE_D;                                  // [F][NSLOT][SIDED]   sites 0, 1 at doubles 0..5
    double* scm = sR + C::SIDE_D;                                 // [NSLOT][CROWD]
    double* scL = scm + C::CM_D;                                  // [NSLOT][SIDED]      c of sites Lx-2, Lx-1 at 14, 15
    double* scR = scL + C::CS_D;                                  // [NSLOT][SIDED]      c of sites 0, 1 at 0, 1
    double* sZ = scR + C::CS_D;                                   // [K][ZS][ROWD]       Z = Y_i of phase A, column = box site index - 1
    double* sUx = sZ + C::Z_D;                                    // [NCW][96]
    uint64_t* full = reinterpret_cast<uint64_t*>(sUx + C::UX_D);
    uint64_t* empty = full + S;
    int* sdep = reinterpret_cast<int*>(empty + S);                // [0] = count, [1..] = CTAs this one exchanges halos with

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const Lat& l = p.l;
    const int Lx = l.Lx, Ly = l.Ly;

    if (threadIdx.x == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NCW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == NCW && lane < 20) asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&maps.m.chunk + lane)) : "memory");
    __syncthreads();
    if (p.done && *p.done) return;

    // column group of this CTA and its place among the group's G CTAs (a launch for one group: G = gridDim.x)
    const int G = p.gpair, grp = (int)blockIdx.x / G, bid = (int)blockIdx.x - grp * G;
    const long long lo = (p.total * bid) / G, hi = (p.total * (bid + 1)) / G;

    if (warp == NCW) {
        // ================================================================ producer warp: all 32 lanes issue TMA boxes
        if (lane == 0) {   // halo partners: CTAs owning sites within two rows / two columns of this CTA's sub-segments
            int nd = 0;
            auto add = [&](int c) {
                for (int i = 1; i <= nd; ++i) if (sdep[i] == c) return;
                if (nd < 60) sdep[++nd] = c; else *p.err = 1;
            };
            auto add_rows = [&](int sx2, int ya, int yb) {
                const int c0 = cta_of((long long)sx2 * Ly + ya, p.total, G), c1 = cta_of((long long)sx2 * Ly + yb, p.total, G);
                for (int c = c0; c <= c1; ++c) add(c);
            };
            add(bid);
            long long q = lo;
            while (q < hi) {
                const int sx = (int)(q / Ly), y0 = (int)(q - (long long)sx * Ly);
                const int nr = (int)((hi - q) < (long long)(Ly - y0) ? (hi - q) : (Ly - y0)), y1 = y0 + nr;   // rows [y0, y1)
                for (int ds = -1; ds <= 1; ++ds) {
                    int s2 = sx + ds;
                    if (s2 < 0) { if (!l.px) continue; s2 += p.nsx; }
                    if (s2 >= p.nsx) { if (!l.px) continue; s2 -= p.nsx; }
                    add_rows(s2, y0 - 2 > 0 ? y0 - 2 : 0, y1 + 1 < Ly ? y1 + 1 : Ly - 1);
                    if (l.py && y0 < 2) add_rows(s2, Ly - 2 + y0 > 0 ? Ly - 2 + y0 : 0, Ly - 1);
                    if (l.py && y1 > Ly - 2) add_rows(s2, 0, y1 + 1 - Ly < Ly ? y1 + 1 - Ly : Ly - 1);
                }
                q += nr;
            }
            sdep[0] = nd;
        }
        __syncwarp();
        constexpr int KINDS = 3 * F + 3;   // per row (or chunk): F main, c main, F left sides, c left, F right sides, c right
        unsigned n = 0;
        for (int pass = 1; pass <= p.npass; ++pass) {
            const FSet& ys = maps.y[pass == 1 ? 0 : ((pass & 1) ? 2 : 1)];
            const bool rev = !(pass & 1);   // even passes sweep every segment bottom-up
            if (pass > 1) {   // every halo partner has published pass - 1 (bounded spin: a lost partner must not hang the GPU)
                const int nd = sdep[0];
                const unsigned long long want = p.epoch + (unsigned long long)(pass - 1);
                for (int d = lane; d < nd; d += 32) {
                    const unsigned long long* f = p.flags + grp * G + sdep[1 + d];
                    unsigned long long v; int spins = 0;
                    do {
                        asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(f) : "memory");
                        if (v >= want) break;
                        __nanosleep(32);
                    } while (++spins < (1 << 22));
                    if (v < want) *p.err = 1;
                }
                __syncwarp();
                asm volatile("fence.proxy.async;" ::: "memory");   // generic-proxy writes of the partners -> this CTA's TMA reads
            }
            long long pos = lo;
            while (pos < hi) {
                const int sx = (int)(pos / Ly), y_start = (int)(pos - (long long)sx * Ly);
                const int nrows = (int)((hi - pos) < (long long)(Ly - y_start) ? (hi - pos) : (Ly - y_start));
                const int y_end = y_start + nrows;
                const int xb = strip_x(sx, Lx, p.nsx), xe = (sx + 1 == p.nsx) ? Lx : strip_x(sx + 1, Lx, p.nsx);
                const bool edgeL = l.px && xb == 0, edgeR = l.px && xe == Lx;
                const int nside = (edgeL ? 1 : 0) + (edgeR ? 1 : 0);
                const int Q = (nrows + 4 + RC - 1) / RC;
                const int x3 = 3 * (xb - 2);   // even: the box start is 16-byte aligned
                for (int j = 0; j < Q; ++j, ++n) {
                    const unsigned s = n % S, ph = (n / S) & 1u;
                    const int r0 = j * RC - 2;                                 // sweep-order index of the first row of this stage
                    const int nvalid = (nrows + 2 - r0) < RC ? (nrows + 2 - r0) : RC;
                    // forward: row r lives at y = y_start + r; reversed: at y = y_end - 1 - r, and a chunk box (ascending y) then
                    // holds descending r, so row i of the stage sits in slot RC - 1 - i
                    const int y0 = rev ? y_end - r0 - RC : y_start + r0;          // lowest-y row of the full chunk box
                    const bool chunk_ok = (nvalid == RC) && (!l.py || (y0 >= 0 && y0 + RC <= Ly));
                    if (lane == 0) {
                        mbar_wait(&empty[s], ph ^ 1u);
                        mbar_expect_tx(&full[s], (unsigned)nvalid * ((F * ROWD + CROWD) * 8 + nside * (F + 1) * SIDED * 8));
                    }
                    __syncwarp();
                    const int nops = (chunk_ok ? 1 : nvalid) * KINDS;
                    for (int t = lane; t < nops; t += 32) {
                        const int i = t / KINDS, kind = t - i * KINDS;
                        int y = chunk_ok ? y0 : (rev ? y_end - 1 - (r0 + i) : y_start + r0 + i);
                        if (!chunk_ok && l.py) { if (y < 0) y += Ly; else if (y >= Ly) y -= Ly; }
                        const int slot = s * RC + (chunk_ok ? 0 : (rev ? RC - 1 - i : i));
                        const int g = kind / (F + 1), f = kind - g * (F + 1);      // g: 0 main, 1 left side, 2 right side; f: field, F = c
                        if (g == 1 && !edgeL) continue;
                        if (g == 2 && !edgeR) continue;
                        const FSet& fs = f == 0 ? maps.m : (f == F ? maps.c : ys);
                        const CUtensorMap* mp = g == 0 ? (chunk_ok ? &fs.chunk : &fs.row) : (chunk_ok ? &fs.schunk : &fs.srow);
                        const int vec = (f == 0 || f == F) ? 0 : K * grp + f - 1;
                        if (f < F) {
                            double* dst = g == 0 ? smain + ((size_t)f * NSLOT + slot) * ROWD : (g == 1 ? sL : sR) + ((size_t)f * NSLOT + slot) * SIDED;
                            tma_load_3d(dst, mp, &full[s], g == 0 ? x3 : (g == 1 ? 3 * Lx - SIDED : 0), y, vec);
                        } else {
                            double* dst = g == 0 ? scm + (size_t)slot * CROWD : (g == 1 ? scL : scR) + (size_t)slot * SIDED;
                            tma_load_3d(dst, mp, &full[s], g == 0 ? xb - 2 : (g == 1 ? Lx - SIDED : 0), y, 0);
                        }
                    }
                }
                pos += nrows;
            }
        }
        return;
    }

    // ==================================================================== consumers
    const int ch = warp & 1, rp = warp >> 1;
    const int col = ch * 32 + lane;          // column of phase A: x = xb - 1 + col, box site index col + 1
    const long long N = (long long)Lx * Ly;
    unsigned n = 0;
    for (int pass = 1; pass <= p.npass; ++pass) {
        const double* cfA = p.coef + 4 * (2 * pass - 2);
        const double* cfB = cfA + 4;
        const double alA = cfA[0], c0A = cfA[1], beA = cfA[2];
        const double alB = cfB[0], c0B = cfB[1], beB = cfB[2];
        // product-form steps (beta = 0, k_cheb_coef) have no third operand: phase A then reads nothing from global memory, and
        // Y_{2 pass - 1} -- wanted by the next pass only as ITS third operand -- never leaves shared memory: a pass moves
        // m, c, Y_{2 pass - 2} in and Y_{2 pass} out, 128 B/site per TWO steps at k = 2
        const size_t goff = (size_t)grp * K * 3 * N;                              // this group's columns inside every block
        const double* UA = (PF || pass == 1 || beA == 0.0) ? nullptr : p.B[(2 * pass - 4) & 3] + goff;   // Y_{2 pass - 3}
        const bool storeA = !PF && pass < p.npass && p.coef[4 * (2 * pass) + 2] != 0.0;
        double* outA = p.Bw[(2 * pass - 2) & 3] + goff;                           // Y_{2 pass - 1}
        double* outB = (pass == p.npass ? p.out : p.Bw[(2 * pass - 1) & 3]) + goff;   // Y_{2 pass}
        // Even passes sweep bottom-up on the point-reflected lattice: row order reversed, left and right neighbours swapped,
        // D -> -D (the stencil is inversion symmetric up to the sign of the DMI vectors), bit-identical to a forward sweep.
        const bool rev = !(pass & 1);
        Lat ls = p.l;
        if (rev) ls.D = -ls.D;
        long long pos = lo;
        while (pos < hi) {
            const int sx = (int)(pos / Ly), y_start = (int)(pos - (long long)sx * Ly);
            const int nrows = (int)((hi - pos) < (long long)(Ly - y_start) ? (hi - pos) : (Ly - y_start));
            const int y_end = y_start + nrows;
            const int xb = strip_x(sx, Lx, p.nsx), xe = (sx + 1 == p.nsx) ? Lx : strip_x(sx + 1, Lx, p.nsx);
            const int w = xe - xb;
            const bool edgeL = l.px && xb == 0, edgeR = l.px && xe == Lx;
            const bool actA = col < w + 2, actB = col >= 1 && col < w + 1;
            int xg = xb - 1 + col;                       // lattice column of this thread (wrapped); xin: inside the lattice
            bool xin = true;
            if (xg < 0) { if (l.px) xg += Lx; else xin = false; }
            else if (xg >= Lx) { if (l.px) xg -= Lx; else xin = false; }
            auto role3 = [&](int i) {   // 3-vector fields
                Role r;
                if (edgeL && i < 2) { r.off = (int)(sL - smain) + 10 + 3 * i; r.pitch = SIDED; r.fstr = NSLOT * SIDED; }
                else if (edgeR && i >= w + 2) { r.off = (int)(sR - smain) + 3 * (i - w - 2); r.pitch = SIDED; r.fstr = NSLOT * SIDED; }
                else { r.off = 3 * i; r.pitch = ROWD; r.fstr = NSLOT * ROWD; }
                return r;
            };
            const Role rLp = role3(col), rC = role3(col + 1), rRp = role3(col + 2);
            const Role rL = rev ? rRp : rLp, rR = rev ? rLp : rRp;     // stencil frame
            int cOff, cPitch;                                           // c at the phase-A centre
            if (edgeL && col + 1 < 2) { cOff = (int)(scL - smain) + 14 + col + 1; cPitch = SIDED; }
            else if (edgeR && col + 1 >= w + 2) { cOff = (int)(scR - smain) + (col + 1 - w - 2); cPitch = SIDED; }
            else { cOff = (int)(scm - smain) + col + 1; cPitch = CROWD; }
            const int Q = (nrows + 4 + RC - 1) / RC, nb = (nrows + 2 + RC - 1) / RC;

            // Three-term operand of phase A (Y_{2 pass - 3} at the Z sites, halo included), read straight from global memory a
            // block ahead.  A lane-per-site read of 24-byte sites costs three 8-byte requests per lane that each touch all 24
            // sectors of the warp's 768-byte row segment (x3 L2 traffic: 20 of 60 us per pass in the round-2 probe), so the warp
            // reads its row segment flat -- lane l takes doubles l, 32 + l, 64 + l -- and transposes it through 768 bytes of
            // shared memory when the values are used.  eo[t]: offset of flat element 32 t + lane inside a lattice row (the halo
            // columns of an edge strip wrap), -1 where the site is outside the strip's Z columns or outside an open lattice.
            int eo[3];
#pragma unroll
            for (int t = 0; t < 3; ++t) {
                const int e = 32 * t + lane, ce = ch * 32 + e / 3;
                int xe_ = xb - 1 + ce;
                bool ok = ce < w + 2;
                if (xe_ < 0) { if (l.px) xe_ += Lx; else ok = false; }
                else if (xe_ >= Lx) { if (l.px) xe_ -= Lx; else ok = false; }
                eo[t] = ok ? 3 * xe_ + e % 3 : -1;
            }
            double uraw[2][K][3];
            auto row_y = [&](int r, bool& yin) {   // lattice row of sweep-order row r (wrapped); yin: inside the lattice
                int y = rev ? y_end - 1 - r : y_start + r;
                yin = true;
                if (y < 0) { if (l.py) y += Ly; else yin = false; }
                else if (y >= Ly) { if (l.py) y -= Ly; else yin = false; }
                return y;
            };
            auto load_u = [&](int jb) {
                const int rA = jb * RC - 1 + 2 * rp;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    bool yin;
                    const int y = row_y(rA + h, yin);
                    const bool rowok = UA && yin && rA + h <= nrows;
#pragma unroll
                    for (int a = 0; a < K; ++a) {
                        const double* rowp = UA + (size_t)a * 3 * N + 3 * (long long)y * Lx;
#pragma unroll
                        for (int t = 0; t < 3; ++t) uraw[h][a][t] = (rowok && eo[t] >= 0) ? __ldcg(rowp + eo[t]) : 0.0;
                    }
                }
            };
            double* scr = sUx + warp * 96;
            auto take_u = [&](int h, int a) {   // this thread's site of row h, field a (all lanes of the warp call it together)
                __syncwarp();
                scr[lane] = uraw[h][a][0]; scr[32 + lane] = uraw[h][a][1]; scr[64 + lane] = uraw[h][a][2];
                __syncwarp();
                return lds3(scr + 3 * lane);
            };
            mbar_wait(&full[n % S], (n / S) & 1u);
            if (!PF && UA) load_u(0);
            for (int j = 0; j < nb; ++j) {
                if (j + 1 < Q) mbar_wait(&full[(n + j + 1) % S], ((n + j + 1) / S) & 1u);
                const int cur = (int)((n + j) % S), nxt = (cur + 1 == S) ? 0 : cur + 1;
                // ---------------------------------------------------------------- phase A: Z rows rA, rA + 1
                const int rA = j * RC - 1 + 2 * rp;
                if (actA && rA <= nrows) {
                    int sr[4];
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const int t = 2 * rp + q;
                        sr[q] = (t < RC ? cur * RC + (rev ? RC - 1 - t : t) : nxt * RC + (rev ? RC - 1 - (t - RC) : t - RC));
                    }
                    const bool haveB = rA + 1 <= nrows;
                    bool yinA, yinB;
                    const int yA = row_y(rA, yinA), yB = row_y(rA + 1, yinB);
                    const bool inA = xin && yinA, inB = xin && yinB && haveB;
                    const d3 m1C = lds3(smain + rC.off + sr[1] * rC.pitch), m2C = lds3(smain + rC.off + sr[2] * rC.pitch);
                    const double cA = smain[cOff + sr[1] * cPitch], cB = smain[cOff + sr[2] * cPitch];
                    const int zA = (rA + 1) % ZS, zB = (rA + 2) % ZS;
                    const bool ownA = actB && rA >= 0 && rA < nrows, ownB = actB && rA + 1 < nrows;
#pragma unroll
                    for (int a = 0; a < K; ++a) {
                        const double* bL = smain + rL.off + (a + 1) * rL.fstr;
                        const double* bC = smain + rC.off + (a + 1) * rC.fstr;
                        const double* bR = smain + rR.off + (a + 1) * rR.fstr;
                        const d3 u0C = lds3(bC + sr[0] * rC.pitch), u0R = lds3(bR + sr[0] * rR.pitch);
                        const d3 u1L = lds3(bL + sr[1] * rL.pitch), u1C = lds3(bC + sr[1] * rC.pitch), u1R = lds3(bR + sr[1] * rR.pitch);
                        const d3 u2L = lds3(bL + sr[2] * rL.pitch), u2C = lds3(bC + sr[2] * rC.pitch), u2R = lds3(bR + sr[2] * rR.pitch);
                        const d3 u3L = lds3(bL + sr[3] * rL.pitch), u3C = lds3(bC + sr[3] * rC.pitch);
                        const d3 LA = stencil_apply(ls, u1R, u1L, u2C, u0C, u2L, u0R, u1C.z);
                        const d3 LB = stencil_apply(ls, u2R, u2L, u3C, u1C, u3L, u1R, u2C.z);
                        d3 oA = scale3(alA, axpy3(-c0A, u1C, axpy3(-cA, u1C, proj3(m1C, LA))));
                        d3 oB = scale3(alA, axpy3(-c0A, u2C, axpy3(-cB, u2C, proj3(m2C, LB))));
                        if (!inA) oA = mk3(0.0, 0.0, 0.0);      // outside an open lattice: absent neighbour contributes 0
                        if (!inB) oB = mk3(0.0, 0.0, 0.0);
                        sts3(sZ + ((size_t)a * ZS + zA) * ROWD + 3 * col, oA);
                        if (haveB) sts3(sZ + ((size_t)a * ZS + zB) * ROWD + 3 * col, oB);
                    }
                }
                // The three-term operand is added last, through a round trip of the partial result in this thread's own Z slots.
                if (!PF && UA && rA <= nrows) {   // warp-uniform: take_u synchronises the warp
                    const bool haveB = rA + 1 <= nrows;
                    bool yinA, yinB;
                    row_y(rA, yinA); row_y(rA + 1, yinB);
                    const bool inA = actA && xin && yinA, inB = actA && xin && yinB && haveB;
                    const int zA = (rA + 1) % ZS, zB = (rA + 2) % ZS;
#pragma unroll
                    for (int a = 0; a < K; ++a) {
                        const d3 ua = take_u(0, a), ub = take_u(1, a);
                        double* zpA = sZ + ((size_t)a * ZS + zA) * ROWD + 3 * col;
                        double* zpB = sZ + ((size_t)a * ZS + zB) * ROWD + 3 * col;
                        if (inA) sts3(zpA, axpy3(beA, ua, lds3(zpA)));
                        if (inB) sts3(zpB, axpy3(beA, ub, lds3(zpB)));
                    }
                }
                if (storeA && actA && rA <= nrows) {   // own sites of Y_{2 pass - 1} to HBM
                    bool yinA, yinB;
                    const int yA = row_y(rA, yinA), yB = row_y(rA + 1, yinB);
                    const int zA = (rA + 1) % ZS, zB = (rA + 2) % ZS;
                    const bool ownA = actB && rA >= 0 && rA < nrows, ownB = actB && rA + 1 < nrows;
#pragma unroll
                    for (int a = 0; a < K; ++a) {
                        if (ownA) st3(outA + (size_t)a * 3 * N, (long long)yA * Lx + xg, lds3(sZ + ((size_t)a * ZS + zA) * ROWD + 3 * col));
                        if (ownB) st3(outA + (size_t)a * 3 * N, (long long)yB * Lx + xg, lds3(sZ + ((size_t)a * ZS + zB) * ROWD + 3 * col));
                    }
                }
                if (!PF && UA && j + 1 < nb) load_u(j + 1);
                asm volatile("bar.sync 1, %0;" ::"n"(NCW * 32) : "memory");      // Z rows of this block complete
                // ---------------------------------------------------------------- phase B: rows rB, rB + 1 of Y_{2 pass}
                const int rB = j * RC - 2 + 2 * rp;
                if (actB && rB + 1 >= 0 && rB < nrows) {
                    const bool haveA = rB >= 0, haveB = rB + 1 < nrows;
                    const int t0 = 2 * rp, t1 = 2 * rp + 1;                         // stage rows of the two centres (always in `cur`)
                    const int sA = cur * RC + (rev ? RC - 1 - t0 : t0), sB = cur * RC + (rev ? RC - 1 - t1 : t1);
                    int z[4];
#pragma unroll
                    for (int q = 0; q < 4; ++q) z[q] = (rB + q + ZS) % ZS;           // Z rows rB - 1 .. rB + 2 (row r in slot (r + 1) mod ZS)
                    const double* zC = sZ + 3 * col;
                    const double* zL = rev ? zC + 3 : zC - 3;
                    const double* zR = rev ? zC - 3 : zC + 3;
                    const double* mC = smain + 3 * (col + 1);
                    const d3 mA = lds3(mC + sA * ROWD), mB = lds3(mC + sB * ROWD);
                    const double cA = scm[sA * CROWD + col + 1], cB = scm[sB * CROWD + col + 1];
                    bool yinA, yinB;
                    const int yA = row_y(rB, yinA), yB = row_y(rB + 1, yinB);
#pragma unroll
                    for (int a = 0; a < K; ++a) {
                        const size_t fo = (size_t)a * ZS * ROWD;
                        const d3 u0C = lds3(zC + fo + z[0] * ROWD), u0R = lds3(zR + fo + z[0] * ROWD);
                        const d3 u1L = lds3(zL + fo + z[1] * ROWD), u1C = lds3(zC + fo + z[1] * ROWD), u1R = lds3(zR + fo + z[1] * ROWD);
                        const d3 u2L = lds3(zL + fo + z[2] * ROWD), u2C = lds3(zC + fo + z[2] * ROWD), u2R = lds3(zR + fo + z[2] * ROWD);
                        const d3 u3L = lds3(zL + fo + z[3] * ROWD), u3C = lds3(zC + fo + z[3] * ROWD);
                        const d3 LA = stencil_apply(ls, u1R, u1L, u2C, u0C, u2L, u0R, u1C.z);
                        const d3 LB = stencil_apply(ls, u2R, u2L, u3C, u1C, u3L, u1R, u2C.z);
                        const double* yp = mC + (size_t)(a + 1) * NSLOT * ROWD;                 // Y_{2 pass - 2} at the centres
                        d3 oA = scale3(alB, axpy3(-c0B, u1C, axpy3(-cA, u1C, proj3(mA, LA))));
                        d3 oB = scale3(alB, axpy3(-c0B, u2C, axpy3(-cB, u2C, proj3(mB, LB))));
                        if (!PF && beB != 0.0) {
                            oA = axpy3(beB, lds3(yp + sA * ROWD), oA);
                            oB = axpy3(beB, lds3(yp + sB * ROWD), oB);
                        }
                        if (haveA) st3(outB + (size_t)a * 3 * N, (long long)yA * Lx + xg, oA);
                        if (haveB) st3(outB + (size_t)a * 3 * N, (long long)yB * Lx + xg, oB);
                    }
                }
                asm volatile("bar.sync 1, %0;" ::"n"(NCW * 32) : "memory");      // phase B done: Z slots and the stage may be reused
                if (lane == 0) mbar_arrive(&empty[cur]);
            }
            if (Q > nb) { if (lane == 0) mbar_arrive(&empty[(n + nb) % S]); }
            n += Q;
            pos += nrows;
        }
        // publish "this CTA has finished pass": every consumer's stores first, then one release store
        // (one fence by the publishing thread after the CTA barrier covers every consumer's stores by cumulativity -- the
        // pattern of a cooperative-groups grid sync; a fence per thread cost ~2 us per step)
        asm volatile("bar.sync 1, %0;" ::"n"(NCW * 32) : "memory");
        if (threadIdx.x == 0) {
            __threadfence();
            const unsigned long long v = p.epoch + (unsigned long long)pass;
            asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p.flags + blockIdx.x), "l"(v) : "memory");
        }
    }
}

bool encode_fset(FSet* v, const double* base, int Lx, int Ly, int nvec, int ncomp) {
    const int mainw = ncomp == 3 ? ROWD : CROWD;
    return encode(&v->chunk, base, Lx, Ly, nvec, mainw, RC, ncomp) && encode(&v->row, base, Lx, Ly, nvec, mainw, 1, ncomp) &&
           encode(&v->schunk, base, Lx, Ly, nvec, SIDED, RC, ncomp) && encode(&v->srow, base, Lx, Ly, nvec, SIDED, 1, ncomp);
}

template <int K, bool PF>
bool launch2(moto_ctx* c, const Maps2& maps, const KParams2& p, int grid) {
    using C = Cfg2<K>;
    static std::atomic<unsigned long long> attr_seen{0};
    if (!ensure_smem_attr(k_cheb2_tma<K, PF>, C::SMEM, attr_seen)) return false;
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(NTHREADS); cfg.dynamicSmemBytes = C::SMEM; cfg.stream = c->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;   // CTAs wait on each other's flags: they must all be resident
    attr[0].val.cooperative = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    if (cudaLaunchKernelEx(&cfg, k_cheb2_tma<K, PF>, maps, p) == cudaSuccess) return true;
    (void)cudaGetLastError();   // the caller falls back to the one-step-per-pass path
    return false;
}

template <int K>
int coop_limit2() {
    using C = Cfg2<K>;
    int dev = 0, sms = 0, per_sm = 0;
    static std::atomic<unsigned long long> attr_seen{0};
    if (cudaGetDevice(&dev) != cudaSuccess) return -1;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1;
    if (!ensure_smem_attr(k_cheb2_tma<K, false>, C::SMEM, attr_seen)) return -1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_cheb2_tma<K, false>, NTHREADS, C::SMEM) != cudaSuccess) return -1;
    return sms * per_sm;
}

}  // namespace

// Two recurrence steps per pass: OUT = Y_d, d even, Y_0 = V, coefficients at d_coef + 4 (i - 1) (device memory); Y_1 .. Y_{d-1}
// rotate through the context's four blocks T1 .. T4.  k <= 2.  Returns the number of launches, 0 if not applicable (the
// caller then takes spin_cheb_multistep / the step-wise path).
// product_form: every coefficient row has beta = 0 (k_cheb_coef): the kernel without the third-operand path.
// ngroups > 1 (k == 2 only): V, OUT and the rotating blocks hold 2 ngroups columns and ONE launch runs the recurrence on all of them,
// column pair g on its own set of CTAs (grid = ngroups x CTAs per pair, each pair synchronising among its own CTAs only): block
// sizes above 2 on lattices too small to fill the GPU with one pair (cfg 2: three 72-us launches bound by the neighbour
// synchronisation of 32 steps become one).
int spin_cheb2_multistep(moto_ctx* c, const double* m, const double* cvec, const double* V, int k, int d, double* OUT,
                         const double* d_coef, const int* d_done, int product_form, int ngroups) {
    if (!spin_tma_applicable(c) || k > 2 || d < 2 || (d & 1) || !c->T1 || !c->T3 || !cvec) return 0;
    if (ngroups < 1 || (ngroups > 1 && (k != 2 || 2 * ngroups > c->kmax))) return 0;
    if (((uintptr_t)m & 15) || ((uintptr_t)V & 15) || ((uintptr_t)cvec & 15)) return 0;
    const int Lx = c->lat.Lx, Ly = c->lat.Ly;
    if (Lx < SIDED || Ly < 4) return 0;   // the side box of c holds 16 sites; two-row halos
    const int nsx = (Lx + TXMAX - 1) / TXMAX;
    const long long total = (long long)nsx * Ly;
    long long g = (total + RC - 1) / RC;
    if (c->coop2_max_ctas == 0) c->coop2_max_ctas = k == 2 ? coop_limit2<2>() : coop_limit2<1>();
    const int cap = (c->coop2_max_ctas < MOTO_NUM_SMS ? c->coop2_max_ctas : MOTO_NUM_SMS) / ngroups;   // CTAs a column group may take
    if (cap < 1) return 0;
    const int gpair = (int)(g > cap ? cap : (g < 1 ? 1 : g));
    const int grid = gpair * ngroups;
    Maps2 maps;
    memset(&maps, 0, sizeof(maps));
    bool ok = encode_fset(&maps.m, m, Lx, Ly, 1, 3) && encode_fset(&maps.c, cvec, Lx, Ly, 1, 1) &&
              encode_fset(&maps.y[0], V, Lx, Ly, k * ngroups, 3) && encode_fset(&maps.y[1], c->T2, Lx, Ly, k * ngroups, 3) &&
              encode_fset(&maps.y[2], c->T4, Lx, Ly, k * ngroups, 3);
    if (!ok) return 0;
    KParams2 p;
    p.l = make_lat(c);
    p.nsx = nsx; p.total = total; p.npass = d / 2; p.coef = d_coef;
    double* T[4] = {c->T1, c->T2, c->T3, c->T4};
    for (int i = 0; i < 4; ++i) { p.B[i] = T[i]; p.Bw[i] = T[i]; }
    p.out = OUT; p.done = d_done;
    p.flags = c->flags; c->epoch += 1024; p.epoch = c->epoch; p.err = &c->st->bad;
    p.gpair = gpair;
    const bool l_ok = product_form ? (k == 2 ? launch2<2, true>(c, maps, p, grid) : launch2<1, true>(c, maps, p, grid))
                                   : (k == 2 ? launch2<2, false>(c, maps, p, grid) : launch2<1, false>(c, maps, p, grid));
    return l_ok ? 1 : 0;
}

// The whole degree-d recurrence OUT = Y_d (Y_0 = V, coefficients at d_coef + 4 (i - 1), device memory) by the fastest path
// the context allows (moto_solver_opts.cheb_mode): one cooperative launch with one step per pass (auto: the fastest as
// measured at 10^6 spins), two steps per pass (+ one single step when d is odd) on request, else d dependent launches.  k <= 2, V tangent, d >= 1.
// Returns the number of launches, or -1 if the TMA K1 path does not apply / a launch failed (nothing usable in OUT).
int spin_cheb_recurrence(moto_ctx* c, const double* m, const double* cvec, const double* V, int k, int d, double* OUT,
                         const double* d_coef, const int* d_done) {
    if (c->nsh > 0) return shell_cheb_recurrence(c, m, cvec, V, k, d, OUT, d_coef, d_done);   // general shells: one launch per step
    const int mode = c->opts.cheb_mode == 0 ? 3 : c->opts.cheb_mode;   // auto: two steps per pass (22.2 vs 24.1 us/step at 10^6 spins)
    double* T[4] = {c->T1, c->T2, c->T3, c->T4};
    if (mode == 3 && d >= 2) {
        const int de = d & ~1;
        // odd d: Y_{d-1} goes to the block it would occupy in the rotation, the last step is a single launch
        int n = spin_cheb2_multistep(c, m, cvec, V, k, de, de == d ? OUT : T[(de - 1) & 3], d_coef, d_done, /*product_form=*/1, 1);
        if (n > 0) {
            if (de == d) return n;
            const int n1 = spin_hvp_tma_ex(c, m, cvec, T[(de - 1) & 3], k, OUT, d_done, nullptr, 1, 0.0, 0.0, 0.0, T[(de - 2) & 3],
                                           d_coef + 4 * (d - 1));
            return n1 > 0 ? n + n1 : -1;
        }
    }
    if ((mode <= 1 || mode == 3) && d >= 2) {
        const int n = spin_cheb_multistep(c, m, cvec, V, k, d, OUT, d_coef, d_done);
        if (n > 0) return n;
    }
    // one launch per step: Y_1 -> T1, Y_2 -> T2, Y_3 -> T1 (in place over its own three-term operand) ...
    int n = 0;
    const double* in = V; const double* prev = nullptr;
    for (int i = 1; i <= d; ++i) {
        double* out = (i == d) ? OUT : ((i & 1) ? c->T1 : c->T2);
        const int n1 = spin_hvp_tma_ex(c, m, cvec, in, k, out, d_done, nullptr, 1, 0.0, 0.0, 0.0, prev, d_coef + 4 * (i - 1));
        if (n1 <= 0) return -1;
        n += n1;
        prev = in; in = out;
    }
    return n;
}
