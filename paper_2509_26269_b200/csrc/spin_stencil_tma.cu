// spin_stencil_tma.cu -- K1, the TMA-staged fast path of the fused gradient + block Riemannian HVP stencil
// (Eq. 4; Hv PAPER.md:156; projected-gradient Jacobian PAPER.md:162; reading A5).
//
// Design (B200, sm_100a): a persistent grid of one CTA per SM.  The lattice is cut into column strips of
// <= 60 sites; the (strip, row) space is linearised and split evenly over the CTAs, so every CTA streams
// one or two vertical strip segments.  One producer warp drives the TMA engine (its 32 lanes issue the boxes of a
// stage in parallel): each 10-row chunk of every field (m, V_1..V_K; 64 sites = 60 + halo columns, 1536 B per row;
// in solver mode also c_i) is one cp.async.bulk.tensor box landing in a ring of shared-memory row slots guarded by
// full/empty mbarriers; the two halo rows of a segment are 1-row boxes, out-of-range coordinates zero-fill (that IS
// the open boundary), periodic wrap in y is a wrapped row coordinate and periodic wrap in x is a 128-byte side box
// per row.  Ten consumer warps (2 column halves x 5 row pairs) compute two rows per thread from shared memory, so
// each site is read from HBM once for all K directions and from shared memory 5x instead of 7x.  Results go straight
// to global memory; the three-term operand is read directly one block ahead (no reuse).  Tensor cores are not used:
// this is a 7-point stencil, HBM-bound.
//
// Modes:  API    (moto_hvp)      HV = P (L Pv) - c Pv with c = m.(Lm - mu B) recomputed, input projected
//         SOLVER (LOBPCG inner)  HV = P (L v) - c v, c given, v tangent; optional per-CTA partials of V^T HV and
//                                optional three-term epilogue out = alpha (HV - c0 v) + beta u
//         MULTI-STEP (solver)    the whole filter recurrence in one cooperative launch, one step per pass: per-step
//                                neighbour flags, ping-pong blocks, alternating sweep direction (see KParams and DESIGN.md 5).
//                                The library's coefficient rows are product-form steps (beta = 0, k_cheb_coef): such a step
//                                skips the third operand (128 B/site at k = 2).  cheb_mode = 1; the default launch of the
//                                recurrence is the two-steps-per-pass kernel of spin_cheb2_tma.cu.
#include "common.cuh"
#include "device_utils.cuh"
#include "stencil_math.cuh"
#include "tma_utils.cuh"

namespace {

using namespace tma;   // TXMAX, ROWD, SIDED, CROWD, mbarrier / TMA wrappers, tensor-map encoding
constexpr int RC = 10;             // rows per chunk (= 2 rows per consumer row-pair x 5)
constexpr int NCW = 10;            // consumer warps: 10 + 1 producer = 11 warps, registers are granted per 4 warps (12)
constexpr int NTHREADS = (NCW + 1) * 32;

constexpr int SMEM_BUDGET = 231 * 1024;

template <int K, bool API> struct Cfg {
    static constexpr int F = K + 1;                                  // fields in the ring: m, V_1..V_K
    static constexpr int FS0 = API ? 0 : 1;                          // first field with x-wrap side boxes (SOLVER: m needs none)
    static constexpr int NFS = F - FS0;
    static constexpr int ROW_BYTES = (F * ROWD + 2 * NFS * SIDED + (API ? 0 : CROWD)) * 8;   // one row slot, everything
    static constexpr int S = SMEM_BUDGET / (ROW_BYTES * RC) > 8 ? 8 : SMEM_BUDGET / (ROW_BYTES * RC);  // stages
    static constexpr int NSLOT = S * RC;
    static constexpr int MAIN_D = F * NSLOT * ROWD;                  // doubles
    static constexpr int SIDE_D = NFS * NSLOT * SIDED;
    static constexpr int C_D = API ? 0 : NSLOT * CROWD;
    static constexpr int RED_D = NCW * 4;                            // V^T HV reduction scratch
    static constexpr size_t SMEM = (size_t)(MAIN_D + 2 * SIDE_D + C_D + RED_D) * 8 + 2 * S * 8 + 64 * 4;
    static_assert(S >= 3, "ring too shallow");
    static_assert(SMEM <= 232448, "over the 227 KB per-CTA limit");
};

struct VSet { CUtensorMap chunk, row, schunk, srow; };   // chunk = RC rows, row = 1 row; main = 64 sites, side = 16 doubles
struct Maps {
    CUtensorMap m_chunk, m_row, m_schunk, m_srow;
    CUtensorMap c_chunk, c_row;   // c [1][Ly][Lx] fp64, box 64 wide (SOLVER)
    VSet vset[3];                 // [0] the input block; [1], [2] the ping-pong blocks T1, T2 of a multi-step launch
};

struct KParams {
    Lat l;
    int nsx;                 // number of strips
    long long total;         // nsx * Ly strip-rows
    const double* cvec;      // [N] (SOLVER)
    double* out;             // [K][N][3]
    const double* U;         // [K][N][3] Chebyshev operand or NULL
    double alpha, c0, beta;  // out = alpha (HV - c0 v) + beta u   (cheb != 0)
    int cheb;
    const double* coef;      // optional device triple {alpha, c0, beta} overriding the three scalars (device-resident recurrence)
    double* waw;             // [grid][K(K+1)/2] or NULL
    const int* done;
    // multi-step launch (nsteps > 1): the whole Chebyshev recurrence Y_1..Y_nsteps in one persistent cooperative kernel.
    // Y_i goes to T1 (i odd) / T2 (i even), the last one to `out`; step i reads Y_{i-1} through TMA (halo) and Y_{i-2}
    // directly; coefficients of step i at coef + 4 (i - 1).  CTAs synchronise with the few neighbours whose sites they
    // read as halo through release/acquire flags (no grid-wide barrier, no launch gap between steps).
    int nsteps;
    const double* V0;        // the input block (three-term operand of step 2)
    double *T1, *T2;
    unsigned long long* flags;   // [grid] last step finished by each CTA, as epoch + step
    unsigned long long epoch;
    int* err;                // set when a neighbour wait times out
    // energy / gradient mode of the <1, API> instantiation (moto_energy_grad, the c_i of a solve): only m is staged; out = the
    // tangent-projected gradient [N][3] or NULL, c_out = c_i = m_i . g_i [N] or NULL, waw = [grid] partial energies or NULL
    int eg = 0;
    double* c_out = nullptr;
    double* e_out = nullptr;          // eg: E itself [1]; the CTA that finishes last sums the partials in `waw` in fixed order
    unsigned* counter = nullptr;      //     (its arrival counter; left at 0), so the call is one launch
    const double* vdot = nullptr;     // eg, pass 1 of the reflected-force step: out = F = -P g, and e_out = F . vdot instead of E
    int gpair = 0;                    // single-step launches on more than K columns: CTAs per column group (CTA b works on columns
                                      // K (b / gpair) .. with the strip-rows of local CTA b % gpair); 0 = one group, the whole grid
};

__device__ __forceinline__ d3 lds3(const double* p) { return mk3(p[0], p[1], p[2]); }

// ---------------------------------------------------------------------------------------------------------
template <int K, bool API>
__global__ void __launch_bounds__(NTHREADS, 1)   // registers are granted per 4 warps: 9 warps count as 12 => 168 regs/thread
k_hvp_tma(const __grid_constant__ Maps maps, const KParams p) {
    using C = Cfg<K, API>;
    constexpr int F = C::F, S = C::S, NSLOT = C::NSLOT, FS0 = C::FS0, NFS = C::NFS;
    constexpr int NK = K * (K + 1) / 2;
    // programmatic dependent launch: let the next K1 in the stream start its prologue as soon as this CTA's SM frees up
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* smain = reinterpret_cast<double*>(smem_raw);          // [F][NSLOT][ROWD]
    double* sL = smain + C::MAIN_D;                               // [NFS][NSLOT][SIDED]  site Lx-1 at doubles 13..15
    double* sR = sL + C::SIDE_D;                                  // [NFS][NSLOT][SIDED]  site 0 at doubles 0..2
    double* sc = sR + C::SIDE_D;                                  // [NSLOT][CROWD]       c_i (SOLVER)
    double* sred = sc + C::C_D;                                   // [NCW][4]
    uint64_t* full = reinterpret_cast<uint64_t*>(sred + C::RED_D);
    uint64_t* empty = full + S;
    int* sdep = reinterpret_cast<int*>(empty + S);                // [0] = count, [1..] = CTAs this one exchanges halos with

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const Lat& l = p.l;
    const int Lx = l.Lx, Ly = l.Ly;

    if (threadIdx.x == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NCW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == NCW && lane < 10) asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&maps.m_chunk + lane)) : "memory");
    const int nsteps = (!API && p.nsteps > 1) ? p.nsteps : 1;
    const bool eg = API && K == 1 && p.eg;
    __syncthreads();
    // everything above overlapped the tail of the previous kernel; nothing it wrote has been touched yet
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (p.done && *p.done) return;

    const int G = p.gpair > 0 ? p.gpair : (int)gridDim.x, grp = (int)blockIdx.x / G, bid = (int)blockIdx.x - grp * G;
    const long long lo = (p.total * bid) / G, hi = (p.total * (bid + 1)) / G;

    if (warp == NCW) {
        // ================================================================ producer warp: all 32 lanes issue TMA boxes
        // kinds of box per row (or per chunk): F main fields, NFS left-wrap sides, NFS right-wrap sides, c (SOLVER)
        constexpr int KINDS = F + 2 * NFS + (API ? 0 : 1);
        if (nsteps > 1) {   // CTAs whose sites this CTA reads as halo (and which read its sites): same strip above/below, strips left/right
            if (lane == 0) {
                int nd = 0;
                auto add = [&](int c) {   // a partner beyond the capacity of sdep would be a silent race: report it instead
                    for (int i = 1; i <= nd; ++i) if (sdep[i] == c) return;
                    if (nd < 60) sdep[++nd] = c; else *p.err = 1;
                };
                auto add_rows = [&](int sx2, int ya, int yb) {   // rows [ya, yb] of strip sx2
                    const int c0 = cta_of((long long)sx2 * Ly + ya, p.total, gridDim.x), c1 = cta_of((long long)sx2 * Ly + yb, p.total, gridDim.x);
                    for (int c = c0; c <= c1; ++c) add(c);
                };
                add((int)blockIdx.x);
                long long q = lo;
                while (q < hi) {
                    const int sx = (int)(q / Ly), y0 = (int)(q - (long long)sx * Ly);
                    const int nr = (int)((hi - q) < (long long)(Ly - y0) ? (hi - q) : (Ly - y0)), y1 = y0 + nr;   // rows [y0, y1)
                    const int ya = y0 > 0 ? y0 - 1 : 0, yb = y1 < Ly ? y1 : Ly - 1;
                    for (int ds = -1; ds <= 1; ++ds) {
                        int s2 = sx + ds;
                        if (s2 < 0) { if (!l.px) continue; s2 += p.nsx; }
                        if (s2 >= p.nsx) { if (!l.px) continue; s2 -= p.nsx; }
                        add_rows(s2, ya, yb);
                        if (l.py && y0 == 0) add_rows(s2, Ly - 1, Ly - 1);
                        if (l.py && y1 == Ly) add_rows(s2, 0, 0);
                    }
                    q += nr;
                }
                sdep[0] = nd;
            }
            __syncwarp();
        }
        unsigned n = 0;
        for (int step = 1; step <= nsteps; ++step) {
        const VSet& vs = maps.vset[step == 1 ? 0 : (((step - 1) & 1) ? 1 : 2)];   // Y_{step-1}: the input, T1 (odd) or T2 (even)
        const bool rev = nsteps > 1 && !(step & 1);   // even steps sweep every segment bottom-up (see the consumers)
        if (step > 1) {   // wait until every halo partner has published step - 1 (bounded spin: a lost partner must not hang the GPU)
            const int nd = sdep[0];
            const unsigned long long want = p.epoch + (unsigned long long)(step - 1);
            for (int d = lane; d < nd; d += 32) {
                const unsigned long long* f = p.flags + sdep[1 + d];
                unsigned long long v; int spins = 0;
                do {
                    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(f) : "memory");
                    if (v >= want) break;
                    __nanosleep(64);
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
            const int xb = strip_x(sx, Lx, p.nsx), xe = (sx + 1 == p.nsx) ? Lx : strip_x(sx + 1, Lx, p.nsx);
            const bool edgeL = l.px && xb == 0, edgeR = l.px && xe == Lx;
            const int nside = (edgeL ? 1 : 0) + (edgeR ? 1 : 0);
            const int Q = (nrows + 2 + RC - 1) / RC;
            // TMA needs a 16-byte aligned box start: the inner coordinate (in doubles) must be even, so the box
            // starts two sites left of the (even) strip start: sites xb-2 .. xb+61 = halo at 1, strip at 2..w+1, halo at w+2
            const int x3 = 3 * (xb - 2);
            for (int j = 0; j < Q; ++j, ++n) {
                const unsigned s = n % S, ph = (n / S) & 1u;
                const int r0 = j * RC - 1;
                const int nvalid = (nrows + 1 - r0) < RC ? (nrows + 1 - r0) : RC;
                // forward: row index r lives at y = y_start + r; reversed: at y = y_end - 1 - r, and a chunk box (ascending y)
                // then holds descending r, so row i of the stage sits in slot RC - 1 - i
                const int y_end = y_start + nrows;
                const int y0 = rev ? y_end - r0 - RC : y_start + r0;          // first (lowest-y) row of the full chunk box
                const bool chunk_ok = (nvalid == RC) && (!l.py || (y0 >= 0 && y0 + RC <= Ly));
                if (lane == 0) {
                    mbar_wait(&empty[s], ph ^ 1u);
                    const int nf = eg ? 1 : F, nfs = eg ? 1 : NFS;   // energy / gradient mode stages m alone
                    mbar_expect_tx(&full[s], (unsigned)nvalid * (nf * ROWD * 8 + nside * nfs * SIDED * 8 + (API ? 0 : CROWD * 8)));
                }
                __syncwarp();
                const int nops = (chunk_ok ? 1 : nvalid) * KINDS;
                for (int t = lane; t < nops; t += 32) {
                    const int i = t / KINDS, kind = t - i * KINDS;     // i: row inside the stage (0 on the chunk path)
                    int y = chunk_ok ? y0 : (rev ? y_end - 1 - (r0 + i) : y_start + r0 + i);
                    if (!chunk_ok && l.py) { if (y < 0) y += Ly; else if (y >= Ly) y -= Ly; }
                    const int slot = s * RC + (chunk_ok ? 0 : (rev ? RC - 1 - i : i));
                    if (kind < F) {
                        const int f = kind;
                        if (eg && f > 0) continue;
                        const CUtensorMap* mp = f == 0 ? (chunk_ok ? &maps.m_chunk : &maps.m_row) : (chunk_ok ? &vs.chunk : &vs.row);
                        tma_load_3d(smain + ((size_t)f * NSLOT + slot) * ROWD, mp, &full[s], x3, y, f == 0 ? 0 : K * grp + f - 1);
                    } else if (kind < F + 2 * NFS) {
                        const int q = kind - F, right = q >= NFS, fi = right ? q - NFS : q, f = fi + FS0;
                        if (eg && f > 0) continue;
                        if (right ? edgeR : edgeL) {
                            const CUtensorMap* ms = f == 0 ? (chunk_ok ? &maps.m_schunk : &maps.m_srow) : (chunk_ok ? &vs.schunk : &vs.srow);
                            tma_load_3d((right ? sR : sL) + ((size_t)fi * NSLOT + slot) * SIDED, ms, &full[s], right ? 0 : 3 * Lx - SIDED, y,
                                        f == 0 ? 0 : K * grp + f - 1);
                        }
                    } else {
                        tma_load_3d(sc + (size_t)slot * CROWD, chunk_ok ? &maps.c_chunk : &maps.c_row, &full[s], xb - 2, y, 0);
                    }
                }
            }
            pos += nrows;
        }
        }   // step
        return;
    }

    // ==================================================================== consumers
    // Address arithmetic is hoisted out of the block loop: per sub-segment a thread fixes where its three stencil columns
    // live (the main row box or, on the edge strips of a periodic lattice, a wrap side box: offset, row pitch and field
    // stride of each), per block only the four row-slot indices change.  (The first version recomputed slots, pitches and
    // 64-bit site indices per load: 330 of its 800 instructions per block were integer work.)
    const int ch = warp & 1, rp = warp >> 1;
    const int col = ch * 32 + lane;
    const long long N = (long long)Lx * Ly;
    double waw[NK > 0 ? NK : 1];
#pragma unroll
    for (int t = 0; t < NK; ++t) waw[t] = 0.0;
    const d3 muB = mk3(l.mu * l.Bx, l.mu * l.By, l.mu * l.Bz);
    const bool use_coef = !API && p.cheb && p.coef;
    struct Role { int off, pitch, fstr; };   // doubles: field-0 / slot-0 offset from smain, row-slot pitch, field stride

    unsigned n = 0;
    for (int step = 1; step <= nsteps; ++step) {
    // per-step operands: coefficients, three-term operand Y_{step-2} (same-site, same-thread data), destination
    const double* cf = use_coef ? p.coef + 4 * (step - 1) : nullptr;
    const double ch_alpha = cf ? cf[0] : p.alpha, ch_c0 = cf ? cf[1] : p.c0, ch_beta = cf ? cf[2] : p.beta;
    const size_t goff = (size_t)grp * K * 3 * N;          // this column group's slice of the blocks (single-step launches)
    const double* Ustep = p.U ? p.U + goff : nullptr;
    double* outp = p.out ? p.out + goff : nullptr;
    if (nsteps > 1) {
        Ustep = step == 1 ? nullptr : (step == 2 ? p.V0 : ((step & 1) ? p.T1 : p.T2));     // Y_{step-2}
        outp = step == nsteps ? p.out : ((step & 1) ? p.T1 : p.T2);                          // Y_step (in place over Y_{step-2})
    }
    const bool use_u = !API && p.cheb && Ustep && ch_beta != 0.0;   // product-form steps (beta = 0) never read Y_{step-2}
    // Even steps of a multi-step launch sweep bottom-up: the rows a CTA wrote (and read) last in step i are the first it
    // touches in step i + 1, so a good part of the 128 MB/step footprint is still in the 126 MB L2.  A reversed sweep is
    // the same code on the point-reflected lattice: row order reversed, left and right neighbours swapped, D -> -D
    // (the stencil is inversion symmetric up to the sign of the DMI vectors, D_{-delta} = -D_delta).
    const bool rev = nsteps > 1 && !(step & 1);
    Lat ls = p.l;
    if (rev) ls.D = -ls.D;
    long long pos = lo;
    while (pos < hi) {
        const int sx = (int)(pos / Ly), y_start = (int)(pos - (long long)sx * Ly);
        const int nrows = (int)((hi - pos) < (long long)(Ly - y_start) ? (hi - pos) : (Ly - y_start));
        const int y_end = y_start + nrows;
        const int xb = strip_x(sx, Lx, p.nsx), xe = (sx + 1 == p.nsx) ? Lx : strip_x(sx + 1, Lx, p.nsx);
        const int w = xe - xb;
        const bool active = col < w;
        const bool wrapL = l.px && xb == 0 && col == 0;        // x - 1 comes from the wrap side box
        const bool wrapR = l.px && xe == Lx && col == w - 1;   // x + 1 comes from the wrap side box
        Role rM, rC, rP;                                        // columns x - 1, x, x + 1
        rC.off = 3 * (col + 2); rC.pitch = ROWD; rC.fstr = NSLOT * ROWD;
        rM.off = 3 * (col + 1); rM.pitch = ROWD; rM.fstr = NSLOT * ROWD;
        rP.off = 3 * (col + 3); rP.pitch = ROWD; rP.fstr = NSLOT * ROWD;
        if (wrapL) { rM.off = (int)(sL - smain) + 13 - FS0 * NSLOT * SIDED; rM.pitch = SIDED; rM.fstr = NSLOT * SIDED; }
        if (wrapR) { rP.off = (int)(sR - smain) - FS0 * NSLOT * SIDED; rP.pitch = SIDED; rP.fstr = NSLOT * SIDED; }
        const Role rL = rev ? rP : rM, rR = rev ? rM : rP;     // stencil frame of the sweep
        const int Q = (nrows + 2 + RC - 1) / RC, nb = (nrows + RC - 1) / RC;
        // this thread's first site and the step to its second row / to the next block, in doubles
        const long long e0 = 3 * ((long long)(rev ? y_end - 1 - 2 * rp : y_start + 2 * rp) * Lx + xb + col);
        const long long eRow = rev ? -3ll * Lx : 3ll * Lx, eBlk = RC * eRow;

        mbar_wait(&full[n % S], (n / S) & 1u);
        // The three-term operand U is read straight from global memory (no reuse, so it does not ride the ring): the loads
        // for block j + 1 are issued at the end of block j, into the registers block j has just finished with, and have
        // the stencil arithmetic of block j + 1 to arrive in.  out may alias U: a site's U is read and written by the same thread.
        d3 uA[K], uB[K];
        auto load_u = [&](int jb) {
            const int r = jb * RC + 2 * rp;
            if (use_u && active && r < nrows) {
                const double* up = Ustep + e0 + (long long)jb * eBlk;
#pragma unroll
                for (int a = 0; a < K; ++a) {
                    uA[a] = ld3(up + (size_t)a * 3 * N, 0);
                    uB[a] = (r + 1 < nrows) ? ld3(up + (size_t)a * 3 * N + eRow, 0) : mk3(0.0, 0.0, 0.0);
                }
            }
        };
        load_u(0);
        int cur = (int)(n % S);
        for (int j = 0; j < nb; ++j) {
            const int nxt = cur + 1 == S ? 0 : cur + 1;
            if (j + 1 < Q) mbar_wait(&full[nxt], ((n + j + 1) / S) & 1u);
            const int rA = j * RC + 2 * rp;
            if (active && rA < nrows) {
                const bool haveB = rA + 1 < nrows;
                int sr[4];   // row slots of stencil rows rA - 1 .. rA + 2 (stage rows 2 rp .. 2 rp + 3, the last ones in the next stage)
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const int t = 2 * rp + q;
                    sr[q] = t < RC ? cur * RC + (rev ? RC - 1 - t : t) : nxt * RC + (rev ? RC - 1 - (t - RC) : t - RC);
                }
                double* oA_p = outp + e0 + (long long)j * eBlk;
                double cA = 0.0, cB = 0.0;
                if (!API) { cA = sc[sr[1] * CROWD + col + 2]; cB = sc[sr[2] * CROWD + col + 2]; }
                // field 0: m.  API: all ten sites (projection of the neighbours + stencil for c); SOLVER: centres only.
                d3 m0C, m0R, m1L, m1C, m1R, m2L, m2C, m2R, m3L, m3C;
                m1C = lds3(smain + rC.off + sr[1] * ROWD);
                m2C = lds3(smain + rC.off + sr[2] * ROWD);
                if (API) {
                    m0C = lds3(smain + rC.off + sr[0] * ROWD); m0R = lds3(smain + rR.off + sr[0] * rR.pitch);
                    m1L = lds3(smain + rL.off + sr[1] * rL.pitch); m1R = lds3(smain + rR.off + sr[1] * rR.pitch);
                    m2L = lds3(smain + rL.off + sr[2] * rL.pitch); m2R = lds3(smain + rR.off + sr[2] * rR.pitch);
                    m3L = lds3(smain + rL.off + sr[3] * rL.pitch); m3C = lds3(smain + rC.off + sr[3] * ROWD);
                    const d3 LmA = stencil_apply(ls, m1R, m1L, m2C, m0C, m2L, m0R, m1C.z);
                    const d3 LmB = stencil_apply(ls, m2R, m2L, m3C, m1C, m3L, m1R, m2C.z);
                    cA = dot3(m1C, LmA) - dot3(m1C, muB);
                    cB = dot3(m2C, LmB) - dot3(m2C, muB);
                    if (eg && p.vdot) {   // F = -P(Lm - mu B) and its dot with v (moto_mmf_step, kr = 1)
                        const double* vp = p.vdot + e0 + (long long)j * eBlk;
                        const d3 FA = scale3(-1.0, axpy3(-cA, m1C, sub3(LmA, muB)));
                        waw[0] += dot3(FA, ld3(vp, 0));
                        st3(oA_p, 0, FA);
                        if (haveB) {
                            const d3 FB = scale3(-1.0, axpy3(-cB, m2C, sub3(LmB, muB)));
                            waw[0] += dot3(FB, ld3(vp + eRow, 0));
                            st3(oA_p + eRow, 0, FB);
                        }
                    } else if (eg) {   // E = sum_i (m.Lm / 2 - mu m.B), g = P(Lm - mu B), c = m.g: the m-stencil is all there is to do
                        waw[0] += 0.5 * dot3(m1C, LmA) - dot3(m1C, muB);
                        if (haveB) waw[0] += 0.5 * dot3(m2C, LmB) - dot3(m2C, muB);
                        if (p.out) {
                            st3(oA_p, 0, axpy3(-cA, m1C, sub3(LmA, muB)));
                            if (haveB) st3(oA_p + eRow, 0, axpy3(-cB, m2C, sub3(LmB, muB)));
                        }
                        if (p.c_out && !p.vdot) {
                            const long long iA = (e0 + (long long)j * eBlk) / 3;
                            p.c_out[iA] = cA;
                            if (haveB) p.c_out[iA + eRow / 3] = cB;
                        }
                    }
                }
                if (!eg) {
                d3 vA[K], hA[K], vB[K], hB[K];
#pragma unroll
                for (int a = 0; a < K; ++a) {
                    const double* bL = smain + rL.off + (a + 1) * rL.fstr;
                    const double* bC = smain + rC.off + (a + 1) * rC.fstr;
                    const double* bR = smain + rR.off + (a + 1) * rR.fstr;
                    d3 u0C = lds3(bC + sr[0] * ROWD), u0R = lds3(bR + sr[0] * rR.pitch);
                    d3 u1L = lds3(bL + sr[1] * rL.pitch), u1C = lds3(bC + sr[1] * ROWD), u1R = lds3(bR + sr[1] * rR.pitch);
                    d3 u2L = lds3(bL + sr[2] * rL.pitch), u2C = lds3(bC + sr[2] * ROWD), u2R = lds3(bR + sr[2] * rR.pitch);
                    d3 u3L = lds3(bL + sr[3] * rL.pitch), u3C = lds3(bC + sr[3] * ROWD);
                    if (API) {
                        u0C = proj3(m0C, u0C); u0R = proj3(m0R, u0R);
                        u1L = proj3(m1L, u1L); u1C = proj3(m1C, u1C); u1R = proj3(m1R, u1R);
                        u2L = proj3(m2L, u2L); u2C = proj3(m2C, u2C); u2R = proj3(m2R, u2R);
                        u3L = proj3(m3L, u3L); u3C = proj3(m3C, u3C);
                    }
                    const d3 LA = stencil_apply(ls, u1R, u1L, u2C, u0C, u2L, u0R, u1C.z);
                    const d3 LB = stencil_apply(ls, u2R, u2L, u3C, u1C, u3L, u1R, u2C.z);
                    vA[a] = u1C; vB[a] = u2C;
                    hA[a] = axpy3(-cA, u1C, proj3(m1C, LA));
                    hB[a] = axpy3(-cB, u2C, proj3(m2C, LB));
                }
                if (NK > 0 && p.waw) {
                    int t = 0;
#pragma unroll
                    for (int a = 0; a < K; ++a)
#pragma unroll
                        for (int b = a; b < K; ++b) {
                            waw[t] += dot3(vA[a], hA[b]);
                            if (haveB) waw[t] += dot3(vB[a], hB[b]);
                            ++t;
                        }
                }
#pragma unroll
                for (int a = 0; a < K; ++a) {
                    d3 oA = hA[a], oB = hB[a];
                    if (!API && p.cheb) {
                        oA = scale3(ch_alpha, axpy3(-ch_c0, vA[a], oA));
                        oB = scale3(ch_alpha, axpy3(-ch_c0, vB[a], oB));
                        if (use_u) {
                            oA = axpy3(ch_beta, uA[a], oA);
                            oB = axpy3(ch_beta, uB[a], oB);
                        }
                    }
                    st3(oA_p + (size_t)a * 3 * N, 0, oA);
                    if (haveB) st3(oA_p + (size_t)a * 3 * N + eRow, 0, oB);
                }
                }   // !eg
            }
            if (j + 1 < nb) load_u(j + 1);
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[cur]);
            cur = nxt;
        }
        if (Q > nb) { __syncwarp(); if (lane == 0) mbar_arrive(&empty[cur]); }
        n += Q;
        pos += nrows;
    }
    if (nsteps > 1) {   // publish "this CTA has finished step": every consumer's stores first, then one release store
        // (one fence by the publishing thread after the CTA barrier covers every consumer's stores by cumulativity -- the
        // pattern of a cooperative-groups grid sync; a fence per thread cost ~2 us per step)
        asm volatile("bar.sync 1, %0;" ::"n"(NCW * 32) : "memory");
        if (threadIdx.x == 0) {
            __threadfence();
            const unsigned long long v = p.epoch + (unsigned long long)step;
            asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p.flags + blockIdx.x), "l"(v) : "memory");
        }
    }
    }   // step

    if (NK > 0 && p.waw) {  // fixed-order reduction over the 320 consumer threads (named barrier 1: the producer warp has left)
#pragma unroll
        for (int t = 0; t < NK; ++t) {
            const double v = warp_sum(waw[t]);
            if (lane == 0) sred[warp * 4 + t] = v;
        }
        asm volatile("bar.sync 1, %0;" ::"n"(NCW * 32) : "memory");
        if (threadIdx.x < NK) {
            double s = 0.0;
            for (int wv = 0; wv < NCW; ++wv) s += sred[wv * 4 + threadIdx.x];
            p.waw[(size_t)blockIdx.x * NK + threadIdx.x] = s;
        }
        if (eg && p.e_out) {   // NK = 1.  Which CTA arrives last varies, the order of the sum does not.
            if (threadIdx.x == 0) { __threadfence(); sdep[0] = atomicAdd(p.counter, 1u) == gridDim.x - 1 ? 1 : 0; }
            asm volatile("bar.sync 1, %0;" ::"n"(NCW * 32) : "memory");
            if (sdep[0] && warp == 0) {
                __threadfence();
                double s = 0.0;
                for (unsigned b = lane; b < gridDim.x; b += 32) s += __ldcg(p.waw + b);
                s = warp_sum(s);
                if (lane == 0) { *p.e_out = s; *p.counter = 0u; }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
bool encode_vset(VSet* v, const double* base, int Lx, int Ly, int nvec) {
    return encode(&v->chunk, base, Lx, Ly, nvec, ROWD, RC) && encode(&v->row, base, Lx, Ly, nvec, ROWD, 1) &&
           encode(&v->schunk, base, Lx, Ly, nvec, SIDED, RC) && encode(&v->srow, base, Lx, Ly, nvec, SIDED, 1);
}

template <int K, bool API>
bool launch(moto_ctx* c, const Maps& maps, const KParams& p, int grid) {
    using C = Cfg<K, API>;
    static std::atomic<unsigned long long> attr_seen{0};   // per device, thread-safe
    if (!ensure_smem_attr(k_hvp_tma<K, API>, C::SMEM, attr_seen)) return false;
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(NTHREADS); cfg.dynamicSmemBytes = C::SMEM; cfg.stream = c->stream;
    cudaLaunchAttribute attr[1];
    if (p.nsteps > 1) {   // CTAs wait on each other's flags: they must all be resident
        attr[0].id = cudaLaunchAttributeCooperative;
        attr[0].val.cooperative = 1;
    } else {
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
    }
    cfg.attrs = attr; cfg.numAttrs = 1;
    if (cudaLaunchKernelEx(&cfg, k_hvp_tma<K, API>, maps, p) == cudaSuccess) return true;
    (void)cudaGetLastError();   // the caller falls back to another path: do not leave the launch error sticky
    return false;
}

}  // namespace

bool spin_tma_applicable(const moto_ctx* c) {
    if (c->kind != MOTO_KIND_TRI2D || c->nsh > 0) return false;   // general neighbour shells take spin_shells.cu
    const int Lx = c->lat.Lx, Ly = c->lat.Ly;
    if (c->opts.hvp_path == 1) return false;                  // hvp_path = generic
    if ((Lx & 1) || Lx < 8 || Ly < 1) return false;          // row stride 24 Lx must be a multiple of 16 B; side box needs 16 doubles
    if (c->opts.hvp_path == 2) return true;                   // hvp_path = tma (forced, tests)
    return (long long)Lx * Ly >= 16384;                       // small lattices are launch-latency bound: generic kernel
}

int spin_tma_grid(const moto_ctx* c) {
    const int Lx = c->lat.Lx, Ly = c->lat.Ly;
    const int nsx = (Lx + TXMAX - 1) / TXMAX;
    const long long total = (long long)nsx * Ly;
    long long g = (total + RC - 1) / RC;
    return (int)(g > MOTO_NUM_SMS ? MOTO_NUM_SMS : (g < 1 ? 1 : g));
}

// Extended entry: SOLVER mode when cvec != NULL (input must be tangent), API mode otherwise.
// waw_partials: optional [spin_tma_grid][k(k+1)/2].  cheb: out = alpha (HV - c0 V) + beta U (U may be NULL).
// Returns the number of kernels launched, 0 if the path does not apply (caller falls back), -1 on error.
int spin_hvp_tma_ex(moto_ctx* c, const double* m, const double* cvec, const double* V, int k, double* HV, const int* d_done,
                    double* waw_partials, int cheb, double alpha, double c0, double beta, const double* U, const double* d_coef) {
    if (!spin_tma_applicable(c)) return 0;
    if (((uintptr_t)m & 15) || ((uintptr_t)V & 15) || ((uintptr_t)cvec & 15)) return 0;
    if (waw_partials && k > 2) return 0;
    const int Lx = c->lat.Lx, Ly = c->lat.Ly;
    const size_t bs = (size_t)3 * c->N;
    int launches = 0, a_first = 0;
    if (k >= 4 && !waw_partials) {
        // all column pairs in ONE launch, pair g on its own share of the SMs (KParams::gpair): below ~10^5 sites a launch is its
        // ramp and tail, and k / 2 of them in a row cost k / 2 times that (moto_hvp at cfg 2, k = 6: 19.3 us in three launches)
        const int ng = k / 2, cap = MOTO_NUM_SMS / ng, g1 = spin_tma_grid(c), gp = g1 < cap ? g1 : cap;
        Maps maps;
        memset(&maps, 0, sizeof(maps));
        bool ok = gp >= 1 && encode(&maps.m_chunk, m, Lx, Ly, 1, ROWD, RC) && encode(&maps.m_row, m, Lx, Ly, 1, ROWD, 1) &&
                  encode(&maps.m_schunk, m, Lx, Ly, 1, SIDED, RC) && encode(&maps.m_srow, m, Lx, Ly, 1, SIDED, 1) &&
                  encode_vset(&maps.vset[0], V, Lx, Ly, 2 * ng);
        if (ok && cvec) ok = encode(&maps.c_chunk, cvec, Lx, Ly, 1, CROWD, RC, 1) && encode(&maps.c_row, cvec, Lx, Ly, 1, CROWD, 1, 1);
        if (ok) {
            KParams p;
            p.l = make_lat(c);
            p.nsx = (Lx + TXMAX - 1) / TXMAX;
            p.total = (long long)p.nsx * Ly;
            p.cvec = cvec; p.out = HV; p.U = U;
            p.alpha = alpha; p.c0 = c0; p.beta = beta; p.cheb = cheb; p.coef = d_coef;
            p.waw = nullptr; p.done = d_done;
            p.nsteps = 1; p.V0 = nullptr; p.T1 = p.T2 = nullptr; p.flags = nullptr; p.epoch = 0; p.err = nullptr;
            p.gpair = gp;
            if (cvec ? launch<2, false>(c, maps, p, gp * ng) : launch<2, true>(c, maps, p, gp * ng)) { ++launches; a_first = 2 * ng; }
        }
    }
    for (int a0 = a_first; a0 < k; a0 += 2) {
        const int kk = (k - a0) >= 2 ? 2 : 1;
        Maps maps;
        memset(&maps, 0, sizeof(maps));
        bool ok = encode(&maps.m_chunk, m, Lx, Ly, 1, ROWD, RC) && encode(&maps.m_row, m, Lx, Ly, 1, ROWD, 1) &&
                  encode(&maps.m_schunk, m, Lx, Ly, 1, SIDED, RC) && encode(&maps.m_srow, m, Lx, Ly, 1, SIDED, 1) &&
                  encode_vset(&maps.vset[0], V + a0 * bs, Lx, Ly, kk);
        if (ok && cvec) ok = encode(&maps.c_chunk, cvec, Lx, Ly, 1, CROWD, RC, 1) && encode(&maps.c_row, cvec, Lx, Ly, 1, CROWD, 1, 1);
        if (!ok) return launches ? -1 : 0;
        KParams p;
        p.l = make_lat(c);
        p.nsx = (Lx + TXMAX - 1) / TXMAX;
        p.total = (long long)p.nsx * Ly;
        p.cvec = cvec; p.out = HV + a0 * bs;
        p.U = U ? U + a0 * bs : nullptr;
        p.alpha = alpha; p.c0 = c0; p.beta = beta; p.cheb = cheb; p.coef = d_coef;
        p.waw = waw_partials; p.done = d_done;
        p.nsteps = 1; p.V0 = nullptr; p.T1 = p.T2 = nullptr; p.flags = nullptr; p.epoch = 0; p.err = nullptr;
        const int grid = spin_tma_grid(c);
        bool l_ok;
        if (cvec) l_ok = kk == 2 ? launch<2, false>(c, maps, p, grid) : launch<1, false>(c, maps, p, grid);
        else l_ok = kk == 2 ? launch<2, true>(c, maps, p, grid) : launch<1, true>(c, maps, p, grid);
        if (!l_ok) return launches ? -1 : 0;
        ++launches;
    }
    return launches;
}

// Energy, tangent-projected gradient and c_i = m_i . g_i through the TMA-staged kernel (its <1, API> instantiation with only m in the
// ring): one pass over m, 24 B/site in and 24 (+ 8) out.  d_E, d_g, d_c may each be NULL.  Returns the number of launches, 0 if the
// path does not apply (the caller takes k_energy_grad).  Lattices below 2^18 sites stay on k_energy_grad (65 536 sites: 17 vs 21 us).
static int eg_launch(moto_ctx* c, const double* m, double* d_sum, double* d_out, double* d_c, const double* vdot) {
    if (!spin_tma_applicable(c) || ((uintptr_t)m & 15)) return 0;
    if (c->opts.hvp_path != 2 && c->N < (1 << 18)) return 0;
    const int Lx = c->lat.Lx, Ly = c->lat.Ly;
    Maps maps;
    memset(&maps, 0, sizeof(maps));
    bool ok = encode(&maps.m_chunk, m, Lx, Ly, 1, ROWD, RC) && encode(&maps.m_row, m, Lx, Ly, 1, ROWD, 1) &&
              encode(&maps.m_schunk, m, Lx, Ly, 1, SIDED, RC) && encode(&maps.m_srow, m, Lx, Ly, 1, SIDED, 1) &&
              encode_vset(&maps.vset[0], m, Lx, Ly, 1);   // never loaded in this mode; a valid descriptor for the prefetch
    if (!ok) return 0;
    KParams p;
    p.l = make_lat(c);
    p.nsx = (Lx + TXMAX - 1) / TXMAX;
    p.total = (long long)p.nsx * Ly;
    p.cvec = nullptr; p.out = d_out; p.U = nullptr;
    p.alpha = p.c0 = p.beta = 0.0; p.cheb = 0; p.coef = nullptr;
    p.waw = d_sum ? c->partials : nullptr; p.done = nullptr;
    p.nsteps = 1; p.V0 = nullptr; p.T1 = p.T2 = nullptr; p.flags = nullptr; p.epoch = 0; p.err = nullptr;
    p.eg = 1; p.c_out = d_c; p.vdot = vdot;
    p.e_out = d_sum; p.counter = reinterpret_cast<unsigned*>(c->flags + 500);   // flags: 512 words, zeroed at create; the K1 launches use < 148
    const int grid = spin_tma_grid(c);
    return launch<1, true>(c, maps, p, grid) ? 1 : 0;
}

int spin_energy_grad_tma(moto_ctx* c, const double* m, double* d_E, double* d_g, double* d_c) { return eg_launch(c, m, d_E, d_g, d_c, nullptr); }

// Pass 1 of the reflected-force step with one mode (moto_mmf_step, kr = 1): Fbuf = F = -P g and *d_alpha = F . v in one launch of
// the same kernel.  Returns 1, or 0 if the path does not apply (the caller takes k_mmf_pass1).
int spin_mmf_pass1_tma(moto_ctx* c, const double* m, const double* v, double* Fbuf, double* d_alpha) {
    if (!v || !Fbuf || !d_alpha) return 0;
    return eg_launch(c, m, d_alpha, Fbuf, nullptr, v);
}

template <int K>
static int coop_limit_of() {
    using C = Cfg<K, false>;
    int dev = 0, sms = 0, per_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(k_hvp_tma<K, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM) != cudaSuccess) return -1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_hvp_tma<K, false>, NTHREADS, C::SMEM) != cudaSuccess) return -1;
    return sms * per_sm;
}
int spin_tma_coop_limit(int k) { return k == 2 ? coop_limit_of<2>() : coop_limit_of<1>(); }

// The whole Chebyshev recurrence of one operator application in ONE persistent cooperative launch:
// OUT = Y_d with Y_0 = V, Y_i = alpha_i (Hess[Y_{i-1}] - c0 Y_{i-1}) + beta_i Y_{i-2}, coefficients at d_coef + 4 (i - 1)
// (device memory), Y_1..Y_{d-1} in the context's T1/T2 blocks.  k <= 2, d >= 2.  Returns launches or 0 if not applicable.
int spin_cheb_multistep(moto_ctx* c, const double* m, const double* cvec, const double* V, int k, int d, double* OUT,
                        const double* d_coef, const int* d_done) {
    if (!spin_tma_applicable(c) || k > 2 || d < 2 || !c->T1 || !cvec) return 0;
    if (((uintptr_t)m & 15) || ((uintptr_t)V & 15) || ((uintptr_t)cvec & 15)) return 0;
    const int Lx = c->lat.Lx, Ly = c->lat.Ly;
    const int grid = spin_tma_grid(c);
    if (c->coop_max_ctas == 0) c->coop_max_ctas = spin_tma_coop_limit(k);
    if (grid > c->coop_max_ctas) return 0;
    Maps maps;
    memset(&maps, 0, sizeof(maps));
    bool ok = encode(&maps.m_chunk, m, Lx, Ly, 1, ROWD, RC) && encode(&maps.m_row, m, Lx, Ly, 1, ROWD, 1) &&
              encode(&maps.m_schunk, m, Lx, Ly, 1, SIDED, RC) && encode(&maps.m_srow, m, Lx, Ly, 1, SIDED, 1) &&
              encode(&maps.c_chunk, cvec, Lx, Ly, 1, CROWD, RC, 1) && encode(&maps.c_row, cvec, Lx, Ly, 1, CROWD, 1, 1) &&
              encode_vset(&maps.vset[0], V, Lx, Ly, k) && encode_vset(&maps.vset[1], c->T1, Lx, Ly, k) &&
              encode_vset(&maps.vset[2], c->T2, Lx, Ly, k);
    if (!ok) return 0;
    KParams p;
    p.l = make_lat(c);
    p.nsx = (Lx + TXMAX - 1) / TXMAX;
    p.total = (long long)p.nsx * Ly;
    p.cvec = cvec; p.out = OUT; p.U = nullptr;
    p.alpha = p.c0 = p.beta = 0.0; p.cheb = 1; p.coef = d_coef;
    p.waw = nullptr; p.done = d_done;
    p.nsteps = d; p.V0 = V; p.T1 = c->T1; p.T2 = c->T2;
    p.flags = c->flags; c->epoch += 1024; p.epoch = c->epoch; p.err = &c->st->bad;
    const bool l_ok = k == 2 ? launch<2, false>(c, maps, p, grid) : launch<1, false>(c, maps, p, grid);
    return l_ok ? 1 : 0;
}

int spin_hvp_tma(moto_ctx* c, const double* m, const double* cvec, const double* V, int k, double* HV, int project_input,
                 const int* d_done) {
    // the two combinations the library uses: (no c, project) = API, (c, no project) = SOLVER
    if ((cvec != nullptr) == (project_input != 0)) return 0;
    int n = spin_hvp_tma_ex(c, m, cvec, V, k, HV, d_done, nullptr, 0, 0.0, 0.0, 0.0, nullptr, nullptr);
    return n < 0 ? 0 : n;
}
