// cart_morse.cu -- K7: Cartesian pair-potential gradient + block HVP over a cell-list neighbour
// structure (the paper's Ni(111) portability case; Morse potential and cell list
// per BASELINE.json north_star (4) / configs[4]).
//
//   g_i     = sum_j phi'(r) n ,                    n = (x_i - x_j)/r (minimum image in-plane, open in z)
//   (Hv)_i  = sum_j [ phi'' n (n.dv) + (phi'/r)(dv - n (n.dv)) ],  dv = v_i - v_j ,  r < rc
// masked: fixed atoms carry v = 0 and get a zero output row (the paper's mask Omega).
//
// Structure: 2-D cell list over the periodic in-plane cell (the slab is thin in z) -> per-atom
// neighbour table with the pair coefficients (n, phi'', phi'/r, phi', phi - phi(rc)) stored once per
// configuration, so every HVP of an eigen-solve is a gather over ~57 stored pairs per atom.
// Deterministic: cells are sorted by atom id, neighbour order is fixed, reductions are fixed-order.
#include <string.h>
#include "common.cuh"
#include "device_utils.cuh"

void launch_mmf_pass2(moto_ctx* c, const double* x, const double* v, int kr, const double* Fbuf, const double* alpha,
                      double dt, double* x_out, int retract);
void launch_final_sum(moto_ctx* c, const double* partials, int nblk, int stride, int nval, double* out, int take_sqrt);

namespace {

constexpr int NC = 7;  // coefficients per pair
constexpr int MAXC = 4096;  // max cells

struct CartGeom {
    double a[2][2];    // cell rows
    double inv[2][2];  // inverse: s = d_xy * inv
    int ncx, ncy, Na;
    double De, alpha, r0, rc, phic;
};

__device__ __forceinline__ void frac(const CartGeom& g, double x, double y, double& s0, double& s1) {
    s0 = x * g.inv[0][0] + y * g.inv[1][0];
    s1 = x * g.inv[0][1] + y * g.inv[1][1];
}

__global__ void k_cell_assign(CartGeom g, const double* __restrict__ x, int* __restrict__ cell_of, int* __restrict__ cell_count) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.Na) return;
    double s0, s1;
    frac(g, x[3 * i], x[3 * i + 1], s0, s1);
    s0 -= floor(s0); s1 -= floor(s1);
    int cx = min(g.ncx - 1, (int)(s0 * g.ncx)), cy = min(g.ncy - 1, (int)(s1 * g.ncy));
    int c = cy * g.ncx + cx;
    cell_of[i] = c;
    atomicAdd(&cell_count[c], 1);
}

// exclusive scan of the cell counts (every CTA redoes it in shared memory, CTA 0 publishes it), then one thread per atom:
// its slot is cell_start + (number of lower-numbered atoms in the same cell), so every cell lists its atoms in ascending id
// (deterministic, no atomics); the rank loop reads cell_of through L1 (Na^2/2 broadcast loads in all: 1.3 M at 1607 atoms)
__global__ void __launch_bounds__(256) k_cell_build(int ncell, int Na, const int* __restrict__ cell_of, const int* __restrict__ cell_count,
                                                    int* __restrict__ cell_start, int* __restrict__ cell_atoms) {
    __shared__ int sstart[MAXC + 1];
    if (threadIdx.x == 0) {
        int s = 0;
        for (int c = 0; c < ncell; ++c) { sstart[c] = s; s += cell_count[c]; }
        sstart[ncell] = s;
    }
    __syncthreads();
    if (blockIdx.x == 0)
        for (int c = threadIdx.x; c <= ncell; c += blockDim.x) cell_start[c] = sstart[c];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= Na) return;
    const int c = cell_of[i];
    int rank = 0;
    for (int j = 0; j < i; ++j) rank += (cell_of[j] == c);
    cell_atoms[sstart[c] + rank] = i;
}

__device__ __forceinline__ void morse(const CartGeom& g, double r, double& phi, double& dphi, double& d2phi) {
    double e = exp(-g.alpha * (r - g.r0));
    phi = g.De * (e * e - 2.0 * e);
    dphi = g.De * (-2.0 * g.alpha * e * e + 2.0 * g.alpha * e);
    d2phi = g.De * (4.0 * g.alpha * g.alpha * e * e - 2.0 * g.alpha * g.alpha * e);
}

// one WARP per atom: neighbour table + pair coefficients.  The lanes test 32 candidates of a cell at a time; the accepted ones
// are compacted in candidate order with a ballot (same order as a serial scan: cells in (oy, ox) order, ascending atom id
// inside a cell), so the table is deterministic.
__global__ void __launch_bounds__(256) k_neighbours(CartGeom g, const double* __restrict__ x, const int* __restrict__ cell_of,
                                                    const int* __restrict__ cell_start, const int* __restrict__ cell_atoms,
                                                    int* __restrict__ nb_count, int* __restrict__ nb_idx, double* __restrict__ nb_coef,
                                                    int* __restrict__ overflow) {
    const int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (i >= g.Na) return;
    const double xi = x[3 * i], yi = x[3 * i + 1], zi = x[3 * i + 2];
    const int c = cell_of[i], cx = c % g.ncx, cy = c / g.ncx;
    const int nx = min(3, g.ncx), ny = min(3, g.ncy);
    int cnt = 0;
    for (int oy = 0; oy < ny; ++oy) {
        const int yy = (cy + oy - (ny == 3 ? 1 : 0) + g.ncy) % g.ncy;
        for (int ox = 0; ox < nx; ++ox) {
            const int xx = (cx + ox - (nx == 3 ? 1 : 0) + g.ncx) % g.ncx;
            const int cc = yy * g.ncx + xx;
            const int t0 = cell_start[cc], t1 = cell_start[cc + 1];
            for (int tb = t0; tb < t1; tb += 32) {
                const int t = tb + lane;
                bool in = false;
                int j = -1;
                double dx = 0.0, dy = 0.0, dz = 0.0, r2 = 0.0;
                if (t < t1) {
                    j = cell_atoms[t];
                    if (j != i) {
                        dx = xi - x[3 * j]; dy = yi - x[3 * j + 1]; dz = zi - x[3 * j + 2];
                        double s0, s1;
                        frac(g, dx, dy, s0, s1);
                        s0 -= rint(s0); s1 -= rint(s1);
                        dx = s0 * g.a[0][0] + s1 * g.a[1][0];
                        dy = s0 * g.a[0][1] + s1 * g.a[1][1];
                        r2 = dx * dx + dy * dy + dz * dz;
                        in = r2 < g.rc * g.rc;
                    }
                }
                const unsigned mask = __ballot_sync(0xffffffffu, in);
                const int slot = cnt + __popc(mask & ((1u << lane) - 1u));
                if (in && slot < MOTO_MAX_NEIGH) {
                    double r = sqrt(r2), phi, dphi, d2phi;
                    morse(g, r, phi, dphi, d2phi);
                    double ir = 1.0 / r;
                    size_t base = (size_t)i * NC * MOTO_MAX_NEIGH + slot;
                    nb_coef[base + 0 * MOTO_MAX_NEIGH] = dx * ir;
                    nb_coef[base + 1 * MOTO_MAX_NEIGH] = dy * ir;
                    nb_coef[base + 2 * MOTO_MAX_NEIGH] = dz * ir;
                    nb_coef[base + 3 * MOTO_MAX_NEIGH] = d2phi;
                    nb_coef[base + 4 * MOTO_MAX_NEIGH] = dphi * ir;
                    nb_coef[base + 5 * MOTO_MAX_NEIGH] = dphi;
                    nb_coef[base + 6 * MOTO_MAX_NEIGH] = phi - g.phic;
                    nb_idx[(size_t)i * MOTO_MAX_NEIGH + slot] = j;
                }
                cnt += __popc(mask);
            }
        }
    }
    if (lane == 0) {
        if (cnt > MOTO_MAX_NEIGH) { atomicExch(overflow, 1); cnt = MOTO_MAX_NEIGH; }
        nb_count[i] = cnt;
    }
}

// warp per atom: E_i = 1/2 sum_j (phi - phi_c),  g_i = sum_j phi' n  (zero row for fixed atoms)
__global__ void __launch_bounds__(256) k_cart_energy_grad(int Na, const uint8_t* __restrict__ fixed, const int* __restrict__ nb_count,
                                                          const double* __restrict__ nb_coef, double* __restrict__ g_out,
                                                          double* __restrict__ e_atom) {
    int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (i >= Na) return;
    const double* cf = nb_coef + (size_t)i * NC * MOTO_MAX_NEIGH;
    double gx = 0, gy = 0, gz = 0, e = 0;
    for (int n = lane; n < nb_count[i]; n += 32) {
        double dphi = cf[5 * MOTO_MAX_NEIGH + n];
        gx = fma(dphi, cf[n], gx); gy = fma(dphi, cf[MOTO_MAX_NEIGH + n], gy); gz = fma(dphi, cf[2 * MOTO_MAX_NEIGH + n], gz);
        e += cf[6 * MOTO_MAX_NEIGH + n];
    }
    gx = warp_sum(gx); gy = warp_sum(gy); gz = warp_sum(gz); e = warp_sum(e);
    if (lane == 0) {
        bool fx = fixed && fixed[i];
        if (g_out) { g_out[3 * i] = fx ? 0.0 : gx; g_out[3 * i + 1] = fx ? 0.0 : gy; g_out[3 * i + 2] = fx ? 0.0 : gz; }
        e_atom[i] = 0.5 * e;
    }
}

// warp per atom, all k columns per pass over the stored pairs
__global__ void __launch_bounds__(256) k_cart_hvp(int Na, int k, const uint8_t* __restrict__ fixed, const int* __restrict__ nb_count,
                                                  const int* __restrict__ nb_idx, const double* __restrict__ nb_coef,
                                                  const double* __restrict__ V, double* __restrict__ HV, const int* __restrict__ done,
                                                  const double* __restrict__ coef) {
    // coef != NULL: a product-form step of the filter recurrence (k_cheb_coef row {alpha, r, ...}): HV = alpha (H V - r V)
    // programmatic dependent launch: the next step's CTAs become resident while this one runs and wait here, so a step of the
    // recurrence does not pay the launch latency (the kernel itself is ~4 us at 1607 atoms)
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (done && *done) return;
    int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (i >= Na) return;
    const bool fxi = fixed && fixed[i];
    const double* cf = nb_coef + (size_t)i * NC * MOTO_MAX_NEIGH;
    const int* idx = nb_idx + (size_t)i * MOTO_MAX_NEIGH;
    double acc[MOTO_KMAX][3];
#pragma unroll
    for (int a = 0; a < MOTO_KMAX; ++a) acc[a][0] = acc[a][1] = acc[a][2] = 0.0;
    if (!fxi) {
        for (int n = lane; n < nb_count[i]; n += 32) {
            const int j = idx[n];
            const bool fxj = fixed && fixed[j];
            d3 nn = mk3(cf[n], cf[MOTO_MAX_NEIGH + n], cf[2 * MOTO_MAX_NEIGH + n]);
            const double d2 = cf[3 * MOTO_MAX_NEIGH + n], d1r = cf[4 * MOTO_MAX_NEIGH + n];
#pragma unroll
            for (int a = 0; a < MOTO_KMAX; ++a) {
                if (a < k) {
                    const double* v = V + (size_t)a * 3 * Na;
                    d3 dv = ld3(v, i);
                    if (!fxj) dv = sub3(dv, ld3(v, j));
                    double nd = dot3(nn, dv);
                    // phi'' n (n.dv) + (phi'/r)(dv - n (n.dv)) = (phi'' - phi'/r)(n.dv) n + (phi'/r) dv
                    double w = (d2 - d1r) * nd;
                    acc[a][0] += fma(w, nn.x, d1r * dv.x);
                    acc[a][1] += fma(w, nn.y, d1r * dv.y);
                    acc[a][2] += fma(w, nn.z, d1r * dv.z);
                }
            }
        }
    }
#pragma unroll
    for (int a = 0; a < MOTO_KMAX; ++a) {
        if (a < k) {
            double x = warp_sum(acc[a][0]), y = warp_sum(acc[a][1]), z = warp_sum(acc[a][2]);
            if (lane == 0) {
                d3 h = mk3(x, y, z);
                if (coef) h = scale3(coef[0], axpy3(-coef[1], ld3(V + (size_t)a * 3 * Na, i), h));
                st3(HV + (size_t)a * 3 * Na, i, h);
            }
        }
    }
}

__global__ void k_cart_mask(int Na, int k, const uint8_t* __restrict__ fixed, double* __restrict__ V) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= Na || !fixed || !fixed[i]) return;
    for (int a = 0; a < k; ++a) st3(V + (size_t)a * 3 * Na, i, mk3(0, 0, 0));
}

// F = -g (masked) ; partial dots alpha_a = F . v_a   (g already in Fbuf, negate in place)
__global__ void __launch_bounds__(256) k_cart_mmf_pass1(int Na, const double* __restrict__ v, int kr, double* __restrict__ Fbuf,
                                                        double* __restrict__ partials) {
    __shared__ double red[32 * MOTO_KMAX];
    double acc[MOTO_KMAX];
#pragma unroll
    for (int a = 0; a < MOTO_KMAX; ++a) acc[a] = 0.0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < Na; i += gridDim.x * blockDim.x) {
        d3 F = scale3(-1.0, ld3(Fbuf, i));
        st3(Fbuf, i, F);
#pragma unroll
        for (int a = 0; a < MOTO_KMAX; ++a)
            if (a < kr) acc[a] += dot3(F, ld3(v + (size_t)a * 3 * Na, i));
    }
    block_sum<MOTO_KMAX>(acc, red);
    if (threadIdx.x == 0)
        for (int a = 0; a < MOTO_KMAX; ++a) partials[blockIdx.x * MOTO_KMAX + a] = acc[a];
}

CartGeom make_geom(const moto_ctx* c) {
    CartGeom g;
    for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) g.a[a][b] = c->lat.cell[a][b];
    double det = g.a[0][0] * g.a[1][1] - g.a[0][1] * g.a[1][0];
    g.inv[0][0] = g.a[1][1] / det; g.inv[0][1] = -g.a[0][1] / det;
    g.inv[1][0] = -g.a[1][0] / det; g.inv[1][1] = g.a[0][0] / det;
    g.ncx = c->cl.ncx; g.ncy = c->cl.ncy; g.Na = c->N;
    g.De = c->mp.De; g.alpha = c->mp.alpha; g.r0 = c->mp.r0; g.rc = c->mp.rc;
    double e = exp(-g.alpha * (g.rc - g.r0));
    g.phic = g.De * (e * e - 2.0 * e);
    return g;
}

}  // namespace

// cells: as many as fit with perpendicular width >= rc along each cell vector (at most 64 x 64)
static void cart_cell_counts(const moto_lattice* lat, double rc, int* ncx, int* ncy, double* h0, double* h1) {
    const double (*a)[2] = lat->cell;
    double area = fabs(a[0][0] * a[1][1] - a[0][1] * a[1][0]);
    double l0 = sqrt(a[0][0] * a[0][0] + a[0][1] * a[0][1]), l1 = sqrt(a[1][0] * a[1][0] + a[1][1] * a[1][1]);
    *h0 = area / l1;  // width of the cell measured perpendicular to a1-lines (fractional coord 0)
    *h1 = area / l0;
    int nx = rc > 0 ? (int)(*h0 / rc) : 1, ny = rc > 0 ? (int)(*h1 / rc) : 1;
    *ncx = nx < 1 ? 1 : (nx > 64 ? 64 : nx);
    *ncy = ny < 1 ? 1 : (ny > 64 ? 64 : ny);
}

bool cart_geometry_ok(const moto_lattice* lat, double rc) {
    int nx, ny; double h0, h1;
    const double (*a)[2] = lat->cell;
    double area = fabs(a[0][0] * a[1][1] - a[0][1] * a[1][0]);
    if (!(area > 0)) return false;
    cart_cell_counts(lat, rc, &nx, &ny, &h0, &h1);
    return rc < 0.5 * h0 && rc < 0.5 * h1;  // minimum image by fractional rounding is exact below half the widths
}

static size_t al256(size_t x) { return (x + 255) & ~(size_t)255; }

size_t cart_lists_bytes(const moto_lattice* lat) {
    size_t Na = (size_t)lat->n_atoms;
    return al256(Na * 4) * 3 + al256((MAXC + 1) * 4) * 2 + al256(Na * MOTO_MAX_NEIGH * 4) +
           al256(Na * MOTO_MAX_NEIGH * NC * 8) + 256;
}

int cart_lists_carve(moto_ctx* c, char* base) {
    size_t Na = (size_t)c->N;
    char* p = base;
    c->cl.cell_of = (int*)p; p += al256(Na * 4);
    c->cl.cell_atoms = (int*)p; p += al256(Na * 4);
    c->cl.nb_count = (int*)p; p += al256(Na * 4);
    c->cl.cell_count = (int*)p; p += al256((MAXC + 1) * 4);
    c->cl.cell_start = (int*)p; p += al256((MAXC + 1) * 4);
    c->cl.nb_idx = (int*)p; p += al256(Na * MOTO_MAX_NEIGH * 4);
    c->cl.nb_coef = (double*)p; p += al256(Na * MOTO_MAX_NEIGH * NC * 8);
    c->cl.overflow = (int*)p; p += 256;
    double h0, h1;
    cart_cell_counts(&c->lat, c->mp.rc, &c->cl.ncx, &c->cl.ncy, &h0, &h1);
    c->cl.ncell = c->cl.ncx * c->cl.ncy;
    return 0;
}

int cart_build_lists(moto_ctx* c, const double* x) {
    CartGeom g = make_geom(c);
    const int Na = c->N, ncell = c->cl.ncell;
    cudaMemsetAsync(c->cl.cell_count, 0, (ncell + 1) * sizeof(int), c->stream);
    cudaMemsetAsync(c->cl.overflow, 0, sizeof(int), c->stream);
    k_cell_assign<<<(Na + 127) / 128, 128, 0, c->stream>>>(g, x, c->cl.cell_of, c->cl.cell_count);
    k_cell_build<<<(Na + 255) / 256, 256, 0, c->stream>>>(ncell, Na, c->cl.cell_of, c->cl.cell_count, c->cl.cell_start, c->cl.cell_atoms);
    k_neighbours<<<(Na * 32 + 255) / 256, 256, 0, c->stream>>>(g, x, c->cl.cell_of, c->cl.cell_start, c->cl.cell_atoms, c->cl.nb_count,
                                                       c->cl.nb_idx, c->cl.nb_coef, c->cl.overflow);
    return 3;
}

int cart_energy_grad(moto_ctx* c, const double* x, double* d_E, double* d_g) {
    (void)x;
    const int Na = c->N;
    double* e_atom = c->c;  // [N] scratch
    k_cart_energy_grad<<<(Na * 32 + 255) / 256, 256, 0, c->stream>>>(Na, c->lat.d_fixed, c->cl.nb_count, c->cl.nb_coef, d_g, e_atom);
    int n = 1;
    if (d_E) { launch_final_sum(c, e_atom, Na, 1, 1, d_E, 0); ++n; }
    return n;
}

static void launch_cart_hvp(moto_ctx* c, const double* V, int k, double* HV, const int* d_done, const double* coef) {
    const int Na = c->N;
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3((Na * 32 + 255) / 256); cfg.blockDim = dim3(256); cfg.dynamicSmemBytes = 0; cfg.stream = c->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    const uint8_t* fixed = c->lat.d_fixed;
    const int* nbc = c->cl.nb_count; const int* nbi = c->cl.nb_idx; const double* nbf = c->cl.nb_coef;
    if (cudaLaunchKernelEx(&cfg, k_cart_hvp, Na, k, fixed, nbc, nbi, nbf, V, HV, d_done, coef) != cudaSuccess) {
        (void)cudaGetLastError();
        k_cart_hvp<<<(Na * 32 + 255) / 256, 256, 0, c->stream>>>(Na, k, fixed, nbc, nbi, nbf, V, HV, d_done, coef);
    }
}

int cart_hvp(moto_ctx* c, const double* V, int k, double* HV, const int* d_done) {
    launch_cart_hvp(c, V, k, HV, d_done, nullptr);
    return 1;
}

// OUT = Y_d of the product-form filter recurrence Y_s = alpha_s (H - r_s) Y_{s-1}, Y_0 = V (masked), rows d_coef [d][4] on the device
// (k_cheb_coef): d launches of k_cart_hvp, Y_s alternating between T1 and T2.  The neighbour table must be current.
int cart_cheb_recurrence(moto_ctx* c, const double* V, int k, int d, double* OUT, const double* d_coef, const int* d_done) {
    if (!c->T1 || !c->T2) return -1;
    const double* in = V;
    for (int i = 1; i <= d; ++i) {
        double* out = (i == d) ? OUT : ((i & 1) ? c->T1 : c->T2);
        launch_cart_hvp(c, in, k, out, d_done, d_coef + 4 * (i - 1));
        in = out;
    }
    return d;
}

// upper bound of the spectrum for the filter interval: block Gershgorin, max_i 2 sum_j max(|phi''_ij|, |phi'_ij / r_ij|)
// (a pair block has eigenvalues phi'' along the bond and phi'/r across it, and sits once on the diagonal and once off it);
// per-CTA maxima to partial_max, *nmax_out = their number
__global__ void __launch_bounds__(256) k_cart_rowbound(int Na, const uint8_t* __restrict__ fixed, const int* __restrict__ nb_count,
                                                       const double* __restrict__ nb_coef, double* __restrict__ partial_max) {
    __shared__ double red[8];
    const int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double s = 0.0;
    if (i < Na && !(fixed && fixed[i])) {
        const double* cf = nb_coef + (size_t)i * NC * MOTO_MAX_NEIGH;
        for (int n = lane; n < nb_count[i]; n += 32) s += fmax(fabs(cf[3 * MOTO_MAX_NEIGH + n]), fabs(cf[4 * MOTO_MAX_NEIGH + n]));
    }
    s = 2.0 * warp_sum(s);
    if (lane == 0) red[warp] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double mx = 0.0;
        for (int w = 0; w < 8; ++w) mx = fmax(mx, red[w]);
        partial_max[blockIdx.x] = mx;
    }
}

int cart_rowbound(moto_ctx* c, double* partial_max, int* nmax_out) {
    const int Na = c->N, g = (Na * 32 + 255) / 256;
    if (g > 1024) return 0;   // (the caller's array of block maxima)
    *nmax_out = g;
    k_cart_rowbound<<<g, 256, 0, c->stream>>>(Na, c->lat.d_fixed, c->cl.nb_count, c->cl.nb_coef, partial_max);
    return 1;
}

int cart_mask(moto_ctx* c, double* V, int k) {
    if (!c->lat.d_fixed) return 0;
    k_cart_mask<<<(c->N + 127) / 128, 128, 0, c->stream>>>(c->N, k, c->lat.d_fixed, V);
    return 1;
}

int cart_mmf_step(moto_ctx* c, const double* x, const double* v, int kr, double dt, double* x_out, double* d_fnorm) {
    const int Na = c->N;
    int n = cart_energy_grad(c, x, nullptr, c->g);
    double* alpha = c->st->scal;
    int blocks = (Na + 255) / 256 < MOTO_RED_BLOCKS ? (Na + 255) / 256 : MOTO_RED_BLOCKS;
    k_cart_mmf_pass1<<<blocks, 256, 0, c->stream>>>(Na, v, kr, c->g, c->partials);
    launch_final_sum(c, c->partials, blocks, MOTO_KMAX, MOTO_KMAX, alpha, 0);
    launch_mmf_pass2(c, x, v, kr, c->g, alpha, dt, x_out, 0);
    n += 3;
    if (d_fnorm) { launch_final_sum(c, c->partials, MOTO_RED_BLOCKS, 1, 1, d_fnorm, 1); ++n; }
    return n;
}
