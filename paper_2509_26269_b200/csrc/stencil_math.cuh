// stencil_math.cuh -- the constant Euclidean Hessian stencil of Eq. 4 shared by the
// generic and the TMA-staged K1 kernels.  Product code: shares nothing with oracle/.
#pragma once
#include "common.cuh"
#include "device_utils.cuh"

struct Lat {
    int Lx, Ly, px, py;
    double J, D, K, Bx, By, Bz, mu;
};

static inline Lat make_lat(const moto_ctx* c) {
    Lat l;
    l.Lx = c->lat.Lx; l.Ly = c->lat.Ly; l.px = c->lat.pbc_x; l.py = c->lat.pbc_y;
    l.J = c->sp.J; l.D = c->sp.D; l.K = c->sp.K; l.mu = c->sp.mu;
    l.Bx = c->sp.B[0]; l.By = c->sp.B[1]; l.Bz = c->sp.B[2];
    return l;
}


#define SQ3H 0.86602540378443864676

// (L u)_i from the six neighbour values (zero where absent) and the site's own u_z
__device__ __forceinline__ d3 stencil_apply(const Lat& l, d3 up1, d3 um1, d3 up2, d3 um2, d3 up3, d3 um3, double uz) {
    d3 s = add3(add3(add3(up1, um1), add3(up2, um2)), add3(up3, um3));
    d3 d1 = sub3(up1, um1), d2 = sub3(up2, um2), d3_ = sub3(up3, um3);
    // sum_p rx_p d_p , sum_p ry_p d_p  with r1=(1,0), r2=(1/2,s), r3=(-1/2,s)
    double ax_z = d1.z + 0.5 * (d2.z - d3_.z);          // sum rx dz
    double ay_z = SQ3H * (d2.z + d3_.z);                // sum ry dz
    double axy = d1.x + 0.5 * (d2.x - d3_.x) + SQ3H * (d2.y + d3_.y);  // sum (rx dx + ry dy)
    d3 r;
    r.x = -2.0 * (l.J * s.x - l.D * ax_z);
    r.y = -2.0 * (l.J * s.y - l.D * ay_z);
    r.z = -2.0 * (l.J * s.z + l.D * axy) - 2.0 * l.K * uz;
    return r;
}

