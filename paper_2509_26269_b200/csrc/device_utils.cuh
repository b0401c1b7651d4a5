// device_utils.cuh -- small device helpers: 3-vectors, deterministic block/grid reductions.
#pragma once
#include <cuda_runtime.h>

struct d3 { double x, y, z; };

__device__ __forceinline__ d3 ld3(const double* __restrict__ p, long long i) {
    d3 r; r.x = p[3 * i]; r.y = p[3 * i + 1]; r.z = p[3 * i + 2]; return r;
}
__device__ __forceinline__ void st3(double* __restrict__ p, long long i, d3 v) {
    p[3 * i] = v.x; p[3 * i + 1] = v.y; p[3 * i + 2] = v.z;
}
__device__ __forceinline__ d3 mk3(double x, double y, double z) { d3 r; r.x = x; r.y = y; r.z = z; return r; }
__device__ __forceinline__ double dot3(d3 a, d3 b) { return fma(a.x, b.x, fma(a.y, b.y, a.z * b.z)); }
__device__ __forceinline__ d3 add3(d3 a, d3 b) { return mk3(a.x + b.x, a.y + b.y, a.z + b.z); }
__device__ __forceinline__ d3 sub3(d3 a, d3 b) { return mk3(a.x - b.x, a.y - b.y, a.z - b.z); }
__device__ __forceinline__ d3 axpy3(double a, d3 x, d3 y) { return mk3(fma(a, x.x, y.x), fma(a, x.y, y.y), fma(a, x.z, y.z)); }
__device__ __forceinline__ d3 scale3(double a, d3 x) { return mk3(a * x.x, a * x.y, a * x.z); }
// tangent projection  v - m (m.v)
__device__ __forceinline__ d3 proj3(d3 m, d3 v) { return axpy3(-dot3(m, v), m, v); }

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Block-wide sum of NV values per thread; result valid in thread 0.  Fixed order => deterministic.
// smem: at least NV * 32 doubles.
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double* smem) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        double s = warp_sum(v[i]);
        if (lane == 0) smem[i * 32 + warp] = s;
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            double s = (lane < nw) ? smem[i * 32 + lane] : 0.0;
            v[i] = warp_sum(s);
        }
    }
    __syncthreads();
}

// Final sum without a second launch: every CTA has written partials[blockIdx.x * stride + v] (v < nval) and then calls this with
// all its threads; the CTA that arrives last adds the partials of all gridDim.x CTAs -- one warp per value, lanes striding over
// the CTAs, shuffle tree: the order of k_final_sum, so the result does not depend on which CTA that is -- and leaves the arrival
// counter at 0 for the next launch.  out == nullptr: nothing to do.
__device__ __forceinline__ void last_cta_sum(const double* partials, int stride, int nval, double* out, int take_sqrt, unsigned* counter) {
    if (!out) return;
    __shared__ int s_last;
    if (threadIdx.x == 0) { __threadfence(); s_last = atomicAdd(counter, 1u) == gridDim.x - 1 ? 1 : 0; }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
    for (int v = warp; v < nval; v += nw) {
        double s = 0.0;
        for (unsigned b = lane; b < gridDim.x; b += 32) s += __ldcg(partials + (size_t)b * stride + v);
        s = warp_sum(s);
        if (lane == 0) out[v] = take_sqrt ? sqrt(s) : s;
    }
    if (threadIdx.x == 0) *counter = 0u;
}
