// lobpcg_blocks.cuh -- the per-site arithmetic of the fused LOBPCG update for block sizes kb <= 2 (K5 + K2 + K3 of SURVEY 8(a)),
// shared by the streaming kernels of lobpcg_fast.cu and the persistent small-lattice solver of lobpcg_persistent.cu so that
// both compute the same numbers.  Product code: shares nothing with oracle/.
#pragma once
#include "common.cuh"
#include "device_utils.cuh"

namespace lob {

template <int KB> struct Tri {
    static constexpr int NS = 3 * KB;
    static constexpr int NT = NS * (NS + 1) / 2;   // upper triangle of one matrix
    static constexpr int NK = KB * (KB + 1) / 2;   // W^T A W block
    static constexpr int NEU = 2 * NT + KB;        // G_B tri, G_A tri, |r_j|^2
    __host__ __device__ static constexpr int idx(int i, int j) { return i * NS - i * (i - 1) / 2 + (j - i); }
};

struct Blk6 { double *X, *W, *P, *AX, *AW, *AP; };


// Accumulate the Gram entries of S = [s_0..s_{NS-1}], AS = [a_0..] for one scalar element.
// skip_waw: leave the (W, AW) block untouched (it comes from K1).
template <int KB, bool SKIP_WAW>
__device__ __forceinline__ void gram_accum(const double (&s)[3 * KB], const double (&a)[3 * KB], double (&acc)[Tri<KB>::NEU]) {
    using T = Tri<KB>;
#pragma unroll
    for (int i = 0; i < T::NS; ++i)
#pragma unroll
        for (int j = i; j < T::NS; ++j) {
            acc[T::idx(i, j)] = fma(s[i], s[j], acc[T::idx(i, j)]);
            const bool waw = (i >= KB && i < 2 * KB && j >= KB && j < 2 * KB);
            if (SKIP_WAW && waw) continue;
            // G_A(i,j) = s_i . a_j ; for a W column on the right use the symmetric form a_i . s_j (A W' not known yet)
            const bool jw = (j >= KB && j < 2 * KB);
            const double v = (SKIP_WAW && jw) ? a[i] * s[j] : s[i] * a[j];
            acc[T::NT + T::idx(i, j)] += v;
        }
}

template <int NV>
__device__ __forceinline__ void block_reduce_store(double (&acc)[NV], double* __restrict__ out) {
    __shared__ double red[8][NV];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        double v = warp_sum(acc[i]);
        if (lane == 0) red[warp][i] = v;
    }
    __syncthreads();
    for (int i = threadIdx.x; i < NV; i += blockDim.x) {
        double s = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) s += red[w][i];
        out[i] = s;
    }
}


// One site of the fused update (see k_update_fused in lobpcg_fast.cu for the algebra): reads the six blocks at this site,
// writes X' = S C, P' = [W,P] C_wp, AX', AP' by the same coefficients and W' = P_m (AX' - X' Theta), and accumulates
// |r_j|^2 and every Gram entry of the next Rayleigh-Ritz except W'^T A W' into acc.
// sC: [3 KB][KB] coefficients followed by theta[KB].  e0 = 3 * site, n3 = 3 N.
// lk[j]: column j is soft-locked -- it gets no new search directions (W'_j = P'_j = AP'_j = 0, in the blocks and in the Gram
// entries alike) but is updated like the others and keeps its residual norm; the Rayleigh-Ritz step drops the null directions.
template <int KB, bool PROJECT>
__device__ __forceinline__ void update_site(const Blk6& b, const double* __restrict__ m, const double* sC, long long e0, long long n3,
                                            double (&acc)[Tri<KB>::NEU], const bool (&lk)[KB]) {
    using T = Tri<KB>;
    double in_s[3][T::NS], in_a[3][T::NS], mm[3];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
#pragma unroll
        for (int i = 0; i < KB; ++i) {
            in_s[q][i] = b.X[i * n3 + e0 + q]; in_s[q][KB + i] = b.W[i * n3 + e0 + q]; in_s[q][2 * KB + i] = b.P[i * n3 + e0 + q];
            in_a[q][i] = b.AX[i * n3 + e0 + q]; in_a[q][KB + i] = b.AW[i * n3 + e0 + q]; in_a[q][2 * KB + i] = b.AP[i * n3 + e0 + q];
        }
        mm[q] = PROJECT ? m[e0 + q] : 0.0;
    }
    double r[3][KB], dm[KB];
#pragma unroll
    for (int j = 0; j < KB; ++j) dm[j] = 0.0;
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        double s[T::NS], a[T::NS];
#pragma unroll
        for (int j = 0; j < KB; ++j) {
            double p = 0.0, ap = 0.0;
#pragma unroll
            for (int i = KB; i < 3 * KB; ++i) { p = fma(sC[i * KB + j], in_s[q][i], p); ap = fma(sC[i * KB + j], in_a[q][i], ap); }
            double x = p, ax = ap;
#pragma unroll
            for (int i = 0; i < KB; ++i) { x = fma(sC[i * KB + j], in_s[q][i], x); ax = fma(sC[i * KB + j], in_a[q][i], ax); }
            const double rt = fma(-sC[3 * KB * KB + j], x, ax);
            acc[2 * T::NT + j] = fma(rt, rt, acc[2 * T::NT + j]);
            const double rr = lk[j] ? 0.0 : rt;
            if (lk[j]) { p = 0.0; ap = 0.0; }
            s[j] = x; s[KB + j] = rr; s[2 * KB + j] = p;
            a[j] = ax; a[KB + j] = 0.0; a[2 * KB + j] = ap;
            r[q][j] = rr;
            dm[j] = fma(mm[q], rr, dm[j]);
            b.X[j * n3 + e0 + q] = x; b.P[j * n3 + e0 + q] = p;
            b.AX[j * n3 + e0 + q] = ax; b.AP[j * n3 + e0 + q] = ap;
        }
        gram_accum<KB, true>(s, a, acc);
    }
#pragma unroll
    for (int i = 0; i < KB; ++i)
#pragma unroll
        for (int j = i; j < KB; ++j) acc[T::idx(KB + i, KB + j)] -= dm[i] * dm[j];
#pragma unroll
    for (int q = 0; q < 3; ++q)
#pragma unroll
        for (int j = 0; j < KB; ++j) b.W[j * n3 + e0 + q] = fma(-dm[j], mm[q], r[q][j]);
}

template <int KB, bool PROJECT>
__device__ __forceinline__ void update_site(const Blk6& b, const double* __restrict__ m, const double* sC, long long e0, long long n3,
                                            double (&acc)[Tri<KB>::NEU]) {
    bool lk[KB];
#pragma unroll
    for (int j = 0; j < KB; ++j) lk[j] = false;
    update_site<KB, PROJECT>(b, m, sC, e0, n3, acc, lk);
}

}  // namespace lob
