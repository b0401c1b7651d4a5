// gram_static.cu -- moto_gram_static: the tall-skinny Gram product K2 (G = S^T T, the reduced pencil of the LOBPCG iteration,
// PAPER.md:54-60, :160) as an entry point that ALLOCATES NOTHING: no context, no workspace, no cudaMalloc / cudaFree and no
// allocating library call, for callers that cannot allocate (CUDA graph capture, tight serving loops, harnesses that forbid
// it).  moto_gram (api.cu -> block_algebra.cu) keeps its per-CTA partial sums in the context's workspace; here they live in
// a file-scope __device__ array of fixed size, which every GPU that loads the library holds until the process exits
// (GS_BLOCKS x GS_MAXE doubles + one ticket slot = 170 752 bytes).
//
// One launch: every CTA writes its partial sums, takes a ticket, and the CTA that draws the last ticket adds the partials in
// CTA order (fixed order: reruns are bit-identical) and resets the ticket.  The ticket must be zero when the kernel starts;
// the host clears it on the caller's stream before every launch, so a call aborted midway cannot poison the next one.
// All calls on a device share the array: two calls that overlap on the GPU (different streams, no dependency) RACE.
#include <atomic>
#include "common.cuh"

namespace {

constexpr int GS_NS = 6;          // largest ns: [X, W, P] at kb = 2
constexpr int GS_NT = 12;         // largest nt: [S, A S]
constexpr int GS_MAXE = GS_NS * GS_NT;
constexpr int GS_BLOCKS = MOTO_RED_BLOCKS;   // 296 CTAs = 2 per SM
constexpr int GS_THREADS = 256;
constexpr int GS_CH = 64;         // flat elements staged per chunk
constexpr int GS_LD = GS_CH + 1;
constexpr int GS_TICKET = GS_BLOCKS * GS_MAXE;   // index (in doubles) of the ticket slot

// In host code this name is a host-side stand-in, not a device address: only cudaGetSymbolAddress gives the pointer a
// kernel may be handed (scratch_ptr below).  Device code names the array directly.
static __device__ __align__(256) double g_gram_scratch[GS_TICKET + 32];

struct Ptrs { const double* s[GS_NS]; const double* t[GS_NT]; };

__global__ void __launch_bounds__(GS_THREADS) k_gram_static(Ptrs P, int ns, int nt, long long n3, double* __restrict__ scratch,
                                                            double* __restrict__ G) {
    __shared__ double sS[GS_NS * GS_LD];
    __shared__ double sT[GS_NT * GS_LD];
    __shared__ unsigned s_ticket;
    const int ne = ns * nt;
    double acc = 0.0;   // thread e < ne owns entry (e / nt, e % nt); ne <= 72 < GS_THREADS
    const int i = threadIdx.x / nt, j = threadIdx.x - i * nt;
    const long long nchunk = (n3 + GS_CH - 1) / GS_CH;
    for (long long ch = blockIdx.x; ch < nchunk; ch += gridDim.x) {
        const long long base = ch * GS_CH;
        for (int t = threadIdx.x; t < (ns + nt) * GS_CH; t += GS_THREADS) {
            const int row = t / GS_CH, q = t - row * GS_CH;
            const long long e = base + q;
            double val = 0.0;
            if (e < n3) val = (row < ns) ? P.s[row][e] : P.t[row - ns][e];
            if (row < ns) sS[row * GS_LD + q] = val; else sT[(row - ns) * GS_LD + q] = val;
        }
        __syncthreads();
        if (threadIdx.x < ne) {
            const double* a = sS + i * GS_LD;
            const double* b = sT + j * GS_LD;
            double s = 0.0;
#pragma unroll 8
            for (int q = 0; q < GS_CH; ++q) s = fma(a[q], b[q], s);
            acc += s;
        }
        __syncthreads();
    }
    if (threadIdx.x < ne) scratch[(size_t)blockIdx.x * GS_MAXE + threadIdx.x] = acc;
    __threadfence();
    __syncthreads();
    unsigned* ticket = reinterpret_cast<unsigned*>(scratch + GS_TICKET);
    if (threadIdx.x == 0) s_ticket = atomicAdd(ticket, 1u);
    __syncthreads();
    if (s_ticket != gridDim.x - 1) return;
    __threadfence();   // last CTA: every other CTA's partials are visible (their fence precedes their ticket)
    if (threadIdx.x < ne) {
        double s = 0.0;
        for (unsigned b = 0; b < gridDim.x; ++b) s += __ldcg(scratch + (size_t)b * GS_MAXE + threadIdx.x);
        G[threadIdx.x] = s;
    }
    if (threadIdx.x == 0) *ticket = 0u;
}

thread_local char t_err[256] = "";

moto_status gs_fail(moto_status s, const char* msg, cudaError_t e = cudaSuccess) {
    if (e != cudaSuccess) snprintf(t_err, sizeof t_err, "%s: %s", msg, cudaGetErrorString(e));
    else snprintf(t_err, sizeof t_err, "%s", msg);
    return s;
}

// device address of g_gram_scratch on the CURRENT device, looked up once per device
std::atomic<double*> g_ptr[64];

moto_status scratch_ptr(double** out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return gs_fail(MOTO_ECUDA, "moto_gram_static: cudaGetDevice", e);
    if (dev < 0 || dev >= 64) return gs_fail(MOTO_EINVAL, "moto_gram_static: device ordinal beyond 63");
    double* p = g_ptr[dev].load(std::memory_order_acquire);
    if (!p) {
        e = cudaGetSymbolAddress((void**)&p, g_gram_scratch);
        if (e != cudaSuccess || !p) return gs_fail(MOTO_ECUDA, "moto_gram_static: cudaGetSymbolAddress", e);
        g_ptr[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return MOTO_OK;
}

}  // namespace

extern "C" {

moto_status moto_gram_static(const double* d_S, int ns, const double* d_T, int nt, int64_t n3, double* d_G, void* stream) {
    if (!d_S || !d_T || !d_G) return gs_fail(MOTO_EINVAL, "moto_gram_static: null argument");
    if (ns < 1 || nt < 1 || n3 < 1) return gs_fail(MOTO_EINVAL, "moto_gram_static: need ns >= 1, nt >= 1, n3 >= 1");
    if (ns > GS_NS || nt > GS_NT) {
        snprintf(t_err, sizeof t_err, "moto_gram_static: ns = %d, nt = %d beyond the static scratch (ns <= %d, nt <= %d); use moto_gram",
                 ns, nt, GS_NS, GS_NT);
        return MOTO_EINVAL;
    }
    double* scratch = nullptr;
    moto_status st = scratch_ptr(&scratch);
    if (st != MOTO_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    Ptrs P = {};
    for (int i = 0; i < ns; ++i) P.s[i] = d_S + (size_t)i * n3;
    for (int j = 0; j < nt; ++j) P.t[j] = d_T + (size_t)j * n3;
    const long long nchunk = (n3 + GS_CH - 1) / GS_CH;
    const int blocks = (int)(nchunk < GS_BLOCKS ? nchunk : GS_BLOCKS);
    cudaError_t e = cudaMemsetAsync(scratch + GS_TICKET, 0, 256, s);
    if (e != cudaSuccess) return gs_fail(MOTO_ECUDA, "moto_gram_static: cudaMemsetAsync", e);
    k_gram_static<<<blocks, GS_THREADS, 0, s>>>(P, ns, nt, (long long)n3, scratch, d_G);
    e = cudaGetLastError();
    if (e != cudaSuccess) return gs_fail(MOTO_ECUDA, "moto_gram_static: launch", e);
    t_err[0] = 0;
    return MOTO_OK;
}

const char* moto_gram_static_last_error(void) { return t_err; }

}  // extern "C"
