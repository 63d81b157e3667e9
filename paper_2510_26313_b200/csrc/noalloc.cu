// noalloc.cu -- lq_project_noalloc: the fp64 eigenvector projection (project.cu) for callers
// that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
//
// project.cu's path takes the per-chunk partial sums of its two-stage reduction from dev_alloc / dev_free on every call.  Here the
// partial sums live in ONE file-scope static __device__ array of LQ_NOALLOC_SCRATCH_BYTES (4 MiB): every GPU that loads the
// library holds it until the process exits, every call on that GPU shares it.  The entry point calls no cudaMalloc, cudaFree or
// allocating library routine and does not synchronise the host: the result is ready when the context's stream reaches this point.
//
// Sharing rules.  The array keeps the last call's contents; nothing has to start at zero, because every partial sum the second
// kernel of a call reads is written by the first kernel of the SAME call (all (t, chunk, spin, j, k) entries below
// Lt * nchunk * 4 * n_ev * n_sol, whatever an earlier, larger call left behind them).  Calls are ordered only by their stream:
// two calls that overlap on the GPU (different streams, different contexts or processes sharing the GPU through one library image)
// race on the array and return garbage without any error.
//
// The array's name in HOST code is a host-side stand-in, not a device address: the kernels get the address that
// cudaGetSymbolAddress returns, looked up once per device with that device current (scratch_address below).
#include <algorithm>
#include <mutex>
#include "internal.cuh"

constexpr size_t NOALLOC_ELEMS = LQ_NOALLOC_SCRATCH_BYTES / sizeof(double2);
static __device__ __align__(256) double2 g_project_scratch[NOALLOC_ELEMS];

constexpr int NOALLOC_MAX_DEVICES = 64;
static double2* g_scratch_addr[NOALLOC_MAX_DEVICES];      // device address of g_project_scratch on each GPU, once looked up
static std::mutex g_scratch_mutex;

// set-up, once per device: c->device must be current
static int scratch_address(lq_ctx* c, double2** out) {
    if (c->device < 0 || c->device >= NOALLOC_MAX_DEVICES) return set_err(c, LQ_EINVAL, "lq_project_noalloc: device index out of range");
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_addr[c->device]) {
        double2* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_project_scratch);
        if (e != cudaSuccess || !p) return set_err(c, LQ_ECUDA, std::string("lq_project_noalloc: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
        g_scratch_addr[c->device] = p;
    }
    *out = g_scratch_addr[c->device];
    return 0;
}

constexpr int NPJ = 4;   // eigenvectors per thread tile (as project.cu)

// The arithmetic and the order of every sum are project.cu's: register tile of 4 eigenvectors x 1 solution x 4 spins, sites strided
// over the chunk's threads, warp shuffle, the block's 4 warps in index order, then the chunks in index order.
__global__ void __launch_bounds__(128) project_noalloc_kernel(int Lt, long long S3, int nchunk, int n_ev, int n_sol, const double2* __restrict__ V,
                                                              const double2* __restrict__ X, double2* __restrict__ partial) {
    const int t = blockIdx.x / nchunk, ch = blockIdx.x - t * nchunk, j0 = blockIdx.y * NPJ, k = blockIdx.z;
    const int nj = min(NPJ, n_ev - j0);
    double ar[NPJ][4], ai[NPJ][4];
#pragma unroll
    for (int j = 0; j < NPJ; j++)
#pragma unroll
        for (int a = 0; a < 4; a++) { ar[j][a] = 0.0; ai[j][a] = 0.0; }
    const double2* xk = X + ((size_t)k * Lt + t) * S3 * 12;
    for (long long s = (long long)ch * blockDim.x + threadIdx.x; s < S3; s += (long long)nchunk * blockDim.x) {
        double2 x[12];
#pragma unroll
        for (int e = 0; e < 12; e++) x[e] = xk[s * 12 + e];
#pragma unroll
        for (int j = 0; j < NPJ; j++) {
            if (j < nj) {
                const double2* vj = V + (((size_t)(j0 + j) * Lt + t) * S3 + s) * 3;
#pragma unroll
                for (int c = 0; c < 3; c++) {
                    const double2 v = vj[c];
#pragma unroll
                    for (int a = 0; a < 4; a++) {
                        ar[j][a] += v.x * x[3 * a + c].x + v.y * x[3 * a + c].y;
                        ai[j][a] += v.x * x[3 * a + c].y - v.y * x[3 * a + c].x;
                    }
                }
            }
        }
    }
    __shared__ double sh[4][NPJ * 4 * 2];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int j = 0; j < NPJ; j++)
#pragma unroll
        for (int a = 0; a < 4; a++) {
            double r = ar[j][a], i = ai[j][a];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) { r += __shfl_xor_sync(0xffffffffu, r, o); i += __shfl_xor_sync(0xffffffffu, i, o); }
            if (lane == 0) { sh[wid][(j * 4 + a) * 2] = r; sh[wid][(j * 4 + a) * 2 + 1] = i; }
        }
    __syncthreads();
    if (threadIdx.x < NPJ * 4) {
        const int j = threadIdx.x / 4, a = threadIdx.x - 4 * j;
        if (j < nj) {
            double r = 0.0, i = 0.0;
            for (int q = 0; q < 4; q++) { r += sh[q][threadIdx.x * 2]; i += sh[q][threadIdx.x * 2 + 1]; }
            partial[((((size_t)t * nchunk + ch) * 4 + a) * n_ev + (j0 + j)) * n_sol + k] = make_double2(r, i);      // [t][chunk][a][j][k]
        }
    }
}
__global__ void project_noalloc_final_kernel(int Lt, int nchunk, int per_t, const double2* __restrict__ partial, double2* __restrict__ out) {
    const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= (long long)Lt * per_t) return;
    const int t = (int)(id / per_t), e = (int)(id - (long long)t * per_t);
    double r = 0.0, i = 0.0;
    for (int c = 0; c < nchunk; c++) { const double2 p = partial[((size_t)t * nchunk + c) * per_t + e]; r += p.x; i += p.y; }
    out[id] = make_double2(r, i);
}

extern "C" int lq_project_noalloc(lq_ctx* c, void* P, const void* evecs, int n_ev, const void* sols, int n_sol) {
    if (!c) return LQ_EINVAL;
    if (!P || !evecs || !sols || n_ev < 1 || n_ev > 1024 || n_sol < 1 || n_sol > 64) return set_err(c, LQ_EINVAL, "lq_project_noalloc: bad argument");
    const int Lt = c->g.L[3];
    const long long S3 = (long long)c->g.L[0] * c->g.L[1] * c->g.L[2];
    const int nchunk = (int)std::max(1LL, std::min(32LL, (S3 + 1023) / 1024));
    const int per_t = 4 * n_ev * n_sol;
    const size_t need = (size_t)Lt * nchunk * per_t;
    if (need > NOALLOC_ELEMS)
        return set_err(c, LQ_EINVAL, "lq_project_noalloc: Lt * nchunk * 4 * n_ev * n_sol = " + std::to_string(need) + " partial sums exceed the static scratch of " +
                                         std::to_string(NOALLOC_ELEMS) + " (LQ_NOALLOC_SCRATCH_BYTES); use lq_project");
    LQ_CUDA(c, cudaSetDevice(c->device));
    double2* partial = nullptr;
    LQ_TRY(scratch_address(c, &partial));
    project_noalloc_kernel<<<dim3(Lt * nchunk, (n_ev + NPJ - 1) / NPJ, n_sol), 128, 0, c->stream>>>(Lt, S3, nchunk, n_ev, n_sol, (const double2*)evecs,
                                                                                                      (const double2*)sols, partial);
    project_noalloc_final_kernel<<<(int)(((long long)Lt * per_t + 127) / 128), 128, 0, c->stream>>>(Lt, nchunk, per_t, partial, (double2*)P);
    c->launches += 2;
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
