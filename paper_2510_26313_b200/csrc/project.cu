// project.cu -- projection of the solutions onto the LapH eigenvectors:
//   P[t][alpha][j][k] = sum_{x, c} conj(v_j(x, t, c)) psi_k(x, t, alpha, c)
// a tall-skinny complex contraction per time-slice (n_ev x 4 n_sol outputs, 3 Ls^3 terms each).  This first version keeps
// fp64 data and fp64 FMAs with a register tile of 4 eigenvectors x 1 solution x 4 spins per thread and a deterministic
// two-stage reduction; the time-slice working set (n_ev eigenvectors + the solution) is re-read from L2, not HBM.
// Next step: fp32 storage with a 3xTF32 tensor-core core (tcgen05), which makes the op HBM-bound.
#include "internal.cuh"

constexpr int PJ = 4;   // eigenvectors per thread tile

__global__ void __launch_bounds__(128) project_kernel(int Lt, long long S3, int nchunk, int n_ev, int n_sol, const double2* __restrict__ V,
                                                      const double2* __restrict__ X, double2* __restrict__ partial) {
    const int t = blockIdx.x / nchunk, ch = blockIdx.x - t * nchunk, j0 = blockIdx.y * PJ, k = blockIdx.z;
    const int nj = min(PJ, n_ev - j0);
    double ar[PJ][4], ai[PJ][4];
#pragma unroll
    for (int j = 0; j < PJ; j++)
#pragma unroll
        for (int a = 0; a < 4; a++) { ar[j][a] = 0.0; ai[j][a] = 0.0; }
    const double2* xk = X + ((size_t)k * Lt + t) * S3 * 12;
    for (long long s = (long long)ch * blockDim.x + threadIdx.x; s < S3; s += (long long)nchunk * blockDim.x) {
        double2 x[12];
#pragma unroll
        for (int e = 0; e < 12; e++) x[e] = xk[s * 12 + e];
#pragma unroll
        for (int j = 0; j < PJ; j++) {
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
    __shared__ double sh[4][PJ * 4 * 2];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int j = 0; j < PJ; j++)
#pragma unroll
        for (int a = 0; a < 4; a++) {
            double r = ar[j][a], i = ai[j][a];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) { r += __shfl_xor_sync(0xffffffffu, r, o); i += __shfl_xor_sync(0xffffffffu, i, o); }
            if (lane == 0) { sh[wid][(j * 4 + a) * 2] = r; sh[wid][(j * 4 + a) * 2 + 1] = i; }
        }
    __syncthreads();
    if (threadIdx.x < PJ * 4) {
        const int j = threadIdx.x / 4, a = threadIdx.x - 4 * j;
        if (j < nj) {
            double r = 0.0, i = 0.0;
            for (int q = 0; q < 4; q++) { r += sh[q][threadIdx.x * 2]; i += sh[q][threadIdx.x * 2 + 1]; }
            // partial[t][chunk][a][j][k]
            partial[((((size_t)t * nchunk + ch) * 4 + a) * n_ev + (j0 + j)) * n_sol + k] = make_double2(r, i);
        }
    }
}
__global__ void project_final_kernel(int Lt, int nchunk, int per_t, const double2* __restrict__ partial, double2* __restrict__ out) {
    const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= (long long)Lt * per_t) return;
    const int t = (int)(id / per_t), e = (int)(id - (long long)t * per_t);
    double r = 0.0, i = 0.0;
    for (int c = 0; c < nchunk; c++) { const double2 p = partial[((size_t)t * nchunk + c) * per_t + e]; r += p.x; i += p.y; }
    out[id] = make_double2(r, i);
}

// dev_V: [n_ev][t][site][3], dev_X: [n_sol][t][site][4][3] complex double on the device; dev_P: [Lt][4][n_ev][n_sol]
int project_device(lq_ctx* c, double* dev_P, const double* dev_V, int n_ev, const double* dev_X, int n_sol) {
    const int Lt = c->g.L[3];
    const long long S3 = (long long)c->g.L[0] * c->g.L[1] * c->g.L[2];
    const int nchunk = (int)std::max(1LL, std::min(32LL, (S3 + 1023) / 1024));
    const int per_t = 4 * n_ev * n_sol;
    double2* partial = (double2*)dev_alloc(c, sizeof(double2) * (size_t)Lt * nchunk * per_t);
    if (!partial) return LQ_ENOMEM;
    project_kernel<<<dim3(Lt * nchunk, (n_ev + PJ - 1) / PJ, n_sol), 128, 0, c->stream>>>(Lt, S3, nchunk, n_ev, n_sol, (const double2*)dev_V, (const double2*)dev_X, partial);
    project_final_kernel<<<(int)(((long long)Lt * per_t + 127) / 128), 128, 0, c->stream>>>(Lt, nchunk, per_t, partial, (double2*)dev_P);
    c->launches += 2;
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    dev_free(c, partial);
    if (e != cudaSuccess) return set_err(c, LQ_ECUDA, std::string("lq_project: ") + cudaGetErrorString(e));
    return 0;
}
