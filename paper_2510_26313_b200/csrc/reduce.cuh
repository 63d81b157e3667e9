// reduce.cuh -- deterministic per-RHS sums over a whole launch (used by the block-BLAS kernels and by the fused
// epilogues of the stencil kernels).  Thread mapping assumed: unit u = global thread / (32 * TPG), RHS group = u % G,
// lane % TPG selects the VW right-hand sides of the thread inside the group; a warp lies inside one unit.
#pragma once
#include "common.cuh"

// part[VW] are this thread's sums for right-hand sides rhs0 + k.  Block size must be a multiple of 32.
template <int VW, int R>
__device__ void reduce_per_rhs(double (&part)[VW], int N, int G, double* partials, unsigned int* counter, double* out) {
    constexpr int TPG = R / VW;
    extern __shared__ double sm[];       // [max(nwarps * R, blockDim.x)]
    const int t = threadIdx.x, nt = blockDim.x, lane = t & 31, w = t >> 5, nw = nt >> 5;
#pragma unroll
    for (int k = 0; k < VW; k++) {
#pragma unroll
        for (int off = 16; off >= TPG; off >>= 1) part[k] += __shfl_xor_sync(0xffffffffu, part[k], off);
    }
    if (lane < TPG) {
#pragma unroll
        for (int k = 0; k < VW; k++) sm[w * R + lane * VW + k] = part[k];
    }
    __syncthreads();
    if (t < N) {
        // warps of this block whose unit belongs to group t / R, in warp order
        const long long gw0 = (long long)blockIdx.x * nw;
        const int grp = t / R, r = t - grp * R;
        double s = 0.0;
        for (int ww = 0; ww < nw; ww++) {
            const long long u = (gw0 + ww) / TPG;
            if ((int)(u % G) == grp) s += sm[ww * R + r];
        }
        partials[(size_t)blockIdx.x * N + t] = s;
    }
    __shared__ bool last;
    __threadfence();
    __syncthreads();
    if (t == 0) last = (atomicInc(counter, gridDim.x - 1) == gridDim.x - 1);
    __syncthreads();
    if (!last) return;
    __threadfence();
    // final: thread t handles RHS r = t % N, slice q = t / N of the blocks; Q = largest power of two with N*Q <= nt
    int Q = 1;
    while (N * Q * 2 <= nt) Q <<= 1;
    const int r = t % N, q = t / N;
    double s = 0.0;
    if (q < Q) {
        // same fixed summation order as a plain loop, but eight loads in flight: this tail runs in ONE block after
        // all others have retired, so its latency is pure serial time of the launch
        unsigned b = q;
        for (; b + 7u * Q < gridDim.x; b += 8u * Q) {
            double v[8];
#pragma unroll
            for (int i = 0; i < 8; i++) v[i] = __ldcg(partials + (size_t)(b + (unsigned)i * Q) * N + r);
#pragma unroll
            for (int i = 0; i < 8; i++) s += v[i];
        }
        for (; b < gridDim.x; b += Q) s += __ldcg(partials + (size_t)b * N + r);
    }
    __syncthreads();
    if (q < Q) sm[t] = s;
    __syncthreads();
    for (int stride = Q >> 1; stride >= 1; stride >>= 1) {
        if (q < stride) sm[t] += sm[t + stride * N];
        __syncthreads();
    }
    if (t < N) out[t] = sm[t];
}

