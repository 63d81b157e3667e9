// reduce.cuh -- deterministic per-RHS sums over a whole launch (used by the block-BLAS kernels and by the fused
// epilogues of the stencil kernels).  Thread mapping assumed: unit u = global thread / (32 * TPG), RHS group = u % G,
// lane % TPG selects the VW right-hand sides of the thread inside the group; a warp lies inside one unit.
//
// Two stages.  (1) Inside the producing kernel (reduce_multi below): fp64 per thread -> warp shuffle -> fixed-order sum over
// the block's warps -> ONE ROW of partial sums per block, written with plain stores: no fence, no atomic, nothing that makes a
// block wait for its own stores (the round-1 version ended every block with __threadfence + atomicInc to elect a "last block";
// on the 248832-block stencil launches of configs[3] that tail cost ~1 ms of a 6 ms kernel, profiles/r02_launches_cfg3.md).
// (2) reduce_finish (blas.cu): a small second launch sums the rows in a fixed order (<= 256 blocks over contiguous row ranges,
// then the last of THOSE blocks -- the only place a fence and an atomic remain -- adds their rows in index order).
// Bitwise reproducible: the order of every addition is fixed by the launch geometry alone.
#pragma once
#include "common.cuh"

// second stage (blas.cu): sums the `nrows` block rows left in lq_ctx::red_partials (nq quantities x n1 right-hand sides) into
// d_out[q * LQ_MAX_RHS + rhs]; enqueued right behind the kernel that produced the rows
int reduce_finish(lq_ctx* c, int nrows, int nq, int n1, double* d_out);

// part[q][VW] are this thread's sums of quantity q for right-hand sides rhs0 + k (NQ quantities reduced in one pass, e.g. the real
// and imaginary part of an inner product and a norm).  Writes partials[blockIdx.x][q * N1 + rhs] (a dense row: zeros for the
// right-hand sides of groups this block does not touch).  Block size must be a multiple of 32 and at least N1.
template <int NQ, int VW, int R>
__device__ __forceinline__ void reduce_multi(double (&part)[NQ][VW], int N1, int G, double* __restrict__ partials) {
    constexpr int TPG = R / VW;
    extern __shared__ double sm[];       // [nwarps * R]
    const int t = threadIdx.x, nt = blockDim.x, lane = t & 31, w = t >> 5, nw = nt >> 5;
    const int N = NQ * N1;               // row width of the partial sums
#pragma unroll
    for (int qq = 0; qq < NQ; qq++) {
#pragma unroll
        for (int k = 0; k < VW; k++) {
#pragma unroll
            for (int off = 16; off >= TPG; off >>= 1) part[qq][k] += __shfl_xor_sync(0xffffffffu, part[qq][k], off);
        }
        if (qq > 0) __syncthreads();
        if (lane < TPG) {
#pragma unroll
            for (int k = 0; k < VW; k++) sm[w * R + lane * VW + k] = part[qq][k];
        }
        __syncthreads();
        if (t < N1) {
            // warps of this block whose unit belongs to group t / R, in warp order
            const long long gw0 = (long long)blockIdx.x * nw;
            const int grp = t / R, r = t - grp * R;
            double s = 0.0;
            for (int ww = 0; ww < nw; ww++) {
                const long long u = (gw0 + ww) / TPG;
                if ((int)(u % G) == grp) s += sm[ww * R + r];
            }
            partials[(size_t)blockIdx.x * N + qq * N1 + t] = s;
        }
    }
}

// part[VW] are this thread's sums for right-hand sides rhs0 + k
template <int VW, int R>
__device__ __forceinline__ void reduce_per_rhs(double (&part)[VW], int N, int G, double* __restrict__ partials) {
    double p1[1][VW];
#pragma unroll
    for (int k = 0; k < VW; k++) p1[0][k] = part[k];
    reduce_multi<1, VW, R>(p1, N, G, partials);
}
