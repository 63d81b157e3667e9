// reduce.cuh -- deterministic per-RHS sums over a whole launch (used by the block-BLAS kernels and by the fused
// epilogues of the stencil kernels).  Thread mapping assumed: unit u = global thread / (32 * TPG), RHS group = u % G,
// lane % TPG selects the VW right-hand sides of the thread inside the group; a warp lies inside one unit.
#pragma once
#include "common.cuh"

// part[q][VW] are this thread's sums of quantity q for right-hand sides rhs0 + k (NQ quantities reduced in one pass, e.g. the real
// and imaginary part of an inner product and a norm).  Result: out[q * LQ_MAX_RHS + rhs].  Block size must be a multiple of 32
// and at least NQ * N.
template <int NQ, int VW, int R>
__device__ void reduce_multi(double (&part)[NQ][VW], int N1, int G, double* partials, unsigned int* counter, double* out) {
    constexpr int TPG = R / VW;
    extern __shared__ double sm[];       // [max(nwarps * R, blockDim.x)]
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
    // Fan-in tree over the blocks (RED_FAN per node, fixed grouping and order: bitwise reproducible).  The last block to
    // finish in a group of RED_FAN adds the group's rows and becomes the group's representative one level up; the tail that
    // runs after all other blocks have retired is then a few short rounds instead of one block reading every partial.
    // Level l rows live behind those of level l-1 in `partials`, its self-resetting counters behind those of level l-1.
    __shared__ bool last;
    int Q = 1;                             // thread t handles RHS t % N, row slice t / N; Q = largest power of two with N*Q <= nt
    while (N * Q * 2 <= nt) Q <<= 1;
    const int r = t % N, q = t / N;
    unsigned idx = blockIdx.x, n = gridDim.x;
    double* src = partials;
    unsigned int* cnt = counter + RED_COUNTER_BASE;
    for (;;) {
        const unsigned grp = idx / RED_FAN, ngrp = (n + RED_FAN - 1) / RED_FAN;
        const unsigned gsize = min((unsigned)RED_FAN, n - grp * RED_FAN);
        __threadfence();
        __syncthreads();
        if (t == 0) last = (atomicInc(cnt + grp, gsize - 1) == gsize - 1);
        __syncthreads();
        if (!last) return;
        __threadfence();
        const double* rows = src + (size_t)grp * RED_FAN * N;
        double s = 0.0;
        if (q < Q) for (unsigned b = q; b < gsize; b += Q) s += __ldcg(rows + (size_t)b * N + r);
        __syncthreads();
        if (q < Q) sm[t] = s;
        __syncthreads();
        for (int stride = Q >> 1; stride >= 1; stride >>= 1) {
            if (q < stride) sm[t] += sm[t + stride * N];
            __syncthreads();
        }
        if (ngrp == 1) { if (t < N) out[(t / N1) * LQ_MAX_RHS + (t % N1)] = sm[t]; return; }
        double* dst = src + (size_t)n * N;
        if (t < N) dst[(size_t)grp * N + t] = sm[t];
        src = dst; cnt += ngrp; idx = grp; n = ngrp;
    }
}

// part[VW] are this thread's sums for right-hand sides rhs0 + k; out[rhs]
template <int VW, int R>
__device__ __forceinline__ void reduce_per_rhs(double (&part)[VW], int N, int G, double* partials, unsigned int* counter, double* out) {
    double p1[1][VW];
#pragma unroll
    for (int k = 0; k < VW; k++) p1[0][k] = part[k];
    reduce_multi<1, VW, R>(p1, N, G, partials, counter, out);
}
