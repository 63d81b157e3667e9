// fmapeak.cu -- plain FP32 ALU peak of the GPU, measured ("measure an FMA microbenchmark on the box and use
// that"): register-only fused multiply-add loops, 16 independent dependency chains per thread, 8 CTAs of 256 threads per SM.
// The stencil kernels are co-limited by HBM and by these pipes for N_rhs >= 8 and for half storage, so bench.py reports
// their counted flops against this number next to the HBM fraction.
#include "internal.cuh"

// mode 0: x_i = fma(x_i, b, c)                    scalar FFMA, 3 distinct source registers
// mode 1: X_i = ffma2(X_i, B, C)                  packed FFMA2, 3 distinct 64-bit sources
// mode 2: X_i = ffma2(A_q, Y_i, X_i), q = i / 4   packed FFMA2, the first source shared by 4 consecutive instructions
//                                                 (the stencil's pattern: one duplicated link element times 4 spinor reals)
template <int MODE>
__global__ void __launch_bounds__(256) fma_peak_kernel(float* out, int iters, float b, float c0) {
    constexpr int NACC = 16;
    const float seed = (float)(threadIdx.x & 7) * 1e-3f;
    if constexpr (MODE == 0) {
        float x[NACC];
#pragma unroll
        for (int i = 0; i < NACC; i++) x[i] = seed + i;
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int r = 0; r < 8; r++)
#pragma unroll
                for (int i = 0; i < NACC; i++) x[i] = fmaf(x[i], b, c0);
        }
        float s = 0.f;
#pragma unroll
        for (int i = 0; i < NACC; i++) s += x[i];
        if (s == 123.456f) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    } else {
        float2 x[NACC];
#pragma unroll
        for (int i = 0; i < NACC; i++) x[i] = make_float2(seed + i, seed - i);
        const float2 b2 = make_float2(b, b * 0.999f), c2 = make_float2(c0, c0 * 1.001f);
        float2 a[4], y[NACC];
#pragma unroll
        for (int q = 0; q < 4; q++) a[q] = make_float2(b * (1.f + 0.01f * q), b * (1.f - 0.01f * q));
#pragma unroll
        for (int i = 0; i < NACC; i++) y[i] = make_float2(c0 + 0.01f * i, c0 - 0.01f * i);
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int r = 0; r < 8; r++) {
#pragma unroll
                for (int i = 0; i < NACC; i++) {
                    if constexpr (MODE == 1) x[i] = __ffma2_rn(x[i], b2, c2);
                    else x[i] = __ffma2_rn(a[i >> 2], y[i], x[i]);
                }
            }
            if constexpr (MODE == 2) {      // keep the operands loop-variant so nothing is hoisted or folded
#pragma unroll
                for (int q = 0; q < 4; q++) a[q].x = -a[q].x;
            }
        }
        float s = 0.f;
#pragma unroll
        for (int i = 0; i < NACC; i++) s += x[i].x + x[i].y;
        if (s == 123.456f) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    }
}

int fma_peak(lq_ctx* c, int mode, double ms, double* tflops) {
    int dev = 0, sms = 0;
    LQ_CUDA(c, cudaGetDevice(&dev));
    LQ_CUDA(c, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int grid = sms * 8, block = 256;
    float* out = (float*)dev_alloc(c, (size_t)grid * block * sizeof(float));
    if (!out) return LQ_ENOMEM;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = 0;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) rc = set_err(c, LQ_ECUDA, "event creation failed");
    auto run = [&](int iters, float* t_ms) -> int {
        cudaEventRecord(e0, c->stream);
        const float b = 0.9999f, c0 = 1e-4f;      // |x| stays bounded: x <- 0.9999 x + 1e-4
        if (mode == 0) fma_peak_kernel<0><<<grid, block, 0, c->stream>>>(out, iters, b, c0);
        else if (mode == 1) fma_peak_kernel<1><<<grid, block, 0, c->stream>>>(out, iters, b, c0);
        else fma_peak_kernel<2><<<grid, block, 0, c->stream>>>(out, iters, 1e-6f, c0);
        LQ_LAUNCHED(c);
        cudaEventRecord(e1, c->stream);
        if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) return set_err(c, LQ_ECUDA, "fma_peak kernel failed");
        cudaEventElapsedTime(t_ms, e0, e1);
        return 0;
    };
    float t = 0.f;
    int iters = 256;
    if (rc == 0) rc = run(iters, &t);                           // warm-up and calibration
    if (rc == 0) rc = run(iters, &t);
    if (rc == 0) {
        double want = ms / (t > 1e-3f ? t : 1e-3f) * iters;
        if (want > 4.0e6) want = 4.0e6;
        if (want < 64) want = 64;
        iters = (int)want;
        rc = run(iters, &t);
    }
    if (rc == 0) {
        const double fma_lanes = (double)grid * block * (double)iters * 8.0 * 16.0 * (mode == 0 ? 1.0 : 2.0);
        *tflops = 2.0 * fma_lanes / (t * 1e-3) * 1e-12;
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    dev_free(c, out);
    return rc;
}
