// fmapeak.cu -- plain FP32 ALU peak of the GPU, measured ("measure an FMA microbenchmark on the box and use
// that"): register-only fused multiply-add loops, 16 independent dependency chains per thread, 8 CTAs of 256 threads per SM.
// The stencil kernels are co-limited by HBM and by these pipes for N_rhs >= 8 and for half storage, so bench.py reports
// their counted flops against this number next to the HBM fraction.
#include "internal.cuh"

// mode 0: x_i = fma(x_i, b, c)                    scalar FFMA, 3 distinct source registers
// mode 1: X_i = ffma2(X_i, B, C)                  packed FFMA2, 3 distinct 64-bit sources
// mode 2: X_i = ffma2(A_q, Y_i, X_i), q = i / 4   packed FFMA2, the first source shared by 4 consecutive instructions
// mode 3: X_i = ffma2((s_q, s_q), Y_i, X_i)       packed FFMA2 whose first source is ONE 32-bit register broadcast to both halves
//                                                 (SASS "R.F32" operand form, what the compiler emits for the stencil's link-element x
//                                                 spinor-pair products), 16 different scalars in rotation so that the operand-reuse
//                                                 cache rarely helps: scalar + two fresh register pairs read one register bank three
//                                                 times and the instruction issues every 3rd cycle instead of every 2nd
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
        float sc[16];
#pragma unroll
        for (int q = 0; q < 4; q++) a[q] = make_float2(b * (1.f + 0.01f * q), b * (1.f - 0.01f * q));
#pragma unroll
        for (int q = 0; q < 16; q++) sc[q] = b * (1.f + 0.01f * q) + seed;
#pragma unroll
        for (int i = 0; i < NACC; i++) y[i] = make_float2(c0 + 0.01f * i, c0 - 0.01f * i);
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int r = 0; r < 8; r++) {
#pragma unroll
                for (int i = 0; i < NACC; i++) {
                    if constexpr (MODE == 1) x[i] = __ffma2_rn(x[i], b2, c2);
                    else if constexpr (MODE == 2) x[i] = __ffma2_rn(a[i >> 2], y[i], x[i]);
                    else { const float sq = sc[(i >> 2) + 4 * (r & 3)]; x[i] = __ffma2_rn(make_float2(sq, sq), y[i], x[i]); }
                }
            }
            if constexpr (MODE >= 2) {      // keep the operands loop-variant so nothing is hoisted or folded
#pragma unroll
                for (int q = 0; q < 4; q++) a[q].x = -a[q].x;
#pragma unroll
                for (int q = 0; q < 16; q++) sc[q] = -sc[q];
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
        else if (mode == 2) fma_peak_kernel<2><<<grid, block, 0, c->stream>>>(out, iters, 1e-6f, c0);
        else fma_peak_kernel<3><<<grid, block, 0, c->stream>>>(out, iters, 1e-6f, c0);
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

// ---- L2 -> SM read bandwidth ------------------------------------------------------------------------------------------------
// Every thread streams 16-byte loads (ld.global.cg: no L1 allocation, 8 independent loads in flight) over a buffer that fits in
// L2 (mode 1, re-read `passes` times) or exceeds it several times (mode 0: HBM).  The stencil kernels fetch every compulsory
// byte ~3x from L2 (the 8 neighbour reads of a site meet in L2, not in L1), so next to HBM this is the second memory-side bound.
__global__ void __launch_bounds__(256) mem_read_kernel(const float4* __restrict__ buf, size_t n16, int passes, float* out) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    float acc = 0.f;
    for (int p = 0; p < passes; p++) {
        size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
        for (; i + 7 * stride < n16; i += 8 * stride) {
            float4 v[8];
#pragma unroll
            for (int u = 0; u < 8; u++) v[u] = __ldcg(buf + i + u * stride);
#pragma unroll
            for (int u = 0; u < 8; u++) acc += v[u].x + v[u].y + v[u].z + v[u].w;
        }
        for (; i < n16; i += stride) { const float4 v = __ldcg(buf + i); acc += v.x + v.y + v.z + v.w; }
    }
    if (acc == 123.456f) out[0] = acc;
}

int mem_peak(lq_ctx* c, int mode, double mbytes, double* gbs) {
    int dev = 0, sms = 0;
    LQ_CUDA(c, cudaGetDevice(&dev));
    LQ_CUDA(c, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const size_t bytes = ((size_t)(mbytes * 1e6) / 4096) * 4096;
    if (bytes < 4096) return set_err(c, LQ_EINVAL, "lq_mem_peak: buffer too small");
    float* buf = (float*)dev_alloc(c, bytes + 256);
    if (!buf) return LQ_ENOMEM;
    int rc = 0;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (cudaMemsetAsync(buf, 0, bytes + 256, c->stream) != cudaSuccess || cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess)
        rc = set_err(c, LQ_ECUDA, "lq_mem_peak: setup failed");
    const int passes = mode == 1 ? 200 : 4;
    const int grid = sms * 8;
    float ms = 0.f;
    if (rc == 0) {
        mem_read_kernel<<<grid, 256, 0, c->stream>>>((const float4*)buf, bytes / 16, 2, buf + bytes / 4);       // warm-up (fills L2 in mode 1)
        cudaEventRecord(e0, c->stream);
        mem_read_kernel<<<grid, 256, 0, c->stream>>>((const float4*)buf, bytes / 16, passes, buf + bytes / 4);
        cudaEventRecord(e1, c->stream);
        c->launches += 2;
        if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) rc = set_err(c, LQ_ECUDA, "lq_mem_peak: kernel failed");
        else cudaEventElapsedTime(&ms, e0, e1);
    }
    if (rc == 0) *gbs = (double)bytes * passes / (ms * 1e-3) * 1e-9;
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    dev_free(c, buf);
    return rc;
}

