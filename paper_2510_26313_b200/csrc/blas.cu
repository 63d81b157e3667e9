// blas.cu -- fused block-BLAS with per-RHS reductions.
//
// A native parity block is 24 planes of Vh*N elements with the RHS index innermost, so every kernel here is
// elementwise over e = cb*N + k.  One thread owns VW = min(N,4) consecutive elements (one site, VW right-hand
// sides) through all 24 planes (needed for the half format's per-(site,rhs) norm).  Per-RHS sums: fp64
// accumulators, fixed-shape shared-memory tree over threads with the same RHS group (block size G*2^m,
// strides multiples of G = N/VW), per-block partials, and a fixed-order final pass by the last block to
// finish.  Deterministic; results stay on the device.
#include "internal.cuh"
#include "dslash.cuh"

template <class S, int VW> struct SiteVec {
    using T = typename S::comp_t;
    T v[24][VW];
    __device__ __forceinline__ void load(const SView<S>& f, size_t plane, size_t e) {
        T sc[VW];
        if constexpr (S::has_norm) {
            float n[VW]; load_norm<VW>(f.n + e, n);
#pragma unroll
            for (int k = 0; k < VW; k++) sc[k] = n[k] * (1.0f / 32767.0f);
        }
#pragma unroll
        for (int j = 0; j < 24; j++) {
            load_comp<S, VW>(f.d + j * plane + e, v[j]);
            if constexpr (S::has_norm) {
#pragma unroll
                for (int k = 0; k < VW; k++) v[j][k] *= sc[k];
            }
        }
    }
    __device__ __forceinline__ void store(const SView<S>& f, size_t plane, size_t e) const {
        if constexpr (S::has_norm) {
            float mx[VW], inv[VW];
#pragma unroll
            for (int k = 0; k < VW; k++) mx[k] = 0.f;
#pragma unroll
            for (int j = 0; j < 24; j++)
#pragma unroll
                for (int k = 0; k < VW; k++) mx[k] = fmaxf(mx[k], fabsf(v[j][k]));
#pragma unroll
            for (int k = 0; k < VW; k++) { inv[k] = mx[k] > 0.f ? 32767.0f / mx[k] : 0.f; f.n[e + k] = mx[k]; }
#pragma unroll
            for (int j = 0; j < 24; j++) {
                T q[VW];
#pragma unroll
                for (int k = 0; k < VW; k++) q[k] = rintf(v[j][k] * inv[k]);
                store_comp<S, VW>(f.d + j * plane + e, q);
            }
        } else {
#pragma unroll
            for (int j = 0; j < 24; j++) store_comp<S, VW>(f.d + j * plane + e, v[j]);
        }
    }
};

// block tree + last-block final pass.  part[VW] are this thread's sums for RHS (threadIdx % G)*VW + k.
template <int VW>
__device__ void reduce_per_rhs(double (&part)[VW], int N, int G, double* partials, unsigned int* counter, double* out) {
    extern __shared__ double sm[];
    const int t = threadIdx.x, nt = blockDim.x;
#pragma unroll
    for (int k = 0; k < VW; k++) sm[t * VW + k] = part[k];
    __syncthreads();
    for (int stride = nt >> 1; stride >= G; stride >>= 1) {
        if (t < stride) {
#pragma unroll
            for (int k = 0; k < VW; k++) sm[t * VW + k] += sm[(t + stride) * VW + k];
        }
        __syncthreads();
    }
    if (t < G) {
#pragma unroll
        for (int k = 0; k < VW; k++) partials[(size_t)blockIdx.x * N + t * VW + k] = sm[t * VW + k];
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
    if (q < Q) for (unsigned b = q; b < gridDim.x; b += Q) s += partials[(size_t)b * N + r];
    __syncthreads();
    if (q < Q) sm[t] = s;
    __syncthreads();
    for (int stride = Q >> 1; stride >= 1; stride >>= 1) {
        if (q < stride) sm[t] += sm[t + stride * N];
        __syncthreads();
    }
    if (t < N) out[t] = sm[t];
}

struct BlasGeom { int N, G; long long elems; size_t plane; };

template <class S, int VW>
__global__ void norm2_kernel(BlasGeom bg, SView<S> x, double* partials, unsigned int* counter, double* out) {
    const long long e = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * VW;
    double part[VW];
#pragma unroll
    for (int k = 0; k < VW; k++) part[k] = 0.0;
    if (e < bg.elems) {
        SiteVec<S, VW> a; a.load(x, bg.plane, e);
#pragma unroll
        for (int j = 0; j < 24; j++)
#pragma unroll
            for (int k = 0; k < VW; k++) part[k] += (double)a.v[j][k] * (double)a.v[j][k];
    }
    reduce_per_rhs<VW>(part, bg.N, bg.G, partials, counter, out);
}

template <class S, int VW>
__global__ void cg_update_xr_kernel(BlasGeom bg, SView<S> x, SView<S> r, SView<S> p, SView<S> q, const double* __restrict__ rr,
                                    const double* __restrict__ pAp, double* partials, unsigned int* counter, double* rr_new) {
    using T = typename S::comp_t;
    const long long e = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * VW;
    double part[VW];
#pragma unroll
    for (int k = 0; k < VW; k++) part[k] = 0.0;
    if (e < bg.elems) {
        const int k0 = (int)(e % bg.N);
        T alpha[VW];
#pragma unroll
        for (int k = 0; k < VW; k++) { const double d = pAp[k0 + k]; alpha[k] = (T)(d > 0.0 ? rr[k0 + k] / d : 0.0); }
        {
            SiteVec<S, VW> a, b; a.load(x, bg.plane, e); b.load(p, bg.plane, e);
#pragma unroll
            for (int j = 0; j < 24; j++)
#pragma unroll
                for (int k = 0; k < VW; k++) a.v[j][k] += alpha[k] * b.v[j][k];
            a.store(x, bg.plane, e);
        }
        {
            SiteVec<S, VW> a, b; a.load(r, bg.plane, e); b.load(q, bg.plane, e);
#pragma unroll
            for (int j = 0; j < 24; j++)
#pragma unroll
                for (int k = 0; k < VW; k++) { a.v[j][k] -= alpha[k] * b.v[j][k]; part[k] += (double)a.v[j][k] * (double)a.v[j][k]; }
            a.store(r, bg.plane, e);
        }
    }
    reduce_per_rhs<VW>(part, bg.N, bg.G, partials, counter, rr_new);
}

template <class S, int VW>
__global__ void cg_update_p_kernel(BlasGeom bg, SView<S> p, SView<S> r, const double* __restrict__ rr_new, const double* __restrict__ rr) {
    using T = typename S::comp_t;
    const long long e = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * VW;
    if (e >= bg.elems) return;
    const int k0 = (int)(e % bg.N);
    T beta[VW];
#pragma unroll
    for (int k = 0; k < VW; k++) { const double d = rr[k0 + k]; beta[k] = (T)(d > 0.0 ? rr_new[k0 + k] / d : 0.0); }
    SiteVec<S, VW> a, b; a.load(p, bg.plane, e); b.load(r, bg.plane, e);
#pragma unroll
    for (int j = 0; j < 24; j++)
#pragma unroll
        for (int k = 0; k < VW; k++) a.v[j][k] = b.v[j][k] + beta[k] * a.v[j][k];
    a.store(p, bg.plane, e);
}

// y (fp64) += s_k * e
template <class S, int VW>
__global__ void axpy_mixed_kernel(BlasGeom bg, double* __restrict__ y, SView<S> ev, const double* __restrict__ scale) {
    const long long e = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * VW;
    if (e >= bg.elems) return;
    const int k0 = (int)(e % bg.N);
    SiteVec<S, VW> a; a.load(ev, bg.plane, e);
#pragma unroll
    for (int j = 0; j < 24; j++)
#pragma unroll
        for (int k = 0; k < VW; k++) y[j * bg.plane + e + k] += scale[k0 + k] * (double)a.v[j][k];
}

// r = b - t (fp64), per-RHS ||r||^2
template <int VW>
__global__ void residual_kernel(BlasGeom bg, double* __restrict__ r, const double* __restrict__ b, const double* __restrict__ tv,
                                double* partials, unsigned int* counter, double* out) {
    const long long e = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * VW;
    double part[VW];
#pragma unroll
    for (int k = 0; k < VW; k++) part[k] = 0.0;
    if (e < bg.elems) {
#pragma unroll
        for (int j = 0; j < 24; j++)
#pragma unroll
            for (int k = 0; k < VW; k++) {
                const size_t i = j * bg.plane + e + k;
                const double d = b[i] - tv[i];
                r[i] = d; part[k] += d * d;
            }
    }
    reduce_per_rhs<VW>(part, bg.N, bg.G, partials, counter, out);
}

// ---- host side -----------------------------------------------------------------------------------------------------
struct Launch { BlasGeom bg; int vw, block, grid; size_t smem; };
static int plan(lq_ctx* c, int nrhs, int maxvw, Launch& L) {
    int vw = nrhs < 4 ? nrhs : 4;
    if (vw > maxvw) vw = maxvw;
    if (nrhs % vw) return set_err(c, LQ_EINVAL, "unsupported nrhs");
    L.vw = vw;
    L.bg.N = nrhs; L.bg.G = nrhs / vw; L.bg.elems = (long long)c->g.Vh * nrhs; L.bg.plane = (size_t)c->g.Vh * nrhs;
    int block = L.bg.G;
    while (block * 2 <= 256) block *= 2;
    L.block = block;
    const long long threads = L.bg.elems / vw;
    L.grid = (int)((threads + block - 1) / block);
    L.smem = (size_t)block * vw * sizeof(double);
    if (L.smem < (size_t)block * sizeof(double)) L.smem = (size_t)block * sizeof(double);
    if ((size_t)L.grid * nrhs > c->red_partials_elems) {
        if (c->red_partials) dev_free(c, c->red_partials);
        c->red_partials_elems = (size_t)L.grid * nrhs * 2;
        c->red_partials = (double*)dev_alloc(c, c->red_partials_elems * sizeof(double));
        if (!c->red_partials) { c->red_partials_elems = 0; return LQ_ENOMEM; }
    }
    return 0;
}
#define VW_DISPATCH(L, MAXVW, CALL4, CALL2, CALL1)          \
    do {                                                       \
        if (L.vw == 4) { if constexpr (MAXVW >= 4) { CALL4; } } \
        else if (L.vw == 2) { CALL2; }                        \
        else { CALL1; }                                        \
    } while (0)

template <class S> static int norm2_t(lq_ctx* c, int nrhs, const void* x, double* d_out) {
    constexpr int MAXVW = S::prec == LQ_FP64 ? 2 : 4;
    Launch L; LQ_TRY(plan(c, nrhs, MAXVW, L));
    SView<S> vx = make_view<S>(c->g, const_cast<void*>(x), nrhs, 0);
    VW_DISPATCH(L, MAXVW,
        (norm2_kernel<S, MAXVW><<<L.grid, L.block, L.smem, c->stream>>>(L.bg, vx, c->red_partials, c->red_counter, d_out)),
        (norm2_kernel<S, 2><<<L.grid, L.block, L.smem, c->stream>>>(L.bg, vx, c->red_partials, c->red_counter, d_out)),
        (norm2_kernel<S, 1><<<L.grid, L.block, L.smem, c->stream>>>(L.bg, vx, c->red_partials, c->red_counter, d_out)));
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
int blas_norm2(lq_ctx* c, int prec, int nrhs, const void* x, double* d_out) {
    if (prec == LQ_FP64) return norm2_t<F64>(c, nrhs, x, d_out);
    if (prec == LQ_FP32) return norm2_t<F32>(c, nrhs, x, d_out);
    return norm2_t<H16>(c, nrhs, x, d_out);
}

template <class S> static int xr_t(lq_ctx* c, int nrhs, void* x, void* r, const void* p, const void* q, const double* rr, const double* pAp, double* rrn) {
    constexpr int MAXVW = S::prec == LQ_FP64 ? 2 : 4;
    Launch L; LQ_TRY(plan(c, nrhs, MAXVW, L));
    SView<S> vx = make_view<S>(c->g, x, nrhs, 0), vr = make_view<S>(c->g, r, nrhs, 0);
    SView<S> vp = make_view<S>(c->g, const_cast<void*>(p), nrhs, 0), vq = make_view<S>(c->g, const_cast<void*>(q), nrhs, 0);
    VW_DISPATCH(L, MAXVW,
        (cg_update_xr_kernel<S, MAXVW><<<L.grid, L.block, L.smem, c->stream>>>(L.bg, vx, vr, vp, vq, rr, pAp, c->red_partials, c->red_counter, rrn)),
        (cg_update_xr_kernel<S, 2><<<L.grid, L.block, L.smem, c->stream>>>(L.bg, vx, vr, vp, vq, rr, pAp, c->red_partials, c->red_counter, rrn)),
        (cg_update_xr_kernel<S, 1><<<L.grid, L.block, L.smem, c->stream>>>(L.bg, vx, vr, vp, vq, rr, pAp, c->red_partials, c->red_counter, rrn)));
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
int blas_cg_update_xr(lq_ctx* c, int prec, int nrhs, void* x, void* r, const void* p, const void* q, const double* d_rr, const double* d_pAp, double* d_rr_new) {
    if (prec == LQ_FP64) return xr_t<F64>(c, nrhs, x, r, p, q, d_rr, d_pAp, d_rr_new);
    if (prec == LQ_FP32) return xr_t<F32>(c, nrhs, x, r, p, q, d_rr, d_pAp, d_rr_new);
    return xr_t<H16>(c, nrhs, x, r, p, q, d_rr, d_pAp, d_rr_new);
}

template <class S> static int p_t(lq_ctx* c, int nrhs, void* p, const void* r, const double* rrn, const double* rr) {
    constexpr int MAXVW = S::prec == LQ_FP64 ? 2 : 4;
    Launch L; LQ_TRY(plan(c, nrhs, MAXVW, L));
    SView<S> vp = make_view<S>(c->g, p, nrhs, 0), vr = make_view<S>(c->g, const_cast<void*>(r), nrhs, 0);
    VW_DISPATCH(L, MAXVW,
        (cg_update_p_kernel<S, MAXVW><<<L.grid, L.block, 0, c->stream>>>(L.bg, vp, vr, rrn, rr)),
        (cg_update_p_kernel<S, 2><<<L.grid, L.block, 0, c->stream>>>(L.bg, vp, vr, rrn, rr)),
        (cg_update_p_kernel<S, 1><<<L.grid, L.block, 0, c->stream>>>(L.bg, vp, vr, rrn, rr)));
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
int blas_cg_update_p(lq_ctx* c, int prec, int nrhs, void* p, const void* r, const double* d_rr_new, const double* d_rr) {
    if (prec == LQ_FP64) return p_t<F64>(c, nrhs, p, r, d_rr_new, d_rr);
    if (prec == LQ_FP32) return p_t<F32>(c, nrhs, p, r, d_rr_new, d_rr);
    return p_t<H16>(c, nrhs, p, r, d_rr_new, d_rr);
}

template <class S> static int axpy_t(lq_ctx* c, int nrhs, void* y, const void* e, const double* s) {
    constexpr int MAXVW = S::prec == LQ_FP64 ? 2 : 4;
    Launch L; LQ_TRY(plan(c, nrhs, MAXVW, L));
    SView<S> ve = make_view<S>(c->g, const_cast<void*>(e), nrhs, 0);
    VW_DISPATCH(L, MAXVW,
        (axpy_mixed_kernel<S, MAXVW><<<L.grid, L.block, 0, c->stream>>>(L.bg, (double*)y, ve, s)),
        (axpy_mixed_kernel<S, 2><<<L.grid, L.block, 0, c->stream>>>(L.bg, (double*)y, ve, s)),
        (axpy_mixed_kernel<S, 1><<<L.grid, L.block, 0, c->stream>>>(L.bg, (double*)y, ve, s)));
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
int blas_axpy_mixed(lq_ctx* c, int prec, int nrhs, void* y64, const void* e, const double* d_scale) {
    if (prec == LQ_FP64) return axpy_t<F64>(c, nrhs, y64, e, d_scale);
    if (prec == LQ_FP32) return axpy_t<F32>(c, nrhs, y64, e, d_scale);
    return axpy_t<H16>(c, nrhs, y64, e, d_scale);
}

int blas_residual(lq_ctx* c, int nrhs, void* r, const void* b, const void* t, double* d_out) {
    Launch L; LQ_TRY(plan(c, nrhs, 2, L));
    if (L.vw == 2) residual_kernel<2><<<L.grid, L.block, L.smem, c->stream>>>(L.bg, (double*)r, (const double*)b, (const double*)t, c->red_partials, c->red_counter, d_out);
    else residual_kernel<1><<<L.grid, L.block, L.smem, c->stream>>>(L.bg, (double*)r, (const double*)b, (const double*)t, c->red_partials, c->red_counter, d_out);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}

int blas_copy(lq_ctx* c, int prec, int nrhs, void* dst, const void* src) {
    LQ_CUDA(c, cudaMemcpyAsync(dst, src, parity_bytes(c->g, nrhs, prec), cudaMemcpyDeviceToDevice, c->stream));
    return 0;
}
