// blas.cu -- fused block-BLAS with per-RHS reductions.
//
// Every kernel here is elementwise over the blocked native layout (common.cuh).  One thread owns one site and VW
// consecutive right-hand sides of one RHS group (VW = R for fp32/half, min(R,2) for fp64) through all 24 reals
// (needed for the half format's per-(site,rhs) norm).  A warp lies inside one unit (site block, RHS group), so
// per-RHS sums are: fp64 accumulators per thread, warp shuffle over the lanes with the same RHS, a fixed-order
// sum over the block's warps of the same group, per-block partials, and a fixed-order final pass by the last
// block to finish.  Deterministic; results stay on the device.
#include "internal.cuh"
#include "dslash_kernel.cuh"
#include "reduce.cuh"

template <int VW, int R> struct BlasIdx {
    static constexpr int TPG = R / VW, UT = SB * TPG, US = 24 * SB * R, UN = SB * R, PL = SB * R;
    size_t own, own_n;
    int rhs0;     // first right-hand side of this thread
    bool valid;
    __device__ __forceinline__ BlasIdx(const Geom& g, int G) {
        const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
        const int u = (int)(tid / UT);
        const int lu = (int)(tid - (long long)u * UT);
        const int s = lu / TPG, hoff = (lu - s * TPG) * VW;
        const int blk = u / G, grp = u - blk * G;
        valid = (u < g.NB * G) && (blk * SB + s < g.Vh);
        own = (size_t)u * US + s * R + hoff;
        own_n = (size_t)u * UN + s * R + hoff;
        rhs0 = grp * R + hoff;
    }
};

struct BlasGeom { Geom g; int N, G; };

template <class S, int VW, int R>
__global__ void norm2_kernel(BlasGeom bg, SView<S> x, double* partials, unsigned int* counter, double* out) {
    using T = typename S::comp_t;
    BlasIdx<VW, R> ix(bg.g, bg.G);
    double part[VW];
#pragma unroll
    for (int k = 0; k < VW; k++) part[k] = 0.0;
    if (ix.valid) {
        T a[24][VW];
        load_site_regs<S, VW, R>(x.d + ix.own, S::has_norm ? x.n + ix.own_n : nullptr, a);
#pragma unroll
        for (int j = 0; j < 24; j++)
#pragma unroll
            for (int k = 0; k < VW; k++) part[k] += (double)a[j][k] * (double)a[j][k];
    }
    reduce_per_rhs<VW, R>(part, bg.N, bg.G, partials, counter, out);
}

// e += alpha p ; p = z + beta p   (alpha = rr / pAp, beta = rr_new / rr)
template <class S, int VW, int R>
__global__ void cg_update_ep_kernel(BlasGeom bg, SView<S> e, SView<S> p, SView<S> z, const double* __restrict__ rr, const double* __restrict__ pAp,
                                    const double* __restrict__ rr_new) {
    using T = typename S::comp_t;
    BlasIdx<VW, R> ix(bg.g, bg.G);
    if (!ix.valid) return;
    T alpha[VW], beta[VW];
#pragma unroll
    for (int k = 0; k < VW; k++) {
        const double d = pAp[ix.rhs0 + k], r0 = rr[ix.rhs0 + k];
        alpha[k] = (T)(d > 0.0 ? r0 / d : 0.0);
        beta[k] = (T)(r0 > 0.0 ? rr_new[ix.rhs0 + k] / r0 : 0.0);
    }
    T a[24][VW], b[24][VW];
    load_site_regs<S, VW, R>(e.d + ix.own, S::has_norm ? e.n + ix.own_n : nullptr, a);
    load_site_regs<S, VW, R>(p.d + ix.own, S::has_norm ? p.n + ix.own_n : nullptr, b);
#pragma unroll
    for (int j = 0; j < 24; j++)
#pragma unroll
        for (int k = 0; k < VW; k++) a[j][k] += alpha[k] * b[j][k];
    store_site_regs<S, VW, R>(e.d + ix.own, S::has_norm ? e.n + ix.own_n : nullptr, a);
    load_site_regs<S, VW, R>(z.d + ix.own, S::has_norm ? z.n + ix.own_n : nullptr, a);
#pragma unroll
    for (int j = 0; j < 24; j++)
#pragma unroll
        for (int k = 0; k < VW; k++) b[j][k] = a[j][k] + beta[k] * b[j][k];
    store_site_regs<S, VW, R>(p.d + ix.own, S::has_norm ? p.n + ix.own_n : nullptr, b);
}

// p <- z_new + c (p - z_old)
template <class S, int VW, int R>
__global__ void keep_direction_kernel(BlasGeom bg, SView<S> p, SView<S> zo, SView<S> zn, const double* __restrict__ cs) {
    using T = typename S::comp_t;
    BlasIdx<VW, R> ix(bg.g, bg.G);
    if (!ix.valid) return;
    T cf[VW];
#pragma unroll
    for (int k = 0; k < VW; k++) cf[k] = (T)cs[ix.rhs0 + k];
    T a[24][VW], b[24][VW];
    load_site_regs<S, VW, R>(p.d + ix.own, S::has_norm ? p.n + ix.own_n : nullptr, a);
    load_site_regs<S, VW, R>(zo.d + ix.own, S::has_norm ? zo.n + ix.own_n : nullptr, b);
#pragma unroll
    for (int j = 0; j < 24; j++)
#pragma unroll
        for (int k = 0; k < VW; k++) a[j][k] = cf[k] * (a[j][k] - b[j][k]);
    load_site_regs<S, VW, R>(zn.d + ix.own, S::has_norm ? zn.n + ix.own_n : nullptr, b);
#pragma unroll
    for (int j = 0; j < 24; j++)
#pragma unroll
        for (int k = 0; k < VW; k++) a[j][k] += b[j][k];
    store_site_regs<S, VW, R>(p.d + ix.own, S::has_norm ? p.n + ix.own_n : nullptr, a);
}

// y (fp64) += s_k * e
template <class S, int VW, int R>
__global__ void axpy_mixed_kernel(BlasGeom bg, double* __restrict__ y, SView<S> ev, const double* __restrict__ scale) {
    using T = typename S::comp_t;
    BlasIdx<VW, R> ix(bg.g, bg.G);
    if (!ix.valid) return;
    T a[24][VW];
    load_site_regs<S, VW, R>(ev.d + ix.own, S::has_norm ? ev.n + ix.own_n : nullptr, a);
#pragma unroll
    for (int j = 0; j < 24; j++)
#pragma unroll
        for (int k = 0; k < VW; k++) y[ix.own + j * ix.PL + k] += scale[ix.rhs0 + k] * (double)a[j][k];
}

// r = b - t (fp64), per-RHS ||r||^2
template <int VW, int R>
__global__ void residual_kernel(BlasGeom bg, double* __restrict__ r, const double* __restrict__ b, const double* __restrict__ tv,
                                double* partials, unsigned int* counter, double* out) {
    BlasIdx<VW, R> ix(bg.g, bg.G);
    double part[VW];
#pragma unroll
    for (int k = 0; k < VW; k++) part[k] = 0.0;
    if (ix.valid) {
#pragma unroll
        for (int j = 0; j < 24; j++)
#pragma unroll
            for (int k = 0; k < VW; k++) {
                const size_t i = ix.own + j * ix.PL + k;
                const double d = b[i] - tv[i];
                r[i] = d; part[k] += d * d;
            }
    }
    reduce_per_rhs<VW, R>(part, bg.N, bg.G, partials, counter, out);
}

// ---- host side -----------------------------------------------------------------------------------------------------
struct Launch { BlasGeom bg; int R, vw, block, grid; size_t smem; };
static int plan(lq_ctx* c, int nrhs, int maxvw, Launch& L) {
    const int R = group_width(nrhs);
    L.R = R; L.vw = R < maxvw ? R : maxvw;
    L.bg.g = c->g; L.bg.N = nrhs; L.bg.G = nrhs / R;
    L.block = 128;
    const long long threads = (long long)c->g.NB * L.bg.G * SB * (R / L.vw);
    L.grid = (int)((threads + L.block - 1) / L.block);
    L.smem = (size_t)L.block * sizeof(double);
    LQ_TRY(ensure_partials(c, (size_t)L.grid * nrhs));
    return 0;
}
// dispatch on (VW, R): fp32/half (4,4) (2,2) (1,1); fp64 (2,4) (2,2) (1,1)
#define VW_DISPATCH(L, S, KERNEL, SMEM, ...)                                                                      \
    do {                                                                                                          \
        constexpr bool F64K_ = S::prec == LQ_FP64;                                                                \
        if (L.R == 4) KERNEL<S, (F64K_ ? 2 : 4), 4><<<L.grid, L.block, SMEM, c->stream>>>(__VA_ARGS__);           \
        else if (L.R == 2) KERNEL<S, 2, 2><<<L.grid, L.block, SMEM, c->stream>>>(__VA_ARGS__);                    \
        else KERNEL<S, 1, 1><<<L.grid, L.block, SMEM, c->stream>>>(__VA_ARGS__);                                  \
    } while (0)

template <class S> static int norm2_t(lq_ctx* c, int nrhs, const void* x, double* d_out) {
    Launch L; LQ_TRY(plan(c, nrhs, S::prec == LQ_FP64 ? 2 : 4, L));
    SView<S> vx = make_view<S>(c->g, const_cast<void*>(x), nrhs, 0);
    VW_DISPATCH(L, S, norm2_kernel, L.smem, L.bg, vx, c->red_partials, c->red_counter, d_out);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
int blas_norm2(lq_ctx* c, int prec, int nrhs, const void* x, double* d_out) {
    if (prec == LQ_FP64) return norm2_t<F64>(c, nrhs, x, d_out);
    if (prec == LQ_FP32) return norm2_t<F32>(c, nrhs, x, d_out);
    return norm2_t<H16>(c, nrhs, x, d_out);
}

template <class S> static int ep_t(lq_ctx* c, int nrhs, void* e, void* p, const void* z, const double* rr, const double* pAp, const double* rrn) {
    Launch L; LQ_TRY(plan(c, nrhs, S::prec == LQ_FP64 ? 2 : 4, L));
    SView<S> ve = make_view<S>(c->g, e, nrhs, 0), vp = make_view<S>(c->g, p, nrhs, 0), vz = make_view<S>(c->g, const_cast<void*>(z), nrhs, 0);
    VW_DISPATCH(L, S, cg_update_ep_kernel, 0, L.bg, ve, vp, vz, rr, pAp, rrn);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
int blas_cg_update_ep(lq_ctx* c, int prec, int nrhs, void* e, void* p, const void* z, const double* d_rr, const double* d_pAp, const double* d_rr_new) {
    if (prec == LQ_FP64) return ep_t<F64>(c, nrhs, e, p, z, d_rr, d_pAp, d_rr_new);
    if (prec == LQ_FP32) return ep_t<F32>(c, nrhs, e, p, z, d_rr, d_pAp, d_rr_new);
    return ep_t<H16>(c, nrhs, e, p, z, d_rr, d_pAp, d_rr_new);
}

template <class S> static int keep_t(lq_ctx* c, int nrhs, void* p, const void* zo, const void* zn, const double* cs) {
    Launch L; LQ_TRY(plan(c, nrhs, S::prec == LQ_FP64 ? 2 : 4, L));
    SView<S> vp = make_view<S>(c->g, p, nrhs, 0), vo = make_view<S>(c->g, const_cast<void*>(zo), nrhs, 0), vn = make_view<S>(c->g, const_cast<void*>(zn), nrhs, 0);
    VW_DISPATCH(L, S, keep_direction_kernel, 0, L.bg, vp, vo, vn, cs);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
int blas_keep_direction(lq_ctx* c, int prec, int nrhs, void* p, const void* z_old, const void* z_new, const double* d_c) {
    if (prec == LQ_FP64) return keep_t<F64>(c, nrhs, p, z_old, z_new, d_c);
    if (prec == LQ_FP32) return keep_t<F32>(c, nrhs, p, z_old, z_new, d_c);
    return keep_t<H16>(c, nrhs, p, z_old, z_new, d_c);
}

template <class S> static int axpy_t(lq_ctx* c, int nrhs, void* y, const void* e, const double* s) {
    Launch L; LQ_TRY(plan(c, nrhs, S::prec == LQ_FP64 ? 2 : 4, L));
    SView<S> ve = make_view<S>(c->g, const_cast<void*>(e), nrhs, 0);
    VW_DISPATCH(L, S, axpy_mixed_kernel, 0, L.bg, (double*)y, ve, s);
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
    double* rp = (double*)r; const double* bp = (const double*)b; const double* tp = (const double*)t;
    if (L.R == 4) residual_kernel<2, 4><<<L.grid, L.block, L.smem, c->stream>>>(L.bg, rp, bp, tp, c->red_partials, c->red_counter, d_out);
    else if (L.R == 2) residual_kernel<2, 2><<<L.grid, L.block, L.smem, c->stream>>>(L.bg, rp, bp, tp, c->red_partials, c->red_counter, d_out);
    else residual_kernel<1, 1><<<L.grid, L.block, L.smem, c->stream>>>(L.bg, rp, bp, tp, c->red_partials, c->red_counter, d_out);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}

int blas_copy(lq_ctx* c, int prec, int nrhs, void* dst, const void* src) {
    LQ_CUDA(c, cudaMemcpyAsync(dst, src, parity_bytes(c->g, nrhs, prec), cudaMemcpyDeviceToDevice, c->stream));
    return 0;
}
