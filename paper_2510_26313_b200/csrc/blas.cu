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

struct BlasGeom { Geom g; int N, G; const int* skip; };   // skip: see lq_ctx::loop_skip
#define LQ_BLAS_SKIP(bg) do { if ((bg).skip != nullptr && *(volatile const int*)(bg).skip) return; } while (0)

template <class S, int VW, int R>
__global__ void norm2_kernel(BlasGeom bg, SView<S> x, double* partials) {
    LQ_BLAS_SKIP(bg);
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
    reduce_per_rhs<VW, R>(part, bg.N, bg.G, partials);
}

// e += alpha p ; p = z + beta p   (alpha = rr / pAp, beta = rr_new / rr)
template <class S, int VW, int R>
__global__ void cg_update_ep_kernel(BlasGeom bg, SView<S> e, SView<S> p, SView<S> z, const double* __restrict__ rr, const double* __restrict__ pAp,
                                    const double* __restrict__ rr_new) {
    LQ_BLAS_SKIP(bg);
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

// p <- z_new + c (p - z_old) ; z_old <- z_new  (the vector buffers keep their roles, so the cached iteration graph stays valid)
template <class S, int VW, int R>
__global__ void keep_direction_kernel(BlasGeom bg, SView<S> p, SView<S> zo, SView<S> zn, const double* __restrict__ cs) {
    LQ_BLAS_SKIP(bg);
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
    store_site_regs<S, VW, R>(zo.d + ix.own, S::has_norm ? zo.n + ix.own_n : nullptr, b);
#pragma unroll
    for (int j = 0; j < 24; j++)
#pragma unroll
        for (int k = 0; k < VW; k++) a[j][k] += b[j][k];
    store_site_regs<S, VW, R>(p.d + ix.own, S::has_norm ? p.n + ix.own_n : nullptr, a);
}

// y (fp64) += s_k * e
template <class S, int VW, int R>
__global__ void axpy_mixed_kernel(BlasGeom bg, double* __restrict__ y, SView<S> ev, const double* __restrict__ scale) {
    LQ_BLAS_SKIP(bg);
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
                                double* partials) {
    LQ_BLAS_SKIP(bg);
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
    reduce_per_rhs<VW, R>(part, bg.N, bg.G, partials);
}

// ---- second stage of every per-RHS reduction (reduce.cuh): rows[nrows][NC] -> out[(col / N1) * LQ_MAX_RHS + col % N1] ----------
// <= 256 blocks, each over a contiguous range of rows (thread = column x row slice, fixed order, shared-memory tree over the
// slices), then the last block to finish adds the block rows in index order.  The only fence / atomic of the whole reduction.
constexpr int RF_THREADS = 256, RF_MAXB = 256;
__global__ void __launch_bounds__(RF_THREADS) reduce_finish_kernel(const double* __restrict__ rows, int nrows, int NC, int N1, double* stage2,
                                                                   unsigned int* counter, double* __restrict__ out, const int* skip) {
    if (skip != nullptr && *(volatile const int*)skip) return;
    __shared__ double sm[RF_THREADS];
    __shared__ bool last;
    const int t = threadIdx.x;
    int Q = 1;                                   // row slices per block: largest power of two with NC * Q <= RF_THREADS
    while (NC * Q * 2 <= RF_THREADS) Q <<= 1;
    const int col = t % NC, q = t / NC;
    const int per = (nrows + gridDim.x - 1) / gridDim.x;
    const int r0 = blockIdx.x * per, r1 = min(nrows, r0 + per);
    double s = 0.0;
    if (q < Q) for (int r = r0 + q; r < r1; r += Q) s += __ldcg(rows + (size_t)r * NC + col);
    if (q < Q) sm[t] = s;
    __syncthreads();
    for (int stride = Q >> 1; stride >= 1; stride >>= 1) {
        if (q < stride) sm[t] += sm[t + stride * NC];
        __syncthreads();
    }
    if (t < NC) stage2[(size_t)blockIdx.x * NC + t] = sm[t];
    __threadfence();
    __syncthreads();
    if (t == 0) last = (atomicInc(counter, gridDim.x - 1) == gridDim.x - 1);
    __syncthreads();
    if (!last) return;
    __threadfence();
    if (t < NC) {
        double f = 0.0;
        for (unsigned b = 0; b < gridDim.x; b++) f += __ldcg(stage2 + (size_t)b * NC + t);
        out[(t / N1) * LQ_MAX_RHS + (t % N1)] = f;
    }
}
int reduce_finish(lq_ctx* c, int nrows, int nq, int n1, double* d_out) {
    const int NC = nq * n1;
    int P = nrows / 64;
    if (P < 1) P = 1;
    if (P > RF_MAXB) P = RF_MAXB;
    reduce_finish_kernel<<<P, RF_THREADS, 0, c->stream>>>(c->red_partials, nrows, NC, n1, c->red_partials + (size_t)nrows * NC,
                                                          c->red_counter + RED_COUNTER_BASE, d_out, c->loop_skip);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}

// ---- host side -----------------------------------------------------------------------------------------------------
struct Launch { BlasGeom bg; int R, vw, block, grid; size_t smem; };
// modelled work of a block-BLAS launch: `streams` passes over a parity batch in precision prec, `fl` flops per site per RHS
#define BLAS_MODEL(c, prec, nrhs, streams, fl) LQ_MODEL(c, (streams) * stream_bytes((c)->g, nrhs, prec), (double)(fl) * (c)->g.Vh * (nrhs))
static int plan(lq_ctx* c, int nrhs, int maxvw, Launch& L) {
    const int R = group_width(nrhs);
    L.R = R; L.vw = R < maxvw ? R : maxvw;
    L.bg.g = c->g; L.bg.N = nrhs; L.bg.G = nrhs / R; L.bg.skip = c->loop_skip;
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
    VW_DISPATCH(L, S, norm2_kernel, L.smem, L.bg, vx, c->red_partials);
    LQ_LAUNCHED(c);
    LQ_TRY(reduce_finish(c, L.grid, 1, nrhs, d_out));
    BLAS_MODEL(c, S::prec, nrhs, 1, 48);
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
    BLAS_MODEL(c, S::prec, nrhs, 5, 96);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
int blas_cg_update_ep(lq_ctx* c, int prec, int nrhs, void* e, void* p, const void* z, const double* d_rr, const double* d_pAp, const double* d_rr_new) {
    if (prec == LQ_FP64) return ep_t<F64>(c, nrhs, e, p, z, d_rr, d_pAp, d_rr_new);
    if (prec == LQ_FP32) return ep_t<F32>(c, nrhs, e, p, z, d_rr, d_pAp, d_rr_new);
    return ep_t<H16>(c, nrhs, e, p, z, d_rr, d_pAp, d_rr_new);
}

template <class S> static int keep_t(lq_ctx* c, int nrhs, void* p, void* zo, const void* zn, const double* cs) {
    Launch L; LQ_TRY(plan(c, nrhs, S::prec == LQ_FP64 ? 2 : 4, L));
    SView<S> vp = make_view<S>(c->g, p, nrhs, 0), vo = make_view<S>(c->g, zo, nrhs, 0), vn = make_view<S>(c->g, const_cast<void*>(zn), nrhs, 0);
    VW_DISPATCH(L, S, keep_direction_kernel, 0, L.bg, vp, vo, vn, cs);
    LQ_LAUNCHED(c);
    BLAS_MODEL(c, S::prec, nrhs, 5, 96);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
int blas_keep_direction(lq_ctx* c, int prec, int nrhs, void* p, void* z_old, const void* z_new, const double* d_c) {
    if (prec == LQ_FP64) return keep_t<F64>(c, nrhs, p, z_old, z_new, d_c);
    if (prec == LQ_FP32) return keep_t<F32>(c, nrhs, p, z_old, z_new, d_c);
    return keep_t<H16>(c, nrhs, p, z_old, z_new, d_c);
}

template <class S> static int axpy_t(lq_ctx* c, int nrhs, void* y, const void* e, const double* s) {
    Launch L; LQ_TRY(plan(c, nrhs, S::prec == LQ_FP64 ? 2 : 4, L));
    SView<S> ve = make_view<S>(c->g, const_cast<void*>(e), nrhs, 0);
    VW_DISPATCH(L, S, axpy_mixed_kernel, 0, L.bg, (double*)y, ve, s);
    LQ_LAUNCHED(c);
    BLAS_MODEL(c, S::prec, nrhs, 1, 48); BLAS_MODEL(c, LQ_FP64, nrhs, 2, 0);
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
    if (L.R == 4) residual_kernel<2, 4><<<L.grid, L.block, L.smem, c->stream>>>(L.bg, rp, bp, tp, c->red_partials);
    else if (L.R == 2) residual_kernel<2, 2><<<L.grid, L.block, L.smem, c->stream>>>(L.bg, rp, bp, tp, c->red_partials);
    else residual_kernel<1, 1><<<L.grid, L.block, L.smem, c->stream>>>(L.bg, rp, bp, tp, c->red_partials);
    LQ_LAUNCHED(c);
    LQ_TRY(reduce_finish(c, L.grid, 1, nrhs, d_out));
    BLAS_MODEL(c, LQ_FP64, nrhs, 3, 72);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}

int blas_copy(lq_ctx* c, int prec, int nrhs, void* dst, const void* src) {
    LQ_CUDA(c, cudaMemcpyAsync(dst, src, parity_bytes(c->g, nrhs, prec), cudaMemcpyDeviceToDevice, c->stream));
    BLAS_MODEL(c, prec, nrhs, 2, 0);
    return 0;
}

// ---- batched BiCGStab block-BLAS (solver variant): per-RHS COMPLEX Krylov scalars ------------------------
// Component j of a site is (re, im) = (2c, 2c+1), c = 3 spin + colour.  Device scalars are kept as raw sums,
//   rho[2][LQ_MAX_RHS] = <rhat0, r>,  c1[3][..] = (<rhat0, v>, ||rhat0||^2),  d2[3][..] = (<t, s>, ||t||^2),
// and every kernel derives alpha = rho / c1, omega = <t, s> / ||t||^2, beta = (rho' / rho)(alpha / omega) from them (zero when a
// denominator is zero: converged or zero right-hand sides stay put).  Two right-hand sides per thread (registers).
namespace {
struct Cplx { double re, im; };
__device__ __forceinline__ Cplx cdiv(double ar, double ai, double br, double bi) {
    const double d = br * br + bi * bi;
    if (!(d > 0.0)) return Cplx{0.0, 0.0};
    return Cplx{(ar * br + ai * bi) / d, (ai * br - ar * bi) / d};
}
__device__ __forceinline__ Cplx cmul(Cplx a, Cplx b) { return Cplx{a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
__device__ __forceinline__ Cplx bicg_alpha(const double* rho, const double* c1, int k) { return cdiv(rho[k], rho[LQ_MAX_RHS + k], c1[k], c1[LQ_MAX_RHS + k]); }
__device__ __forceinline__ Cplx bicg_omega(const double* d2, int k) {
    const double tt = d2[2 * LQ_MAX_RHS + k];
    return tt > 0.0 ? Cplx{d2[k] / tt, d2[LQ_MAX_RHS + k] / tt} : Cplx{0.0, 0.0};
}
// y[c] (+)= s * x[c] for the 12 complex components of VW right-hand sides
template <class T, int VW, bool ACCUM>
__device__ __forceinline__ void caxpy_regs(const T (&sr)[VW], const T (&si)[VW], const T (&x)[24][VW], T (&y)[24][VW]) {
#pragma unroll
    for (int cc = 0; cc < 12; cc++)
#pragma unroll
        for (int k = 0; k < VW; k++) {
            const T xr = x[2 * cc][k], xi = x[2 * cc + 1][k];
            const T pr = sr[k] * xr - si[k] * xi, pi = sr[k] * xi + si[k] * xr;
            if (ACCUM) { y[2 * cc][k] += pr; y[2 * cc + 1][k] += pi; } else { y[2 * cc][k] = pr; y[2 * cc + 1][k] = pi; }
        }
}
}  // namespace

// out = (Re <a, b>, Im <a, b>, ||a||^2) per RHS, <a, b> = sum conj(a) b
template <class S, int VW, int R>
__global__ void cdot3_kernel(BlasGeom bg, SView<S> a, SView<S> b, double* partials) {
    LQ_BLAS_SKIP(bg);
    using T = typename S::comp_t;
    BlasIdx<VW, R> ix(bg.g, bg.G);
    double part[3][VW];
#pragma unroll
    for (int q = 0; q < 3; q++)
#pragma unroll
        for (int k = 0; k < VW; k++) part[q][k] = 0.0;
    if (ix.valid) {
        T x[24][VW], y[24][VW];
        load_site_regs<S, VW, R>(a.d + ix.own, S::has_norm ? a.n + ix.own_n : nullptr, x);
        load_site_regs<S, VW, R>(b.d + ix.own, S::has_norm ? b.n + ix.own_n : nullptr, y);
#pragma unroll
        for (int cc = 0; cc < 12; cc++)
#pragma unroll
            for (int k = 0; k < VW; k++) {
                const double ar = x[2 * cc][k], ai = x[2 * cc + 1][k], br = y[2 * cc][k], bi = y[2 * cc + 1][k];
                part[0][k] += ar * br + ai * bi; part[1][k] += ar * bi - ai * br; part[2][k] += ar * ar + ai * ai;
            }
    }
    reduce_multi<3, VW, R>(part, bg.N, bg.G, partials);
}

// s = r - alpha v
template <class S, int VW, int R>
__global__ void bicg_s_kernel(BlasGeom bg, SView<S> s, SView<S> r, SView<S> v, const double* __restrict__ rho, const double* __restrict__ c1) {
    LQ_BLAS_SKIP(bg);
    using T = typename S::comp_t;
    BlasIdx<VW, R> ix(bg.g, bg.G);
    if (!ix.valid) return;
    T ar[VW], ai[VW];
#pragma unroll
    for (int k = 0; k < VW; k++) { const Cplx a = bicg_alpha(rho, c1, ix.rhs0 + k); ar[k] = (T)(-a.re); ai[k] = (T)(-a.im); }
    T x[24][VW], y[24][VW];
    load_site_regs<S, VW, R>(r.d + ix.own, S::has_norm ? r.n + ix.own_n : nullptr, y);
    load_site_regs<S, VW, R>(v.d + ix.own, S::has_norm ? v.n + ix.own_n : nullptr, x);
    caxpy_regs<T, VW, true>(ar, ai, x, y);
    store_site_regs<S, VW, R>(s.d + ix.own, S::has_norm ? s.n + ix.own_n : nullptr, y);
}

// e += alpha p + omega s ; r = s - omega t ; out = (<rhat0, r>, ||rhat0||^2 (unused), ...) -> (Re, Im <rhat0, r>, ||r||^2)
template <class S, int VW, int R>
__global__ void bicg_xr_kernel(BlasGeom bg, SView<S> e, SView<S> r, SView<S> p, SView<S> s, SView<S> tv, SView<S> rhat,
                               const double* __restrict__ rho, const double* __restrict__ c1, const double* __restrict__ d2,
                               double* partials) {
    LQ_BLAS_SKIP(bg);
    using T = typename S::comp_t;
    BlasIdx<VW, R> ix(bg.g, bg.G);
    double part[3][VW];
#pragma unroll
    for (int q = 0; q < 3; q++)
#pragma unroll
        for (int k = 0; k < VW; k++) part[q][k] = 0.0;
    if (ix.valid) {
        T ar[VW], ai[VW], wr[VW], wi[VW], mwr[VW], mwi[VW];
#pragma unroll
        for (int k = 0; k < VW; k++) {
            const Cplx a = bicg_alpha(rho, c1, ix.rhs0 + k), w = bicg_omega(d2, ix.rhs0 + k);
            ar[k] = (T)a.re; ai[k] = (T)a.im; wr[k] = (T)w.re; wi[k] = (T)w.im; mwr[k] = (T)(-w.re); mwi[k] = (T)(-w.im);
        }
        T x[24][VW], y[24][VW], z[24][VW];
        load_site_regs<S, VW, R>(s.d + ix.own, S::has_norm ? s.n + ix.own_n : nullptr, x);       // x = s
        load_site_regs<S, VW, R>(e.d + ix.own, S::has_norm ? e.n + ix.own_n : nullptr, y);       // y = e
        caxpy_regs<T, VW, true>(wr, wi, x, y);                                                    // e += omega s
        load_site_regs<S, VW, R>(p.d + ix.own, S::has_norm ? p.n + ix.own_n : nullptr, z);       // z = p
        caxpy_regs<T, VW, true>(ar, ai, z, y);                                                    // e += alpha p
        store_site_regs<S, VW, R>(e.d + ix.own, S::has_norm ? e.n + ix.own_n : nullptr, y);
        load_site_regs<S, VW, R>(tv.d + ix.own, S::has_norm ? tv.n + ix.own_n : nullptr, z);     // z = t
        caxpy_regs<T, VW, true>(mwr, mwi, z, x);                                                  // x = s - omega t = r
        store_site_regs<S, VW, R>(r.d + ix.own, S::has_norm ? r.n + ix.own_n : nullptr, x);
        load_site_regs<S, VW, R>(rhat.d + ix.own, S::has_norm ? rhat.n + ix.own_n : nullptr, z); // z = rhat0
#pragma unroll
        for (int cc = 0; cc < 12; cc++)
#pragma unroll
            for (int k = 0; k < VW; k++) {
                const double hr = z[2 * cc][k], hi = z[2 * cc + 1][k], rr = x[2 * cc][k], ri = x[2 * cc + 1][k];
                part[0][k] += hr * rr + hi * ri; part[1][k] += hr * ri - hi * rr; part[2][k] += rr * rr + ri * ri;
            }
    }
    reduce_multi<3, VW, R>(part, bg.N, bg.G, partials);
}

// p = r + beta (p - omega v), beta = (rho_new / rho)(alpha / omega)
template <class S, int VW, int R>
__global__ void bicg_p_kernel(BlasGeom bg, SView<S> p, SView<S> r, SView<S> v, const double* __restrict__ rho, const double* __restrict__ rho_new,
                              const double* __restrict__ c1, const double* __restrict__ d2) {
    LQ_BLAS_SKIP(bg);
    using T = typename S::comp_t;
    BlasIdx<VW, R> ix(bg.g, bg.G);
    if (!ix.valid) return;
    T br[VW], bi[VW], mwr[VW], mwi[VW];
#pragma unroll
    for (int k = 0; k < VW; k++) {
        const int rh = ix.rhs0 + k;
        const Cplx a = bicg_alpha(rho, c1, rh), w = bicg_omega(d2, rh);
        const Cplx q1 = cdiv(rho_new[rh], rho_new[LQ_MAX_RHS + rh], rho[rh], rho[LQ_MAX_RHS + rh]), q2 = cdiv(a.re, a.im, w.re, w.im);
        const Cplx b = cmul(q1, q2);
        br[k] = (T)b.re; bi[k] = (T)b.im; mwr[k] = (T)(-w.re); mwi[k] = (T)(-w.im);
    }
    T x[24][VW], y[24][VW], z[24][VW];
    load_site_regs<S, VW, R>(p.d + ix.own, S::has_norm ? p.n + ix.own_n : nullptr, y);       // y = p
    load_site_regs<S, VW, R>(v.d + ix.own, S::has_norm ? v.n + ix.own_n : nullptr, x);       // x = v
    caxpy_regs<T, VW, true>(mwr, mwi, x, y);                                                  // y = p - omega v
    load_site_regs<S, VW, R>(r.d + ix.own, S::has_norm ? r.n + ix.own_n : nullptr, z);       // z = r
    caxpy_regs<T, VW, true>(br, bi, y, z);                                                    // z = r + beta y
    store_site_regs<S, VW, R>(p.d + ix.own, S::has_norm ? p.n + ix.own_n : nullptr, z);
}

// two right-hand sides per thread for every precision: (2,4) (2,2) (1,1)
#define VW2_DISPATCH(L, S, KERNEL, SMEM, ...)                                                  \
    do {                                                                                       \
        if (L.R == 4) KERNEL<S, 2, 4><<<L.grid, L.block, SMEM, c->stream>>>(__VA_ARGS__);      \
        else if (L.R == 2) KERNEL<S, 2, 2><<<L.grid, L.block, SMEM, c->stream>>>(__VA_ARGS__); \
        else KERNEL<S, 1, 1><<<L.grid, L.block, SMEM, c->stream>>>(__VA_ARGS__);               \
    } while (0)
#define PREC_SWITCH(FN, ...)                                   \
    do {                                                       \
        if (prec == LQ_FP64) return FN<F64>(c, __VA_ARGS__);   \
        if (prec == LQ_FP32) return FN<F32>(c, __VA_ARGS__);   \
        return FN<H16>(c, __VA_ARGS__);                        \
    } while (0)

template <class S> static int cdot3_t(lq_ctx* c, int nrhs, const void* a, const void* b, double* d_out) {
    Launch L; LQ_TRY(plan(c, nrhs, 2, L));
    LQ_TRY(ensure_partials(c, (size_t)L.grid * nrhs * 3));
    SView<S> va = make_view<S>(c->g, const_cast<void*>(a), nrhs, 0), vb = make_view<S>(c->g, const_cast<void*>(b), nrhs, 0);
    VW2_DISPATCH(L, S, cdot3_kernel, L.smem, L.bg, va, vb, c->red_partials);
    LQ_LAUNCHED(c);
    LQ_TRY(reduce_finish(c, L.grid, 3, nrhs, d_out));
    BLAS_MODEL(c, S::prec, nrhs, 2, 144);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
int blas_cdot3(lq_ctx* c, int prec, int nrhs, const void* a, const void* b, double* d_out) { PREC_SWITCH(cdot3_t, nrhs, a, b, d_out); }

template <class S> static int bicg_s_t(lq_ctx* c, int nrhs, void* s, const void* r, const void* v, const double* rho, const double* c1) {
    Launch L; LQ_TRY(plan(c, nrhs, 2, L));
    SView<S> vs = make_view<S>(c->g, s, nrhs, 0), vr = make_view<S>(c->g, const_cast<void*>(r), nrhs, 0), vv = make_view<S>(c->g, const_cast<void*>(v), nrhs, 0);
    VW2_DISPATCH(L, S, bicg_s_kernel, 0, L.bg, vs, vr, vv, rho, c1);
    LQ_LAUNCHED(c);
    BLAS_MODEL(c, S::prec, nrhs, 3, 96);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
int blas_bicg_s(lq_ctx* c, int prec, int nrhs, void* s, const void* r, const void* v, const double* d_rho, const double* d_c1) { PREC_SWITCH(bicg_s_t, nrhs, s, r, v, d_rho, d_c1); }

template <class S> static int bicg_xr_t(lq_ctx* c, int nrhs, void* e, void* r, const void* p, const void* s, const void* t, const void* rhat,
                                        const double* rho, const double* c1, const double* d2, double* d_out) {
    Launch L; LQ_TRY(plan(c, nrhs, 2, L));
    LQ_TRY(ensure_partials(c, (size_t)L.grid * nrhs * 3));
    SView<S> ve = make_view<S>(c->g, e, nrhs, 0), vr = make_view<S>(c->g, r, nrhs, 0), vp = make_view<S>(c->g, const_cast<void*>(p), nrhs, 0),
             vs = make_view<S>(c->g, const_cast<void*>(s), nrhs, 0), vt = make_view<S>(c->g, const_cast<void*>(t), nrhs, 0),
             vh = make_view<S>(c->g, const_cast<void*>(rhat), nrhs, 0);
    VW2_DISPATCH(L, S, bicg_xr_kernel, L.smem, L.bg, ve, vr, vp, vs, vt, vh, rho, c1, d2, c->red_partials);
    LQ_LAUNCHED(c);
    LQ_TRY(reduce_finish(c, L.grid, 3, nrhs, d_out));
    BLAS_MODEL(c, S::prec, nrhs, 7, 432);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
int blas_bicg_xr(lq_ctx* c, int prec, int nrhs, void* e, void* r, const void* p, const void* s, const void* t, const void* rhat,
                 const double* d_rho, const double* d_c1, const double* d_d2, double* d_out) {
    PREC_SWITCH(bicg_xr_t, nrhs, e, r, p, s, t, rhat, d_rho, d_c1, d_d2, d_out);
}

template <class S> static int bicg_p_t(lq_ctx* c, int nrhs, void* p, const void* r, const void* v, const double* rho, const double* rho_new,
                                       const double* c1, const double* d2) {
    Launch L; LQ_TRY(plan(c, nrhs, 2, L));
    SView<S> vp = make_view<S>(c->g, p, nrhs, 0), vr = make_view<S>(c->g, const_cast<void*>(r), nrhs, 0), vv = make_view<S>(c->g, const_cast<void*>(v), nrhs, 0);
    VW2_DISPATCH(L, S, bicg_p_kernel, 0, L.bg, vp, vr, vv, rho, rho_new, c1, d2);
    LQ_LAUNCHED(c);
    BLAS_MODEL(c, S::prec, nrhs, 4, 192);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
int blas_bicg_p(lq_ctx* c, int prec, int nrhs, void* p, const void* r, const void* v, const double* d_rho, const double* d_rho_new,
                const double* d_c1, const double* d_d2) {
    PREC_SWITCH(bicg_p_t, nrhs, p, r, v, d_rho, d_rho_new, d_c1, d_d2);
}
