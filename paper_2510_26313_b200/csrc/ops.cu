// ops.cu -- precision dispatch of the single-parity building blocks.
#include "internal.cuh"
#include "dslash_kernel.cuh"

template <class S>
static DslashArgs<S> base_args(lq_ctx* c, int nrhs, int out_parity, void* out, const void* in, const void* x, int dagger) {
    using T = typename S::comp_t;
    DslashArgs<S> a;
    a.g = c->g; a.parity = out_parity; a.N = nrhs; a.G = 0;
    a.out = make_view<S>(c->g, out, nrhs, 0);
    a.in = make_view<S>(c->g, const_cast<void*>(in), nrhs, 0);
    a.x = make_view<S>(c->g, const_cast<void*>(x), nrhs, 0);
    if constexpr (S::prec == LQ_FP64) a.gauge = c->gauge64; else a.gauge = c->gauge32;
    a.clover = nullptr;
    a.coef = T(1); a.tsign = T(c->t_bc); a.dsign = dagger ? T(-1) : T(1);
    return a;
}

template <class S, int FORM>
static int run_form(lq_ctx* c, DslashArgs<S> a) {
    if constexpr (S::prec == LQ_FP64) return launch_dslash<S, 18, FORM>(c, a, c->dslash_rpt);
    else {
        if (c->recon32 == 12) return launch_dslash<S, 12, FORM>(c, a, c->dslash_rpt);
        return launch_dslash<S, 18, FORM>(c, a, c->dslash_rpt);
    }
}

template <class S> static const typename S::comp_t* clover_ptr(lq_ctx* c, int parity, int inverse) {
    if constexpr (S::prec == LQ_FP64) return (inverse ? c->clovinv64 : c->clov64) + (size_t)parity * 72 * c->g.Vh;
    else return (inverse ? c->clovinv32 : c->clov32) + (size_t)parity * 72 * c->g.Vh;
}

int op_hop(lq_ctx* c, int prec, int nrhs, int out_parity, void* out, const void* in, int dagger) {
    if (prec == LQ_FP64) return run_form<F64, FORM_HOP>(c, base_args<F64>(c, nrhs, out_parity, out, in, nullptr, dagger));
    if (prec == LQ_FP32) return run_form<F32, FORM_HOP>(c, base_args<F32>(c, nrhs, out_parity, out, in, nullptr, dagger));
    return run_form<H16, FORM_HOP>(c, base_args<H16>(c, nrhs, out_parity, out, in, nullptr, dagger));
}

template <class S> static int kernel_a_t(lq_ctx* c, int nrhs, int out_parity, void* out, const void* in, int dagger) {
    auto a = base_args<S>(c, nrhs, out_parity, out, in, nullptr, dagger);
    a.clover = clover_ptr<S>(c, out_parity, 1);
    return run_form<S, FORM_A>(c, a);
}
int op_kernel_a(lq_ctx* c, int prec, int nrhs, int out_parity, void* out, const void* in, int dagger) {
    if (prec == LQ_FP64) return kernel_a_t<F64>(c, nrhs, out_parity, out, in, dagger);
    if (prec == LQ_FP32) return kernel_a_t<F32>(c, nrhs, out_parity, out, in, dagger);
    return kernel_a_t<H16>(c, nrhs, out_parity, out, in, dagger);
}

template <class S> static int kernel_b_t(lq_ctx* c, int nrhs, int out_parity, void* out, const void* x, const void* in, double coef, int use_clover, int dagger) {
    auto a = base_args<S>(c, nrhs, out_parity, out, in, x, dagger);
    a.clover = use_clover ? clover_ptr<S>(c, out_parity, 0) : nullptr;
    a.coef = (typename S::comp_t)coef;
    return run_form<S, FORM_B>(c, a);
}
int op_kernel_b(lq_ctx* c, int prec, int nrhs, int out_parity, void* out, const void* x, const void* in, double coef, int use_clover, int dagger) {
    if (prec == LQ_FP64) return kernel_b_t<F64>(c, nrhs, out_parity, out, x, in, coef, use_clover, dagger);
    if (prec == LQ_FP32) return kernel_b_t<F32>(c, nrhs, out_parity, out, x, in, coef, use_clover, dagger);
    return kernel_b_t<H16>(c, nrhs, out_parity, out, x, in, coef, use_clover, dagger);
}

// ---- site-local clover apply: out = C x --------------------------------------------------------------------
template <class S, int RPT>
__global__ void __launch_bounds__(256) clover_apply_kernel(Geom g, int N, int G, SView<S> out, SView<S> x, const typename S::comp_t* __restrict__ clover) {
    using T = typename S::comp_t;
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= g.Vh * G) return;
    const int cb = tid / G, goff = (tid - cb * G) * RPT;
    const size_t plane = (size_t)g.Vh * N;
    T sc[RPT];
    if constexpr (S::has_norm) {
        float nrm[RPT];
        load_norm<RPT>(x.n + (size_t)cb * N + goff, nrm);
#pragma unroll
        for (int k = 0; k < RPT; k++) sc[k] = nrm[k] * (1.0f / 32767.0f);
    }
    T res[24][RPT];
#pragma unroll
    for (int b = 0; b < 2; b++) {
        T v[6][2][RPT], o[6][2][RPT], cl[36];
#pragma unroll
        for (int i = 0; i < 6; i++)
#pragma unroll
            for (int ri = 0; ri < 2; ri++) {
                load_comp<S, RPT>(x.d + (size_t)(12 * b + 2 * i + ri) * plane + (size_t)cb * N + goff, v[i][ri]);
                if constexpr (S::has_norm) {
#pragma unroll
                    for (int k = 0; k < RPT; k++) v[i][ri][k] *= sc[k];
                }
            }
        load_planes<T, 36>(clover + (size_t)b * 36 * g.Vh, g.Vh, cb, cl);
        clover_block_mul<T, RPT>(cl, v, o);
#pragma unroll
        for (int i = 0; i < 6; i++)
#pragma unroll
            for (int ri = 0; ri < 2; ri++)
#pragma unroll
                for (int k = 0; k < RPT; k++) res[12 * b + 2 * i + ri][k] = o[i][ri][k];
    }
    typename S::store_t* ob = out.d + (size_t)cb * N + goff;
    if constexpr (S::has_norm) {
        float mx[RPT], inv[RPT];
#pragma unroll
        for (int k = 0; k < RPT; k++) mx[k] = 0.f;
#pragma unroll
        for (int j = 0; j < 24; j++)
#pragma unroll
            for (int k = 0; k < RPT; k++) mx[k] = fmaxf(mx[k], fabsf(res[j][k]));
#pragma unroll
        for (int k = 0; k < RPT; k++) { inv[k] = mx[k] > 0.f ? 32767.0f / mx[k] : 0.f; out.n[(size_t)cb * N + goff + k] = mx[k]; }
#pragma unroll
        for (int j = 0; j < 24; j++) {
            T q[RPT];
#pragma unroll
            for (int k = 0; k < RPT; k++) q[k] = rintf(res[j][k] * inv[k]);
            store_comp<S, RPT>(ob + (size_t)j * plane, q);
        }
    } else {
#pragma unroll
        for (int j = 0; j < 24; j++) store_comp<S, RPT>(ob + (size_t)j * plane, res[j]);
    }
}

template <class S> static int clover_t(lq_ctx* c, int nrhs, int parity, void* out, const void* x, int inverse) {
    SView<S> vo = make_view<S>(c->g, out, nrhs, 0), vx = make_view<S>(c->g, const_cast<void*>(x), nrhs, 0);
    const typename S::comp_t* cl = clover_ptr<S>(c, parity, inverse);
    const int rpt = (nrhs % 2 == 0) ? 2 : 1;
    const int G = nrhs / rpt;
    const long long threads = (long long)c->g.Vh * G;
    const int block = 128, grid = (int)((threads + block - 1) / block);
    if (rpt == 2) clover_apply_kernel<S, 2><<<grid, block, 0, c->stream>>>(c->g, nrhs, G, vo, vx, cl);
    else clover_apply_kernel<S, 1><<<grid, block, 0, c->stream>>>(c->g, nrhs, G, vo, vx, cl);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
int op_clover(lq_ctx* c, int prec, int nrhs, int parity, void* out, const void* x, int inverse) {
    if (prec == LQ_FP64) return clover_t<F64>(c, nrhs, parity, out, x, inverse);
    if (prec == LQ_FP32) return clover_t<F32>(c, nrhs, parity, out, x, inverse);
    return clover_t<H16>(c, nrhs, parity, out, x, inverse);
}
