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
    if constexpr (S::prec == LQ_FP64) a.gauge = c->gauge64;
    else if constexpr (sizeof(typename S::link_t) == 2) a.gauge = c->gauge16;
    else a.gauge = c->gauge32;
    a.clover = nullptr;
    a.coef = T(1); a.tsign = T(c->t_bc); a.dsign = dagger ? T(-1) : T(1);
    a.epi = EPI_NONE; a.epi_num = a.epi_den = nullptr; a.epi_out = nullptr; a.red_partials = nullptr; a.red_counter = nullptr;
    a.epi_v = a.out; a.epi_conj = 0;
    a.skip = c->loop_skip;
    return a;
}

template <class S, int FORM>
static int run_form(lq_ctx* c, DslashArgs<S> a) {
    {   // SURVEY 8(d) model: every input site read once, output written once, 8 links + the clover block once per launch
        const int recon = (S::prec == LQ_FP64 || sizeof(typename S::link_t) == 2) ? 18 : c->recon32;
        const double cb = S::prec == LQ_FP64 ? 8.0 : 4.0;      // bytes per clover real
        const double lb = (double)sizeof(typename S::link_t);   // bytes per link real
        int streams = FORM == FORM_B ? 3 : 2;
        if (FORM == FORM_B && (a.epi == EPI_XMAY || a.epi == EPI_CDOT)) streams++;
        const double bytes = streams * stream_bytes(c->g, a.N, S::prec) + (double)c->g.Vh * (8.0 * recon * lb + (a.clover ? 72.0 : 0.0) * cb);
        const double flops = (double)c->g.Vh * a.N * (1320.0 + (a.clover ? 504.0 : 0.0) + (FORM == FORM_B ? 48.0 : 0.0) +
                                                      (FORM == FORM_B && a.epi != EPI_NONE ? 48.0 : 0.0) + (FORM == FORM_B && a.epi == EPI_CDOT ? 96.0 : 0.0));
        LQ_MODEL(c, bytes, flops);
    }
    if constexpr (S::prec == LQ_FP64 || sizeof(typename S::link_t) == 2) return launch_dslash<S, 18, FORM>(c, a, c->dslash_rpt, c->dslash_variant);
    else {
        if (c->recon32 == 12) return launch_dslash<S, 12, FORM>(c, a, c->dslash_rpt, c->dslash_variant);
        return launch_dslash<S, 18, FORM>(c, a, c->dslash_rpt, c->dslash_variant);
    }
}

template <class S> static const typename S::comp_t* clover_ptr(lq_ctx* c, int parity, int inverse) {
    if constexpr (S::prec == LQ_FP64) return clover_block(inverse ? c->clovinv64 : c->clov64, c->g.NB, parity, 0);
    else return clover_block(inverse ? c->clovinv32 : c->clov32, c->g.NB, parity, 0);
}

int op_hop(lq_ctx* c, int prec, int nrhs, int out_parity, void* out, const void* in, int dagger) {
    if (prec == LQ_FP64) return run_form<F64, FORM_HOP>(c, base_args<F64>(c, nrhs, out_parity, out, in, nullptr, dagger));
    if (prec == LQ_FP32) return run_form<F32, FORM_HOP>(c, base_args<F32>(c, nrhs, out_parity, out, in, nullptr, dagger));
    if (c->half_links) return run_form<H16L, FORM_HOP>(c, base_args<H16L>(c, nrhs, out_parity, out, in, nullptr, dagger));
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
    if (c->half_links) return kernel_a_t<H16L>(c, nrhs, out_parity, out, in, dagger);
    return kernel_a_t<H16>(c, nrhs, out_parity, out, in, dagger);
}

int op_probe_loads(lq_ctx* c, int prec, int nrhs, int out_parity, void* out, const void* in) {
    if (c->recon32 != 18 || (prec != LQ_FP32 && prec != LQ_HALF)) return set_err(c, LQ_EINVAL, "LQ_OP_PROBE_LOADS: fp32 or half storage with 18-real links only");
    if (prec == LQ_FP32) {
        auto a = base_args<F32>(c, nrhs, out_parity, out, in, nullptr, 0);
        a.clover = clover_ptr<F32>(c, out_parity, 1);
        return launch_dslash<F32, 18, FORM_PROBE>(c, a, c->dslash_rpt, c->dslash_variant);
    }
    auto a = base_args<H16>(c, nrhs, out_parity, out, in, nullptr, 0);
    a.clover = clover_ptr<H16>(c, out_parity, 1);
    return launch_dslash<H16, 18, FORM_PROBE>(c, a, c->dslash_rpt, c->dslash_variant);
}

template <class S> static int kernel_b_t(lq_ctx* c, int nrhs, int out_parity, void* out, const void* x, const void* in, double coef, int use_clover, int dagger,
                                         int epi, const double* num, const double* den, double* epi_out) {
    auto a = base_args<S>(c, nrhs, out_parity, out, in, x, dagger);
    a.clover = use_clover ? clover_ptr<S>(c, out_parity, 0) : nullptr;
    a.coef = (typename S::comp_t)coef;
    a.epi = epi; a.epi_num = num; a.epi_den = den; a.epi_out = epi_out;
    return run_form<S, FORM_B>(c, a);
}
int op_kernel_b_epi(lq_ctx* c, int prec, int nrhs, int out_parity, void* out, const void* x, const void* in, double coef, int use_clover, int dagger,
                    int epi, const double* num, const double* den, double* epi_out) {
    if (prec == LQ_FP64) return kernel_b_t<F64>(c, nrhs, out_parity, out, x, in, coef, use_clover, dagger, epi, num, den, epi_out);
    if (prec == LQ_FP32) return kernel_b_t<F32>(c, nrhs, out_parity, out, x, in, coef, use_clover, dagger, epi, num, den, epi_out);
    if (c->half_links) return kernel_b_t<H16L>(c, nrhs, out_parity, out, x, in, coef, use_clover, dagger, epi, num, den, epi_out);
    return kernel_b_t<H16>(c, nrhs, out_parity, out, x, in, coef, use_clover, dagger, epi, num, den, epi_out);
}
// kernel B with the fused complex inner product <h, out> (conj: <out, h>) and ||out||^2: epi_out = 3 x LQ_MAX_RHS doubles
template <class S> static int kernel_b_cdot_t(lq_ctx* c, int nrhs, int out_parity, void* out, const void* x, const void* in, double coef, int use_clover, int dagger,
                                              const void* h, int conj, double* epi_out) {
    auto a = base_args<S>(c, nrhs, out_parity, out, in, x, dagger);
    a.clover = use_clover ? clover_ptr<S>(c, out_parity, 0) : nullptr;
    a.coef = (typename S::comp_t)coef;
    a.epi = EPI_CDOT; a.epi_num = a.epi_den = nullptr; a.epi_out = epi_out;
    a.epi_v = make_view<S>(c->g, const_cast<void*>(h), nrhs, 0); a.epi_conj = conj;
    return run_form<S, FORM_B>(c, a);
}
int op_kernel_b_cdot(lq_ctx* c, int prec, int nrhs, int out_parity, void* out, const void* x, const void* in, double coef, int use_clover, int dagger,
                     const void* h, int conj, double* epi_out) {
    if (prec == LQ_FP64) return kernel_b_cdot_t<F64>(c, nrhs, out_parity, out, x, in, coef, use_clover, dagger, h, conj, epi_out);
    if (prec == LQ_FP32) return kernel_b_cdot_t<F32>(c, nrhs, out_parity, out, x, in, coef, use_clover, dagger, h, conj, epi_out);
    if (c->half_links) return kernel_b_cdot_t<H16L>(c, nrhs, out_parity, out, x, in, coef, use_clover, dagger, h, conj, epi_out);
    return kernel_b_cdot_t<H16>(c, nrhs, out_parity, out, x, in, coef, use_clover, dagger, h, conj, epi_out);
}
int op_kernel_b(lq_ctx* c, int prec, int nrhs, int out_parity, void* out, const void* x, const void* in, double coef, int use_clover, int dagger) {
    return op_kernel_b_epi(c, prec, nrhs, out_parity, out, x, in, coef, use_clover, dagger, EPI_NONE, nullptr, nullptr, nullptr);
}

// ---- site-local clover apply: out = C x --------------------------------------------------------------------
template <class S, int RPT, int R>
__global__ void __launch_bounds__(128) clover_apply_kernel(Geom g, int G, SView<S> out, SView<S> x, const typename S::comp_t* __restrict__ clover) {
    using T = typename S::comp_t;
    constexpr int TPG = R / RPT, UT = SB * TPG, US = 24 * SB * R, UN = SB * R;
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int u = tid / UT;
    if (u >= g.NB * G) return;
    const int lu = tid - u * UT;
    const int s = lu / TPG, hoff = (lu - s * TPG) * RPT;
    const int blk = u / G;
    if (blk * SB + s >= g.Vh) return;
    const size_t own = (size_t)u * US + s * R + hoff, own_n = (size_t)u * UN + s * R + hoff;
    T v[24][RPT];
    load_site_regs<S, RPT, R>(x.d + own, S::has_norm ? x.n + own_n : nullptr, v);
    clover_apply_regs<T, RPT>(clover + (size_t)blk * (72 * SB), s, v);
    store_site_regs<S, RPT, R>(out.d + own, S::has_norm ? out.n + own_n : nullptr, v);
}

template <class S> static int clover_t(lq_ctx* c, int nrhs, int parity, void* out, const void* x, int inverse) {
    SView<S> vo = make_view<S>(c->g, out, nrhs, 0), vx = make_view<S>(c->g, const_cast<void*>(x), nrhs, 0);
    const typename S::comp_t* cl = clover_ptr<S>(c, parity, inverse);
    const int R = group_width(nrhs), G = nrhs / R;
    const int block = 128;
    if (R >= 2) {   // two right-hand sides per thread
        const long long threads = (long long)c->g.NB * G * SB * (R / 2);
        const int grid = (int)((threads + block - 1) / block);
        if (R == 4) clover_apply_kernel<S, 2, 4><<<grid, block, 0, c->stream>>>(c->g, G, vo, vx, cl);
        else clover_apply_kernel<S, 2, 2><<<grid, block, 0, c->stream>>>(c->g, G, vo, vx, cl);
    } else {
        const long long threads = (long long)c->g.NB * G * SB;
        const int grid = (int)((threads + block - 1) / block);
        clover_apply_kernel<S, 1, 1><<<grid, block, 0, c->stream>>>(c->g, G, vo, vx, cl);
    }
    LQ_LAUNCHED(c);
    LQ_MODEL(c, 2 * stream_bytes(c->g, nrhs, S::prec) + (double)c->g.Vh * 72.0 * (S::prec == LQ_FP64 ? 8.0 : 4.0), 504.0 * c->g.Vh * nrhs);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
int op_clover(lq_ctx* c, int prec, int nrhs, int parity, void* out, const void* x, int inverse) {
    if (prec == LQ_FP64) return clover_t<F64>(c, nrhs, parity, out, x, inverse);
    if (prec == LQ_FP32) return clover_t<F32>(c, nrhs, parity, out, x, inverse);
    return clover_t<H16>(c, nrhs, parity, out, x, inverse);
}
