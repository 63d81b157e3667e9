// dslash_launch.cuh -- launcher body; each dslash_*.cu instantiates it for one (storage type, link reals, form).
#pragma once
#include "dslash_kernel.cuh"

template <class S, int RPT, int R, int RECON, int FORM, int MINB>
static int launch_one(lq_ctx* c, DslashArgs<S> a) {
    constexpr int BLOCK = 128;
    const long long threads = (long long)a.g.NB * a.G * SB * (R / RPT);
    const int grid = (int)((threads + BLOCK - 1) / BLOCK);
    if (FORM == FORM_B && a.epi != EPI_NONE) {
        LQ_TRY(ensure_partials(c, (size_t)grid * a.N * (a.epi == EPI_CDOT ? 3 : 1)));
        a.red_partials = c->red_partials; a.red_counter = c->red_counter;
    }
    const size_t smem = FORM == FORM_B ? BLOCK * sizeof(double) : 0;      // scratch of the fused reduction
    if constexpr (FORM == FORM_B) {
        switch (a.epi) {
        case EPI_NORM: dslash_kernel<S, RPT, R, RECON, FORM, BLOCK, MINB, EPI_NORM><<<grid, BLOCK, smem, c->stream>>>(a); break;
        case EPI_XMAY: dslash_kernel<S, RPT, R, RECON, FORM, BLOCK, MINB, EPI_XMAY><<<grid, BLOCK, smem, c->stream>>>(a); break;
        case EPI_CDOT: dslash_kernel<S, RPT, R, RECON, FORM, BLOCK, MINB, EPI_CDOT><<<grid, BLOCK, smem, c->stream>>>(a); break;
        default: dslash_kernel<S, RPT, R, RECON, FORM, BLOCK, MINB, EPI_NONE><<<grid, BLOCK, smem, c->stream>>>(a); break;
        }
    } else {
        dslash_kernel<S, RPT, R, RECON, FORM, BLOCK, MINB, EPI_NONE><<<grid, BLOCK, smem, c->stream>>>(a);
    }
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    if (FORM == FORM_B && a.epi != EPI_NONE) LQ_TRY(reduce_finish(c, grid, a.epi == EPI_CDOT ? 3 : 1, a.N, a.epi_out));
    return 0;
}

// Sweep order (DslashArgs::zc): chunk the z extent so that one time-slice of a chunk of the input batch is <= ~6.5 MB and the
// slices t-1, t, t+1 of the chunk plus the streamed links / clover / output stay inside the 126 MB L2 between their uses.
// Needs whole x-y planes per site block (Lx/2 * Ly % 32 == 0); otherwise memory order.
template <class S>
static void plan_sweep(lq_ctx* c, DslashArgs<S>& a) {
    a.zc = 0; a.nby = 1; a.dnby = a.dzc = a.dLt = make_fastdiv(1);
    if (c->dslash_zc < 0 || a.g.Vh % SB != 0 || (a.g.Lxh * a.g.L[1]) % SB != 0) return;
    const int Lz = a.g.L[2];
    int zc = c->dslash_zc;
    if (zc == 0) {
        const double layer = (double)a.g.Lxh * a.g.L[1] * a.N * 24.0 * sizeof(typename S::store_t);
        const double slice = layer * Lz;
        if (slice <= 6.6e6) return;                   // measured on B200: chunks of <= ~6.5 MB per time-slice are best
        zc = 1;
        for (int d = 1; d <= Lz; d++) if (Lz % d == 0 && d * layer <= 6.6e6) zc = d;
    }
    if (zc >= Lz || Lz % zc != 0) return;
    a.zc = zc; a.nby = a.g.Lxh * a.g.L[1] / SB;
    a.dnby = make_fastdiv(a.nby); a.dzc = make_fastdiv(zc); a.dLt = make_fastdiv(a.g.L[3]);
}

// Register budget per thread = 65536 / (128 * MINB): MINB 2 -> 255, 3 -> 168, 4 -> 128, 5 -> 96 (rounded by ptxas).
// `variant` (tuning knob): 0 = default budget, 1 = alternative budget (fp32 only).
template <class S, int RPT, int R, int RECON, int FORM>
static int launch_rpt(lq_ctx* c, DslashArgs<S> a, int variant) {
    constexpr bool F64K = S::prec == LQ_FP64;
    constexpr int DEF = F64K ? (RPT == 2 ? 2 : 3) : (RPT == 4 ? 2 : (RPT == 2 ? 3 : 4));
    a.G = a.N / R;
    a.dG = make_fastdiv(a.G);
    a.pfd = c->dslash_pfd;
    plan_sweep<S>(c, a);
    if constexpr (S::prec != LQ_FP64) {
        constexpr int ALT = RPT == 4 ? 3 : (RPT == 2 ? 4 : 5);
        if ((variant & 1) == 1) return launch_one<S, RPT, R, RECON, FORM, ALT>(c, a);
    }
    return launch_one<S, RPT, R, RECON, FORM, DEF>(c, a);
}

// rpt = right-hand sides per thread; 0 = default: 2 for groups of 4 (measured best on B200 for fp32 at N = 4, 8, 16:
// 168 registers, 12 warps per SM), else the group width; fp64 caps at 2.
template <class S, int RECON, int FORM>
int launch_dslash(lq_ctx* c, DslashArgs<S> a, int rpt, int variant) {
    constexpr int MAXRPT = (S::prec == LQ_FP64) ? 2 : 4;
    const int R = group_width(a.N);
    if (rpt <= 0) rpt = (R == 4) ? 2 : R;
    if (rpt > MAXRPT) rpt = MAXRPT;
    if (rpt > R) rpt = R;
    if (R % rpt != 0) return set_err(c, LQ_EINVAL, "rhs-per-thread must divide the RHS group width");
    if (R == 4) {
        if constexpr (MAXRPT == 4) { if (rpt == 4) return launch_rpt<S, 4, 4, RECON, FORM>(c, a, variant); }
        if (rpt == 2) return launch_rpt<S, 2, 4, RECON, FORM>(c, a, variant);
        return launch_rpt<S, 1, 4, RECON, FORM>(c, a, variant);
    }
    if (R == 2) {
        if (rpt == 2) return launch_rpt<S, 2, 2, RECON, FORM>(c, a, variant);
        return launch_rpt<S, 1, 2, RECON, FORM>(c, a, variant);
    }
    return launch_rpt<S, 1, 1, RECON, FORM>(c, a, variant);
}

#define INSTANTIATE_DSLASH(S, RECON, FORM) template int launch_dslash<S, RECON, FORM>(lq_ctx*, DslashArgs<S>, int, int);
