// dslash_launch.cuh -- launcher body; each dslash_*.cu instantiates it for one storage type.
#pragma once
#include "dslash_kernel.cuh"

template <class S, int RPT, int RECON, int FORM>
static int launch_one(lq_ctx* c, DslashArgs<S> a, int block) {
    a.G = a.N / RPT;
    const long long threads = (long long)a.g.Vh * a.G;
    const int grid = (int)((threads + block - 1) / block);
    dslash_kernel<S, RPT, RECON, FORM><<<grid, block, 0, c->stream>>>(a);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}

template <class S, int RECON, int FORM>
int launch_dslash(lq_ctx* c, DslashArgs<S> a, int rpt_override) {
    constexpr int MAXRPT = (S::prec == LQ_FP64) ? 2 : 4;
    int rpt = rpt_override > 0 ? rpt_override : ((a.N % 4 == 0) ? 4 : ((a.N % 2 == 0) ? 2 : 1));
    if (rpt > MAXRPT) rpt = MAXRPT;
    if (a.N % rpt != 0) return set_err(c, LQ_EINVAL, "nrhs not divisible by rhs-per-thread");
    const int block = c->dslash_block > 0 ? c->dslash_block : 128;
    if (rpt == 1) return launch_one<S, 1, RECON, FORM>(c, a, block);
    if (rpt == 2) return launch_one<S, 2, RECON, FORM>(c, a, block);
    if constexpr (MAXRPT == 4) { if (rpt == 4) return launch_one<S, 4, RECON, FORM>(c, a, block); }
    return set_err(c, LQ_EINVAL, "bad rhs-per-thread");
}

#define INSTANTIATE_DSLASH(S, RECON)                                                   \
    template int launch_dslash<S, RECON, FORM_HOP>(lq_ctx*, DslashArgs<S>, int);       \
    template int launch_dslash<S, RECON, FORM_A>(lq_ctx*, DslashArgs<S>, int);         \
    template int launch_dslash<S, RECON, FORM_B>(lq_ctx*, DslashArgs<S>, int);
