// solver.cu -- batched even-odd CGNR / BiCGStab inside an fp64 defect correction
// (8(c.1) steps 8, 11; PAPER.md L135-140 batched solves, L116/L164 mixed precision).
//
// Every RHS k has its own Krylov scalars (no block-Krylov coupling, reading #26); the batch shares only the operator
// application.  All per-RHS scalars live on the device.  The body of `check_every` inner iterations plus a one-warp
// convergence test is ONE CUDA graph, captured once per (precision, batch, tuning) and cached in the context.  The test
// raises a device flag that turns every kernel of the body into a no-op, so the host may queue the next graph before it
// knows the outcome of the previous one: it reads the flag (mirrored into pinned host memory) one graph behind and the
// GPU never waits for the host inside a cycle.  Host synchronisations per defect-correction cycle: one (the fp64 residual
// norms that decide whether another cycle is needed).
#include <math.h>
#include <string.h>
#include "internal.cuh"

// control block of one inner solve (device; `done` and `iters` are mirrored to pinned host memory)
struct InnerCtl {
    int done;                    // 1: every RHS is below its threshold (or produced a NaN): the queued body is skipped
    int iters;                   // inner iterations executed in this cycle
    int pad[2];
    int met[LQ_MAX_RHS];         // iteration at which RHS k went (and stayed) below its threshold, -1: not yet
    double thresh[LQ_MAX_RHS];   // threshold on the recursive residual norm^2 of RHS k
};

struct GraphKey {
    int prec, n, check_every, alg, recon, rpt, variant, pfd, zc, t_bc;
    double kappa;
    const void *partials, *gauge, *clov, *clovinv;
    unsigned gen;                // workspace generation (buffers reallocated -> new graph)
    bool operator==(const GraphKey& o) const {
        return prec == o.prec && n == o.n && check_every == o.check_every && alg == o.alg && recon == o.recon && rpt == o.rpt && variant == o.variant &&
               pfd == o.pfd && zc == o.zc && t_bc == o.t_bc && kappa == o.kappa && partials == o.partials && gauge == o.gauge && clov == o.clov &&
               clovinv == o.clovinv && gen == o.gen;
    }
};

struct SolverWorkspace {
    int nrhs = 0, prec = -1;
    unsigned gen = 0;
    void *bhat = nullptr, *r = nullptr, *t64 = nullptr, *tmp64 = nullptr;          // fp64, one parity each
    void *e = nullptr, *z = nullptr, *p = nullptr, *t = nullptr, *q = nullptr, *tmp = nullptr, *rt = nullptr, *s = nullptr;  // inner precision
    double* d_scal = nullptr;    // 10 x LQ_MAX_RHS doubles
    double* d_bicg = nullptr;    // 12 x LQ_MAX_RHS doubles (BiCGStab sums)
    InnerCtl* d_ctl = nullptr;
    InnerCtl* h_ctl = nullptr;   // pinned host mirror
    cudaEvent_t ev[2] = {nullptr, nullptr}, t0 = nullptr, t1 = nullptr;
    cudaGraphExec_t gexec = nullptr;
    GraphKey key;
    bool body_ran = false;       // the body has run un-captured with these buffers (every lazy allocation has happened)
    double iter_bytes = 0, iter_flops = 0;   // modelled work of one inner iteration
    int iter_launches = 0;
};

static void ws_release(lq_ctx* c, SolverWorkspace* w) {
    void** all[] = {&w->bhat, &w->r, &w->t64, &w->tmp64, &w->e, &w->z, &w->p, &w->t, &w->q, &w->tmp, &w->rt, &w->s,
                    (void**)&w->d_scal, (void**)&w->d_bicg, (void**)&w->d_ctl};
    for (void** p : all) if (*p) { dev_free(c, *p); *p = nullptr; }
    if (w->gexec) { cudaGraphExecDestroy(w->gexec); w->gexec = nullptr; }
    w->nrhs = 0; w->prec = -1; w->body_ran = false;
}
// called by lq_destroy (before the context's allocations are returned)
void solver_release(lq_ctx* c) {
    SolverWorkspace* w = c->ws;
    if (!w) return;
    ws_release(c, w);
    for (cudaEvent_t* e : {&w->ev[0], &w->ev[1], &w->t0, &w->t1}) if (*e) cudaEventDestroy(*e);
    if (w->h_ctl) cudaFreeHost(w->h_ctl);
    delete w;
    c->ws = nullptr;
}
static int ws_prepare(lq_ctx* c, int nrhs, int prec) {
    if (!c->ws) {
        c->ws = new SolverWorkspace();
        SolverWorkspace* w = c->ws;
        for (cudaEvent_t* e : {&w->ev[0], &w->ev[1]}) LQ_CUDA(c, cudaEventCreateWithFlags(e, cudaEventDisableTiming));
        LQ_CUDA(c, cudaEventCreate(&w->t0)); LQ_CUDA(c, cudaEventCreate(&w->t1));
        LQ_CUDA(c, cudaMallocHost((void**)&w->h_ctl, sizeof(InnerCtl)));
        memset(w->h_ctl, 0, sizeof(InnerCtl));
    }
    SolverWorkspace* w = c->ws;
    if (w->nrhs == nrhs && w->prec == prec) return 0;
    ws_release(c, w);
    w->gen++;
    const size_t b64 = parity_bytes(c->g, nrhs, LQ_FP64), bin = parity_bytes(c->g, nrhs, prec);
    void** p64[] = {&w->bhat, &w->r, &w->t64, &w->tmp64};
    for (void** p : p64) { *p = dev_alloc(c, b64); if (!*p) { ws_release(c, w); return LQ_ENOMEM; } }
    void** pin[] = {&w->e, &w->z, &w->p, &w->t, &w->q, &w->tmp, &w->rt, &w->s};
    for (void** p : pin) { *p = dev_alloc(c, bin); if (!*p) { ws_release(c, w); return LQ_ENOMEM; } }
    w->d_scal = (double*)dev_alloc(c, 10 * LQ_MAX_RHS * sizeof(double));
    w->d_bicg = (double*)dev_alloc(c, 12 * LQ_MAX_RHS * sizeof(double));
    w->d_ctl = (InnerCtl*)dev_alloc(c, sizeof(InnerCtl));
    if (!w->d_scal || !w->d_bicg || !w->d_ctl) { ws_release(c, w); return LQ_ENOMEM; }
    w->nrhs = nrhs; w->prec = prec;
    return 0;
}

// ---- device-side control of the inner solve (one warp each) ---------------------------------------------------------
// thresh_k = (fac_k)^2 * cur_k: the reduction of the recursive residual asked of this cycle
__global__ void inner_begin_kernel(InnerCtl* ctl, volatile int* h_done, int n, const double* __restrict__ cur, const double* __restrict__ fac) {
    const int k = threadIdx.x;
    if (k == 0) { ctl->done = 0; ctl->iters = 0; h_done[0] = 0; h_done[1] = 0; }
    if (k < LQ_MAX_RHS) { ctl->thresh[k] = k < n ? fac[k] * fac[k] * cur[k] : 0.0; ctl->met[k] = -1; }
}
// after `step` more iterations: which RHS are below their threshold; all of them -> raise the flag
__global__ void inner_check_kernel(InnerCtl* ctl, volatile int* h_done, int n, const double* __restrict__ cur, int step) {
    if (ctl->done) return;
    const int k = threadIdx.x;
    const int it = ctl->iters + step;
    bool ok = true;
    if (k < n) {
        const double v = cur[k];
        ok = (v <= ctl->thresh[k]) || !(v == v);
        if (ok) { if (ctl->met[k] < 0) ctl->met[k] = it; } else ctl->met[k] = -1;
    }
    const bool all = __all_sync(0xffffffffu, ok);
    __syncwarp();
    if (k == 0) {
        ctl->iters = it; h_done[1] = it;
        if (all) { ctl->done = 1; __threadfence_system(); h_done[0] = 1; }
    }
}

// out_e = Mhat in_e  (2 stencil kernels: A then B); dagger -> Mhat^dag
static int apply_mhat(lq_ctx* c, int prec, int n, void* out_e, const void* in_e, void* tmp_o, int dagger) {
    LQ_TRY(op_kernel_a(c, prec, n, 1, tmp_o, in_e, dagger));
    return op_kernel_b(c, prec, n, 0, out_e, in_e, tmp_o, -c->kappa * c->kappa, 1, dagger);
}
int mhat_native(lq_ctx* c, int prec, int n, void* out_e, const void* in_e, int dagger) {
    void* tmp = dev_alloc(c, parity_bytes(c->g, n, prec));
    if (!tmp) return LQ_ENOMEM;
    int rc = apply_mhat(c, prec, n, out_e, in_e, tmp, dagger);
    if (rc == 0 && cudaStreamSynchronize(c->stream) != cudaSuccess) rc = set_err(c, LQ_ECUDA, "sync failed");
    dev_free(c, tmp);
    return rc;
}

static int fetch(lq_ctx* c, const double* d, int n, double* h) {
    LQ_CUDA(c, cudaMemcpyAsync(c->h_scalars, d, n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    LQ_CUDA(c, cudaStreamSynchronize(c->stream));
    memcpy(h, c->h_scalars, n * sizeof(double));
    return 0;
}

// pointers of the device scalars (per RHS, LQ_MAX_RHS apart)
struct Scal {
    double *rr, *rrn, *pAp, *rn, *bn_e, *bn_o, *scale, *cs, *fac;
    double *rho, *rho_new, *c1, *d2;    // BiCGStab: 3 x LQ_MAX_RHS each
};

// one inner CG iteration (5 launches).  The two block-BLAS reductions and the residual update ride in the kernel-B epilogues
// (SURVEY 8(a) rows a4/a6): q = Mhat^dag t is never stored.  rr / rrn alternate; an even number of iterations restores them.
static int cg_iteration(lq_ctx* c, SolverWorkspace* w, int prec, int n, double* rr, double* pAp, double* rrn) {
    const double k2 = -c->kappa * c->kappa;
    LQ_TRY(op_kernel_a(c, prec, n, 1, w->tmp, w->p, 0));
    LQ_TRY(op_kernel_b_epi(c, prec, n, 0, w->t, w->p, w->tmp, k2, 1, 0, EPI_NORM, nullptr, nullptr, pAp));   // t = Mhat p, pAp = ||t||^2
    LQ_TRY(op_kernel_a(c, prec, n, 1, w->tmp, w->t, 1));
    LQ_TRY(op_kernel_b_epi(c, prec, n, 0, w->z, w->t, w->tmp, k2, 1, 1, EPI_XMAY, rr, pAp, rrn));          // z -= alpha Mhat^dag t, rrn = ||z||^2
    return blas_cg_update_ep(c, prec, n, w->e, w->p, w->z, rr, pAp, rrn);                                    // e += alpha p ; p = z + beta p
}
// one batched BiCGStab iteration on Mhat e = rt (7 launches): rhat0 = rt, r = z, v = q
static int bicg_iteration(lq_ctx* c, SolverWorkspace* w, int prec, int n, double* rho, double* rho_new, double* c1, double* d2) {
    const double k2 = -c->kappa * c->kappa;
    LQ_TRY(op_kernel_a(c, prec, n, 1, w->tmp, w->p, 0));                              // v = Mhat p with <rhat0, v> in the epilogue
    LQ_TRY(op_kernel_b_cdot(c, prec, n, 0, w->q, w->p, w->tmp, k2, 1, 0, w->rt, 0, c1));
    LQ_TRY(blas_bicg_s(c, prec, n, w->s, w->z, w->q, rho, c1));                       // s = r - alpha v
    LQ_TRY(op_kernel_a(c, prec, n, 1, w->tmp, w->s, 0));                              // t = Mhat s with <t, s> = conj <s, t> and ||t||^2
    LQ_TRY(op_kernel_b_cdot(c, prec, n, 0, w->t, w->s, w->tmp, k2, 1, 0, w->s, 1, d2));
    LQ_TRY(blas_bicg_xr(c, prec, n, w->e, w->z, w->p, w->s, w->t, w->rt, rho, c1, d2, rho_new));   // e, r, rho', ||r||^2
    return blas_bicg_p(c, prec, n, w->p, w->z, w->q, rho, rho_new, c1, d2);            // p
}

// `check_every` (even) iterations followed by the convergence test, enqueued on the context's stream
static int enqueue_block(lq_ctx* c, SolverWorkspace* w, int alg, int prec, int n, int check_every, const Scal& S) {
    c->loop_skip = &w->d_ctl->done;
    int rc = 0;
    if (alg == LQ_ALG_BICGSTAB) {
        double *rho = S.rho, *rho_new = S.rho_new;
        for (int j = 0; j < check_every && rc == 0; j++) { rc = bicg_iteration(c, w, prec, n, rho, rho_new, S.c1, S.d2); double* sw = rho; rho = rho_new; rho_new = sw; }
    } else {
        double *rr = S.rr, *rrn = S.rrn;
        for (int j = 0; j < check_every && rc == 0; j++) { rc = cg_iteration(c, w, prec, n, rr, S.pAp, rrn); double* sw = rr; rr = rrn; rrn = sw; }
    }
    c->loop_skip = nullptr;
    if (rc) return rc;
    const double* cur = alg == LQ_ALG_BICGSTAB ? S.rho + 2 * LQ_MAX_RHS : S.rr;
    inner_check_kernel<<<1, 32, 0, c->stream>>>(w->d_ctl, (volatile int*)&w->h_ctl->done, n, cur, check_every);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}

static GraphKey make_key(lq_ctx* c, SolverWorkspace* w, int alg, int prec, int n, int check_every) {
    GraphKey k;
    k.prec = prec; k.n = n; k.check_every = check_every; k.alg = alg; k.recon = c->recon32; k.rpt = c->dslash_rpt; k.variant = c->dslash_variant;
    k.pfd = c->dslash_pfd; k.zc = c->dslash_zc; k.t_bc = c->t_bc; k.kappa = c->kappa; k.partials = c->red_partials;
    k.gauge = prec == LQ_FP64 ? (const void*)c->gauge64 : ((prec == LQ_HALF && c->half_links) ? (const void*)c->gauge16 : (const void*)c->gauge32);
    k.clov = prec == LQ_FP64 ? (const void*)c->clov64 : (const void*)c->clov32;
    k.clovinv = prec == LQ_FP64 ? (const void*)c->clovinv64 : (const void*)c->clovinv32;
    k.gen = w->gen;
    return k;
}

// capture the block into a graph (only after the block has run un-captured once: no allocation may happen in a capture)
static int build_graph(lq_ctx* c, SolverWorkspace* w, int alg, int prec, int n, int check_every, const Scal& S) {
    if (w->gexec) { cudaGraphExecDestroy(w->gexec); w->gexec = nullptr; }
    if (c->stream == nullptr || c->stream == cudaStreamLegacy) return 1;          // the legacy default stream cannot be captured
    if (cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); return 1; }
    const long long l0 = c->launches;
    const double mb = c->model_bytes, mf = c->model_flops;
    const int rc = enqueue_block(c, w, alg, prec, n, check_every, S);
    c->launches = l0; c->model_bytes = mb; c->model_flops = mf;
    cudaGraph_t graph = nullptr;
    const cudaError_t ce = cudaStreamEndCapture(c->stream, &graph);              // always close the capture, even on failure
    if (rc != 0 || ce != cudaSuccess || !graph) { if (graph) cudaGraphDestroy(graph); cudaGetLastError(); return rc ? rc : 1; }
    const cudaError_t ci = cudaGraphInstantiate(&w->gexec, graph, 0);
    cudaGraphDestroy(graph);
    if (ci != cudaSuccess) { w->gexec = nullptr; cudaGetLastError(); return 1; }
    w->key = make_key(c, w, alg, prec, n, check_every);
    return 0;
}

int solve_native(lq_ctx* c, void* x_full, const void* b_full, int n, const lq_solve_param* prm, lq_solve_info* info) {
    if (!c->has_gauge || !c->has_clover) return set_err(c, LQ_ESTATE, "gauge field and clover term must be loaded before lq_solve");
    const int prec = prm->inner_prec, alg = prm->algorithm;
    if (prec != LQ_FP64 && prec != LQ_FP32 && prec != LQ_HALF) return set_err(c, LQ_EINVAL, "bad inner precision");
    if (alg != LQ_ALG_CGNR && alg != LQ_ALG_BICGSTAB) return set_err(c, LQ_EINVAL, "bad solver algorithm");
    LQ_TRY(ws_prepare(c, n, prec));
    SolverWorkspace* w = c->ws;
    const size_t pb64 = parity_bytes(c->g, n, LQ_FP64);
    const char* b_e = (const char*)b_full; const char* b_o = b_e + pb64;
    char* x_e = (char*)x_full; char* x_o = x_e + pb64;
    Scal S;
    {
        double* q = w->d_scal;
        S.rr = q; S.rrn = q + LQ_MAX_RHS; S.pAp = q + 2 * LQ_MAX_RHS; S.rn = q + 3 * LQ_MAX_RHS; S.bn_e = q + 4 * LQ_MAX_RHS; S.bn_o = q + 5 * LQ_MAX_RHS;
        S.scale = q + 6 * LQ_MAX_RHS; S.cs = q + 7 * LQ_MAX_RHS; S.fac = q + 8 * LQ_MAX_RHS;
        S.rho = w->d_bicg; S.rho_new = S.rho + 3 * LQ_MAX_RHS; S.c1 = S.rho + 6 * LQ_MAX_RHS; S.d2 = S.rho + 9 * LQ_MAX_RHS;
    }
    const double kappa = c->kappa;
    int check_every = prm->check_every > 0 ? prm->check_every : 10;
    if (check_every & 1) check_every++;                       // a block must leave the alternating scalar buffers un-swapped
    memset(info, 0, sizeof(*info));
    info->nrhs = n;
    const double mb0 = c->model_bytes, mf0 = c->model_flops;

    LQ_CUDA(c, cudaEventRecord(w->t0, c->stream));
    // ||b_k|| over both parities
    LQ_TRY(blas_norm2(c, LQ_FP64, n, b_e, S.bn_e));
    LQ_TRY(blas_norm2(c, LQ_FP64, n, b_o, S.bn_o));
    // a2: bhat_e = b_e + kappa D_eo A_oo^{-1} b_o
    LQ_TRY(op_clover(c, LQ_FP64, n, 1, w->tmp64, b_o, 1));
    LQ_TRY(op_kernel_b(c, LQ_FP64, n, 0, w->bhat, b_e, w->tmp64, kappa, 0, 0));
    if (prm->use_x0) {
        // r = bhat - Mhat x_e for the caller's initial guess (only the even sites of x matter: x_o is reconstructed)
        LQ_TRY(apply_mhat(c, LQ_FP64, n, w->t64, x_e, w->tmp64, 0));
        LQ_TRY(blas_residual(c, n, w->r, w->bhat, w->t64, S.rn));
    } else {
        LQ_TRY(spinor_zero_parity(c, x_e, n, LQ_FP64));
        LQ_TRY(blas_copy(c, LQ_FP64, n, w->r, w->bhat));
        LQ_TRY(blas_norm2(c, LQ_FP64, n, w->r, S.rn));
    }

    bool done[LQ_MAX_RHS];
    double bnorm[LQ_MAX_RHS], prev_rnorm[LQ_MAX_RHS];
    for (int k = 0; k < n; k++) { done[k] = false; info->iters[k] = 0; prev_rnorm[k] = 0.0; bnorm[k] = 0.0; }
    int status = LQ_ENOTCONVERGED;
    int total_inner = 0, cycle = 0, last_it = 0;
    bool have_inner = false;                                   // an inner solve has been queued whose counters are still on the device
    double loop_bytes = 0, loop_flops = 0;
    for (;; cycle++) {
        // the one host synchronisation of the cycle: fp64 residual norms (+ ||b|| the first time, + the counters of the inner solve)
        double hs[3 * LQ_MAX_RHS], rnorm[LQ_MAX_RHS];
        if (have_inner) LQ_CUDA(c, cudaMemcpyAsync(w->h_ctl, w->d_ctl, sizeof(InnerCtl), cudaMemcpyDeviceToHost, c->stream));
        LQ_TRY(fetch(c, S.rn, 3 * LQ_MAX_RHS, hs));
        if (cycle == 0) for (int k = 0; k < n; k++) bnorm[k] = sqrt(hs[LQ_MAX_RHS + k] + hs[2 * LQ_MAX_RHS + k]);
        if (have_inner) {
            last_it = w->h_ctl->iters;
            total_inner += last_it;
            for (int k = 0; k < n; k++) if (!done[k]) info->iters[k] = total_inner - last_it + (w->h_ctl->met[k] > 0 ? w->h_ctl->met[k] : last_it);
            loop_bytes += last_it * w->iter_bytes; loop_flops += last_it * w->iter_flops;
            have_inner = false;
        }
        bool all = true;
        for (int k = 0; k < n; k++) {
            rnorm[k] = sqrt(hs[k]);
            info->true_rel_residual[k] = bnorm[k] > 0 ? rnorm[k] / bnorm[k] : 0.0;
            const bool ok = info->true_rel_residual[k] <= prm->tol;      // a NaN compares false
            if (ok && !done[k]) { done[k] = true; if (info->iters[k] == 0) info->iters[k] = total_inner; }
            if (!ok) { done[k] = false; all = false; }
        }
        if (all) { status = 0; break; }
        if (cycle >= prm->max_outer) break;
        // per-RHS scale ||r_k||, direction-carrying factor c_k and the inner reduction factor f_k, one upload
        {
            double up[3 * LQ_MAX_RHS];
            memset(up, 0, sizeof(up));
            for (int k = 0; k < n; k++) {
                up[k] = rnorm[k];
                up[LQ_MAX_RHS + k] = (rnorm[k] > 0 && prev_rnorm[k] > 0) ? prev_rnorm[k] / rnorm[k] : 0.0;
                const double want = (rnorm[k] > 0) ? 0.25 * prm->tol * bnorm[k] / rnorm[k] : 1.0;   // reduction still needed
                double f = prm->delta > want ? prm->delta : want;
                if (f > 0.5) f = 0.5;
                up[2 * LQ_MAX_RHS + k] = f;
            }
            memcpy(c->h_scalars, up, sizeof(up));            // pinned; the previous fetch has been consumed
            LQ_CUDA(c, cudaMemcpyAsync(S.scale, c->h_scalars, sizeof(up), cudaMemcpyHostToDevice, c->stream));
        }
        // rt = lowprec(r / ||r_k||): per-RHS scaling keeps fp32 / half in range
        LQ_TRY(spinor_convert(c, w->rt, prec, w->r, LQ_FP64, n, S.scale, 1));
        const double* cur;
        if (alg == LQ_ALG_BICGSTAB) {
            LQ_TRY(blas_copy(c, prec, n, w->z, w->rt));
            LQ_TRY(blas_copy(c, prec, n, w->p, w->rt));
            LQ_TRY(spinor_zero_parity(c, w->e, n, prec));
            LQ_TRY(blas_cdot3(c, prec, n, w->rt, w->rt, S.rho));                     // rho = <rhat0, r> = ||rt||^2
            cur = S.rho + 2 * LQ_MAX_RHS;
            for (int k = 0; k < n; k++) prev_rnorm[k] = 0.0;                         // no CG direction to carry over
        } else {
            // z = Mhat^dag rt ; e = 0 ; p = z (restart) or, with reliable updates, p <- z + c (p - z_old): the old direction
            // survives the residual refresh, rescaled by c_k = ||r_k||_old / ||r_k||_new because the inner system is
            // normalised by ||r_k|| (in exact arithmetic z = c z_old, so the correction only carries the rounding difference)
            if (prm->keep_direction && cycle > 0) {
                LQ_TRY(apply_mhat(c, prec, n, w->q, w->rt, w->tmp, 1));
                LQ_TRY(blas_keep_direction(c, prec, n, w->p, w->z, w->q, S.cs));    // also z <- q
            } else {
                LQ_TRY(apply_mhat(c, prec, n, w->z, w->rt, w->tmp, 1));
                LQ_TRY(blas_copy(c, prec, n, w->p, w->z));
            }
            for (int k = 0; k < n; k++) prev_rnorm[k] = rnorm[k];
            LQ_TRY(spinor_zero_parity(c, w->e, n, prec));
            LQ_TRY(blas_norm2(c, prec, n, w->z, S.rr));
            cur = S.rr;
        }
        inner_begin_kernel<<<1, 32, 0, c->stream>>>(w->d_ctl, (volatile int*)&w->h_ctl->done, n, cur, S.fac);
        LQ_LAUNCHED(c);
        LQ_CUDA(c, cudaGetLastError());

        // ---- inner loop: blocks of check_every iterations; the host runs one block ahead of the flag it reads
        const double mb1 = c->model_bytes, mf1 = c->model_flops;
        int blocks = 0;
        for (int it = 0; it < prm->max_inner; it += check_every, blocks++) {
            bool graphed = false;
            if (prm->use_graph && w->body_ran) {
                const GraphKey key = make_key(c, w, alg, prec, n, check_every);
                if (!w->gexec || !(key == w->key)) {
                    const int rc = build_graph(c, w, alg, prec, n, check_every, S);
                    if (rc < 0) return rc;                     // rc == 1: capture unavailable, run un-captured
                }
                if (w->gexec) {
                    LQ_CUDA(c, cudaGraphLaunch(w->gexec, c->stream));
                    c->launches += (long long)w->iter_launches * check_every + 1;
                    graphed = true;
                }
            }
            if (!graphed) {
                const long long l0 = c->launches;
                const double b0 = c->model_bytes, f0 = c->model_flops;
                LQ_TRY(enqueue_block(c, w, alg, prec, n, check_every, S));
                w->iter_launches = (int)((c->launches - l0 - 1) / check_every);
                w->iter_bytes = (c->model_bytes - b0) / check_every; w->iter_flops = (c->model_flops - f0) / check_every;
                w->body_ran = true;
            }
            LQ_CUDA(c, cudaEventRecord(w->ev[blocks & 1], c->stream));
            if (blocks >= 1) {
                LQ_CUDA(c, cudaEventSynchronize(w->ev[(blocks - 1) & 1]));
                if (*(volatile int*)&w->h_ctl->done) break;
            }
        }
        c->model_bytes = mb1; c->model_flops = mf1;            // the loop's work is added from the executed iteration count
        have_inner = true;
        // x += ||r|| e ; r = bhat - Mhat x
        LQ_TRY(blas_axpy_mixed(c, prec, n, x_e, w->e, S.scale));
        LQ_TRY(apply_mhat(c, LQ_FP64, n, w->t64, x_e, w->tmp64, 0));
        LQ_TRY(blas_residual(c, n, w->r, w->bhat, w->t64, S.rn));
        for (int k = 0; k < n; k++) done[k] = false;           // re-decided from the fresh true residual
    }
    info->outer_cycles = cycle;
    info->inner_iters = total_inner;
    // a10: x_o = A_oo^{-1} (b_o + kappa D_oe x_e)
    LQ_TRY(op_kernel_b(c, LQ_FP64, n, 1, w->tmp64, b_o, x_e, kappa, 0, 0));
    LQ_TRY(op_clover(c, LQ_FP64, n, 1, x_o, w->tmp64, 1));
    LQ_CUDA(c, cudaEventRecord(w->t1, c->stream));
    LQ_CUDA(c, cudaEventSynchronize(w->t1));
    float ms = 0;
    LQ_CUDA(c, cudaEventElapsedTime(&ms, w->t0, w->t1));
    info->seconds = ms * 1e-3;
    info->dslash_applies = (double)(4LL * total_inner + 2LL * cycle + (alg == LQ_ALG_BICGSTAB ? 0LL : 2LL * cycle) + 2 + (prm->use_x0 ? 2 : 0));
    c->model_bytes += loop_bytes; c->model_flops += loop_flops;
    info->model_bytes = c->model_bytes - mb0; info->model_flops = c->model_flops - mf0;
    if (status != 0) return set_err(c, LQ_ENOTCONVERGED, "lq_solve: tolerance not reached within the iteration caps");
    return 0;
}
