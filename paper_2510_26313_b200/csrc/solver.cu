// solver.cu -- batched even-odd CGNR inside an fp64 restart defect correction
// (8(c.1) steps 8, 11; PAPER.md L135-140 batched solves, L116/L164 mixed precision).
//
// Every RHS k has its own alpha_k, beta_k (no block-Krylov coupling, reading #26); the batch shares only the
// operator application.  Per-RHS scalars live on the device; the host polls N numbers every `check_every`
// inner iterations and once per outer cycle.  The inner iteration body can be replayed as a CUDA graph.
#include <math.h>
#include <string.h>
#include "internal.cuh"

struct Workspace {
    int nrhs = 0, prec = -1;
    void *bhat = nullptr, *r = nullptr, *t64 = nullptr, *tmp64 = nullptr;          // fp64, one parity each
    void *e = nullptr, *z = nullptr, *p = nullptr, *t = nullptr, *q = nullptr, *tmp = nullptr, *rt = nullptr, *s = nullptr;  // inner precision
    double* d_scal = nullptr;                                                       // 8 x LQ_MAX_RHS doubles
    double* d_bicg = nullptr;                                                       // 12 x LQ_MAX_RHS doubles (BiCGStab sums)
};

struct WsHolder { lq_ctx* c; Workspace ws; };
static std::vector<WsHolder> g_ws;      // one cached workspace per context

static Workspace* ws_for(lq_ctx* c) {
    for (auto& h : g_ws) if (h.c == c) return &h.ws;
    g_ws.push_back(WsHolder{c, Workspace()});
    return &g_ws.back().ws;
}
void solver_forget(lq_ctx* c) {
    for (size_t i = 0; i < g_ws.size(); i++) if (g_ws[i].c == c) { g_ws.erase(g_ws.begin() + i); return; }
}
static void ws_release(lq_ctx* c, Workspace* w) {
    void** all[] = {&w->bhat, &w->r, &w->t64, &w->tmp64, &w->e, &w->z, &w->p, &w->t, &w->q, &w->tmp, &w->rt, &w->s, (void**)&w->d_scal, (void**)&w->d_bicg};
    for (void** p : all) if (*p) { dev_free(c, *p); *p = nullptr; }
    w->nrhs = 0; w->prec = -1;
}
static int ws_prepare(lq_ctx* c, Workspace* w, int nrhs, int prec) {
    if (w->nrhs == nrhs && w->prec == prec) return 0;
    ws_release(c, w);
    const size_t b64 = parity_bytes(c->g, nrhs, LQ_FP64), bin = parity_bytes(c->g, nrhs, prec);
    void** p64[] = {&w->bhat, &w->r, &w->t64, &w->tmp64};
    for (void** p : p64) { *p = dev_alloc(c, b64); if (!*p) return LQ_ENOMEM; }
    void** pin[] = {&w->e, &w->z, &w->p, &w->t, &w->q, &w->tmp, &w->rt, &w->s};
    for (void** p : pin) { *p = dev_alloc(c, bin); if (!*p) return LQ_ENOMEM; }
    w->d_scal = (double*)dev_alloc(c, 8 * LQ_MAX_RHS * sizeof(double));
    w->d_bicg = (double*)dev_alloc(c, 12 * LQ_MAX_RHS * sizeof(double));
    if (!w->d_scal || !w->d_bicg) return LQ_ENOMEM;
    w->nrhs = nrhs; w->prec = prec;
    return 0;
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

// one inner CG iteration (5 launches); rr/rrn are swapped by the caller.  The two block-BLAS reductions and the residual
// update ride in the kernel-B epilogues: q = Mhat^dag t is never stored.
static int cg_iteration(lq_ctx* c, Workspace* w, int prec, int n, double* rr, double* pAp, double* rrn) {
    const double k2 = -c->kappa * c->kappa;
    LQ_TRY(op_kernel_a(c, prec, n, 1, w->tmp, w->p, 0));
    LQ_TRY(op_kernel_b_epi(c, prec, n, 0, w->t, w->p, w->tmp, k2, 1, 0, EPI_NORM, nullptr, nullptr, pAp));   // t = Mhat p, pAp = ||t||^2
    LQ_TRY(op_kernel_a(c, prec, n, 1, w->tmp, w->t, 1));
    LQ_TRY(op_kernel_b_epi(c, prec, n, 0, w->z, w->t, w->tmp, k2, 1, 1, EPI_XMAY, rr, pAp, rrn));          // z -= alpha Mhat^dag t, rrn = ||z||^2
    return blas_cg_update_ep(c, prec, n, w->e, w->p, w->z, rr, pAp, rrn);                                    // e += alpha p ; p = z + beta p
}
static const int KERNELS_PER_ITER = 5;

int solve_native(lq_ctx* c, void* x_full, const void* b_full, int n, const lq_solve_param* prm, lq_solve_info* info) {
    if (!c->has_gauge || !c->has_clover) return set_err(c, LQ_ESTATE, "gauge field and clover term must be loaded before lq_solve");
    const int prec = prm->inner_prec;
    if (prec != LQ_FP64 && prec != LQ_FP32 && prec != LQ_HALF) return set_err(c, LQ_EINVAL, "bad inner precision");
    if (prm->algorithm != LQ_ALG_CGNR && prm->algorithm != LQ_ALG_BICGSTAB) return set_err(c, LQ_EINVAL, "bad solver algorithm");
    Workspace* w = ws_for(c);
    LQ_TRY(ws_prepare(c, w, n, prec));
    const size_t pb64 = parity_bytes(c->g, n, LQ_FP64);
    const char* b_e = (const char*)b_full; const char* b_o = b_e + pb64;
    char* x_e = (char*)x_full; char* x_o = x_e + pb64;
    double* S = w->d_scal;
    double *d_rr = S, *d_rrn = S + LQ_MAX_RHS, *d_pAp = S + 2 * LQ_MAX_RHS, *d_rn = S + 3 * LQ_MAX_RHS, *d_bn = S + 4 * LQ_MAX_RHS,
           *d_scale = S + 6 * LQ_MAX_RHS, *d_cs = S + 7 * LQ_MAX_RHS;
    const double kappa = c->kappa;
    int check_every = prm->check_every > 0 ? prm->check_every : 10;
    if (prm->use_graph && (check_every & 1)) check_every++;           // graph body must leave rr/rrn un-swapped
    memset(info, 0, sizeof(*info));
    info->nrhs = n;

    cudaEvent_t ev0, ev1;
    LQ_CUDA(c, cudaEventCreate(&ev0)); LQ_CUDA(c, cudaEventCreate(&ev1));
    LQ_CUDA(c, cudaEventRecord(ev0, c->stream));
    const long long launches0 = c->launches;

    // ||b_k|| over both parities
    double bn[2 * LQ_MAX_RHS], bnorm[LQ_MAX_RHS];
    LQ_TRY(blas_norm2(c, LQ_FP64, n, b_e, d_bn));
    LQ_TRY(blas_norm2(c, LQ_FP64, n, b_o, d_bn + LQ_MAX_RHS));
    // a2: bhat_e = b_e + kappa D_eo A_oo^{-1} b_o
    LQ_TRY(op_clover(c, LQ_FP64, n, 1, w->tmp64, b_o, 1));
    LQ_TRY(op_kernel_b(c, LQ_FP64, n, 0, w->bhat, b_e, w->tmp64, kappa, 0, 0));
    LQ_TRY(fetch(c, d_bn, 2 * LQ_MAX_RHS, bn));
    for (int k = 0; k < n; k++) bnorm[k] = sqrt(bn[k] + bn[LQ_MAX_RHS + k]);
    // x_e = 0, r = bhat
    LQ_TRY(spinor_zero_parity(c, x_e, n, LQ_FP64));
    LQ_TRY(blas_copy(c, LQ_FP64, n, w->r, w->bhat));
    LQ_TRY(blas_norm2(c, LQ_FP64, n, w->r, d_rn));

    bool done[LQ_MAX_RHS];
    for (int k = 0; k < n; k++) { done[k] = false; info->iters[k] = 0; }
    int status = LQ_ENOTCONVERGED;
    cudaGraphExec_t gexec = nullptr;
    int total_inner = 0, cycle = 0;
    double prev_rnorm[LQ_MAX_RHS];
    for (int k = 0; k < n; k++) prev_rnorm[k] = 0.0;
    for (;; cycle++) {
        double rn2[LQ_MAX_RHS], rnorm[LQ_MAX_RHS];
        LQ_TRY(fetch(c, d_rn, n, rn2));
        bool all = true;
        for (int k = 0; k < n; k++) {
            rnorm[k] = sqrt(rn2[k]);
            info->true_rel_residual[k] = bnorm[k] > 0 ? rnorm[k] / bnorm[k] : 0.0;
            const bool ok = info->true_rel_residual[k] <= prm->tol;
            if (ok && !done[k]) { done[k] = true; if (info->iters[k] == 0) info->iters[k] = total_inner; }
            if (!ok) { done[k] = false; all = false; }
        }
        if (all) { status = 0; break; }
        if (cycle >= prm->max_outer) break;
        // rt = lowprec(r / ||r_k||): per-RHS scaling keeps fp32 / half in range
        LQ_CUDA(c, cudaMemcpyAsync(d_scale, rnorm, n * sizeof(double), cudaMemcpyHostToDevice, c->stream));
        LQ_TRY(spinor_convert(c, w->rt, prec, w->r, LQ_FP64, n, d_scale, 1));
        int it = 0;
        int met[LQ_MAX_RHS];
        double thresh[LQ_MAX_RHS];
        if (prm->algorithm == LQ_ALG_BICGSTAB) {
            // ---- batched BiCGStab on Mhat e = rt: rhat0 = rt, r = z, v = q; complex per-RHS scalars on the device
            const double k2b = -c->kappa * c->kappa;
            double* rho = w->d_bicg; double* rho_new = rho + 3 * LQ_MAX_RHS; double* c1 = rho + 6 * LQ_MAX_RHS; double* d2 = rho + 9 * LQ_MAX_RHS;
            LQ_TRY(blas_copy(c, prec, n, w->z, w->rt));
            LQ_TRY(blas_copy(c, prec, n, w->p, w->rt));
            LQ_TRY(spinor_zero_parity(c, w->e, n, prec));
            LQ_TRY(blas_cdot3(c, prec, n, w->rt, w->rt, rho));                       // rho = <rhat0, r> = ||rt||^2
            double rr0[LQ_MAX_RHS];
            LQ_TRY(fetch(c, rho + 2 * LQ_MAX_RHS, n, rr0));
            for (int k = 0; k < n; k++) {
                double want = (rnorm[k] > 0) ? 0.25 * prm->tol * bnorm[k] / rnorm[k] : 1.0;   // reduction still needed
                double f = prm->delta > want ? prm->delta : want;
                if (f > 0.5) f = 0.5;
                thresh[k] = f * f * rr0[k];
                met[k] = -1;
            }
            while (it < prm->max_inner) {
                for (int j = 0; j < check_every; j++) {
                    LQ_TRY(op_kernel_a(c, prec, n, 1, w->tmp, w->p, 0));             // v = Mhat p with <rhat0, v> in the epilogue
                    LQ_TRY(op_kernel_b_cdot(c, prec, n, 0, w->q, w->p, w->tmp, k2b, 1, 0, w->rt, 0, c1));
                    LQ_TRY(blas_bicg_s(c, prec, n, w->s, w->z, w->q, rho, c1));      // s = r - alpha v
                    LQ_TRY(op_kernel_a(c, prec, n, 1, w->tmp, w->s, 0));             // t = Mhat s with <t, s> = conj <s, t> and ||t||^2
                    LQ_TRY(op_kernel_b_cdot(c, prec, n, 0, w->t, w->s, w->tmp, k2b, 1, 0, w->s, 1, d2));
                    LQ_TRY(blas_bicg_xr(c, prec, n, w->e, w->z, w->p, w->s, w->t, w->rt, rho, c1, d2, rho_new));   // e, r, rho', ||r||^2
                    LQ_TRY(blas_bicg_p(c, prec, n, w->p, w->z, w->q, rho, rho_new, c1, d2));                      // p
                    double* sw = rho; rho = rho_new; rho_new = sw;
                }
                it += check_every;
                double cur[LQ_MAX_RHS];
                LQ_TRY(fetch(c, rho + 2 * LQ_MAX_RHS, n, cur));
                bool conv = true;
                for (int k = 0; k < n; k++) {
                    if (cur[k] <= thresh[k] || !(cur[k] == cur[k])) { if (met[k] < 0) met[k] = it; }
                    else { met[k] = -1; conv = false; }
                }
                if (conv) break;
            }
            for (int k = 0; k < n; k++) prev_rnorm[k] = 0.0;                         // no CG direction to carry over
        } else {
            // z = Mhat^dag rt ; e = 0 ; p = z (restart) or, with reliable updates, p <- z + c (p - z_old): the old direction
            // survives the residual refresh, rescaled by c_k = ||r_k||_old / ||r_k||_new because the inner system is
            // normalised by ||r_k|| (in exact arithmetic z = c z_old, so the correction only carries the rounding difference)
            if (prm->keep_direction && cycle > 0) {
                double cs[LQ_MAX_RHS];
                for (int k = 0; k < n; k++) cs[k] = (rnorm[k] > 0 && prev_rnorm[k] > 0) ? prev_rnorm[k] / rnorm[k] : 0.0;
                LQ_CUDA(c, cudaMemcpyAsync(d_cs, cs, n * sizeof(double), cudaMemcpyHostToDevice, c->stream));
                LQ_TRY(apply_mhat(c, prec, n, w->q, w->rt, w->tmp, 1));
                LQ_TRY(blas_keep_direction(c, prec, n, w->p, w->z, w->q, d_cs));
                void* sw = w->z; w->z = w->q; w->q = sw;
            } else {
                LQ_TRY(apply_mhat(c, prec, n, w->z, w->rt, w->tmp, 1));
                LQ_TRY(blas_copy(c, prec, n, w->p, w->z));
            }
            for (int k = 0; k < n; k++) prev_rnorm[k] = rnorm[k];
            LQ_TRY(spinor_zero_parity(c, w->e, n, prec));
            LQ_TRY(blas_norm2(c, prec, n, w->z, d_rr));
            double rr0[LQ_MAX_RHS];
            LQ_TRY(fetch(c, d_rr, n, rr0));
            for (int k = 0; k < n; k++) {
                double want = (rnorm[k] > 0) ? 0.25 * prm->tol * bnorm[k] / rnorm[k] : 1.0;   // reduction still needed
                double f = prm->delta > want ? prm->delta : want;
                if (f > 0.5) f = 0.5;
                thresh[k] = f * f * rr0[k];
                met[k] = -1;
            }
            double *rr = d_rr, *rrn = d_rrn;
            it = 0;
            bool graph_ready = false;
            while (it < prm->max_inner) {
                if (prm->use_graph && it >= check_every) {
                    if (!graph_ready) {
                        if (gexec) { cudaGraphExecDestroy(gexec); gexec = nullptr; }
                        cudaGraph_t graph;
                        LQ_CUDA(c, cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
                        const long long l0 = c->launches;
                        int rc = 0;
                        for (int j = 0; j < check_every && rc == 0; j++) { rc = cg_iteration(c, w, prec, n, rr, d_pAp, rrn); double* s = rr; rr = rrn; rrn = s; }
                        c->launches = l0;
                        cudaError_t ce = cudaStreamEndCapture(c->stream, &graph);   // always close the capture, even on failure
                        if (rc) { if (ce == cudaSuccess && graph) cudaGraphDestroy(graph); cudaGetLastError(); return rc; }
                        LQ_CUDA(c, ce);
                        LQ_CUDA(c, cudaGraphInstantiate(&gexec, graph, 0));
                        cudaGraphDestroy(graph);
                        graph_ready = true;
                    }
                    LQ_CUDA(c, cudaGraphLaunch(gexec, c->stream));
                    c->launches += (long long)KERNELS_PER_ITER * check_every;
                } else {
                    for (int j = 0; j < check_every; j++) { LQ_TRY(cg_iteration(c, w, prec, n, rr, d_pAp, rrn)); double* s = rr; rr = rrn; rrn = s; }
                }
                it += check_every;
                double cur[LQ_MAX_RHS];
                LQ_TRY(fetch(c, rr, n, cur));
                bool conv = true;
                for (int k = 0; k < n; k++) {
                    if (cur[k] <= thresh[k] || !(cur[k] == cur[k])) { if (met[k] < 0) met[k] = it; }
                    else { met[k] = -1; conv = false; }
                }
                if (conv) break;
            }
        }
        total_inner += it;
        for (int k = 0; k < n; k++) if (!done[k]) info->iters[k] = total_inner - it + (met[k] > 0 ? met[k] : it);
        // x += ||r|| e ; r = bhat - Mhat x
        LQ_TRY(blas_axpy_mixed(c, prec, n, x_e, w->e, d_scale));
        LQ_TRY(apply_mhat(c, LQ_FP64, n, w->t64, x_e, w->tmp64, 0));
        LQ_TRY(blas_residual(c, n, w->r, w->bhat, w->t64, d_rn));
        for (int k = 0; k < n; k++) done[k] = false;   // re-decided from the fresh true residual
        // iters[k] stays as the estimate of when k was done; overwritten while k is not converged
    }
    if (gexec) cudaGraphExecDestroy(gexec);
    info->outer_cycles = cycle;
    info->inner_iters = total_inner;
    // a10: x_o = A_oo^{-1} (b_o + kappa D_oe x_e)
    LQ_TRY(op_kernel_b(c, LQ_FP64, n, 1, w->tmp64, b_o, x_e, kappa, 0, 0));
    LQ_TRY(op_clover(c, LQ_FP64, n, 1, x_o, w->tmp64, 1));
    LQ_CUDA(c, cudaEventRecord(ev1, c->stream));
    LQ_CUDA(c, cudaEventSynchronize(ev1));
    float ms = 0;
    LQ_CUDA(c, cudaEventElapsedTime(&ms, ev0, ev1));
    cudaEventDestroy(ev0); cudaEventDestroy(ev1);
    info->seconds = ms * 1e-3;
    info->dslash_applies = (double)(4LL * total_inner + 2LL * cycle + 2LL * cycle + 2);
    (void)launches0;
    if (status != 0) return set_err(c, LQ_ENOTCONVERGED, "lq_solve: tolerance not reached within the iteration caps");
    return 0;
}
