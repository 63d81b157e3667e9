// multigrid.cu -- host side of the two-level adaptive multigrid (include/lqcd_b200.h "two-level adaptive multigrid";
// SURVEY.md 8(f) #4).  Kernels: mg_kernels.cuh.  The fine operator is the library's own stencil
// (two kernel-B launches per application of M, ops.cu); everything here is batched over the N right-hand sides of the call.
#include <string.h>
#include <math.h>
#include <functional>
#include "internal.cuh"
#include "mg_kernels.cuh"

using mg::MgGeom;

constexpr int MG_MAX_RESTART = 16;

struct MgState {
    MgGeom m;
    lq_mg_param prm;
    bool ready;
    int* site_f; int* nbr; int* status;
    float2* P; float2* Ac;
    double* d_s;             // device scalars: slots of 3 * LQ_MAX_RHS doubles
    int probes;
    // workspace for `wn` right-hand sides
    int wn;
    float *res, *t;                       // smoother residual, M * (...)
    float *d, *rho;                       // even-odd smoother: correction, Schur residual (even half) / scratch (odd half)
    float *r32, *e32;                     // outer FGCR right-hand side / solution
    std::vector<float*> Z, W;             // outer FGCR directions
    float2 *rc, *ec;                      // coarse right-hand side / solution
    std::vector<float2*> Zc, Wc;          // coarse GCR directions
    double m_applies;
};

static size_t fine_bytes(const lq_ctx* c, int n) { return 2 * parity_bytes(c->g, n, LQ_FP32); }
static size_t coarse_bytes(const MgState* s, int n) { return (size_t)s->m.Vc * s->m.nc * n * sizeof(float2); }
static double* slot(MgState* s, int i) { return s->d_s + (size_t)i * 3 * LQ_MAX_RHS; }

static void work_release(lq_ctx* c, MgState* s) {
    void* single[] = {s->res, s->t, s->d, s->rho, s->r32, s->e32, s->rc, s->ec};
    for (void* p : single) if (p) dev_free(c, p);
    s->res = s->t = s->d = s->rho = s->r32 = s->e32 = nullptr; s->rc = s->ec = nullptr;
    for (auto p : s->Z) dev_free(c, p);
    for (auto p : s->W) dev_free(c, p);
    for (auto p : s->Zc) dev_free(c, p);
    for (auto p : s->Wc) dev_free(c, p);
    s->Z.clear(); s->W.clear(); s->Zc.clear(); s->Wc.clear();
    s->wn = 0;
}
void mg_release(lq_ctx* c) {
    MgState* s = c->mg;
    if (!s) return;
    work_release(c, s);
    void* single[] = {s->site_f, s->nbr, s->status, s->P, s->Ac, s->d_s};
    for (void* p : single) if (p) dev_free(c, p);
    delete s;
    c->mg = nullptr;
}
void mg_invalidate(lq_ctx* c) { if (c->mg) c->mg->ready = false; }

// workspace: `outer` also allocates the outer FGCR vectors (lq_mg_solve); the cycle alone needs res, t and the coarse vectors
static int work_ensure(lq_ctx* c, MgState* s, int n, bool outer) {
    if (s->wn != n) work_release(c, s);
    s->wn = n;
    const size_t fb = fine_bytes(c, n), cb = coarse_bytes(s, n);
    auto need = [&](void** p, size_t bytes) -> int { if (!*p) { *p = dev_alloc(c, bytes); if (!*p) return LQ_ENOMEM; } return 0; };
    LQ_TRY(need((void**)&s->res, fb)); LQ_TRY(need((void**)&s->t, fb));
    if (s->prm.smoother == LQ_MG_SMOOTH_EO) { LQ_TRY(need((void**)&s->d, fb)); LQ_TRY(need((void**)&s->rho, fb)); }
    LQ_TRY(need((void**)&s->rc, cb)); LQ_TRY(need((void**)&s->ec, cb));
    const int mc = s->prm.coarse_iters < MG_MAX_RESTART ? s->prm.coarse_iters : MG_MAX_RESTART;
    while ((int)s->Zc.size() < mc) {
        float2* z = (float2*)dev_alloc(c, cb); if (!z) return LQ_ENOMEM; s->Zc.push_back(z);
        float2* w = (float2*)dev_alloc(c, cb); if (!w) return LQ_ENOMEM; s->Wc.push_back(w);
    }
    if (outer) {
        LQ_TRY(need((void**)&s->r32, fb)); LQ_TRY(need((void**)&s->e32, fb));
        while ((int)s->Z.size() < s->prm.restart) {
            float* z = (float*)dev_alloc(c, fb); if (!z) return LQ_ENOMEM; s->Z.push_back(z);
            float* w = (float*)dev_alloc(c, fb); if (!w) return LQ_ENOMEM; s->W.push_back(w);
        }
    }
    return 0;
}

// ---- launches ---------------------------------------------------------------------------------------------------------------
#define MG_R_DISPATCH(R_, CALL4, CALL2, CALL1) do { if ((R_) == 4) { CALL4; } else if ((R_) == 2) { CALL2; } else { CALL1; } } while (0)

static int fine_M(lq_ctx* c, MgState* s, int n, float* out, const float* in) {       // out = M in (fp32)
    const size_t pb = parity_bytes(c->g, n, LQ_FP32);
    char* oe = (char*)out; const char* ie = (const char*)in;
    LQ_TRY(op_kernel_b(c, LQ_FP32, n, 0, oe, ie, ie + pb, -c->kappa, 1, 0));
    LQ_TRY(op_kernel_b(c, LQ_FP32, n, 1, oe + pb, ie + pb, ie, -c->kappa, 1, 0));
    s->m_applies += 1;
    return 0;
}
// parities: 2 = full-lattice vectors, 1 = one parity block
static int fine_cdot3(lq_ctx* c, int n, const float* a, const float* b, double* d_out, int parities = 2) {
    const int R = group_width(n), G = n / R, units = parities * c->g.NB * G;
    const int block = 128, grid = (units * 32 + block - 1) / block;
    LQ_TRY(ensure_partials(c, (size_t)grid * 3 * n));
    const size_t smem = (block / 32) * R * sizeof(double);
    MG_R_DISPATCH(R, (mg::fine_cdot3_kernel<4><<<grid, block, smem, c->stream>>>(units, n, G, a, b, c->red_partials)),
                     (mg::fine_cdot3_kernel<2><<<grid, block, smem, c->stream>>>(units, n, G, a, b, c->red_partials)),
                     (mg::fine_cdot3_kernel<1><<<grid, block, smem, c->stream>>>(units, n, G, a, b, c->red_partials)));
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return reduce_finish(c, grid, 3, n, d_out);
}
// y1 += s1 c x1 ; y2 += s2 c x2 with c_k from (da + db); d_norm != null: ||y2||^2
static int fine_caxpy2(lq_ctx* c, int n, float* y1, const float* x1, float s1, float* y2, const float* x2, float s2,
                       const double* da, const double* db, double* d_norm, int parities = 2) {
    const int R = group_width(n), G = n / R, units = parities * c->g.NB * G;
    const int block = 128, grid = (units * 32 + block - 1) / block;
    const size_t smem = (block / 32) * R * sizeof(double);
    if (d_norm) {
        LQ_TRY(ensure_partials(c, (size_t)grid * n));
        MG_R_DISPATCH(R, (mg::fine_caxpy2_kernel<4, true><<<grid, block, smem, c->stream>>>(units, n, G, y1, x1, s1, y2, x2, s2, da, db, c->red_partials)),
                         (mg::fine_caxpy2_kernel<2, true><<<grid, block, smem, c->stream>>>(units, n, G, y1, x1, s1, y2, x2, s2, da, db, c->red_partials)),
                         (mg::fine_caxpy2_kernel<1, true><<<grid, block, smem, c->stream>>>(units, n, G, y1, x1, s1, y2, x2, s2, da, db, c->red_partials)));
    } else {
        MG_R_DISPATCH(R, (mg::fine_caxpy2_kernel<4, false><<<grid, block, 0, c->stream>>>(units, n, G, y1, x1, s1, y2, x2, s2, da, db, nullptr)),
                         (mg::fine_caxpy2_kernel<2, false><<<grid, block, 0, c->stream>>>(units, n, G, y1, x1, s1, y2, x2, s2, da, db, nullptr)),
                         (mg::fine_caxpy2_kernel<1, false><<<grid, block, 0, c->stream>>>(units, n, G, y1, x1, s1, y2, x2, s2, da, db, nullptr)));
    }
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    if (d_norm) return reduce_finish(c, grid, 1, n, d_norm);
    return 0;
}
static int fine_sub(lq_ctx* c, int n, float* out, const float* a, const float* b, float sign = -1.f) {   // out = a + sign b
    const size_t n4 = fine_bytes(c, n) / 16;
    const int block = 256, grid = (int)((n4 + block - 1) / block);
    mg::sub4_kernel<<<grid, block, 0, c->stream>>>(n4, (float4*)out, (const float4*)a, (const float4*)b, sign);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
static int do_restrict(lq_ctx* c, MgState* s, int n, float2* yc, const float* x) {
    const int R = group_width(n), G = n / R, KG = s->m.nv * G;
    int S = 256 / KG;
    if (S < 1) S = 1;
    if (S > s->m.ns) S = s->m.ns;
    const int block = ((KG * S + 31) / 32) * 32, grid = s->m.Vc * 2;
    const size_t smem = (size_t)S * KG * R * sizeof(float2);
    MG_R_DISPATCH(R, (mg::restrict_kernel<4><<<grid, block, smem, c->stream>>>(s->m, n, S, s->site_f, s->P, x, yc)),
                     (mg::restrict_kernel<2><<<grid, block, smem, c->stream>>>(s->m, n, S, s->site_f, s->P, x, yc)),
                     (mg::restrict_kernel<1><<<grid, block, smem, c->stream>>>(s->m, n, S, s->site_f, s->P, x, yc)));
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
static int do_prolong(lq_ctx* c, MgState* s, int n, float* x, const float2* yc, bool accumulate) {
    const int R = group_width(n);
    const int block = 256, grid = s->m.Vc * 2;
    const size_t smem = (size_t)s->m.nv * n * sizeof(float2);
    if (accumulate)
        MG_R_DISPATCH(R, (mg::prolong_kernel<4, true><<<grid, block, smem, c->stream>>>(s->m, n, s->site_f, s->P, yc, x)),
                         (mg::prolong_kernel<2, true><<<grid, block, smem, c->stream>>>(s->m, n, s->site_f, s->P, yc, x)),
                         (mg::prolong_kernel<1, true><<<grid, block, smem, c->stream>>>(s->m, n, s->site_f, s->P, yc, x)));
    else
        MG_R_DISPATCH(R, (mg::prolong_kernel<4, false><<<grid, block, smem, c->stream>>>(s->m, n, s->site_f, s->P, yc, x)),
                         (mg::prolong_kernel<2, false><<<grid, block, smem, c->stream>>>(s->m, n, s->site_f, s->P, yc, x)),
                         (mg::prolong_kernel<1, false><<<grid, block, smem, c->stream>>>(s->m, n, s->site_f, s->P, yc, x)));
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
static int coarse_M(lq_ctx* c, MgState* s, int n, float2* y, const float2* x) {
    const int nch = n % 8 == 0 ? 8 : (n % 4 == 0 ? 4 : n);      // right-hand sides per CTA
    const dim3 grid(s->m.Vc, n / nch);
    const size_t smem = (size_t)9 * s->m.nc * nch * sizeof(float2);
    if (nch == 8) mg::coarse_apply_kernel<8><<<grid, 288, smem, c->stream>>>(s->m, n, s->nbr, s->Ac, x, y);
    else if (nch == 4) mg::coarse_apply_kernel<4><<<grid, 288, smem, c->stream>>>(s->m, n, s->nbr, s->Ac, x, y);
    else if (nch == 2) mg::coarse_apply_kernel<2><<<grid, 288, smem, c->stream>>>(s->m, n, s->nbr, s->Ac, x, y);
    else mg::coarse_apply_kernel<1><<<grid, 288, smem, c->stream>>>(s->m, n, s->nbr, s->Ac, x, y);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
struct CoarseLaunch { dim3 block; int grid; size_t smem; };
static CoarseLaunch coarse_plan(const MgState* s, int n) {
    CoarseLaunch L;
    int by = 256 / n; if (by < 1) by = 1;
    L.block = dim3(n, by, 1);
    const long long rows = (long long)s->m.Vc * s->m.nc;
    long long g = (rows + by - 1) / by;
    if (g > 148 * 8) g = 148 * 8;
    L.grid = (int)g;
    L.smem = (size_t)by * n * sizeof(double);
    return L;
}
static int coarse_cdot3(lq_ctx* c, MgState* s, int n, const float2* a, const float2* b, double* d_out) {
    const CoarseLaunch L = coarse_plan(s, n);
    LQ_TRY(ensure_partials(c, (size_t)L.grid * 3 * n));
    mg::coarse_cdot3_kernel<<<L.grid, L.block, L.smem, c->stream>>>((long long)s->m.Vc * s->m.nc, n, a, b, c->red_partials);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return reduce_finish(c, L.grid, 3, n, d_out);
}
static int coarse_caxpy2(lq_ctx* c, MgState* s, int n, float2* y1, const float2* x1, float s1, float2* y2, const float2* x2, float s2,
                         const double* da, double* d_norm) {
    const CoarseLaunch L = coarse_plan(s, n);
    const long long rows = (long long)s->m.Vc * s->m.nc;
    if (d_norm) {
        LQ_TRY(ensure_partials(c, (size_t)L.grid * n));
        mg::coarse_caxpy2_kernel<true><<<L.grid, L.block, L.smem, c->stream>>>(rows, n, y1, x1, s1, y2, x2, s2, da, c->red_partials);
    } else mg::coarse_caxpy2_kernel<false><<<L.grid, L.block, 0, c->stream>>>(rows, n, y1, x1, s1, y2, x2, s2, da, nullptr);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    if (d_norm) return reduce_finish(c, L.grid, 1, n, d_norm);
    return 0;
}

// ---- GCR(m) with device-resident coefficients, shared by the two levels -------------------------------------------------------
// x = 0 and r = right-hand side on entry; on exit x is the approximate solution and r the recursively updated residual.
// Iteration k (inside the restart cycle): z_k = precond(r) (or r), w_k = Op z_k, modified Gram-Schmidt of w_k against w_0 .. w_{k-1}
// (the same combination applied to z_k), alpha = <w_k, r> / <w_k, w_k>, x += alpha z_k, r -= alpha w_k.  No host
// synchronisation unless `h_target2` is given: then ||r_k||^2 is fetched after every iteration and the loop stops when every
// right-hand side is at or below its target.
struct Krylov {
    std::function<int(void* out, const void* in)> op;
    std::function<int(void* z, const void* r)> precond;          // empty: z = r
    std::function<int(const void* a, const void* b, double* d)> cdot3;
    std::function<int(void* y1, const void* x1, float s1, void* y2, const void* x2, float s2, const double* d, double* d_norm)> caxpy2;
    size_t bytes;
};
static int gcr(lq_ctx* c, MgState* s, const Krylov& K, int n, void* x, void* r, void* const* Z, void* const* W, int m, int iters,
               const double* h_target2, int* iters_done) {
    double* d0 = slot(s, 0); double* d1 = slot(s, 1); double* d_rn = slot(s, 2);
    int it = 0;
    for (; it < iters; it++) {
        const int k = it % m;
        if (K.precond) LQ_TRY(K.precond(Z[k], r));
        else LQ_CUDA(c, cudaMemcpyAsync(Z[k], r, K.bytes, cudaMemcpyDeviceToDevice, c->stream));
        LQ_TRY(K.op(W[k], Z[k]));
        for (int i = 0; i < k; i++) {
            LQ_TRY(K.cdot3(W[i], W[k], d0));
            LQ_TRY(K.caxpy2(W[k], W[i], -1.f, Z[k], Z[i], -1.f, d0, nullptr));
        }
        LQ_TRY(K.cdot3(W[k], r, d1));
        LQ_TRY(K.caxpy2(x, Z[k], 1.f, r, W[k], -1.f, d1, h_target2 ? d_rn : nullptr));
        if (h_target2) {
            LQ_CUDA(c, cudaMemcpyAsync(c->h_scalars, d_rn, n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
            LQ_CUDA(c, cudaStreamSynchronize(c->stream));
            bool all = true;
            for (int q = 0; q < n; q++) if (!(c->h_scalars[q] <= h_target2[q])) all = false;
            if (all) { it++; break; }
        }
    }
    if (iters_done) *iters_done = it;
    return 0;
}

static Krylov coarse_level(lq_ctx* c, MgState* s, int n) {
    Krylov K;
    K.op = [=](void* out, const void* in) { return coarse_M(c, s, n, (float2*)out, (const float2*)in); };
    K.cdot3 = [=](const void* a, const void* b, double* d) { return coarse_cdot3(c, s, n, (const float2*)a, (const float2*)b, d); };
    K.caxpy2 = [=](void* y1, const void* x1, float s1, void* y2, const void* x2, float s2, const double* d, double* dn) {
        return coarse_caxpy2(c, s, n, (float2*)y1, (const float2*)x1, s1, (float2*)y2, (const float2*)x2, s2, d, dn); };
    K.bytes = coarse_bytes(s, n);
    return K;
}

// LQ_MG_SMOOTH_MR: minimal-residual steps on (z, res): t = M res, w = <t, res> / <t, t>, z += w res, res -= w t
static int smooth_mr(lq_ctx* c, MgState* s, int n, float* z, int steps) {
    for (int i = 0; i < steps; i++) {
        LQ_TRY(fine_M(c, s, n, s->t, s->res));
        LQ_TRY(fine_cdot3(c, n, s->t, s->res, slot(s, 3)));
        LQ_TRY(fine_caxpy2(c, n, z, s->res, 1.f, s->res, s->t, -1.f, slot(s, 3), nullptr, nullptr));
    }
    return 0;
}
// LQ_MG_SMOOTH_EO: delta ~ M^{-1} res through the even-odd Schur system (steps 8-10 of the solver, with `steps` minimal-residual
// steps instead of CG): rho_e = res_e + kappa D_eo A_oo^{-1} res_o; delta_e from Mhat delta_e = rho_e; delta_o = A_oo^{-1} (res_o +
// kappa D_oe delta_e).  z = delta or z += delta.  On exit res = (rho_e, 0), exactly the residual of the updated z: the odd rows are
// solved exactly.  Cost: `steps` applications of Mhat (kernel A + kernel B) and two hops; Mhat's spectrum lambda (2 - lambda) folds
// the lambda ~ 2 end of M's spectrum onto the low modes, which plain minimal residual on M leaves undamped.
static int smooth_eo(lq_ctx* c, MgState* s, int n, float* z, bool accumulate, int steps) {
    const size_t pb = parity_bytes(c->g, n, LQ_FP32);
    const double k = c->kappa;
    float* d = accumulate ? s->d : z;
    char *res_e = (char*)s->res, *res_o = res_e + pb, *t_e = (char*)s->t, *t_o = t_e + pb, *d_e = (char*)d, *d_o = d_e + pb;
    char* rho_e = (char*)s->rho;
    LQ_TRY(op_clover(c, LQ_FP32, n, 1, t_o, res_o, 1));
    LQ_TRY(op_kernel_b(c, LQ_FP32, n, 0, rho_e, res_e, t_o, k, 0, 0));
    LQ_CUDA(c, cudaMemsetAsync(d_e, 0, pb, c->stream));
    for (int i = 0; i < steps; i++) {
        LQ_TRY(op_kernel_a(c, LQ_FP32, n, 1, t_o, rho_e, 0));
        // t_e = Mhat rho_e with <t, rho> and ||t||^2 from the kernel's fused epilogue (the BiCGStab omega of solver.cu)
        LQ_TRY(op_kernel_b_cdot(c, LQ_FP32, n, 0, t_e, rho_e, t_o, -k * k, 1, 0, rho_e, 1, slot(s, 3)));
        s->m_applies += 1;
        LQ_TRY(fine_caxpy2(c, n, (float*)d_e, (float*)rho_e, 1.f, (float*)rho_e, (float*)t_e, -1.f, slot(s, 3), nullptr, nullptr, 1));
    }
    LQ_TRY(op_kernel_b(c, LQ_FP32, n, 1, t_o, res_o, d_e, k, 0, 0));
    LQ_TRY(op_clover(c, LQ_FP32, n, 1, d_o, t_o, 1));
    s->m_applies += 1;        // the two hops and clover applications of the source and the reconstruction
    if (accumulate) LQ_TRY(fine_sub(c, n, z, z, s->d, 1.f));
    LQ_CUDA(c, cudaMemcpyAsync(res_e, rho_e, pb, cudaMemcpyDeviceToDevice, c->stream));
    LQ_CUDA(c, cudaMemsetAsync(res_o, 0, pb, c->stream));
    return 0;
}
// z ~ M^{-1} r  (the two-grid cycle of the header; r is not modified, z must not alias r)
static int vcycle(lq_ctx* c, MgState* s, int n, float* z, const float* r) {
    const size_t fb = fine_bytes(c, n), cb = coarse_bytes(s, n);
    const bool eo = s->prm.smoother == LQ_MG_SMOOTH_EO;
    LQ_CUDA(c, cudaMemcpyAsync(s->res, r, fb, cudaMemcpyDeviceToDevice, c->stream));
    if (eo && s->prm.nu_pre > 0) LQ_TRY(smooth_eo(c, s, n, z, false, s->prm.nu_pre));
    else {
        LQ_CUDA(c, cudaMemsetAsync(z, 0, fb, c->stream));
        LQ_TRY(smooth_mr(c, s, n, z, s->prm.nu_pre));
    }
    // coarse correction
    LQ_TRY(do_restrict(c, s, n, s->rc, s->res));
    LQ_CUDA(c, cudaMemsetAsync(s->ec, 0, cb, c->stream));
    const int mc = (int)s->Zc.size();
    const Krylov K = coarse_level(c, s, n);
    LQ_TRY(gcr(c, s, K, n, s->ec, s->rc, (void* const*)s->Zc.data(), (void* const*)s->Wc.data(), mc, s->prm.coarse_iters, nullptr, nullptr));
    LQ_TRY(do_prolong(c, s, n, z, s->ec, true));
    if (s->prm.nu_post > 0) {
        LQ_TRY(fine_M(c, s, n, s->t, z));
        LQ_TRY(fine_sub(c, n, s->res, r, s->t));
        if (eo) LQ_TRY(smooth_eo(c, s, n, z, true, s->prm.nu_post));
        else LQ_TRY(smooth_mr(c, s, n, z, s->prm.nu_post));
    }
    return 0;
}

// ---- setup ------------------------------------------------------------------------------------------------------------------
static int smallest_divisor_ge3(int L) { for (int d = 3; d <= L; d++) if (L % d == 0) return d; return L; }

static float ms_between(cudaEvent_t a, cudaEvent_t b) { float ms = 0.f; cudaEventElapsedTime(&ms, a, b); return ms; }

static int check_param(lq_ctx* c, const lq_mg_param* p) {
    if (!p) return set_err(c, LQ_EINVAL, "lq_mg_setup: null parameters");
    for (int mu = 0; mu < 4; mu++)
        if (p->block[mu] < 1 || c->g.L[mu] % p->block[mu] != 0) return set_err(c, LQ_EINVAL, "lq_mg_setup: block must divide the lattice extent");
    const int nv = p->n_vec;
    if (!(nv == 1 || nv == 2 || (nv >= 4 && nv <= LQ_MAX_RHS && nv % 4 == 0))) return set_err(c, LQ_EINVAL, "lq_mg_setup: n_vec must be 1, 2 or a multiple of 4 up to 32");
    if (p->nu_pre < 0 || p->nu_post < 0 || p->coarse_iters < 1 || p->restart < 1 || p->restart > MG_MAX_RESTART ||
        (p->smoother != LQ_MG_SMOOTH_MR && p->smoother != LQ_MG_SMOOTH_EO))
        return set_err(c, LQ_EINVAL, "lq_mg_setup: bad cycle parameters");
    if (c->g.Vh % SB != 0) return set_err(c, LQ_EINVAL, "lq_mg_setup: the multigrid needs V % 64 == 0");
    const long long ns = (long long)p->block[0] * p->block[1] * p->block[2] * p->block[3];
    if (ns < 2) return set_err(c, LQ_EINVAL, "lq_mg_setup: an aggregate needs at least 2 sites");
    if (6 * ns < nv) return set_err(c, LQ_EINVAL, "lq_mg_setup: more near-null vectors than degrees of freedom per aggregate and chirality");
    if (!c->has_gauge || !c->has_clover) return set_err(c, LQ_ESTATE, "lq_mg_setup: gauge field and clover term first");
    return 0;
}

// vecs32: native fp32 full-lattice batch of n_vec near-null vectors (device)
static int setup_from_native(lq_ctx* c, const lq_mg_param* p, const float* vecs32, lq_mg_info* info) {
    mg_release(c);
    MgState* s = new MgState();
    c->mg = s;
    s->prm = *p; s->ready = false; s->wn = 0; s->m_applies = 0; s->probes = 0;
    s->site_f = s->nbr = s->status = nullptr; s->P = s->Ac = nullptr; s->d_s = nullptr;
    s->res = s->t = s->d = s->rho = s->r32 = s->e32 = nullptr; s->rc = s->ec = nullptr;
    MgGeom& m = s->m;
    m.Vc = 1; m.ns = 1;
    for (int mu = 0; mu < 4; mu++) { m.b[mu] = p->block[mu]; m.Lc[mu] = c->g.L[mu] / p->block[mu]; m.Vc *= m.Lc[mu]; m.ns *= m.b[mu]; }
    m.nv = p->n_vec; m.nc = 2 * m.nv; m.M = 6 * m.ns;
    const size_t Pbytes = (size_t)m.Vc * 2 * m.M * m.nv * sizeof(float2);
    const size_t Abytes = (size_t)m.Vc * 9 * m.nc * m.nc * sizeof(float2);
    s->site_f = (int*)dev_alloc(c, (size_t)m.Vc * m.ns * sizeof(int));
    s->nbr = (int*)dev_alloc(c, (size_t)m.Vc * 9 * sizeof(int));
    s->status = (int*)dev_alloc(c, 256);
    s->P = (float2*)dev_alloc(c, Pbytes);
    s->Ac = (float2*)dev_alloc(c, Abytes);
    s->d_s = (double*)dev_alloc(c, (size_t)8 * 3 * LQ_MAX_RHS * sizeof(double));
    if (!s->site_f || !s->nbr || !s->status || !s->P || !s->Ac || !s->d_s) return LQ_ENOMEM;
    struct Events { cudaEvent_t e[3] = {nullptr, nullptr, nullptr}; ~Events() { for (cudaEvent_t x : e) if (x) cudaEventDestroy(x); } } evs;   // also on the error returns
    cudaEvent_t (&ev)[3] = evs.e;
    for (auto& e : ev) LQ_CUDA(c, cudaEventCreate(&e));
    LQ_CUDA(c, cudaEventRecord(ev[0], c->stream));
    // tables
    {
        const long long th = (long long)m.Vc * m.ns;
        mg::tables_kernel<<<(int)((th + 255) / 256), 256, 0, c->stream>>>(c->g, m, s->site_f);
        LQ_LAUNCHED(c);
        std::vector<int> nb((size_t)m.Vc * 9);
        for (int a = 0; a < m.Vc; a++) {
            int ac[4], q = a;
            for (int mu = 0; mu < 4; mu++) { ac[mu] = q % m.Lc[mu]; q /= m.Lc[mu]; }
            nb[(size_t)a * 9] = a;
            for (int mu = 0; mu < 4; mu++) {
                int stride = 1;
                for (int nu = 0; nu < mu; nu++) stride *= m.Lc[nu];
                const int fwd = a + (((ac[mu] + 1) % m.Lc[mu]) - ac[mu]) * stride;
                const int bwd = a + (((ac[mu] + m.Lc[mu] - 1) % m.Lc[mu]) - ac[mu]) * stride;
                nb[(size_t)a * 9 + 1 + 2 * mu] = m.Lc[mu] >= 2 ? fwd : -1;
                nb[(size_t)a * 9 + 2 + 2 * mu] = m.Lc[mu] >= 3 ? bwd : -1;
            }
        }
        LQ_CUDA(c, cudaMemcpyAsync(s->nbr, nb.data(), nb.size() * sizeof(int), cudaMemcpyHostToDevice, c->stream));
        LQ_CUDA(c, cudaStreamSynchronize(c->stream));      // nb goes out of scope
    }
    // prolongator
    {
        const int R = group_width(m.nv);
        const long long th = (long long)m.Vc * 2 * m.M * m.nv;
        const int grid = (int)((th + 255) / 256);
        MG_R_DISPATCH(R, (mg::gather_P_kernel<4><<<grid, 256, 0, c->stream>>>(m, s->site_f, vecs32, s->P)),
                         (mg::gather_P_kernel<2><<<grid, 256, 0, c->stream>>>(m, s->site_f, vecs32, s->P)),
                         (mg::gather_P_kernel<1><<<grid, 256, 0, c->stream>>>(m, s->site_f, vecs32, s->P)));
        LQ_LAUNCHED(c);
        LQ_CUDA(c, cudaMemsetAsync(s->status, 0, 256, c->stream));
        mg::orthonormalise_kernel<<<m.Vc * 2, 256, 0, c->stream>>>(m, s->P, s->status);
        LQ_LAUNCHED(c);
        int st = 0;
        LQ_CUDA(c, cudaMemcpyAsync(&st, s->status, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
        LQ_CUDA(c, cudaEventRecord(ev[1], c->stream));
        LQ_CUDA(c, cudaStreamSynchronize(c->stream));
        if (st != 0) return set_err(c, LQ_ESINGULAR, "lq_mg_setup: near-null vectors are linearly dependent on an aggregate");
    }
    // coarse operator by probing (mg_kernels.cuh, "Galerkin coarse operator by probing")
    {
        LQ_CUDA(c, cudaMemsetAsync(s->Ac, 0, Abytes, c->stream));
        struct Probe { int col, mu, colour, ncol; };
        std::vector<Probe> probes;
        for (int col = 0; col < m.nc; col++) probes.push_back({col, -1, 0, 1});
        for (int mu = 0; mu < 4; mu++) {
            if (m.Lc[mu] < 2) continue;
            const int ncol = m.Lc[mu] == 2 ? 2 : smallest_divisor_ge3(m.Lc[mu]);
            for (int cl = 0; cl < ncol; cl++)
                for (int col = 0; col < m.nc; col++) probes.push_back({col, mu, cl, ncol});
        }
        const int nb = 16, R = 4;      // probing batch
        const size_t fb = fine_bytes(c, nb);
        float* x = (float*)dev_alloc(c, fb); float* y = (float*)dev_alloc(c, fb);
        float2* yc = (float2*)dev_alloc(c, coarse_bytes(s, nb));
        int rc = (!x || !y || !yc) ? LQ_ENOMEM : 0;
        for (size_t p0 = 0; p0 < probes.size() && rc == 0; p0 += nb) {
            mg::ProbeDesc pd;
            for (int k = 0; k < LQ_MAX_RHS; k++) { pd.col[k] = -1; pd.mu[k] = -1; pd.colour[k] = 0; pd.ncol[k] = 1; }
            for (int k = 0; k < nb && p0 + k < probes.size(); k++) {
                const Probe& q = probes[p0 + k];
                pd.col[k] = q.col; pd.mu[k] = q.mu; pd.colour[k] = q.colour; pd.ncol[k] = q.ncol;
            }
            const long long th = (long long)m.Vc * m.ns * nb;
            mg::probe_fill_kernel<R><<<(int)((th + 255) / 256), 256, 0, c->stream>>>(m, nb, pd, s->site_f, s->P, x);
            LQ_LAUNCHED(c);
            rc = fine_M(c, s, nb, y, x);
            if (rc == 0) rc = do_restrict(c, s, nb, yc, y);
            if (rc == 0) {
                const long long th2 = (long long)m.Vc * m.nc * nb;
                mg::probe_scatter_kernel<<<(int)((th2 + 255) / 256), 256, 0, c->stream>>>(m, nb, pd, yc, s->Ac);
                LQ_LAUNCHED(c);
                if (cudaGetLastError() != cudaSuccess) rc = set_err(c, LQ_ECUDA, "lq_mg_setup: probing launch failed");
            }
        }
        s->probes = (int)probes.size();
        if (rc == 0) {
            const long long th = (long long)m.Vc * m.nc * m.nc;
            mg::self_fix_kernel<<<(int)((th + 255) / 256), 256, 0, c->stream>>>(m, s->nbr, s->Ac);
            LQ_LAUNCHED(c);
        }
        cudaEventRecord(ev[2], c->stream);
        if (cudaStreamSynchronize(c->stream) != cudaSuccess && rc == 0) rc = set_err(c, LQ_ECUDA, std::string("lq_mg_setup: ") + cudaGetErrorString(cudaGetLastError()));
        void* tofree[] = {x, y, yc};
        for (void* q : tofree) if (q) dev_free(c, q);
        if (rc != 0) return rc;
    }
    s->m_applies = 0;
    s->ready = true;
    if (info) {
        for (int mu = 0; mu < 4; mu++) info->coarse_dims[mu] = m.Lc[mu];
        info->coarse_dof = (long long)m.Vc * m.nc;
        info->probes = s->probes;
        info->seconds_prolongator = ms_between(ev[0], ev[1]) * 1e-3;
        info->seconds_coarse_op = ms_between(ev[1], ev[2]) * 1e-3;
        info->bytes = Pbytes + Abytes + (size_t)m.Vc * (m.ns + 9) * sizeof(int);
    }
    return 0;
}

int mg_setup_vectors(lq_ctx* c, const lq_mg_param* p, const void* dev_canonical64, lq_mg_info* info) {
    LQ_TRY(check_param(c, p));
    if (info) memset(info, 0, sizeof(*info));
    float* v32 = (float*)dev_alloc(c, fine_bytes(c, p->n_vec));
    if (!v32) return LQ_ENOMEM;
    int rc = spinor_pack(c, v32, dev_canonical64, p->n_vec, LQ_FP32, LQ_FP64);
    if (rc == 0) rc = setup_from_native(c, p, v32, info);
    if (cudaStreamSynchronize(c->stream) != cudaSuccess && rc == 0) rc = set_err(c, LQ_ECUDA, "lq_mg_setup_from_vectors failed");
    dev_free(c, v32);
    if (rc != 0) mg_release(c);
    return rc;
}

int mg_setup_adaptive(lq_ctx* c, const lq_mg_param* p, lq_mg_info* info) {
    LQ_TRY(check_param(c, p));
    if (!(p->setup_tol > 0) || !(p->setup_tol < 1)) return set_err(c, LQ_EINVAL, "lq_mg_setup: setup_tol must lie in (0, 1)");
    if (p->refine < 0 || p->refine > 16) return set_err(c, LQ_EINVAL, "lq_mg_setup: refine must lie in 0 .. 16");
    if (info) memset(info, 0, sizeof(*info));
    const int nv = p->n_vec;
    const size_t pb64 = parity_bytes(c->g, nv, LQ_FP64), pb32 = parity_bytes(c->g, nv, LQ_FP32);
    void* eta = dev_alloc(c, 2 * pb64); void* v64 = dev_alloc(c, 2 * pb64);
    float* v32 = (float*)dev_alloc(c, 2 * pb32);
    int rc = (!eta || !v64 || !v32) ? LQ_ENOMEM : 0;
    double secs = 0;
    if (rc == 0) rc = fill_spinor(c, eta, nv, LQ_FP64, p->seed, 0, 0);
    if (rc == 0) {
        lq_solve_param sp;
        memset(&sp, 0, sizeof(sp));
        sp.tol = p->setup_tol; sp.max_outer = 10; sp.max_inner = 2000; sp.inner_prec = LQ_FP32; sp.delta = 0.1; sp.check_every = 10;
        sp.use_graph = 1; sp.keep_direction = 1; sp.algorithm = LQ_ALG_CGNR; sp.use_x0 = 0;
        lq_solve_info si;
        memset(&si, 0, sizeof(si));
        rc = solve_native(c, v64, eta, nv, &sp, &si);
        if (rc == LQ_ENOTCONVERGED) rc = 0;      // loosely solved vectors are still rich in low modes
        secs = si.seconds;
    }
    if (rc == 0) rc = spinor_convert(c, v32, LQ_FP32, v64, LQ_FP64, nv, nullptr, 0);
    if (rc == 0) rc = spinor_convert(c, (char*)v32 + pb32, LQ_FP32, (char*)v64 + pb64, LQ_FP64, nv, nullptr, 0);
    if (rc == 0) rc = setup_from_native(c, p, v32, info);
    // adaptive refinement: with the hierarchy just built, v <- v - cycle(M v) for all vectors at once, then rebuild P and A_c
    double t_p = info ? info->seconds_prolongator : 0.0, t_a = info ? info->seconds_coarse_op : 0.0;
    int probes = info ? info->probes : 0;
    for (int pass = 0; pass < p->refine && rc == 0; pass++) {
        MgState* s = c->mg;
        rc = work_ensure(c, s, nv, false);
        float* r = nullptr; float* z = nullptr;
        if (rc == 0) { r = (float*)dev_alloc(c, 2 * pb32); z = (float*)dev_alloc(c, 2 * pb32); if (!r || !z) rc = LQ_ENOMEM; }
        if (rc == 0) rc = fine_M(c, s, nv, r, v32);
        if (rc == 0) rc = vcycle(c, s, nv, z, r);
        if (rc == 0) rc = fine_sub(c, nv, v32, v32, z, -1.f);
        if (cudaStreamSynchronize(c->stream) != cudaSuccess && rc == 0) rc = set_err(c, LQ_ECUDA, "lq_mg_setup: refinement failed");
        if (r) dev_free(c, r);
        if (z) dev_free(c, z);
        if (rc == 0) rc = setup_from_native(c, p, v32, info);
        if (rc == 0 && info) { t_p += info->seconds_prolongator; t_a += info->seconds_coarse_op; probes += info->probes; }
    }
    if (rc == 0 && info) { info->seconds_prolongator = t_p; info->seconds_coarse_op = t_a; info->probes = probes; }
    if (cudaStreamSynchronize(c->stream) != cudaSuccess && rc == 0) rc = set_err(c, LQ_ECUDA, "lq_mg_setup failed");
    void* tofree[] = {eta, v64, v32};
    for (void* q : tofree) if (q) dev_free(c, q);
    if (rc != 0) mg_release(c);
    else if (info) info->seconds_vectors = secs;
    return rc;
}

static int mg_ready(lq_ctx* c, const char* who) {
    if (!c->mg || !c->mg->ready) return set_err(c, LQ_ESTATE, std::string(who) + ": no multigrid hierarchy (run lq_mg_setup; gauge or clover changes invalidate it)");
    return 0;
}

// ---- the pieces at the boundary: device canonical fp64 fine vectors, device complex fp64 coarse vectors [rhs][Vc][nc] -------
static int coarse_in(lq_ctx* c, MgState* s, int n, float2* dst, const double* src) {
    const long long rows = (long long)s->m.Vc * s->m.nc, th = rows * n;
    mg::coarse_pack_kernel<<<(int)((th + 255) / 256), 256, 0, c->stream>>>(rows, n, src, dst);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
static int coarse_out(lq_ctx* c, MgState* s, int n, double* dst, const float2* src) {
    const long long rows = (long long)s->m.Vc * s->m.nc, th = rows * n;
    mg::coarse_unpack_kernel<<<(int)((th + 255) / 256), 256, 0, c->stream>>>(rows, n, src, dst);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
size_t mg_coarse_canonical_bytes(const lq_ctx* c, int n) { return c->mg ? (size_t)c->mg->m.Vc * c->mg->m.nc * n * 2 * sizeof(double) : 0; }

int mg_restrict_dev(lq_ctx* c, double* coarse64, const void* fine_canonical64, int n) {
    LQ_TRY(mg_ready(c, "lq_mg_restrict"));
    MgState* s = c->mg;
    float* x = (float*)dev_alloc(c, fine_bytes(c, n)); float2* y = (float2*)dev_alloc(c, coarse_bytes(s, n));
    int rc = (!x || !y) ? LQ_ENOMEM : 0;
    if (rc == 0) rc = spinor_pack(c, x, fine_canonical64, n, LQ_FP32, LQ_FP64);
    if (rc == 0) rc = do_restrict(c, s, n, y, x);
    if (rc == 0) rc = coarse_out(c, s, n, coarse64, y);
    if (cudaStreamSynchronize(c->stream) != cudaSuccess && rc == 0) rc = set_err(c, LQ_ECUDA, "lq_mg_restrict failed");
    if (x) dev_free(c, x);
    if (y) dev_free(c, y);
    return rc;
}
int mg_prolong_dev(lq_ctx* c, void* fine_canonical64, const double* coarse64, int n) {
    LQ_TRY(mg_ready(c, "lq_mg_prolong"));
    MgState* s = c->mg;
    float* x = (float*)dev_alloc(c, fine_bytes(c, n)); float2* y = (float2*)dev_alloc(c, coarse_bytes(s, n));
    int rc = (!x || !y) ? LQ_ENOMEM : 0;
    if (rc == 0) rc = coarse_in(c, s, n, y, coarse64);
    if (rc == 0) rc = do_prolong(c, s, n, x, y, false);
    if (rc == 0) rc = spinor_unpack(c, fine_canonical64, x, n, LQ_FP32, LQ_FP64);
    if (cudaStreamSynchronize(c->stream) != cudaSuccess && rc == 0) rc = set_err(c, LQ_ECUDA, "lq_mg_prolong failed");
    if (x) dev_free(c, x);
    if (y) dev_free(c, y);
    return rc;
}
int mg_coarse_apply_dev(lq_ctx* c, double* out64, const double* in64, int n) {
    LQ_TRY(mg_ready(c, "lq_mg_coarse_apply"));
    MgState* s = c->mg;
    float2* x = (float2*)dev_alloc(c, coarse_bytes(s, n)); float2* y = (float2*)dev_alloc(c, coarse_bytes(s, n));
    int rc = (!x || !y) ? LQ_ENOMEM : 0;
    if (rc == 0) rc = coarse_in(c, s, n, x, in64);
    if (rc == 0) rc = coarse_M(c, s, n, y, x);
    if (rc == 0) rc = coarse_out(c, s, n, out64, y);
    if (cudaStreamSynchronize(c->stream) != cudaSuccess && rc == 0) rc = set_err(c, LQ_ECUDA, "lq_mg_coarse_apply failed");
    if (x) dev_free(c, x);
    if (y) dev_free(c, y);
    return rc;
}
int mg_vcycle_dev(lq_ctx* c, void* z_canonical64, const void* r_canonical64, int n) {
    LQ_TRY(mg_ready(c, "lq_mg_vcycle"));
    MgState* s = c->mg;
    LQ_TRY(work_ensure(c, s, n, false));
    float* r = (float*)dev_alloc(c, fine_bytes(c, n)); float* z = (float*)dev_alloc(c, fine_bytes(c, n));
    int rc = (!r || !z) ? LQ_ENOMEM : 0;
    if (rc == 0) rc = spinor_pack(c, r, r_canonical64, n, LQ_FP32, LQ_FP64);
    if (rc == 0) rc = vcycle(c, s, n, z, r);
    if (rc == 0) rc = spinor_unpack(c, z_canonical64, z, n, LQ_FP32, LQ_FP64);
    if (cudaStreamSynchronize(c->stream) != cudaSuccess && rc == 0) rc = set_err(c, LQ_ECUDA, "lq_mg_vcycle failed");
    if (r) dev_free(c, r);
    if (z) dev_free(c, z);
    return rc;
}

// ---- solve: FGCR(restart) preconditioned by the cycle, fp32, inside an fp64 defect correction --------------------------------
static int fine_M64(lq_ctx* c, MgState* s, int n, void* out, const void* in) {
    const size_t pb = parity_bytes(c->g, n, LQ_FP64);
    char* oe = (char*)out; const char* ie = (const char*)in;
    LQ_TRY(op_kernel_b(c, LQ_FP64, n, 0, oe, ie, ie + pb, -c->kappa, 1, 0));
    LQ_TRY(op_kernel_b(c, LQ_FP64, n, 1, oe + pb, ie + pb, ie, -c->kappa, 1, 0));
    s->m_applies += 1;
    return 0;
}
// per-RHS sums of the two parity results sitting in slots a and b
static int fetch2(lq_ctx* c, const double* da, const double* db, int n, double* h) {
    LQ_CUDA(c, cudaMemcpyAsync(c->h_scalars, da, n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    LQ_CUDA(c, cudaMemcpyAsync(c->h_scalars + LQ_MAX_RHS, db, n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    LQ_CUDA(c, cudaStreamSynchronize(c->stream));
    for (int k = 0; k < n; k++) h[k] = c->h_scalars[k] + c->h_scalars[LQ_MAX_RHS + k];
    return 0;
}

int mg_solve_native(lq_ctx* c, void* x64, const void* b64, int n, double tol, int max_iter, lq_mg_solve_info* info) {
    LQ_TRY(mg_ready(c, "lq_mg_solve"));
    MgState* s = c->mg;
    memset(info, 0, sizeof(*info));
    LQ_TRY(work_ensure(c, s, n, true));
    const size_t pb64 = parity_bytes(c->g, n, LQ_FP64), pb32 = parity_bytes(c->g, n, LQ_FP32);
    void* r64 = dev_alloc(c, 2 * pb64); void* t64 = dev_alloc(c, 2 * pb64);
    if (!r64 || !t64) { if (r64) dev_free(c, r64); if (t64) dev_free(c, t64); return LQ_ENOMEM; }
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = 0, status = LQ_ENOTCONVERGED;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) rc = set_err(c, LQ_ECUDA, "event creation failed");
    s->m_applies = 0;
    double bn[LQ_MAX_RHS], rn[LQ_MAX_RHS], target2[LQ_MAX_RHS];
    double* d_a = slot(s, 4); double* d_b = slot(s, 5); double* d_scale = slot(s, 6);

    Krylov K;
    K.op = [=](void* out, const void* in) { return fine_M(c, s, n, (float*)out, (const float*)in); };
    K.precond = [=](void* z, const void* r) { return vcycle(c, s, n, (float*)z, (const float*)r); };
    K.cdot3 = [=](const void* a, const void* b, double* d) { return fine_cdot3(c, n, (const float*)a, (const float*)b, d); };
    K.caxpy2 = [=](void* y1, const void* x1, float s1, void* y2, const void* x2, float s2, const double* d, double* dn) {
        return fine_caxpy2(c, n, (float*)y1, (const float*)x1, s1, (float*)y2, (const float*)x2, s2, d, nullptr, dn); };
    K.bytes = 2 * pb32;

    auto body = [&]() -> int {
        LQ_CUDA(c, cudaEventRecord(e0, c->stream));
        LQ_CUDA(c, cudaMemsetAsync(x64, 0, 2 * pb64, c->stream));
        LQ_CUDA(c, cudaMemcpyAsync(r64, b64, 2 * pb64, cudaMemcpyDeviceToDevice, c->stream));
        LQ_TRY(blas_norm2(c, LQ_FP64, n, b64, d_a));
        LQ_TRY(blas_norm2(c, LQ_FP64, n, (const char*)b64 + pb64, d_b));
        LQ_TRY(fetch2(c, d_a, d_b, n, bn));
        for (int k = 0; k < n; k++) rn[k] = bn[k];
        int iters = 0, cycle = 0;
        for (;; cycle++) {
            bool all = true;
            for (int k = 0; k < n; k++) {
                info->true_rel_residual[k] = bn[k] > 0 ? sqrt(rn[k] / bn[k]) : 0.0;
                if (!(info->true_rel_residual[k] <= tol)) all = false;
            }
            if (all) { status = 0; break; }
            if (iters >= max_iter || cycle >= 20) break;
            // normalised inner system M e = r / ||r||, reduced to what is still needed (at most the fp32 floor 1e-5)
            double up[LQ_MAX_RHS];
            for (int k = 0; k < n; k++) {
                up[k] = sqrt(rn[k]);
                double want = rn[k] > 0 ? 0.5 * tol * sqrt(bn[k] / rn[k]) : 1.0;
                if (want < 1e-5) want = 1e-5;
                if (want > 0.5) want = 0.5;
                target2[k] = rn[k] > 0 ? want * want : 1e300;
            }
            memcpy(c->h_scalars, up, n * sizeof(double));
            LQ_CUDA(c, cudaMemcpyAsync(d_scale, c->h_scalars, n * sizeof(double), cudaMemcpyHostToDevice, c->stream));
            LQ_TRY(spinor_convert(c, s->r32, LQ_FP32, r64, LQ_FP64, n, d_scale, 1));
            LQ_TRY(spinor_convert(c, (char*)s->r32 + pb32, LQ_FP32, (char*)r64 + pb64, LQ_FP64, n, d_scale, 1));
            LQ_CUDA(c, cudaMemsetAsync(s->e32, 0, 2 * pb32, c->stream));
            int done = 0;
            LQ_TRY(gcr(c, s, K, n, s->e32, s->r32, (void* const*)s->Z.data(), (void* const*)s->W.data(), s->prm.restart, max_iter - iters, target2, &done));
            iters += done;
            // x += ||r|| e ; r = b - M x
            LQ_TRY(blas_axpy_mixed(c, LQ_FP32, n, x64, s->e32, d_scale));
            LQ_TRY(blas_axpy_mixed(c, LQ_FP32, n, (char*)x64 + pb64, (char*)s->e32 + pb32, d_scale));
            LQ_TRY(fine_M64(c, s, n, t64, x64));
            LQ_TRY(blas_residual(c, n, r64, b64, t64, d_a));
            LQ_TRY(blas_residual(c, n, (char*)r64 + pb64, (const char*)b64 + pb64, (char*)t64 + pb64, d_b));
            LQ_TRY(fetch2(c, d_a, d_b, n, rn));
        }
        info->iters = iters; info->outer_cycles = cycle;
        LQ_CUDA(c, cudaEventRecord(e1, c->stream));
        LQ_CUDA(c, cudaEventSynchronize(e1));
        float ms = 0.f;
        LQ_CUDA(c, cudaEventElapsedTime(&ms, e0, e1));
        info->seconds = ms * 1e-3;
        info->m_applies = s->m_applies;
        return 0;
    };
    if (rc == 0) rc = body();
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    dev_free(c, r64); dev_free(c, t64);
    if (rc != 0) return rc;
    if (status != 0) return set_err(c, LQ_ENOTCONVERGED, "lq_mg_solve: tolerance not reached within max_iter");
    return 0;
}
