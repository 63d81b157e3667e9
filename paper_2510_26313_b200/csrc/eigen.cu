// eigen.cu -- time-batched thick-restart Lanczos for the lowest eigenpairs of -Laplacian on every time-slice
// ("a highly-scalable batched Lanczos eigensolver", the time extent is the batch).
//
// All Lt slices advance in lockstep through the same kernels; every scalar of the iteration (Gram-Schmidt coefficients,
// norms, projected matrices, Ritz rotations) exists once per slice.  The operator handed to Lanczos is the Chebyshev
// polynomial B = T_d((2A - (a+b)) / (b-a)) of A = -Laplacian: eigenvalues of A below the cut `a` are mapped to the
// largest |eigenvalues| of B, which Lanczos finds first.  The Krylov basis is kept fully orthogonal (two classical
// Gram-Schmidt passes per step), so the projected matrix T = V^dag B V is real symmetric and is simply re-diagonalised at every
// restart ON THE DEVICE (ritz_jacobi_kernel: one CTA per time-slice, parallel two-sided Jacobi, all slices in one launch); the k
// best Ritz vectors and the residual vector seed the next sweep (thick restart).  Eigenvalues of A are returned as Rayleigh quotients <v, A v> of the final Ritz vectors.
#include <math.h>
#include <string.h>
#include <algorithm>
#include <vector>
#include "internal.cuh"
#include "eigen_kernels.cuh"

namespace {

struct Eig {
    lq_ctx* c; SliceGeom sg; int Lt, nchunk; size_t fbytes;
    double2 *d_partial, *d_H;     // dot partials; coefficient rows [m+2][Lt]
    double* d_scale;              // [Lt]
    std::vector<double2> h_H;
    long long lap_applies = 0;
};

int grid_sites(const Eig& e) { return (int)((2LL * e.sg.Vh + 127) / 128); }

int dot(Eig& e, const double* a, const double* b, double2* d_out) {
    slice_dot_kernel<<<e.Lt * e.nchunk, 256, 0, e.c->stream>>>(e.sg, e.nchunk, a, b, e.d_partial);
    slice_dot_final_kernel<<<(e.Lt + 63) / 64, 64, 0, e.c->stream>>>(e.Lt, e.nchunk, e.d_partial, d_out);
    e.c->launches += 2;
    LQ_CUDA(e.c, cudaGetLastError());
    return 0;
}
__global__ void negate_kernel(int n, double2* h) { const int i = blockIdx.x * blockDim.x + threadIdx.x; if (i < n) { h[i].x = -h[i].x; h[i].y = -h[i].y; } }
__global__ void inv_norm_kernel(int Lt, const double2* nn, double* inv, double* beta) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= Lt) return;
    const double b = sqrt(fmax(nn[t].x, 0.0));
    beta[t] = b; inv[t] = b > 0.0 ? 1.0 / b : 0.0;
}

// w <- B w0 = T_d(L) w0, L = (2A - (a+b))/(b-a), A = -Laplacian; y0, y1, tmp are scratch fields
int chebyshev(Eig& e, double* out, const double* v, int degree, double a, double b, double* y0, double* y1, double* tmp) {
    const double c1 = -2.0 / (b - a), c0 = -(b + a) / (b - a);
    (void)tmp;
    // y1 = L v = c1 Lap v + c0 v  (A = -Lap): the recurrence rides in the Laplacian kernel's epilogue
    LQ_TRY(laplacian_native_axpby(e.c, y1, v, 1, LQ_FP64, c1, c0, 0.0, nullptr)); e.lap_applies++;
    if (degree == 1) { LQ_CUDA(e.c, cudaMemcpyAsync(out, y1, e.fbytes, cudaMemcpyDeviceToDevice, e.c->stream)); return 0; }
    LQ_CUDA(e.c, cudaMemcpyAsync(y0, v, e.fbytes, cudaMemcpyDeviceToDevice, e.c->stream));
    double *prev = y0, *cur = y1;
    for (int n = 1; n < degree; n++) {
        // prev <- 2 L cur - prev
        LQ_TRY(laplacian_native_axpby(e.c, prev, cur, 1, LQ_FP64, 2.0 * c1, 2.0 * c0, -1.0, prev)); e.lap_applies++;
        std::swap(prev, cur);
    }
    LQ_CUDA(e.c, cudaMemcpyAsync(out, cur, e.fbytes, cudaMemcpyDeviceToDevice, e.c->stream));
    LQ_CUDA(e.c, cudaGetLastError());
    return 0;
}

}  // namespace

int laph_eigensolve(lq_ctx* c, double* h_evals, double* dev_canon_evecs, const lq_eig_param* p, lq_eig_info* info) {
    const int Lt = c->g.L[3], n_ev = p->n_ev, m = p->m;
    constexpr int MMAX = 512;
    if (n_ev < 1 || m < n_ev + 2 || m > MMAX || p->cheb_degree < 1 || !(p->cheb_b > p->cheb_a) || !(p->tol > 0) || p->max_restarts < 1)
        return set_err(c, LQ_EINVAL, "lq_laph_eigensolve: bad parameters (need n_ev + 2 <= m <= 512, degree >= 1, cheb_a < cheb_b)");
    const int S3h = c->g.Lxh * c->g.L[1] * c->g.L[2];
    if (n_ev > 6 * S3h - 1) return set_err(c, LQ_EINVAL, "lq_laph_eigensolve: more eigenpairs than the slice dimension");
    Eig e; e.c = c; e.Lt = Lt;
    e.sg.Vh = c->g.Vh; e.sg.S3h = S3h; e.sg.Lt = Lt; e.sg.dS3h = make_fastdiv(S3h);
    e.fbytes = cv_native_bytes(c, 1, LQ_FP64); e.sg.pbe = e.fbytes / 2 / sizeof(double);
    e.nchunk = std::max(1, std::min(64, (2 * S3h + 2047) / 2048));
    const int keep = std::min(m - 2, n_ev + std::max(2, n_ev / 4));      // Ritz vectors kept at a restart

    std::vector<void*> allocs;
    auto alloc = [&](size_t bytes) { void* q = dev_alloc(c, bytes); if (q) allocs.push_back(q); return q; };
    auto cleanup = [&]() { for (void* q : allocs) dev_free(c, q); };
    std::vector<double*> V(m + 1), W(m);
    bool ok = true;
    for (int i = 0; i <= m; i++) { V[i] = (double*)alloc(e.fbytes); ok = ok && V[i]; }
    for (int i = 0; i < keep; i++) { W[i] = (double*)alloc(e.fbytes); ok = ok && W[i]; }
    double* w = (double*)alloc(e.fbytes); double* y0 = (double*)alloc(e.fbytes); double* y1 = (double*)alloc(e.fbytes); double* tmp = (double*)alloc(e.fbytes);
    e.d_partial = (double2*)alloc(sizeof(double2) * Lt * e.nchunk);
    e.d_H = (double2*)alloc(sizeof(double2) * (size_t)(2 * m + 4) * Lt);
    e.d_scale = (double*)alloc(sizeof(double) * 2 * Lt);
    const int nT = (m + 1) & ~1;                                   // leading dimension of the projected matrices (even, for the Jacobi pairing)
    double* d_Q = (double*)alloc(sizeof(double) * (size_t)Lt * m * m);
    double* d_T = (double*)alloc(sizeof(double) * (size_t)Lt * nT * nT);
    double* d_QT = (double*)alloc(sizeof(double) * (size_t)Lt * nT * nT);
    double* d_ritz = (double*)alloc(sizeof(double) * (size_t)Lt * (m + n_ev + 2));      // theta [Lt][m], residual estimates [Lt][n_ev], beta [Lt]
    int* d_sweeps = (int*)alloc(sizeof(int) * Lt);
    double** d_ptr = (double**)alloc(sizeof(double*) * (size_t)(2 * m + 2));
    double2* d_mpart = (double2*)alloc(sizeof(double2) * (size_t)Lt * e.nchunk * (m + 1));
    ok = ok && w && y0 && y1 && tmp && e.d_partial && e.d_H && e.d_scale && d_Q && d_ptr && d_mpart && d_T && d_QT && d_ritz && d_sweeps;
    if (!ok) { cleanup(); return LQ_ENOMEM; }
    const int grid = grid_sites(e);
    cudaEvent_t ev0, ev1, evA, evB;
    cudaEventCreate(&ev0); cudaEventCreate(&ev1); cudaEventCreate(&evA); cudaEventCreate(&evB);
    cudaEventRecord(ev0, c->stream);
    double t_ortho = 0.0, t_ritz = 0.0;

    int rc = 0;
#define EIG_TRY(x) do { rc = (x); if (rc) goto done; } while (0)
#define EIG_CUDA(x) do { if ((x) != cudaSuccess) { rc = set_err(c, LQ_ECUDA, #x); goto done; } } while (0)
    {
    std::vector<double2> hH((size_t)(2 * m + 4) * Lt);
    struct EventList { std::vector<cudaEvent_t> v; ~EventList() { for (cudaEvent_t ev : v) if (ev) cudaEventDestroy(ev); } } evlist;
    evlist.v.assign(2 * (size_t)m, nullptr);                   // per-step event pairs around the orthogonalisation (read after the sweep)
    std::vector<cudaEvent_t>& evs = evlist.v;
    for (auto& ev : evs) EIG_CUDA(cudaEventCreate(&ev));
    EIG_CUDA(cudaMemsetAsync(d_T, 0, sizeof(double) * (size_t)Lt * nT * nT, c->stream));
    std::vector<double> theta((size_t)Lt * m), hres((size_t)Lt * n_ev);
    double* d_theta = d_ritz; double* d_res = d_ritz + (size_t)Lt * m; double* d_beta = d_res + (size_t)Lt * n_ev;
    int k = 0, restarts = 0; bool converged = false; double worst = 0.0;
    // v_0: pseudo-random, normalised on every slice; zero the padding first
    EIG_CUDA(cudaMemsetAsync(V[0], 0, e.fbytes, c->stream));
    for (int i = 1; i <= m; i++) EIG_CUDA(cudaMemsetAsync(V[i], 0, e.fbytes, c->stream));
    EIG_CUDA(cudaMemsetAsync(w, 0, e.fbytes, c->stream)); EIG_CUDA(cudaMemsetAsync(y0, 0, e.fbytes, c->stream));
    EIG_CUDA(cudaMemsetAsync(y1, 0, e.fbytes, c->stream)); EIG_CUDA(cudaMemsetAsync(tmp, 0, e.fbytes, c->stream));
    for (int i = 0; i < keep; i++) EIG_CUDA(cudaMemsetAsync(W[i], 0, e.fbytes, c->stream));
    EIG_TRY(cv_fill(c, tmp, 1, LQ_FP64, 0x5EEDull + p->seed));
    {   // copy only real sites (padding stays zero): scale by 1 through the slice kernel
        std::vector<double> ones(Lt, 1.0);
        EIG_CUDA(cudaMemcpyAsync(e.d_scale, ones.data(), sizeof(double) * Lt, cudaMemcpyHostToDevice, c->stream));
        slice_scale_kernel<<<grid, 128, 0, c->stream>>>(e.sg, V[0], tmp, e.d_scale); c->launches++;
        EIG_CUDA(cudaStreamSynchronize(c->stream));
    }
    EIG_TRY(dot(e, V[0], V[0], e.d_H));
    inv_norm_kernel<<<(Lt + 63) / 64, 64, 0, c->stream>>>(Lt, e.d_H, e.d_scale, e.d_scale + Lt);
    slice_scale_kernel<<<grid, 128, 0, c->stream>>>(e.sg, V[0], V[0], e.d_scale); c->launches += 2;

    for (restarts = 0; restarts < p->max_restarts; restarts++) {
        {   // device table of the basis vectors (changes at every restart)
            std::vector<double*> ptrs(V.begin(), V.end());
            EIG_CUDA(cudaMemcpyAsync(d_ptr, ptrs.data(), sizeof(double*) * (size_t)(m + 1), cudaMemcpyHostToDevice, c->stream));
            EIG_CUDA(cudaStreamSynchronize(c->stream));
        }
        for (int j = k; j < m; j++) {
            EIG_TRY(chebyshev(e, w, V[j], p->cheb_degree, p->cheb_a, p->cheb_b, y0, y1, tmp));
            // two classical Gram-Schmidt passes against v_0 .. v_j; the coefficients are the column j of T
            cudaEventRecord(evs[2 * (size_t)j], c->stream);
            // pass 0 is LOCAL: against v_{j-1}, v_j only (the three-term recurrence carries all of the weight there), except on the
            // first step after a restart, where the arrow couples w to every kept Ritz vector; pass 1 is the full reorthogonalisation
            // against v_0 .. v_j.  After pass 0 the components left along the older vectors are rounding-level, so one full classical
            // Gram-Schmidt pass restores orthogonality to working precision at half the basis traffic of two full passes.
            // Nothing of a step goes through the host: the coefficients stay in d_H and t_column_kernel / t_beta_kernel write
            // column j of the projected matrices, so the whole sweep is enqueued without a synchronisation.
            for (int pass = 0; pass < 2; pass++) {
                const int first = (pass == 0 && j > k) ? j - 1 : 0;
                const int nv = j + 1 - first;
                double2* H = e.d_H + (size_t)pass * (m + 1) * Lt + (size_t)first * Lt;
                slice_multidot_kernel<<<dim3(Lt * e.nchunk, (nv + 7) / 8), 256, 0, c->stream>>>(e.sg, e.nchunk, nv, d_ptr + first, w, d_mpart);
                slice_multidot_final_kernel<<<(Lt * nv + 127) / 128, 128, 0, c->stream>>>(Lt, e.nchunk, nv, d_mpart, H);
                slice_multiaxpy_kernel<<<grid, 128, 0, c->stream>>>(e.sg, nv, w, d_ptr + first, H);
                c->launches += 3;
            }
            t_column_kernel<<<(Lt * (j + 1) + 127) / 128, 128, 0, c->stream>>>(Lt, nT, j, k, j > k ? j - 1 : 0, e.d_H, e.d_H + (size_t)(m + 1) * Lt, d_T);
            EIG_TRY(dot(e, w, w, e.d_H + (size_t)(2 * m + 2) * Lt));
            inv_norm_kernel<<<(Lt + 63) / 64, 64, 0, c->stream>>>(Lt, e.d_H + (size_t)(2 * m + 2) * Lt, e.d_scale, e.d_scale + Lt);
            slice_scale_kernel<<<grid, 128, 0, c->stream>>>(e.sg, V[j + 1], w, e.d_scale);
            t_beta_kernel<<<(Lt + 63) / 64, 64, 0, c->stream>>>(Lt, nT, j, m, e.d_scale + Lt, d_T, d_beta); c->launches += 4;
            cudaEventRecord(evs[2 * (size_t)j + 1], c->stream);
            EIG_CUDA(cudaGetLastError());
        }
        const int k_sweep = k;
        // Ritz pairs of every slice
        cudaEventRecord(evA, c->stream);
        worst = 0.0; converged = true;
        // all Lt projected eigenproblems in one launch; the kernel leaves the sorted eigenvalues, the residual estimates and the
        // first `keep` eigenvectors (d_Q, the layout slice_rotate_kernel reads) on the device
        ritz_jacobi_kernel<<<Lt * RITZ_CLUSTER, RITZ_THREADS, 0, c->stream>>>(m, keep, n_ev, d_T, d_QT, d_beta, d_theta, d_Q, d_res, d_sweeps); c->launches++;
        EIG_CUDA(cudaGetLastError());
        EIG_CUDA(cudaMemcpyAsync(theta.data(), d_theta, sizeof(double) * (size_t)Lt * m, cudaMemcpyDeviceToHost, c->stream));
        EIG_CUDA(cudaMemcpyAsync(hres.data(), d_res, sizeof(double) * (size_t)Lt * n_ev, cudaMemcpyDeviceToHost, c->stream));
        EIG_CUDA(cudaStreamSynchronize(c->stream));
        for (int jj = k_sweep; jj < m; jj++) { float tms = 0; cudaEventElapsedTime(&tms, evs[2 * (size_t)jj], evs[2 * (size_t)jj + 1]); t_ortho += tms * 1e-3; }
        for (int t = 0; t < Lt; t++)
            for (int cidx = 0; cidx < n_ev; cidx++) {
                const double rel = hres[(size_t)t * n_ev + cidx];
                worst = fmax(worst, rel);
                if (!(rel <= p->tol)) converged = false;
            }
        // thick restart: V[0..keep) <- V Q[:, 0..keep), V[keep] <- v_m, T <- diag(theta) (the arrow is rebuilt by the sweep)
        {
            std::vector<double*> ptrs(2 * m + 2);
            for (int i = 0; i < m; i++) ptrs[i] = V[i];
            for (int i = 0; i < keep; i++) ptrs[m + i] = W[i];
            EIG_CUDA(cudaMemcpyAsync(d_ptr, ptrs.data(), sizeof(double*) * (size_t)(2 * m + 2), cudaMemcpyHostToDevice, c->stream));
            slice_rotate_kernel<<<grid, 128, 0, c->stream>>>(e.sg, m, keep, d_ptr, d_ptr + m, d_Q); c->launches++;
            EIG_CUDA(cudaStreamSynchronize(c->stream));
            for (int i = 0; i < keep; i++) std::swap(V[i], W[i]);
            std::swap(V[keep], V[m]);
        }
        cudaEventRecord(evB, c->stream);
        EIG_CUDA(cudaEventSynchronize(evB));
        { float tms = 0; cudaEventElapsedTime(&tms, evA, evB); t_ritz += tms * 1e-3; }
        t_reset_kernel<<<(int)(((long long)Lt * nT * nT + 255) / 256), 256, 0, c->stream>>>(Lt, nT, keep, m, d_theta, d_T); c->launches++;
        k = keep;
        if (converged) { restarts++; break; }
    }
    // eigenvalues of A = -Laplacian as Rayleigh quotients, true residuals, canonical eigenvectors
    double maxres = 0.0;
    for (int i = 0; i < n_ev; i++) {
        EIG_TRY(laplacian_native(c, tmp, V[i], 1, LQ_FP64)); e.lap_applies++;
        EIG_TRY(dot(e, V[i], tmp, e.d_H));
        EIG_CUDA(cudaMemcpyAsync(hH.data(), e.d_H, sizeof(double2) * Lt, cudaMemcpyDeviceToHost, c->stream));
        EIG_CUDA(cudaStreamSynchronize(c->stream));
        std::vector<double2> lam(Lt);
        for (int t = 0; t < Lt; t++) { h_evals[(size_t)t * n_ev + i] = -hH[t].x; lam[t] = make_double2(-hH[t].x, 0.0); }
        // r = A v - lambda v = -(tmp) - lambda v  ->  tmp += lambda v ; ||tmp||
        EIG_CUDA(cudaMemcpyAsync(e.d_H, lam.data(), sizeof(double2) * Lt, cudaMemcpyHostToDevice, c->stream));
        slice_axpy_kernel<<<grid, 128, 0, c->stream>>>(e.sg, tmp, V[i], e.d_H); c->launches++;
        EIG_TRY(dot(e, tmp, tmp, e.d_H + Lt));
        EIG_CUDA(cudaMemcpyAsync(hH.data(), e.d_H + Lt, sizeof(double2) * Lt, cudaMemcpyDeviceToHost, c->stream));
        EIG_CUDA(cudaStreamSynchronize(c->stream));
        for (int t = 0; t < Lt; t++) maxres = fmax(maxres, sqrt(fmax(hH[t].x, 0.0)));
        if (dev_canon_evecs) EIG_TRY(cv_unpack(c, dev_canon_evecs + (size_t)i * c->g.V * 6, V[i], 1, LQ_FP64));
    }
    cudaEventRecord(ev1, c->stream);
    EIG_CUDA(cudaEventSynchronize(ev1));
    float ms = 0; cudaEventElapsedTime(&ms, ev0, ev1);
    info->restarts = restarts; info->converged = converged ? 1 : 0; info->lap_applies = (double)e.lap_applies;
    info->max_ritz_residual = worst; info->max_true_residual = maxres; info->seconds = ms * 1e-3;
    info->seconds_ritz = t_ritz; info->seconds_ortho = t_ortho;
    if (!converged) rc = LQ_ENOTCONVERGED;
    }
done:
    cudaStreamSynchronize(c->stream);
    cudaEventDestroy(ev0); cudaEventDestroy(ev1); cudaEventDestroy(evA); cudaEventDestroy(evB);
    cleanup();
    return rc;
#undef EIG_TRY
#undef EIG_CUDA
}
