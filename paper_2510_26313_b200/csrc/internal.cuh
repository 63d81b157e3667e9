// internal.cuh -- cross-file declarations of the CUDA path (not part of the C ABI).
#pragma once
#include "common.cuh"
#include "dslash.cuh"

// dslash_*.cu
template <class S, int RECON, int FORM>
int launch_dslash(lq_ctx* c, DslashArgs<S> a, int rpt, int variant);

// ops.cu : typed single-parity building blocks on native fields
// out(parity) = [C] D in(1-parity) ; form A uses A^{-1}, form HOP nothing
int op_hop(lq_ctx* c, int prec, int nrhs, int out_parity, void* out, const void* in, int dagger);
int op_kernel_a(lq_ctx* c, int prec, int nrhs, int out_parity, void* out, const void* in, int dagger);
// bench only: kernel A's memory accesses with trivial arithmetic (fp32 / half storage, 18-real links)
int op_probe_loads(lq_ctx* c, int prec, int nrhs, int out_parity, void* out, const void* in);
// out(parity) = C x + coef D in ; use_clover: 1 -> A(parity), 0 -> identity
int op_kernel_b(lq_ctx* c, int prec, int nrhs, int out_parity, void* out, const void* x, const void* in, double coef, int use_clover, int dagger);
// kernel B with a fused block-BLAS epilogue: EPI_NORM: epi_out[k] = ||out_k||^2 ; EPI_XMAY: out_k <- out_k - (num_k/den_k) (C x + coef D in)_k
// and epi_out[k] = ||out_k||^2 (out is read and written)
int op_kernel_b_epi(lq_ctx* c, int prec, int nrhs, int out_parity, void* out, const void* x, const void* in, double coef, int use_clover, int dagger,
                    int epi, const double* num, const double* den, double* epi_out);
int op_kernel_b_cdot(lq_ctx* c, int prec, int nrhs, int out_parity, void* out, const void* x, const void* in, double coef, int use_clover, int dagger,
                     const void* h, int conj, double* epi_out);
// out(parity) = A x or A^{-1} x (site-local)
int op_clover(lq_ctx* c, int prec, int nrhs, int parity, void* out, const void* x, int inverse);

// reorder.cu
int gauge_ingest(lq_ctx* c, const void* dev_canonical, int in_prec);            // canonical (device) -> native fp64
int gauge_make_fp32(lq_ctx* c, int recon);
int gauge_make_int16(lq_ctx* c);                                                  // native fp64 -> int16 fixed point (18 reals), for H16L                                       // native fp64 -> native fp32 (18 or 12)
int spinor_pack(lq_ctx* c, void* native_full, const void* dev_canonical, int nrhs, int prec, int in_prec);
int spinor_unpack(lq_ctx* c, void* dev_canonical, const void* native_full, int nrhs, int prec, int out_prec);
// the same for right-hand sides k0 .. k0+nk-1 only: dev_canonical holds just those nk fields (host buffers are staged in such chunks)
int spinor_pack_part(lq_ctx* c, void* native_full, const void* dev_canonical, int nrhs, int k0, int nk, int prec, int in_prec);
int spinor_unpack_part(lq_ctx* c, void* dev_canonical, const void* native_full, int nrhs, int k0, int nk, int prec, int out_prec);
int spinor_convert(lq_ctx* c, void* dst, int dst_prec, const void* src, int src_prec, int nrhs, const double* d_scale /*per rhs, multiplies*/, int invert_scale);
int spinor_zero_parity(lq_ctx* c, void* parity_block, int nrhs, int prec);
int spinor_gather_sites(lq_ctx* c, double* dev_out, const void* parity_block, int nrhs, int prec, long long nsites, const int* dev_sites);
int canonical_zero_parity(lq_ctx* c, void* dev_canonical, int nrhs, int prec, int parity);

// clover.cu
int clover_build(lq_ctx* c, double kappa, double csw);

// blas.cu : per-RHS block BLAS on one parity block; results stay on the device
int blas_norm2(lq_ctx* c, int prec, int nrhs, const void* x, double* d_out);                       // d_out[k] = ||x_k||^2
// y (fp64) += s_k * e (prec)       (defect-correction accumulate)
// fused CG vector update: alpha_k = rr_k / pAp_k, beta_k = rr_new_k / rr_k;  e += alpha p;  p = z + beta p
int blas_cg_update_ep(lq_ctx* c, int prec, int nrhs, void* e, void* p, const void* z, const double* d_rr, const double* d_pAp, const double* d_rr_new);
// reliable update of the search direction: p_k <- z_new_k + c_k (p_k - z_old_k), then z_old <- z_new; c per RHS on the device
int blas_keep_direction(lq_ctx* c, int prec, int nrhs, void* p, void* z_old, const void* z_new, const double* d_c);
int blas_axpy_mixed(lq_ctx* c, int prec, int nrhs, void* y64, const void* e, const double* d_scale);
// r = b - t (fp64), d_out[k] = ||r_k||^2
int blas_residual(lq_ctx* c, int nrhs, void* r, const void* b, const void* t, double* d_out);
int blas_copy(lq_ctx* c, int prec, int nrhs, void* dst, const void* src);
// batched BiCGStab (complex per-RHS scalars kept as raw sums on the device; d_out = 3 x LQ_MAX_RHS doubles)
int blas_cdot3(lq_ctx* c, int prec, int nrhs, const void* a, const void* b, double* d_out);        // Re <a,b>, Im <a,b>, ||a||^2
int blas_bicg_s(lq_ctx* c, int prec, int nrhs, void* s, const void* r, const void* v, const double* d_rho, const double* d_c1);
int blas_bicg_xr(lq_ctx* c, int prec, int nrhs, void* e, void* r, const void* p, const void* s, const void* t, const void* rhat,
                 const double* d_rho, const double* d_c1, const double* d_d2, double* d_out);       // -> Re, Im <rhat,r>, ||r||^2
int blas_bicg_p(lq_ctx* c, int prec, int nrhs, void* p, const void* r, const void* v, const double* d_rho, const double* d_rho_new,
                const double* d_c1, const double* d_d2);

// fill.cu
int fill_gauge(lq_ctx* c, uint64_t seed, double eps);
int fill_spinor(lq_ctx* c, void* native, int nrhs, int prec, uint64_t seed, int parity_only, int parity);

// fmapeak.cu
int fma_peak(lq_ctx* c, int mode, double ms, double* tflops);
int mem_peak(lq_ctx* c, int mode, double mbytes, double* gbs);

// solver.cu
void solver_release(lq_ctx* c);
int mhat_native(lq_ctx* c, int prec, int n, void* out_e, const void* in_e, int dagger);
int solve_native(lq_ctx* c, void* x_full64, const void* b_full64, int nrhs, const lq_solve_param* p, lq_solve_info* info);

// laplace.cu : batched 3-d gauge-covariant Laplacian on native colour-vector fields
int laplacian_native(lq_ctx* c, void* out, const void* in, int nvec, int prec);
// out = ca * Lap(in) + cb * in + cc * y, y = nullptr or any field (may be `out`); out must not alias in
int laplacian_native_axpby(lq_ctx* c, void* out, const void* in, int nvec, int prec, double ca, double cb, double cc, const void* y);
size_t cv_native_bytes(const lq_ctx* c, int nvec, int prec);
int cv_pack(lq_ctx* c, void* native, const double* dev_canon, int nvec, int prec);
int cv_unpack(lq_ctx* c, double* dev_canon, const void* native, int nvec, int prec);
int cv_fill(lq_ctx* c, void* native, int nvec, int prec, unsigned long long seed);

// eigen.cu : time-batched thick-restart Lanczos on the Chebyshev-filtered -Laplacian
int laph_eigensolve(lq_ctx* c, double* h_evals, double* dev_canon_evecs, const lq_eig_param* p, lq_eig_info* info);

// project.cu : projection of solutions onto LapH eigenvectors
int project_device(lq_ctx* c, double* dev_P, const double* dev_V, int n_ev, const double* dev_X, int n_sol);
// project_tc.cu : the same contraction on tcgen05 tensor cores (3xTF32, fp32 TMEM accumulator, fp64 split-K sum)
int project_device_tc(lq_ctx* c, double* dev_P, const double* dev_V, int n_ev, const double* dev_X, int n_sol);
// project_tc32.cu : the tensor-core kernel for complex-float fields (two operand buffers: conversion overlaps the MMAs)
int project_device_tc32(lq_ctx* c, double* dev_P, const float* dev_V, int n_ev, const float* dev_X, int n_sol);

// multigrid.cu : two-level adaptive multigrid; canonical / coarse arrays below are DEVICE arrays
void mg_release(lq_ctx* c);
void mg_invalidate(lq_ctx* c);
int mg_setup_vectors(lq_ctx* c, const lq_mg_param* p, const void* dev_canonical64, lq_mg_info* info);
int mg_setup_adaptive(lq_ctx* c, const lq_mg_param* p, lq_mg_info* info);
size_t mg_coarse_canonical_bytes(const lq_ctx* c, int n);
int mg_restrict_dev(lq_ctx* c, double* coarse64, const void* fine_canonical64, int n);
int mg_prolong_dev(lq_ctx* c, void* fine_canonical64, const double* coarse64, int n);
int mg_coarse_apply_dev(lq_ctx* c, double* out64, const double* in64, int n);
int mg_vcycle_dev(lq_ctx* c, void* z_canonical64, const void* r_canonical64, int n);
int mg_solve_native(lq_ctx* c, void* x64, const void* b64, int n, double tol, int max_iter, lq_mg_solve_info* info);
