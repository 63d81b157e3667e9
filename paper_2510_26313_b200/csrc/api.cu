// api.cu -- the C ABI of include/lqcd_b200.h: context, ingest, apply, pack/unpack, solve.
#include <algorithm>
#include <string.h>
#include "internal.cuh"


int set_err(lq_ctx* c, int code, const std::string& msg) {
    if (c) c->err = msg;
    return code;
}
void* dev_alloc(lq_ctx* c, size_t bytes) {
    void* p = nullptr;
    if (bytes == 0) bytes = 256;
    if (c->alloc_fn) p = c->alloc_fn(bytes, c->alloc_user);
    else if (cudaMalloc(&p, bytes) != cudaSuccess) { cudaGetLastError(); p = nullptr; }
    if (!p) { set_err(c, LQ_ENOMEM, "device allocation of " + std::to_string(bytes) + " bytes failed"); return nullptr; }
    c->owned.push_back(p);
    return p;
}
void dev_free(lq_ctx* c, void* p) {
    if (!p) return;
    auto it = std::find(c->owned.begin(), c->owned.end(), p);
    if (it != c->owned.end()) c->owned.erase(it);
    if (c->free_fn) c->free_fn(p, c->alloc_user);
    else if (!c->alloc_fn) cudaFree(p);
}

int ensure_partials(lq_ctx* c, size_t elems) {
    if (elems + 256 * 3 * LQ_MAX_RHS <= c->red_partials_elems) return 0;
    if (c->red_partials) dev_free(c, c->red_partials);
    c->red_partials_elems = elems + elems / 8 + 256 * 3 * LQ_MAX_RHS;   // the block rows and the rows of the second stage (reduce.cuh)
    c->red_partials = (double*)dev_alloc(c, c->red_partials_elems * sizeof(double));
    if (!c->red_partials) { c->red_partials_elems = 0; return LQ_ENOMEM; }
    return 0;
}
static bool nrhs_ok(int n) { return n == 1 || n == 2 || (n >= 4 && n <= LQ_MAX_RHS && n % 4 == 0); }

extern "C" {

int lq_create(lq_ctx** out, const int dims[4], int device, void* cuda_stream) {
    if (!out || !dims) return LQ_EINVAL;
    *out = nullptr;
    for (int k = 0; k < 4; k++) if (dims[k] < 2 || (dims[k] & 1)) return LQ_EINVAL;
    const long long V = (long long)dims[0] * dims[1] * dims[2] * dims[3];
    if (V / 2 * LQ_MAX_RHS >= (1LL << 31)) return LQ_EINVAL;
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return LQ_ECUDA; }
    lq_ctx* c = new lq_ctx();
    for (int k = 0; k < 4; k++) c->g.L[k] = dims[k];
    c->g.Lxh = dims[0] / 2; c->g.V = V; c->g.Vh = (int)(V / 2); c->g.NB = (c->g.Vh + SB - 1) / SB;
    c->g.dLxh = make_fastdiv(c->g.Lxh); c->g.dLy = make_fastdiv(dims[1]); c->g.dLz = make_fastdiv(dims[2]);
    c->device = device; c->stream = (cudaStream_t)cuda_stream; c->t_bc = -1;
    c->gauge64 = nullptr; c->gauge32 = nullptr; c->recon32 = 18; c->gauge16 = nullptr; c->half_links = false;
    c->clov64 = c->clovinv64 = nullptr; c->clov32 = c->clovinv32 = nullptr;
    c->kappa = c->csw = 0; c->has_gauge = c->has_clover = false;
    c->alloc_fn = nullptr; c->free_fn = nullptr; c->alloc_user = nullptr;
    c->launches = 0; c->dslash_rpt = 0; c->dslash_variant = 0; c->dslash_pfd = LQ_DEFAULT_PFD; c->dslash_zc = 0;
    c->red_partials = nullptr; c->red_partials_elems = 0; c->red_counter = nullptr; c->h_scalars = nullptr; c->d_flag = nullptr;
    c->ws = nullptr; c->mg = nullptr; c->loop_skip = nullptr; c->model_bytes = c->model_flops = 0.0; c->proj_scratch = nullptr; c->proj_scratch_bytes = 0;
    if (cudaMalloc(&c->red_counter, RED_COUNTER_BYTES) != cudaSuccess || cudaMemset(c->red_counter, 0, RED_COUNTER_BYTES) != cudaSuccess ||
        cudaMallocHost(&c->h_scalars, 8 * LQ_MAX_RHS * sizeof(double)) != cudaSuccess) { cudaGetLastError(); delete c; return LQ_ECUDA; }
    c->d_flag = (int*)(c->red_counter + 16);
    *out = c;
    return 0;
}

int lq_destroy(lq_ctx* c) {
    if (!c) return LQ_EINVAL;
    cudaSetDevice(c->device);
    cudaStreamSynchronize(c->stream);
    solver_release(c);
    mg_release(c);
    std::vector<void*> owned = c->owned;
    for (void* p : owned) dev_free(c, p);
    cudaFree(c->red_counter);
    cudaFreeHost(c->h_scalars);
    delete c;
    return 0;
}

const char* lq_last_error(const lq_ctx* c) { return c ? c->err.c_str() : "null context"; }

int lq_set_allocator(lq_ctx* c, lq_alloc_fn alloc, lq_free_fn release, void* user) {
    if (!c) return LQ_EINVAL;
    if (!c->owned.empty()) return set_err(c, LQ_ESTATE, "allocator must be installed before the first allocation");
    c->alloc_fn = alloc; c->free_fn = release; c->alloc_user = user;
    return 0;
}

int lq_set_tuning(lq_ctx* c, int dslash_variant, int dslash_rpt, int dslash_pfd) {
    if (!c) return LQ_EINVAL;
    c->dslash_zc = (dslash_variant >> 8) == 0xFF ? -1 : (dslash_variant >> 8);     // bits 8.. : z-chunk (0 auto, 0xFF memory order)
    dslash_variant &= 0xFF;
    c->dslash_variant = dslash_variant; c->dslash_rpt = dslash_rpt; c->dslash_pfd = dslash_pfd < 0 ? LQ_DEFAULT_PFD : dslash_pfd;
    return 0;
}

long long lq_kernel_launches(const lq_ctx* c) { return c ? c->launches : 0; }

static int ensure_gauge_storage(lq_ctx* c, int recon) {
    if (recon != 18 && recon != 12) return set_err(c, LQ_EINVAL, "recon must be 18 or 12");
    if (!c->gauge64) { c->gauge64 = (double*)dev_alloc(c, (size_t)8 * 18 * c->g.NB * SB * sizeof(double)); if (!c->gauge64) return LQ_ENOMEM; }
    if (!c->gauge32) { c->gauge32 = (float*)dev_alloc(c, (size_t)8 * 18 * c->g.NB * SB * sizeof(float)); if (!c->gauge32) return LQ_ENOMEM; }
    return 0;
}

int lq_load_gauge(lq_ctx* c, const void* links, int in_prec, int loc, int recon, int t_bc) {
    if (!c || !links) return LQ_EINVAL;
    if (in_prec != LQ_FP64 && in_prec != LQ_FP32) return set_err(c, LQ_EINVAL, "gauge precision must be fp64 or fp32");
    if (t_bc != 1 && t_bc != -1) return set_err(c, LQ_EINVAL, "t_bc must be +1 or -1");
    cudaSetDevice(c->device);
    LQ_TRY(ensure_gauge_storage(c, recon));
    const size_t bytes = (size_t)4 * c->g.V * 18 * elem_bytes(in_prec);
    const void* dev = links;
    void* staging = nullptr;
    if (loc == LQ_HOST) {
        staging = dev_alloc(c, bytes);
        if (!staging) return LQ_ENOMEM;
        LQ_CUDA(c, cudaMemcpyAsync(staging, links, bytes, cudaMemcpyHostToDevice, c->stream));
        dev = staging;
    }
    int rc = gauge_ingest(c, dev, in_prec);
    if (rc == 0) rc = gauge_make_fp32(c, recon);
    if (rc == 0 && c->half_links) rc = gauge_make_int16(c);
    if (rc == 0 && cudaStreamSynchronize(c->stream) != cudaSuccess) rc = set_err(c, LQ_ECUDA, "gauge ingest failed");
    if (staging) dev_free(c, staging);
    if (rc) return rc;
    c->t_bc = t_bc; c->has_gauge = true; c->has_clover = false;
    mg_invalidate(c);
    return 0;
}

int lq_fill_gauge_random(lq_ctx* c, uint64_t seed, double eps, int recon, int t_bc) {
    if (!c) return LQ_EINVAL;
    if (t_bc != 1 && t_bc != -1) return set_err(c, LQ_EINVAL, "t_bc must be +1 or -1");
    cudaSetDevice(c->device);
    LQ_TRY(ensure_gauge_storage(c, recon));
    LQ_TRY(fill_gauge(c, seed, eps));
    LQ_TRY(gauge_make_fp32(c, recon));
    if (c->half_links) LQ_TRY(gauge_make_int16(c));
    LQ_CUDA(c, cudaStreamSynchronize(c->stream));
    c->t_bc = t_bc; c->has_gauge = true; c->has_clover = false;
    mg_invalidate(c);
    return 0;
}

int lq_set_half_links(lq_ctx* c, int enable) {
    if (!c) return LQ_EINVAL;
    cudaSetDevice(c->device);
    if (enable) {
        if (!c->has_gauge) return set_err(c, LQ_ESTATE, "load the gauge field before lq_set_half_links");
        LQ_TRY(gauge_make_int16(c));
        LQ_CUDA(c, cudaStreamSynchronize(c->stream));
    }
    c->half_links = enable != 0;
    return 0;
}

int lq_build_clover(lq_ctx* c, double kappa, double csw) {
    if (!c) return LQ_EINVAL;
    if (!c->has_gauge) return set_err(c, LQ_ESTATE, "load the gauge field before building the clover term");
    cudaSetDevice(c->device);
    mg_invalidate(c);
    return clover_build(c, kappa, csw);
}

size_t lq_native_bytes(const lq_ctx* c, int nrhs, int prec, int parity_only) {
    if (!c || nrhs < 1) return 0;
    return parity_bytes(c->g, nrhs, prec) * (parity_only ? 1 : 2);
}

// stage a canonical array on the device if it lives on the host; returns the device pointer (or nullptr on failure)
static const void* stage_in(lq_ctx* c, const void* p, size_t bytes, int loc, void** staging) {
    *staging = nullptr;
    if (loc == LQ_DEVICE) return p;
    *staging = dev_alloc(c, bytes);
    if (!*staging) return nullptr;
    if (cudaMemcpyAsync(*staging, p, bytes, cudaMemcpyHostToDevice, c->stream) != cudaSuccess) { set_err(c, LQ_ECUDA, "H2D copy failed"); return nullptr; }
    return *staging;
}

// Host canonical arrays are staged through ONE device buffer of at most ~2 GiB, a few right-hand sides at a time: the device
// never holds a canonical copy of the whole batch (configs[3]: 24.5 GB per field).  nk = right-hand sides per chunk.
static int chunk_rhs(const lq_ctx* c, int nrhs) {
    const size_t per = (size_t)c->g.V * 24 * sizeof(double);
    size_t nk = ((size_t)2 << 30) / per;
    if (nk < 1) nk = 1;
    return nk > (size_t)nrhs ? nrhs : (int)nk;
}
// canonical complex double (host or device) -> native full-lattice batch
static int pack_any(lq_ctx* c, void* native_out, const void* canonical_in, int nrhs, int prec, int loc) {
    if (loc == LQ_DEVICE) return spinor_pack(c, native_out, canonical_in, nrhs, prec, LQ_FP64);
    const size_t per = (size_t)c->g.V * 24 * sizeof(double);
    const int nk = chunk_rhs(c, nrhs);
    void* st = dev_alloc(c, per * nk);
    if (!st) return LQ_ENOMEM;
    int rc = 0;
    for (int k0 = 0; k0 < nrhs && rc == 0; k0 += nk) {
        const int m = nrhs - k0 < nk ? nrhs - k0 : nk;
        if (cudaMemcpyAsync(st, (const char*)canonical_in + per * k0, per * m, cudaMemcpyHostToDevice, c->stream) != cudaSuccess) rc = set_err(c, LQ_ECUDA, "H2D copy failed");
        if (rc == 0) rc = spinor_pack_part(c, native_out, st, nrhs, k0, m, prec, LQ_FP64);
    }
    if (cudaStreamSynchronize(c->stream) != cudaSuccess && rc == 0) rc = set_err(c, LQ_ECUDA, "pack failed");
    dev_free(c, st);
    return rc;
}
static int unpack_any(lq_ctx* c, void* canonical_out, const void* native_in, int nrhs, int prec, int loc) {
    if (loc == LQ_DEVICE) return spinor_unpack(c, canonical_out, native_in, nrhs, prec, LQ_FP64);
    const size_t per = (size_t)c->g.V * 24 * sizeof(double);
    const int nk = chunk_rhs(c, nrhs);
    void* st = dev_alloc(c, per * nk);
    if (!st) return LQ_ENOMEM;
    int rc = 0;
    for (int k0 = 0; k0 < nrhs && rc == 0; k0 += nk) {
        const int m = nrhs - k0 < nk ? nrhs - k0 : nk;
        rc = spinor_unpack_part(c, st, native_in, nrhs, k0, m, prec, LQ_FP64);
        if (rc == 0 && cudaMemcpyAsync((char*)canonical_out + per * k0, st, per * m, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) rc = set_err(c, LQ_ECUDA, "D2H copy failed");
    }
    if (cudaStreamSynchronize(c->stream) != cudaSuccess && rc == 0) rc = set_err(c, LQ_ECUDA, "unpack failed");
    dev_free(c, st);
    return rc;
}

int lq_pack(lq_ctx* c, void* native_out, const void* canonical_in, int nrhs, int prec, int loc) {
    if (!c || !native_out || !canonical_in || !nrhs_ok(nrhs)) return set_err(c, LQ_EINVAL, "lq_pack: bad argument");
    cudaSetDevice(c->device);
    int rc = pack_any(c, native_out, canonical_in, nrhs, prec, loc);
    if (rc == 0 && cudaStreamSynchronize(c->stream) != cudaSuccess) rc = set_err(c, LQ_ECUDA, "pack failed");
    return rc;
}
int lq_unpack(lq_ctx* c, void* canonical_out, const void* native_in, int nrhs, int prec, int loc) {
    if (!c || !canonical_out || !native_in || !nrhs_ok(nrhs)) return set_err(c, LQ_EINVAL, "lq_unpack: bad argument");
    cudaSetDevice(c->device);
    int rc = unpack_any(c, canonical_out, native_in, nrhs, prec, loc);
    if (rc == 0 && cudaStreamSynchronize(c->stream) != cudaSuccess) rc = set_err(c, LQ_ECUDA, "unpack failed");
    return rc;
}

int lq_native_index(const lq_ctx* c, int nrhs, int prec, int x, int y, int z, int t, int rhs, int j,
                    size_t* elem_offset, size_t* norm_offset, size_t* parity_block_byte, size_t* norm_array_byte) {
    if (!c || !nrhs_ok(nrhs) || rhs < 0 || rhs >= nrhs || j < 0 || j >= 24 || (prec != LQ_FP64 && prec != LQ_FP32 && prec != LQ_HALF)) return LQ_EINVAL;
    const int xs[4] = {x, y, z, t};
    for (int k = 0; k < 4; k++) if (xs[k] < 0 || xs[k] >= c->g.L[k]) return LQ_EINVAL;
    int parity, cb;
    coords_to_cb(c->g, x, y, z, t, parity, cb);
    if (elem_offset) *elem_offset = sp_index(nrhs, cb, rhs, j);
    if (norm_offset) *norm_offset = prec == LQ_HALF ? nrm_index(nrhs, cb, rhs) : 0;
    if (parity_block_byte) *parity_block_byte = (size_t)parity * parity_bytes(c->g, nrhs, prec);
    if (norm_array_byte) *norm_array_byte = prec == LQ_HALF ? round256((size_t)24 * c->g.NB * SB * nrhs * elem_bytes(prec)) : 0;
    return 0;
}

int lq_mem_peak(lq_ctx* c, int mode, double mbytes, double* gbs) {
    if (!c || !gbs || mode < 0 || mode > 1 || !(mbytes > 0)) return set_err(c, LQ_EINVAL, "lq_mem_peak: bad argument");
    cudaSetDevice(c->device);
    return mem_peak(c, mode, mbytes, gbs);
}

int lq_fma_peak(lq_ctx* c, int mode, double ms, double* tflops) {
    if (!c || !tflops || mode < 0 || mode > 3 || !(ms > 0)) return set_err(c, LQ_EINVAL, "lq_fma_peak: bad argument");
    cudaSetDevice(c->device);
    return fma_peak(c, mode, ms, tflops);
}

int lq_fill_spinor_random(lq_ctx* c, void* native_out, int nrhs, int prec, uint64_t seed, int parity_only, int parity) {
    if (!c || !native_out || !nrhs_ok(nrhs)) return set_err(c, LQ_EINVAL, "lq_fill_spinor_random: bad argument");
    cudaSetDevice(c->device);
    return fill_spinor(c, native_out, nrhs, prec, seed, parity_only, parity);
}

int lq_gather_sites(lq_ctx* c, double* out, const void* native_parity_block, int nrhs, int prec, long long nsites, const int* sites_xyzt) {
    if (!c || !out || !native_parity_block || !sites_xyzt || !nrhs_ok(nrhs) || nsites < 1) return set_err(c, LQ_EINVAL, "lq_gather_sites: bad argument");
    if (prec != LQ_FP64 && prec != LQ_FP32 && prec != LQ_HALF) return set_err(c, LQ_EINVAL, "bad precision");
    for (long long n = 0; n < nsites; n++)
        for (int k = 0; k < 4; k++) if (sites_xyzt[4 * n + k] < 0 || sites_xyzt[4 * n + k] >= c->g.L[k]) return set_err(c, LQ_EINVAL, "lq_gather_sites: site out of range");
    cudaSetDevice(c->device);
    int* d_sites = (int*)dev_alloc(c, (size_t)nsites * 4 * sizeof(int));
    double* d_out = (double*)dev_alloc(c, (size_t)nsites * nrhs * 24 * sizeof(double));
    int rc = (!d_sites || !d_out) ? LQ_ENOMEM : 0;
    if (rc == 0 && cudaMemcpyAsync(d_sites, sites_xyzt, (size_t)nsites * 4 * sizeof(int), cudaMemcpyHostToDevice, c->stream) != cudaSuccess) rc = set_err(c, LQ_ECUDA, "H2D copy failed");
    if (rc == 0) rc = spinor_gather_sites(c, d_out, native_parity_block, nrhs, prec, nsites, d_sites);
    if (rc == 0 && cudaMemcpyAsync(out, d_out, (size_t)nsites * nrhs * 24 * sizeof(double), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) rc = set_err(c, LQ_ECUDA, "D2H copy failed");
    if (cudaStreamSynchronize(c->stream) != cudaSuccess && rc == 0) rc = set_err(c, LQ_ECUDA, "lq_gather_sites failed");
    if (d_sites) dev_free(c, d_sites);
    if (d_out) dev_free(c, d_out);
    return rc;
}
int lq_laplacian_native(lq_ctx* c, void* out, const void* in, int nvec, int prec) {
    if (!c || !out || !in || out == in || !nrhs_ok(nvec)) return set_err(c, LQ_EINVAL, "lq_laplacian_native: bad argument");
    if (prec != LQ_FP64 && prec != LQ_FP32) return set_err(c, LQ_EINVAL, "Laplacian precision must be fp64 or fp32");
    if (!c->has_gauge) return set_err(c, LQ_ESTATE, "gauge field not loaded");
    cudaSetDevice(c->device);
    return laplacian_native(c, out, in, nvec, prec);
}
size_t lq_cv_native_bytes(const lq_ctx* c, int nvec, int prec) {
    if (!c || nvec < 1 || (prec != LQ_FP64 && prec != LQ_FP32)) return 0;
    return cv_native_bytes(c, nvec, prec);
}
int lq_cv_fill_random(lq_ctx* c, void* native_out, int nvec, int prec, uint64_t seed) {
    if (!c || !native_out || !nrhs_ok(nvec) || (prec != LQ_FP64 && prec != LQ_FP32)) return set_err(c, LQ_EINVAL, "lq_cv_fill_random: bad argument");
    cudaSetDevice(c->device);
    return cv_fill(c, native_out, nvec, prec, seed);
}
int lq_laplacian(lq_ctx* c, void* out, const void* in, int nvec, int prec, int loc) {
    if (!c || !out || !in || out == in || !nrhs_ok(nvec)) return set_err(c, LQ_EINVAL, "lq_laplacian: bad argument");
    if (prec != LQ_FP64 && prec != LQ_FP32) return set_err(c, LQ_EINVAL, "Laplacian precision must be fp64 or fp32");
    if (!c->has_gauge) return set_err(c, LQ_ESTATE, "gauge field not loaded");
    cudaSetDevice(c->device);
    const size_t cbytes = (size_t)nvec * c->g.V * 6 * sizeof(double), nbytes = cv_native_bytes(c, nvec, prec);
    void *st_in = nullptr, *st_out = nullptr;
    void *n_in = dev_alloc(c, nbytes), *n_out = dev_alloc(c, nbytes);
    int rc = (!n_in || !n_out) ? LQ_ENOMEM : 0;
    const void* d_in = nullptr;
    if (rc == 0) { d_in = stage_in(c, in, cbytes, loc, &st_in); if (!d_in) rc = LQ_ENOMEM; }
    if (rc == 0 && cudaMemsetAsync(n_in, 0, nbytes, c->stream) != cudaSuccess) rc = set_err(c, LQ_ECUDA, "memset failed");
    if (rc == 0) rc = cv_pack(c, n_in, (const double*)d_in, nvec, prec);
    if (rc == 0) rc = laplacian_native(c, n_out, n_in, nvec, prec);
    void* d_out = out;
    if (rc == 0 && loc == LQ_HOST) { st_out = dev_alloc(c, cbytes); if (!st_out) rc = LQ_ENOMEM; d_out = st_out; }
    if (rc == 0) rc = cv_unpack(c, (double*)d_out, n_out, nvec, prec);
    if (rc == 0 && st_out && cudaMemcpyAsync(out, st_out, cbytes, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) rc = set_err(c, LQ_ECUDA, "D2H copy failed");
    if (cudaStreamSynchronize(c->stream) != cudaSuccess && rc == 0) rc = set_err(c, LQ_ECUDA, std::string("lq_laplacian: ") + cudaGetErrorString(cudaGetLastError()));
    void* tofree[] = {st_in, st_out, n_in, n_out};
    for (void* p : tofree) if (p) dev_free(c, p);
    return rc;
}
int lq_laph_eigensolve(lq_ctx* c, double* evals, void* evecs, int loc, const lq_eig_param* param, lq_eig_info* info) {
    if (!c || !evals || !param || !info) return set_err(c, LQ_EINVAL, "lq_laph_eigensolve: null argument");
    if (!c->has_gauge) return set_err(c, LQ_ESTATE, "gauge field not loaded");
    cudaSetDevice(c->device);
    memset(info, 0, sizeof(*info));
    const size_t cbytes = (size_t)(param->n_ev > 0 ? param->n_ev : 0) * c->g.V * 6 * sizeof(double);
    void* st = nullptr; double* d_ev = (double*)evecs;
    if (evecs && loc == LQ_HOST) { st = dev_alloc(c, cbytes); if (!st) return LQ_ENOMEM; d_ev = (double*)st; }
    int rc = laph_eigensolve(c, evals, d_ev, param, info);
    if ((rc == 0 || rc == LQ_ENOTCONVERGED) && st) {
        if (cudaMemcpyAsync(evecs, st, cbytes, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess || cudaStreamSynchronize(c->stream) != cudaSuccess)
            rc = set_err(c, LQ_ECUDA, "D2H copy failed");
    }
    if (st) dev_free(c, st);
    return rc;
}
int lq_project(lq_ctx* c, void* P, const void* evecs, int n_ev, const void* sols, int n_sol, int loc, int prec) {
    if (!c || !P || !evecs || !sols || n_ev < 1 || n_ev > 1024 || n_sol < 1 || n_sol > 64) return set_err(c, LQ_EINVAL, "lq_project: bad argument");
    if (prec != LQ_FP64 && prec != LQ_FP32) return set_err(c, LQ_EINVAL, "lq_project: precision must be fp64 or fp32");
    cudaSetDevice(c->device);
    const size_t vb = (size_t)n_ev * c->g.V * 6 * sizeof(double), xb = (size_t)n_sol * c->g.V * 24 * sizeof(double);
    const size_t pb = (size_t)c->g.L[3] * 4 * n_ev * n_sol * 2 * sizeof(double);
    void *st_v = nullptr, *st_x = nullptr, *st_p = nullptr;
    const void* d_v = stage_in(c, evecs, vb, loc, &st_v);
    const void* d_x = d_v ? stage_in(c, sols, xb, loc, &st_x) : nullptr;
    int rc = (!d_v || !d_x) ? LQ_ENOMEM : 0;
    void* d_p = P;
    if (rc == 0 && loc == LQ_HOST) { st_p = dev_alloc(c, pb); if (!st_p) rc = LQ_ENOMEM; d_p = st_p; }
    if (rc == 0) rc = prec == LQ_FP64 ? project_device(c, (double*)d_p, (const double*)d_v, n_ev, (const double*)d_x, n_sol)
                                      : project_device_tc(c, (double*)d_p, (const double*)d_v, n_ev, (const double*)d_x, n_sol);
    if (rc == 0 && st_p) {
        if (cudaMemcpyAsync(P, st_p, pb, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess || cudaStreamSynchronize(c->stream) != cudaSuccess) rc = set_err(c, LQ_ECUDA, "D2H copy failed");
    }
    void* tofree[] = {st_v, st_x, st_p};
    for (void* q : tofree) if (q) dev_free(c, q);
    return rc;
}
int lq_project_c64(lq_ctx* c, void* P, const void* evecs, int n_ev, const void* sols, int n_sol, int loc) {
    if (!c) return LQ_EINVAL;
    if (!P || !evecs || !sols || n_ev < 1 || n_ev > 1024 || n_sol < 1 || n_sol > 64) return set_err(c, LQ_EINVAL, "lq_project_c64: bad argument");
    cudaSetDevice(c->device);
    const size_t vb = (size_t)n_ev * c->g.V * 3 * 2 * sizeof(float), xb = (size_t)n_sol * c->g.V * 12 * 2 * sizeof(float);
    const size_t pb = (size_t)c->g.L[3] * 4 * n_ev * n_sol * 2 * sizeof(double);
    void *st_v = nullptr, *st_x = nullptr, *st_p = nullptr;
    const void* d_v = stage_in(c, evecs, vb, loc, &st_v);
    const void* d_x = d_v ? stage_in(c, sols, xb, loc, &st_x) : nullptr;
    int rc = (!d_v || !d_x) ? LQ_ENOMEM : 0;
    void* d_p = P;
    if (rc == 0 && loc == LQ_HOST) { st_p = dev_alloc(c, pb); if (!st_p) rc = LQ_ENOMEM; d_p = st_p; }
    if (rc == 0) rc = project_device_tc32(c, (double*)d_p, (const float*)d_v, n_ev, (const float*)d_x, n_sol);
    if (rc == 0 && st_p) {
        if (cudaMemcpyAsync(P, st_p, pb, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess || cudaStreamSynchronize(c->stream) != cudaSuccess) rc = set_err(c, LQ_ECUDA, "D2H copy failed");
    }
    void* tofree[] = {st_v, st_x, st_p};
    for (void* q : tofree) if (q) dev_free(c, q);
    return rc;
}
// the operator on native buffers
static int apply_native(lq_ctx* c, int op, void* out, const void* in, const void* in2, int n, int prec) {
    const size_t pb = parity_bytes(c->g, n, prec);
    char* out_e = (char*)out; char* out_o = out_e + pb;
    const char* in_e = (const char*)in; const char* in_o = in_e + pb;
    const double k = c->kappa;
    switch (op) {
    case LQ_OP_HOP:
        LQ_TRY(op_hop(c, prec, n, 0, out_e, in_o, 0));
        return op_hop(c, prec, n, 1, out_o, in_e, 0);
    case LQ_OP_M: case LQ_OP_MDAG: {
        const int dag = op == LQ_OP_MDAG;
        LQ_TRY(op_kernel_b(c, prec, n, 0, out_e, in_e, in_o, -k, 1, dag));
        return op_kernel_b(c, prec, n, 1, out_o, in_o, in_e, -k, 1, dag);
    }
    case LQ_OP_CLOVER: case LQ_OP_CLOVER_INV: {
        const int inv = op == LQ_OP_CLOVER_INV;
        LQ_TRY(op_clover(c, prec, n, 0, out_e, in_e, inv));
        return op_clover(c, prec, n, 1, out_o, in_o, inv);
    }
    case LQ_OP_HOP_EO: return op_hop(c, prec, n, 0, out, in, 0);
    case LQ_OP_HOP_OE: return op_hop(c, prec, n, 1, out, in, 0);
    case LQ_OP_MHAT: return mhat_native(c, prec, n, out, in, 0);
    case LQ_OP_MHAT_DAG: return mhat_native(c, prec, n, out, in, 1);
    case LQ_OP_KERNEL_A: return op_kernel_a(c, prec, n, 1, out, in, 0);
    case LQ_OP_KERNEL_B: return op_kernel_b(c, prec, n, 0, out, in, in2, -k * k, 1, 0);
    case LQ_OP_PROBE_LOADS: return op_probe_loads(c, prec, n, 1, out, in);
    default: return set_err(c, LQ_EINVAL, "unknown operator");
    }
}

int lq_apply(lq_ctx* c, int op, void* out, const void* in, const void* in2, int nrhs, int prec, int loc, int layout) {
    if (!c || !out || !in) return set_err(c, LQ_EINVAL, "lq_apply: null argument");
    if (!nrhs_ok(nrhs)) return set_err(c, LQ_EINVAL, "nrhs must be 1, 2 or a multiple of 4 up to 32");
    if (prec != LQ_FP64 && prec != LQ_FP32 && prec != LQ_HALF) return set_err(c, LQ_EINVAL, "bad precision");
    if (op < 0 || op > LQ_OP_PROBE_LOADS) return set_err(c, LQ_EINVAL, "unknown operator");
    if (op == LQ_OP_PROBE_LOADS && layout != LQ_NATIVE) return set_err(c, LQ_EINVAL, "LQ_OP_PROBE_LOADS is a native-layout bench probe");
    if (op == LQ_OP_KERNEL_B && !in2) return set_err(c, LQ_EINVAL, "LQ_OP_KERNEL_B needs in2");
    if (out == in || out == in2) return set_err(c, LQ_EINVAL, "out must not alias an input");
    if (!c->has_gauge) return set_err(c, LQ_ESTATE, "gauge field not loaded");
    const bool needs_clover = !(op == LQ_OP_HOP || op == LQ_OP_HOP_EO || op == LQ_OP_HOP_OE);
    if (needs_clover && !c->has_clover) return set_err(c, LQ_ESTATE, "clover term not built");
    cudaSetDevice(c->device);
    if (layout == LQ_NATIVE) {
        if (loc != LQ_DEVICE) return set_err(c, LQ_EINVAL, "native buffers must be device buffers");
        return apply_native(c, op, out, in, in2, nrhs, prec);
    }
    // canonical: stage, pack, apply, unpack
    const int cprec = prec == LQ_FP64 ? LQ_FP64 : LQ_FP32;
    const size_t cbytes = (size_t)nrhs * c->g.V * 24 * elem_bytes(cprec);
    const size_t pb = parity_bytes(c->g, nrhs, prec);
    const bool full = op <= LQ_OP_CLOVER_INV;
    int in_par = 0, out_par = 0;       // parity blocks used by parity ops
    if (op == LQ_OP_HOP_EO) { in_par = 1; out_par = 0; }
    if (op == LQ_OP_HOP_OE || op == LQ_OP_KERNEL_A) { in_par = 0; out_par = 1; }
    void *st_in = nullptr, *st_in2 = nullptr, *st_out = nullptr;
    void *n_in = dev_alloc(c, 2 * pb), *n_in2 = in2 ? dev_alloc(c, 2 * pb) : nullptr, *n_out = dev_alloc(c, 2 * pb);
    int rc = (!n_in || !n_out || (in2 && !n_in2)) ? LQ_ENOMEM : 0;
    const void* d_in = nullptr; const void* d_in2 = nullptr;
    if (rc == 0) { d_in = stage_in(c, in, cbytes, loc, &st_in); if (!d_in) rc = LQ_ENOMEM; }
    if (rc == 0 && in2) { d_in2 = stage_in(c, in2, cbytes, loc, &st_in2); if (!d_in2) rc = LQ_ENOMEM; }
    if (rc == 0) rc = spinor_pack(c, n_in, d_in, nrhs, prec, cprec);
    if (rc == 0 && in2) rc = spinor_pack(c, n_in2, d_in2, nrhs, prec, cprec);
    if (rc == 0 && cudaMemsetAsync(n_out, 0, 2 * pb, c->stream) != cudaSuccess) rc = set_err(c, LQ_ECUDA, "memset failed");
    if (rc == 0) {
        if (full) rc = apply_native(c, op, n_out, n_in, nullptr, nrhs, prec);
        else rc = apply_native(c, op, (char*)n_out + out_par * pb, (char*)n_in + in_par * pb, in2 ? (char*)n_in2 + pb : nullptr, nrhs, prec);
    }
    void* d_out = out;
    if (rc == 0 && loc == LQ_HOST) { st_out = dev_alloc(c, cbytes); if (!st_out) rc = LQ_ENOMEM; d_out = st_out; }
    if (rc == 0) rc = spinor_unpack(c, d_out, n_out, nrhs, prec, cprec);
    if (rc == 0 && st_out && cudaMemcpyAsync(out, st_out, cbytes, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) rc = set_err(c, LQ_ECUDA, "D2H copy failed");
    if (cudaStreamSynchronize(c->stream) != cudaSuccess && rc == 0) rc = set_err(c, LQ_ECUDA, std::string("lq_apply: ") + cudaGetErrorString(cudaGetLastError()));
    void* tofree[] = {st_in, st_in2, st_out, n_in, n_in2, n_out};
    for (void* p : tofree) if (p) dev_free(c, p);
    return rc;
}

int lq_solve(lq_ctx* c, void* x, const void* b, int nrhs, int loc, int layout, const lq_solve_param* param, lq_solve_info* info) {
    if (!c || !x || !b || !param || !info) return set_err(c, LQ_EINVAL, "lq_solve: null argument");
    if (!nrhs_ok(nrhs)) return set_err(c, LQ_EINVAL, "nrhs must be 1, 2 or a multiple of 4 up to 32");
    if (!(param->tol > 0) || param->max_outer < 1 || param->max_inner < 1) return set_err(c, LQ_EINVAL, "bad solve parameters");
    cudaSetDevice(c->device);
    if (layout == LQ_NATIVE) {
        if (loc != LQ_DEVICE) return set_err(c, LQ_EINVAL, "native buffers must be device buffers");
        return solve_native(c, x, b, nrhs, param, info);
    }
    const size_t pb = parity_bytes(c->g, nrhs, LQ_FP64);
    void *n_b = dev_alloc(c, 2 * pb), *n_x = dev_alloc(c, 2 * pb);
    int rc = (!n_b || !n_x) ? LQ_ENOMEM : 0;
    if (rc == 0) rc = pack_any(c, n_b, b, nrhs, LQ_FP64, loc);
    if (rc == 0 && param->use_x0) rc = pack_any(c, n_x, x, nrhs, LQ_FP64, loc);
    int src = 0;
    if (rc == 0) { src = solve_native(c, n_x, n_b, nrhs, param, info); if (src != 0 && src != LQ_ENOTCONVERGED) rc = src; }
    if (rc == 0) rc = unpack_any(c, x, n_x, nrhs, LQ_FP64, loc);
    if (cudaStreamSynchronize(c->stream) != cudaSuccess && rc == 0) rc = set_err(c, LQ_ECUDA, std::string("lq_solve: ") + cudaGetErrorString(cudaGetLastError()));
    void* tofree[] = {n_b, n_x};
    for (void* p : tofree) if (p) dev_free(c, p);
    return rc ? rc : src;
}

// ---- two-level multigrid (multigrid.cu) ---------------------------------------------------------------------------------------
int lq_mg_setup(lq_ctx* c, const lq_mg_param* param, lq_mg_info* info) {
    if (!c) return LQ_EINVAL;
    cudaSetDevice(c->device);
    return mg_setup_adaptive(c, param, info);
}
int lq_mg_setup_from_vectors(lq_ctx* c, const lq_mg_param* param, const void* vecs, int loc, lq_mg_info* info) {
    if (!c) return LQ_EINVAL;
    if (!param || !vecs || param->n_vec < 1 || param->n_vec > LQ_MAX_RHS) return set_err(c, LQ_EINVAL, "lq_mg_setup_from_vectors: bad argument");
    cudaSetDevice(c->device);
    void* st = nullptr;
    const void* d = stage_in(c, vecs, (size_t)param->n_vec * c->g.V * 24 * sizeof(double), loc, &st);
    int rc = d ? mg_setup_vectors(c, param, d, info) : LQ_ENOMEM;
    if (st) { cudaStreamSynchronize(c->stream); dev_free(c, st); }
    return rc;
}
int lq_mg_free(lq_ctx* c) {
    if (!c) return LQ_EINVAL;
    cudaSetDevice(c->device);
    cudaStreamSynchronize(c->stream);
    mg_release(c);
    return 0;
}
// one of the four pieces: in / out are fine (canonical) or coarse arrays at `loc`
static int mg_piece(lq_ctx* c, int which, void* out, const void* in, int nrhs, int loc) {
    if (!c) return LQ_EINVAL;
    if (!out || !in || out == in || !nrhs_ok(nrhs)) return set_err(c, LQ_EINVAL, "lq_mg_*: bad argument");
    if (!c->mg) return set_err(c, LQ_ESTATE, "lq_mg_*: no multigrid hierarchy");
    cudaSetDevice(c->device);
    const size_t fb = (size_t)nrhs * c->g.V * 24 * sizeof(double), cb = mg_coarse_canonical_bytes(c, nrhs);
    const bool in_fine = which == 0 || which == 3, out_fine = which == 1 || which == 3;
    const size_t ib = in_fine ? fb : cb, ob = out_fine ? fb : cb;
    void *st_in = nullptr, *st_out = nullptr;
    const void* d_in = stage_in(c, in, ib, loc, &st_in);
    int rc = d_in ? 0 : LQ_ENOMEM;
    void* d_out = out;
    if (rc == 0 && loc == LQ_HOST) { st_out = dev_alloc(c, ob); if (!st_out) rc = LQ_ENOMEM; d_out = st_out; }
    if (rc == 0) {
        if (which == 0) rc = mg_restrict_dev(c, (double*)d_out, d_in, nrhs);
        else if (which == 1) rc = mg_prolong_dev(c, d_out, (const double*)d_in, nrhs);
        else if (which == 2) rc = mg_coarse_apply_dev(c, (double*)d_out, (const double*)d_in, nrhs);
        else rc = mg_vcycle_dev(c, d_out, d_in, nrhs);
    }
    if (rc == 0 && st_out && cudaMemcpyAsync(out, st_out, ob, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) rc = set_err(c, LQ_ECUDA, "D2H copy failed");
    if (cudaStreamSynchronize(c->stream) != cudaSuccess && rc == 0) rc = set_err(c, LQ_ECUDA, std::string("lq_mg_*: ") + cudaGetErrorString(cudaGetLastError()));
    if (st_in) dev_free(c, st_in);
    if (st_out) dev_free(c, st_out);
    return rc;
}
int lq_mg_restrict(lq_ctx* c, void* coarse_out, const void* fine_in, int nrhs, int loc) { return mg_piece(c, 0, coarse_out, fine_in, nrhs, loc); }
int lq_mg_prolong(lq_ctx* c, void* fine_out, const void* coarse_in, int nrhs, int loc) { return mg_piece(c, 1, fine_out, coarse_in, nrhs, loc); }
int lq_mg_coarse_apply(lq_ctx* c, void* coarse_out, const void* coarse_in, int nrhs, int loc) { return mg_piece(c, 2, coarse_out, coarse_in, nrhs, loc); }
int lq_mg_vcycle(lq_ctx* c, void* z, const void* r, int nrhs, int loc) { return mg_piece(c, 3, z, r, nrhs, loc); }

int lq_mg_solve(lq_ctx* c, void* x, const void* b, int nrhs, int loc, double tol, int max_iter, lq_mg_solve_info* info) {
    if (!c) return LQ_EINVAL;
    if (!x || !b || !info || !nrhs_ok(nrhs) || !(tol > 0) || max_iter < 1) return set_err(c, LQ_EINVAL, "lq_mg_solve: bad argument");
    cudaSetDevice(c->device);
    const size_t pb = parity_bytes(c->g, nrhs, LQ_FP64);
    void *n_b = dev_alloc(c, 2 * pb), *n_x = dev_alloc(c, 2 * pb);
    int rc = (!n_b || !n_x) ? LQ_ENOMEM : 0;
    if (rc == 0) rc = pack_any(c, n_b, b, nrhs, LQ_FP64, loc);
    int src = 0;
    if (rc == 0) { src = mg_solve_native(c, n_x, n_b, nrhs, tol, max_iter, info); if (src != 0 && src != LQ_ENOTCONVERGED) rc = src; }
    if (rc == 0) rc = unpack_any(c, x, n_x, nrhs, LQ_FP64, loc);
    if (cudaStreamSynchronize(c->stream) != cudaSuccess && rc == 0) rc = set_err(c, LQ_ECUDA, std::string("lq_mg_solve: ") + cudaGetErrorString(cudaGetLastError()));
    void* tofree[] = {n_b, n_x};
    for (void* p : tofree) if (p) dev_free(c, p);
    return rc ? rc : src;
}

}  // extern "C"
