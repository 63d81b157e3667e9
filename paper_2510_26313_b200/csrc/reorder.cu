// reorder.cu -- canonical <-> native reorders and precision conversion.
#include "internal.cuh"

// ---- gauge ---------------------------------------------------------------------------------------------------
template <typename Tin>
__global__ void gauge_ingest_kernel(Geom g, const Tin* __restrict__ canon, double* __restrict__ native) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 8LL * g.Vh) return;
    const int cb = (int)(tid % g.Vh);
    const int pm = (int)(tid / g.Vh);           // parity*4 + mu
    const int parity = pm >> 2, mu = pm & 3;
    int xh, y, z, t, odd;
    cb_coords(g, parity, cb, xh, y, z, t, odd);
    const long long site = (2 * xh + odd) + (long long)g.L[0] * (y + (long long)g.L[1] * (z + (long long)g.L[2] * t));
    const Tin* src = canon + ((long long)mu * g.V + site) * 18;
    double r[18];
#pragma unroll
    for (int k = 0; k < 18; k++) r[k] = (double)src[k];
    store_planes<double, 18>(link_block(native, g.NB, 18, parity, cb / SB, mu), cb % SB, r);
}
int gauge_ingest(lq_ctx* c, const void* dev_canonical, int in_prec) {
    const long long threads = 8LL * c->g.Vh;
    const int block = 128; const int grid = (int)((threads + block - 1) / block);
    if (in_prec == LQ_FP64) gauge_ingest_kernel<double><<<grid, block, 0, c->stream>>>(c->g, (const double*)dev_canonical, c->gauge64);
    else if (in_prec == LQ_FP32) gauge_ingest_kernel<float><<<grid, block, 0, c->stream>>>(c->g, (const float*)dev_canonical, c->gauge64);
    else return set_err(c, LQ_EINVAL, "gauge precision must be fp64 or fp32");
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
template <int RECON>
__global__ void gauge_to_fp32_kernel(int Vh, int NB, const double* __restrict__ src, float* __restrict__ dst) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 8LL * Vh) return;
    const int cb = (int)(tid % Vh), pm = (int)(tid / Vh);
    double r[18]; float f[18];
    load_planes<double, 18>(link_block(src, NB, 18, pm >> 2, cb / SB, pm & 3), cb % SB, r);
#pragma unroll
    for (int k = 0; k < RECON; k++) f[k] = (float)r[k];
    store_planes<float, RECON>(link_block(dst, NB, RECON, pm >> 2, cb / SB, pm & 3), cb % SB, f);
}
int gauge_make_fp32(lq_ctx* c, int recon) {
    const long long threads = 8LL * c->g.Vh;
    const int block = 128; const int grid = (int)((threads + block - 1) / block);
    if (recon == 18) gauge_to_fp32_kernel<18><<<grid, block, 0, c->stream>>>(c->g.Vh, c->g.NB, c->gauge64, c->gauge32);
    else gauge_to_fp32_kernel<12><<<grid, block, 0, c->stream>>>(c->g.Vh, c->g.NB, c->gauge64, c->gauge32);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    c->recon32 = recon;
    return 0;
}

// int16 fixed-point copy of the 18-real links for the half-storage kernels (H16L): q = rint(32767 u), |u| <= 1
__global__ void gauge_to_int16_kernel(int Vh, int NB, const double* __restrict__ src, short* __restrict__ dst) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 8LL * Vh) return;
    const int cb = (int)(tid % Vh), pm = (int)(tid / Vh);
    double r[18];
    load_planes<double, 18>(link_block(src, NB, 18, pm >> 2, cb / SB, pm & 3), cb % SB, r);
    short* blk = dst + ((size_t)((pm >> 2) * NB + cb / SB) * 4 + (pm & 3)) * (size_t)(18 * SB);
    const int s = cb % SB;
#pragma unroll
    for (int k = 0; k < 18; k++) {
        const float q = rintf(fminf(fmaxf((float)r[k], -1.0f), 1.0f) * 32767.0f);
        const int plane = k / 8, e = k % 8;
        if (plane < 2) blk[plane * 8 * SB + s * 8 + e] = (short)q; else blk[16 * SB + s * 2 + e] = (short)q;
    }
}
int gauge_make_int16(lq_ctx* c) {
    if (!c->gauge16) { c->gauge16 = (short*)dev_alloc(c, (size_t)8 * 18 * c->g.NB * SB * sizeof(short)); if (!c->gauge16) return LQ_ENOMEM; }
    LQ_CUDA(c, cudaMemsetAsync(c->gauge16, 0, (size_t)8 * 18 * c->g.NB * SB * sizeof(short), c->stream));
    const long long threads = 8LL * c->g.Vh;
    const int block = 128; const int grid = (int)((threads + block - 1) / block);
    gauge_to_int16_kernel<<<grid, block, 0, c->stream>>>(c->g.Vh, c->g.NB, c->gauge64, c->gauge16);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}

// ---- scalar element access of a native parity block ---------------------------------------------------------------
template <class S>
__device__ __forceinline__ void load_site(const SView<S>& v, int N, int cb, int k, double* o) {
    const int PL = SB * group_width(N);
    const size_t off = sp_index(N, cb, k, 0);
    double sc = 1.0;
    if constexpr (S::has_norm) sc = (double)(v.n[nrm_index(N, cb, k)] * (1.0f / 32767.0f));
#pragma unroll
    for (int j = 0; j < 24; j++) o[j] = (double)v.d[off + (size_t)j * PL] * sc;
}
template <class S>
__device__ __forceinline__ void store_site(const SView<S>& v, int N, int cb, int k, const double* o) {
    const int PL = SB * group_width(N);
    const size_t off = sp_index(N, cb, k, 0);
    if constexpr (S::has_norm) {
        float mx = 0.f;
#pragma unroll
        for (int j = 0; j < 24; j++) mx = fmaxf(mx, fabsf((float)o[j]));
        v.n[nrm_index(N, cb, k)] = mx;
        const float inv = mx > 0.f ? 32767.0f / mx : 0.f;
#pragma unroll
        for (int j = 0; j < 24; j++) v.d[off + (size_t)j * PL] = (short)rintf((float)o[j] * inv);
    } else {
#pragma unroll
        for (int j = 0; j < 24; j++) v.d[off + (size_t)j * PL] = (typename S::store_t)o[j];
    }
}

// ---- spinor pack / unpack ---------------------------------------------------------------------------------------------
// `canon` holds right-hand sides k0 .. k0+nk-1 of the batch of N (canonical [rhs][site][24]); the native buffer holds all N.
template <class S, typename Tc, bool PACK>
__global__ void spinor_reorder_kernel(Geom g, int N, int k0, int nk, SView<S> even, SView<S> odd, Tc* canon) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 2LL * g.Vh * nk) return;
    const int kl = (int)(tid % nk), k = k0 + kl;
    const long long r = tid / nk;
    const int cb = (int)(r % g.Vh), parity = (int)(r / g.Vh);
    int xh, y, z, t, odd_;
    cb_coords(g, parity, cb, xh, y, z, t, odd_);
    const long long site = (2 * xh + odd_) + (long long)g.L[0] * (y + (long long)g.L[1] * (z + (long long)g.L[2] * t));
    Tc* p = canon + ((long long)kl * g.V + site) * 24;
    const SView<S>& v = parity ? odd : even;
    double o[24];
    if constexpr (PACK) {
#pragma unroll
        for (int j = 0; j < 24; j++) o[j] = (double)p[j];
        store_site<S>(v, N, cb, k, o);
    } else {
        load_site<S>(v, N, cb, k, o);
#pragma unroll
        for (int j = 0; j < 24; j++) p[j] = (Tc)o[j];
    }
}
template <class S, bool PACK>
static int reorder_t(lq_ctx* c, void* native_full, void* canon, int nrhs, int k0, int nk, int cprec) {
    SView<S> e = make_view<S>(c->g, native_full, nrhs, 0), o = make_view<S>(c->g, native_full, nrhs, 1);
    const long long threads = 2LL * c->g.Vh * nk;
    const int block = 128; const int grid = (int)((threads + block - 1) / block);
    if (cprec == LQ_FP64) spinor_reorder_kernel<S, double, PACK><<<grid, block, 0, c->stream>>>(c->g, nrhs, k0, nk, e, o, (double*)canon);
    else spinor_reorder_kernel<S, float, PACK><<<grid, block, 0, c->stream>>>(c->g, nrhs, k0, nk, e, o, (float*)canon);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
int spinor_pack_part(lq_ctx* c, void* native_full, const void* dev_canonical, int nrhs, int k0, int nk, int prec, int in_prec) {
    void* cn = const_cast<void*>(dev_canonical);
    if (prec == LQ_FP64) return reorder_t<F64, true>(c, native_full, cn, nrhs, k0, nk, in_prec);
    if (prec == LQ_FP32) return reorder_t<F32, true>(c, native_full, cn, nrhs, k0, nk, in_prec);
    return reorder_t<H16, true>(c, native_full, cn, nrhs, k0, nk, in_prec);
}
int spinor_unpack_part(lq_ctx* c, void* dev_canonical, const void* native_full, int nrhs, int k0, int nk, int prec, int out_prec) {
    void* nf = const_cast<void*>(native_full);
    if (prec == LQ_FP64) return reorder_t<F64, false>(c, nf, dev_canonical, nrhs, k0, nk, out_prec);
    if (prec == LQ_FP32) return reorder_t<F32, false>(c, nf, dev_canonical, nrhs, k0, nk, out_prec);
    return reorder_t<H16, false>(c, nf, dev_canonical, nrhs, k0, nk, out_prec);
}
int spinor_pack(lq_ctx* c, void* native_full, const void* dev_canonical, int nrhs, int prec, int in_prec) {
    return spinor_pack_part(c, native_full, dev_canonical, nrhs, 0, nrhs, prec, in_prec);
}
int spinor_unpack(lq_ctx* c, void* dev_canonical, const void* native_full, int nrhs, int prec, int out_prec) {
    return spinor_unpack_part(c, dev_canonical, native_full, nrhs, 0, nrhs, prec, out_prec);
}

// ---- precision conversion of one parity block, with an optional per-RHS scale ----------------------------------------------
template <class SD, class SS>
__global__ void convert_kernel(int Vh, int N, SView<SD> dst, SView<SS> src, const double* __restrict__ scale, int invert) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= (long long)Vh * N) return;
    const int k = (int)(tid % N), cb = (int)(tid / N);
    double o[24];
    load_site<SS>(src, N, cb, k, o);
    if (scale) {
        double s = scale[k];
        if (invert) s = (s != 0.0) ? 1.0 / s : 0.0;
#pragma unroll
        for (int j = 0; j < 24; j++) o[j] *= s;
    }
    store_site<SD>(dst, N, cb, k, o);
}
template <class SD, class SS>
static int convert_t(lq_ctx* c, void* dst, const void* src, int nrhs, const double* d_scale, int invert) {
    SView<SD> d = make_view<SD>(c->g, dst, nrhs, 0);
    SView<SS> s = make_view<SS>(c->g, const_cast<void*>(src), nrhs, 0);
    const long long threads = (long long)c->g.Vh * nrhs;
    const int block = 128; const int grid = (int)((threads + block - 1) / block);
    convert_kernel<SD, SS><<<grid, block, 0, c->stream>>>(c->g.Vh, nrhs, d, s, d_scale, invert);
    LQ_LAUNCHED(c);
    LQ_MODEL(c, stream_bytes(c->g, nrhs, SD::prec) + stream_bytes(c->g, nrhs, SS::prec), 24.0 * c->g.Vh * nrhs);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
template <class SD>
static int convert_d(lq_ctx* c, void* dst, const void* src, int src_prec, int nrhs, const double* d_scale, int invert) {
    if (src_prec == LQ_FP64) return convert_t<SD, F64>(c, dst, src, nrhs, d_scale, invert);
    if (src_prec == LQ_FP32) return convert_t<SD, F32>(c, dst, src, nrhs, d_scale, invert);
    return convert_t<SD, H16>(c, dst, src, nrhs, d_scale, invert);
}
int spinor_convert(lq_ctx* c, void* dst, int dst_prec, const void* src, int src_prec, int nrhs, const double* d_scale, int invert) {
    if (dst_prec == LQ_FP64) return convert_d<F64>(c, dst, src, src_prec, nrhs, d_scale, invert);
    if (dst_prec == LQ_FP32) return convert_d<F32>(c, dst, src, src_prec, nrhs, d_scale, invert);
    return convert_d<H16>(c, dst, src, src_prec, nrhs, d_scale, invert);
}

int spinor_zero_parity(lq_ctx* c, void* parity_block, int nrhs, int prec) {
    LQ_CUDA(c, cudaMemsetAsync(parity_block, 0, parity_bytes(c->g, nrhs, prec), c->stream));
    return 0;
}

template <typename Tc>
__global__ void canonical_zero_parity_kernel(Geom g, int N, Tc* canon, int parity) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= (long long)g.Vh * N) return;
    const int cb = (int)(tid % g.Vh), k = (int)(tid / g.Vh);
    int xh, y, z, t, odd_;
    cb_coords(g, parity, cb, xh, y, z, t, odd_);
    const long long site = (2 * xh + odd_) + (long long)g.L[0] * (y + (long long)g.L[1] * (z + (long long)g.L[2] * t));
    Tc* p = canon + ((long long)k * g.V + site) * 24;
#pragma unroll
    for (int j = 0; j < 24; j++) p[j] = Tc(0);
}
int canonical_zero_parity(lq_ctx* c, void* dev_canonical, int nrhs, int prec, int parity) {
    const long long threads = (long long)c->g.Vh * nrhs;
    const int block = 128; const int grid = (int)((threads + block - 1) / block);
    if (prec == LQ_FP64) canonical_zero_parity_kernel<double><<<grid, block, 0, c->stream>>>(c->g, nrhs, (double*)dev_canonical, parity);
    else canonical_zero_parity_kernel<float><<<grid, block, 0, c->stream>>>(c->g, nrhs, (float*)dev_canonical, parity);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}

// ---- read back selected sites of one parity block ----------------------------------------------------------------
template <class S>
__global__ void gather_sites_kernel(Geom g, int N, SView<S> v, long long nsites, const int* __restrict__ sites, double* __restrict__ out) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= nsites * N) return;
    const int k = (int)(tid % N);
    const long long n = tid / N;
    int parity, cb;
    coords_to_cb(g, sites[4 * n], sites[4 * n + 1], sites[4 * n + 2], sites[4 * n + 3], parity, cb);
    double o[24];
    load_site<S>(v, N, cb, k, o);
#pragma unroll
    for (int j = 0; j < 24; j++) out[(n * N + k) * 24 + j] = o[j];
}
int spinor_gather_sites(lq_ctx* c, double* dev_out, const void* parity_block, int nrhs, int prec, long long nsites, const int* dev_sites) {
    const long long threads = nsites * nrhs;
    const int block = 128; const int grid = (int)((threads + block - 1) / block);
    void* pb = const_cast<void*>(parity_block);
    if (prec == LQ_FP64) gather_sites_kernel<F64><<<grid, block, 0, c->stream>>>(c->g, nrhs, make_view<F64>(c->g, pb, nrhs, 0), nsites, dev_sites, dev_out);
    else if (prec == LQ_FP32) gather_sites_kernel<F32><<<grid, block, 0, c->stream>>>(c->g, nrhs, make_view<F32>(c->g, pb, nrhs, 0), nsites, dev_sites, dev_out);
    else gather_sites_kernel<H16><<<grid, block, 0, c->stream>>>(c->g, nrhs, make_view<H16>(c->g, pb, nrhs, 0), nsites, dev_sites, dev_out);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
