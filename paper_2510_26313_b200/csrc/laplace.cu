// laplace.cu -- batched 3-d gauge-covariant Laplacian:
//   (Lap v)(x) = sum_{i = x,y,z} [ U_i(x) v(x+i) + U_i(x-i)^dag v(x-i) ] - 6 v(x)       on every time-slice,
// for N colour-vector fields at once (the batch index is innermost, so a link is loaded once per batch group, exactly
// as in the Dslash kernels; the time extent is an independent batching dimension).
//
// Native colour-vector layout (one parity): [blk][g][j = 0..5][s = 0..31][r = 0..R-1], j = 2*colour + (re|im):
// the spinor layout of common.cuh with 6 instead of 24 reals per site.  A full field = even block, then odd block.
#include "internal.cuh"
#include "dslash_kernel.cuh"

inline size_t cv_parity_bytes(const Geom& g, int nvec, int prec) { return round256((size_t)6 * g.NB * SB * nvec * elem_bytes(prec)); }
__host__ __device__ inline size_t cv_index(int N, int cb, int k, int j) {
    const int R = group_width(N), G = N / R;
    const size_t u = (size_t)(cb / SB) * G + k / R;
    return (u * 6 + j) * (SB * R) + (size_t)(cb % SB) * R + k % R;
}

template <typename T> struct StoreOf;
template <> struct StoreOf<float> { using S = F32; };
template <> struct StoreOf<double> { using S = F64; };

template <typename T, int RPT, int R, int RECON>
// Fused epilogue (the three-term Chebyshev recurrence of the Lanczos filter without a separate vector kernel and without
// storing Lap v): out = ca * (Lap in) + cb * in + cc * y, y optional (may be `out` itself: every thread reads its own site of y
// before it writes it); ca = 1, cb = cc = 0 is the plain operator.  out must not alias in.
__global__ void __launch_bounds__(128) laplace_kernel(Geom g, int G, FastDiv d2G, int pfd, T* out_full, const T* __restrict__ in_full,
                                                      size_t pb_elems, const T* __restrict__ gauge, T ca, T cb, T cc, const T* y_full) {
    using S = typename StoreOf<T>::S;
    constexpr int TPG = R / RPT, UT = SB * TPG, US = 6 * SB * R, PL = SB * R;
    const int tid = blockIdx.x * 128 + threadIdx.x;
    // one launch covers both parities: work item w -> (site block, parity, RHS group), parity and group fastest, so the
    // link slab that parity p reads as forward links is read as backward links by parity 1-p of the same and the
    // neighbouring blocks a moment later and is still in L2 (each link then costs one HBM read per application)
    const int w = tid / UT;
    if (w >= 2 * g.NB * G) return;
    const int lu = tid - w * UT;
    const int blk = d2G.div(w);
    const int rem = w - blk * 2 * G;
    const int parity = rem >= G ? 1 : 0, grp = rem - parity * G;
    const int u = blk * G + grp;
    T* out = out_full + (size_t)parity * pb_elems;
    const T* in_own = in_full + (size_t)parity * pb_elems;
    const T* in_opp = in_full + (size_t)(1 - parity) * pb_elems;
    const int s = lu / TPG, hoff = (lu - s * TPG) * RPT;
    SiteCtx sc;
    sc.cb = blk * SB + s;
    if (sc.cb >= g.Vh) return;
    cb_coords(g, parity, sc.cb, sc.xh, sc.y, sc.z, sc.t, sc.odd);
    sc.Lxh = g.Lxh; sc.Ly = g.L[1]; sc.Lz = g.L[2]; sc.Lt = g.L[3];
    const size_t own = (size_t)u * US + s * R + hoff;
    const T* gown = gauge + ((size_t)(parity * g.NB + blk) * 4) * (RECON * SB);
    const T* gopp = gauge + ((size_t)((1 - parity) * g.NB) * 4) * (RECON * SB);
    const T* inb = in_opp + (size_t)grp * US + hoff;
    const size_t bstride = (size_t)G * US;

    // distance prefetch into L2 (same reasoning as in dslash_kernel.cuh): what the unit `pfd` blocks ahead touches first
    if (R == 4 && pfd > 0 && blk + pfd < g.NB) {
        const int pb = blk + pfd;
        constexpr int LINE = 128;
        const int sz32 = (sc.Lxh * sc.Ly) / SB;
        int pbz = pb + sz32; if (pbz >= g.NB) pbz -= g.NB;
#define LQ_PF_LINES(base, nlines) { _Pragma("unroll") for (int i0_ = 0; i0_ < (nlines); i0_ += UT) { const int i_ = i0_ + lu; \
            if (i_ < (nlines)) asm volatile("prefetch.global.L2 [%0];" ::"l"((base) + (size_t)i_ * LINE)); } }
        const char* q0 = (const char*)(in_opp + ((size_t)pbz * G + grp) * US);
        const char* q1 = (const char*)(in_own + ((size_t)pb * G + grp) * US);
        LQ_PF_LINES(q0, (int)(US * sizeof(T) / LINE))
        LQ_PF_LINES(q1, (int)(US * sizeof(T) / LINE))
        constexpr int GL = 3 * RECON * SB * sizeof(T) / LINE;      // x, y, z slabs of one (parity, block)
        if (grp == 0 % G) { const char* l = (const char*)(gauge + ((size_t)(parity * g.NB + pb) * 4) * (RECON * SB)); LQ_PF_LINES(l, GL) }
        if (grp == 1 % G) { const char* l = (const char*)(gauge + ((size_t)((1 - parity) * g.NB + pb) * 4) * (RECON * SB)); LQ_PF_LINES(l, GL) }
#undef LQ_PF_LINES
    }
    T acc[6][RPT], vown[6][RPT];
#pragma unroll
    for (int j = 0; j < 6; j++) {
        load_comp<S, RPT>(in_own + own + j * PL, vown[j]);
#pragma unroll
        for (int k = 0; k < RPT; k++) acc[j][k] = vown[j][k] * T(-6);
    }
#define LQ_LAP(D) { const int nb_ = neighbour<D>(sc); constexpr bool FWD_ = ((D) & 1) == 0; \
        const T* p_ = inb + (size_t)(nb_ >> 5) * bstride + (nb_ & 31) * R; \
        T u_[18], v_[6][RPT]; \
        load_link<T, RECON>(FWD_ ? gown + ((D) >> 1) * (RECON * SB) : gopp + ((size_t)(nb_ >> 5) * 4 + ((D) >> 1)) * (RECON * SB), FWD_ ? s : (nb_ & 31), u_); \
        _Pragma("unroll") for (int j = 0; j < 6; j++) load_comp<S, RPT>(p_ + j * PL, v_[j]); \
        _Pragma("unroll") for (int r = 0; r < 3; r++) _Pragma("unroll") for (int c = 0; c < 3; c++) { \
            const T ur_ = FWD_ ? u_[2 * (3 * r + c)] : u_[2 * (3 * c + r)]; \
            const T ui_ = FWD_ ? u_[2 * (3 * r + c) + 1] : -u_[2 * (3 * c + r) + 1]; \
            _Pragma("unroll") for (int k = 0; k < RPT; k++) { \
                acc[2 * r][k] = fm(ur_, v_[2 * c][k], acc[2 * r][k]); acc[2 * r][k] = fm(-ui_, v_[2 * c + 1][k], acc[2 * r][k]); \
                acc[2 * r + 1][k] = fm(ur_, v_[2 * c + 1][k], acc[2 * r + 1][k]); acc[2 * r + 1][k] = fm(ui_, v_[2 * c][k], acc[2 * r + 1][k]); } } }
    LQ_LAP(0) LQ_LAP(1) LQ_LAP(2) LQ_LAP(3) LQ_LAP(4) LQ_LAP(5)
#undef LQ_LAP
    if (ca != T(1) || cb != T(0) || y_full != nullptr) {
        const T* y = y_full != nullptr ? y_full + (size_t)parity * pb_elems : nullptr;
#pragma unroll
        for (int j = 0; j < 6; j++) {
            T yv[RPT];
            if (y != nullptr) {
                // plain loads: y may be the buffer this thread is about to overwrite
                if constexpr (RPT == 1) yv[0] = y[own + j * PL];
                else {
#pragma unroll
                    for (int k = 0; k < RPT; k++) yv[k] = y[own + j * PL + k];
                }
            }
#pragma unroll
            for (int k = 0; k < RPT; k++) acc[j][k] = ca * acc[j][k] + cb * vown[j][k] + (y != nullptr ? cc * yv[k] : T(0));
        }
    }
#pragma unroll
    for (int j = 0; j < 6; j++) store_comp<S, RPT>(out + own + j * PL, acc[j]);
}

template <typename T, int RECON>
static int launch_laplace(lq_ctx* c, int nvec, T* out, const T* in, const T* gauge, int prec, double a, double b, double cc_, const void* yv) {
    const T ca = (T)a, cb = (T)b, cc = (T)cc_;
    const T* y = (const T*)yv;
    const int R = group_width(nvec), G = nvec / R;
    constexpr int MAXRPT = sizeof(T) == 8 ? 2 : 4;
    const int rpt = R < MAXRPT ? R : MAXRPT;
    const long long threads = 2LL * c->g.NB * G * SB * (R / rpt);
    const int grid = (int)((threads + 127) / 128);
    const FastDiv d2G = make_fastdiv(2 * G);
    const size_t pbe = cv_parity_bytes(c->g, nvec, prec) / sizeof(T);
    const int pfd = c->dslash_pfd;
    if (R == 4 && rpt == 4) { if constexpr (MAXRPT == 4) laplace_kernel<T, 4, 4, RECON><<<grid, 128, 0, c->stream>>>(c->g, G, d2G, pfd, out, in, pbe, gauge, ca, cb, cc, y); }
    else if (R == 4) laplace_kernel<T, 2, 4, RECON><<<grid, 128, 0, c->stream>>>(c->g, G, d2G, pfd, out, in, pbe, gauge, ca, cb, cc, y);
    else if (R == 2) laplace_kernel<T, 2, 2, RECON><<<grid, 128, 0, c->stream>>>(c->g, G, d2G, pfd, out, in, pbe, gauge, ca, cb, cc, y);
    else laplace_kernel<T, 1, 1, RECON><<<grid, 128, 0, c->stream>>>(c->g, G, d2G, pfd, out, in, pbe, gauge, ca, cb, cc, y);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}

// out, in: native full colour-vector fields (even block then odd block)
// out = ca * Lap(in) + cb * in + cc * y  (y may be nullptr or `out`)
int laplacian_native_axpby(lq_ctx* c, void* out, const void* in, int nvec, int prec, double ca, double cb, double cc, const void* y) {
    if (prec == LQ_FP64) return launch_laplace<double, 18>(c, nvec, (double*)out, (const double*)in, c->gauge64, prec, ca, cb, cc, y);
    if (c->recon32 == 12) return launch_laplace<float, 12>(c, nvec, (float*)out, (const float*)in, c->gauge32, prec, ca, cb, cc, y);
    return launch_laplace<float, 18>(c, nvec, (float*)out, (const float*)in, c->gauge32, prec, ca, cb, cc, y);
}
int laplacian_native(lq_ctx* c, void* out, const void* in, int nvec, int prec) {
    return laplacian_native_axpby(c, out, in, nvec, prec, 1.0, 0.0, 0.0, nullptr);
}
size_t cv_native_bytes(const lq_ctx* c, int nvec, int prec) { return 2 * cv_parity_bytes(c->g, nvec, prec); }

// ---- canonical [vec][t][z][y][x][3] complex double <-> native -------------------------------------------------------
template <typename T, bool PACK>
__global__ void cv_reorder_kernel(Geom g, int N, T* native, size_t pb_elems, double* canon) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 2LL * g.Vh * N) return;
    const int k = (int)(tid % N);
    const long long r = tid / N;
    const int cb = (int)(r % g.Vh), parity = (int)(r / g.Vh);
    int xh, y, z, t, odd_;
    cb_coords(g, parity, cb, xh, y, z, t, odd_);
    const long long site = (2 * xh + odd_) + (long long)g.L[0] * (y + (long long)g.L[1] * (z + (long long)g.L[2] * t));
    double* p = canon + ((long long)k * g.V + site) * 6;
    T* nb = native + (size_t)parity * pb_elems;
    const int PLs = SB * group_width(N);
    const size_t off = cv_index(N, cb, k, 0);
#pragma unroll
    for (int j = 0; j < 6; j++) {
        if constexpr (PACK) nb[off + (size_t)j * PLs] = (T)p[j];
        else p[j] = (double)nb[off + (size_t)j * PLs];
    }
}
int cv_pack(lq_ctx* c, void* native, const double* dev_canon, int nvec, int prec) {
    const long long threads = 2LL * c->g.Vh * nvec;
    const int grid = (int)((threads + 127) / 128);
    const size_t pbe = cv_parity_bytes(c->g, nvec, prec) / elem_bytes(prec);
    if (prec == LQ_FP64) cv_reorder_kernel<double, true><<<grid, 128, 0, c->stream>>>(c->g, nvec, (double*)native, pbe, const_cast<double*>(dev_canon));
    else cv_reorder_kernel<float, true><<<grid, 128, 0, c->stream>>>(c->g, nvec, (float*)native, pbe, const_cast<double*>(dev_canon));
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
int cv_unpack(lq_ctx* c, double* dev_canon, const void* native, int nvec, int prec) {
    const long long threads = 2LL * c->g.Vh * nvec;
    const int grid = (int)((threads + 127) / 128);
    const size_t pbe = cv_parity_bytes(c->g, nvec, prec) / elem_bytes(prec);
    if (prec == LQ_FP64) cv_reorder_kernel<double, false><<<grid, 128, 0, c->stream>>>(c->g, nvec, (double*)const_cast<void*>(native), pbe, dev_canon);
    else cv_reorder_kernel<float, false><<<grid, 128, 0, c->stream>>>(c->g, nvec, (float*)const_cast<void*>(native), pbe, dev_canon);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}

// ---- bench only: pseudo-random colour vectors written straight into a native buffer ---------------------------------
template <typename T>
__global__ void cv_fill_kernel(T* native, size_t n, unsigned long long seed) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    unsigned long long z = seed + i * 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL; z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL; z ^= z >> 31;
    native[i] = (T)((double)(z >> 11) * (1.0 / 9007199254740992.0) - 0.5);
}
int cv_fill(lq_ctx* c, void* native, int nvec, int prec, unsigned long long seed) {
    const size_t n = cv_native_bytes(c, nvec, prec) / elem_bytes(prec);
    const int grid = (int)((n + 255) / 256);
    if (prec == LQ_FP64) cv_fill_kernel<double><<<grid, 256, 0, c->stream>>>((double*)native, n, seed);
    else cv_fill_kernel<float><<<grid, 256, 0, c->stream>>>((float*)native, n, seed);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
