// common.cuh -- geometry, native-layout accessors and the context of the CUDA path.
// Native layout: SURVEY.md 8(a) "Native layout" (even/odd checkerboards, SoA, RHS innermost).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>
#include "../../include/lqcd_b200.h"

// ------------------------------------------------------------------ geometry
struct Geom {
    int L[4];      // Lx, Ly, Lz, Lt
    int Lxh;       // Lx / 2
    int Vh;        // sites per parity
    long long V;   // all sites
};

// checkerboard index -> coordinates.  cb = xh + Lxh*(y + Ly*(z + Lz*t)), x = 2*xh + ((y+z+t+parity)&1)
__host__ __device__ inline void cb_coords(const Geom& g, int parity, int cb, int& xh, int& y, int& z, int& t, int& odd) {
    xh = cb % g.Lxh; int r = cb / g.Lxh;
    y = r % g.L[1]; r /= g.L[1];
    z = r % g.L[2]; t = r / g.L[2];
    odd = (y + z + t + parity) & 1;
}
// full coordinates -> (parity, cb)
__host__ __device__ inline void coords_to_cb(const Geom& g, int x, int y, int z, int t, int& parity, int& cb) {
    parity = (x + y + z + t) & 1;
    cb = (x >> 1) + g.Lxh * (y + g.L[1] * (z + g.L[2] * t));
}

// ------------------------------------------------------------------ storage traits
struct F64 { using store_t = double; using comp_t = double; static constexpr int prec = LQ_FP64; static constexpr bool has_norm = false; };
struct F32 { using store_t = float;  using comp_t = float;  static constexpr int prec = LQ_FP32; static constexpr bool has_norm = false; };
struct H16 { using store_t = short;  using comp_t = float;  static constexpr int prec = LQ_HALF; static constexpr bool has_norm = true; };

// one parity of a native spinor batch
template <class S> struct SView {
    typename S::store_t* d;   // payload [24][Vh][N]
    float* n;                 // norms [Vh][N] (H16 only)
};

inline size_t elem_bytes(int prec) { return prec == LQ_FP64 ? 8 : (prec == LQ_FP32 ? 4 : 2); }
inline size_t round256(size_t b) { return (b + 255) & ~size_t(255); }
// bytes of one parity block of a native spinor batch
inline size_t parity_bytes(const Geom& g, int nrhs, int prec) {
    size_t pay = round256((size_t)24 * g.Vh * nrhs * elem_bytes(prec));
    if (prec == LQ_HALF) pay += round256((size_t)g.Vh * nrhs * sizeof(float));
    return pay;
}
template <class S> inline SView<S> make_view(const Geom& g, void* base, int nrhs, int parity_block) {
    char* p = (char*)base + (size_t)parity_block * parity_bytes(g, nrhs, S::prec);
    SView<S> v;
    v.d = (typename S::store_t*)p;
    v.n = S::has_norm ? (float*)(p + round256((size_t)24 * g.Vh * nrhs * elem_bytes(S::prec))) : nullptr;
    return v;
}

// ------------------------------------------------------------------ vector-plane storage of per-site constants
// A per-site record of R reals (link: 18 or 12, clover: 72) is stored as planes of VL = 16/sizeof(T)
// reals: plane q holds reals [q*VL, q*VL+VL) of every site, offset q*VL*Vh + cb*VL; a remainder of
// R % VL reals (2 for an 18-real fp32 link) forms a last, narrower plane.  All lanes of a warp that
// work on consecutive sites read consecutive 16-byte vectors; lanes that share a site broadcast.
template <typename T> struct VecOf;
template <> struct VecOf<float>  { using v_t = float4;  static constexpr int VL = 4; };
template <> struct VecOf<double> { using v_t = double2; static constexpr int VL = 2; };

template <typename T, int R>
__device__ __forceinline__ void load_planes(const T* __restrict__ base, int Vh, int cb, T* out) {
    constexpr int VL = VecOf<T>::VL;
    constexpr int NF = R / VL;
    constexpr int REM = R - NF * VL;
#pragma unroll
    for (int q = 0; q < NF; q++) {
        if constexpr (VL == 4) {
            float4 v = __ldg(reinterpret_cast<const float4*>(base + (size_t)q * 4 * Vh) + cb);
            out[4 * q] = v.x; out[4 * q + 1] = v.y; out[4 * q + 2] = v.z; out[4 * q + 3] = v.w;
        } else {
            double2 v = __ldg(reinterpret_cast<const double2*>(base + (size_t)q * 2 * Vh) + cb);
            out[2 * q] = v.x; out[2 * q + 1] = v.y;
        }
    }
    if constexpr (REM == 2) {
        float2 v = __ldg(reinterpret_cast<const float2*>(base + (size_t)NF * VL * Vh) + cb);
        out[NF * VL] = v.x; out[NF * VL + 1] = v.y;
    }
}
template <typename T, int R>
__device__ __forceinline__ void store_planes(T* __restrict__ base, int Vh, int cb, const T* in) {
    constexpr int VL = VecOf<T>::VL;
    constexpr int NF = R / VL;
    constexpr int REM = R - NF * VL;
#pragma unroll
    for (int q = 0; q < NF; q++)
#pragma unroll
        for (int e = 0; e < VL; e++) base[(size_t)q * VL * Vh + (size_t)cb * VL + e] = in[q * VL + e];
#pragma unroll
    for (int e = 0; e < REM; e++) base[(size_t)NF * VL * Vh + (size_t)cb * REM + e] = in[NF * VL + e];
}

// ------------------------------------------------------------------ context
struct lq_ctx {
    Geom g;
    int device;
    cudaStream_t stream;
    int t_bc;
    // gauge: [parity][mu] blocks of R*Vh reals
    double* gauge64;  // R = 18
    float* gauge32;   // R = recon32
    int recon32;
    // clover: [parity] blocks of 72*Vh reals; A and A^{-1}
    double *clov64, *clovinv64;
    float *clov32, *clovinv32;
    double kappa, csw;
    bool has_gauge, has_clover;
    lq_alloc_fn alloc_fn; lq_free_fn free_fn; void* alloc_user;
    std::vector<void*> owned;       // everything from dev_alloc still alive
    long long launches;
    int dslash_block;               // tuning knob (0 = default)
    int dslash_rpt;                 // tuning knob (0 = auto)
    std::string err;
    // reduction scratch
    double* red_partials; size_t red_partials_elems;
    unsigned int* red_counter;
    double* h_scalars;              // pinned host, 8*LQ_MAX_RHS doubles
    int* d_flag;                    // device error flag
};

int set_err(lq_ctx* c, int code, const std::string& msg);
void* dev_alloc(lq_ctx* c, size_t bytes);          // nullptr on failure (error recorded)
void dev_free(lq_ctx* c, void* p);

#define LQ_CUDA(ctx, call)                                                                     \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess) return set_err(ctx, LQ_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
    } while (0)
#define LQ_TRY(x) do { int r_ = (x); if (r_ != 0) return r_; } while (0)
#define LQ_LAUNCHED(ctx) do { (ctx)->launches++; } while (0)

inline const double* gauge64_block(const lq_ctx* c, int parity, int mu) { return c->gauge64 + ((size_t)(parity * 4 + mu)) * 18 * c->g.Vh; }
inline const float* gauge32_block(const lq_ctx* c, int parity, int mu) { return c->gauge32 + ((size_t)(parity * 4 + mu)) * c->recon32 * c->g.Vh; }
