// common.cuh -- geometry, native-layout accessors and the context of the CUDA path.
// Native layout: SURVEY.md 8(a) "Native layout" (even/odd checkerboards, SoA, RHS innermost).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>
#include "../../include/lqcd_b200.h"

// ------------------------------------------------------------------ geometry
constexpr int SB = 32;   // sites per native block (one warp-wide row of every plane)
constexpr int LQ_DEFAULT_PFD = 64;    // default L2 prefetch distance of the stencil kernels, in site blocks

// division of a non-negative int < 2^31 by a fixed positive divisor: q = (umulhi(m, n) + n) >> l  (Granlund-Montgomery)
struct FastDiv {
    unsigned m, l;
    __host__ __device__ inline int div(int n) const {
#ifdef __CUDA_ARCH__
        return (int)((__umulhi(m, (unsigned)n) + (unsigned)n) >> l);
#else
        return (int)(((unsigned)(((unsigned long long)m * (unsigned)n) >> 32) + (unsigned)n) >> l);
#endif
    }
};
inline FastDiv make_fastdiv(int d) {
    FastDiv f; unsigned l = 0;
    while ((1u << l) < (unsigned)d) l++;
    f.l = l;
    f.m = (unsigned)((((unsigned long long)1 << 32) * ((1ull << l) - (unsigned)d)) / (unsigned)d + 1);
    return f;
}

struct Geom {
    FastDiv dLxh, dLy, dLz;   // divisions by Lx/2, Ly, Lz
    int L[4];      // Lx, Ly, Lz, Lt
    int Lxh;       // Lx / 2
    int Vh;        // sites per parity
    int NB;        // native site blocks per parity = ceil(Vh / SB); sites cb >= Vh of the last block are padding
    long long V;   // all sites
};

// checkerboard index -> coordinates.  cb = xh + Lxh*(y + Ly*(z + Lz*t)), x = 2*xh + ((y+z+t+parity)&1)
__host__ __device__ inline void cb_coords(const Geom& g, int parity, int cb, int& xh, int& y, int& z, int& t, int& odd) {
    int r = g.dLxh.div(cb); xh = cb - r * g.Lxh;
    int q = g.dLy.div(r); y = r - q * g.L[1];
    t = g.dLz.div(q); z = q - t * g.L[2];
    odd = (y + z + t + parity) & 1;
}
// full coordinates -> (parity, cb)
__host__ __device__ inline void coords_to_cb(const Geom& g, int x, int y, int z, int t, int& parity, int& cb) {
    parity = (x + y + z + t) & 1;
    cb = (x >> 1) + g.Lxh * (y + g.L[1] * (z + g.L[2] * t));
}

// ------------------------------------------------------------------ storage traits
// link_t: storage type of the gauge links the stencil kernels read
struct F64 { using store_t = double; using comp_t = double; using link_t = double; static constexpr int prec = LQ_FP64; static constexpr bool has_norm = false; };
struct F32 { using store_t = float;  using comp_t = float;  using link_t = float;  static constexpr int prec = LQ_FP32; static constexpr bool has_norm = false; };
struct H16 { using store_t = short;  using comp_t = float;  using link_t = float;  static constexpr int prec = LQ_HALF; static constexpr bool has_norm = true; };
// half-storage spinors AND int16 fixed-point links (SURVEY 8(f) #3, 8(c.2) reading #13: entries of an SU(3) matrix lie in [-1, 1],
// q = rint(32767 u), no norm needed): 36 instead of 72 bytes per link
struct H16L { using store_t = short; using comp_t = float;  using link_t = short;  static constexpr int prec = LQ_HALF; static constexpr bool has_norm = true; };

// ------------------------------------------------------------------ native spinor layout (one parity, N right-hand sides)
// The batch is cut into G = N/R groups of R = 4 (N % 4 == 0), 2 (N even) or 1 consecutive right-hand sides and the
// sites into blocks of SB = 32 consecutive checkerboard sites:
//     payload[blk][g][j = 0..23][s = 0..31][r = 0..R-1]      real j = 2*(3*spin + colour) + (re|im)
//     norm   [blk][g][s][r]                                   (half storage only)
// The RHS index is innermost (BASELINE.json north_star, layout item 1): a thread that owns (site, group) reads one
// 16-byte vector per real (R = 4, fp32), a warp reads one contiguous 512-byte row, and every row of a neighbour
// unit sits at a COMPILE-TIME offset j*SB*R from the unit base, so the 24 loads of a neighbour share one address.
__host__ __device__ inline int group_width(int N) { return (N % 4 == 0) ? 4 : ((N % 2 == 0) ? 2 : 1); }

// one parity of a native spinor batch
template <class S> struct SView {
    typename S::store_t* d;   // payload
    float* n;                 // norms (H16 only)
};
// element offset of (rhs k, site cb, real j) in the payload, and of (k, cb) in the norms
__host__ __device__ inline size_t sp_index(int N, int cb, int k, int j) {
    const int R = group_width(N), G = N / R;
    const size_t u = (size_t)(cb / SB) * G + k / R;
    return (u * 24 + j) * (SB * R) + (size_t)(cb % SB) * R + k % R;
}
__host__ __device__ inline size_t nrm_index(int N, int cb, int k) {
    const int R = group_width(N), G = N / R;
    const size_t u = (size_t)(cb / SB) * G + k / R;
    return u * (SB * R) + (size_t)(cb % SB) * R + k % R;
}

inline size_t elem_bytes(int prec) { return prec == LQ_FP64 ? 8 : (prec == LQ_FP32 ? 4 : 2); }
inline size_t round256(size_t b) { return (b + 255) & ~size_t(255); }
// bytes of one parity block of a native spinor batch (padded to whole site blocks)
inline size_t parity_bytes(const Geom& g, int nrhs, int prec) {
    size_t pay = round256((size_t)24 * g.NB * SB * nrhs * elem_bytes(prec));
    if (prec == LQ_HALF) pay += round256((size_t)g.NB * SB * nrhs * sizeof(float));
    return pay;
}
// algorithmic bytes of one pass over one parity of a batch (payload + norms)
inline double stream_bytes(const Geom& g, int nrhs, int prec) { return (double)g.Vh * nrhs * (24.0 * elem_bytes(prec) + (prec == LQ_HALF ? 4.0 : 0.0)); }
template <class S> inline SView<S> make_view(const Geom& g, void* base, int nrhs, int parity_block) {
    char* p = (char*)base + (size_t)parity_block * parity_bytes(g, nrhs, S::prec);
    SView<S> v;
    v.d = (typename S::store_t*)p;
    v.n = S::has_norm ? (float*)(p + round256((size_t)24 * g.NB * SB * nrhs * elem_bytes(S::prec))) : nullptr;
    return v;
}

// ------------------------------------------------------------------ blocked vector-plane storage of per-site constants
// A per-site record of R reals (link: 18 or 12, clover: 72) of the SB sites of one block is stored as planes of
// VL = 16/sizeof(T) reals: plane q holds reals [q*VL, q*VL+VL) of the 32 sites (offset q*VL*SB + s*VL); a remainder
// of R % VL reals (2 for an 18-real fp32 link) forms a last, narrower plane.  All offsets inside a block are
// compile-time constants; a warp working on the 32 sites of a block reads 512 contiguous bytes per plane.
//   gauge : [parity][blk][mu][planes][s]      block of (parity, blk) = 4*RECON*SB reals
//   clover: [parity][blk][planes][s]          block = 72*SB reals
template <typename T> struct VecOf;
template <> struct VecOf<float>  { using v_t = float4;  static constexpr int VL = 4; };
template <> struct VecOf<double> { using v_t = double2; static constexpr int VL = 2; };

// SMEM: blockbase points into shared memory (a staged copy of the block, same plane layout): plain loads instead of ld.global.nc
template <typename T, int R, bool SMEM = false>
__device__ __forceinline__ void load_planes(const T* __restrict__ blockbase, int s, T* out) {
    constexpr int VL = VecOf<T>::VL;
    constexpr int NF = R / VL;
    constexpr int REM = R - NF * VL;
#pragma unroll
    for (int q = 0; q < NF; q++) {
        if constexpr (VL == 4) {
            const float4* p = reinterpret_cast<const float4*>(blockbase + q * 4 * SB) + s;
            float4 v;
            if constexpr (SMEM) v = *p; else v = __ldg(p);
            out[4 * q] = v.x; out[4 * q + 1] = v.y; out[4 * q + 2] = v.z; out[4 * q + 3] = v.w;
        } else {
            const double2* p = reinterpret_cast<const double2*>(blockbase + q * 2 * SB) + s;
            double2 v;
            if constexpr (SMEM) v = *p; else v = __ldg(p);
            out[2 * q] = v.x; out[2 * q + 1] = v.y;
        }
    }
    if constexpr (REM == 2) {
        const float2* p = reinterpret_cast<const float2*>(blockbase + NF * VL * SB) + s;
        float2 v;
        if constexpr (SMEM) v = *p; else v = __ldg(p);
        out[NF * VL] = v.x; out[NF * VL + 1] = v.y;
    }
}
template <typename T, int R>
__device__ __forceinline__ void store_planes(T* __restrict__ blockbase, int s, const T* in) {
    constexpr int VL = VecOf<T>::VL;
    constexpr int NF = R / VL;
    constexpr int REM = R - NF * VL;
#pragma unroll
    for (int q = 0; q < NF; q++)
#pragma unroll
        for (int e = 0; e < VL; e++) blockbase[q * VL * SB + s * VL + e] = in[q * VL + e];
#pragma unroll
    for (int e = 0; e < REM; e++) blockbase[NF * VL * SB + s * REM + e] = in[NF * VL + e];
}
// base of the link block of (parity, site block, mu) / of the clover block of (parity, site block)
template <typename T> __host__ __device__ inline T* link_block(T* gauge, int NB, int recon, int parity, int blk, int mu) {
    return gauge + ((size_t)(parity * NB + blk) * 4 + mu) * (size_t)(recon * SB);
}
template <typename T> __host__ __device__ inline T* clover_block(T* clov, int NB, int parity, int blk) {
    return clov + (size_t)(parity * NB + blk) * (size_t)(72 * SB);
}

// ------------------------------------------------------------------ context
struct lq_ctx {
    Geom g;
    int device;
    cudaStream_t stream;
    int t_bc;
    // gauge: [parity][blk][mu] blocks of R*SB reals
    double* gauge64;  // R = 18
    float* gauge32;   // R = recon32
    int recon32;
    short* gauge16;   // int16 copy of the 18-real links (lq_set_half_links), or nullptr
    bool half_links;  // LQ_HALF stencil kernels read gauge16
    // clover: [parity][blk] blocks of 72*SB reals; A and A^{-1}
    double *clov64, *clovinv64;
    float *clov32, *clovinv32;
    double kappa, csw;
    bool has_gauge, has_clover;
    lq_alloc_fn alloc_fn; lq_free_fn free_fn; void* alloc_user;
    std::vector<void*> owned;       // everything from dev_alloc still alive
    long long launches;
    int dslash_rpt;                 // tuning knob (0 = auto)
    int dslash_variant;             // tuning knob: kernel variant (0 = default)
    int dslash_pfd;                 // tuning knob: L2 prefetch distance in site blocks (0 = off)
    int dslash_zc;                  // tuning knob: z-chunk of the sweep order (0 = auto, -1 = memory order)
    std::string err;
    // reduction scratch
    double* red_partials; size_t red_partials_elems;
    unsigned int* red_counter;
    double* h_scalars;              // pinned host, 8*LQ_MAX_RHS doubles
    int* d_flag;                    // device error flag
    // solver state (solver.cu): workspace with the cached iteration graph, owned by the context
    struct SolverWorkspace* ws;
    // two-level multigrid hierarchy (multigrid.cu), or nullptr
    struct MgState* mg;
    // while the solver enqueues the body of an inner iteration: device flag that makes every kernel of the body return
    // at once when set (the inner solve has converged; launches already queued behind the flag become no-ops)
    const int* loop_skip;
    // modelled work of everything launched so far (SURVEY 8(d) byte / flop model; lq_solve_info)
    double model_bytes, model_flops;
    // projection scratch kept between calls (project_tc.cu)
    void* proj_scratch; size_t proj_scratch_bytes;
};

int set_err(lq_ctx* c, int code, const std::string& msg);
void* dev_alloc(lq_ctx* c, size_t bytes);          // nullptr on failure (error recorded)
void dev_free(lq_ctx* c, void* p);
// second stage of the deterministic reductions (reduce.cuh, blas.cu): its one self-resetting counter sits behind the first 64
// words of lq_ctx::red_counter (flags)
constexpr int RED_COUNTER_BASE = 64;
constexpr size_t RED_COUNTER_BYTES = (size_t)(RED_COUNTER_BASE + 64) * sizeof(unsigned int);
int ensure_partials(lq_ctx* c, size_t elems);      // reduction scratch of at least `elems` doubles

#define LQ_CUDA(ctx, call)                                                                     \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess) return set_err(ctx, LQ_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
    } while (0)
#define LQ_TRY(x) do { int r_ = (x); if (r_ != 0) return r_; } while (0)
#define LQ_LAUNCHED(ctx) do { (ctx)->launches++; } while (0)
// modelled (algorithmic) bytes and counted flops of one launch
#define LQ_MODEL(ctx, bytes, flops) do { (ctx)->model_bytes += (double)(bytes); (ctx)->model_flops += (double)(flops); } while (0)

