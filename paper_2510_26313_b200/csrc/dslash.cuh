// dslash.cuh -- the fused single-parity Wilson-clover stencil kernels.
//
//   FORM_HOP : out = D in
//   FORM_A   : out = C (D in)            C = A^{-1} of the output parity      ("kernel A")
//   FORM_B   : out = C x + coef (D in)   C = A of the output parity or 1      ("kernel B")
// with D replaced by g5 D g5 when dsign = -1 (dagger, row a5: only the projector signs flip because the
// clover blocks commute with g5 = diag(1,1,-1,-1)).
//
// Thread mapping on the blocked native layout (common.cuh): a "unit" is (site block of 32 sites, RHS group of
// R right-hand sides).  One thread owns one output site and RPT consecutive right-hand sides of the group
// (RPT divides R; R/RPT adjacent lanes share a site).  With RPT = R = 4 (fp32) a warp is exactly one unit: every
// real of a neighbour is one 16-byte load per lane, 512 contiguous bytes per warp, at a compile-time offset from
// ONE per-neighbour address; the link and the clover block of the site are loaded once per thread as 16-byte
// vectors and reused in registers across the thread's right-hand sides (the paper's stencil-coefficient reuse,
// PAPER.md L136); the other RHS groups of the same sites run in adjacent warps and find the links in L1.
// All complex arithmetic is written as explicit fused multiply-adds (1128 FP instructions per site per RHS for
// kernel A: 8 x (12 project + 72 SU(3) + 24 accumulate) + 264 clover).  Spin projection uses the DeGrand-Rossi
// rank-2 structure of (1 -+ gamma_mu); boundaries are wrapped in-kernel and the antiperiodic sign multiplies the
// hopped term (never the stored link, so 12-real reconstruction stays valid).
#pragma once
#include "common.cuh"

enum { FORM_HOP = 0, FORM_A = 1, FORM_B = 2, FORM_PROBE = 3 };   // FORM_PROBE: kernel A's memory accesses with trivial arithmetic (bench only)
// fused epilogues of kernel B: per-RHS ||out||^2, or out <- out - (num/den)_k * result with per-RHS ||out||^2
// or (EPI_CDOT, BiCGStab) the complex inner product of a vector h with the result: (Re, Im <h, out>, ||out||^2), Im negated if epi_conj
enum { EPI_NONE = 0, EPI_NORM = 1, EPI_XMAY = 2, EPI_CDOT = 3 };

template <class S> struct DslashArgs {
    using T = typename S::comp_t;
    Geom g;
    int parity;            // parity of the output sites
    int N, G;              // right-hand sides, RHS groups (N / R)
    FastDiv dG;            // division by G
    SView<S> out, in, x;   // out / x on `parity`, in on 1-parity
    const typename S::link_t* gauge;   // [parity][blk][mu] blocks of RECON*SB reals (fp64 / fp32, or int16 fixed point for H16L)
    const T* clover;       // [blk] blocks of 72*SB reals of the output parity, or nullptr (identity)
    T coef;                // FORM_B
    T tsign;               // t_bc
    T dsign;               // +1, -1 = dagger
    int pfd;               // L2 prefetch distance in site blocks (0 = off)
    // sweep order: launch-order block index -> site block, [z chunk][t][z in chunk][y-x blocks], so that the three
    // time-slices a chunk needs stay in L2 between their uses (zc = 0: memory order)
    int zc, nby; FastDiv dnby, dzc, dLt;
    int epi;               // FORM_B epilogue
    const double *epi_num, *epi_den;   // EPI_XMAY: alpha_k = num_k / den_k (device, per RHS)
    double* epi_out;                   // per-RHS sums (device); EPI_CDOT: 3 x LQ_MAX_RHS
    SView<S> epi_v; int epi_conj;      // EPI_CDOT: h (on `parity`), conjugate the inner product
    double* red_partials; unsigned int* red_counter;   // reduction scratch of the context
    const int* skip;       // device flag or nullptr: when set the launch is a no-op (lq_ctx::loop_skip, solver.cu)
};

__device__ __forceinline__ float fm(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double fm(double a, double b, double c) { return fma(a, b, c); }

// two int16 packed in a 32-bit word -> two floats
__device__ __forceinline__ void s16x2_to_f32(unsigned w, float& lo, float& hi) {
    int a, b;
    asm("prmt.b32 %0, %1, 0, 0x9910;" : "=r"(a) : "r"(w));   // bytes b0 b1 sign(b1) sign(b1)
    asm("prmt.b32 %0, %1, 0, 0xBB32;" : "=r"(b) : "r"(w));   // bytes b2 b3 sign(b3) sign(b3)
    lo = (float)a; hi = (float)b;
}

// ---- RPT-wide loads / stores of one real of one site ------------------------------------------------
template <class S, int RPT>
__device__ __forceinline__ void load_comp(const typename S::store_t* __restrict__ p, typename S::comp_t* o) {
    if constexpr (S::prec == LQ_FP32) {
        if constexpr (RPT == 4) { float4 v = __ldg((const float4*)p); o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w; }
        else if constexpr (RPT == 2) { float2 v = __ldg((const float2*)p); o[0] = v.x; o[1] = v.y; }
        else { o[0] = __ldg(p); }
    } else if constexpr (S::prec == LQ_FP64) {
        if constexpr (RPT == 4) {
            double2 v = __ldg((const double2*)p), w = __ldg((const double2*)p + 1);
            o[0] = v.x; o[1] = v.y; o[2] = w.x; o[3] = w.y;
        } else if constexpr (RPT == 2) { double2 v = __ldg((const double2*)p); o[0] = v.x; o[1] = v.y; }
        else { o[0] = __ldg(p); }
    } else {
        // int16 -> fp32 as byte-permute sign extension + I2FP.F32.S32 (full rate); the direct I2F.S16 form that the
        // compiler picks for (float)short runs on the 16-lane conversion unit and made this kernel slower than fp32
        if constexpr (RPT == 4) { uint2 v = __ldg((const uint2*)p); s16x2_to_f32(v.x, o[0], o[1]); s16x2_to_f32(v.y, o[2], o[3]); }
        else if constexpr (RPT == 2) { unsigned v = __ldg((const unsigned*)p); s16x2_to_f32(v, o[0], o[1]); }
        else { int v = __ldg(p); int w; asm("mov.b32 %0, %1;" : "=r"(w) : "r"(v)); o[0] = (float)w; }
    }
}
template <int RPT> __device__ __forceinline__ void load_norm(const float* __restrict__ p, float* o) {
    if constexpr (RPT == 4) { float4 v = __ldg((const float4*)p); o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w; }
    else if constexpr (RPT == 2) { float2 v = __ldg((const float2*)p); o[0] = v.x; o[1] = v.y; }
    else { o[0] = __ldg(p); }
}
template <int RPT> __device__ __forceinline__ void store_norm(float* __restrict__ p, const float* o) {
    if constexpr (RPT == 4) *(float4*)p = make_float4(o[0], o[1], o[2], o[3]);
    else if constexpr (RPT == 2) *(float2*)p = make_float2(o[0], o[1]);
    else *p = o[0];
}
template <class S, int RPT>
__device__ __forceinline__ void store_comp(typename S::store_t* __restrict__ p, const typename S::comp_t* o) {
    if constexpr (S::prec == LQ_FP32) {
        if constexpr (RPT == 4) *(float4*)p = make_float4(o[0], o[1], o[2], o[3]);
        else if constexpr (RPT == 2) *(float2*)p = make_float2(o[0], o[1]);
        else *p = o[0];
    } else if constexpr (S::prec == LQ_FP64) {
        if constexpr (RPT == 4) { *(double2*)p = make_double2(o[0], o[1]); *((double2*)p + 1) = make_double2(o[2], o[3]); }
        else if constexpr (RPT == 2) *(double2*)p = make_double2(o[0], o[1]);
        else *p = o[0];
    } else {
        if constexpr (RPT == 4) *(short4*)p = make_short4((short)o[0], (short)o[1], (short)o[2], (short)o[3]);
        else if constexpr (RPT == 2) *(short2*)p = make_short2((short)o[0], (short)o[1]);
        else *p = (short)o[0];
    }
}

// ---- link load (+ 12-real reconstruction: third row = conj(row0 x row1)) -----------------------------
template <typename T, int RECON, bool SMEM = false>
__device__ __forceinline__ void load_link(const T* __restrict__ blockbase, int s, T* u) {
    load_planes<T, RECON, SMEM>(blockbase, s, u);
    if constexpr (RECON == 12) {
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
            // (a x b)_c = a_c1 b_c2 - a_c2 b_c1, conjugated
            T re = u[2 * c1] * u[6 + 2 * c2];
            re = fm(-u[2 * c1 + 1], u[6 + 2 * c2 + 1], re);
            re = fm(-u[2 * c2], u[6 + 2 * c1], re);
            re = fm(u[2 * c2 + 1], u[6 + 2 * c1 + 1], re);
            T im = u[2 * c1] * u[6 + 2 * c2 + 1];
            im = fm(u[2 * c1 + 1], u[6 + 2 * c2], im);
            im = fm(-u[2 * c2], u[6 + 2 * c1 + 1], im);
            im = fm(-u[2 * c2 + 1], u[6 + 2 * c1], im);
            u[12 + 2 * c] = re; u[12 + 2 * c + 1] = -im;
        }
    }
}

// int16 fixed-point links (H16L): the 18 values of a site are two 16-byte planes of 8 int16 and one 4-byte plane of 2
__device__ __forceinline__ void load_link(const short* __restrict__ blockbase, int s, float* u) {
    const uint4 a = __ldg(reinterpret_cast<const uint4*>(blockbase) + s);
    const uint4 b = __ldg(reinterpret_cast<const uint4*>(blockbase + 8 * SB) + s);
    const unsigned c = __ldg(reinterpret_cast<const unsigned*>(blockbase + 16 * SB) + s);
    s16x2_to_f32(a.x, u[0], u[1]); s16x2_to_f32(a.y, u[2], u[3]); s16x2_to_f32(a.z, u[4], u[5]); s16x2_to_f32(a.w, u[6], u[7]);
    s16x2_to_f32(b.x, u[8], u[9]); s16x2_to_f32(b.y, u[10], u[11]); s16x2_to_f32(b.z, u[12], u[13]); s16x2_to_f32(b.w, u[14], u[15]);
    s16x2_to_f32(c, u[16], u[17]);
#pragma unroll
    for (int i = 0; i < 18; i++) u[i] *= (1.0f / 32767.0f);
}

// ---- SU(3) x projected half spinor, spin reconstruction and accumulation --------------------------------
// acc += cuk * (upper rows) and +-clk * (lower rows) of (1 - sigma gamma_MU) W h,  W = U (FWD) or U^dag.
template <typename T, int RPT, int MU, bool FWD>
__device__ __forceinline__ void hop_mulacc(const T (&h)[2][3][2][RPT], const T (&u)[18], const T (&cuk)[RPT], const T (&clk)[RPT],
                                           T (&acc)[24][RPT]) {
#pragma unroll
    for (int s = 0; s < 2; s++)
#pragma unroll
        for (int r = 0; r < 3; r++) {
            T wr[RPT], wi[RPT];
#pragma unroll
            for (int c = 0; c < 3; c++) {
                // FWD: U[r][c];  backward: conj(U[c][r])
                const T ur = FWD ? u[2 * (3 * r + c)] : u[2 * (3 * c + r)];
                const T ui = FWD ? u[2 * (3 * r + c) + 1] : -u[2 * (3 * c + r) + 1];
#pragma unroll
                for (int k = 0; k < RPT; k++) {
                    if (c == 0) { wr[k] = ur * h[s][c][0][k]; wi[k] = ur * h[s][c][1][k]; }
                    else { wr[k] = fm(ur, h[s][c][0][k], wr[k]); wi[k] = fm(ur, h[s][c][1][k], wi[k]); }
                    wr[k] = fm(-ui, h[s][c][1][k], wr[k]);
                    wi[k] = fm(ui, h[s][c][0][k], wi[k]);
                }
            }
            // upper spin rows: acc_s += cu w_s
            const int ju = 2 * (3 * s + r);
#pragma unroll
            for (int k = 0; k < RPT; k++) { acc[ju][k] = fm(cuk[k], wr[k], acc[ju][k]); acc[ju + 1][k] = fm(cuk[k], wi[k], acc[ju + 1][k]); }
            // lower spin rows (reconstruction)
            if constexpr (MU == 0) {        // row2 = (s i) w1, row3 = (s i) w0
                const int jl = 2 * (3 * (3 - s) + r);
#pragma unroll
                for (int k = 0; k < RPT; k++) { acc[jl][k] = fm(-clk[k], wi[k], acc[jl][k]); acc[jl + 1][k] = fm(clk[k], wr[k], acc[jl + 1][k]); }
            } else if constexpr (MU == 1) { // row2 = -s w1, row3 = +s w0
                const int jl = 2 * (3 * (3 - s) + r);
                if (s == 0) {
#pragma unroll
                    for (int k = 0; k < RPT; k++) { acc[jl][k] = fm(clk[k], wr[k], acc[jl][k]); acc[jl + 1][k] = fm(clk[k], wi[k], acc[jl + 1][k]); }
                } else {
#pragma unroll
                    for (int k = 0; k < RPT; k++) { acc[jl][k] = fm(-clk[k], wr[k], acc[jl][k]); acc[jl + 1][k] = fm(-clk[k], wi[k], acc[jl + 1][k]); }
                }
            } else if constexpr (MU == 2) { // row2 = (s i) w0, row3 = -(s i) w1
                const int jl = 2 * (3 * (2 + s) + r);
                if (s == 0) {
#pragma unroll
                    for (int k = 0; k < RPT; k++) { acc[jl][k] = fm(-clk[k], wi[k], acc[jl][k]); acc[jl + 1][k] = fm(clk[k], wr[k], acc[jl + 1][k]); }
                } else {
#pragma unroll
                    for (int k = 0; k < RPT; k++) { acc[jl][k] = fm(clk[k], wi[k], acc[jl][k]); acc[jl + 1][k] = fm(-clk[k], wr[k], acc[jl + 1][k]); }
                }
            } else {                        // row2 = -s w0, row3 = -s w1
                const int jl = 2 * (3 * (2 + s) + r);
#pragma unroll
                for (int k = 0; k < RPT; k++) { acc[jl][k] = fm(-clk[k], wr[k], acc[jl][k]); acc[jl + 1][k] = fm(-clk[k], wi[k], acc[jl + 1][k]); }
            }
        }
}

// ---- packed-FP32 variant of hop_mulacc for 2 right-hand sides per thread (sm_100 FFMA2: one instruction = the same FMA
// on both right-hand sides; the link element is duplicated into a register pair).  Same arithmetic, same rounding.
#ifdef LQ_USE_FFMA2
template <int RPT, int MU, bool FWD>
__device__ __forceinline__ void hop_mulacc_f2(const float (&h)[2][3][2][RPT], const float (&u)[18], const float (&cuk)[RPT], const float (&clk)[RPT],
                                              float (&acc)[24][RPT]) {
#pragma unroll
  for (int k0 = 0; k0 < RPT; k0 += 2) {
    const float2 cu2 = make_float2(cuk[k0], cuk[k0 + 1]), cl2 = make_float2(clk[k0], clk[k0 + 1]), ncl2 = make_float2(-clk[k0], -clk[k0 + 1]);
#define A2(j) make_float2(acc[j][k0], acc[j][k0 + 1])
#define SETA(j, v) { const float2 t_ = (v); acc[j][k0] = t_.x; acc[j][k0 + 1] = t_.y; }
#pragma unroll
    for (int r = 0; r < 3; r++) {
        float2 wr[2], wi[2];
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const float ur = FWD ? u[2 * (3 * r + c)] : u[2 * (3 * c + r)];
            const float ui = FWD ? u[2 * (3 * r + c) + 1] : -u[2 * (3 * c + r) + 1];
            const float2 ur2 = make_float2(ur, ur), ui2 = make_float2(ui, ui), nui2 = make_float2(-ui, -ui);
#pragma unroll
            for (int s = 0; s < 2; s++) {
                const float2 hr = make_float2(h[s][c][0][k0], h[s][c][0][k0 + 1]), hi = make_float2(h[s][c][1][k0], h[s][c][1][k0 + 1]);
                if (c == 0) { wr[s] = __fmul2_rn(ur2, hr); wi[s] = __fmul2_rn(ur2, hi); }
                else { wr[s] = __ffma2_rn(ur2, hr, wr[s]); wi[s] = __ffma2_rn(ur2, hi, wi[s]); }
                wr[s] = __ffma2_rn(nui2, hi, wr[s]);
                wi[s] = __ffma2_rn(ui2, hr, wi[s]);
            }
        }
#pragma unroll
        for (int s = 0; s < 2; s++) {
            const int ju = 2 * (3 * s + r);
            SETA(ju, __ffma2_rn(cu2, wr[s], A2(ju))) SETA(ju + 1, __ffma2_rn(cu2, wi[s], A2(ju + 1)))
            if constexpr (MU == 0) {
                const int jl = 2 * (3 * (3 - s) + r);
                SETA(jl, __ffma2_rn(ncl2, wi[s], A2(jl))) SETA(jl + 1, __ffma2_rn(cl2, wr[s], A2(jl + 1)))
            } else if constexpr (MU == 1) {
                const int jl = 2 * (3 * (3 - s) + r);
                if (s == 0) { SETA(jl, __ffma2_rn(cl2, wr[s], A2(jl))) SETA(jl + 1, __ffma2_rn(cl2, wi[s], A2(jl + 1))) }
                else { SETA(jl, __ffma2_rn(ncl2, wr[s], A2(jl))) SETA(jl + 1, __ffma2_rn(ncl2, wi[s], A2(jl + 1))) }
            } else if constexpr (MU == 2) {
                const int jl = 2 * (3 * (2 + s) + r);
                if (s == 0) { SETA(jl, __ffma2_rn(ncl2, wi[s], A2(jl))) SETA(jl + 1, __ffma2_rn(cl2, wr[s], A2(jl + 1))) }
                else { SETA(jl, __ffma2_rn(cl2, wi[s], A2(jl))) SETA(jl + 1, __ffma2_rn(ncl2, wr[s], A2(jl + 1))) }
            } else {
                const int jl = 2 * (3 * (2 + s) + r);
                SETA(jl, __ffma2_rn(ncl2, wr[s], A2(jl))) SETA(jl + 1, __ffma2_rn(ncl2, wi[s], A2(jl + 1)))
            }
        }
    }
#undef A2
#undef SETA
  }
}
#endif

// ---- spin projection of one colour: h[s][c] = rows of (1 - sigma gamma_MU) p, DeGrand-Rossi rank-2 structure ------------------
template <typename T, int RPT, int MU>
__device__ __forceinline__ void project_half(const T (&p)[4][2][RPT], T sigma, int c, T (&h)[2][3][2][RPT]) {
#ifdef LQ_USE_FFMA2
        if constexpr (sizeof(T) == 4 && RPT % 2 == 0) {
#pragma unroll
            for (int k = 0; k < RPT; k += 2) {
                const float2 sg = make_float2(sigma, sigma), ns = make_float2(-sigma, -sigma);
#define P2(s_, ri_) make_float2(p[s_][ri_][k], p[s_][ri_][k + 1])
#define SETH(s_, ri_, v) { const float2 t_ = (v); h[s_][c][ri_][k] = t_.x; h[s_][c][ri_][k + 1] = t_.y; }
                if constexpr (MU == 0) {
                    SETH(0, 0, __ffma2_rn(sg, P2(3, 1), P2(0, 0))) SETH(0, 1, __ffma2_rn(ns, P2(3, 0), P2(0, 1)))
                    SETH(1, 0, __ffma2_rn(sg, P2(2, 1), P2(1, 0))) SETH(1, 1, __ffma2_rn(ns, P2(2, 0), P2(1, 1)))
                } else if constexpr (MU == 1) {
                    SETH(0, 0, __ffma2_rn(sg, P2(3, 0), P2(0, 0))) SETH(0, 1, __ffma2_rn(sg, P2(3, 1), P2(0, 1)))
                    SETH(1, 0, __ffma2_rn(ns, P2(2, 0), P2(1, 0))) SETH(1, 1, __ffma2_rn(ns, P2(2, 1), P2(1, 1)))
                } else if constexpr (MU == 2) {
                    SETH(0, 0, __ffma2_rn(sg, P2(2, 1), P2(0, 0))) SETH(0, 1, __ffma2_rn(ns, P2(2, 0), P2(0, 1)))
                    SETH(1, 0, __ffma2_rn(ns, P2(3, 1), P2(1, 0))) SETH(1, 1, __ffma2_rn(sg, P2(3, 0), P2(1, 1)))
                } else {
                    SETH(0, 0, __ffma2_rn(ns, P2(2, 0), P2(0, 0))) SETH(0, 1, __ffma2_rn(ns, P2(2, 1), P2(0, 1)))
                    SETH(1, 0, __ffma2_rn(ns, P2(3, 0), P2(1, 0))) SETH(1, 1, __ffma2_rn(ns, P2(3, 1), P2(1, 1)))
                }
#undef P2
#undef SETH
            }
        } else
#endif
        {
#pragma unroll
        for (int k = 0; k < RPT; k++) {
            if constexpr (MU == 0) {        // h0 = p0 - s i p3, h1 = p1 - s i p2
                h[0][c][0][k] = fm(sigma, p[3][1][k], p[0][0][k]);  h[0][c][1][k] = fm(-sigma, p[3][0][k], p[0][1][k]);
                h[1][c][0][k] = fm(sigma, p[2][1][k], p[1][0][k]);  h[1][c][1][k] = fm(-sigma, p[2][0][k], p[1][1][k]);
            } else if constexpr (MU == 1) { // h0 = p0 + s p3, h1 = p1 - s p2
                h[0][c][0][k] = fm(sigma, p[3][0][k], p[0][0][k]);  h[0][c][1][k] = fm(sigma, p[3][1][k], p[0][1][k]);
                h[1][c][0][k] = fm(-sigma, p[2][0][k], p[1][0][k]); h[1][c][1][k] = fm(-sigma, p[2][1][k], p[1][1][k]);
            } else if constexpr (MU == 2) { // h0 = p0 - s i p2, h1 = p1 + s i p3
                h[0][c][0][k] = fm(sigma, p[2][1][k], p[0][0][k]);  h[0][c][1][k] = fm(-sigma, p[2][0][k], p[0][1][k]);
                h[1][c][0][k] = fm(-sigma, p[3][1][k], p[1][0][k]); h[1][c][1][k] = fm(sigma, p[3][0][k], p[1][1][k]);
            } else {                        // h0 = p0 - s p2, h1 = p1 - s p3
                h[0][c][0][k] = fm(-sigma, p[2][0][k], p[0][0][k]); h[0][c][1][k] = fm(-sigma, p[2][1][k], p[0][1][k]);
                h[1][c][0][k] = fm(-sigma, p[3][0][k], p[1][0][k]); h[1][c][1][k] = fm(-sigma, p[3][1][k], p[1][1][k]);
            }
        }
        }
}

// ---- one of the eight hopping terms -------------------------------------------------------------------
// acc[j][k] += cu * (1 - sigma*gamma_MU) W psi(nb),  W = U (FWD) or U^dag (backward), sigma = +-1.
// `nb` points at real 0 of the neighbour's RPT right-hand sides; real j is at nb + j*SB*R.
template <class S, int RPT, int R, int RECON, int MU, bool FWD, bool SMLINK = false>
__device__ __forceinline__ void hop_dir(const typename S::store_t* __restrict__ nb, const float* __restrict__ nb_norm,
                                        const typename S::link_t* __restrict__ link_blk, int link_s,
                                        typename S::comp_t cu, typename S::comp_t sigma, typename S::comp_t (&acc)[24][RPT]) {
    using T = typename S::comp_t;
    constexpr int PL = SB * R;   // elements between consecutive reals of a site
    T u[18];
    if constexpr (sizeof(typename S::link_t) == 2) load_link(link_blk, link_s, u);
    else load_link<T, RECON, SMLINK>(link_blk, link_s, u);

    T cuk[RPT], clk[RPT];
    if constexpr (S::has_norm) {
        float nrm[RPT];
        load_norm<RPT>(nb_norm, nrm);
#pragma unroll
        for (int k = 0; k < RPT; k++) cuk[k] = cu * nrm[k] * (1.0f / 32767.0f);
    } else {
#pragma unroll
        for (int k = 0; k < RPT; k++) cuk[k] = cu;
    }
#pragma unroll
    for (int k = 0; k < RPT; k++) clk[k] = sigma * cuk[k];

    // projected half spinor h[s][c][ri][k]
    T h[2][3][2][RPT];
#pragma unroll
    for (int c = 0; c < 3; c++) {
        T p[4][2][RPT];
#pragma unroll
        for (int s = 0; s < 4; s++)
#pragma unroll
            for (int ri = 0; ri < 2; ri++) load_comp<S, RPT>(nb + (2 * (3 * s + c) + ri) * PL, p[s][ri]);
        project_half<T, RPT, MU>(p, sigma, c, h);
    }
#ifdef LQ_USE_FFMA2
    if constexpr (sizeof(T) == 4 && RPT % 2 == 0) { hop_mulacc_f2<RPT, MU, FWD>(h, u, cuk, clk, acc); return; }
#endif
    hop_mulacc<T, RPT, MU, FWD>(h, u, cuk, clk, acc);
}

// ---- bench-only probe: the loads of one hopping term (link, 24 rows of the neighbour, norm) with ONE multiply-add per loaded
// value.  Kernel FORM_PROBE = kernel A's address stream, prefetches and stores without its arithmetic: its time is the floor
// that the memory path (L1 misses in flight, L2 -> SM transfers, HBM) sets for this access pattern (bench.py --op cfgN:probe:...).
template <class S, int RPT, int R, int RECON, bool SMLINK = false>
__device__ __forceinline__ void hop_dir_probe(const typename S::store_t* __restrict__ nb, const float* __restrict__ nb_norm,
                                              const typename S::link_t* __restrict__ link_blk, int link_s, typename S::comp_t (&acc)[24][RPT]) {
    using T = typename S::comp_t;
    constexpr int PL = SB * R;
    T u[18];
    if constexpr (sizeof(typename S::link_t) == 2) load_link(link_blk, link_s, u);
    else {
        load_planes<T, RECON, SMLINK>(link_blk, link_s, u);
        if constexpr (RECON == 12) {
#pragma unroll
            for (int i = 12; i < 18; i++) u[i] = u[i - 12];
        }
    }
    T sc[RPT];
    if constexpr (S::has_norm) { float nrm[RPT]; load_norm<RPT>(nb_norm, nrm);
#pragma unroll
        for (int k = 0; k < RPT; k++) sc[k] = nrm[k];
    } else {
#pragma unroll
        for (int k = 0; k < RPT; k++) sc[k] = T(1);
    }
#pragma unroll
    for (int j = 0; j < 24; j++) {
        T p[RPT];
        load_comp<S, RPT>(nb + j * PL, p);
#pragma unroll
        for (int k = 0; k < RPT; k++) acc[j][k] = fm(p[k] * sc[k], u[j % 18], acc[j][k]);
    }
}

