// dslash_kernel.cuh -- kernel body, clover block multiply, half-storage epilogue and the launcher declaration.
#pragma once
#include "dslash.cuh"
#include "reduce.cuh"

// o = C v for one chirality block: cl = 6 real diagonal entries then 15 complex lower-triangular entries
// L(i,j), i > j, at index i(i-1)/2 + j (clover as 2 x (6x6 Hermitian), 72 reals per site).
// 22 FP instructions per output row and RHS: 2 multiplies by the real diagonal + 5 complex fused multiply-adds.
template <typename T, int RPT>
__device__ __forceinline__ void clover_block_mul(const T* cl, const T (&v)[6][2][RPT], T (&o)[6][2][RPT]) {
#ifdef LQ_USE_FFMA2
    if constexpr (sizeof(T) == 4 && RPT % 2 == 0) {      // packed FP32: one FFMA2 per pair of right-hand sides
#pragma unroll
        for (int k = 0; k < RPT; k += 2) {
#define V2(j_, ri_) make_float2(v[j_][ri_][k], v[j_][ri_][k + 1])
#pragma unroll
            for (int i = 0; i < 6; i++) {
                const float2 d2 = make_float2(cl[i], cl[i]);
                float2 orr = __fmul2_rn(d2, V2(i, 0)), oi = __fmul2_rn(d2, V2(i, 1));
#pragma unroll
                for (int j = 0; j < 6; j++) {
                    if (j == i) continue;
                    const int idx = (i > j) ? (i * (i - 1) / 2 + j) : (j * (j - 1) / 2 + i);
                    const float lr = cl[6 + 2 * idx];
                    const float li = (i > j) ? cl[7 + 2 * idx] : -cl[7 + 2 * idx];
                    const float2 lr2 = make_float2(lr, lr), li2 = make_float2(li, li), nli2 = make_float2(-li, -li);
                    orr = __ffma2_rn(lr2, V2(j, 0), orr); orr = __ffma2_rn(nli2, V2(j, 1), orr);
                    oi = __ffma2_rn(lr2, V2(j, 1), oi); oi = __ffma2_rn(li2, V2(j, 0), oi);
                }
                o[i][0][k] = orr.x; o[i][0][k + 1] = orr.y; o[i][1][k] = oi.x; o[i][1][k + 1] = oi.y;
            }
#undef V2
        }
        return;
    }
#endif
#pragma unroll
    for (int i = 0; i < 6; i++) {
#pragma unroll
        for (int k = 0; k < RPT; k++) { o[i][0][k] = cl[i] * v[i][0][k]; o[i][1][k] = cl[i] * v[i][1][k]; }
#pragma unroll
        for (int j = 0; j < 6; j++) {
            if (j == i) continue;
            const int idx = (i > j) ? (i * (i - 1) / 2 + j) : (j * (j - 1) / 2 + i);
            const T lr = cl[6 + 2 * idx];
            const T li = (i > j) ? cl[7 + 2 * idx] : -cl[7 + 2 * idx];
#pragma unroll
            for (int k = 0; k < RPT; k++) {
                o[i][0][k] = fm(lr, v[j][0][k], o[i][0][k]);
                o[i][0][k] = fm(-li, v[j][1][k], o[i][0][k]);
                o[i][1][k] = fm(lr, v[j][1][k], o[i][1][k]);
                o[i][1][k] = fm(li, v[j][0][k], o[i][1][k]);
            }
        }
    }
}

// acc (24 reals x RPT) <- C acc, one chirality block at a time
template <typename T, int RPT, bool SMEM = false>
__device__ __forceinline__ void clover_apply_regs(const T* __restrict__ clov_blk, int s, T (&acc)[24][RPT]) {
#pragma unroll
    for (int b = 0; b < 2; b++) {
        T cl[36], v[6][2][RPT], o[6][2][RPT];
        load_planes<T, 36, SMEM>(clov_blk + b * 36 * SB, s, cl);
#pragma unroll
        for (int i = 0; i < 6; i++)
#pragma unroll
            for (int ri = 0; ri < 2; ri++)
#pragma unroll
                for (int k = 0; k < RPT; k++) v[i][ri][k] = acc[12 * b + 2 * i + ri][k];
        clover_block_mul<T, RPT>(cl, v, o);
#pragma unroll
        for (int i = 0; i < 6; i++)
#pragma unroll
            for (int ri = 0; ri < 2; ri++)
#pragma unroll
                for (int k = 0; k < RPT; k++) acc[12 * b + 2 * i + ri][k] = o[i][ri][k];
    }
}

// load one site's 24 reals (RPT right-hand sides) into registers, dequantising half storage
template <class S, int RPT, int R>
__device__ __forceinline__ void load_site_regs(const typename S::store_t* __restrict__ p, const float* __restrict__ pn,
                                               typename S::comp_t (&v)[24][RPT]) {
    constexpr int PL = SB * R;
#pragma unroll
    for (int j = 0; j < 24; j++) load_comp<S, RPT>(p + j * PL, v[j]);
    if constexpr (S::has_norm) {
        float nrm[RPT];
        load_norm<RPT>(pn, nrm);
#pragma unroll
        for (int k = 0; k < RPT; k++) {
            const float sc = nrm[k] * (1.0f / 32767.0f);
#pragma unroll
            for (int j = 0; j < 24; j++) v[j][k] *= sc;
        }
    }
}
// store one site's 24 reals; half storage: int16 fixed point with a per-(site, rhs) fp32 max-abs norm
// (SURVEY 8(c.2) reading #12)
template <class S, int RPT, int R>
__device__ __forceinline__ void store_site_regs(typename S::store_t* __restrict__ p, float* __restrict__ pn,
                                                const typename S::comp_t (&v)[24][RPT]) {
    using T = typename S::comp_t;
    constexpr int PL = SB * R;
    if constexpr (S::has_norm) {
        float mx[RPT], inv[RPT];
#pragma unroll
        for (int k = 0; k < RPT; k++) mx[k] = 0.f;
#pragma unroll
        for (int j = 0; j < 24; j++)
#pragma unroll
            for (int k = 0; k < RPT; k++) mx[k] = fmaxf(mx[k], fabsf(v[j][k]));
#pragma unroll
        for (int k = 0; k < RPT; k++) inv[k] = mx[k] > 0.f ? 32767.0f / mx[k] : 0.f;
        store_norm<RPT>(pn, mx);
        // q = round-to-nearest-even(v * 32767 / max) without the conversion unit: ONE fused multiply-add onto 1.5 * 2^23 leaves the rounded
        // integer, as two's complement, in the low 16 bits of the result (|q| <= 32767 << 2^22; rounded once, where rintf(v * inv)
        // rounds twice); a byte permute packs two of them.  (FRND + F2I, the straightforward form, run on the 16-lane unit.)
#pragma unroll
        for (int j = 0; j < 24; j++) {
            unsigned b[RPT];
#pragma unroll
            for (int k = 0; k < RPT; k++) b[k] = __float_as_uint(fmaf(v[j][k], inv[k], 12582912.0f));
            short* q = p + j * PL;
            if constexpr (RPT == 4) *(uint2*)q = make_uint2(__byte_perm(b[0], b[1], 0x5410), __byte_perm(b[2], b[3], 0x5410));
            else if constexpr (RPT == 2) *(unsigned*)q = __byte_perm(b[0], b[1], 0x5410);
            else *q = (short)(b[0] & 0xFFFFu);
        }
    } else {
#pragma unroll
        for (int j = 0; j < 24; j++) store_comp<S, RPT>(p + j * PL, v[j]);
    }
}

// site coordinates and strides of one thread, and its neighbour in direction D = 2*mu + (0 forward | 1 backward)
struct SiteCtx { int cb, xh, y, z, t, odd, Lxh, Ly, Lz, Lt; };
template <int D> __device__ __forceinline__ int neighbour(const SiteCtx& c) {
    constexpr int mu = D >> 1; constexpr bool fwd = (D & 1) == 0;
    if constexpr (mu == 0) {
        const int xn = fwd ? (c.odd ? (c.xh + 1 == c.Lxh ? 0 : c.xh + 1) : c.xh) : (c.odd ? c.xh : (c.xh == 0 ? c.Lxh - 1 : c.xh - 1));
        return c.cb - c.xh + xn;
    } else if constexpr (mu == 1) {
        const int sy = c.Lxh;
        return fwd ? ((c.y + 1 == c.Ly) ? c.cb - (c.Ly - 1) * sy : c.cb + sy) : ((c.y == 0) ? c.cb + (c.Ly - 1) * sy : c.cb - sy);
    } else if constexpr (mu == 2) {
        const int sz = c.Lxh * c.Ly;
        return fwd ? ((c.z + 1 == c.Lz) ? c.cb - (c.Lz - 1) * sz : c.cb + sz) : ((c.z == 0) ? c.cb + (c.Lz - 1) * sz : c.cb - sz);
    } else {
        const int st = c.Lxh * c.Ly * c.Lz;
        return fwd ? ((c.t + 1 == c.Lt) ? c.cb - (c.Lt - 1) * st : c.cb + st) : ((c.t == 0) ? c.cb + (c.Lt - 1) * st : c.cb - st);
    }
}

// launch-order block index -> site block (see DslashArgs::zc)
template <class S> __device__ __forceinline__ int sweep_block(const DslashArgs<S>& a, int b) {
    if (a.zc == 0) return b;
    int r = a.dnby.div(b); const int yb = b - r * a.nby;
    int q = a.dzc.div(r); const int zi = r - q * a.zc;
    const int zch = a.dLt.div(q); const int t = q - zch * a.g.L[3];
    return yb + a.nby * ((zch * a.zc + zi) + a.g.L[2] * t);
}

// EPI: the fused block-BLAS epilogue of kernel B, a template parameter so that every launch carries only the code it runs
// (one kernel with all three epilogues was 90 KB of instructions for half storage: instruction-fetch stalls)
template <class S, int RPT, int R, int RECON, int FORM, int BLOCK, int MINB, int EPI = EPI_NONE>
__global__ void __launch_bounds__(BLOCK, MINB) dslash_kernel(const DslashArgs<S> a) {
    using T = typename S::comp_t;
    using ST = typename S::store_t;
    if (a.skip != nullptr && *(volatile const int*)a.skip) return;      // the inner solve has converged (grid-uniform)
    constexpr int TPG = R / RPT;            // lanes per (site, group)
    constexpr int UT = SB * TPG;            // threads per unit
    constexpr int US = 24 * SB * R;         // payload elements per unit
    constexpr int UN = SB * R;              // norm elements per unit
    const int G = a.G;
    const int tid = blockIdx.x * BLOCK + threadIdx.x;
    const int u = tid / UT;                 // unit = blk*G + grp
    const int lu = tid - u * UT;
    const int lblk = a.dG.div(u), grp = u - lblk * G;      // launch-order block
    const int blk = sweep_block(a, lblk);
    const int s = lu / TPG, hoff = (lu - s * TPG) * RPT;
    SiteCtx sc;
    sc.cb = blk * SB + s;
    // threads beyond the last unit and padding sites of the last block do no work (but reach the fused reduction)
    const bool valid = (u < a.g.NB * G) && (sc.cb < a.g.Vh);
    double part[RPT], part_c[2][RPT];       // part_c: EPI_CDOT only
#pragma unroll
    for (int k = 0; k < RPT; k++) { part[k] = 0.0; part_c[0][k] = 0.0; part_c[1][k] = 0.0; }
    if (valid) {
    cb_coords(a.g, a.parity, sc.cb, sc.xh, sc.y, sc.z, sc.t, sc.odd);
    sc.Lxh = a.g.Lxh; sc.Ly = a.g.L[1]; sc.Lz = a.g.L[2]; sc.Lt = a.g.L[3];

    const size_t own = (size_t)(blk * G + grp) * US + s * R + hoff;
    const size_t own_n = (size_t)(blk * G + grp) * UN + s * R + hoff;

    const int NB = a.g.NB;
    // forward links live on the output site, backward links on the neighbour (other parity)
    using LT = typename S::link_t;
    const LT* gown = a.gauge + ((size_t)(a.parity * NB + blk) * 4) * (RECON * SB);
    const LT* gopp = a.gauge + ((size_t)((1 - a.parity) * NB) * 4) * (RECON * SB);
    const ST* inb = a.in.d + (size_t)grp * US + hoff;
    const float* inn = S::has_norm ? a.in.n + (size_t)grp * UN + hoff : nullptr;
    const size_t bstride = (size_t)G * US, nstride = (size_t)G * UN;
#define LQ_NB_PTR(nb) (inb + (size_t)((nb) >> 5) * bstride + ((nb) & 31) * R)
#define LQ_NB_NRM(nb) (S::has_norm ? inn + (size_t)((nb) >> 5) * nstride + ((nb) & 31) * R : nullptr)
#define LQ_LINK(D, nb) (((D) & 1) ? gopp + ((size_t)((nb) >> 5) * 4 + ((D) >> 1)) * (RECON * SB) : gown + ((D) >> 1) * (RECON * SB))
#define LQ_LINK_S(D, nb) (((D) & 1) ? ((nb) & 31) : s)

    // ---- distance prefetch into L2 ------------------------------------------------------------------------
    // An SM can keep only a few KB of L1 misses in flight, so a demand load that goes to HBM (~2.5x the latency of
    // an L2 hit) costs ~2.5x the L1 miss-slot time: the kernel is bound by (bytes fetched) x (their latency), not by
    // HBM bandwidth.  Every unit therefore asks L2, with fire-and-forget prefetches, for the data that the unit
    // `pfd` site blocks further along the sweep will touch FIRST: the input unit one time-slice ahead (the +t
    // neighbours; every other neighbour was touched by earlier blocks), both parities' link slabs and the clover
    // block.  One 128-byte line per lane per instruction; ~10 instructions per thread.
    {
        if (a.pfd > 0) {
            const int lpb = lblk + a.pfd;
            if (lpb < NB) {
                const int pb = sweep_block(a, lpb);
                constexpr int LINE = 128;
#define LQ_PF_LINES(base, nlines) { _Pragma("unroll") for (int i0_ = 0; i0_ < (nlines); i0_ += UT) { const int i_ = i0_ + lu; \
                    if (i_ < (nlines)) asm volatile("prefetch.global.L2 [%0];" ::"l"((base) + (size_t)i_ * LINE)); } }
                const int st32 = (sc.Lxh * sc.Ly * sc.Lz) / SB;
                int pbt = pb + st32; if (pbt >= NB) pbt -= NB;
                const char* q = (const char*)(a.in.d + ((size_t)pbt * G + grp) * US);
                LQ_PF_LINES(q, (int)(US * sizeof(ST) / LINE))
                if constexpr (FORM == FORM_B) {
                    const char* qx = (const char*)(a.x.d + ((size_t)pb * G + grp) * US);
                    LQ_PF_LINES(qx, (int)(US * sizeof(ST) / LINE))
                    if constexpr (EPI == EPI_XMAY) {          // the epilogue reads the vector it updates
                        const char* qz = (const char*)(a.out.d + ((size_t)pb * G + grp) * US);
                        LQ_PF_LINES(qz, (int)(US * sizeof(ST) / LINE))
                    } else if constexpr (EPI == EPI_CDOT) {
                        const char* qh = (const char*)(a.epi_v.d + ((size_t)pb * G + grp) * US);
                        LQ_PF_LINES(qh, (int)(US * sizeof(ST) / LINE))
                    }
                }
                constexpr int GL = 4 * RECON * SB * sizeof(typename S::link_t) / LINE;     // lines of one (parity, block) link slab
                constexpr int CL = 72 * SB * sizeof(T) / LINE;            // lines of one clover block
                if (grp == 0 % G) {
                    const char* l = (const char*)(a.gauge + ((size_t)(a.parity * NB + pb) * 4) * (RECON * SB));
                    LQ_PF_LINES(l, GL)
                }
                if (grp == 1 % G) {
                    const char* l = (const char*)(a.gauge + ((size_t)((1 - a.parity) * NB + pb) * 4) * (RECON * SB));
                    LQ_PF_LINES(l, GL)
                }
                if (grp == 2 % G && a.clover != nullptr) {
                    const char* l = (const char*)(a.clover + (size_t)pb * (72 * SB));
                    LQ_PF_LINES(l, CL)
                }
#undef LQ_PF_LINES
            }
        }
    }

    T acc[24][RPT];
    // ---- prologue (FORM_B): acc = C x  (or x when no clover) -----------------------------------------
    if constexpr (FORM == FORM_B) {
        load_site_regs<S, RPT, R>(a.x.d + own, S::has_norm ? a.x.n + own_n : nullptr, acc);
        if (a.clover != nullptr) clover_apply_regs<T, RPT>(a.clover + (size_t)blk * (72 * SB), s, acc);
    } else {
#pragma unroll
        for (int j = 0; j < 24; j++)
#pragma unroll
            for (int k = 0; k < RPT; k++) acc[j][k] = 0;
    }

    // ---- the eight hops ---------------------------------------------------------------------------------
    const T c0 = (FORM == FORM_B) ? a.coef : T(1);
    const T cp = (sc.t + 1 == sc.Lt) ? c0 * a.tsign : c0;     // boundary sign on the wrapped t terms
    const T cm = (sc.t == 0) ? c0 * a.tsign : c0;
#define LQ_HOP(D) { const int nb_ = neighbour<D>(sc); \
        if constexpr (FORM == FORM_PROBE) hop_dir_probe<S, RPT, R, RECON>(LQ_NB_PTR(nb_), LQ_NB_NRM(nb_), LQ_LINK(D, nb_), LQ_LINK_S(D, nb_), acc); \
        else hop_dir<S, RPT, R, RECON, ((D) >> 1), (((D) & 1) == 0)>(LQ_NB_PTR(nb_), LQ_NB_NRM(nb_), LQ_LINK(D, nb_), LQ_LINK_S(D, nb_), \
                (D) == 6 ? cp : ((D) == 7 ? cm : c0), ((D) & 1) ? -a.dsign : a.dsign, acc); }
    LQ_HOP(0) LQ_HOP(1) LQ_HOP(2) LQ_HOP(3) LQ_HOP(4) LQ_HOP(5) LQ_HOP(6) LQ_HOP(7)
#undef LQ_HOP
#undef LQ_NB_PTR
#undef LQ_NB_NRM
#undef LQ_LINK
#undef LQ_LINK_S

    // ---- epilogue (FORM_A): acc <- C acc -----------------------------------------------------------------
    if constexpr (FORM == FORM_A) clover_apply_regs<T, RPT>(a.clover + (size_t)blk * (72 * SB), s, acc);
    if constexpr (FORM == FORM_PROBE) {       // the clover block's loads, one multiply-add per loaded value
        T cl[72];
        load_planes<T, 72>(a.clover + (size_t)blk * (72 * SB), s, cl);
#pragma unroll
        for (int j = 0; j < 72; j++)
#pragma unroll
            for (int k = 0; k < RPT; k++) acc[j % 24][k] = fm(cl[j], T(0.5), acc[j % 24][k]);
    }

    // ---- fused block-BLAS epilogues of kernel B and store ---------------------------------
    if constexpr (FORM == FORM_B) {
        if constexpr (EPI == EPI_XMAY) {
            // out <- out - alpha_k acc  (the CG residual update z -= alpha q without ever storing q), alpha = rr / pAp
            T zv[24][RPT], al[RPT];
            load_site_regs<S, RPT, R>(a.out.d + own, S::has_norm ? a.out.n + own_n : nullptr, zv);
#pragma unroll
            for (int k = 0; k < RPT; k++) { const double d = a.epi_den[grp * R + hoff + k]; al[k] = (T)(d > 0.0 ? a.epi_num[grp * R + hoff + k] / d : 0.0); }
#pragma unroll
            for (int j = 0; j < 24; j++)
#pragma unroll
                for (int k = 0; k < RPT; k++) acc[j][k] = zv[j][k] - al[k] * acc[j][k];
        }
        if constexpr (EPI == EPI_CDOT) {
            // <h, out> for the 12 complex components, summed in the compute type per site like the norms below
            T hv[24][RPT], pr[RPT], pi[RPT];
            load_site_regs<S, RPT, R>(a.epi_v.d + own, S::has_norm ? a.epi_v.n + own_n : nullptr, hv);
#pragma unroll
            for (int k = 0; k < RPT; k++) { pr[k] = 0; pi[k] = 0; }
#pragma unroll
            for (int cc = 0; cc < 12; cc++)
#pragma unroll
                for (int k = 0; k < RPT; k++) {
                    pr[k] = fm(hv[2 * cc][k], acc[2 * cc][k], fm(hv[2 * cc + 1][k], acc[2 * cc + 1][k], pr[k]));
                    pi[k] = fm(hv[2 * cc][k], acc[2 * cc + 1][k], fm(-hv[2 * cc + 1][k], acc[2 * cc][k], pi[k]));
                }
#pragma unroll
            for (int k = 0; k < RPT; k++) { part_c[0][k] = (double)pr[k]; part_c[1][k] = a.epi_conj ? -(double)pi[k] : (double)pi[k]; }
        }
        if constexpr (EPI != EPI_NONE) {
            // the 24 squares of one site are summed in the compute type (relative error ~1e-7 in fp32, far below the
            // solver's use of these norms); sites are summed in fp64 by the reduction
            T ps[RPT];
#pragma unroll
            for (int k = 0; k < RPT; k++) ps[k] = 0;
#pragma unroll
            for (int j = 0; j < 24; j++)
#pragma unroll
                for (int k = 0; k < RPT; k++) ps[k] = fm(acc[j][k], acc[j][k], ps[k]);
#pragma unroll
            for (int k = 0; k < RPT; k++) part[k] = (double)ps[k];
        }
    }
    store_site_regs<S, RPT, R>(a.out.d + own, S::has_norm ? a.out.n + own_n : nullptr, acc);
    }   // valid
    if constexpr (FORM == FORM_B) {
        if constexpr (EPI == EPI_CDOT) {
            double p3[3][RPT];
#pragma unroll
            for (int k = 0; k < RPT; k++) { p3[0][k] = part_c[0][k]; p3[1][k] = part_c[1][k]; p3[2][k] = part[k]; }
            reduce_multi<3, RPT, R>(p3, a.N, G, a.red_partials);
        } else if constexpr (EPI != EPI_NONE) reduce_per_rhs<RPT, R>(part, a.N, G, a.red_partials);
    }
}

// ---- launcher -----------------------------------------------------------------------------------------------
// rpt: right-hand sides per thread (0 = default: the group width R, capped at 2 for fp64); variant: tuning bits.
template <class S, int RECON, int FORM>
int launch_dslash(lq_ctx* c, DslashArgs<S> a, int rpt, int variant);
