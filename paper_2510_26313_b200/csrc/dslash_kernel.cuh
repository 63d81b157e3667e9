// dslash_kernel.cuh -- kernel body, clover block multiply, half-storage epilogue and the launcher declaration.
#pragma once
#include "dslash.cuh"

// o = C v for one chirality block: cl = 6 real diagonal entries then 15 complex lower-triangular entries
// L(i,j), i > j, at index i(i-1)/2 + j (clover as 2 x (6x6 Hermitian), 72 reals per site).
// 22 FP instructions per output row and RHS: 2 multiplies by the real diagonal + 5 complex fused multiply-adds.
template <typename T, int RPT>
__device__ __forceinline__ void clover_block_mul(const T* cl, const T (&v)[6][2][RPT], T (&o)[6][2][RPT]) {
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
template <typename T, int RPT>
__device__ __forceinline__ void clover_apply_regs(const T* __restrict__ clov_blk, int s, T (&acc)[24][RPT]) {
#pragma unroll
    for (int b = 0; b < 2; b++) {
        T cl[36], v[6][2][RPT], o[6][2][RPT];
        load_planes<T, 36>(clov_blk + b * 36 * SB, s, cl);
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
#pragma unroll
        for (int j = 0; j < 24; j++) {
            T q[RPT];
#pragma unroll
            for (int k = 0; k < RPT; k++) q[k] = rintf(v[j][k] * inv[k]);
            store_comp<S, RPT>(p + j * PL, q);
        }
    } else {
#pragma unroll
        for (int j = 0; j < 24; j++) store_comp<S, RPT>(p + j * PL, v[j]);
    }
}

template <class S, int RPT, int R, int RECON, int FORM, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB) dslash_kernel(const DslashArgs<S> a) {
    using T = typename S::comp_t;
    using ST = typename S::store_t;
    constexpr int TPG = R / RPT;            // lanes per (site, group)
    constexpr int UT = SB * TPG;            // threads per unit
    constexpr int US = 24 * SB * R;         // payload elements per unit
    constexpr int UN = SB * R;              // norm elements per unit
    const int tid = blockIdx.x * BLOCK + threadIdx.x;
    const int G = a.G;
    const int u = tid / UT;                 // unit = blk*G + grp
    if (u >= a.g.NB * G) return;
    const int lu = tid - u * UT;
    const int s = lu / TPG, hoff = (lu - s * TPG) * RPT;
    const int blk = u / G, grp = u - blk * G;
    const int cb = blk * SB + s;
    if (cb >= a.g.Vh) return;               // padding sites of the last block
    int xh, y, z, t, odd;
    cb_coords(a.g, a.parity, cb, xh, y, z, t, odd);

    const size_t own = (size_t)u * US + s * R + hoff;
    const size_t own_n = (size_t)u * UN + s * R + hoff;

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
    const int NB = a.g.NB;
    // forward links live on the output site, backward links on the neighbour (other parity)
    const T* gown = a.gauge + ((size_t)(a.parity * NB + blk) * 4) * (RECON * SB);
    const T* gopp = a.gauge + ((size_t)((1 - a.parity) * NB) * 4) * (RECON * SB);
    const int Lxh = a.g.Lxh, Ly = a.g.L[1], Lz = a.g.L[2], Lt = a.g.L[3];
    const int sy = Lxh, sz = Lxh * Ly, st = Lxh * Ly * Lz;
    const ST* inb = a.in.d + (size_t)grp * US + hoff;
    const float* inn = S::has_norm ? a.in.n + (size_t)grp * UN + hoff : nullptr;
    const size_t bstride = (size_t)G * US, nstride = (size_t)G * UN;
#define LQ_NB_PTR(nb) (inb + (size_t)((nb) >> 5) * bstride + ((nb) & 31) * R)
#define LQ_NB_NRM(nb) (S::has_norm ? inn + (size_t)((nb) >> 5) * nstride + ((nb) & 31) * R : nullptr)
#define LQ_BWD_LINK(nb, mu) (gopp + ((size_t)((nb) >> 5) * 4 + (mu)) * (RECON * SB))
    {   // x
        const int xp = odd ? (xh + 1 == Lxh ? 0 : xh + 1) : xh;
        const int xm = odd ? xh : (xh == 0 ? Lxh - 1 : xh - 1);
        const int nbp = cb - xh + xp, nbm = cb - xh + xm;
        hop_dir<S, RPT, R, RECON, 0, true>(LQ_NB_PTR(nbp), LQ_NB_NRM(nbp), gown, s, c0, a.dsign, acc);
        hop_dir<S, RPT, R, RECON, 0, false>(LQ_NB_PTR(nbm), LQ_NB_NRM(nbm), LQ_BWD_LINK(nbm, 0), nbm & 31, c0, -a.dsign, acc);
    }
    {   // y
        const int nbp = (y + 1 == Ly) ? cb - (Ly - 1) * sy : cb + sy;
        const int nbm = (y == 0) ? cb + (Ly - 1) * sy : cb - sy;
        hop_dir<S, RPT, R, RECON, 1, true>(LQ_NB_PTR(nbp), LQ_NB_NRM(nbp), gown + RECON * SB, s, c0, a.dsign, acc);
        hop_dir<S, RPT, R, RECON, 1, false>(LQ_NB_PTR(nbm), LQ_NB_NRM(nbm), LQ_BWD_LINK(nbm, 1), nbm & 31, c0, -a.dsign, acc);
    }
    {   // z
        const int nbp = (z + 1 == Lz) ? cb - (Lz - 1) * sz : cb + sz;
        const int nbm = (z == 0) ? cb + (Lz - 1) * sz : cb - sz;
        hop_dir<S, RPT, R, RECON, 2, true>(LQ_NB_PTR(nbp), LQ_NB_NRM(nbp), gown + 2 * RECON * SB, s, c0, a.dsign, acc);
        hop_dir<S, RPT, R, RECON, 2, false>(LQ_NB_PTR(nbm), LQ_NB_NRM(nbm), LQ_BWD_LINK(nbm, 2), nbm & 31, c0, -a.dsign, acc);
    }
    {   // t (boundary sign on the wrapped term)
        const int nbp = (t + 1 == Lt) ? cb - (Lt - 1) * st : cb + st;
        const int nbm = (t == 0) ? cb + (Lt - 1) * st : cb - st;
        const T cp = (t + 1 == Lt) ? c0 * a.tsign : c0;
        const T cm = (t == 0) ? c0 * a.tsign : c0;
        hop_dir<S, RPT, R, RECON, 3, true>(LQ_NB_PTR(nbp), LQ_NB_NRM(nbp), gown + 3 * RECON * SB, s, cp, a.dsign, acc);
        hop_dir<S, RPT, R, RECON, 3, false>(LQ_NB_PTR(nbm), LQ_NB_NRM(nbm), LQ_BWD_LINK(nbm, 3), nbm & 31, cm, -a.dsign, acc);
    }
#undef LQ_NB_PTR
#undef LQ_NB_NRM
#undef LQ_BWD_LINK

    // ---- epilogue (FORM_A): acc <- C acc -----------------------------------------------------------------
    if constexpr (FORM == FORM_A) clover_apply_regs<T, RPT>(a.clover + (size_t)blk * (72 * SB), s, acc);

    // ---- store ----------------------------------------------------------------------------------------------
    store_site_regs<S, RPT, R>(a.out.d + own, S::has_norm ? a.out.n + own_n : nullptr, acc);
}

// ---- launcher -----------------------------------------------------------------------------------------------
// rpt: right-hand sides per thread (0 = default: the group width R, capped at 2 for fp64); variant: tuning bits.
template <class S, int RECON, int FORM>
int launch_dslash(lq_ctx* c, DslashArgs<S> a, int rpt, int variant);
