// dslash_kernel.cuh -- kernel body, clover block multiply, half-storage epilogue and the launcher.
#pragma once
#include "dslash.cuh"

// o = C v for one chirality block: cl = 6 real diagonal entries then 15 complex lower-triangular entries
// L(i,j), i > j, at index i(i-1)/2 + j (clover as 2 x (6x6 Hermitian), 72 reals per site).
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
                o[i][0][k] += lr * v[j][0][k] - li * v[j][1][k];
                o[i][1][k] += lr * v[j][1][k] + li * v[j][0][k];
            }
        }
    }
}

template <class S, int RPT, int RECON, int FORM>
__global__ void __launch_bounds__(256) dslash_kernel(const DslashArgs<S> a) {
    using T = typename S::comp_t;
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int Vh = a.g.Vh, N = a.N;
    if (tid >= Vh * a.G) return;
    const int cb = tid / a.G;
    const int goff = (tid - cb * a.G) * RPT;
    int xh, y, z, t, odd;
    cb_coords(a.g, a.parity, cb, xh, y, z, t, odd);
    const size_t plane = (size_t)Vh * N;

    T acc[24][RPT];
    // ---- prologue (FORM_B): acc = C x  (or x when no clover) -----------------------------------------
    if constexpr (FORM == FORM_B) {
        T sc[RPT];
        if constexpr (S::has_norm) {
            float nrm[RPT];
            load_norm<RPT>(a.x.n + (size_t)cb * N + goff, nrm);
#pragma unroll
            for (int k = 0; k < RPT; k++) sc[k] = nrm[k] * (1.0f / 32767.0f);
        }
        const typename S::store_t* xb = a.x.d + (size_t)cb * N + goff;
#pragma unroll
        for (int b = 0; b < 2; b++) {
            T v[6][2][RPT];
#pragma unroll
            for (int i = 0; i < 6; i++)
#pragma unroll
                for (int ri = 0; ri < 2; ri++) {
                    load_comp<S, RPT>(xb + (size_t)(12 * b + 2 * i + ri) * plane, v[i][ri]);
                    if constexpr (S::has_norm) {
#pragma unroll
                        for (int k = 0; k < RPT; k++) v[i][ri][k] *= sc[k];
                    }
                }
            if (a.clover != nullptr) {
                T cl[36], o[6][2][RPT];
                load_planes<T, 36>(a.clover + (size_t)b * 36 * Vh, Vh, cb, cl);
                clover_block_mul<T, RPT>(cl, v, o);
#pragma unroll
                for (int i = 0; i < 6; i++)
#pragma unroll
                    for (int ri = 0; ri < 2; ri++)
#pragma unroll
                        for (int k = 0; k < RPT; k++) acc[12 * b + 2 * i + ri][k] = o[i][ri][k];
            } else {
#pragma unroll
                for (int i = 0; i < 6; i++)
#pragma unroll
                    for (int ri = 0; ri < 2; ri++)
#pragma unroll
                        for (int k = 0; k < RPT; k++) acc[12 * b + 2 * i + ri][k] = v[i][ri][k];
            }
        }
    } else {
#pragma unroll
        for (int j = 0; j < 24; j++)
#pragma unroll
            for (int k = 0; k < RPT; k++) acc[j][k] = 0;
    }

    // ---- the eight hops ---------------------------------------------------------------------------------
    const T c0 = (FORM == FORM_B) ? a.coef : T(1);
    const int op = 1 - a.parity;
    const T* gown = a.gauge + (size_t)(a.parity * 4) * RECON * Vh;   // forward links live on the output site
    const T* gopp = a.gauge + (size_t)(op * 4) * RECON * Vh;         // backward links on the neighbour
    const size_t gmu = (size_t)RECON * Vh;
    const int Lxh = a.g.Lxh, Ly = a.g.L[1], Lz = a.g.L[2], Lt = a.g.L[3];
    const int sy = Lxh, sz = Lxh * Ly, st = Lxh * Ly * Lz;
    {   // x
        const int xp = odd ? (xh + 1 == Lxh ? 0 : xh + 1) : xh;
        const int xm = odd ? xh : (xh == 0 ? Lxh - 1 : xh - 1);
        const int nbp = cb - xh + xp, nbm = cb - xh + xm;
        hop_dir<S, RPT, RECON, 0, true>(a, nbp, gown, cb, c0, a.dsign, goff, acc);
        hop_dir<S, RPT, RECON, 0, false>(a, nbm, gopp, nbm, c0, -a.dsign, goff, acc);
    }
    {   // y
        const int nbp = (y + 1 == Ly) ? cb - (Ly - 1) * sy : cb + sy;
        const int nbm = (y == 0) ? cb + (Ly - 1) * sy : cb - sy;
        hop_dir<S, RPT, RECON, 1, true>(a, nbp, gown + gmu, cb, c0, a.dsign, goff, acc);
        hop_dir<S, RPT, RECON, 1, false>(a, nbm, gopp + gmu, nbm, c0, -a.dsign, goff, acc);
    }
    {   // z
        const int nbp = (z + 1 == Lz) ? cb - (Lz - 1) * sz : cb + sz;
        const int nbm = (z == 0) ? cb + (Lz - 1) * sz : cb - sz;
        hop_dir<S, RPT, RECON, 2, true>(a, nbp, gown + 2 * gmu, cb, c0, a.dsign, goff, acc);
        hop_dir<S, RPT, RECON, 2, false>(a, nbm, gopp + 2 * gmu, nbm, c0, -a.dsign, goff, acc);
    }
    {   // t (boundary sign on the wrapped term)
        const int nbp = (t + 1 == Lt) ? cb - (Lt - 1) * st : cb + st;
        const int nbm = (t == 0) ? cb + (Lt - 1) * st : cb - st;
        const T cp = (t + 1 == Lt) ? c0 * a.tsign : c0;
        const T cm = (t == 0) ? c0 * a.tsign : c0;
        hop_dir<S, RPT, RECON, 3, true>(a, nbp, gown + 3 * gmu, cb, cp, a.dsign, goff, acc);
        hop_dir<S, RPT, RECON, 3, false>(a, nbm, gopp + 3 * gmu, nbm, cm, -a.dsign, goff, acc);
    }

    // ---- epilogue (FORM_A): acc <- C acc -----------------------------------------------------------------
    if constexpr (FORM == FORM_A) {
#pragma unroll
        for (int b = 0; b < 2; b++) {
            T cl[36], v[6][2][RPT], o[6][2][RPT];
            load_planes<T, 36>(a.clover + (size_t)b * 36 * Vh, Vh, cb, cl);
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

    // ---- store ----------------------------------------------------------------------------------------------
    typename S::store_t* ob = a.out.d + (size_t)cb * N + goff;
    if constexpr (S::has_norm) {
        // int16 fixed point with a per-(site, rhs) fp32 max-abs norm (SURVEY 8(c.2) reading #12)
        float mx[RPT], inv[RPT];
#pragma unroll
        for (int k = 0; k < RPT; k++) mx[k] = 0.f;
#pragma unroll
        for (int j = 0; j < 24; j++)
#pragma unroll
            for (int k = 0; k < RPT; k++) mx[k] = fmaxf(mx[k], fabsf(acc[j][k]));
#pragma unroll
        for (int k = 0; k < RPT; k++) inv[k] = mx[k] > 0.f ? 32767.0f / mx[k] : 0.f;
        if constexpr (RPT == 4) *(float4*)(a.out.n + (size_t)cb * N + goff) = make_float4(mx[0], mx[1], mx[2], mx[3]);
        else if constexpr (RPT == 2) *(float2*)(a.out.n + (size_t)cb * N + goff) = make_float2(mx[0], mx[1]);
        else a.out.n[(size_t)cb * N + goff] = mx[0];
#pragma unroll
        for (int j = 0; j < 24; j++) {
            T q[RPT];
#pragma unroll
            for (int k = 0; k < RPT; k++) q[k] = rintf(acc[j][k] * inv[k]);
            store_comp<S, RPT>(ob + (size_t)j * plane, q);
        }
    } else {
#pragma unroll
        for (int j = 0; j < 24; j++) store_comp<S, RPT>(ob + (size_t)j * plane, acc[j]);
    }
}

// ---- launcher -----------------------------------------------------------------------------------------------
// rpt_for: right-hand sides per thread.  fp32/half: 4 when N % 4 == 0; fp64: 2 when N % 2 == 0.
template <class S, int RECON, int FORM>
int launch_dslash(lq_ctx* c, DslashArgs<S> a, int rpt_override);
