// mg_kernels.cuh -- device side of the two-level adaptive multigrid (the
// construction of the paper's ref. [19]): aggregates x chirality, block-orthonormal prolongator P, Galerkin coarse operator
// A_c = P^dag M P as a 9-point stencil of dense (2 Nv)^2 blocks, all batched over N right-hand sides ("Batching ...
// especially important in the context of multi-grid, where the coarse grids have limited parallelism").
//
// Data (fp32; the multigrid cycle is a preconditioner inside an fp64 defect correction):
//   fine vectors   full-lattice NATIVE batches: the even and the odd parity block of common.cuh back to back.  MG needs
//                  Vh % 32 == 0 (no padded sites), so a full vector is one array [2 NB][G][24][32][R] and a site is addressed by
//                  its "full checkerboard index" f = parity * Vh + cb.
//   site_f         [Vc][ns]  f of the i-th site of aggregate a, i = ix + bx (iy + by (iz + bz it))
//   P              [Vc][2][M = 6 ns][Nv] float2: column k of aggregate a, chirality chi; row m = 6 i + (3 (spin % 2) + colour)
//   coarse vectors [Vc][nc = 2 Nv][N] float2, row = chi * Nv + k, right-hand side innermost
//   A_c            [Vc][9][nc (column)][nc (row)] float2; direction 0 = self, 1 + 2 mu = +mu, 2 + 2 mu = -mu
//   nbr            [Vc][9] coarse neighbour, -1 where the block is merged into another one (Lc_mu = 2: -mu into +mu; Lc_mu = 1: both
//                  into self)
#pragma once
#include "common.cuh"
#include "reduce.cuh"

namespace mg {

struct MgGeom {
    int b[4], Lc[4];
    int Vc, ns, nv, nc, M;    // coarse sites, sites per aggregate, near-null vectors, 2 nv, 6 ns
};

template <int R> __device__ __forceinline__ void ldv(const float* p, float (&v)[R]) {
    if constexpr (R == 4) { const float4 q = *reinterpret_cast<const float4*>(p); v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w; }
    else if constexpr (R == 2) { const float2 q = *reinterpret_cast<const float2*>(p); v[0] = q.x; v[1] = q.y; }
    else v[0] = *p;
}
template <int R> __device__ __forceinline__ void stv(float* p, const float (&v)[R]) {
    if constexpr (R == 4) *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
    else if constexpr (R == 2) *reinterpret_cast<float2*>(p) = make_float2(v[0], v[1]);
    else *p = v[0];
}
// element offset of (full index f, group g, real j = 0) in a full-lattice native fp32 batch of G groups of R
template <int R> __device__ __forceinline__ size_t fine_base(int f, int G, int g) {
    return ((size_t)(f >> 5) * G + g) * (size_t)(24 * SB * R) + (size_t)(f & 31) * R;
}

// ---- tables ---------------------------------------------------------------------------------------------------------------
__global__ void tables_kernel(Geom g, MgGeom m, int* __restrict__ site_f) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= (long long)m.Vc * m.ns) return;
    int a = (int)(tid / m.ns), i = (int)(tid % m.ns);
    int x[4];
    for (int mu = 0; mu < 4; mu++) {
        const int am = a % m.Lc[mu], im = i % m.b[mu];
        a /= m.Lc[mu]; i /= m.b[mu];
        x[mu] = am * m.b[mu] + im;
    }
    int parity, cb;
    coords_to_cb(g, x[0], x[1], x[2], x[3], parity, cb);
    site_f[tid] = parity * g.Vh + cb;
}

// ---- prolongator from Nv near-null vectors (native fp32 batch of Nv right-hand sides) ------------------------------------
template <int R>
__global__ void gather_P_kernel(MgGeom m, const int* __restrict__ site_f, const float* __restrict__ v, float2* __restrict__ P) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)m.Vc * 2 * m.M * m.nv;
    if (tid >= total) return;
    const int k = (int)(tid % m.nv);
    long long q = tid / m.nv;
    const int mm = (int)(q % m.M); q /= m.M;
    const int chi = (int)(q & 1), a = (int)(q >> 1);
    const int i = mm / 6, c6 = mm - 6 * i;
    const int f = site_f[(size_t)a * m.ns + i];
    const int G = m.nv / R;
    const size_t base = fine_base<R>(f, G, k / R) + (k % R);
    const int j = 2 * (chi * 6 + c6);
    P[tid] = make_float2(v[base + (size_t)j * (SB * R)], v[base + (size_t)(j + 1) * (SB * R)]);
}

// block-wide sum of NQ doubles, result broadcast to every thread (fixed order: warp shuffle, then the warps in index order)
template <int NQ>
__device__ __forceinline__ void block_sum(double (&v)[NQ], double* sm /* [NQ * 32] */) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int q = 0; q < NQ; q++)
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) v[q] += __shfl_xor_sync(0xffffffffu, v[q], off);
    __syncthreads();
    if (lane == 0) {
#pragma unroll
        for (int q = 0; q < NQ; q++) sm[q * 32 + w] = v[q];
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < NQ; q++) {
        double s = 0.0;
        for (int ww = 0; ww < nw; ww++) s += sm[q * 32 + ww];
        v[q] = s;
    }
}

// Gram-Schmidt over k = 0, 1, ... inside every (aggregate, chirality) block: column k against the earlier columns, twice, then
// normalised.  One CTA of 8 warps per block; the columns stay in global memory (L1 / L2 resident).  Each of the two passes is
// classical Gram-Schmidt in two phases -- all inner products <col_j, col_k>, j < k, at once (warp w takes j = w, w + 8, ..., its lanes
// stride the rows, fp64 sums), then one update col_k -= sum_j d_j col_j -- instead of 2 k dependent dot / update rounds; two
// classical passes give the Q factor of the oracle's (modified, twice) order to rounding: the factor is unique.
// status[0] is set when a column has (nearly) no component left: linearly dependent near-null vectors.
__global__ void __launch_bounds__(256) orthonormalise_kernel(MgGeom m, float2* __restrict__ P, int* __restrict__ status) {
    __shared__ double sm[2 * 32];
    __shared__ float2 dj[LQ_MAX_RHS];
    float2* Pb = P + (size_t)blockIdx.x * m.M * m.nv;
    const int t = threadIdx.x, nt = blockDim.x, lane = t & 31, w = t >> 5, nw = nt >> 5;
    for (int k = 0; k < m.nv; k++) {
        double n0[1] = {0.0};
        for (int r = t; r < m.M; r += nt) { const float2 b = Pb[(size_t)r * m.nv + k]; n0[0] += (double)b.x * b.x + (double)b.y * b.y; }
        block_sum<1>(n0, sm);
        for (int pass = 0; pass < 2 && k > 0; pass++) {
            for (int j = w; j < k; j += nw) {
                double dr = 0.0, di = 0.0;
                for (int r = lane; r < m.M; r += 32) {
                    const float2 a = Pb[(size_t)r * m.nv + j], b = Pb[(size_t)r * m.nv + k];
                    dr += (double)a.x * b.x + (double)a.y * b.y;
                    di += (double)a.x * b.y - (double)a.y * b.x;
                }
#pragma unroll
                for (int off = 16; off >= 1; off >>= 1) { dr += __shfl_xor_sync(0xffffffffu, dr, off); di += __shfl_xor_sync(0xffffffffu, di, off); }
                if (lane == 0) dj[j] = make_float2((float)dr, (float)di);
            }
            __syncthreads();
            for (int r = t; r < m.M; r += nt) {
                float2 b = Pb[(size_t)r * m.nv + k];
                for (int j = 0; j < k; j++) {
                    const float2 a = Pb[(size_t)r * m.nv + j], d = dj[j];
                    b.x -= d.x * a.x - d.y * a.y;
                    b.y -= d.x * a.y + d.y * a.x;
                }
                Pb[(size_t)r * m.nv + k] = b;
            }
            __syncthreads();
        }
        double n[1] = {0.0};
        for (int r = t; r < m.M; r += nt) { const float2 b = Pb[(size_t)r * m.nv + k]; n[0] += (double)b.x * b.x + (double)b.y * b.y; }
        block_sum<1>(n, sm);
        if (!(n[0] > 1e-8 * n0[0])) { if (t == 0) atomicExch(status, 1); n[0] = 1.0; }    // less than 1e-4 of the column is new
        const float sc = (float)(1.0 / sqrt(n[0]));
        for (int r = t; r < m.M; r += nt) { float2 b = Pb[(size_t)r * m.nv + k]; b.x *= sc; b.y *= sc; Pb[(size_t)r * m.nv + k] = b; }
        __syncthreads();
    }
}

// ---- restriction y = P^dag x and prolongation x (+)= P y, N right-hand sides ------------------------------------------------
// One CTA per (aggregate, chirality).  restrict: thread = (k, RHS group, row slice), sums over the rows of its slice of its column
// (P coalesced over k, x broadcast), slices added in order.  prolong: the 2 Nv x N coarse values of the block sit in shared memory, thread = (row, RHS group).
template <int R>
__global__ void __launch_bounds__(256) restrict_kernel(MgGeom m, int N, int S, const int* __restrict__ site_f, const float2* __restrict__ P,
                                                       const float* __restrict__ x, float2* __restrict__ yc) {
    // thread = (k, RHS group, slice): slice sl of S takes the sites i = sl, sl + S, ... of the aggregate; the slices' partial sums are
    // added in slice order through shared memory
    extern __shared__ float2 rs[];     // [S][nv * G][R]
    const int G = N / R, KG = m.nv * G;
    const int a = blockIdx.x >> 1, chi = blockIdx.x & 1;
    const int t = threadIdx.x;
    const int kg = t % KG, sl = t / KG;
    const int k = kg % m.nv, g = kg / m.nv;
    float ar[R], ai[R];
#pragma unroll
    for (int r = 0; r < R; r++) ar[r] = ai[r] = 0.f;
    if (sl < S) {
        const float2* Pb = P + (size_t)blockIdx.x * m.M * m.nv + k;
        const int* sf = site_f + (size_t)a * m.ns;
#pragma unroll 2
        for (int i = sl; i < m.ns; i += S) {
            const size_t base = fine_base<R>(sf[i], G, g) + (size_t)(12 * chi) * (SB * R);
#pragma unroll
            for (int c6 = 0; c6 < 6; c6++) {
                float xr[R], xi[R];
                ldv<R>(x + base + (size_t)(2 * c6) * (SB * R), xr);
                ldv<R>(x + base + (size_t)(2 * c6 + 1) * (SB * R), xi);
                const float2 p = __ldg(Pb + (size_t)(6 * i + c6) * m.nv);
#pragma unroll
                for (int r = 0; r < R; r++) { ar[r] += p.x * xr[r] + p.y * xi[r]; ai[r] += p.x * xi[r] - p.y * xr[r]; }
            }
        }
#pragma unroll
        for (int r = 0; r < R; r++) rs[((size_t)sl * KG + kg) * R + r] = make_float2(ar[r], ai[r]);
    }
    __syncthreads();
    if (t < KG) {
        float2* o = yc + ((size_t)a * m.nc + chi * m.nv + k) * N + g * R;
#pragma unroll
        for (int r = 0; r < R; r++) {
            float2 sum = make_float2(0.f, 0.f);
            for (int q = 0; q < S; q++) { const float2 v = rs[((size_t)q * KG + kg) * R + r]; sum.x += v.x; sum.y += v.y; }
            o[r] = sum;
        }
    }
}

template <int R, bool ACCUM>
__global__ void __launch_bounds__(256) prolong_kernel(MgGeom m, int N, const int* __restrict__ site_f, const float2* __restrict__ P,
                                                      const float2* __restrict__ yc, float* __restrict__ x) {
    extern __shared__ float2 ys[];     // [nv][N]
    const int G = N / R;
    const int a = blockIdx.x >> 1, chi = blockIdx.x & 1;
    const float2* src = yc + ((size_t)a * m.nc + chi * m.nv) * N;
    for (int q = threadIdx.x; q < m.nv * N; q += blockDim.x) ys[q] = src[q];
    __syncthreads();
    const float2* Pb = P + (size_t)blockIdx.x * m.M * m.nv;
    const int* sf = site_f + (size_t)a * m.ns;
    for (int w = threadIdx.x; w < m.M * G; w += blockDim.x) {
        const int mm = w % m.M, g = w / m.M;
        const int i = mm / 6, c6 = mm - 6 * i;
        float xr[R], xi[R];
#pragma unroll
        for (int r = 0; r < R; r++) xr[r] = xi[r] = 0.f;
        const float2* pr = Pb + (size_t)mm * m.nv;
        if ((m.nv & 1) == 0) {          // two columns per 16-byte load
            const float4* pr4 = reinterpret_cast<const float4*>(pr);
#pragma unroll 4
            for (int k2 = 0; k2 < (m.nv >> 1); k2++) {
                const float4 p = __ldg(pr4 + k2);
#pragma unroll
                for (int r = 0; r < R; r++) {
                    const float2 y0 = ys[(2 * k2) * N + g * R + r], y1 = ys[(2 * k2 + 1) * N + g * R + r];
                    xr[r] += p.x * y0.x - p.y * y0.y + p.z * y1.x - p.w * y1.y;
                    xi[r] += p.x * y0.y + p.y * y0.x + p.z * y1.y + p.w * y1.x;
                }
            }
        } else {
            for (int k = 0; k < m.nv; k++) {
                const float2 p = pr[k];
#pragma unroll
                for (int r = 0; r < R; r++) {
                    const float2 y = ys[k * N + g * R + r];
                    xr[r] += p.x * y.x - p.y * y.y;
                    xi[r] += p.x * y.y + p.y * y.x;
                }
            }
        }
        float* o = x + fine_base<R>(sf[i], G, g) + (size_t)(2 * (6 * chi + c6)) * (SB * R);
        if (ACCUM) {
            float or_[R], oi_[R];
            ldv<R>(o, or_); ldv<R>(o + SB * R, oi_);
#pragma unroll
            for (int r = 0; r < R; r++) { xr[r] += or_[r]; xi[r] += oi_[r]; }
        }
        stv<R>(o, xr); stv<R>(o + SB * R, xi);
    }
}

// ---- coarse operator y[a] = sum_d A_c[a][d] x[nbr(a, d)], N right-hand sides ------------------------------------------------
// One CTA of 9 warps per (coarse site, chunk of NCH right-hand sides): warp d streams the block of stencil direction d, lane l owns
// the row pair (2l, 2l+1) (one 16-byte load per column, 4 columns in flight), the neighbour's values of a column are NCH
// consecutive float2 that every lane reads from the same address (one L1 broadcast).  The 9 partial results meet in shared memory and
// are added in direction order 0..8 (deterministic).  HBM-bound on A_c: every entry read once feeds NCH complex multiply-adds per
// chunk -- the batched coarse operator is the matrix-matrix form of PAPER.md L133-137; 2 Nv <= 64 keeps a block row inside one warp.
template <int NCH>
__global__ void __launch_bounds__(288) coarse_apply_kernel(MgGeom m, int N, const int* __restrict__ nbr, const float2* __restrict__ Ac,
                                                           const float2* __restrict__ x, float2* __restrict__ y) {
    extern __shared__ float2 red[];     // [9][nc][NCH]
    const int a = blockIdx.x, r0 = blockIdx.y * NCH;
    const int d = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nc = m.nc;
    const int nb = nbr[a * 9 + d];
    float2 acc[2][NCH];
#pragma unroll
    for (int q = 0; q < 2; q++)
#pragma unroll
        for (int r = 0; r < NCH; r++) acc[q][r] = make_float2(0.f, 0.f);
    if (nb >= 0 && 2 * lane < nc) {
        const float4* A = reinterpret_cast<const float4*>(Ac + ((size_t)(a * 9 + d) * nc) * nc) + lane;      // column stride nc / 2 float4
        const float2* xv = x + (size_t)nb * nc * N + r0;
        const int cs = nc >> 1;
        constexpr int U = 4;            // columns per batch; the next batch's 16-byte loads are issued before this batch's arithmetic
        float4 cur[U], nxt[U];
#pragma unroll
        for (int u = 0; u < U; u++) cur[u] = u < nc ? __ldg(A + (size_t)u * cs) : make_float4(0.f, 0.f, 0.f, 0.f);
        for (int col0 = 0; col0 < nc; col0 += U) {
#pragma unroll
            for (int u = 0; u < U; u++) nxt[u] = col0 + U + u < nc ? __ldg(A + (size_t)(col0 + U + u) * cs) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
            for (int u = 0; u < U; u++) {
                const int col = col0 + u < nc ? col0 + u : nc - 1;      // a padded column multiplies zeros
                float2 v[NCH];
                if constexpr (NCH >= 2) {
#pragma unroll
                    for (int r = 0; r < NCH; r += 2) {
                        const float4 w = __ldg(reinterpret_cast<const float4*>(xv + (size_t)col * N + r));
                        v[r] = make_float2(w.x, w.y); v[r + 1] = make_float2(w.z, w.w);
                    }
                } else v[0] = __ldg(xv + (size_t)col * N);
                const float4 c = cur[u];
#pragma unroll
                for (int r = 0; r < NCH; r++) {
                    acc[0][r].x = fmaf(c.x, v[r].x, acc[0][r].x); acc[0][r].x = fmaf(-c.y, v[r].y, acc[0][r].x);
                    acc[0][r].y = fmaf(c.x, v[r].y, acc[0][r].y); acc[0][r].y = fmaf(c.y, v[r].x, acc[0][r].y);
                    acc[1][r].x = fmaf(c.z, v[r].x, acc[1][r].x); acc[1][r].x = fmaf(-c.w, v[r].y, acc[1][r].x);
                    acc[1][r].y = fmaf(c.z, v[r].y, acc[1][r].y); acc[1][r].y = fmaf(c.w, v[r].x, acc[1][r].y);
                }
            }
#pragma unroll
            for (int u = 0; u < U; u++) cur[u] = nxt[u];
        }
    }
    if (2 * lane < nc) {
#pragma unroll
        for (int q = 0; q < 2; q++)
#pragma unroll
            for (int r = 0; r < NCH; r++) red[((size_t)d * nc + 2 * lane + q) * NCH + r] = acc[q][r];
    }
    __syncthreads();
    for (int e = threadIdx.x; e < nc * NCH; e += blockDim.x) {
        float2 sum = make_float2(0.f, 0.f);
#pragma unroll
        for (int dd = 0; dd < 9; dd++) { const float2 v = red[(size_t)dd * nc * NCH + e]; sum.x += v.x; sum.y += v.y; }
        const int row = e / NCH, r = e - row * NCH;
        y[((size_t)a * nc + row) * N + r0 + r] = sum;
    }
}

// ---- Galerkin coarse operator by probing -----------------------------------------------------------------------------------
// Right-hand side r of a probing batch carries column col of P (chirality col / Nv, vector col % Nv of EVERY aggregate), masked to
// the aggregates with a_mu % ncol == colour (mu < 0: unmasked).  After y = P^dag M (probe), row block a' of y is
//   unmasked              : sum over all 9 blocks of column col         -> self block (the others are subtracted afterwards)
//   a'_mu + 1 == colour   : the +mu block of a' (its +mu neighbour is the only coloured aggregate among its 9)
//   a'_mu - 1 == colour   : the -mu block
//   ncol == 2 (Lc_mu = 2) : a'_mu != colour: +mu and -mu neighbour coincide, the sum is stored as the +mu block
struct ProbeDesc { int col[LQ_MAX_RHS], mu[LQ_MAX_RHS], colour[LQ_MAX_RHS], ncol[LQ_MAX_RHS]; };

__device__ __forceinline__ int coarse_coord(const MgGeom& m, int a, int mu) {
    for (int n = 0; n < mu; n++) a /= m.Lc[n];
    return a % m.Lc[mu];
}

template <int R>
__global__ void probe_fill_kernel(MgGeom m, int N, ProbeDesc pd, const int* __restrict__ site_f, const float2* __restrict__ P, float* __restrict__ x) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= (long long)m.Vc * m.ns * N) return;
    const int k = (int)(tid % N);
    const long long q = tid / N;
    const int i = (int)(q % m.ns), a = (int)(q / m.ns);
    const int G = N / R;
    const int col = pd.col[k], chi = col / m.nv, kv = col % m.nv;
    bool on = col >= 0;
    if (on && pd.mu[k] >= 0) on = (coarse_coord(m, a, pd.mu[k]) % pd.ncol[k]) == pd.colour[k];
    float* o = x + fine_base<R>(site_f[(size_t)a * m.ns + i], G, k / R) + (k % R);
    const float2* Pb = P + ((size_t)(a * 2 + (on ? chi : 0)) * m.M + 6 * i) * m.nv + (on ? kv : 0);
#pragma unroll
    for (int c = 0; c < 12; c++) {
        float2 v = make_float2(0.f, 0.f);
        if (on && c / 6 == chi) v = Pb[(size_t)(c % 6) * m.nv];
        o[(size_t)(2 * c) * (SB * R)] = v.x;
        o[(size_t)(2 * c + 1) * (SB * R)] = v.y;
    }
}

__global__ void probe_scatter_kernel(MgGeom m, int N, ProbeDesc pd, const float2* __restrict__ yc, float2* __restrict__ Ac) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= (long long)m.Vc * m.nc * N) return;
    const int k = (int)(tid % N);
    const long long q = tid / N;
    const int row = (int)(q % m.nc), a = (int)(q / m.nc);
    const int col = pd.col[k];
    if (col < 0) return;
    int d = -1;
    if (pd.mu[k] < 0) d = 0;
    else {
        const int am = coarse_coord(m, a, pd.mu[k]), nc_ = pd.ncol[k], cl = pd.colour[k];
        if (nc_ == 2) { if (am % 2 != cl) d = 1 + 2 * pd.mu[k]; }
        else if ((am + 1) % nc_ == cl) d = 1 + 2 * pd.mu[k];
        else if ((am + nc_ - 1) % nc_ == cl) d = 2 + 2 * pd.mu[k];
    }
    if (d < 0) return;
    Ac[((size_t)(a * 9 + d) * m.nc + col) * m.nc + row] = yc[tid];
}

// self block = (sum of all blocks) - (the stored neighbour blocks)
__global__ void self_fix_kernel(MgGeom m, const int* __restrict__ nbr, float2* __restrict__ Ac) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int n2 = m.nc * m.nc;
    if (tid >= (long long)m.Vc * n2) return;
    const int e = (int)(tid % n2), a = (int)(tid / n2);
    float2 s = Ac[(size_t)(a * 9) * n2 + e];
    for (int d = 1; d < 9; d++) {
        if (nbr[a * 9 + d] < 0) continue;
        const float2 v = Ac[(size_t)(a * 9 + d) * n2 + e];
        s.x -= v.x; s.y -= v.y;
    }
    Ac[(size_t)(a * 9) * n2 + e] = s;
}

// ---- per-RHS complex block-BLAS of the Krylov solvers, fine (native fp32, both parities in one launch) and coarse ----------
// Device scalars are raw sums d[0..2][LQ_MAX_RHS] = (Re <a,b>, Im <a,b>, ||a||^2) with <a,b> = sum conj(a) b; the consumer
// derives its coefficient c_k = (Re + i Im) / ||a||^2 (zero when the denominator is zero).  Two sets (da, db) are added first:
// the stencil kernel's fused epilogue delivers one set per parity.
__device__ __forceinline__ void coef_of(const double* __restrict__ da, const double* __restrict__ db, int k, float& cr, float& ci) {
    double re = da[k], im = da[LQ_MAX_RHS + k], den = da[2 * LQ_MAX_RHS + k];
    if (db) { re += db[k]; im += db[LQ_MAX_RHS + k]; den += db[2 * LQ_MAX_RHS + k]; }
    if (den > 0.0) { cr = (float)(re / den); ci = (float)(im / den); } else { cr = 0.f; ci = 0.f; }
}

// fine: thread = (unit, site) with the R right-hand sides of the unit's group; a warp = one unit (reduce.cuh's mapping, VW = R)
template <int R>
__global__ void __launch_bounds__(128) fine_cdot3_kernel(int units, int N, int G, const float* __restrict__ a, const float* __restrict__ b, double* partials) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int u = (int)(tid >> 5), s = (int)(tid & 31);
    double part[3][R];
#pragma unroll
    for (int q = 0; q < 3; q++)
#pragma unroll
        for (int r = 0; r < R; r++) part[q][r] = 0.0;
    if (u < units) {
        const size_t own = (size_t)u * (24 * SB * R) + (size_t)s * R;
#pragma unroll
        for (int c = 0; c < 12; c++) {
            float ar[R], ai[R], br[R], bi[R];
            ldv<R>(a + own + (size_t)(2 * c) * (SB * R), ar); ldv<R>(a + own + (size_t)(2 * c + 1) * (SB * R), ai);
            ldv<R>(b + own + (size_t)(2 * c) * (SB * R), br); ldv<R>(b + own + (size_t)(2 * c + 1) * (SB * R), bi);
#pragma unroll
            for (int r = 0; r < R; r++) {
                part[0][r] += (double)(ar[r] * br[r] + ai[r] * bi[r]);
                part[1][r] += (double)(ar[r] * bi[r] - ai[r] * br[r]);
                part[2][r] += (double)(ar[r] * ar[r] + ai[r] * ai[r]);
            }
        }
    }
    reduce_multi<3, R, R>(part, N, G, partials);
}

// y1 += s1 c x1 ; y2 += s2 c x2 (y1 / x1 may be null; x1 may be y2: the minimal-residual step z += w res, res -= w t reads res
// before it updates it, so the vector pointers carry no __restrict__); NORM: partial rows of ||y2||^2
template <int R, bool NORM>
__global__ void __launch_bounds__(128) fine_caxpy2_kernel(int units, int N, int G, float* y1, const float* x1, float s1, float* y2, const float* x2, float s2,
                                                          const double* __restrict__ da, const double* __restrict__ db, double* partials) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int u = (int)(tid >> 5), s = (int)(tid & 31);
    double part[R];
#pragma unroll
    for (int r = 0; r < R; r++) part[r] = 0.0;
    if (u < units) {
        const int rhs0 = (u % G) * R;
        float cr[R], ci[R];
#pragma unroll
        for (int r = 0; r < R; r++) coef_of(da, db, rhs0 + r, cr[r], ci[r]);
        const size_t own = (size_t)u * (24 * SB * R) + (size_t)s * R;
#pragma unroll
        for (int c = 0; c < 12; c++) {
            const size_t o0 = own + (size_t)(2 * c) * (SB * R), o1 = o0 + SB * R;
            float xr[R], xi[R], yr[R], yi[R];
            if (y1 != nullptr) {
                ldv<R>(x1 + o0, xr); ldv<R>(x1 + o1, xi); ldv<R>(y1 + o0, yr); ldv<R>(y1 + o1, yi);
#pragma unroll
                for (int r = 0; r < R; r++) { yr[r] += s1 * (cr[r] * xr[r] - ci[r] * xi[r]); yi[r] += s1 * (cr[r] * xi[r] + ci[r] * xr[r]); }
                stv<R>(y1 + o0, yr); stv<R>(y1 + o1, yi);
            }
            ldv<R>(x2 + o0, xr); ldv<R>(x2 + o1, xi); ldv<R>(y2 + o0, yr); ldv<R>(y2 + o1, yi);
#pragma unroll
            for (int r = 0; r < R; r++) {
                yr[r] += s2 * (cr[r] * xr[r] - ci[r] * xi[r]); yi[r] += s2 * (cr[r] * xi[r] + ci[r] * xr[r]);
                if (NORM) part[r] += (double)(yr[r] * yr[r] + yi[r] * yi[r]);
            }
            stv<R>(y2 + o0, yr); stv<R>(y2 + o1, yi);
        }
    }
    if constexpr (NORM) reduce_per_rhs<R, R>(part, N, G, partials);
}

// coarse: arrays [n][N] float2; block = (N, BY): thread (x = rhs, y = row slot), rows grid-strided; per-block partial rows in the
// format reduce_finish expects ([q * N + rhs])
template <int NQ>
__device__ __forceinline__ void coarse_block_rows(double (&part)[NQ], int N, double* partials) {
    extern __shared__ double csm[];     // [BY][N]
    const int tx = threadIdx.x, ty = threadIdx.y, BY = blockDim.y;
#pragma unroll
    for (int q = 0; q < NQ; q++) {
        __syncthreads();
        csm[ty * N + tx] = part[q];
        __syncthreads();
        if (ty == 0) {
            double s = 0.0;
            for (int yy = 0; yy < BY; yy++) s += csm[yy * N + tx];
            partials[(size_t)blockIdx.x * (NQ * N) + q * N + tx] = s;
        }
    }
}
__global__ void coarse_cdot3_kernel(long long n, int N, const float2* __restrict__ a, const float2* __restrict__ b, double* partials) {
    double part[3] = {0.0, 0.0, 0.0};
    for (long long i = (long long)blockIdx.x * blockDim.y + threadIdx.y; i < n; i += (long long)gridDim.x * blockDim.y) {
        const float2 av = a[i * N + threadIdx.x], bv = b[i * N + threadIdx.x];
        part[0] += (double)(av.x * bv.x + av.y * bv.y);
        part[1] += (double)(av.x * bv.y - av.y * bv.x);
        part[2] += (double)(av.x * av.x + av.y * av.y);
    }
    coarse_block_rows<3>(part, N, partials);
}
template <bool NORM>
__global__ void coarse_caxpy2_kernel(long long n, int N, float2* y1, const float2* x1, float s1, float2* y2, const float2* x2, float s2,
                                     const double* __restrict__ da, double* partials) {
    float cr, ci;
    coef_of(da, nullptr, threadIdx.x, cr, ci);
    double part[1] = {0.0};
    for (long long i = (long long)blockIdx.x * blockDim.y + threadIdx.y; i < n; i += (long long)gridDim.x * blockDim.y) {
        const long long e = i * N + threadIdx.x;
        if (y1 != nullptr) {
            const float2 x = x1[e]; float2 y = y1[e];
            y.x += s1 * (cr * x.x - ci * x.y); y.y += s1 * (cr * x.y + ci * x.x);
            y1[e] = y;
        }
        const float2 x = x2[e]; float2 y = y2[e];
        y.x += s2 * (cr * x.x - ci * x.y); y.y += s2 * (cr * x.y + ci * x.x);
        y2[e] = y;
        if (NORM) part[0] += (double)(y.x * y.x + y.y * y.y);
    }
    if constexpr (NORM) coarse_block_rows<1>(part, N, partials);
}

// out = a + sign b (out may be a)
__global__ void sub4_kernel(size_t n4, float4* out, const float4* a, const float4* __restrict__ b, float sign) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n4) return;
    const float4 x = a[i], y = b[i];
    out[i] = make_float4(x.x + sign * y.x, x.y + sign * y.y, x.z + sign * y.z, x.w + sign * y.w);
}

// ---- boundary conversions of coarse vectors: host/canonical complex fp64 [rhs][Vc][nc] <-> internal float2 [Vc][nc][N] ----
__global__ void coarse_pack_kernel(long long n, int N, const double* __restrict__ in, float2* __restrict__ out) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= n * N) return;
    const int k = (int)(tid % N);
    const long long i = tid / N;
    out[tid] = make_float2((float)in[2 * ((long long)k * n + i)], (float)in[2 * ((long long)k * n + i) + 1]);
}
__global__ void coarse_unpack_kernel(long long n, int N, const float2* __restrict__ in, double* __restrict__ out) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= n * N) return;
    const int k = (int)(tid % N);
    const long long i = tid / N;
    const float2 v = in[tid];
    out[2 * ((long long)k * n + i)] = v.x; out[2 * ((long long)k * n + i) + 1] = v.y;
}

}  // namespace mg
