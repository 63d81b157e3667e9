// eigen_kernels.cuh -- per-time-slice vector kernels of the batched Lanczos eigensolver (
// "batched Lanczos", the time extent is the batch).  One colour-vector field = native cv layout
// with N = 1 (common layout of laplace.cu): element (parity, cb, j) at parity*pbe + ((cb/32)*6 + j)*32 + cb%32, fp64.
// Every kernel takes per-slice coefficients: the Lt time-slices are independent eigenproblems advancing in lockstep.
#pragma once
#include <cooperative_groups.h>
#include "common.cuh"

struct SliceGeom { int Vh, S3h, Lt; size_t pbe; FastDiv dS3h; };   // S3h = sites of one time-slice per parity

// thread i < 2*Vh -> (parity, cb); returns the element offset of real 0 and the slice
__device__ __forceinline__ bool slice_site(const SliceGeom& g, long long i, size_t& off, int& t) {
    if (i >= 2LL * g.Vh) return false;
    const int parity = i >= g.Vh ? 1 : 0;
    const int cb = (int)(i - (long long)parity * g.Vh);
    t = g.dS3h.div(cb);
    off = (size_t)parity * g.pbe + (size_t)(cb / SB) * (6 * SB) + (cb % SB);
    return true;
}

// partial[t][chunk] = sum over the sites of the chunk of conj(a) b  (complex); chunks never straddle slices:
// grid = Lt * nchunk blocks of 256 threads, each thread strides over the slice's 2*S3h sites.
__global__ void slice_dot_kernel(SliceGeom g, int nchunk, const double* __restrict__ a, const double* __restrict__ b, double2* __restrict__ partial) {
    const int t = blockIdx.x / nchunk, ch = blockIdx.x - t * nchunk;
    double sr = 0.0, si = 0.0;
    const int per_slice = 2 * g.S3h;
    for (int i = ch * blockDim.x + threadIdx.x; i < per_slice; i += nchunk * blockDim.x) {
        const int parity = i >= g.S3h ? 1 : 0;
        const int cb = t * g.S3h + (i - parity * g.S3h);
        const size_t off = (size_t)parity * g.pbe + (size_t)(cb / SB) * (6 * SB) + (cb % SB);
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const double ar = a[off + (2 * c) * SB], ai = a[off + (2 * c + 1) * SB];
            const double br = b[off + (2 * c) * SB], bi = b[off + (2 * c + 1) * SB];
            sr += ar * br + ai * bi; si += ar * bi - ai * br;
        }
    }
    __shared__ double shr[256], shi[256];
    shr[threadIdx.x] = sr; shi[threadIdx.x] = si;
    __syncthreads();
    for (int s = blockDim.x >> 1; s > 0; s >>= 1) {
        if (threadIdx.x < s) { shr[threadIdx.x] += shr[threadIdx.x + s]; shi[threadIdx.x] += shi[threadIdx.x + s]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = make_double2(shr[0], shi[0]);
}
// out[t] = sum over chunks in fixed order
__global__ void slice_dot_final_kernel(int Lt, int nchunk, const double2* __restrict__ partial, double2* __restrict__ out) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= Lt) return;
    double sr = 0.0, si = 0.0;
    for (int c = 0; c < nchunk; c++) { sr += partial[t * nchunk + c].x; si += partial[t * nchunk + c].y; }
    out[t] = make_double2(sr, si);
}

// y += coef[t] * x   (complex coefficient per slice)
__global__ void slice_axpy_kernel(SliceGeom g, double* __restrict__ y, const double* __restrict__ x, const double2* __restrict__ coef) {
    size_t off; int t;
    if (!slice_site(g, (long long)blockIdx.x * blockDim.x + threadIdx.x, off, t)) return;
    const double cr = coef[t].x, ci = coef[t].y;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const double xr = x[off + (2 * c) * SB], xi = x[off + (2 * c + 1) * SB];
        y[off + (2 * c) * SB] += cr * xr - ci * xi;
        y[off + (2 * c + 1) * SB] += cr * xi + ci * xr;
    }
}
// y = s[t] * x   (real scale per slice; y may alias x)
__global__ void slice_scale_kernel(SliceGeom g, double* __restrict__ y, const double* __restrict__ x, const double* __restrict__ s) {
    size_t off; int t;
    if (!slice_site(g, (long long)blockIdx.x * blockDim.x + threadIdx.x, off, t)) return;
    const double f = s[t];
#pragma unroll
    for (int j = 0; j < 6; j++) y[off + j * SB] = f * x[off + j * SB];
}
// z = alpha x + beta y + gamma z   (global real scalars: the Chebyshev three-term recurrence)
__global__ void cv_axpbypcz_kernel(SliceGeom g, double* __restrict__ z, double alpha, const double* __restrict__ x, double beta, const double* __restrict__ y, double gamma) {
    size_t off; int t;
    if (!slice_site(g, (long long)blockIdx.x * blockDim.x + threadIdx.x, off, t)) return;
#pragma unroll
    for (int j = 0; j < 6; j++) {
        const size_t e = off + j * SB;
        z[e] = alpha * x[e] + beta * y[e] + (gamma != 0.0 ? gamma * z[e] : 0.0);
    }
}
// basis rotation: out[c] = sum_i Q[t][i][c] * V[i]  for c < k (real Q from the projected eigenproblem of slice t): a tall-skinny
// GEMM per slice; one thread = one real element row, 16 output columns per pass (the basis is re-read from L1/L2 once per pass)
__global__ void slice_rotate_kernel(SliceGeom g, int m, int k, const double* const* __restrict__ V, double* const* __restrict__ out, const double* __restrict__ Q) {
    constexpr int TC = 16;
    size_t off; int t;
    if (!slice_site(g, (long long)blockIdx.x * blockDim.x + threadIdx.x, off, t)) return;
    const double* q = Q + (size_t)t * m * k;
    for (int j = 0; j < 6; j++) {
        for (int c0 = 0; c0 < k; c0 += TC) {
            const int nc = min(TC, k - c0);
            double acc[TC];
#pragma unroll
            for (int cc = 0; cc < TC; cc++) acc[cc] = 0.0;
            for (int i = 0; i < m; i++) {
                const double v = V[i][off + j * SB];
                const double* qi = q + (size_t)i * k + c0;
#pragma unroll
                for (int cc = 0; cc < TC; cc++) if (cc < nc) acc[cc] += qi[cc] * v;
            }
#pragma unroll
            for (int cc = 0; cc < TC; cc++) if (cc < nc) out[c0 + cc][off + j * SB] = acc[cc];
        }
    }
}

// Gram-Schmidt as two batched kernels (the tall-skinny GEMV pair of the Lanczos step):
// multidot:  partial[t][chunk][i] = sum over the chunk of conj(V[i0+i]) w  for up to 8 vectors per block (blockIdx.y = tile)
__global__ void slice_multidot_kernel(SliceGeom g, int nchunk, int nv, const double* const* __restrict__ V, const double* __restrict__ w,
                                      double2* __restrict__ partial /*[Lt*nchunk][nv]*/) {
    constexpr int TV = 8;
    const int t = blockIdx.x / nchunk, ch = blockIdx.x - t * nchunk, i0 = blockIdx.y * TV;
    const int nt = min(TV, nv - i0);
    double sr[TV], si[TV];
#pragma unroll
    for (int i = 0; i < TV; i++) { sr[i] = 0.0; si[i] = 0.0; }
    const int per_slice = 2 * g.S3h;
    for (int s = ch * blockDim.x + threadIdx.x; s < per_slice; s += nchunk * blockDim.x) {
        const int parity = s >= g.S3h ? 1 : 0;
        const int cb = t * g.S3h + (s - parity * g.S3h);
        const size_t off = (size_t)parity * g.pbe + (size_t)(cb / SB) * (6 * SB) + (cb % SB);
        double wv[6];
#pragma unroll
        for (int j = 0; j < 6; j++) wv[j] = w[off + j * SB];
#pragma unroll
        for (int i = 0; i < TV; i++) {
            if (i < nt) {
                const double* v = V[i0 + i];
#pragma unroll
                for (int c = 0; c < 3; c++) {
                    const double ar = v[off + (2 * c) * SB], ai = v[off + (2 * c + 1) * SB];
                    sr[i] += ar * wv[2 * c] + ai * wv[2 * c + 1]; si[i] += ar * wv[2 * c + 1] - ai * wv[2 * c];
                }
            }
        }
    }
    __shared__ double sh[8][2 * TV];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int i = 0; i < TV; i++) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) { sr[i] += __shfl_xor_sync(0xffffffffu, sr[i], o); si[i] += __shfl_xor_sync(0xffffffffu, si[i], o); }
        if (lane == 0) { sh[wid][2 * i] = sr[i]; sh[wid][2 * i + 1] = si[i]; }
    }
    __syncthreads();
    if (threadIdx.x < nt) {
        double a = 0.0, b = 0.0;
        for (int q = 0; q < (int)(blockDim.x >> 5); q++) { a += sh[q][2 * threadIdx.x]; b += sh[q][2 * threadIdx.x + 1]; }
        partial[(size_t)blockIdx.x * nv + i0 + threadIdx.x] = make_double2(a, b);
    }
}
// out[i][t] = sum over chunks (fixed order)
__global__ void slice_multidot_final_kernel(int Lt, int nchunk, int nv, const double2* __restrict__ partial, double2* __restrict__ out) {
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= Lt * nv) return;
    const int i = id / Lt, t = id - i * Lt;
    double sr = 0.0, si = 0.0;
    for (int c = 0; c < nchunk; c++) { const double2 p = partial[(size_t)(t * nchunk + c) * nv + i]; sr += p.x; si += p.y; }
    out[(size_t)i * Lt + t] = make_double2(sr, si);
}
// w -= sum_i H[i][t] V[i]
__global__ void slice_multiaxpy_kernel(SliceGeom g, int nv, double* __restrict__ w, const double* const* __restrict__ V, const double2* __restrict__ H) {
    size_t off; int t;
    if (!slice_site(g, (long long)blockIdx.x * blockDim.x + threadIdx.x, off, t)) return;
    double acc[6];
#pragma unroll
    for (int j = 0; j < 6; j++) acc[j] = w[off + j * SB];
    for (int i = 0; i < nv; i++) {
        const double cr = H[(size_t)i * g.Lt + t].x, ci = H[(size_t)i * g.Lt + t].y;
        const double* v = V[i];
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const double xr = v[off + (2 * c) * SB], xi = v[off + (2 * c + 1) * SB];
            acc[2 * c] -= cr * xr - ci * xi;
            acc[2 * c + 1] -= cr * xi + ci * xr;
        }
    }
#pragma unroll
    for (int j = 0; j < 6; j++) w[off + j * SB] = acc[j];
}

// ---- the projected matrices T[t] = V^dag B V are assembled ON THE DEVICE (no host round trip inside a Lanczos sweep) ----------
// column j from the Gram-Schmidt coefficients of step j: H0 (local pass, rows first0 .. j) + H1 (full pass, rows 0 .. j), rows
// [i][Lt] of double2; rows i < k (the kept Ritz vectors) couple to column j only in the first step after a restart (the arrow)
__global__ void t_column_kernel(int Lt, int nT, int j, int k, int first0, const double2* __restrict__ H0, const double2* __restrict__ H1, double* __restrict__ T) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= Lt * (j + 1)) return;
    const int t = idx % Lt, i = idx / Lt;
    const double h = (i >= first0 ? H0[(size_t)i * Lt + t].x : 0.0) + H1[(size_t)i * Lt + t].x;
    if (i >= k || j == k || i == j) {
        double* Tt = T + (size_t)t * nT * nT;
        Tt[(size_t)i * nT + j] = h; Tt[(size_t)j * nT + i] = h;
    }
}
// sub-diagonal entry beta_j = ||w|| of step j, or the residual norm beta_m of the last step
__global__ void t_beta_kernel(int Lt, int nT, int j, int m, const double* __restrict__ beta, double* __restrict__ T, double* __restrict__ beta_m) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= Lt) return;
    if (j + 1 < m) { double* Tt = T + (size_t)t * nT * nT; Tt[(size_t)(j + 1) * nT + j] = beta[t]; Tt[(size_t)j * nT + j + 1] = beta[t]; }
    else beta_m[t] = beta[t];
}
// thick restart: T <- diag(theta_0 .. theta_{keep-1})
__global__ void t_reset_kernel(int Lt, int nT, int keep, int m, const double* __restrict__ theta, double* __restrict__ T) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)Lt * nT * nT) return;
    const int t = (int)(idx / ((long long)nT * nT)), e = (int)(idx - (long long)t * nT * nT), i = e / nT, jj = e - i * nT;
    T[idx] = (i == jj && i < keep) ? theta[(size_t)t * m + i] : 0.0;
}


// ---- Ritz step on the device: all Lt projected matrices at once, one CTA per time-slice ---------------------------------------
// Parallel two-sided Jacobi (Brent-Luk round-robin ordering): in every step the n/2 disjoint index pairs (p, q) get their
// rotations from the current 2x2 diagonal blocks; the matrix then splits into (n/2)^2 independent 2x2 blocks B(P,Q) that become
// R_P^T B R_Q in place (each element belongs to exactly one block), and rows p, q of Q^T are rotated.  n - 1 steps = one sweep;
// sweeps repeat until the off-diagonal Frobenius norm is below 1e-14 of the matrix norm.  A and Q^T live in global memory (they
// stay in L2: 2 x 8 n^2 bytes per slice).  A slice is worked on by a CLUSTER of RITZ_CLUSTER thread blocks (one CTA alone is bound by
// its SM's L1 bandwidth: 0.13 s for m = 288): every CTA derives the same rotations, takes every RITZ_CLUSTER-th chunk of the block
// updates and meets the others at a cluster barrier (which also invalidates L1) once per step.  Afterwards the eigenvalues are ranked by |theta| descending (the Chebyshev map sends
// the wanted end of the spectrum to the largest |T_d|) and the first `keep` eigenvectors, the Ritz residual estimates
// |beta_m q_{m-1,i}| / |theta_0| and the sorted eigenvalues are written in the layouts the restart needs.
constexpr int RITZ_THREADS = 1024;
constexpr int RITZ_MAXN = 512;
constexpr int RITZ_CLUSTER = 4;

__global__ void __cluster_dims__(RITZ_CLUSTER, 1, 1) __launch_bounds__(RITZ_THREADS) ritz_jacobi_kernel(int m, int keep, int n_ev, double* __restrict__ Aall /*[Lt][n][n], n = m rounded up to even*/,
                                                                   double* __restrict__ QTall /*[Lt][n][n]*/, const double* __restrict__ beta /*[Lt]*/,
                                                                   double* __restrict__ theta /*[Lt][m]*/, double* __restrict__ Qk /*[Lt][m][keep]*/,
                                                                   double* __restrict__ res /*[Lt][n_ev]*/, int* __restrict__ sweeps_out /*[Lt]*/) {
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank();
    const int n = (m + 1) & ~1, half = n / 2;
    const int t = blockIdx.x / RITZ_CLUSTER, tid = threadIdx.x, nt = blockDim.x;
    const int gtid = rank * nt + tid, gnt = RITZ_CLUSTER * nt;      // thread index / count within the cluster
    double* A = Aall + (size_t)t * n * n;
    double* QT = QTall + (size_t)t * n * n;
    __shared__ double s_c[RITZ_MAXN / 2], s_s[RITZ_MAXN / 2];
    __shared__ int s_p[RITZ_MAXN / 2], s_q[RITZ_MAXN / 2];
    __shared__ double s_red[RITZ_THREADS / 32];
    __shared__ double s_off, s_tot;
    for (int i = gtid; i < n * n; i += gnt) QT[i] = (i / n == i % n) ? 1.0 : 0.0;
    __threadfence();
    cluster.sync();
    int sweep = 0;
    for (; sweep < 40; sweep++) {
        // convergence: off-diagonal norm against the whole norm (fixed-order block reduction)
        double off = 0.0, tot = 0.0;
        for (int i = tid; i < n * n; i += nt) { const double v = __ldcg(A + i); tot += v * v; if (i / n != i % n) off += v * v; }
        for (int pass = 0; pass < 2; pass++) {
            double v = pass == 0 ? off : tot;
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if ((tid & 31) == 0) s_red[tid >> 5] = v;
            __syncthreads();
            if (tid == 0) { double sum = 0.0; for (int w = 0; w < nt / 32; w++) sum += s_red[w]; if (pass == 0) s_off = sum; else s_tot = sum; }
            __syncthreads();
        }
        if (s_off <= 1e-28 * s_tot) break;
        for (int step = 0; step < n - 1; step++) {
            // rotations of this step's pairs from the current diagonal blocks
            if (tid < half) {
                int p, q;
                if (tid == 0) { p = n - 1; q = step; }
                else { p = (step + tid) % (n - 1); q = (step - tid + (n - 1)) % (n - 1); }
                const double apq = __ldcg(A + (size_t)p * n + q), app = __ldcg(A + (size_t)p * n + p), aqq = __ldcg(A + (size_t)q * n + q);
                double cs = 1.0, sn = 0.0;
                if (fabs(apq) > 1e-300) {
                    const double th = (aqq - app) / (2.0 * apq);
                    const double tt = (th >= 0.0 ? 1.0 : -1.0) / (fabs(th) + sqrt(th * th + 1.0));
                    cs = 1.0 / sqrt(tt * tt + 1.0); sn = tt * cs;
                }
                s_c[tid] = cs; s_s[tid] = sn; s_p[tid] = p; s_q[tid] = q;
            }
            __syncthreads();
            // A <- J^T A J by independent 2x2 blocks; Q^T rows
            for (int b = gtid; b < half * half; b += gnt) {
                const int k1 = b / half, k2 = b - k1 * half;
                const int p1 = s_p[k1], q1 = s_q[k1], p2 = s_p[k2], q2 = s_q[k2];
                const double c1 = s_c[k1], s1 = s_s[k1], c2 = s_c[k2], s2 = s_s[k2];
                const double bpp = __ldcg(A + (size_t)p1 * n + p2), bpq = __ldcg(A + (size_t)p1 * n + q2), bqp = __ldcg(A + (size_t)q1 * n + p2), bqq = __ldcg(A + (size_t)q1 * n + q2);
                const double tpp = c2 * bpp - s2 * bpq, tpq = s2 * bpp + c2 * bpq, tqp = c2 * bqp - s2 * bqq, tqq = s2 * bqp + c2 * bqq;
                double opp = c1 * tpp - s1 * tqp, opq = c1 * tpq - s1 * tqq, oqp = s1 * tpp + c1 * tqp, oqq = s1 * tpq + c1 * tqq;
                if (k1 == k2) { opq = 0.0; oqp = 0.0; }
                A[(size_t)p1 * n + p2] = opp; A[(size_t)p1 * n + q2] = opq; A[(size_t)q1 * n + p2] = oqp; A[(size_t)q1 * n + q2] = oqq;
            }
            for (int b = gtid; b < half * n; b += gnt) {
                const int k = b / n, j = b - k * n;
                const int p = s_p[k], q = s_q[k];
                const double cs = s_c[k], sn = s_s[k];
                const double vp = __ldcg(QT + (size_t)p * n + j), vq = __ldcg(QT + (size_t)q * n + j);
                QT[(size_t)p * n + j] = cs * vp - sn * vq; QT[(size_t)q * n + j] = sn * vp + cs * vq;
            }
            __threadfence();
            cluster.sync();          // the other CTAs' updates are visible (and the barrier drops this SM's stale L1 lines)
        }
    }
    if (rank != 0) return;           // ranking and output by the first CTA of the cluster
    if (tid == 0) sweeps_out[t] = sweep;
    // rank by |theta| descending (ties by index): rank_i = number of eigenvalues that come before i
    __shared__ int s_ord[RITZ_MAXN];
    for (int i = tid; i < RITZ_MAXN; i += nt) s_ord[i] = 0;       // a NaN in the matrix must not leave an index unset
    __syncthreads();
    for (int i = tid; i < m; i += nt) {
        const double di = fabs(__ldcg(A + (size_t)i * n + i));
        int r = 0;
        for (int j = 0; j < m; j++) { const double dj = fabs(__ldcg(A + (size_t)j * n + j)); if (dj > di || (dj == di && j < i)) r++; }
        s_ord[r] = i;
        theta[(size_t)t * m + r] = __ldcg(A + (size_t)i * n + i);
    }
    __syncthreads();
    const double th0 = fmax(fabs(__ldcg(A + (size_t)s_ord[0] * n + s_ord[0])), 1e-300);
    for (int b = tid; b < m * keep; b += nt) {
        const int i = b / keep, cidx = b - i * keep;
        Qk[((size_t)t * m + i) * keep + cidx] = __ldcg(QT + (size_t)s_ord[cidx] * n + i);
    }
    for (int cidx = tid; cidx < n_ev; cidx += nt) res[(size_t)t * n_ev + cidx] = fabs(beta[t] * __ldcg(QT + (size_t)s_ord[cidx] * n + (m - 1))) / th0;
}

