// clover.cu -- clover term and its inverse on the device (8(c.1) steps 5, 6).
//
// F_{mu nu} = (Q - Q^dag)/(8i) from the four plaquette leaves around x (periodic wrap, no boundary sign).
// In the DeGrand-Rossi basis sigma_{mu nu} = i gamma_mu gamma_nu is block diagonal in chirality:
//   sigma_xy = diag(s3, s3)   sigma_xz = diag(s2, s2)   sigma_yz = diag(s1, s1)
//   sigma_xt = diag(-s1, s1)  sigma_yt = diag(s2, -s2)  sigma_zt = diag(-s3, s3)      (s_k = Pauli matrices)
// so with k = kappa*csw the two 6x6 Hermitian blocks (index 3*spin_in_block + colour) are
//   A+- = [[1 - k B3, -k (B1 - i B2)], [-k (B1 + i B2), 1 + k B3]]
//   A+ : B3 = F_xy - F_zt, B2 = F_xz + F_yt, B1 = F_yz - F_xt
//   A- : B3 = F_xy + F_zt, B2 = F_xz - F_yt, B1 = F_yz + F_xt
// Each block is stored as 6 real diagonal entries + 15 complex lower-triangular entries (36 reals), and is
// inverted in fp64 by Gauss-Jordan elimination without pivoting (positive definite => positive pivots).
#include "internal.cuh"

struct M3 { double re[9], im[9]; };

__device__ inline void m3_identity(M3& a) {
#pragma unroll
    for (int k = 0; k < 9; k++) { a.re[k] = (k % 4 == 0) ? 1.0 : 0.0; a.im[k] = 0.0; }
}
// o = a * b   or   o = a * b^dag
template <bool BDAG> __device__ inline void m3_mul(const M3& a, const M3& b, M3& o) {
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            double sr = 0, si = 0;
#pragma unroll
            for (int k = 0; k < 3; k++) {
                const double br = BDAG ? b.re[3 * j + k] : b.re[3 * k + j];
                const double bi = BDAG ? -b.im[3 * j + k] : b.im[3 * k + j];
                sr += a.re[3 * i + k] * br - a.im[3 * i + k] * bi;
                si += a.re[3 * i + k] * bi + a.im[3 * i + k] * br;
            }
            o.re[3 * i + j] = sr; o.im[3 * i + j] = si;
        }
}
__device__ inline void load_link64(const double* __restrict__ gauge, const Geom& g, const int* x, int mu, M3& u) {
    int parity, cb;
    coords_to_cb(g, x[0], x[1], x[2], x[3], parity, cb);
    double r[18];
    load_planes<double, 18>(link_block(gauge, g.NB, 18, parity, cb / SB, mu), cb % SB, r);
#pragma unroll
    for (int k = 0; k < 9; k++) { u.re[k] = r[2 * k]; u.im[k] = r[2 * k + 1]; }
}
// walk one link: forward P <- P U_mu(x), x += mu ; backward x -= mu, P <- P U_mu(x)^dag
__device__ inline void step(const double* gauge, const Geom& g, int* x, int mu, int dir, M3& P) {
    M3 u, t;
    if (dir > 0) {
        load_link64(gauge, g, x, mu, u);
        m3_mul<false>(P, u, t);
        x[mu] = (x[mu] + 1 == g.L[mu]) ? 0 : x[mu] + 1;
    } else {
        x[mu] = (x[mu] == 0) ? g.L[mu] - 1 : x[mu] - 1;
        load_link64(gauge, g, x, mu, u);
        m3_mul<true>(P, u, t);
    }
    P = t;
}
// F_{mu nu}(x): Hermitian 3x3
__device__ void field_strength(const double* gauge, const Geom& g, const int* x0, int mu, int nu, M3& F) {
    M3 Q;
#pragma unroll
    for (int k = 0; k < 9; k++) { Q.re[k] = 0; Q.im[k] = 0; }
    // the four leaves, all counter-clockwise in the (mu,nu) plane, starting and ending at x0
    const int d1[4] = {mu, nu, mu, nu};
    const int s1[4][4] = {{+1, +1, -1, -1}, {+1, -1, -1, +1}, {-1, -1, +1, +1}, {-1, +1, +1, -1}};
    for (int leaf = 0; leaf < 4; leaf++) {
        int x[4] = {x0[0], x0[1], x0[2], x0[3]};
        M3 P; m3_identity(P);
        // leaf 0: +mu +nu -mu -nu ; leaf 1: +nu -mu -nu +mu ; leaf 2: -mu -nu +mu +nu ; leaf 3: -nu +mu +nu -mu
        const bool start_nu = (leaf == 1 || leaf == 3);
        for (int k = 0; k < 4; k++) {
            const int dir = start_nu ? d1[(k + 1) & 3] : d1[k];
            step(gauge, g, x, dir, s1[leaf][k], P);
        }
#pragma unroll
        for (int k = 0; k < 9; k++) { Q.re[k] += P.re[k]; Q.im[k] += P.im[k]; }
    }
    // F = (Q - Q^dag)/(8i) = -i (Q - Q^dag)/8
#pragma unroll
    for (int a = 0; a < 3; a++)
#pragma unroll
        for (int b = 0; b < 3; b++) {
            const double dr = Q.re[3 * a + b] - Q.re[3 * b + a];
            const double di = Q.im[3 * a + b] + Q.im[3 * b + a];
            F.re[3 * a + b] = di * 0.125;
            F.im[3 * a + b] = -dr * 0.125;
        }
}

// in-place inverse of a Hermitian positive-definite 6x6 (complex, dense); returns false if a pivot is <= 0
__device__ bool invert6(double (&mr)[6][6], double (&mi)[6][6]) {
    double ar[6][12], ai[6][12];
    for (int i = 0; i < 6; i++)
        for (int j = 0; j < 6; j++) { ar[i][j] = mr[i][j]; ai[i][j] = mi[i][j]; ar[i][6 + j] = (i == j) ? 1.0 : 0.0; ai[i][6 + j] = 0.0; }
    bool ok = true;
    for (int k = 0; k < 6; k++) {
        const double pr = ar[k][k], pi = ai[k][k];
        if (!(pr > 0.0)) ok = false;
        const double den = pr * pr + pi * pi;
        const double ir = pr / den, ii = -pi / den;
        for (int j = 0; j < 12; j++) { const double r = ar[k][j] * ir - ai[k][j] * ii, m = ar[k][j] * ii + ai[k][j] * ir; ar[k][j] = r; ai[k][j] = m; }
        for (int i = 0; i < 6; i++) {
            if (i == k) continue;
            const double fr = ar[i][k], fi = ai[i][k];
            for (int j = 0; j < 12; j++) { ar[i][j] -= fr * ar[k][j] - fi * ai[k][j]; ai[i][j] -= fr * ai[k][j] + fi * ar[k][j]; }
        }
    }
    for (int i = 0; i < 6; i++) for (int j = 0; j < 6; j++) { mr[i][j] = ar[i][6 + j]; mi[i][j] = ai[i][6 + j]; }
    return ok;
}
__device__ inline void pack_block(const double (&mr)[6][6], const double (&mi)[6][6], double* out36) {
    for (int i = 0; i < 6; i++) out36[i] = mr[i][i];
    for (int i = 1; i < 6; i++) for (int j = 0; j < i; j++) { const int idx = i * (i - 1) / 2 + j; out36[6 + 2 * idx] = mr[i][j]; out36[7 + 2 * idx] = mi[i][j]; }
}

__global__ void __launch_bounds__(64) clover_build_kernel(Geom g, const double* __restrict__ gauge, double k, double* clov, double* clovinv, int* flag) {
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 2 * g.Vh) return;
    const int parity = tid / g.Vh, cb = tid - parity * g.Vh;
    int xh, y, z, t, odd;
    cb_coords(g, parity, cb, xh, y, z, t, odd);
    const int x0[4] = {2 * xh + odd, y, z, t};
    M3 F[6];   // xy xz xt yz yt zt
    int p = 0;
    for (int mu = 0; mu < 4; mu++) for (int nu = mu + 1; nu < 4; nu++) field_strength(gauge, g, x0, mu, nu, F[p++]);
    double rec[72], recinv[72];
    for (int b = 0; b < 2; b++) {
        const double s = b == 0 ? -1.0 : 1.0;
        double mr[6][6], mi[6][6];
        for (int a = 0; a < 3; a++) for (int c = 0; c < 3; c++) {
            const int e = 3 * a + c;
            const double b3r = F[0].re[e] + s * F[5].re[e], b3i = F[0].im[e] + s * F[5].im[e];
            const double b2r = F[1].re[e] - s * F[4].re[e], b2i = F[1].im[e] - s * F[4].im[e];
            const double b1r = F[3].re[e] + s * F[2].re[e], b1i = F[3].im[e] + s * F[2].im[e];
            const double d = (a == c) ? 1.0 : 0.0;
            mr[a][c] = d - k * b3r;          mi[a][c] = -k * b3i;
            mr[3 + a][3 + c] = d + k * b3r;  mi[3 + a][3 + c] = k * b3i;
            // upper right: -k (B1 - i B2) ; lower left: -k (B1 + i B2)
            mr[a][3 + c] = -k * (b1r + b2i); mi[a][3 + c] = -k * (b1i - b2r);
            mr[3 + a][c] = -k * (b1r - b2i); mi[3 + a][c] = -k * (b1i + b2r);
        }
        pack_block(mr, mi, rec + 36 * b);
        if (!invert6(mr, mi)) atomicExch(flag, 1);
        pack_block(mr, mi, recinv + 36 * b);
    }
    store_planes<double, 72>(clover_block(clov, g.NB, parity, cb / SB), cb % SB, rec);
    store_planes<double, 72>(clover_block(clovinv, g.NB, parity, cb / SB), cb % SB, recinv);
}

__global__ void clover_to_fp32_kernel(int Vh, int NB, const double* __restrict__ src, float* __restrict__ dst) {
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 2 * Vh) return;
    const int parity = tid / Vh, cb = tid - parity * Vh;
    double r[72]; float f[72];
    load_planes<double, 72>(clover_block(src, NB, parity, cb / SB), cb % SB, r);
#pragma unroll
    for (int k = 0; k < 72; k++) f[k] = (float)r[k];
    store_planes<float, 72>(clover_block(dst, NB, parity, cb / SB), cb % SB, f);
}

int clover_build(lq_ctx* c, double kappa, double csw) {
    const size_t n = (size_t)2 * 72 * c->g.NB * SB;
    if (!c->clov64) {
        c->clov64 = (double*)dev_alloc(c, n * 8); c->clovinv64 = (double*)dev_alloc(c, n * 8);
        c->clov32 = (float*)dev_alloc(c, n * 4); c->clovinv32 = (float*)dev_alloc(c, n * 4);
        if (!c->clov64 || !c->clovinv64 || !c->clov32 || !c->clovinv32) return LQ_ENOMEM;
    }
    c->has_clover = false;      // the stored blocks are overwritten below: valid again only if every block is positive definite
    LQ_CUDA(c, cudaMemsetAsync(c->d_flag, 0, sizeof(int), c->stream));
    const int threads = 2 * c->g.Vh;
    clover_build_kernel<<<(threads + 63) / 64, 64, 0, c->stream>>>(c->g, c->gauge64, kappa * csw, c->clov64, c->clovinv64, c->d_flag);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    clover_to_fp32_kernel<<<(threads + 127) / 128, 128, 0, c->stream>>>(c->g.Vh, c->g.NB, c->clov64, c->clov32);
    LQ_LAUNCHED(c);
    clover_to_fp32_kernel<<<(threads + 127) / 128, 128, 0, c->stream>>>(c->g.Vh, c->g.NB, c->clovinv64, c->clovinv32);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    int flag = 0;
    LQ_CUDA(c, cudaMemcpyAsync(&flag, c->d_flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    LQ_CUDA(c, cudaStreamSynchronize(c->stream));
    if (flag) return set_err(c, LQ_ESINGULAR, "clover block not positive definite");
    c->kappa = kappa; c->csw = csw; c->has_clover = true;
    return 0;
}
