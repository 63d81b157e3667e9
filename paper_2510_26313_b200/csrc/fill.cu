// fill.cu -- device-side seeded inputs for the bench configurations that never exist on the host
// (BASELINE.json configs[2], configs[4]; SURVEY.md 8(c.2) reading #4).  This is the CUDA copy of the
// counter-based generator specified in paper_2510_26313_b200/inputs.py (same streams and index conventions);
// it contains none of the method's arithmetic beyond the SU(3) row projection of the input recipe.
#include "internal.cuh"

__host__ __device__ inline uint64_t mix64(uint64_t z) {
    z += 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
__host__ __device__ inline uint64_t stream_key(uint64_t seed, uint64_t stream) { return mix64(mix64(seed) + stream); }
__device__ inline void cgauss(uint64_t key, uint64_t idx, double& re, double& im) {
    const uint64_t b0 = mix64(key + 2 * idx), b1 = mix64(key + 2 * idx + 1);
    const double u1 = ((double)(b0 >> 11) + 0.5) * (1.0 / 9007199254740992.0);
    const double u2 = (double)(b1 >> 11) * (1.0 / 9007199254740992.0);
    const double r = sqrt(-log(u1));
    double s, c;
    sincospi(2.0 * u2, &s, &c);
    re = r * c; im = r * s;
}

__global__ void fill_gauge_kernel(Geom g, uint64_t key, double eps, double* __restrict__ native) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 8LL * g.Vh) return;
    const int cb = (int)(tid % g.Vh), pm = (int)(tid / g.Vh);
    const int parity = pm >> 2, mu = pm & 3;
    int xh, y, z, t, odd;
    cb_coords(g, parity, cb, xh, y, z, t, odd);
    const uint64_t site = (uint64_t)(2 * xh + odd) + (uint64_t)g.L[0] * (y + (uint64_t)g.L[1] * (z + (uint64_t)g.L[2] * t));
    double wr[9], wi[9];
    for (int e = 0; e < 9; e++) {
        double a, b;
        cgauss(key, (site * 4 + mu) * 9 + e, a, b);
        wr[e] = eps * a + ((e % 4 == 0) ? 1.0 : 0.0);
        wi[e] = eps * b;
    }
    // rows a = w[0..2], b = w[3..5]: a <- a/|a| ; b <- b - (a^dag b) a ; b <- b/|b| ; c = conj(a x b)
    double n = 0;
    for (int k = 0; k < 3; k++) n += wr[k] * wr[k] + wi[k] * wi[k];
    n = 1.0 / sqrt(n);
    for (int k = 0; k < 3; k++) { wr[k] *= n; wi[k] *= n; }
    double dr = 0, di = 0;
    for (int k = 0; k < 3; k++) { dr += wr[k] * wr[3 + k] + wi[k] * wi[3 + k]; di += wr[k] * wi[3 + k] - wi[k] * wr[3 + k]; }
    for (int k = 0; k < 3; k++) { wr[3 + k] -= dr * wr[k] - di * wi[k]; wi[3 + k] -= dr * wi[k] + di * wr[k]; }
    n = 0;
    for (int k = 0; k < 3; k++) n += wr[3 + k] * wr[3 + k] + wi[3 + k] * wi[3 + k];
    n = 1.0 / sqrt(n);
    for (int k = 0; k < 3; k++) { wr[3 + k] *= n; wi[3 + k] *= n; }
    for (int k = 0; k < 3; k++) {
        const int k1 = (k + 1) % 3, k2 = (k + 2) % 3;
        const double cr = wr[k1] * wr[3 + k2] - wi[k1] * wi[3 + k2] - (wr[k2] * wr[3 + k1] - wi[k2] * wi[3 + k1]);
        const double ci = wr[k1] * wi[3 + k2] + wi[k1] * wr[3 + k2] - (wr[k2] * wi[3 + k1] + wi[k2] * wr[3 + k1]);
        wr[6 + k] = cr; wi[6 + k] = -ci;
    }
    double r[18];
    for (int e = 0; e < 9; e++) { r[2 * e] = wr[e]; r[2 * e + 1] = wi[e]; }
    store_planes<double, 18>(link_block(native, g.NB, 18, parity, cb / SB, mu), cb % SB, r);
}
int fill_gauge(lq_ctx* c, uint64_t seed, double eps) {
    const long long threads = 8LL * c->g.Vh;
    const int block = 128; const int grid = (int)((threads + block - 1) / block);
    fill_gauge_kernel<<<grid, block, 0, c->stream>>>(c->g, stream_key(seed, 1), eps, c->gauge64);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}

template <class S>
__global__ void fill_spinor_kernel(Geom g, int N, uint64_t key, SView<S> even, SView<S> odd, int only, int only_parity) {
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (only ? 1LL : 2LL) * g.Vh * N;
    if (tid >= total) return;
    const int k = (int)(tid % N);
    const long long r = tid / N;
    const int cb = (int)(r % g.Vh);
    const int parity = only ? only_parity : (int)(r / g.Vh);
    int xh, y, z, t, odd_;
    cb_coords(g, parity, cb, xh, y, z, t, odd_);
    const uint64_t site = (uint64_t)(2 * xh + odd_) + (uint64_t)g.L[0] * (y + (uint64_t)g.L[1] * (z + (uint64_t)g.L[2] * t));
    double o[24];
    for (int e = 0; e < 12; e++) cgauss(key, ((uint64_t)k * (uint64_t)g.V + site) * 12 + e, o[2 * e], o[2 * e + 1]);
    const SView<S>& v = (only || parity == 0) ? even : odd;
    const size_t plane = (size_t)SB * group_width(N), off = sp_index(N, cb, k, 0);
    if constexpr (S::has_norm) {
        float mx = 0.f;
        for (int j = 0; j < 24; j++) mx = fmaxf(mx, fabsf((float)o[j]));
        v.n[nrm_index(N, cb, k)] = mx;
        const float inv = mx > 0.f ? 32767.0f / mx : 0.f;
        for (int j = 0; j < 24; j++) v.d[j * plane + off] = (short)rintf((float)o[j] * inv);
    } else {
        for (int j = 0; j < 24; j++) v.d[j * plane + off] = (typename S::store_t)o[j];
    }
}
template <class S> static int fill_spinor_t(lq_ctx* c, void* native, int nrhs, uint64_t seed, int only, int parity) {
    SView<S> e = make_view<S>(c->g, native, nrhs, 0), o = make_view<S>(c->g, native, nrhs, only ? 0 : 1);
    const long long threads = (only ? 1LL : 2LL) * c->g.Vh * nrhs;
    const int block = 128; const int grid = (int)((threads + block - 1) / block);
    fill_spinor_kernel<S><<<grid, block, 0, c->stream>>>(c->g, nrhs, stream_key(seed, 2), e, o, only, parity);
    LQ_LAUNCHED(c);
    LQ_CUDA(c, cudaGetLastError());
    return 0;
}
int fill_spinor(lq_ctx* c, void* native, int nrhs, int prec, uint64_t seed, int parity_only, int parity) {
    if (prec == LQ_FP64) return fill_spinor_t<F64>(c, native, nrhs, seed, parity_only, parity);
    if (prec == LQ_FP32) return fill_spinor_t<F32>(c, native, nrhs, seed, parity_only, parity);
    return fill_spinor_t<H16>(c, native, nrhs, seed, parity_only, parity);
}
