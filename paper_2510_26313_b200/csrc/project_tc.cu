// project_tc.cu -- eigenvector projection on the 5th-generation tensor cores (tcgen05.mma kind::tf32, accumulator in TMEM).
//
// Per time-slice the projection P[j][(k,alpha)] = sum_{x,c} conj(v_j) psi_k,alpha is a tall-skinny complex GEMM
// (PAPER.md L131-133).  It is run as a REAL GEMM C'[j][n'] = sum_kk A'[j][kk] B'[n'][kk] with
//   kk = ((site, colour), re|im),  A'[j][kk] = (Re v, Im v),  B'[2n][kk] = (Re psi, Im psi),  B'[2n+1][kk] = (Im psi, -Re psi),
// so that C'[j][2n] = Re P, C'[j][2n+1] = Im P.  Precision: every fp32 operand is split into two TF32 numbers,
// x = hi + lo, and three MMAs (lo*hi, hi*lo, hi*hi) are accumulated in the fp32 TMEM accumulator ("3xTF32", ~2^-21 per
// product) over 16 sites at a time; the 16-site sums are carried in fp64 registers, K is split over CTAs (256 sites each)
// and the partial sums are added in fp64 in a fixed order.
// One CTA = 512 threads: all threads load fp64, convert and lay out the operands in shared memory (canonical no-swizzle
// K-major UMMA layout: 8-row x 16-byte core matrices; lanes are mapped so that a quarter-warp stores one 128-byte core
// matrix row group: no bank conflicts, and every global request covers whole 128-byte lines), thread 0 issues the MMAs and
// commits them to an mbarrier, the 16 warps read their TMEM lane quadrant x column group back with tcgen05.ld.
// M = 128 eigenvectors (zero padded), N = 64 or 256 = (8 or 32 solutions) x 4 spins x (re, im).
#include "internal.cuh"

namespace {
constexpr int TM = 128, SITES_PER_CTA = 256, NT = 512;

__device__ __forceinline__ uint32_t s32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
// shared-memory matrix descriptor (cute::UMMA::SmemDescriptor bit layout): start >> 4, leading byte offset >> 4 at bit 16,
// stride byte offset >> 4 at bit 32, version 1 at bit 46, no swizzle
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo, uint32_t sbo) {
    return (uint64_t)((addr >> 4) & 0x3FFF) | ((uint64_t)((lbo >> 4) & 0x3FFF) << 16) | ((uint64_t)((sbo >> 4) & 0x3FFF) << 32) | ((uint64_t)1 << 46);
}
__device__ __forceinline__ void split_tf32(float x, float& hi, float& lo) {
    hi = __uint_as_float(__float_as_uint(x) & 0xFFFFE000u);
    lo = x - hi;
}
__device__ __forceinline__ void split4(float4 x, float4& h, float4& l) {
    split_tf32(x.x, h.x, l.x); split_tf32(x.y, h.y, l.y); split_tf32(x.z, h.z, l.z); split_tf32(x.w, h.w, l.w);
}
// float4 index of (row r, 16-byte K chunk) in an operand tile with ROWS rows: chunks outermost, then 8-row groups of 128 bytes
template <int ROWS> __device__ __forceinline__ int chunk_index(int r, int chunk) { return chunk * ROWS + r; }
__device__ __forceinline__ void mma_tf32(uint32_t tmem, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}\n" ::"r"(tmem), "l"(da), "l"(db), "r"(idesc), "r"(accumulate) : "memory");
}

// TN = accumulator columns (8 per solution), SPB = sites per shared-memory stage (K = 6 SPB real terms)
template <int TN, int SPB>
__global__ void __launch_bounds__(NT) project_tc_kernel(int Lt, int S3, int nchunk, int n_ev, int n_sol, int j0, int k0,
                                                        const double2* __restrict__ V, const double2* __restrict__ X, float* __restrict__ partial, int* __restrict__ err) {
    constexpr int KB = SPB * 6, NCH = KB / 4;                 // real K terms and 16-byte chunks per stage
    constexpr int A_UNITS = (TM / 8) * (NCH / 4) / (NT / 32);  // (8 rows x 4 chunks) units per warp
    constexpr int B_TASKS = (TN / 8) * 4 * NCH;                // (solution, spin, chunk) tasks per stage
    constexpr int B_PER_THREAD = (B_TASKS + NT - 1) / NT;
    constexpr int COLS = TN / 4;                               // accumulator columns per warp (4 column groups x 4 lane quadrants)
    static_assert((TM / 8) * (NCH / 4) % (NT / 32) == 0 && NCH % 4 == 0, "stage shape");
    extern __shared__ __align__(1024) unsigned char smem[];
    float4* sAh = (float4*)smem;               // [NCH][TM/8][8] x 16 bytes
    float4* sAl = sAh + TM * NCH;
    float4* sBh = sAl + TM * NCH;              // [NCH][TN/8][8] x 16 bytes
    float4* sBl = sBh + TN * NCH;
    uint64_t* bar = (uint64_t*)(sBl + TN * NCH);
    uint32_t* tptr = (uint32_t*)(bar + 1);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int t = blockIdx.x / nchunk, ch = blockIdx.x - t * nchunk;
    if (tid == 0) { asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(s32(bar))); asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(s32(tptr)), "n"(TN));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tmem = *tptr;
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(TN >> 3) << 17) | ((uint32_t)(TM >> 4) << 24);   // F32 acc, TF32 x TF32, K-major
    const int s_begin = ch * SITES_PER_CTA, s_end = min(S3, s_begin + SITES_PER_CTA);
    const int nj = min(TM, n_ev - j0), nk = min(TN / 8, n_sol - k0);
    uint32_t phase = 0;
    bool ok = true;
    float acc[COLS];                           // TMEM lanes 32 (warp % 4) + lane, columns COLS (warp / 4) ..., summed over the stages
#pragma unroll
    for (int i = 0; i < COLS; i++) acc[i] = 0.f;
    // global loads of one stage into registers; issued for stage i+1 right after the MMAs of stage i, so that their latency
    // overlaps the tensor-core work and the accumulator read-out
    double2 va[A_UNITS][2], xb[B_PER_THREAD][2];
    auto load_stage = [&](int sb) {
        const int e_end = (s_end - sb) * 3;    // complex elements of V left in this CTA's range (<= 0: nothing)
        // ---- A': rows = eigenvectors j0 .. j0+127; lane = (row % 8, chunk % 4): a quarter-warp stores one 128-byte row group
#pragma unroll
        for (int u = 0; u < A_UNITS; u++) {
            const int unit = warp * A_UNITS + u, r = (unit / (NCH / 4)) * 8 + (lane & 7), chunk = (unit % (NCH / 4)) * 4 + (lane >> 3);
            const double2* src = V + (((size_t)(j0 + r) * Lt + t) * S3 + sb) * 3 + 2 * chunk;
            const bool row = r < nj;
            va[u][0] = (row && 2 * chunk < e_end) ? src[0] : make_double2(0.0, 0.0);
            va[u][1] = (row && 2 * chunk + 1 < e_end) ? src[1] : make_double2(0.0, 0.0);
        }
        // ---- B': rows 2n, 2n+1 with n = (solution, spin); task = (solution, chunk, spin), spin fastest across lanes
#pragma unroll
        for (int u = 0; u < B_PER_THREAD; u++) {
            const int q = tid + u * NT, a = q & 3, chunk = (q >> 2) % NCH, kl = (q >> 2) / NCH;
            xb[u][0] = xb[u][1] = make_double2(0.0, 0.0);
            if (q < B_TASKS && kl < nk) {
                const double2* base = X + ((size_t)(k0 + kl) * Lt + t) * S3 * 12 + 3 * a;
                const int e0 = 2 * chunk, e1 = e0 + 1;
                if (e0 < e_end) xb[u][0] = base[(size_t)(sb + e0 / 3) * 12 + e0 % 3];
                if (e1 < e_end) xb[u][1] = base[(size_t)(sb + e1 / 3) * 12 + e1 % 3];
            }
        }
    };
    load_stage(s_begin);
    for (int sb = s_begin; sb < s_end; sb += SPB) {
#pragma unroll
        for (int u = 0; u < A_UNITS; u++) {
            const int unit = warp * A_UNITS + u, r = (unit / (NCH / 4)) * 8 + (lane & 7), chunk = (unit % (NCH / 4)) * 4 + (lane >> 3);
            float4 h, l;
            split4(make_float4((float)va[u][0].x, (float)va[u][0].y, (float)va[u][1].x, (float)va[u][1].y), h, l);
            sAh[chunk_index<TM>(r, chunk)] = h; sAl[chunk_index<TM>(r, chunk)] = l;
        }
#pragma unroll
        for (int u = 0; u < B_PER_THREAD; u++) {
            const int q = tid + u * NT, a = q & 3, chunk = (q >> 2) % NCH, kl = (q >> 2) / NCH;
            if (q < B_TASKS) {
                float4 h, l;
                split4(make_float4((float)xb[u][0].x, (float)xb[u][0].y, (float)xb[u][1].x, (float)xb[u][1].y), h, l);
                const float4 h1 = make_float4(h.y, -h.x, h.w, -h.z), l1 = make_float4(l.y, -l.x, l.w, -l.z);
                const int r0 = 2 * (kl * 4 + a);
                // odd chunks store the odd row first: the 8 lanes of a quarter-warp then cover the 8 rows of one core matrix
                if (chunk & 1) {
                    sBh[chunk_index<TN>(r0 + 1, chunk)] = h1; sBh[chunk_index<TN>(r0, chunk)] = h;
                    sBl[chunk_index<TN>(r0 + 1, chunk)] = l1; sBl[chunk_index<TN>(r0, chunk)] = l;
                } else {
                    sBh[chunk_index<TN>(r0, chunk)] = h; sBh[chunk_index<TN>(r0 + 1, chunk)] = h1;
                    sBl[chunk_index<TN>(r0, chunk)] = l; sBl[chunk_index<TN>(r0 + 1, chunk)] = l1;
                }
            }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        asm volatile("tcgen05.fence::after_thread_sync;");
        if (tid == 0) {
#pragma unroll 1
            for (int s = 0; s < KB / 8; s++) {
                const uint64_t ah = smem_desc(s32(sAh) + (2 * s) * (TM * 16), TM * 16, 128), al = smem_desc(s32(sAl) + (2 * s) * (TM * 16), TM * 16, 128);
                const uint64_t bh = smem_desc(s32(sBh) + (2 * s) * (TN * 16), TN * 16, 128), bl = smem_desc(s32(sBl) + (2 * s) * (TN * 16), TN * 16, 128);
                mma_tf32(tmem, al, bh, idesc, s == 0 ? 0u : 1u);
                mma_tf32(tmem, ah, bl, idesc, 1u);
                mma_tf32(tmem, ah, bh, idesc, 1u);
            }
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(s32(bar)) : "memory");
        }
        load_stage(sb + SPB);
        // every thread waits for the MMAs of this stage (bounded spin: a fault must not hang the GPU)
        bool done = false;
        for (int spin = 0; spin < 20000000 && !done; spin++) {
            uint32_t r;
            asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }" : "=r"(r) : "r"(s32(bar)), "r"(phase) : "memory");
            done = r != 0;
        }
        if (!done) { ok = false; break; }
        phase ^= 1;
        asm volatile("tcgen05.fence::after_thread_sync;");
        // the tensor core adds into its fp32 accumulator with truncation: keep its chains short (one stage) and carry the
        // running sum in registers (round to nearest)
#pragma unroll
        for (int c0 = 0; c0 < COLS; c0 += 8) {
            uint32_t v[8];
            const uint32_t taddr = tmem + ((uint32_t)((warp & 3) * 32) << 16) + (warp >> 2) * COLS + c0;
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                         : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]) : "r"(taddr));
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
            for (int i = 0; i < 8; i++) acc[c0 + i] += __uint_as_float(v[i]);
        }
        asm volatile("tcgen05.fence::before_thread_sync;");
    }
    if (!ok && lane == 0) atomicAdd(err, 1);
    // accumulator row r = TMEM lane r, column n'; partial[t][chunk][r][n']
    const int r = (warp & 3) * 32 + lane;
    if (ok && r < nj) {
        float* dst = partial + (((size_t)t * nchunk + ch) * TM + r) * TN + (warp >> 2) * COLS;
#pragma unroll
        for (int c0 = 0; c0 < COLS; c0 += 4) *(float4*)(dst + c0) = make_float4(acc[c0], acc[c0 + 1], acc[c0 + 2], acc[c0 + 3]);
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(TN));
}

// out[t][alpha][j0+r][k0+kl] = fixed-order fp64 sum over chunks of partial[t][chunk][r][2*(kl*4+alpha) + (re|im)]
__global__ void project_tc_final_kernel(int Lt, int nchunk, int n_ev, int n_sol, int j0, int k0, int TN, const float* __restrict__ partial, double2* __restrict__ out) {
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    const int nj = min(TM, n_ev - j0), nk = min(TN / 8, n_sol - k0);
    if (id >= Lt * nj * nk * 4) return;
    int q = id;
    const int kl = q % nk; q /= nk;
    const int r = q % nj; q /= nj;
    const int a = q % 4; const int t = q / 4;
    double re = 0.0, im = 0.0;
    for (int c = 0; c < nchunk; c++) {
        const float* p = partial + (((size_t)t * nchunk + c) * TM + r) * TN + 2 * (kl * 4 + a);
        re += (double)p[0]; im += (double)p[1];
    }
    out[(((size_t)t * 4 + a) * n_ev + (j0 + r)) * n_sol + (k0 + kl)] = make_double2(re, im);
}

template <int TN, int SPB>
int project_tc_run(lq_ctx* c, int Lt, int S3, int n_ev, int n_sol, const double* dev_V, const double* dev_X, double* dev_P) {
    const int nchunk = (S3 + SITES_PER_CTA - 1) / SITES_PER_CTA;
    const size_t smem = (size_t)(2 * TM + 2 * TN) * SPB * 6 * sizeof(float) + 64;
    static bool configured = false;
    if (!configured) { LQ_CUDA(c, cudaFuncSetAttribute(project_tc_kernel<TN, SPB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); configured = true; }
    float* partial = (float*)dev_alloc(c, sizeof(float) * (size_t)Lt * nchunk * TM * TN);
    int* d_err = (int*)dev_alloc(c, sizeof(int));
    if (!partial || !d_err) { if (partial) dev_free(c, partial); if (d_err) dev_free(c, d_err); return LQ_ENOMEM; }
    cudaMemsetAsync(d_err, 0, sizeof(int), c->stream);
    int rc = 0;
    for (int j0 = 0; j0 < n_ev && rc == 0; j0 += TM)
        for (int k0 = 0; k0 < n_sol && rc == 0; k0 += TN / 8) {
            project_tc_kernel<TN, SPB><<<Lt * nchunk, NT, smem, c->stream>>>(Lt, S3, nchunk, n_ev, n_sol, j0, k0, (const double2*)dev_V, (const double2*)dev_X, partial, d_err);
            const int nj = std::min(TM, n_ev - j0), nk = std::min(TN / 8, n_sol - k0);
            project_tc_final_kernel<<<(Lt * nj * nk * 4 + 127) / 128, 128, 0, c->stream>>>(Lt, nchunk, n_ev, n_sol, j0, k0, TN, partial, (double2*)dev_P);
            c->launches += 2;
            if (cudaGetLastError() != cudaSuccess) rc = set_err(c, LQ_ECUDA, "lq_project: launch failed");
        }
    int herr = 0;
    if (rc == 0 && (cudaMemcpyAsync(&herr, d_err, sizeof(int), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess || cudaStreamSynchronize(c->stream) != cudaSuccess))
        rc = set_err(c, LQ_ECUDA, "lq_project: tensor-core kernel failed");
    if (rc == 0 && herr) rc = set_err(c, LQ_ECUDA, "lq_project: tcgen05 completion barrier timed out");
    dev_free(c, partial); dev_free(c, d_err);
    return rc;
}
}  // namespace

int project_device_tc(lq_ctx* c, double* dev_P, const double* dev_V, int n_ev, const double* dev_X, int n_sol) {
    const int Lt = c->g.L[3];
    const long long S3l = (long long)c->g.L[0] * c->g.L[1] * c->g.L[2];
    if (S3l > (1LL << 30)) return set_err(c, LQ_EINVAL, "lq_project: slice too large");
    // 8 solutions per pass (N = 64, 16-site stages) or 32 (N = 256, 8-site stages): the eigenvectors are read once per pass
    if (n_sol <= 8) return project_tc_run<64, 16>(c, Lt, (int)S3l, n_ev, n_sol, dev_V, dev_X, dev_P);
    return project_tc_run<256, 8>(c, Lt, (int)S3l, n_ev, n_sol, dev_V, dev_X, dev_P);
}
