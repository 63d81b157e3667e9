// project_tc.cu -- eigenvector projection on the 5th-generation tensor cores (tcgen05.mma kind::tf32, accumulator in TMEM).
//
// Per time-slice the projection P[j][(k,alpha)] = sum_{x,c} conj(v_j) psi_k,alpha is a tall-skinny complex GEMM
// (PAPER.md L131-133).  It is run as a REAL GEMM C'[j][n'] = sum_kk A'[j][kk] B'[n'][kk] with
//   kk = ((site, colour), re|im),  A'[j][kk] = (Re v, Im v),  B'[2n][kk] = (Re psi, Im psi),  B'[2n+1][kk] = (Im psi, -Re psi),
// so that C'[j][2n] = Re P, C'[j][2n+1] = Im P.  Precision: every fp32 operand is split into two TF32 numbers,
// x = hi + lo, and three MMAs (lo*hi, hi*lo, hi*hi) are accumulated in the fp32 TMEM accumulator ("3xTF32", ~2^-21 per
// product) over 16 sites at a time; the 16-site sums are carried in fp64 registers, K is split over CTAs (64 .. 1024 sites each)
// and the partial sums are added in fp64 in a fixed order.
// One CTA = 512 threads: all threads load fp64, convert and lay out the operands in shared memory (canonical no-swizzle
// K-major UMMA layout: 8-row x 16-byte core matrices; lanes are mapped so that a quarter-warp stores one 128-byte core
// matrix row group: no bank conflicts, and every global request covers whole 128-byte lines), thread 0 issues the MMAs and
// commits them to an mbarrier, the 16 warps read their TMEM lane quadrant x column group back with tcgen05.ld.
// M = 128 eigenvectors (zero padded), N = 64 or 256 = (8 or 32 solutions) x 4 spins x (re, im).
#include "internal.cuh"

namespace {
constexpr int TM = 128, NT = 512;

__device__ __forceinline__ uint32_t s32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
// shared-memory matrix descriptor (cute::UMMA::SmemDescriptor bit layout): start >> 4, leading byte offset >> 4 at bit 16,
// stride byte offset >> 4 at bit 32, version 1 at bit 46, no swizzle
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo, uint32_t sbo) {
    return (uint64_t)((addr >> 4) & 0x3FFF) | ((uint64_t)((lbo >> 4) & 0x3FFF) << 16) | ((uint64_t)((sbo >> 4) & 0x3FFF) << 32) | ((uint64_t)1 << 46);
}
__device__ __forceinline__ void split_tf32(float x, float& hi, float& lo) {
    // round to nearest, ties away (cvt.rna.tf32.f32 written as two full-rate integer instructions): the error of the low
    // part, which the tensor core truncates, then has no preferred sign
    hi = __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xFFFFE000u);
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

// TN = accumulator columns (8 per solution), SPB = sites per stage (K = 6 SPB real terms), RING = raw stages in flight.
// Pipeline per stage i: cp.async brings the fp64 fields of stage i+RING into a raw shared-memory ring (no registers held in
// flight; each thread's copies arrive on the slot's mbarrier, cp.async.mbarrier.arrive.noinc); all threads convert raw stage i
// into the operand tiles once the MMAs of stage i-1 have released them; one CTA barrier; one thread of the last warp issues
// the MMAs of stage i into TMEM bank i%2; the accumulator of stage i-1 (other bank) is then added into registers
// while the tensor core works.  The tensor core adds into its fp32 accumulator with truncation, so its chains are kept to
// one stage and the running sum is carried in registers (round to nearest).
template <int TN, int SPB, int RING>
struct TcShape {
    static constexpr int KB = SPB * 6, NCH = KB / 4;                       // real K terms / 16-byte operand chunks per stage
    static constexpr int A_STRIDE = SPB * 48 + 16;                         // raw bytes per eigenvector row (+16: bank-conflict-free reads)
    // raw solutions in pairs, the odd one 64 bytes further than its size: two solutions per quarter-warp read without conflicts
    static constexpr int B_PAIR = 2 * SPB * 192 + 64;
    __host__ __device__ static constexpr int b_offset(int kl) { return (kl >> 1) * B_PAIR + (kl & 1) * (SPB * 192 + 64); }
    static constexpr int A_RAW = TM * A_STRIDE, B_RAW = (TN / 16) * B_PAIR, RAW = A_RAW + B_RAW;
    static constexpr int OPER = (2 * TM + 2 * TN) * KB * 4;
    static constexpr size_t SMEM = (size_t)OPER + (size_t)RING * RAW + 64;
};

__device__ __forceinline__ void cp_async16(void* dst, const void* src, bool valid) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s32(dst)), "l"(src), "r"(valid ? 16 : 0) : "memory");
}

template <int TN, int SPB, int RING>
__global__ void __launch_bounds__(NT) project_tc_kernel(int Lt, int S3, int nchunk, int spc, int n_ev, int n_sol, int j0, int k0,
                                                        const double2* __restrict__ V, const double2* __restrict__ X, float* __restrict__ partial, int* __restrict__ err) {
    using Sh = TcShape<TN, SPB, RING>;
    constexpr int KB = Sh::KB, NCH = Sh::NCH;
    constexpr int A_PIECES = TM * SPB * 3, B_PIECES = (TN / 8) * SPB * 12;   // 16-byte pieces per raw stage
    constexpr int A_TASKS = TM * NCH, B_TASKS = (TN / 8) * 4 * NCH;          // float4 conversion tasks per stage
    constexpr int COLS = TN / 4;                               // accumulator columns per warp (4 column groups x 4 lane quadrants)
    static_assert(NCH % 2 == 0 && 2 * TN <= 512 && A_TASKS % 32 == 0, "stage shape");
    extern __shared__ __align__(1024) unsigned char smem[];
    float4* sAh = (float4*)smem;               // [NCH][TM/8][8] x 16 bytes
    float4* sAl = sAh + TM * NCH;
    float4* sBh = sAl + TM * NCH;              // [NCH][TN/8][8] x 16 bytes
    float4* sBl = sBh + TN * NCH;
    unsigned char* raw = smem + Sh::OPER;      // RING x { A rows [TM][A_STRIDE], B [TN/8][SPB][12] double2 }
    uint64_t* bar = (uint64_t*)(raw + (size_t)RING * Sh::RAW);
    uint64_t* full = bar + 1;                  // full[slot]: every thread's copies of the raw stage in this slot have landed
    uint32_t* tptr = (uint32_t*)(full + RING);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int t = blockIdx.x / nchunk, ch = blockIdx.x - t * nchunk;
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(s32(bar)));
        for (int k = 0; k < RING; k++) asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(s32(full + k)), "r"(NT));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(s32(tptr)), "n"(2 * TN));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tmem = *tptr;
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(TN >> 3) << 17) | ((uint32_t)(TM >> 4) << 24);   // F32 acc, TF32 x TF32, K-major
    const int s_begin = ch * spc, s_end = min(S3, s_begin + spc);          // spc = sites per CTA (a multiple of 8)
    const int nst = (s_end - s_begin + SPB - 1) / SPB;
    const int nj = min(TM, n_ev - j0), nk = min(TN / 8, n_sol - k0);
    const double2* Vt = V + ((size_t)j0 * Lt + t) * S3 * 3;    // row r: + r * Lt * S3 * 3
    const double2* Xt = X + ((size_t)k0 * Lt + t) * S3 * 12;   // solution kl: + kl * Lt * S3 * 12
    const size_t vrow = (size_t)Lt * S3 * 3, xrow = (size_t)Lt * S3 * 12;

    // Per-thread copy pieces and conversion tasks are the same in every stage (the slice size is a multiple of 8 sites, so a
    // stage is never ragged): precompute their addresses once, the stage loop only adds the stage offset.
    constexpr int NPA = (A_PIECES + NT - 1) / NT, NPB = (B_PIECES + NT - 1) / NT;
    const double2* srcA[NPA]; uint32_t dstA[NPA];              // source of stage 0, byte offset in the raw slot; dst = ~0: no piece
    const double2* srcB[NPB]; uint32_t dstB[NPB];
#pragma unroll
    for (int k = 0; k < NPA; k++) {
        const int p = tid + k * NT, r = p / (SPB * 3), e = p - r * (SPB * 3);
        const bool have = p < A_PIECES;
        dstA[k] = have ? (uint32_t)(r * Sh::A_STRIDE + e * 16) : 0xFFFFFFFFu;
        srcA[k] = (have && r < nj) ? Vt + r * vrow + (size_t)s_begin * 3 + e : nullptr;
    }
#pragma unroll
    for (int k = 0; k < NPB; k++) {
        const int p = tid + k * NT, kl = p / (SPB * 12), w = p - kl * (SPB * 12);
        const bool have = p < B_PIECES;
        dstB[k] = have ? (uint32_t)(Sh::A_RAW + Sh::b_offset(kl) + w * 16) : 0xFFFFFFFFu;
        srcB[k] = (have && kl < nk) ? Xt + kl * xrow + (size_t)s_begin * 12 + w : nullptr;
    }
    // raw stage `st` -> ring slot st % RING; rows / solutions beyond the problem are zero-filled
    auto fetch_stage = [&](int st) {
        if (st < nst) {
            unsigned char* slot = raw + (size_t)(st % RING) * Sh::RAW;
#pragma unroll
            for (int k = 0; k < NPA; k++)
                if (dstA[k] != 0xFFFFFFFFu) cp_async16(slot + dstA[k], srcA[k] ? srcA[k] + (size_t)st * (SPB * 3) : V, srcA[k] != nullptr);
#pragma unroll
            for (int k = 0; k < NPB; k++)
                if (dstB[k] != 0xFFFFFFFFu) cp_async16(slot + dstB[k], srcB[k] ? srcB[k] + (size_t)st * (SPB * 12) : X, srcB[k] != nullptr);
        }
        // the copies of this thread arrive on the slot's mbarrier when they complete (count = all NT threads): the consumers wait
        // on the barrier, no wait_group + CTA barrier
        if (st < nst) asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(s32(full + st % RING)) : "memory");
    };
    // conversion tasks: the A' tasks followed by the B' tasks form one list dealt round-robin to the threads (every thread gets
    // the same number, +-1); per task: the byte offsets of its two raw complex numbers in the slot, the float4 index in the
    // operand tile, and its kind (0 none, 1 A', 2 B'; uniform inside a warp because A_TASKS is a multiple of 32)
    constexpr int NTK = (A_TASKS + B_TASKS + NT - 1) / NT;
    uint32_t raw0[NTK], raw1[NTK], op[NTK];
    int kind[NTK];
#pragma unroll
    for (int k = 0; k < NTK; k++) {
        const int g = tid + k * NT;
        if (g < A_TASKS) {
            // unit = 16 rows x 2 chunks; lane = (row % 8, chunk % 2, (row / 8) % 2): a quarter-warp reads 8 raw rows without bank
            // conflicts and stores one 128-byte core-matrix row group
            const int unit = g >> 5, r = ((unit / (NCH / 2)) * 2 + (lane >> 4)) * 8 + (lane & 7), chunk = (unit % (NCH / 2)) * 2 + ((lane >> 3) & 1);
            raw0[k] = (uint32_t)(r * Sh::A_STRIDE + chunk * 32); raw1[k] = raw0[k] + 16;
            op[k] = (uint32_t)chunk_index<TM>(r, chunk); kind[k] = 1;
        } else if (g < A_TASKS + B_TASKS) {
            // rows 2n, 2n+1 with n = (solution, spin); lane = (spin, solution % 2, chunk % 4): a quarter-warp reads two solutions x
            // four spins of one chunk (conflict-free with the pair layout) and, odd solutions storing the odd row first, covers
            // the 8 rows of a core matrix in each store
            const int q = g - A_TASKS, a = q & 3, chunk = (q >> 3) % NCH, kl = 2 * ((q >> 3) / NCH) + ((q >> 2) & 1);
            const int e0 = 2 * chunk, e1 = e0 + 1;
            const uint32_t base = (uint32_t)(Sh::A_RAW + Sh::b_offset(kl) + a * 48);
            raw0[k] = base + ((e0 / 3) * 12 + e0 % 3) * 16;
            raw1[k] = base + ((e1 / 3) * 12 + e1 % 3) * 16;
            op[k] = (uint32_t)chunk_index<TN>(2 * (kl * 4 + a), chunk); kind[k] = 2;
        } else { raw0[k] = raw1[k] = op[k] = 0; kind[k] = 0; }
    }
    auto flush_bank = [&](int bank, float* acc) {
#pragma unroll
        for (int c0 = 0; c0 < COLS; c0 += 8) {
            uint32_t v[8];
            const uint32_t taddr = tmem + ((uint32_t)((warp & 3) * 32) << 16) + bank * TN + (warp >> 2) * COLS + c0;
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                         : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]) : "r"(taddr));
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
            for (int i = 0; i < 8; i++) acc[c0 + i] += __uint_as_float(v[i]);
        }
        asm volatile("tcgen05.fence::before_thread_sync;");
    };
    // every thread waits for the MMAs of one stage (bounded spin: a fault must not hang the GPU)
    auto wait_bar = [&](uint64_t* b, uint32_t parity) {
        bool done = false;
        for (int spin = 0; spin < 20000000 && !done; spin++) {
            uint32_t r;
            asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }" : "=r"(r) : "r"(s32(b)), "r"(parity) : "memory");
            done = r != 0;
        }
        return done;
    };
    auto wait_mma = [&](uint32_t parity) {
        const bool done = wait_bar(bar, parity);
        asm volatile("tcgen05.fence::after_thread_sync;");
        return done;
    };

    float acc[COLS];                           // TMEM lanes 32 (warp % 4) + lane, columns COLS (warp / 4) ..., summed over the stages
#pragma unroll
    for (int i = 0; i < COLS; i++) acc[i] = 0.f;
    bool ok = true;
#pragma unroll
    for (int st = 0; st < RING; st++) fetch_stage(st);
    for (int i = 0; i < nst; i++) {
        bool arrived = wait_bar(full + i % RING, (uint32_t)((i / RING) & 1));                   // raw stage i has landed (all threads' copies)
        if (arrived && i > 0) arrived = wait_mma((uint32_t)((i - 1) & 1));                       // operand tiles released by the MMAs of stage i-1
        if (__syncthreads_or(!arrived)) { ok = false; break; }                                   // a timeout anywhere ends the loop for the whole CTA
        const unsigned char* slot = raw + (size_t)(i % RING) * Sh::RAW;
#pragma unroll
        for (int k = 0; k < NTK; k++) {
            if (kind[k] == 0) continue;
            const double2 x0 = *(const double2*)(slot + raw0[k]), x1 = *(const double2*)(slot + raw1[k]);
            float4 h, l;
            split4(make_float4((float)x0.x, (float)x0.y, (float)x1.x, (float)x1.y), h, l);
            if (kind[k] == 1) {
                sAh[op[k]] = h; sAl[op[k]] = l;
            } else {
                const float4 h1 = make_float4(h.y, -h.x, h.w, -h.z), l1 = make_float4(l.y, -l.x, l.w, -l.z);
                // odd solutions store the odd row first (selects, not branches: one store instruction must cover all 8 rows)
                const bool odd = (lane >> 2) & 1;
                const uint32_t i0 = op[k] + (odd ? 1u : 0u), i1 = op[k] + (odd ? 0u : 1u);
                const float4 ha = odd ? h1 : h, hb = odd ? h : h1, la = odd ? l1 : l, lb = odd ? l : l1;
                sBh[i0] = ha; sBl[i0] = la;
                sBh[i1] = hb; sBl[i1] = lb;
            }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;");
        __syncthreads();                                         // operands visible; raw slot i % RING is free again
        asm volatile("tcgen05.fence::after_thread_sync;");
        if (tid == NT - 32) {
            const uint32_t d = tmem + (i & 1) * TN;
            // descriptors of k-step 0; k-step s starts 2 s chunks further: the 14-bit start-address field (bytes >> 4) grows by a constant
            // (the operand tiles lie below 72 KB, the field holds 256 KB: no carry into the next field)
            uint64_t ah = smem_desc(s32(sAh), TM * 16, 128), al = smem_desc(s32(sAl), TM * 16, 128);
            uint64_t bh = smem_desc(s32(sBh), TN * 16, 128), bl = smem_desc(s32(sBl), TN * 16, 128);
#pragma unroll
            for (int s = 0; s < KB / 8; s++) {
                mma_tf32(d, al, bh, idesc, s == 0 ? 0u : 1u);
                mma_tf32(d, ah, bl, idesc, 1u);
                mma_tf32(d, ah, bh, idesc, 1u);
                ah += (2 * TM * 16) >> 4; al += (2 * TM * 16) >> 4; bh += (2 * TN * 16) >> 4; bl += (2 * TN * 16) >> 4;
            }
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(s32(bar)) : "memory");
        }
        fetch_stage(i + RING);
        if (i > 0) flush_bank((i - 1) & 1, acc);                 // overlaps the MMAs of stage i (other bank)
    }
    asm volatile("cp.async.wait_all;" ::: "memory");
    if (ok && nst > 0) {
        ok = wait_mma((uint32_t)((nst - 1) & 1));
        if (ok) flush_bank((nst - 1) & 1, acc);
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
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(2 * TN));
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

template <int TN, int SPB, int RING>
int project_tc_run(lq_ctx* c, int Lt, int S3, int n_ev, int n_sol, const double* dev_V, const double* dev_X, double* dev_P) {
    // K split: spc sites per CTA (multiple of 8), chosen among 64 .. 1024 to minimise (waves of CTAs over the SMs) x (stages per
    // CTA): with one CTA per SM the last wave otherwise idles up to half of the machine (16^3x32: 512 CTAs of 256 sites = 3.5
    // waves on 148 SMs -> 288 CTAs of 456 sites = 1.95 waves)
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device);
    int spc = std::min(256, S3);
    {
        long long best = -1;
        for (int cand = 64; cand <= 1024 && cand <= S3; cand += 8) {
            const long long nch = (S3 + cand - 1) / cand, waves = ((long long)Lt * nch + sms - 1) / sms;
            const long long cost = waves * ((cand + SPB - 1) / SPB + 3);       // + a few stage-times of prologue / epilogue per CTA
            if (best < 0 || cost < best) { best = cost; spc = cand; }
        }
    }
    const int nchunk = (S3 + spc - 1) / spc;
    const size_t smem = TcShape<TN, SPB, RING>::SMEM;
    static_assert(TcShape<TN, SPB, RING>::SMEM <= 232448, "shared memory per CTA");
    // the attribute is per device: set it on every call (cheap) rather than once per process
    LQ_CUDA(c, cudaFuncSetAttribute(project_tc_kernel<TN, SPB, RING>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    // scratch (error word + split-K partials) lives in the context between calls
    const size_t need = 256 + sizeof(float) * (size_t)Lt * nchunk * TM * TN;
    if (c->proj_scratch_bytes < need) {
        if (c->proj_scratch) dev_free(c, c->proj_scratch);
        c->proj_scratch = dev_alloc(c, need);
        c->proj_scratch_bytes = c->proj_scratch ? need : 0;
        if (!c->proj_scratch) return LQ_ENOMEM;
    }
    int* d_err = (int*)c->proj_scratch;
    float* partial = (float*)((char*)c->proj_scratch + 256);
    cudaMemsetAsync(d_err, 0, sizeof(int), c->stream);
    int rc = 0;
    for (int j0 = 0; j0 < n_ev && rc == 0; j0 += TM)
        for (int k0 = 0; k0 < n_sol && rc == 0; k0 += TN / 8) {
            project_tc_kernel<TN, SPB, RING><<<Lt * nchunk, NT, smem, c->stream>>>(Lt, S3, nchunk, spc, n_ev, n_sol, j0, k0, (const double2*)dev_V, (const double2*)dev_X, partial, d_err);
            const int nj = std::min(TM, n_ev - j0), nk = std::min(TN / 8, n_sol - k0);
            project_tc_final_kernel<<<(Lt * nj * nk * 4 + 127) / 128, 128, 0, c->stream>>>(Lt, nchunk, n_ev, n_sol, j0, k0, TN, partial, (double2*)dev_P);
            c->launches += 2;
            if (cudaGetLastError() != cudaSuccess) rc = set_err(c, LQ_ECUDA, "lq_project: launch failed");
        }
    int herr = 0;
    if (rc == 0 && (cudaMemcpyAsync(&herr, d_err, sizeof(int), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess || cudaStreamSynchronize(c->stream) != cudaSuccess))
        rc = set_err(c, LQ_ECUDA, "lq_project: tensor-core kernel failed");
    if (rc == 0 && herr) rc = set_err(c, LQ_ECUDA, "lq_project: tcgen05 completion barrier timed out");
    return rc;
}
}  // namespace

int project_device_tc(lq_ctx* c, double* dev_P, const double* dev_V, int n_ev, const double* dev_X, int n_sol) {
    const int Lt = c->g.L[3];
    const long long S3l = (long long)c->g.L[0] * c->g.L[1] * c->g.L[2];
    if (S3l > (1LL << 30) || S3l % 8 != 0) return set_err(c, LQ_EINVAL, "lq_project: bad slice size");   // even extents: 8 | S3
    // 8 solutions per pass (N = 64, 8-site stages) or 32 (N = 256, 4-site stages): the eigenvectors are read once per pass
    if (n_sol <= 8) return project_tc_run<64, 8, 2>(c, Lt, (int)S3l, n_ev, n_sol, dev_V, dev_X, dev_P);
    return project_tc_run<256, 4, 3>(c, Lt, (int)S3l, n_ev, n_sol, dev_V, dev_X, dev_P);
}
