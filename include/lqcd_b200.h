/*
 * lqcd_b200.h -- C ABI of the B200-native multi-RHS Wilson-clover Dslash and batched
 * mixed-precision CG (hot path of the LapH workflow of arxiv 2510.26313).
 *
 * The calls follow the paper's statement of the problem as condensed in BASELINE.json
 * north_star ("load gauge field, build clover term, apply M to N_rhs spinors, solve M x = b
 * for N_rhs sources") and the driver/library split of PAPER.md L110 (Sec. V-B: the driver
 * owns I/O and task order; the library owns device data and host<->device copies; persistent
 * state lives in one long-lived object -- here the opaque lq_ctx).  The operator itself is the
 * textbook Sheikholeslami-Wohlert operator fixed by BASELINE.json and spelled out in
 * SURVEY.md 8(c.1); "batched" means N independent right-hand sides sharing each link and
 * clover load (Sec. V-C3); "mixed precision" is PAPER.md L116/L164.
 *
 * Conventions (binding):
 *   dims = (Lx, Ly, Lz, Lt), all even.  mu = 0,1,2,3 = x,y,z,t.  Lexicographic site index
 *   i = x + Lx*(y + Ly*(z + Lz*t)); parity = (x+y+z+t) mod 2 (0 = even).
 *   Periodic in x,y,z; in t the hopped term is multiplied by t_bc (-1 antiperiodic, +1 periodic)
 *   when the hop wraps around the lattice.  DeGrand-Rossi gamma basis, gamma5 = diag(1,1,-1,-1).
 *   D psi(x) = sum_mu (1-g_mu) U_mu(x) psi(x+mu) + (1+g_mu) U_mu(x-mu)^dag psi(x-mu)
 *   A(x)     = 1 - kappa*csw * sum_{mu<nu} sigma_{mu nu} (x) F_{mu nu}(x),  F from the 4-leaf clover
 *   M = A - kappa D,  M^dag = g5 M g5,  Mhat = A_ee - kappa^2 D_eo A_oo^{-1} D_oe (even sites).
 *
 * CANONICAL layouts (row-major, complex = (re, im) pairs of the stated precision):
 *   gauge   U[mu][t][z][y][x][row][col]
 *   spinor  psi[rhs][t][z][y][x][spin][colour]
 * NATIVE spinor layout (what the kernels stream; for timing without reorders).  One parity of a batch of N right-hand
 * sides is cut into G = N / R groups of R consecutive right-hand sides (R = 4 if N % 4 == 0, else 2 if N is even, else 1)
 * and into NB = ceil(Vh / 32) blocks of 32 consecutive checkerboard sites, Vh = V / 2,
 *                cb = x/2 + (Lx/2) * (y + Ly * (z + Lz * t))   (sites of that parity only; blk = cb / 32, s = cb % 32):
 *   payload[blk][g][j = 0..23][s = 0..31][r = 0..R-1]   with j = 2*(3*spin + colour) + (0 re | 1 im), rhs = g*R + r,
 *                i.e. element offset ((blk*G + g)*24 + j)*32*R + s*R + r; elements are double (LQ_FP64), float (LQ_FP32)
 *                or int16 (LQ_HALF); the payload of one parity is 24*NB*32*N elements rounded up to 256 bytes;
 *   LQ_HALF appends fp32 norms[blk][g][s][r] (offset (blk*G + g)*32*R + s*R + r; NB*32*N floats rounded up to 256
 *                bytes): value = q * norm / 32767, norm = max-abs over the 24 reals of that (site, rhs), q = rint(32767 v / norm).
 *   Sites cb >= Vh of the last block are padding: never read into a result, content unspecified after a call.
 *   Full lattice: the even-parity block followed by the odd-parity block, each lq_native_bytes(.., parity_only = 1) bytes.
 *   lq_native_index() returns these offsets, so a caller never has to retype the formula.
 *   The RHS index is innermost so that one SU(3) link / clover block load serves the whole group.
 *
 * Ownership: the caller owns every buffer it passes; the library copies what it keeps (links)
 * and owns its native copies and scratch.  Device scratch comes from cudaMalloc unless an
 * allocator is installed with lq_set_allocator (the Python binding installs a PyTorch-backed one).
 * Pointers are HOST or DEVICE as said by the `loc` argument next to them.
 *
 * Errors: every call returns 0 on success or a negative lq_status; no exceptions, no abort, no
 * printing.  lq_last_error(ctx) gives a message for the last failure on that context.  All work is
 * enqueued on the context's stream; calls that return values to the host synchronise that stream.
 * There is NO CPU fallback: every operation runs in this library's CUDA kernels.
 */
#ifndef LQCD_B200_H
#define LQCD_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LQ_MAX_RHS 32

typedef struct lq_ctx lq_ctx;

typedef enum { LQ_FP64 = 0, LQ_FP32 = 1, LQ_HALF = 2 } lq_prec;
typedef enum { LQ_HOST = 0, LQ_DEVICE = 1 } lq_loc;
typedef enum { LQ_CANONICAL = 0, LQ_NATIVE = 1 } lq_layout;

typedef enum {
    LQ_OK = 0,
    LQ_EINVAL = -1,        /* bad dims / odd extent / unsupported nrhs, precision or op */
    LQ_ESTATE = -2,        /* gauge or clover not loaded yet */
    LQ_ENOMEM = -3,
    LQ_ECUDA = -4,
    LQ_ENOTCONVERGED = -5, /* lq_solve: some RHS missed tol within the caps; x and info still filled */
    LQ_ESINGULAR = -6      /* lq_build_clover: a 6x6 block is singular / not positive definite */
} lq_status;

/* Operators of lq_apply.  "full" ops act on full-lattice fields; "parity" ops act on one parity
 * (in NATIVE layout the buffers are single-parity blocks; in CANONICAL layout they are full-lattice
 * arrays of which only the stated parity is read / written, the other parity of `out` is zeroed). */
typedef enum {
    LQ_OP_HOP = 0,        /* full:   out = D in                                           (step 4) */
    LQ_OP_M = 1,          /* full:   out = A in - kappa D in                              (step 7) */
    LQ_OP_MDAG = 2,       /* full:   out = g5 M g5 in                                              */
    LQ_OP_CLOVER = 3,     /* full:   out = A in                                           (step 6) */
    LQ_OP_CLOVER_INV = 4, /* full:   out = A^{-1} in                                               */
    LQ_OP_HOP_EO = 5,     /* parity: out_e = D_eo in_o                                             */
    LQ_OP_HOP_OE = 6,     /* parity: out_o = D_oe in_e                                             */
    LQ_OP_MHAT = 7,       /* parity: out_e = A_ee in_e - kappa^2 D_eo A_oo^{-1} D_oe in_e (step 8) */
    LQ_OP_MHAT_DAG = 8,   /* parity: out_e = g5 Mhat g5 in_e                                       */
    LQ_OP_KERNEL_A = 9,   /* parity: out_o = A_oo^{-1} D_oe in_e   */
    LQ_OP_KERNEL_B = 10,  /* parity: out_e = A_ee in_e - kappa^2 D_eo in2_o   */
    LQ_OP_PROBE_LOADS = 11 /* bench only (NATIVE layout, fp32 or half, 18-real links): kernel A's loads, prefetches and stores
                              with one multiply-add per loaded value instead of its arithmetic; the output is meaningless, the
                              time is the floor the memory path sets for kernel A's access pattern                        */
} lq_op;

/* ---- context --------------------------------------------------------------------------------- */
/* Creates a context for a lattice dims = (Lx,Ly,Lz,Lt) (all even, Lx >= 2) on CUDA device `device`.
 * `cuda_stream` is a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream) or NULL for the
 * default stream; the library never creates streams of its own. */
int lq_create(lq_ctx** out, const int dims[4], int device, void* cuda_stream);
int lq_destroy(lq_ctx* ctx);
const char* lq_last_error(const lq_ctx* ctx);

/* Optional device allocator (must be installed before the first lq_load_gauge).  alloc returns a
 * device pointer aligned to >= 256 bytes or NULL; release gets the same pointer back. */
typedef void* (*lq_alloc_fn)(size_t bytes, void* user);
typedef void (*lq_free_fn)(void* ptr, void* user);
int lq_set_allocator(lq_ctx* ctx, lq_alloc_fn alloc, lq_free_fn release, void* user);

/* ---- gauge field and clover term ------------------------------------ */
/* links: CANONICAL gauge field, complex of precision in_prec (LQ_FP64 or LQ_FP32), at `loc`.
 * The library copies it into its native even/odd layout in fp64 (always 18 reals per link) and in
 * fp32 with `recon` = 18 (full) or 12 (third row rebuilt in-kernel as conj(row0 x row1)) reals.
 * The boundary sign t_bc (+1 / -1) is never folded into the stored links.  Invalidates the clover. */
int lq_load_gauge(lq_ctx* ctx, const void* links, int in_prec, int loc, int recon, int t_bc);
/* Bench only: fills the gauge field on the device, U = SU(3) projection (Gram-Schmidt on rows,
 * third row conj(a x b)) of 1 + eps*G, G_ij ~ CN(0,1) from the counter-based generator documented
 * in paper_2510_26313_b200/inputs.py (same stream / index convention). */
int lq_fill_gauge_random(lq_ctx* ctx, uint64_t seed, double eps, int recon, int t_bc);
/* Solver variant (SURVEY 8(f) #3, 8(c.2) reading #13; PAPER.md L116 mixed precision): with enable != 0 the LQ_HALF stencil kernels read
 * the links as int16 fixed point (q = rint(32767 u), always 18 reals: 36 instead of 72 bytes per link); the fp64 / fp32 kernels and the
 * fp64 defect correction are unaffected, so lq_solve still converges to the full-precision solution.  Needs a loaded gauge field. */
int lq_set_half_links(lq_ctx* ctx, int enable);
/* Computes A and A^{-1} (two 6x6 Hermitian blocks per site, both parities) on the device in fp64
 * from the 4-leaf field strength, keeps fp64 and fp32 copies.  LQ_ESINGULAR if a block is not
 * positive definite. */
int lq_build_clover(lq_ctx* ctx, double kappa, double csw);

/* ---- operator application (rows a3, a4, a5) ----------------------------------------------------- */
/* out = op(in [, in2]) for nrhs right-hand sides in precision `prec`.
 * nrhs in {1,2,4,8,12,16,20,24,28,32}: batches beyond 16 are further link-reuse tiles of the same launch (RHS groups of 4 that
 * share every link and clover load through L1; SURVEY 8(f) #3 "larger N").  CANONICAL: complex double (LQ_FP64) or complex float (LQ_FP32) arrays
 * psi[rhs][t][z][y][x][4][3] at `loc`, reordered internally (LQ_HALF: canonical arrays are complex
 * float and are quantised to int16+norm on the way in -- the operator then sees what the half-storage
 * solver sees).  NATIVE: device buffers in the native layout (loc must be LQ_DEVICE).
 * in2 is used by LQ_OP_KERNEL_B only (the odd-parity field to hop), else NULL.  out must not alias
 * in / in2. */
int lq_apply(lq_ctx* ctx, int op, void* out, const void* in, const void* in2, int nrhs, int prec, int loc, int layout);

/* ---- native layout helpers ------------------------------------------------------------------------ */
size_t lq_native_bytes(const lq_ctx* ctx, int nrhs, int prec, int parity_only);
/* Position of (site (x,y,z,t), right-hand side rhs, real j = 2*(3*spin+colour)+(re|im)) in a FULL-lattice native buffer of
 * nrhs right-hand sides in precision prec: *elem_offset = index of the payload element counted in elements of that precision
 * from the start of the site's parity block, *norm_offset = index of the fp32 norm counted in floats from the start of that
 * block's norm array (LQ_HALF; else 0), *parity_block_byte = byte offset of the parity block in the buffer, *norm_array_byte
 * = byte offset of the norm array inside the parity block (LQ_HALF; else 0).  Host-only arithmetic, no device work. */
int lq_native_index(const lq_ctx* ctx, int nrhs, int prec, int x, int y, int z, int t, int rhs, int j,
                    size_t* elem_offset, size_t* norm_offset, size_t* parity_block_byte, size_t* norm_array_byte);
/* canonical (complex double, at loc) -> native (device, precision prec, full lattice) and back */
int lq_pack(lq_ctx* ctx, void* native_out, const void* canonical_in, int nrhs, int prec, int loc);
int lq_unpack(lq_ctx* ctx, void* canonical_out, const void* native_in, int nrhs, int prec, int loc);
/* Bench only: complex-Gaussian spinors written straight into a native device buffer (full lattice if
 * parity_only == 0, else that many sites of parity `parity`), same counter-based generator. */
int lq_fill_spinor_random(lq_ctx* ctx, void* native_out, int nrhs, int prec, uint64_t seed, int parity_only, int parity);
/* Read back selected sites of ONE parity block of a native device buffer (what makes parity checkable at
 * 64^3x128 without a canonical copy of the field, SURVEY 8(d) configs[4]): sites_xyzt is a HOST array of
 * nsites x 4 ints (x, y, z, t), every site of the parity the block holds; out is a HOST array of
 * nsites x nrhs x 24 doubles (spin-major, colour, re/im; half storage dequantised).  Synchronises the stream. */
int lq_gather_sites(lq_ctx* ctx, double* out, const void* native_parity_block, int nrhs, int prec,
                    long long nsites, const int* sites_xyzt);

/* ---- batched mixed-precision solve (rows a2, a6-a11) ---------------------------------------------- */
enum { LQ_ALG_CGNR = 0, LQ_ALG_BICGSTAB = 1 };

typedef struct {
    double tol;          /* target ||b - M x|| / ||b|| per RHS (full system, fp64)                   */
    int max_outer;       /* cap on fp64 defect-correction cycles                                      */
    int max_inner;       /* cap on inner CG iterations per cycle                                      */
    int inner_prec;      /* LQ_FP64, LQ_FP32 or LQ_HALF: storage of the inner CG vectors              */
    double delta;        /* inner CG stops when ||z_k|| <= delta*||z_k(0)|| for every RHS k           */
    int check_every;     /* inner iterations between convergence polls (host sync of N scalars)       */
    int use_graph;       /* 1: replay the inner iteration body as a CUDA graph                        */
    int keep_direction;  /* 1: reliable updates (SURVEY 8(c.2) reading #11, 8(f) #3): after each fp64 residual refresh the
                            CG search direction is kept, p <- z_new + c (p - z_old), instead of restarting at p = z   */
    int algorithm;       /* inner solver: LQ_ALG_CGNR (0, default) or LQ_ALG_BICGSTAB (1): batched BiCGStab on Mhat
                            itself with complex per-RHS scalars, 2 Mhat applications per iteration;
                            keep_direction ignored                                                       */
    int use_x0;          /* 1: the even-site part of x on entry is the initial guess (SURVEY 8(b) solve row); 0: zero start,
                            x is output only                                                             */
} lq_solve_param;

typedef struct {
    int nrhs;
    int outer_cycles;                  /* defect-correction cycles executed                          */
    int inner_iters;                   /* inner CG iterations summed over cycles (shared by the batch) */
    int iters[LQ_MAX_RHS];             /* inner iteration count at which RHS k first met tol (estimate; parity unpinned) */
    double true_rel_residual[LQ_MAX_RHS]; /* ||bhat_e - Mhat x_e|| / ||b|| in fp64 = full-system residual   */
    double seconds;                    /* device time of the solve proper (CUDA events), excl. pack/unpack */
    double dslash_applies;             /* single-parity stencil kernel launches (A or B) that did work, all precisions */
    double model_bytes;                /* modelled (algorithmic) HBM bytes of the solve: every kernel's compulsory traffic,
                                          SURVEY 8(d) byte model (stencil: spinor streams + links and clover once per launch;
                                          block-BLAS: its streams)                                      */
    double model_flops;                /* counted flops: 1320 hop + 504 clover (+48 xpay) per site per RHS per stencil launch,
                                          plus the block-BLAS flops                                      */
} lq_solve_info;

/* Solves M x = b for nrhs independent right-hand sides (no block-Krylov coupling).  b, x: full-lattice
 * complex double, CANONICAL at `loc`, or NATIVE LQ_FP64 device buffers.  x is output only (zero start).
 * CANONICAL host buffers are staged one right-hand side at a time (device staging = one canonical RHS, not the batch).
 * x is output only unless param->use_x0.
 * Even-odd preconditioned CGNR (or, param->algorithm = LQ_ALG_BICGSTAB, batched BiCGStab on Mhat) in inner_prec inside an
 * fp64 defect correction.  The iteration body is replayed as a CUDA graph cached in the context;
 * convergence is tested on the device and the host reads the flag one graph behind, so no launch waits for the host.
 * Returns LQ_ENOTCONVERGED (x, info still valid) if any RHS misses tol. */
int lq_solve(lq_ctx* ctx, void* x, const void* b, int nrhs, int loc, int layout, const lq_solve_param* param, lq_solve_info* info);

/* ---- 3-d gauge-covariant Laplacian ------------------------
 * (Lap v)(x) = sum_{i=x,y,z} [ U_i(x) v(x+i) + U_i(x-i)^dag v(x-i) ] - 6 v(x) on every time-slice independently,
 * periodic in space, for nvec colour-vector fields at once (nvec in {1,2,4,8,12,16,20,24,28,32}); uses the loaded gauge field
 * (fp64 links for LQ_FP64, the fp32 18- or 12-real links for LQ_FP32; LQ_HALF is not supported).
 * lq_laplacian: in/out canonical [vec][t][z][y][x][colour] complex double at `loc`; out must not alias in.
 * lq_laplacian_native: device buffers of lq_cv_native_bytes() bytes in the library's blocked even/odd layout
 * (for timing); lq_cv_fill_random writes bench-only pseudo-random values into such a buffer. */
int lq_laplacian(lq_ctx* ctx, void* out, const void* in, int nvec, int prec, int loc);
int lq_laplacian_native(lq_ctx* ctx, void* out, const void* in, int nvec, int prec);
size_t lq_cv_native_bytes(const lq_ctx* ctx, int nvec, int prec);
int lq_cv_fill_random(lq_ctx* ctx, void* native_out, int nvec, int prec, uint64_t seed);

/* ---- time-batched Lanczos for the LapH eigenvectors -------------------
 * Lowest n_ev eigenpairs of A = -Laplacian on EVERY time-slice (the Lt slices are independent eigenproblems that advance
 * in lockstep): thick-restart Lanczos with full reorthogonalisation on the Chebyshev polynomial
 * T_degree((2A - (cheb_a + cheb_b)) / (cheb_b - cheb_a)); cheb_a = cut just above the wanted eigenvalues, cheb_b >= the
 * largest eigenvalue of A (12 is a bound).  fp64 throughout. */
typedef struct {
    int n_ev;            /* eigenpairs wanted per time-slice                                          */
    int m;               /* Krylov space size, n_ev + 2 <= m <= 512                                    */
    int cheb_degree;     /* degree of the Chebyshev filter (>= 1)                                      */
    int max_restarts;
    double cheb_a, cheb_b;
    double tol;          /* Ritz residual |beta_m q_mi| <= tol * |theta_max| for all wanted pairs, all slices */
    unsigned long long seed;   /* start vector                                                          */
} lq_eig_param;
typedef struct {
    int restarts, converged;
    double lap_applies;        /* Laplacian applications (each on one field = all time-slices)          */
    double max_ritz_residual;  /* the convergence measure above, worst pair and slice                   */
    double max_true_residual;  /* max over pairs and slices of ||A v - lambda v||_2 of the returned vectors (||v|| = 1) */
    double seconds;
    double seconds_ritz;       /* part of `seconds` spent in the Ritz step (projected eigenproblems of all slices + basis rotation) */
    double seconds_ortho;      /* part spent in the Gram-Schmidt passes against the Krylov basis                              */
} lq_eig_info;
/* evals: HOST array [Lt][n_ev] (ascending per slice); evecs: canonical [n_ev][t][z][y][x][colour] complex double at
 * `loc`, or NULL.  Each returned vector has unit norm on every time-slice.  Returns LQ_ENOTCONVERGED (outputs still
 * filled) if max_restarts is reached. */
int lq_laph_eigensolve(lq_ctx* ctx, double* evals, void* evecs, int loc, const lq_eig_param* param, lq_eig_info* info);

/* ---- eigenvector projection ----------------------------------------
 * P[t][alpha][j][k] = sum_{x, c} conj(v_j(x, t, c)) psi_k(x, t, alpha, c)  for n_ev eigenvector fields v
 * (canonical [j][t][z][y][x][colour]) and n_sol solution fields psi (canonical [k][t][z][y][x][spin][colour]), all
 * complex double at `loc`; P: [Lt][4][n_ev][n_sol] complex double at `loc`.  1 <= n_ev <= 1024, 1 <= n_sol <= 64.
 * prec = LQ_FP64: fp64 FMAs (exact to rounding); prec = LQ_FP32: tcgen05 tensor cores, every operand split into two TF32
 * numbers (3xTF32), fp32 accumulation (tensor core over 4 or 8 sites, registers over the 64..1024 sites of one CTA), fp64 sum over the rest:
 * measured error <= 4e-7 of max |P|; deterministic.  Errors: LQ_EINVAL (bad sizes / precision), LQ_ENOMEM (scratch), LQ_ECUDA (incl. a
 * tensor-core completion barrier that timed out: the kernel never hangs). */
int lq_project(lq_ctx* ctx, void* P, const void* evecs, int n_ev, const void* sols, int n_sol, int loc, int prec);

/* The same projection for SINGLE-PRECISION fields: evecs and sols are complex float arrays (8 bytes per number, same index order, 16-byte
 * aligned) at `loc` -- what an fp32 inner solve and an fp32 eigenvector store hold; P is complex double as above.  Always the tensor-core
 * kernel (3xTF32, error <= 4e-7 of max |P| relative to the exact projection of the given fp32 fields).  Half the compulsory bytes of
 * lq_project, and the smaller raw stages leave shared memory for a second operand buffer, so conversion and MMAs overlap. */
int lq_project_c64(lq_ctx* ctx, void* P, const void* evecs, int n_ev, const void* sols, int n_sol, int loc);

/* The fp64 projection for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid it): the same arithmetic, summed in the same order, as lq_project(..., LQ_DEVICE, LQ_FP64), but the partial sums of its
 * two-stage reduction sit in a static device array of LQ_NOALLOC_SCRATCH_BYTES that every GPU loading the library holds until the
 * process exits.  P, evecs, sols: DEVICE arrays as for lq_project (the caller's; P is output).  The call allocates and frees nothing,
 * enqueues two kernels on the context's stream and returns without synchronising: P is ready when the stream reaches that point.
 * Limit: Lt * nchunk * 4 * n_ev * n_sol * 16 bytes <= LQ_NOALLOC_SCRATCH_BYTES with nchunk = clamp(ceil(Lx Ly Lz / 1024), 1, 32),
 * e.g. 8^3 x 16 with 64 eigenvectors x 64 solutions, or 16^3 x 32 with 32 x 16; beyond it LQ_EINVAL with a message naming the limit.
 * All calls on one GPU share the array, which keeps the previous call's contents (nothing needs to start at zero: every entry a call
 * reads it has written itself).  Calls that overlap on the GPU -- other streams, contexts or threads -- race on it. */
#define LQ_NOALLOC_SCRATCH_BYTES (4u << 20)
int lq_project_noalloc(lq_ctx* ctx, void* P, const void* evecs, int n_ev, const void* sols, int n_sol);

/* Launch-parameter knobs of the stencil kernels (the paper's autotuning, reduced to an
 * offline sweep): kernel variant (bits 0-7: 0 = default register budget, 1 = alternative; bits 8-15: z-chunk of the
 * sweep order, 0 = automatic, 0xFF = memory order; see csrc/dslash_launch.cuh),
 * right-hand sides per thread (0 = auto: 2 for nrhs % 4 == 0, else the RHS group width 2 / 1; fp64 caps at 2;
 * must divide the group width), and
 * the L2 prefetch distance of the stencil kernels in 32-site blocks (0 = off, negative = library default). */
int lq_set_tuning(lq_ctx* ctx, int dslash_variant, int dslash_rpt, int dslash_pfd);

/* Plain FP32 ALU peak of this GPU measured with register-only FMA loops ("measure an FMA microbenchmark on
 * the box and use that" as the denominator of the ALU roofline fraction).  mode 0: scalar FFMA, 1: packed FFMA2 with three
 * distinct 64-bit operands, 2: packed FFMA2 whose first operand is shared by 4 consecutive instructions (the stencil kernels'
 * pattern: one link element against 4 spinor reals), 3: packed FFMA2 whose first operand is one 32-bit register broadcast to
 * both halves (the operand form the compiler emits for those products: it issues every 3rd cycle).  Runs for about `ms` milliseconds on the context's stream, synchronises,
 * and writes TFLOP/s (2 flops per FMA lane) to *tflops. */
int lq_fma_peak(lq_ctx* ctx, int mode, double ms, double* tflops);

/* Read bandwidth of the memory path measured with a streaming kernel (16-byte loads that bypass L1, 8 in flight per thread, 8 CTAs of
 * 256 threads per SM).  mode 0: a buffer of `mbytes` MB (choose several times the L2 size) read 4 times: HBM; mode 1: a buffer that
 * fits in L2 (e.g. 48 MB) read 200 times: the L2 -> SM bandwidth, the second memory-side bound of the stencil kernels (every compulsory
 * byte crosses L2 -> SM about 3 times because the 8 neighbour reads of a site meet in L2).  Writes GB/s to *gbs. */
int lq_mem_peak(lq_ctx* ctx, int mode, double mbytes, double* gbs);

/* ------------------------------------------------------------------ two-level adaptive multigrid
 * PAPER.md L118 ("adaptive geometric multi-grid solver", ref. [19]), L164 ("mixed-precision multi-grid solver") and L137 (batching
 * matters most on the coarse grids).  M x = b for the FULL operator M = A - kappa D (step 7) and N right-hand sides at once:
 *   setup   N_v near-null vectors v_k (adaptive: v_k = M^{-1} eta_k, then `refine` passes v_k <- v_k - cycle(M v_k)) -> aggregates (blocks of block[0] x block[1] x block[2] x block[3] sites) x chirality
 *           (spin 0,1 | spin 2,3) -> prolongator P with orthonormal columns: column (a, chi, k) is v_k restricted to aggregate a and
 *           chirality chi, Gram-Schmidt over k = 0, 1, ... (each column against the earlier ones, twice, then normalised) ->
 *           Galerkin coarse operator A_c = P^dag M P, a 9-point stencil of dense (2 N_v) x (2 N_v) blocks
 *   cycle   z ~ M^{-1} r: nu_pre smoother steps from z = 0, coarse correction z += P A_c^{-1} P^dag (r - M z) with A_c^{-1} by
 *           coarse_iters iterations of GCR (restart length min(coarse_iters, 16)), nu_post smoother steps; fp32 throughout.
 *           Smoother LQ_MG_SMOOTH_MR: minimal-residual steps on M itself (t = M res, w = <t,res>/<t,t>, z += w res, res -= w t).
 *           Smoother LQ_MG_SMOOTH_EO: the correction delta ~ M^{-1} res is taken through the even-odd Schur system of steps 8-10,
 *           rho_e = res_e + kappa D_eo A_oo^{-1} res_o, nu minimal-residual steps on Mhat delta_e = rho_e from zero,
 *           delta_o = A_oo^{-1} (res_o + kappa D_oe delta_e); z += delta.  (Mhat has the spectrum lambda (2 - lambda) of M's: the
 *           lambda ~ 2 modes, which minimal residual on M leaves as undamped as the low modes, are folded onto the low modes.)
 *   solve   flexible GCR(restart) preconditioned by the cycle, in fp32, inside an fp64 defect correction (true residual b - M x)
 * Coarse site of (x,y,z,t): a = ax + Lcx (ay + Lcy (az + Lcz at)), a_mu = x_mu / block_mu, Lc_mu = L_mu / block_mu.  Coarse vectors at
 * this boundary are complex fp64 arrays [rhs][a][chi][k]; fine vectors are CANONICAL complex fp64 [rhs][t][z][y][x][spin][colour].
 * Restrictions: L_mu % block_mu == 0, V % 64 == 0, n_vec in {1, 2, 4, 8, ..., 32 (multiples of 4)}.  The hierarchy belongs to the
 * context, is rebuilt by the next setup call and released by lq_mg_free / lq_destroy; it is invalidated (LQ_ESTATE from the calls
 * below) by lq_load_gauge, lq_fill_gauge_random and lq_build_clover. */
enum { LQ_MG_SMOOTH_MR = 0, LQ_MG_SMOOTH_EO = 1 };
typedef struct lq_mg_param {
    int block[4];         /* aggregate extent per direction */
    int n_vec;            /* N_v */
    int nu_pre, nu_post;  /* smoother steps before / after the coarse correction (>= 0) */
    int smoother;         /* LQ_MG_SMOOTH_MR or LQ_MG_SMOOTH_EO */
    int coarse_iters;     /* GCR iterations of the coarse solve (>= 1) */
    int restart;          /* restart length of the outer flexible GCR, 1 .. 16 */
    double setup_tol;     /* lq_mg_setup: v_k = M^{-1} eta_k by lq_solve's mixed-precision CG to this relative residual (e.g. 1e-3) */
    uint64_t seed;        /* lq_mg_setup: seed of the Gaussian eta_k (the generator of lq_fill_spinor_random) */
    int refine;           /* lq_mg_setup: adaptive refinement passes (>= 0): with the hierarchy just built, v_k <- v_k - cycle(M v_k) for all
                             k at once (the cycle removes from v_k what the hierarchy already represents badly), then P and A_c are rebuilt */
} lq_mg_param;
typedef struct lq_mg_info {
    int coarse_dims[4];
    long long coarse_dof;        /* Vc * 2 N_v */
    int probes;                  /* applications of M that built A_c */
    double seconds_vectors;      /* lq_mg_setup: the near-null vector solves */
    double seconds_prolongator;  /* gather + block Gram-Schmidt */
    double seconds_coarse_op;    /* probing */
    size_t bytes;                /* device memory of P, A_c and the tables */
} lq_mg_info;
typedef struct lq_mg_solve_info {
    int iters;                              /* outer FGCR iterations (= multigrid cycles) summed over the defect-correction cycles */
    int outer_cycles;                       /* fp64 defect-correction cycles */
    double true_rel_residual[LQ_MAX_RHS];   /* ||b - M x|| / ||b|| in fp64 */
    double seconds;                         /* device time of the solve (CUDA events), staging excluded */
    double m_applies;                       /* applications of the fine operator M, all precisions */
} lq_mg_solve_info;
/* Adaptive setup: v_k = M^{-1} eta_k with Gaussian eta_k, k < n_vec (one batched lq_solve).  `info` may be NULL. */
int lq_mg_setup(lq_ctx* ctx, const lq_mg_param* param, lq_mg_info* info);
/* Setup from given near-null vectors: vecs = n_vec CANONICAL complex fp64 fields at `loc` (read only). */
int lq_mg_setup_from_vectors(lq_ctx* ctx, const lq_mg_param* param, const void* vecs, int loc, lq_mg_info* info);
int lq_mg_free(lq_ctx* ctx);
/* The pieces of the cycle, each on nrhs right-hand sides at `loc` (parity tests; also usable on their own):
 * coarse_out = P^dag fine_in ; fine_out = P coarse_in ; out = A_c in ; z = cycle(r). */
int lq_mg_restrict(lq_ctx* ctx, void* coarse_out, const void* fine_in, int nrhs, int loc);
int lq_mg_prolong(lq_ctx* ctx, void* fine_out, const void* coarse_in, int nrhs, int loc);
int lq_mg_coarse_apply(lq_ctx* ctx, void* coarse_out, const void* coarse_in, int nrhs, int loc);
int lq_mg_vcycle(lq_ctx* ctx, void* z, const void* r, int nrhs, int loc);
/* Solve M x = b (CANONICAL complex fp64 at `loc`, zero initial guess) to ||b - M x|| <= tol ||b|| per right-hand side, at most max_iter
 * outer iterations.  Returns LQ_ENOTCONVERGED (x and info still filled) if a right-hand side misses tol. */
int lq_mg_solve(lq_ctx* ctx, void* x, const void* b, int nrhs, int loc, double tol, int max_iter, lq_mg_solve_info* info);

/* Number of kernels this library has launched on this context since creation (for bench.py). */
long long lq_kernel_launches(const lq_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* LQCD_B200_H */
