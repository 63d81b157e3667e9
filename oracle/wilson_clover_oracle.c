/*
 * oracle/wilson_clover_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of what the hot path computes: the Wilson-clover
 * Dirac operator M = A - kappa*D, its even-odd Schur complement, and a textbook CG
 * on the normal equations.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call this.  It shares no code with the
 * CUDA path under paper_2510_26313_b200/csrc/.
 *
 * Authority: the paper ("inverse x source", L116 bandwidth-bound sparse
 * computation, L135-140 batched solves, L164 mixed-precision solver) never writes the
 * operator down; BASELINE.json north_star/configs fix it (Wilson-clover, kappa, c_sw,
 * DeGrand-Rossi, periodic space / antiperiodic time, even-odd CG on MdagM) and
 * SURVEY.md 8(c.1) steps 1-9 give the binding definition followed here, step by step,
 * with full 4x4 gamma matrices and dense 12x12 clover blocks: no spin projection, no
 * chirality packing, no checkerboard storage, no blocking or fusion.
 *
 * Layouts (canonical, row-major, complex128):
 *   gauge   U[mu][t][z][y][x][row][col]      mu = 0,1,2,3 = x,y,z,t
 *   spinor  psi[t][z][y][x][spin][colour]    (one right-hand side)
 *   clover  A[t][z][y][x][12][12]            index 3*spin+colour
 * Site index i = x + Lx*(y + Ly*(z + Lz*t)); parity = (x+y+z+t) mod 2.
 *
 * Pins (tests/test_oracle_pins.py): Clifford algebra + gamma5; free-field plane-wave
 * closed form (incl. the worked values of SURVEY 8(c.3)); twisted free field; uniform
 * Abelian flux clover closed form; gamma5-hermiticity; gauge covariance; Sigma D Sigma
 * = -D; dense 192x192 brute force on 2^4 built independently in numpy; Schur identity;
 * CG vs dense solve.  Iteration counts: parity unpinned (only x and the residual are).
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

/* ---------------------------------------------------------------- geometry */
/* SURVEY 8(c.1) step 1 */
typedef struct { int L[4]; long V; } geom_t;

static geom_t make_geom(const int *dims) {
    geom_t g;
    for (int k = 0; k < 4; k++) g.L[k] = dims[k];
    g.V = (long)dims[0] * dims[1] * dims[2] * dims[3];
    return g;
}
static inline long site_index(const geom_t *g, const int *c) {
    return c[0] + (long)g->L[0] * (c[1] + (long)g->L[1] * (c[2] + (long)g->L[2] * c[3]));
}
static inline void site_coords(const geom_t *g, long i, int *c) {
    c[0] = (int)(i % g->L[0]); i /= g->L[0];
    c[1] = (int)(i % g->L[1]); i /= g->L[1];
    c[2] = (int)(i % g->L[2]); i /= g->L[2];
    c[3] = (int)i;
}
/* coordinates of c shifted by `steps` (may be negative) in direction mu, periodic wrap */
static inline void shifted(const geom_t *g, const int *c, int mu, int steps, int *o) {
    for (int k = 0; k < 4; k++) o[k] = c[k];
    int L = g->L[mu];
    o[mu] = ((c[mu] + steps) % L + L) % L;
}
static inline int parity_of(const int *c) { return (c[0] + c[1] + c[2] + c[3]) & 1; }

/* ---------------------------------------------------------------- gamma matrices */
/* DeGrand-Rossi basis, rows as listed there. */
static void gamma_matrix(int mu, cplx g[4][4]) {
    memset(g, 0, 16 * sizeof(cplx));
    switch (mu) {
    case 0: g[0][3] = I;  g[1][2] = I;  g[2][1] = -I; g[3][0] = -I; break;
    case 1: g[0][3] = -1; g[1][2] = 1;  g[2][1] = 1;  g[3][0] = -1; break;
    case 2: g[0][2] = I;  g[1][3] = -I; g[2][0] = -I; g[3][1] = I;  break;
    case 3: g[0][2] = 1;  g[1][3] = 1;  g[2][0] = 1;  g[3][1] = 1;  break;
    case 5: { /* gamma5 = gx gy gz gt */
        cplx a[4][4], b[4][4], t[4][4];
        gamma_matrix(0, a); gamma_matrix(1, b);
        for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) { t[i][j] = 0; for (int k = 0; k < 4; k++) t[i][j] += a[i][k] * b[k][j]; }
        gamma_matrix(2, b);
        for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) { a[i][j] = 0; for (int k = 0; k < 4; k++) a[i][j] += t[i][k] * b[k][j]; }
        gamma_matrix(3, b);
        for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) { g[i][j] = 0; for (int k = 0; k < 4; k++) g[i][j] += a[i][k] * b[k][j]; }
        break; }
    default: break;
    }
}
void orc_gamma(int mu, cplx *out) { cplx g[4][4]; gamma_matrix(mu, g); memcpy(out, g, sizeof g); }

/* sigma_{mu nu} = (i/2) [gamma_mu, gamma_nu]   (step 2) */
static void sigma_matrix(int mu, int nu, cplx s[4][4]) {
    cplx a[4][4], b[4][4];
    gamma_matrix(mu, a); gamma_matrix(nu, b);
    for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) {
        cplx ab = 0, ba = 0;
        for (int k = 0; k < 4; k++) { ab += a[i][k] * b[k][j]; ba += b[i][k] * a[k][j]; }
        s[i][j] = 0.5 * I * (ab - ba);
    }
}
void orc_sigma(int mu, int nu, cplx *out) { cplx s[4][4]; sigma_matrix(mu, nu, s); memcpy(out, s, sizeof s); }

/* ---------------------------------------------------------------- 3x3 helpers */
static inline void m3_mul(const cplx *a, const cplx *b, cplx *o) {      /* o = a b */
    for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) {
        cplx s = 0; for (int k = 0; k < 3; k++) s += a[3 * i + k] * b[3 * k + j]; o[3 * i + j] = s; }
}
static inline void m3_dag(const cplx *a, cplx *o) {
    for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) o[3 * i + j] = conj(a[3 * j + i]);
}

/* ---------------------------------------------------------------- input sources */
/* The operator routines below read links and spinors through these two accessors, so that the same
 * arithmetic serves host arrays (full-lattice entry points) and inputs regenerated per site from the
 * counter-based generator (site-local entry points, reading #4).
 * The generator is the oracle's OWN C statement of the recipe in paper_2510_26313_b200/inputs.py:
 *   mix(z): z += 0x9E3779B97F4A7C15; z = (z ^ z>>30)*0xBF58476D1CE4E5B9; z = (z ^ z>>27)*0x94D049BB133111EB; z ^ z>>31
 *   key = mix(mix(seed) + stream); b_w = mix(key + 2*i + w); u1 = ((b_0>>11)+0.5)/2^53; u2 = (b_1>>11)/2^53
 *   cgauss = sqrt(-ln u1) * exp(2 pi i u2)                          (CN(0,1), reading #2)
 * streams: 1 gauge (index (site*4+mu)*9 + 3*row+col), 2 spinor (index (k*V+site)*12 + 3*spin+colour). */
static uint64_t mix64(uint64_t z) {
    z += 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
static cplx cgauss(uint64_t seed, uint64_t stream, uint64_t idx) {
    uint64_t key = mix64(mix64(seed) + stream);
    uint64_t b0 = mix64(key + 2 * idx), b1 = mix64(key + 2 * idx + 1);
    double u1 = ((double)(b0 >> 11) + 0.5) * (1.0 / 9007199254740992.0);
    double u2 = (double)(b1 >> 11) * (1.0 / 9007199254740992.0);
    return sqrt(-log(u1)) * cexp(2.0 * 3.14159265358979323846 * u2 * I);
}
typedef struct { const cplx *U; uint64_t seed; double eps; } linksrc_t;       /* U != NULL: host array */
typedef struct { const cplx *psi; uint64_t seed; long rhs; } spinsrc_t;       /* psi != NULL: host array */

/* step 3: W = 1 + eps G; rows a, b: a <- a/|a|; b <- b - (a^dag b) a; b <- b/|b|; c = conj(a x b) */
static void generated_link(const geom_t *g, const linksrc_t *src, int mu, const int *c, cplx *u) {
    uint64_t base = ((uint64_t)site_index(g, c) * 4 + (uint64_t)mu) * 9;
    cplx w[9];
    for (int e = 0; e < 9; e++) w[e] = src->eps * cgauss(src->seed, 1, base + e) + ((e % 4 == 0) ? 1.0 : 0.0);
    double n = 0; for (int k = 0; k < 3; k++) n += creal(w[k] * conj(w[k]));
    n = sqrt(n); for (int k = 0; k < 3; k++) w[k] /= n;
    cplx d = 0; for (int k = 0; k < 3; k++) d += conj(w[k]) * w[3 + k];
    for (int k = 0; k < 3; k++) w[3 + k] -= d * w[k];
    n = 0; for (int k = 0; k < 3; k++) n += creal(w[3 + k] * conj(w[3 + k]));
    n = sqrt(n); for (int k = 0; k < 3; k++) w[3 + k] /= n;
    for (int k = 0; k < 3; k++) { int k1 = (k + 1) % 3, k2 = (k + 2) % 3; w[6 + k] = conj(w[k1] * w[3 + k2] - w[k2] * w[3 + k1]); }
    memcpy(u, w, sizeof w);
}
static inline void get_link(const geom_t *g, const linksrc_t *src, int mu, const int *c, cplx *u) {
    if (src->U) memcpy(u, src->U + ((long)mu * g->V + site_index(g, c)) * 9, 9 * sizeof(cplx));
    else generated_link(g, src, mu, c, u);
}
static inline void get_spinor(const geom_t *g, const spinsrc_t *src, const int *c, cplx *p) {
    long i = site_index(g, c);
    if (src->psi) memcpy(p, src->psi + i * 12, 12 * sizeof(cplx));
    else for (int e = 0; e < 12; e++) p[e] = cgauss(src->seed, 2, ((uint64_t)src->rhs * (uint64_t)g->V + (uint64_t)i) * 12 + e);
}

/* ---------------------------------------------------------------- hopping term */
/* step 4: (D psi)(x) = sum_mu [ (1-g_mu) U_mu(x) psi(x+mu) + (1+g_mu) U_mu(x-mu)^dag psi(x-mu) ],
 * step 1: a hop that wraps around t multiplies the hopped term by t_bc (-1 antiperiodic). */
static void hop_site(const geom_t *g, int t_bc, const linksrc_t *ls, const spinsrc_t *ss, cplx gam[4][4][4], const int *c, cplx acc[4][3]) {
    int cn[4];
    memset(acc, 0, 12 * sizeof(cplx));
    for (int mu = 0; mu < 4; mu++) {
        cplx tmp[4][3], u[9], p[12];
        /* forward */
        shifted(g, c, mu, +1, cn);
        get_link(g, ls, mu, c, u);
        get_spinor(g, ss, cn, p);
        double sgn = (mu == 3 && c[3] == g->L[3] - 1) ? (double)t_bc : 1.0;
        for (int s = 0; s < 4; s++) for (int a = 0; a < 3; a++) {
            cplx z = 0; for (int b = 0; b < 3; b++) z += u[3 * a + b] * p[3 * s + b]; tmp[s][a] = z; }
        for (int s = 0; s < 4; s++) for (int a = 0; a < 3; a++) {
            cplx z = 0;
            for (int sp = 0; sp < 4; sp++) z += ((s == sp ? 1.0 : 0.0) - gam[mu][s][sp]) * tmp[sp][a];
            acc[s][a] += sgn * z; }
        /* backward */
        shifted(g, c, mu, -1, cn);
        get_link(g, ls, mu, cn, u);
        get_spinor(g, ss, cn, p);
        sgn = (mu == 3 && c[3] == 0) ? (double)t_bc : 1.0;
        for (int s = 0; s < 4; s++) for (int a = 0; a < 3; a++) {
            cplx z = 0; for (int b = 0; b < 3; b++) z += conj(u[3 * b + a]) * p[3 * s + b]; tmp[s][a] = z; }
        for (int s = 0; s < 4; s++) for (int a = 0; a < 3; a++) {
            cplx z = 0;
            for (int sp = 0; sp < 4; sp++) z += ((s == sp ? 1.0 : 0.0) + gam[mu][s][sp]) * tmp[sp][a];
            acc[s][a] += sgn * z; }
    }
}
void orc_hop(const int *dims, int t_bc, const cplx *U, const cplx *in, cplx *out) {
    geom_t g = make_geom(dims);
    cplx gam[4][4][4];
    for (int mu = 0; mu < 4; mu++) gamma_matrix(mu, gam[mu]);
    linksrc_t ls = {U, 0, 0.0}; spinsrc_t ss = {in, 0, 0};
#pragma omp parallel for schedule(static)
    for (long i = 0; i < g.V; i++) {
        int c[4];
        site_coords(&g, i, c);
        cplx acc[4][3];
        hop_site(&g, t_bc, &ls, &ss, gam, c, acc);
        memcpy(out + i * 12, acc, sizeof acc);
    }
}

/* ---------------------------------------------------------------- field strength */
/* step 5: Q_{mu nu}(x) = sum of the four plaquette leaves starting and ending at x, all with
 * the same orientation; F = (Q - Q^dag)/(8i).  Periodic wrap, no boundary sign. */
static void clover_leaf_sum(const geom_t *g, const linksrc_t *ls, const int *x, int mu, int nu, cplx *Q) {
    int a[4], b[4], c[4];
    cplx t1[9], t2[9], d1[9], d2[9], u1[9], u2[9], u3[9], u4[9];
    memset(Q, 0, 9 * sizeof(cplx));
    /* leaf 1: U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag */
    shifted(g, x, mu, 1, a); shifted(g, x, nu, 1, b);
    get_link(g, ls, mu, x, u1); get_link(g, ls, nu, a, u2); get_link(g, ls, mu, b, u3); get_link(g, ls, nu, x, u4);
    m3_mul(u1, u2, t1);
    m3_dag(u3, d1); m3_mul(t1, d1, t2);
    m3_dag(u4, d2); m3_mul(t2, d2, t1);
    for (int k = 0; k < 9; k++) Q[k] += t1[k];
    /* leaf 2: U_nu(x) U_mu(x-mu+nu)^dag U_nu(x-mu)^dag U_mu(x-mu) */
    shifted(g, x, mu, -1, a); shifted(g, a, nu, 1, b);
    get_link(g, ls, nu, x, u1); get_link(g, ls, mu, b, u2); get_link(g, ls, nu, a, u3); get_link(g, ls, mu, a, u4);
    m3_dag(u2, d1); m3_mul(u1, d1, t1);
    m3_dag(u3, d2); m3_mul(t1, d2, t2);
    m3_mul(t2, u4, t1);
    for (int k = 0; k < 9; k++) Q[k] += t1[k];
    /* leaf 3: U_mu(x-mu)^dag U_nu(x-mu-nu)^dag U_mu(x-mu-nu) U_nu(x-nu) */
    shifted(g, x, mu, -1, a); shifted(g, a, nu, -1, b); shifted(g, x, nu, -1, c);
    get_link(g, ls, mu, a, u1); get_link(g, ls, nu, b, u2); get_link(g, ls, mu, b, u3); get_link(g, ls, nu, c, u4);
    m3_dag(u1, d1); m3_dag(u2, d2); m3_mul(d1, d2, t1);
    m3_mul(t1, u3, t2); m3_mul(t2, u4, t1);
    for (int k = 0; k < 9; k++) Q[k] += t1[k];
    /* leaf 4: U_nu(x-nu)^dag U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^dag */
    shifted(g, x, nu, -1, a); shifted(g, a, mu, 1, b);
    get_link(g, ls, nu, a, u1); get_link(g, ls, mu, a, u2); get_link(g, ls, nu, b, u3); get_link(g, ls, mu, x, u4);
    m3_dag(u1, d1); m3_mul(d1, u2, t1);
    m3_mul(t1, u3, t2);
    m3_dag(u4, d2); m3_mul(t2, d2, t1);
    for (int k = 0; k < 9; k++) Q[k] += t1[k];
}
static void field_strength_site(const geom_t *g, const linksrc_t *ls, const int *x, int mu, int nu, cplx *F) {
    cplx Q[9], Qd[9];
    clover_leaf_sum(g, ls, x, mu, nu, Q);
    m3_dag(Q, Qd);
    for (int k = 0; k < 9; k++) F[k] = (Q[k] - Qd[k]) / (8.0 * I);
}
/* F[plane][site][3][3], planes ordered (mu,nu) = (0,1),(0,2),(0,3),(1,2),(1,3),(2,3) */
void orc_field_strength(const int *dims, const cplx *U, cplx *F) {
    geom_t g = make_geom(dims);
    static const int PL[6][2] = {{0, 1}, {0, 2}, {0, 3}, {1, 2}, {1, 3}, {2, 3}};
    linksrc_t ls = {U, 0, 0.0};
#pragma omp parallel for schedule(static)
    for (long i = 0; i < g.V; i++) {
        int c[4]; site_coords(&g, i, c);
        for (int p = 0; p < 6; p++) field_strength_site(&g, &ls, c, PL[p][0], PL[p][1], F + ((long)p * g.V + i) * 9);
    }
}

/* ---------------------------------------------------------------- clover term */
/* step 6: A(x) = 1 - kappa*csw * sum_{mu<nu} sigma_{mu nu} (x) F_{mu nu}(x), dense 12x12. */
static void clover_site(const geom_t *g, const linksrc_t *ls, const int *x, double kappa, double csw, cplx *A) {
    for (int r = 0; r < 12; r++) for (int c = 0; c < 12; c++) A[12 * r + c] = (r == c) ? 1.0 : 0.0;
    for (int mu = 0; mu < 4; mu++) for (int nu = mu + 1; nu < 4; nu++) {
        cplx F[9], sg[4][4];
        field_strength_site(g, ls, x, mu, nu, F);
        sigma_matrix(mu, nu, sg);
        for (int s = 0; s < 4; s++) for (int sp = 0; sp < 4; sp++)
            for (int a = 0; a < 3; a++) for (int b = 0; b < 3; b++)
                A[12 * (3 * s + a) + (3 * sp + b)] -= kappa * csw * sg[s][sp] * F[3 * a + b];
    }
}
void orc_clover(const int *dims, const cplx *U, double kappa, double csw, cplx *A) {
    geom_t g = make_geom(dims);
    linksrc_t ls = {U, 0, 0.0};
#pragma omp parallel for schedule(static)
    for (long i = 0; i < g.V; i++) { int c[4]; site_coords(&g, i, c); clover_site(&g, &ls, c, kappa, csw, A + i * 144); }
}

/* general complex n x n inverse, Gauss-Jordan with partial pivoting; returns 0 ok, -1 singular */
static int dense_inverse(int n, const cplx *Ain, cplx *Ainv) {
    cplx *w = (cplx *)malloc(sizeof(cplx) * n * 2 * n);
    for (int r = 0; r < n; r++) for (int c = 0; c < n; c++) { w[r * 2 * n + c] = Ain[r * n + c]; w[r * 2 * n + n + c] = (r == c) ? 1.0 : 0.0; }
    for (int k = 0; k < n; k++) {
        int piv = k; double best = cabs(w[k * 2 * n + k]);
        for (int r = k + 1; r < n; r++) { double v = cabs(w[r * 2 * n + k]); if (v > best) { best = v; piv = r; } }
        if (best == 0.0) { free(w); return -1; }
        if (piv != k) for (int c = 0; c < 2 * n; c++) { cplx t = w[k * 2 * n + c]; w[k * 2 * n + c] = w[piv * 2 * n + c]; w[piv * 2 * n + c] = t; }
        cplx d = w[k * 2 * n + k];
        for (int c = 0; c < 2 * n; c++) w[k * 2 * n + c] /= d;
        for (int r = 0; r < n; r++) if (r != k) {
            cplx f = w[r * 2 * n + k];
            if (f != 0) for (int c = 0; c < 2 * n; c++) w[r * 2 * n + c] -= f * w[k * 2 * n + c];
        }
    }
    for (int r = 0; r < n; r++) for (int c = 0; c < n; c++) Ainv[r * n + c] = w[r * 2 * n + n + c];
    free(w);
    return 0;
}
int orc_clover_inverse(long nsites, const cplx *A, cplx *Ainv) {
    int bad = 0;
#pragma omp parallel for schedule(static) reduction(| : bad)
    for (long i = 0; i < nsites; i++) if (dense_inverse(12, A + i * 144, Ainv + i * 144)) bad |= 1;
    return bad ? -1 : 0;
}
/* out(x) = C(x) in(x) for a site-diagonal 12x12 field C */
void orc_apply_site_matrix(long nsites, const cplx *C, const cplx *in, cplx *out) {
#pragma omp parallel for schedule(static)
    for (long i = 0; i < nsites; i++) {
        cplx t[12];
        for (int r = 0; r < 12; r++) { cplx z = 0; for (int c = 0; c < 12; c++) z += C[i * 144 + 12 * r + c] * in[i * 12 + c]; t[r] = z; }
        memcpy(out + i * 12, t, sizeof t);
    }
}

/* ---------------------------------------------------------------- full operator */
static void gamma5_inplace(long nsites, cplx *v) {   /* gamma5 = diag(1,1,-1,-1) is *checked* in the pins;
                                                        here it is applied as the product matrix itself */
    cplx g5[4][4]; gamma_matrix(5, g5);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < nsites; i++) {
        cplx t[12];
        for (int s = 0; s < 4; s++) for (int a = 0; a < 3; a++) { cplx z = 0; for (int sp = 0; sp < 4; sp++) z += g5[s][sp] * v[i * 12 + 3 * sp + a]; t[3 * s + a] = z; }
        memcpy(v + i * 12, t, sizeof t);
    }
}
/* step 7: M = A - kappa D;  dagger: M^dag = g5 M g5 */
void orc_M(const int *dims, int t_bc, const cplx *U, const cplx *A, double kappa, int dagger, const cplx *in, cplx *out) {
    geom_t g = make_geom(dims);
    cplx *v = (cplx *)malloc(sizeof(cplx) * 12 * g.V), *d = (cplx *)malloc(sizeof(cplx) * 12 * g.V);
    memcpy(v, in, sizeof(cplx) * 12 * g.V);
    if (dagger) gamma5_inplace(g.V, v);
    orc_hop(dims, t_bc, U, v, d);
    orc_apply_site_matrix(g.V, A, v, out);
#pragma omp parallel for schedule(static)
    for (long k = 0; k < 12 * g.V; k++) out[k] -= kappa * d[k];
    if (dagger) gamma5_inplace(g.V, out);
    free(v); free(d);
}

/* ---------------------------------------------------------------- even-odd Schur form */
static void mask_parity(const geom_t *g, int keep, cplx *v) {   /* zero every site whose parity != keep */
#pragma omp parallel for schedule(static)
    for (long i = 0; i < g->V; i++) { int c[4]; site_coords(g, i, c); if (parity_of(c) != keep) memset(v + i * 12, 0, 12 * sizeof(cplx)); }
}
/* step 8: Mhat = A_ee - kappa^2 D_eo A_oo^{-1} D_oe on even sites (odd sites of `out` are zero;
 * odd sites of `in` are ignored).  Mhat^dag = g5 Mhat g5. */
void orc_Mhat(const int *dims, int t_bc, const cplx *U, const cplx *A, const cplx *Ainv, double kappa, int dagger,
              const cplx *in, cplx *out) {
    geom_t g = make_geom(dims);
    size_t nb = sizeof(cplx) * 12 * g.V;
    cplx *xe = (cplx *)malloc(nb), *t1 = (cplx *)malloc(nb), *t2 = (cplx *)malloc(nb);
    memcpy(xe, in, nb); mask_parity(&g, 0, xe);
    if (dagger) gamma5_inplace(g.V, xe);
    orc_hop(dims, t_bc, U, xe, t1);            /* D_oe x_e lives on odd sites */
    mask_parity(&g, 1, t1);
    orc_apply_site_matrix(g.V, Ainv, t1, t2);  /* A_oo^{-1} */
    orc_hop(dims, t_bc, U, t2, t1);            /* D_eo */
    mask_parity(&g, 0, t1);
    orc_apply_site_matrix(g.V, A, xe, out);    /* A_ee x_e */
#pragma omp parallel for schedule(static)
    for (long k = 0; k < 12 * g.V; k++) out[k] -= kappa * kappa * t1[k];
    if (dagger) gamma5_inplace(g.V, out);
    free(xe); free(t1); free(t2);
}
/* bhat_e = b_e + kappa D_eo A_oo^{-1} b_o  (odd sites of out zero) */
void orc_schur_source(const int *dims, int t_bc, const cplx *U, const cplx *Ainv, double kappa, const cplx *b, cplx *bhat) {
    geom_t g = make_geom(dims);
    size_t nb = sizeof(cplx) * 12 * g.V;
    cplx *bo = (cplx *)malloc(nb), *t = (cplx *)malloc(nb);
    memcpy(bo, b, nb); mask_parity(&g, 1, bo);
    orc_apply_site_matrix(g.V, Ainv, bo, t);
    orc_hop(dims, t_bc, U, t, bo);
    mask_parity(&g, 0, bo);
    memcpy(bhat, b, nb); mask_parity(&g, 0, bhat);
#pragma omp parallel for schedule(static)
    for (long k = 0; k < 12 * g.V; k++) bhat[k] += kappa * bo[k];
    free(bo); free(t);
}
/* x_o = A_oo^{-1} (b_o + kappa D_oe x_e); on entry x holds x_e (odd part ignored), on exit the full x */
void orc_schur_reconstruct(const int *dims, int t_bc, const cplx *U, const cplx *Ainv, double kappa, const cplx *b, cplx *x) {
    geom_t g = make_geom(dims);
    size_t nb = sizeof(cplx) * 12 * g.V;
    cplx *t = (cplx *)malloc(nb), *s = (cplx *)malloc(nb);
    mask_parity(&g, 0, x);
    orc_hop(dims, t_bc, U, x, t);
#pragma omp parallel for schedule(static)
    for (long k = 0; k < 12 * g.V; k++) t[k] = b[k] + kappa * t[k];
    mask_parity(&g, 1, t);
    orc_apply_site_matrix(g.V, Ainv, t, s);
#pragma omp parallel for schedule(static)
    for (long k = 0; k < 12 * g.V; k++) x[k] += s[k];
    free(t); free(s);
}

/* ---------------------------------------------------------------- vector helpers */
static double norm2(long n, const cplx *v) {
    double s = 0;
#pragma omp parallel for schedule(static) reduction(+ : s)
    for (long k = 0; k < n; k++) s += creal(v[k]) * creal(v[k]) + cimag(v[k]) * cimag(v[k]);
    return s;
}
double orc_norm2(long n, const cplx *v) { return norm2(n, v); }

/* ---------------------------------------------------------------- solvers */
/* step 9: plain CG on Mhat^dag Mhat x_e = Mhat^dag bhat_e (CGNR), zero start, one RHS.
 * Stop when the explicitly recomputed ||bhat - Mhat x|| / ||b|| <= tol (recomputed every iteration:
 * the oracle can afford the extra apply).  b is the FULL source; returns the FULL solution x
 * (odd sites reconstructed).  Returns iterations, or -1 if maxit reached. */
int orc_solve_eo(const int *dims, int t_bc, const cplx *U, const cplx *A, const cplx *Ainv, double kappa,
                 const cplx *b, cplx *x, double tol, int maxit, double *relres_out) {
    geom_t g = make_geom(dims);
    long n = 12 * g.V; size_t nb = sizeof(cplx) * n;
    cplx *bhat = (cplx *)malloc(nb), *r = (cplx *)malloc(nb), *z = (cplx *)malloc(nb), *p = (cplx *)malloc(nb),
         *t = (cplx *)malloc(nb), *q = (cplx *)malloc(nb);
    double bnorm = sqrt(norm2(n, b));
    orc_schur_source(dims, t_bc, U, Ainv, kappa, b, bhat);
    memset(x, 0, nb);
    orc_Mhat(dims, t_bc, U, A, Ainv, kappa, 1, bhat, z);       /* z = Mhat^dag bhat */
    memcpy(p, z, nb);
    double rr = norm2(n, z);
    int it = 0, status = -1;
    double rel = (bnorm > 0) ? sqrt(norm2(n, bhat)) / bnorm : 0.0;
    if (bnorm == 0 || rel <= tol) status = 0;
    while (status < 0 && it < maxit) {
        orc_Mhat(dims, t_bc, U, A, Ainv, kappa, 0, p, t);       /* t = Mhat p */
        double alpha = rr / norm2(n, t);
#pragma omp parallel for schedule(static)
        for (long k = 0; k < n; k++) x[k] += alpha * p[k];
        orc_Mhat(dims, t_bc, U, A, Ainv, kappa, 1, t, q);       /* q = Mhat^dag t */
#pragma omp parallel for schedule(static)
        for (long k = 0; k < n; k++) z[k] -= alpha * q[k];
        double rr1 = norm2(n, z), beta = rr1 / rr; rr = rr1;
#pragma omp parallel for schedule(static)
        for (long k = 0; k < n; k++) p[k] = z[k] + beta * p[k];
        it++;
        orc_Mhat(dims, t_bc, U, A, Ainv, kappa, 0, x, r);       /* true residual */
#pragma omp parallel for schedule(static)
        for (long k = 0; k < n; k++) r[k] = bhat[k] - r[k];
        rel = sqrt(norm2(n, r)) / bnorm;
        if (rel <= tol) status = it;
    }
    orc_schur_reconstruct(dims, t_bc, U, Ainv, kappa, b, x);
    if (relres_out) *relres_out = rel;
    free(bhat); free(r); free(z); free(p); free(t); free(q);
    return status;
}

/* cross-check of step 9: CG on the unpreconditioned M^dag M x = M^dag b */
int orc_solve_full(const int *dims, int t_bc, const cplx *U, const cplx *A, double kappa,
                   const cplx *b, cplx *x, double tol, int maxit, double *relres_out) {
    geom_t g = make_geom(dims);
    long n = 12 * g.V; size_t nb = sizeof(cplx) * n;
    cplx *r = (cplx *)malloc(nb), *z = (cplx *)malloc(nb), *p = (cplx *)malloc(nb), *t = (cplx *)malloc(nb), *q = (cplx *)malloc(nb);
    double bnorm = sqrt(norm2(n, b));
    memset(x, 0, nb);
    orc_M(dims, t_bc, U, A, kappa, 1, b, z);
    memcpy(p, z, nb);
    double rr = norm2(n, z), rel = 1.0;
    int it = 0, status = -1;
    if (bnorm == 0) status = 0;
    while (status < 0 && it < maxit) {
        orc_M(dims, t_bc, U, A, kappa, 0, p, t);
        double alpha = rr / norm2(n, t);
#pragma omp parallel for schedule(static)
        for (long k = 0; k < n; k++) x[k] += alpha * p[k];
        orc_M(dims, t_bc, U, A, kappa, 1, t, q);
#pragma omp parallel for schedule(static)
        for (long k = 0; k < n; k++) z[k] -= alpha * q[k];
        double rr1 = norm2(n, z), beta = rr1 / rr; rr = rr1;
#pragma omp parallel for schedule(static)
        for (long k = 0; k < n; k++) p[k] = z[k] + beta * p[k];
        it++;
        orc_M(dims, t_bc, U, A, kappa, 0, x, r);
#pragma omp parallel for schedule(static)
        for (long k = 0; k < n; k++) r[k] = b[k] - r[k];
        rel = sqrt(norm2(n, r)) / bnorm;
        if (rel <= tol) status = it;
    }
    if (relres_out) *relres_out = rel;
    free(r); free(z); free(p); free(t); free(q);
    return status;
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------- site-local evaluators */
/* hop / kernel-A / kernel-B output at single sites, with links and input spinors
 * either taken from host arrays (U, psi != NULL: used to pin this routine against the full-lattice one) or
 * regenerated on the fly from the counter-based generator (U == NULL: gauge seed/eps; psi == NULL: spinor seed,
 * rhs index), building F_{mu nu}, A and A^{-1} for the site from its 4-leaf neighbourhood.  This is what makes
 * parity checkable at 32^3x64 and 64^3x128 without host copies of the fields.
 *   kind 0: out = (D in)(x)
 *   kind 1: out = A(x)^{-1} (D in)(x)                               "kernel A"
 *   kind 2: out = A(x) xin(x) + coef (D in)(x)                      "kernel B" (row a4; coef = -kappa^2 there)
 * sites[n][4] = (x, y, z, t); out[n][12].  `in` lives on the parity opposite to the listed sites; the
 * generated spinor stream gives every site of the lattice a value, only the neighbours are read. */
int orc_site_eval(const int *dims, int t_bc, int kind, double kappa, double csw, double coef,
                  const cplx *U, uint64_t gauge_seed, double eps,
                  const cplx *psi, uint64_t in_seed, const cplx *xin, uint64_t x_seed, long rhs,
                  long nsites, const int *sites, cplx *out) {
    geom_t g = make_geom(dims);
    cplx gam[4][4][4];
    for (int mu = 0; mu < 4; mu++) gamma_matrix(mu, gam[mu]);
    linksrc_t ls = {U, gauge_seed, eps};
    spinsrc_t ss = {psi, in_seed, rhs};
    spinsrc_t xs = {xin, x_seed, rhs};
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 16) reduction(| : bad)
    for (long n = 0; n < nsites; n++) {
        const int *c = sites + 4 * n;
        cplx d[4][3], A[144], Ainv[144], r[12];
        hop_site(&g, t_bc, &ls, &ss, gam, c, d);
        const cplx *dv = &d[0][0];
        if (kind == 0) { memcpy(out + n * 12, dv, 12 * sizeof(cplx)); continue; }
        clover_site(&g, &ls, c, kappa, csw, A);
        if (kind == 1) {
            if (dense_inverse(12, A, Ainv)) { bad |= 1; continue; }
            for (int i = 0; i < 12; i++) { cplx z = 0; for (int j = 0; j < 12; j++) z += Ainv[12 * i + j] * dv[j]; r[i] = z; }
        } else {
            cplx xv[12];
            get_spinor(&g, &xs, c, xv);
            for (int i = 0; i < 12; i++) { cplx z = 0; for (int j = 0; j < 12; j++) z += A[12 * i + j] * xv[j]; r[i] = z + coef * dv[i]; }
        }
        memcpy(out + n * 12, r, sizeof r);
    }
    return bad ? -1 : 0;
}

/* ---------------------------------------------------------------- 3-d gauge-covariant Laplacian */
/* The LapH smearing operator of PAPER.md L98, L106: on every time-slice t independently (L127: "the temporal
 * extent ... is an independent batching dimension") and for each colour-vector field v,
 *   (Lap v)(x) = sum_{i = x,y,z} [ U_i(x) v(x + i) + U_i(x - i)^dag v(x - i) - 2 v(x) ],
 * periodic in space, no boundary sign (colour vectors carry no spin), the time links are not used.
 * Layouts: U[mu][t][z][y][x][3][3] (as everywhere), v[vec][t][z][y][x][3]. */
void orc_laplacian(const int *dims, const cplx *U, long nvec, const cplx *v, cplx *out) {
    geom_t g = make_geom(dims);
    linksrc_t ls = {U, 0, 0.0};
#pragma omp parallel for schedule(static) collapse(2)
    for (long k = 0; k < nvec; k++)
        for (long i = 0; i < g.V; i++) {
            int c[4], cn[4];
            site_coords(&g, i, c);
            const cplx *vk = v + k * g.V * 3;
            cplx acc[3] = {0, 0, 0}, u[9];
            for (int mu = 0; mu < 3; mu++) {
                shifted(&g, c, mu, +1, cn);
                get_link(&g, &ls, mu, c, u);
                const cplx *p = vk + site_index(&g, cn) * 3;
                for (int a = 0; a < 3; a++) for (int b = 0; b < 3; b++) acc[a] += u[3 * a + b] * p[b];
                shifted(&g, c, mu, -1, cn);
                get_link(&g, &ls, mu, cn, u);
                p = vk + site_index(&g, cn) * 3;
                for (int a = 0; a < 3; a++) for (int b = 0; b < 3; b++) acc[a] += conj(u[3 * b + a]) * p[b];
                for (int a = 0; a < 3; a++) acc[a] -= 2.0 * vk[i * 3 + a];
            }
            memcpy(out + (k * g.V + i) * 3, acc, sizeof acc);
        }
}
