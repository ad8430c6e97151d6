/*
 * sww_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, obviously-correct CPU implementation of the Dirichlet-to-Neumann hot path of
 * Wilkening & Yu, "Overdetermined shooting methods for computing standing water waves with spectral
 * accuracy" (arXiv 1210.5672; text in /root/reference/PAPER.md, cited below as PAPER.md:<line>).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may call it.
 * It shares no code with the CUDA path (paper_1210_5672_b200/csrc) and neither includes the other.
 *
 * One source, one working type REAL, chosen at compile time (the paper's own typedef trick):
 *     -DORC_F64  double        (speed baseline)          symbols orc_f64_*
 *     -DORC_LD   long double   (oracle for the fp64 bar) symbols orc_ld_*
 *     -DORC_Q    __float128    (oracle for the dd bar)   symbols orc_q_*
 * Every array crosses the interface as a (hi, lo) pair of double arrays, value = hi + lo (lo may be
 * NULL = 0 on input / discarded on output).  Batches are column-major N x nrhs (column c at c*N).
 * Matrices K, G are row-major here: K[i*N + j], i = target point alpha_i, j = source point alpha_j.
 *
 * The method is exact linear algebra on a fixed discretisation, so the oracle is the plain definition:
 *   - explicit O(N^2) DFT sums for every Fourier multiplier (no FFT);
 *   - K, G entry by entry from (2.13) with the two-branch cot of PAPER.md:154;
 *   - Gaussian elimination with partial pivoting for (2.7);
 *   - a straight loop over the Runge-Kutta stages.
 *
 * Readings of the paper (full list with justification: DESIGN.md §3):
 *   R1  image kernels are SUBTRACTED: K = K1 - K2, G = G1 - G2, as (A.2),(A.3),(A.8) print them
 *       (PAPER.md:637,643,663); the "+" of (2.7),(2.8),(A.4),(A.6),(A.9),(A.11) is a sign erratum.
 *       Pinned by the flat-surface symbol k tanh(kh) (4.34).
 *   R2  API eta is the elevation about the mean level; the bottom is y=0 and the surface is
 *       y = h + eta ("absorb the mean fluid depth into eta").  The system matrix that is
 *       factored is A = I/2 + K ("LU-factorization of K").
 *   R3  uniform grid xi(alpha)=alpha (rho_1 = 1), so 1/|xi'| = 1 in (2.8), unless set_mesh() selects a
 *       refined mesh (2.10): then zeta = xi + i eta o xi, d/dx = (1/xi') d/dalpha, P removes the mean over x.
 *   R4  Nyquist mode (N even): symbol 0 for D, H, |D|; eta'' = D(D eta); filter factor exp(-36) there.
 *   R5  the 36th-order filter (2.14) multiplies every evaluated right-hand side and the solution after
 *       every step; flag to switch it off.
 *   R6  "an 8th-order explicit Runge-Kutta": the paper cites DOP853 without printing it;
 *       the 11-stage order-8 Cooper-Verner tableau with coefficients in Q(sqrt 21) is used
 *       (SURVEY.md §8(c)-A12); pinned by the rooted-tree order conditions in tests/.
 *   R7  g eta vs g (h + eta) in (2.1b) differ by a constant that P removes; sigma = 0.
 *   PARITY UNPINNED (conventions that no printed value or identity fixes; the CUDA path takes the same ones):
 *       the filter being on by default and applied to every right-hand side and after every step (R5); the symbol 0 of D, H, |D| at the
 *       Nyquist mode (R4); on a refined mesh, the filter acting on the Fourier modes in alpha of the stored samples (R16).
 *       Everything else below is pinned in tests/test_oracle_pins.py and tests/test_oracle_mesh.py.
 *   R8  every Fourier multiplier (D, H, |D|, P, filter) is summed in __float128 in the ld and q builds
 *       (see multiplier_w below); the dense O(N^2)/O(N^3) steps run in REAL.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#if defined(ORC_Q)
#include <quadmath.h>
typedef __float128 REAL;
#define NAME(x) orc_q_##x
#define R_SIN sinq
#define R_COS cosq
#define R_SINH sinhq
#define R_COSH coshq
#define R_EXP expq
#define R_POW powq
#define R_SQRT sqrtq
#define R_FABS fabsq
#define R_PI M_PIq
#define R_ISINF isinfq
#elif defined(ORC_LD)
typedef long double REAL;
#define NAME(x) orc_ld_##x
#define R_SIN sinl
#define R_COS cosl
#define R_SINH sinhl
#define R_COSH coshl
#define R_EXP expl
#define R_POW powl
#define R_SQRT sqrtl
#define R_FABS fabsl
#define R_PI 3.141592653589793238462643383279502884L
#define R_ISINF isinf
#else
typedef double REAL;
#define NAME(x) orc_f64_##x
#define R_SIN sin
#define R_COS cos
#define R_SINH sinh
#define R_COSH cosh
#define R_EXP exp
#define R_POW pow
#define R_SQRT sqrt
#define R_FABS fabs
#define R_PI 3.14159265358979323846
#define R_ISINF isinf
#endif

/* WIDE: the type every Fourier multiplier is summed in (reading R8 below). */
#if defined(ORC_F64)
typedef double WIDE;
#define W_SIN sin
#define W_COS cos
#define W_EXP exp
#define W_POW pow
#define W_PI 3.14159265358979323846
#else
#include <quadmath.h>
typedef __float128 WIDE;
#define W_SIN sinq
#define W_COS cosq
#define W_EXP expq
#define W_POW powq
#define W_PI M_PIq
#endif

#define ORC_OK 0
#define ORC_EINVAL (-1)
#define ORC_ENOMEM (-2)
#define ORC_EBOTTOM (-4)
#define ORC_ESINGULAR (-5)

/* ---------- hi/lo marshalling ---------- */
static void load_hl(REAL *dst, const double *hi, const double *lo, long n) {
    for (long i = 0; i < n; i++) dst[i] = (REAL)hi[i] + (lo ? (REAL)lo[i] : (REAL)0);
}
static void store_hl(const REAL *src, double *hi, double *lo, long n) {
    for (long i = 0; i < n; i++) {
        double h = (double)src[i];
        if (hi) hi[i] = h;
        if (lo) lo[i] = (double)(src[i] - (REAL)h);
    }
}
static REAL *ralloc(long n) { return (REAL *)malloc((size_t)(n > 0 ? n : 1) * sizeof(REAL)); }

/* ---------- trigonometric tables: cos, sin(2 pi m / N), m = 0..N-1, by direct evaluation ---------- */
/* cos, sin(2 pi m / N) with the angle reduced EXACTLY (integer arithmetic) to [0, pi/4] before the library call, so
 * that small values keep full RELATIVE accuracy: the kernels (2.13) multiply sin x by ~N^2/(2 pi^2) next to the diagonal,
 * and sinl(2 pi (N-1)/N) evaluated at a rounded argument near 2 pi is only absolutely accurate. */
#define DEF_TRIG_EXACT(FN, T, PI_, SIN_, COS_)                                                      \
    static void FN(long m, long N, T *c, T *s) {                                                    \
        long t = 4 * (m % N), quad = t / N, r = t - quad * N; /* angle = quad*pi/2 + (pi/2) r/N */  \
        int swap = 0;                                                                               \
        if (2 * r > N) { r = N - r; swap = 1; }             /* (pi/2) r/N -> pi/2 - (pi/2) r'/N */  \
        T phi = (PI_ / 2) * (T)r / (T)N, cc = COS_(phi), ss = SIN_(phi);                            \
        if (r == 0) { cc = 1; ss = 0; }                                                             \
        if (2 * r == N) { cc = ss; }  /* pi/4: keep cos == sin exactly */                           \
        if (swap) { T tmp = cc; cc = ss; ss = tmp; }                                                \
        switch (quad) {                                                                             \
        case 0: *c = cc; *s = ss; break;                                                            \
        case 1: *c = -ss; *s = cc; break;                                                           \
        case 2: *c = -cc; *s = -ss; break;                                                          \
        default: *c = ss; *s = -cc; break;                                                          \
        }                                                                                           \
    }
DEF_TRIG_EXACT(trig_exact_r, REAL, R_PI, R_SIN, R_COS)
DEF_TRIG_EXACT(trig_exact_w, WIDE, W_PI, W_SIN, W_COS)

typedef struct { int N; REAL *c, *s; WIDE *wc, *ws; } trig_t;
static int trig_init(trig_t *t, int N) {
    t->N = N; t->c = ralloc(N); t->s = ralloc(N);
    t->wc = (WIDE *)malloc(sizeof(WIDE) * N); t->ws = (WIDE *)malloc(sizeof(WIDE) * N);
    if (!t->c || !t->s || !t->wc || !t->ws) return ORC_ENOMEM;
    for (int m = 0; m < N; m++) {
        trig_exact_r(m, N, &t->c[m], &t->s[m]);
        trig_exact_w(m, N, &t->wc[m], &t->ws[m]);
    }
    return ORC_OK;
}
static void trig_free(trig_t *t) { free(t->c); free(t->s); free(t->wc); free(t->ws); }

/* ---------- Fourier multipliers by explicit DFT sums ----------
 * f_j real, alpha_j = 2 pi j/N.  a_k = (1/N) sum_j f_j cos(k alpha_j), b_k = (1/N) sum_j f_j sin(k alpha_j),
 * so fhat_k = a_k - i b_k and f_j = a_0 + 2 sum_{0<k<N/2} (a_k cos + b_k sin) + a_{N/2} cos(N/2 alpha_j).
 * A multiplier m_k = p_k + i q_k (m_{-k} = conj m_k) maps this to
 *   out_j = p_0 a_0 + 2 sum_{0<k<N/2} [ (p a + q b) cos(k alpha_j) - (q a - p b) sin(k alpha_j) ] + p_{N/2} a_{N/2} cos(N/2 alpha_j).
 */
enum { MUL_D = 1,      /* d/dalpha: i k, Nyquist 0                 */
       MUL_H = 2,      /* Hilbert transform: -i sgn k, Nyquist 0   */
       MUL_ABSD = 3,   /* |D| = H D: |k|, Nyquist 0                               */
       MUL_FILTER = 4, /* exp(-36 (|k|/(N/2))^36) (2.14)            */
       MUL_P = 5,      /* projection to zero mean (2.2)              */
       MUL_PFILTER = 6 /* filter o P                                              */ };

static void symbol(int which, int k, int N, WIDE *p, WIDE *q) {
    int nyq = (2 * k == N);
    *p = 0; *q = 0;
    switch (which) {
    case MUL_D: *q = nyq ? 0 : (WIDE)k; break;
    case MUL_H: *q = (k == 0 || nyq) ? 0 : (WIDE)(-1); break;
    case MUL_ABSD: *p = nyq ? 0 : (WIDE)k; break;
    case MUL_FILTER: *p = W_EXP(-36 * W_POW((WIDE)k / ((WIDE)N / 2), (WIDE)36)); break;
    case MUL_P: *p = (k == 0) ? 0 : 1; break;
    case MUL_PFILTER: *p = (k == 0) ? 0 : W_EXP(-36 * W_POW((WIDE)k / ((WIDE)N / 2), (WIDE)36)); break;
    }
}

/* R8: the sums run in WIDE (= __float128 in the ld and q builds, double in the f64 speed-baseline build).
 * D is the one unbounded step of the procedure: it multiplies rounding noise by ~N/4, and the
 * near-singular kernels (2.13) turn noise d in eta' into ~(N^2/20) d in the result.  Plain O(N^2) DFT sums in
 * the working type carry ~sqrt(N) x more noise per coefficient than an FFT would, which made the long-double
 * oracle no better than a careful fp64 pipeline (measured 1.2e-13 at N=512).  Same definition, more digits. */
static void multiplier_w(const trig_t *t, int which, const WIDE *f, WIDE *out) {
    int N = t->N, K = N / 2;
    WIDE *a = (WIDE *)malloc(sizeof(WIDE) * (K + 1)), *b = (WIDE *)malloc(sizeof(WIDE) * (K + 1));
#pragma omp parallel for schedule(static)
    for (int k = 0; k <= K; k++) {
        WIDE sa = 0, sb = 0;
        for (int j = 0; j < N; j++) {
            int m = (int)(((long)k * j) % N);
            sa += f[j] * t->wc[m]; sb += f[j] * t->ws[m];
        }
        WIDE p, q;
        symbol(which, k, N, &p, &q);
        sa /= (WIDE)N; sb /= (WIDE)N;
        a[k] = p * sa + q * sb;   /* R_k */
        b[k] = q * sa - p * sb;   /* I_k */
    }
#pragma omp parallel for schedule(static)
    for (int j = 0; j < N; j++) {
        WIDE s = a[0];
        for (int k = 1; k < K; k++) {
            int m = (int)(((long)k * j) % N);
            s += 2 * (a[k] * t->wc[m] - b[k] * t->ws[m]);
        }
        if (N % 2 == 0) { int m = (int)(((long)K * j) % N); s += a[K] * t->wc[m]; }
        else { int m = (int)(((long)K * j) % N); s += 2 * (a[K] * t->wc[m] - b[K] * t->ws[m]); }
        out[j] = s;
    }
    free(a); free(b);
}
static void multiplier(const trig_t *t, int which, const REAL *f, REAL *out) {
    int N = t->N;
    WIDE *wf = (WIDE *)malloc(sizeof(WIDE) * N), *wo = (WIDE *)malloc(sizeof(WIDE) * N);
    for (int j = 0; j < N; j++) wf[j] = (WIDE)f[j];
    multiplier_w(t, which, wf, wo);
    for (int j = 0; j < N; j++) out[j] = (REAL)wo[j];
    free(wf); free(wo);
}

/* ---------- mesh refinement: the change of variables x = xi(alpha), (2.10)-(2.11), PAPER.md:122-136 ----------
 *   E(alpha) = 1 - P[A sin^4(alpha/2)]  (refine near x = pi)   or   1 - P[A cos^4(alpha/2)]  (refine near x = 0),
 *   A = 8 (1 - rho) / (5 + 3 rho),  xi(alpha) = int_0^alpha E,  P removes the mean (3/8 for both fourth powers).
 * With sin^4(a/2) = 3/8 - cos(a)/2 + cos(2a)/8 and cos^4(a/2) = 3/8 + cos(a)/2 + cos(2a)/8 the primitive is elementary:
 *   xi - alpha = +-A sin(alpha)/2 - A sin(2 alpha)/16   (+ near pi, - near 0).
 * The state (eta, phi and the columns) is stored at the points x_j = xi(alpha_j); rho = 1 is the uniform mesh (E = 1).
 * The setting is process-wide (set_mesh below) and read when a surface is set up; it is not changed while a call runs. */
static REAL g_mesh_rho = 1;
static int g_mesh_where = 0;   /* 0: refine near x = pi, 1: refine near x = 0 */
static int mesh_on(void) { return g_mesh_rho != 1; }
/* xp = xi - alpha, E = xi', E1 = xi'' at alpha_j = 2 pi j / N */
static void mesh_tables(int N, REAL *xp, REAL *E, REAL *E1) {
    REAL A = 8 * (1 - g_mesh_rho) / (5 + 3 * g_mesh_rho);
    for (int j = 0; j < N; j++) {
        REAL ch, sh, c1, s1, c2, s2;
        trig_exact_r(j, 2L * N, &ch, &sh);          /* alpha_j / 2 */
        trig_exact_r(j, N, &c1, &s1);               /* alpha_j     */
        trig_exact_r(2L * j, N, &c2, &s2);          /* 2 alpha_j   */
        if (g_mesh_where == 0) {
            E[j] = 1 - A * (sh * sh * sh * sh - (REAL)3 / 8);
            E1[j] = -2 * A * sh * sh * sh * ch;
            xp[j] = A * s1 / 2 - A * s2 / 16;
        } else {
            E[j] = 1 - A * (ch * ch * ch * ch - (REAL)3 / 8);
            E1[j] = 2 * A * ch * ch * ch * sh;
            xp[j] = -A * s1 / 2 - A * s2 / 16;
        }
    }
}

/* O1: eta' = D eta, eta'' = D(D eta); the intermediate eta' stays in WIDE (R8). */
static void surface_derivs(const trig_t *t, const REAL *eta, REAL *d1, REAL *d2) {
    int N = t->N;
    WIDE *f = (WIDE *)malloc(sizeof(WIDE) * N), *g1 = (WIDE *)malloc(sizeof(WIDE) * N), *g2 = (WIDE *)malloc(sizeof(WIDE) * N);
    for (int j = 0; j < N; j++) f[j] = (WIDE)eta[j];
    multiplier_w(t, MUL_D, f, g1);
    multiplier_w(t, MUL_D, g1, g2);
    for (int j = 0; j < N; j++) { d1[j] = (REAL)g1[j]; d2[j] = (REAL)g2[j]; }
    free(f); free(g1); free(g2);
}

/* ---------- (c_r, c_i) = (1/2) cot((x + i y)/2), two-branch form of PAPER.md:154 ----------
 * cot((x+iy)/2) = (cos x + cosh y)/(sin x + i sinh y)         if cos x >= 0
 *               = (sin x - i sinh y)/(cosh y - cos x)         if cos x <  0
 * and 1/(sin x + i sinh y) = (sin x - i sinh y)/(sin^2 x + sinh^2 y).                       */
static void half_cot(REAL sx, REAL cx, REAL y, REAL *cr, REAL *ci) {
    REAL sh = R_SINH(y), ch = R_COSH(y), p;
    if (cx >= 0) p = (cx + ch) / (sx * sx + sh * sh);
    else p = 1 / (ch - cx);
    *cr = p * sx / 2;
    *ci = -p * sh / 2;
}

/* ---------- O1-O3: K and G from (2.13), with reading R1 ---------- */
/* On a refined mesh zeta(alpha) = xi(alpha) + i eta(xi(alpha)) (2.5): zeta' = E + i d1, zeta'' = E1 + i d2 (d1, d2: alpha-derivatives
 * of the stored values) and Re(zeta_i - zeta_j) = (alpha_i - alpha_j) + (xp_i - xp_j); xp = NULL is the uniform mesh. */
static int assemble(const trig_t *t, REAL h, const REAL *eta, const REAL *d1, const REAL *d2,
                    const REAL *xp, const REAL *E, const REAL *E1, REAL *K, REAL *G) {
    int N = t->N;
    int finite = !R_ISINF(h);
    if (finite) for (int i = 0; i < N; i++) if (!(h + eta[i] > 0)) return ORC_EBOTTOM;
    /* (1/2) cot((alpha_i - alpha_j)/2) depends on (i-j) mod N only: "computed once and for all" PAPER.md:150 */
    REAL *c0 = ralloc(N);
    c0[0] = 0;
    for (int m = 1; m < N; m++) { REAL ch, sh; trig_exact_r(m, 2L * N, &ch, &sh); c0[m] = ch / sh / 2; }   /* angle pi m/N */
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; i++) {
        for (int j = 0; j < N; j++) {
            int m = ((i - j) % N + N) % N;
            REAL sx = t->s[m], cx = t->c[m];
            REAL k1, g1, k2 = 0, g2 = 0, cr, ci;
            REAL Ei = xp ? E[i] : 1, Ej = xp ? E[j] : 1;
            if (xp) {                                    /* sin, cos of (alpha_i - alpha_j) + (xp_i - xp_j) */
                REAL dl = xp[i] - xp[j], sd = R_SIN(dl), cd = R_COS(dl);
                REAL s0 = sx, c0m = cx;
                sx = s0 * cd + c0m * sd;
                cx = c0m * cd - s0 * sd;
            }
            if (i != j) {
                REAL y1 = eta[i] - eta[j];               /* Im(zeta_i - zeta_j), from the raw inputs */
                half_cot(sx, cx, y1, &cr, &ci);
                k1 = Ej * ci + d1[j] * cr;               /* Im{ zeta'_j/2 cot } ; zeta' = E + i eta~' (E = 1: uniform) */
                g1 = Ei * cr - d1[i] * ci - c0[m];       /* Re{ zeta'_i/2 cot } - (1/2)cot((alpha_i - alpha_j)/2)       */
            } else {                                     /* continuous limits */
                REAL den = 2 * (Ei * Ei + d1[i] * d1[i]);
                REAL Ep = xp ? E1[i] : 0;                /* zeta'' = E' + i eta~'' */
                k1 = -(d2[i] * Ei - Ep * d1[i]) / den;   /* -Im{ zeta''/(2 zeta') } = -Im{ zeta'' conj(zeta') } / (2 |zeta'|^2) */
                g1 = (Ep * Ei + d1[i] * d2[i]) / den;    /*  Re{ zeta''/(2 zeta') }                  */
            }
            if (finite) {
                REAL y2 = (h + eta[i]) + (h + eta[j]);   /* Im(zeta_i - conj zeta_j) > 0 */
                half_cot(sx, cx, y2, &cr, &ci);
                k2 = Ej * ci - d1[j] * cr;               /* Im{ conj(zeta'_j)/2 cot } */
                g2 = Ei * cr - d1[i] * ci;               /* Re{ zeta'_i/2 cot }       */
            }
            K[(long)i * N + j] = (k1 - k2) / (REAL)N;    /* R1 */
            G[(long)i * N + j] = (g1 - g2) / (REAL)N;
        }
    }
    free(c0);
    return ORC_OK;
}

/* ---------- Gaussian elimination with partial pivoting, in place; piv[k] = row swapped with k ---------- */
static int lu_factor(int N, REAL *A, int *piv) {
    for (int k = 0; k < N; k++) {
        int p = k; REAL best = R_FABS(A[(long)k * N + k]);
        for (int i = k + 1; i < N; i++) { REAL v = R_FABS(A[(long)i * N + k]); if (v > best) { best = v; p = i; } }
        piv[k] = p;
        if (best == 0) return ORC_ESINGULAR;
        if (p != k) for (int j = 0; j < N; j++) { REAL tmp = A[(long)k * N + j]; A[(long)k * N + j] = A[(long)p * N + j]; A[(long)p * N + j] = tmp; }
        REAL piv_v = A[(long)k * N + k];
#pragma omp parallel for schedule(static) if (N - k > 64)
        for (int i = k + 1; i < N; i++) {
            REAL l = A[(long)i * N + k] / piv_v;
            A[(long)i * N + k] = l;
            const REAL *rk = A + (long)k * N;
            REAL *ri = A + (long)i * N;
            for (int j = k + 1; j < N; j++) ri[j] -= l * rk[j];
        }
    }
    return ORC_OK;
}
static void lu_solve(int N, const REAL *LU, const int *piv, REAL *x) {
    for (int k = 0; k < N; k++) { int p = piv[k]; if (p != k) { REAL t = x[k]; x[k] = x[p]; x[p] = t; } }
    for (int i = 1; i < N; i++) { REAL s = x[i]; const REAL *r = LU + (long)i * N; for (int j = 0; j < i; j++) s -= r[j] * x[j]; x[i] = s; }
    for (int i = N - 1; i >= 0; i--) { REAL s = x[i]; const REAL *r = LU + (long)i * N; for (int j = i + 1; j < N; j++) s -= r[j] * x[j]; x[i] = s / r[i]; }
}
static void matvec(int N, const REAL *M, const REAL *x, REAL *y) {
    for (int i = 0; i < N; i++) { REAL s = 0; const REAL *r = M + (long)i * N; for (int j = 0; j < N; j++) s += r[j] * x[j]; y[i] = s; }
}

/* ---------- a "setup": everything that depends on the surface only ---------- */
typedef struct {
    int N; REAL h; trig_t t;
    REAL *eta, *d1, *d2;   /* eta, eta', eta'' */
    REAL *K, *G, *LU; int *piv;
    REAL *xp, *E, *E1;     /* mesh (2.10): xi - alpha, xi', xi''; NULL on the uniform mesh */
} setup_t;

static void setup_free(setup_t *s) {
    trig_free(&s->t); free(s->eta); free(s->d1); free(s->d2); free(s->K); free(s->G); free(s->LU); free(s->piv);
    free(s->xp); free(s->E); free(s->E1);
}
static int setup_make(setup_t *s, int N, REAL h, const REAL *eta) {
    memset(s, 0, sizeof(*s));
    if (N < 4) return ORC_EINVAL;
    s->N = N; s->h = h;
    int rc = trig_init(&s->t, N); if (rc) return rc;
    s->eta = ralloc(N); s->d1 = ralloc(N); s->d2 = ralloc(N);
    s->K = ralloc((long)N * N); s->G = ralloc((long)N * N); s->LU = ralloc((long)N * N);
    s->piv = (int *)malloc(sizeof(int) * N);
    if (!s->eta || !s->d1 || !s->d2 || !s->K || !s->G || !s->LU || !s->piv) { setup_free(s); return ORC_ENOMEM; }
    memcpy(s->eta, eta, sizeof(REAL) * N);
    surface_derivs(&s->t, s->eta, s->d1, s->d2);  /* O1: eta', eta'' = D(D eta)  (R8) */
    if (mesh_on()) {
        s->xp = ralloc(N); s->E = ralloc(N); s->E1 = ralloc(N);
        if (!s->xp || !s->E || !s->E1) { setup_free(s); return ORC_ENOMEM; }
        mesh_tables(N, s->xp, s->E, s->E1);
    }
    rc = assemble(&s->t, h, s->eta, s->d1, s->d2, s->xp, s->E, s->E1, s->K, s->G); if (rc) { setup_free(s); return rc; }
    for (long i = 0; i < (long)N * N; i++) s->LU[i] = s->K[i];
    for (int i = 0; i < N; i++) s->LU[(long)i * N + i] += (REAL)0.5;   /* A = I/2 + K, (2.7) PAPER.md:105 */
    rc = lu_factor(N, s->LU, s->piv); if (rc) { setup_free(s); return rc; }
    return ORC_OK;
}

/* O4-O5: w = G(eta) b :  solve (I/2 + K) mu = b ; gamma = D mu ; w = H gamma / 2 + G gamma   (2.7),(2.8) */
static void dtn_one(const setup_t *s, const REAL *b, REAL *w, REAL *mu_out) {
    int N = s->N;
    REAL *mu = ralloc(N), *gam = ralloc(N), *hg = ralloc(N);
    memcpy(mu, b, sizeof(REAL) * N);
    lu_solve(N, s->LU, s->piv, mu);
    multiplier(&s->t, MUL_D, mu, gam);
    multiplier(&s->t, MUL_H, gam, hg);
    matvec(N, s->G, gam, w);
    for (int i = 0; i < N; i++) w[i] += hg[i] / 2;
    if (s->E) for (int i = 0; i < N; i++) w[i] /= s->E[i];      /* the factor 1/|xi'(alpha)| of (2.8) */
    if (mu_out) memcpy(mu_out, mu, sizeof(REAL) * N);
    free(mu); free(gam); free(hg);
}

/* d/dx of a function stored on the mesh: (1/xi') d/dalpha  (chain rule for f(xi(alpha))) */
static void deriv_x(const setup_t *s, const REAL *f, REAL *out) {
    multiplier(&s->t, MUL_D, f, out);
    if (s->E) for (int i = 0; i < s->N; i++) out[i] /= s->E[i];
}
/* P (2.2) and the filter (2.14) on the mesh: the filter acts on the stored samples (Fourier modes in alpha); the mean that P
 * removes is the mean over x, (1/2pi) int f dx = (1/N) sum_j f_j E_j by the trapezoidal rule with dx = E dalpha. */
static void project_x(const setup_t *s, int filter, const REAL *r, REAL *out) {
    int N = s->N;
    if (!s->E) { multiplier(&s->t, filter ? MUL_PFILTER : MUL_P, r, out); return; }
    if (filter) multiplier(&s->t, MUL_FILTER, r, out); else memcpy(out, r, sizeof(REAL) * N);
    REAL m = 0;
    for (int i = 0; i < N; i++) m += out[i] * s->E[i];
    m /= (REAL)N;
    for (int i = 0; i < N; i++) out[i] -= m;
}

/* O6: base state about which the problem is linearised; (2.9) PAPER.md:116 */
typedef struct { REAL *dphi, *W0, *u, *v; } base_t;
static void base_free(base_t *b) { free(b->dphi); free(b->W0); free(b->u); free(b->v); }
static void base_make(const setup_t *s, const REAL *phi0, base_t *b) {
    int N = s->N;
    b->dphi = ralloc(N); b->W0 = ralloc(N); b->u = ralloc(N); b->v = ralloc(N);
    deriv_x(s, phi0, b->dphi);
    dtn_one(s, phi0, b->W0, NULL);
    for (int i = 0; i < N; i++) {
        REAL e1 = s->E ? s->d1[i] / s->E[i] : s->d1[i], den = 1 + e1 * e1;   /* eta'(x) */
        b->u[i] = (b->dphi[i] - e1 * b->W0[i]) / den;     /* phi_x */
        b->v[i] = (e1 * b->dphi[i] + b->W0[i]) / den;     /* phi_y */
    }
}

/* ================= exported entry points ================= */

/* out = multiplier(which) f, one column.  Used by the tests to pin D, H, |D|, filter, P. */
int NAME(multiplier)(int N, int which, const double *fhi, const double *flo, double *ohi, double *olo) {
    trig_t t; int rc = trig_init(&t, N); if (rc) return rc;
    REAL *f = ralloc(N), *o = ralloc(N);
    load_hl(f, fhi, flo, N);
    multiplier(&t, which, f, o);
    store_hl(o, ohi, olo, N);
    free(f); free(o); trig_free(&t);
    return ORC_OK;
}

/* K, G (row-major N x N) and eta', eta''. Any output pointer may be NULL. */
int NAME(assemble)(int N, double h, const double *ehi, const double *elo,
                   double *Khi, double *Klo, double *Ghi, double *Glo,
                   double *d1hi, double *d1lo, double *d2hi, double *d2lo) {
    REAL *eta = ralloc(N); load_hl(eta, ehi, elo, N);
    setup_t s; int rc = setup_make(&s, N, (REAL)h, eta); free(eta); if (rc) return rc;
    if (Khi || Klo) store_hl(s.K, Khi, Klo, (long)N * N);
    if (Ghi || Glo) store_hl(s.G, Ghi, Glo, (long)N * N);
    if (d1hi || d1lo) store_hl(s.d1, d1hi, d1lo, N);
    if (d2hi || d2lo) store_hl(s.d2, d2hi, d2lo, N);
    setup_free(&s);
    return ORC_OK;
}

/* out_c = G(eta) phi_c, c < nrhs.  mu (optional) returns the dipole densities. */
int NAME(dtn_apply)(int N, double h, const double *ehi, const double *elo, int nrhs,
                    const double *phi_hi, const double *phi_lo, double *out_hi, double *out_lo,
                    double *mu_hi, double *mu_lo) {
    REAL *eta = ralloc(N); load_hl(eta, ehi, elo, N);
    setup_t s; int rc = setup_make(&s, N, (REAL)h, eta); free(eta); if (rc) return rc;
#pragma omp parallel for schedule(dynamic) if (nrhs > 1)
    for (int c = 0; c < nrhs; c++) {
        REAL *b = ralloc(N), *w = ralloc(N), *mu = ralloc(N);
        load_hl(b, phi_hi + (long)c * N, phi_lo ? phi_lo + (long)c * N : NULL, N);
        dtn_one(&s, b, w, mu);
        store_hl(w, out_hi + (long)c * N, out_lo ? out_lo + (long)c * N : NULL, N);
        if (mu_hi || mu_lo) store_hl(mu, mu_hi ? mu_hi + (long)c * N : NULL, mu_lo ? mu_lo + (long)c * N : NULL, N);
        free(b); free(w); free(mu);
    }
    setup_free(&s);
    return ORC_OK;
}

/* O7: out_c = d/de G(eta + e deta_c)[phi0 + e dphi_c] at e=0 = G[dphi_c - v deta_c] - D(u deta_c)   (B.1d),(B.2)
 * PAPER.md:699-708.  base_out (optional, 4N: phi0', W0, u, v as hi then lo) exposes the base state. */
int NAME(dtn_linearized)(int N, double h, const double *ehi, const double *elo,
                         const double *p0hi, const double *p0lo, int nrhs,
                         const double *dehi, const double *delo, const double *dphi, const double *dplo,
                         double *out_hi, double *out_lo, double *base_hi, double *base_lo) {
    REAL *eta = ralloc(N), *phi0 = ralloc(N);
    load_hl(eta, ehi, elo, N); load_hl(phi0, p0hi, p0lo, N);
    setup_t s; int rc = setup_make(&s, N, (REAL)h, eta); free(eta); if (rc) { free(phi0); return rc; }
    base_t bs; base_make(&s, phi0, &bs); free(phi0);
    if (base_hi || base_lo) {
        store_hl(bs.dphi, base_hi, base_lo, N);
        store_hl(bs.W0, base_hi ? base_hi + N : NULL, base_lo ? base_lo + N : NULL, N);
        store_hl(bs.u, base_hi ? base_hi + 2 * N : NULL, base_lo ? base_lo + 2 * N : NULL, N);
        store_hl(bs.v, base_hi ? base_hi + 3 * N : NULL, base_lo ? base_lo + 3 * N : NULL, N);
    }
#pragma omp parallel for schedule(dynamic) if (nrhs > 1)
    for (int c = 0; c < nrhs; c++) {
        REAL *de = ralloc(N), *dp = ralloc(N), *b = ralloc(N), *w = ralloc(N), *ud = ralloc(N), *dud = ralloc(N);
        load_hl(de, dehi + (long)c * N, delo ? delo + (long)c * N : NULL, N);
        load_hl(dp, dphi + (long)c * N, dplo ? dplo + (long)c * N : NULL, N);
        for (int i = 0; i < N; i++) { b[i] = dp[i] - bs.v[i] * de[i]; ud[i] = bs.u[i] * de[i]; }
        dtn_one(&s, b, w, NULL);
        deriv_x(&s, ud, dud);
        for (int i = 0; i < N; i++) w[i] -= dud[i];
        store_hl(w, out_hi + (long)c * N, out_lo ? out_lo + (long)c * N : NULL, N);
        free(de); free(dp); free(b); free(w); free(ud); free(dud);
    }
    base_free(&bs); setup_free(&s);
    return ORC_OK;
}

/* O8: right-hand sides of (2.1) and of the variational equation (B.1)-(B.3) at one state.
 * eta_t = W0 ; phi_t = P[ v W0 - u^2/2 - v^2/2 - g eta ]                                  (2.1)
 * deta_t = w_c - D(u deta_c)                                                              (B.2)
 * dphi_t = P[ -D(deta_c u v) - u D(b_c) + v w_c - g deta_c ], b_c = dphi_c - v deta_c      (B.1f)+(B.3)
 * each multiplied by the filter (2.14) when filter != 0 (R5).  All arrays REAL, columns at c*N.
 * Surface tension (sigma = sigma/rho of (2.1b); zero in sections 4.1-4.5, one in section 4.6):
 *   phi_t  += P[ sigma D( eta' / sqrt(1 + eta'^2) ) ]                                      (2.1b)
 *   dphi_t += P[ sigma D( D(deta_c) / (1 + eta'^2)^(3/2) ) ]                                (B.4) */
static int rhs_eval(int N, REAL h, REAL g, REAL sigma, int filter, const REAL *eta, const REAL *phi, int ncols,
                    const REAL *deta, const REAL *dphi, REAL *eta_t, REAL *phi_t, REAL *deta_t, REAL *dphi_t, REAL *energy) {
    setup_t s; int rc = setup_make(&s, N, h, eta); if (rc) return rc;
    base_t bs; base_make(&s, phi, &bs);
    REAL *tmp = ralloc(N);
    for (int i = 0; i < N; i++) tmp[i] = bs.v[i] * bs.W0[i] - bs.u[i] * bs.u[i] / 2 - bs.v[i] * bs.v[i] / 2 - g * eta[i];
    if (sigma != 0) {
        REAL *cv = ralloc(N), *dcv = ralloc(N);
        for (int i = 0; i < N; i++) { REAL e1 = s.E ? s.d1[i] / s.E[i] : s.d1[i]; cv[i] = e1 / R_SQRT(1 + e1 * e1); }
        deriv_x(&s, cv, dcv);
        for (int i = 0; i < N; i++) tmp[i] += sigma * dcv[i];
        free(cv); free(dcv);
    }
    if (eta_t) { if (filter) multiplier(&s.t, MUL_FILTER, bs.W0, eta_t); else memcpy(eta_t, bs.W0, sizeof(REAL) * N); }
    if (phi_t) project_x(&s, filter, tmp, phi_t);
    if (energy) {   /* E = (1/2) int (phi G phi + g eta^2) dx; dx = xi' dalpha on a refined mesh */
        REAL e = 0; for (int i = 0; i < N; i++) e += (phi[i] * bs.W0[i] + g * eta[i] * eta[i]) * (s.E ? s.E[i] : 1);
        *energy = e * R_PI / (REAL)N;
    }
    free(tmp);
#pragma omp parallel for schedule(dynamic) if (ncols > 1)
    for (int c = 0; c < ncols; c++) {
        const REAL *de = deta + (long)c * N, *dp = dphi + (long)c * N;
        REAL *b = ralloc(N), *w = ralloc(N), *t1 = ralloc(N), *t2 = ralloc(N), *db = ralloc(N), *r = ralloc(N);
        for (int i = 0; i < N; i++) b[i] = dp[i] - bs.v[i] * de[i];
        dtn_one(&s, b, w, NULL);
        for (int i = 0; i < N; i++) t1[i] = bs.u[i] * de[i];
        deriv_x(&s, t1, t2);
        for (int i = 0; i < N; i++) r[i] = w[i] - t2[i];
        if (filter) multiplier(&s.t, MUL_FILTER, r, deta_t + (long)c * N); else memcpy(deta_t + (long)c * N, r, sizeof(REAL) * N);
        for (int i = 0; i < N; i++) t1[i] = de[i] * bs.u[i] * bs.v[i];
        deriv_x(&s, t1, t2);
        deriv_x(&s, b, db);
        for (int i = 0; i < N; i++) r[i] = -t2[i] - bs.u[i] * db[i] + bs.v[i] * w[i] - g * de[i];
        if (sigma != 0) {
            deriv_x(&s, de, t1);
            for (int i = 0; i < N; i++) { REAL e1 = s.E ? s.d1[i] / s.E[i] : s.d1[i], den = 1 + e1 * e1; t1[i] = t1[i] / (den * R_SQRT(den)); }
            deriv_x(&s, t1, t2);
            for (int i = 0; i < N; i++) r[i] += sigma * t2[i];
        }
        project_x(&s, filter, r, dphi_t + (long)c * N);
        free(b); free(w); free(t1); free(t2); free(db); free(r);
    }
    base_free(&bs); setup_free(&s);
    return ORC_OK;
}

int NAME(rhs)(int N, double h, double g, double sigma, int filter, const double *ehi, const double *elo, const double *phi_hi, const double *phi_lo,
              int ncols, const double *dehi, const double *delo, const double *dphi, const double *dplo,
              double *out_hi, double *out_lo /* 2N(1+ncols): eta_t, phi_t, deta_t[ncols], dphi_t[ncols] */, double *energy_hl /* 2 */) {
    long n1 = N, nc = (long)N * ncols;
    REAL *eta = ralloc(n1), *phi = ralloc(n1), *de = ralloc(nc), *dp = ralloc(nc);
    REAL *o = ralloc(2 * n1 + 2 * nc), E = 0;
    load_hl(eta, ehi, elo, n1); load_hl(phi, phi_hi, phi_lo, n1);
    if (ncols) { load_hl(de, dehi, delo, nc); load_hl(dp, dphi, dplo, nc); }
    int rc = rhs_eval(N, (REAL)h, (REAL)g, (REAL)sigma, filter, eta, phi, ncols, de, dp, o, o + n1, o + 2 * n1, o + 2 * n1 + nc, &E);
    if (!rc) {
        store_hl(o, out_hi, out_lo, 2 * n1 + 2 * nc);
        if (energy_hl) store_hl(&E, energy_hl, energy_hl + 1, 1);
    }
    free(eta); free(phi); free(de); free(dp); free(o);
    return rc;
}

/* The adjoint system (B.6): right-hand side of q~_s = DF(q)^* q~ at the state q = (eta, phi) for ncols adjoint
 * vectors (eta~_c, phi~_c), with u = phi_x, v = phi_y on the surface (2.9):
 *   chi_c     = eta~_c + v P phi~_c                                                              (B.6d)
 *   phi~_s,c  = G chi_c + D( u P phi~_c )                                                        (B.6e), G chi = chi_y - eta' chi_x
 *   eta~_s,c  = -v G chi_c + u D eta~_c - v D(u) P phi~_c - g P phi~_c + sigma D( D(phi~_c) / (1 + eta'^2)^(3/2) )   (B.6f)
 * (no filter: the adjoint identity <DF(q) qdot, q~> = <qdot, DF(q)^* q~> is stated for the unfiltered operators). */
static int adjoint_eval(int N, REAL h, REAL g, REAL sigma, const REAL *eta, const REAL *phi, int ncols,
                        const REAL *etat, const REAL *phit, REAL *eta_s, REAL *phi_s) {
    setup_t s; int rc = setup_make(&s, N, h, eta); if (rc) return rc;   /* refined mesh: D = d/dx, P = mean over x (deriv_x, project_x) */
    base_t bs; base_make(&s, phi, &bs);
    REAL *du = ralloc(N);
    deriv_x(&s, bs.u, du);
#pragma omp parallel for schedule(dynamic) if (ncols > 1)
    for (int c = 0; c < ncols; c++) {
        const REAL *et = etat + (long)c * N, *pt = phit + (long)c * N;
        REAL *pp = ralloc(N), *chi = ralloc(N), *w = ralloc(N), *t1 = ralloc(N), *t2 = ralloc(N), *det = ralloc(N);
        project_x(&s, 0, pt, pp);
        for (int i = 0; i < N; i++) chi[i] = et[i] + bs.v[i] * pp[i];
        dtn_one(&s, chi, w, NULL);
        for (int i = 0; i < N; i++) t1[i] = bs.u[i] * pp[i];
        deriv_x(&s, t1, t2);
        for (int i = 0; i < N; i++) phi_s[(long)c * N + i] = w[i] + t2[i];
        deriv_x(&s, et, det);
        for (int i = 0; i < N; i++) eta_s[(long)c * N + i] = -bs.v[i] * w[i] + bs.u[i] * det[i] - bs.v[i] * du[i] * pp[i] - g * pp[i];
        if (sigma != 0) {
            deriv_x(&s, pt, t1);
            for (int i = 0; i < N; i++) { REAL e1 = s.E ? s.d1[i] / s.E[i] : s.d1[i], den = 1 + e1 * e1; t1[i] = t1[i] / (den * R_SQRT(den)); }
            deriv_x(&s, t1, t2);
            for (int i = 0; i < N; i++) eta_s[(long)c * N + i] += sigma * t2[i];
        }
        free(pp); free(chi); free(w); free(t1); free(t2); free(det);
    }
    free(du); base_free(&bs); setup_free(&s);
    return ORC_OK;
}
int NAME(adjoint_rhs)(int N, double h, double g, double sigma, const double *ehi, const double *elo, const double *phi_hi, const double *phi_lo,
                      int ncols, const double *ethi, const double *etlo, const double *pthi, const double *ptlo,
                      double *out_hi, double *out_lo /* 2 N ncols: eta~_s[ncols], phi~_s[ncols] */) {
    long n1 = N, nc = (long)N * ncols;
    REAL *eta = ralloc(n1), *phi = ralloc(n1), *et = ralloc(nc), *pt = ralloc(nc), *o = ralloc(2 * nc);
    load_hl(eta, ehi, elo, n1); load_hl(phi, phi_hi, phi_lo, n1);
    load_hl(et, ethi, etlo, nc); load_hl(pt, pthi, ptlo, nc);
    int rc = adjoint_eval(N, (REAL)h, (REAL)g, (REAL)sigma, eta, phi, ncols, et, pt, o, o + nc);
    if (!rc) store_hl(o, out_hi, out_lo, 2 * nc);
    free(eta); free(phi); free(et); free(pt); free(o);
    return rc;
}

/* ---------- R6: 11-stage, order-8 explicit Runge-Kutta tableau, coefficients in Q(sqrt 21) ---------- */
#define RK_S 11
static void rk_tableau(REAL a[RK_S][RK_S], REAL b[RK_S], REAL c[RK_S]) {
    REAL s = R_SQRT((REAL)21);
    memset(a, 0, sizeof(REAL) * RK_S * RK_S);
    for (int i = 0; i < RK_S; i++) b[i] = 0;
    c[0] = 0; c[1] = (REAL)1 / 2; c[2] = (REAL)1 / 2; c[3] = (7 + s) / 14; c[4] = (7 + s) / 14; c[5] = (REAL)1 / 2;
    c[6] = (7 - s) / 14; c[7] = (7 - s) / 14; c[8] = (REAL)1 / 2; c[9] = (7 + s) / 14; c[10] = 1;
    b[0] = (REAL)1 / 20; b[7] = (REAL)49 / 180; b[8] = (REAL)16 / 45; b[9] = (REAL)49 / 180; b[10] = (REAL)1 / 20;
    a[1][0] = (REAL)1 / 2;
    a[2][0] = (REAL)1 / 4; a[2][1] = (REAL)1 / 4;
    a[3][0] = (REAL)1 / 7; a[3][1] = (-7 - 3 * s) / 98; a[3][2] = (21 + 5 * s) / 49;
    a[4][0] = (11 + s) / 84; a[4][2] = (18 + 4 * s) / 63; a[4][3] = (21 - s) / 252;
    a[5][0] = (5 + s) / 48; a[5][2] = (9 + s) / 36; a[5][3] = (-231 + 14 * s) / 360; a[5][4] = (63 - 7 * s) / 80;
    a[6][0] = (10 - s) / 42; a[6][2] = (-432 + 92 * s) / 315; a[6][3] = (633 - 145 * s) / 90; a[6][4] = (-504 + 115 * s) / 70; a[6][5] = (63 - 13 * s) / 35;
    a[7][0] = (REAL)1 / 14; a[7][4] = (14 - 3 * s) / 126; a[7][5] = (13 - 3 * s) / 63; a[7][6] = (REAL)1 / 9;
    a[8][0] = (REAL)1 / 32; a[8][4] = (91 - 21 * s) / 576; a[8][5] = (REAL)11 / 72; a[8][6] = (-385 - 75 * s) / 1152; a[8][7] = (63 + 13 * s) / 128;
    a[9][0] = (REAL)1 / 14; a[9][4] = (REAL)1 / 9; a[9][5] = (-733 - 147 * s) / 2205; a[9][6] = (515 + 111 * s) / 504; a[9][7] = (-51 - 11 * s) / 56; a[9][8] = (132 + 28 * s) / 245;
    a[10][4] = (-42 + 7 * s) / 18; a[10][5] = (-18 + 28 * s) / 45; a[10][6] = (-273 - 53 * s) / 72; a[10][7] = (301 + 53 * s) / 72; a[10][8] = (28 - 28 * s) / 45; a[10][9] = (49 - 7 * s) / 18;
}

/* tableau as hi/lo doubles: a (11x11 row-major), b (11), c (11) */
int NAME(rk_tableau)(double *a_hi, double *a_lo, double *b_hi, double *b_lo, double *c_hi, double *c_lo) {
    REAL a[RK_S][RK_S], b[RK_S], c[RK_S];
    rk_tableau(a, b, c);
    store_hl(&a[0][0], a_hi, a_lo, RK_S * RK_S); store_hl(b, b_hi, b_lo, RK_S); store_hl(c, c_hi, c_lo, RK_S);
    return ORC_OK;
}

/* generic explicit RK step driver on y' = f(y), used by the tests to pin the tableau on ODEs with known solutions:
 * y' = lambda y (complex lambda = lr + i li, y complex), nsteps of size dt; returns y(T) as hi/lo of (re, im). */
int NAME(rk_linear_test)(double lr, double li, double dt, int nsteps, double *y_hi, double *y_lo) {
    REAL a[RK_S][RK_S], b[RK_S], c[RK_S];
    rk_tableau(a, b, c);
    REAL yr = 1, yi = 0, kr[RK_S], ki[RK_S], h = (REAL)dt, Lr = (REAL)lr, Li = (REAL)li;
    for (int n = 0; n < nsteps; n++) {
        for (int i = 0; i < RK_S; i++) {
            REAL sr = yr, si = yi;
            for (int j = 0; j < i; j++) { sr += h * a[i][j] * kr[j]; si += h * a[i][j] * ki[j]; }
            kr[i] = Lr * sr - Li * si; ki[i] = Lr * si + Li * sr;
        }
        for (int i = 0; i < RK_S; i++) { yr += h * b[i] * kr[i]; yi += h * b[i] * ki[i]; }
    }
    REAL y[2] = { yr, yi };
    store_hl(y, y_hi, y_lo, 2);
    return ORC_OK;
}
/* y' = -y^2 (nonlinear, non-autonomous-free), y(0) = 1, exact y(t) = 1/(1+t) */
int NAME(rk_riccati_test)(double dt, int nsteps, double *y_hi, double *y_lo) {
    REAL a[RK_S][RK_S], b[RK_S], c[RK_S];
    rk_tableau(a, b, c);
    REAL y = 1, k[RK_S], h = (REAL)dt;
    for (int n = 0; n < nsteps; n++) {
        for (int i = 0; i < RK_S; i++) { REAL s = y; for (int j = 0; j < i; j++) s += h * a[i][j] * k[j]; k[i] = -s * s; }
        for (int i = 0; i < RK_S; i++) y += h * b[i] * k[i];
    }
    store_hl(&y, y_hi, y_lo, 1);
    return ORC_OK;
}

/* O9: advance (eta, phi, deta[ncols], dphi[ncols]) by nsteps RK8 steps of size dt, in place; (3.32) PAPER.md:301.
 * The state is filtered after every step when filter != 0 (R5).  energies (optional, nsteps+1 hi then nsteps+1 lo). */
int NAME(rk_advance)(int N, double h, double g, double sigma, int filter, double dt, int nsteps,
                     double *ehi, double *elo, double *phi_hi, double *phi_lo,
                     int ncols, double *dehi, double *delo, double *dphi, double *dplo, double *energies) {
    long n1 = N, nc = (long)N * ncols, L = 2 * n1 + 2 * nc;
    REAL a[RK_S][RK_S], b[RK_S], c[RK_S];
    rk_tableau(a, b, c);
    REAL *y = ralloc(L), *ys = ralloc(L), *k = ralloc(L * RK_S), *tmp = ralloc(N);
    if (!y || !ys || !k) return ORC_ENOMEM;
    load_hl(y, ehi, elo, n1); load_hl(y + n1, phi_hi, phi_lo, n1);
    if (ncols) { load_hl(y + 2 * n1, dehi, delo, nc); load_hl(y + 2 * n1 + nc, dphi, dplo, nc); }
    trig_t t; trig_init(&t, N);
    REAL H = (REAL)dt; int rc = ORC_OK;
    for (int n = 0; n < nsteps && !rc; n++) {
        for (int i = 0; i < RK_S && !rc; i++) {
            for (long q = 0; q < L; q++) { REAL s = y[q]; for (int j = 0; j < i; j++) if (a[i][j] != 0) s += H * a[i][j] * k[(long)j * L + q]; ys[q] = s; }
            REAL E, *ki = k + (long)i * L;
            rc = rhs_eval(N, (REAL)h, (REAL)g, (REAL)sigma, filter, ys, ys + n1, ncols, ys + 2 * n1, ys + 2 * n1 + nc,
                          ki, ki + n1, ki + 2 * n1, ki + 2 * n1 + nc, (i == 0 && energies) ? &E : NULL);
            if (i == 0 && energies && !rc) store_hl(&E, energies + n, energies + (nsteps + 1) + n, 1);
        }
        for (long q = 0; q < L; q++) { REAL s = y[q]; for (int i = 0; i < RK_S; i++) if (b[i] != 0) s += H * b[i] * k[(long)i * L + q]; y[q] = s; }
        if (filter) for (long col = 0; col < 2 + 2 * (long)ncols; col++) { multiplier(&t, MUL_FILTER, y + col * N, tmp); memcpy(y + col * N, tmp, sizeof(REAL) * N); }
    }
    if (!rc && energies) {
        REAL E; rc = rhs_eval(N, (REAL)h, (REAL)g, (REAL)sigma, filter, y, y + n1, 0, NULL, NULL, NULL, NULL, NULL, NULL, &E);
        if (!rc) store_hl(&E, energies + nsteps, energies + (nsteps + 1) + nsteps, 1);
    }
    if (!rc) {
        store_hl(y, ehi, elo, n1); store_hl(y + n1, phi_hi, phi_lo, n1);
        if (ncols) { store_hl(y + 2 * n1, dehi, delo, nc); store_hl(y + 2 * n1 + nc, dphi, dplo, nc); }
    }
    trig_free(&t); free(y); free(ys); free(k); free(tmp);
    return rc;
}

/* ---------- SDC15: spectral deferred correction on 8 Radau IIa nodes (reading R15 of DESIGN.md) ----------
 * Nodes c_1 < ... < c_s = 1: the right Radau points, ((x + 1)/2 for the roots x of P_s - P_{s-1} on (-1, 1]).
 * Integration matrix S_mj = int_0^{c_m} l_j(tau) dtau, l_j the Lagrange basis on the nodes (the coefficient matrix of the Radau IIa
 * collocation method), by an n-point Gauss-Legendre rule with 2 n - 1 >= s - 1 on [0, c_m] (exact);
 * b_j = S_sj.  One step y_n -> y_{n+1} of size h:
 *   predictor  : Y_0 = y_n, Y_m = classical RK4 step from Y_{m-1} over (c_m - c_{m-1}) h      ("initial values ... via fourth order Runge-Kutta")
 *   10 sweeps  : Y_m <- y_n + h sum_j S_mj F(Y_j), m = 1..s, all from the previous sweep     ("pure Picard corrections")
 *   final      : y_{n+1} = y_n + h sum_j b_j F(Y_j)                                            ("the final integration step")
 * The Picard iteration converges to the Radau IIa collocation solution (order 2 s - 1 = 15); every sweep gains one order on the
 * RK4 predictor.  F is rhs_eval (filtered when filter != 0); the state is filtered after every step as in rk_advance. */
#define SDC_S 8
#define SDC_SWEEPS 10
static REAL legendre(int n, REAL x, REAL *dp) {   /* P_n(x) and P_n'(x) by the three-term recurrence */
    REAL p0 = 1, p1 = x;
    if (n == 0) { if (dp) *dp = 0; return 1; }
    for (int k = 2; k <= n; k++) { REAL p2 = ((2 * k - 1) * x * p1 - (k - 1) * p0) / k; p0 = p1; p1 = p2; }
    if (dp) *dp = n * (x * p1 - p0) / (x * x - 1);
    return p1;
}
static void sdc_tables(int s, REAL *c, REAL *S /* s x s row-major */) {
    /* roots of f = P_s - P_{s-1} in (-1, 1): bracket by a scan, then bisection to the last bit; the root x = 1 is known */
    int found = 0; const int scan = 4000;
    REAL xa = -1, fa = legendre(s, xa, NULL) - legendre(s - 1, xa, NULL);
    for (int i = 1; i < scan && found < s - 1; i++) {
        REAL xb = -1 + (REAL)2 * i / scan, fb = legendre(s, xb, NULL) - legendre(s - 1, xb, NULL);
        if ((fa < 0) != (fb < 0)) {
            REAL lo = xa, hi = xb, flo = fa;
            for (int it = 0; it < 200; it++) {
                REAL mid = (lo + hi) / 2, fm = legendre(s, mid, NULL) - legendre(s - 1, mid, NULL);
                if (mid == lo || mid == hi) break;
                if ((fm < 0) == (flo < 0)) { lo = mid; flo = fm; } else hi = mid;
            }
            c[found++] = ((lo + hi) / 2 + 1) / 2;
        }
        xa = xb; fa = fb;
    }
    c[s - 1] = 1;
    /* Gauss-Legendre rule with ng points on [-1, 1] (2 ng - 1 >= s - 1): nodes by Newton from the Chebyshev guesses */
    const int ng = (s + 1) / 2 + 1;
    REAL gx[16], gw[16];
    for (int i = 0; i < ng; i++) {
        REAL x = R_COS(R_PI * (i + (REAL)0.75) / (ng + (REAL)0.5)), dp;
        for (int it = 0; it < 100; it++) { REAL p = legendre(ng, x, &dp); REAL dx = p / dp; x -= dx; if (R_FABS(dx) < (REAL)1e-40) break; }
        legendre(ng, x, &dp);
        gx[i] = x; gw[i] = 2 / ((1 - x * x) * dp * dp);
    }
    for (int m = 0; m < s; m++)
        for (int j = 0; j < s; j++) {
            REAL acc = 0;
            for (int q = 0; q < ng; q++) {
                REAL tau = c[m] * (gx[q] + 1) / 2, l = 1;
                for (int i = 0; i < s; i++) if (i != j) l *= (tau - c[i]) / (c[j] - c[i]);
                acc += gw[q] * l;
            }
            S[m * s + j] = acc * c[m] / 2;
        }
}
int NAME(sdc_tables)(int s, double *c_hi, double *c_lo, double *S_hi, double *S_lo) {
    if (s < 1 || s > 12) return ORC_EINVAL;
    REAL c[12], S[144];
    sdc_tables(s, c, S);
    store_hl(c, c_hi, c_lo, s); store_hl(S, S_hi, S_lo, (long)s * s);
    return ORC_OK;
}
/* the same driver on y' = lambda y (complex), for the order test: returns y(nsteps dt) */
int NAME(sdc_linear_test)(double lr, double li, double dt, int nsteps, double *y_hi, double *y_lo) {
    REAL c[SDC_S], S[SDC_S * SDC_S], h = (REAL)dt, Lr = (REAL)lr, Li = (REAL)li;
    sdc_tables(SDC_S, c, S);
    REAL yr = 1, yi = 0;
#define LAM(ar, ai, or_, oi) do { (or_) = Lr * (ar) - Li * (ai); (oi) = Lr * (ai) + Li * (ar); } while (0)
    for (int n = 0; n < nsteps; n++) {
        REAL Yr[SDC_S], Yi[SDC_S], Fr[SDC_S], Fi[SDC_S], pr = yr, pi = yi;
        for (int m = 0; m < SDC_S; m++) {   /* RK4 predictor */
            REAL hm = (c[m] - (m ? c[m - 1] : 0)) * h, k1r, k1i, k2r, k2i, k3r, k3i, k4r, k4i;
            LAM(pr, pi, k1r, k1i);
            LAM(pr + hm / 2 * k1r, pi + hm / 2 * k1i, k2r, k2i);
            LAM(pr + hm / 2 * k2r, pi + hm / 2 * k2i, k3r, k3i);
            LAM(pr + hm * k3r, pi + hm * k3i, k4r, k4i);
            pr += hm / 6 * (k1r + 2 * k2r + 2 * k3r + k4r); pi += hm / 6 * (k1i + 2 * k2i + 2 * k3i + k4i);
            Yr[m] = pr; Yi[m] = pi;
        }
        for (int m = 0; m < SDC_S; m++) LAM(Yr[m], Yi[m], Fr[m], Fi[m]);
        for (int sw = 0; sw < SDC_SWEEPS; sw++) {
            for (int m = 0; m < SDC_S; m++) {
                REAL sr = yr, si = yi;
                for (int j = 0; j < SDC_S; j++) { sr += h * S[m * SDC_S + j] * Fr[j]; si += h * S[m * SDC_S + j] * Fi[j]; }
                Yr[m] = sr; Yi[m] = si;
            }
            for (int m = 0; m < SDC_S; m++) LAM(Yr[m], Yi[m], Fr[m], Fi[m]);
        }
        for (int j = 0; j < SDC_S; j++) { yr += h * S[(SDC_S - 1) * SDC_S + j] * Fr[j]; yi += h * S[(SDC_S - 1) * SDC_S + j] * Fi[j]; }
    }
#undef LAM
    REAL y[2] = { yr, yi };
    store_hl(y, y_hi, y_lo, 2);
    return ORC_OK;
}
/* advance (eta, phi, deta[ncols], dphi[ncols]) by nsteps SDC15 steps of size dt, in place (same arguments as rk_advance) */
int NAME(sdc_advance)(int N, double h, double g, double sigma, int filter, double dt, int nsteps,
                      double *ehi, double *elo, double *phi_hi, double *phi_lo,
                      int ncols, double *dehi, double *delo, double *dphi, double *dplo, double *energies) {
    long n1 = N, nc = (long)N * ncols, L = 2 * n1 + 2 * nc;
    REAL c[SDC_S], S[SDC_S * SDC_S];
    sdc_tables(SDC_S, c, S);
    REAL *y = ralloc(L), *Y = ralloc(L * SDC_S), *F = ralloc(L * SDC_S), *k = ralloc(L * 4), *ys = ralloc(L), *tmp = ralloc(N);
    if (!y || !Y || !F || !k || !ys) return ORC_ENOMEM;
    load_hl(y, ehi, elo, n1); load_hl(y + n1, phi_hi, phi_lo, n1);
    if (ncols) { load_hl(y + 2 * n1, dehi, delo, nc); load_hl(y + 2 * n1 + nc, dphi, dplo, nc); }
    trig_t t; trig_init(&t, N);
    REAL H = (REAL)dt; int rc = ORC_OK;
#define EVAL(state, out, en) rhs_eval(N, (REAL)h, (REAL)g, (REAL)sigma, filter, (state), (state) + n1, ncols, (state) + 2 * n1, (state) + 2 * n1 + nc, \
                                      (out), (out) + n1, (out) + 2 * n1, (out) + 2 * n1 + nc, (en))
    for (int n = 0; n < nsteps && !rc; n++) {
        REAL E;
        for (int m = 0; m < SDC_S && !rc; m++) {   /* predictor: RK4 from node to node */
            const REAL *prev = m ? Y + (long)(m - 1) * L : y;
            REAL hm = (c[m] - (m ? c[m - 1] : 0)) * H, *k1 = k, *k2 = k + L, *k3 = k + 2 * L, *k4 = k + 3 * L, *Ym = Y + (long)m * L;
            if (m == 0) { rc = EVAL(y, k1, energies ? &E : NULL); if (energies && !rc) store_hl(&E, energies + n, energies + (nsteps + 1) + n, 1); }
            else memcpy(k1, F + (long)(m - 1) * L, sizeof(REAL) * L);
            for (long q = 0; q < L; q++) ys[q] = prev[q] + hm / 2 * k1[q];
            if (!rc) rc = EVAL(ys, k2, NULL);
            for (long q = 0; q < L; q++) ys[q] = prev[q] + hm / 2 * k2[q];
            if (!rc) rc = EVAL(ys, k3, NULL);
            for (long q = 0; q < L; q++) ys[q] = prev[q] + hm * k3[q];
            if (!rc) rc = EVAL(ys, k4, NULL);
            for (long q = 0; q < L; q++) Ym[q] = prev[q] + hm / 6 * (k1[q] + 2 * k2[q] + 2 * k3[q] + k4[q]);
            if (!rc) rc = EVAL(Ym, F + (long)m * L, NULL);
        }
        for (int sw = 0; sw < SDC_SWEEPS && !rc; sw++) {
            for (int m = 0; m < SDC_S; m++)
                for (long q = 0; q < L; q++) { REAL s = y[q]; for (int j = 0; j < SDC_S; j++) s += H * S[m * SDC_S + j] * F[(long)j * L + q]; Y[(long)m * L + q] = s; }
            for (int m = 0; m < SDC_S && !rc; m++) rc = EVAL(Y + (long)m * L, F + (long)m * L, NULL);
        }
        for (long q = 0; q < L; q++) { REAL s = y[q]; for (int j = 0; j < SDC_S; j++) s += H * S[(SDC_S - 1) * SDC_S + j] * F[(long)j * L + q]; y[q] = s; }
        if (filter) for (long col = 0; col < 2 + 2 * (long)ncols; col++) { multiplier(&t, MUL_FILTER, y + col * N, tmp); memcpy(y + col * N, tmp, sizeof(REAL) * N); }
    }
    if (!rc && energies) {
        REAL E; rc = rhs_eval(N, (REAL)h, (REAL)g, (REAL)sigma, filter, y, y + n1, 0, NULL, NULL, NULL, NULL, NULL, NULL, &E);
        if (!rc) store_hl(&E, energies + nsteps, energies + (nsteps + 1) + nsteps, 1);
    }
#undef EVAL
    if (!rc) {
        store_hl(y, ehi, elo, n1); store_hl(y + n1, phi_hi, phi_lo, n1);
        if (ncols) { store_hl(y + 2 * n1, dehi, delo, nc); store_hl(y + 2 * n1 + nc, dphi, dplo, nc); }
    }
    trig_free(&t); free(y); free(Y); free(F); free(k); free(ys); free(tmp);
    return rc;
}

/* thread count of the following calls (no arithmetic: small problems run faster on one thread than through the OpenMP barriers) */
/* ---------- mesh refinement: setting, tables, respacing (2.10)-(2.11), PAPER.md:122-136 ---------- */
/* rho in (0, 1]; where = 0 refines near x = pi, 1 near x = 0.  rho = 1: the uniform mesh. */
int NAME(set_mesh)(double rho, int where) {
    if (!(rho > 0 && rho <= 1) || (where != 0 && where != 1)) return ORC_EINVAL;
    g_mesh_rho = (REAL)rho; g_mesh_where = where;
    return ORC_OK;
}
/* xi(alpha_j) - alpha_j, E = xi', E1 = xi'' of the current setting at alpha_j = 2 pi j / N */
int NAME(mesh_tables)(int N, double *xp_hi, double *xp_lo, double *E_hi, double *E_lo, double *E1_hi, double *E1_lo) {
    REAL *xp = ralloc(N), *E = ralloc(N), *E1 = ralloc(N);
    mesh_tables(N, xp, E, E1);
    store_hl(xp, xp_hi, xp_lo, N); store_hl(E, E_hi, E_lo, N); store_hl(E1, E1_hi, E1_lo, N);
    free(xp); free(E); free(E1);
    return ORC_OK;
}
/* xi(b) and xi'(b) at an arbitrary parameter value b */
static void mesh_xi(REAL rho, int where, REAL b, REAL *xi, REAL *E) {
    REAL A = 8 * (1 - rho) / (5 + 3 * rho), sg = where == 0 ? 1 : -1;
    *xi = b + sg * A * R_SIN(b) / 2 - A * R_SIN(2 * b) / 16;
    *E = 1 + sg * A * R_COS(b) / 2 - A * R_COS(2 * b) / 8;
}
/* Respacing from segment l to l+1: f o xi_new(alpha_j) = (f o xi_old)(beta_j), beta_j = xi_old^{-1}(xi_new(alpha_j))
 * by Newton's method, alpha_j = 2 pi j / Mn; f o xi_old is evaluated at beta_j through its trigonometric interpolant on the
 * old mesh (Mo points): a_k, b_k as in the multipliers above, the Nyquist mode as a cosine.  Columns of f at c*Mo, of out at c*Mn. */
int NAME(respace)(int Mo, double rho_o, int where_o, int Mn, double rho_n, int where_n, int ncols,
                  const double *fhi, const double *flo, double *ohi, double *olo) {
    if (Mo < 4 || Mn < 4 || (Mo & 1)) return ORC_EINVAL;
    REAL *beta = ralloc(Mn);
    for (int j = 0; j < Mn; j++) {
        REAL al = 2 * R_PI * (REAL)j / (REAL)Mn, x, e, b, xb, eb;
        mesh_xi((REAL)rho_n, where_n, al, &x, &e);
        b = x;
        for (int it = 0; it < 60; it++) {
            mesh_xi((REAL)rho_o, where_o, b, &xb, &eb);
            REAL step = (xb - x) / eb;
            b -= step;
            if (step == 0) break;
        }
        beta[j] = b;
    }
#pragma omp parallel for schedule(dynamic) if (ncols > 1)
    for (int c = 0; c < ncols; c++) {
        REAL *f = ralloc(Mo), *a = ralloc(Mo / 2 + 1), *bb = ralloc(Mo / 2 + 1), *o = ralloc(Mn);
        load_hl(f, fhi + (long)c * Mo, flo ? flo + (long)c * Mo : NULL, Mo);
        for (int k = 0; k <= Mo / 2; k++) {
            REAL sa = 0, sb = 0;
            for (int j = 0; j < Mo; j++) {
                REAL cc, ss; trig_exact_r((long)k * j, Mo, &cc, &ss);
                sa += f[j] * cc; sb += f[j] * ss;
            }
            a[k] = sa / (REAL)Mo; bb[k] = sb / (REAL)Mo;
        }
        for (int j = 0; j < Mn; j++) {
            REAL v = a[0];
            for (int k = 1; k < Mo / 2; k++) v += 2 * (a[k] * R_COS(k * beta[j]) + bb[k] * R_SIN(k * beta[j]));
            v += a[Mo / 2] * R_COS((Mo / 2) * beta[j]);
            o[j] = v;
        }
        store_hl(o, ohi + (long)c * Mn, olo ? olo + (long)c * Mn : NULL, Mn);
        free(f); free(a); free(bb); free(o);
    }
    free(beta);
    return ORC_OK;
}

void NAME(set_num_threads)(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
int NAME(num_threads)(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
int NAME(sizeof_real)(void) { return (int)sizeof(REAL); }
