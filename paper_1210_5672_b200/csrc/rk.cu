// rk.cu -- S8/S9: right-hand sides of the free-surface Euler equations (2.1) and of the batched variational
// equation (B.1)-(B.3), (3.32), the 36th-order filter (2.14), and the explicit
// 11-stage order-8 Runge-Kutta stepper (reading R6 of DESIGN.md section 3: the paper cites DOP853 without printing it).
//
//   eta_t   = W0                         phi_t   = P[ v W0 - u^2/2 - v^2/2 - g eta ]
//   deta_t  = w_c - D(u deta_c)          dphi_t  = P[ -D(deta_c u v) - u D(b_c) + v w_c - g deta_c ],  b_c = dphi_c - v deta_c,
//   w_c = G[b_c],  every right-hand side multiplied by the filter, the state filtered after every step (R5).
// One DtN setup (S0-S2), one base state and one batched linearized solve per stage, all through the entry points of api.cu.
// State layout: y = [eta (N) | phi (N) | deta (N x nc) | dphi (N x nc)] = L doubles; double-double states are planar (hi plane of
// L doubles, then lo plane) and run through the kernels of rk_dd.cu.  Product code; shares nothing with oracle/.
#include "common.cuh"
#include "fft.cuh"
#include "rk_dd.cuh"
#include <new>
#include <cstring>

using namespace sww;

#include "rk.cuh"

namespace sww {

// ---- the tableau in double-double: (p + q sqrt 21) / r with small integers p, q, r, by error-free transformations on the host
struct hdd {
    double hi, lo;
};
static hdd h_two_sum(double a, double b) {
    const double s = a + b, bb = s - a;
    return hdd{s, (a - (s - bb)) + (b - bb)};
}
static hdd h_add(hdd a, hdd b) {
    hdd s = h_two_sum(a.hi, b.hi);
    s.lo += a.lo + b.lo;
    return h_two_sum(s.hi, s.lo);
}
static hdd h_mul_d(hdd a, double b) {
    const double p = a.hi * b, e = fma(a.hi, b, -p) + a.lo * b;
    return h_two_sum(p, e);
}
static hdd h_div_d(hdd a, double b) {  // b a small integer
    const double q1 = a.hi / b;
    const double r = fma(-q1, b, a.hi) + a.lo;  // exact remainder of the high word (fma) plus the low word
    return h_two_sum(q1, r / b);
}
static hdd h_sqrt21() {
    const double x = sqrt(21.0);
    const double x2 = x * x, e = fma(x, x, -x2);            // x^2 = x2 + e exactly
    return h_two_sum(x, ((21.0 - x2) - e) / (2.0 * x));      // one Newton step carried in the low word
}
static hdd h_coef(int p, int q, int r) {  // (p + q sqrt 21) / r
    return h_div_d(h_add(hdd{(double)p, 0.0}, h_mul_d(h_sqrt21(), (double)q)), (double)r);
}
static void rk_tableau_dd(double a[RK_S][RK_S], double alo[RK_S][RK_S], double b[RK_S], double blo[RK_S]) {
    memset(a, 0, sizeof(double) * RK_S * RK_S);
    memset(alo, 0, sizeof(double) * RK_S * RK_S);
    memset(b, 0, sizeof(double) * RK_S);
    memset(blo, 0, sizeof(double) * RK_S);
    auto A = [&](int i, int j, int p, int q, int r) {
        const hdd v = h_coef(p, q, r);
        a[i][j] = v.hi;
        alo[i][j] = v.lo;
    };
    auto B = [&](int i, int p, int r) {
        const hdd v = h_coef(p, 0, r);
        b[i] = v.hi;
        blo[i] = v.lo;
    };
    B(0, 1, 20); B(7, 49, 180); B(8, 16, 45); B(9, 49, 180); B(10, 1, 20);
    A(1, 0, 1, 0, 2);
    A(2, 0, 1, 0, 4); A(2, 1, 1, 0, 4);
    A(3, 0, 1, 0, 7); A(3, 1, -7, -3, 98); A(3, 2, 21, 5, 49);
    A(4, 0, 11, 1, 84); A(4, 2, 18, 4, 63); A(4, 3, 21, -1, 252);
    A(5, 0, 5, 1, 48); A(5, 2, 9, 1, 36); A(5, 3, -231, 14, 360); A(5, 4, 63, -7, 80);
    A(6, 0, 10, -1, 42); A(6, 2, -432, 92, 315); A(6, 3, 633, -145, 90); A(6, 4, -504, 115, 70); A(6, 5, 63, -13, 35);
    A(7, 0, 1, 0, 14); A(7, 4, 14, -3, 126); A(7, 5, 13, -3, 63); A(7, 6, 1, 0, 9);
    A(8, 0, 1, 0, 32); A(8, 4, 91, -21, 576); A(8, 5, 11, 0, 72); A(8, 6, -385, -75, 1152); A(8, 7, 63, 13, 128);
    A(9, 0, 1, 0, 14); A(9, 4, 1, 0, 9); A(9, 5, -733, -147, 2205); A(9, 6, 515, 111, 504); A(9, 7, -51, -11, 56); A(9, 8, 132, 28, 245);
    A(10, 4, -42, 7, 18); A(10, 5, -18, 28, 45); A(10, 6, -273, -53, 72); A(10, 7, 301, 53, 72); A(10, 8, 28, -28, 45); A(10, 9, 49, -7, 18);
}

// the tableau of DESIGN.md section 3 (R6): coefficients in Q(sqrt 21), evaluated in double
static void rk_tableau(double a[RK_S][RK_S], double b[RK_S], double c[RK_S]) {
    const double s = sqrt(21.0);
    memset(a, 0, sizeof(double) * RK_S * RK_S);
    memset(b, 0, sizeof(double) * RK_S);
    const double cv[RK_S] = {0.0, 0.5, 0.5, (7 + s) / 14, (7 + s) / 14, 0.5, (7 - s) / 14, (7 - s) / 14, 0.5, (7 + s) / 14, 1.0};
    memcpy(c, cv, sizeof(cv));
    b[0] = 1.0 / 20; b[7] = 49.0 / 180; b[8] = 16.0 / 45; b[9] = 49.0 / 180; b[10] = 1.0 / 20;
    a[1][0] = 0.5;
    a[2][0] = 0.25; a[2][1] = 0.25;
    a[3][0] = 1.0 / 7; a[3][1] = (-7 - 3 * s) / 98; a[3][2] = (21 + 5 * s) / 49;
    a[4][0] = (11 + s) / 84; a[4][2] = (18 + 4 * s) / 63; a[4][3] = (21 - s) / 252;
    a[5][0] = (5 + s) / 48; a[5][2] = (9 + s) / 36; a[5][3] = (-231 + 14 * s) / 360; a[5][4] = (63 - 7 * s) / 80;
    a[6][0] = (10 - s) / 42; a[6][2] = (-432 + 92 * s) / 315; a[6][3] = (633 - 145 * s) / 90; a[6][4] = (-504 + 115 * s) / 70; a[6][5] = (63 - 13 * s) / 35;
    a[7][0] = 1.0 / 14; a[7][4] = (14 - 3 * s) / 126; a[7][5] = (13 - 3 * s) / 63; a[7][6] = 1.0 / 9;
    a[8][0] = 1.0 / 32; a[8][4] = (91 - 21 * s) / 576; a[8][5] = 11.0 / 72; a[8][6] = (-385 - 75 * s) / 1152; a[8][7] = (63 + 13 * s) / 128;
    a[9][0] = 1.0 / 14; a[9][4] = 1.0 / 9; a[9][5] = (-733 - 147 * s) / 2205; a[9][6] = (515 + 111 * s) / 504; a[9][7] = (-51 - 11 * s) / 56; a[9][8] = (132 + 28 * s) / 245;
    a[10][4] = (-42 + 7 * s) / 18; a[10][5] = (-18 + 28 * s) / 45; a[10][6] = (-273 - 53 * s) / 72; a[10][7] = (301 + 53 * s) / 72; a[10][8] = (28 - 28 * s) / 45; a[10][9] = (49 - 7 * s) / 18;
}

// S9: out = y + sum_j coef[j] k_j   (coef = dt a_ij or dt b_j; zero coefficients are skipped on the host side)
struct Comb {
    int n;
    int idx[RK_S];
    double coef[RK_S];
};
__global__ void k_rk_combine(size_t L, const double* __restrict__ y, const double* __restrict__ k, Comb cb, double* __restrict__ out) {
    size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= L) return;
    double s = y[q];
    for (int j = 0; j < cb.n; j++) s = fma(cb.coef[j], k[(size_t)cb.idx[j] * L + q], s);
    out[q] = s;
}

__device__ __forceinline__ int dft_index(int p, int logN) { return (int)(__brev((unsigned)p) >> (32 - logN)); }

// S8, base state: eta_t = F[W0], phi_t = F P[v W0 - u^2/2 - v^2/2 - g eta]   (2.1), one CTA; F = filter (or identity), P = zero mean
__global__ void __launch_bounds__(1024) k_rhs_base(int N, int logN, const double2* __restrict__ tw, const double* __restrict__ filt,
                                                   int filter_on, double g, const double* __restrict__ eta, const double* __restrict__ W0,
                                                   const double* __restrict__ u, const double* __restrict__ v, double* __restrict__ eta_t,
                                                   double* __restrict__ phi_t) {
    extern __shared__ __align__(16) double2 z[];
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const double w = W0[j], uu = u[j], vv = v[j];
        z[j] = make_double2(w, fma(vv, w, -0.5 * uu * uu) - 0.5 * vv * vv - g * eta[j]);
    }
    __syncthreads();
    fft_dif(z, N, tw);
    const double rN = 1.0 / (double)N;
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        const double f = (filter_on ? filt[dft_index(p, logN)] : 1.0) * rN;
        double2 t = z[p];
        t.x *= f;
        t.y = (p == 0) ? 0.0 : t.y * f;  // P: the mean of phi_t is removed (2.2)
        z[p] = t;
    }
    __syncthreads();
    ifft_dit(z, N, tw);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        eta_t[j] = z[j].x;
        phi_t[j] = z[j].y;
    }
}

// S8, variational columns (B.1)-(B.3): one CTA per column pair.  wout = w_c - D(u deta_c) is the linearized DtN (api.cu).
//   deta_t = F[wout] ;  dphi_t = F P[ -D(deta u v) - u D(b) + v w - g deta ],  w = wout + D(u deta),  b = dphi - v deta
__global__ void __launch_bounds__(1024) k_rhs_cols(int N, int logN, const double2* __restrict__ tw, const double* __restrict__ filt,
                                                   int filter_on, double g, int ncols, const double* __restrict__ u, const double* __restrict__ v,
                                                   const double* __restrict__ deta, const double* __restrict__ dphi, const double* __restrict__ wout,
                                                   double* __restrict__ deta_t, double* __restrict__ dphi_t) {
    extern __shared__ __align__(16) double2 z[];
    double2* z2 = z + N;
    const int c0 = 2 * blockIdx.x, c1 = c0 + 1;
    const bool has1 = c1 < ncols;
    const size_t o0 = (size_t)c0 * N, o1 = (size_t)c1 * N;
    const double rN = 1.0 / (double)N;
    auto deriv_inplace = [&]() {  // z <- D z (natural order in and out)
        __syncthreads();
        fft_dif(z, N, tw);
        for (int p = threadIdx.x; p < N; p += blockDim.x) {
            const double k = (double)wavenumber(p, N, logN) * rN;
            const double2 t = z[p];
            z[p] = make_double2(-k * t.y, k * t.x);
        }
        __syncthreads();
        ifft_dit(z, N, tw);
    };
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const double uu = u[j];
        z[j] = make_double2(uu * deta[o0 + j], has1 ? uu * deta[o1 + j] : 0.0);
    }
    deriv_inplace();  // z = D(u deta)
    double2 wv[FFT_MAX_PER_THREAD];
#pragma unroll
    for (int r = 0; r < FFT_MAX_PER_THREAD; r++) {
        const int j = threadIdx.x + r * blockDim.x;
        if (j < N) wv[r] = make_double2(wout[o0 + j] + z[j].x, has1 ? wout[o1 + j] + z[j].y : 0.0);
    }
    __syncthreads();
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const double vv = v[j];
        z[j] = make_double2(fma(-vv, deta[o0 + j], dphi[o0 + j]), has1 ? fma(-vv, deta[o1 + j], dphi[o1 + j]) : 0.0);
    }
    deriv_inplace();  // z = D(b)
#pragma unroll
    for (int r = 0; r < FFT_MAX_PER_THREAD; r++) {
        const int j = threadIdx.x + r * blockDim.x;
        if (j < N) {
            const double uu = u[j], vv = v[j];
            const double2 a3 = z[j];
            const double d0 = deta[o0 + j], d1 = has1 ? deta[o1 + j] : 0.0;
            z[j] = make_double2(fma(vv, wv[r].x, -uu * a3.x) - g * d0, fma(vv, wv[r].y, -uu * a3.y) - g * d1);
        }
    }
    __syncthreads();
    fft_dif(z, N, tw);
    for (int p = threadIdx.x; p < N; p += blockDim.x) z2[p] = z[p];
    __syncthreads();
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const double uv = u[j] * v[j];
        z[j] = make_double2(uv * deta[o0 + j], has1 ? uv * deta[o1 + j] : 0.0);
    }
    __syncthreads();
    fft_dif(z, N, tw);
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        const double k = (double)wavenumber(p, N, logN);
        const double f = (filter_on ? filt[dft_index(p, logN)] : 1.0) * rN;
        const double2 q = z2[p], t = z[p];
        z2[p] = (p == 0) ? make_double2(0.0, 0.0) : make_double2(f * fma(k, t.y, q.x), f * fma(-k, t.x, q.y));  // F P (q^ - i k t^)
    }
    __syncthreads();
    ifft_dit(z2, N, tw);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        dphi_t[o0 + j] = z2[j].x;
        if (has1) dphi_t[o1 + j] = z2[j].y;
        z[j] = make_double2(wout[o0 + j], has1 ? wout[o1 + j] : 0.0);
    }
    __syncthreads();
    fft_dif(z, N, tw);
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        const double f = (filter_on ? filt[dft_index(p, logN)] : 1.0) * rN;
        z[p] = make_double2(f * z[p].x, f * z[p].y);
    }
    __syncthreads();
    ifft_dit(z, N, tw);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        deta_t[o0 + j] = z[j].x;
        if (has1) deta_t[o1 + j] = z[j].y;
    }
}

// Surface tension, base state: phi_t += F P[ sigma D( eta' / sqrt(1 + eta'^2) ) ]   (2.1b); one CTA.
// F and P are linear, so the term is added to the phi_t that k_rhs_base has already filtered and projected.
__global__ void __launch_bounds__(1024) k_st_base(int N, int logN, const double2* __restrict__ tw, const double* __restrict__ filt,
                                                  int filter_on, double sigma, const double* __restrict__ d1, double* __restrict__ phi_t) {
    extern __shared__ __align__(16) double2 z[];
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const double e1 = d1[j];
        z[j] = make_double2(e1 / sqrt(fma(e1, e1, 1.0)), 0.0);
    }
    __syncthreads();
    fft_dif(z, N, tw);
    const double rN = 1.0 / (double)N;
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        const double k = (double)wavenumber(p, N, logN) * (filter_on ? filt[dft_index(p, logN)] : 1.0) * rN;  // k = 0 at p = 0: P
        const double2 t = z[p];
        z[p] = make_double2(-k * t.y, k * t.x);
    }
    __syncthreads();
    ifft_dit(z, N, tw);
    for (int j = threadIdx.x; j < N; j += blockDim.x) phi_t[j] = fma(sigma, z[j].x, phi_t[j]);
}

// Surface tension, variational columns: dphi_t += F P[ sigma D( D(deta_c) / (1 + eta'^2)^(3/2) ) ]   (B.4), PAPER.md:718;
// one CTA per column pair.
__global__ void __launch_bounds__(1024) k_st_cols(int N, int logN, const double2* __restrict__ tw, const double* __restrict__ filt,
                                                  int filter_on, double sigma, int ncols, const double* __restrict__ d1,
                                                  const double* __restrict__ deta, double* __restrict__ dphi_t) {
    extern __shared__ __align__(16) double2 z[];
    const int c0 = 2 * blockIdx.x, c1 = c0 + 1;
    const bool has1 = c1 < ncols;
    const size_t o0 = (size_t)c0 * N, o1 = (size_t)c1 * N;
    const double rN = 1.0 / (double)N;
    for (int j = threadIdx.x; j < N; j += blockDim.x) z[j] = make_double2(deta[o0 + j], has1 ? deta[o1 + j] : 0.0);
    __syncthreads();
    fft_dif(z, N, tw);
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        const double k = (double)wavenumber(p, N, logN) * rN;
        const double2 t = z[p];
        z[p] = make_double2(-k * t.y, k * t.x);
    }
    __syncthreads();
    ifft_dit(z, N, tw);  // D(deta)
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const double e1 = d1[j], den = fma(e1, e1, 1.0), q = 1.0 / (den * sqrt(den));
        z[j] = make_double2(z[j].x * q, z[j].y * q);
    }
    __syncthreads();
    fft_dif(z, N, tw);
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        const double k = (double)wavenumber(p, N, logN) * (filter_on ? filt[dft_index(p, logN)] : 1.0) * rN;
        const double2 t = z[p];
        z[p] = make_double2(-k * t.y, k * t.x);
    }
    __syncthreads();
    ifft_dit(z, N, tw);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        dphi_t[o0 + j] = fma(sigma, z[j].x, dphi_t[o0 + j]);
        if (has1) dphi_t[o1 + j] = fma(sigma, z[j].y, dphi_t[o1 + j]);
    }
}

// ------------------------------------------------------------------------------------------------ refined mesh (mesh.cu)
// On the mesh x = xi(alpha) of (2.10) the stored samples are functions of alpha: d/dx = (1/xi') d/dalpha in every term of (2.1) and
// (B.1)-(B.4), the filter acts on the samples (modes in alpha), and P removes the mean over x,
//     (1/2pi) int f dx = (1/N) sum_j f_j E_j = f^_0 + a1 Re f^_1 + a2 Re f^_2     for E = 1 + a1 cos(alpha) + a2 cos(2 alpha).
// W0, u, v and the linearized DtN output arrive in physical form (ddpath.cu, api.cu divide by xi').  The uniform-mesh kernels
// above fold some of the derivatives into the last transform; here each derivative is taken on its own, then divided by xi'.
//
// z: the spectrum (scaled, bit-reversed order: mode k at position brev(k)) of a packed pair x + i y of real signals.  Returns the
// part a1 Re f^_1 + a2 Re f^_2 of both means: with X_k = (Z_k + conj Z_-k)/2 and Y_k = (Z_k - conj Z_-k)/(2i),
// Re X_k = (Re Z_k + Re Z_-k)/2 and Re Y_k = (Im Z_k + Im Z_-k)/2.
__device__ __forceinline__ double2 mesh_mean_pair(const double2* z, int N, int logN, double a1, double a2) {
    const double2 p1 = z[dft_index(1, logN)], m1 = z[dft_index(N - 1, logN)], p2 = z[dft_index(2, logN)], m2 = z[dft_index(N - 2, logN)];
    return make_double2(0.5 * (a1 * (p1.x + m1.x) + a2 * (p2.x + m2.x)), 0.5 * (a1 * (p1.y + m1.y) + a2 * (p2.y + m2.y)));
}

struct MeshRk {
    const double* xE;  // xi' (hi words)
    double a1, a2;
};

// z <- (1/xi') D z for a packed pair (natural order in and out); every thread of the CTA calls it
__device__ __forceinline__ void mesh_deriv_x(double2* z, int N, int logN, const double2* __restrict__ tw, const double* __restrict__ xE) {
    const double rN = 1.0 / (double)N;
    __syncthreads();
    fft_dif(z, N, tw);
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        const double k = (double)wavenumber(p, N, logN) * rN;
        const double2 t = z[p];
        z[p] = make_double2(-k * t.y, k * t.x);
    }
    __syncthreads();
    ifft_dit(z, N, tw);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const double re = 1.0 / xE[j];
        z[j] = make_double2(z[j].x * re, z[j].y * re);
    }
    __syncthreads();
}
// z <- F z for a packed pair; P (mean over x) on the y part if proj_y, on the x part if proj_x
__device__ __forceinline__ void mesh_filter_project(double2* z, int N, int logN, const double2* __restrict__ tw, const double* __restrict__ filt,
                                                    int filter_on, MeshRk ms, bool proj_x, bool proj_y) {
    const double rN = 1.0 / (double)N;
    __syncthreads();
    fft_dif(z, N, tw);
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        const double f = (filter_on ? filt[dft_index(p, logN)] : 1.0) * rN;
        z[p] = make_double2(f * z[p].x, f * z[p].y);
    }
    __syncthreads();
    if (threadIdx.x == 0 && (proj_x || proj_y)) {
        const double2 m = mesh_mean_pair(z, N, logN, ms.a1, ms.a2);
        if (proj_x) z[0].x = -m.x;   // mean over alpha z[0] minus the mean over x (z[0] + m)
        if (proj_y) z[0].y = -m.y;
    }
    __syncthreads();
    ifft_dit(z, N, tw);
}

// base state on the refined mesh: eta_t = F[W0] ; phi_t = F P[ v W0 - u^2/2 - v^2/2 - g eta + sigma d/dx( eta_x / sqrt(1 + eta_x^2) ) ],
// eta_x = d1 / xi'   (2.1); one CTA
__global__ void __launch_bounds__(1024) k_rhs_base_mesh(int N, int logN, const double2* __restrict__ tw, const double* __restrict__ filt,
                                                        int filter_on, double g, double sigma, MeshRk ms, const double* __restrict__ eta,
                                                        const double* __restrict__ d1, const double* __restrict__ W0, const double* __restrict__ u,
                                                        const double* __restrict__ v, double* __restrict__ eta_t, double* __restrict__ phi_t) {
    extern __shared__ __align__(16) double2 z[];
    double cur[FFT_MAX_PER_THREAD];
#pragma unroll
    for (int r = 0; r < FFT_MAX_PER_THREAD; r++) cur[r] = 0.0;
    if (sigma != 0.0) {
        for (int j = threadIdx.x; j < N; j += blockDim.x) {
            const double e1 = d1[j] / ms.xE[j];
            z[j] = make_double2(e1 / sqrt(fma(e1, e1, 1.0)), 0.0);
        }
        mesh_deriv_x(z, N, logN, tw, ms.xE);
#pragma unroll
        for (int r = 0; r < FFT_MAX_PER_THREAD; r++) {
            const int j = threadIdx.x + r * blockDim.x;
            if (j < N) cur[r] = sigma * z[j].x;
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < FFT_MAX_PER_THREAD; r++) {
        const int j = threadIdx.x + r * blockDim.x;
        if (j < N) {
            const double w = W0[j], uu = u[j], vv = v[j];
            z[j] = make_double2(w, fma(vv, w, -0.5 * uu * uu) - 0.5 * vv * vv - g * eta[j] + cur[r]);
        }
    }
    mesh_filter_project(z, N, logN, tw, filt, filter_on, ms, false, true);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        eta_t[j] = z[j].x;
        phi_t[j] = z[j].y;
    }
}

// variational columns on the refined mesh (B.1)-(B.4), one CTA per column pair; wout = G b - d/dx(u deta) (physical, api.cu):
//   deta_t = F[wout] ;  dphi_t = F P[ -d/dx(deta u v) - u d/dx(b) + v w - g deta + sigma d/dx( d/dx(deta) / (1 + eta_x^2)^(3/2) ) ],
//   w = wout + d/dx(u deta),  b = dphi - v deta
__global__ void __launch_bounds__(1024) k_rhs_cols_mesh(int N, int logN, const double2* __restrict__ tw, const double* __restrict__ filt,
                                                        int filter_on, double g, double sigma, MeshRk ms, int ncols, const double* __restrict__ d1,
                                                        const double* __restrict__ u, const double* __restrict__ v, const double* __restrict__ deta,
                                                        const double* __restrict__ dphi, const double* __restrict__ wout,
                                                        double* __restrict__ deta_t, double* __restrict__ dphi_t) {
    extern __shared__ __align__(16) double2 z[];
    const int c0 = 2 * blockIdx.x, c1 = c0 + 1;
    const bool has1 = c1 < ncols;
    const size_t o0 = (size_t)c0 * N, o1 = (size_t)c1 * N;
    double2 acc[FFT_MAX_PER_THREAD];
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const double uu = u[j];
        z[j] = make_double2(uu * deta[o0 + j], has1 ? uu * deta[o1 + j] : 0.0);
    }
    mesh_deriv_x(z, N, logN, tw, ms.xE);  // d/dx(u deta)
#pragma unroll
    for (int r = 0; r < FFT_MAX_PER_THREAD; r++) {
        const int j = threadIdx.x + r * blockDim.x;
        if (j < N) {
            const double vv = v[j];
            acc[r] = make_double2(vv * (wout[o0 + j] + z[j].x) - g * deta[o0 + j], has1 ? vv * (wout[o1 + j] + z[j].y) - g * deta[o1 + j] : 0.0);  // v w - g deta
        }
    }
    __syncthreads();
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const double vv = v[j];
        z[j] = make_double2(fma(-vv, deta[o0 + j], dphi[o0 + j]), has1 ? fma(-vv, deta[o1 + j], dphi[o1 + j]) : 0.0);
    }
    mesh_deriv_x(z, N, logN, tw, ms.xE);  // d/dx(b)
#pragma unroll
    for (int r = 0; r < FFT_MAX_PER_THREAD; r++) {
        const int j = threadIdx.x + r * blockDim.x;
        if (j < N) {
            const double uu = u[j];
            acc[r].x = fma(-uu, z[j].x, acc[r].x);
            acc[r].y = fma(-uu, z[j].y, acc[r].y);
        }
    }
    __syncthreads();
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const double uv = u[j] * v[j];
        z[j] = make_double2(uv * deta[o0 + j], has1 ? uv * deta[o1 + j] : 0.0);
    }
    mesh_deriv_x(z, N, logN, tw, ms.xE);  // d/dx(deta u v)
#pragma unroll
    for (int r = 0; r < FFT_MAX_PER_THREAD; r++) {
        const int j = threadIdx.x + r * blockDim.x;
        if (j < N) {
            acc[r].x -= z[j].x;
            acc[r].y -= z[j].y;
        }
    }
    __syncthreads();
    if (sigma != 0.0) {
        for (int j = threadIdx.x; j < N; j += blockDim.x) z[j] = make_double2(deta[o0 + j], has1 ? deta[o1 + j] : 0.0);
        mesh_deriv_x(z, N, logN, tw, ms.xE);
        for (int j = threadIdx.x; j < N; j += blockDim.x) {
            const double e1 = d1[j] / ms.xE[j], den = fma(e1, e1, 1.0), q = 1.0 / (den * sqrt(den));
            z[j] = make_double2(z[j].x * q, z[j].y * q);
        }
        mesh_deriv_x(z, N, logN, tw, ms.xE);
#pragma unroll
        for (int r = 0; r < FFT_MAX_PER_THREAD; r++) {
            const int j = threadIdx.x + r * blockDim.x;
            if (j < N) {
                acc[r].x = fma(sigma, z[j].x, acc[r].x);
                acc[r].y = fma(sigma, z[j].y, acc[r].y);
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < FFT_MAX_PER_THREAD; r++) {
        const int j = threadIdx.x + r * blockDim.x;
        if (j < N) z[j] = acc[r];
    }
    mesh_filter_project(z, N, logN, tw, filt, filter_on, ms, true, true);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        dphi_t[o0 + j] = z[j].x;
        if (has1) dphi_t[o1 + j] = z[j].y;
    }
    __syncthreads();
    for (int j = threadIdx.x; j < N; j += blockDim.x) z[j] = make_double2(wout[o0 + j], has1 ? wout[o1 + j] : 0.0);
    mesh_filter_project(z, N, logN, tw, filt, filter_on, ms, false, false);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        deta_t[o0 + j] = z[j].x;
        if (has1) deta_t[o1 + j] = z[j].y;
    }
}

// the filter (2.14) applied in place to ncols columns (the state after every step)
__global__ void __launch_bounds__(1024) k_filter_cols(int N, int logN, const double2* __restrict__ tw, const double* __restrict__ filt,
                                                      int ncols, double* __restrict__ y) {
    extern __shared__ __align__(16) double2 z[];
    const int c0 = 2 * blockIdx.x, c1 = c0 + 1;
    const bool has1 = c1 < ncols;
    const size_t o0 = (size_t)c0 * N, o1 = (size_t)c1 * N;
    for (int j = threadIdx.x; j < N; j += blockDim.x) z[j] = make_double2(y[o0 + j], has1 ? y[o1 + j] : 0.0);
    __syncthreads();
    fft_dif(z, N, tw);
    const double rN = 1.0 / (double)N;
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        const double f = filt[dft_index(p, logN)] * rN;
        z[p] = make_double2(f * z[p].x, f * z[p].y);
    }
    __syncthreads();
    ifft_dit(z, N, tw);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        y[o0 + j] = z[j].x;
        if (has1) y[o1 + j] = z[j].y;
    }
}

// E = (pi/N) sum_j [ phi_j (G phi)_j + g eta_j^2 ], one CTA, pairwise tree in shared memory
// xE (refined mesh, else nullptr): dx = xi' dalpha
__global__ void __launch_bounds__(256) k_energy(int N, double g, const double* __restrict__ eta, const double* __restrict__ phi,
                                                const double* __restrict__ W0, const double* __restrict__ xE, double* __restrict__ out) {
    __shared__ double s[256];
    double a = 0.0;
    for (int j = threadIdx.x; j < N; j += 256) a += fma(phi[j], W0[j], g * eta[j] * eta[j]) * (xE ? xE[j] : 1.0);
    s[threadIdx.x] = a;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) s[threadIdx.x] += s[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) out[0] = s[0] * 3.14159265358979323846 / (double)N;
}

}  // namespace sww

namespace sww {

static int rk_set_attrs() {
    static DeviceOnce done;
    if (done.first()) {
        SWW_CUDA(cudaFuncSetAttribute(k_rhs_base, cudaFuncAttributeMaxDynamicSharedMemorySize, 8192 * 16));
        SWW_CUDA(cudaFuncSetAttribute(k_rhs_cols, cudaFuncAttributeMaxDynamicSharedMemorySize, 4096 * 32));
        SWW_CUDA(cudaFuncSetAttribute(k_filter_cols, cudaFuncAttributeMaxDynamicSharedMemorySize, 8192 * 16));
        SWW_CUDA(cudaFuncSetAttribute(k_st_base, cudaFuncAttributeMaxDynamicSharedMemorySize, 8192 * 16));
        SWW_CUDA(cudaFuncSetAttribute(k_st_cols, cudaFuncAttributeMaxDynamicSharedMemorySize, 8192 * 16));
        SWW_CUDA(cudaFuncSetAttribute(k_rhs_base_mesh, cudaFuncAttributeMaxDynamicSharedMemorySize, 8192 * 16));
        SWW_CUDA(cudaFuncSetAttribute(k_rhs_cols_mesh, cudaFuncAttributeMaxDynamicSharedMemorySize, 8192 * 16));
    }
    return SWW_OK;
}

// one evaluation of the right-hand sides at the stage state ys -> kout (same layout as the state)
static int rk_rhs_dd(sww_state_s* s, const double* ys, double* kout) {
    const int N = s->N, nc = s->nc;
    const size_t L = s->L;
    sww_dtn_s* d = s->dtn;
    SWW_TRY(ensure_workspace(d, nc > 0 ? nc : 1));
    SWW_TRY(setup_surface(d, ys, ys + L));          // S0-S2 for this stage's surface (eta: high and low planes)
    SWW_TRY(accurate_base(d, ys + N, L));           // W0 = G phi, u, v of (2.9)
    d->has_base = true;
    const bool st_apart = s->sigma != 0.0 && !d->mesh_on;  // on a refined mesh the surface-tension terms are inside the mesh kernels
    SWW_TRY(rkdd_rhs_base(d, s->filter, s->g, s->sigma, L, ys, kout));
    if (st_apart) SWW_TRY(rkdd_st_base(d, s->filter, s->sigma, L, kout));
    if (nc > 0) {
        const double* deta = ys + 2 * (size_t)N;
        const double* dphi = deta + (size_t)N * nc;
        SWW_TRY(dd_linearized(d, deta, dphi, nc, s->w, L, 0));   // w_c - D(u deta_c)   (B.1d), (B.2)
        SWW_TRY(rkdd_rhs_cols(d, s->filter, s->g, s->sigma, nc, L, ys, s->w, kout));
        if (st_apart) SWW_TRY(rkdd_st_cols(d, s->filter, s->sigma, nc, L, ys, kout));
    }
    return SWW_OK;
}

int rk_rhs(sww_state_s* s, const double* ys, double* kout) {
    if (s->prec == SWW_DD) return rk_rhs_dd(s, ys, kout);
    const int N = s->N, nc = s->nc, logN = fft_ilog2(N), thr = fft_threads(N);
    sww_dtn_s* d = s->dtn;
    cudaStream_t st = s->stream;
    const double* eta = ys;
    const double* phi = ys + N;
    SWW_TRY(sww_dtn_refactor(d, eta));   // S0-S2 for this stage's surface
    if (nc == 0 && N <= 1024 && d->prec == SWW_F64) {  // nothing is linearized about this state: the plain fp64 base state (ddpath.cu)
        SWW_TRY(ensure_workspace(d, 1));
        SWW_TRY(fast_base_f64(d, phi));
        d->has_base = true;
    } else {
        SWW_TRY(sww_dtn_set_base(d, phi));   // W0 = G phi, u, v of (2.9)
    }
    const Tables* t = d->tab;
    if (d->mesh_on) {  // the refined mesh (2.10): kernels with d/dx = (1/xi') d/dalpha and the mean over x
        const MeshRk ms{d->mesh.xE, d->mesh_a1, d->mesh_a2};
        SWW_BEGIN(KC_FFT, st);
        k_rhs_base_mesh<<<1, thr, sizeof(double2) * (size_t)N, st>>>(N, logN, t->tw, t->filt, s->filter ? 1 : 0, s->g, s->sigma, ms, eta, d->d1,
                                                                       d->bW0, d->bu, d->bv, kout, kout + N);
        SWW_LAUNCHED();
        SWW_CUDA(cudaGetLastError());
        if (nc > 0) {
            const double* deta = ys + 2 * (size_t)N;
            const double* dphi = deta + (size_t)N * nc;
            SWW_TRY(sww_dtn_linearized_apply(d, deta, dphi, nc, s->w));  // G b - d/dx(u deta_c)   (B.1d), (B.2)
            SWW_BEGIN(KC_FFT, st);
            k_rhs_cols_mesh<<<(nc + 1) / 2, thr, sizeof(double2) * (size_t)N, st>>>(N, logN, t->tw, t->filt, s->filter ? 1 : 0, s->g, s->sigma, ms, nc,
                                                                                    d->d1, d->bu, d->bv, deta, dphi, s->w, kout + 2 * (size_t)N,
                                                                                    kout + 2 * (size_t)N + (size_t)N * nc);
            SWW_LAUNCHED();
            SWW_CUDA(cudaGetLastError());
        }
        return SWW_OK;
    }
    SWW_BEGIN(KC_FFT, st);
    k_rhs_base<<<1, thr, sizeof(double2) * (size_t)N, st>>>(N, logN, t->tw, t->filt, s->filter ? 1 : 0, s->g, eta, d->bW0, d->bu, d->bv, kout,
                                                              kout + N);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    if (s->sigma != 0.0) {
        SWW_BEGIN(KC_FFT, st);
        k_st_base<<<1, thr, sizeof(double2) * (size_t)N, st>>>(N, logN, t->tw, t->filt, s->filter ? 1 : 0, s->sigma, d->d1, kout + N);
        SWW_LAUNCHED();
        SWW_CUDA(cudaGetLastError());
    }
    if (nc > 0) {
        const double* deta = ys + 2 * (size_t)N;
        const double* dphi = deta + (size_t)N * nc;
        SWW_TRY(sww_dtn_linearized_apply(d, deta, dphi, nc, s->w));  // w_c - D(u deta_c)   (B.1d), (B.2)
        SWW_BEGIN(KC_FFT, st);
        k_rhs_cols<<<(nc + 1) / 2, thr, sizeof(double2) * 2 * (size_t)N, st>>>(N, logN, t->tw, t->filt, s->filter ? 1 : 0, s->g, nc, d->bu, d->bv,
                                                                                deta, dphi, s->w, kout + 2 * (size_t)N,
                                                                                kout + 2 * (size_t)N + (size_t)N * nc);
        SWW_LAUNCHED();
        SWW_CUDA(cudaGetLastError());
        if (s->sigma != 0.0) {
            SWW_BEGIN(KC_FFT, st);
            k_st_cols<<<(nc + 1) / 2, thr, sizeof(double2) * (size_t)N, st>>>(N, logN, t->tw, t->filt, s->filter ? 1 : 0, s->sigma, nc, d->d1, deta,
                                                                              kout + 2 * (size_t)N + (size_t)N * nc);
            SWW_LAUNCHED();
            SWW_CUDA(cudaGetLastError());
        }
    }
    return SWW_OK;
}

// out = base + dt sum_j coef_j kbuf[j]   (kbuf: n state vectors, slot j at j L mul)
static int rk_combine_ex(sww_state_s* s, const double* base, const double* kbuf, const double* coef, const double* coef_lo, int n, double dt,
                         double* out);
static int rk_combine(sww_state_s* s, const double* coef, const double* coef_lo, int n, double dt, double* out) {
    return rk_combine_ex(s, s->y, s->k, coef, coef_lo, n, dt, out);
}
static int rk_combine_ex(sww_state_s* s, const double* base, const double* kbuf, const double* coef, const double* coef_lo, int n, double dt,
                         double* out) {
    if (s->prec == SWW_DD) {
        CombDD cd;
        cd.n = 0;
        for (int j = 0; j < n; j++)
            if (coef[j] != 0.0) {
                const hdd v = h_mul_d(hdd{coef[j], coef_lo[j]}, dt);
                cd.idx[cd.n] = j;
                cd.chi[cd.n] = v.hi;
                cd.clo[cd.n] = v.lo;
                cd.n++;
            }
        return rkdd_combine(s->stream, s->L, base, kbuf, cd, out);
    }
    Comb cb;
    cb.n = 0;
    for (int j = 0; j < n; j++)
        if (coef[j] != 0.0) {
            cb.idx[cb.n] = j;
            cb.coef[cb.n] = dt * coef[j];
            cb.n++;
        }
    SWW_BEGIN(KC_OTHER, s->stream);
    k_rk_combine<<<(unsigned)((s->L + 255) / 256), 256, 0, s->stream>>>(s->L, base, kbuf, cb, out);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

}  // namespace sww

extern "C" {

int sww_state_create(int N, double h, double g, int prec, int ncols, const void* eta, const void* phi, const void* deta,
                     const void* dphi, unsigned flags, void* stream, sww_state_t* out) {
    if (!out || !eta || !phi || ncols < 0 || (ncols > 0 && (!deta || !dphi))) return SWW_EINVAL;
    if (prec != SWW_F64 && prec != SWW_DD) return SWW_EINVAL;
    // k_rhs_cols / k_rhs_cols_dd keep two N-point complex arrays in shared memory (include/sww.h states the limits)
    if (N > (prec == SWW_DD ? RKDD_MAX_N : 4096)) return SWW_EINVAL;
    sww_state_s* s = new (std::nothrow) sww_state_s();
    if (!s) return SWW_ENOMEM;
    memset(s, 0, sizeof(*s));
    s->N = N; s->nc = ncols; s->prec = prec; s->h = h; s->g = g;
    s->filter = !(flags & 1u);
    s->stream = (cudaStream_t)stream;
    s->L = 2 * (size_t)N * (1 + (size_t)ncols);
    rk_tableau(s->a, s->b, s->c);
    if (prec == SWW_DD) rk_tableau_dd(s->a, s->alo, s->b, s->blo);
    int rc = sww_dtn_setup(eta, N, h, prec, stream, &s->dtn);  // validates N, h; also the first factorisation
    if (rc) { delete s; return rc; }
    const size_t mul = s->mul();
    bool ok = cudaMalloc(&s->y, sizeof(double) * s->L * mul) == cudaSuccess && cudaMalloc(&s->ys, sizeof(double) * s->L * mul) == cudaSuccess &&
              cudaMalloc(&s->k, sizeof(double) * s->L * mul * RK_S) == cudaSuccess &&
              cudaMalloc(&s->w, sizeof(double) * mul * (size_t)N * (ncols > 0 ? ncols : 1)) == cudaSuccess &&
              cudaMalloc(&s->red, 2 * sizeof(double)) == cudaSuccess;
    if (!ok) { sww_state_destroy(s); return SWW_ENOMEM; }
    const size_t v = sizeof(double) * N, bsz = v * ncols;
    cudaStream_t st = s->stream;
    // double-double inputs are planar per array (hi block, lo block); the state keeps one hi plane and one lo plane of L doubles
    for (size_t pl = 0; pl < mul; pl++) {
        double* y = s->y + pl * s->L;
        const double *e = (const double*)eta + pl * N, *p = (const double*)phi + pl * N;
        const double *de = ncols ? (const double*)deta + pl * (size_t)N * ncols : nullptr, *dp = ncols ? (const double*)dphi + pl * (size_t)N * ncols : nullptr;
        if (cudaMemcpyAsync(y, e, v, cudaMemcpyDeviceToDevice, st) || cudaMemcpyAsync(y + N, p, v, cudaMemcpyDeviceToDevice, st) ||
            (ncols && (cudaMemcpyAsync(y + 2 * (size_t)N, de, bsz, cudaMemcpyDeviceToDevice, st) ||
                       cudaMemcpyAsync(y + 2 * (size_t)N + (size_t)N * ncols, dp, bsz, cudaMemcpyDeviceToDevice, st)))) {
            sww_state_destroy(s);
            return SWW_ECUDA;
        }
    }
    rc = rk_set_attrs();
    if (!rc && prec == SWW_DD) rc = rkdd_set_attrs();
    if (rc) { sww_state_destroy(s); return rc; }
    *out = s;
    return SWW_OK;
}

int sww_state_set_sigma(sww_state_t s, double sigma) {
    if (!s || !(sigma >= 0.0)) return SWW_EINVAL;
    s->sigma = sigma;
    return SWW_OK;
}

int sww_rk_advance(sww_state_t s, double dt, int nsteps) {
    if (!s || nsteps < 0) return SWW_EINVAL;
    const int N = s->N, logN = fft_ilog2(N);
    for (int n = 0; n < nsteps; n++) {
        for (int i = 0; i < RK_S; i++) {
            const double* ys = s->y;
            if (i > 0) {
                SWW_TRY(rk_combine(s, s->a[i], s->alo[i], i, dt, s->ys));
                ys = s->ys;
            }
            if (s->tape && s->prec == SWW_F64) {
                if (n >= s->tape_steps) return SWW_EINVAL;
                SWW_CUDA(cudaMemcpyAsync(s->tape + ((size_t)n * RK_S + i) * 2 * N, ys, sizeof(double) * 2 * N, cudaMemcpyDeviceToDevice, s->stream));
            }
            SWW_TRY(rk_rhs(s, ys, s->k + (size_t)i * s->L * s->mul()));
        }
        SWW_TRY(rk_combine(s, s->b, s->blo, RK_S, dt, s->y));
        if (s->filter && s->prec == SWW_DD) {
            SWW_TRY(rkdd_filter_state(s->dtn, 2 + 2 * s->nc, s->L, s->y));
        } else if (s->filter) {
            const int ncol = 2 + 2 * s->nc;
            SWW_BEGIN(KC_FFT, s->stream);
            k_filter_cols<<<(ncol + 1) / 2, fft_threads(N), sizeof(double2) * (size_t)N, s->stream>>>(N, logN, s->dtn->tab->tw, s->dtn->tab->filt,
                                                                                                       ncol, s->y);
            SWW_LAUNCHED();
            SWW_CUDA(cudaGetLastError());
        }
        s->t += dt;
    }
    return SWW_OK;
}

// ---- SDC15 (R15): 8 Radau IIa nodes, RK4 predictor from node to node, 10 Picard sweeps
// Y_m <- y_n + h sum_j S_mj F(Y_j), final quadrature y_{n+1} = y_n + h sum_j b_j F(Y_j); every F is one rk_rhs (setup + batched
// linearized DtN), 113 per step.  The tables come from sdc_tables.cpp (host, __float128) as double-double pairs; the fp64 stepper
// uses their high words.  Work space: slots F[8], Fnew[8], K1..K4, Ya, Yb.
constexpr int SDC_S = 8, SDC_SWEEPS = 10, SDC_SLOTS = 2 * SDC_S + 6;

int sww_sdc_advance(sww_state_t s, double dt, int nsteps) {
    if (!s || nsteps < 0) return SWW_EINVAL;
    static double c_hi[SDC_S], c_lo[SDC_S], dc_hi[SDC_S], dc_lo[SDC_S], S_hi[SDC_S * SDC_S], S_lo[SDC_S * SDC_S];
    static bool have = false;
    if (!have) {
        if (sdc_tables_host(SDC_S, c_hi, c_lo, dc_hi, dc_lo, S_hi, S_lo)) return SWW_EINVAL;
        have = true;
    }
    const size_t Lm = s->L * s->mul();
    if (!s->sdc && cudaMalloc(&s->sdc, sizeof(double) * Lm * SDC_SLOTS) != cudaSuccess) return SWW_ENOMEM;
    double* F = s->sdc;                       // F(Y_m) of the previous sweep, m = 1..8
    double* Fn = F + Lm * SDC_S;              // ... of the sweep being formed
    double* K = Fn + Lm * SDC_S;              // K1..K4 of the predictor (contiguous: slots 0..3 of one combination)
    double* Ya = K + Lm * 4;
    double* Yb = Ya + Lm;
    const int N = s->N, logN = fft_ilog2(N);
    const bool isdd = s->prec == SWW_DD;
    for (int n = 0; n < nsteps; n++) {
        // predictor
        const double* prev = s->y;
        for (int m = 0; m < SDC_S; m++) {
            double* Ym = (m & 1) ? Yb : Ya;
            if (m == 0) SWW_TRY(rk_rhs(s, s->y, K));
            else SWW_CUDA(cudaMemcpyAsync(K, F + Lm * (m - 1), sizeof(double) * Lm, cudaMemcpyDeviceToDevice, s->stream));
            const hdd d = hdd{dc_hi[m], isdd ? dc_lo[m] : 0.0}, dh = h_mul_d(d, 0.5), d6 = h_div_d(d, 6.0), d3 = h_div_d(d, 3.0);
            double ch[4], cl[4];
            ch[0] = dh.hi; cl[0] = dh.lo;
            SWW_TRY(rk_combine_ex(s, prev, K, ch, cl, 1, dt, s->ys));             // prev + hm/2 K1
            SWW_TRY(rk_rhs(s, s->ys, K + Lm));
            ch[0] = 0.0; cl[0] = 0.0; ch[1] = dh.hi; cl[1] = dh.lo;
            SWW_TRY(rk_combine_ex(s, prev, K, ch, cl, 2, dt, s->ys));             // prev + hm/2 K2
            SWW_TRY(rk_rhs(s, s->ys, K + 2 * Lm));
            ch[1] = 0.0; cl[1] = 0.0; ch[2] = d.hi; cl[2] = d.lo;
            SWW_TRY(rk_combine_ex(s, prev, K, ch, cl, 3, dt, s->ys));             // prev + hm K3
            SWW_TRY(rk_rhs(s, s->ys, K + 3 * Lm));
            ch[0] = d6.hi; cl[0] = d6.lo; ch[1] = d3.hi; cl[1] = d3.lo; ch[2] = d3.hi; cl[2] = d3.lo; ch[3] = d6.hi; cl[3] = d6.lo;
            SWW_TRY(rk_combine_ex(s, prev, K, ch, cl, 4, dt, Ym));                // Y_m
            SWW_TRY(rk_rhs(s, Ym, F + Lm * m));
            prev = Ym;
        }
        // Picard sweeps
        for (int sw = 0; sw < SDC_SWEEPS; sw++) {
            for (int m = 0; m < SDC_S; m++) {
                SWW_TRY(rk_combine_ex(s, s->y, F, S_hi + m * SDC_S, S_lo + m * SDC_S, SDC_S, dt, s->ys));
                SWW_TRY(rk_rhs(s, s->ys, Fn + Lm * m));
            }
            double* t = F; F = Fn; Fn = t;
        }
        SWW_TRY(rk_combine_ex(s, s->y, F, S_hi + (SDC_S - 1) * SDC_S, S_lo + (SDC_S - 1) * SDC_S, SDC_S, dt, s->ys));
        SWW_CUDA(cudaMemcpyAsync(s->y, s->ys, sizeof(double) * Lm, cudaMemcpyDeviceToDevice, s->stream));
        if (s->filter && isdd) {
            SWW_TRY(rkdd_filter_state(s->dtn, 2 + 2 * s->nc, s->L, s->y));
        } else if (s->filter) {
            const int ncol = 2 + 2 * s->nc;
            SWW_BEGIN(KC_FFT, s->stream);
            k_filter_cols<<<(ncol + 1) / 2, fft_threads(N), sizeof(double2) * (size_t)N, s->stream>>>(N, logN, s->dtn->tab->tw, s->dtn->tab->filt,
                                                                                                       ncol, s->y);
            SWW_LAUNCHED();
            SWW_CUDA(cudaGetLastError());
        }
        s->t += dt;
    }
    return SWW_OK;
}

int sww_state_read(sww_state_t s, void* eta, void* phi, void* deta, void* dphi, double* t) {
    if (!s) return SWW_EINVAL;
    const size_t v = sizeof(double) * s->N, bsz = v * s->nc;
    cudaStream_t st = s->stream;
    for (size_t pl = 0; pl < s->mul(); pl++) {  // double-double: each output is planar (hi block, lo block)
        const double* y = s->y + pl * s->L;
        if (eta) SWW_CUDA(cudaMemcpyAsync((double*)eta + pl * s->N, y, v, cudaMemcpyDeviceToDevice, st));
        if (phi) SWW_CUDA(cudaMemcpyAsync((double*)phi + pl * s->N, y + s->N, v, cudaMemcpyDeviceToDevice, st));
        if (deta && s->nc) SWW_CUDA(cudaMemcpyAsync((double*)deta + pl * (size_t)s->N * s->nc, y + 2 * (size_t)s->N, bsz, cudaMemcpyDeviceToDevice, st));
        if (dphi && s->nc)
            SWW_CUDA(cudaMemcpyAsync((double*)dphi + pl * (size_t)s->N * s->nc, y + 2 * (size_t)s->N + (size_t)s->N * s->nc, bsz, cudaMemcpyDeviceToDevice, st));
    }
    if (t) *t = s->t;
    return sww_dtn_status(s->dtn);  // synchronises the stream
}

int sww_state_energy(sww_state_t s, double* energy_hl) {
    if (!s || !energy_hl) return SWW_EINVAL;
    sww_dtn_s* d = s->dtn;
    if (s->prec == SWW_DD) {
        SWW_TRY(ensure_workspace(d, 1));
        SWW_TRY(setup_surface(d, s->y, s->y + s->L));
        SWW_TRY(accurate_base(d, s->y + s->N, s->L));
        d->has_base = true;
        SWW_TRY(rkdd_energy(d, s->g, s->L, s->y, s->red));
        SWW_CUDA(cudaMemcpyAsync(energy_hl, s->red, 2 * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
        return sww_dtn_status(d);
    }
    SWW_TRY(sww_dtn_refactor(d, s->y));
    SWW_TRY(sww_dtn_set_base(d, s->y + s->N));
    SWW_BEGIN(KC_OTHER, s->stream);
    k_energy<<<1, 256, 0, s->stream>>>(s->N, s->g, s->y, s->y + s->N, d->bW0, d->mesh_on ? d->mesh.xE : nullptr, s->red);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    SWW_CUDA(cudaMemcpyAsync(energy_hl, s->red, sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    energy_hl[1] = 0.0;
    return sww_dtn_status(d);
}

int sww_state_destroy(sww_state_t s) {
    if (!s) return SWW_EINVAL;
    if (s->dtn) sww_dtn_destroy(s->dtn);
    cudaFree(s->y); cudaFree(s->ys); cudaFree(s->k); cudaFree(s->w); cudaFree(s->red); cudaFree(s->sdc); cudaFree(s->rsp_R);
    delete s;
    return SWW_OK;
}

}  // extern "C"
