// rk_dd.cu -- the double-double instances of S8/S9: right-hand sides of (2.1) and of the variational equation
// (B.1)-(B.3), (3.32), the filter (2.14), the stage combination and the energy
// (PAPER.md:501), all in error-free-transformation arithmetic on the CUDA cores with double-double FFTs in shared memory --
// the paper's quadruple-precision time stepping.  Same formulas and the same order as rk.cu.
// State layout: planar, hi plane of L = 2 N (1 + nc) doubles then lo plane; within a plane [eta | phi | deta (N x nc) | dphi].
// Product code; shares nothing with oracle/.
#include "common.cuh"
#include "dd.cuh"
#include "ddfft.cuh"
#include "rk_dd.cuh"

namespace sww {

constexpr int DDF_MAX_PER_THREAD = 4;  // ceil(N / blockDim.x): 2 up to N = 1024 (N/2 threads), 4 at N = 2048 (512 threads)

__device__ __forceinline__ int dft_index_dd(int p, int logN) { return (int)(__brev((unsigned)p) >> (32 - logN)); }
__device__ __forceinline__ dd ldp(const double* p, size_t plane, size_t o) { return dd{p[o], p[plane + o]}; }
__device__ __forceinline__ void stp(double* p, size_t plane, size_t o, dd v) {
    p[o] = v.hi;
    p[plane + o] = v.lo;
}

// S9: out = y + sum_j coef_j k_j, coefficients dt a_ij (or dt b_j) as double-double pairs
__global__ void k_rk_combine_dd(size_t L, const double* __restrict__ y, const double* __restrict__ k, CombDD cb, double* __restrict__ out) {
    size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= L) return;
    dd s = ldp(y, L, q);
    for (int j = 0; j < cb.n; j++) {
        const double* kj = k + (size_t)cb.idx[j] * 2 * L;
        s = dd_fma(dd{cb.chi[j], cb.clo[j]}, ldp(kj, L, q), s);
    }
    stp(out, L, q, s);
}

// S8, base state: eta_t = F[W0], phi_t = F P[v W0 - u^2/2 - v^2/2 - g eta]   (2.1); one CTA
__global__ void __launch_bounds__(512) k_rhs_base_dd(int N, int logN, const double* __restrict__ cs, const double* __restrict__ sn,
                                                     const double* __restrict__ filt, int filter_on, double g, size_t L,
                                                     const double* __restrict__ eta /* planes L apart */, const double* __restrict__ W0,
                                                     const double* __restrict__ u, const double* __restrict__ v /* planes N apart */,
                                                     double* __restrict__ eta_t, double* __restrict__ phi_t /* planes L apart */) {
    extern __shared__ __align__(16) unsigned char rkdd_sm[];
    cdd* z = reinterpret_cast<cdd*>(rkdd_sm);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const dd w = ldp(W0, N, j), uu = ldp(u, N, j), vv = ldp(v, N, j), e = ldp(eta, L, j);
        dd r = dd_sub(dd_mul(vv, w), dd_half(dd_sqr(uu)));
        r = dd_sub(r, dd_half(dd_sqr(vv)));
        r = dd_sub(r, dd_mul_d(e, g));
        z[j] = cdd{w, r};
    }
    __syncthreads();
    fft_dif_dd(z, N, cs, sn);
    const double rN = 1.0 / (double)N;
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        dd f = filter_on ? ldp(filt, N, dft_index_dd(p, logN)) : dd{1.0, 0.0};
        f = dd_mul_d(f, rN);  // exact: a power of two
        cdd t = z[p];
        t.re = dd_mul(t.re, f);
        t.im = (p == 0) ? dd{0.0, 0.0} : dd_mul(t.im, f);  // P: the mean of phi_t is removed (2.2)
        z[p] = t;
    }
    __syncthreads();
    ifft_dit_dd(z, N, cs, sn);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        stp(eta_t, L, j, z[j].re);
        stp(phi_t, L, j, z[j].im);
    }
}

// S8, variational columns (B.1)-(B.3): one CTA per column pair.  wout = w_c - D(u deta_c) is the linearized DtN.
//   deta_t = F[wout] ;  dphi_t = F P[ -D(deta u v) - u D(b) + v w - g deta ],  w = wout + D(u deta),  b = dphi - v deta
__global__ void __launch_bounds__(512) k_rhs_cols_dd(int N, int logN, const double* __restrict__ cs, const double* __restrict__ sn,
                                                     const double* __restrict__ filt, int filter_on, double g, int ncols, size_t L,
                                                     size_t Lw, const double* __restrict__ u, const double* __restrict__ v,
                                                     const double* __restrict__ deta, const double* __restrict__ dphi /* planes L apart */,
                                                     const double* __restrict__ wout /* planes Lw apart */, double* __restrict__ deta_t,
                                                     double* __restrict__ dphi_t /* planes L apart */) {
    extern __shared__ __align__(16) unsigned char rkdd_sm[];
    cdd* z = reinterpret_cast<cdd*>(rkdd_sm);
    cdd* z2 = z + N;
    const int c0 = 2 * blockIdx.x, c1 = c0 + 1;
    const bool has1 = c1 < ncols;
    const size_t o0 = (size_t)c0 * N, o1 = (size_t)c1 * N;
    const double rN = 1.0 / (double)N;
    const dd zero{0.0, 0.0};
    auto deriv_inplace = [&]() {  // z <- D z (natural order in and out)
        __syncthreads();
        fft_dif_dd(z, N, cs, sn);
        for (int p = threadIdx.x; p < N; p += blockDim.x) {
            const double k = (double)wavenumber_dd(p, N, logN) * rN;
            const cdd t = z[p];
            z[p] = cdd{dd_mul_d(t.im, -k), dd_mul_d(t.re, k)};
        }
        __syncthreads();
        ifft_dit_dd(z, N, cs, sn);
    };
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const dd uu = ldp(u, N, j);
        z[j] = cdd{dd_mul(uu, ldp(deta, L, o0 + j)), has1 ? dd_mul(uu, ldp(deta, L, o1 + j)) : zero};
    }
    deriv_inplace();  // z = D(u deta)
    cdd wv[DDF_MAX_PER_THREAD];
#pragma unroll
    for (int r = 0; r < DDF_MAX_PER_THREAD; r++) {
        const int j = threadIdx.x + r * blockDim.x;
        if (j < N) wv[r] = cdd{dd_add(ldp(wout, Lw, o0 + j), z[j].re), has1 ? dd_add(ldp(wout, Lw, o1 + j), z[j].im) : zero};
    }
    __syncthreads();
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const dd vv = ldp(v, N, j);
        z[j] = cdd{dd_sub(ldp(dphi, L, o0 + j), dd_mul(vv, ldp(deta, L, o0 + j))),
                   has1 ? dd_sub(ldp(dphi, L, o1 + j), dd_mul(vv, ldp(deta, L, o1 + j))) : zero};
    }
    deriv_inplace();  // z = D(b)
#pragma unroll
    for (int r = 0; r < DDF_MAX_PER_THREAD; r++) {
        const int j = threadIdx.x + r * blockDim.x;
        if (j < N) {
            const dd uu = ldp(u, N, j), vv = ldp(v, N, j);
            const cdd a3 = z[j];
            const dd d0 = ldp(deta, L, o0 + j), d1 = has1 ? ldp(deta, L, o1 + j) : zero;
            z[j] = cdd{dd_sub(dd_sub(dd_mul(vv, wv[r].re), dd_mul(uu, a3.re)), dd_mul_d(d0, g)),
                       dd_sub(dd_sub(dd_mul(vv, wv[r].im), dd_mul(uu, a3.im)), dd_mul_d(d1, g))};
        }
    }
    __syncthreads();
    fft_dif_dd(z, N, cs, sn);
    for (int p = threadIdx.x; p < N; p += blockDim.x) z2[p] = z[p];
    __syncthreads();
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const dd uv = dd_mul(ldp(u, N, j), ldp(v, N, j));
        z[j] = cdd{dd_mul(uv, ldp(deta, L, o0 + j)), has1 ? dd_mul(uv, ldp(deta, L, o1 + j)) : zero};
    }
    __syncthreads();
    fft_dif_dd(z, N, cs, sn);
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        const double k = (double)wavenumber_dd(p, N, logN);
        dd f = filter_on ? ldp(filt, N, dft_index_dd(p, logN)) : dd{1.0, 0.0};
        f = dd_mul_d(f, rN);
        const cdd q = z2[p], t = z[p];
        // F P (q^ - i k t^)
        z2[p] = (p == 0) ? cdd{zero, zero} : cdd{dd_mul(f, dd_add(q.re, dd_mul_d(t.im, k))), dd_mul(f, dd_sub(q.im, dd_mul_d(t.re, k)))};
    }
    __syncthreads();
    ifft_dit_dd(z2, N, cs, sn);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        stp(dphi_t, L, o0 + j, z2[j].re);
        if (has1) stp(dphi_t, L, o1 + j, z2[j].im);
        z[j] = cdd{ldp(wout, Lw, o0 + j), has1 ? ldp(wout, Lw, o1 + j) : zero};
    }
    __syncthreads();
    fft_dif_dd(z, N, cs, sn);
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        dd f = filter_on ? ldp(filt, N, dft_index_dd(p, logN)) : dd{1.0, 0.0};
        f = dd_mul_d(f, rN);
        z[p] = cdd{dd_mul(f, z[p].re), dd_mul(f, z[p].im)};
    }
    __syncthreads();
    ifft_dit_dd(z, N, cs, sn);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        stp(deta_t, L, o0 + j, z[j].re);
        if (has1) stp(deta_t, L, o1 + j, z[j].im);
    }
}

// Surface tension in double-double.  Base state: phi_t += F P[ sigma D( eta' / sqrt(1 + eta'^2) ) ]   (2.1b); one CTA.
__global__ void __launch_bounds__(512) k_st_base_dd(int N, int logN, const double* __restrict__ cs, const double* __restrict__ sn,
                                                    const double* __restrict__ filt, int filter_on, double sigma, size_t L,
                                                    const double* __restrict__ d1, double* __restrict__ phi_t) {
    extern __shared__ __align__(16) unsigned char rkdd_sm[];
    cdd* z = reinterpret_cast<cdd*>(rkdd_sm);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const dd e1 = ldp(d1, N, j);
        z[j] = cdd{dd_div(e1, dd_sqrt(dd_add_d(dd_sqr(e1), 1.0))), dd{0.0, 0.0}};
    }
    __syncthreads();
    fft_dif_dd(z, N, cs, sn);
    const double rN = 1.0 / (double)N;
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        const double k = (double)wavenumber_dd(p, N, logN) * rN;   // exact; 0 at p = 0: the projection P
        dd f = dd{k, 0.0};
        if (filter_on) f = dd_mul_d(ldp(filt, N, dft_index_dd(p, logN)), k);
        const cdd t = z[p];
        z[p] = cdd{dd_neg(dd_mul(f, t.im)), dd_mul(f, t.re)};
    }
    __syncthreads();
    ifft_dit_dd(z, N, cs, sn);
    for (int j = threadIdx.x; j < N; j += blockDim.x) stp(phi_t, L, j, dd_add(ldp(phi_t, L, j), dd_mul_d(z[j].re, sigma)));
}

// Variational columns: dphi_t += F P[ sigma D( D(deta_c) / (1 + eta'^2)^(3/2) ) ]   (B.4); one CTA per column pair.
__global__ void __launch_bounds__(512) k_st_cols_dd(int N, int logN, const double* __restrict__ cs, const double* __restrict__ sn,
                                                    const double* __restrict__ filt, int filter_on, double sigma, int ncols, size_t L,
                                                    const double* __restrict__ d1, const double* __restrict__ deta, double* __restrict__ dphi_t) {
    extern __shared__ __align__(16) unsigned char rkdd_sm[];
    cdd* z = reinterpret_cast<cdd*>(rkdd_sm);
    const int c0 = 2 * blockIdx.x, c1 = c0 + 1;
    const bool has1 = c1 < ncols;
    const size_t o0 = (size_t)c0 * N, o1 = (size_t)c1 * N;
    const double rN = 1.0 / (double)N;
    for (int j = threadIdx.x; j < N; j += blockDim.x) z[j] = cdd{ldp(deta, L, o0 + j), has1 ? ldp(deta, L, o1 + j) : dd{0.0, 0.0}};
    __syncthreads();
    fft_dif_dd(z, N, cs, sn);
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        const double k = (double)wavenumber_dd(p, N, logN) * rN;
        const cdd t = z[p];
        z[p] = cdd{dd_mul_d(t.im, -k), dd_mul_d(t.re, k)};
    }
    __syncthreads();
    ifft_dit_dd(z, N, cs, sn);   // D(deta)
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const dd e1 = ldp(d1, N, j), den = dd_add_d(dd_sqr(e1), 1.0), q = dd_mul(den, dd_sqrt(den));
        z[j] = cdd{dd_div(z[j].re, q), dd_div(z[j].im, q)};
    }
    __syncthreads();
    fft_dif_dd(z, N, cs, sn);
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        const double k = (double)wavenumber_dd(p, N, logN) * rN;
        dd f = dd{k, 0.0};
        if (filter_on) f = dd_mul_d(ldp(filt, N, dft_index_dd(p, logN)), k);
        const cdd t = z[p];
        z[p] = cdd{dd_neg(dd_mul(f, t.im)), dd_mul(f, t.re)};
    }
    __syncthreads();
    ifft_dit_dd(z, N, cs, sn);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        stp(dphi_t, L, o0 + j, dd_add(ldp(dphi_t, L, o0 + j), dd_mul_d(z[j].re, sigma)));
        if (has1) stp(dphi_t, L, o1 + j, dd_add(ldp(dphi_t, L, o1 + j), dd_mul_d(z[j].im, sigma)));
    }
}

// ------------------------------------------------------------------------------------------------ refined mesh (mesh.cu), double-double
// The same kernels as k_rhs_base_mesh / k_rhs_cols_mesh of rk.cu: d/dx = (1/xi') d/dalpha term by term, the filter on the modes in alpha,
// P removes the mean over x, f^_0 + a1 Re f^_1 + a2 Re f^_2 for E = 1 + a1 cos(alpha) + a2 cos(2 alpha).  xE, coef: mesh tables (dd).
struct MeshRkDD {
    const double* xE;    // xi', dd planar 2N
    const double* coef;  // a1 (hi, lo), a2 (hi, lo)
};
__device__ __forceinline__ void mesh_deriv_x_dd(cdd* z, int N, int logN, const double* __restrict__ cs, const double* __restrict__ sn,
                                                const double* __restrict__ xE) {
    const double rN = 1.0 / (double)N;
    __syncthreads();
    fft_dif_dd(z, N, cs, sn);
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        const double k = (double)wavenumber_dd(p, N, logN) * rN;
        const cdd t = z[p];
        z[p] = cdd{dd_mul_d(t.im, -k), dd_mul_d(t.re, k)};
    }
    __syncthreads();
    ifft_dit_dd(z, N, cs, sn);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const dd e = ldp(xE, N, j);
        z[j] = cdd{dd_div(z[j].re, e), dd_div(z[j].im, e)};
    }
    __syncthreads();
}
__device__ __forceinline__ void mesh_filter_project_dd(cdd* z, int N, int logN, const double* __restrict__ cs, const double* __restrict__ sn,
                                                       const double* __restrict__ filt, int filter_on, MeshRkDD ms, bool proj_re, bool proj_im) {
    const double rN = 1.0 / (double)N;
    __syncthreads();
    fft_dif_dd(z, N, cs, sn);
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        dd f = filter_on ? ldp(filt, N, dft_index_dd(p, logN)) : dd{1.0, 0.0};
        f = dd_mul_d(f, rN);
        z[p] = cdd{dd_mul(z[p].re, f), dd_mul(z[p].im, f)};
    }
    __syncthreads();
    if (threadIdx.x == 0 && (proj_re || proj_im)) {
        const dd a1{ms.coef[0], ms.coef[1]}, a2{ms.coef[2], ms.coef[3]};
        const cdd p1 = z[dft_index_dd(1, logN)], m1 = z[dft_index_dd(N - 1, logN)], p2 = z[dft_index_dd(2, logN)], m2 = z[dft_index_dd(N - 2, logN)];
        // Re X_k = (Re Z_k + Re Z_-k)/2, Re Y_k = (Im Z_k + Im Z_-k)/2 for the packed pair x + i y
        if (proj_re) z[0].re = dd_neg(dd_half(dd_add(dd_mul(a1, dd_add(p1.re, m1.re)), dd_mul(a2, dd_add(p2.re, m2.re)))));
        if (proj_im) z[0].im = dd_neg(dd_half(dd_add(dd_mul(a1, dd_add(p1.im, m1.im)), dd_mul(a2, dd_add(p2.im, m2.im)))));
    }
    __syncthreads();
    ifft_dit_dd(z, N, cs, sn);
}

__global__ void __launch_bounds__(512) k_rhs_base_mesh_dd(int N, int logN, const double* __restrict__ cs, const double* __restrict__ sn,
                                                          const double* __restrict__ filt, int filter_on, double g, double sigma, MeshRkDD ms, size_t L,
                                                          const double* __restrict__ eta, const double* __restrict__ d1, const double* __restrict__ W0,
                                                          const double* __restrict__ u, const double* __restrict__ v, double* __restrict__ eta_t,
                                                          double* __restrict__ phi_t) {
    extern __shared__ __align__(16) unsigned char rkdd_sm[];
    cdd* z = reinterpret_cast<cdd*>(rkdd_sm);
    const dd zero{0.0, 0.0};
    dd cur[DDF_MAX_PER_THREAD];
#pragma unroll
    for (int r = 0; r < DDF_MAX_PER_THREAD; r++) cur[r] = zero;
    if (sigma != 0.0) {
        for (int j = threadIdx.x; j < N; j += blockDim.x) {
            const dd e1 = dd_div(ldp(d1, N, j), ldp(ms.xE, N, j));
            z[j] = cdd{dd_div(e1, dd_sqrt(dd_add_d(dd_sqr(e1), 1.0))), zero};
        }
        mesh_deriv_x_dd(z, N, logN, cs, sn, ms.xE);
#pragma unroll
        for (int r = 0; r < DDF_MAX_PER_THREAD; r++) {
            const int j = threadIdx.x + r * blockDim.x;
            if (j < N) cur[r] = dd_mul_d(z[j].re, sigma);
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < DDF_MAX_PER_THREAD; r++) {
        const int j = threadIdx.x + r * blockDim.x;
        if (j < N) {
            const dd w = ldp(W0, N, j), uu = ldp(u, N, j), vv = ldp(v, N, j), e = ldp(eta, L, j);
            dd q = dd_sub(dd_mul(vv, w), dd_half(dd_sqr(uu)));
            q = dd_sub(q, dd_half(dd_sqr(vv)));
            q = dd_sub(q, dd_mul_d(e, g));
            z[j] = cdd{w, dd_add(q, cur[r])};
        }
    }
    mesh_filter_project_dd(z, N, logN, cs, sn, filt, filter_on, ms, false, true);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        stp(eta_t, L, j, z[j].re);
        stp(phi_t, L, j, z[j].im);
    }
}

__global__ void __launch_bounds__(512) k_rhs_cols_mesh_dd(int N, int logN, const double* __restrict__ cs, const double* __restrict__ sn,
                                                          const double* __restrict__ filt, int filter_on, double g, double sigma, MeshRkDD ms, int ncols,
                                                          size_t L, size_t Lw, const double* __restrict__ d1, const double* __restrict__ u,
                                                          const double* __restrict__ v, const double* __restrict__ deta, const double* __restrict__ dphi,
                                                          const double* __restrict__ wout, double* __restrict__ deta_t, double* __restrict__ dphi_t) {
    extern __shared__ __align__(16) unsigned char rkdd_sm[];
    cdd* z = reinterpret_cast<cdd*>(rkdd_sm);
    const int c0 = 2 * blockIdx.x, c1 = c0 + 1;
    const bool has1 = c1 < ncols;
    const size_t o0 = (size_t)c0 * N, o1 = (size_t)c1 * N;
    const dd zero{0.0, 0.0};
    cdd acc[DDF_MAX_PER_THREAD];
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const dd uu = ldp(u, N, j);
        z[j] = cdd{dd_mul(uu, ldp(deta, L, o0 + j)), has1 ? dd_mul(uu, ldp(deta, L, o1 + j)) : zero};
    }
    mesh_deriv_x_dd(z, N, logN, cs, sn, ms.xE);  // d/dx(u deta)
#pragma unroll
    for (int r = 0; r < DDF_MAX_PER_THREAD; r++) {
        const int j = threadIdx.x + r * blockDim.x;
        if (j < N) {
            const dd vv = ldp(v, N, j);
            acc[r].re = dd_sub(dd_mul(vv, dd_add(ldp(wout, Lw, o0 + j), z[j].re)), dd_mul_d(ldp(deta, L, o0 + j), g));  // v w - g deta
            acc[r].im = has1 ? dd_sub(dd_mul(vv, dd_add(ldp(wout, Lw, o1 + j), z[j].im)), dd_mul_d(ldp(deta, L, o1 + j), g)) : zero;
        }
    }
    __syncthreads();
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const dd vv = ldp(v, N, j);
        z[j] = cdd{dd_sub(ldp(dphi, L, o0 + j), dd_mul(vv, ldp(deta, L, o0 + j))),
                   has1 ? dd_sub(ldp(dphi, L, o1 + j), dd_mul(vv, ldp(deta, L, o1 + j))) : zero};
    }
    mesh_deriv_x_dd(z, N, logN, cs, sn, ms.xE);  // d/dx(b)
#pragma unroll
    for (int r = 0; r < DDF_MAX_PER_THREAD; r++) {
        const int j = threadIdx.x + r * blockDim.x;
        if (j < N) {
            const dd uu = ldp(u, N, j);
            acc[r].re = dd_sub(acc[r].re, dd_mul(uu, z[j].re));
            acc[r].im = dd_sub(acc[r].im, dd_mul(uu, z[j].im));
        }
    }
    __syncthreads();
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const dd uv = dd_mul(ldp(u, N, j), ldp(v, N, j));
        z[j] = cdd{dd_mul(uv, ldp(deta, L, o0 + j)), has1 ? dd_mul(uv, ldp(deta, L, o1 + j)) : zero};
    }
    mesh_deriv_x_dd(z, N, logN, cs, sn, ms.xE);  // d/dx(deta u v)
#pragma unroll
    for (int r = 0; r < DDF_MAX_PER_THREAD; r++) {
        const int j = threadIdx.x + r * blockDim.x;
        if (j < N) {
            acc[r].re = dd_sub(acc[r].re, z[j].re);
            acc[r].im = dd_sub(acc[r].im, z[j].im);
        }
    }
    __syncthreads();
    if (sigma != 0.0) {
        for (int j = threadIdx.x; j < N; j += blockDim.x) z[j] = cdd{ldp(deta, L, o0 + j), has1 ? ldp(deta, L, o1 + j) : zero};
        mesh_deriv_x_dd(z, N, logN, cs, sn, ms.xE);
        for (int j = threadIdx.x; j < N; j += blockDim.x) {
            const dd e1 = dd_div(ldp(d1, N, j), ldp(ms.xE, N, j)), den = dd_add_d(dd_sqr(e1), 1.0), q = dd_mul(den, dd_sqrt(den));
            z[j] = cdd{dd_div(z[j].re, q), dd_div(z[j].im, q)};
        }
        mesh_deriv_x_dd(z, N, logN, cs, sn, ms.xE);
#pragma unroll
        for (int r = 0; r < DDF_MAX_PER_THREAD; r++) {
            const int j = threadIdx.x + r * blockDim.x;
            if (j < N) {
                acc[r].re = dd_add(acc[r].re, dd_mul_d(z[j].re, sigma));
                acc[r].im = dd_add(acc[r].im, dd_mul_d(z[j].im, sigma));
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < DDF_MAX_PER_THREAD; r++) {
        const int j = threadIdx.x + r * blockDim.x;
        if (j < N) z[j] = acc[r];
    }
    mesh_filter_project_dd(z, N, logN, cs, sn, filt, filter_on, ms, true, true);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        stp(dphi_t, L, o0 + j, z[j].re);
        if (has1) stp(dphi_t, L, o1 + j, z[j].im);
    }
    __syncthreads();
    for (int j = threadIdx.x; j < N; j += blockDim.x) z[j] = cdd{ldp(wout, Lw, o0 + j), has1 ? ldp(wout, Lw, o1 + j) : zero};
    mesh_filter_project_dd(z, N, logN, cs, sn, filt, filter_on, ms, false, false);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        stp(deta_t, L, o0 + j, z[j].re);
        if (has1) stp(deta_t, L, o1 + j, z[j].im);
    }
}

// the filter (2.14) applied in place to ncols columns of the state (column c at offset c N of each plane)
__global__ void __launch_bounds__(512) k_filter_cols_dd(int N, int logN, const double* __restrict__ cs, const double* __restrict__ sn,
                                                        const double* __restrict__ filt, int ncols, size_t L, double* __restrict__ y) {
    extern __shared__ __align__(16) unsigned char rkdd_sm[];
    cdd* z = reinterpret_cast<cdd*>(rkdd_sm);
    const int c0 = 2 * blockIdx.x, c1 = c0 + 1;
    const bool has1 = c1 < ncols;
    const size_t o0 = (size_t)c0 * N, o1 = (size_t)c1 * N;
    for (int j = threadIdx.x; j < N; j += blockDim.x) z[j] = cdd{ldp(y, L, o0 + j), has1 ? ldp(y, L, o1 + j) : dd{0.0, 0.0}};
    __syncthreads();
    fft_dif_dd(z, N, cs, sn);
    const double rN = 1.0 / (double)N;
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        const dd f = dd_mul_d(ldp(filt, N, dft_index_dd(p, logN)), rN);
        z[p] = cdd{dd_mul(f, z[p].re), dd_mul(f, z[p].im)};
    }
    __syncthreads();
    ifft_dit_dd(z, N, cs, sn);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        stp(y, L, o0 + j, z[j].re);
        if (has1) stp(y, L, o1 + j, z[j].im);
    }
}

// E = (pi/N) sum_j [ phi_j (G phi)_j + g eta_j^2 ] in double-double; one CTA, out: hi, lo
__global__ void __launch_bounds__(256) k_energy_dd(int N, double g, size_t L, const double* __restrict__ eta, const double* __restrict__ phi,
                                                   const double* __restrict__ W0, const double* __restrict__ xE, double* __restrict__ out) {
    __shared__ double sh[256], sl[256];
    dd a{0.0, 0.0};
    for (int j = threadIdx.x; j < N; j += 256) {
        const dd e = ldp(eta, L, j);
        dd t = dd_add(dd_mul(ldp(phi, L, j), ldp(W0, N, j)), dd_mul_d(dd_sqr(e), g));
        if (xE) t = dd_mul(t, ldp(xE, N, j));  // dx = xi' dalpha on a refined mesh
        a = dd_add(a, t);
    }
    sh[threadIdx.x] = a.hi;
    sl[threadIdx.x] = a.lo;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) {
            const dd s = dd_add(dd{sh[threadIdx.x], sl[threadIdx.x]}, dd{sh[threadIdx.x + o], sl[threadIdx.x + o]});
            sh[threadIdx.x] = s.hi;
            sl[threadIdx.x] = s.lo;
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const dd e = dd_mul_d(dd_mul(dd{sh[0], sl[0]}, dd_pi()), 1.0 / (double)N);
        out[0] = e.hi;
        out[1] = e.lo;
    }
}

static int ddf_threads(int N) { return N / 2 > 512 ? 512 : (N / 2 < 32 ? 32 : N / 2); }
static int ddf_log2(int n) {
    int l = 0;
    while ((1 << l) < n) l++;
    return l;
}

int rkdd_set_attrs() {
    static DeviceOnce once;
    if (once.first()) {
        SWW_CUDA(cudaFuncSetAttribute(k_rhs_base_dd, cudaFuncAttributeMaxDynamicSharedMemorySize, RKDD_MAX_N * 32));
        SWW_CUDA(cudaFuncSetAttribute(k_rhs_cols_dd, cudaFuncAttributeMaxDynamicSharedMemorySize, RKDD_MAX_N * 64));
        SWW_CUDA(cudaFuncSetAttribute(k_filter_cols_dd, cudaFuncAttributeMaxDynamicSharedMemorySize, RKDD_MAX_N * 32));
        SWW_CUDA(cudaFuncSetAttribute(k_st_base_dd, cudaFuncAttributeMaxDynamicSharedMemorySize, RKDD_MAX_N * 32));
        SWW_CUDA(cudaFuncSetAttribute(k_st_cols_dd, cudaFuncAttributeMaxDynamicSharedMemorySize, RKDD_MAX_N * 32));
        SWW_CUDA(cudaFuncSetAttribute(k_rhs_base_mesh_dd, cudaFuncAttributeMaxDynamicSharedMemorySize, RKDD_MAX_N * 32));
        SWW_CUDA(cudaFuncSetAttribute(k_rhs_cols_mesh_dd, cudaFuncAttributeMaxDynamicSharedMemorySize, RKDD_MAX_N * 32));
    }
    return SWW_OK;
}

int rkdd_combine(cudaStream_t st, size_t L, const double* y, const double* k, const CombDD& cb, double* out) {
    SWW_BEGIN(KC_OTHER, st);
    k_rk_combine_dd<<<(unsigned)((L + 255) / 256), 256, 0, st>>>(L, y, k, cb, out);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

int rkdd_rhs_base(sww_dtn_s* d, bool filter, double g, double sigma, size_t L, const double* ys, double* kout) {
    const int N = d->N;
    const Tables* t = d->tab;
    SWW_BEGIN(KC_FFT, d->stream);
    if (d->mesh_on) {  // refined mesh: the surface-tension term is inside the kernel
        k_rhs_base_mesh_dd<<<1, ddf_threads(N), (size_t)N * 32, d->stream>>>(N, ddf_log2(N), t->cs, t->sn, t->filt_dd, filter ? 1 : 0, g, sigma,
                                                                             MeshRkDD{d->mesh.xE, d->mesh.coef}, L, ys, d->d1, d->bW0, d->bu, d->bv, kout,
                                                                             kout + N);
        SWW_LAUNCHED();
        SWW_CUDA(cudaGetLastError());
        return SWW_OK;
    }
    k_rhs_base_dd<<<1, ddf_threads(N), (size_t)N * 32, d->stream>>>(N, ddf_log2(N), t->cs, t->sn, t->filt_dd, filter ? 1 : 0, g, L, ys, d->bW0, d->bu,
                                                                    d->bv, kout, kout + N);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

int rkdd_rhs_cols(sww_dtn_s* d, bool filter, double g, double sigma, int nc, size_t L, const double* ys, const double* wout, double* kout) {
    const int N = d->N;
    const Tables* t = d->tab;
    const size_t od = 2 * (size_t)N, op = od + (size_t)N * nc;
    SWW_BEGIN(KC_FFT, d->stream);
    if (d->mesh_on) {
        k_rhs_cols_mesh_dd<<<(nc + 1) / 2, ddf_threads(N), (size_t)N * 32, d->stream>>>(N, ddf_log2(N), t->cs, t->sn, t->filt_dd, filter ? 1 : 0, g, sigma,
                                                                                        MeshRkDD{d->mesh.xE, d->mesh.coef}, nc, L, (size_t)N * nc, d->d1,
                                                                                        d->bu, d->bv, ys + od, ys + op, wout, kout + od, kout + op);
        SWW_LAUNCHED();
        SWW_CUDA(cudaGetLastError());
        return SWW_OK;
    }
    k_rhs_cols_dd<<<(nc + 1) / 2, ddf_threads(N), (size_t)N * 64, d->stream>>>(N, ddf_log2(N), t->cs, t->sn, t->filt_dd, filter ? 1 : 0, g, nc, L,
                                                                               (size_t)N * nc, d->bu, d->bv, ys + od, ys + op, wout, kout + od,
                                                                               kout + op);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

int rkdd_st_base(sww_dtn_s* d, bool filter, double sigma, size_t L, double* kout) {
    const int N = d->N;
    const Tables* t = d->tab;
    SWW_BEGIN(KC_FFT, d->stream);
    k_st_base_dd<<<1, ddf_threads(N), (size_t)N * 32, d->stream>>>(N, ddf_log2(N), t->cs, t->sn, t->filt_dd, filter ? 1 : 0, sigma, L, d->d1, kout + N);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

int rkdd_st_cols(sww_dtn_s* d, bool filter, double sigma, int nc, size_t L, const double* ys, double* kout) {
    const int N = d->N;
    const Tables* t = d->tab;
    const size_t od = 2 * (size_t)N, op = od + (size_t)N * nc;
    SWW_BEGIN(KC_FFT, d->stream);
    k_st_cols_dd<<<(nc + 1) / 2, ddf_threads(N), (size_t)N * 32, d->stream>>>(N, ddf_log2(N), t->cs, t->sn, t->filt_dd, filter ? 1 : 0, sigma, nc, L,
                                                                              d->d1, ys + od, kout + op);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

int rkdd_filter_state(sww_dtn_s* d, int ncol, size_t L, double* y) {
    const int N = d->N;
    const Tables* t = d->tab;
    SWW_BEGIN(KC_FFT, d->stream);
    k_filter_cols_dd<<<(ncol + 1) / 2, ddf_threads(N), (size_t)N * 32, d->stream>>>(N, ddf_log2(N), t->cs, t->sn, t->filt_dd, ncol, L, y);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

int rkdd_energy(sww_dtn_s* d, double g, size_t L, const double* y, double* out2) {
    SWW_BEGIN(KC_OTHER, d->stream);
    k_energy_dd<<<1, 256, 0, d->stream>>>(d->N, g, L, y, y + d->N, d->bW0, d->mesh_on ? d->mesh.xE : nullptr, out2);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

}  // namespace sww
