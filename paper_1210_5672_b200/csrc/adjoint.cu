// adjoint.cu -- right-hand side of the adjoint system (B.6), PAPER.md:730-747 (the "same structure as the forward and linearized
// problems, with a Dirichlet to Neumann map"): for the state q = (eta, phi) held by the handle (surface set up, base
// state set: u = phi_x, v = phi_y on the surface) and nrhs adjoint vectors (eta~_c, phi~_c):
//     chi_c     = eta~_c + v P phi~_c                                                                              (B.6d)
//     phi~_s,c  = G chi_c + D( u P phi~_c )                                                                        (B.6e)
//     eta~_s,c  = -v G chi_c + u D eta~_c - v D(u) P phi~_c - g P phi~_c + sigma D( D(phi~_c) / (1 + eta'^2)^(3/2) )  (B.6f)
// One batched DtN apply (S3-S6 of the hot path) between two small kernels, in fp64 and in double-double (planar hi / lo blocks,
// N <= 2048 like the double-double stepper).  On the refined mesh (2.10) (mesh.cu) D is d/dx = (1/xi') d/dalpha and P removes the mean
// over x; G chi, u, v arrive in physical form.  Product code; shares nothing with oracle/.
#include "common.cuh"
#include "fft.cuh"
#include "ddfft.cuh"

namespace sww {

// per column: pp = P phi~ (mean removed) -> PP ; chi = eta~ + v pp -> X.  One CTA per column.
// xE (refined mesh (2.10), else nullptr): P removes the mean over x, (1/N) sum_j f_j xi'(alpha_j)
__global__ void __launch_bounds__(256) k_adj_prep(int N, const double* __restrict__ v, const double* __restrict__ xE, const double* __restrict__ eta_t,
                                                  const double* __restrict__ phi_t, double* __restrict__ PP, double* __restrict__ X) {
    __shared__ double s[256];
    const size_t o = (size_t)blockIdx.x * N;
    double a = 0.0;
    for (int j = threadIdx.x; j < N; j += 256) a += xE ? phi_t[o + j] * xE[j] : phi_t[o + j];
    s[threadIdx.x] = a;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if (threadIdx.x < w) s[threadIdx.x] += s[threadIdx.x + w];
        __syncthreads();
    }
    const double mean = s[0] / (double)N;
    for (int j = threadIdx.x; j < N; j += 256) {
        const double pp = phi_t[o + j] - mean, e = eta_t[o + j];  // read before the stores: PP / X may alias the inputs' partners
        PP[o + j] = pp;
        X[o + j] = fma(v[j], pp, e);
    }
}

// one CTA per column pair; PPg (= eta_s on entry) holds P phi~, W (= phi_s on entry) holds G chi; both are overwritten by the result
__global__ void __launch_bounds__(1024) k_adj_rhs(int N, int logN, const double2* __restrict__ tw, double g, double sigma, int ncols,
                                                  const double* __restrict__ u, const double* __restrict__ v, const double* __restrict__ du,
                                                  const double* __restrict__ d1, const double* __restrict__ xE, const double* __restrict__ eta_t,
                                                  const double* __restrict__ phi_t, double* __restrict__ eta_s, double* __restrict__ phi_s) {
    extern __shared__ __align__(16) double2 z[];
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
        if (xE) {  // refined mesh: d/dx = (1/xi') d/dalpha
            for (int j = threadIdx.x; j < N; j += blockDim.x) {
                const double re = 1.0 / xE[j];
                z[j] = make_double2(z[j].x * re, z[j].y * re);
            }
            __syncthreads();
        }
    };
    double2 pp[FFT_MAX_PER_THREAD], w[FFT_MAX_PER_THREAD], es[FFT_MAX_PER_THREAD];
#pragma unroll
    for (int r = 0; r < FFT_MAX_PER_THREAD; r++) {
        const int j = threadIdx.x + r * blockDim.x;
        if (j < N) {
            pp[r] = make_double2(eta_s[o0 + j], has1 ? eta_s[o1 + j] : 0.0);
            w[r] = make_double2(phi_s[o0 + j], has1 ? phi_s[o1 + j] : 0.0);
            z[j] = make_double2(u[j] * pp[r].x, u[j] * pp[r].y);
        }
    }
    deriv_inplace();  // D(u P phi~)
#pragma unroll
    for (int r = 0; r < FFT_MAX_PER_THREAD; r++) {
        const int j = threadIdx.x + r * blockDim.x;
        if (j < N) {
            phi_s[o0 + j] = w[r].x + z[j].x;   // (B.6e)
            if (has1) phi_s[o1 + j] = w[r].y + z[j].y;
        }
    }
    __syncthreads();
    for (int j = threadIdx.x; j < N; j += blockDim.x) z[j] = make_double2(eta_t[o0 + j], has1 ? eta_t[o1 + j] : 0.0);
    deriv_inplace();  // D eta~
#pragma unroll
    for (int r = 0; r < FFT_MAX_PER_THREAD; r++) {
        const int j = threadIdx.x + r * blockDim.x;
        if (j < N) {
            const double uu = u[j], vv = v[j], c = fma(vv, du[j], g);   // v D(u) + g
            es[r] = make_double2(fma(uu, z[j].x, -vv * w[r].x) - c * pp[r].x, fma(uu, z[j].y, -vv * w[r].y) - c * pp[r].y);
        }
    }
    if (sigma != 0.0) {
        __syncthreads();
        for (int j = threadIdx.x; j < N; j += blockDim.x) z[j] = make_double2(phi_t[o0 + j], has1 ? phi_t[o1 + j] : 0.0);
        deriv_inplace();  // D phi~
        for (int j = threadIdx.x; j < N; j += blockDim.x) {
            const double e1 = xE ? d1[j] / xE[j] : d1[j], den = fma(e1, e1, 1.0), q = 1.0 / (den * sqrt(den));
            z[j] = make_double2(z[j].x * q, z[j].y * q);
        }
        deriv_inplace();
#pragma unroll
        for (int r = 0; r < FFT_MAX_PER_THREAD; r++) {
            const int j = threadIdx.x + r * blockDim.x;
            if (j < N) es[r] = make_double2(fma(sigma, z[j].x, es[r].x), fma(sigma, z[j].y, es[r].y));
        }
    }
#pragma unroll
    for (int r = 0; r < FFT_MAX_PER_THREAD; r++) {
        const int j = threadIdx.x + r * blockDim.x;
        if (j < N) {
            eta_s[o0 + j] = es[r].x;   // (B.6f)
            if (has1) eta_s[o1 + j] = es[r].y;
        }
    }
}

// ------------------------------------------------------------------------------------------------ double-double
__device__ __forceinline__ dd adj_ld(const double* p, size_t plane, size_t o) { return dd{p[o], p[plane + o]}; }
__device__ __forceinline__ void adj_st(double* p, size_t plane, size_t o, dd v) {
    p[o] = v.hi;
    p[plane + o] = v.lo;
}

// per column (user arrays: planes of L = N nrhs): pp = P phi~ -> PP ; chi = eta~ + v pp -> X
__global__ void __launch_bounds__(256) k_adj_prep_dd(int N, size_t L, const double* __restrict__ v, const double* __restrict__ xE,
                                                     const double* __restrict__ eta_t, const double* __restrict__ phi_t, double* __restrict__ PP,
                                                     double* __restrict__ X) {
    __shared__ double sh[256], sl[256];
    const size_t o = (size_t)blockIdx.x * N;
    dd a{0.0, 0.0};
    for (int j = threadIdx.x; j < N; j += 256) a = dd_add(a, xE ? dd_mul(adj_ld(phi_t, L, o + j), adj_ld(xE, N, j)) : adj_ld(phi_t, L, o + j));
    sh[threadIdx.x] = a.hi;
    sl[threadIdx.x] = a.lo;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if (threadIdx.x < w) {
            const dd s = dd_add(dd{sh[threadIdx.x], sl[threadIdx.x]}, dd{sh[threadIdx.x + w], sl[threadIdx.x + w]});
            sh[threadIdx.x] = s.hi;
            sl[threadIdx.x] = s.lo;
        }
        __syncthreads();
    }
    const dd mean = dd_mul_d(dd{sh[0], sl[0]}, 1.0 / (double)N);  // N a power of two: exact scaling
    for (int j = threadIdx.x; j < N; j += 256) {
        const dd pp = dd_sub(adj_ld(phi_t, L, o + j), mean), e = adj_ld(eta_t, L, o + j);
        adj_st(PP, L, o + j, pp);
        adj_st(X, L, o + j, dd_add(e, dd_mul(adj_ld(v, N, j), pp)));
    }
}

// one CTA per column pair; PP holds P phi~, W holds G chi (user layout, planes L); results to OE, OP (work space, planes Lws)
__global__ void __launch_bounds__(512) k_adj_rhs_dd(int N, int logN, const double* __restrict__ cs, const double* __restrict__ sn, double g,
                                                    double sigma, int ncols, size_t L, size_t Lws, const double* __restrict__ u,
                                                    const double* __restrict__ v, const double* __restrict__ du, const double* __restrict__ d1,
                                                    const double* __restrict__ xE, const double* __restrict__ eta_t, const double* __restrict__ phi_t,
                                                    const double* __restrict__ PP, const double* __restrict__ W, double* __restrict__ OE,
                                                    double* __restrict__ OP) {
    extern __shared__ __align__(16) unsigned char adj_sm[];
    cdd* z = reinterpret_cast<cdd*>(adj_sm);
    const int c0 = 2 * blockIdx.x, c1 = c0 + 1;
    const bool has1 = c1 < ncols;
    const size_t o0 = (size_t)c0 * N, o1 = (size_t)c1 * N;
    const double rN = 1.0 / (double)N;
    const dd zero{0.0, 0.0};
    auto deriv_inplace = [&]() {
        __syncthreads();
        fft_dif_dd(z, N, cs, sn);
        for (int p = threadIdx.x; p < N; p += blockDim.x) {
            const double k = (double)wavenumber_dd(p, N, logN) * rN;
            const cdd t = z[p];
            z[p] = cdd{dd_mul_d(t.im, -k), dd_mul_d(t.re, k)};
        }
        __syncthreads();
        ifft_dit_dd(z, N, cs, sn);
        if (xE) {
            for (int j = threadIdx.x; j < N; j += blockDim.x) {
                const dd e = adj_ld(xE, N, j);
                z[j] = cdd{dd_div(z[j].re, e), dd_div(z[j].im, e)};
            }
            __syncthreads();
        }
    };
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const dd uu = adj_ld(u, N, j);
        z[j] = cdd{dd_mul(uu, adj_ld(PP, L, o0 + j)), has1 ? dd_mul(uu, adj_ld(PP, L, o1 + j)) : zero};
    }
    deriv_inplace();  // D(u P phi~)
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        adj_st(OP, Lws, o0 + j, dd_add(adj_ld(W, L, o0 + j), z[j].re));   // (B.6e)
        if (has1) adj_st(OP, Lws, o1 + j, dd_add(adj_ld(W, L, o1 + j), z[j].im));
    }
    __syncthreads();
    for (int j = threadIdx.x; j < N; j += blockDim.x) z[j] = cdd{adj_ld(eta_t, L, o0 + j), has1 ? adj_ld(eta_t, L, o1 + j) : zero};
    deriv_inplace();  // D eta~
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const dd uu = adj_ld(u, N, j), vv = adj_ld(v, N, j), c = dd_add_d(dd_mul(vv, adj_ld(du, N, j)), g);   // v D(u) + g
        const dd e0 = dd_sub(dd_sub(dd_mul(uu, z[j].re), dd_mul(vv, adj_ld(W, L, o0 + j))), dd_mul(c, adj_ld(PP, L, o0 + j)));
        adj_st(OE, Lws, o0 + j, e0);
        if (has1) {
            const dd e1 = dd_sub(dd_sub(dd_mul(uu, z[j].im), dd_mul(vv, adj_ld(W, L, o1 + j))), dd_mul(c, adj_ld(PP, L, o1 + j)));
            adj_st(OE, Lws, o1 + j, e1);
        }
    }
    if (sigma != 0.0) {
        __syncthreads();
        for (int j = threadIdx.x; j < N; j += blockDim.x) z[j] = cdd{adj_ld(phi_t, L, o0 + j), has1 ? adj_ld(phi_t, L, o1 + j) : zero};
        deriv_inplace();  // D phi~
        for (int j = threadIdx.x; j < N; j += blockDim.x) {
            const dd e1 = xE ? dd_div(adj_ld(d1, N, j), adj_ld(xE, N, j)) : adj_ld(d1, N, j), den = dd_add_d(dd_sqr(e1), 1.0), q = dd_mul(den, dd_sqrt(den));
            z[j] = cdd{dd_div(z[j].re, q), dd_div(z[j].im, q)};
        }
        deriv_inplace();
        for (int j = threadIdx.x; j < N; j += blockDim.x) {
            adj_st(OE, Lws, o0 + j, dd_add(adj_ld(OE, Lws, o0 + j), dd_mul_d(z[j].re, sigma)));   // (B.6f)
            if (has1) adj_st(OE, Lws, o1 + j, dd_add(adj_ld(OE, Lws, o1 + j), dd_mul_d(z[j].im, sigma)));
        }
    }
}

// planar copy: n entries per plane, planes Lin -> Lout
__global__ void k_adj_copy_dd(size_t n, size_t Lin, size_t Lout, const double* __restrict__ in, double* __restrict__ out) {
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    out[e] = in[e];
    out[Lout + e] = in[Lin + e];
}

int circ_dd(sww_dtn_s* d, int mode, const double* in, double* out);   // ddpath.cu: the double-double circulants D (mode 0), H (mode 1)

static int adjoint_dd(sww_dtn_s* d, const double* eta_t, const double* phi_t, int nrhs, double g, double sigma, double* eta_s, double* phi_s) {
    const int N = d->N;
    if (N > 2048) return SWW_EINVAL;  // one N-point complex double-double array in shared memory and the stepper's limit (include/sww.h)
    cudaStream_t st = d->stream;
    const size_t L = (size_t)N * nrhs;
    double* du = d->tmp;  // 2 N of the base-state scratch
    const double* xE = d->mesh_on ? d->mesh.xE : nullptr;
    SWW_TRY(circ_dd(d, 0, d->bu, du));
    SWW_TRY(mesh_scale_out(d, du, 1, N));  // refined mesh: d/dx(u) = D(u) / xi'
    SWW_BEGIN(KC_OTHER, st);
    k_adj_prep_dd<<<nrhs, 256, 0, st>>>(N, L, d->bv, xE, eta_t, phi_t, eta_s, phi_s);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    SWW_TRY(sww_dtn_apply(d, phi_s, nrhs, phi_s));  // G chi in double-double, in place
    Workspace& w = d->ws;
    const size_t Lws = (size_t)N * w.cap_cols;
    static DeviceOnce attr_once;
    if (attr_once.first()) SWW_CUDA(cudaFuncSetAttribute(k_adj_rhs_dd, cudaFuncAttributeMaxDynamicSharedMemorySize, 2048 * 32));
    int lg = 0;
    while ((1 << lg) < N) lg++;
    const int thr = N / 2 > 512 ? 512 : (N / 2 < 32 ? 32 : N / 2);
    SWW_BEGIN(KC_FFT, st);
    k_adj_rhs_dd<<<(nrhs + 1) / 2, thr, (size_t)N * sizeof(cdd), st>>>(N, lg, d->tab->cs, d->tab->sn, g, sigma, nrhs, L, Lws, d->bu, d->bv, du, d->d1, xE, eta_t,
                                                                      phi_t, eta_s, phi_s, w.T, w.Gam);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    const unsigned blocks = (unsigned)((L + 255) / 256);
    SWW_BEGIN(KC_OTHER, st);
    k_adj_copy_dd<<<blocks, 256, 0, st>>>(L, Lws, L, w.T, eta_s);
    SWW_LAUNCHED();
    SWW_BEGIN(KC_OTHER, st);
    k_adj_copy_dd<<<blocks, 256, 0, st>>>(L, Lws, L, w.Gam, phi_s);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

}  // namespace sww

using namespace sww;

extern "C" int sww_dtn_adjoint_rhs(sww_dtn_t d, const void* eta_t, const void* phi_t, int nrhs, double g, double sigma, void* eta_s, void* phi_s) {
    if (!d || nrhs < 0 || !(sigma >= 0.0)) return SWW_EINVAL;
    if (!d->has_base) return SWW_ENOBASE;
    if (nrhs == 0) return SWW_OK;
    if (!eta_t || !phi_t || !eta_s || !phi_s || eta_s == phi_s || eta_s == eta_t || eta_s == phi_t || phi_s == eta_t || phi_s == phi_t)
        return SWW_EINVAL;
    if (d->prec == SWW_DD)
        return adjoint_dd(d, (const double*)eta_t, (const double*)phi_t, nrhs, g, sigma, (double*)eta_s, (double*)phi_s);
    const int N = d->N;
    cudaStream_t st = d->stream;
    double* du = d->tmp;  // scratch of the base-state flow (14 N doubles), idle once the base state is set
    const double* xE = d->mesh_on ? d->mesh.xE : nullptr;
    SWW_TRY(spectral_deriv(d, d->bu, du, 1));  // D(u) = "phi_x'" of (B.6f)
    SWW_TRY(mesh_scale_out(d, du, 1, 0));      // refined mesh: d/dx(u) = D(u) / xi'
    SWW_BEGIN(KC_OTHER, st);
    k_adj_prep<<<nrhs, 256, 0, st>>>(N, d->bv, xE, (const double*)eta_t, (const double*)phi_t, (double*)eta_s, (double*)phi_s);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    SWW_TRY(sww_dtn_apply(d, phi_s, nrhs, phi_s));  // G chi, in place (S3-S6)
    static DeviceOnce attr_once;
    if (attr_once.first()) SWW_CUDA(cudaFuncSetAttribute(k_adj_rhs, cudaFuncAttributeMaxDynamicSharedMemorySize, 8192 * 16));
    SWW_BEGIN(KC_FFT, st);
    k_adj_rhs<<<(nrhs + 1) / 2, fft_threads(N), sizeof(double2) * (size_t)N, st>>>(N, fft_ilog2(N), d->tab->tw, g, sigma, nrhs, d->bu, d->bv, du, d->d1, xE,
                                                                                  (const double*)eta_t, (const double*)phi_t, (double*)eta_s,
                                                                                  (double*)phi_s);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}
