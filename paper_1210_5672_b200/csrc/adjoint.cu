// adjoint.cu -- right-hand side of the adjoint system (B.6), PAPER.md:730-747 (the "same structure as the forward and linearized
// problems, with a Dirichlet to Neumann map"): for the state q = (eta, phi) held by the handle (surface set up, base
// state set: u = phi_x, v = phi_y on the surface) and nrhs adjoint vectors (eta~_c, phi~_c):
//     chi_c     = eta~_c + v P phi~_c                                                                              (B.6d)
//     phi~_s,c  = G chi_c + D( u P phi~_c )                                                                        (B.6e)
//     eta~_s,c  = -v G chi_c + u D eta~_c - v D(u) P phi~_c - g P phi~_c + sigma D( D(phi~_c) / (1 + eta'^2)^(3/2) )  (B.6f)
// One batched DtN apply (S3-S6 of the hot path) between two small kernels.  fp64 handles.  Product code; shares nothing with oracle/.
#include "common.cuh"
#include "fft.cuh"

namespace sww {

// per column: pp = P phi~ (mean removed) -> PP ; chi = eta~ + v pp -> X.  One CTA per column.
__global__ void __launch_bounds__(256) k_adj_prep(int N, const double* __restrict__ v, const double* __restrict__ eta_t,
                                                  const double* __restrict__ phi_t, double* __restrict__ PP, double* __restrict__ X) {
    __shared__ double s[256];
    const size_t o = (size_t)blockIdx.x * N;
    double a = 0.0;
    for (int j = threadIdx.x; j < N; j += 256) a += phi_t[o + j];
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
                                                  const double* __restrict__ d1, const double* __restrict__ eta_t,
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
            const double e1 = d1[j], den = fma(e1, e1, 1.0), q = 1.0 / (den * sqrt(den));
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

}  // namespace sww

using namespace sww;

extern "C" int sww_dtn_adjoint_rhs(sww_dtn_t d, const void* eta_t, const void* phi_t, int nrhs, double g, double sigma, void* eta_s, void* phi_s) {
    if (!d || nrhs < 0 || !(sigma >= 0.0)) return SWW_EINVAL;
    if (d->prec != SWW_F64) return SWW_EINVAL;  // include/sww.h: fp64 handles
    if (!d->has_base) return SWW_ENOBASE;
    if (nrhs == 0) return SWW_OK;
    if (!eta_t || !phi_t || !eta_s || !phi_s || eta_s == phi_s || eta_s == eta_t || eta_s == phi_t || phi_s == eta_t || phi_s == phi_t)
        return SWW_EINVAL;
    const int N = d->N;
    cudaStream_t st = d->stream;
    double* du = d->tmp;  // scratch of the base-state flow (14 N doubles), idle once the base state is set
    SWW_TRY(spectral_deriv(d, d->bu, du, 1));  // D(u) = "phi_x'" of (B.6f)
    SWW_BEGIN(KC_OTHER, st);
    k_adj_prep<<<nrhs, 256, 0, st>>>(N, d->bv, (const double*)eta_t, (const double*)phi_t, (double*)eta_s, (double*)phi_s);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    SWW_TRY(sww_dtn_apply(d, phi_s, nrhs, phi_s));  // G chi, in place (S3-S6)
    static DeviceOnce attr_once;
    if (attr_once.first()) SWW_CUDA(cudaFuncSetAttribute(k_adj_rhs, cudaFuncAttributeMaxDynamicSharedMemorySize, 8192 * 16));
    SWW_BEGIN(KC_FFT, st);
    k_adj_rhs<<<(nrhs + 1) / 2, fft_threads(N), sizeof(double2) * (size_t)N, st>>>(N, fft_ilog2(N), d->tab->tw, g, sigma, nrhs, d->bu, d->bv, du, d->d1,
                                                                                  (const double*)eta_t, (const double*)phi_t, (double*)eta_s,
                                                                                  (double*)phi_s);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}
