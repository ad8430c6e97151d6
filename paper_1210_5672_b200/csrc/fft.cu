// fft.cu -- S5/S7: hand-written shared-memory FFTs and the Fourier multipliers of the method (no cuFFT):
//   D = d/dalpha (symbol i k), H = Hilbert transform (-i sgn k), |D| = H D (|k|), all with symbol 0 at the
//   Nyquist mode k = N/2 (R4); "the FFT is used to compute mu', H gamma ...".
// One CTA transforms one PAIR of real columns packed as z = a + i b: every multiplier here has m(-k) = conj m(k), so it maps
// real columns to real columns and acts on a and b independently -- no untangling pass is needed.
// Forward transform: radix-2 decimation in frequency (natural order in, bit-reversed out); the symbol is applied in bit-reversed
// order; inverse transform: radix-2 decimation in time (bit-reversed in, natural out).  No permutation pass.
// Twiddles exp(-2 pi i m/N) come from the dd-accurate table rounded to fp64 (tables.cu).
// Product code; shares nothing with oracle/.
#include "common.cuh"
#include "fft.cuh"

namespace sww {


// Gam_c = D M_c ;  W_c = |D| M_c / 2 - (T ? D T_c : 0)     for the column pair (2*blockIdx.x, 2*blockIdx.x + 1)
// Mp (optional, ncols = 2): column 1 is read from Mp instead of M + N -- the single-vector base state rides phi0 along with mu0 so that
// Gam_1 = D phi0 comes out of the same transform pair (one launch less per stage of the stepper)
__global__ void __launch_bounds__(1024) k_spectral_gamma_w(int N, int logN, const double2* __restrict__ tw, const double* __restrict__ M,
                                   const double* __restrict__ T, double* __restrict__ Gam, double* __restrict__ W, int ncols,
                                   int w_cols, const double* __restrict__ Mp) {
    extern __shared__ __align__(16) double2 z[];
    const int c0 = 2 * blockIdx.x, c1 = c0 + 1;
    const bool has1 = c1 < ncols;
    const int per = (N + blockDim.x - 1) / blockDim.x;
    double2 zt[FFT_MAX_PER_THREAD];
    if (T) {
        for (int j = threadIdx.x; j < N; j += blockDim.x)
            z[j] = make_double2(T[(size_t)c0 * N + j], has1 ? T[(size_t)c1 * N + j] : 0.0);
        __syncthreads();
        fft_dif(z, N, tw);
#pragma unroll
        for (int r = 0; r < FFT_MAX_PER_THREAD; r++)
            if (r < per && threadIdx.x + r * blockDim.x < N) zt[r] = z[threadIdx.x + r * blockDim.x];
        __syncthreads();
    }
    for (int j = threadIdx.x; j < N; j += blockDim.x)
        z[j] = make_double2(M[(size_t)c0 * N + j], has1 ? (Mp ? Mp[j] : M[(size_t)c1 * N + j]) : 0.0);
    __syncthreads();
    fft_dif(z, N, tw);
    double2 zm[FFT_MAX_PER_THREAD];
    const double rN = 1.0 / (double)N;
#pragma unroll
    for (int r = 0; r < FFT_MAX_PER_THREAD; r++)
        if (r < per && threadIdx.x + r * blockDim.x < N) {
            int p = threadIdx.x + r * blockDim.x;
            zm[r] = z[p];
            double k = (double)wavenumber(p, N, logN) * rN;  // fold the 1/N of the inverse transform into the symbol
            z[p] = make_double2(-k * zm[r].y, k * zm[r].x);  // i k zhat
        }
    __syncthreads();
    ifft_dit(z, N, tw);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        double2 v = z[j];
        Gam[(size_t)c0 * N + j] = v.x;
        Gam[(size_t)c1 * N + j] = has1 ? v.y : 0.0;  // Gam is a padded buffer: the odd partner column is zeroed
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < FFT_MAX_PER_THREAD; r++)
        if (r < per && threadIdx.x + r * blockDim.x < N) {
            int p = threadIdx.x + r * blockDim.x;
            double k = (double)wavenumber(p, N, logN) * rN;
            double ha = 0.5 * fabs(k);
            double2 v = make_double2(ha * zm[r].x, ha * zm[r].y);
            if (T) {
                v.x += k * zt[r].y;  // - i k that
                v.y -= k * zt[r].x;
            }
            z[p] = v;
        }
    __syncthreads();
    ifft_dit(z, N, tw);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        double2 v = z[j];
        if (c0 < w_cols) W[(size_t)c0 * N + j] = v.x;
        if (c1 < w_cols) W[(size_t)c1 * N + j] = v.y;
    }
}

// out_c = D in_c
__global__ void __launch_bounds__(1024) k_spectral_deriv(int N, int logN, const double2* __restrict__ tw, const double* __restrict__ in,
                                 double* __restrict__ out, int ncols) {
    extern __shared__ __align__(16) double2 z[];
    const int c0 = 2 * blockIdx.x, c1 = c0 + 1;
    const bool has1 = c1 < ncols;
    for (int j = threadIdx.x; j < N; j += blockDim.x) z[j] = make_double2(in[(size_t)c0 * N + j], has1 ? in[(size_t)c1 * N + j] : 0.0);
    __syncthreads();
    fft_dif(z, N, tw);
    const double rN = 1.0 / (double)N;
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        double2 v = z[p];
        double k = (double)wavenumber(p, N, logN) * rN;
        z[p] = make_double2(-k * v.y, k * v.x);
    }
    __syncthreads();
    ifft_dit(z, N, tw);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        double2 v = z[j];
        out[(size_t)c0 * N + j] = v.x;
        if (has1) out[(size_t)c1 * N + j] = v.y;
    }
}

int spectral_gamma_w(sww_dtn_s* d, const double* M, const double* T, double* Gam, double* W, int ncols, int w_cols, const double* Mp) {
    const int N = d->N;
    size_t smem = sizeof(double2) * (size_t)N;
    static DeviceOnce attr_once;
    if (attr_once.first()) {
        SWW_CUDA(cudaFuncSetAttribute(k_spectral_gamma_w, cudaFuncAttributeMaxDynamicSharedMemorySize, 8192 * 16));
        SWW_CUDA(cudaFuncSetAttribute(k_spectral_deriv, cudaFuncAttributeMaxDynamicSharedMemorySize, 8192 * 16));
    }
    SWW_BEGIN(KC_FFT, d->stream);
    // 512 threads at N = 2048, 4096: two CTAs per SM hide each other's barriers (0.072 -> 0.062 ms at the metric point); the per-thread
    // register arrays hold N / threads <= 8 entries
    const int thr = (N == 2048 || N == 4096) ? 512 : fft_threads(N);
    k_spectral_gamma_w<<<(ncols + 1) / 2, thr, smem, d->stream>>>(N, fft_ilog2(N), d->tab->tw, M, T, Gam, W, ncols, w_cols, Mp);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

int spectral_deriv(sww_dtn_s* d, const double* in, double* out, int ncols) {
    const int N = d->N;
    size_t smem = sizeof(double2) * (size_t)N;
    static DeviceOnce attr_once;
    if (attr_once.first()) {
        SWW_CUDA(cudaFuncSetAttribute(k_spectral_deriv, cudaFuncAttributeMaxDynamicSharedMemorySize, 8192 * 16));
    }
    SWW_BEGIN(KC_FFT, d->stream);
    k_spectral_deriv<<<(ncols + 1) / 2, fft_threads(N), smem, d->stream>>>(N, fft_ilog2(N), d->tab->tw, in, out, ncols);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

}  // namespace sww
