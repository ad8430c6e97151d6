// ddfft.cuh -- double-double complex arithmetic and the shared-memory FFTs of the double-double path (ddpath.cu, rk_dd.cu):
// radix-2 decimation in frequency forward (natural in, bit-reversed out), radix-2 decimation in time inverse (bit-reversed in,
// natural out, unscaled), twiddles exp(-+2 pi i m/N) from the dd tables cs, sn (planar, tables.cu).  "custom FFT ... in
// quadruple precision".  Product code; shares nothing with oracle/.
#pragma once
#include "common.cuh"
#include "dd.cuh"

namespace sww {

struct cdd {
    dd re, im;
};
__device__ __forceinline__ cdd cdd_add(cdd a, cdd b) { return cdd{dd_add(a.re, b.re), dd_add(a.im, b.im)}; }
__device__ __forceinline__ cdd cdd_sub(cdd a, cdd b) { return cdd{dd_sub(a.re, b.re), dd_sub(a.im, b.im)}; }
// a * (wr + i wi)
__device__ __forceinline__ cdd cdd_mul(cdd a, dd wr, dd wi) {
    return cdd{dd_sub(dd_mul(a.re, wr), dd_mul(a.im, wi)), dd_add(dd_mul(a.re, wi), dd_mul(a.im, wr))};
}
static __device__ void fft_dif_dd(cdd* z, int N, const double* __restrict__ cs, const double* __restrict__ sn) {
    for (int half = N >> 1; half >= 1; half >>= 1) {
        int tstride = N / (2 * half);
        for (int t = threadIdx.x; t < N / 2; t += blockDim.x) {
            int blk = t / half, o = t - blk * half, i = blk * 2 * half + o, m = o * tstride;
            cdd a = z[i], b = z[i + half];
            dd wr = dd_load(cs, N, m), wi = dd_neg(dd_load(sn, N, m));  // exp(-2 pi i m/N)
            z[i] = cdd_add(a, b);
            z[i + half] = cdd_mul(cdd_sub(a, b), wr, wi);
        }
        __syncthreads();
    }
}
static __device__ void ifft_dit_dd(cdd* z, int N, const double* __restrict__ cs, const double* __restrict__ sn) {
    for (int half = 1; half < N; half <<= 1) {
        int tstride = N / (2 * half);
        for (int t = threadIdx.x; t < N / 2; t += blockDim.x) {
            int blk = t / half, o = t - blk * half, i = blk * 2 * half + o, m = o * tstride;
            cdd a = z[i];
            cdd b = cdd_mul(z[i + half], dd_load(cs, N, m), dd_load(sn, N, m));  // conj twiddle exp(+2 pi i m/N)
            z[i] = cdd_add(a, b);
            z[i + half] = cdd_sub(a, b);
        }
        __syncthreads();
    }
}
__device__ __forceinline__ int wavenumber_dd(int p, int N, int logN) {
    int k = (int)(__brev((unsigned)p) >> (32 - logN));
    if (2 * k == N) return 0;
    return (2 * k < N) ? k : k - N;
}

}  // namespace sww
