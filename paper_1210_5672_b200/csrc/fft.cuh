// fft.cuh -- device helpers of the hand-written shared-memory FFTs (fft.cu, rk.cu): radix-2 decimation in frequency forward
// (natural in, bit-reversed out), radix-2 decimation in time inverse (bit-reversed in, natural out, unscaled), and the signed
// wavenumber of a bit-reversed position.  Product code; shares nothing with oracle/.
#pragma once
#include "common.cuh"

namespace sww {

__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
    return make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ double2 cmulc(double2 a, double2 b) {  // a * conj(b)
    return make_double2(fma(a.x, b.x, a.y * b.y), fma(a.y, b.x, -a.x * b.y));
}

// in-place forward DIF FFT of z[0..N) in shared memory; output in bit-reversed order
static __device__ void fft_dif(double2* z, int N, const double2* __restrict__ tw) {
    for (int half = N >> 1; half >= 1; half >>= 1) {
        int tstride = N / (2 * half);
        for (int t = threadIdx.x; t < N / 2; t += blockDim.x) {
            int blk = t / half, o = t - blk * half;
            int i = blk * 2 * half + o;
            double2 a = z[i], b = z[i + half];
            double2 w = tw[o * tstride];
            z[i] = make_double2(a.x + b.x, a.y + b.y);
            z[i + half] = cmul(make_double2(a.x - b.x, a.y - b.y), w);
        }
        __syncthreads();
    }
}
// in-place inverse DIT FFT (input bit-reversed, output natural), unscaled
static __device__ void ifft_dit(double2* z, int N, const double2* __restrict__ tw) {
    for (int half = 1; half < N; half <<= 1) {
        int tstride = N / (2 * half);
        for (int t = threadIdx.x; t < N / 2; t += blockDim.x) {
            int blk = t / half, o = t - blk * half;
            int i = blk * 2 * half + o;
            double2 a = z[i];
            double2 b = cmulc(z[i + half], tw[o * tstride]);
            z[i] = make_double2(a.x + b.x, a.y + b.y);
            z[i + half] = make_double2(a.x - b.x, a.y - b.y);
        }
        __syncthreads();
    }
}
// signed wavenumber of bit-reversed position p (Nyquist -> 0: every multiplier here vanishes there, R4)
__device__ __forceinline__ int wavenumber(int p, int N, int logN) {
    int k = (int)(__brev((unsigned)p) >> (32 - logN));
    if (2 * k == N) return 0;
    return (2 * k < N) ? k : k - N;
}

constexpr int FFT_MAX_PER_THREAD = 8;  // ceil(N / blockDim.x) <= 8

static inline int fft_ilog2(int n) {
    int l = 0;
    while ((1 << l) < n) l++;
    return l;
}
static inline int fft_threads(int N) {
    int t = N / 2;
    if (t > 1024) t = 1024;
    if (t < 32) t = 32;
    return t;
}

}  // namespace sww
