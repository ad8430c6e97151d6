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

__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ int fft_log2(int n) { return 31 - __clz(n); }

// in-place forward DIF FFT of z[0..N) in shared memory; output in bit-reversed order.  Two radix-2 stages are fused per pass
// (radix 4 in registers: half the barriers and half the shared-memory traffic), with one plain radix-2 pass when log2 N is odd.
// The arithmetic is exactly that of the radix-2 stages (same twiddles from the table, same order), only the exchange differs.
static __device__ void fft_dif(double2* z, int N, const double2* __restrict__ tw) {
    int half = N >> 1;
    for (; half >= 2; half >>= 2) {                    // stages `half` and `half / 2`
        const int q = half >> 1, lq = fft_log2(q), ts = N / (2 * half);
        for (int t = threadIdx.x; t < N / 4; t += blockDim.x) {
            const int blk = t >> lq, o = t & (q - 1), base = blk * 2 * half + o;
            double2 a0 = z[base], a1 = z[base + q], a2 = z[base + half], a3 = z[base + half + q];
            const double2 w0 = tw[o * ts], w1 = tw[(o + q) * ts], w2 = tw[o * 2 * ts];
            const double2 b0 = cadd(a0, a2), b2 = cmul(csub(a0, a2), w0);
            const double2 b1 = cadd(a1, a3), b3 = cmul(csub(a1, a3), w1);
            z[base] = cadd(b0, b1);
            z[base + q] = cmul(csub(b0, b1), w2);
            z[base + half] = cadd(b2, b3);
            z[base + half + q] = cmul(csub(b2, b3), w2);
        }
        __syncthreads();
    }
    if (half == 1) {                                   // log2 N odd: the last stage alone (twiddle 1)
        for (int t = threadIdx.x; t < N / 2; t += blockDim.x) {
            const double2 a = z[2 * t], b = z[2 * t + 1];
            z[2 * t] = cadd(a, b);
            z[2 * t + 1] = cmul(csub(a, b), tw[0]);
        }
        __syncthreads();
    }
}
// in-place inverse DIT FFT (input bit-reversed, output natural), unscaled; the mirror image of fft_dif
static __device__ void ifft_dit(double2* z, int N, const double2* __restrict__ tw) {
    int half = 1;
    if (fft_log2(N) & 1) {                             // log2 N odd: the first stage alone
        for (int t = threadIdx.x; t < N / 2; t += blockDim.x) {
            const double2 a = z[2 * t], b = cmulc(z[2 * t + 1], tw[0]);
            z[2 * t] = cadd(a, b);
            z[2 * t + 1] = csub(a, b);
        }
        __syncthreads();
        half = 2;
    }
    for (; half < N; half <<= 2) {                     // stages `half` and `2 half`
        const int lh = fft_log2(half), ts = N / (4 * half);   // ts: twiddle stride of the second stage; the first uses 2 ts
        for (int t = threadIdx.x; t < N / 4; t += blockDim.x) {
            const int blk = t >> lh, o = t & (half - 1), base = blk * 4 * half + o;
            const double2 w0 = tw[o * 2 * ts], w1 = tw[o * ts], w2 = tw[(o + half) * ts];
            const double2 a0 = z[base], a1 = cmulc(z[base + half], w0);
            const double2 a2 = z[base + 2 * half], a3 = cmulc(z[base + 3 * half], w0);
            const double2 b0 = cadd(a0, a1), b1 = csub(a0, a1), b2 = cadd(a2, a3), b3 = csub(a2, a3);
            const double2 c2 = cmulc(b2, w1), c3 = cmulc(b3, w2);
            z[base] = cadd(b0, c2);
            z[base + 2 * half] = csub(b0, c2);
            z[base + half] = cadd(b1, c3);
            z[base + 3 * half] = csub(b1, c3);
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
