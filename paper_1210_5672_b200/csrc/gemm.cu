// gemm.cu -- S6: the product with G of (2.8) ("the device also applies G") as an FP64 dense
// contraction on the FP64 tensor pipe: DMMA.8x8x4 = mma.sync.m8n8k4.f64, the only FP64 MMA shape that is native on sm_100a
// (tcgen05 has no f64 kind), with cp.async multi-stage shared-memory staging.
//
//   C[M x Nc] = alpha * A[M x K] * B[K x Nc] + beta * C        (all column-major, leading dimensions lda, ldb, ldc)
//
// Requirements: M % BM == 0, K % BK == 0 (the library pads: N is a power of two >= 16, column counts are padded to 64);
// Nc may be ragged: columns >= Nc of B are never read (zero-filled in shared memory) and columns >= n_valid of C never stored.
// The LU and the triangular solves have their own persistent dataflow kernels (lu.cu); a stage without variational columns
// applies G to one vector through the streamed GEMV at the bottom of this file.
#include "common.cuh"

namespace sww {

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
// src_bytes = 0 -> the 16 destination bytes are zero-filled and the source is not read
__device__ __forceinline__ void cp_async16_zfill(void* smem, const void* gmem, int src_bytes) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int n>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;\n" ::"n"(n));
}

// CTA tile BM x BN, k-slab BK, WR x WC warps, each warp (BM/WR) x (BN/WC).
template <int BM, int BN, int BK, int WR, int WC, int STAGES>
struct GemmCfg {
    static constexpr int THREADS = WR * WC * 32;
    static constexpr int WM = BM / WR, WN = BN / WC;
    static constexpr int FM = WM / 8, FN = WN / 8;  // DMMA fragments per warp
    static constexpr int LDA_S = BM + 4;            // As[k][m], stride = 4 mod 16 doubles -> conflict-free fragment loads
    static constexpr int LDB_S = BK + 4;            // Bs[n][k]
    static constexpr int A_STAGE = BK * LDA_S, B_STAGE = BN * LDB_S;
    static constexpr size_t SMEM = sizeof(double) * (size_t)STAGES * (A_STAGE + B_STAGE);
};

template <class Cfg, int BM, int BN, int BK, int STAGES>
__global__ void __launch_bounds__(Cfg::THREADS) k_gemm_f64(int M, int Nc, int K, double alpha, const double* __restrict__ A, int lda,
                                                           const double* __restrict__ B, int ldb, double beta, double* C, int ldc,
                                                           int n_valid) {
    extern __shared__ __align__(16) double smem[];
    double* As = smem;
    double* Bs = smem + STAGES * Cfg::A_STAGE;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wr = warp % (BM / Cfg::WM), wc = warp / (BM / Cfg::WM);
    const int m0 = blockIdx.x * BM, n0 = blockIdx.y * BN;
    const double* Ag = A + m0;
    const double* Bg = B + (size_t)n0 * ldb;

    auto load_stage = [&](int stage, int kt) {
        double* as = As + stage * Cfg::A_STAGE;
        double* bs = Bs + stage * Cfg::B_STAGE;
        const int k0 = kt * BK;
        // A slab: BK columns of BM contiguous doubles -> BK*BM/2 chunks of 16 B
        for (int c = tid; c < BK * BM / 2; c += Cfg::THREADS) {
            int kk = c / (BM / 2), mm = (c % (BM / 2)) * 2;
            cp_async16(as + kk * Cfg::LDA_S + mm, Ag + (size_t)(k0 + kk) * lda + mm);
        }
        // B slab: BN columns, BK contiguous doubles each
        for (int c = tid; c < BN * BK / 2; c += Cfg::THREADS) {
            int nn = c / (BK / 2), kk = (c % (BK / 2)) * 2;
            bool ok = (n0 + nn) < Nc;
            cp_async16_zfill(bs + nn * Cfg::LDB_S + kk, ok ? Bg + (size_t)nn * ldb + k0 + kk : B, ok ? 16 : 0);
        }
    };

    double acc[Cfg::FM][Cfg::FN][2];
#pragma unroll
    for (int i = 0; i < Cfg::FM; i++)
#pragma unroll
        for (int j = 0; j < Cfg::FN; j++) acc[i][j][0] = acc[i][j][1] = 0.0;

    const int KT = K / BK;
#pragma unroll
    for (int s = 0; s < STAGES - 1; s++) {
        if (s < KT) load_stage(s, s);
        cp_async_commit();
    }
    const int fr = lane >> 2, fk = lane & 3;  // fragment row (or col) and k index of this lane
    for (int kt = 0; kt < KT; kt++) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        {
            int nk = kt + STAGES - 1;
            if (nk < KT) load_stage(nk % STAGES, nk);
            cp_async_commit();
        }
        const double* as = As + (kt % STAGES) * Cfg::A_STAGE + wr * Cfg::WM + fr;
        const double* bs = Bs + (kt % STAGES) * Cfg::B_STAGE + (wc * Cfg::WN + fr) * Cfg::LDB_S;
#pragma unroll
        for (int k4 = 0; k4 < BK; k4 += 4) {
            double af[Cfg::FM], bf[Cfg::FN];
#pragma unroll
            for (int i = 0; i < Cfg::FM; i++) af[i] = as[(k4 + fk) * Cfg::LDA_S + i * 8];
#pragma unroll
            for (int j = 0; j < Cfg::FN; j++) bf[j] = bs[j * 8 * Cfg::LDB_S + k4 + fk];
#pragma unroll
            for (int i = 0; i < Cfg::FM; i++)
#pragma unroll
                for (int j = 0; j < Cfg::FN; j++) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
    }
    cp_async_wait<0>();
    // epilogue: lane holds C(row = fr, cols = 2*fk, 2*fk+1) of each 8x8 fragment
#pragma unroll
    for (int i = 0; i < Cfg::FM; i++) {
        int row = m0 + wr * Cfg::WM + i * 8 + fr;
#pragma unroll
        for (int j = 0; j < Cfg::FN; j++) {
#pragma unroll
            for (int e = 0; e < 2; e++) {
                int col = n0 + wc * Cfg::WN + j * 8 + 2 * fk + e;
                if (col < n_valid) {
                    double* p = C + (size_t)col * ldc + row;
                    double v = alpha * acc[i][j][e];
                    if (beta != 0.0) v = fma(beta, *p, v);
                    *p = v;
                }
            }
        }
    }
}

// small / ragged fallback (M < 64 or K % 16 != 0): one thread per output element
__global__ void k_gemm_naive(int M, int Nc, int K, double alpha, const double* A, int lda, const double* B, int ldb, double beta,
                             double* C, int ldc) {
    int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (i >= M || j >= Nc) return;
    double s = 0.0;
    for (int k = 0; k < K; k++) s = fma(A[(size_t)k * lda + i], B[(size_t)j * ldb + k], s);
    double* p = C + (size_t)j * ldc + i;
    double v = alpha * s;
    if (beta != 0.0) v = fma(beta, *p, v);
    *p = v;
}

template <int BM, int BN, int BK, int WR, int WC, int STAGES>
static int launch_gemm(cudaStream_t st, int M, int Nc, int K, double alpha, const double* A, int lda, const double* B, int ldb,
                       double beta, double* C, int ldc, int n_valid) {
    using Cfg = GemmCfg<BM, BN, BK, WR, WC, STAGES>;
    auto kern = k_gemm_f64<Cfg, BM, BN, BK, STAGES>;
    static DeviceOnce attr_once;
    if (attr_once.first()) {
        SWW_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM));
    }
    dim3 grid(M / BM, (Nc + BN - 1) / BN);
    SWW_BEGIN(KC_GEMM, st);
    kern<<<grid, Cfg::THREADS, Cfg::SMEM, st>>>(M, Nc, K, alpha, A, lda, B, ldb, beta, C, ldc, n_valid);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

int gemm_f64(cudaStream_t st, int M, int Nc, int K, double alpha, const double* A, int lda, const double* B, int ldb, double beta,
             double* C, int ldc, int n_valid) {
    if (M <= 0 || Nc <= 0) return SWW_OK;
    if (n_valid > Nc) n_valid = Nc;
    if (M % 64 != 0 || K % 16 != 0) {
        dim3 grid((M + 63) / 64, n_valid);
        SWW_BEGIN(KC_GEMM, st);
        k_gemm_naive<<<grid, 64, 0, st>>>(M, n_valid, K, alpha, A, lda, B, ldb, beta, C, ldc);
        SWW_LAUNCHED();
        SWW_CUDA(cudaGetLastError());
        return SWW_OK;
    }
    // tile choice: fill the 148 SMs.  128x128 tiles when that still gives >= ~2 waves of CTAs, else 64x64.
    long tiles128 = (M % 128 == 0) ? (long)(M / 128) * ((Nc + 127) / 128) : 0;
    if (tiles128 >= 148) return launch_gemm<128, 128, 16, 4, 2, 3>(st, M, Nc, K, alpha, A, lda, B, ldb, beta, C, ldc, n_valid);
    // 64x64: k-slabs of 32 when K allows (measured on the G product 2048 x 512 x 2048: 0.173 ms against 0.181 with slabs of 16;
    // 128x64, 64x128, 128x32 and 64x32 tiles were all slower there)
    if (K % 32 == 0) return launch_gemm<64, 64, 32, 2, 2, 3>(st, M, Nc, K, alpha, A, lda, B, ldb, beta, C, ldc, n_valid);
    return launch_gemm<64, 64, 16, 2, 2, 3>(st, M, Nc, K, alpha, A, lda, B, ldb, beta, C, ldc, n_valid);
}

// ------------------------------------------------------------------------------------------------ few columns: C += A B as a GEMV
// A stage of the time stepper without variational columns applies G to ONE vector: the tiled kernel would run 8 CTAs over a
// 33 MB matrix.  Here the matrix is streamed once by (M / 32) x ny CTAs: block = 8 warps x 32 rows, warp q takes the columns
// j = q (mod 8) of its block's column range, eight loads in flight per thread; the ny partial sums of a row block are combined by
// the last CTA to arrive (counter per row block, left at zero), in a fixed order -- the result is deterministic.
template <int NC>
__global__ void __launch_bounds__(256) k_gemv_few(int M, int K, const double* __restrict__ A, int lda, const double* __restrict__ B, int ldb,
                                                  double* __restrict__ C, int ldc, double* __restrict__ part, unsigned* __restrict__ count) {
    __shared__ double red[8][NC][32];
    __shared__ unsigned s_last;
    const int lane = threadIdx.x & 31, q = threadIdx.x >> 5;
    const int i = blockIdx.x * 32 + lane;
    const int ny = gridDim.y, jn = K / ny, jb = blockIdx.y * jn, je = jb + jn;
    double acc[NC];
#pragma unroll
    for (int c = 0; c < NC; c++) acc[c] = 0.0;
    for (int j0 = jb + q; j0 < je; j0 += 64) {
        double a[8];
#pragma unroll
        for (int u = 0; u < 8; u++) a[u] = (j0 + 8 * u < je) ? A[(size_t)(j0 + 8 * u) * lda + i] : 0.0;
#pragma unroll
        for (int u = 0; u < 8; u++) {
            const int j = min(j0 + 8 * u, je - 1);
#pragma unroll
            for (int c = 0; c < NC; c++) acc[c] = fma(a[u], B[(size_t)c * ldb + j], acc[c]);
        }
    }
#pragma unroll
    for (int c = 0; c < NC; c++) red[q][c][lane] = acc[c];
    __syncthreads();
    if (q != 0) return;
#pragma unroll
    for (int c = 0; c < NC; c++)
        for (int w = 1; w < 8; w++) acc[c] += red[w][c][lane];
    if (ny > 1) {
#pragma unroll
        for (int c = 0; c < NC; c++) part[((size_t)blockIdx.y * NC + c) * M + i] = acc[c];
        __threadfence();
        __syncwarp();
        if (lane == 0) s_last = (atomicAdd(count + blockIdx.x, 1u) == (unsigned)(ny - 1));
        __syncwarp();
        if (!s_last) return;
        __threadfence();
        if (lane == 0) count[blockIdx.x] = 0;
#pragma unroll
        for (int c = 0; c < NC; c++) {
            acc[c] = 0.0;
            for (int y = 0; y < ny; y++) acc[c] += __ldcg(part + ((size_t)y * NC + c) * M + i);
        }
    }
#pragma unroll
    for (int c = 0; c < NC; c++) C[(size_t)c * ldc + i] += acc[c];
}

// C[M x nc] += A[M x K] B[K x nc], nc <= 4, M a multiple of 32, K a multiple of 64 ny; part: >= 4 * 4 * M doubles, count: M / 32
// zeroed counters (both owned by the handle)
int gemv_few_f64(cudaStream_t st, int M, int nc, int K, const double* A, int lda, const double* B, int ldb, double* C, int ldc, double* part,
                 unsigned* count) {
    const int ny = (K % 256 == 0 && M >= 256) ? 4 : 1;
    dim3 grid(M / 32, ny);
    SWW_BEGIN(KC_GEMM, st);
    switch (nc) {
        case 1: k_gemv_few<1><<<grid, 256, 0, st>>>(M, K, A, lda, B, ldb, C, ldc, part, count); break;
        case 2: k_gemv_few<2><<<grid, 256, 0, st>>>(M, K, A, lda, B, ldb, C, ldc, part, count); break;
        case 3: k_gemv_few<3><<<grid, 256, 0, st>>>(M, K, A, lda, B, ldb, C, ldc, part, count); break;
        default: k_gemv_few<4><<<grid, 256, 0, st>>>(M, K, A, lda, B, ldb, C, ldc, part, count); break;
    }
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

}  // namespace sww
