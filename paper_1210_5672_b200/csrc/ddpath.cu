// ddpath.cu -- double-double ("quadruple precision") kernels of the DtN path, all error-free-transformation FMA
// code on the CUDA cores, and the two flows that use them:
//   (1) the ACCURATE BASE STATE (both precisions): W0 = G phi0, u, v of (2.9) with mu0 carried as a dd pair out
//       of iterative refinement, differentiated by the dd circulant, so that the noise of a first-order operator applied to a
//       rounded fp64 density (~N eps) does not get amplified a second time by the linearized solve;
//   (2) the dd DtN apply / linearized apply: "iterative refinement around the double-precision LU ... residuals by a blocked quad
//       matrix-matrix multiply": mu = sum of fp64 corrections, each from the fp64 LU applied to a dd residual.
// Product code; shares nothing with oracle/.
#include "common.cuh"
#include "dd.cuh"
#include "ddfft.cuh"

namespace sww {

// Solves per right-hand side in the refinement around the fp64 factors.  The compensated fp64 solve returns hi + lo with a
// relative error near 1e-17, so the second solve (on the dd residual of the first) already lands below the dd rounding of the
// residual itself: measured E_col with 2 and with 3 solves is the same to two digits (config 4: 1.48e-28 / 1.43e-28, N = 1024:
// 8.83e-28 / 8.86e-28; bar 1e-25), and the third solve with its dd residual GEMM was a quarter of the dd step.
constexpr int DD_SWEEPS = 2;

// ------------------------------------------------------------------------------------------------ dd circulants: D and H
// mode 0: out = D f,  coefficient (1/2)(-1)^m cot(pi m/N)                       (Fourier differentiation, Nyquist symbol 0, R4)
// mode 1: out = H f,  coefficient (1/N) cot(pi m/N) (1 - (-1)^m) = 4 c0[m]/N for odd m, 0 for even m   (symbol -i sgn k)
// Both kernels are odd in m, so out_i = sum_{m=1}^{N/2-1} coef[m] (f_{i-m} - f_{i+m}).  Four warps per output node (two nodes per
// CTA): the time of the kernel is the length of the per-lane chain of dependent dd operations behind scattered loads.
// blockIdx.y = 1 (two-vector launches) applies the same circulant to a second, independent vector f2 -> out2.
__global__ void __launch_bounds__(256) k_circ_dd(int N, int mode, const double* __restrict__ dc, const double* __restrict__ c0,
                                                 const double* __restrict__ f, double* __restrict__ out, const double* __restrict__ f2,
                                                 double* __restrict__ out2) {
    __shared__ double part[2][4][2];
    if (blockIdx.y) {
        f = f2;
        out = out2;
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, node = warp >> 2, q = warp & 3;
    const int i = blockIdx.x * 2 + node, mask = N - 1;
    const int l128 = q * 32 + lane;
    // four independent dd accumulators per lane: one dd multiply-add is a chain of ~30 dependent fp64 instructions
    dd acc4[4] = {{0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}};
    const double hs = (mode == 0) ? 1.0 : 4.0 / (double)N;  // exact (power of two)
    const double* coef = (mode == 0) ? dc : c0;
    const int step = (mode == 0) ? 1 : 2;                   // H: odd m only
    if (i < N) {
        // both tables hold 0 at m = N/2, so when the stride divides N/2 the last group may run over it unguarded and the
        // 24 loads of a group are issued together (the kernel is bound by their latency otherwise)
        const bool full = ((N / 2) % (4 * 128 * step)) == 0;
        for (int m0 = 1 + step * l128; m0 < N / 2; m0 += 4 * 128 * step) {
            if (full) {
                dd c[4], a[4], b[4];
#pragma unroll
                for (int u = 0; u < 4; u++) {
                    const int m = m0 + u * 128 * step;
                    c[u] = dd_load(coef, N, m);
                    a[u] = dd_load(f, N, (i - m) & mask);
                    b[u] = dd_load(f, N, (i + m) & mask);
                }
#pragma unroll
                for (int u = 0; u < 4; u++) acc4[u] = dd_fma(dd{c[u].hi * hs, c[u].lo * hs}, dd_sub(a[u], b[u]), acc4[u]);
            } else {
#pragma unroll
                for (int u = 0; u < 4; u++) {
                    const int m = m0 + u * 128 * step;
                    if (m < N / 2) {
                        dd c = dd_load(coef, N, m);
                        c.hi *= hs;
                        c.lo *= hs;
                        dd a = dd_load(f, N, (i - m) & mask), b = dd_load(f, N, (i + m) & mask);
                        acc4[u] = dd_fma(c, dd_sub(a, b), acc4[u]);
                    }
                }
            }
        }
    }
    dd acc = dd_add(dd_add(acc4[0], acc4[1]), dd_add(acc4[2], acc4[3]));
    acc = dd_warp_sum(acc);
    if (lane == 0) {
        part[node][q][0] = acc.hi;
        part[node][q][1] = acc.lo;
    }
    __syncthreads();
    if (q == 0 && lane == 0 && i < N) {
        for (int r = 1; r < 4; r++) acc = dd_add(acc, dd{part[node][r][0], part[node][r][1]});
        dd_store(out, N, i, acc);
    }
}

int circ_dd(sww_dtn_s* d, int mode, const double* in, double* out) {
    const int N = d->N;
    SWW_BEGIN(KC_OTHER, d->stream);
    k_circ_dd<<<(N + 1) / 2, 256, 0, d->stream>>>(N, mode, d->tab->dc, d->tab->c0, in, out, nullptr, nullptr);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}
// two independent vectors in one launch
static int circ_dd2(sww_dtn_s* d, int mode, const double* in1, double* out1, const double* in2, double* out2) {
    const int N = d->N;
    SWW_BEGIN(KC_OTHER, d->stream);
    k_circ_dd<<<dim3((N + 1) / 2, 2), 256, 0, d->stream>>>(N, mode, d->tab->dc, d->tab->c0, in1, out1, in2, out2);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

// ------------------------------------------------------------------------------------------------ dd mat-vec (one column)
// y = zs * z + beta * x + alpha * (A x), accumulated in dd.  A column-major N x N, fp64 (Alo == nullptr) or dd (Alo = lo plane).
// x, z, y dd planar (2N).  y_f64 (optional) receives y rounded to fp64.  zs, beta, alpha must be powers of two or 0 (exact).
// Block = 8 warps x 32 rows: warp q sums the columns j = q (mod 8) of this block's column range for 32 consecutive rows
// (coalesced 256 B per load, eight loads in flight per thread: the kernel streams A once and is bound by memory latency).
// gridDim.y blocks share a row block: each writes its partial dd sums to part[y][2][N]; the last one to arrive (counter per
// row block, left at zero again) adds them up and applies the epilogue.
__global__ void __launch_bounds__(256) k_matvec_dd(int N, const double* __restrict__ A, const double* __restrict__ Alo,
                                                   const double* __restrict__ x, double zs, const double* __restrict__ z, double beta,
                                                   double alpha, double* __restrict__ y, double* __restrict__ y_f64,
                                                   double* __restrict__ part, unsigned* __restrict__ count) {
    __shared__ double red_hi[8][32], red_lo[8][32];
    __shared__ unsigned s_last;
    const int lane = threadIdx.x & 31, q = threadIdx.x >> 5;
    const int i = blockIdx.x * 32 + lane;
    const int ny = gridDim.y, jn = N / ny, jb = blockIdx.y * jn, je = jb + jn;
    dd acc4[4] = {{0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}};  // independent chains (see k_circ_dd)
    if (i < N) {
        if ((jn & 63) == 0) {
            for (int j0 = jb + q; j0 < je; j0 += 64) {
                dd a[8], xj[8];
#pragma unroll
                for (int u = 0; u < 8; u++) {
                    const int j = j0 + 8 * u;
                    const size_t o = (size_t)j * N + i;
                    a[u] = dd{A[o], Alo ? Alo[o] : 0.0};
                    xj[u] = dd_load(x, N, j);
                }
#pragma unroll
                for (int u = 0; u < 8; u++) acc4[u & 3] = dd_fma(a[u], xj[u], acc4[u & 3]);
            }
        } else {
            for (int j = jb + q; j < je; j += 8) {
                dd xj = dd_load(x, N, j);
                size_t o = (size_t)j * N + i;
                acc4[0] = dd_fma(dd{A[o], Alo ? Alo[o] : 0.0}, xj, acc4[0]);
            }
        }
    }
    dd acc = dd_add(dd_add(acc4[0], acc4[1]), dd_add(acc4[2], acc4[3]));
    red_hi[q][lane] = acc.hi;
    red_lo[q][lane] = acc.lo;
    __syncthreads();
    if (q != 0) return;
    for (int w = 1; w < 8; w++) acc = dd_add(acc, dd{red_hi[w][lane], red_lo[w][lane]});
    if (ny > 1) {
        if (i < N) {
            part[((size_t)blockIdx.y * 2) * N + i] = acc.hi;
            part[((size_t)blockIdx.y * 2 + 1) * N + i] = acc.lo;
        }
        __threadfence();
        __syncwarp();
        if (lane == 0) s_last = (atomicAdd(count + blockIdx.x, 1u) == (unsigned)(ny - 1));
        __syncwarp();
        if (!s_last) return;
        __threadfence();
        if (lane == 0) count[blockIdx.x] = 0;  // ready for the next launch
        acc = dd{0.0, 0.0};
        if (i < N)
            for (int c = 0; c < ny; c++)
                acc = dd_add(acc, dd{__ldcg(part + ((size_t)c * 2) * N + i), __ldcg(part + ((size_t)c * 2 + 1) * N + i)});
    }
    if (i < N) {
        dd r{alpha * acc.hi, alpha * acc.lo};
        if (beta != 0.0) {
            dd xi = dd_load(x, N, i);
            r = dd_add(r, dd{beta * xi.hi, beta * xi.lo});
        }
        if (zs != 0.0) {
            dd zi = dd_load(z, N, i);
            r = dd_add(r, dd{zs * zi.hi, zs * zi.lo});
        }
        dd_store(y, N, i, r);
        if (y_f64) y_f64[i] = r.hi;
    }
}

static int matvec_dd(sww_dtn_s* d, const double* A, const double* Alo, const double* x, double zs, const double* z, double beta,
                     double alpha, double* y, double* y_f64) {
    const int N = d->N;
    // column splits: the per-thread chain of dd operations behind the loads sets the time (part = d->bp_part: bp_chunks * 4 * N
    // doubles >= ny * 2 * N; every split keeps a multiple of 64 columns)
    const int ny = (N >= 2048 && d->bp_chunks >= 8) ? 16 : ((N >= 512 && d->bp_chunks >= 2) ? 4 : 1);
    SWW_BEGIN(KC_DDGEMM, d->stream);
    k_matvec_dd<<<dim3((N + 31) / 32, ny), 256, 0, d->stream>>>(N, A, Alo, x, zs, z, beta, alpha, y, y_f64, d->bp_part, d->mv_count);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

// ------------------------------------------------------------------------------------------------ dd GEMM (many columns)
// Y = zs * Z + beta * X + alpha * (A X): A dd (or fp64) N x N, X, Z, Y dd planar N x ncols (plane size L = N * ld_cols).
// CTA tile 64 rows x 32 columns, 256 threads, thread tile 4 x 2 (rows ty + 16 r, columns tx + 16 c), k-slab 16.
// CN = columns per thread: 2 (tile 64 x 32) or 1 (tile 64 x 16, used when there would be fewer than 100 wide tiles).
constexpr int DG_BM = 64, DG_BK = 16, DG_XLD = DG_BK + 2;  // even padding: 16-byte cp.async destinations
// 16 bytes global -> shared, zero-filled when !valid (cp.async src-size 0)
__device__ __forceinline__ void dg_cp16(void* smem, const void* gmem, bool valid) {
    unsigned s_ = (unsigned)__cvta_generic_to_shared(smem);
    int sz = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s_), "l"(gmem), "r"(sz));
}
template <int CN>
struct DgSmem {
    static constexpr int BN = 16 * CN;
    static constexpr int A_PLANE = DG_BK * DG_BM, X_PLANE = BN * DG_XLD;
    static constexpr int STAGE = 2 * A_PLANE + 2 * X_PLANE;  // doubles: A hi, A lo, X hi, X lo
    static constexpr int BYTES = 2 * STAGE * (int)sizeof(double);
};
// The k-slabs are double-buffered through cp.async: slab s + 1 is in flight while slab s is multiplied.
template <int CN>
__global__ void __launch_bounds__(256) k_gemm_dd(int N, int ncols, size_t L, const double* __restrict__ A, const double* __restrict__ Alo,
                                                 const double* __restrict__ X, double zs, const double* __restrict__ Z, double beta,
                                                 double alpha, double* __restrict__ Y, double* __restrict__ Y_f64) {
    using S = DgSmem<CN>;
    constexpr int DG_BN = S::BN;
    extern __shared__ __align__(16) double dg_sm[];
    const int tid = threadIdx.x, ty = tid & 15, tx = tid >> 4;
    const int i0 = blockIdx.x * DG_BM, c0 = blockIdx.y * DG_BN;
    auto issue = [&](int k0, int st) {
        double* base = dg_sm + st * S::STAGE;
        for (int e = tid; e < S::A_PLANE / 2; e += 256) {  // A: rows contiguous
            const int kk = e / (DG_BM / 2), ii = (e % (DG_BM / 2)) * 2;
            const size_t o = (size_t)(k0 + kk) * N + i0 + ii;
            dg_cp16(base + kk * DG_BM + ii, A + o, true);
            dg_cp16(base + S::A_PLANE + kk * DG_BM + ii, Alo ? Alo + o : A + o, Alo != nullptr);
        }
        for (int e = tid; e < DG_BN * DG_BK / 2; e += 256) {  // X: k contiguous
            const int cc = e / (DG_BK / 2), kk = (e % (DG_BK / 2)) * 2;
            const int c = c0 + cc;
            const bool ok = c < ncols;
            const size_t o = (size_t)(ok ? c : 0) * N + k0 + kk;
            dg_cp16(base + 2 * S::A_PLANE + cc * DG_XLD + kk, X + o, ok);
            dg_cp16(base + 2 * S::A_PLANE + S::X_PLANE + cc * DG_XLD + kk, X + L + o, ok);
        }
        asm volatile("cp.async.commit_group;\n" ::);
    };
    dd acc[4][CN];
#pragma unroll
    for (int r = 0; r < 4; r++)
#pragma unroll
        for (int c = 0; c < CN; c++) acc[r][c] = dd{0.0, 0.0};
    issue(0, 0);
    for (int k0 = 0, st = 0; k0 < N; k0 += DG_BK, st ^= 1) {
        if (k0 + DG_BK < N) {
            issue(k0 + DG_BK, st ^ 1);  // its buffer was released by the barrier that ended the previous slab
            asm volatile("cp.async.wait_group 1;\n" ::);
        } else {
            asm volatile("cp.async.wait_group 0;\n" ::);
        }
        __syncthreads();
        const double* As_hi = dg_sm + st * S::STAGE;
        const double* As_lo = As_hi + S::A_PLANE;
        const double* Xs_hi = As_hi + 2 * S::A_PLANE;
        const double* Xs_lo = Xs_hi + S::X_PLANE;
#pragma unroll 4
        for (int kk = 0; kk < DG_BK; kk++) {
            dd a[4], x[CN];
#pragma unroll
            for (int r = 0; r < 4; r++) a[r] = dd{As_hi[kk * DG_BM + ty + 16 * r], As_lo[kk * DG_BM + ty + 16 * r]};
#pragma unroll
            for (int c = 0; c < CN; c++) x[c] = dd{Xs_hi[(tx + 16 * c) * DG_XLD + kk], Xs_lo[(tx + 16 * c) * DG_XLD + kk]};
#pragma unroll
            for (int r = 0; r < 4; r++)
#pragma unroll
                for (int c = 0; c < CN; c++) dd_fma_lazy(a[r], x[c], acc[r][c]);
        }
        // the accumulators are renormalised once per k-slab (16 terms), not per term: 12 instead of 15 flops per multiply-add
#pragma unroll
        for (int r = 0; r < 4; r++)
#pragma unroll
            for (int c = 0; c < CN; c++) acc[r][c] = dd_renorm(acc[r][c]);
        __syncthreads();
    }
#pragma unroll
    for (int c = 0; c < CN; c++) {
        int col = c0 + tx + 16 * c;
        if (col >= ncols) continue;
#pragma unroll
        for (int r = 0; r < 4; r++) {
            int i = i0 + ty + 16 * r;
            size_t o = (size_t)col * N + i;
            dd v{alpha * acc[r][c].hi, alpha * acc[r][c].lo};
            if (beta != 0.0) v = dd_add(v, dd{beta * X[o], beta * X[L + o]});
            if (zs != 0.0) v = dd_add(v, dd{zs * Z[o], zs * Z[L + o]});
            Y[o] = v.hi;
            Y[L + o] = v.lo;
            if (Y_f64) Y_f64[o] = v.hi;
        }
    }
}

// N < 64 (one tile would be mostly padding): Y = zs Z + beta X + alpha A X, one thread per element
__global__ void k_gemm_dd_small(int N, size_t L, const double* __restrict__ A, const double* __restrict__ Alo, const double* __restrict__ X,
                                double zs, const double* __restrict__ Z, double beta, double alpha, double* __restrict__ Y,
                                double* __restrict__ Y_f64) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y;
    if (i >= N) return;
    dd acc{0.0, 0.0};
    for (int k = 0; k < N; k++) {
        const size_t o = (size_t)k * N + i, ox = (size_t)c * N + k;
        acc = dd_fma(dd{A[o], Alo ? Alo[o] : 0.0}, dd{X[ox], X[L + ox]}, acc);
    }
    const size_t o = (size_t)c * N + i;
    dd v{alpha * acc.hi, alpha * acc.lo};
    if (beta != 0.0) v = dd_add(v, dd{beta * X[o], beta * X[L + o]});
    if (zs != 0.0) v = dd_add(v, dd{zs * Z[o], zs * Z[L + o]});
    Y[o] = v.hi;
    Y[L + o] = v.lo;
    if (Y_f64) Y_f64[o] = v.hi;
}

static int gemm_dd(sww_dtn_s* d, int ncols, size_t L, const double* A, const double* Alo, const double* X, double zs, const double* Z,
                   double beta, double alpha, double* Y, double* Y_f64) {
    const int N = d->N;
    if (N < DG_BM) {  // N = 16, 32: one thread per output element
        dim3 grid((N + 31) / 32, ncols);
        SWW_BEGIN(KC_DDGEMM, d->stream);
        k_gemm_dd_small<<<grid, 32, 0, d->stream>>>(N, L, A, Alo, X, zs, Z, beta, alpha, Y, Y_f64);
        SWW_LAUNCHED();
        SWW_CUDA(cudaGetLastError());
        return SWW_OK;
    }
    const bool narrow = (long)(N / DG_BM) * ((ncols + 31) / 32) < 100;  // too few wide tiles to occupy the chip
    const int bn = narrow ? 16 : 32;
    dim3 grid(N / DG_BM, (ncols + bn - 1) / bn);
    SWW_BEGIN(KC_DDGEMM, d->stream);
    static DeviceOnce attr_once;
    if (attr_once.first()) {
        SWW_CUDA(cudaFuncSetAttribute(k_gemm_dd<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, DgSmem<1>::BYTES));
        SWW_CUDA(cudaFuncSetAttribute(k_gemm_dd<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, DgSmem<2>::BYTES));
    }
    if (narrow)
        k_gemm_dd<1><<<grid, 256, DgSmem<1>::BYTES, d->stream>>>(N, ncols, L, A, Alo, X, zs, Z, beta, alpha, Y, Y_f64);
    else
        k_gemm_dd<2><<<grid, 256, DgSmem<2>::BYTES, d->stream>>>(N, ncols, L, A, Alo, X, zs, Z, beta, alpha, Y, Y_f64);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

// ------------------------------------------------------------------------------------------------ pointwise dd helpers
// mu += delta + delta_lo (the compensated fp64 solve's two words), planar with plane size L; first sweep: mu = delta + delta_lo
__global__ void k_dd_axpy_f64(size_t n, size_t L, int first, const double* __restrict__ delta, const double* __restrict__ delta_lo,
                              double* __restrict__ mu) {
    size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    if (first) {
        mu[e] = delta[e];
        mu[L + e] = delta_lo[e];
    } else {
        dd m = dd_add(dd{mu[e], mu[L + e]}, dd{delta[e], delta_lo[e]});
        mu[e] = m.hi;
        mu[L + e] = m.lo;
    }
}
// planar copy with a different plane stride: dst (plane Ld) <- src (plane Ls), n elements per plane; src_lo may be absent
__global__ void k_dd_copy(size_t n, size_t Ls, size_t Ld, int has_lo, const double* __restrict__ src, double* __restrict__ dst,
                          double* __restrict__ dst_f64) {
    size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    double hi = src[e], lo = has_lo ? src[Ls + e] : 0.0;
    dst[e] = hi;
    dst[Ld + e] = lo;
    if (dst_f64) dst_f64[e] = hi;
}
// (2.9), in dd
// W0 = Wa (+ Wb when given; stored to W0out) and the surface velocities (2.9) from it
// xE (refined mesh, else nullptr): the inputs are alpha-derivatives and the bracket of (2.8); eta'(x) = d1 / xi', phi'(x) = dphi / xi',
// G phi = W / |xi'|, and phi' and G phi are stored back in that form (dphi_out, W0out)
__global__ void k_base_uv_dd(int N, const double* __restrict__ d1, const double* dphi, const double* Wa, const double* Wb,
                             double* W0out, double* __restrict__ u, double* __restrict__ v, const double* __restrict__ xE, double* dphi_out) {
    int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    dd e1 = dd_load(d1, N, j), p = dd_load(dphi, N, j), w = dd_load(Wa, N, j);
    if (Wb) w = dd_add(w, dd_load(Wb, N, j));
    if (xE) {
        const dd e = dd_load(xE, N, j);
        e1 = dd_div(e1, e);
        p = dd_div(p, e);
        w = dd_div(w, e);
        dd_store(dphi_out, N, j, p);
    }
    if (Wb || xE) dd_store(W0out, N, j, w);
    dd den = dd_add_d(dd_sqr(e1), 1.0);
    dd_store(u, N, j, dd_div(dd_sub(p, dd_mul(e1, w)), den));
    dd_store(v, N, j, dd_div(dd_add(dd_mul(e1, p), w), den));
}
// linearized right-hand sides in dd: B_c = dphi_c - v deta_c (B.1d) ; T_c = u deta_c ; also the fp64 rounding of B for the LU
__global__ void k_rhs_lin_dd(int N, size_t total, size_t Lin, size_t Lws, const double* __restrict__ deta, const double* __restrict__ dphi,
                             const double* __restrict__ u, const double* __restrict__ v, double* __restrict__ B, double* __restrict__ T,
                             double* __restrict__ R) {
    size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= total) return;
    int j = (int)(e & (size_t)(N - 1));
    dd de{deta[e], deta[Lin + e]}, dp{dphi[e], dphi[Lin + e]};
    dd uj = dd_load(u, N, j), vj = dd_load(v, N, j);
    dd b = dd_sub(dp, dd_mul(vj, de));
    dd t = dd_mul(uj, de);
    B[e] = b.hi;
    B[Lws + e] = b.lo;
    T[e] = t.hi;
    T[Lws + e] = t.lo;
    R[e] = b.hi;
}

// Gam_c = D M_c ;  W_c = |D| M_c / 2 - (T ? D T_c : 0), dd planar in/out (plane sizes Lws for M, T, Gam; Lw for W)
__global__ void __launch_bounds__(512) k_spectral_gamma_w_dd(int N, int logN, const double* __restrict__ cs, const double* __restrict__ sn,
                                                             size_t Lws, size_t Lw, const double* __restrict__ M, const double* __restrict__ T,
                                                             double* __restrict__ Gam, double* __restrict__ W, int ncols, int w_cols) {
    extern __shared__ __align__(16) unsigned char dd_fft_sm[];
    cdd* z = reinterpret_cast<cdd*>(dd_fft_sm);
    cdd* zt = z + N;  // second buffer: transform of T (only touched when T != nullptr)
    const int c0 = 2 * blockIdx.x, c1 = c0 + 1;
    const bool has1 = c1 < ncols;
    const double rN = 1.0 / (double)N;
    if (T) {
        for (int j = threadIdx.x; j < N; j += blockDim.x) {
            size_t o0 = (size_t)c0 * N + j, o1 = (size_t)c1 * N + j;
            zt[j] = cdd{dd{T[o0], T[Lws + o0]}, has1 ? dd{T[o1], T[Lws + o1]} : dd{0, 0}};
        }
        __syncthreads();
        fft_dif_dd(zt, N, cs, sn);
    }
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        size_t o0 = (size_t)c0 * N + j, o1 = (size_t)c1 * N + j;
        z[j] = cdd{dd{M[o0], M[Lws + o0]}, has1 ? dd{M[o1], M[Lws + o1]} : dd{0, 0}};
    }
    __syncthreads();
    fft_dif_dd(z, N, cs, sn);
    // zt <- |k|/2 zhat - i k that (kept for the second inverse transform);  z <- i k zhat
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        double k = (double)wavenumber_dd(p, N, logN) * rN;  // exact: integer times a power of two
        cdd v = z[p];
        cdd w{dd_mul_d(v.re, 0.5 * fabs(k)), dd_mul_d(v.im, 0.5 * fabs(k))};
        if (T) {
            cdd t = zt[p];
            w.re = dd_add(w.re, dd_mul_d(t.im, k));
            w.im = dd_sub(w.im, dd_mul_d(t.re, k));
        }
        zt[p] = w;
        z[p] = cdd{dd_mul_d(v.im, -k), dd_mul_d(v.re, k)};
    }
    __syncthreads();
    ifft_dit_dd(z, N, cs, sn);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        cdd v = z[j];
        size_t o0 = (size_t)c0 * N + j, o1 = (size_t)c1 * N + j;
        Gam[o0] = v.re.hi;
        Gam[Lws + o0] = v.re.lo;
        Gam[o1] = has1 ? v.im.hi : 0.0;
        Gam[Lws + o1] = has1 ? v.im.lo : 0.0;
    }
    ifft_dit_dd(zt, N, cs, sn);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        cdd v = zt[j];
        size_t o0 = (size_t)c0 * N + j, o1 = (size_t)c1 * N + j;
        if (c0 < w_cols) {
            W[o0] = v.re.hi;
            W[Lw + o0] = v.re.lo;
        }
        if (c1 < w_cols) {
            W[o1] = v.im.hi;
            W[Lw + o1] = v.im.lo;
        }
    }
}

// One multiplier per launch, one complex dd array in shared memory (N = 4096: 128 KB; the fused kernel above needs two):
// out_c (+)= sign * m(D) in_c for the column pair (2 b, 2 b + 1);  mode 0: m = i k (D), mode 1: m = |k| / 2.
__global__ void __launch_bounds__(512) k_spectral_pass_dd(int N, int logN, const double* __restrict__ cs, const double* __restrict__ sn,
                                                          int mode, double sign, int accumulate, size_t Lin, size_t Lout,
                                                          const double* __restrict__ in, double* __restrict__ out, int ncols, int out_cols,
                                                          int zero_partner) {
    extern __shared__ __align__(16) unsigned char dd_fft_sm[];
    cdd* z = reinterpret_cast<cdd*>(dd_fft_sm);
    const int c0 = 2 * blockIdx.x, c1 = c0 + 1;
    const bool has1 = c1 < ncols;
    const double rN = 1.0 / (double)N;
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const size_t o0 = (size_t)c0 * N + j, o1 = (size_t)c1 * N + j;
        z[j] = cdd{dd{in[o0], in[Lin + o0]}, has1 ? dd{in[o1], in[Lin + o1]} : dd{0, 0}};
    }
    __syncthreads();
    fft_dif_dd(z, N, cs, sn);
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        const double k = (double)wavenumber_dd(p, N, logN) * rN;  // exact: an integer times a power of two (1/N of the inverse folded in)
        const double a = sign * k, h = sign * 0.5 * fabs(k);
        const cdd v = z[p];
        z[p] = (mode == 0) ? cdd{dd_mul_d(v.im, -a), dd_mul_d(v.re, a)} : cdd{dd_mul_d(v.re, h), dd_mul_d(v.im, h)};
    }
    __syncthreads();
    ifft_dit_dd(z, N, cs, sn);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const cdd v = z[j];
        const size_t o0 = (size_t)c0 * N + j, o1 = (size_t)c1 * N + j;
        if (c0 < out_cols) {
            const dd r = accumulate ? dd_add(dd{out[o0], out[Lout + o0]}, v.re) : v.re;
            out[o0] = r.hi;
            out[Lout + o0] = r.lo;
        }
        if (c1 < out_cols) {
            const dd r = accumulate ? dd_add(dd{out[o1], out[Lout + o1]}, v.im) : v.im;
            out[o1] = r.hi;
            out[Lout + o1] = r.lo;
        } else if (zero_partner && !has1) {  // padded buffer: the odd partner column is zeroed
            out[o1] = 0.0;
            out[Lout + o1] = 0.0;
        }
    }
}

static int ilog2(int n) {
    int l = 0;
    while ((1 << l) < n) l++;
    return l;
}

// two independent sums in one launch: o1 = a1 + b1, o2 = a2 + b2 (dd planar, plane size N; outputs may alias their inputs)
__global__ void k_dd_add2(int N, const double* a1, const double* b1, double* o1, const double* a2, const double* b2, double* o2) {
    int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    dd_store(o1, N, j, dd_add(dd_load(a1, N, j), dd_load(b1, N, j)));
    dd_store(o2, N, j, dd_add(dd_load(a2, N, j), dd_load(b2, N, j)));
}

// ------------------------------------------------------------------------------------------------ flow (1): accurate base state
// phi0: dd planar when d->prec == SWW_DD (lo plane at phi0 + phi_plane; 0 = N), N doubles otherwise.  Uses d->tmp (14N doubles) and column 0 of ws.T|R and ws.S.
//   dd handle : mu0 by refinement sweeps around the fp64 LU with residuals from the stored dd K; W0 from the stored dd G.
//   f64 handle: the stored K, G are fp64-rounded, which is not enough here (their rounding alone leaves ~2e-15 of white noise in
//               v at N = 2048, and every linearized column multiplies v into its right-hand side and differentiates: 3e-12 in
//               the output).  One fused pass evaluates the kernels in dd on the fly (assembly.cu, base_pass_dd):
//               mu~ = LU \ phi0 ; gam~ = D mu~ ; [res, w~] = [phi0 - mu~/2 - K mu~, G gam~] (dd) ; delta = LU \ res ;
//               mu0 = mu~ + delta ; W0 = H D mu0 / 2 + w~ + G_f64 (D delta)   (2.7), (2.8).
int accurate_base(sww_dtn_s* d, const double* phi0, size_t phi_plane) {
    const int N = d->N;
    cudaStream_t st = d->stream;
    const bool isdd = d->prec == SWW_DD;
    const size_t NN = (size_t)N * N;
    double* b = d->tmp;             // phi0 as dd planar
    double* mu = d->tmp + 2 * N;    // mu0 dd
    double* gam = d->tmp + 4 * N;   // gamma = D mu0
    double* hg = d->tmp + 6 * N;    // H gamma
    double* res = d->tmp + 8 * N;   // residual dd / delta dd
    double* wt = d->tmp + 10 * N;   // w~ = G gam~
    double* dgam = d->tmp + 12 * N; // D delta
    // fp64 scratch column for the LU solves (+ its low word in ws.S)
    double* rcol = isdd ? d->ws.R : d->ws.T;
    double* rlo = d->ws.S;
    unsigned blocks = (unsigned)((N + 255) / 256);
    SWW_BEGIN(KC_OTHER, st);
    k_dd_copy<<<blocks, 256, 0, st>>>((size_t)N, phi_plane ? phi_plane : (size_t)N, (size_t)N, isdd ? 1 : 0, phi0, b, rcol);
    SWW_LAUNCHED();
    if (isdd) {
        const int nsweep = DD_SWEEPS;
        for (int s = 0; s < nsweep; s++) {
            SWW_TRY(run_solve(d, rcol, rlo, 1));  // delta = (LU)^{-1} round(r)
            SWW_BEGIN(KC_OTHER, st);
            k_dd_axpy_f64<<<blocks, 256, 0, st>>>((size_t)N, (size_t)N, s == 0, rcol, rlo, mu);
            SWW_LAUNCHED();
            if (s + 1 < nsweep)  // r = b - mu/2 - K mu   (2.7)
                SWW_TRY(matvec_dd(d, d->K, d->K + NN, mu, 1.0, b, -0.5, -1.0, res, rcol));
        }
        SWW_TRY(circ_dd(d, 0, mu, gam));                                                   // gamma = D mu
        SWW_TRY(circ_dd(d, 1, gam, hg));                                                   // H gamma
        SWW_TRY(matvec_dd(d, d->G, d->G + NN, gam, 0.5, hg, 0.0, 1.0, d->bW0, nullptr));   // W0 = H gamma / 2 + G gamma   (2.8)
    } else {
        SWW_TRY(run_solve(d, rcol, rlo, 1));
        SWW_BEGIN(KC_OTHER, st);
        k_dd_axpy_f64<<<blocks, 256, 0, st>>>((size_t)N, (size_t)N, 1, rcol, rlo, mu);     // mu~
        SWW_LAUNCHED();
        SWW_TRY(circ_dd2(d, 0, mu, gam, b, d->bphi));                                      // gam~ = D mu~ ; phi0' = D phi0
        SWW_TRY(base_pass_dd(d, b, mu, gam, res, rcol, wt));
        SWW_TRY(run_solve(d, rcol, rlo, 1));                                               // delta
        SWW_BEGIN(KC_OTHER, st);
        k_dd_axpy_f64<<<blocks, 256, 0, st>>>((size_t)N, (size_t)N, 1, rcol, rlo, res);    // res <- delta as dd
        SWW_LAUNCHED();
        SWW_TRY(circ_dd(d, 0, res, dgam));                                                 // D delta
        SWW_BEGIN(KC_OTHER, st);
        k_dd_add2<<<blocks, 256, 0, st>>>(N, mu, res, mu, gam, dgam, gam);                 // mu0 = mu~ + delta ; gamma = D mu0
        SWW_LAUNCHED();
        SWW_TRY(circ_dd(d, 1, gam, hg));                                                   // H gamma
        SWW_TRY(matvec_dd(d, d->G, nullptr, dgam, 0.5, hg, 0.0, 1.0, res, nullptr));       // H gamma / 2 + G_f64 (D delta)
    }
    if (isdd) SWW_TRY(circ_dd(d, 0, b, d->bphi));                                          // phi0' (fp64 handles: done with gam~ above)
    SWW_BEGIN(KC_OTHER, st);
    const double* xE = d->mesh_on ? d->mesh.xE : nullptr;
    if (isdd) k_base_uv_dd<<<blocks, 256, 0, st>>>(N, d->d1, d->bphi, d->bW0, nullptr, d->bW0, d->bu, d->bv, xE, d->bphi);
    else k_base_uv_dd<<<blocks, 256, 0, st>>>(N, d->d1, d->bphi, res, wt, d->bW0, d->bu, d->bv, xE, d->bphi);   // W0 = res + w~ (2.8), then u, v
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

// ------------------------------------------------------------------------------------------------ plain fp64 base state
// (2.9) for a state that is NOT linearized about: phi0', W0 = G phi0, u, v straight from the fp64 pipeline (one solve, one
// spectral pass, one product with G), written as dd pairs with zero low words.  The time stepper without variational columns
// uses it for N <= 1024: there u, v enter the right-hand sides of (2.1) only, nothing differentiates them a second time, and the
// rounding noise of the first-order operator (~2 N eps) stays three digits under the parity bar (SURVEY.md section 0, fact 4:
// fp64 against long double over config 2's full period: 3e-14 / 2e-13).
__global__ void k_base_uv_f64(int N, const double* __restrict__ d1, const double* __restrict__ dphi, const double* __restrict__ W0,
                              double* __restrict__ bphi, double* __restrict__ bW0, double* __restrict__ u, double* __restrict__ v,
                              const double* __restrict__ xE) {
    int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    double e1 = d1[j], p = dphi[j], w = W0[j];
    if (xE) {  // refined mesh: x-derivatives and the factor 1/|xi'| of (2.8)
        const double re = 1.0 / xE[j];
        e1 *= re; p *= re; w *= re;
    }
    const double rden = 1.0 / fma(e1, e1, 1.0);
    bphi[j] = p;       bphi[N + j] = 0.0;
    bW0[j] = w;        bW0[N + j] = 0.0;
    u[j] = (p - e1 * w) * rden;       u[N + j] = 0.0;
    v[j] = fma(e1, p, w) * rden;      v[N + j] = 0.0;
}

int fast_base_f64(sww_dtn_s* d, const double* phi0) {
    const int N = d->N;
    cudaStream_t st = d->stream;
    Workspace& w = d->ws;
    SWW_CUDA(cudaMemcpyAsync(w.B, phi0, sizeof(double) * N, cudaMemcpyDeviceToDevice, st));
    SWW_TRY(run_solve(d, w.B, w.S, 1));                               // mu0
    // gamma = D mu0 ; W = |D| mu0 / 2 ; phi0 rides along as the partner column of the transform pair: Gam column 1 = D phi0
    SWW_TRY(spectral_gamma_w(d, w.B, nullptr, w.Gam, w.W, 2, 1, phi0));
    if (N >= 128 && (size_t)d->bp_chunks * 4 >= 16)
        SWW_TRY(gemv_few_f64(st, N, 1, N, d->G, N, w.Gam, N, w.W, N, d->bp_part, d->mv_count));
    else
        SWW_TRY(gemm_f64(st, N, 1, N, 1.0, d->G, N, w.Gam, N, 1.0, w.W, N, 1));
    SWW_BEGIN(KC_OTHER, st);
    k_base_uv_f64<<<(N + 255) / 256, 256, 0, st>>>(N, d->d1, w.Gam + N, w.W, d->bphi, d->bW0, d->bu, d->bv, d->mesh_on ? d->mesh.xE : nullptr);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

// ------------------------------------------------------------------------------------------------ flow (2): dd apply
// rhs: dd planar N x nrhs with plane size Lin (0 = N * nrhs; ignored when rhs_in_ws: ws.B (dd) and ws.R (fp64 rounding) are
// already filled).  Tcols: dd planar in ws layout or nullptr.  out: dd planar N x nrhs, plane size Lout (0 = N * nrhs).
int dd_apply(sww_dtn_s* d, const double* rhs, bool rhs_in_ws, const double* Tcols, int nrhs, double* out, size_t Lin, size_t Lout) {
    const int N = d->N;
    if (N > 4096) return SWW_EINVAL;  // one N-point complex dd array in shared memory: 32 B x N <= 128 KB (include/sww.h states it)
    cudaStream_t st = d->stream;
    Workspace& w = d->ws;
    const size_t NN = (size_t)N * N, Lws = (size_t)N * w.cap_cols, n = (size_t)N * nrhs, Lio = Lout ? Lout : n;
    unsigned blocks = (unsigned)((n + 255) / 256);
    if (!rhs_in_ws) {
        SWW_BEGIN(KC_OTHER, st);
        k_dd_copy<<<blocks, 256, 0, st>>>(n, Lin ? Lin : n, Lws, 1, rhs, w.B, w.R);
        SWW_LAUNCHED();
    }
    double* mu = w.W;  // dd planar, ws layout
    const int nsweep = DD_SWEEPS;
    for (int s = 0; s < nsweep; s++) {
        SWW_TRY(run_solve(d, w.R, w.S, nrhs));
        SWW_BEGIN(KC_OTHER, st);
        k_dd_axpy_f64<<<blocks, 256, 0, st>>>(n, Lws, s == 0, w.R, w.S, mu);
        SWW_LAUNCHED();
        if (s + 1 < nsweep) {  // R = B - mu/2 - K mu in dd, rounded to fp64 for the next LU solve
            SWW_TRY(gemm_dd(d, nrhs, Lws, d->K, d->K + NN, mu, 1.0, w.B, -0.5, -1.0, w.Gam, w.R));
        }
    }
    static DeviceOnce attr_once;
    if (attr_once.first()) {
        SWW_CUDA(cudaFuncSetAttribute(k_spectral_gamma_w_dd, cudaFuncAttributeMaxDynamicSharedMemorySize, 2048 * 32 * 2));
        SWW_CUDA(cudaFuncSetAttribute(k_spectral_pass_dd, cudaFuncAttributeMaxDynamicSharedMemorySize, 4096 * 32));
    }
    int threads = N / 2 > 512 ? 512 : (N / 2 < 32 ? 32 : N / 2);
    // Gam = D mu (ws layout) ; out = |D| mu / 2 - D T  (user layout)
    if (N <= 2048) {
        size_t smem = (size_t)N * sizeof(cdd) * 2;
        SWW_BEGIN(KC_FFT, st);
        k_spectral_gamma_w_dd<<<(nrhs + 1) / 2, threads, smem, st>>>(N, ilog2(N), d->tab->cs, d->tab->sn, Lws, Lio, mu, Tcols, w.Gam, out, nrhs, nrhs);
        SWW_LAUNCHED();
    } else {  // N = 4096: the two transforms of a column pair do not fit side by side; one multiplier per launch
        const size_t smem = (size_t)N * sizeof(cdd);
        const int nb = (nrhs + 1) / 2, lg = ilog2(N);
        SWW_BEGIN(KC_FFT, st);
        k_spectral_pass_dd<<<nb, threads, smem, st>>>(N, lg, d->tab->cs, d->tab->sn, 0, 1.0, 0, Lws, Lws, mu, w.Gam, nrhs, nrhs, 1);
        SWW_LAUNCHED();
        SWW_BEGIN(KC_FFT, st);
        k_spectral_pass_dd<<<nb, threads, smem, st>>>(N, lg, d->tab->cs, d->tab->sn, 1, 1.0, 0, Lws, Lio, mu, out, nrhs, nrhs, 0);
        SWW_LAUNCHED();
        if (Tcols) {
            SWW_BEGIN(KC_FFT, st);
            k_spectral_pass_dd<<<nb, threads, smem, st>>>(N, lg, d->tab->cs, d->tab->sn, 0, -1.0, 1, Lws, Lio, Tcols, out, nrhs, nrhs, 0);
            SWW_LAUNCHED();
        }
    }
    SWW_CUDA(cudaGetLastError());
    // out += G Gam : Y = 1*Z + 0*X + 1*(A X) with Z = out (plane Lio) -- the kernel takes one plane size, so go through w.B:
    SWW_BEGIN(KC_OTHER, st);
    k_dd_copy<<<blocks, 256, 0, st>>>(n, Lio, Lws, 1, out, w.B, nullptr);
    SWW_LAUNCHED();
    SWW_TRY(gemm_dd(d, nrhs, Lws, d->G, d->G + NN, w.Gam, 1.0, w.B, 0.0, 1.0, w.T == Tcols ? w.W : w.T, nullptr));
    SWW_BEGIN(KC_OTHER, st);
    k_dd_copy<<<blocks, 256, 0, st>>>(n, Lws, Lio, 1, w.T == Tcols ? w.W : w.T, out, nullptr);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return mesh_scale_out(d, out, nrhs, Lio);  // the factor 1/|xi'| of (2.8) on a refined mesh
}

int dd_linearized(sww_dtn_s* d, const double* deta, const double* dphi, int nrhs, double* out, size_t Lin, size_t Lout) {
    const int N = d->N;
    Workspace& w = d->ws;
    const size_t Lws = (size_t)N * w.cap_cols, n = (size_t)N * nrhs;
    SWW_BEGIN(KC_OTHER, d->stream);
    k_rhs_lin_dd<<<(unsigned)((n + 255) / 256), 256, 0, d->stream>>>(N, n, Lin ? Lin : n, Lws, deta, dphi, d->bu, d->bv, w.B, w.T, w.R);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return dd_apply(d, nullptr, true, w.T, nrhs, out, 0, Lout);
}

}  // namespace sww
