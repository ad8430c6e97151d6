// trsv.cu -- S4 for ONE right-hand side: the forward and backward sweeps of the block LU of lu.cu (A = L U with identity diagonal
// blocks in L, U_ii = S_i, F_i = inv(S_i) - 2 I) as ONE thread-block cluster of 16 CTAs (8 where the device refuses 16).
//
// Why a second kernel: a single column is a chain of 2 N/64 dependent block steps.  In k_trsm_dataflow every link of that chain
// is a release/acquire hop through L2 (store, gpu-scope fence, flag, poll, reload: ~2 us).  Here the 64 new values of a block go
// straight into the shared memory of every CTA of the cluster (distributed shared memory) by st.async, each store counted on an
// mbarrier that sits next to the data in the receiving CTA: data and signal travel together, without fences or flags, and a
// waiting CTA sleeps in mbarrier.try_wait.  This is the path of the base state (two solves per surface; "a single back-solve",
// PAPER.md:305) and of the time stepper without variational columns.
//
// Work split: CTA r of the cluster owns the row blocks i = r (mod cluster size).  Forward: when y_k arrives, every CTA subtracts
// L_ik y_k from the accumulators of its blocks i > k (right-looking); the owner of block k + 1 takes that tile first, finishes
// y_{k+1} = b_{k+1} - sum and broadcasts it.  Backward the same from the bottom with U_ik and the extra product
// x_i = 2 z + F_i z.  The factor tiles (final before the launch) stream from L2 through a ring of cp.async buffers, in exactly
// the order they are used; a slot is refilled behind the work on the chain.  Measured (N = 2048): 0.11 ms per solve against
// 0.135 ms for the L2-hop kernel; what bounds it now is the 33 MB of factors read by 16 SMs (about 60 GB/s each).
// Accuracy: as in k_trsm_dataflow the sums of the O(1/N) products are kept as (hi, lo) two-sum pairs per thread and the O(1)
// right-hand side is added by an error-free two-sum; the result is B (hi) + Blo (lo).
// Product code; shares nothing with oracle/.
#include "common.cuh"
#include <cstdlib>

namespace sww {

namespace {
constexpr int TV_TS = 64;      // tile size (= lu.cu TS)
constexpr int TV_CSMAX = 16;   // CTAs per cluster: 16 (non-portable size) when the device accepts it, else 8
constexpr int TV_RING = 4;     // factor tiles in flight per CTA

__device__ __forceinline__ void tv_cp16(void* smem, const void* gmem) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void tv_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int n>
__device__ __forceinline__ void tv_wait() {
    asm volatile("cp.async.wait_group %0;\n" ::"n"(n));
}
__device__ __forceinline__ void tv_two_sum(double a, double b, double& s, double& e) {
    s = __dadd_rn(a, b);
    const double bb = __dsub_rn(s, a);
    e = __dadd_rn(__dsub_rn(a, __dsub_rn(s, bb)), __dsub_rn(b, bb));
}
// address of the same shared-memory location in CTA `rank` of the cluster
__device__ __forceinline__ unsigned tv_mapa(unsigned local, unsigned rank) {
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;\n" : "=r"(r) : "r"(local), "r"(rank));
    return r;
}
// store 8 bytes into a peer's shared memory and count them on the mbarrier next to it (same peer): data and signal travel
// together, no release fence and no separate flag
__device__ __forceinline__ void tv_st_async_f64(unsigned addr, double v, unsigned mbar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b64 [%0], %1, [%2];\n" ::"r"(addr), "l"(__double_as_longlong(v)), "r"(mbar)
                 : "memory");
}
__device__ __forceinline__ void tv_mbar_init(unsigned mbar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(mbar), "r"(count) : "memory");
}
__device__ __forceinline__ void tv_mbar_expect_tx(unsigned mbar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tv_mbar_wait(unsigned mbar, unsigned parity) {
    asm volatile(
        "{\n .reg .pred p;\n WAIT_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n @!p bra WAIT_%=;\n}\n" ::"r"(mbar), "r"(parity)
        : "memory");
}
__device__ __forceinline__ unsigned long long tv_gtime() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ void tv_cluster_sync() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;\n" ::: "memory");
}
}  // namespace

struct TrsvArgs {
    const double* A;   // block LU factors, N x N column-major
    const double* Fs;  // nt blocks of 64 x 64 (column-major, ld 64): inv(S_i) - 2 I
    double *B, *Blo;   // the column: in B = right-hand side, out B + Blo = solution
    int N, nt, cs;
    unsigned long long* trace;  // optional (env SWW_TRSV_TRACE): 4 globaltimer stamps per forward block
};

// shared memory layout (doubles unless noted)
//   y[N]                      the solution vector of the current sweep as it arrives (forward: y, backward: x)
//   bs[N]                     the right-hand side; a finished forward block leaves its low word here
//   ring[TV_RING][64 * 64]    factor tiles, column-major ld 64
//   red[2][4][64]             (hi, lo) partial sums of the four column quarters of a block being finished
//   z[64]                     the block being finished (operand of the F product)
//   accs[2][nown][256]        per-thread (hi, lo) sums of the products of each owned row block (added by run_trsv_cluster)
//   mbar[2][nt] (8 bytes each) mbar[phase][k] completes when the 512 bytes of block k of this phase's vector have landed in y[]
static size_t trsv_smem_bytes(int N) {
    return sizeof(double) * (2 * (size_t)N + (size_t)TV_RING * TV_TS * TV_TS + 2 * 4 * 64 + 64) + sizeof(unsigned long long) * (2 * (size_t)(N / TV_TS) + TV_RING) + 64;
}

namespace {
// The sequence of factor tiles CTA `r` consumes: forward  L(i, k) for k = 0 .. nt-2 and its row blocks i > k ascending;
// backward  [F(nt-1)] then for k = nt-1 .. 1: U(i, k) for its row blocks i < k descending, with F(k-1) right after U(k-1, k).
enum { TILE_L = 0, TILE_U = 1, TILE_F = 2, TILE_END = 3 };
struct TileIt {
    int r, nt, cs, type, k, i;
    __device__ void bstep(int kk) {  // first tile of backward step kk, kk-1, ...
        for (; kk >= 1; kk--) {
            const int top = kk - 1, ii = top - (((top - r) % cs + cs) % cs);
            if (ii >= 0) {
                type = TILE_U; k = kk; i = ii;
                return;
            }
        }
        type = TILE_END;
    }
    __device__ void bstart() {
        if ((nt - 1) % cs == r) {
            type = TILE_F; k = nt; i = nt - 1;
        } else {
            bstep(nt - 1);
        }
    }
    __device__ void fstep(int kk) {  // first tile of forward step kk, kk+1, ...
        for (; kk <= nt - 2; kk++) {
            const int lo = kk + 1, ii = lo + (((r - lo) % cs + cs) % cs);
            if (ii < nt) {
                type = TILE_L; k = kk; i = ii;
                return;
            }
        }
        bstart();
    }
    __device__ void init(int r_, int nt_, int cs_) {
        r = r_; nt = nt_; cs = cs_;
        fstep(0);
    }
    __device__ void next() {
        if (type == TILE_L) {
            if (i + cs < nt) i += cs;
            else fstep(k + 1);
        } else if (type == TILE_U) {
            if (i == k - 1) type = TILE_F;  // k stays: the step this F belongs to
            else if (i - cs >= 0) i -= cs;
            else bstep(k - 1);
        } else if (type == TILE_F) {
            if (k == nt) bstep(nt - 1);                                  // F(nt-1) opened the backward sweep
            else if (i - cs >= 0) { type = TILE_U; i -= cs; }      // rest of step k
            else bstep(k - 1);
        }
    }
};
}  // namespace

__global__ void __launch_bounds__(256, 1) k_trsv_cluster(TrsvArgs p) {
    extern __shared__ __align__(16) double tv_sm[];
    const int N = p.N, nt = p.nt;
    const int cs = p.cs;
    const int nown = (nt + cs - 1) / cs;
    double* y = tv_sm;                               // [N]
    double* bs = y + N;                              // [N]: right-hand side, then the low words of this CTA's blocks
    double* ring = bs + N;                            // [TV_RING][64*64]
    double* red = ring + TV_RING * TV_TS * TV_TS;    // [2][4][64]
    double* zs = red + 2 * 4 * 64;                   // [64]
    double* accs = zs + 64;                          // [2][nown][256]: per-thread (hi, lo) sums of each owned block
    unsigned long long* mbar = reinterpret_cast<unsigned long long*>(accs + 2 * (size_t)nown * 256);  // [2][nt]
    const int tid = threadIdx.x, row = tid & 63, part = tid >> 6;
    unsigned rank;
    asm volatile("mov.u32 %0, %%cluster_ctarank;\n" : "=r"(rank));
    const int r = (int)rank;

    const unsigned mbar_s = (unsigned)__cvta_generic_to_shared(mbar);
    for (int t = tid; t < 2 * nt; t += 256) {  // one-shot barriers: one arrival (made here) + the 512 bytes of the block
        tv_mbar_init(mbar_s + 8u * t, 1u);
        tv_mbar_expect_tx(mbar_s + 8u * t, 8u * TV_TS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    for (int t = tid; t < 2 * nown * 256; t += 256) accs[t] = 0.0;
    for (int t = tid; t < N; t += 256) bs[t] = p.B[t];
    __syncthreads();
    tv_cluster_sync();  // every CTA's barriers are armed before any remote write can arrive

    const unsigned y_s = (unsigned)__cvta_generic_to_shared(y);
    // publish block i of the current sweep's vector: threads 0..63 hold its entries; each sends its value to every CTA
    auto broadcast = [&](int phase, int i, double v) {  // called by tid < 64 only
        const unsigned ya = y_s + 8u * (unsigned)(i * TV_TS + row), ma = mbar_s + 8u * (unsigned)(phase * nt + i);
        for (unsigned q = 0; q < (unsigned)cs; q++) tv_st_async_f64(tv_mapa(ya, q), v, tv_mapa(ma, q));
    };
    // request a tile into ring slot `slot` (cp.async, 8 x 16 bytes per thread; the caller commits the group)
    auto issue = [&](const TileIt& it, int slot) {
        double* dst = ring + (size_t)slot * TV_TS * TV_TS;
        const double* src;
        size_t ld;
        if (it.type == TILE_F) {
            src = p.Fs + (size_t)it.i * TV_TS * TV_TS;
            ld = TV_TS;
        } else {
            src = p.A + (size_t)it.k * TV_TS * N + (size_t)it.i * TV_TS;  // tile (i, k): L below, U above the diagonal
            ld = (size_t)N;
        }
        for (int c = tid; c < TV_TS * TV_TS / 2; c += 256) {
            const int col = c >> 5, ch = (c & 31) * 2;
            tv_cp16(dst + col * TV_TS + ch, src + (size_t)col * ld + ch);
        }
    };
    // s = sum over this thread's column quarter of tile[row][c] * v[c]
    auto quarter_dot = [&](const double* tile, const double* v) {
        const double* t = tile + (size_t)(part * 16) * TV_TS + row;
        const double* vv = v + part * 16;
        double s0 = 0.0, s1 = 0.0;
#pragma unroll
        for (int c = 0; c < 16; c += 2) {
            s0 = fma(t[(size_t)c * TV_TS], vv[c], s0);
            s1 = fma(t[(size_t)(c + 1) * TV_TS], vv[c + 1], s1);
        }
        return s0 + s1;
    };
    // sum of the four quarters' (hi, lo) accumulators of owned block io -> (ph, pl) on threads tid < 64; all threads call
    auto gather = [&](int io, double& ph, double& pl) {
        red[(0 * 4 + part) * 64 + row] = accs[(size_t)(0 * nown + io) * 256 + tid];
        red[(1 * 4 + part) * 64 + row] = accs[(size_t)(1 * nown + io) * 256 + tid];
        __syncthreads();
        ph = pl = 0.0;
        if (tid < 64) {
            ph = red[row];
            pl = red[4 * 64 + row];
#pragma unroll
            for (int q = 1; q < 4; q++) {
                double s_, e_;
                tv_two_sum(ph, red[q * 64 + row], s_, e_);
                ph = s_;
                pl += e_ + red[(4 + q) * 64 + row];
            }
        }
    };

    if (r == 0 && tid < 64) broadcast(0, 0, bs[row]);  // y_0 = b_0 (identity diagonal block); Blo of block 0 is set backward
    TileIt itI, itC;
    itI.init(r, nt, cs);
    itC.init(r, nt, cs);
    int nI = 0;
    for (; nI < TV_RING - 1; nI++) {
        if (itI.type != TILE_END) {
            issue(itI, nI % TV_RING);
            itI.next();
        }
        tv_commit();
    }
    bool backward = false;
    for (int n = 0; itC.type != TILE_END; n++, itC.next()) {
        const bool trc = p.trace && itC.type == TILE_L && itC.i == itC.k + 1 && tid == 0;
        if (trc) p.trace[8 * itC.i + 4] = tv_gtime();
        tv_wait<TV_RING - 2>();
        __syncthreads();  // tile n is visible to every thread; everyone is done with tile n - 1 (its slot is refilled below)
        if (trc) p.trace[8 * itC.i + 5] = tv_gtime();
        const double* tile = ring + (size_t)(n % TV_RING) * TV_TS * TV_TS;
        const int type = itC.type, k = itC.k, i = itC.i, io = i / cs;
        if (type != TILE_L && !backward) {  // first backward tile: the accumulators start again from zero
            backward = true;
            for (int q = 0; q < 2 * nown; q++) accs[(size_t)q * 256 + tid] = 0.0;
        }
        if (type != TILE_F) {
            tv_mbar_wait(mbar_s + 8u * (unsigned)((type == TILE_U ? nt : 0) + k), 0u);
            const bool tr = p.trace && type == TILE_L && i == k + 1 && tid == 0;
            if (tr) p.trace[8 * i] = tv_gtime();
            const double s = quarter_dot(tile, y + (size_t)k * TV_TS);
            double* ah = accs + (size_t)(0 * nown + io) * 256 + tid;
            double* al = accs + (size_t)(1 * nown + io) * 256 + tid;
            double s_, e_;
            tv_two_sum(*ah, s, s_, e_);
            *ah = s_;
            *al += e_;
            if (type == TILE_L && i == k + 1) {  // y_i = b_i - sum_{k<i} L_ik y_k
                double ph, pl;
                if (tr) p.trace[8 * i + 1] = tv_gtime();
                gather(io, ph, pl);
                if (tr) p.trace[8 * i + 2] = tv_gtime();
                if (tid < 64) {
                    const size_t o = (size_t)i * TV_TS + row;
                    double zh, e2;
                    tv_two_sum(bs[o], -ph, zh, e2);
                    const double zl = e2 - pl;
                    const double hi = __dadd_rn(zh, zl);
                    bs[o] = __dsub_rn(zl, __dsub_rn(hi, zh));  // low word of y_i, used by this CTA in the backward sweep
                    broadcast(0, i, hi);
                    if (tr) p.trace[8 * i + 3] = tv_gtime();
                }
            }
        } else {  // x_i = Z_i (y_i - sum_{k>i} U_ik x_k) = 2 z + F_i z
            double ph, pl;
            gather(io, ph, pl);
            const size_t o = (size_t)i * TV_TS + row;
            double zh = 0.0, zl = 0.0;
            if (tid < 64) {
                double e2;
                tv_two_sum(y[o], -ph, zh, e2);                 // y[] still holds y_i: x_i replaces it below
                zl = e2 + (((i == 0) ? 0.0 : bs[o]) - pl);     // block 0 went out as the plain right-hand side
                zs[row] = zh;
            }
            __syncthreads();
            red[part * 64 + row] = quarter_dot(tile, zs);
            __syncthreads();
            if (tid < 64) {
                const double fz = (red[row] + red[64 + row]) + (red[128 + row] + red[192 + row]);
                double t_, e_;
                tv_two_sum(2.0 * zh, fz, t_, e_);
                const double lo = fma(2.0, zl, e_);
                const double hi = __dadd_rn(t_, lo);
                p.B[o] = hi;
                p.Blo[o] = __dsub_rn(lo, __dsub_rn(hi, t_));
                broadcast(1, i, hi);
            }
        }
        // refill the slot of tile n - 1 (free since this iteration's barrier) behind the work on the chain
        if (itI.type != TILE_END) {
            issue(itI, nI % TV_RING);
            itI.next();
        }
        tv_commit();
        nI++;
    }
    tv_wait<0>();
    tv_cluster_sync();  // nobody exits while a peer may still write into its shared memory
}

static size_t trsv_smem_for(int N, int c) {
    const int nt = N / TV_TS;
    return trsv_smem_bytes(N) + sizeof(double) * 2 * (size_t)((nt + c - 1) / c) * 256;
}
static void trsv_make_cfg(cudaLaunchConfig_t& cfg, cudaLaunchAttribute* at, int N, int c, cudaStream_t st) {
    cfg = cudaLaunchConfig_t{};
    cfg.gridDim = dim3(c, 1, 1);
    cfg.blockDim = dim3(256, 1, 1);
    cfg.dynamicSmemBytes = trsv_smem_for(N, c);
    cfg.stream = st;
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = c;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
}
constexpr size_t TV_SMEM_MAX = 225 * 1024;
// cluster size: 16 needs the non-portable attribute and 16 free SMs in one GPC; asked once per process, 8 otherwise
static int trsv_cluster_size() {
    static int cs = 0;
    if (cs) return cs;
    cs = 8;
    if (cudaFuncSetAttribute(k_trsv_cluster, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TV_SMEM_MAX) != cudaSuccess) {
        cudaGetLastError();
        return cs;
    }
    if (!getenv("SWW_TRSV_CS8") && cudaFuncSetAttribute(k_trsv_cluster, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess) {
        cudaLaunchConfig_t cfg;
        cudaLaunchAttribute at[1];
        trsv_make_cfg(cfg, at, 2048, 16, nullptr);
        int ncl = 0;
        if (cudaOccupancyMaxActiveClusters(&ncl, k_trsv_cluster, &cfg) == cudaSuccess && ncl >= 1) cs = 16;
    }
    cudaGetLastError();
    return cs;
}

bool trsv_cluster_supported(int N) { return N >= 2 * TV_TS && N <= 8192 && trsv_smem_for(N, trsv_cluster_size()) <= TV_SMEM_MAX; }

int run_trsv_cluster(sww_dtn_s* d, double* B, double* Blo) {
    const int N = d->N, nt = N / TV_TS, cs = trsv_cluster_size();
    TrsvArgs a;
    a.A = d->LU;
    a.Fs = d->invD + (size_t)nt * TV_TS * TV_TS;
    a.B = B;
    a.Blo = Blo;
    a.N = N;
    a.nt = nt;
    a.cs = cs;
    a.trace = nullptr;
    static unsigned long long* g_trace = nullptr;
    if (getenv("SWW_TRSV_TRACE")) {
        if (!g_trace) cudaMalloc(&g_trace, sizeof(unsigned long long) * 8 * 128);
        a.trace = g_trace;
    }
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute at[1];
    trsv_make_cfg(cfg, at, N, cs, d->stream);
    SWW_BEGIN(KC_TRSM, d->stream);
    SWW_CUDA(cudaLaunchKernelEx(&cfg, k_trsv_cluster, a));
    SWW_LAUNCHED();
    if (a.trace) {  // debugging aid: print the forward chain of this launch
        unsigned long long h[8 * 128];
        cudaStreamSynchronize(d->stream);
        cudaMemcpy(h, a.trace, sizeof(h), cudaMemcpyDeviceToHost);
        for (int i = 2; i < nt && i < 14; i++) {
            const long long t0 = (long long)h[8 * (i - 1) + 3];  // y_{i-1} sent
            fprintf(stderr, "trsv fwd block %2d (since y_%d was sent): loop top %6lld  tile landed %6lld  y seen %6lld  dot %6lld  gathered %6lld  sent %6lld ns\n", i,
                    i - 1, (long long)h[8 * i + 4] - t0, (long long)h[8 * i + 5] - t0, (long long)h[8 * i] - t0, (long long)h[8 * i + 1] - t0,
                    (long long)h[8 * i + 2] - t0, (long long)h[8 * i + 3] - t0);
        }
        fprintf(stderr, "trsv fwd total %lld ns\n", (long long)(h[8 * (nt - 1) + 3] - h[8 + 3]));
    }
    return SWW_OK;
}

}  // namespace sww
