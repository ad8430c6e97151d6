// lu.cu -- S2: unpivoted BLOCK LU of A = I/2 + K (the matrix of (2.7); "LU-factorization") and
// S4: the multi-right-hand-side triangular solves ("a single back-solve", "level 3 BLAS speed").
//
// No pivoting: the second-kind operator is benign -- sigma(A) in [0.46, 1.01], partial pivoting performs zero row swaps on every
// workload family; a guard on every pivot reports SWW_ESINGULAR instead of producing garbage.
//
// Factorisation = ONE persistent kernel (k_lu_dataflow) over 64 x 64 tiles.  The diagonal blocks are not factored but INVERTED:
// A = L U with identity diagonal blocks in L and the Schur complements S_m on the block diagonal of U; what is stored is
// L_im = X_im Z_m (i > m), U_mj = X_mj (j > m) and F_m = Z_m - 2 I, Z_m = inv(S_m).  Block 0 (the "spine") runs the recurrence of
// the diagonal blocks; every other CTA is a worker claiming tile tasks from a counter in dependency order.  Tiles are handed
// over through release/acquire flags in global memory: no grid barrier, no host round trip.  Details at k_lu_dataflow.
// N <= 64 (one padded tile) goes through k_lu_single (a scalar 64-step GETRF with explicit triangular inverses).
//
// Storage convention of the LU buffer: the DIAGONAL holds kappa_ii = A_ii - 1/2 (the assembly writes K, not I/2 + K): every
// update then rounds at the O(1/N) scale of the kernel entries instead of the O(1) scale of the pivot, and the inverse
// diagonal blocks are carried as deviations F_m = inv(S_m) - 2 I.
// Product code; shares nothing with oracle/.
#include "common.cuh"
#include "bgj.cuh"
#include <algorithm>
#include <vector>

namespace sww {

constexpr double PIVOT_GUARD = BGJ_PIVOT_GUARD;
constexpr int TR_MAXNS = 256;  // column slabs per TRSM launch (more columns: several launches)
constexpr int TS = 64;    // tile size
constexpr int LDT = 65;   // leading dimension of the row-major work tiles T, Eb, Fb (element (r,c) at r*LDT + c)
constexpr int LDO = 68;   // leading dimension of the DMMA operand tiles (conflict-free fragment loads)

__device__ __forceinline__ void lu_dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp16(void* smem, const void* gmem) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int n>
__device__ __forceinline__ void cp_wait() {
    asm volatile("cp.async.wait_group %0;\n" ::"n"(n));
}
__device__ __forceinline__ unsigned ld_acquire(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned ld_relaxed(const unsigned* p) {
    unsigned v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(unsigned* p, unsigned v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;\n" ::"l"(p), "r"(v) : "memory");
}

// ---- mbarrier helpers (shared-memory barriers with phase parity: the full / empty pairs of the operand rings)
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_test(unsigned long long* bar, unsigned parity) {
    unsigned ok;
    asm volatile(
        "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
        : "=r"(ok)
        : "r"((unsigned)__cvta_generic_to_shared(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    while (!mbar_test(bar, parity)) {
    }
}
// arrival on `bar` when every cp.async this thread has issued so far has landed (counted in the barrier's expected arrivals)
__device__ __forceinline__ void cp_arrive_on(unsigned long long* bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}

// ------------------------------------------------------------------------------------------------ 64 x 64 GETRF in shared memory
// One rolled loop of 64 elimination steps by a 256-thread CTA; thread (ty, tx) of a 16 x 16 grid keeps the 4 x 4 register tile
// rows ty + 16 q, columns tx + 16 b of three matrices:
//     a : the block itself (diagonal = U_jj - 1/2)           -> L\U in place (unit-lower multipliers, U with the 1/2 implicit)
//     x : starts as I, receives the same ROW operations      -> inv(L)
//     y : starts as I, receives the COLUMN operations col_c -= (u_jc / u_jj) col_j   -> inv(U') with U' = diag(U)^-1 U,
//         so that inv(U) = y diag(1/u_jj).
// Per step the owners publish column j of a and y and row j of a and x in shared memory (double-buffered: one barrier per
// step); everything else is 48 register FMAs per thread.  The code is a compact loop on purpose: a fully unrolled in-warp
// variant was 5x slower because its straight-line code (600 KB) misses the instruction cache on every diagonal tile.
// Results go to global memory: Ag (leading dimension lda) <- L\U, Eg <- inv(L) - I, Fg <- inv(U) - 2 I (both lde); entries with
// row or column >= nb are not stored (N < 64: the tile is padded with kappa = 0, i.e. pivots 1/2 and no coupling).
// vec: 512 + 64 doubles of shared memory.  Every thread of the CTA must call it; T is read before the first barrier only.
// the 16 elimination steps j = 16 JB .. 16 JB + 15: only the 16 x 16 sub-blocks that can change are touched (static in JB)
template <int JB>
__device__ __forceinline__ void getrf64_steps(double (&a)[4][4], double (&x)[4][4], double (&y)[4][4], double* vec, int* status, int tid) {
    const int ty = tid & 15, tx = tid >> 4;
    double* rinv = vec + 512;
#pragma unroll 1
    for (int jt = 0; jt < 16; jt++) {
        const int j = 16 * JB + jt;
        double* colA = vec + (jt & 1) * 256;
        double* rowA = colA + 64;
        double* rowX = colA + 128;
        double* colY = colA + 192;
        if (tx == jt) {
#pragma unroll
            for (int q = 0; q < 4; q++) {
                if (q >= JB) colA[ty + 16 * q] = a[q][JB];
                if (q <= JB) colY[ty + 16 * q] = y[q][JB];
            }
        }
        if (ty == jt) {
#pragma unroll
            for (int b = 0; b < 4; b++) {
                if (b >= JB) rowA[tx + 16 * b] = a[JB][b];
                if (b <= JB) rowX[tx + 16 * b] = x[JB][b];
            }
        }
        __syncthreads();
        const double piv = 0.5 + rowA[j];  // the diagonal holds U_jj - 1/2
        const double ri = 1.0 / piv;
        if (tid == 0) {
            rinv[j] = ri;
            if (!(fabs(piv) >= PIVOT_GUARD)) atomicCAS(status, SWW_OK, SWW_ESINGULAR);
        }
        double l[4], u[4], ut[4], xr[4], yc[4];
#pragma unroll
        for (int q = 0; q < 4; q++) {
            const int row = ty + 16 * q;
            if (q >= JB) l[q] = (row > j) ? colA[row] * ri : 0.0;
            if (q <= JB) yc[q] = colY[row];  // Y[r][j] = 0 for r > j already
        }
#pragma unroll
        for (int b = 0; b < 4; b++) {
            const int col = tx + 16 * b;
            if (b >= JB) {
                u[b] = (col > j) ? rowA[col] : 0.0;
                ut[b] = u[b] * ri;
            }
            if (b <= JB) xr[b] = rowX[col];  // X[j][c] = 0 for c > j already
        }
#pragma unroll
        for (int q = 0; q < 4; q++)
#pragma unroll
            for (int b = 0; b < 4; b++) {
                if (q >= JB && b >= JB) a[q][b] = fma(-l[q], u[b], a[q][b]);
                if (q >= JB && b == JB && tx == jt && ty + 16 * q > j) a[q][b] = l[q];  // keep the multiplier
                if (q >= JB && b <= JB) x[q][b] = fma(-l[q], xr[b], x[q][b]);
                if (q <= JB && b >= JB) y[q][b] = fma(-yc[q], ut[b], y[q][b]);
            }
    }
}

__device__ __noinline__ void getrf64(const double* T, double* vec, int* status, int tid, double* Ag, size_t lda, double* Eg,
                                     double* Fg, int lde, int nb) {
    const int ty = tid & 15, tx = tid >> 4;
    double* rinv = vec + 512;
    double a[4][4], x[4][4], y[4][4];
#pragma unroll
    for (int q = 0; q < 4; q++)
#pragma unroll
        for (int b = 0; b < 4; b++) {
            a[q][b] = T[(ty + 16 * q) * LDT + tx + 16 * b];
            x[q][b] = y[q][b] = (ty + 16 * q == tx + 16 * b) ? 1.0 : 0.0;
        }
    getrf64_steps<0>(a, x, y, vec, status, tid);
    getrf64_steps<1>(a, x, y, vec, status, tid);
    getrf64_steps<2>(a, x, y, vec, status, tid);
    getrf64_steps<3>(a, x, y, vec, status, tid);
    __syncthreads();  // rinv complete
#pragma unroll
    for (int b = 0; b < 4; b++) {
        const int col = tx + 16 * b;
        const double rc = rinv[col];
#pragma unroll
        for (int q = 0; q < 4; q++) {
            const int row = ty + 16 * q;
            if (row < nb && col < nb) {
                Ag[(size_t)col * lda + row] = a[q][b];
                Eg[col * lde + row] = (row > col) ? x[q][b] : 0.0;
                Fg[col * lde + row] = (row < col) ? y[q][b] * rc : ((row == col) ? -2.0 * a[q][b] * rc : 0.0);  // F_rr = 1/U_rr - 2 without cancellation
            }
        }
    }
}

// N <= 64: the whole matrix is one (padded) tile
__global__ void __launch_bounds__(256) k_lu_single(double* __restrict__ A, int nb, double* __restrict__ Eout, double* __restrict__ Fout, int* status) {
    extern __shared__ double lu_sm[];
    double* T = lu_sm;
    double* vec = T + TS * LDT;
    const int tid = threadIdx.x;
    for (int e = tid; e < TS * TS; e += 256) {
        const int r = e & 63, c = e >> 6;
        T[r * LDT + c] = (r < nb && c < nb) ? A[(size_t)c * nb + r] : 0.0;  // padding: kappa = 0 -> pivot 1/2, no coupling
    }
    __syncthreads();
    getrf64(T, vec, status, tid, A, (size_t)nb, Eout, Fout, nb, nb);
}

// ------------------------------------------------------------------------------------------------ the persistent dataflow LU
// BLOCK LU without pivoting, 64 x 64 tiles:  A = L U  with identity diagonal blocks in L and the Schur complements S_m on the
// block diagonal of U; what is stored is  L_im = X_im Z_m  (i > m),  U_mj = X_mj  (j > m)  and  F_m = Z_m - 2 I,  Z_m = inv(S_m),
// where  X_ij = A_ij - sum_{k < min(i,j)} L_ik U_kj.  (Well posed: every S_m is I/2 plus a small block.)
//
// The recurrence of the diagonal,  S_m = P_m - X_{m,m-1} Z_{m-1} U_{m-1,m}  with  P_m = A_mm - sum_{k<m-1} L_mk U_km,  is the
// critical path.  It runs on a dedicated cluster of two CTAs (the "spine", blocks 0 and 1): blocked Gauss-Jordan inverse of
// S_{m-1} on the tensor pipe (bgj.cuh; both CTAs, redundantly), then V = Z_{m-1} U_{m-1,m} and S_m = P_m - X_{m,m-1} V with the
// columns split between the two CTAs and the halves exchanged through distributed shared memory; the three inputs are fetched
// while the previous inverse runs.  Everything else is done by worker CTAs claiming tile tasks from a counter.  A tile of level l = min(i,j) sums its terms k < l-1 from finished tiles; its LAST term needs Z_{l-1}, which has only
// just been published -- waiting for a neighbour task to turn X_{i,l-1} into L_{i,l-1} first would put two tasks and two trips
// through L2 between consecutive inverses.  So every task forms the L it needs for its last term itself, L = X Z_{l-1} (a
// chained pair of products right behind the flag of Z_{l-1}), from an X that is available long before:
//     lower (i > j)  : sum over k < j-1; wait for Z_{j-1}; L_{i,j-1} = X_{i,j-1} Z_{j-1}; X_ij = sum - L_{i,j-1} U_{j-1,j}, stored in
//                      place (xready) -- for j = i-1 in the staging block Xs[i] (xflags), the tile itself keeps A; then the
//                      finished L_{i,j-1} overwrites X_{i,j-1} (final).  Every lower tile is finished by its right neighbour.
//     upper (i < j)  : sum over k < i-1; wait for Z_{i-1}; L_{i,i-1} = Xs[i] Z_{i-1}; U_ij = sum - L_{i,i-1} U_{i-1,j} (final); the
//                      tile next to the diagonal (j = i+1) also stores L_{i,i-1} (row nt-1 has a task that does only that).
//     P (i, i)       : partial sum P_i over k < i-2, then the term of k = i-2 from X_{i,i-2} in the same way, in place; it
//                      tells the task of tile (i, i-1) when it has read X_{i,i-2} (pflags), which may then overwrite it.
// A tile is published by a release store of the launch's epoch into its flag; consumers acquire-poll.  Tasks are claimed in
// order of the generation g of the inverse Z_g they wait for (build_order); every other dependency of a task is on a task of an
// earlier generation (pflags: earlier in the same generation), and the spine computing Z_m waits only for tasks of
// generation m - 2: a claimed task waits only for tasks claimed earlier or for the spine -- no deadlock, no grid barrier.
constexpr int LU_THREADS = BGJ_CTA_THREADS;  // 352: 8 MMA warps (tid < 256) + the extra warps the inversion's role map needs
enum LuTaskType { T_U = 0, T_L = 1, T_P = 2 };
__host__ __device__ constexpr int lu_task(int type, int i, int j) { return (type << 28) | (i << 14) | j; }
// kl: the term a tile forms from X and Z on the fly (upper: i-1, lower: j-1, diagonal P: i-2); its plain terms are k < kl
__host__ __device__ constexpr int lu_kl(int i, int j) { return i < j ? i - 1 : (i > j ? j - 1 : i - 2); }

struct LuArgs {
    double* A;         // N x N column-major, in place
    int N, nt;         // nt = N / 64 tiles per side
    int ntasks;
    const int* order;  // worker tasks in claim order: lu_task(type, i, j)
    unsigned* flags;   // nt*nt: flags[i*nt + j] == epoch  <=>  tile (i,j) is final (i != j) / P_i is ready (i == j)
    unsigned* xready;  // nt*nt: X_ij is in place (lower tiles, j < i-1)
    unsigned* xflags;  // nt: X_{m,m-1} is in Xs[m]
    unsigned* pflags;  // nt: the P task of row m has read X_{m,m-2}
    unsigned* zflags;  // nt: F_m is in Fs
    unsigned epoch;
    unsigned* counter;  // next task to claim (zeroed before the launch)
    double* Fs;        // nt blocks of 64 x 64 (column-major, ld 64): inv(S_m) - 2 I
    double* Xs;        // nt blocks of 64 x 64 (column-major, ld 64): staging of X_{m,m-1}
    double* Vs;        // nt blocks of 64 x 64 (column-major, ld 64): V_m = inv(S_m) U_{m,m+1}, the front term of the backward sweep
    int* status;
};

// spine: sX, sF (64 columns), sU, sV, sP (32 columns), two work tiles, bgj64 scratch; workers: a ring of three operand tile pairs
constexpr int LU_SMEM_SPINE = (2 * TS * LDO + 3 * 32 * LDO + 2 * TS * BGJ_TLD + BGJ_SCRATCH) * (int)sizeof(double);
constexpr int LU_RING = 3;          // stages of the workers' operand ring (one L tile + one U tile per stage)
constexpr int LU_SMEM_WORKER = 2 * LU_RING * TS * LDO * (int)sizeof(double) + 256;
constexpr int LU_SMEM_BYTES = LU_SMEM_SPINE > LU_SMEM_WORKER ? LU_SMEM_SPINE : LU_SMEM_WORKER;

// fragment coordinates of this lane (threads 0..255): rows wr*32 + x*8 + fr (x < 4), columns wc*16 + y*8 + 2 fk + e (y, e < 2)
struct Frag {
    int wr, wc, fr, fk;
    __device__ __forceinline__ Frag(int tid) : wr((tid >> 5) & 1), wc((tid >> 6) & 3), fr((tid & 31) >> 2), fk(tid & 3) {}
    __device__ __forceinline__ int row(int x) const { return wr * 32 + x * 8 + fr; }
    __device__ __forceinline__ int col(int y, int e) const { return wc * 16 + y * 8 + 2 * fk + e; }
};
#define SWW_FRAG_LOOP for (int x = 0; x < 4; x++) for (int y = 0; y < 2; y++) for (int e = 0; e < 2; e++)

// acc += As x Bs over one 64-deep slab; As[k][r] (ld LDO), Bs[n][k] (ld LDO)
__device__ __forceinline__ void mma_tile64(double (&acc)[4][2][2], const double* a, const double* b, const Frag& f) {
    const double* as = a + f.wr * 32 + f.fr;
    const double* bs = b + (f.wc * 16 + f.fr) * LDO;
#pragma unroll
    for (int k4 = 0; k4 < TS; k4 += 4) {
        double af[4], bf[2];
#pragma unroll
        for (int x = 0; x < 4; x++) af[x] = as[(k4 + f.fk) * LDO + x * 8];
#pragma unroll
        for (int y = 0; y < 2; y++) bf[y] = bs[y * 8 * LDO + k4 + f.fk];
#pragma unroll
        for (int x = 0; x < 4; x++)
#pragma unroll
            for (int y = 0; y < 2; y++) lu_dmma884(acc[x][y][0], acc[x][y][1], af[x], bf[y]);
    }
}
// 64 x 64 column-major tile (leading dimension ld) -> shared, ld LDO, same orientation; thread t of nthr, cp.async (not committed)
__device__ __forceinline__ void tile_async(double* dst, const double* src, size_t ld, int t, int nthr) {
    for (int c = t; c < TS * TS / 2; c += nthr) {
        const int col = c >> 5, ch = (c & 31) * 2;
        cp16(dst + col * LDO + ch, src + (size_t)col * ld + ch);
    }
}

__device__ __forceinline__ void spin_until(const unsigned* f, unsigned epoch) {
    while (ld_acquire(f) != epoch) __nanosleep(20);
}
// for the few waits that sit on the spine's critical path: no back-off
__device__ __forceinline__ void spin_tight(const unsigned* f, unsigned epoch) {
    while (ld_acquire(f) != epoch) {
    }
}

#ifdef SWW_LU_TRACE  // development aid, compiled out of the product (build.py never defines it): per-step time stamps of the spine
__device__ unsigned long long g_lu_trace[4 * 128 + 3 * 8 * 128];
__device__ __forceinline__ void lu_stamp(int m, int k) {
    if (threadIdx.x == 0) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
        g_lu_trace[4 * m + k] = t;
    }
}
#define SWW_STAMP(m, k) lu_stamp(m, k)
// worker stamps of the three tasks that feed the spine: which = 0 (tile (i, i-1)), 1 (tile (i-1, i)), 2 (P_i); 8 stamps per task
#define SWW_WSTAMP(k)                                                                                              \
    do {                                                                                                           \
        const int which_ = (type == T_L && j == i - 1) ? 0 : (type == T_U && j == i + 1) ? 1 : (type == T_P) ? 2 : -1; \
        if (which_ >= 0 && threadIdx.x == 0) {                                                                     \
            unsigned long long t_;                                                                                 \
            asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t_));                                                 \
            g_lu_trace[4 * 128 + (which_ * 128 + (which_ == 1 ? i + 1 : i)) * 8 + (k)] = t_;                      \
        }                                                                                                          \
    } while (0)
#else
#define SWW_STAMP(m, k)
#define SWW_WSTAMP(k)
#endif

// ---- thread-block cluster helpers (the spine is a cluster of two CTAs)
__device__ __forceinline__ unsigned cluster_rank() {
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {  // every thread of both CTAs
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// the address of my shared-memory location p in the shared memory of CTA `rank` of the cluster
__device__ __forceinline__ unsigned cluster_map(const void* p, unsigned rank) {
    unsigned a = (unsigned)__cvta_generic_to_shared(p), r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(rank));
    return r;
}

// fragment coordinates for a 64 x 32 half tile (threads 0..255): rows wr*16 + x*8 + fr (x < 2), columns wc*16 + y*8 + 2 fk + e
struct FragH {
    int wr, wc, fr, fk;
    __device__ __forceinline__ FragH(int tid) : wr((tid >> 5) & 3), wc((tid >> 7) & 1), fr((tid & 31) >> 2), fk(tid & 3) {}
    __device__ __forceinline__ int row(int x) const { return wr * 16 + x * 8 + fr; }
    __device__ __forceinline__ int col(int y, int e) const { return wc * 16 + y * 8 + 2 * fk + e; }
};
#define SWW_FRAGH_LOOP for (int x = 0; x < 2; x++) for (int y = 0; y < 2; y++) for (int e = 0; e < 2; e++)
// acc (64 x 32) += As (64 x 64) x Bs (64 x 32); As[k][r] (ld LDO), Bs[n][k] (ld LDO, 32 columns)
__device__ __forceinline__ void mma_half(double (&acc)[2][2][2], const double* a, const double* b, const FragH& f) {
    const double* as = a + f.wr * 16 + f.fr;
    const double* bs = b + (f.wc * 16 + f.fr) * LDO;
#pragma unroll
    for (int k4 = 0; k4 < TS; k4 += 4) {
        double af[2], bf[2];
#pragma unroll
        for (int x = 0; x < 2; x++) af[x] = as[(k4 + f.fk) * LDO + x * 8];
#pragma unroll
        for (int y = 0; y < 2; y++) bf[y] = bs[y * 8 * LDO + k4 + f.fk];
#pragma unroll
        for (int x = 0; x < 2; x++)
#pragma unroll
            for (int y = 0; y < 2; y++) lu_dmma884(acc[x][y][0], acc[x][y][1], af[x], bf[y]);
    }
}
// 32 columns of a 64-row column-major tile -> shared, ld LDO; thread t of nthr, cp.async (not committed)
__device__ __forceinline__ void half_async(double* dst, const double* src, size_t ld, int t, int nthr) {
    for (int c = t; c < TS * 32 / 2; c += nthr) {
        const int col = c >> 5, ch = (c & 31) * 2;
        cp16(dst + col * LDO + ch, src + (size_t)col * ld + ch);
    }
}

// ---- the spine: the cluster of blocks 0 and 1.  Both CTAs invert S_{m-1} (the same instructions on the same data: the same
// bits), then each forms one half of the columns of V = Z_{m-1} U_{m-1,m} and of S_m = P_m - X_{m,m-1} V (two 64 x 64 x 32 products
// instead of two 64^3), and writes its half of kappa_m = S_m - I/2 into both CTAs' work tiles through distributed shared
// memory; one cluster barrier per step.  CTA 0 publishes F_m.
__device__ void lu_spine(const LuArgs& p, double* sm) {
    double* sX = sm;                  // X_{m,m-1}                               (A operand: As[k][r])
    double* sF = sX + TS * LDO;       // F_{m-1}, written by bgj64               (A operand)
    double* sU = sF + TS * LDO;       // my 32 columns of U_{m-1,m}              (B operand: Bs[n][k])
    double* sV = sU + 32 * LDO;       // my 32 columns of V = Z_{m-1} U_{m-1,m}  (B operand)
    double* sP = sV + 32 * LDO;       // my 32 columns of P_m (column-major, ld LDO)
    double* sK = sP + 32 * LDO;       // 2 work tiles kappa_m = S_m - I/2 (row-major, ld BGJ_TLD) for bgj64, alternating by step
    double* scr = sK + 2 * TS * BGJ_TLD;
    const int tid = threadIdx.x;
    const FragH f(tid);
    const bool mm = tid < 256;        // the 8 MMA warps of the two products
    const int N = p.N, nt = p.nt;
    const unsigned epoch = p.epoch;
    const unsigned rank = cluster_rank(), peer = rank ^ 1u;
    const int cb = 32 * (int)rank;    // my columns of the step: cb .. cb + 31
    const int role = bgj_role(tid >> 5);
    // the three input flags of step m: Xs[m], tile (m-1, m), P_m (P_1 is the raw diagonal tile)
    auto input_flag = [&](int m, int q) -> const unsigned* {
        if (q == 0) return p.xflags + m;
        if (q == 1) return p.flags + (size_t)(m - 1) * nt + m;
        return (m >= 2) ? p.flags + (size_t)m * nt + m : nullptr;
    };
    // The two warps that have no role in the inversion (bgj_role < 0) fetch the inputs of the next step meanwhile: they wait for
    // the three flags (acquire) and issue the tile copies, which land in sX, sU, sP while the other warps invert.
    const int it = (tid >> 5) == 4 ? (tid & 31) : 32 + (tid & 31);  // index among the 64 idle threads (warps 4 and 8)
    auto fetch_inputs = [&](int m) {  // warp 4: P_m, then X_{m,m-1}, together with warp 8, which first fetches U_{m-1,m}
        const int lane = tid & 31;
        if ((tid >> 5) == 8) {
            if (lane == 0) spin_tight(input_flag(m, 1), epoch);
            __syncwarp();
            half_async(sU, p.A + ((size_t)m * TS + cb) * N + (size_t)(m - 1) * TS, N, lane, 32);   // tile (m-1, m), my columns
        } else {
            if (lane == 0 && input_flag(m, 2)) spin_tight(input_flag(m, 2), epoch);
            __syncwarp();
            half_async(sP, p.A + ((size_t)m * TS + cb) * N + (size_t)m * TS, N, lane, 32);         // tile (m, m), my columns
        }
        if (it == 0) spin_tight(input_flag(m, 0), epoch);
        asm volatile("bar.sync 4, 64;" ::: "memory");  // the two idle warps
        tile_async(sX, p.Xs + (size_t)m * TS * TS, TS, it, 64);
        cp_commit();
        cp_wait<0>();
    };
    for (int m = 0; m < nt; m++) {
        double* T = sK + (m & 1) * TS * BGJ_TLD;
        SWW_STAMP(m, 0);
        if (m == 0) {
            for (int e = tid; e < TS * TS; e += LU_THREADS) {
                const int r = e & 63, c = e >> 6;
                T[r * BGJ_TLD + c] = p.A[(size_t)c * N + r];
            }
        } else {
            SWW_STAMP(m, 1);
            double v[2][2][2], c0[2][2][2];
            if (mm) {  // V = Z_{m-1} U_{m-1,m} = 2 U + F U, my columns
#pragma unroll
                SWW_FRAGH_LOOP v[x][y][e] = 2.0 * sU[f.col(y, e) * LDO + f.row(x)];
                mma_half(v, sF, sU, f);
#pragma unroll
                SWW_FRAGH_LOOP sV[f.col(y, e) * LDO + f.row(x)] = v[x][y][e];
            }
            __syncthreads();
            if (!mm) {  // V is kept for the triangular solves: the warps that have no part in the products copy it out meanwhile
                double* Vg = p.Vs + (size_t)(m - 1) * TS * TS + (size_t)cb * TS;
                for (int c = tid - 256; c < 32 * TS / 2; c += LU_THREADS - 256) {
                    const int col = c >> 5, ch = (c & 31) * 2;
                    *reinterpret_cast<double2*>(Vg + col * TS + ch) = *reinterpret_cast<const double2*>(sV + col * LDO + ch);
                }
            }
            if (mm) {  // S_m = P_m - X_{m,m-1} V, my columns -> both CTAs' work tiles
#pragma unroll
                SWW_FRAGH_LOOP {
                    c0[x][y][e] = sP[f.col(y, e) * LDO + f.row(x)];
                    v[x][y][e] = 0.0;
                }
                mma_half(v, sX, sV, f);
                const unsigned Tpeer = cluster_map(T, peer);
#pragma unroll
                for (int x = 0; x < 2; x++)
#pragma unroll
                    for (int y = 0; y < 2; y++) {  // the two entries of a fragment row are neighbours in the row-major tile: one 16-byte store each way
                        const int o = f.row(x) * BGJ_TLD + cb + f.col(y, 0);
                        const double k0 = c0[x][y][0] - v[x][y][0], k1 = c0[x][y][1] - v[x][y][1];
                        *reinterpret_cast<double2*>(T + o) = make_double2(k0, k1);
                        asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};" ::"r"(Tpeer + 8u * (unsigned)o), "d"(k0), "d"(k1) : "memory");
                    }
            }
        }
        cluster_sync_all();  // kappa_m complete in both CTAs (also the CTA barrier: sX, sU, sV, sP free)
        SWW_STAMP(m, 2);
        bgj64(T, scr, p.status, tid, rank == 0 ? p.Fs + (size_t)m * TS * TS : nullptr, sF);
        if (role < 0 && m + 1 < nt) fetch_inputs(m + 1);
        __syncthreads();  // F_m in sF and in global memory; the inputs of step m + 1 in shared memory
        SWW_STAMP(m, 3);
        if (rank == 0 && tid == LU_THREADS - 32) st_release(p.zflags + m, epoch);  // a lane of a warp that has no part in the products
    }
    cluster_sync_all();  // neither CTA leaves while the other may still write into its shared memory
}

__global__ void __launch_bounds__(LU_THREADS, 1) k_lu_dataflow(LuArgs p) {
    extern __shared__ __align__(16) double lu_sm[];
    const int tid = threadIdx.x;
    if (blockIdx.x < 2) {  // cluster 0
        lu_spine(p, lu_sm);
        return;
    }
    double* sA = lu_sm;                         // LU_RING stages of L_ik as As[k][r]
    double* sB = sA + LU_RING * TS * LDO;       // LU_RING stages of U_kj as Bs[n][k]
    __shared__ unsigned long long full[LU_RING], empty[LU_RING];
    __shared__ int s_task;
    if (tid == 0)
        for (int q = 0; q < LU_RING; q++) {
            mbar_init(&full[q], LU_THREADS - 256);   // the producer threads, each when its copies of the stage have landed
            mbar_init(&empty[q], 8);                 // the eight MMA warps
        }
    unsigned it = 0;  // ring position: plain terms done so far by this CTA (the same number in every thread)
    const Frag f(tid);
    const bool mm = tid < 256;
    const int N = p.N, nt = p.nt;
    const unsigned epoch = p.epoch;
    auto tile = [&](int r, int c) { return p.A + (size_t)c * TS * N + (size_t)r * TS; };
    // after a CTA barrier behind the stores: the barrier orders every thread's stores before thread 0's release (which is a
    // gpu-scope fence followed by the store; a separate __threadfence in front of it would fence twice)
    auto publish = [&](unsigned* flag) {
        if (tid == 0) st_release(flag, epoch);
    };

    if (blockIdx.x == 2) {  // block row 0 and block column 0 are A itself: final / X-ready from the start
        for (int t = tid; t < nt; t += LU_THREADS) {
            st_release(p.flags + t, epoch);
            st_release(p.xready + (size_t)t * nt, epoch);
        }
    }
    for (;;) {
        __syncthreads();  // the previous task is finished with s_task and the shared tiles
        if (tid == 0) s_task = (int)atomicAdd(p.counter, 1u);
        __syncthreads();
        const int task = s_task;
        if (task >= p.ntasks) break;
        const int code = p.order[task], type = code >> 28, i = (code >> 14) & 0x3fff, j = code & 0x3fff;
        const bool has_tile = j < nt;  // the upper task (nt-1, nt) only finishes L_{nt-1,nt-2}
        // kl: the term that is formed from X and Z on the fly (-1: none); the plain left-looking sum runs over k < m
        const int kl = has_tile ? lu_kl(i, j) : i - 1;
        const int m = (has_tile && kl > 0) ? kl : 0;
        double* Cg = has_tile ? tile(i, j) : nullptr;
        SWW_WSTAMP(0);

        // own tile -> registers (fragment layout), sum = 0
        double c0[4][2][2], acc[4][2][2];
#pragma unroll
        SWW_FRAG_LOOP {
            c0[x][y][e] = (mm && has_tile) ? Cg[(size_t)f.col(y, e) * N + f.row(x)] : 0.0;
            acc[x][y][e] = 0.0;
        }
        // The plain terms k < m, warp-specialized: the three warps that have no part in the products are the PRODUCERS -- they wait for
        // the flags of the two operand tiles of term k (U_kj is final a generation before L_ik), fetch them into the next stage of
        // the ring as soon as the MMA warps have released it, and go on to term k + 1; each producer thread's arrival on the
        // stage's full barrier fires when its copies have landed.  The eight MMA warps do nothing but wait, multiply and release.
        if (mm) {
            for (int k = 0; k < m; k++) {
                const unsigned g = it + (unsigned)k;
                const int buf = (int)(g % LU_RING);
                mbar_wait(&full[buf], (g / LU_RING) & 1u);
                mma_tile64(acc, sA + buf * TS * LDO, sB + buf * TS * LDO, f);
                __syncwarp();
                if ((tid & 31) == 0) mbar_arrive(&empty[buf]);
            }
        } else {
            const int t = tid - 256;  // 0..95
            for (int k = 0; k < m; k++) {
                const unsigned g = it + (unsigned)k;
                const int buf = (int)(g % LU_RING);
                if (t == 0) {
                    spin_tight(p.flags + (size_t)k * nt + j, epoch);
                    spin_tight(p.flags + (size_t)i * nt + k, epoch);
                }
                asm volatile("bar.sync 6, 96;" ::: "memory");  // the producers: the acquire of lane 0 orders everybody's copies behind the flags
                mbar_wait(&empty[buf], ((g / LU_RING) & 1u) ^ 1u);
                tile_async(sA + buf * TS * LDO, tile(i, k), N, t, LU_THREADS - 256);
                tile_async(sB + buf * TS * LDO, tile(k, j), N, t, LU_THREADS - 256);
                cp_arrive_on(&full[buf]);
            }
            cp_commit();
            cp_wait<0>();  // nothing of mine is in flight when the task goes on to its last term (which re-uses the stages)
        }
        it += (unsigned)m;
        __syncthreads();  // every plain term is in acc; the ring is free
        auto store_tile = [&](double* dst, size_t ld, const double (&v)[4][2][2]) {
            if (mm) {
#pragma unroll
                SWW_FRAG_LOOP dst[(size_t)f.col(y, e) * ld + f.row(x)] = v[x][y][e];
            }
        };
        // ---- the last term, k = kl: L = X Z_kl = 2 X + X F_kl formed here, then sum += L U_{kl,j}
        // X: the left neighbour X_{i,kl} in place (lower tiles, P) or the staging block Xs[i] (upper tiles)
        double l[4][2][2];
        const bool finish_left = kl >= 0 && (type == T_L || (type == T_U && j == i + 1));
        SWW_WSTAMP(1);
        if (kl >= 0) {
            const bool upper = (type == T_U);
            const double* Xg = upper ? p.Xs + (size_t)i * TS * TS : tile(i, kl);
            const size_t ldx = upper ? (size_t)TS : (size_t)N;
            if (tid < 2) {  // inputs that are final long before Z_kl
                const unsigned* fl = (tid == 0) ? (upper ? p.xflags + i : p.xready + (size_t)i * nt + kl)
                                                : (has_tile ? p.flags + (size_t)kl * nt + j : nullptr);
                if (fl) spin_until(fl, epoch);
            }
            __syncthreads();
            tile_async(sA, Xg, ldx, tid, LU_THREADS);                                  // X_{i,kl}
            if (has_tile) tile_async(sB + TS * LDO, tile(kl, j), N, tid, LU_THREADS);  // U_{kl,j}
            cp_commit();
            SWW_WSTAMP(2);
            if (tid == 0) spin_tight(p.zflags + kl, epoch);
            __syncthreads();
            SWW_WSTAMP(3);
            tile_async(sB, p.Fs + (size_t)kl * TS * TS, TS, tid, LU_THREADS);          // F_kl
            cp_commit();
            cp_wait<0>();
            __syncthreads();
            SWW_WSTAMP(4);
            if (type == T_P && tid == 0) st_release(p.pflags + i, epoch);  // X_{i,i-2} has been read (nothing was written: no fence)
            if (mm) {
#pragma unroll
                SWW_FRAG_LOOP l[x][y][e] = 2.0 * sA[f.col(y, e) * LDO + f.row(x)];
                mma_tile64(l, sA, sB, f);
#pragma unroll
                SWW_FRAG_LOOP sA[TS * LDO + f.col(y, e) * LDO + f.row(x)] = l[x][y][e];  // L as an A operand, second stage
            }
            __syncthreads();
            // The finished left neighbour L_{i,kl} goes out at once (the tasks of the next generation sum it as a plain term and
            // must be through with that before Z_{kl+1} arrives) -- by the three warps that have no part in the products, from
            // the shared-memory copy, while the MMA warps go on with the last term.
            if (mm) {
                if (has_tile) mma_tile64(acc, sA + TS * LDO, sB + TS * LDO, f);
            } else if (finish_left) {
                const int t = tid - 256;  // 0..95
                if (type == T_L && j == i - 1 && i >= 2 && t == 0) spin_until(p.pflags + i, epoch);  // P of this row reads X_{i,i-2} too
                asm volatile("bar.sync 5, 96;" ::: "memory");
                double* Lg = tile(i, kl);
                const double* Ls = sA + TS * LDO;
                for (int c = t; c < TS * TS / 2; c += 96) {
                    const int col = c >> 5, ch = (c & 31) * 2;
                    *reinterpret_cast<double2*>(Lg + (size_t)col * N + ch) = *reinterpret_cast<const double2*>(Ls + col * LDO + ch);
                }
                asm volatile("bar.sync 5, 96;" ::: "memory");
                if (t == 0) st_release(p.flags + (size_t)i * nt + kl, epoch);
            }
        }
        SWW_WSTAMP(5);
#pragma unroll
        SWW_FRAG_LOOP c0[x][y][e] -= acc[x][y][e];
        // ---- publish X_ij / U_ij / P_i
        if (has_tile) {
            const bool staged = (type == T_L && j == i - 1);
            store_tile(staged ? p.Xs + (size_t)i * TS * TS : Cg, staged ? (size_t)TS : (size_t)N, c0);
            __syncthreads();
            publish(staged ? p.xflags + i : (type == T_L ? p.xready + (size_t)i * nt + j : p.flags + (size_t)i * nt + j));
            SWW_WSTAMP(6);
        }
    }
}

// Claim order: generation g = -1, 0, 1, ... of the inverse Z_g a task waits for; within a generation first what the spine
// needs for step g + 2 (P_{g+2} -- ahead of the task of tile (g+2, g+1), which waits for its pflag --, the tiles (g+2, g+1) and
// (g+1, g+2)), then block column g+1 / block row g+1 by distance from the diagonal.  Block row 0 and block column 0 need no
// task (A itself), except tile (1, 0), which is copied to its staging block.
static void build_order(int nt, std::vector<int>& o) {
    o.clear();
    for (int g = -1; g <= nt - 2; g++) {
        if (g + 2 >= 2 && g + 2 <= nt - 1) o.push_back(lu_task(T_P, g + 2, g + 2));
        if (g + 2 <= nt - 1) o.push_back(lu_task(T_L, g + 2, g + 1));
        if (g >= 0) o.push_back(lu_task(T_U, g + 1, g + 2));  // j = nt for the last row: only finishes L_{nt-1,nt-2}
        if (g >= 0)
            for (int d = 1; g + 2 + d <= nt - 1; d++) {
                o.push_back(lu_task(T_L, g + 2 + d, g + 1));
                o.push_back(lu_task(T_U, g + 1, g + 2 + d));
            }
    }
}

int lu_alloc(sww_dtn_s* d) {
    const int N = d->N;
    d->lu_order = nullptr;
    d->lu_flags = nullptr;
    d->lu_epoch = 0;
    d->tr_flags = nullptr;
    if (N <= TS) return SWW_OK;
    const int nt = N / TS;
    std::vector<int> o;
    build_order(nt, o);
    d->lu_ntasks = (int)o.size();
    const size_t nflags = 2 * (size_t)nt * nt + 3 * nt + 1;
    if (cudaMalloc(&d->lu_order, sizeof(int) * o.size()) != cudaSuccess) return SWW_ENOMEM;
    if (cudaMalloc(&d->lu_flags, sizeof(unsigned) * nflags) != cudaSuccess) return SWW_ENOMEM;
    SWW_CUDA(cudaMemcpyAsync(d->lu_order, o.data(), sizeof(int) * o.size(), cudaMemcpyHostToDevice, d->stream));
    SWW_CUDA(cudaMemsetAsync(d->lu_flags, 0, sizeof(unsigned) * nflags, d->stream));
    if (cudaMalloc(&d->tr_flags, sizeof(unsigned)) != cudaSuccess) return SWW_ENOMEM;  // the claim counter of the dataflow solves
    SWW_CUDA(cudaMemsetAsync(d->tr_flags, 0, sizeof(unsigned), d->stream));
    SWW_CUDA(cudaStreamSynchronize(d->stream));  // o goes out of scope
    return SWW_OK;
}

int run_lu(sww_dtn_s* d) {
    const int N = d->N, nb = (N < NB) ? N : NB, nblk = N / nb;
    cudaStream_t st = d->stream;
    double* Es = d->invD;                           // N <= 64: inv(L) - I ; larger N: the staging blocks Xs of the dataflow LU
    double* Fs = d->invD + (size_t)nblk * nb * nb;
    constexpr int SINGLE_SMEM = (TS * LDT + 576) * (int)sizeof(double);
    static DeviceOnce attr_once;
    if (attr_once.first()) {
        SWW_CUDA(cudaFuncSetAttribute(k_lu_single, cudaFuncAttributeMaxDynamicSharedMemorySize, SINGLE_SMEM));
        SWW_CUDA(cudaFuncSetAttribute(k_lu_dataflow, cudaFuncAttributeMaxDynamicSharedMemorySize, LU_SMEM_BYTES));
    }
    if (nblk == 1) {
        SWW_BEGIN(KC_LU, st);
        k_lu_single<<<1, 256, SINGLE_SMEM, st>>>(d->LU, nb, Es, Fs, d->status);
        SWW_LAUNCHED();
        SWW_CUDA(cudaGetLastError());
        return SWW_OK;
    }
    LuArgs a;
    a.A = d->LU;
    a.N = N;
    a.nt = nblk;
    a.ntasks = d->lu_ntasks;
    a.order = d->lu_order;
    a.counter = d->lu_flags;
    a.flags = d->lu_flags + 1;
    a.xready = a.flags + (size_t)nblk * nblk;
    a.xflags = a.xready + (size_t)nblk * nblk;
    a.pflags = a.xflags + nblk;
    a.zflags = a.pflags + nblk;
    a.epoch = ++d->lu_epoch;
    a.Fs = Fs;
    a.Xs = Es;
    a.Vs = d->invD + 2 * (size_t)nblk * nb * nb;
    a.status = d->status;
    SWW_CUDA(cudaMemsetAsync(a.counter, 0, sizeof(unsigned), st));
    // clusters of two CTAs: cluster 0 is the spine, every other CTA works on its own (an even grid, one CTA per SM)
    const int grid = std::min(sm_count() & ~1, (3 + a.ntasks) & ~1);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(LU_THREADS);
    cfg.dynamicSmemBytes = LU_SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    SWW_BEGIN(KC_LU, st);
    SWW_CUDA(cudaLaunchKernelEx(&cfg, k_lu_dataflow, a));
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

#ifdef SWW_LU_TRACE
extern "C" int sww_debug_lu_trace(unsigned long long* dst, int n) {
    return cudaMemcpyFromSymbol(dst, g_lu_trace, sizeof(unsigned long long) * n) == cudaSuccess ? 0 : -3;
}
#endif

// N <= 64 (a single diagonal block): one CTA per column, x = (2 I + F)(I + E) b with the same compensation as below
__global__ void __launch_bounds__(64) k_solve_small(int N, const double* __restrict__ E, const double* __restrict__ F,
                                                    double* __restrict__ B, double* __restrict__ Blo) {
    __shared__ double v[64];
    const int i = threadIdx.x;
    double* b = B + (size_t)blockIdx.x * N;
    double bi = 0.0;
    if (i < N) v[i] = bi = b[i];
    __syncthreads();
    double acc = 0.0;
    if (i < N)
        for (int c = 0; c < i; c++) acc = fma(E[(size_t)c * N + i], v[c], acc);
    double yh = bi + acc;
    double bb = yh - bi;
    double yl = (bi - (yh - bb)) + (acc - bb);
    __syncthreads();
    if (i < N) v[i] = yh;
    __syncthreads();
    if (i < N) {
        acc = 0.0;
        for (int c = i; c < N; c++) acc = fma(F[(size_t)c * N + i], v[c], acc);
        double c2 = 2.0 * yh;
        double s = __dadd_rn(c2, acc);
        bb = __dsub_rn(s, c2);
        double err = __dadd_rn(__dsub_rn(c2, __dsub_rn(s, bb)), __dsub_rn(acc, bb));
        double lo = fma(2.0, yl, err);
        double t = __dadd_rn(s, lo);
        b[i] = t;
        Blo[(size_t)blockIdx.x * N + i] = __dsub_rn(lo, __dsub_rn(t, s));
    }
}

// ------------------------------------------------------------------------------------------------ the persistent dataflow TRSM
// Solve L Y = B, then U X = Y (block LU of k_lu_dataflow), for a batch of columns, in place, as ONE persistent kernel in the
// same style.  A task is (phase, row block i, column slab s of WS columns).  Forward:  Y_i = B_i - sum_{k<i} L_ik Y_k;
// backward:  X_i = (2 I + F_i)(Y_i - sum_{k>i} U_ik X_k),  2 I + F_i = inv(S_i).  The sums run left-looking in DMMA fragments over the blocks that are
// already final; the chain of a slab is sequential in i, different slabs and the accumulation over old blocks run in parallel.
// Tasks are claimed in dependency order (forward i ascending, then backward i descending), so a claimed task only waits for
// tasks claimed earlier.
// Hand-over between tasks: THE DATA IS THE FLAG.  The forward results go to Yh / Yl and the backward results to Xh, scratch
// buffers filled with an all-ones bit pattern (a NaN no computation produces) before the launch; a consumer loads the block
// it needs (cp.async.cg / ld.cg, i.e. from L2) and simply reloads while any entry still shows the pattern.  Every entry is one
// aligned 8-byte store, so it is either absent or final: no fence, no release/acquire pair, no separate flag -- a link of the
// chain costs one store-to-L2 plus one load-from-L2 latency instead of store + fence + flag + poll + load (~2 us).
// Accuracy: the O(1) vectors are carried as hi + lo (B + Blo).  P = sum L_ik Y_k is accumulated from zero (its terms are
// O(1/N)) and folded into a two-sum (hi, lo) pair every TR_FOLD blocks; B_i - P and the diagonal-block products are added by
// error-free two-sums, so each block of the result is the correctly rounded sum plus a remainder word -- the density is
// differentiated afterwards, which amplifies white rounding noise by ~N/3.
struct TrsmArgs {
    const double* A;     // LU factors, N x N column-major (L multipliers below the diagonal, U above)
    const double* Fs;    // nt blocks of 64 x 64 (column-major, ld 64): inv(S_i) - 2 I
    const double* Vs;    // nt blocks of 64 x 64 (column-major, ld 64): V_i = inv(S_i) U_{i,i+1}
    double *B, *Blo;     // N x (ns*WS) column-major, ld = N; in: right-hand sides (Blo ignored), out: solution hi, lo
    int N, nt, ns;       // nt row blocks of 64, ns column slabs
    double *Yh, *Yl, *Xh;  // scratch, same shape as B: forward result (hi, lo) and backward result (hi); pre-filled with TR_ABSENT
    unsigned* counter;
    int* status;
};
constexpr long long TR_ABSENT = -1LL;       // bit pattern of "not written yet" (cudaMemset 0xFF)
constexpr int TR_SPIN_LIMIT = 1 << 17;      // reloads (~1 us each) before a task gives up: SWW_ECUDA, and every other task stops polling
constexpr int TR_FOLD = 4;
// The reserved pattern never enters the scratch vectors: a NaN with that payload (an input column filled with 0xFF bytes, say)
// is replaced by the canonical quiet NaN where right-hand sides are loaded and before every hand-over store.
__device__ __forceinline__ double tr_canon(double v) {
    return (__double_as_longlong(v) == TR_ABSENT) ? __longlong_as_double(0x7FF8000000000000LL) : v;
}
__device__ __forceinline__ int ld_status(const int* p) {
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ void two_sum_d(double a, double b, double& s, double& e) {
    s = __dadd_rn(a, b);
    const double bb = __dsub_rn(s, a);
    e = __dadd_rn(__dsub_rn(a, __dsub_rn(s, bb)), __dsub_rn(b, bb));
}

template <int WS>
struct TrsmCfg {
    static constexpr int WC = WS / 8;               // warps across the slab's columns (8 columns per warp): 1, 2 or 4
    static constexpr int WR = 8 / WC;               // warps across the 64 rows
    static constexpr int FM = (TS / WR) / 8;        // 8 x 8 fragments per warp along the rows
    static constexpr int WSP = WC * 8;              // columns covered = WS
    static constexpr int SMEM = (3 * TS * LDO + 3 * WS * LDO) * (int)sizeof(double) + 256;
};

template <int WS>
__global__ void __launch_bounds__(256, 1) k_trsm_dataflow(TrsmArgs p) {
    using C = TrsmCfg<WS>;
    extern __shared__ __align__(16) double tr_sm[];
    double* sA = tr_sm;                    // 2 stages of the factor tile as As[k][r]
    double* sD = sA + 2 * TS * LDO;        // the diagonal block F_i of the backward sweep, as As[k][r]
    double* sB = sD + TS * LDO;            // 2 stages of the solution tile as Bs[n][k]
    double* sZ = sB + 2 * WS * LDO;        // z as Bs[n][k] (the B operand of the diagonal product)
    __shared__ int s_task, s_abort;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wr = warp % C::WR, wc = warp / C::WR, fr = lane >> 2, fk = lane & 3;
    const int N = p.N, nt = p.nt, ns = p.ns;
    const int row0 = wr * (TS / C::WR) + fr;   // + 8 x : row of this lane's fragment element
    const int col0 = wc * 8 + 2 * fk;          // + e   : column within the slab

    for (;;) {
        __syncthreads();
        if (tid == 0) {
            s_task = (int)atomicAdd(p.counter, 1u);
            s_abort = ld_status(p.status) != SWW_OK;
        }
        __syncthreads();
        int task = s_task;
        if (task >= 2 * nt * ns) break;
        if (s_abort) break;  // some task gave up (or the handle already carries an error): stop polling, leave at once
        const int phase = task >= nt * ns;
        if (phase) task -= nt * ns;
        const int s = task % ns, i = phase ? nt - 1 - task / ns : task / ns;
        const int m = phase ? nt - 1 - i : i;  // number of finished blocks this one depends on
        const size_t blk = (size_t)s * WS * N + (size_t)i * TS;
        double* Bg = p.B + blk;
        double* Lg = p.Blo + blk;
        const double* Vin = phase ? p.Xh : p.Yh;  // the vector this sweep consumes block by block
        auto kblock = [&](int kk) { return phase ? nt - 1 - kk : kk; };
        // the factors are final before this kernel starts: their tiles are requested one step ahead of the flags, so that
        // only the (small) solution block is loaded behind the flag on the chain of a slab
        auto issueA = [&](int kk, int buf) {
            const int k = kblock(kk);
            const bool front = phase && kk == m - 1;  // backward: the term of block i + 1 goes through V_i = inv(S_i) U_{i,i+1}
            const double* Ag = front ? p.Vs + (size_t)i * TS * TS : p.A + (size_t)k * TS * N + (size_t)i * TS;  // factor tile (i, k)
            const size_t lda = front ? (size_t)TS : (size_t)N;
            double* a = sA + buf * TS * LDO;
            for (int c = tid; c < TS * TS / 2; c += 256) {
                const int col = c >> 5, ch = (c & 31) * 2;
                cp16(a + col * LDO + ch, Ag + col * lda + ch);
            }
        };
        // true if any of the entries THIS thread requested in issueY is still absent (call after its cp.async group completed)
        auto absentY = [&](int buf) {
            const double* b = sB + buf * WS * LDO;
            bool bad = false;
            for (int c = tid; c < WS * TS / 2; c += 256) {
                const int col = c >> 5, ch = (c & 31) * 2;
                bad |= (__double_as_longlong(b[col * LDO + ch]) == TR_ABSENT) | (__double_as_longlong(b[col * LDO + ch + 1]) == TR_ABSENT);
            }
            return bad;
        };
        // CTA-uniform: true when this wait must end -- the spin limit is hit (this task records SWW_ECUDA) or, looked at every
        // 64 reloads, some other task already did
        auto spin_out = [&](int spin) -> bool {
            if (spin > TR_SPIN_LIMIT) {
                if (tid == 0) atomicCAS(p.status, SWW_OK, SWW_ECUDA);
                return true;
            }
            if ((spin & 63) != 63) return false;
            return __syncthreads_or(tid == 0 && ld_status(p.status) != SWW_OK) != 0;
        };
        auto issueY = [&](int kk, int buf) {
            const int k = kblock(kk);
            const double* Yg = Vin + (size_t)s * WS * N + (size_t)k * TS;          // solution block k of this slab
            double* b = sB + buf * WS * LDO;
            for (int c = tid; c < WS * TS / 2; c += 256) {
                const int col = c >> 5, ch = (c & 31) * 2;
                cp16(b + col * LDO + ch, Yg + (size_t)col * N + ch);
            }
        };
        double acc[C::FM][2];
        auto mma_tile = [&](const double* a, const double* b) {
            const double* as = a + row0;
            const double* bs = b + (wc * 8 + fr) * LDO;
#pragma unroll
            for (int k4 = 0; k4 < TS; k4 += 4) {
                const double bf = bs[k4 + fk];
#pragma unroll
                for (int x = 0; x < C::FM; x++) lu_dmma884(acc[x][0], acc[x][1], as[(k4 + fk) * LDO + x * 8], bf);
            }
        };

        double bh[C::FM][2], bl[C::FM][2], ph[C::FM][2], pl[C::FM][2];
        for (int spin = 0;; spin++) {  // backward: the block's own forward result (hi and lo), reloaded until all of it is there
            bool bad = false;
#pragma unroll
            for (int x = 0; x < C::FM; x++)
#pragma unroll
                for (int e = 0; e < 2; e++) {
                    const size_t o = (size_t)(col0 + e) * N + row0 + x * 8;
                    if (phase) {
                        bh[x][e] = __ldcg(p.Yh + blk + o);
                        bl[x][e] = __ldcg(p.Yl + blk + o);
                        bad |= (__double_as_longlong(bh[x][e]) == TR_ABSENT) | (__double_as_longlong(bl[x][e]) == TR_ABSENT);
                    } else {
                        bh[x][e] = tr_canon(Bg[o]);
                        bl[x][e] = 0.0;  // the forward sweep starts from plain fp64 right-hand sides
                    }
                    acc[x][e] = ph[x][e] = pl[x][e] = 0.0;
                }
            if (!phase || !__syncthreads_or(bad)) break;
            if (spin_out(spin)) break;
        }
        auto fold = [&]() {  // (ph, pl) += acc, error-free; acc = 0
#pragma unroll
            for (int x = 0; x < C::FM; x++)
#pragma unroll
                for (int e = 0; e < 2; e++) {
                    double s_, e_;
                    two_sum_d(ph[x][e], acc[x][e], s_, e_);
                    ph[x][e] = s_;
                    pl[x][e] += e_;
                    acc[x][e] = 0.0;
                }
        };
        if (phase) {  // block LU: L has identity diagonal blocks, only the backward sweep has a diagonal product
            const double* Dg = p.Fs + (size_t)i * TS * TS;
            for (int c = tid; c < TS * TS / 2; c += 256) {
                const int col = c >> 5, ch = (c & 31) * 2;
                cp16(sD + col * LDO + ch, Dg + col * TS + ch);  // As[k][r] = D[r][k]
            }
            cp_commit();
        }
        // The factor tile of step kk + 1 is requested while step kk computes (its buffer was released by the barrier that ended
        // step kk - 1); the solution block is asked for at its own step (asking one step early did not pay: on the chain it
        // is never there yet, behind the front the load is hidden by the other resident work).
        if (m > 0) {
            issueA(0, 0);
            cp_commit();
        }
        // one term: the solution block is asked for at its own step and reloaded until complete, then the product
        auto term = [&](int kk, bool more) {
            issueY(kk, kk & 1);
            cp_commit();
            if (more) {
                issueA(kk + 1, (kk + 1) & 1);
                cp_commit();
                cp_wait<1>();
            } else {
                cp_wait<0>();
            }
            // Not there yet (the chain front): every thread polls ITS chunks with plain L2 loads into registers until none shows
            // the absent pattern and puts them into the tile by hand -- no copy, wait and CTA-wide vote per round, one barrier at
            // the end (which also makes the tiles visible to all).  A thread that gives up records SWW_ECUDA; the others look at
            // the status word every 256 rounds.
            if (absentY(kk & 1)) {
                const double* Yg = Vin + (size_t)s * WS * N + (size_t)kblock(kk) * TS;
                double* b = sB + (kk & 1) * WS * LDO;
                constexpr int NCH = (WS * TS / 2 + 255) / 256;
                double2 v[NCH];
                for (int spin = 0;; spin++) {
                    bool miss = false;
#pragma unroll
                    for (int q = 0; q < NCH; q++) {
                        const int c = tid + q * 256;
                        if (c < WS * TS / 2) {
                            const int col = c >> 5, ch = (c & 31) * 2;
                            v[q] = __ldcg(reinterpret_cast<const double2*>(Yg + (size_t)col * N + ch));
                            miss |= (__double_as_longlong(v[q].x) == TR_ABSENT) | (__double_as_longlong(v[q].y) == TR_ABSENT);
                        }
                    }
                    if (!miss) break;
                    if (spin > 8 * TR_SPIN_LIMIT) {
                        atomicCAS(p.status, SWW_OK, SWW_ECUDA);
                        break;
                    }
                    if ((spin & 255) == 255 && ld_status(p.status) != SWW_OK) break;
                }
#pragma unroll
                for (int q = 0; q < NCH; q++) {
                    const int c = tid + q * 256;
                    if (c < WS * TS / 2) {
                        const int col = c >> 5, ch = (c & 31) * 2;
                        *reinterpret_cast<double2*>(b + col * LDO + ch) = v[q];
                    }
                }
            }
            __syncthreads();
            mma_tile(sA + (kk & 1) * TS * LDO, sB + (kk & 1) * WS * LDO);
        };
        // forward: all m terms; backward: the terms of the blocks k > i + 1 (the front term comes last, through V_i)
        const int mb = phase ? (m > 0 ? m - 1 : 0) : m;
        for (int kk = 0; kk < mb; kk++) {
            term(kk, kk + 1 < m);
            if ((kk % TR_FOLD) == TR_FOLD - 1) fold();
            __syncthreads();
        }
        fold();
        // z = (bh + bl) - (ph + pl) as sh + sl
        double sh[C::FM][2], sl[C::FM][2];
#pragma unroll
        for (int x = 0; x < C::FM; x++)
#pragma unroll
            for (int e = 0; e < 2; e++) {
                double s_, e_;
                two_sum_d(bh[x][e], -ph[x][e], s_, e_);
                sh[x][e] = s_;
                sl[x][e] = e_ + (bl[x][e] - pl[x][e]);
                if (phase) sZ[(col0 + e) * LDO + row0 + x * 8] = s_;  // Bs[n][k] = z[k][n]
            }
        if (phase) {
            // backward: w = Z_i z = 2 z + F_i z (before the front block is there), then x_i = w - V_i x_{i+1}
            if (m >= 1) cp_wait<1>();  // F_i (the oldest group); the front factor tile may still be in flight
            else cp_wait<0>();
            __syncthreads();
            mma_tile(sD, sZ);
#pragma unroll
            for (int x = 0; x < C::FM; x++)
#pragma unroll
                for (int e = 0; e < 2; e++) {
                    double t_, e_;
                    two_sum_d(2.0 * sh[x][e], acc[x][e], t_, e_);
                    sh[x][e] = t_;
                    sl[x][e] = fma(2.0, sl[x][e], e_);
                    acc[x][e] = 0.0;
                }
            if (m > 0) {
                term(m - 1, false);
#pragma unroll
                for (int x = 0; x < C::FM; x++)
#pragma unroll
                    for (int e = 0; e < 2; e++) {
                        double t_, e_;
                        two_sum_d(sh[x][e], -acc[x][e], t_, e_);
                        sh[x][e] = t_;
                        sl[x][e] += e_;
                    }
            }
        }
#pragma unroll
        for (int x = 0; x < C::FM; x++)
#pragma unroll
            for (int e = 0; e < 2; e++) {  // first what the chain waits for: the high words of the whole block
                const size_t o = (size_t)(col0 + e) * N + row0 + x * 8;
                const double hi = __dadd_rn(sh[x][e], sl[x][e]);
                sl[x][e] = __dsub_rn(sl[x][e], __dsub_rn(hi, sh[x][e]));
                sh[x][e] = hi;
                (phase ? p.Xh : p.Yh)[blk + o] = tr_canon(hi);
            }
#pragma unroll
        for (int x = 0; x < C::FM; x++)
#pragma unroll
            for (int e = 0; e < 2; e++) {
                const size_t o = (size_t)(col0 + e) * N + row0 + x * 8;
                if (phase) {  // x_i: the result (hi, lo)
                    Bg[o] = sh[x][e];
                    Lg[o] = sl[x][e];
                } else {      // y_i: the low word for this block's backward task
                    p.Yl[blk + o] = tr_canon(sl[x][e]);
                }
            }
    }
}

// ------------------------------------------------------------------------------------------------ the same solve, warp-specialized
// k_trsm_ws: the tasks, the hand-over protocol and the compensated arithmetic of k_trsm_dataflow, but the operands come through
// a ring of ST stages filled by two dedicated LOADER warps (cp.async, mbarrier full / empty pairs) while the eight MMA warps do
// nothing but fragment loads and DMMAs: the loaders run up to ST - 1 steps ahead of the products, look for the absent pattern
// in the solution blocks they fetched (each thread in its own chunks) and ask L2 again until a block is complete, so the MMA
// warps never poll, never issue a copy and meet no CTA-wide barrier inside a task.
// Backward sweep: x_i = Z_i (y_i - sum_{k>i+1} U_ik x_k) - V_i x_{i+1} with V_i = Z_i U_{i,i+1} kept by the LU spine: the product
// with the diagonal block is done before the front block x_{i+1} arrives, a link of the chain is one product in both sweeps.
// named barrier 1 with an OR reduction among the 256 threads of the MMA warps
__device__ __forceinline__ bool mma_bar_or(bool pred) {
    int r;
    asm volatile(
        "{\n.reg .pred p, q;\nsetp.ne.b32 p, %1, 0;\nbar.red.or.pred q, 1, 256, p;\nselp.b32 %0, 1, 0, q;\n}"
        : "=r"(r)
        : "r"((int)pred)
        : "memory");
    return r != 0;
}

template <int WS>
struct TrsmWsCfg {
    static constexpr int WC = WS / 8;               // MMA warps across the slab's columns (8 columns per warp)
    static constexpr int WR = 8 / WC;               // MMA warps across the 64 rows
    static constexpr int FM = (TS / WR) / 8;        // 8 x 8 fragments per warp along the rows
    static constexpr int ST = WS <= 32 ? 3 : 2;     // stages of the operand ring
    static constexpr int THREADS = 320;             // 8 MMA warps + 2 loader warps
    static constexpr int NLOAD = 64;
    // ring (factor tile + solution tile per stage), F_i, z (the B operand of the diagonal product)
    static constexpr int SMEM = ((ST + 1) * TS * LDO + (ST + 1) * WS * LDO) * (int)sizeof(double) + 256;
};

template <int WS>
__global__ void __launch_bounds__(320, 1) k_trsm_ws(TrsmArgs p) {
    using C = TrsmWsCfg<WS>;
    constexpr int ST = C::ST, NL = C::NLOAD;
    extern __shared__ __align__(16) double tr_sm[];
    double* sA = tr_sm;                    // ST stages of the factor tile as As[k][r]
    double* sD = sA + ST * TS * LDO;       // the diagonal block F_i of the backward sweep, as As[k][r]
    double* sB = sD + TS * LDO;            // ST stages of the solution tile as Bs[n][k]
    double* sZ = sB + ST * WS * LDO;       // z as Bs[n][k]
    __shared__ unsigned long long full[ST], empty[ST], fullD;
    __shared__ int s_task, s_abort;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool loader = warp >= 8;
    const int lt = tid - 256;                  // loader thread index 0..63
    const int wr = warp % C::WR, wc = warp / C::WR, fr = lane >> 2, fk = lane & 3;
    const int N = p.N, nt = p.nt, ns = p.ns;
    const int row0 = wr * (TS / C::WR) + fr;   // + 8 x : row of this lane's fragment element
    const int col0 = wc * 8 + 2 * fk;          // + e   : column within the slab
    if (tid == 0) {
        for (int s = 0; s < ST; s++) {
            mbar_init(&full[s], NL);
            mbar_init(&empty[s], 8);
        }
        mbar_init(&fullD, NL);
        s_abort = 0;
    }
    unsigned it = 0;   // ring position: products done so far by this CTA (the same number in every thread)
    unsigned nd = 0;   // backward tasks done so far (phase of fullD)

    for (;;) {
        __syncthreads();  // the previous task is through with the ring, sD and sZ; the barriers are initialised
        if (tid == 0) {
            s_task = (int)atomicAdd(p.counter, 1u);
            if (ld_status(p.status) != SWW_OK) s_abort = 1;
        }
        __syncthreads();
        int task = s_task;
        if (task >= 2 * nt * ns) break;
        if (s_abort) break;  // some task gave up (or the handle already carries an error): stop polling, leave at once
        const int phase = task >= nt * ns;
        if (phase) task -= nt * ns;
        const int s = task % ns, i = phase ? nt - 1 - task / ns : task / ns;
        const int m = phase ? nt - 1 - i : i;  // number of finished blocks this one depends on
        const size_t blk = (size_t)s * WS * N + (size_t)i * TS;
        const double* Vin = phase ? p.Xh : p.Yh;  // the vector this sweep consumes block by block

        if (loader) {
            // ---------------------------------------------------------------------------------- the loader warps
            auto kblock = [&](int kk) { return phase ? nt - 1 - kk : kk; };
            auto issueA = [&](int kk, int buf) {
                const bool front = phase && kk == m - 1;  // backward: the term of block i + 1 goes through V_i = inv(S_i) U_{i,i+1}
                const double* Ag = front ? p.Vs + (size_t)i * TS * TS : p.A + (size_t)kblock(kk) * TS * N + (size_t)i * TS;  // factor tile (i, k)
                const size_t lda = front ? (size_t)TS : (size_t)N;
                double* a = sA + buf * TS * LDO;
#pragma unroll 4
                for (int c = lt; c < TS * TS / 2; c += NL) {
                    const int col = c >> 5, ch = (c & 31) * 2;
                    cp16(a + col * LDO + ch, Ag + col * lda + ch);
                }
            };
            auto issueY = [&](int kk, int buf) {
                const double* Yg = Vin + (size_t)s * WS * N + (size_t)kblock(kk) * TS;   // solution block k of this slab
                double* b = sB + buf * WS * LDO;
#pragma unroll 4
                for (int c = lt; c < WS * TS / 2; c += NL) {
                    const int col = c >> 5, ch = (c & 31) * 2;
                    cp16(b + col * LDO + ch, Yg + (size_t)col * N + ch);
                }
            };
            if (phase) {  // block LU: L has identity diagonal blocks, only the backward sweep has a diagonal product
                const double* Dg = p.Fs + (size_t)i * TS * TS;
                for (int c = lt; c < TS * TS / 2; c += NL) {
                    const int col = c >> 5, ch = (c & 31) * 2;
                    cp16(sD + col * LDO + ch, Dg + col * TS + ch);  // As[k][r] = D[r][k]
                }
                cp_commit();
            }
            int issued = 0;
            auto issue_stage = [&]() {
                const unsigned g = it + (unsigned)issued;
                const int buf = (int)(g % ST);
                mbar_wait(&empty[buf], ((g / ST) & 1u) ^ 1u);  // the products of the stage that used this buffer are done
                issueA(issued, buf);
                issueY(issued, buf);
                cp_commit();
                issued++;
            };
            while (issued < m && issued < ST - 1) issue_stage();
            for (int kk = 0; kk < m; kk++) {
                const int buf = (int)((it + (unsigned)kk) % ST);
                if (issued - 1 - kk >= 1) cp_wait<1>();
                else cp_wait<0>();
                if (kk == 0 && phase) mbar_arrive(&fullD);  // the group of F_i is older than that of stage 0
                // My part of the block as the copy brought it: complete?  If not (the chain front: the producer has not stored it
                // yet), poll with plain L2 loads into registers -- first one sentinel chunk (1 KB of polling traffic per CTA and
                // round; every row below waits for the same block), then all of my chunks until none shows the absent pattern --
                // and put the block into the stage by hand.  A round of register loads is a third of a cp.async round + rescan.
                const double* Yg = Vin + (size_t)s * WS * N + (size_t)kblock(kk) * TS;
                double* b = sB + buf * WS * LDO;
                constexpr int NCH = WS * TS / 2 / NL;  // 16-byte chunks per loader thread
                bool bad = false;
#pragma unroll
                for (int q = 0; q < NCH; q++) {
                    const int c = lt + q * NL, col = c >> 5, ch = (c & 31) * 2;
                    const double2 v = *reinterpret_cast<const double2*>(b + col * LDO + ch);
                    bad |= (__double_as_longlong(v.x) == TR_ABSENT) | (__double_as_longlong(v.y) == TR_ABSENT);
                }
                if (bad) {
                    bool out = false;
                    // the task whose LAST dependency this block is sits on the chain of its slab: it polls all of its chunks from
                    // the start (one round trip less when the block lands); every other waiting task probes a sentinel first
                    if (kk != m - 1) {
                        const int col = lt >> 5, ch = (lt & 31) * 2;
                        const double2* g0 = reinterpret_cast<const double2*>(Yg + (size_t)col * N + ch);
                        for (int spin = 0;; spin++) {
                            const double2 v = __ldcg(g0);
                            if (!((__double_as_longlong(v.x) == TR_ABSENT) | (__double_as_longlong(v.y) == TR_ABSENT))) break;
                            if (spin > 8 * TR_SPIN_LIMIT) {
                                atomicCAS(p.status, SWW_OK, SWW_ECUDA);
                                s_abort = 1;
                                out = true;
                                break;
                            }
                            if ((spin & 255) == 255 && (s_abort || ld_status(p.status) != SWW_OK)) {
                                s_abort = 1;
                                out = true;
                                break;
                            }
                        }
                    }
                    double2 v[NCH];
                    for (int spin = 0; !out; spin++) {
                        bool miss = false;
#pragma unroll
                        for (int q = 0; q < NCH; q++) {
                            const int c = lt + q * NL, col = c >> 5, ch = (c & 31) * 2;
                            v[q] = __ldcg(reinterpret_cast<const double2*>(Yg + (size_t)col * N + ch));
                        }
#pragma unroll
                        for (int q = 0; q < NCH; q++)
                            miss |= (__double_as_longlong(v[q].x) == TR_ABSENT) | (__double_as_longlong(v[q].y) == TR_ABSENT);
                        if (!miss) break;
                        if (spin > TR_SPIN_LIMIT) {
                            atomicCAS(p.status, SWW_OK, SWW_ECUDA);
                            s_abort = 1;
                            break;
                        }
                        if ((spin & 63) == 63 && (s_abort || ld_status(p.status) != SWW_OK)) {
                            s_abort = 1;
                            break;
                        }
                    }
                    if (!out) {
#pragma unroll
                        for (int q = 0; q < NCH; q++) {
                            const int c = lt + q * NL, col = c >> 5, ch = (c & 31) * 2;
                            *reinterpret_cast<double2*>(b + col * LDO + ch) = v[q];
                        }
                    }
                }
                mbar_arrive(&full[buf]);
                if (issued < m) issue_stage();
            }
            if (phase && m == 0) {
                cp_wait<0>();
                mbar_arrive(&fullD);
            }
        } else {
            // ---------------------------------------------------------------------------------- the MMA warps
            double* Bg = p.B + blk;
            double* Lg = p.Blo + blk;
            double acc[C::FM][2], ph[C::FM][2], pl[C::FM][2];
#pragma unroll
            for (int x = 0; x < C::FM; x++)
#pragma unroll
                for (int e = 0; e < 2; e++) acc[x][e] = ph[x][e] = pl[x][e] = 0.0;
            auto mma_tile = [&](const double* a, const double* b) {
                const double* as = a + row0;
                const double* bs = b + (wc * 8 + fr) * LDO;
#pragma unroll
                for (int k4 = 0; k4 < TS; k4 += 4) {
                    const double bf = bs[k4 + fk];
#pragma unroll
                    for (int x = 0; x < C::FM; x++) lu_dmma884(acc[x][0], acc[x][1], as[(k4 + fk) * LDO + x * 8], bf);
                }
            };
            auto fold = [&]() {  // (ph, pl) += acc, error-free; acc = 0
#pragma unroll
                for (int x = 0; x < C::FM; x++)
#pragma unroll
                    for (int e = 0; e < 2; e++) {
                        double s_, e_;
                        two_sum_d(ph[x][e], acc[x][e], s_, e_);
                        ph[x][e] = s_;
                        pl[x][e] += e_;
                        acc[x][e] = 0.0;
                    }
            };
            // the block's own right-hand side: forward B_i (plain fp64), backward the forward result (hi, lo), reloaded until
            // all of it is there (it is final long before, except at the turn of the sweeps); the loaders work meanwhile
            double bh[C::FM][2], bl[C::FM][2];
            for (int spin = 0;; spin++) {
                bool bad = false;
#pragma unroll
                for (int x = 0; x < C::FM; x++)
#pragma unroll
                    for (int e = 0; e < 2; e++) {
                        const size_t o = (size_t)(col0 + e) * N + row0 + x * 8;
                        if (phase) {
                            bh[x][e] = __ldcg(p.Yh + blk + o);
                            bl[x][e] = __ldcg(p.Yl + blk + o);
                            bad |= (__double_as_longlong(bh[x][e]) == TR_ABSENT) | (__double_as_longlong(bl[x][e]) == TR_ABSENT);
                        } else {
                            bh[x][e] = tr_canon(Bg[o]);
                            bl[x][e] = 0.0;  // the forward sweep starts from plain fp64 right-hand sides
                        }
                    }
                if (!phase || !mma_bar_or(bad)) break;
                if (spin > TR_SPIN_LIMIT) {
                    if (tid == 0) atomicCAS(p.status, SWW_OK, SWW_ECUDA);
                    break;
                }
                if ((spin & 63) == 63 && mma_bar_or(tid == 0 && ld_status(p.status) != SWW_OK)) break;
            }
            auto step = [&](int kk) {
                const unsigned g = it + (unsigned)kk;
                const int buf = (int)(g % ST);
                mbar_wait(&full[buf], (g / ST) & 1u);
                mma_tile(sA + buf * TS * LDO, sB + buf * WS * LDO);
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[buf]);
            };
            // forward: all m terms; backward: the terms of the blocks k > i + 1 (the front term comes last, through V_i)
            const int mb = phase ? (m > 0 ? m - 1 : 0) : m;
            for (int kk = 0; kk < mb; kk++) {
                step(kk);
                if ((kk % TR_FOLD) == TR_FOLD - 1) fold();
            }
            fold();
            // z = (bh + bl) - (ph + pl) as sh + sl
            double sh[C::FM][2], sl[C::FM][2];
#pragma unroll
            for (int x = 0; x < C::FM; x++)
#pragma unroll
                for (int e = 0; e < 2; e++) {
                    double s_, e_;
                    two_sum_d(bh[x][e], -ph[x][e], s_, e_);
                    sh[x][e] = s_;
                    sl[x][e] = e_ + (bl[x][e] - pl[x][e]);
                    if (phase) sZ[(col0 + e) * LDO + row0 + x * 8] = s_;  // Bs[n][k] = z[k][n]
                }
            if (phase) {
                // backward: w = Z_i z = 2 z + F_i z (before the front block is there), then x_i = w - V_i x_{i+1}
                asm volatile("bar.sync 1, 256;" ::: "memory");  // z complete (the MMA warps only)
                mbar_wait(&fullD, nd & 1u);
                mma_tile(sD, sZ);
#pragma unroll
                for (int x = 0; x < C::FM; x++)
#pragma unroll
                    for (int e = 0; e < 2; e++) {
                        double t_, e_;
                        two_sum_d(2.0 * sh[x][e], acc[x][e], t_, e_);
                        sh[x][e] = t_;
                        sl[x][e] = fma(2.0, sl[x][e], e_);
                        acc[x][e] = 0.0;
                    }
                if (m > 0) {
                    step(m - 1);
#pragma unroll
                    for (int x = 0; x < C::FM; x++)
#pragma unroll
                        for (int e = 0; e < 2; e++) {
                            double t_, e_;
                            two_sum_d(sh[x][e], -acc[x][e], t_, e_);
                            sh[x][e] = t_;
                            sl[x][e] += e_;
                        }
                }
            }
#pragma unroll
            for (int x = 0; x < C::FM; x++)
#pragma unroll
                for (int e = 0; e < 2; e++) {  // first what the chain waits for: the high words of the whole block
                    const size_t o = (size_t)(col0 + e) * N + row0 + x * 8;
                    const double hi = __dadd_rn(sh[x][e], sl[x][e]);
                    sl[x][e] = __dsub_rn(sl[x][e], __dsub_rn(hi, sh[x][e]));
                    sh[x][e] = hi;
                    (phase ? p.Xh : p.Yh)[blk + o] = tr_canon(hi);
                }
#pragma unroll
            for (int x = 0; x < C::FM; x++)
#pragma unroll
                for (int e = 0; e < 2; e++) {
                    const size_t o = (size_t)(col0 + e) * N + row0 + x * 8;
                    if (phase) {  // x_i: the result (hi, lo)
                        Bg[o] = sh[x][e];
                        Lg[o] = sl[x][e];
                    } else {      // y_i: the low word for this block's backward task
                        p.Yl[blk + o] = tr_canon(sl[x][e]);
                    }
                }
        }
        it += (unsigned)m;
        nd += (unsigned)phase;
    }
}

template <int WS>
static int launch_trsm(sww_dtn_s* d, double* B, double* Blo, int ns) {
    using C = TrsmCfg<WS>;
    const int N = d->N, nt = N / TS;
    TrsmArgs a;
    a.A = d->LU;
    a.Fs = d->invD + (size_t)nt * TS * TS;
    a.Vs = d->invD + 2 * (size_t)nt * TS * TS;
    a.B = B;
    a.Blo = Blo;
    a.N = N;
    a.nt = nt;
    a.ns = ns;
    a.counter = d->tr_flags;
    a.status = d->status;
    const size_t span = (size_t)N * ns * WS;  // doubles per scratch vector
    if (d->tr_scr_cap < 3 * span) {
        SWW_CUDA(cudaStreamSynchronize(d->stream));
        cudaFree(d->tr_scr);
        d->tr_scr = nullptr;
        d->tr_scr_cap = 0;
        if (cudaMalloc(&d->tr_scr, sizeof(double) * 3 * span) != cudaSuccess) return SWW_ENOMEM;
        d->tr_scr_cap = 3 * span;
    }
    a.Yh = d->tr_scr;
    a.Yl = d->tr_scr + span;
    a.Xh = d->tr_scr + 2 * span;
    SWW_CUDA(cudaMemsetAsync(d->tr_scr, 0xFF, sizeof(double) * 3 * span, d->stream));  // every entry "absent"
    SWW_CUDA(cudaMemsetAsync(a.counter, 0, sizeof(unsigned), d->stream));
    const int grid = std::min(sm_count(), 2 * nt * ns);
    SWW_BEGIN(WS == 8 ? KC_TRSV : KC_TRSM, d->stream);  // the 8-column instantiation serves the single-vector solves: chain-latency-bound
    if constexpr (WS >= 16) {  // batches: the warp-specialized kernel
        using W = TrsmWsCfg<WS>;
        static DeviceOnce attr_ws;
        if (attr_ws.first()) SWW_CUDA(cudaFuncSetAttribute(k_trsm_ws<WS>, cudaFuncAttributeMaxDynamicSharedMemorySize, W::SMEM));
        k_trsm_ws<WS><<<grid, W::THREADS, W::SMEM, d->stream>>>(a);
    } else {                   // up to 64 columns (the single-vector solves): pure chain latency, every warp polls and multiplies
        static DeviceOnce attr_once;
        if (attr_once.first()) SWW_CUDA(cudaFuncSetAttribute(k_trsm_dataflow<WS>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM));
        k_trsm_dataflow<WS><<<grid, 256, C::SMEM, d->stream>>>(a);
    }
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

// Solve (LU) X = B for ncols columns, in place; B and Blo are N x (ncols rounded up to the slab width) buffers (the padding
// columns are solved too and ignored).  On return B + Blo is the solution (B = its fp64 rounding).
int run_solve(sww_dtn_s* d, double* B, double* Blo, int ncols) {
    const int N = d->N, nb = (N < NB) ? N : NB, nblk = N / nb;
    cudaStream_t st = d->stream;
    if (nblk == 1) {
        const double* Es = d->invD;
        const double* Fs = d->invD + (size_t)nblk * nb * nb;
        SWW_BEGIN(KC_GEMM, st);
        k_solve_small<<<ncols, 64, 0, st>>>(N, Es, Fs, B, Blo);
        SWW_LAUNCHED();
        SWW_CUDA(cudaGetLastError());
        return SWW_OK;
    }
    // slab width: the chain of a slab is 2 N/64 links of (flag hop + one or two 64 x 64 x WS products), so narrow slabs finish
    // sooner as long as there are few of them; every slab re-reads the factors from L2, so many columns want wide slabs
    // (measured at N = 2048: 128 columns 0.19 ms with 16-column slabs against 0.27 ms with 32; 512 columns 0.36 against 0.34)
    const int ws = ncols <= 64 ? 8 : (ncols <= 256 ? 16 : 32);
    for (int c0 = 0; c0 < ncols; c0 += TR_MAXNS * ws) {
        const int nc = std::min(ncols - c0, TR_MAXNS * ws);
        double *b = B + (size_t)c0 * N, *bl = Blo + (size_t)c0 * N;
        if (ws == 8)
            SWW_TRY(launch_trsm<8>(d, b, bl, (nc + 7) / 8));
        else if (ws == 16)
            SWW_TRY(launch_trsm<16>(d, b, bl, (nc + 15) / 16));
        else
            SWW_TRY(launch_trsm<32>(d, b, bl, (nc + 31) / 32));
    }
    return SWW_OK;
}

}  // namespace sww
