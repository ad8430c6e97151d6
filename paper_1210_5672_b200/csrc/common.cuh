// common.cuh -- shared declarations of the sww CUDA library (product code; shares nothing with oracle/).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <cmath>
#include <cstdlib>
#include "../../include/sww.h"

namespace sww {

// ---------------------------------------------------------------- launch accounting / error capture
extern unsigned long long g_launches;
extern char g_cuda_err[256];
int note_cuda(cudaError_t e, const char* where);
#define SWW_CUDA(call)                                                        \
    do {                                                                      \
        cudaError_t e_ = (call);                                              \
        if (e_ != cudaSuccess) return ::sww::note_cuda(e_, #call);            \
    } while (0)
#define SWW_TRY(call)                                                         \
    do {                                                                      \
        int rc_ = (call);                                                     \
        if (rc_ != SWW_OK) return rc_;                                        \
    } while (0)
// Per-kernel-class device timing (sww_timing_enable / sww_timing_read): when enabled, SWW_BEGIN / SWW_LAUNCHED bracket every
// launch with a CUDA event pair on the launching stream; off by default (no events, no overhead beyond a branch).
enum KClass { KC_ASM = 0, KC_LU = 1, KC_GEMM = 2, KC_FFT = 3, KC_DDGEMM = 4, KC_OTHER = 5, KC_TRSM = 6, KC_TRSV = 7, KC_COUNT = 8 };
extern bool g_timing;
void timing_begin(int cls, cudaStream_t st);
void timing_end();
#define SWW_BEGIN(cls, st)                                   \
    do {                                                     \
        if (::sww::g_timing) ::sww::timing_begin(cls, st);   \
    } while (0)
#define SWW_LAUNCHED()                                       \
    do {                                                     \
        ++::sww::g_launches;                                 \
        if (::sww::g_timing) ::sww::timing_end();            \
    } while (0)

// ---------------------------------------------------------------- per-device state
// first() is true exactly once per device for each instance: guards the per-device opt-ins (cudaFuncSetAttribute for more than
// 48 KB of dynamic shared memory) at their call sites.  Not thread-safe (like the rest of the library's host side).
struct DeviceOnce {
    unsigned long long seen[4] = {0, 0, 0, 0};
    bool first() {
        int dev = 0;
        cudaGetDevice(&dev);
        dev &= 255;
        const unsigned long long bit = 1ull << (dev & 63);
        if (seen[dev >> 6] & bit) return false;
        seen[dev >> 6] |= bit;
        return true;
    }
};
int sm_count();  // multiprocessors of the current device (cached per device)

// ---------------------------------------------------------------- per-N constant tables (device, cached per N per device)
// "computed once and for all".  All double-double, planar (hi[N], lo[N]).
struct Tables {
    int N;
    double* cs;    // cos(2 pi m / N), m = 0..N-1        (hi at [m], lo at [N+m])
    double* sn;    // sin(2 pi m / N)
    double* c0;    // (1/2) cot(pi m / N), m >= 1; c0[0] = 0
    double* s2;    // sin^2(pi m / N)
    double* dc;    // differentiation circulant: (1/2) (-1)^m cot(pi m / N), m >= 1; dc[0] = 0, dc[N/2] = 0
    double* dc2;   // the circulant of D(D .): symbol -k^2, Nyquist 0; the entry of m = N/2 stored halved (tables.cu)
    double2* tw;   // fp64 FFT twiddles exp(-2 pi i m / N) = (cs, -sn) rounded, m = 0..N-1
    double* filt;  // 36th-order filter exp(-36 (|k|/(N/2))^36) of (2.14) at DFT index m (|k| = min(m, N - m))
    double* filt_dd;  // the same in double-double (planar 2N)
};
int get_tables(int N, cudaStream_t st, const Tables** out);

// ---------------------------------------------------------------- mesh refinement (2.10), PAPER.md:122-136 (mesh.cu)
// per-node tables of the change of variables x = xi(alpha), each double-double planar 2N; all nullptr on the uniform mesh
struct MeshDev {
    const double* xE;   // xi'(alpha_j) = E of (2.10)
    const double* xE1;  // xi''(alpha_j)
    const double* xS;   // sin(xi(alpha_j) - alpha_j)
    const double* xC;   // cos(xi(alpha_j) - alpha_j)
    const double* coef; // 4 doubles: a1 (hi, lo), a2 (hi, lo) of E = 1 + a1 cos(alpha) + a2 cos(2 alpha)
};

// ---------------------------------------------------------------- the DtN handle
struct Workspace {
    int cap_cols = 0;          // padded column capacity
    double* B = nullptr;       // right-hand sides / mu           (f64: N*cap ; dd: 2*N*cap planar)
    double* Gam = nullptr;     // gamma = D mu
    double* W = nullptr;       // result accumulator
    double* T = nullptr;       // scratch columns (u*deta etc.)
    double* R = nullptr;       // dd: fp64 residual / correction
    double* S = nullptr;       // low words of the compensated triangular solves (N*cap)
};

}  // namespace sww

struct sww_dtn_s {
    int N, prec;
    double h;
    bool finite;
    cudaStream_t stream;
    const sww::Tables* tab;
    // node vectors, each dd planar 2N (lo = 0-filled / unused in the f64 path)
    double *eta, *d1, *d2;
    // f64 node tables: E = exp(-(h+eta)), Dm = 1 - E;   dd node tables: sinh(eta), cosh(eta), E, Dm (planar 2N each)
    double *E, *Dm, *Sh, *Ch;
    double *K, *G;        // column-major N x N (dd: planar 2*N*N)
    double *LU;           // fp64 LU factors of I/2 + K (unit lower L below the diagonal, U on and above), column-major
    double *invD;         // inverses of the diagonal blocks of L and U: 2 * (N/NB) blocks of NB x NB
    int* lu_order;        // dataflow LU (lu.cu): task order, tile flags (+ the claim counter in slot 0), epoch of the last run
    unsigned* lu_flags;
    unsigned lu_epoch;
    int lu_ntasks;
    unsigned* tr_flags;   // dataflow TRSM: the claim counter
    double* tr_scr;       // dataflow TRSM: forward (hi, lo) and backward (hi) results, the hand-over buffers between tasks
    size_t tr_scr_cap;    // doubles
    // base state (dd planar 2N each): phi0', W0, u, v
    double *bphi, *bW0, *bu, *bv;
    double *bp_part;      // partial sums of the dd base-state pass: bp_chunks x 4 x N doubles
    int bp_chunks;
    unsigned* mv_count;   // k_matvec_dd: arrival counters per 32-row block (zero between launches)
    double *tmp;          // 14 N doubles: dd scratch vectors of the accurate base state (ddpath.cu)
    bool has_base;
    // mesh refinement (sww_dtn_set_mesh): E = 1 + a1 cos(alpha) + a2 cos(2 alpha); mesh_buf holds the four tables of `mesh`
    bool mesh_on;
    double mesh_rho, mesh_a1, mesh_a2;
    int mesh_where;
    double* mesh_buf;
    sww::MeshDev mesh;
    int* status;          // device sticky status
    sww::Workspace ws;
};

namespace sww {

// block size of the LU / triangular-solve blocking (diag blocks are inverted explicitly)
constexpr int NB = 64;

int ensure_workspace(sww_dtn_s* d, int nrhs);

// node prep + assembly (assembly.cu)
int run_setup_f64(sww_dtn_s* d);
int run_setup_dd(sww_dtn_s* d);
// LU (lu.cu)
int lu_alloc(sww_dtn_s* d);
int run_lu(sww_dtn_s* d);
// multi-RHS triangular solves with the factors in d->LU; B is N x ncols (ld = N), in place; Blo (same shape) receives the
// low word of the compensated solution (B already holds RN(B + Blo)); Blo's incoming content is ignored
int run_solve(sww_dtn_s* d, double* B, double* Blo, int ncols);
// GEMM (gemm.cu): C[M x Nc] = alpha * A[M x K] * B[K x Nc] + beta * C, all column-major fp64; C must not alias A or B.
// n_valid: columns >= n_valid are not stored.
int gemm_f64(cudaStream_t st, int M, int Nc, int K, double alpha, const double* A, int lda, const double* B, int ldb,
             double beta, double* C, int ldc, int n_valid);
// C[M x nc] += A B for nc <= 4 columns as a streamed GEMV (gemm.cu); part / count: the handle's bp_part / mv_count
int gemv_few_f64(cudaStream_t st, int M, int nc, int K, const double* A, int lda, const double* B, int ldb, double* C, int ldc, double* part,
                 unsigned* count);
// accurate base state (ddpath.cu): phi0', W0, u, v of (2.9) with mu0 refined to dd; phi0 is dd planar iff prec == SWW_DD
int accurate_base(sww_dtn_s* d, const double* phi0, size_t phi_plane = 0);
// double-double apply / linearized apply (ddpath.cu); Lin, Lout: plane sizes of the dd planar inputs / output (0 = N * nrhs)
int dd_apply(sww_dtn_s* d, const double* rhs_dev, bool rhs_in_ws, const double* Tcols, int nrhs, double* out, size_t Lin = 0, size_t Lout = 0);
int dd_linearized(sww_dtn_s* d, const double* deta, const double* dphi, int nrhs, double* out, size_t Lin = 0, size_t Lout = 0);
// S0-S2 for a new surface (api.cu); eta_lo: low words of a double-double surface held apart from the high words (nullptr: at eta + N)
int setup_surface(sww_dtn_s* d, const double* eta, const double* eta_lo);
// the plain fp64 base state (fp64 handles only; see ddpath.cu for when the stepper may use it)
int fast_base_f64(sww_dtn_s* d, const double* phi0);
// fused dd pass (assembly.cu): res = b - mu/2 - K mu, w = G gam with the kernel entries evaluated in dd on the fly; all dd planar 2N
int base_pass_dd(sww_dtn_s* d, const double* b, const double* mu, const double* gam, double* res, double* res_f64, double* w);
// refined mesh (mesh.cu): out_c <- out_c / xi' for nrhs columns (no-op on the uniform mesh); L: dd plane size (0 = N * nrhs)
int mesh_scale_out(sww_dtn_s* d, double* out, int nrhs, size_t L);
// spectral (fft.cu)
enum SpecMode { SPEC_APPLY = 0, SPEC_LIN = 1 };
// For each column c < ncols: Gam_c = D M_c ;  W_c = |D| M_c / 2  - (T ? D T_c : 0)
// Mp (optional, ncols = 2): the source of column 1 (see fft.cu)
int spectral_gamma_w(sww_dtn_s* d, const double* M, const double* T, double* Gam, double* W, int ncols, int w_cols, const double* Mp = nullptr);
// out_c = D in_c
int spectral_deriv(sww_dtn_s* d, const double* in, double* out, int ncols);

}  // namespace sww
