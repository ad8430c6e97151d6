// rk_dd.cuh -- host-side interface of the double-double stepper kernels (rk_dd.cu), used by rk.cu.
// Product code; shares nothing with oracle/.
#pragma once
#include "common.cuh"

namespace sww {

constexpr int RKDD_MAX_N = 2048;  // k_rhs_cols_dd keeps two N-point complex double-double arrays in shared memory (64 B x N)

// S9 in double-double: indices and coefficients dt a_ij (or dt b_j) of the non-zero terms of one stage combination
struct CombDD {
    int n;
    int idx[11];
    double chi[11], clo[11];
};

// all pointers DEVICE; state vectors planar with plane size L = 2 N (1 + nc): [eta | phi | deta | dphi] in each plane
int rkdd_set_attrs();
int rkdd_combine(cudaStream_t st, size_t L, const double* y, const double* k, const CombDD& cb, double* out);
// eta_t, phi_t of (2.1) at the stage state ys from the base state held by d (set_base done) -> kout
int rkdd_rhs_base(sww_dtn_s* d, bool filter, double g, double sigma, size_t L, const double* ys, double* kout);  // sigma: used on a refined mesh only
// deta_t, dphi_t of (B.1)-(B.3) for nc columns; wout: the linearized DtN of the columns, dd planar with plane size N nc
int rkdd_rhs_cols(sww_dtn_s* d, bool filter, double g, double sigma, int nc, size_t L, const double* ys, const double* wout, double* kout);
// surface tension (2.1b), (B.4): the curvature term and its variation added to phi_t / dphi_t in kout (sigma != 0 only)
int rkdd_st_base(sww_dtn_s* d, bool filter, double sigma, size_t L, double* kout);
int rkdd_st_cols(sww_dtn_s* d, bool filter, double sigma, int nc, size_t L, const double* ys, double* kout);
int rkdd_filter_state(sww_dtn_s* d, int ncol, size_t L, double* y);
// E of PAPER.md:501 for the state y -> out2 (DEVICE, hi and lo); the handle's base state must belong to y
int rkdd_energy(sww_dtn_s* d, double g, size_t L, const double* y, double* out2);

}  // namespace sww
