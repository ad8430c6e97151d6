// rk.cuh -- the time-stepper state shared by rk.cu (S8, S9) and shoot.cu (the shooting map).  Product code; shares nothing with oracle/.
#pragma once
#include "common.cuh"

constexpr int RK_S = 11;

struct sww_state_s {
    int N, nc, prec;
    double h, g;
    double sigma;        // surface tension sigma / rho of (2.1b) (0: none)
    bool filter;
    cudaStream_t stream;
    sww_dtn_t dtn;
    size_t L;            // 2 N (1 + nc)
    double* y;           // state
    double* ys;          // stage state
    double* k;           // RK_S stage derivatives, L each
    double* w;           // N x nc: unfiltered deta_t of the current stage
    double* red;         // 2 doubles: energy reduction (hi, lo)
    double* sdc;         // SDC15 work space (SDC_SLOTS state vectors), allocated by the first sww_sdc_advance
    double t;
    // sww_shoot_gradient (grad.cu): when set, sww_rk_advance records the stage states (eta, phi) of every step here, stage i of step n at
    // (n RK_S + i) 2N (fp64 steppers); tape_steps = the steps that fit
    double* tape;
    int tape_steps;
    // sww_state_respace into this state (mesh.cu): the interpolation matrix of the last pair of meshes, kept for the next call
    double* rsp_R;
    int rsp_Mo, rsp_where_o, rsp_where_n;
    double rsp_rho_o, rsp_rho_n;
    double a[RK_S][RK_S], b[RK_S], c[RK_S];
    double alo[RK_S][RK_S], blo[RK_S];  // low words of the tableau (double-double states)
    size_t mul() const { return prec == SWW_DD ? 2 : 1; }
};

namespace sww {
// one evaluation of the right-hand sides (2.1), (B.1)-(B.3) at the stage state ys -> kout (same layout as the state)   (rk.cu)
int rk_rhs(sww_state_s* s, const double* ys, double* kout);
// Radau IIa nodes c, their spacings dc and the integration matrix S (s x s row-major) as double-double pairs   (sdc_tables.cpp, host)
int sdc_tables_host(int s, double* c_hi, double* c_lo, double* dc_hi, double* dc_lo, double* S_hi, double* S_lo);
}  // namespace sww
