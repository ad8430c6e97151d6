// rk.cu -- time stepper (placeholder until the RK kernels land; returns SWW_EINVAL)
#include "common.cuh"
extern "C" {
int sww_state_create(int, double, double, int, int, const void*, const void*, const void*, const void*, unsigned, void*, sww_state_t*) { return SWW_EINVAL; }
int sww_rk_advance(sww_state_t, double, int) { return SWW_EINVAL; }
int sww_state_read(sww_state_t, void*, void*, void*, void*, double*) { return SWW_EINVAL; }
int sww_state_energy(sww_state_t, double*) { return SWW_EINVAL; }
int sww_state_destroy(sww_state_t) { return SWW_EINVAL; }
}
