// ddpath.cu -- double-double DtN apply (placeholder until the dd kernels land; returns SWW_EINVAL)
#include "common.cuh"
namespace sww {
int dd_apply(sww_dtn_s*, const double*, bool, const double*, int, double*) { return SWW_EINVAL; }
int dd_set_base(sww_dtn_s*, const double*) { return SWW_EINVAL; }
int dd_linearized(sww_dtn_s*, const double*, const double*, int, double*) { return SWW_EINVAL; }
}
