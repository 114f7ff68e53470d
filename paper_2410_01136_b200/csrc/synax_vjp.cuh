// synax_vjp.cuh -- adjoint kernels for the analytic models (A9-A11).
#pragma once
#include "synax_forward.cuh"
#include "../../include/synax.h"

namespace synax {

static synax_status analytic_vjp(int code, const FreqTab& ft, const Geometry& geo, const BatchConsts* bc, int batch,
                                 int n_params, int G, const float* dI, const float* dQ, const float* dU, float* grad,
                                 cudaStream_t st, int64_t* launches) {
  return SYNAX_ERR_UNSUPPORTED;
}

}  // namespace synax
