// synax_grid.cuh -- gridded-B forward (A3') and adjoint with scatter-add (A11').
#pragma once
#include "synax_forward.cuh"
#include "../../include/synax.h"

namespace synax {

static synax_status grid_forward(const FreqTab& ft, const ForwardArgs& a, const synax_model* m, const float* grid,
                                 int precision, double escalate_rad, cudaStream_t st, int64_t* launches) {
  return SYNAX_ERR_UNSUPPORTED;
}
static synax_status grid_vjp(const FreqTab& ft, const Geometry& geo, const BatchConsts* bc, const synax_model* m,
                             const float* grid, const float* dI, const float* dQ, const float* dU, float* grad,
                             cudaStream_t st, int64_t* launches) {
  return SYNAX_ERR_UNSUPPORTED;
}

}  // namespace synax
