// adjoint kernels of one model code (see synax_launch.h)
#include "synax_vjp_impl.cuh"
namespace synax {
SYNAX_INSTANTIATE_VJP(kAnalyticFull)
}
