// forward kernels of one model code (see synax_launch.h)
#include "synax_fwd_impl.cuh"
namespace synax {
SYNAX_INSTANTIATE_FWD(kUniform)
}
