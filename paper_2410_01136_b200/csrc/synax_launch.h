// synax_launch.h -- host-side launchers of the template kernels.  Each model code is instantiated in its own
// translation unit (synax_fwd_<code>.cu, synax_vjp_<code>.cu) so that the library builds in parallel; synax_api.cu and
// synax_vjp_driver.cu see only these declarations.
#pragma once
#include "../../include/synax.h"
#include "synax_forward.cuh"
#include "synax_vjp.cuh"

namespace synax {

// ---- forward (synax_fwd_impl.cuh, explicitly instantiated per CODE)
template <int CODE> void fwd_launch_pilot(unsigned blocks, cudaStream_t st, const ForwardArgs& a, int64_t stride, int64_t n_pilot, int* ctrl);
template <int CODE> void fwd_launch_classify(unsigned blocks, cudaStream_t st, const ForwardArgs& a, int* ctrl);
template <int CODE> void fwd_launch_fast(bool list, int G, int nf, int64_t n_sl, cudaStream_t st, const ForwardArgs& a, const FreqTab& ft);
// batched fp32 forward (forward_batched_kernel; DISC4 and FULL16, one frequency, one thread per sightline), nb = 2 or 4
template <int CODE> void fwd_launch_batched(int nb, cudaStream_t st, const ForwardArgs& a, const FreqTab& ft);
template <int CODE> void fwd_launch_f64(int G, int nf, unsigned blocks, cudaStream_t st, const ForwardArgs& a, const FreqTab& ft);

// ---- adjoint (synax_vjp_impl.cuh, explicitly instantiated per CODE)
template <int CODE> void vjp_launch(int pmode, int G, int nf, dim3 grid, cudaStream_t st, const VjpArgs& a, const FreqTab& ft);
// forward-order lean adjoint (vjp_batched_kernel; DISC4 and FULL16, one frequency), nb = 1, 2 or 4 parameter vectors per
// thread, grid = (n_blocks, ceil(batch / nb))
template <int CODE> void vjp_launch_batched(int nb, dim3 grid, cudaStream_t st, const VjpArgs& a, const FreqTab& ft);
template <int CODE> void vjp_launch_classify(int G, dim3 grid, cudaStream_t st, const VjpArgs& a, unsigned char* cta_sel);

// dispatch on the run-time model code (kAnalyticDisc, kAnalyticFull, kStack16, kUniform)
#define SYNAX_DISPATCH_CODE(code, FN, ...)                                   \
  do {                                                                       \
    if ((code) == kAnalyticDisc) FN<kAnalyticDisc>(__VA_ARGS__);             \
    else if ((code) == kStack16) FN<kStack16>(__VA_ARGS__);                  \
    else if ((code) == kAnalyticFull) FN<kAnalyticFull>(__VA_ARGS__);        \
    else FN<kUniform>(__VA_ARGS__);                                          \
  } while (0)

// ---- plan-owned workspace (synax_api.cu)
// Per-call scratch (constants, lists, block partials, the gridded path's repacked grid and accumulation buffer ...) is cut
// from one buffer that stays with the plan, in stack order, instead of coming from the device's stream-ordered memory pool:
// with CUDA's default release threshold (0) the pool gives everything back at every stream synchronisation, and the first
// allocation after one waits ~0.23 ms for memory to be mapped again -- more than a whole cfg-1 forward.  The buffer grows
// (cudaFree + cudaMalloc: synchronises the device, like the plan's other buffers) at the start of a call when an earlier
// call needed more, up to kWorkspaceMax; what does not fit, and everything inside a stream capture (a captured graph must
// not hold pointers into a buffer that may be reallocated later), comes from the pool as before.  A plan is not used by two
// calls at a time (synax.h), and calls that follow each other are ordered by their streams, so a later call may reuse the
// bytes of an earlier one.
struct Workspace {
  char* base; size_t cap;     // zero-initialised with the plan
  size_t used;                // stack pointer of the call in progress (virtual: counts what went to the pool too)
  size_t want;                // high-water mark
  int depth;                  // nesting of WorkspaceScope
};
constexpr size_t kWorkspaceMax = (size_t)256 << 20;
void* ws_alloc(Workspace* ws, size_t bytes, cudaStream_t st, bool* pooled);   // nullptr when nothing is to be had
inline void ws_release(void* p, bool pooled, cudaStream_t st) { if (p && pooled) cudaFreeAsync(p, st); }
void ws_enter(Workspace* ws, cudaStream_t st, size_t* mark);                  // grows the buffer at the outermost level
inline void ws_leave(Workspace* ws, size_t mark) { if (ws) { ws->used = mark; --ws->depth; } }

// ---- synax_vjp_driver.cu
synax_status analytic_vjp(int code, const FreqTab& ft, const Geometry& geo, const BatchConsts* bc,
                          const BatchConstsD* bd, int batch, int n_params, int G, const ScalarGridDesc& sg_ne,
                          const ScalarGridDesc& sg_n0, int precision, double escalate_rad, int batch_share, const double* phi, const int* phi_ok,
                          const double* phi_base, const unsigned char* phi_has, int* ctrl,
                          cudaStream_t aux, cudaEvent_t ev_fork, cudaEvent_t ev_join,
                          const float* dI, const float* dQ, const float* dU, float* grad, Workspace* ws, cudaStream_t st,
                          int64_t* launches);

// ---- synax_grid.cu
synax_status grid_forward(const FreqTab& ft, const ForwardArgs& a0, const synax_model* m, const float* grid,
                          int precision, double escalate_rad, int sms, int* d_flag_count, int* h_flag_count,
                          Workspace* ws, cudaStream_t st, int64_t* launches);
synax_status grid_vjp(const FreqTab& ft, const Geometry& geo, const BatchConsts* bc, const BatchConstsD* bd,
                      const synax_model* m, const ScalarGridDesc& sg_ne, const ScalarGridDesc& sg_n0,
                      const float* grid, const float* dI, const float* dQ, const float* dU, float* grad,
                      int precision, double escalate_rad, int sms, Workspace* ws, cudaStream_t st, int64_t* launches);

// ---- synax_dd.cu: the all-float64 path (synax_forward_f64 / synax_vjp_f64)
size_t dd_consts_bytes(int batch);
int dd_vjp_blocks(int64_t npix, int G);
synax_status dd_forward(int code, const FreqTab& ft, const Geometry& geo, const double* params, int n_params, int batch,
                        const AuxHost& aux, const ScalarGridDesc& sg_ne, const ScalarGridDesc& sg_n0, int G, void* bc64,
                        double* I, double* Q, double* U, cudaStream_t st, int64_t* launches);
synax_status dd_vjp(int code, const FreqTab& ft, const Geometry& geo, const double* params, int n_params, int batch,
                    const AuxHost& aux, const ScalarGridDesc& sg_ne, const ScalarGridDesc& sg_n0, int G, void* bc64,
                    double* partial, const double* dI, const double* dQ, const double* dU, double* grad, cudaStream_t st,
                    int64_t* launches);
// the adjoint on the library's static scratch array (synax_vjp_f64_noalloc): capacity, bytes a call needs, the call
size_t dd_noalloc_capacity();
size_t dd_noalloc_bytes(int64_t npix, int G, int batch);
synax_status dd_vjp_noalloc(int device, int code, const FreqTab& ft, const Geometry& geo, const double* params, int n_params,
                            int batch, const AuxHost& aux, const ScalarGridDesc& sg_ne, const ScalarGridDesc& sg_n0, int G,
                            const double* dI, const double* dQ, const double* dU, double* grad, cudaStream_t st,
                            int64_t* launches, cudaError_t* cuda_error);

}  // namespace synax
