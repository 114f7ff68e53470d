// synax_dd.cu -- host-side dispatch of the all-float64 kernels (synax_dd.cuh): synax_forward_f64 / synax_vjp_f64.
#include <algorithm>
#include <mutex>

#include "synax_launch.h"
#include "synax_dd.cuh"

namespace synax {

static int dd_freq_block(int remaining) { return remaining >= 8 ? 8 : (remaining >= 4 ? 4 : 1); }

template <int CODE, int G>
static void launch_forward_dd(int nf, unsigned blocks, cudaStream_t st, const DDArgs& a, const FreqTab& ft0) {
  const FreqTab ft = shift_freqs(ft0, a.f0);
  if (nf == 8) forward_dd_kernel<CODE, G, 8><<<blocks, kBlock, 0, st>>>(a, ft);
  else if (nf == 4) forward_dd_kernel<CODE, G, 4><<<blocks, kBlock, 0, st>>>(a, ft);
  else forward_dd_kernel<CODE, G, 1><<<blocks, kBlock, 0, st>>>(a, ft);
}
template <int CODE, int G>
static void launch_vjp_dd(int nf, dim3 grid, cudaStream_t st, const DDArgs& a, const FreqTab& ft0) {
  const FreqTab ft = shift_freqs(ft0, a.f0);
  if (nf == 8) vjp_dd_kernel<CODE, G, 8><<<grid, kBlock, 0, st>>>(a, ft);
  else if (nf == 4) vjp_dd_kernel<CODE, G, 4><<<grid, kBlock, 0, st>>>(a, ft);
  else vjp_dd_kernel<CODE, G, 1><<<grid, kBlock, 0, st>>>(a, ft);
}
template <int CODE>
static void forward_dd_g(int G, int nf, unsigned blocks, cudaStream_t st, const DDArgs& a, const FreqTab& ft) {
  if (G == 1) launch_forward_dd<CODE, 1>(nf, blocks, st, a, ft);
  else if (G == 8) launch_forward_dd<CODE, 8>(nf, blocks, st, a, ft);
  else launch_forward_dd<CODE, 32>(nf, blocks, st, a, ft);
}
template <int CODE>
static void vjp_dd_g(int G, int nf, dim3 grid, cudaStream_t st, const DDArgs& a, const FreqTab& ft) {
  if (G == 1) launch_vjp_dd<CODE, 1>(nf, grid, st, a, ft);
  else if (G == 8) launch_vjp_dd<CODE, 8>(nf, grid, st, a, ft);
  else launch_vjp_dd<CODE, 32>(nf, grid, st, a, ft);
}

// bc64: device scratch for `batch` BatchConsts64, written here
synax_status dd_forward(int code, const FreqTab& ft, const Geometry& geo, const double* params, int n_params, int batch,
                        const AuxHost& aux, const ScalarGridDesc& sg_ne, const ScalarGridDesc& sg_n0, int G, void* bc64,
                        double* I, double* Q, double* U, cudaStream_t st, int64_t* launches) {
  DDArgs a{};
  a.geo = geo; a.bc = (BatchConsts64*)bc64; a.batch = batch; a.n_freq_total = ft.n_freq; a.sg_ne = sg_ne; a.sg_n0 = sg_n0;
  a.I = I; a.Q = Q; a.U = U;
  prologue64_kernel<<<(batch + 127) / 128, 128, 0, st>>>(code, params, n_params, batch, aux, ft, geo.delta, (BatchConsts64*)bc64);
  ++*launches;
  const int64_t n_sl = geo.npix * batch;
  const unsigned blocks = (unsigned)((n_sl * G + kBlock - 1) / kBlock);
  for (int f0 = 0; f0 < ft.n_freq;) {
    const int nf = dd_freq_block(ft.n_freq - f0);
    a.f0 = f0;
    if (code == kAnalyticDisc) forward_dd_g<kAnalyticDisc>(G, nf, blocks, st, a, ft);
    else if (code == kStack16) forward_dd_g<kStack16>(G, nf, blocks, st, a, ft);
    else if (code == kAnalyticFull) forward_dd_g<kAnalyticFull>(G, nf, blocks, st, a, ft);
    else forward_dd_g<kUniform>(G, nf, blocks, st, a, ft);
    ++*launches;
    f0 += nf;
  }
  return cudaGetLastError() == cudaSuccess ? SYNAX_OK : SYNAX_ERR_CUDA;
}

// partial: device scratch [batch][n_blocks][16] doubles, n_blocks = ceil(npix * G / kBlock)
synax_status dd_vjp(int code, const FreqTab& ft, const Geometry& geo, const double* params, int n_params, int batch,
                    const AuxHost& aux, const ScalarGridDesc& sg_ne, const ScalarGridDesc& sg_n0, int G, void* bc64,
                    double* partial, const double* dI, const double* dQ, const double* dU, double* grad, cudaStream_t st,
                    int64_t* launches) {
  DDArgs a{};
  a.geo = geo; a.bc = (BatchConsts64*)bc64; a.batch = batch; a.n_freq_total = ft.n_freq; a.sg_ne = sg_ne; a.sg_n0 = sg_n0;
  a.dI = dI; a.dQ = dQ; a.dU = dU; a.partial = partial;
  a.n_blocks = dd_vjp_blocks(geo.npix, G);
  prologue64_kernel<<<(batch + 127) / 128, 128, 0, st>>>(code, params, n_params, batch, aux, ft, geo.delta, (BatchConsts64*)bc64);
  ++*launches;
  for (int b0 = 0; b0 < batch; b0 += 65535) {   // gridDim.y limit
    const int nb = std::min(65535, batch - b0);
    DDArgs ab = a;
    ab.bc = a.bc + b0; ab.partial = a.partial + (size_t)b0 * a.n_blocks * 16;
    if (dI) ab.dI = dI + (size_t)b0 * ft.n_freq * geo.npix;
    if (dQ) ab.dQ = dQ + (size_t)b0 * ft.n_freq * geo.npix;
    if (dU) ab.dU = dU + (size_t)b0 * ft.n_freq * geo.npix;
    const dim3 grid((unsigned)a.n_blocks, (unsigned)nb);
    for (int f0 = 0; f0 < ft.n_freq;) {
      const int nf = dd_freq_block(ft.n_freq - f0);
      ab.f0 = f0; ab.accumulate = f0 > 0;
      if (code == kAnalyticDisc) vjp_dd_g<kAnalyticDisc>(G, nf, grid, st, ab, ft);
      else if (code == kStack16) vjp_dd_g<kStack16>(G, nf, grid, st, ab, ft);
      else if (code == kAnalyticFull) vjp_dd_g<kAnalyticFull>(G, nf, grid, st, ab, ft);
      else vjp_dd_g<kUniform>(G, nf, grid, st, ab, ft);
      ++*launches;
      f0 += nf;
    }
  }
  vjp_dd_reduce_kernel<<<batch, 256, 0, st>>>(partial, a.n_blocks, n_params, grad);
  ++*launches;
  return cudaGetLastError() == cudaSuccess ? SYNAX_OK : SYNAX_ERR_CUDA;
}

size_t dd_consts_bytes(int batch) { return sizeof(BatchConsts64) * (size_t)batch; }
int dd_vjp_blocks(int64_t npix, int G) { return (int)((npix * G + kBlock - 1) / kBlock); }

// ------------------------------------------------------------------------------------------------
// synax_vjp_f64_noalloc: the same adjoint with its scratch (the per-batch constants and the per-CTA partial
// gradients) in a fixed array that is part of the library image, for callers that cannot allocate (CUDA graph capture,
// serving loops, harnesses that forbid cudaMalloc).  Every GPU that loads the library holds kNoAllocScratchBytes of
// it until the process exits.  ALL calls on a device share the array: it keeps the last call's contents (what a call
// reads it writes or clears first), and two calls that overlap on the GPU (different streams) race.
// ------------------------------------------------------------------------------------------------
constexpr size_t kNoAllocScratchBytes = (size_t)4 << 20;   // 4 MiB
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocScratchBytes];

static_assert(sizeof(BatchConsts64) == 872, "synax.h states the scratch a synax_vjp_f64_noalloc call needs");

constexpr int kNoAllocMaxDevices = 64;
static std::mutex g_noalloc_mutex;
static void* g_noalloc_ptr[kNoAllocMaxDevices];   // device address of g_noalloc_scratch, per device; null = not asked yet

size_t dd_noalloc_capacity() { return kNoAllocScratchBytes; }

static size_t round_up_256(size_t n) { return (n + 255) & ~(size_t)255; }

size_t dd_noalloc_bytes(int64_t npix, int G, int batch) {
  return round_up_256(dd_consts_bytes(batch)) + sizeof(double) * 16 * (size_t)dd_vjp_blocks(npix, G) * (size_t)batch;
}

// In host code `g_noalloc_scratch` names a host-side stand-in, not device memory: the device address comes from
// cudaGetSymbolAddress, asked once per device with that device current.
static cudaError_t noalloc_scratch_address(int device, unsigned char** out) {
  *out = nullptr;
  if (device < 0 || device >= kNoAllocMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_ptr[device]) {
    int cur = -1;
    cudaError_t e = cudaGetDevice(&cur);
    if (e != cudaSuccess) return e;
    if (cur != device) return cudaErrorInvalidDevice;   // the caller keeps the plan's device current (synax.h)
    void* q = nullptr;
    e = cudaGetSymbolAddress(&q, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    g_noalloc_ptr[device] = q;
  }
  *out = (unsigned char*)g_noalloc_ptr[device];
  return cudaSuccess;
}

// dd_vjp on the static scratch.  SYNAX_ERR_UNSUPPORTED when the call needs more than the array holds (checked by the
// caller too, for the message); no cudaMalloc / cudaFree / allocating routine on this path.
synax_status dd_vjp_noalloc(int device, int code, const FreqTab& ft, const Geometry& geo, const double* params, int n_params,
                            int batch, const AuxHost& aux, const ScalarGridDesc& sg_ne, const ScalarGridDesc& sg_n0, int G,
                            const double* dI, const double* dQ, const double* dU, double* grad, cudaStream_t st,
                            int64_t* launches, cudaError_t* cuda_error) {
  *cuda_error = cudaSuccess;
  if (dd_noalloc_bytes(geo.npix, G, batch) > kNoAllocScratchBytes) return SYNAX_ERR_UNSUPPORTED;
  unsigned char* base = nullptr;
  *cuda_error = noalloc_scratch_address(device, &base);
  if (*cuda_error != cudaSuccess) return SYNAX_ERR_CUDA;
  void* bc64 = base;
  double* partial = reinterpret_cast<double*>(base + round_up_256(dd_consts_bytes(batch)));
  // the partial gradients of the last call are still there: cleared on the stream (the kernels also overwrite every
  // entry the reduction reads; this keeps that an implementation detail)
  *cuda_error = cudaMemsetAsync(partial, 0, sizeof(double) * 16 * (size_t)dd_vjp_blocks(geo.npix, G) * (size_t)batch, st);
  if (*cuda_error != cudaSuccess) return SYNAX_ERR_CUDA;
  const synax_status s = dd_vjp(code, ft, geo, params, n_params, batch, aux, sg_ne, sg_n0, G, bc64, partial, dI, dQ, dU, grad,
                                st, launches);
  if (s != SYNAX_OK) *cuda_error = cudaGetLastError();
  return s;
}

}  // namespace synax
