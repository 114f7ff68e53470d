// synax_dd.cu -- host-side dispatch of the all-float64 kernels (synax_dd.cuh): synax_forward_f64 / synax_vjp_f64.
#include <algorithm>

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

}  // namespace synax
