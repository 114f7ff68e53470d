// synax_fwd_impl.cuh -- definitions of the forward launchers of synax_launch.h for one model code; included by the
// synax_fwd_<code>.cu translation units, which instantiate them explicitly.
#pragma once
#include "synax_launch.h"

namespace synax {

template <int CODE>
void fwd_launch_pilot(unsigned blocks, cudaStream_t st, const ForwardArgs& a, int64_t stride, int64_t n_pilot, int* ctrl) {
  pilot_kernel<CODE><<<blocks, kBlock, 0, st>>>(a, stride, n_pilot, ctrl);
}
template <int CODE>
void fwd_launch_classify(unsigned blocks, cudaStream_t st, const ForwardArgs& a, int* ctrl) {
  classify_kernel<CODE><<<blocks, kBlock, 0, st>>>(a, ctrl);
}

template <int CODE, int G, bool LIST>
static void launch_forward_nf(int nf, unsigned blocks, cudaStream_t st, const ForwardArgs& a, const FreqTab& ft0) {
  const FreqTab ft = shift_freqs(ft0, a.f0);
  switch (nf) {
    case 0: forward_kernel<CODE, G, 0, LIST><<<blocks, kBlock, 0, st>>>(a, ft); break;   // Faraday-only pass (synax_vjp)
    case 1: forward_kernel<CODE, G, 1, LIST><<<blocks, kBlock, 0, st>>>(a, ft); break;
    case 2: forward_kernel<CODE, G, 2, LIST><<<blocks, kBlock, 0, st>>>(a, ft); break;
    case 3: forward_kernel<CODE, G, 3, LIST><<<blocks, kBlock, 0, st>>>(a, ft); break;
    case 4: forward_kernel<CODE, G, 4, LIST><<<blocks, kBlock, 0, st>>>(a, ft); break;
    default: forward_kernel<CODE, G, 8, LIST><<<blocks, kBlock, 0, st>>>(a, ft); break;
  }
}
template <int CODE, bool LIST>
static void launch_forward_g(int G, int nf, int64_t n_sl, cudaStream_t st, const ForwardArgs& a, const FreqTab& ft) {
  const unsigned blocks = (unsigned)((n_sl * G + kBlock - 1) / kBlock);
  if (G == 1) launch_forward_nf<CODE, 1, LIST>(nf, blocks, st, a, ft);
  else if (G == 8) launch_forward_nf<CODE, 8, LIST>(nf, blocks, st, a, ft);
  else launch_forward_nf<CODE, 32, LIST>(nf, blocks, st, a, ft);
}
template <int CODE>
void fwd_launch_fast(bool list, int G, int nf, int64_t n_sl, cudaStream_t st, const ForwardArgs& a, const FreqTab& ft) {
  if (list) launch_forward_g<CODE, true>(G, nf, n_sl, st, a, ft);
  else launch_forward_g<CODE, false>(G, nf, n_sl, st, a, ft);
}

template <int CODE>
void fwd_launch_batched(int nb, cudaStream_t st, const ForwardArgs& a, const FreqTab& ft0) {
  if constexpr (CODE == kAnalyticDisc || CODE == kAnalyticFull) {
    const FreqTab ft = shift_freqs(ft0, a.f0);
    const int64_t threads = a.geo.npix * ((a.batch + nb - 1) / nb);
    const unsigned blocks = (unsigned)((threads + kBlock - 1) / kBlock);
    if (nb == 4) forward_batched_kernel<CODE, 4><<<blocks, kBlock, 0, st>>>(a, ft);
    else forward_batched_kernel<CODE, 2><<<blocks, kBlock, 0, st>>>(a, ft);
  }
}

template <int CODE, int G>
static void launch_f64_nf(int nf, unsigned blocks, cudaStream_t st, const ForwardArgs& a, const FreqTab& ft0) {
  const FreqTab ft = shift_freqs(ft0, a.f0);
  switch (nf) {
    case 0: forward_f64_kernel<CODE, G, 0><<<blocks, kBlockD, 0, st>>>(a, ft); break;
    case 1: forward_f64_kernel<CODE, G, 1><<<blocks, kBlockD, 0, st>>>(a, ft); break;
    case 2: forward_f64_kernel<CODE, G, 2><<<blocks, kBlockD, 0, st>>>(a, ft); break;
    case 3: forward_f64_kernel<CODE, G, 3><<<blocks, kBlockD, 0, st>>>(a, ft); break;
    case 4: forward_f64_kernel<CODE, G, 4><<<blocks, kBlockD, 0, st>>>(a, ft); break;
    default: forward_f64_kernel<CODE, G, 8><<<blocks, kBlockD, 0, st>>>(a, ft); break;
  }
}
template <int CODE>
void fwd_launch_f64(int G, int nf, unsigned blocks, cudaStream_t st, const ForwardArgs& a, const FreqTab& ft) {
  if (G == 1) launch_f64_nf<CODE, 1>(nf, blocks, st, a, ft);
  else if (G == 8) launch_f64_nf<CODE, 8>(nf, blocks, st, a, ft);
  else launch_f64_nf<CODE, 32>(nf, blocks, st, a, ft);
}

#define SYNAX_INSTANTIATE_FWD(CODE)                                                                                       \
  template void fwd_launch_pilot<CODE>(unsigned, cudaStream_t, const ForwardArgs&, int64_t, int64_t, int*);                \
  template void fwd_launch_classify<CODE>(unsigned, cudaStream_t, const ForwardArgs&, int*);                               \
  template void fwd_launch_fast<CODE>(bool, int, int, int64_t, cudaStream_t, const ForwardArgs&, const FreqTab&);          \
  template void fwd_launch_batched<CODE>(int, cudaStream_t, const ForwardArgs&, const FreqTab&);                           \
  template void fwd_launch_f64<CODE>(int, int, unsigned, cudaStream_t, const ForwardArgs&, const FreqTab&);

}  // namespace synax
