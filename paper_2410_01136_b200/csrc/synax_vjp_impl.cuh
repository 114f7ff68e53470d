// synax_vjp_impl.cuh -- definitions of the adjoint launchers of synax_launch.h for one model code; included by the
// synax_vjp_<code>.cu translation units, which instantiate them explicitly.
#pragma once
#include "synax_launch.h"

namespace synax {

template <int CODE>
void vjp_launch_classify(int G, dim3 grid, cudaStream_t st, const VjpArgs& a, unsigned char* cta_sel) {
  if (G == 1) vjp_classify_kernel<CODE, 1><<<grid, kBlock, 0, st>>>(a, cta_sel);
  else if (G == 8) vjp_classify_kernel<CODE, 8><<<grid, kBlock, 0, st>>>(a, cta_sel);
  else vjp_classify_kernel<CODE, 32><<<grid, kBlock, 0, st>>>(a, cta_sel);
}

template <int CODE>
void vjp_launch_batched(int nb, dim3 grid, cudaStream_t st, const VjpArgs& a, const FreqTab& ft0) {
  if constexpr (CODE == kAnalyticDisc || CODE == kAnalyticFull) {
    const FreqTab ft = shift_freqs(ft0, a.f0);
    if (nb == 4) vjp_batched_kernel<CODE, 4><<<grid, kBlock, 0, st>>>(a, ft);
    else if (nb == 2) vjp_batched_kernel<CODE, 2><<<grid, kBlock, 0, st>>>(a, ft);
    else vjp_batched_kernel<CODE, 1><<<grid, kBlock, 0, st>>>(a, ft);
  }
}

template <int CODE, int G, int PMODE>
static void launch_vjp_nf(int nf, dim3 grid, cudaStream_t st, const VjpArgs& a, const FreqTab& ft0) {
  const FreqTab ft = shift_freqs(ft0, a.f0);
  switch (nf) {
    case 1: vjp_kernel<CODE, G, 1, PMODE><<<grid, kBlock, 0, st>>>(a, ft); break;
    case 2: vjp_kernel<CODE, G, 2, PMODE><<<grid, kBlock, 0, st>>>(a, ft); break;
    case 3: vjp_kernel<CODE, G, 3, PMODE><<<grid, kBlock, 0, st>>>(a, ft); break;
    case 4: vjp_kernel<CODE, G, 4, PMODE><<<grid, kBlock, 0, st>>>(a, ft); break;
    default: vjp_kernel<CODE, G, 8, PMODE><<<grid, kBlock, 0, st>>>(a, ft); break;
  }
}
template <int CODE, int PMODE>
static void launch_vjp_g(int G, int nf, dim3 grid, cudaStream_t st, const VjpArgs& a, const FreqTab& ft) {
  if (G == 1) launch_vjp_nf<CODE, 1, PMODE>(nf, grid, st, a, ft);
  else if (G == 8) launch_vjp_nf<CODE, 8, PMODE>(nf, grid, st, a, ft);
  else launch_vjp_nf<CODE, 32, PMODE>(nf, grid, st, a, ft);
}
template <int CODE>
void vjp_launch(int pmode, int G, int nf, dim3 grid, cudaStream_t st, const VjpArgs& a, const FreqTab& ft) {
  if (pmode == 0) launch_vjp_g<CODE, 0>(G, nf, grid, st, a, ft);
  else if (pmode == 1) launch_vjp_g<CODE, 1>(G, nf, grid, st, a, ft);
  else launch_vjp_g<CODE, 2>(G, nf, grid, st, a, ft);
}

#define SYNAX_INSTANTIATE_VJP(CODE)                                                                           \
  template void vjp_launch<CODE>(int, int, int, dim3, cudaStream_t, const VjpArgs&, const FreqTab&);           \
  template void vjp_launch_batched<CODE>(int, dim3, cudaStream_t, const VjpArgs&, const FreqTab&);             \
  template void vjp_launch_classify<CODE>(int, dim3, cudaStream_t, const VjpArgs&, unsigned char*);

}  // namespace synax
