// synax_vjp_driver.cu -- host-side orchestration of the analytic adjoint: pilot, per-CTA pair on two streams,
// frequency passes, deterministic reduction ("VJP").
#include <algorithm>

#include "synax_launch.h"

namespace synax {

// decide_kernel lives in synax_api.cu's translation unit (synax_plan_kernels.cuh)
void launch_decide(int* ctrl, int64_t n_pilot, int num, int den, int mode_yes, cudaStream_t st);

static void launch_pmode(int code, int pmode, int G, int nf, dim3 grid, cudaStream_t st, const VjpArgs& a, const FreqTab& ft) {
  SYNAX_DISPATCH_CODE(code, vjp_launch, pmode, G, nf, grid, st, a, ft);
}

// the lean fp32 variant, or its batched form (nb parameter vectors per thread sharing the sightline geometry, A12)
static void launch_lean(int code, int nb, int G, int nf, dim3 grid, cudaStream_t st, const VjpArgs& a, const FreqTab& ft) {
  if (nb > 0) {
    const dim3 gb(grid.x, (unsigned)((a.batch + nb - 1) / nb));
    SYNAX_DISPATCH_CODE(code, vjp_launch_batched, nb, gb, st, a, ft);
  } else {
    launch_pmode(code, 0, G, nf, grid, st, a, ft);
  }
}

// partial[b][n_blocks][16] -> grad[b][n_params], float64 accumulation, deterministic order
__global__ void vjp_reduce_kernel(const float* __restrict__ partial, int n_blocks, int n_params, float* __restrict__ grad) {
  const int b = blockIdx.x;
  const int j = threadIdx.x & 15;
  const int part = threadIdx.x >> 4;        // 16 partial sums per parameter
  __shared__ double sh[16][17];
  double s = 0.0;
  if (j < n_params)
    for (int k = part; k < n_blocks; k += 16) s += (double)partial[((size_t)b * n_blocks + k) * 16 + j];
  sh[part][j] = s;
  __syncthreads();
  if (threadIdx.x < n_params) {
    double t = 0.0;
    for (int k = 0; k < 16; ++k) t += sh[k][threadIdx.x];
    grad[(size_t)b * n_params + threadIdx.x] = (float)t;
  }
}

// precision 0: per sightline (PMODE 2), threshold = the forward's, escalate_rad (300 rad) -- unless a pilot over ~8k sightlines
// finds none above HALF that threshold, in which case the lean fp32 variant (PMODE 0: fewer registers, no estimate) runs
// (cfg 2 at 23 GHz: 8.2 instead of 9.5 ms).  Decided on the device, no host sync.
// (Until late in round 2 the adjoint used 10/3 x escalate_rad = 1000 rad, on the argument that a gradient is a sum over all
// pixels with a 1e-3 bound.  A cotangent that is non-zero on a few hundred pixels only -- a masked likelihood -- takes that
// averaging away: of 400 seeded random mid-size workloads with such cotangents, 6 missed the bound by up to 5e-2 at 1000 rad,
// one still at 500 rad, none at 300 rad.  The adjoint after a forward was never affected: it works on the forward's own selection.)
constexpr double kVjpEscalateFactor = 1.0;   // x escalate_rad
constexpr int kStandAloneVectors = 1;   // vectors per thread of the stand-alone forward-order adjoint (2: 8.25 ms at cfg 2)

synax_status analytic_vjp(int code, const FreqTab& ft, const Geometry& geo, const BatchConsts* bc,
                                 const BatchConstsD* bd, int batch, int n_params, int G, const ScalarGridDesc& sg_ne,
                                 const ScalarGridDesc& sg_n0, int precision, double escalate_rad, int batch_share, const double* phi, const int* phi_ok,
                          const double* phi_base, const unsigned char* phi_has, int* ctrl,
                                 cudaStream_t aux, cudaEvent_t ev_fork, cudaEvent_t ev_join,
                                 const float* dI, const float* dQ, const float* dU, float* grad, Workspace* ws, cudaStream_t st,
                                 int64_t* launches) {
  VjpArgs a;
  a.geo = geo; a.bc = bc; a.bd = bd; a.batch = batch; a.n_freq_total = ft.n_freq;
  a.dI = dI; a.dQ = dQ; a.dU = dU; a.sg_ne = sg_ne; a.sg_n0 = sg_n0;
  a.n_blocks = (int)((geo.npix * G + kBlock - 1) / kBlock);
  float k_max = 0.f;
  for (int f = 0; f < ft.n_freq; ++f) k_max = fmaxf(k_max, ft.k_rad[f]);
  a.flag_S = (float)(kVjpEscalateFactor * escalate_rad / (double)k_max);
  a.mode = nullptr; a.cta_sel = nullptr;
  a.phi = phi; a.phi_ok = phi_ok; a.phi_base = phi_base; a.phi_has = phi_has; a.only_with_bases = 0;
  // Long calls with one thread per sightline: the work is split per CTA between the lean fp32 variant and the
  // float64-angle variant (vjp_classify_kernel) instead of deciding per sightline inside one heavier kernel
  // (cfg 4 stand-alone with nothing stored by a forward: DESIGN.md section 5).
  // (G lanes per sightline, G > 1: a CTA holds 128 / G sightlines; worth its three extra launches from ~1M threads)
  const bool split = precision == 0 && (G == 1 ? geo.npix * batch >= 262144 : geo.npix * batch * G >= 1000000);
  if (precision == 0) {
    ForwardArgs pa;
    pa.geo = geo; pa.bc = bc; pa.bd = bd; pa.batch = batch; pa.sg_ne = sg_ne; pa.sg_n0 = sg_n0;
    pa.flag_S = 0.5f * a.flag_S; pa.flag_T = 0.0f;
    const int64_t n_sl = geo.npix * batch;
    const int64_t stride = (n_sl / 8192) | 1;
    const int64_t n_pilot = (n_sl + stride - 1) / stride;
    const unsigned pb = (unsigned)((n_pilot * 32 + kBlock - 1) / kBlock);
    if (cudaMemsetAsync(ctrl, 0, kCtrlWords * sizeof(int), st) != cudaSuccess) return SYNAX_ERR_CUDA;
    SYNAX_DISPATCH_CODE(code, fwd_launch_pilot, pb, st, pa, stride, n_pilot, ctrl);
    // any sampled sightline above half the threshold: per-sightline variant, or (long calls) the per-CTA pair
    launch_decide(ctrl, n_pilot, 0, 1, split ? kModeSplit : kModeAllF64, st);
    *launches += 2;
    a.mode = ctrl + kCtrlMode;
  }
  unsigned char* cta_sel = nullptr;
  bool sel_pooled = false, partial_pooled = false;
  if (split && !(cta_sel = static_cast<unsigned char*>(ws_alloc(ws, (size_t)a.n_blocks * (size_t)batch, st, &sel_pooled))))
    return SYNAX_ERR_ALLOC;
  // measured at cfg 2 (256 vectors, B200): sharing pays in the forward (5.09 -> 4.68 ms at 4 vectors per thread) but not here
  // -- two or four sets of 27 gradient accumulators per thread cost more occupancy than the shared geometry saves (8.46 ->
  // 8.82 / 9.53 ms) -- so the adjoint shares only on request (option "batch_share")
  // nb: 0 = vjp_kernel (backward sweep), 1 / 2 / 4 = vjp_batched_kernel (forward order, that many vectors per thread).
  // The backward sweep needs the sightline's Faraday total first.  After a forward of this plan it is there (phi); a call
  // the host knows to be stand-alone would pay a pre-pass for it -- a second evaluation of the fields, 70 % on top at one
  // frequency (cfg 2: 11.6 against 6.7 ms) -- so it takes the forward-order kernel instead, whose prefix-form scan needs no
  // total (cfg 2 stand-alone: 7.7 ms).  With tile bases on offer the lean vjp_kernel is the one that uses them.
  const bool fo_ok = G == 1 && ft.n_freq == 1 && (code == kAnalyticDisc || code == kAnalyticFull) && !sg_ne.g && !sg_n0.g && batch <= 65535;
  int nb = 0;
  if (fo_ok && batch_share > 1 && !phi_base) nb = batch_share;
  else if (fo_ok && !phi) nb = kStandAloneVectors;
  float* partial = static_cast<float*>(ws_alloc(ws, sizeof(float) * 16 * (size_t)a.n_blocks * (size_t)batch, st, &partial_pooled));
  if (!partial) {
    ws_release(cta_sel, sel_pooled, st);
    return SYNAX_ERR_ALLOC;
  }
  a.partial = partial;
  cudaError_t stream_err = cudaSuccess;   // fork / join of the second stream
  for (int b0 = 0; b0 < batch; b0 += 65535) {   // gridDim.y limit
    const dim3 grid((unsigned)a.n_blocks, (unsigned)std::min(65535, batch - b0));
    a.b0 = b0;
    if (split) {
      SYNAX_DISPATCH_CODE(code, vjp_launch_classify, G, grid, st, a, cta_sel);
      ++*launches;
      cudaError_t r = cudaEventRecord(ev_fork, st);
      if (r == cudaSuccess) r = cudaStreamWaitEvent(aux, ev_fork, 0);
      if (r != cudaSuccess) { stream_err = r; break; }   // nothing launched on the second stream yet: clean up below
    }
    for (int f0 = 0; f0 < ft.n_freq;) {
      const int rem = ft.n_freq - f0;
      const int nf = rem >= 8 ? 8 : (rem >= 4 ? 4 : rem);
      a.f0 = f0; a.accumulate = f0 > 0;
      if (precision == 1) launch_lean(code, nb, G, nf, grid, st, a, ft);
      else if (precision == 2) {
        launch_pmode(code, 1, G, nf, grid, st, a, ft);
        if (phi_base) {   // ... or, when the forward left tile bases for every sightline, the lean variant on those (the float64
          VjpArgs ab = a;  // variant stands aside then)
          ab.only_with_bases = 1;
          launch_pmode(code, 0, G, nf, grid, st, ab, ft);
          ++*launches;
        }
      }
      else {
        launch_lean(code, nb, G, nf, grid, st, a, ft);
        if (split) {
          // the per-CTA pair (runs in kModeSplit).  Every CTA's partial belongs to exactly one member, so the two run
          // concurrently: the float64-angle member (few, long CTAs: 2.7 waves at cfg 4) on the plan's second stream,
          // forked after the classify kernel and joined before the reduction, fills its tail with the other's CTAs.
          VjpArgs as = a;
          as.cta_sel = cta_sel;
          launch_pmode(code, 1, G, nf, grid, aux, as, ft);
          launch_pmode(code, 0, G, nf, grid, st, as, ft);
          ++*launches;
        } else {
          launch_pmode(code, 2, G, nf, grid, st, a, ft);
        }
        ++*launches;
      }
      ++*launches;
      f0 += nf;
    }
    if (split) {
      cudaError_t r = cudaEventRecord(ev_join, aux);
      if (r == cudaSuccess) r = cudaStreamWaitEvent(st, ev_join, 0);
      if (r != cudaSuccess) { stream_err = r; cudaStreamSynchronize(aux); break; }   // join by hand, then clean up
    }
  }
  if (stream_err == cudaSuccess) {
    vjp_reduce_kernel<<<batch, 256, 0, st>>>(partial, a.n_blocks, n_params, grad);
    ++*launches;
  }
  cudaError_t e = cudaGetLastError();
  if (stream_err != cudaSuccess) e = stream_err;
  ws_release(partial, partial_pooled, st);
  ws_release(cta_sel, sel_pooled, st);
  return e == cudaSuccess ? SYNAX_OK : SYNAX_ERR_CUDA;
}

}  // namespace synax
