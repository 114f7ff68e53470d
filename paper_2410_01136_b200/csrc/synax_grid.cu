// synax_grid.cu -- host-side dispatch of the gridded-B kernels (synax_grid.cuh).
#include <algorithm>
#include <numeric>

#include "synax_launch.h"
#include "synax_grid.cuh"

namespace synax {

// ------------------------------------------------------------------------------------------------
// host-side dispatch
// ------------------------------------------------------------------------------------------------
static GridDesc make_grid_desc(const synax_model* m, const float* grid) {
  GridDesc g;
  g.g = grid; g.g4 = nullptr; g.nx = m->nx; g.ny = m->ny; g.nz = m->nz;
  g.sx = (double)(m->nx - 1) / (double)m->lx; g.sy = (double)(m->ny - 1) / (double)m->ly; g.sz = (double)(m->nz - 1) / (double)m->lz;
  g.bx = 0.5 * (double)(m->nx - 1); g.by = 0.5 * (double)(m->ny - 1); g.bz = 0.5 * (double)(m->nz - 1);
  g.hx = 0.5 * (double)m->lx; g.hy = 0.5 * (double)m->ly; g.hz = 0.5 * (double)m->lz;
  return g;
}

// Repacked per-call copy of the grid (GridDesc::g4) from the plan's workspace (or the stream-ordered pool); 0 on success.
static synax_status pack_grid(GridDesc& g, Workspace* ws, bool* pooled, cudaStream_t st, int64_t* launches) {
  const int64_t n_nodes = (int64_t)g.nx * g.ny * g.nz;
  float4* g4 = static_cast<float4*>(ws_alloc(ws, sizeof(float4) * (size_t)n_nodes, st, pooled));
  if (!g4) return SYNAX_ERR_ALLOC;
  grid_pack_kernel<<<(unsigned)((n_nodes + 255) / 256), 256, 0, st>>>(g.g, n_nodes, g4);
  ++*launches;
  g.g4 = g4;
  return SYNAX_OK;
}
static void unpack_grid(const GridDesc& g, bool pooled, cudaStream_t st) {
  ws_release((void*)g.g4, pooled, st);
}

static void launch_grid_forward(int nf, unsigned blocks, cudaStream_t st, const GridFwdArgs& a, const FreqTab& ft0) {
  const FreqTab ft = shift_freqs(ft0, a.f.f0);
  const bool sg = a.f.sg_ne.g || a.f.sg_n0.g;   // gridded n_e / N_0: separate instantiation keeps the common path lean
#define SYNAX_GF(NFV)                                                                  \
  do {                                                                                 \
    if (sg) grid_forward_kernel<NFV, true><<<blocks, kBlock, 0, st>>>(a, ft);          \
    else grid_forward_kernel<NFV, false><<<blocks, kBlock, 0, st>>>(a, ft);            \
  } while (0)
  switch (nf) {
    case 1: SYNAX_GF(1); break;
    case 2: SYNAX_GF(2); break;
    case 3: SYNAX_GF(3); break;
    case 4: SYNAX_GF(4); break;
    default: SYNAX_GF(8); break;
  }
#undef SYNAX_GF
}

synax_status grid_forward(const FreqTab& ft, const ForwardArgs& a0, const synax_model* m, const float* grid,
                                 int precision, double escalate_rad, int sms, int* d_flag_count, int* h_flag_count,
                                 Workspace* ws, cudaStream_t st, int64_t* launches) {
  GridFwdArgs ga;
  ga.f = a0; ga.grid = make_grid_desc(m, grid); ga.mode = precision;
  float k_max = 0.f;
  for (int f = 0; f < ft.n_freq; ++f) k_max = fmaxf(k_max, ft.k_rad[f]);
  ga.f.flag_list = nullptr; ga.f.flag_count = d_flag_count;
  ga.f.flag_S = (float)(escalate_rad / (double)k_max);
  cudaMemsetAsync(d_flag_count, 0, kCtrlWords * sizeof(int), st);
  bool g4_pooled = false;
  const synax_status ps = pack_grid(ga.grid, ws, &g4_pooled, st, launches);
  if (ps != SYNAX_OK) return ps;
  // one warp per sightline; the hardware block scheduler balances the CTAs (a persistent grid of 16 CTAs/SM ran 2.3
  // waves of the 7 CTAs/SM that fit, with a thin last wave)
  const unsigned blocks = (unsigned)((a0.geo.npix * 32 + kBlock - 1) / kBlock);
  for (int f0 = 0; f0 < ft.n_freq;) {
    const int rem = ft.n_freq - f0, nf = rem >= 8 ? 8 : (rem >= 4 ? 4 : rem);
    ga.f.f0 = f0;
    launch_grid_forward(nf, blocks, st, ga, ft); ++*launches;
    f0 += nf;
  }
  const cudaError_t e = cudaGetLastError();
  unpack_grid(ga.grid, g4_pooled, st);
  cudaMemcpyAsync(h_flag_count, d_flag_count, kCtrlWords * sizeof(int), cudaMemcpyDeviceToHost, st);
  return e == cudaSuccess ? SYNAX_OK : SYNAX_ERR_CUDA;
}

synax_status grid_vjp(const FreqTab& ft, const Geometry& geo, const BatchConsts* bc, const BatchConstsD* bd,
                             const synax_model* m, const ScalarGridDesc& sg_ne, const ScalarGridDesc& sg_n0,
                             const float* grid, const float* dI, const float* dQ, const float* dU, float* grad,
                             int precision, double escalate_rad, int sms, Workspace* ws, cudaStream_t st, int64_t* launches) {
  GridVjpArgs a;
  a.geo = geo; a.bc = bc; a.bd = bd; a.grid = make_grid_desc(m, grid); a.sg_ne = sg_ne; a.sg_n0 = sg_n0;
  a.n_freq_total = ft.n_freq; a.dI = dI; a.dQ = dQ; a.dU = dU;
  const int64_t n_nodes = (int64_t)m->nx * m->ny * m->nz;
  int cl = 0;
  while ((32 << cl) < geo.n_los) ++cl;
  a.chunk_log2 = cl;
  float k_max = 0.f;
  for (int f = 0; f < ft.n_freq; ++f) k_max = fmaxf(k_max, ft.k_rad[f]);
  a.mode = precision; a.flag_S = (float)(escalate_rad / (double)k_max);
  // order of the pixel groups (grid_vjp_kernel): a stride of about the golden section of their count, coprime to it
  a.n_groups = (geo.npix + kGridGroup - 1) / kGridGroup;
  a.group_stride = std::max<int64_t>(1, (int64_t)(0.6180339887 * (double)a.n_groups));
  while (std::gcd(a.group_stride, a.n_groups) != 1) ++a.group_stride;
  a.group_stride %= a.n_groups;   // (n_groups = 1: stride 0, the one group)
  const size_t smem = (size_t)(kBlock / 32) * 3 * 32 * ((1u << cl) + 1) * sizeof(float);
  if (smem > 200 * 1024) return SYNAX_ERR_UNSUPPORTED;  // n_los too large for the shared-memory hand-over
  // (+ one 8-byte ticket counter per frequency block behind the accumulation buffer, cleared with it)
  const size_t acc_bytes = sizeof(float4) * (size_t)n_nodes + 8 * kMaxFreq;
  bool acc_pooled = false, g4_pooled = false;
  a.grad4 = static_cast<float*>(ws_alloc(ws, acc_bytes, st, &acc_pooled));
  if (!a.grad4) return SYNAX_ERR_ALLOC;
  unsigned long long* tickets = reinterpret_cast<unsigned long long*>(a.grad4 + (size_t)n_nodes * 4);
  if (cudaMemsetAsync(a.grad4, 0, acc_bytes, st) != cudaSuccess) {
    ws_release(a.grad4, acc_pooled, st);
    return SYNAX_ERR_CUDA;
  }
  const synax_status ps = pack_grid(a.grid, ws, &g4_pooled, st, launches);
  if (ps != SYNAX_OK) {
    ws_release(a.grad4, acc_pooled, st);
    return ps;
  }
  const int64_t max_blocks = (geo.npix * 32 + kBlock - 1) / kBlock;
  for (int f0 = 0; f0 < ft.n_freq;) {
    const int rem = ft.n_freq - f0, nf = rem >= 8 ? 8 : (rem >= 4 ? 4 : rem);
    a.f0 = f0;
    a.ticket = tickets + f0;
    const bool sg = a.sg_ne.g || a.sg_n0.g;
#define SYNAX_GV(NFV)                                                                                              \
  do {                                                                                                             \
    /* persistent warps (per-warp shared-memory state): exactly the CTAs that are resident at once, so no thin last wave */ \
    if (sg) {                                                                                                      \
      cudaFuncSetAttribute(grid_vjp_kernel<NFV, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);    \
      int occ = 1;                                                                                                 \
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, grid_vjp_kernel<NFV, true>, kBlock, smem);               \
      const unsigned blocks = (unsigned)std::min<int64_t>((int64_t)sms * std::max(occ, 1), max_blocks);            \
      grid_vjp_kernel<NFV, true><<<blocks, kBlock, smem, st>>>(a, shift_freqs(ft, a.f0));                          \
    } else {                                                                                                       \
      cudaFuncSetAttribute(grid_vjp_kernel<NFV, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);   \
      int occ = 1;                                                                                                 \
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, grid_vjp_kernel<NFV, false>, kBlock, smem);              \
      const unsigned blocks = (unsigned)std::min<int64_t>((int64_t)sms * std::max(occ, 1), max_blocks);            \
      grid_vjp_kernel<NFV, false><<<blocks, kBlock, smem, st>>>(a, shift_freqs(ft, a.f0));                         \
    }                                                                                                              \
  } while (0)
    switch (nf) {
      case 1: SYNAX_GV(1); break;
      case 2: SYNAX_GV(2); break;
      case 3: SYNAX_GV(3); break;
      case 4: SYNAX_GV(4); break;
      default: SYNAX_GV(8); break;
    }
#undef SYNAX_GV
    ++*launches;
    f0 += nf;
  }
  grid_grad_compact_kernel<<<(unsigned)((n_nodes + 255) / 256), 256, 0, st>>>(reinterpret_cast<const float4*>(a.grad4), n_nodes, grad);
  ++*launches;
  const cudaError_t e = cudaGetLastError();
  ws_release(a.grad4, acc_pooled, st);
  unpack_grid(a.grid, g4_pooled, st);
  return e == cudaSuccess ? SYNAX_OK : SYNAX_ERR_CUDA;
}

}  // namespace synax
