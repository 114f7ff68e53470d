// grid_streams.cu -- "achievable" ceilings for the gridded path (microbenchmarks (G) and (R)):
// the memory-system work of grid_forward_kernel / grid_vjp_kernel on config 3's ACTUAL index stream
// (nside 64, 512 samples over 20 kpc, 128x128x32x3 grid over 40x40x8 kpc, observer (-8.3, 0, 0.006)) with the
// arithmetic of the method removed:
//   G  one warp per sightline, lanes on consecutive samples, the 8-corner x 3-component gather (24 loads per
//      sample) summed into one float per sightline;
//   R  one warp per sightline, lanes on contiguous chunks, one red.global.add.f32 x 24 each time a lane leaves a
//      cell (per-cell aggregation as in grid_vjp_kernel sweep 2), and the un-aggregated variant (24 per sample).
// Build + run: python -m paper_2410_01136_b200.ubench   (nvcc, sm_100a; prints one line per stream)
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <numeric>
#include <vector>

#include "../csrc/synax_grid.cuh"
#include "../csrc/synax_plan_kernels.cuh"

using namespace synax;

__global__ void gather_stream(Geometry geo, GridDesc G, float* __restrict__ out) {
  const int lane = threadIdx.x & 31;
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t n_warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  for (int64_t pix = warp; pix < geo.npix; pix += n_warps) {
    const Triad T = load_triad(geo.dirs, pix);
    float acc = 0.f;
    for (int nt = 0; nt < geo.n_los; nt += 32) {
      const double s_d = ((double)(nt + lane) + 0.5) * geo.delta;
      const Cell c = locate(G, fma(s_d, T.nxd, geo.obs[0]), fma(s_d, T.nyd, geo.obs[1]), fma(s_d, T.nzd, geo.obs[2]));
      if (c.inbox && nt + lane < geo.n_los) {
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          const float* p = G.g + 3 * (c.base + corner_offset(G, q));
          acc += __ldg(p) + __ldg(p + 1) + __ldg(p + 2);
        }
      }
    }
    acc = group_sum<32>(acc);
    if (lane == 0) out[pix] = acc;
  }
}

// the same stream on the padded [node][4] copy the kernels gather from: one 16-byte load per corner
__global__ void gather_stream_v4(Geometry geo, GridDesc G, float* __restrict__ out) {
  const int lane = threadIdx.x & 31;
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t n_warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  for (int64_t pix = warp; pix < geo.npix; pix += n_warps) {
    const Triad T = load_triad(geo.dirs, pix);
    float acc = 0.f;
    for (int nt = 0; nt < geo.n_los; nt += 32) {
      const double s_d = ((double)(nt + lane) + 0.5) * geo.delta;
      const Cell c = locate(G, fma(s_d, T.nxd, geo.obs[0]), fma(s_d, T.nyd, geo.obs[1]), fma(s_d, T.nzd, geo.obs[2]));
      if (c.inbox && nt + lane < geo.n_los) {
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          const float4 v = __ldg(G.g4 + c.base + corner_offset(G, q));
          acc += v.x + v.y + v.z;
        }
      }
    }
    acc = group_sum<32>(acc);
    if (lane == 0) out[pix] = acc;
  }
}

template <bool AGGREGATE>
__global__ void red_stream(Geometry geo, GridDesc G, float* __restrict__ grad, unsigned long long* __restrict__ count) {
  const int lane = threadIdx.x & 31;
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t n_warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  const int C = (geo.n_los + 31) / 32;
  unsigned long long mine = 0;
  for (int64_t pix = warp; pix < geo.npix; pix += n_warps) {
    const Triad T = load_triad(geo.dirs, pix);
    const int m0 = min(lane * C, geo.n_los), m1 = min(m0 + C, geo.n_los);
    int cur = -1;
    for (int m = m1 - 1; m >= m0 - 1; --m) {
      int cell = -1;
      if (m >= m0) {
        const double s_d = ((double)m + 0.5) * geo.delta;
        const Cell c = locate(G, fma(s_d, T.nxd, geo.obs[0]), fma(s_d, T.nyd, geo.obs[1]), fma(s_d, T.nzd, geo.obs[2]));
        cell = c.inbox ? c.base : -1;
      }
      const bool flush = AGGREGATE ? (cell != cur && cur >= 0) : (cur >= 0);
      if (flush) {
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          float* p = grad + 3 * (cur + corner_offset(G, q));
          atomicAdd(p, 1.0f); atomicAdd(p + 1, 1.0f); atomicAdd(p + 2, 1.0f);
        }
        mine += 24;
      }
      cur = cell;
    }
  }
  atomicAdd(count, mine);
}

__device__ __forceinline__ void red_add_v4(float* p, float a, float b, float c, float d) {
  asm volatile("red.global.v4.f32.add [%0], {%1, %2, %3, %4};" :: "l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
// the same stream into a gradient padded to 4 floats per node: one 16-byte vector red per corner
// group_stride > 0: the sightlines in grid_vjp_kernel's order (groups of kGridGroup neighbouring pixels, group q -> q * stride mod n)
__global__ void red_stream_v4(Geometry geo, GridDesc G, float* __restrict__ grad4, unsigned long long* __restrict__ count,
                              int64_t n_groups, int64_t group_stride) {
  const int lane = threadIdx.x & 31;
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t n_warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  const int C = (geo.n_los + 31) / 32;
  unsigned long long mine = 0;
  for (int64_t pidx = warp; pidx < n_groups * kGridGroup; pidx += n_warps) {
    const int64_t pix = group_stride > 0 ? (((pidx / kGridGroup) * group_stride) % n_groups) * kGridGroup + pidx % kGridGroup : pidx;
    if (pix >= geo.npix) continue;
    const Triad T = load_triad(geo.dirs, pix);
    const int m0 = min(lane * C, geo.n_los), m1 = min(m0 + C, geo.n_los);
    int cur = -1;
    for (int m = m1 - 1; m >= m0 - 1; --m) {
      int cell = -1;
      if (m >= m0) {
        const double s_d = ((double)m + 0.5) * geo.delta;
        const Cell c = locate(G, fma(s_d, T.nxd, geo.obs[0]), fma(s_d, T.nyd, geo.obs[1]), fma(s_d, T.nzd, geo.obs[2]));
        cell = c.inbox ? c.base : -1;
      }
      if (cell != cur && cur >= 0) {
#pragma unroll
        for (int q = 0; q < 8; ++q) red_add_v4(grad4 + (size_t)(cur + corner_offset(G, q)) * 4, 1.0f, 1.0f, 1.0f, 0.0f);
        mine += 8;
      }
      cur = cell;
    }
  }
  atomicAdd(count, mine);
}

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { printf("CUDA error %s at %s:%d\n", cudaGetErrorString(e_), __FILE__, __LINE__); return 1; } } while (0)

int main() {
  const int nside = 64, n_los = 512, nx = 128, ny = 128, nz = 32;
  const double s_max = 20.0;
  const int64_t npix = 12LL * nside * nside;
  double* dirs; float *grid, *out, *grad; unsigned long long* count;
  const size_t ngrid = (size_t)nx * ny * nz * 3;
  CK(cudaMalloc(&dirs, npix * 4 * sizeof(double)));
  CK(cudaMalloc(&grid, ngrid * 4)); CK(cudaMalloc(&grad, ngrid * 4)); CK(cudaMalloc(&out, npix * 4));
  CK(cudaMalloc(&count, 8));
  CK(cudaMemset(grid, 0, ngrid * 4)); CK(cudaMemset(grad, 0, ngrid * 4));
  pix2ang_kernel<<<(unsigned)((npix + 255) / 256), 256>>>(nside, 0, 1, npix, dirs);
  Geometry geo; geo.npix = npix; geo.n_los = n_los; geo.delta = s_max / n_los;
  geo.obs[0] = -8.3; geo.obs[1] = 0.0; geo.obs[2] = 0.006; geo.obsf[0] = -8.3f; geo.obsf[1] = 0.f; geo.obsf[2] = 0.006f; geo.dirs = dirs; geo.path = nullptr;
  float4* grid4; CK(cudaMalloc(&grid4, ngrid / 3 * sizeof(float4))); CK(cudaMemset(grid4, 0, ngrid / 3 * sizeof(float4)));
  GridDesc G; G.g = grid; G.g4 = grid4; G.nx = nx; G.ny = ny; G.nz = nz;
  G.sx = (nx - 1) / 40.0; G.sy = (ny - 1) / 40.0; G.sz = (nz - 1) / 8.0;
  G.bx = 0.5 * (nx - 1); G.by = 0.5 * (ny - 1); G.bz = 0.5 * (nz - 1);
  G.hx = 20.0; G.hy = 20.0; G.hz = 4.0;
  int sms = 148; cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  const double samples = (double)npix * n_los;
  auto time_it = [&](auto launch, const char* name, double units, const char* unit) {
    launch(); launch();
    cudaEventRecord(e0);
    for (int i = 0; i < 10; ++i) launch();
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1); ms /= 10;
    printf("%-40s %.4f ms  %.3e %s/s  (%.3e samples/s)\n", name, ms, units / (ms * 1e-3), unit, samples / (ms * 1e-3));
    return (double)ms;
  };
  double best_g = 1e30, best_g4 = 1e30, best_r4 = 1e30;
  for (int bps : {8, 16, 32}) {
    char name[64]; snprintf(name, sizeof(name), "G gather 96 B/sample, %d CTAs/SM", bps);
    best_g = std::min(best_g, time_it([&] { gather_stream<<<sms * bps, 128>>>(geo, G, out); }, name, samples * 96.0, "B"));
  }
  for (int bps : {8, 16, 32}) {
    char name[64]; snprintf(name, sizeof(name), "G4 gather 8 x 16 B/sample, %d CTAs/SM", bps);
    best_g4 = std::min(best_g4, time_it([&] { gather_stream_v4<<<sms * bps, 128>>>(geo, G, out); }, name, samples * 128.0, "B"));
  }
  unsigned long long h = 0;
  CK(cudaMemset(count, 0, 8));
  red_stream<true><<<sms * 16, 128>>>(geo, G, grad, count);
  CK(cudaMemcpy(&h, count, 8, cudaMemcpyDeviceToHost));
  const double n_agg = (double)h;
  CK(cudaMemset(count, 0, 8));
  red_stream<false><<<sms * 16, 128>>>(geo, G, grad, count);
  CK(cudaMemcpy(&h, count, 8, cudaMemcpyDeviceToHost));
  const double n_raw = (double)h;
  printf("atomics per call: per-cell aggregated %.4e, un-aggregated %.4e (ratio %.2f)\n", n_agg, n_raw, n_raw / n_agg);
  for (int bps : {8, 16, 32}) {
    char name[64]; snprintf(name, sizeof(name), "R red.add per-cell aggregated, %d CTAs/SM", bps);
    time_it([&] { red_stream<true><<<sms * bps, 128>>>(geo, G, grad, count); }, name, n_agg, "red");
  }
  time_it([&] { red_stream<false><<<sms * 16, 128>>>(geo, G, grad, count); }, "R red.add un-aggregated, 16 CTAs/SM", n_raw, "red");
  float* grad4; CK(cudaMalloc(&grad4, ngrid / 3 * 4 * 4)); CK(cudaMemset(grad4, 0, ngrid / 3 * 4 * 4));
  const int64_t n_groups = (npix + kGridGroup - 1) / kGridGroup;
  int64_t group_stride = std::max<int64_t>(1, (int64_t)(0.6180339887 * (double)n_groups));   // as grid_vjp() chooses it
  while (std::gcd(group_stride, n_groups) != 1) ++group_stride;
  double best_r4p = 1e30;
  for (int bps : {8, 16}) {
    char name[80]; snprintf(name, sizeof(name), "R red.add.v4 per-cell aggregated, pixel order, %d CTAs/SM", bps);
    best_r4 = std::min(best_r4, time_it([&] { red_stream_v4<<<sms * bps, 128>>>(geo, G, grad4, count, n_groups, 0); }, name, n_agg / 3, "red.v4"));
  }
  for (int bps : {5, 8, 16}) {
    char name[80]; snprintf(name, sizeof(name), "R red.add.v4, the adjoint's group order, %d CTAs/SM", bps);
    best_r4p = std::min(best_r4p, time_it([&] { red_stream_v4<<<sms * bps, 128>>>(geo, G, grad4, count, n_groups, group_stride); }, name, n_agg / 3, "red.v4"));
  }
  // one machine-readable line for bench.py --config 3 (the ceilings of the gridded path, best over the CTA counts)
  printf("JSON {\"gather_ms\": %.5f, \"gather_v4_ms\": %.5f, \"red_v4_ms\": %.5f, \"red_v4_group_order_ms\": %.5f, \"gather_bytes\": %.6e, \"red_v4_count\": %.6e, \"samples\": %.6e}\n",
         best_g, best_g4, best_r4, best_r4p, samples * 96.0, n_agg / 3, samples);
  CK(cudaDeviceSynchronize());
  return 0;
}
