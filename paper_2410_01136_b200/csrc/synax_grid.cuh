// synax_grid.cuh -- gridded-B model (cfg 3): forward with trilinear gathers (A3') and the adjoint with
// scatter-add into the grid gradient (A11').  One warp per sightline.
//   forward / adjoint sweep 1: lanes take CONSECUTIVE samples (neighbouring lanes read neighbouring
//     cells -> gathers coalesce), Faraday depth by a warp inclusive scan per 32-sample tile plus a
//     float64 carry;
//   adjoint sweep 2: lanes take CONTIGUOUS chunks, so a lane stays in one cell for several samples and
//     accumulates its 8x3 corner contributions in registers, flushing with red.global.add only when
//     the cell changes.  Per-sample cotangents travel from sweep 1 to sweep 2 through shared memory.
#pragma once
#include "../../include/synax.h"
#include "synax_forward.cuh"

namespace synax {

struct GridDesc {
  const float* g;       // caller's grid [nx][ny][nz][3]
  // Per-call repacked copy (grid_pack_kernel; L2-resident like the grid itself).  The kernels are bound by L1 gather
  // wavefronts (ncu: l1tex data pipe 70 %, long-scoreboard stalls), so a node is padded to one 16-byte vector: a corner
  // costs one LDG.128 instead of three LDG.32.  The float64 chain converts the 24 values of a sample in registers -- a
  // float64 copy of the nodes (two LDG.128 per corner) was slower: 0.256 vs 0.241 ms for cfg 3's forward.
  const float4* g4;     // [node] = (Bx, By, Bz, 0)
  int nx, ny, nz;
  double sx, sy, sz;    // (n-1)/l
  double bx, by, bz;    // (n-1)/2
  double hx, hy, hz;    // l/2
};

struct Cell {
  int base;             // node index of corner (i,j,k)
  int i, j, k;
  float tx, ty, tz;
  bool inbox;
};

__device__ __forceinline__ Cell locate(const GridDesc& G, double x, double y, double z) {
  const double ux = fma(x, G.sx, G.bx), uy = fma(y, G.sy, G.by), uz = fma(z, G.sz, G.bz);
  Cell c;
  c.inbox = (ux >= 0.0) && (ux <= (double)(G.nx - 1)) && (uy >= 0.0) && (uy <= (double)(G.ny - 1)) &&
            (uz >= 0.0) && (uz <= (double)(G.nz - 1));
  int i = __double2int_rd(ux), j = __double2int_rd(uy), k = __double2int_rd(uz);
  i = max(0, min(i, G.nx - 2)); j = max(0, min(j, G.ny - 2)); k = max(0, min(k, G.nz - 2));
  c.tx = (float)(ux - (double)i); c.ty = (float)(uy - (double)j); c.tz = (float)(uz - (double)k);
  c.base = (i * G.ny + j) * G.nz + k;
  c.i = i; c.j = j; c.k = k;
  return c;
}

// trilinear weights in the order (a,b,d) = (0,0,0),(0,0,1),(0,1,0),(0,1,1),(1,0,0),...
__device__ __forceinline__ void weights(const Cell& c, float w[8]) {
  const float x0 = 1.0f - c.tx, y0 = 1.0f - c.ty, z0 = 1.0f - c.tz;
  const float a00 = x0 * y0, a01 = x0 * c.ty, a10 = c.tx * y0, a11 = c.tx * c.ty;
  w[0] = a00 * z0; w[1] = a00 * c.tz; w[2] = a01 * z0; w[3] = a01 * c.tz;
  w[4] = a10 * z0; w[5] = a10 * c.tz; w[6] = a11 * z0; w[7] = a11 * c.tz;
}

__device__ __forceinline__ int corner_offset(const GridDesc& G, int q) {  // q = a*4 + b*2 + d
  return ((q >> 2) * G.ny + ((q >> 1) & 1)) * G.nz + (q & 1);   // in nodes
}

__device__ __forceinline__ void gather_B(const GridDesc& G, const Cell& c, float B[3]) {
  float w[8];
  weights(c, w);
  B[0] = B[1] = B[2] = 0.f;
  if (!c.inbox) return;
#pragma unroll
  for (int q = 0; q < 8; ++q) {
    const float4 v = __ldg(G.g4 + c.base + corner_offset(G, q));
    B[0] = fmaf(w[q], v.x, B[0]);
    B[1] = fmaf(w[q], v.y, B[1]);
    B[2] = fmaf(w[q], v.z, B[2]);
  }
}

// CR and thermal-electron exponential discs from aux (fp32 chain), Eq.(12)
__device__ __forceinline__ void densities_f32(const BatchConsts& P, float rho2, float z, float& N0, float& ne) {
  const float rho = rho2 * mufu_rsqrt(fmaxf(rho2, 1e-30f));
  const float az = fabsf(z);
  const float ez = mufu_ex2(P.k_hz * az), dz = 1.0f + ez;
  N0 = 4.0f * P.p[9] * mufu_ex2(P.k_hr * rho) * ez * mufu_rcp(dz * dz);
  const float ee = mufu_ex2(P.k_hez * az), de = 1.0f + ee;
  ne = 4.0f * P.p[13] * mufu_ex2(P.k_her * rho) * ee * mufu_rcp(de * de);
}

__device__ __forceinline__ float warp_inclusive_scan(float v, int lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const float o = __shfl_up_sync(0xffffffffu, v, d);
    if (lane >= d) v += o;
  }
  return v;
}
// sin/cos of the Faraday angle k_turn * S for a float64 S (turn reduction in float64)
__device__ __forceinline__ void faraday_sincos(double k_turn, double S, float& c, float& s) {
  double t = k_turn * S;
  t -= rint(t);
  const float a = (float)t * 6.283185307179586f;
  c = mufu_cos(a); s = mufu_sin(a);
}

// CR density only (fp32 MUFU chain), Eq.(12) P:L173 -- the emission needs no more than that
__device__ __forceinline__ float n0_f32(const BatchConsts& P, float rho2, float z) {
  const float rho = rho2 * mufu_rsqrt(fmaxf(rho2, 1e-30f));
  const float ez = mufu_ex2(P.k_hz * fabsf(z)), dz = 1.0f + ez;
  return 4.0f * P.p[9] * mufu_ex2(P.k_hr * rho) * ez * mufu_rcp(dz * dz);
}

// float64 chain for one sample: coordinates, trilinear weights and interpolation in float64, n_e in float64 from
// the short polynomials of synax_f64.cuh; N_0 stays fp32.
__device__ __forceinline__ void fields_f64(const GridDesc& G, const BatchConsts& P, const BatchConstsD& D,
                                           const double4 dir, double xd, double yd, double zd, double& Bpar,
                                           double& BN, double& BE, float& N0, double& ne) {
  const double ux = fma(xd, G.sx, G.bx), uy = fma(yd, G.sy, G.by), uz = fma(zd, G.sz, G.bz);
  const bool inbox = (ux >= 0.0) && (ux <= (double)(G.nx - 1)) && (uy >= 0.0) && (uy <= (double)(G.ny - 1)) &&
                     (uz >= 0.0) && (uz <= (double)(G.nz - 1));
  int i = __double2int_rd(ux), j = __double2int_rd(uy), k = __double2int_rd(uz);
  i = max(0, min(i, G.nx - 2)); j = max(0, min(j, G.ny - 2)); k = max(0, min(k, G.nz - 2));
  const double tx = ux - (double)i, ty = uy - (double)j, tz = uz - (double)k;
  double B[3] = {0.0, 0.0, 0.0};
  if (inbox) {
    const int base = (i * G.ny + j) * G.nz + k;
    const double x0 = 1.0 - tx, y0 = 1.0 - ty, z0 = 1.0 - tz;
    const double wxy[4] = {x0 * y0, x0 * ty, tx * y0, tx * ty};
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      const double w = wxy[q >> 1] * ((q & 1) ? tz : z0);
      const float4 v = __ldg(G.g4 + base + corner_offset(G, q));
      B[0] = fma(w, (double)v.x, B[0]); B[1] = fma(w, (double)v.y, B[1]); B[2] = fma(w, (double)v.z, B[2]);
    }
  }
  const double rho2 = fma(xd, xd, yd * yd);
  const double rho = rho2 * rsqrt_d(rho2);
  const double xs[2] = {D.k_hez * fabs(zd), D.k_her * rho};
  double o[2];
  exp2_d_n<2>(xs, o);
  const double de = 1.0 + o[0];
  ne = D.ne0x4 * o[1] * o[0] * rcp_d(de * de);
  N0 = n0_f32(P, (float)rho2, (float)zd);
  Bpar = B[0] * (dir.z * dir.x) + B[1] * (dir.z * dir.y) + B[2] * dir.w;
  BN = B[2] * dir.z - dir.w * (B[0] * dir.x + B[1] * dir.y);
  BE = B[1] * dir.x - B[0] * dir.y;
}

__device__ __forceinline__ double warp_inclusive_scan_d(double v, int lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const double o = shfl_up_d(v, d, 32);
    if (lane >= d) v += o;
  }
  return v;
}
__device__ __forceinline__ double warp_bcast_d(double v, int src) {
  int lo = __double2loint(v), hi = __double2hiint(v);
  lo = __shfl_sync(0xffffffffu, lo, src); hi = __shfl_sync(0xffffffffu, hi, src);
  return __hiloint2double(hi, lo);
}

struct GridFwdArgs {
  ForwardArgs f;
  GridDesc grid;
  int mode;            // 0 auto, 1 fp32 chain only, 2 float64 Faraday chain for every sightline
};

// Samples n_lo <= n < n_hi of a sightline that can lie inside the grid box -- a conservative superset (slab
// intersection of the ray with the box in float64, one sample of margin at either end); the exact per-sample box test
// stays in the sweeps.  Outside the box B = 0: such a sample adds nothing to I, Q, U, the Faraday depth or any
// cotangent, so the sweeps skip the tiles before n_lo and after n_hi (cfg 3: the 40 x 40 x 8 kpc box holds less than
// half of the samples of the 20-kpc sightlines).  Warp-uniform.
__device__ __forceinline__ void box_sample_range(const GridDesc& G, const Geometry& geo, const Triad& T, int& n_lo, int& n_hi) {
  // in units of samples: s / delta (reciprocals by rcp_d, ~1e-12 relative: far inside the one-sample margin)
  const double inv_delta = rcp_d(geo.delta * T.scale);
  double u_in = 0.0, u_out = (double)geo.n_los;
  const double dir[3] = {T.nxd, T.nyd, T.nzd};
  const double half[3] = {G.hx, G.hy, G.hz};
  bool empty = false;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double o = geo.obs[a];
    if (fabs(dir[a]) > 1.0e-200) {
      const double inv = rcp_d(dir[a]) * inv_delta;
      const double t1 = (-half[a] - o) * inv, t2 = (half[a] - o) * inv;
      u_in = fmax(u_in, fmin(t1, t2));
      u_out = fmin(u_out, fmax(t1, t2));
    } else if (fabs(o) > half[a]) {
      empty = true;
    }
  }
  if (empty || !(u_out >= u_in)) { n_lo = 0; n_hi = 0; return; }
  n_lo = max(0, __double2int_rd(u_in - 0.5) - 1);
  n_hi = min(geo.n_los, __double2int_ru(u_out - 0.5) + 2);
  if (n_hi < n_lo) n_hi = n_lo;
}

// Round-off scale of a sightline's Faraday sum, k-independent part: sum_n |n_e| (|B_LOS| + |B_N| + |B_E|),
// estimated with the fp32 chain from 32 samples spread over the in-box range [n_lo, n_hi), B taken at the NEAREST node
// (one gather per sample: with the lanes in 32 different cells a trilinear gather costs 8 x 32 L1 wavefronts).  It only
// routes the sightline -- the fp32 sweep checks the exact sum afterwards.  Whole warp; the same value in every lane.
template <bool SG>
__device__ __forceinline__ float grid_roundoff_estimate(const GridDesc& G, const BatchConsts& P, const Triad& T,
                                                        const Geometry& geo, const ScalarGridDesc& sg_ne, int lane,
                                                        int n_lo, int n_hi) {
  const int stride = (n_hi - n_lo + 31) >> 5;
  const int n = n_lo + lane * stride + (stride >> 1);
  float acc = 0.f;
  if (n < n_hi) {
    const double s_d = ((double)n + 0.5) * geo.delta * T.scale;
    const double xd = fma(s_d, T.nxd, geo.obs[0]), yd = fma(s_d, T.nyd, geo.obs[1]), zd = fma(s_d, T.nzd, geo.obs[2]);
    const double ux = fma(xd, G.sx, G.bx), uy = fma(yd, G.sy, G.by), uz = fma(zd, G.sz, G.bz);
    const int i = __double2int_rn(ux), j = __double2int_rn(uy), k = __double2int_rn(uz);
    if (i >= 0 && i < G.nx && j >= 0 && j < G.ny && k >= 0 && k < G.nz) {
      const float4 B = __ldg(G.g4 + (i * G.ny + j) * G.nz + k);
      float N0, ne;
      densities_f32(P, (float)fma(xd, xd, yd * yd), (float)zd, N0, ne);
      if (SG && sg_ne.g) ne = scalar_grid_at<float>(sg_ne, xd, yd, zd);
      const float Bpar = fmaf(B.x, T.nx, fmaf(B.y, T.ny, B.z * T.nz));
      const float BN = fmaf(B.x, T.eNx, fmaf(B.y, T.eNy, B.z * T.eNz));
      const float BE = fmaf(B.x, T.eEx, B.y * T.eEy);
      acc = fabsf(ne) * (fabsf(Bpar) + fabsf(BN) + fabsf(BE));
    }
  }
  return (float)stride * T.scalef * group_sum<32>(acc);
}

// One sightline, whole warp, lanes on CONSECUTIVE samples (neighbouring lanes gather neighbouring cells).
// PRECISE = float64 trilinear weights / n_e / scan.  Returns the (exact, not estimated) round-off scale.
template <int NF, bool PRECISE, bool SG>
__device__ __forceinline__ float grid_forward_sweep(const ForwardArgs& A, const GridDesc& G, const FreqTab& ft,
                                                    const BatchConsts& P, const BatchConstsD& D, const Triad& T,
                                                    const double4 dir, int lane, int n_lo, int n_hi, float& accI,
                                                    float (&accQ)[NF], float (&accU)[NF]) {
  accI = 0.f;
#pragma unroll
  for (int f = 0; f < NF; ++f) { accQ[f] = 0.f; accU[f] = 0.f; }
  double carry = 0.0;
  float absS = 0.f;
  const double delta = A.geo.delta * T.scale;
  for (int nt = n_lo & ~31; nt < n_hi; nt += 32) {
    const int n = nt + lane;
    const bool active = n < A.geo.n_los;
    const double s_d = ((double)n + 0.5) * delta;
    const double xd = fma(s_d, T.nxd, A.geo.obs[0]);
    const double yd = fma(s_d, T.nyd, A.geo.obs[1]);
    const double zd = fma(s_d, T.nzd, A.geo.obs[2]);
    float eI = 0.f, a = 0.f, bq = 0.f;
    double S_here;  // sum_{m<n} g_m + g_n/2 relative to the start of the sightline
    if (!PRECISE) {
      const Cell c = locate(G, xd, yd, zd);
      float B[3];
      gather_B(G, c, B);
      float N0, ne;
      densities_f32(P, (float)fma(xd, xd, yd * yd), (float)zd, N0, ne);
      if (SG && A.sg_ne.g) ne = scalar_grid_at<float>(A.sg_ne, xd, yd, zd);
      if (SG && A.sg_n0.g) N0 = scalar_grid_at<float>(A.sg_n0, xd, yd, zd);
      ne *= T.scalef;
      const float Bpar = fmaf(B[0], T.nx, fmaf(B[1], T.ny, B[2] * T.nz));
      const float BN = fmaf(B[0], T.eNx, fmaf(B[1], T.eNy, B[2] * T.eNz));
      const float BE = fmaf(B[0], T.eEx, B[1] * T.eEy);
      if (active) emission(P, BN, BE, N0, eI, a, bq);
      const float gn = active ? ne * Bpar : 0.f;
      if (active) absS = fmaf(fabsf(ne), fabsf(Bpar) + fabsf(BN) + fabsf(BE), absS);
      const float incl = warp_inclusive_scan(gn, lane);
      S_here = carry + (double)(incl - 0.5f * gn);
      carry += (double)__shfl_sync(0xffffffffu, incl, 31);   // the tile's fp32 sum, as the lanes saw it
    } else {
      double Bpar, BN, BE, ne;
      float N0;
      fields_f64(G, P, D, dir, xd, yd, zd, Bpar, BN, BE, N0, ne);
      if (SG && A.sg_ne.g) ne = scalar_grid_at<double>(A.sg_ne, xd, yd, zd);
      if (SG && A.sg_n0.g) N0 = scalar_grid_at<float>(A.sg_n0, xd, yd, zd);
      ne *= T.scale;
      if (active) emission(P, (float)BN, (float)BE, N0, eI, a, bq);
      const double gn = active ? ne * Bpar : 0.0;
      const double incl = warp_inclusive_scan_d(gn, lane);
      S_here = carry + incl - 0.5 * gn;
      carry += warp_bcast_d(incl, 31);
    }
    accI += eI;
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      float c, s;
      faraday_sincos(ft.k_turn[f], S_here, c, s);
      accQ[f] = fmaf(a, c, fmaf(-bq, s, accQ[f]));
      accU[f] = fmaf(a, s, fmaf(bq, c, accU[f]));
    }
  }
  accI = group_sum<32>(accI);
#pragma unroll
  for (int f = 0; f < NF; ++f) { accQ[f] = group_sum<32>(accQ[f]); accU[f] = group_sum<32>(accU[f]); }
  return group_sum<32>(absS);
}

// ------------------------------------------------------------------------------------------------
// Forward: persistent warps striding over sightlines.  Per sightline (warp-uniform): a cheap estimate of the
// round-off scale from every 8th sample sends it straight to the float64 chain when the Faraday rotation is
// strong; otherwise the fp32 sweep runs and is redone in float64 only if its exact criterion fires.
// ------------------------------------------------------------------------------------------------
template <int NF, bool SG>
__global__ void __launch_bounds__(kBlock) grid_forward_kernel(const __grid_constant__ GridFwdArgs GA,
                                                              const __grid_constant__ FreqTab ft) {
  const ForwardArgs& A = GA.f;
  const GridDesc& G = GA.grid;
  const int lane = threadIdx.x & 31;
  const int64_t warp = ((int64_t)blockIdx.x * kBlock + threadIdx.x) >> 5;
  const int64_t n_warps = ((int64_t)gridDim.x * kBlock) >> 5;
  const BatchConsts& P = A.bc[0];
  const BatchConstsD D = A.bd[0];
  for (int64_t pix = warp; pix < A.geo.npix; pix += n_warps) {
    const double4 dir = *reinterpret_cast<const double4*>(A.geo.dirs + 4 * pix);
    const Triad T = load_triad(A.geo, pix);
    float accI, accQ[NF], accU[NF];
    int n_lo, n_hi;   // the samples that can lie inside the box
    box_sample_range(G, A.geo, T, n_lo, n_hi);
    bool precise = GA.mode == 2;
    if (GA.mode == 0) precise = grid_roundoff_estimate<SG>(G, P, T, A.geo, A.sg_ne, lane, n_lo, n_hi) > A.flag_S;
    if (!precise) {
      const float scale = grid_forward_sweep<NF, false, SG>(A, G, ft, P, D, T, dir, lane, n_lo, n_hi, accI, accQ, accU);
      precise = GA.mode == 0 && scale > A.flag_S;
    }
    if (precise) grid_forward_sweep<NF, true, SG>(A, G, ft, P, D, T, dir, lane, n_lo, n_hi, accI, accQ, accU);
    if (lane == 0) {
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        const int64_t o = (int64_t)(A.f0 + f) * A.geo.npix + pix;
        A.I[o] = P.coefI[A.f0 + f] * T.scalef * accI;
        A.Q[o] = P.coefP[A.f0 + f] * T.scalef * accQ[f];
        A.U[o] = P.coefP[A.f0 + f] * T.scalef * accU[f];
      }
      if (precise && GA.mode == 0 && A.f0 == 0) atomicAdd(A.flag_count, 1);
    }
  }
}

// red.global.add of (a, b, c, 0) to a 16-byte aligned node {gx, gy, gz, pad} (sm_90+ vector reduction)
__device__ __forceinline__ void red_add_v4(float* p, float a, float b, float c) {
  asm volatile("red.global.v4.f32.add [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(0.0f) : "memory");
}

// caller's [node][3] grid -> padded fp32 nodes
__global__ void grid_pack_kernel(const float* __restrict__ g, int64_t n_nodes, float4* __restrict__ g4) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_nodes) return;
  const float x = g[3 * i], y = g[3 * i + 1], z = g[3 * i + 2];
  g4[i] = make_float4(x, y, z, 0.f);
}

// [n][4] accumulation buffer -> caller's [n][3] gradient
__global__ void grid_grad_compact_kernel(const float4* __restrict__ g4, int64_t n_nodes, float* __restrict__ grad) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_nodes) return;
  const float4 v = g4[i];
  grad[3 * i] = v.x; grad[3 * i + 1] = v.y; grad[3 * i + 2] = v.z;
}

// ------------------------------------------------------------------------------------------------
// Adjoint.  grad_grid must be zero on entry (the host wrapper clears it).
// Dynamic shared memory: 3 float arrays of 32*(C+1) per warp, C = chunk length (power of two).
// ------------------------------------------------------------------------------------------------
constexpr int kGridGroup = kBlock / 32;   // grid_vjp_kernel: neighbouring pixels taken together (the warps of a CTA)
struct GridVjpArgs {
  Geometry geo;
  ScalarGridDesc sg_ne, sg_n0;
  const BatchConsts* bc;
  const BatchConstsD* bd;
  GridDesc grid;
  int f0, n_freq_total;
  const float* dI; const float* dQ; const float* dU;
  float* grad4;         // internal accumulation buffer [nx][ny][nz][4] (16-byte nodes), zero on entry
  int chunk_log2;       // C = 1 << chunk_log2, 32*C >= n_los
  int mode;             // 0 auto, 1 fp32 chain, 2 float64 Faraday chain
  float flag_S;         // auto: redo a sightline in float64 when max |sum n_e B_LOS| exceeds this
  int64_t n_groups;     // ceil(npix / kGridGroup): groups of neighbouring pixels, one per CTA pass
  unsigned long long* ticket;   // zero on entry: next index of the permuted sequence
  int64_t group_stride; // coprime to n_groups, ~0.618 n_groups: the order in which the groups are taken (grid_vjp_kernel)
};

// Sweep 2's per-lane accumulators: the 8 x 3 corner contributions of the cell the lane is in.  A ray leaves a cell
// through a face, and the 4 nodes of that face belong to the next cell too: only the 4 nodes left behind are
// flushed (red.global.add), the shared ones stay in their registers.  So that nothing has to move, the registers
// are addressed in "slot" coordinates: slot bit s of an axis means corner bit s ^ flip of that axis, and crossing a
// face toggles the axis' flip (the kept registers were the far face of the old cell and are the near face of the new
// one).  The trilinear weights follow by using 1 - t for a flipped axis.
struct CornerAcc {
  float acc[24];        // [slot q = (sa << 2) | (sb << 1) | sd][component]
  int ci, cj, ck;       // the cell
  int flip;             // bit 2: x, bit 1: y, bit 0: z
  bool valid;           // in a cell (acc may be non-zero)
};

// node index of slot q of the current cell
__device__ __forceinline__ int slot_node(const GridDesc& G, const CornerAcc& S, int q) {
  const int a = ((q >> 2) ^ (S.flip >> 2)) & 1, b = ((q >> 1) ^ (S.flip >> 1)) & 1, d = (q ^ S.flip) & 1;
  return ((S.ci + a) * G.ny + (S.cj + b)) * G.nz + (S.ck + d);
}

// flush (and clear) the slots whose bit of axis AX (2: x, 1: y, 0: z) equals h
template <int AX>
__device__ __forceinline__ void flush_half(const GridDesc& G, float* grad4, CornerAcc& S, int h) {
  if (h == 0) {
#pragma unroll
    for (int q = 0; q < 8; ++q)
      if (((q >> AX) & 1) == 0) {
        red_add_v4(grad4 + (size_t)slot_node(G, S, q) * 4, S.acc[3 * q], S.acc[3 * q + 1], S.acc[3 * q + 2]);
        S.acc[3 * q] = 0.f; S.acc[3 * q + 1] = 0.f; S.acc[3 * q + 2] = 0.f;
      }
  } else {
#pragma unroll
    for (int q = 0; q < 8; ++q)
      if (((q >> AX) & 1) == 1) {
        red_add_v4(grad4 + (size_t)slot_node(G, S, q) * 4, S.acc[3 * q], S.acc[3 * q + 1], S.acc[3 * q + 2]);
        S.acc[3 * q] = 0.f; S.acc[3 * q + 1] = 0.f; S.acc[3 * q + 2] = 0.f;
      }
  }
}

// step to the neighbouring cell across the face of axis AX, `wd` = +1 or -1 cells
template <int AX>
__device__ __forceinline__ void cross_face(const GridDesc& G, float* grad4, CornerAcc& S, int wd) {
  const int leave = wd > 0 ? 0 : 1;                       // corner bit of the face left behind
  flush_half<AX>(G, grad4, S, leave ^ ((S.flip >> AX) & 1));
  S.flip ^= 1 << AX;
  if (AX == 2) S.ci += wd; else if (AX == 1) S.cj += wd; else S.ck += wd;
}

__device__ __forceinline__ void flush_all(const GridDesc& G, float* grad4, CornerAcc& S) {
#pragma unroll
  for (int q = 0; q < 8; ++q) {
    // one 16-byte vector reduction per corner node (measured 2.6x the throughput of three scalar reds)
    red_add_v4(grad4 + (size_t)slot_node(G, S, q) * 4, S.acc[3 * q], S.acc[3 * q + 1], S.acc[3 * q + 2]);
    S.acc[3 * q] = 0.f; S.acc[3 * q + 1] = 0.f; S.acc[3 * q + 2] = 0.f;
  }
}

// Sweep 1 of the gridded adjoint for one sightline (whole warp): per-sample forward quantities, cotangent
// fan-out (A9) and the per-sample hand-over to sweep 2 through shared memory.  Returns sum n_e (|B_LOS| + |B_N| + |B_E|).
template <int NF, bool PRECISE, bool SG>
__device__ __forceinline__ float grid_vjp_sweep1(const GridVjpArgs& A, const FreqTab& ft, const GridDesc& G,
                                                 const BatchConsts& P, const BatchConstsD& D, const Triad& T,
                                                 const double4 dir, int lane,
                                                 float cI, const float (&cQ)[NF], const float (&cU)[NF],
                                                 const float (&kr)[NF], int n_lo, int n_hi, int cl2,
                                                 float* st_w, float* st_n, float* st_e) {
  const int C = 1 << cl2, Cp = C + 1;   // this sightline's chunk length: 32 C >= n_hi - n_lo
  const double delta = A.geo.delta * T.scale;
  double carry = 0.0;
  float absS = 0.f;
  for (int nt = n_lo; nt < n_hi; nt += 32) {
    const int n = nt + lane;
    const bool active = n < n_hi;
    const double s_d = ((double)n + 0.5) * delta;
    const double xd = fma(s_d, T.nxd, A.geo.obs[0]);
    const double yd = fma(s_d, T.nyd, A.geo.obs[1]);
    const double zd = fma(s_d, T.nzd, A.geo.obs[2]);
    float BN, BE, N0, ne;
    double S_here;
    if (!PRECISE) {
      const Cell c = locate(G, xd, yd, zd);
      float B[3];
      gather_B(G, c, B);
      densities_f32(P, (float)fma(xd, xd, yd * yd), (float)zd, N0, ne);
      if (SG && A.sg_ne.g) ne = scalar_grid_at<float>(A.sg_ne, xd, yd, zd);
      if (SG && A.sg_n0.g) N0 = scalar_grid_at<float>(A.sg_n0, xd, yd, zd);
      ne *= T.scalef;
      const float Bpar = fmaf(B[0], T.nx, fmaf(B[1], T.ny, B[2] * T.nz));
      BN = fmaf(B[0], T.eNx, fmaf(B[1], T.eNy, B[2] * T.eNz));
      BE = fmaf(B[0], T.eEx, B[1] * T.eEy);
      const float gn = active ? ne * Bpar : 0.f;
      if (active) absS = fmaf(fabsf(ne), fabsf(Bpar) + fabsf(BN) + fabsf(BE), absS);
      const float incl = warp_inclusive_scan(gn, lane);
      S_here = carry + (double)(incl - 0.5f * gn);
      carry += (double)__shfl_sync(0xffffffffu, incl, 31);
    } else {
      double Bpar, BNd, BEd, ned;
      fields_f64(G, P, D, dir, xd, yd, zd, Bpar, BNd, BEd, N0, ned);
      if (SG && A.sg_ne.g) ned = scalar_grid_at<double>(A.sg_ne, xd, yd, zd);
      if (SG && A.sg_n0.g) N0 = scalar_grid_at<float>(A.sg_n0, xd, yd, zd);
      ned *= T.scale;
      BN = (float)BNd; BE = (float)BEd; ne = (float)ned;
      const double gn = active ? ned * Bpar : 0.0;
      const double incl = warp_inclusive_scan_d(gn, lane);
      S_here = carry + incl - 0.5 * gn;
      carry += warp_bcast_d(incl, 31);
    }
    const float bn2 = BN * BN, be2 = BE * BE, Bt2 = bn2 + be2;
    float w = 1.0f;
    if (!P.alpha_is_3) w = (Bt2 > 0.f) ? mufu_ex2(P.q_exp * mufu_lg2(Bt2)) : 0.f;
    const float M = active ? w * N0 : 0.f;
    const float d2 = be2 - bn2, p2 = 2.0f * BE * BN;
    float Xc = 0.f, Xs = 0.f, Yc = 0.f, Ys = 0.f;
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      float cc, ss;
      faraday_sincos(ft.k_turn[f], S_here, cc, ss);
      const float u = fmaf(cQ[f], cc, cU[f] * ss);
      const float v = fmaf(cU[f], cc, -cQ[f] * ss);
      Xc += u; Xs += v;
      Yc = fmaf(kr[f], u, Yc); Ys = fmaf(kr[f], v, Ys);
    }
    const float K = fmaf(cI, Bt2, fmaf(Xc, d2, Xs * p2));
    const float MK = M * K;
    const float Sbar = M * fmaf(d2, Ys, -p2 * Yc);   // cotangent of this sample's Faraday sum
    const float tq_ = (Bt2 > 0.f) ? P.q_exp * MK / Bt2 : 0.f;
    const float BEb = 2.0f * fmaf(M, fmaf(BE, cI + Xc, BN * Xs), BE * tq_);
    const float BNb = 2.0f * fmaf(M, fmaf(BN, cI - Xc, BE * Xs), BN * tq_);
    if (active) {
      const int idx = ((n - n_lo) >> cl2) * Cp + ((n - n_lo) & (C - 1));
      st_w[idx] = Sbar; st_n[idx] = BNb; st_e[idx] = BEb;
    }
  }
  return group_sum<32>(absS);
}

template <int NF, bool SG>
// (one frequency: a sixth CTA per SM for 8 bytes of spill, 0.535 -> 0.525 ms at cfg 3; no gain with 4 or 8 frequencies)
__global__ void __launch_bounds__(kBlock, NF == 1 ? 6 : 5) grid_vjp_kernel(const __grid_constant__ GridVjpArgs A,
                                                          const __grid_constant__ FreqTab ft) {
  extern __shared__ float smem[];
  const GridDesc& G = A.grid;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int C = 1 << A.chunk_log2, Cp = C + 1;
  float* st_w = smem + (size_t)wid * 3 * 32 * Cp;   // Sbar_m: cotangent of the Faraday sum at sample m
  float* st_n = st_w + 32 * Cp;                     // BbarN (direct)
  float* st_e = st_n + 32 * Cp;                     // BbarE (direct)
  const int64_t warp = ((int64_t)blockIdx.x * kBlock + threadIdx.x) >> 5;
  const int64_t n_warps = ((int64_t)gridDim.x * kBlock) >> 5;
  const BatchConsts& P = A.bc[0];
  const BatchConstsD D = A.bd[0];
  // Sightline order: the warps of a CTA take neighbouring pixels (their gathers share L1 lines), but the CTAs that run at the
  // same time are spread over the sky -- group q of kBlock / 32 pixels is the (q * group_stride mod n_groups)-th of the map
  // (group_stride coprime to n_groups: a permutation).  In pixel order the ~3,000 sightlines in flight cross the same cells
  // at the same time and their red.global.add to the same nodes queue up in L2 (cfg 3: 0.67 -> 0.545 ms).
  constexpr int64_t kW = kGridGroup;
  for (;;) {
    // the next sightline of that sequence goes to whichever warp is free (costs differ: in-box length, fp32 or float64
    // chain): 0.545 -> 0.536 ms
    unsigned long long tk = 0;
    if (lane == 0) tk = atomicAdd(A.ticket, 1ULL);
    const int64_t pidx = (int64_t)__shfl_sync(0xffffffffu, tk, 0);
    if (pidx >= A.n_groups * kW) break;
    const int64_t pix = (((pidx / kW) * A.group_stride) % A.n_groups) * kW + pidx % kW;
    if (pix >= A.geo.npix) continue;   // the last group of a map whose size is no multiple of kW (warp-uniform)
    const Triad T = load_triad(A.geo, pix);
    const double delta = A.geo.delta * T.scale;
    const double4 dir = *reinterpret_cast<const double4*>(A.geo.dirs + 4 * pix);
    float cI = 0.f, cQ[NF], cU[NF], kr[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const int64_t o = (int64_t)(A.f0 + f) * A.geo.npix + pix;
      cI = fmaf(A.dI ? __ldg(A.dI + o) : 0.f, P.coefI[A.f0 + f] * T.scalef, cI);
      cQ[f] = (A.dQ ? __ldg(A.dQ + o) : 0.f) * P.coefP[A.f0 + f] * T.scalef;
      cU[f] = (A.dU ? __ldg(A.dU + o) : 0.f) * P.coefP[A.f0 + f] * T.scalef;
      kr[f] = ft.k_rad[f];
    }
    // ---- sweep 1: consecutive samples per lane; fp32 chain first, redone with the float64 Faraday chain
    // when the rotation angle of this sightline is large (warp-uniform decision)
    // the samples that can lie inside the box (the others add nothing to the gradient), cut into 32 chunks of
    // C2 = 2^cl2 samples: the layout of the hand-over and of sweep 2's lanes
    int n_lo, n_hi;
    box_sample_range(G, A.geo, T, n_lo, n_hi);
    int cl2 = 0;
    while ((32 << cl2) < n_hi - n_lo) ++cl2;
    float absS = 0.f;
    bool precise = A.mode == 2;
    if (A.mode == 0) precise = grid_roundoff_estimate<SG>(G, P, T, A.geo, A.sg_ne, lane, n_lo, n_hi) > A.flag_S;
    if (!precise) absS = grid_vjp_sweep1<NF, false, SG>(A, ft, G, P, D, T, dir, lane, cI, cQ, cU, kr, n_lo, n_hi, cl2, st_w, st_n, st_e);
    if (precise || (A.mode == 0 && absS > A.flag_S)) {
      __syncwarp();
      grid_vjp_sweep1<NF, true, SG>(A, ft, G, P, D, T, dir, lane, cI, cQ, cU, kr, n_lo, n_hi, cl2, st_w, st_n, st_e);
    }
    __syncwarp();
    // ---- sweep 2: contiguous chunk per lane walked BACKWARDS, so that the suffix sum of Sbar that the
    // transposed half-cell scan needs (gbar_m = sum_{n>m} Sbar_n + Sbar_m / 2) is a running sum with no
    // cancellation; register accumulation per cell, red.global.add only when the cell changes.
    const int C2 = 1 << cl2, Cq = C2 + 1;
    const int mb = n_lo + (lane << cl2);                // this lane's chunk [mb, mb + C2) of the in-box range
    const int m0 = min(mb, n_hi), m1 = min(mb + C2, n_hi);
    float tot = 0.f;
    for (int m = m0; m < m1; ++m) tot += st_w[lane * Cq + (m - mb)];
    float incl = tot;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const float o = __shfl_down_sync(0xffffffffu, incl, d);
      if (lane + d < 32) incl += o;
    }
    float suf = incl - tot;      // sum of Sbar over all later lanes
    CornerAcc S;
#pragma unroll
    for (int q = 0; q < 24; ++q) S.acc[q] = 0.f;
    S.ci = S.cj = S.ck = 0; S.flip = 0; S.valid = false;
    // walking backwards along the sightline the cell indices move against the direction (warp-uniform)
    const int wdx = T.nxd > 0.0 ? -1 : 1, wdy = T.nyd > 0.0 ? -1 : 1, wdz = T.nzd > 0.0 ? -1 : 1;
    for (int m = m1 - 1; m >= m0 - 1; --m) {
      Cell c; c.base = -1; c.i = c.j = c.k = 0; c.inbox = false; c.tx = c.ty = c.tz = 0.f;
      float ne_m = 0.f;   // recomputed (fp32, 4 MUFU) rather than handed over: 25 % less shared memory per warp
      if (m >= m0) {
        const double s_d = ((double)m + 0.5) * delta;
        const double xd = fma(s_d, T.nxd, A.geo.obs[0]), yd = fma(s_d, T.nyd, A.geo.obs[1]), zd = fma(s_d, T.nzd, A.geo.obs[2]);
        c = locate(G, xd, yd, zd);
        float N0_unused;
        densities_f32(P, (float)fma(xd, xd, yd * yd), (float)zd, N0_unused, ne_m);
        if (SG && A.sg_ne.g) ne_m = scalar_grid_at<float>(A.sg_ne, xd, yd, zd);
        ne_m *= T.scalef;
      }
      const bool have = m >= m0 && c.inbox;
      if (S.valid) {
        const int di = c.i - S.ci, dj = c.j - S.cj, dk = c.k - S.ck;
        if (!have || (di != 0 && di != wdx) || (dj != 0 && dj != wdy) || (dk != 0 && dk != wdz)) {
          flush_all(G, A.grad4, S);      // end of the chunk, out of the box, or not a face neighbour
          S.valid = false;
        } else {
          if (di != 0) cross_face<2>(G, A.grad4, S, wdx);
          if (dj != 0) cross_face<1>(G, A.grad4, S, wdy);
          if (dk != 0) cross_face<0>(G, A.grad4, S, wdz);
        }
      }
      if (have && !S.valid) { S.ci = c.i; S.cj = c.j; S.ck = c.k; S.valid = true; }
      if (m >= m0) {
        const int idx = lane * Cq + (m - mb);
        const float Sb = st_w[idx];
        const float gbar = fmaf(0.5f, Sb, suf);
        suf += Sb;
        if (have) {
          const float BNb = st_n[idx], BEb = st_e[idx], gn = gbar * ne_m;
          const float bx = fmaf(BNb, T.eNx, fmaf(BEb, T.eEx, gn * T.nx));
          const float by = fmaf(BNb, T.eNy, fmaf(BEb, T.eEy, gn * T.ny));
          const float bz = fmaf(BNb, T.eNz, gn * T.nz);
          Cell cs = c;   // weights in slot coordinates
          if (S.flip & 4) cs.tx = 1.0f - c.tx;
          if (S.flip & 2) cs.ty = 1.0f - c.ty;
          if (S.flip & 1) cs.tz = 1.0f - c.tz;
          float w[8];
          weights(cs, w);
#pragma unroll
          for (int q = 0; q < 8; ++q) {
            S.acc[3 * q] = fmaf(w[q], bx, S.acc[3 * q]);
            S.acc[3 * q + 1] = fmaf(w[q], by, S.acc[3 * q + 1]);
            S.acc[3 * q + 2] = fmaf(w[q], bz, S.acc[3 * q + 2]);
          }
        }
      }
    }
    __syncwarp();
  }
}

}  // namespace synax
