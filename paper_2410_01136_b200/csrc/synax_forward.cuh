// synax_forward.cuh -- plan geometry kernel (A1), per-batch prologue, forward kernels (A2-A8, A12).
#pragma once
#include "synax_device.cuh"
#include "synax_f64.cuh"

namespace synax {

constexpr int kBlock = 128;   // threads per CTA for the sightline kernels
constexpr int kTile = 32;     // samples between re-basing of the local Faraday sum
constexpr int kTileDMax = 16;  // float64-chain kernel: at most this many samples per tile (BatchConsts::tile_d)
#ifndef SYNAX_UNROLL_D
#define SYNAX_UNROLL_D 1
#endif
constexpr int kUnrollD = SYNAX_UNROLL_D;  // ... samples advanced in lockstep per iteration
constexpr float kTilePhase = 96.0f;  // ... and at most about this much Faraday angle (rad) inside a tile

enum ModelCode { kAnalyticDisc = 0, kAnalyticFull = 1, kGridB = 2, kUniform = 3, kStack16 = 4 };

// ------------------------------------------------------------------------------------------------
// small warp helpers over groups of G lanes (G = 1, 2, 4, ..., 32; groups are aligned)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double shfl_up_d(double v, int d, int width) {
  int lo = __double2loint(v), hi = __double2hiint(v);
  lo = __shfl_up_sync(0xffffffffu, lo, d, width);
  hi = __shfl_up_sync(0xffffffffu, hi, d, width);
  return __hiloint2double(hi, lo);
}

// exclusive prefix sum over the G lanes of a group
template <int G>
__device__ __forceinline__ double group_exclusive_scan(double v, int g) {
  double incl = v;
#pragma unroll
  for (int d = 1; d < G; d <<= 1) {
    const double o = shfl_up_d(incl, d, G);
    if (g >= d) incl += o;
  }
  return incl - v;
}

template <int G>
__device__ __forceinline__ float group_sum(float v) {
#pragma unroll
  for (int d = G / 2; d >= 1; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d, G);
  return v;
}
template <int G>
__device__ __forceinline__ double group_sum_d(double v) {
#pragma unroll
  for (int d = G / 2; d >= 1; d >>= 1) {
    int lo = __double2loint(v), hi = __double2hiint(v);
    lo = __shfl_xor_sync(0xffffffffu, lo, d, G); hi = __shfl_xor_sync(0xffffffffu, hi, d, G);
    v += __hiloint2double(hi, lo);
  }
  return v;
}
template <int G>
__device__ __forceinline__ float group_max(float v) {
#pragma unroll
  for (int d = G / 2; d >= 1; d >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, d, G));
  return v;
}

// rotate (q,u) by the Faraday angle of a float64 offset: turns reduced in float64 (never form a
// large angle in fp32), sin/cos of the reduced angle on the MUFU.
__device__ __forceinline__ void rotate_by_offset(double k_turn, double S, float& q, float& u) {
  double t = k_turn * S;
  t -= rint(t);
  const float a = (float)t * 6.283185307179586f;
  const float c = mufu_cos(a), s = mufu_sin(a);
  const float q2 = q * c - u * s;
  u = fmaf(q, s, u * c);
  q = q2;
}

// emission terms of one sample (A5): e~ = N0 (B_perp^2)^((alpha+1)/4), and e~ e^{2 i chi0}
// = N0 (B_perp^2)^((alpha-3)/4) (B_E + i B_N)^2  -- no atan2, no division (S:C-2#19 for B_perp = 0).
__device__ __forceinline__ void emission(const BatchConsts& P, float BN, float BE, float N0, float& eI,
                                         float& a, float& b) {
  const float bn2 = BN * BN, be2 = BE * BE;
  const float Bt2 = bn2 + be2;
  float w = N0;
  if (!P.alpha_is_3) w = (Bt2 > 0.0f) ? N0 * mufu_ex2(P.q_exp * mufu_lg2(Bt2)) : 0.0f;
  eI = w * Bt2;
  a = w * (be2 - bn2);
  b = w * (2.0f * BE * BN);
}

// ------------------------------------------------------------------------------------------------
// Forward, fp32 fast chain.  G lanes per sightline, each lane owns a contiguous chunk of samples
// (no per-sample scan: each lane integrates with a chunk-local Faraday depth and its partial Q+iU
// is rotated once by the float64 offset of the preceding lanes).  NF frequencies per pass.
// ------------------------------------------------------------------------------------------------
// Sample positions for the fp32 field chain, evaluated in fp32 on their own: s = s0 + n Delta_i from an exactly represented
// sample counter, then one fused multiply-add per coordinate (error ~2 ulp of the coordinate, the accuracy class of the
// rest of that chain).  The float64 positions are still formed for the decisions (annulus / box tests) and the float64
// chain, but are no longer CONVERTED per sample: four F2F.F32.F64 were 10 % of the XU-pipe work of the fp32 kernels,
// which are bound by that pipe (ncu: XU 86 % in the fp32 forward).
struct PosF {
  float s0, dlt, nf;
  __device__ __forceinline__ void init(double delta, int n_first) {
    s0 = (float)(((double)n_first + 0.5) * delta); dlt = (float)delta; nf = 0.f;
  }
  // position of the current sample, then step by `dir` samples (+1 forward sweeps, -1 backward sweeps)
  __device__ __forceinline__ void next(const Geometry& geo, const Triad& T, float dir, float& x, float& y, float& z, float& rho2) {
    const float sf = fmaf(nf, dlt, s0);
    nf += dir;
    x = fmaf(sf, T.nx, geo.obsf[0]); y = fmaf(sf, T.ny, geo.obsf[1]); z = fmaf(sf, T.nz, geo.obsf[2]);
    rho2 = fmaf(x, x, y * y);
  }
};

struct ForwardArgs {
  Geometry geo;
  const BatchConsts* bc;
  const BatchConstsD* bd; // float64 constants (float64 Faraday chain only)
  int batch;
  int f0;                 // first frequency of this pass
  float* I; float* Q; float* U;
  int n_freq_total;
  float flag_S;           // flag a sightline when max |sum n_e B_LOS| exceeds this (<=0: never)
  float flag_T;           // ... or when the Faraday sum inside one 32-sample tile of the fp32 chain exceeds this (<=0: never)
  int* flag_count;        // device counter
  int* flag_list;         // device list of flagged sightline ids (b * npix + p)
  ScalarGridDesc sg_ne, sg_n0;  // gridded n_e / N_0 replacing the analytic discs (DISC4, GRID_B), g == nullptr: unused
  const int* mode;        // device: kModeFastThenList / kModeAllF64 / kModeSplit (written by decide_kernel), or null
  int run_when;           // forward_f64_kernel: 0 always, 1 only in mode fast-then-list (flag list), 2 only in mode
                          // all-float64 (every sightline), 3 in both all-float64 (every sightline) and split (flag list),
                          // 4 only in mode split (flag list)
  int* append_count;      // where forward_kernel appends the sightlines its exact criterion flags: the flag list itself
  int* append_list;       // (fast-then-list), or a separate "missed" list in split mode, where the float64 kernel reads
                          // the flag list concurrently on the plan's second stream
  double* phi;            // [batch][npix]: every sightline's Faraday sum sum_n n_e B_LOS Delta_i / Delta, stored for the plan's
                          // next adjoint (which sweeps backwards and needs the total first), or null
  double* phi_base;       // [k][batch * npix], k = 1 .. ceil(n_los / 32) - 1: Faraday sum over the samples BEFORE sample 32 k, stored by
                          // the float64-chain kernel for its sightlines: the adjoint then runs fp32 tile-local angles on exact
                          // tile bases and needs no float64 chain of its own; phi_has[sl] = 1 marks those sightlines.  Or null.
  unsigned char* phi_has;
  int* list_u;            // kModeSplit: sightlines classify_kernel left to the fp32 kernel (count in ctrl[kCtrlCountU])
  const int* count_u;
};

// kModeSplit: classify_kernel sorts the sightlines by an estimate of the round-off scale into the flag list (float64
// chain) and list_u (fp32 kernel, whose exact criterion still appends what the estimate missed to the flag list).
enum { kModeFastThenList = 0, kModeAllF64 = 1, kModeSplit = 2 };
enum { kCtrlFlagCount = 0, kCtrlPilotFlagged = 1, kCtrlMode = 2, kCtrlCountU = 3, kCtrlCountM = 4, kCtrlWords = 8 };

// Estimate of one lane's share of the round-off scale  sum_n |n_e| (|B_LOS| + |B_N| + |B_E|)  over samples [n0, n1):
// every 16th sample (all of them for short chunks), MUFU-grade fp32 chain; the caller sums the lanes of the
// sightline and multiplies by Triad::scalef.
// kTileMax: also *tile_max = estimate of the largest |signed Faraday sum inside one 32-sample tile| (forward_kernel's second
// criterion, ForwardArgs::flag_T), from the same samples (its own instantiation: the bookkeeping costs the plain one 10 %).
template <int CODE, bool kTileMax = false>
__device__ __forceinline__ float roundoff_scale_estimate(const Geometry& geo, const BatchConsts& P, const Triad& T,
                                                         const ScalarGridDesc& sg_ne, int n0, int n1, float* tile_max = nullptr) {
  const int step = (n1 - n0 >= 32) ? 16 : 1;
  const double delta = geo.delta * T.scale;
  float est = 0.f;
  float tsum = 0.f, tmax = 0.f;
  int tcur = -1;
  for (int n = n0 + step / 2; n < n1; n += step) {
    const double s_e = ((double)n + 0.5) * delta;
    const double xd = fma(s_e, T.nxd, geo.obs[0]), yd = fma(s_e, T.nyd, geo.obs[1]), zd = fma(s_e, T.nzd, geo.obs[2]);
    SampleF S;
    if (CODE == kUniform) {
      S.Bpar = fabsf(P.uB[0]) + fabsf(P.uB[1]) + fabsf(P.uB[2]); S.BN = 0.f; S.BE = 0.f; S.ne = P.une;
    } else {
      const double rho2d = fma(xd, xd, yd * yd);
      const bool inside = (rho2d > 9.0) && (rho2d < 400.0);
      if (CODE == kStack16) {
        StackAux sa;
        eval_stack16_f32<true>(P, T, (float)xd, (float)yd, (float)zd, (float)rho2d, inside, S, sa);
      } else {
        AnalyticAux aux;
        eval_analytic_f32<CODE == kAnalyticFull, true>(P, T, (float)xd, (float)yd, (float)zd, (float)rho2d, inside, S, aux);
      }
      if ((CODE == kAnalyticDisc || CODE == kStack16) && sg_ne.g) S.ne = scalar_grid_at<float>(sg_ne, xd, yd, zd);
    }
    est = fmaf(fabsf(S.ne), fabsf(S.Bpar) + fabsf(S.BN) + fabsf(S.BE), est);
    if (kTileMax) {
      const int t = (n - n0) >> 5;
      if (t != tcur) { tmax = fmaxf(tmax, fabsf(tsum)); tsum = 0.f; tcur = t; }
      tsum = fmaf(S.ne, CODE == kUniform ? fmaf(P.uB[0], T.nx, fmaf(P.uB[1], T.ny, P.uB[2] * T.nz)) : S.Bpar, tsum);
    }
  }
  if (kTileMax) *tile_max = fmaxf(tmax, fabsf(tsum)) * (float)step;
  return est * (float)step;
}

// LIST = false: every sightline, runs in kModeFastThenList (or without a pilot); LIST = true: the sightlines of
// list_u, runs in kModeSplit.  (Two instantiations rather than a run-time switch: the switch put two more
// F2F conversions per sample into the loop of the NF = 1 kernel, +4 % at cfg 2.)
template <int CODE, int G, int NF, bool LIST>
__global__ void __launch_bounds__(kBlock) forward_kernel(const __grid_constant__ ForwardArgs A,
                                                         const __grid_constant__ FreqTab ft) {
  if (LIST ? (*A.mode != kModeSplit) : (A.mode && *A.mode != kModeFastThenList)) return;
  constexpr int NFA = NF > 0 ? NF : 1;   // NF = 0: the adjoint's Faraday-only pass (totals and flags, no maps)
  const int64_t tid = (int64_t)blockIdx.x * kBlock + threadIdx.x;
  const int g = (int)(tid % G);
  int64_t sl = tid / G;
  const int64_t n_sl = LIST ? (int64_t)(*A.count_u) : A.geo.npix * A.batch;
  if (LIST && sl - ((threadIdx.x & 31) / G) >= n_sl) return;   // the whole warp is past the end of the list
  const bool valid = sl < n_sl;
  if (!valid) sl = n_sl - 1;  // keep the lane alive for the shuffles
  if (LIST) sl = (int64_t)A.list_u[sl];
  const int b = (int)(sl / A.geo.npix);
  const int64_t pix = sl - (int64_t)b * A.geo.npix;
  const BatchConsts& P = A.bc[b];
  const Triad T = load_triad(A.geo, pix);

  const int C = (A.geo.n_los + G - 1) / G;
  const int n0 = g * C;
  const int n1 = min(n0 + C, A.geo.n_los);
  const double delta = A.geo.delta * T.scale;
  double s_d = ((double)n0 + 0.5) * delta;
  PosF pf;
  pf.init(delta, n0);

  float k_rad[NFA];
#pragma unroll
  for (int f = 0; f < NF; ++f) k_rad[f] = ft.k_rad[f];

  float accI = 0.0f, accQ[NFA], accU[NFA];
#pragma unroll
  for (int f = 0; f < NF; ++f) { accQ[f] = 0.0f; accU[f] = 0.0f; }
  double carry = 0.0;            // chunk-local sum of n_e B_LOS over finished tiles
  float gabs = 0.0f;             // sum n_e (|B_LOS| + |B_N| + |B_E|): scale of the fp32 round-off in the Faraday sum
  float tmax = 0.0f;             // largest |tile-local Faraday sum|: the fp32 rotation angle inside a tile is k_f times this

  for (int ts = n0; ts < n1; ts += kTile) {
    const int te = min(ts + kTile, n1);
    float hi = 0.0f, lo = 0.0f;  // tile-local two-float sum of n_e B_LOS
    float tq[NFA], tu[NFA];
#pragma unroll
    for (int f = 0; f < NF; ++f) { tq[f] = 0.0f; tu[f] = 0.0f; }
    for (int n = ts; n < te; ++n) {
      // A2: midpoint position in float64 (mask decisions), rounded once to fp32 for the fields
      const double xd = fma(s_d, T.nxd, A.geo.obs[0]);
      const double yd = fma(s_d, T.nyd, A.geo.obs[1]);
      const double zd = fma(s_d, T.nzd, A.geo.obs[2]);
      s_d += delta;
      float xf, yf, zf, rho2f;
      pf.next(A.geo, T, 1.0f, xf, yf, zf, rho2f);
      SampleF S;
      if (CODE == kUniform) {
        S.Bpar = fmaf(P.uB[0], T.nx, fmaf(P.uB[1], T.ny, P.uB[2] * T.nz));
        S.BN = fmaf(P.uB[0], T.eNx, fmaf(P.uB[1], T.eNy, P.uB[2] * T.eNz));
        S.BE = fmaf(P.uB[0], T.eEx, P.uB[1] * T.eEy);
        S.N0 = P.uN0; S.ne = P.une;
      } else if (CODE == kStack16) {
        const double rho2d = fma(xd, xd, yd * yd);
        StackAux sa;
        eval_stack16_f32<false>(P, T, xf, yf, zf, rho2f, (rho2d > 9.0) && (rho2d < 400.0), S, sa);
      } else {
        const double rho2d = fma(xd, xd, yd * yd);
        const bool inside = (rho2d > 9.0) && (rho2d < 400.0);
        AnalyticAux aux;
        eval_analytic_f32<CODE == kAnalyticFull, false>(P, T, xf, yf, zf, rho2f, inside, S, aux);
      }
      if (CODE == kAnalyticDisc || CODE == kStack16) {
        if (A.sg_ne.g) S.ne = scalar_grid_at<float>(A.sg_ne, xd, yd, zd);
        if (A.sg_n0.g) S.N0 = scalar_grid_at<float>(A.sg_n0, xd, yd, zd);
      }
      S.ne *= T.scalef;
      float eI, a, bq;
      emission(P, S.BN, S.BE, S.N0, eI, a, bq);
      accI += eI;
      // A6: half-cell Faraday sum (S:C-2#5), tile-local, compensated
      const float gn = S.ne * S.Bpar;
      gabs = fmaf(fabsf(S.ne), fabsf(S.Bpar) + fabsf(S.BN) + fabsf(S.BE), gabs);
      const float ph = fmaf(0.5f, gn, hi);
      const float sum = hi + gn;
      lo += gn - (sum - hi);
      hi = sum;
      // A7: rotate and accumulate per frequency
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        const float th = k_rad[f] * ph;
        const float c = mufu_cos(th), s = mufu_sin(th);
        tq[f] = fmaf(a, c, fmaf(-bq, s, tq[f]));
        tu[f] = fmaf(a, s, fmaf(bq, c, tu[f]));
      }
    }
    if (ts == n0) {
#pragma unroll
      for (int f = 0; f < NF; ++f) { accQ[f] = tq[f]; accU[f] = tu[f]; }
    } else {
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        rotate_by_offset(ft.k_turn[f], carry, tq[f], tu[f]);
        accQ[f] += tq[f]; accU[f] += tu[f];
      }
    }
    carry += (double)hi + (double)lo;
    tmax = fmaxf(tmax, fabsf(hi));
  }

  // combine the G lanes of the sightline
  float absS;
  const double phi_total = G > 1 ? group_sum_d<G>(carry) : carry;
  if (G > 1) {
    const double off = group_exclusive_scan<G>(carry, g);
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      if (g > 0) rotate_by_offset(ft.k_turn[f], off, accQ[f], accU[f]);
      accQ[f] = group_sum<G>(accQ[f]);
      accU[f] = group_sum<G>(accU[f]);
    }
    accI = group_sum<G>(accI);
    absS = group_sum<G>(gabs);
    tmax = group_max<G>(tmax);
  } else {
    absS = gabs;
  }
  if (valid && g == 0) {
    const int64_t npix = A.geo.npix;
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const int64_t o = ((int64_t)b * A.n_freq_total + A.f0 + f) * npix + pix;
      A.I[o] = P.coefI[A.f0 + f] * T.scalef * accI;
      A.Q[o] = P.coefP[A.f0 + f] * T.scalef * accQ[f];
      A.U[o] = P.coefP[A.f0 + f] * T.scalef * accU[f];
    }
    if (A.f0 == 0 && A.phi) A.phi[sl] = phi_total;
    if (A.f0 == 0 && A.phi_has) A.phi_has[sl] = 0;
    if (A.f0 == 0 && A.flag_S > 0.0f && (absS > A.flag_S || tmax > A.flag_T)) {
      const int k = atomicAdd(A.append_count, 1);
      A.append_list[k] = (int)sl;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Forward, fp32 chain, batched (S:8(a) A12, "batch acceleration"): one thread integrates the SAME sightline for
// NB consecutive parameter vectors of the batch, so everything that does not depend on the parameters -- the float64
// sample position and annulus test, their four conversions to fp32, 1/rho, ln(rho/8), tanh z (8 of the ~29 XU
// operations per sample and vector at cfg 2, where this kernel is XU-bound) -- is evaluated once per sample instead
// of once per vector.  One frequency, one thread per sightline (the shape of HMC-style batches: many vectors, modest
// maps).  Per vector the arithmetic, and so every map value, is that of forward_kernel<CODE, 1, 1, false>.
// ------------------------------------------------------------------------------------------------
template <int CODE, int NB>
__global__ void __launch_bounds__(kBlock) forward_batched_kernel(const __grid_constant__ ForwardArgs A,
                                                                 const __grid_constant__ FreqTab ft) {
  static_assert(CODE == kAnalyticDisc || CODE == kAnalyticFull, "analytic models only");
  if (A.mode && *A.mode != kModeFastThenList) return;
  const int64_t tid = (int64_t)blockIdx.x * kBlock + threadIdx.x;
  const int n_groups = (A.batch + NB - 1) / NB;
  if (tid >= A.geo.npix * n_groups) return;
  const int bg = (int)(tid / A.geo.npix);
  const int64_t pix = tid - (int64_t)bg * A.geo.npix;
  int bj[NB];
  bool live[NB];
#pragma unroll
  for (int j = 0; j < NB; ++j) { live[j] = bg * NB + j < A.batch; bj[j] = live[j] ? bg * NB + j : A.batch - 1; }
  const Triad T = load_triad(A.geo, pix);
  const double delta = A.geo.delta * T.scale;
  double s_d = 0.5 * delta;
  PosF pf;
  pf.init(delta, 0);
  const float k_rad = ft.k_rad[0];

  float accI[NB], accQ[NB], accU[NB], gabs[NB];
  float tmax = 0.f;   // largest |tile-local Faraday sum| of the NB vectors together (one register; flags all NB when it fires)
  double carry[NB];
#pragma unroll
  for (int j = 0; j < NB; ++j) { accI[j] = 0.f; accQ[j] = 0.f; accU[j] = 0.f; gabs[j] = 0.f; carry[j] = 0.0; }
  for (int ts = 0; ts < A.geo.n_los; ts += kTile) {
    const int te = min(ts + kTile, A.geo.n_los);
    float hi[NB], lo[NB], tq[NB], tu[NB];
#pragma unroll
    for (int j = 0; j < NB; ++j) { hi[j] = 0.f; lo[j] = 0.f; tq[j] = 0.f; tu[j] = 0.f; }
    for (int n = ts; n < te; ++n) {
      const double xd = fma(s_d, T.nxd, A.geo.obs[0]);
      const double yd = fma(s_d, T.nyd, A.geo.obs[1]);
      s_d += delta;
      const double rho2d = fma(xd, xd, yd * yd);
      const bool inside = (rho2d > 9.0) && (rho2d < 400.0);
      float xf, yf, zf, rho2f;
      pf.next(A.geo, T, 1.0f, xf, yf, zf, rho2f);
      SharedGeomF geom;
      analytic_shared_f32(xf, yf, zf, rho2f, geom);
#pragma unroll
      for (int j = 0; j < NB; ++j) {
        const BatchConsts& P = A.bc[bj[j]];
        SampleF S;
        AnalyticAux aux;
        analytic_fields_f32<CODE == kAnalyticFull, false>(P, T, geom, zf, inside, S, aux);
        S.ne *= T.scalef;
        float eI, a, bq;
        emission(P, S.BN, S.BE, S.N0, eI, a, bq);
        accI[j] += eI;
        const float gn = S.ne * S.Bpar;
        gabs[j] = fmaf(fabsf(S.ne), fabsf(S.Bpar) + fabsf(S.BN) + fabsf(S.BE), gabs[j]);
        const float ph = fmaf(0.5f, gn, hi[j]);
        const float sum = hi[j] + gn;
        lo[j] += gn - (sum - hi[j]);
        hi[j] = sum;
        const float th = k_rad * ph;
        const float c = mufu_cos(th), sn = mufu_sin(th);
        tq[j] = fmaf(a, c, fmaf(-bq, sn, tq[j]));
        tu[j] = fmaf(a, sn, fmaf(bq, c, tu[j]));
      }
    }
#pragma unroll
    for (int j = 0; j < NB; ++j) {
      if (ts == 0) {
        accQ[j] = tq[j]; accU[j] = tu[j];
      } else {
        rotate_by_offset(ft.k_turn[0], carry[j], tq[j], tu[j]);
        accQ[j] += tq[j]; accU[j] += tu[j];
      }
      carry[j] += (double)hi[j] + (double)lo[j];
      tmax = fmaxf(tmax, fabsf(hi[j]));
    }
  }
#pragma unroll
  for (int j = 0; j < NB; ++j) {
    if (!live[j]) continue;
    const BatchConsts& P = A.bc[bj[j]];
    const int64_t o = ((int64_t)bj[j] * A.n_freq_total + A.f0) * A.geo.npix + pix;
    A.I[o] = P.coefI[A.f0] * T.scalef * accI[j];
    A.Q[o] = P.coefP[A.f0] * T.scalef * accQ[j];
    A.U[o] = P.coefP[A.f0] * T.scalef * accU[j];
    if (A.f0 == 0 && A.phi) A.phi[(int64_t)bj[j] * A.geo.npix + pix] = carry[j];
    if (A.f0 == 0 && A.phi_has) A.phi_has[(int64_t)bj[j] * A.geo.npix + pix] = 0;
    if (A.f0 == 0 && A.flag_S > 0.0f && (gabs[j] > A.flag_S || tmax > A.flag_T)) {
      const int k = atomicAdd(A.append_count, 1);
      A.append_list[k] = (int)((int64_t)bj[j] * A.geo.npix + pix);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Forward, float64 Faraday chain (synax_f64.cuh): B and n_e in float64 from short polynomials, the
// Faraday sum in float64; emission, N_0 and the per-frequency rotation in fp32 as in the fast kernel
// (the rotation angle is taken relative to the start of a 32-sample tile, whose own float64 angle is
// reduced to turns exactly).  G lanes per sightline; groups stride over the flag list written by
// forward_kernel, or over all sightlines when the list is null.
// ------------------------------------------------------------------------------------------------
#ifndef SYNAX_F64_MINB
#define SYNAX_F64_MINB 4
#endif
#ifndef SYNAX_F64_BLOCK
#define SYNAX_F64_BLOCK 128
#endif
constexpr int kBlockD = SYNAX_F64_BLOCK;   // threads per CTA of the float64-chain forward
template <int CODE, int G, int NF>
__global__ void __launch_bounds__(kBlockD, SYNAX_F64_MINB) forward_f64_kernel(const __grid_constant__ ForwardArgs A,
                                                             const __grid_constant__ FreqTab ft) {
  const int64_t tid = (int64_t)blockIdx.x * kBlockD + threadIdx.x;
  const int g = (int)(tid % G);
  const int64_t n_groups = ((int64_t)gridDim.x * kBlockD) / G;
  const int64_t n_sl = A.geo.npix * A.batch;
  constexpr int NFA = NF > 0 ? NF : 1;   // NF = 0: the adjoint's Faraday-only pass
  if (A.run_when == 1 && *A.mode != kModeFastThenList) return;
  if (A.run_when == 2 && *A.mode != kModeAllF64) return;
  if (A.run_when == 3 && *A.mode == kModeFastThenList) return;
  if (A.run_when == 4 && *A.mode != kModeSplit) return;
  const bool use_list = A.flag_list && (A.run_when == 3 ? *A.mode == kModeSplit : A.run_when != 2);
  const int64_t count = use_list ? (int64_t)(*A.flag_count) : n_sl;
  const int C = (A.geo.n_los + G - 1) / G;
  const int n0 = g * C;
  const int n1 = min(n0 + C, A.geo.n_los);
  const double delta0 = A.geo.delta;
  float k_rad[NFA];
#pragma unroll
  for (int f = 0; f < NF; ++f) k_rad[f] = ft.k_rad[f];

  for (int64_t it = tid / G;; it += n_groups) {
    if (it - ((threadIdx.x & 31) / G) >= count) break;   // first group of this warp: warp-uniform exit
    const bool valid = it < count;
    const int64_t item = valid ? it : count - 1;
    const int64_t sl = use_list ? (int64_t)A.flag_list[item] : item;
    const int b = (int)(sl / A.geo.npix);
    const int64_t pix = sl - (int64_t)b * A.geo.npix;
    const BatchConsts& P = A.bc[b];
    const BatchConstsD D = A.bd[b];   // by value: kept in registers across the sample loop
    const Triad T = load_triad(A.geo, pix);
    const double delta = delta0 * T.scale;
    double s_d = ((double)n0 + 0.5) * delta;
    float accI = 0.0f, accQ[NFA], accU[NFA];
#pragma unroll
    for (int f = 0; f < NF; ++f) { accQ[f] = 0.0f; accU[f] = 0.0f; }
    double S_loc = 0.0;      // sum of n_e B_LOS over this lane's finished samples
    const int tile = P.tile_d;
    const bool one_sample_tiles = tile == 1;
    for (int ts = n0; ts < n1; ts += tile) {
      const int te = min(ts + tile, n1);
      const double S_tile = S_loc;
      // tile bases for the adjoint: the Faraday sum before every 32nd sample.  One thread per sightline: tiles (a power of
      // two long, from sample 0) start on those samples.  Several lanes: see the sample loop.
      if (G == 1 && A.phi_base && A.f0 == 0 && valid && (ts & 31) == 0 && ts > 0)
        A.phi_base[(size_t)(ts >> 5) * (size_t)n_sl + sl] = S_loc;
      float tq[NFA], tu[NFA];
#pragma unroll
      for (int f = 0; f < NF; ++f) { tq[f] = 0.0f; tu[f] = 0.0f; }
      for (int n = ts; n < te; n += kUnrollD) {
        // kUnrollD consecutive samples advanced together (latency hiding); those past the tile end are computed
        // at harmless positions and masked out
        double xd[kUnrollD], yd[kUnrollD], zd[kUnrollD], rho2d[kUnrollD], Bx[kUnrollD], By[kUnrollD], Bz[kUnrollD],
            ne[kUnrollD];
        bool inside[kUnrollD], live[kUnrollD];
        float N0[kUnrollD];
#pragma unroll
        for (int j = 0; j < kUnrollD; ++j) {
          live[j] = n + j < te;
          xd[j] = fma(s_d, T.nxd, A.geo.obs[0]);
          yd[j] = fma(s_d, T.nyd, A.geo.obs[1]);
          zd[j] = fma(s_d, T.nzd, A.geo.obs[2]);
          if (live[j]) s_d += delta;
          rho2d[j] = fma(xd[j], xd[j], yd[j] * yd[j]);
          inside[j] = (rho2d[j] > 9.0) && (rho2d[j] < 400.0);
        }
        if (CODE == kUniform) {
#pragma unroll
          for (int j = 0; j < kUnrollD; ++j) {
            Bx[j] = (double)P.uB[0]; By[j] = (double)P.uB[1]; Bz[j] = (double)P.uB[2]; ne[j] = (double)P.une * T.scale; N0[j] = P.uN0;
          }
        } else {
          if (CODE == kStack16) {
#pragma unroll
            for (int j = 0; j < kUnrollD; ++j) eval_stack16_d(D, xd[j], yd[j], zd[j], rho2d[j], inside[j], Bx[j], By[j], Bz[j], ne[j]);
          } else {
            eval_analytic_dm<CODE == kAnalyticFull, kUnrollD>(D, xd, yd, zd, rho2d, inside, Bx, By, Bz, ne);
          }
#pragma unroll
          for (int j = 0; j < kUnrollD; ++j) {
            if ((CODE == kAnalyticDisc || CODE == kStack16) && A.sg_ne.g) ne[j] = scalar_grid_at<double>(A.sg_ne, xd[j], yd[j], zd[j]);
            ne[j] *= T.scale;
          }
#pragma unroll
          for (int j = 0; j < kUnrollD; ++j) {
            // N_0 (emission only): fp32 MUFU chain, Eq.(12)
            const float rho2f = fmaxf((float)rho2d[j], 1.0e-30f);
            const float rho = rho2f * mufu_rsqrt(rho2f);
            const float ez = mufu_ex2(P.k_hz * fabsf((float)zd[j]));
            const float dz = 1.0f + ez;
            N0[j] = 4.0f * P.p[9] * mufu_ex2(P.k_hr * rho) * ez * mufu_rcp(dz * dz);
            if ((CODE == kAnalyticDisc || CODE == kStack16) && A.sg_n0.g) N0[j] = scalar_grid_at<float>(A.sg_n0, xd[j], yd[j], zd[j]);
          }
        }
#pragma unroll
        for (int j = 0; j < kUnrollD; ++j) {
          double gn = ne[j] * fma(Bx[j], T.nxd, fma(By[j], T.nyd, Bz[j] * T.nzd));   // n_e B.n, signed (S:C-2#3)
          if (!live[j]) gn = 0.0;
          // several lanes per sightline (chunks start anywhere): the lane-local sum before every 32nd sample, per sample;
          // the lanes add their offset below
          if (G > 1 && A.phi_base && A.f0 == 0 && live[j] && valid && ((n + j) & 31) == 0 && n + j > 0)
            A.phi_base[(size_t)((n + j) >> 5) * (size_t)n_sl + sl] = S_loc;
          // half-cell (S:C-2#5), tile-local.  Tile length 1 (under-resolved: one sample already turns by more than 24 rad at the
          // lowest frequency): the half-cell angle joins the tile offset, which is reduced to turns in float64 below, instead
          // of being formed in fp32 here -- two selects, the frequency loop stays as it is
          const float ph = one_sample_tiles ? 0.0f : (float)fma(0.5, gn, S_loc - S_tile);
          S_loc += gn;
          const float bx = (float)Bx[j], by = (float)By[j], bz = (float)Bz[j];
          const float BN = fmaf(bx, T.eNx, fmaf(by, T.eNy, bz * T.eNz));
          const float BE = fmaf(bx, T.eEx, by * T.eEy);
          float eI, a, bq;
          emission(P, BN, BE, live[j] ? N0[j] : 0.0f, eI, a, bq);
          accI += eI;
#pragma unroll
          for (int f = 0; f < NF; ++f) {
            const float th = k_rad[f] * ph;
            const float c = mufu_cos(th), s = mufu_sin(th);
            tq[f] = fmaf(a, c, fmaf(-bq, s, tq[f]));
            tu[f] = fmaf(a, s, fmaf(bq, c, tu[f]));
          }
        }
      }
      // one-sample tiles: the sample's half-cell term g_n / 2 = (S_loc - S_tile) / 2 is rotated exactly with the tile offset
      const double tile_off = one_sample_tiles ? 0.5 * (S_tile + S_loc) : S_tile;
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        rotate_by_offset(ft.k_turn[f], tile_off, tq[f], tu[f]);
        accQ[f] += tq[f]; accU[f] += tu[f];
      }
    }
    const double phi_total = G > 1 ? group_sum_d<G>(S_loc) : S_loc;
    if (G > 1) {
      const double off = group_exclusive_scan<G>(S_loc, g);
      if (A.phi_base && A.f0 == 0 && valid && g > 0)   // this lane's tile bases were stored relative to its chunk start
        for (int k = (n0 + 31) >> 5; (k << 5) < n1; ++k)
          if (k > 0) A.phi_base[(size_t)k * (size_t)n_sl + sl] += off;
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        rotate_by_offset(ft.k_turn[f], off, accQ[f], accU[f]);
        accQ[f] = group_sum<G>(accQ[f]);
        accU[f] = group_sum<G>(accU[f]);
      }
      accI = group_sum<G>(accI);
    }
    if (valid && g == 0) {
      const int64_t npix = A.geo.npix;
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        const int64_t o = ((int64_t)b * A.n_freq_total + A.f0 + f) * npix + pix;
        A.I[o] = P.coefI[A.f0 + f] * T.scalef * accI;
        A.Q[o] = P.coefP[A.f0 + f] * T.scalef * accQ[f];
        A.U[o] = P.coefP[A.f0 + f] * T.scalef * accU[f];
      }
      if (A.f0 == 0 && A.phi) A.phi[sl] = phi_total;
      if (A.f0 == 0 && A.phi_has) A.phi_has[sl] = 1;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Pilot: Faraday sums only (MUFU-grade fp32 chain), one warp per sampled sightline (every `stride`-th),
// counting those whose rotation angle exceeds the escalation threshold.  decide_kernel then picks the
// forward strategy on the device -- no host synchronisation: fp32 pass + float64 redo of the flagged
// list when they are few, or the float64-chain kernel for every sightline when they are many.
// ------------------------------------------------------------------------------------------------
template <int CODE>
__global__ void __launch_bounds__(kBlock) pilot_kernel(const __grid_constant__ ForwardArgs A, int64_t stride,
                                                       int64_t n_pilot, int* __restrict__ ctrl) {
  const int lane = threadIdx.x & 31;
  const int64_t j = ((int64_t)blockIdx.x * kBlock + threadIdx.x) >> 5;
  if (j >= n_pilot) return;
  const int64_t sl = j * stride;
  const int b = (int)(sl / A.geo.npix);
  const int64_t pix = sl - (int64_t)b * A.geo.npix;
  const BatchConsts& P = A.bc[b];
  const Triad T = load_triad(A.geo, pix);
  // every 16th sample of the sightline (all of them below 32), spread over the lanes: the estimate classify_kernel and the
  // adjoint use.  It only picks the strategy -- the fp32 kernels check the exact sum -- and costs 1/16 of a full pass
  // (cfg 1: 12.7 -> see profiles/r02_launches.md; before, the pilot was 8 % of that forward).
  const int step = A.geo.n_los >= 32 ? 16 : 1;
  float gabs = 0.0f;
  for (int n = step / 2 + lane * step; n < A.geo.n_los; n += 32 * step) {
    const double s_d = ((double)n + 0.5) * A.geo.delta * T.scale;
    float gn;
    if (CODE == kUniform) {
      gn = fabsf(P.une) * (fabsf(P.uB[0]) + fabsf(P.uB[1]) + fabsf(P.uB[2]));
    } else {
      const double xd = fma(s_d, T.nxd, A.geo.obs[0]);
      const double yd = fma(s_d, T.nyd, A.geo.obs[1]);
      const double zd = fma(s_d, T.nzd, A.geo.obs[2]);
      const double rho2d = fma(xd, xd, yd * yd);
      SampleF Sm;
      if (CODE == kStack16) {
        StackAux sa;
        eval_stack16_f32<true>(P, T, (float)xd, (float)yd, (float)zd, (float)rho2d, (rho2d > 9.0) && (rho2d < 400.0), Sm, sa);
      } else {
        AnalyticAux aux;
        eval_analytic_f32<CODE == kAnalyticFull, false>(P, T, (float)xd, (float)yd, (float)zd, (float)rho2d,
                                                        (rho2d > 9.0) && (rho2d < 400.0), Sm, aux);
      }
      if ((CODE == kAnalyticDisc || CODE == kStack16) && A.sg_ne.g) Sm.ne = scalar_grid_at<float>(A.sg_ne, xd, yd, zd);
      gn = fabsf(Sm.ne) * (fabsf(Sm.Bpar) + fabsf(Sm.BN) + fabsf(Sm.BE));
    }
    gabs += gn;
  }
  const float absS = T.scalef * (float)step * group_sum<32>(gabs);
  if (lane == 0 && absS > A.flag_S) atomicAdd(ctrl + kCtrlPilotFlagged, 1);
}

// kModeSplit: one thread per sightline; sightlines whose estimated round-off scale exceeds flag_S go to the head of
// the flag list (float64 chain), the others to list_u (fp32 kernel).  Block-ordered compaction: within a CTA the
// sightlines keep their order (neighbouring pixels stay neighbours in the lists); the CTAs' segments land in the
// order their atomics arrive -- the maps do not depend on it.
template <int CODE>
__global__ void __launch_bounds__(kBlock) classify_kernel(const __grid_constant__ ForwardArgs A, int* __restrict__ ctrl) {
  if (ctrl[kCtrlMode] != kModeSplit) return;
  __shared__ int w_cnt[2][kBlock / 32];
  __shared__ int w_base[2][kBlock / 32];
  const int64_t n_sl = A.geo.npix * A.batch;
  for (int64_t chunk = blockIdx.x; chunk * kBlock < n_sl; chunk += gridDim.x) {   // block-uniform trip count
  const int64_t sl = chunk * kBlock + threadIdx.x;
  const bool valid = sl < n_sl;
  bool flagged = false;
  if (valid) {
    const int b = (int)(sl / A.geo.npix);
    const int64_t pix = sl - (int64_t)b * A.geo.npix;
    const BatchConsts& P = A.bc[b];
    const Triad T = load_triad(A.geo, pix);
    // (3 % under the threshold: a sightline the estimate misses by a little is redone after the join, alone on the GPU --
    // cfg 4: that redo 0.18 -> 0.11 ms for 10,003 more sightlines on the float64 chain's list, forward 9.17 -> 9.09 ms.
    // The kernel's second criterion, the Faraday sum inside one 32-sample tile, is estimated from the same samples: at
    // nside 128 x 256 samples the redo of what it flagged took 0.15 of 0.89 ms.)
    // (only where a tile is a sizeable part of the sightline, <= 512 samples: longer ones stay far below it per tile unless
    // the first criterion flags them anyway, and the bookkeeping costs cfg 4 0.01 ms; a miss is only redone later)
    float tile_est = 0.f, est;
    if (A.flag_T > 0.f && A.geo.n_los <= 512) est = roundoff_scale_estimate<CODE, true>(A.geo, P, T, A.sg_ne, 0, A.geo.n_los, &tile_est) * T.scalef;
    else est = roundoff_scale_estimate<CODE>(A.geo, P, T, A.sg_ne, 0, A.geo.n_los) * T.scalef;
    flagged = est > 0.97f * A.flag_S || (A.flag_T > 0.f && tile_est * T.scalef > 0.97f * A.flag_T);
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned mf = __ballot_sync(0xffffffffu, valid && flagged), mu = __ballot_sync(0xffffffffu, valid && !flagged);
  if (lane == 0) { w_cnt[0][warp] = __popc(mf); w_cnt[1][warp] = __popc(mu); }
  __syncthreads();
  if (threadIdx.x < 2) {
    int tot = 0;
    for (int w = 0; w < kBlock / 32; ++w) { w_base[threadIdx.x][w] = tot; tot += w_cnt[threadIdx.x][w]; }
    const int base = tot ? atomicAdd(ctrl + (threadIdx.x == 0 ? kCtrlFlagCount : kCtrlCountU), tot) : 0;
    for (int w = 0; w < kBlock / 32; ++w) w_base[threadIdx.x][w] += base;
  }
  __syncthreads();
  if (valid) {
    const unsigned below = (1u << lane) - 1u;
    if (flagged) A.flag_list[w_base[0][warp] + __popc(mf & below)] = (int)sl;
    else A.list_u[w_base[1][warp] + __popc(mu & below)] = (int)sl;
  }
  __syncthreads();
  }
}

}  // namespace synax
