// synax_forward.cuh -- plan geometry kernel (A1), per-batch prologue, forward kernels (A2-A8, A12).
#pragma once
#include "synax_device.cuh"
#include "synax_f64.cuh"

namespace synax {

#ifndef SYNAX_FWD_FASTTRIG
#define SYNAX_FWD_FASTTRIG false
#endif
#ifndef SYNAX_FAST_ACC
#define SYNAX_FAST_ACC false
#endif
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
// A1: HEALPix RING pixel -> (cos l, sin l, cos b, sin b) in float64 (Gorski et al. 2005).
// Integer ring arithmetic as in DESIGN.md section 4; once per plan.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int64_t isqrt_i64(int64_t v) {
  int64_t r = (int64_t)sqrt((double)v);
  while (r * r > v) --r;
  while ((r + 1) * (r + 1) <= v) ++r;
  return r;
}

// Writes dirs[i] for the `count` pixels p = pix0 + i of the nside map (a plan may hold a shard of the sky).
__global__ void pix2ang_kernel(int64_t nside, int64_t pix0, int64_t count, double* __restrict__ dirs) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= count) return;
  const int64_t p = pix0 + idx;
  const int64_t npix = 12 * nside * nside;
  const int64_t ncap = 2 * nside * (nside - 1);
  double z, phi, omz;  // omz = 1 - |z| kept separately for accurate cos b near the poles
  if (p < ncap) {
    const int64_t i = (1 + isqrt_i64(1 + 2 * p)) / 2;
    const int64_t j = p + 1 - 2 * i * (i - 1);
    omz = (double)(i * i) / (3.0 * (double)(nside * nside));
    z = 1.0 - omz;
    phi = ((double)j - 0.5) * SYNAX_PI / (2.0 * (double)i);
  } else if (p < npix - ncap) {
    const int64_t pp = p - ncap;
    const int64_t i = pp / (4 * nside) + nside;
    const int64_t j = pp % (4 * nside) + 1;
    const double s = ((i + nside) & 1) ? 1.0 : 0.5;
    z = (double)(2 * nside - i) * 2.0 / (3.0 * (double)nside);
    omz = 1.0 - fabs(z);
    phi = ((double)j - s) * SYNAX_PI / (2.0 * (double)nside);
  } else {
    const int64_t pp = npix - p;
    const int64_t i = (1 + isqrt_i64(2 * pp - 1)) / 2;
    const int64_t j = 4 * i + 1 - (pp - 2 * i * (i - 1));
    omz = (double)(i * i) / (3.0 * (double)(nside * nside));
    z = -1.0 + omz;
    phi = ((double)j - 0.5) * SYNAX_PI / (2.0 * (double)i);
  }
  double sl, cl;
  sincos(phi, &sl, &cl);
  const double cb = sqrt(omz * (1.0 + fabs(z)));  // sin(theta) = sqrt((1-|z|)(1+|z|))
  dirs[4 * idx + 0] = cl; dirs[4 * idx + 1] = sl; dirs[4 * idx + 2] = cb; dirs[4 * idx + 3] = z;
}

// Path length of every sightline of the plan from the observer (strictly inside the box) to the face of a box of
// side lengths `box` centred on the Galactic centre, in units of s_ref (Fig. 1): path[i] = L_i / s_ref.
__global__ void box_path_kernel(const double* __restrict__ dirs, int64_t count, double ox, double oy, double oz,
                                double hx, double hy, double hz, double inv_s_ref, double* __restrict__ path) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= count) return;
  const double4 d = *reinterpret_cast<const double4*>(dirs + 4 * i);   // cos l, sin l, cos b, sin b
  const double n[3] = {d.z * d.x, d.z * d.y, d.w};
  const double o[3] = {ox, oy, oz}, h[3] = {hx, hy, hz};
  double L = 1.0e300;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    if (n[k] > 0.0) L = fmin(L, (h[k] - o[k]) / n[k]);
    else if (n[k] < 0.0) L = fmin(L, (-h[k] - o[k]) / n[k]);
  }
  path[i] = L * inv_s_ref;
}

// ------------------------------------------------------------------------------------------------
// Prologue: raw parameters -> BatchConsts (float64 math, once per batch element per call).
// Folds Eq.(2)'s constants, the Rayleigh-Jeans conversion (S:C-2#1) and the units into
// c_f(alpha) so that I_f = c_f Delta sum_n N_0 (B_perp^2)^((alpha+1)/4)  with B in uG.
// ------------------------------------------------------------------------------------------------
struct AuxHost { float v[7]; };  // C0, h_r, h_z, alpha, ne0, h_er, h_ez

__global__ void prologue_kernel(int code, const float* __restrict__ params, int n_params, int batch,
                                AuxHost aux, FreqTab ft, double delta, BatchConsts* __restrict__ out,
                                BatchConstsD* __restrict__ outd) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= batch) return;
  BatchConsts c;
  for (int j = 0; j < 16; ++j) c.sp[j] = 0.0f;
  double p[16];
  for (int j = 0; j < 16; ++j) p[j] = 0.0;
  double alpha;
  if (code == kAnalyticFull) {
    for (int j = 0; j < 16; ++j) p[j] = (double)params[(size_t)b * n_params + j];
  } else if (code == kUniform) {
    const float* q = params + (size_t)b * n_params;
    c.uB[0] = q[0]; c.uB[1] = q[1]; c.uB[2] = q[2]; c.uN0 = q[3]; c.une = q[4];
    p[12] = (double)q[5];
    p[4] = p[7] = p[8] = p[10] = p[11] = p[14] = p[15] = 1.0;
  } else {  // DISC4, STACK16 or GRID_B: densities and alpha from aux
    if (code == kStack16)
      for (int j = 0; j < 16; ++j) c.sp[j] = params[(size_t)b * n_params + j];
    if (code == kAnalyticDisc)
      for (int j = 0; j < 4; ++j) p[j] = (double)params[(size_t)b * n_params + j];
    p[4] = 1.0;  // unused: k_hb = 0
    p[6] = 0.0; p[7] = 1.0; p[8] = 1.0;
    p[9] = aux.v[0]; p[10] = aux.v[1]; p[11] = aux.v[2]; p[12] = aux.v[3];
    p[13] = aux.v[4]; p[14] = aux.v[5]; p[15] = aux.v[6];
  }
  alpha = p[12];
  for (int j = 0; j < 16; ++j) c.p[j] = (float)p[j];
  const double log2e = 1.4426950408889634;
  c.k_hb = (code == kAnalyticFull) ? (float)(-log2e / p[4]) : 0.0f;
  c.k_hb_lo = (code == kAnalyticFull) ? (float)(-log2e / p[4] - (double)c.k_hb) : 0.0f;
  c.inv_wh = (float)(1.0 / p[8]);
  c.inv_rh = (float)(1.0 / p[7]);
  c.k_hr = (float)(-log2e / p[10]);
  c.k_hz = (float)(-2.0 * log2e / fabs(p[11]));
  c.k_her = (float)(-log2e / p[14]);
  c.k_her_lo = (float)(-log2e / p[14] - (double)c.k_her);
  c.k_hez = (float)(-2.0 * log2e / fabs(p[15]));
  c.q_exp = (float)((alpha - 3.0) * 0.25);
  c.pi_frac = (float)((alpha + 1.0) / (alpha + 7.0 / 3.0));
  c.alpha_is_3 = (c.p[12] == 3.0f) ? 1 : 0;
  c.angles_small = (fabs(p[1]) + fabs(p[2]) <= 0.78 && fabs(p[3]) <= 0.78) ? 1 : 0;   // 0.78 < pi/4; |ln(rho/8)| < 1 in the annulus
  c.dpi_dalpha_over_pi = (float)(1.0 / (alpha + 1.0) - 1.0 / (alpha + 7.0 / 3.0));
  // Eq.(2) prefactor with B^((1+alpha)/2) nu^((1-alpha)/2) factored out
  const double g1 = tgamma(alpha * 0.25 - 1.0 / 12.0), g2 = tgamma(alpha * 0.25 + 19.0 / 12.0);
  const double w = 4.0 * SYNAX_PI * SYNAX_ME * SYNAX_C / (3.0 * SYNAX_QE);
  const double A_I = sqrt(3.0) * SYNAX_QE * SYNAX_QE * SYNAX_QE / (8.0 * SYNAX_PI * SYNAX_ME * SYNAX_C * SYNAX_C) *
                     pow(w, (1.0 - alpha) * 0.5) * pow(2.0, (alpha + 1.0) * 0.5) / (alpha + 1.0) * g1 * g2;
  const double dlnA = -0.5 * log(w) + 0.5 * log(2.0) - 1.0 / (alpha + 1.0) +
                      0.25 * digamma_d(alpha * 0.25 - 1.0 / 12.0) + 0.25 * digamma_d(alpha * 0.25 + 19.0 / 12.0) +
                      0.5 * log(1.0e-6);
  for (int f = 0; f < kMaxFreq; ++f) {
    if (f < ft.n_freq) {
      const double nu = ft.freq[f];
      const double TRJ = SYNAX_C * SYNAX_C / (2.0 * SYNAX_KB * nu * nu);
      const double cf = TRJ * A_I * pow(nu, (1.0 - alpha) * 0.5) * pow(1.0e-6, (alpha + 1.0) * 0.5) * SYNAX_KPC * delta;
      c.coefI[f] = (float)cf;
      c.coefP[f] = (float)(cf * (alpha + 1.0) / (alpha + 7.0 / 3.0));
      c.dlnc_dalpha[f] = (float)(dlnA - 0.5 * log(nu));
    } else {
      c.coefI[f] = c.coefP[f] = c.dlnc_dalpha[f] = 0.0f;
    }
  }
  // Tile length of the float64-chain kernel: the fp32 angle k_f * (tile-local Faraday sum) must stay small
  // enough for its 6e-8 relative round-off not to matter.  Bound on |n_e B_LOS| per sample:
  {
    double gmax;
    if (code == kUniform) {
      gmax = fabs((double)c.une) * (fabs((double)c.uB[0]) + fabs((double)c.uB[1]) + fabs((double)c.uB[2]));
    } else {
      double bmax = fabs(p[0]);
      if (code == kStack16) bmax = 0.6 * fabs((double)c.sp[0]) + 0.3 * fabs((double)c.sp[4]) + 0.1 * fabs((double)c.sp[8]) + 0.3 * fabs((double)c.sp[12]);
      if (code == kAnalyticFull) bmax = bmax * fmax(exp(5.0 / p[4]), exp(-12.0 / p[4])) + fabs(p[5]);
      gmax = fabs(p[13]) * bmax;
    }
    double kmax = 0.0;
    for (int f = 0; f < ft.n_freq; ++f) kmax = fmax(kmax, (double)ft.k_rad[f]);
    const double per_step = kmax * gmax;
    int t = kTileDMax;
    if (per_step * t > (double)kTilePhase) t = (int)((double)kTilePhase / per_step);
    if (t > kUnrollD) t -= t % kUnrollD;
    c.tile_d = t < 1 ? 1 : t;
  }
  out[b] = c;
  if (outd) {
    BatchConstsD d;
    d.b0 = p[0]; d.psi0 = p[1]; d.psi1 = p[2]; d.chi0 = p[3];
    d.k_hb = (code == kAnalyticFull) ? -log2e / p[4] : 0.0;
    d.Bh = p[5]; d.zh0 = p[6]; d.inv_rh = 1.0 / p[7]; d.inv_wh = 1.0 / p[8];
    d.ne0x4 = 4.0 * p[13]; d.k_her = -log2e / p[14]; d.k_hez = -2.0 * log2e / fabs(p[15]);
    d.psi1_small = fabs(p[2]) <= 0.05 ? 1 : 0;
    d.angles_small = (fabs(p[1]) + fabs(p[2]) <= 0.78 && fabs(p[3]) <= 0.78) ? 1 : 0;   // 0.78 < pi/4
    d.hez_is_one = (p[15] == 1.0 || p[15] == -1.0) ? 1 : 0;
    for (int k = 0; k < 4; ++k) {
      const bool st = code == kStack16;
      const double w = k == 0 ? 0.6 : (k == 2 ? 0.1 : 0.3);
      d.sb0[k] = st ? w * (double)c.sp[4 * k] : 0.0; d.spsi0[k] = st ? (double)c.sp[4 * k + 1] : 0.0;
      d.spsi1[k] = st ? (double)c.sp[4 * k + 2] : 0.0; d.schi0[k] = st ? (double)c.sp[4 * k + 3] : 0.0;
    }
    outd[b] = d;
  }
}

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
struct ForwardArgs {
  Geometry geo;
  const BatchConsts* bc;
  const BatchConstsD* bd; // float64 constants (float64 Faraday chain only)
  int batch;
  int f0;                 // first frequency of this pass
  float* I; float* Q; float* U;
  int n_freq_total;
  float flag_S;           // flag a sightline when max |sum n_e B_LOS| exceeds this (<=0: never)
  int* flag_count;        // device counter
  int* flag_list;         // device list of flagged sightline ids (b * npix + p)
  ScalarGridDesc sg_ne, sg_n0;  // gridded n_e / N_0 replacing the analytic discs (DISC4, GRID_B), g == nullptr: unused
  const int* mode;        // device: kModeFastThenList / kModeAllF64 / kModeSplit (written by decide_kernel), or null
  int run_when;           // forward_f64_kernel: 0 always, 1 only in mode fast-then-list (flag list), 2 only in mode
                          // all-float64 (every sightline), 3 in both all-float64 (every sightline) and split (flag list)
  int* list_u;            // kModeSplit: sightlines classify_kernel left to the fp32 kernel (count in ctrl[kCtrlCountU])
  const int* count_u;
};

// kModeSplit: classify_kernel sorts the sightlines by an estimate of the round-off scale into the flag list (float64
// chain) and list_u (fp32 kernel, whose exact criterion still appends what the estimate missed to the flag list).
enum { kModeFastThenList = 0, kModeAllF64 = 1, kModeSplit = 2 };
enum { kCtrlFlagCount = 0, kCtrlPilotFlagged = 1, kCtrlMode = 2, kCtrlCountU = 3, kCtrlWords = 4 };

// Estimate of one lane's share of the round-off scale  sum_n |n_e| (|B_LOS| + |B_N| + |B_E|)  over samples [n0, n1):
// every 16th sample (all of them for short chunks), MUFU-grade fp32 chain; the caller sums the lanes of the
// sightline and multiplies by Triad::scalef.
template <int CODE>
__device__ __forceinline__ float roundoff_scale_estimate(const Geometry& geo, const BatchConsts& P, const Triad& T,
                                                         const ScalarGridDesc& sg_ne, int n0, int n1) {
  const int step = (n1 - n0 >= 32) ? 16 : 1;
  const double delta = geo.delta * T.scale;
  float est = 0.f;
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
        eval_analytic_f32<CODE == kAnalyticFull, false, true>(P, T, (float)xd, (float)yd, (float)zd, (float)rho2d, inside, S, aux);
      }
      if ((CODE == kAnalyticDisc || CODE == kStack16) && sg_ne.g) S.ne = scalar_grid_at<float>(sg_ne, xd, yd, zd);
    }
    est = fmaf(fabsf(S.ne), fabsf(S.Bpar) + fabsf(S.BN) + fabsf(S.BE), est);
  }
  return est * (float)step;
}

// LIST = false: every sightline, runs in kModeFastThenList (or without a pilot); LIST = true: the sightlines of
// list_u, runs in kModeSplit.  (Two instantiations rather than a run-time switch: the switch put two more
// F2F conversions per sample into the loop of the NF = 1 kernel, +4 % at cfg 2.)
template <int CODE, int G, int NF, bool LIST>
__global__ void __launch_bounds__(kBlock) forward_kernel(const __grid_constant__ ForwardArgs A,
                                                         const __grid_constant__ FreqTab ft) {
  if (LIST ? (*A.mode != kModeSplit) : (A.mode && *A.mode != kModeFastThenList)) return;
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

  float k_rad[NF];
#pragma unroll
  for (int f = 0; f < NF; ++f) k_rad[f] = ft.k_rad[f];

  float accI = 0.0f, accQ[NF], accU[NF];
#pragma unroll
  for (int f = 0; f < NF; ++f) { accQ[f] = 0.0f; accU[f] = 0.0f; }
  double carry = 0.0;            // chunk-local sum of n_e B_LOS over finished tiles
  float gabs = 0.0f;             // sum n_e (|B_LOS| + |B_N| + |B_E|): scale of the fp32 round-off in the Faraday sum

  for (int ts = n0; ts < n1; ts += kTile) {
    const int te = min(ts + kTile, n1);
    float hi = 0.0f, lo = 0.0f;  // tile-local two-float sum of n_e B_LOS
    float tq[NF], tu[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) { tq[f] = 0.0f; tu[f] = 0.0f; }
    for (int n = ts; n < te; ++n) {
      // A2: midpoint position in float64 (mask decisions), rounded once to fp32 for the fields
      const double xd = fma(s_d, T.nxd, A.geo.obs[0]);
      const double yd = fma(s_d, T.nyd, A.geo.obs[1]);
      const double zd = fma(s_d, T.nzd, A.geo.obs[2]);
      s_d += delta;
      SampleF S;
      if (CODE == kUniform) {
        S.Bpar = fmaf(P.uB[0], T.nx, fmaf(P.uB[1], T.ny, P.uB[2] * T.nz));
        S.BN = fmaf(P.uB[0], T.eNx, fmaf(P.uB[1], T.eNy, P.uB[2] * T.eNz));
        S.BE = fmaf(P.uB[0], T.eEx, P.uB[1] * T.eEy);
        S.N0 = P.uN0; S.ne = P.une;
      } else if (CODE == kStack16) {
        const double rho2d = fma(xd, xd, yd * yd);
        StackAux sa;
        eval_stack16_f32<false>(P, T, (float)xd, (float)yd, (float)zd, (float)rho2d, (rho2d > 9.0) && (rho2d < 400.0), S, sa);
      } else {
        const double rho2d = fma(xd, xd, yd * yd);
        const bool inside = (rho2d > 9.0) && (rho2d < 400.0);
        AnalyticAux aux;
        eval_analytic_f32<CODE == kAnalyticFull, SYNAX_FAST_ACC, SYNAX_FWD_FASTTRIG>(P, T, (float)xd, (float)yd, (float)zd, (float)rho2d, inside, S, aux);
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
  }

  // combine the G lanes of the sightline
  float absS;
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
    if (A.f0 == 0 && A.flag_S > 0.0f && absS > A.flag_S) {
      const int k = atomicAdd(A.flag_count, 1);
      A.flag_list[k] = (int)sl;
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
  if (A.run_when == 1 && *A.mode != kModeFastThenList) return;
  if (A.run_when == 2 && *A.mode != kModeAllF64) return;
  if (A.run_when == 3 && *A.mode == kModeFastThenList) return;
  const bool use_list = A.flag_list && (A.run_when == 3 ? *A.mode == kModeSplit : A.run_when != 2);
  const int64_t count = use_list ? (int64_t)(*A.flag_count) : n_sl;
  const int C = (A.geo.n_los + G - 1) / G;
  const int n0 = g * C;
  const int n1 = min(n0 + C, A.geo.n_los);
  const double delta0 = A.geo.delta;
  float k_rad[NF];
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
    float accI = 0.0f, accQ[NF], accU[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) { accQ[f] = 0.0f; accU[f] = 0.0f; }
    double S_loc = 0.0;      // sum of n_e B_LOS over this lane's finished samples
    const int tile = P.tile_d;
    for (int ts = n0; ts < n1; ts += tile) {
      const int te = min(ts + tile, n1);
      const double S_tile = S_loc;
      float tq[NF], tu[NF];
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
          const float ph = (float)fma(0.5, gn, S_loc - S_tile);                  // half-cell (S:C-2#5), tile-local
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
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        rotate_by_offset(ft.k_turn[f], S_tile, tq[f], tu[f]);
        accQ[f] += tq[f]; accU[f] += tu[f];
      }
    }
    if (G > 1) {
      const double off = group_exclusive_scan<G>(S_loc, g);
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
  const int C = (A.geo.n_los + 31) / 32;
  const int n0 = lane * C, n1 = min(n0 + C, A.geo.n_los);
  float gabs = 0.0f;
  for (int n = n0; n < n1; ++n) {
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
  const float absS = T.scalef * group_sum<32>(gabs);
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
    flagged = roundoff_scale_estimate<CODE>(A.geo, P, T, A.sg_ne, 0, A.geo.n_los) * T.scalef > A.flag_S;
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

// Forward: the pilot's flagged share picks the mode -- below 1/50: fp32 pass + float64 redo of its flag list; above
// 3/4: float64 chain for every sightline; in between: split by classify_kernel.  (cfg 4 @ 408 MHz, fp32 pass 7.2 ms,
// float64 pass 11.1 ms: measured split 11.9 / 10.4 / 9.1 ms at 78 / 50 / 28 % flagged.)
__global__ void decide_forward_kernel(int* __restrict__ ctrl, int64_t n_pilot) {
  const int64_t f = ctrl[kCtrlPilotFlagged];
  ctrl[kCtrlMode] = (50 * f <= n_pilot) ? kModeFastThenList : (4 * f > 3 * n_pilot) ? kModeAllF64 : kModeSplit;
}

__global__ void decide_kernel(int* __restrict__ ctrl, int64_t n_pilot, int num, int den, int mode_yes) {
  // short forward calls (1/4): more than a quarter flagged -> one float64-chain pass costs less than fp32 + redo.
  // adjoint (0/1): any sampled sightline above half the threshold, see analytic_vjp.
  ctrl[kCtrlMode] = ((int64_t)den * ctrl[kCtrlPilotFlagged] > (int64_t)num * n_pilot) ? mode_yes : kModeFastThenList;
}

}  // namespace synax
