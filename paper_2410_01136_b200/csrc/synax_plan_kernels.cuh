// synax_plan_kernels.cuh -- the non-template kernels of the plan and of the per-call prologue: A1 pixel directions,
// box path lengths, per-batch constants, device-side strategy decisions.  Included by synax_api.cu only.
#pragma once
#include "synax_forward.cuh"

namespace synax {

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

// Writes dirs[i] for the `count` pixels p = pix0 + i * stride of the nside map (a plan may hold a shard of the sky: a
// contiguous range, stride 1, or every stride-th pixel).
__global__ void pix2ang_kernel(int64_t nside, int64_t pix0, int64_t stride, int64_t count, double* __restrict__ dirs) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= count) return;
  const int64_t p = pix0 + idx * stride;
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

// max |g[i]| of a non-negative-comparable float array into *out (zero on entry): non-negative floats order like ints
__global__ void absmax_kernel(const float* __restrict__ g, int64_t n, float* __restrict__ out) {
  float m = 0.f;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) m = fmaxf(m, fabsf(__ldg(g + i)));
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, d));
  if ((threadIdx.x & 31) == 0 && m > 0.f) atomicMax(reinterpret_cast<int*>(out), __float_as_int(m));
}

// *ok = 1 when the n floats of `now` equal `saved` bit for bit (the parameters the plan's last forward ran with), else 0.
// One block.
__global__ void phi_validate_kernel(const float* __restrict__ now, const float* __restrict__ saved, int64_t n, int* __restrict__ ok) {
  int same = 1;
  for (int64_t i = threadIdx.x; i < n; i += blockDim.x)
    if (__float_as_int(now[i]) != __float_as_int(saved[i])) same = 0;
  same = __syncthreads_and(same);
  if (threadIdx.x == 0) *ok = same;
}

// ne_max: device scalar max |ne_grid| when a gridded n_e replaces the analytic disc, else null
__global__ void prologue_kernel(int code, const float* __restrict__ params, int n_params, int batch,
                                AuxHost aux, FreqTab ft, double delta, int n_los, const float* __restrict__ ne_max,
                                BatchConsts* __restrict__ out, BatchConstsD* __restrict__ outd) {
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
  c.inv_wh = (float)(1.0 / p[8]);
  c.inv_rh = (float)(1.0 / p[7]);
  c.k_hr = (float)(-log2e / p[10]);
  c.k_hz = (float)(-2.0 * log2e / fabs(p[11]));
  c.k_her = (float)(-log2e / p[14]);
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
                     exp((1.0 - alpha) * 0.5 * log(w)) * exp2((alpha + 1.0) * 0.5) / (alpha + 1.0) * g1 * g2;
  const double dlnA = -0.5 * log(w) + 0.5 * log(2.0) - 1.0 / (alpha + 1.0) +
                      0.25 * digamma_d(alpha * 0.25 - 1.0 / 12.0) + 0.25 * digamma_d(alpha * 0.25 + 19.0 / 12.0) +
                      0.5 * log(1.0e-6);
  c.dlnA_dalpha = (float)dlnA;
  // (nu^((1 - alpha) / 2) as exp of the logarithm the alpha derivative needs anyway: this kernel is one serial float64 chain
  // in front of every call, and each pow() in it costs ~0.8 us)
  const double unit_B = exp((alpha + 1.0) * 0.5 * log(1.0e-6)) * SYNAX_KPC * delta;
  for (int f = 0; f < kMaxFreq; ++f) {
    if (f < ft.n_freq) {
      const double nu = ft.freq[f], ln_nu = log(nu);
      const double TRJ = SYNAX_C * SYNAX_C / (2.0 * SYNAX_KB * nu * nu);
      const double cf = TRJ * A_I * exp((1.0 - alpha) * 0.5 * ln_nu) * unit_B;
      c.coefI[f] = (float)cf;
      c.coefP[f] = (float)(cf * (alpha + 1.0) / (alpha + 7.0 / 3.0));
      c.dlnc_dalpha[f] = (float)(dlnA - 0.5 * ln_nu);
    } else {
      c.coefI[f] = c.coefP[f] = c.dlnc_dalpha[f] = 0.0f;
    }
  }
  // Tile length of the float64-chain kernel: the fp32 angle k_f * (tile-local Faraday sum) must stay small
  // enough for its 6e-8 relative round-off not to matter.  Bound on |n_e B_LOS| per sample:
  double per_step_rad;   // ... times the largest k_f: bound on the rotation of one sample
  {
    double gmax;
    if (code == kUniform) {
      gmax = fabs((double)c.une) * (fabs((double)c.uB[0]) + fabs((double)c.uB[1]) + fabs((double)c.uB[2]));
    } else {
      double bmax = fabs(p[0]);
      if (code == kStack16) bmax = 0.6 * fabs((double)c.sp[0]) + 0.3 * fabs((double)c.sp[4]) + 0.1 * fabs((double)c.sp[8]) + 0.3 * fabs((double)c.sp[12]);
      if (code == kAnalyticFull) bmax = bmax * fmax(exp(5.0 / p[4]), exp(-12.0 / p[4])) + fabs(p[5]);
      gmax = (ne_max ? (double)*ne_max : fabs(p[13])) * bmax;
    }
    double kmax = 0.0;
    for (int f = 0; f < ft.n_freq; ++f) kmax = fmax(kmax, (double)ft.k_rad[f]);
    const double per_step = kmax * gmax;
    per_step_rad = per_step;
    int t = kTileDMax;
    if (per_step * t > (double)kTilePhase) t = (int)((double)kTilePhase / per_step);
    if (t > kUnrollD) t -= t % kUnrollD;
    t = t < 1 ? 1 : t;
    while (t & (t - 1)) t &= t - 1;   // a power of two: tiles from sample 0 then start on every multiple of 32, where the
    c.tile_d = t;                     // float64-chain forward stores its Faraday depth for the adjoint (ForwardArgs::phi_base)
  }
  out[b] = c;
  if (outd) {
    BatchConstsD d;
    d.b0 = p[0]; d.psi0 = p[1]; d.psi1 = p[2]; d.chi0 = p[3];
    d.k_hb = (code == kAnalyticFull) ? -log2e / p[4] : 0.0;
    d.Bh = p[5]; d.zh0 = p[6]; d.inv_rh = 1.0 / p[7]; d.inv_wh = 1.0 / p[8];
    d.ne0x4 = 4.0 * p[13]; d.k_her = -log2e / p[14]; d.k_hez = -2.0 * log2e / fabs(p[15]);
    // ln(rho/8) from the MUFU lg2 (abs err ~5e-7, pseudo-random from sample to sample) turns the disc field by psi1 x that:
    // a relative error of ~|psi1| x 7e-7 in a sample's Faraday term, ~|psi1| x 7e-7 x (rotation per sample) x sqrt(n_los) in
    // the sightline's angle.  Kept below ~1e-5 rad: a run with ONE sample of 1,800 rad (psi1 0.014) was off by 2e-5 rad,
    // 1.1e-4 x RMS; 256 samples of <= 25 rad each (the same model at nside 128 x 256) stay at 4e-6 and keep the fast path.
    d.psi1_small = (fabs(p[2]) <= 0.05 && fabs(p[2]) * per_step_rad * sqrt((double)n_los) <= 10.0) ? 1 : 0;
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
