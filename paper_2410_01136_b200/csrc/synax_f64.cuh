// synax_f64.cuh -- float64 evaluation of the Faraday integrand n_e B_LOS for the analytic models, built
// from short polynomials instead of libm calls.
//
// Why: at 408 MHz the Faraday angle of an in-plane sightline reaches ~1500 rad while the depolarised Q/U
// maps have an RMS ~100x below the intrinsic polarised intensity of those pixels, so the parity bound
// (1e-4 x map RMS) asks for ~1e-9 relative accuracy of sum_n n_e B_LOS -- below fp32 round-off (measured:
// an fp32 integrand, however carefully evaluated, gives 2-7e-4).  The accuracy that
// IS needed (~1e-10) is far below what libm's float64 functions deliver, so every function here is a
// range reduction plus a polynomial just long enough for 1e-11: ~12 DFMA per exp, ~19 per sincos,
// 2 per reciprocal / 5 per square root (MUFU seed + one Newton step).  B200 issues 64 DFMA/clk/SM on a
// pipe separate from the FP32 and XU pipes, so this chain overlaps with the per-frequency fp32 work.
#pragma once
#include "synax_device.cuh"

namespace synax {

// 2^x, x <= ~60; relative error < 1e-11 (Taylor in f ln2, |f| <= 1/2, degree 9).  Returns 0 below 2^-1000.
__device__ __forceinline__ double exp2_d(double x) {
  const double kMagic = 6755399441055744.0;  // 1.5 * 2^52
  const double t = x + kMagic;
  const int k = __double2loint(t);
  const double f = x - (t - kMagic);         // exact, |f| <= 1/2
  double p = 1.0178086009239699e-7;          // ln2^9 / 9!
  p = fma(p, f, 1.3215486790144307e-6);
  p = fma(p, f, 1.5252733804059841e-5);
  p = fma(p, f, 1.5403530393381609e-4);
  p = fma(p, f, 1.3333558146428443e-3);
  p = fma(p, f, 9.6181291076284772e-3);
  p = fma(p, f, 5.5504108664821580e-2);
  p = fma(p, f, 2.4022650695910071e-1);
  p = fma(p, f, 6.9314718055994531e-1);
  p = fma(p, f, 1.0);
  const int hi = __double2hiint(p) + (k << 20);
  return (x < -1000.0) ? 0.0 : __hiloint2double(hi, __double2loint(p));
}

// 1/x for finite x with |x| in fp32 range: MUFU.RCP seed (1e-7) + one Newton step (-> 1e-14)
__device__ __forceinline__ double rcp_d(double x) {
  const double y = (double)mufu_rcp((float)x);
  return fma(y, fma(-x, y, 1.0), y);
}

// 1/sqrt(x) for x > 0 in fp32 range: MUFU.RSQ seed + one Newton step (-> ~4e-15)
__device__ __forceinline__ double rsqrt_d(double x) {
  const double y = (double)mufu_rsqrt((float)x);
  const double e = fma(-x * y, y, 1.0);
  return fma(0.5 * y, e, y);
}

// sin and cos, |x| < ~1e6; absolute error < 1e-11 (reduction by pi/2, odd degree 11 / even degree 12)
__device__ __forceinline__ void sincos_d(double x, double& s, double& c) {
  const double kMagic = 6755399441055744.0;
  const double t = fma(x, 0.63661977236758134308, kMagic);
  const int q = __double2loint(t);
  const double k = t - kMagic;
  double r = fma(k, -1.5707963267948966192, x);
  r = fma(k, -6.1232339957367658860e-17, r);
  const double r2 = r * r;
  double ps = -2.5052108385441718775e-8;      // -1/11!
  ps = fma(ps, r2, 2.7557319223985890653e-6);
  ps = fma(ps, r2, -1.9841269841269841270e-4);
  ps = fma(ps, r2, 8.3333333333333333333e-3);
  ps = fma(ps, r2, -1.6666666666666666667e-1);
  ps = fma(ps * r2, r, r);
  double pc = 2.0876756987868098979e-9;       // 1/12!
  pc = fma(pc, r2, -2.7557319223985890653e-7);
  pc = fma(pc, r2, 2.4801587301587301587e-5);
  pc = fma(pc, r2, -1.3888888888888888889e-3);
  pc = fma(pc, r2, 4.1666666666666666667e-2);
  pc = fma(pc, r2, -0.5);
  pc = fma(pc, r2, 1.0);
  const double ss = (q & 1) ? pc : ps;
  const double cs = (q & 1) ? ps : pc;
  s = (q & 2) ? -ss : ss;
  c = ((q + 1) & 2) ? -cs : cs;
}

// natural logarithm of a positive normal number; absolute error < 1e-11
__device__ __forceinline__ double log_d(double v) {
  int hi = __double2hiint(v);
  const int lo = __double2loint(v);
  int e = ((hi >> 20) & 0x7ff) - 1023;
  hi = (hi & 0x000fffff) | 0x3ff00000;         // mantissa in [1, 2)
  if (hi >= 0x3ff6a09f) { hi -= 0x00100000; ++e; }  // -> [sqrt(1/2), sqrt(2))
  const double m = __hiloint2double(hi, lo);
  const double s = (m - 1.0) * rcp_d(m + 1.0);
  const double s2 = s * s;
  double p = 1.0 / 13.0;
  p = fma(p, s2, 1.0 / 11.0);
  p = fma(p, s2, 1.0 / 9.0);
  p = fma(p, s2, 1.0 / 7.0);
  p = fma(p, s2, 1.0 / 5.0);
  p = fma(p, s2, 1.0 / 3.0);
  p = fma(p * s2, s, s);
  return fma((double)e, 0.69314718055994530942, 2.0 * p);
}

// Per-batch-element float64 constants of the analytic model (prologue_kernel writes them).
struct BatchConstsD {
  double b0, psi0, psi1, chi0;
  double k_hb;            // -log2(e)/h_b, 0 for DISC4
  double Bh, zh0, inv_rh, inv_wh;
  double ne0x4, k_her, k_hez;   // 4 ne0, -log2(e)/h_er, -2 log2(e)/|h_ez|
  int psi1_small;         // |psi1| <= 0.05: the MUFU lg2 (abs err 2e-7) is accurate enough for ln(rho/8)
};

// B (Cartesian, uG) and n_e (cm^-3) at a point, float64 with the short polynomials above.
// Eq.(12)-(13) P:L173-180 and the halo of DESIGN.md section 3 (S:App.C); `inside` as in the fp32 chain.
template <bool kHalo>
__device__ __forceinline__ void eval_analytic_d(const BatchConstsD& D, double x, double y, double z, double rho2,
                                                bool inside, double& Bx, double& By, double& Bz, double& ne) {
  const double kLog2e = 1.4426950408889634074;
  rho2 = fmax(rho2, 1.0e-30);
  const double ir = rsqrt_d(rho2);
  const double rho = rho2 * ir;
  const double xr = x * ir, yr = y * ir;
  const double az = fabs(z);
  double Brho = 0.0, Bphi = 0.0;
  Bz = 0.0;
  if (inside) {   // warp-divergent only at the annulus edges
    const double lr = D.psi1_small ? (double)((mufu_lg2((float)rho2) - 6.0f) * 0.34657359027997264f)
                                   : 0.5 * log_d(rho2 * 0.015625);
    double sp, cp, sc, cc;
    sincos_d(fma(D.psi1, lr, D.psi0), sp, cp);
    const double e1 = exp2_d(-2.0 * kLog2e * az);               // tanh|z| = (1 - e)/(1 + e)
    const double th = (1.0 - e1) * rcp_d(1.0 + e1);
    sincos_d(D.chi0 * copysign(th, z), sc, cc);
    double A = D.b0;
    if (D.k_hb != 0.0) A *= exp2_d(D.k_hb * (rho - 8.0));
    const double Acc = A * cc;
    Brho = Acc * cp; Bphi = Acc * sp; Bz = A * sc;
  }
  if (kHalo) {
    const double u = (az - D.zh0) * D.inv_wh;
    const double L = rcp_d(fma(u, u, 1.0));
    const double q = rho * D.inv_rh;
    Bphi = fma(D.Bh * L, q * exp2_d(kLog2e * (1.0 - q)), Bphi);
  }
  Bx = Brho * xr - Bphi * yr;
  By = fma(Brho, yr, Bphi * xr);
  const double ee = exp2_d(D.k_hez * az);                       // sech^2 w = 4 e / (1 + e)^2
  const double de = 1.0 + ee;
  ne = D.ne0x4 * exp2_d(D.k_her * rho) * ee * rcp_d(de * de);
}

}  // namespace synax
