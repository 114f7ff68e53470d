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

// Polynomial coefficients live in constant memory so that DFMA takes them as c[bank][offset] operands
// (a 64-bit literal costs two UMOV issue slots each time it is used).
static __constant__ double kExp2C[9] = {   // ln2^k / k!, k = 9 .. 1
    1.0178086009239699e-7, 1.3215486790144307e-6, 1.5252733804059841e-5, 1.5403530393381609e-4,
    1.3333558146428443e-3, 9.6181291076284772e-3, 5.5504108664821580e-2, 2.4022650695910071e-1,
    6.9314718055994531e-1};
static __constant__ double kSinC[5] = {-2.5052108385441718775e-8, 2.7557319223985890653e-6, -1.9841269841269841270e-4,
                                8.3333333333333333333e-3, -1.6666666666666666667e-1};
static __constant__ double kCosC[6] = {2.0876756987868098979e-9, -2.7557319223985890653e-7, 2.4801587301587301587e-5,
                                -1.3888888888888888889e-3, 4.1666666666666666667e-2, -0.5};
static __constant__ double kMiscC[4] = {6755399441055744.0,          // 1.5 * 2^52
                                 0.63661977236758134308,      // 2/pi
                                 -1.5707963267948966192,      // -pi/2 hi
                                 -6.1232339957367658860e-17}; // -pi/2 lo

// 2^x, x <= ~60; relative error < 1e-11 (Taylor in f ln2, |f| <= 1/2, degree 9).  Below 2^-1000 the result is
// pinned at ~2^-1000 (1e-301), which is zero for every use here.
__device__ __forceinline__ double exp2_d(double x) {
  const double t = x + kMiscC[0];
  const int k = max(__double2loint(t), -1000);
  const double f = x - (t - kMiscC[0]);         // exact, |f| <= 1/2 (garbage but finite when k was clamped)
  double p = kExp2C[0];
#pragma unroll
  for (int i = 1; i < 9; ++i) p = fma(p, f, kExp2C[i]);
  p = fma(p, f, 1.0);
  return __hiloint2double(__double2hiint(p) + (k << 20), __double2loint(p));
}

// MUFU.RCP64H / MUFU.RSQ64H: reciprocal and reciprocal square root seeds taken from the HIGH word of a double
// (20 mantissa bits, relative error ~1e-6, low word zero) -- one XU instruction, where a seed through fp32
// costs two F2F conversions on the same pipe besides (measured 13.6 lanes/clk/SM, 20 cycles each way).
__device__ __forceinline__ double mufu_rcp64h(double x) { double y; asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x)); return y; }
__device__ __forceinline__ double mufu_rsq64h(double x) { double y; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x)); return y; }

// 1/x for finite normal x: MUFU.RCP64H seed (~1e-6) + one Newton step (-> ~1e-12)
__device__ __forceinline__ double rcp_d(double x) {
  const double y = mufu_rcp64h(x);
  return fma(y, fma(-x, y, 1.0), y);
}

// 1/sqrt(x) for x >= 0: MUFU.RSQ64H seed + one Newton step (-> ~2e-12); finite (huge) for x -> 0
__device__ __forceinline__ double rsqrt_d(double x) {
  x = fmax(x, 1.0e-30);
  const double y = mufu_rsq64h(x);
  const double e = fma(-x * y, y, 1.0);
  return fma(0.5 * y, e, y);
}

// sin and cos, |x| < ~1e6; absolute error < 1e-11 (reduction by pi/2, odd degree 11 / even degree 12)
__device__ __forceinline__ void sincos_d(double x, double& s, double& c) {
  const double t = fma(x, kMiscC[1], kMiscC[0]);
  const int q = __double2loint(t);
  const double k = t - kMiscC[0];
  double r = fma(k, kMiscC[2], x);
  r = fma(k, kMiscC[3], r);
  const double r2 = r * r;
  double ps = kSinC[0];
#pragma unroll
  for (int i = 1; i < 5; ++i) ps = fma(ps, r2, kSinC[i]);
  ps = fma(ps * r2, r, r);
  double pc = kCosC[0];
#pragma unroll
  for (int i = 1; i < 6; ++i) pc = fma(pc, r2, kCosC[i]);
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

// N independent 2^x evaluated in lockstep: the compiler emits each Horner chain serially when they sit in
// different basic blocks (a DFMA depends on the previous one, ~8 cycles apart), so the exponentials of one
// sample are gathered here and advanced together -- N chains in flight instead of one.
template <int N>
__device__ __forceinline__ void exp2_d_n(const double (&x)[N], double (&out)[N]) {
  double f[N], p[N];
  int k[N];
#pragma unroll
  for (int j = 0; j < N; ++j) {
    const double t = x[j] + kMiscC[0];
    k[j] = max(__double2loint(t), -1000);
    f[j] = x[j] - (t - kMiscC[0]);
    p[j] = kExp2C[0];
  }
#pragma unroll
  for (int i = 1; i < 9; ++i) {
#pragma unroll
    for (int j = 0; j < N; ++j) p[j] = fma(p[j], f[j], kExp2C[i]);
  }
#pragma unroll
  for (int j = 0; j < N; ++j) {
    p[j] = fma(p[j], f[j], 1.0);
    out[j] = __hiloint2double(__double2hiint(p[j]) + (k[j] << 20), __double2loint(p[j]));
  }
}

// Per-batch-element float64 constants of the analytic model (prologue_kernel writes them).
struct BatchConstsD {
  double b0, psi0, psi1, chi0;
  double k_hb;            // -log2(e)/h_b, 0 for DISC4
  double Bh, zh0, inv_rh, inv_wh;
  double ne0x4, k_her, k_hez;   // 4 ne0, -log2(e)/h_er, -2 log2(e)/|h_ez|
  int psi1_small;         // |psi1| <= 0.05 and |psi1| x (bound on one sample's rotation) x sqrt(n_los) <= 10 rad: the MUFU lg2 is accurate enough for ln(rho/8)
  int angles_small;       // |psi0| + |psi1| <= pi/4 and |chi0| <= pi/4: psi (|ln(rho/8)| < 1 inside the annulus) and
                          // chi = chi0 tanh z never leave [-pi/4, pi/4], so sincos needs no range reduction
  int hez_is_one;         // h_ez == 1 kpc exactly: exp(-2|z|/h_ez) is the tanh(z / 1 kpc) exponential, evaluated once
  double sb0[4], spsi0[4], spsi1[4], schi0[4];   // STACK16 only: the four stacked spirals (b0 already times its weight)
};

// M independent sincos in lockstep (same polynomials as sincos_d)
template <int M>
__device__ __forceinline__ void sincos_d_n(const double (&x)[M], double (&s)[M], double (&c)[M]) {
  double r[M], r2[M], ps[M], pc[M];
  int q[M];
#pragma unroll
  for (int j = 0; j < M; ++j) {
    const double t = fma(x[j], kMiscC[1], kMiscC[0]);
    q[j] = __double2loint(t);
    const double k = t - kMiscC[0];
    r[j] = fma(k, kMiscC[3], fma(k, kMiscC[2], x[j]));
    r2[j] = r[j] * r[j];
    ps[j] = kSinC[0]; pc[j] = kCosC[0];
  }
#pragma unroll
  for (int i = 1; i < 6; ++i) {
#pragma unroll
    for (int j = 0; j < M; ++j) {
      if (i < 5) ps[j] = fma(ps[j], r2[j], kSinC[i]);
      pc[j] = fma(pc[j], r2[j], kCosC[i]);
    }
  }
#pragma unroll
  for (int j = 0; j < M; ++j) {
    ps[j] = fma(ps[j] * r2[j], r[j], r[j]);
    pc[j] = fma(pc[j], r2[j], 1.0);
    const double ss = (q[j] & 1) ? pc[j] : ps[j];
    const double cs = (q[j] & 1) ? ps[j] : pc[j];
    s[j] = (q[j] & 2) ? -ss : ss;
    c[j] = ((q[j] + 1) & 2) ? -cs : cs;
  }
}

// the same polynomials without range reduction, for arguments known to lie in [-pi/4, pi/4]
template <int M>
__device__ __forceinline__ void sincos_d_small_n(const double (&x)[M], double (&s)[M], double (&c)[M]) {
  double r2[M], ps[M], pc[M];
#pragma unroll
  for (int j = 0; j < M; ++j) { r2[j] = x[j] * x[j]; ps[j] = kSinC[0]; pc[j] = kCosC[0]; }
#pragma unroll
  for (int i = 1; i < 6; ++i) {
#pragma unroll
    for (int j = 0; j < M; ++j) {
      if (i < 5) ps[j] = fma(ps[j], r2[j], kSinC[i]);
      pc[j] = fma(pc[j], r2[j], kCosC[i]);
    }
  }
#pragma unroll
  for (int j = 0; j < M; ++j) {
    s[j] = fma(ps[j] * r2[j], x[j], x[j]);
    c[j] = fma(pc[j], r2[j], 1.0);
  }
}

// B (Cartesian, uG) and n_e (cm^-3) at M consecutive samples of one sightline, float64 with the short
// polynomials above.  Eq.(12)-(13) P:L173-180 and the halo of DESIGN.md section 3 (S:App.C); `inside` as in
// the fp32 chain.  Everything is advanced in lockstep over the M samples and over the independent functions
// of one sample (the kernel is bound by dependent-issue latency, not by a pipe: ncu "wait" stalls), with two
// straight-line variants: some sample inside the disc annulus (the others masked) / all outside.
template <bool kHalo, int M>
__device__ __forceinline__ void eval_analytic_dm(const BatchConstsD& D, const double (&x)[M], const double (&y)[M],
                                                 const double (&z)[M], const double (&rho2)[M], const bool (&inside)[M],
                                                 double (&Bx)[M], double (&By)[M], double (&Bz)[M], double (&ne)[M]) {
  const double kLog2e = 1.4426950408889634074;
  double ir[M], rho[M], az[M], q[M], u[M];
  bool any = false;
#pragma unroll
  for (int j = 0; j < M; ++j) {
    ir[j] = rsqrt_d(rho2[j]);
    rho[j] = rho2[j] * ir[j];
    az[j] = fabs(z[j]);
    q[j] = rho[j] * D.inv_rh;
    u[j] = (az[j] - D.zh0) * D.inv_wh;
    any = any || inside[j];
  }
  double Brho[M], Bphi[M], ee[M], er[M], eh[M];
  if (any) {
    // exponentials of this sample in lockstep: n_e's two, tanh's (skipped when it IS n_e's z-exponential), halo's two
    constexpr int NE = kHalo ? 5 : 3;
    double xs[NE * M], o[NE * M];
#pragma unroll
    for (int j = 0; j < M; ++j) {
      xs[j] = D.k_hez * az[j];
      xs[M + j] = D.k_her * rho[j];
      if (kHalo) {
        xs[2 * M + j] = kLog2e * (1.0 - q[j]);
        xs[3 * M + j] = D.k_hb * (rho[j] - 8.0);
        xs[4 * M + j] = -2.0 * kLog2e * az[j];
      } else {
        xs[2 * M + j] = -2.0 * kLog2e * az[j];
      }
    }
    if (D.hez_is_one) {
      double xr[(NE - 1) * M], orr[(NE - 1) * M];
#pragma unroll
      for (int j = 0; j < (NE - 1) * M; ++j) xr[j] = xs[j];
      exp2_d_n<(NE - 1) * M>(xr, orr);
#pragma unroll
      for (int j = 0; j < (NE - 1) * M; ++j) o[j] = orr[j];
#pragma unroll
      for (int j = 0; j < M; ++j) o[(NE - 1) * M + j] = orr[j];
    } else {
      exp2_d_n<NE * M>(xs, o);
    }
    double ang[2 * M], sn[2 * M], cs[2 * M], A[M];
#pragma unroll
    for (int j = 0; j < M; ++j) {
      ee[j] = o[j]; er[j] = o[M + j];
      const double e1 = o[(NE - 1) * M + j];
      eh[j] = kHalo ? o[2 * M + j] : 0.0;
      A[j] = inside[j] ? (kHalo ? D.b0 * o[3 * M + j] : D.b0) : 0.0;
      const double lr = D.psi1_small ? (double)((mufu_lg2((float)rho2[j]) - 6.0f) * 0.34657359027997264f)
                                     : 0.5 * log_d(rho2[j] * 0.015625);
      const double th = (1.0 - e1) * rcp_d(1.0 + e1);           // tanh|z| = (1 - e)/(1 + e)
      ang[j] = fma(D.psi1, lr, D.psi0);
      ang[M + j] = D.chi0 * copysign(th, z[j]);
    }
    if (D.angles_small) sincos_d_small_n<2 * M>(ang, sn, cs);
    else sincos_d_n<2 * M>(ang, sn, cs);
#pragma unroll
    for (int j = 0; j < M; ++j) {
      const double Acc = A[j] * cs[M + j];
      Brho[j] = Acc * cs[j]; Bphi[j] = Acc * sn[j]; Bz[j] = A[j] * sn[M + j];
    }
  } else {
    constexpr int NE = kHalo ? 3 : 2;
    double xs[NE * M], o[NE * M];
#pragma unroll
    for (int j = 0; j < M; ++j) {
      xs[j] = D.k_hez * az[j];
      xs[M + j] = D.k_her * rho[j];
      if (kHalo) xs[2 * M + j] = kLog2e * (1.0 - q[j]);
    }
    exp2_d_n<NE * M>(xs, o);
#pragma unroll
    for (int j = 0; j < M; ++j) {
      ee[j] = o[j]; er[j] = o[M + j];
      eh[j] = kHalo ? o[2 * M + j] : 0.0;
      Brho[j] = 0.0; Bphi[j] = 0.0; Bz[j] = 0.0;
    }
  }
#pragma unroll
  for (int j = 0; j < M; ++j) {
    const double de = 1.0 + ee[j];                              // sech^2 w = 4 e / (1 + e)^2
    double ide2;                                                // 1 / (1 + e)^2
    if (kHalo) {   // one reciprocal serves the halo's Lorentzian and sech^2
      const double lu = fma(u[j], u[j], 1.0), de2 = de * de;
      const double inv = rcp_d(lu * de2);
      ide2 = inv * lu;
      Bphi[j] = fma(D.Bh * (inv * de2), q[j] * eh[j], Bphi[j]);
    } else {
      ide2 = rcp_d(de * de);
    }
    const double xr = x[j] * ir[j], yr = y[j] * ir[j];
    Bx[j] = Brho[j] * xr - Bphi[j] * yr;
    By[j] = fma(Brho[j], yr, Bphi[j] * xr);
    ne[j] = D.ne0x4 * er[j] * ee[j] * ide2;
  }
}

// STACK16 (Eq.(16)), float64: shared geometry, n_e's exponentials and tanh, then eight sincos in lockstep.
__device__ __forceinline__ void eval_stack16_d(const BatchConstsD& D, double x, double y, double z, double rho2,
                                               bool inside, double& Bx, double& By, double& Bz, double& ne) {
  const double kLog2e = 1.4426950408889634074;
  const double ir = rsqrt_d(rho2);
  const double rho = rho2 * ir;
  const double xr = x * ir, yr = y * ir;
  const double az = fabs(z);
  double B[3] = {0.0, 0.0, 0.0};
  double ee, er;
  if (inside) {
    const double xs[3] = {D.k_hez * az, D.k_her * rho, -2.0 * kLog2e * az};
    double o[3];
    exp2_d_n<3>(xs, o);
    ee = o[0]; er = o[1];
    const double th = copysign((1.0 - o[2]) * rcp_d(1.0 + o[2]), z);
    const double lr = 0.5 * log_d(rho2 * 0.015625);      // Table 3's psi1 are O(1): the MUFU lg2 is not enough
    double ang[8], sn[8], cs[8];
#pragma unroll
    for (int k = 0; k < 4; ++k) { ang[k] = fma(D.spsi1[k], lr, D.spsi0[k]); ang[4 + k] = D.schi0[k] * th; }
    sincos_d_n<8>(ang, sn, cs);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const double A = D.sb0[k];
      const double Brho = A * cs[k] * cs[4 + k], Bphi = A * sn[k] * cs[4 + k];
      const double comp[3] = {Brho * xr - Bphi * yr, fma(Brho, yr, Bphi * xr), A * sn[4 + k]};
#pragma unroll
      for (int c = 0; c < 3; ++c) B[c] += comp[stack_src(k, c)];
    }
  } else {
    const double xs[2] = {D.k_hez * az, D.k_her * rho};
    double o[2];
    exp2_d_n<2>(xs, o);
    ee = o[0]; er = o[1];
  }
  Bx = B[0]; By = B[1]; Bz = B[2];
  const double de = 1.0 + ee;
  ne = D.ne0x4 * er * ee * rcp_d(de * de);
}

}  // namespace synax
