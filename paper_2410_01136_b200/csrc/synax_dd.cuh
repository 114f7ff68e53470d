// synax_dd.cuh -- the paper's own arithmetic: EVERY step of the path in float64 (section 2.4: "the default
// precision is double ... for all examples").  Entry points synax_forward_f64 / synax_vjp_f64 (include/synax.h):
// float64 parameters in, float64 maps / gradients out, CUDA's float64 math library throughout (exp, log, sincos,
// tanh, cosh, pow, sincospi: <= 2 ulp), no MUFU approximations, no tiles, no mixed precision.  Same sightline <-> lane
// mapping as the fp32 kernels (G lanes own consecutive chunks; the partial Q + iU of a chunk is rotated once by the
// Faraday angle of the preceding lanes) and the same adjoint (prefix form of the reverse scan, synax_vjp.cuh,
// instantiated with R = double).  Analytic models only.
#pragma once
#include "synax_forward.cuh"
#include "synax_vjp.cuh"

namespace synax {

// per-batch constants in float64 (prologue64_kernel)
struct BatchConsts64 {
  double p[kMaxAnalyticParams];   // canonical FULL16 order; DISC4 / STACK16: densities and alpha from aux
  double sp[16];                  // STACK16: the four spirals
  double uB[3], uN0, une;         // UNIFORM
  double inv_wh, inv_rh;
  double alpha, q_exp, pi_frac, dpi_dalpha_over_pi, dlnA_dalpha;
  int alpha_is_3;
  double coefI[kMaxFreq], coefP[kMaxFreq];   // c_f(alpha) Delta, Pi c_f(alpha) Delta
};

struct TriadD {
  double nx, ny, nz, eNx, eNy, eNz, eEx, eEy;
  double scale, scalef;   // (scalef: the name the shared gradient structs use)
};
__device__ __forceinline__ TriadD load_triad_d(const Geometry& geo, int64_t pix) {
  const double4 d = *reinterpret_cast<const double4*>(geo.dirs + 4 * pix);   // cos l, sin l, cos b, sin b
  TriadD t;
  t.nx = d.z * d.x; t.ny = d.z * d.y; t.nz = d.w;
  t.eNx = -d.w * d.x; t.eNy = -d.w * d.y; t.eNz = d.z;
  t.eEx = -d.y; t.eEy = d.x;
  t.scale = geo.path ? geo.path[pix] : 1.0;
  t.scalef = t.scale;
  return t;
}

struct SampleDD { double Bpar, BN, BE, N0, ne; };
struct AuxDD {   // what the adjoint needs again (same names as AnalyticAux)
  double rho, xr, yr, lr, sp, cp, sc, cc, t, A, u, L, R, thz, thez, N0u, neu;
};
struct StackAuxDD {
  double xr, yr, lr, t, mask;
  double sp[4], cp[4], sc[4], cc[4];
};

__device__ __forceinline__ double sech2_d(double w) { const double c = cosh(w); return 1.0 / (c * c); }

__device__ __forceinline__ void project_dd(const TriadD& T, double Bx, double By, double Bz, SampleDD& S) {
  S.Bpar = fma(Bx, T.nx, fma(By, T.ny, Bz * T.nz));          // B.n, signed (S:C-2#3)
  S.BN = fma(Bx, T.eNx, fma(By, T.eNy, Bz * T.eNz));         // Eq.(8) numerator
  S.BE = fma(Bx, T.eEx, By * T.eEy);                         // Eq.(8) denominator (S:C-2#4)
}

// Eq.(12)-(13) P:L173-180 and the halo / radial scale of DESIGN.md section 3 (S:App.C)
template <bool kHalo>
__device__ __forceinline__ void eval_analytic_dd(const BatchConsts64& P, const TriadD& T, double x, double y, double z,
                                                 SampleDD& S, AuxDD& a) {
  const double rho2 = fma(x, x, y * y);
  a.rho = sqrt(rho2);
  const bool inside = (rho2 > 9.0) && (rho2 < 400.0);
  const double ir = a.rho > 0.0 ? 1.0 / a.rho : 0.0;
  a.xr = x * ir; a.yr = y * ir;
  a.lr = a.rho > 0.0 ? log(a.rho * 0.125) : 0.0;
  sincos(fma(P.p[2], a.lr, P.p[1]), &a.sp, &a.cp);
  a.t = tanh(z);
  sincos(P.p[3] * a.t, &a.sc, &a.cc);
  a.A = inside ? (kHalo ? exp(-(a.rho - 8.0) / P.p[4]) : 1.0) : 0.0;
  const double Ab = P.p[0] * a.A;
  const double Brho = Ab * a.cp * a.cc;
  double Bphi = Ab * a.sp * a.cc;
  const double Bz = Ab * a.sc;
  if (kHalo) {
    a.u = (fabs(z) - P.p[6]) * P.inv_wh;
    a.L = 1.0 / fma(a.u, a.u, 1.0);
    const double q = a.rho * P.inv_rh;
    a.R = q * exp(1.0 - q);
    Bphi = fma(P.p[5] * a.L, a.R, Bphi);
  } else {
    a.u = 0.0; a.L = 0.0; a.R = 0.0;
  }
  project_dd(T, Brho * a.xr - Bphi * a.yr, fma(Brho, a.yr, Bphi * a.xr), Bz, S);
  a.N0u = exp(-a.rho / P.p[10]) * sech2_d(z / P.p[11]);
  a.thz = tanh(z / P.p[11]);
  S.N0 = P.p[9] * a.N0u;
  a.neu = exp(-a.rho / P.p[14]) * sech2_d(z / P.p[15]);
  a.thez = tanh(z / P.p[15]);
  S.ne = P.p[13] * a.neu;
}

// Eq.(16) P:L283-289 (weights and component permutations as printed; C-2#21)
__device__ __forceinline__ void eval_stack16_dd(const BatchConsts64& P, const TriadD& T, double x, double y, double z,
                                                SampleDD& S, StackAuxDD& a) {
  const double rho2 = fma(x, x, y * y), rho = sqrt(rho2);
  const double ir = rho > 0.0 ? 1.0 / rho : 0.0;
  a.xr = x * ir; a.yr = y * ir;
  a.lr = rho > 0.0 ? log(rho * 0.125) : 0.0;
  a.t = tanh(z);
  a.mask = ((rho2 > 9.0) && (rho2 < 400.0)) ? 1.0 : 0.0;
  double B[3] = {0.0, 0.0, 0.0};
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    sincos(fma(P.sp[4 * k + 2], a.lr, P.sp[4 * k + 1]), &a.sp[k], &a.cp[k]);
    sincos(P.sp[4 * k + 3] * a.t, &a.sc[k], &a.cc[k]);
    const double A = a.mask * stack_w_d(k) * P.sp[4 * k];
    const double Brho = A * a.cp[k] * a.cc[k], Bphi = A * a.sp[k] * a.cc[k];
    const double comp[3] = {Brho * a.xr - Bphi * a.yr, fma(Brho, a.yr, Bphi * a.xr), A * a.sc[k]};
#pragma unroll
    for (int c = 0; c < 3; ++c) B[c] += comp[stack_src(k, c)];
  }
  project_dd(T, B[0], B[1], B[2], S);
  S.N0 = P.p[9] * exp(-rho / P.p[10]) * sech2_d(z / P.p[11]);
  S.ne = P.p[13] * exp(-rho / P.p[14]) * sech2_d(z / P.p[15]);
}

// cos, sin of the Faraday angle 2 pi k_turn S, the turn count reduced before the trigonometric call
__device__ __forceinline__ void faraday_phasor_d(double k_turn, double S, double& c, double& s) {
  double t = k_turn * S;
  t -= rint(t);
  sincospi(2.0 * t, &s, &c);
}

struct DDArgs {
  Geometry geo;
  const BatchConsts64* bc;
  int batch, f0, n_freq_total;
  ScalarGridDesc sg_ne, sg_n0;
  double* I; double* Q; double* U;                        // forward
  const double* dI; const double* dQ; const double* dU;   // adjoint (any may be null)
  double* partial;                                        // adjoint: [batch][n_blocks][16]
  int n_blocks, accumulate;
};

// one sample: fields, projections (shared by the forward and the adjoint)
template <int CODE>
__device__ __forceinline__ void sample_dd(const DDArgs& A, const BatchConsts64& P, const TriadD& T, double x, double y,
                                          double z, SampleDD& S, AuxDD& aux, StackAuxDD& sa) {
  if constexpr (CODE == kUniform) {
    project_dd(T, P.uB[0], P.uB[1], P.uB[2], S);
    S.N0 = P.uN0; S.ne = P.une;
  } else if constexpr (CODE == kStack16) {
    eval_stack16_dd(P, T, x, y, z, S, sa);
  } else {
    eval_analytic_dd<CODE == kAnalyticFull>(P, T, x, y, z, S, aux);
  }
  if constexpr (CODE == kAnalyticDisc || CODE == kStack16) {
    if (A.sg_ne.g) S.ne = scalar_grid_at<double>(A.sg_ne, x, y, z);
    if (A.sg_n0.g) S.N0 = scalar_grid_at<double>(A.sg_n0, x, y, z);
  }
  S.ne *= T.scale;   // n_e enters only through the Faraday integrand n_e B_LOS Delta_i
}

// ------------------------------------------------------------------------------------------------
// Forward (A2-A8, A12), float64.  grid.x covers batch * npix * G threads.
// ------------------------------------------------------------------------------------------------
template <int CODE, int G, int NF>
__global__ void __launch_bounds__(kBlock) forward_dd_kernel(const __grid_constant__ DDArgs A, const __grid_constant__ FreqTab ft) {
  const int64_t tid = (int64_t)blockIdx.x * kBlock + threadIdx.x;
  const int g = (int)(tid % G);
  int64_t sl = tid / G;
  const int64_t n_sl = A.geo.npix * A.batch;
  const bool valid = sl < n_sl;
  if (!valid) sl = n_sl - 1;   // keep the lane alive for the shuffles
  const int b = (int)(sl / A.geo.npix);
  const int64_t pix = sl - (int64_t)b * A.geo.npix;
  const BatchConsts64& P = A.bc[b];
  const TriadD T = load_triad_d(A.geo, pix);
  const int C = (A.geo.n_los + G - 1) / G;
  const int n0 = g * C, n1 = min(n0 + C, A.geo.n_los);
  const double delta = A.geo.delta * T.scale;
  double accI = 0.0, accQ[NF], accU[NF];
#pragma unroll
  for (int f = 0; f < NF; ++f) { accQ[f] = 0.0; accU[f] = 0.0; }
  double S_loc = 0.0;   // sum of n_e B_LOS over this lane's finished samples
  for (int n = n0; n < n1; ++n) {
    const double s_d = ((double)n + 0.5) * delta;                                  // A2: midpoint
    const double x = fma(s_d, T.nx, A.geo.obs[0]), y = fma(s_d, T.ny, A.geo.obs[1]), z = fma(s_d, T.nz, A.geo.obs[2]);
    SampleDD S; AuxDD aux; StackAuxDD sa;
    sample_dd<CODE>(A, P, T, x, y, z, S, aux, sa);
    const double bn2 = S.BN * S.BN, be2 = S.BE * S.BE, Bt2 = bn2 + be2;
    double w = S.N0;                                                               // A5: e~ = N0 (B_perp^2)^((alpha+1)/4)
    if (!P.alpha_is_3) w = Bt2 > 0.0 ? S.N0 * pow(Bt2, P.q_exp) : 0.0;
    accI += w * Bt2;
    const double a = w * (be2 - bn2), bq = w * (2.0 * S.BE * S.BN);                // e~ e^{2 i chi0}, no atan2
    const double gn = S.ne * S.Bpar;
    const double ph = fma(0.5, gn, S_loc);                                         // A6: half-cell (S:C-2#5)
    S_loc += gn;
#pragma unroll
    for (int f = 0; f < NF; ++f) {                                                 // A7
      double c, s;
      faraday_phasor_d(ft.k_turn[f], ph, c, s);
      accQ[f] = fma(a, c, fma(-bq, s, accQ[f]));
      accU[f] = fma(a, s, fma(bq, c, accU[f]));
    }
  }
  if (G > 1) {                                                                     // A8: combine the lanes
    const double off = group_exclusive_scan<G>(S_loc, g);
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      double c, s;
      faraday_phasor_d(ft.k_turn[f], off, c, s);
      const double q = accQ[f] * c - accU[f] * s;
      accU[f] = fma(accQ[f], s, accU[f] * c);
      accQ[f] = group_sum_d<G>(q);
      accU[f] = group_sum_d<G>(accU[f]);
    }
    accI = group_sum_d<G>(accI);
  }
  if (valid && g == 0) {
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const int64_t o = ((int64_t)b * A.n_freq_total + A.f0 + f) * A.geo.npix + pix;
      A.I[o] = P.coefI[A.f0 + f] * T.scale * accI;
      A.Q[o] = P.coefP[A.f0 + f] * T.scale * accQ[f];
      A.U[o] = P.coefP[A.f0 + f] * T.scale * accU[f];
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Adjoint (A9-A11), float64: one forward-order sweep, nothing stored per sample.  grid = (n_blocks, batch).
// ------------------------------------------------------------------------------------------------
template <int CODE, int G, int NF>
__global__ void __launch_bounds__(kBlock) vjp_dd_kernel(const __grid_constant__ DDArgs A, const __grid_constant__ FreqTab ft) {
  constexpr bool kAlpha = (CODE == kAnalyticFull || CODE == kUniform);
  const int b = blockIdx.y;
  const int64_t tid = (int64_t)blockIdx.x * kBlock + threadIdx.x;
  const int g = (int)(tid % G);
  int64_t pix = tid / G;
  const bool valid = pix < A.geo.npix;
  if (!valid) pix = A.geo.npix - 1;
  const BatchConsts64& P = A.bc[b];
  const TriadD T = load_triad_d(A.geo, pix);
  const int C = (A.geo.n_los + G - 1) / G;
  const int n0 = g * C, n1 = min(n0 + C, A.geo.n_los);
  const double delta = A.geo.delta * T.scale;
  const double kTwoPi = 6.283185307179586476925;

  // Faraday sum of the preceding lanes
  double off = 0.0;
  if (G > 1) {
    double Sl = 0.0;
    for (int n = n0; n < n1; ++n) {
      const double s_d = ((double)n + 0.5) * delta;
      const double x = fma(s_d, T.nx, A.geo.obs[0]), y = fma(s_d, T.ny, A.geo.obs[1]), z = fma(s_d, T.nz, A.geo.obs[2]);
      SampleDD S; AuxDD aux; StackAuxDD sa;
      sample_dd<CODE>(A, P, T, x, y, z, S, aux, sa);
      Sl += S.ne * S.Bpar;
    }
    off = group_exclusive_scan<G>(Sl, g);
  }
  // cotangents, coefficients folded in and rotated by the angle of the preceding lanes (zero for padded lanes)
  double cI = 0.0, cIa = 0.0, rq[NF], ru[NF], kr[NF], lnu[NF];
#pragma unroll
  for (int f = 0; f < NF; ++f) {
    const int64_t o = ((int64_t)b * A.n_freq_total + A.f0 + f) * A.geo.npix + pix;
    const double vI = (valid && A.dI) ? A.dI[o] * P.coefI[A.f0 + f] * T.scale : 0.0;
    lnu[f] = log(ft.freq[f]);
    cI += vI;
    cIa = fma(vI, P.dlnA_dalpha - 0.5 * lnu[f], cIa);
    const double q = (valid && A.dQ) ? A.dQ[o] * P.coefP[A.f0 + f] * T.scale : 0.0;
    const double u = (valid && A.dU) ? A.dU[o] * P.coefP[A.f0 + f] * T.scale : 0.0;
    double c, s;
    faraday_phasor_d(ft.k_turn[f], off, c, s);
    rq[f] = q * c + u * s; ru[f] = u * c - q * s;    // Qb cos(t0 + t) + Ub sin(t0 + t) = Qb' cos t + Ub' sin t
    kr[f] = kTwoPi * ft.k_turn[f];
  }
  typename GradOf<CODE, double>::type acc;
  acc.zero();
  double gAlpha = 0.0, sumE = 0.0, gPol = 0.0, Pl = 0.0, S_loc = 0.0;
  const double cPol = kAlpha ? P.dlnA_dalpha + P.dpi_dalpha_over_pi : 0.0;
  for (int n = n0; n < n1; ++n) {
    const double s_d = ((double)n + 0.5) * delta;
    const double x = fma(s_d, T.nx, A.geo.obs[0]), y = fma(s_d, T.ny, A.geo.obs[1]), z = fma(s_d, T.nz, A.geo.obs[2]);
    SampleDD S; AuxDD aux; StackAuxDD sa;
    sample_dd<CODE>(A, P, T, x, y, z, S, aux, sa);
    const double bn2 = S.BN * S.BN, be2 = S.BE * S.BE, Bt2 = bn2 + be2;
    double w = 1.0, lnB = 0.0;
    if (kAlpha || !P.alpha_is_3) {
      lnB = Bt2 > 0.0 ? log(Bt2) : 0.0;
      if (!P.alpha_is_3) w = Bt2 > 0.0 ? exp(P.q_exp * lnB) : 0.0;
    }
    const double M = w * S.N0;
    const double d2 = be2 - bn2, p2 = 2.0 * S.BE * S.BN;
    const double a = M * d2, bq = M * p2;
    const double gn = S.ne * S.Bpar;
    const double ph = fma(0.5, gn, S_loc);
    S_loc += gn;
    double Xc = 0.0, Xs = 0.0, Yc = 0.0, Ys = 0.0, Zc = 0.0, Zs = 0.0;
#pragma unroll
    for (int f = 0; f < NF; ++f) {                 // A9: fan-out
      double c, s;
      faraday_phasor_d(ft.k_turn[f], ph, c, s);
      const double u = fma(rq[f], c, ru[f] * s), v = fma(ru[f], c, -rq[f] * s);
      Xc += u; Xs += v;
      Yc = fma(kr[f], u, Yc); Ys = fma(kr[f], v, Ys);
      if (kAlpha) { Zc = fma(lnu[f], u, Zc); Zs = fma(lnu[f], v, Zs); }
    }
    if (kAlpha) gPol = fma(a, fma(cPol, Xc, -0.5 * Zc), fma(bq, fma(cPol, Xs, -0.5 * Zs), gPol));
    const double K = fma(cI, Bt2, fma(Xc, d2, Xs * p2));
    const double MK = M * K;
    sumE = fma(M, Bt2, sumE);
    if (kAlpha) gAlpha = fma(lnB, MK, gAlpha);
    const double Sbar = fma(a, Ys, -bq * Yc);      // cotangent of the Faraday sum at this sample
    Pl += Sbar;
    double tq_ = 0.0;
    if (!P.alpha_is_3 && Bt2 > 0.0) tq_ = P.q_exp * MK / Bt2;
    const double BEb = 2.0 * fma(M, fma(S.BE, cI + Xc, S.BN * Xs), S.BE * tq_);
    const double BNb = 2.0 * fma(M, fma(S.BN, cI - Xc, S.BE * Xs), S.BN * tq_);
    if constexpr (CODE == kUniform) acc.add(T, S, BNb, BEb, Sbar, w * K);
    else if constexpr (CODE == kStack16) acc.add(P, T, sa, S, BNb, BEb, Sbar);
    else acc.add(P, T, aux, S, z, BNb, BEb, Sbar, w * aux.N0u * K);
  }
  acc.template combine<G>(Pl, g);
  double out[16];
#pragma unroll
  for (int j = 0; j < 16; ++j) out[j] = 0.0;
  acc.finish(P, out);
  if (kAlpha) out[CODE == kUniform ? 5 : 12] = fma(0.25, gAlpha, fma(cIa, sumE, gPol));

  constexpr int NP = (CODE == kUniform) ? 6 : ((CODE == kAnalyticFull || CODE == kStack16) ? 16 : 4);
  __shared__ double red[kBlock / 32][16];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int j = 0; j < NP; ++j) {
    const double v = group_sum_d<32>(out[j]);
    if (lane == 0) red[wid][j] = v;
  }
  __syncthreads();
  if (threadIdx.x < NP) {
    double v = 0.0;
#pragma unroll
    for (int k = 0; k < kBlock / 32; ++k) v += red[k][threadIdx.x];
    double* dst = A.partial + ((size_t)b * A.n_blocks + blockIdx.x) * 16 + threadIdx.x;
    *dst = A.accumulate ? (*dst + v) : v;
  }
}

// partial[b][n_blocks][16] -> grad[b][n_params], fixed order (deterministic)
__global__ void vjp_dd_reduce_kernel(const double* __restrict__ partial, int n_blocks, int n_params, double* __restrict__ grad) {
  const int b = blockIdx.x;
  const int j = threadIdx.x & 15, part = threadIdx.x >> 4;
  __shared__ double sh[16][17];
  double s = 0.0;
  if (j < n_params)
    for (int k = part; k < n_blocks; k += 16) s += partial[((size_t)b * n_blocks + k) * 16 + j];
  sh[part][j] = s;
  __syncthreads();
  if (threadIdx.x < n_params) {
    double t = 0.0;
    for (int k = 0; k < 16; ++k) t += sh[k][threadIdx.x];
    grad[(size_t)b * n_params + threadIdx.x] = t;
  }
}

// Per-batch constants in float64: folds Eq.(2)'s prefactor, the Rayleigh-Jeans conversion (S:C-2#1) and the units
// into c_f(alpha) (as prologue_kernel does for the fp32 kernels, without rounding to fp32).
__global__ void prologue64_kernel(int code, const double* __restrict__ params, int n_params, int batch, AuxHost aux,
                                  FreqTab ft, double delta, BatchConsts64* __restrict__ out) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= batch) return;
  BatchConsts64 c;
  for (int j = 0; j < 16; ++j) { c.p[j] = 0.0; c.sp[j] = 0.0; }
  c.uB[0] = c.uB[1] = c.uB[2] = c.uN0 = c.une = 0.0;
  const double* q = params + (size_t)b * n_params;
  if (code == kAnalyticFull) {
    for (int j = 0; j < 16; ++j) c.p[j] = q[j];
  } else if (code == kUniform) {
    c.uB[0] = q[0]; c.uB[1] = q[1]; c.uB[2] = q[2]; c.uN0 = q[3]; c.une = q[4];
    c.p[12] = q[5];
    c.p[4] = c.p[7] = c.p[8] = c.p[10] = c.p[11] = c.p[14] = c.p[15] = 1.0;
  } else {
    if (code == kStack16) for (int j = 0; j < 16; ++j) c.sp[j] = q[j];
    if (code == kAnalyticDisc) for (int j = 0; j < 4; ++j) c.p[j] = q[j];
    c.p[4] = 1.0; c.p[6] = 0.0; c.p[7] = 1.0; c.p[8] = 1.0;
    c.p[9] = aux.v[0]; c.p[10] = aux.v[1]; c.p[11] = aux.v[2]; c.p[12] = aux.v[3];
    c.p[13] = aux.v[4]; c.p[14] = aux.v[5]; c.p[15] = aux.v[6];
  }
  const double alpha = c.p[12];
  c.alpha = alpha;
  c.inv_wh = 1.0 / c.p[8]; c.inv_rh = 1.0 / c.p[7];
  c.q_exp = (alpha - 3.0) * 0.25;
  c.pi_frac = (alpha + 1.0) / (alpha + 7.0 / 3.0);
  c.alpha_is_3 = alpha == 3.0 ? 1 : 0;
  c.dpi_dalpha_over_pi = 1.0 / (alpha + 1.0) - 1.0 / (alpha + 7.0 / 3.0);
  const double g1 = tgamma(alpha * 0.25 - 1.0 / 12.0), g2 = tgamma(alpha * 0.25 + 19.0 / 12.0);
  const double w = 4.0 * SYNAX_PI * SYNAX_ME * SYNAX_C / (3.0 * SYNAX_QE);
  const double A_I = sqrt(3.0) * SYNAX_QE * SYNAX_QE * SYNAX_QE / (8.0 * SYNAX_PI * SYNAX_ME * SYNAX_C * SYNAX_C) *
                     pow(w, (1.0 - alpha) * 0.5) * pow(2.0, (alpha + 1.0) * 0.5) / (alpha + 1.0) * g1 * g2;
  c.dlnA_dalpha = -0.5 * log(w) + 0.5 * log(2.0) - 1.0 / (alpha + 1.0) + 0.25 * digamma_d(alpha * 0.25 - 1.0 / 12.0) +
                  0.25 * digamma_d(alpha * 0.25 + 19.0 / 12.0) + 0.5 * log(1.0e-6);
  for (int f = 0; f < kMaxFreq; ++f) {
    if (f < ft.n_freq) {
      const double nu = ft.freq[f];
      const double TRJ = SYNAX_C * SYNAX_C / (2.0 * SYNAX_KB * nu * nu);
      const double cf = TRJ * A_I * pow(nu, (1.0 - alpha) * 0.5) * pow(1.0e-6, (alpha + 1.0) * 0.5) * SYNAX_KPC * delta;
      c.coefI[f] = cf; c.coefP[f] = cf * c.pi_frac;
    } else {
      c.coefI[f] = c.coefP[f] = 0.0;
    }
  }
  out[b] = c;
}

}  // namespace synax
