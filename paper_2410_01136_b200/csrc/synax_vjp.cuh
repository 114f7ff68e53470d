// synax_vjp.cuh -- adjoint (VJP) kernels for the analytic models: A9 cotangent fan-out, A10 reverse
// half-cell scan (vjp_kernel sweeps each sightline BACKWARDS, where that scan is a running sum; the batched and the
// float64 kernels sweep forwards with a running prefix per parameter), A11 field partials and
// reductions.  Nothing per SAMPLE is stored: the fields are recomputed; per SIGHTLINE the adjoint uses, when valid, the
// Faraday total (and tile bases) the plan's last forward left (VjpArgs::phi, phi_base).
#pragma once
#include <algorithm>
#include <type_traits>

#include "../../include/synax.h"
#include "synax_forward.cuh"

namespace synax {

// ------------------------------------------------------------------------------------------------
// Per-lane gradient accumulators.  The Faraday-coupled part of a parameter gradient is
//   sum_m gbar_m h_mj,   gbar_m = sum_{n>m} Sbar_n + Sbar_m / 2  (transposed half-cell scan, S:App.D.2),
// h_mj = d(n_e B_LOS)_m / d theta_j.  Swapping the order of summation,
//   sum_m gbar_m h_mj = sum_n Sbar_n (H_{j,n-1} + h_nj / 2),   H_{j,n} = sum_{m<=n} h_mj,
// which one forward-order sweep evaluates with a running prefix H_j per parameter and no subtraction of large
// terms (the earlier T - P_m form, S:App.D.4, lost the w_h component to cancellation on under-resolved
// sightlines: 1.1e-2 at nside 16 x 256 samples with the box clip).
// Amplitude parameters (b0, B_h, n0, ne0, ...) are accumulated with the UNIT-amplitude field, so their derivative
// needs no division by the parameter and stays finite when the amplitude is exactly zero.
// ------------------------------------------------------------------------------------------------
// rho/phi/z components of a Cartesian vector at a point with unit vectors rho_hat = (xr, yr, 0)
__device__ __forceinline__ float fma_r(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double fma_r(double a, double b, double c) { return fma(a, b, c); }

template <typename R>
__device__ __forceinline__ void to_cyl(R vx, R vy, R xr, R yr, R& vr, R& vp) {
  vr = fma_r(vx, xr, vy * yr);
  vp = fma_r(vy, xr, -vx * yr);
}

// g += d1 + Sbar * H (H = prefix over the earlier samples), then H += d2
template <typename R>
__device__ __forceinline__ void prefix_update(R& g, R& H, R Sbar, R d1, R d2) {
  g = fma_r(Sbar, H, g + d1);
  H += d2;
}

// lanes of a group own consecutive chunks: add Sbar-total-of-this-lane x (prefix H of the preceding lanes)
template <int G, typename R>
__device__ __forceinline__ void prefix_combine(R& g, R H, R Pl, int lane_in_group) {
  if (G > 1) g = fma_r((R)group_exclusive_scan<G>((double)H, lane_in_group), Pl, g);
}

// R = float (the fp32 kernels) or double (the all-float64 kernels of synax_dd.cuh); P, T, a, S are the matching structs
template <bool kFull, typename R = float>
struct AnalyticGrad {
  static constexpr int NB = kFull ? 9 : 4;
  R g[NB], H[NB];        // B parameters (unit amplitudes)
  R n1[3];               // CR density parameters (direct only)
  R ge[3], He[3];        // n_e parameters
  __device__ __forceinline__ void zero() {
#pragma unroll
    for (int j = 0; j < NB; ++j) { g[j] = (R)0.0; H[j] = (R)0.0; }
#pragma unroll
    for (int j = 0; j < 3; ++j) { n1[j] = (R)0.0; ge[j] = (R)0.0; He[j] = (R)0.0; }
  }
  // V1 = BbarN e_N + BbarE e_E + Sbar/2 ne n ; V2 = ne n ; MKu = N0bar * N0 / n0 ; a.A, a.N0u, a.neu: unit amplitudes
  template <typename PT, typename TT, typename AT, typename ST>
  __device__ __forceinline__ void add(const PT& P, const TT& T, const AT& a, const ST& S,
                                      R z, R BNb, R BEb, R Sbar, R MKu) {
    const R hs = (R)0.5 * Sbar * S.ne;
    const R v1x = fma_r(BNb, T.eNx, fma_r(BEb, T.eEx, hs * T.nx));
    const R v1y = fma_r(BNb, T.eNy, fma_r(BEb, T.eEy, hs * T.ny));
    const R v1z = fma_r(BNb, T.eNz, hs * T.nz);
    R v1r, v1p, nr, np;
    to_cyl(v1x, v1y, a.xr, a.yr, v1r, v1p);
    to_cyl(T.nx, T.ny, a.xr, a.yr, nr, np);
    const R v2r = S.ne * nr, v2p = S.ne * np, v2z = S.ne * T.nz;
    // disc: B = b0 A [cp cc rho_hat + sp cc phi_hat + sc z_hat], A = exp(-(rho-8)/h_b) inside the annulus.
    // Every accumulator first takes Sbar x (its prefix H), then the direct term is fused into its last FMAs.
#pragma unroll
    for (int j = 0; j < NB; ++j) g[j] = fma_r(Sbar, H[j], g[j]);
    const R Acc = a.A * a.cc, Asc = a.A * a.sc;
    {
      const R al1 = fma_r(a.cp, v1r, a.sp * v1p), al2 = fma_r(a.cp, v2r, a.sp * v2p);
      if (kFull) {
        const R d1 = fma_r(Acc, al1, Asc * v1z), d2 = fma_r(Acc, al2, Asc * v2z);   // (B_disc / b0) . V
        const R dr = a.rho - (R)8.0;
        g[0] += d1; H[0] += d2;
        g[4] = fma_r(dr, d1, g[4]); H[4] = fma_r(dr, d2, H[4]);                    // * b0 / h_b^2
      } else {
        g[0] = fma_r(Acc, al1, fma_r(Asc, v1z, g[0])); H[0] = fma_r(Acc, al2, fma_r(Asc, v2z, H[0]));
      }
      const R p1 = Acc * fma_r(a.cp, v1p, -a.sp * v1r);                            // (dB/dpsi0) / b0 . V
      const R p2 = Acc * fma_r(a.cp, v2p, -a.sp * v2r);
      g[1] += p1; H[1] += p2;
      g[2] = fma_r(a.lr, p1, g[2]); H[2] = fma_r(a.lr, p2, H[2]);
      const R tAcc = a.t * Acc, tAsc = a.t * Asc;                                  // (dB/dchi0) / b0 = t A (cc z_hat - sc (...))
      g[3] = fma_r(tAcc, v1z, fma_r(-tAsc, al1, g[3])); H[3] = fma_r(tAcc, v2z, fma_r(-tAsc, al2, H[3]));
    }
    if (kFull) {  // halo: B_h L R phi_hat
      const R LR = a.L * a.R;
      g[5] = fma_r(LR, v1p, g[5]); H[5] = fma_r(LR, v2p, H[5]);
      const R RuL2 = a.R * a.u * a.L * a.L;
      g[6] = fma_r(RuL2, v1p, g[6]); H[6] = fma_r(RuL2, v2p, H[6]);                // * 2 B_h / w_h
      const R q = LR * fma_r(a.rho, P.inv_rh, (R)-1.0);
      g[7] = fma_r(q, v1p, g[7]); H[7] = fma_r(q, v2p, H[7]);                      // * B_h / r_h
      const R Ru2L2 = RuL2 * a.u;
      g[8] = fma_r(Ru2L2, v1p, g[8]); H[8] = fma_r(Ru2L2, v2p, H[8]);              // * 2 B_h / w_h
    }
    if (kFull) {
      // N_0 = n0 exp(-rho/h_r) sech^2(z/h_z):  dN0/dn0 = N0/n0, /dh_r = N0 rho/h_r^2, /dh_z = N0 2 tanh(z/h_z) z/h_z^2
      n1[0] += MKu; n1[1] = fma_r(MKu, a.rho, n1[1]); n1[2] = fma_r(MKu * a.thz, z, n1[2]);
      const R h = T.scalef * a.neu * S.Bpar;   // d(ne Bpar Delta_i/Delta) / d ne0
      const R hh = (R)0.5 * Sbar * h;
#pragma unroll
      for (int j = 0; j < 3; ++j) ge[j] = fma_r(Sbar, He[j], ge[j]);
      ge[0] += hh; He[0] += h;
      ge[1] = fma_r(hh, a.rho, ge[1]); He[1] = fma_r(h, a.rho, He[1]);
      const R tz = a.thez * z;
      ge[2] = fma_r(hh, tz, ge[2]); He[2] = fma_r(h, tz, He[2]);
    }
  }
  // Backward sweep (vjp_kernel): the reverse Faraday scan's gbar_m = sum_{n>m} Sbar_n + Sbar_m / 2 is a running suffix
  // sum there, so B's whole cotangent W = BbarN e_N + BbarE e_E + gbar ne n is known at the sample and every parameter
  // needs ONE functional and one accumulator.  kLanes (G > 1): the suffix over the LATER lanes of the sightline is
  // known only after the sweep, so the lane also sums the Faraday terms h alone (H, He) for combine_suffix().
  template <bool kLanes, typename PT, typename TT, typename AT, typename ST>
  __device__ __forceinline__ void add_w(const PT& P, const TT& T, const AT& a, const ST& S, R z, R BNb, R BEb, R gbar, R MKu) {
    const R gne = gbar * S.ne;
    const R wx = fma_r(BNb, T.eNx, fma_r(BEb, T.eEx, gne * T.nx));
    const R wy = fma_r(BNb, T.eNy, fma_r(BEb, T.eEy, gne * T.ny));
    const R wz = fma_r(BNb, T.eNz, gne * T.nz);
    R wr, wp;
    to_cyl(wx, wy, a.xr, a.yr, wr, wp);
    const R Acc = a.A * a.cc, Asc = a.A * a.sc;
    apply(P, a, wr, wp, wz, Acc, Asc, g);
    if (kLanes) {
      R nr, np;
      to_cyl((R)T.nx, (R)T.ny, a.xr, a.yr, nr, np);
      apply(P, a, S.ne * nr, S.ne * np, S.ne * (R)T.nz, Acc, Asc, H);
    }
    if (kFull) {
      n1[0] += MKu; n1[1] = fma_r(MKu, a.rho, n1[1]); n1[2] = fma_r(MKu * a.thz, z, n1[2]);
      const R h = T.scalef * a.neu * S.Bpar;   // d(ne Bpar Delta_i/Delta) / d ne0
      const R tz = a.thez * z;
      const R gh = gbar * h;
      ge[0] += gh; ge[1] = fma_r(gh, a.rho, ge[1]); ge[2] = fma_r(gh, tz, ge[2]);
      if (kLanes) { He[0] += h; He[1] = fma_r(h, a.rho, He[1]); He[2] = fma_r(h, tz, He[2]); }
    }
  }
  // acc[j] += (dB/dtheta_j at unit amplitude) . (vr, vp, vz)
  template <typename PT, typename AT>
  __device__ __forceinline__ void apply(const PT& P, const AT& a, R vr, R vp, R vz, R Acc, R Asc, R (&acc)[NB]) {
    const R al = fma_r(a.cp, vr, a.sp * vp);
    const R d = fma_r(Acc, al, Asc * vz);                       // (B_disc / b0) . V
    acc[0] += d;
    const R pp = Acc * fma_r(a.cp, vp, -a.sp * vr);             // (dB/dpsi0) / b0 . V
    acc[1] += pp;
    acc[2] = fma_r(a.lr, pp, acc[2]);
    acc[3] = fma_r(a.t, fma_r(Acc, vz, -Asc * al), acc[3]);     // (dB/dchi0) / b0 . V
    if (kFull) {
      acc[4] = fma_r(a.rho - (R)8.0, d, acc[4]);                // * b0 / h_b^2
      const R LR = a.L * a.R;                                   // halo: B_h L R phi_hat
      acc[5] = fma_r(LR, vp, acc[5]);
      const R RuL2 = a.R * a.u * a.L * a.L;
      acc[6] = fma_r(RuL2, vp, acc[6]);                         // * 2 B_h / w_h
      acc[7] = fma_r(LR * fma_r(a.rho, P.inv_rh, (R)-1.0), vp, acc[7]);   // * B_h / r_h
      acc[8] = fma_r(RuL2 * a.u, vp, acc[8]);                   // * 2 B_h / w_h
    }
  }
  // G > 1: add (sum of Sbar over the later lanes of the sightline) x (this lane's sum of Faraday terms)
  template <int G>
  __device__ __forceinline__ void combine_suffix(R later) {
    if (G > 1) {
#pragma unroll
      for (int j = 0; j < NB; ++j) g[j] = fma_r(later, H[j], g[j]);
      if (kFull) {
#pragma unroll
        for (int j = 0; j < 3; ++j) ge[j] = fma_r(later, He[j], ge[j]);
      }
    }
  }
  template <int G>
  __device__ __forceinline__ void combine(R Pl, int lane_in_group) {
#pragma unroll
    for (int j = 0; j < NB; ++j) prefix_combine<G, R>(g[j], H[j], Pl, lane_in_group);
    if (kFull) {
#pragma unroll
      for (int j = 0; j < 3; ++j) prefix_combine<G, R>(ge[j], He[j], Pl, lane_in_group);
    }
  }
  // out[0..15] in canonical order (alpha handled by the caller)
  template <typename PT>
  __device__ __forceinline__ void finish(const PT& P, R* out) {
    const R b0 = P.p[0];
    out[0] = g[0];
    out[1] = b0 * g[1]; out[2] = b0 * g[2]; out[3] = b0 * g[3];
    if (kFull) {
      out[4] = b0 * g[4] / (P.p[4] * P.p[4]);
      out[5] = g[5];
      out[6] = g[6] * (R)2.0 * P.p[5] * P.inv_wh;
      out[7] = g[7] * P.p[5] * P.inv_rh;
      out[8] = g[8] * (R)2.0 * P.p[5] * P.inv_wh;
      out[9] = n1[0];
      out[10] = P.p[9] * n1[1] / (P.p[10] * P.p[10]);
      out[11] = P.p[9] * n1[2] * (R)2.0 / (P.p[11] * P.p[11]);
      out[13] = ge[0];
      out[14] = P.p[13] * ge[1] / (P.p[14] * P.p[14]);
      out[15] = P.p[13] * ge[2] * (R)2.0 / (P.p[15] * P.p[15]);
    }
  }
};

template <typename R = float>
struct UniformGrad {
  R g[3], H[3], n1, ge, He;
  __device__ __forceinline__ void zero() {
    for (int j = 0; j < 3; ++j) { g[j] = (R)0.0; H[j] = (R)0.0; }
    n1 = ge = He = (R)0.0;
  }
  // wK = N0bar (the cotangent of N0 itself: M K / N0)
  template <typename TT, typename ST>
  __device__ __forceinline__ void add(const TT& T, const ST& S, R BNb, R BEb, R Sbar, R wK) {
    const R hs = (R)0.5 * Sbar * S.ne;
    prefix_update(g[0], H[0], Sbar, fma_r(BNb, T.eNx, fma_r(BEb, T.eEx, hs * T.nx)), S.ne * T.nx);
    prefix_update(g[1], H[1], Sbar, fma_r(BNb, T.eNy, fma_r(BEb, T.eEy, hs * T.ny)), S.ne * T.ny);
    prefix_update(g[2], H[2], Sbar, fma_r(BNb, T.eNz, hs * T.nz), S.ne * T.nz);
    n1 += wK;
    const R h = T.scalef * S.Bpar;   // d(scale ne Bpar)/d ne = scale Bpar (S.ne carries scale)
    prefix_update(ge, He, Sbar, (R)0.5 * Sbar * h, h);
  }
  template <bool kLanes, typename TT, typename ST>
  __device__ __forceinline__ void add_w(const TT& T, const ST& S, R BNb, R BEb, R gbar, R wK) {
    const R gne = gbar * S.ne;
    g[0] += fma_r(BNb, T.eNx, fma_r(BEb, T.eEx, gne * T.nx));
    g[1] += fma_r(BNb, T.eNy, fma_r(BEb, T.eEy, gne * T.ny));
    g[2] += fma_r(BNb, T.eNz, gne * T.nz);
    n1 += wK;
    const R h = T.scalef * S.Bpar;
    ge = fma_r(gbar, h, ge);
    if (kLanes) { H[0] += S.ne * T.nx; H[1] += S.ne * T.ny; H[2] += S.ne * T.nz; He += h; }
  }
  template <int G>
  __device__ __forceinline__ void combine_suffix(R later) {
    if (G > 1) {
      for (int j = 0; j < 3; ++j) g[j] = fma_r(later, H[j], g[j]);
      ge = fma_r(later, He, ge);
    }
  }
  template <int G>
  __device__ __forceinline__ void combine(R Pl, int lane_in_group) {
    for (int j = 0; j < 3; ++j) prefix_combine<G, R>(g[j], H[j], Pl, lane_in_group);
    prefix_combine<G, R>(ge, He, Pl, lane_in_group);
  }
  template <typename PT>
  __device__ __forceinline__ void finish(const PT& P, R* out) {
    for (int j = 0; j < 3; ++j) out[j] = g[j];
    out[3] = n1;
    out[4] = ge;
  }
};

// STACK16 (Eq.(16)): (b0, psi0, psi1, chi0) of the four stacked spirals.  The cotangent of B_k is the
// un-permuted total cotangent; amplitudes are accumulated per unit b0_k (weight w_k and annulus mask only).
template <typename R = float>
struct StackGrad {
  R g[16], H[16];
  __device__ __forceinline__ void zero() {
#pragma unroll
    for (int j = 0; j < 16; ++j) { g[j] = (R)0.0; H[j] = (R)0.0; }
  }
  template <typename PT, typename TT, typename AT, typename ST>
  __device__ __forceinline__ void add(const PT& P, const TT& T, const AT& a, const ST& S,
                                      R BNb, R BEb, R Sbar) {
    const R hs = (R)0.5 * Sbar * S.ne;
    const R v1[3] = {fma_r(BNb, T.eNx, fma_r(BEb, T.eEx, hs * T.nx)), fma_r(BNb, T.eNy, fma_r(BEb, T.eEy, hs * T.ny)),
                         fma_r(BNb, T.eNz, hs * T.nz)};
    const R v2[3] = {S.ne * T.nx, S.ne * T.ny, S.ne * T.nz};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      R u1[3], u2[3];
#pragma unroll
      for (int c = 0; c < 3; ++c) { u1[stack_src(k, c)] = v1[c]; u2[stack_src(k, c)] = v2[c]; }
      R u1r, u1p, u2r, u2p;
      to_cyl(u1[0], u1[1], a.xr, a.yr, u1r, u1p);
      to_cyl(u2[0], u2[1], a.xr, a.yr, u2r, u2p);
      const R A = a.mask * stack_weight<R>(k);
      const R Acc = A * a.cc[k], Asc = A * a.sc[k];
      const R h1 = fma_r(a.cp[k], u1r, a.sp[k] * u1p), h2 = fma_r(a.cp[k], u2r, a.sp[k] * u2p);
      prefix_update(g[4 * k], H[4 * k], Sbar, fma_r(Acc, h1, Asc * u1[2]), fma_r(Acc, h2, Asc * u2[2]));   // (B_k / b0_k) . V
      const R p1 = Acc * fma_r(a.cp[k], u1p, -a.sp[k] * u1r), p2 = Acc * fma_r(a.cp[k], u2p, -a.sp[k] * u2r);
      prefix_update(g[4 * k + 1], H[4 * k + 1], Sbar, p1, p2);
      prefix_update(g[4 * k + 2], H[4 * k + 2], Sbar, a.lr * p1, a.lr * p2);
      prefix_update(g[4 * k + 3], H[4 * k + 3], Sbar, a.t * fma_r(Acc, u1[2], -Asc * h1), a.t * fma_r(Acc, u2[2], -Asc * h2));
    }
  }
  template <bool kLanes, typename PT, typename TT, typename AT, typename ST>
  __device__ __forceinline__ void add_w(const PT& P, const TT& T, const AT& a, const ST& S, R BNb, R BEb, R gbar) {
    const R gne = gbar * S.ne;
    const R w1[3] = {fma_r(BNb, T.eNx, fma_r(BEb, T.eEx, gne * T.nx)), fma_r(BNb, T.eNy, fma_r(BEb, T.eEy, gne * T.ny)),
                     fma_r(BNb, T.eNz, gne * T.nz)};
    const R v2[3] = {S.ne * T.nx, S.ne * T.ny, S.ne * T.nz};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const R A = a.mask * stack_weight<R>(k);
      const R Acc = A * a.cc[k], Asc = A * a.sc[k];
      apply_k(a, k, w1, Acc, Asc, g);
      if (kLanes) apply_k(a, k, v2, Acc, Asc, H);
    }
  }
  template <typename AT>
  __device__ __forceinline__ void apply_k(const AT& a, int k, const R (&v)[3], R Acc, R Asc, R (&acc)[16]) {
    R u[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) u[stack_src(k, c)] = v[c];
    R ur, up;
    to_cyl(u[0], u[1], a.xr, a.yr, ur, up);
    const R h = fma_r(a.cp[k], ur, a.sp[k] * up);
    acc[4 * k] += fma_r(Acc, h, Asc * u[2]);                                   // (B_k / b0_k) . V
    const R pp = Acc * fma_r(a.cp[k], up, -a.sp[k] * ur);
    acc[4 * k + 1] += pp;
    acc[4 * k + 2] = fma_r(a.lr, pp, acc[4 * k + 2]);
    acc[4 * k + 3] = fma_r(a.t, fma_r(Acc, u[2], -Asc * h), acc[4 * k + 3]);
  }
  template <int G>
  __device__ __forceinline__ void combine_suffix(R later) {
    if (G > 1) {
#pragma unroll
      for (int j = 0; j < 16; ++j) g[j] = fma_r(later, H[j], g[j]);
    }
  }
  template <int G>
  __device__ __forceinline__ void combine(R Pl, int lane_in_group) {
#pragma unroll
    for (int j = 0; j < 16; ++j) prefix_combine<G, R>(g[j], H[j], Pl, lane_in_group);
  }
  template <typename PT>
  __device__ __forceinline__ void finish(const PT& P, R* out) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      out[4 * k] = g[4 * k];
#pragma unroll
      for (int j = 1; j < 4; ++j) out[4 * k + j] = P.sp[4 * k] * g[4 * k + j];
    }
  }
};

template <int CODE, typename R = float> struct GradOf { using type = AnalyticGrad<CODE == kAnalyticFull, R>; };
template <typename R> struct GradOf<kUniform, R> { using type = UniformGrad<R>; };
template <typename R> struct GradOf<kStack16, R> { using type = StackGrad<R>; };

constexpr int kMinTileForBases = 4;   // vjp_kernel: BatchConsts::tile_d from which the forward's tile bases are used

struct VjpArgs {
  Geometry geo;
  const BatchConsts* bc;
  int batch, f0, n_freq_total;
  int b0;           // first batch element of this launch (gridDim.y <= 65535 per launch)
  const BatchConstsD* bd;   // float64 constants (float64 Faraday chain variant)
  float flag_S;     // PMODE 2: sightlines whose round-off scale exceeds this take the float64 chain
  const int* mode;  // auto: device word from decide_kernel -- kModeAllF64 = "some sightline is near the threshold: run the
                    // per-sightline variant (PMODE 2)", kModeSplit = "... run the per-CTA pair (cta_sel)", else the lean
                    // fp32 variant (PMODE 0) runs; the variants the word does not name exit; or null
  const unsigned char* cta_sel;   // kModeSplit: [batch][n_blocks] from vjp_classify_kernel, 1 = some sightline of this CTA
                    // is above the threshold -> the CTA is done by the PMODE 1 launch, 0 -> by the PMODE 0 launch; or null
  const float* dI; const float* dQ; const float* dU;   // may be null
  ScalarGridDesc sg_ne, sg_n0;   // gridded n_e / N_0 (DISC4), g == nullptr: unused
  const double* phi;      // [batch][npix] Faraday sum of every sightline as the plan's last forward stored it, or null
  const int* phi_ok;      // device word: 1 = that forward ran with exactly these parameters (phi_validate_kernel)
  const double* phi_base; // [k][batch * npix]: Faraday sum before sample 32 k of the sightlines the forward's float64 chain did
  const unsigned char* phi_has;   // [batch * npix]: 1 = phi_base holds this sightline (ForwardArgs::phi_base), or null
  int only_with_bases;    // this launch runs only in the "bases" case (precision 2: the lean variant beside the float64 one)
  float* partial;   // [batch][n_blocks][16]
  int n_blocks;     // blocks per batch element (gridDim.x)
  int accumulate;   // 0: overwrite partials (first frequency block), 1: add
};

// n_e B_LOS Delta_i / Delta of one sample from the float64 chain (synax_f64.cuh) -- the adjoint's Faraday ANGLE needs
// the same accuracy as the forward's when the rotation is strong (measured: fp32 angle, n_e doubled at 408 MHz ->
// gradient errors 2.4e-3); the adjoint algebra itself stays fp32.
template <int CODE>
__device__ __forceinline__ double faraday_term_d(const BatchConsts& P, const BatchConstsD& D, const Triad& T,
                                                 const ScalarGridDesc& sg_ne, double xd, double yd, double zd) {
  double Bx, By, Bz, ne;
  if (CODE == kUniform) {
    Bx = (double)P.uB[0]; By = (double)P.uB[1]; Bz = (double)P.uB[2]; ne = (double)P.une;
  } else {
    const double rho2d = fma(xd, xd, yd * yd);
    const bool inside = (rho2d > 9.0) && (rho2d < 400.0);
    if (CODE == kStack16) {
      eval_stack16_d(D, xd, yd, zd, rho2d, inside, Bx, By, Bz, ne);
    } else {
      const double x1[1] = {xd}, y1[1] = {yd}, z1[1] = {zd}, r1[1] = {rho2d};
      const bool in1[1] = {inside};
      double bx[1], by[1], bz[1], n1[1];
      eval_analytic_dm<CODE == kAnalyticFull, 1>(D, x1, y1, z1, r1, in1, bx, by, bz, n1);
      Bx = bx[0]; By = by[0]; Bz = bz[0]; ne = n1[0];
    }
    if ((CODE == kAnalyticDisc || CODE == kStack16) && sg_ne.g) ne = scalar_grid_at<double>(sg_ne, xd, yd, zd);
  }
  return T.scale * ne * fma(Bx, T.nxd, fma(By, T.nyd, Bz * T.nzd));
}

// grid = (n_blocks, batch); block = kBlock threads; G lanes per sightline.
// PMODE 0: fp32 Faraday angles; 1: Faraday sums and angles from the float64 chain for every sightline; 2: decided per
// sightline -- its round-off scale k_max sum |n_e|(|B_LOS|+|B_N|+|B_E|), estimated from every 16th sample, against
// A.flag_S (= escalate_rad / k_max): sightlines below it carry an angle error <= ~3e-7 x 300 rad = 1e-4 rad,
// inside the 1e-3 gradient bound; the others take the float64 chain.  The tile length is warp-uniform.
#ifndef SYNAX_VJP_MINB
#define SYNAX_VJP_MINB 1
#endif
template <int CODE, int G, int NF, int PMODE>
__global__ void __launch_bounds__(kBlock, (PMODE == 0 && G == 1 && SYNAX_VJP_MINB < 3) ? 3 : SYNAX_VJP_MINB) vjp_kernel(const __grid_constant__ VjpArgs A, const __grid_constant__ FreqTab ft) {
  constexpr bool kAlpha = (CODE == kAnalyticFull || CODE == kUniform);  // alpha is a parameter
  // The forward of this plan left, for these very parameters, the Faraday depth at every 32nd sample of each sightline
  // its float64 chain integrated: fp32 tile-local angles on those exact tile bases are as good as float64 angles, so the
  // lean variant does EVERY sightline and the float64-angle variants (and their classification) stand aside.
  // (Not for under-resolved runs: the bases are 32 samples apart, and the fp32 angle inside a tile must stay below ~800 rad
  // -- tile_d >= 4 means at most 24 rad per step -- for its 6e-8 relative round-off to stay inside the gradient bound.)
  const bool bases = G == 1 && A.phi_base != nullptr && A.phi != nullptr && *A.phi_ok != 0 && A.bc[A.b0 + blockIdx.y].tile_d >= kMinTileForBases;
  if (bases) {
    if (PMODE != 0 || A.cta_sel) return;
  } else if (A.only_with_bases) {
    return;
  } else if (A.mode) {
    const int m = *A.mode;
    if (A.cta_sel ? (m != kModeSplit) : (m == kModeSplit || (m == kModeAllF64) != (PMODE == 2))) return;
  }
  const int b = A.b0 + blockIdx.y;
  // the other launch of the pair does this CTA (and owns its partial: the two launches run concurrently)
  if (A.cta_sel && (A.cta_sel[(size_t)b * A.n_blocks + blockIdx.x] != 0) != (PMODE == 1)) return;
  const int64_t tid = (int64_t)blockIdx.x * kBlock + threadIdx.x;
  const int g = (int)(tid % G);
  int64_t pix = tid / G;
  const bool valid = pix < A.geo.npix;
  if (!valid) pix = A.geo.npix - 1;
  const BatchConsts& P = A.bc[b];
  BatchConstsD D;
  if (PMODE != 0) D = A.bd[b];
  const Triad T = load_triad(A.geo, pix);
  const int C = (A.geo.n_los + G - 1) / G;
  const int n0 = g * C, n1 = min(n0 + C, A.geo.n_los);
  const double delta = A.geo.delta * T.scale;

  bool prec = PMODE == 1;
  if (PMODE == 2) {
    float est = roundoff_scale_estimate<CODE>(A.geo, P, T, A.sg_ne, n0, n1);
    est = group_sum<G>(est) * T.scalef;
    prec = est > A.flag_S;
  }
  const bool warp_prec = PMODE == 1 || (PMODE == 2 && __any_sync(0xffffffffu, prec));

  // cotangents of this sightline, coefficients folded in (zero for padded lanes)
  // (dQ, dU are re-read at every tile start -- L1 hits -- instead of being held in 2 NF registers)
  float cI = 0.f;
  float cIa = 0.f;   // sum_f Ibar_f c_f d ln c_f / d alpha (alpha gradient)
  const int64_t o0 = ((int64_t)b * A.n_freq_total + A.f0) * A.geo.npix + pix;
#pragma unroll
  for (int f = 0; f < NF; ++f) {
    const float vI = (valid && A.dI) ? A.dI[o0 + f * A.geo.npix] : 0.f;
    cI = fmaf(vI, P.coefI[A.f0 + f], cI);
    if (kAlpha) cIa = fmaf(vI * P.coefI[A.f0 + f], P.dlnc_dalpha[A.f0 + f], cIa);
  }
  cI *= T.scalef;   // the maps are scale * coef * sums (per-sightline segment length, synax_plan_set_box)
  cIa *= T.scalef;

  // ---- Faraday sum of this lane's chunk.  The sweep below runs BACKWARDS (far end first), where the reverse scan of the
  // Faraday cotangent (S:App.D.2) is a running sum; the forward Faraday depth of a sample is then
  //   phi_n = (sum over the whole sightline) - (sum over the samples after n) - g_n / 2,
  // so the sightline total is needed first: taken from the value the last forward of this plan stored for exactly these
  // parameters (A.phi, validated on the device: *A.phi_ok) when the thread owns the whole sightline, else from a
  // forward-order pre-pass over the Faraday integrand alone.
  double Sl = 0.0;
  const bool cached = G == 1 && A.phi != nullptr && *A.phi_ok != 0;
  if (cached) {
    Sl = A.phi[(int64_t)b * A.geo.npix + pix];
  } else {
    double s_d = ((double)n0 + 0.5) * delta;
    float hi = 0.f, lo = 0.f;
    for (int n = n0; n < n1; ++n) {
      const double xd = fma(s_d, T.nxd, A.geo.obs[0]);
      const double yd = fma(s_d, T.nyd, A.geo.obs[1]);
      const double zd = fma(s_d, T.nzd, A.geo.obs[2]);
      s_d += delta;
      if (PMODE != 0 && prec) { Sl += faraday_term_d<CODE>(P, D, T, A.sg_ne, xd, yd, zd); continue; }
      SampleF S;
      if (CODE == kUniform) {
        S.Bpar = fmaf(P.uB[0], T.nx, fmaf(P.uB[1], T.ny, P.uB[2] * T.nz)); S.ne = P.une;
      } else if (CODE == kStack16) {
        const double rho2d = fma(xd, xd, yd * yd);
        StackAux sa;
        eval_stack16_f32<true>(P, T, (float)xd, (float)yd, (float)zd, (float)rho2d, (rho2d > 9.0) && (rho2d < 400.0), S, sa);
        if (A.sg_ne.g) S.ne = scalar_grid_at<float>(A.sg_ne, xd, yd, zd);
      } else {
        const double rho2d = fma(xd, xd, yd * yd);
        AnalyticAux aux;
        eval_analytic_f32<CODE == kAnalyticFull, true>(P, T, (float)xd, (float)yd, (float)zd, (float)rho2d,
                                                 (rho2d > 9.0) && (rho2d < 400.0), S, aux);
        if (CODE == kAnalyticDisc && A.sg_ne.g) S.ne = scalar_grid_at<float>(A.sg_ne, xd, yd, zd);
      }
      const float gn = T.scalef * S.ne * S.Bpar;
      const float sum = hi + gn;
      lo += gn - (sum - hi);
      hi = sum;
      if (((n - n0) & (kTile - 1)) == kTile - 1) { Sl += (double)hi + (double)lo; hi = 0.f; lo = 0.f; }
    }
    Sl += (double)hi + (double)lo;
  }
  double total = Sl, after = 0.0;   // Faraday sum of the whole sightline / of the lanes after this one
  if (G > 1) {
    const double before = group_exclusive_scan<G>(Sl, g);
    total = group_sum_d<G>(Sl);
    after = total - before - Sl;
  }

  // ---- main sweep, backwards
  typename GradOf<CODE>::type acc;
  acc.zero();
  float gAlpha = 0.f;          // sum_n 1/4 ln(B_perp^2) M K
  float sumE = 0.f;            // sum_n e~_n
  float gPol = 0.f;            // sum_f (d ln c_f / d alpha + d ln Pi / d alpha) (Qbar_f Q_f + Ubar_f U_f)
  // d ln c_f / d alpha = dlnA - ln(nu_f) / 2: the frequency-dependent part comes from the constant bank (ft.ln_nu)
  const float cPol = kAlpha ? P.dlnA_dalpha + P.dpi_dalpha_over_pi : 0.f;
  float suf = 0.f;             // sum of Sbar over this lane's samples after the current one
  double carry = after;        // Faraday sum over everything after the current tile
  const int tile = warp_prec ? P.tile_d : kTile;
  const int64_t slb = (int64_t)b * A.geo.npix + pix;
  const bool has_base = PMODE == 0 && bases && A.phi_has[slb] != 0;
  for (int te = n1; te > n0;) {
    const int ts = max(((te - 1) / tile) * tile, n0);   // tiles are aligned to multiples of the tile length from sample 0
    // Faraday depth at the far end of this tile: the forward's float64 value where it stored one, else total - (sum after)
    const double phi_te = (has_base && te < A.geo.n_los) ? A.phi_base[(size_t)(te >> 5) * ((size_t)A.geo.npix * A.batch) + slb] : total - carry;
    // cotangents rotated by the Faraday angle at the far end of this tile
    float rq[NF], ru[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      // Qb cos(tb + tl) + Ub sin(tb + tl) = Qb' cos tl + Ub' sin tl,  Qb' = Qb cb + Ub sb, Ub' = -Qb sb + Ub cb
      float q = (valid && A.dQ) ? __ldg(A.dQ + o0 + f * A.geo.npix) * P.coefP[A.f0 + f] * T.scalef : 0.f;
      float u = (valid && A.dU) ? __ldg(A.dU + o0 + f * A.geo.npix) * P.coefP[A.f0 + f] * T.scalef : 0.f;
      rotate_by_offset(-ft.k_turn[f], phi_te, q, u);
      rq[f] = q; ru[f] = u;
    }
    float hi = 0.f, lo = 0.f;    // tile-local Faraday sum over the samples after the current one (two-float)
    double dl = 0.0;             // the same in float64 (float64-chain sightlines)
    double s_d = ((double)te - 0.5) * delta;   // midpoint of sample te - 1
    PosF pf;
    pf.init(delta, te - 1);
    for (int n = te - 1; n >= ts; --n) {
      const double xd = fma(s_d, T.nxd, A.geo.obs[0]);
      const double yd = fma(s_d, T.nyd, A.geo.obs[1]);
      const double zd = fma(s_d, T.nzd, A.geo.obs[2]);
      s_d -= delta;
      float xf, yf, zf, rho2f;
      pf.next(A.geo, T, -1.0f, xf, yf, zf, rho2f);
      SampleF S;
      AnalyticAux aux;
      StackAux sa;
      if (CODE == kStack16) {
        const double rho2d = fma(xd, xd, yd * yd);
        eval_stack16_f32<true>(P, T, xf, yf, zf, rho2f, (rho2d > 9.0) && (rho2d < 400.0), S, sa);
        if (A.sg_ne.g) S.ne = scalar_grid_at<float>(A.sg_ne, xd, yd, zd);
        if (A.sg_n0.g) S.N0 = scalar_grid_at<float>(A.sg_n0, xd, yd, zd);
      } else if (CODE == kUniform) {
        S.Bpar = fmaf(P.uB[0], T.nx, fmaf(P.uB[1], T.ny, P.uB[2] * T.nz));
        S.BN = fmaf(P.uB[0], T.eNx, fmaf(P.uB[1], T.eNy, P.uB[2] * T.eNz));
        S.BE = fmaf(P.uB[0], T.eEx, P.uB[1] * T.eEy);
        S.N0 = P.uN0; S.ne = P.une;
      } else {
        const double rho2d = fma(xd, xd, yd * yd);
        eval_analytic_f32<CODE == kAnalyticFull, true>(P, T, xf, yf, zf, rho2f, (rho2d > 9.0) && (rho2d < 400.0), S, aux);
        if (CODE == kAnalyticDisc) {
          if (A.sg_ne.g) S.ne = scalar_grid_at<float>(A.sg_ne, xd, yd, zd);
          if (A.sg_n0.g) S.N0 = scalar_grid_at<float>(A.sg_n0, xd, yd, zd);
        }
      }
      S.ne *= T.scalef;   // n_e enters only through the Faraday integrand n_e B_LOS Delta_i
      // emission terms
      const float bn2 = S.BN * S.BN, be2 = S.BE * S.BE;
      const float Bt2 = bn2 + be2;
      float w = 1.0f, lgB = 0.f;
      if (kAlpha || !P.alpha_is_3) {
        lgB = (Bt2 > 0.f) ? mufu_lg2(Bt2) : 0.f;
        if (!P.alpha_is_3) w = (Bt2 > 0.f) ? mufu_ex2(P.q_exp * lgB) : 0.f;
      }
      const float M = w * S.N0;
      const float d2 = be2 - bn2, p2 = 2.0f * S.BE * S.BN;
      const float a = M * d2, bq = M * p2;
      // Faraday phase of this sample relative to the far end of the tile: -(sum after it within the tile + g_n / 2)
      float ph;
      double phd = 0.0;   // the same in float64 (float64-chain sightlines)
      if (PMODE != 0 && prec) {
        const double gd = faraday_term_d<CODE>(P, D, T, A.sg_ne, xd, yd, zd);
        phd = -fma(0.5, gd, dl);
        ph = (float)phd;
        dl += gd;
      } else {
        const float gn = S.ne * S.Bpar;
        ph = -fmaf(0.5f, gn, hi);
        const float sum = hi + gn;
        lo += gn - (sum - hi);
        hi = sum;
      }
      // A9: fan-out over frequencies
      float Xc = 0.f, Xs = 0.f, Yc = 0.f, Ys = 0.f, Zc = 0.f, Zs = 0.f;
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        float th = ft.k_rad[f] * ph;
        if (PMODE != 0 && prec && tile == 1) {   // under-resolved: one sample turns by more than 24 rad at the lowest frequency --
          double t = ft.k_turn[f] * phd;          // its half-cell angle is reduced to turns in float64, not formed in fp32
          t -= rint(t);
          th = (float)t * 6.283185307179586f;
        }
        const float c = mufu_cos(th), s = mufu_sin(th);
        const float u = fmaf(rq[f], c, ru[f] * s);
        const float v = fmaf(ru[f], c, -rq[f] * s);
        Xc += u; Xs += v;
        Yc = fmaf(ft.k_rad[f], u, Yc); Ys = fmaf(ft.k_rad[f], v, Ys);
        if (kAlpha) { Zc = fmaf(ft.ln_nu[f], u, Zc); Zs = fmaf(ft.ln_nu[f], v, Zs); }
      }
      if (kAlpha) gPol = fmaf(a, fmaf(cPol, Xc, -0.5f * Zc), fmaf(bq, fmaf(cPol, Xs, -0.5f * Zs), gPol));
      // L_n = M K,  K = cI Bt2 + Xc d2 + Xs p2
      const float K = fmaf(cI, Bt2, fmaf(Xc, d2, Xs * p2));
      const float MK = M * K;
      sumE = fmaf(M, Bt2, sumE);
      if (kAlpha) gAlpha = fmaf(lgB, MK, gAlpha);
      // A10: cotangent Sbar of the Faraday sum at this sample; transposed half-cell scan gbar = sum_{later} Sbar + Sbar / 2
      const float Sbar = fmaf(a, Ys, -bq * Yc);
      const float gbar = fmaf(0.5f, Sbar, suf);
      suf += Sbar;
      // B_N, B_E cotangents (direct): from M, d2, p2, Bt2 and the (B_perp^2)^q factor
      float tq_ = 0.f;                                             // d/dBt2 through w (alpha != 3 only)
      if (!P.alpha_is_3 && Bt2 > 0.f) tq_ = P.q_exp * MK * mufu_rcp(Bt2);
      const float BEb = 2.0f * fmaf(M, fmaf(S.BE, cI + Xc, S.BN * Xs), S.BE * tq_);
      const float BNb = 2.0f * fmaf(M, fmaf(S.BN, cI - Xc, S.BE * Xs), S.BN * tq_);
      // A11: field partials
      if constexpr (CODE == kUniform) acc.template add_w<(G > 1)>(T, S, BNb, BEb, gbar, w * K);
      else if constexpr (CODE == kStack16) acc.template add_w<(G > 1)>(P, T, sa, S, BNb, BEb, gbar);
      else acc.template add_w<(G > 1)>(P, T, aux, S, zf, BNb, BEb, gbar, w * aux.N0u * K);
    }
    carry += (PMODE != 0 && prec) ? dl : (double)hi + (double)lo;
    te = ts;
  }

  // ---- lanes of a sightline: the Sbar totals of the LATER lanes weight this lane's Faraday terms
  if (G > 1) {
    const float before = (float)group_exclusive_scan<G>((double)suf, g);
    const float all = group_sum<G>(suf);
    acc.template combine_suffix<G>(all - before - suf);
  }
  float out[16];
#pragma unroll
  for (int j = 0; j < 16; ++j) out[j] = 0.f;
  acc.finish(P, out);
  if (kAlpha) {
    // alpha: 1/4 ln(B_perp^2) term + d ln c_f / d alpha * (Ibar I + Qbar Q + Ubar U) + dPi/Pi * (Qbar Q + Ubar U)
    out[CODE == kUniform ? 5 : 12] = fmaf(0.25f * 0.6931471805599453f, gAlpha, fmaf(cIa, sumE, gPol));
  }

  // ---- block reduction -> partial[b][block][16]
  constexpr int NP = (CODE == kUniform) ? 6 : ((CODE == kAnalyticFull || CODE == kStack16) ? 16 : 4);
  __shared__ float red[kBlock / 32][16];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int j = 0; j < NP; ++j) {
    float v = out[j];
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    if (lane == 0) red[wid][j] = v;
  }
  __syncthreads();
  if (threadIdx.x < NP) {
    float v = 0.f;
#pragma unroll
    for (int k = 0; k < kBlock / 32; ++k) v += red[k][threadIdx.x];
    float* dst = A.partial + ((size_t)b * A.n_blocks + blockIdx.x) * 16 + threadIdx.x;
    *dst = A.accumulate ? (*dst + v) : v;
  }
}

// ------------------------------------------------------------------------------------------------
// Adjoint, batched (S:8(a) A12): the lean variant (fp32 Faraday angles, one thread per sightline, one frequency) for NB
// consecutive parameter vectors per thread, sharing the sample geometry as forward_batched_kernel does.  Per vector the
// arithmetic is that of vjp_kernel<CODE, 1, 1, 0>, but in FORWARD order (prefix form of the reverse scan): no Faraday total
// is needed first, so NB = 1 is also the stand-alone adjoint at one frequency.  grid = (n_blocks, ceil(batch / NB)).
// ------------------------------------------------------------------------------------------------
template <int CODE, int NB>
__global__ void __launch_bounds__(kBlock) vjp_batched_kernel(const __grid_constant__ VjpArgs A, const __grid_constant__ FreqTab ft) {
  static_assert(CODE == kAnalyticDisc || CODE == kAnalyticFull, "analytic models only");
  constexpr bool kAlpha = CODE == kAnalyticFull;
  if (A.mode) {   // runs where the lean fp32 variant would
    const int m = *A.mode;
    if (m == kModeSplit || m == kModeAllF64) return;
  }
  int64_t pix = (int64_t)blockIdx.x * kBlock + threadIdx.x;
  const bool valid = pix < A.geo.npix;
  if (!valid) pix = A.geo.npix - 1;
  int bj[NB];
  bool live[NB];
#pragma unroll
  for (int j = 0; j < NB; ++j) { live[j] = (int)blockIdx.y * NB + j < A.batch; bj[j] = live[j] ? (int)blockIdx.y * NB + j : A.batch - 1; }
  const Triad T = load_triad(A.geo, pix);
  const double delta = A.geo.delta * T.scale;
  const float k_rad = ft.k_rad[0], ln_nu = ft.ln_nu[0];

  typename GradOf<CODE>::type acc[NB];
  float cI[NB], cIa[NB], cq[NB], cu[NB], gAlpha[NB], sumE[NB], gPol[NB], cPol[NB], Pl[NB];
  double carry[NB];
#pragma unroll
  for (int j = 0; j < NB; ++j) {
    const BatchConsts& P = A.bc[bj[j]];
    const int64_t o = ((int64_t)bj[j] * A.n_freq_total + A.f0) * A.geo.npix + pix;
    const bool on = valid && live[j];
    const float vI = (on && A.dI) ? A.dI[o] : 0.f;
    cI[j] = vI * P.coefI[A.f0] * T.scalef;
    cIa[j] = kAlpha ? vI * P.coefI[A.f0] * P.dlnc_dalpha[A.f0] * T.scalef : 0.f;
    cq[j] = (on && A.dQ) ? __ldg(A.dQ + o) * P.coefP[A.f0] * T.scalef : 0.f;
    cu[j] = (on && A.dU) ? __ldg(A.dU + o) * P.coefP[A.f0] * T.scalef : 0.f;
    cPol[j] = kAlpha ? P.dlnA_dalpha + P.dpi_dalpha_over_pi : 0.f;
    acc[j].zero();
    gAlpha[j] = 0.f; sumE[j] = 0.f; gPol[j] = 0.f; Pl[j] = 0.f; carry[j] = 0.0;
  }
  double s_d = 0.5 * delta;
  PosF pf;
  pf.init(delta, 0);
  for (int ts = 0; ts < A.geo.n_los; ts += kTile) {
    const int te = min(ts + kTile, A.geo.n_los);
    float rq[NB], ru[NB], hi[NB], lo[NB];
#pragma unroll
    for (int j = 0; j < NB; ++j) {   // cotangents rotated by the Faraday angle of everything before this tile
      float q = cq[j], u = cu[j];
      rotate_by_offset(-ft.k_turn[0], carry[j], q, u);
      rq[j] = q; ru[j] = u; hi[j] = 0.f; lo[j] = 0.f;
    }
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
        analytic_fields_f32<CODE == kAnalyticFull, true>(P, T, geom, zf, inside, S, aux);
        S.ne *= T.scalef;
        const float bn2 = S.BN * S.BN, be2 = S.BE * S.BE;
        const float Bt2 = bn2 + be2;
        float w = 1.0f, lgB = 0.f;
        if (kAlpha || !P.alpha_is_3) {
          lgB = (Bt2 > 0.f) ? mufu_lg2(Bt2) : 0.f;
          if (!P.alpha_is_3) w = (Bt2 > 0.f) ? mufu_ex2(P.q_exp * lgB) : 0.f;
        }
        const float M = w * S.N0;
        const float d2 = be2 - bn2, p2 = 2.0f * S.BE * S.BN;
        const float a = M * d2, bq = M * p2;
        const float gn = S.ne * S.Bpar;
        const float ph = fmaf(0.5f, gn, hi[j]);
        const float sum = hi[j] + gn;
        lo[j] += gn - (sum - hi[j]);
        hi[j] = sum;
        const float th = k_rad * ph;
        const float c = mufu_cos(th), sn = mufu_sin(th);
        const float Xc = fmaf(rq[j], c, ru[j] * sn);
        const float Xs = fmaf(ru[j], c, -rq[j] * sn);
        const float Yc = k_rad * Xc, Ys = k_rad * Xs;
        if (kAlpha) gPol[j] = fmaf(a, fmaf(cPol[j], Xc, -0.5f * ln_nu * Xc), fmaf(bq, fmaf(cPol[j], Xs, -0.5f * ln_nu * Xs), gPol[j]));
        const float K = fmaf(cI[j], Bt2, fmaf(Xc, d2, Xs * p2));
        const float MK = M * K;
        sumE[j] = fmaf(M, Bt2, sumE[j]);
        if (kAlpha) gAlpha[j] = fmaf(lgB, MK, gAlpha[j]);
        const float Sbar = fmaf(a, Ys, -bq * Yc);
        Pl[j] += Sbar;
        float tq_ = 0.f;
        if (!P.alpha_is_3 && Bt2 > 0.f) tq_ = P.q_exp * MK * mufu_rcp(Bt2);
        const float BEb = 2.0f * fmaf(M, fmaf(S.BE, cI[j] + Xc, S.BN * Xs), S.BE * tq_);
        const float BNb = 2.0f * fmaf(M, fmaf(S.BN, cI[j] - Xc, S.BE * Xs), S.BN * tq_);
        acc[j].add(P, T, aux, S, zf, BNb, BEb, Sbar, w * aux.N0u * K);
      }
    }
#pragma unroll
    for (int j = 0; j < NB; ++j) carry[j] += (double)hi[j] + (double)lo[j];
  }
  constexpr int NP = CODE == kAnalyticFull ? 16 : 4;
  __shared__ float red[kBlock / 32][16];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int j = 0; j < NB; ++j) {
    const BatchConsts& P = A.bc[bj[j]];
    float out[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) out[k] = 0.f;
    acc[j].finish(P, out);
    if (kAlpha) out[12] = fmaf(0.25f * 0.6931471805599453f, gAlpha[j], fmaf(cIa[j], sumE[j], gPol[j]));
#pragma unroll
    for (int k = 0; k < NP; ++k) {
      float v = out[k];
#pragma unroll
      for (int d = 16; d >= 1; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
      if (lane == 0) red[wid][k] = v;
    }
    __syncthreads();
    if (threadIdx.x < NP && live[j]) {
      float v = 0.f;
#pragma unroll
      for (int k = 0; k < kBlock / 32; ++k) v += red[k][threadIdx.x];
      float* dst = A.partial + ((size_t)bj[j] * A.n_blocks + blockIdx.x) * 16 + threadIdx.x;
      *dst = A.accumulate ? (*dst + v) : v;
    }
    __syncthreads();
  }
}

// kModeSplit (long calls): the G lanes of a sightline estimate its round-off scale exactly as PMODE 2 does; a
// CTA with any sightline above the threshold is handed to the PMODE 1 launch (float64 Faraday angles for its 128 / G
// sightlines), the others to the lean PMODE 0 launch.  The thread <-> sightline mapping, and so the order of every
// sum, is the one of a full launch: the gradient stays deterministic.  (In RING order the strongly rotating
// sightlines -- low latitudes towards the inner Galaxy -- are contiguous runs, so CTA granularity loses little.)
template <int CODE, int G>
__global__ void __launch_bounds__(kBlock) vjp_classify_kernel(const __grid_constant__ VjpArgs A,
                                                              unsigned char* __restrict__ cta_sel) {
  if (*A.mode != kModeSplit) return;
  if (G == 1 && A.phi_base != nullptr && A.phi != nullptr && *A.phi_ok != 0 && A.bc[A.b0 + blockIdx.y].tile_d >= kMinTileForBases) return;   // vjp_kernel: "bases"
  const int b = A.b0 + blockIdx.y;
  const int64_t tid = (int64_t)blockIdx.x * kBlock + threadIdx.x;
  const int g = (int)(tid % G);
  int64_t pix = tid / G;
  const bool valid = pix < A.geo.npix;
  if (!valid) pix = A.geo.npix - 1;   // keep the lane alive for the shuffles
  const BatchConsts& P = A.bc[b];
  const Triad T = load_triad(A.geo, pix);
  const int C = (A.geo.n_los + G - 1) / G;
  const int n0 = g * C, n1 = min(n0 + C, A.geo.n_los);
  float est = roundoff_scale_estimate<CODE>(A.geo, P, T, A.sg_ne, n0, n1);   // as PMODE 2 does, lane by lane
  est = group_sum<G>(est) * T.scalef;
  const int any = __syncthreads_or((valid && est > A.flag_S) ? 1 : 0);
  if (threadIdx.x == 0) cta_sel[(size_t)b * A.n_blocks + blockIdx.x] = any ? 1 : 0;
}
}  // namespace synax
