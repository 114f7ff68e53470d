// synax_device.cuh -- device-side building blocks of libsynax (sm_100a): math helpers, per-batch
// constants, analytic field evaluators (fp32 fast chain, fp64 precise chain).
// Shares nothing with oracle/ (see DESIGN.md).  Citations: P:L<n> = paper text line, S:<tag> =
// DESIGN.md section 3 reading.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace synax {

constexpr int kMaxFreq = 32;
constexpr int kMaxAnalyticParams = 16;

// ---- physical constants, Gaussian CGS (CODATA 2018) -- used on the host and in the fp64 prologue
#define SYNAX_QE 4.80320471257e-10
#define SYNAX_ME 9.1093837015e-28
#define SYNAX_C 2.99792458e10
#define SYNAX_KB 1.380649e-16
#define SYNAX_KPC 3.0856775814913673e21
#define SYNAX_PI 3.14159265358979323846

// ------------------------------------------------------------------------------------------------
// fp32 hardware approximations (XU / MUFU pipe), flush-to-zero.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float mufu_ex2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_lg2(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_rcp(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_rsqrt(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_sin(float x) { float y; asm("sin.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_cos(float x) { float y; asm("cos.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// sin and cos on the FMA pipe, ~1 ulp for |x| < ~200 (Cody-Waite reduction by pi/2 + minimax
// polynomials on [-pi/4, pi/4]).  Used where the MUFU's 5e-7 absolute error would be systematic
// along a sightline (the pitch / tilt angles of the disc field), see DESIGN.md section 5.
__device__ __forceinline__ void sincos_fma(float x, float& s, float& c) {
  const float t = fmaf(x, 0.636619772367581343f, 12582912.0f);  // 1.5 * 2^23: round to nearest int
  const int q = __float_as_int(t);
  const float k = t - 12582912.0f;
  float r = fmaf(k, -1.57079625129699707031f, x);
  r = fmaf(k, -7.54978941586159635335e-08f, r);
  const float r2 = r * r;
  float ps = fmaf(r2, -1.9515295891e-4f, 8.3321608736e-3f);
  ps = fmaf(ps, r2, -1.6666654611e-1f);
  ps = fmaf(ps * r2, r, r);                                     // sin(r)
  float pc = fmaf(r2, 2.443315711809948e-5f, -1.388731625493765e-3f);
  pc = fmaf(pc, r2, 4.166664568298827e-2f);
  pc = fmaf(pc * r2, r2, fmaf(r2, -0.5f, 1.0f));                // cos(r)
  const float ss = (q & 1) ? pc : ps;
  const float cs = (q & 1) ? ps : pc;
  s = (q & 2) ? -ss : ss;
  c = ((q + 1) & 2) ? -cs : cs;
}

// the same polynomials without the reduction, for |x| <= pi/4 (BatchConsts::angles_small)
__device__ __forceinline__ void sincos_fma_small(float r, float& s, float& c) {
  const float r2 = r * r;
  float ps = fmaf(r2, -1.9515295891e-4f, 8.3321608736e-3f);
  ps = fmaf(ps, r2, -1.6666654611e-1f);
  s = fmaf(ps * r2, r, r);
  float pc = fmaf(r2, 2.443315711809948e-5f, -1.388731625493765e-3f);
  pc = fmaf(pc, r2, 4.166664568298827e-2f);
  c = fmaf(pc * r2, r2, fmaf(r2, -0.5f, 1.0f));
}

// ------------------------------------------------------------------------------------------------
// Per-batch-element constants, written by prologue_kernel (fp64 math, rounded once).
// Canonical 16-parameter analytic model; DISC4 maps onto it with h_b = inf, B_h = 0.
// ------------------------------------------------------------------------------------------------
struct BatchConsts {
  // raw parameters, canonical FULL16 order (S:App.C), as float and double
  float p[kMaxAnalyticParams];
  float sp[16];      // STACK16 only: (b0, psi0, psi1, chi0) of the four stacked spirals (p[] then holds the aux densities)
  // derived fp32
  float k_hb;        // -log2(e)/h_b      (0 for DISC4)
  float inv_wh, inv_rh;
  float k_hr, k_hz;  // -log2(e)/h_r, -2 log2(e)/h_z
  float k_her, k_hez;
  float q_exp;       // (alpha-3)/4 : (B_perp^2)^q_exp
  float pi_frac;     // (alpha+1)/(alpha+7/3)   Eq.(5)/Eq.(2)
  int alpha_is_3;
  int angles_small;  // |psi0| + |psi1| <= pi/4 and |chi0| <= pi/4: psi and chi never leave [-pi/4, pi/4] (no range reduction)
  int tile_d;        // samples per tile of the float64-chain kernel (prologue_kernel)
  float coefI[kMaxFreq];  // c_f(alpha) * Delta  [K per (cm^-3 uG^((alpha+1)/2))]
  float coefP[kMaxFreq];  // pi_frac * coefI
  // VJP only
  float dlnc_dalpha[kMaxFreq];  // d ln c_f / d alpha
  float dpi_dalpha_over_pi;     // d ln Pi / d alpha
  float dlnA_dalpha;            // d ln c_f / d alpha + ln(nu_f) / 2 (the frequency-independent part)
  // uniform model
  float uB[3], uN0, une;
};

struct AuxHost { float v[7]; };  // synax_model::aux by value: C0, h_r, h_z, alpha, ne0, h_er, h_ez

struct FreqTab {
  int n_freq;
  float k_rad[kMaxFreq];    // 2 lambda_f^2 K_F Delta : Faraday angle (rad) per unit sum(n_e B_LOS)
  double k_turn[kMaxFreq];  // the same / (2 pi), float64, for exact turn reduction of large offsets
  double freq[kMaxFreq];
  float ln_nu[kMaxFreq];    // ln(nu_f / Hz)
};

// the table of one frequency pass: entries f0 .. f0 + n - 1 moved to the front, so that the kernels index it with
// compile-time constants (k_rad[f], k_turn[f] become constant-bank operands instead of registers)
static inline FreqTab shift_freqs(const FreqTab& ft, int f0) {
  FreqTab o = ft;
  for (int f = 0; f < kMaxFreq; ++f) {
    const int g = f0 + f < kMaxFreq ? f0 + f : kMaxFreq - 1;
    o.k_rad[f] = ft.k_rad[g]; o.k_turn[f] = ft.k_turn[g]; o.freq[f] = ft.freq[g]; o.ln_nu[f] = ft.ln_nu[g];
  }
  return o;
}

struct Geometry {
  int64_t npix;
  int n_los;
  double delta;   // s_max / n_los  (kpc)
  double obs[3];
  float obsf[3];  // the observer rounded to fp32 (constant-bank operands of the fp32 position FMAs)
  const double* dirs;  // [npix][4] = cos l, sin l, cos b, sin b
  const double* path;  // [npix] path length of the sightline in units of s_max = n_los * delta, or null (= 1):
                       // set by synax_plan_set_box (integration from the observer to the box face)
};

// Gridded scalar field (n_e or N_0): regular grid [nx][ny][nz] fp32, nodes on the faces of a box
// centred on the Galactic centre, trilinear interpolation, zero outside.  g == nullptr: not used (analytic disc).
struct ScalarGridDesc {
  const float* g;
  int nx, ny, nz;
  double sx, sy, sz;    // (n-1)/l
  double bx, by, bz;    // (n-1)/2
};

// coordinates, box test and cell in float64 (as for the B grid); weights and sum in fp32 or float64
template <typename R>
__device__ __forceinline__ R scalar_grid_at(const ScalarGridDesc& G, double x, double y, double z) {
  const double ux = fma(x, G.sx, G.bx), uy = fma(y, G.sy, G.by), uz = fma(z, G.sz, G.bz);
  const bool inbox = (ux >= 0.0) && (ux <= (double)(G.nx - 1)) && (uy >= 0.0) && (uy <= (double)(G.ny - 1)) &&
                     (uz >= 0.0) && (uz <= (double)(G.nz - 1));
  if (!inbox) return (R)0;
  int i = __double2int_rd(ux), j = __double2int_rd(uy), k = __double2int_rd(uz);
  i = min(i, G.nx - 2); j = min(j, G.ny - 2); k = min(k, G.nz - 2);
  const R tx = (R)(ux - (double)i), ty = (R)(uy - (double)j), tz = (R)(uz - (double)k);
  const R x0 = (R)1 - tx, y0 = (R)1 - ty, z0 = (R)1 - tz;
  const float* p = G.g + ((size_t)i * G.ny + j) * G.nz + k;
  const size_t dy = (size_t)G.nz, dx = (size_t)G.ny * G.nz;
  const R c00 = z0 * (R)__ldg(p) + tz * (R)__ldg(p + 1);
  const R c01 = z0 * (R)__ldg(p + dy) + tz * (R)__ldg(p + dy + 1);
  const R c10 = z0 * (R)__ldg(p + dx) + tz * (R)__ldg(p + dx + 1);
  const R c11 = z0 * (R)__ldg(p + dx + dy) + tz * (R)__ldg(p + dx + dy + 1);
  return x0 * (y0 * c00 + ty * c01) + tx * (y0 * c10 + ty * c11);
}

// per-sightline direction triad
struct Triad {
  double nxd, nyd, nzd;    // line of sight, float64 (positions, mask)
  float nx, ny, nz;
  float nxl, nyl, nzl;     // n - (float)n: low parts, so that B.n does not carry a per-sightline 3e-8 bias
  float eNx, eNy, eNz;     // towards Galactic north
  float eEx, eEy;          // towards increasing l (z component is 0)
  double scale;            // Delta_i / delta: this sightline's segment length relative to the plan's (1 without a box)
  float scalef;
};

__device__ __forceinline__ Triad load_triad(const double* __restrict__ dirs, int64_t pix) {
  const double4 d = *reinterpret_cast<const double4*>(dirs + 4 * pix);  // cl, sl, cb, sb
  Triad t;
  t.nxd = d.z * d.x; t.nyd = d.z * d.y; t.nzd = d.w;
  t.nx = (float)t.nxd; t.ny = (float)t.nyd; t.nz = (float)t.nzd;
  t.nxl = (float)(t.nxd - (double)t.nx); t.nyl = (float)(t.nyd - (double)t.ny); t.nzl = (float)(t.nzd - (double)t.nz);
  t.eNx = (float)(-d.w * d.x); t.eNy = (float)(-d.w * d.y); t.eNz = (float)d.z;
  t.eEx = (float)(-d.y); t.eEy = (float)d.x;
  t.scale = 1.0; t.scalef = 1.0f;
  return t;
}
// With the per-sightline segment length: positions step by delta * scale, and because the Faraday constants k_f and
// the intensity coefficients c_f are folded with the plan's delta, n_e (which enters only through the Faraday
// integrand n_e B_LOS Delta) and the final sums (cotangents in the adjoint) are multiplied by scale.
__device__ __forceinline__ Triad load_triad(const Geometry& geo, int64_t pix) {
  Triad t = load_triad(geo.dirs, pix);
  if (geo.path) { t.scale = geo.path[pix]; t.scalef = (float)t.scale; }
  return t;
}

// What one sample hands to the integrator (fp32): B projections, densities.
struct SampleF {
  float Bpar, BN, BE;  // uG
  float N0, ne;
};

// ------------------------------------------------------------------------------------------------
// Analytic model, fp32 fast chain.  x,y,z,rho2 are the float64 sample coordinates rounded to fp32;
// `inside` is the annulus test 3 < rho < 20 kpc taken in float64 (S:C-2#7).
// Everything needed by the adjoint is kept in AnalyticAux.
// ------------------------------------------------------------------------------------------------
struct AnalyticAux {
  float ir, rho, xr, yr;   // 1/rho, rho, x/rho, y/rho
  float lr;                // ln(rho/8)
  float sp, cp, sc, cc;    // sin/cos psi, sin/cos chi
  float t;                 // tanh(z / 1 kpc)
  float A;                 // exp(-(rho-8)/h_b) inside the annulus, else 0 (unit amplitude: B_disc = b0 A [...])
  float N0u, neu;          // N_0 / n0 and n_e / ne0 (unit amplitudes)
  float u, L, R;           // halo: u, 1/(1+u^2), (rho/r_h) exp(1-rho/r_h)
  float thz, thez;         // tanh(z/h_z), tanh(z/h_ez)
};

// The part of the analytic evaluation that does not depend on the model parameters (S:8(a) A12: shared by the
// parameter vectors of a batch): cylindrical geometry, ln(rho/8), tanh(z / 1 kpc).  4 MUFU.
struct SharedGeomF {
  float ir, rho, xr, yr;   // 1/rho, rho, x/rho, y/rho
  float lr;                // ln(rho/8)
  float az, t;             // |z|, tanh(z / 1 kpc)
};
__device__ __forceinline__ void analytic_shared_f32(float x, float y, float z, float rho2, SharedGeomF& g) {
  const float kLog2e = 1.4426950408889634f;
  rho2 = fmaxf(rho2, 1.0e-30f);
  g.ir = mufu_rsqrt(rho2);
  g.rho = rho2 * g.ir;
  g.xr = x * g.ir; g.yr = y * g.ir;
  g.az = fabsf(z);
  g.lr = (mufu_lg2(rho2) - 6.0f) * 0.34657359027997264f;        // ln(rho/8) = ln2/2 (lg2 rho^2 - 6)
  const float e1 = mufu_ex2(-2.0f * kLog2e * g.az);             // tanh(|z|) = (1-e)/(1+e)
  g.t = copysignf((1.0f - e1) * mufu_rcp(1.0f + e1), z);
}

// The parameter-dependent part.  kFastTrig: sin/cos of the pitch and tilt angles on the MUFU (abs err 5e-7: enough for
// the 1e-3 gradient bound)
template <bool kHalo, bool kFastTrig>
__device__ __forceinline__ void analytic_fields_f32(const BatchConsts& P, const Triad& T, const SharedGeomF& g, float z,
                                                    bool inside, SampleF& S, AnalyticAux& a) {
  const float kLog2e = 1.4426950408889634f;
  a.ir = g.ir; a.rho = g.rho; a.xr = g.xr; a.yr = g.yr; a.lr = g.lr; a.t = g.t;
  const float az = g.az;
  // --- disc: B = A [cos psi cos chi rho_hat + sin psi cos chi phi_hat + sin chi z_hat]   Eq.(13)
  const float psi = fmaf(P.p[2], a.lr, P.p[1]);
  if (kFastTrig) { a.sp = mufu_sin(psi); a.cp = mufu_cos(psi); }
  else if (P.angles_small) sincos_fma_small(psi, a.sp, a.cp);
  else sincos_fma(psi, a.sp, a.cp);
  const float chi = P.p[3] * a.t;
  if (kFastTrig) { a.sc = mufu_sin(chi); a.cc = mufu_cos(chi); }
  else if (P.angles_small) sincos_fma_small(chi, a.sc, a.cc);
  else sincos_fma(chi, a.sc, a.cc);
  float rad = 1.0f;
  if (P.k_hb != 0.0f) rad = mufu_ex2(P.k_hb * (a.rho - 8.0f));
  a.A = inside ? rad : 0.0f;
  const float Ab = P.p[0] * a.A;
  const float Brho = Ab * a.cp * a.cc;
  float Bphi = Ab * a.sp * a.cc;
  const float Bz = Ab * a.sc;
  // The three reciprocals of a sample -- the halo's Lorentzian 1/(1+u^2) and the two sech^2 denominators 1/(1+e)^2 --
  // share ONE MUFU.RCP of their product (the kernels are XU-bound: a reciprocal costs 8 issue cycles of that pipe, a
  // multiply one of the FMA pipe); every factor is >= 1, the product stays far below the fp32 range.
  const float ez = mufu_ex2(P.k_hz * az);
  const float dz = 1.0f + ez, dz2 = dz * dz;
  const float ee = mufu_ex2(P.k_hez * az);
  const float de = 1.0f + ee, de2 = de * de;
  float iz, ie;
  if (kHalo) {  // toroidal halo, S:App.C
    a.u = (az - P.p[6]) * P.inv_wh;
    const float q = a.rho * P.inv_rh;
    const float lu = fmaf(a.u, a.u, 1.0f), dd = dz2 * de2;
    const float inv = mufu_rcp(lu * dd);
    a.L = inv * dd;
    const float il = inv * lu;
    iz = il * de2; ie = il * dz2;
    a.R = q * mufu_ex2(kLog2e * (1.0f - q));
    Bphi = fmaf(P.p[5] * a.L, a.R, Bphi);
  } else {
    const float inv = mufu_rcp(dz2 * de2);
    iz = inv * de2; ie = inv * dz2;
  }
  const float Bx = Brho * a.xr - Bphi * a.yr;
  const float By = fmaf(Brho, a.yr, Bphi * a.xr);
  S.Bpar = fmaf(Bx, T.nx, fmaf(By, T.ny, Bz * T.nz));           // B.n, signed (S:C-2#3)
  S.BN = fmaf(Bx, T.eNx, fmaf(By, T.eNy, Bz * T.eNz));          // Eq.(8) numerator
  S.BE = fmaf(Bx, T.eEx, By * T.eEy);                           // Eq.(8) denominator (S:C-2#4)
  // --- N_0 = n0 exp(-rho/h_r) sech^2(z/h_z)  Eq.(12);  sech^2 w = 4e/(1+e)^2, e = exp(-2|w|)
  a.N0u = 4.0f * mufu_ex2(P.k_hr * a.rho) * ez * iz;
  S.N0 = P.p[9] * a.N0u;
  a.thz = copysignf((1.0f - ez) * dz * iz, z);                  // tanh = (1-e)/(1+e)
  a.neu = 4.0f * mufu_ex2(P.k_her * a.rho) * ee * ie;
  S.ne = P.p[13] * a.neu;
  a.thez = copysignf((1.0f - ee) * de * ie, z);
}

template <bool kHalo, bool kFastTrig = false>
__device__ __forceinline__ void eval_analytic_f32(const BatchConsts& P, const Triad& T, float x, float y,
                                                  float z, float rho2, bool inside, SampleF& S,
                                                  AnalyticAux& a) {
  SharedGeomF g;
  analytic_shared_f32(x, y, z, rho2, g);
  analytic_fields_f32<kHalo, kFastTrig>(P, T, g, z, inside, S, a);
}

// ------------------------------------------------------------------------------------------------
// The paper's own 16-parameter model, Eq.(16) P:L283-289 (Table 3): four WMAP spirals B_k stacked with
// the printed weights and component permutations,
//   B_x = .6 B1x + .3 B2x + .1 B3z + .3 B4y,  B_y = .6 B1y + .3 B2z + .1 B3y + .3 B4x,  B_z = .6 B1z + .3 B2y + .1 B3x + .3 B4z
// (DESIGN.md section 3 on the "rotation before stacking").  CR / n_e / alpha from aux as for DISC4.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float stack_w(int k) { return k == 0 ? 0.6f : (k == 2 ? 0.1f : 0.3f); }
__device__ __forceinline__ double stack_w_d(int k) { return k == 0 ? 0.6 : (k == 2 ? 0.1 : 0.3); }
template <typename R> __device__ __forceinline__ R stack_weight(int k);
template <> __device__ __forceinline__ float stack_weight<float>(int k) { return stack_w(k); }
template <> __device__ __forceinline__ double stack_weight<double>(int k) { return stack_w_d(k); }
// component of B_k that feeds component c of the total
__device__ __forceinline__ constexpr int stack_src(int k, int c) {
  return k == 0 ? c : (k == 1 ? (c == 0 ? 0 : (c == 1 ? 2 : 1)) : (k == 2 ? (c == 0 ? 2 : (c == 1 ? 1 : 0)) : (c == 0 ? 1 : (c == 1 ? 0 : 2))));
}

struct StackAux {
  float ir, rho, xr, yr, lr, t;
  float sp[4], cp[4], sc[4], cc[4];
  float mask;              // 1 inside the annulus 3 < rho < 20 kpc, else 0
};

template <bool kFastTrig>
__device__ __forceinline__ void eval_stack16_f32(const BatchConsts& P, const Triad& T, float x, float y, float z,
                                                 float rho2, bool inside, SampleF& S, StackAux& a) {
  const float kLog2e = 1.4426950408889634f;
  rho2 = fmaxf(rho2, 1.0e-30f);
  a.ir = mufu_rsqrt(rho2);
  a.rho = rho2 * a.ir;
  a.xr = x * a.ir; a.yr = y * a.ir;
  const float az = fabsf(z);
  a.lr = (mufu_lg2(rho2) - 6.0f) * 0.34657359027997264f;
  const float e1 = mufu_ex2(-2.0f * kLog2e * az);
  a.t = copysignf((1.0f - e1) * mufu_rcp(1.0f + e1), z);
  a.mask = inside ? 1.0f : 0.0f;
  float B[3] = {0.0f, 0.0f, 0.0f};
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const float psi = fmaf(P.sp[4 * k + 2], a.lr, P.sp[4 * k + 1]);
    const float chi = P.sp[4 * k + 3] * a.t;
    if (kFastTrig) { a.sp[k] = mufu_sin(psi); a.cp[k] = mufu_cos(psi); a.sc[k] = mufu_sin(chi); a.cc[k] = mufu_cos(chi); }
    else { sincos_fma(psi, a.sp[k], a.cp[k]); sincos_fma(chi, a.sc[k], a.cc[k]); }
    const float A = a.mask * stack_w(k) * P.sp[4 * k];
    const float Brho = A * a.cp[k] * a.cc[k], Bphi = A * a.sp[k] * a.cc[k];
    const float comp[3] = {Brho * a.xr - Bphi * a.yr, fmaf(Brho, a.yr, Bphi * a.xr), A * a.sc[k]};
#pragma unroll
    for (int c = 0; c < 3; ++c) B[c] += comp[stack_src(k, c)];
  }
  S.Bpar = fmaf(B[0], T.nx, fmaf(B[1], T.ny, B[2] * T.nz));
  S.BN = fmaf(B[0], T.eNx, fmaf(B[1], T.eNy, B[2] * T.eNz));
  S.BE = fmaf(B[0], T.eEx, B[1] * T.eEy);
  const float ez = mufu_ex2(P.k_hz * az), dz = 1.0f + ez;
  S.N0 = 4.0f * P.p[9] * mufu_ex2(P.k_hr * a.rho) * ez * mufu_rcp(dz * dz);
  const float ee = mufu_ex2(P.k_hez * az), de = 1.0f + ee;
  S.ne = 4.0f * P.p[13] * mufu_ex2(P.k_her * a.rho) * ee * mufu_rcp(de * de);
}

// ------------------------------------------------------------------------------------------------
// Analytic model, float64 chain for the Faraday integrand (and, reused, for the emission inputs).
// Used only for sightlines whose Faraday rotation is so large that fp32 round-off in n_e B_LOS
// would exceed the parity tolerance.
// ------------------------------------------------------------------------------------------------
// digamma for x > 0 (prologue only)
__device__ inline double digamma_d(double x) {
  double r = 0.0;
  while (x < 10.0) { r -= 1.0 / x; x += 1.0; }
  const double f = 1.0 / (x * x);
  const double ser = f * (1.0 / 12.0 - f * (1.0 / 120.0 - f * (1.0 / 252.0 - f * (1.0 / 240.0 - f * (1.0 / 132.0)))));
  return r + log(x) - 0.5 / x - ser;
}

}  // namespace synax
