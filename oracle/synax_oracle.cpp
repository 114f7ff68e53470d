// synax_oracle.cpp -- float64 CPU ORACLE for the synax line-of-sight hot path.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
// It shares no source, header, table or constant generator with the CUDA library
// (paper_2410_01136_b200/csrc); neither includes nor imports the other.
//
// It is a plain, slow, step-by-step restatement of arXiv:2410.01136 ("synax"), sections
// 2.1-2.3, in the paper's order and notation (citations: P:L<n> = PAPER.md line n;
// S:<tag> = SURVEY.md section 8(c) reading, all listed again in DESIGN.md):
//
//   step 1  direction of HEALPix RING pixel i -> (l_i, b_i)             P:L108, Gorski+05
//   step 2  N_int equal segments, midpoints r_{i,n} = r_obs + s_n n     P:L108, r_obs P:L49
//   step 3  fields B, N_0, n_e, alpha at r_{i,n}                        P:L99-110, Eq.12-13
//   step 4  B_LOS = B.n (signed, S:C-2#3), B_N, B_E (Eq.8, S:C-2#4)
//   step 5  j_I  Eq.(2) in Gaussian CGS, literally
//   step 6  j_P  Eq.(5) in Gaussian CGS, literally
//   step 7  chi_0 = atan2(B_N, B_E)    Eq.(8)
//   step 8  RM_n = K_F * Delta*(sum_{m<n} n_e B_LOS + 1/2 (n_e B_LOS)_n)   Eq.(7), S:C-2#5
//   step 9  chi = RM lambda^2 + chi_0  Eq.(6)
//   step 10 I,Q,U = sum_n j * {1, cos 2chi, sin 2chi} * Delta_r  Eq.(9)
//           converted to Rayleigh-Jeans brightness temperature (K), S:C-2#1
//
// and of the reverse-mode derivative (VJP) of steps 1-10 w.r.t. the model parameters,
// derived by hand (the paper uses JAX AD) and pinned in tests/ by central
// finite differences of the forward.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): uniform-slab closed forms Eq.(10), the
// discrete Burn-slab closed form of Eq.(11), HEALPix ring facts, Gamma/digamma textbook
// values, the 0.812 Faraday constant, invariants, gridded==uniform, convergence order,
// finite differences for every gradient.  Functions without such a pin: none known;
// absolute map values of the spiral/halo models are pinned only through those
// invariants and spot values ("parity unpinned" beyond them).
//
// Build:  g++ -O2 -fopenmp -shared -fPIC -o liboracle.so synax_oracle.cpp   (no fast-math)

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <limits>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---------------------------------------------------------------------------------------
// Physical constants, Gaussian CGS, CODATA 2018 (exact SI values converted).
// ---------------------------------------------------------------------------------------
const double QE_ESU   = 4.80320471257e-10;      // esu
const double ME_G   = 9.1093837015e-28;       // g
const double C_CMS   = 2.99792458e10;          // cm / s
const double KB_ERG   = 1.380649e-16;           // erg / K
const double PC_CM = 3.0856775814913673e18;  // cm
const double KPC_CM = 1.0e3 * PC_CM;
const double PI = 3.14159265358979323846264338327950288;

// model kinds (the oracle's own numbering; the python wrapper maps names to these)
enum { KIND_DISC4 = 0, KIND_FULL16 = 1, KIND_GRID_B = 2, KIND_UNIFORM = 3, KIND_STACK16 = 4 };

struct Model {
  int kind;
  const double* params;  // DISC4: 4, FULL16: 16, UNIFORM: 6, GRID_B: grid [nx][ny][nz][3]
  const double* aux;     // DISC4/GRID_B: {C0,h_r,h_z,alpha,ne0,h_er,h_ez}; UNIFORM: {R0} or NULL
  int64_t nx, ny, nz;    // GRID_B
  double lx, ly, lz;     // GRID_B box lengths (kpc), centred on the Galactic centre
  const double* observer;  // r_obs (kpc), used by the UNIFORM toy sphere
};

int n_params_of(const Model& m) {
  switch (m.kind) {
    case KIND_DISC4: return 4;
    case KIND_FULL16: return 16;
    case KIND_UNIFORM: return 6;
    case KIND_STACK16: return 16;
    case KIND_GRID_B: return (int)(m.nx * m.ny * m.nz * 3);
  }
  return -1;
}

struct Fields {
  double B[3];   // micro-gauss
  double N0;     // cm^-3
  double ne;     // cm^-3
  double alpha;  // CR spectral index
};

// digamma psi(x), x > 0: upward recurrence to x >= 12, then the asymptotic series.
double digamma(double x) {
  double r = 0.0;
  while (x < 12.0) { r -= 1.0 / x; x += 1.0; }
  const double f = 1.0 / (x * x);
  // ln x - 1/(2x) - sum B_2k / (2k x^2k)
  const double series = f * (1.0 / 12.0 - f * (1.0 / 120.0 - f * (1.0 / 252.0 - f * (1.0 / 240.0 -
                        f * (1.0 / 132.0 - f * (691.0 / 32760.0 - f * (1.0 / 12.0)))))));
  return r + std::log(x) - 0.5 / x - series;
}

double sech2(double w) { const double c = std::cosh(w); return 1.0 / (c * c); }

// WMAP cosmic-ray density, Eq.(12):  N_0 = C_0 exp(-rho/h_r) sech^2(z/h_z)
double exp_disc(double amp, double hr, double hz, double rho, double z) {
  return amp * std::exp(-rho / hr) * sech2(z / hz);
}

// WMAP logarithmic spiral, Eq.(13), times exp(-(rho-8)/h_b) (S:App.C; h_b=inf for
// DISC4).  Zero outside the open annulus 3 < rho < 20 kpc (S:C-2#7).
void disc_field(double b0, double psi0, double psi1, double chi0, double inv_hb,
                double x, double y, double z, double B[3]) {
  B[0] = B[1] = B[2] = 0.0;
  const double rho = std::sqrt(x * x + y * y);
  if (!(rho > 3.0 && rho < 20.0)) return;
  const double psi = psi0 + psi1 * std::log(rho / 8.0);
  const double chi = chi0 * std::tanh(z / 1.0);
  const double A = b0 * std::exp(-(rho - 8.0) * inv_hb);
  const double rhat[2] = {x / rho, y / rho};
  const double phat[2] = {-y / rho, x / rho};
  const double Brho = A * std::cos(psi) * std::cos(chi);
  const double Bphi = A * std::sin(psi) * std::cos(chi);
  B[0] = Brho * rhat[0] + Bphi * phat[0];
  B[1] = Brho * rhat[1] + Bphi * phat[1];
  B[2] = A * std::sin(chi);
}

// Toroidal halo (S:App.C, not in PAPER.md): B_h L(z) R(rho) phi_hat,
// L = 1/(1+u^2), u = (|z|-z_h0)/w_h, R = (rho/r_h) exp(1 - rho/r_h).
void halo_field(double Bh, double zh0, double rh, double wh, double x, double y, double z, double B[3]) {
  B[0] = B[1] = B[2] = 0.0;
  const double rho = std::sqrt(x * x + y * y);
  if (rho == 0.0) return;  // R(0) = 0
  const double u = (std::fabs(z) - zh0) / wh;
  const double L = 1.0 / (1.0 + u * u);
  const double R = (rho / rh) * std::exp(1.0 - rho / rh);
  const double Bphi = Bh * L * R;
  B[0] = Bphi * (-y / rho);
  B[1] = Bphi * (x / rho);
}

// Trilinear interpolation on a regular grid with nodes on the box faces (S:C-2#12, App.C):
// x_i = -lx/2 + i lx/(nx-1); layout [ix][iy][iz][c]; zero outside the box.  P:L106-110.
bool grid_cell(const Model& m, double x, double y, double z, int64_t idx[3], double t[3]) {
  const double p[3] = {x, y, z};
  const double len[3] = {m.lx, m.ly, m.lz};
  const int64_t n[3] = {m.nx, m.ny, m.nz};
  for (int a = 0; a < 3; ++a) {
    const double u = (p[a] + 0.5 * len[a]) * (double)(n[a] - 1) / len[a];
    if (!(u >= 0.0 && u <= (double)(n[a] - 1))) return false;
    int64_t i = (int64_t)std::floor(u);
    if (i < 0) i = 0;
    if (i > n[a] - 2) i = n[a] - 2;
    idx[a] = i;
    t[a] = u - (double)i;
  }
  return true;
}

void grid_field(const Model& m, double x, double y, double z, double B[3]) {
  B[0] = B[1] = B[2] = 0.0;
  int64_t i[3]; double t[3];
  if (!grid_cell(m, x, y, z, i, t)) return;
  for (int a = 0; a < 2; ++a)
    for (int b = 0; b < 2; ++b)
      for (int d = 0; d < 2; ++d) {
        const double w = (a ? t[0] : 1.0 - t[0]) * (b ? t[1] : 1.0 - t[1]) * (d ? t[2] : 1.0 - t[2]);
        const double* g = m.params + (((i[0] + a) * m.ny + (i[1] + b)) * m.nz + (i[2] + d)) * 3;
        B[0] += w * g[0]; B[1] += w * g[1]; B[2] += w * g[2];
      }
}

// Gridded scalar fields (the paper's n_e is the YMW16 model sampled on a (256,256,64) grid;
// N_0 may be gridded the same way): regular grid [nx][ny][nz], nodes on the faces of a box centred on the
// Galactic centre, trilinear interpolation, zero outside.  Set process-wide by oracle_set_scalar_grids; they
// REPLACE the analytic exponential discs of the DISC4 and GRID_B models (whose n_e / N_0 are not differentiated).
struct ScalarGrid { const double* g = nullptr; int64_t n[3] = {0, 0, 0}; double len[3] = {0, 0, 0}; };
ScalarGrid g_ne_grid, g_n0_grid;
double scalar_grid_value(const ScalarGrid& S, double x, double y, double z) {
  const double p[3] = {x, y, z};
  int64_t i[3]; double t[3];
  for (int a = 0; a < 3; ++a) {
    const double u = (p[a] + 0.5 * S.len[a]) * (double)(S.n[a] - 1) / S.len[a];
    if (!(u >= 0.0 && u <= (double)(S.n[a] - 1))) return 0.0;
    int64_t k = (int64_t)std::floor(u);
    if (k > S.n[a] - 2) k = S.n[a] - 2;
    i[a] = k; t[a] = u - (double)k;
  }
  double v = 0.0;
  for (int a = 0; a < 2; ++a)
    for (int b = 0; b < 2; ++b)
      for (int d = 0; d < 2; ++d)
        v += (a ? t[0] : 1.0 - t[0]) * (b ? t[1] : 1.0 - t[1]) * (d ? t[2] : 1.0 - t[2]) *
             S.g[((i[0] + a) * S.n[1] + (i[1] + b)) * S.n[2] + (i[2] + d)];
  return v;
}

// The paper's 16-parameter model, Eq.(16): four WMAP spirals B_k (parameters (b0, psi0, psi1, chi0)_k,
// k = 1..4, Table 3) stacked with the printed weights and component permutations:
//   B_x = 0.6 B1x + 0.3 B2x + 0.1 B3z + 0.3 B4y
//   B_y = 0.6 B1y + 0.3 B2z + 0.1 B3y + 0.3 B4x
//   B_z = 0.6 B1z + 0.3 B2y + 0.1 B3x + 0.3 B4z
// kStackSrc[k][c] = which component of B_k feeds component c of the total.  (The text also says B_2..4 "are
// rotated before stacking" without giving the rotation; the permutations printed in Eq.(16) are taken as
// that rotation -- DESIGN.md section 3.)
const double kStackW[4] = {0.6, 0.3, 0.1, 0.3};
const int kStackSrc[4][3] = {{0, 1, 2}, {0, 2, 1}, {2, 1, 0}, {1, 0, 2}};

// step 3: all fields at one point.
void eval_fields(const Model& m, const double r[3], Fields& F) {
  const double x = r[0], y = r[1], z = r[2];
  const double rho = std::sqrt(x * x + y * y);
  const double* p = m.params;
  switch (m.kind) {
    case KIND_DISC4: {
      disc_field(p[0], p[1], p[2], p[3], 0.0, x, y, z, F.B);
      const double* a = m.aux;
      F.N0 = exp_disc(a[0], a[1], a[2], rho, z);
      F.alpha = a[3];
      F.ne = exp_disc(a[4], a[5], a[6], rho, z);
    } break;
    case KIND_FULL16: {
      double Bd[3], Bh[3];
      disc_field(p[0], p[1], p[2], p[3], 1.0 / p[4], x, y, z, Bd);
      halo_field(p[5], p[6], p[7], p[8], x, y, z, Bh);
      for (int c = 0; c < 3; ++c) F.B[c] = Bd[c] + Bh[c];
      F.N0 = exp_disc(p[9], p[10], p[11], rho, z);
      F.alpha = p[12];
      F.ne = exp_disc(p[13], p[14], p[15], rho, z);
    } break;
    case KIND_GRID_B: {
      grid_field(m, x, y, z, F.B);
      const double* a = m.aux;
      F.N0 = exp_disc(a[0], a[1], a[2], rho, z);
      F.alpha = a[3];
      F.ne = exp_disc(a[4], a[5], a[6], rho, z);
    } break;
    case KIND_STACK16: {
      F.B[0] = F.B[1] = F.B[2] = 0.0;
      for (int k = 0; k < 4; ++k) {
        double Bk[3];
        disc_field(p[4 * k], p[4 * k + 1], p[4 * k + 2], p[4 * k + 3], 0.0, x, y, z, Bk);
        for (int c = 0; c < 3; ++c) F.B[c] += kStackW[k] * Bk[kStackSrc[k][c]];
      }
      const double* a = m.aux;
      F.N0 = exp_disc(a[0], a[1], a[2], rho, z);
      F.alpha = a[3];
      F.ne = exp_disc(a[4], a[5], a[6], rho, z);
    } break;
    case KIND_UNIFORM: {
      // homogeneous toy fields; aux[0] = R0 > 0 confines them to a sphere of radius
      // R0 around the observer ("zero outside").
      bool inside = true;
      if (m.aux && m.aux[0] > 0.0) {
        const double dx = x - m.observer[0], dy = y - m.observer[1], dz = z - m.observer[2];
        inside = (dx * dx + dy * dy + dz * dz) <= m.aux[0] * m.aux[0];
      }
      F.B[0] = inside ? p[0] : 0.0; F.B[1] = inside ? p[1] : 0.0; F.B[2] = inside ? p[2] : 0.0;
      F.N0 = inside ? p[3] : 0.0;
      F.ne = inside ? p[4] : 0.0;
      F.alpha = p[5];
    } break;
  }
  if (m.kind == KIND_DISC4 || m.kind == KIND_GRID_B || m.kind == KIND_STACK16) {
    if (g_ne_grid.g) F.ne = scalar_grid_value(g_ne_grid, x, y, z);
    if (g_n0_grid.g) F.N0 = scalar_grid_value(g_n0_grid, x, y, z);
  }
}

// Transpose of step 3: field cotangents (Bbar, N0bar, nebar, alphabar) -> parameter gradient.
// grad has n_params entries (grid: the whole grid), accumulated (+=).
void disc_field_vjp(double b0, double psi0, double psi1, double chi0, double hb, bool has_hb,
                    double x, double y, double z, const double Bb[3],
                    double* g_b0, double* g_psi0, double* g_psi1, double* g_chi0, double* g_hb) {
  const double rho = std::sqrt(x * x + y * y);
  if (!(rho > 3.0 && rho < 20.0)) return;
  const double lr = std::log(rho / 8.0);
  const double psi = psi0 + psi1 * lr;
  const double t = std::tanh(z / 1.0);
  const double chi = chi0 * t;
  const double s = has_hb ? std::exp(-(rho - 8.0) / hb) : 1.0;
  const double A = b0 * s;
  const double cp = std::cos(psi), sp = std::sin(psi), cc = std::cos(chi), sc = std::sin(chi);
  // cylindrical components of the cotangent
  const double Bb_rho = (Bb[0] * x + Bb[1] * y) / rho;
  const double Bb_phi = (-Bb[0] * y + Bb[1] * x) / rho;
  const double Bb_z = Bb[2];
  const double B_dot_Bb = A * (cp * cc * Bb_rho + sp * cc * Bb_phi + sc * Bb_z);
  // dB/db0 = B_disc / b0 (App. D.3), written as the unit-amplitude field so that b0 = 0 is not 0/0
  *g_b0 += s * (cp * cc * Bb_rho + sp * cc * Bb_phi + sc * Bb_z);
  const double dpsi = A * cc * (-sp * Bb_rho + cp * Bb_phi);
  *g_psi0 += dpsi;
  *g_psi1 += lr * dpsi;
  *g_chi0 += t * A * (-sc * (cp * Bb_rho + sp * Bb_phi) + cc * Bb_z);
  if (has_hb) *g_hb += B_dot_Bb * (rho - 8.0) / (hb * hb);
}

void halo_field_vjp(double Bh, double zh0, double rh, double wh, double x, double y, double z,
                    const double Bb[3], double* g) {  // g[0..3] = d/d(Bh, zh0, rh, wh)
  const double rho = std::sqrt(x * x + y * y);
  if (rho == 0.0) return;
  const double u = (std::fabs(z) - zh0) / wh;
  const double L = 1.0 / (1.0 + u * u);
  const double R = (rho / rh) * std::exp(1.0 - rho / rh);
  const double Bb_phi = (-Bb[0] * y + Bb[1] * x) / rho;
  g[0] += L * R * Bb_phi;
  // dL/du = -2u L^2 ; du/dzh0 = -1/wh ; du/dwh = -u/wh
  g[1] += Bh * R * (2.0 * u * L * L / wh) * Bb_phi;
  g[3] += Bh * R * (2.0 * u * u * L * L / wh) * Bb_phi;
  // dR/drh = R (rho/rh - 1)/rh
  g[2] += Bh * L * R * (rho / rh - 1.0) / rh * Bb_phi;
}

void exp_disc_vjp(double amp, double hr, double hz, double rho, double z, double bar,
                  double* g_amp, double* g_hr, double* g_hz) {
  const double v = exp_disc(amp, hr, hz, rho, z);
  *g_amp += bar * exp_disc(1.0, hr, hz, rho, z);   // d/d amp = profile at unit amplitude (App. D.3), finite at amp = 0
  *g_hr += bar * v * rho / (hr * hr);
  *g_hz += bar * v * 2.0 * std::tanh(z / hz) * z / (hz * hz);
}

void fields_vjp(const Model& m, const double r[3], const double Bb[3], double N0b, double neb,
                double alphab, double* grad) {
  const double x = r[0], y = r[1], z = r[2];
  const double rho = std::sqrt(x * x + y * y);
  const double* p = m.params;
  switch (m.kind) {
    case KIND_DISC4: {
      double dummy = 0.0;
      disc_field_vjp(p[0], p[1], p[2], p[3], 0.0, false, x, y, z, Bb, &grad[0], &grad[1], &grad[2],
                     &grad[3], &dummy);
      // CR / n_e / alpha come from aux and are not differentiated (S:App.C)
    } break;
    case KIND_STACK16: {
      for (int k = 0; k < 4; ++k) {   // transpose of the stacking: cotangent of B_k's component kStackSrc[k][c] += w_k Bb[c]
        double Bbk[3] = {0.0, 0.0, 0.0}, dummy = 0.0;
        for (int c = 0; c < 3; ++c) Bbk[kStackSrc[k][c]] += kStackW[k] * Bb[c];
        disc_field_vjp(p[4 * k], p[4 * k + 1], p[4 * k + 2], p[4 * k + 3], 0.0, false, x, y, z, Bbk, &grad[4 * k],
                       &grad[4 * k + 1], &grad[4 * k + 2], &grad[4 * k + 3], &dummy);
      }
    } break;
    case KIND_FULL16: {
      disc_field_vjp(p[0], p[1], p[2], p[3], p[4], true, x, y, z, Bb, &grad[0], &grad[1], &grad[2],
                     &grad[3], &grad[4]);
      halo_field_vjp(p[5], p[6], p[7], p[8], x, y, z, Bb, &grad[5]);
      exp_disc_vjp(p[9], p[10], p[11], rho, z, N0b, &grad[9], &grad[10], &grad[11]);
      grad[12] += alphab;
      exp_disc_vjp(p[13], p[14], p[15], rho, z, neb, &grad[13], &grad[14], &grad[15]);
    } break;
    case KIND_GRID_B: {
      int64_t i[3]; double t[3];
      if (!grid_cell(m, x, y, z, i, t)) return;
      for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b)
          for (int d = 0; d < 2; ++d) {
            const double w = (a ? t[0] : 1.0 - t[0]) * (b ? t[1] : 1.0 - t[1]) * (d ? t[2] : 1.0 - t[2]);
            double* g = grad + (((i[0] + a) * m.ny + (i[1] + b)) * m.nz + (i[2] + d)) * 3;
            g[0] += w * Bb[0]; g[1] += w * Bb[1]; g[2] += w * Bb[2];
          }
    } break;
    case KIND_UNIFORM: {
      bool inside = true;
      if (m.aux && m.aux[0] > 0.0) {
        const double dx = x - m.observer[0], dy = y - m.observer[1], dz = z - m.observer[2];
        inside = (dx * dx + dy * dy + dz * dz) <= m.aux[0] * m.aux[0];
      }
      if (inside) { grad[0] += Bb[0]; grad[1] += Bb[1]; grad[2] += Bb[2]; grad[3] += N0b; grad[4] += neb; }
      grad[5] += alphab;
    } break;
  }
}

// ---------------------------------------------------------------------------------------
// Emissivities, Eq.(2) and Eq.(5), literally, in Gaussian CGS (erg s^-1 cm^-3 Hz^-1 sr^-1).
// B_trans in gauss, N_0 in cm^-3, nu in Hz.
// ---------------------------------------------------------------------------------------
double emissivity_I(double nu, double Btrans, double N0, double alpha) {
  if (Btrans <= 0.0) return 0.0;  // S:C-2#19
  return std::sqrt(3.0) * QE_ESU * QE_ESU * QE_ESU * Btrans * N0 / (8.0 * PI * ME_G * C_CMS * C_CMS) *
         std::pow(4.0 * PI * nu * ME_G * C_CMS / (3.0 * QE_ESU * Btrans), (1.0 - alpha) / 2.0) *
         std::pow(2.0, (alpha + 1.0) / 2.0) / (alpha + 1.0) *
         std::tgamma(alpha / 4.0 - 1.0 / 12.0) * std::tgamma(alpha / 4.0 + 19.0 / 12.0);
}
double emissivity_P(double nu, double Btrans, double N0, double alpha) {
  if (Btrans <= 0.0) return 0.0;
  return std::sqrt(3.0) * QE_ESU * QE_ESU * QE_ESU * Btrans * N0 / (8.0 * PI * ME_G * C_CMS * C_CMS) *
         std::pow(4.0 * PI * nu * ME_G * C_CMS / (3.0 * QE_ESU * Btrans), (1.0 - alpha) / 2.0) *
         std::pow(2.0, (alpha - 3.0) / 2.0) *
         std::tgamma(alpha / 4.0 - 1.0 / 12.0) * std::tgamma(alpha / 4.0 + 7.0 / 12.0);
}
// d ln j / d alpha at fixed (nu, Btrans, N0)
double dln_emissivity_I_dalpha(double nu, double Btrans, double alpha) {
  return -0.5 * std::log(4.0 * PI * nu * ME_G * C_CMS / (3.0 * QE_ESU * Btrans)) + 0.5 * std::log(2.0) -
         1.0 / (alpha + 1.0) + 0.25 * digamma(alpha / 4.0 - 1.0 / 12.0) +
         0.25 * digamma(alpha / 4.0 + 19.0 / 12.0);
}
double dln_emissivity_P_dalpha(double nu, double Btrans, double alpha) {
  return -0.5 * std::log(4.0 * PI * nu * ME_G * C_CMS / (3.0 * QE_ESU * Btrans)) + 0.5 * std::log(2.0) +
         0.25 * digamma(alpha / 4.0 - 1.0 / 12.0) + 0.25 * digamma(alpha / 4.0 + 7.0 / 12.0);
}

// Faraday constant of Eq.(7): q_e^3 / (2 pi m_e^2 c^4)  [rad cm^-2 per (cm^-3 G cm)],
// converted so that RM is in rad m^-2 when n_e is in cm^-3, B in micro-gauss, path in kpc.
double faraday_K_per_kpc() {
  const double K_cgs = QE_ESU * QE_ESU * QE_ESU / (2.0 * PI * ME_G * ME_G * C_CMS * C_CMS * C_CMS * C_CMS);
  return K_cgs * 1.0e4 /* cm^-2 -> m^-2 */ * 1.0e-6 /* uG -> G */ * KPC_CM;
}

// Rayleigh-Jeans brightness temperature per unit specific intensity (S:C-2#1).
double rayleigh_jeans(double nu) { return C_CMS * C_CMS / (2.0 * KB_ERG * nu * nu); }

// ---------------------------------------------------------------------------------------
// step 1: HEALPix RING pixel centre (Gorski et al. 2005), S:App.B.  z = cos(theta).
// ---------------------------------------------------------------------------------------
int64_t isqrt64(int64_t v) {
  int64_t r = (int64_t)std::floor(std::sqrt((double)v));
  while (r * r > v) --r;
  while ((r + 1) * (r + 1) <= v) ++r;
  return r;
}

void pix2ang_ring(int64_t nside, int64_t p, double* z, double* phi) {
  const int64_t npix = 12 * nside * nside;
  const int64_t ncap = 2 * nside * (nside - 1);
  if (p < ncap) {  // north polar cap
    const int64_t i = (1 + isqrt64(1 + 2 * p)) / 2;
    const int64_t j = p + 1 - 2 * i * (i - 1);
    *z = 1.0 - (double)(i * i) / (3.0 * (double)(nside * nside));
    *phi = ((double)j - 0.5) * PI / (2.0 * (double)i);
  } else if (p < npix - ncap) {  // equatorial belt
    const int64_t pp = p - ncap;
    const int64_t i = pp / (4 * nside) + nside;
    const int64_t j = pp % (4 * nside) + 1;
    const double s = ((i + nside) % 2 == 1) ? 1.0 : 0.5;
    *z = (double)(2 * nside - i) * 2.0 / (3.0 * (double)nside);
    *phi = ((double)j - s) * PI / (2.0 * (double)nside);
  } else {  // south polar cap
    const int64_t pp = npix - p;
    const int64_t i = (1 + isqrt64(2 * pp - 1)) / 2;
    const int64_t j = 4 * i + 1 - (pp - 2 * i * (i - 1));
    *z = -1.0 + (double)(i * i) / (3.0 * (double)(nside * nside));
    *phi = ((double)j - 0.5) * PI / (2.0 * (double)i);
  }
}

// Direction triad from (l, b): n (line of sight, away from the observer), e_N (towards Galactic
// north), e_E (towards increasing l).  S:C-1 step 1.
struct Triad { double n[3], eN[3], eE[3], l, b; };
void make_triad(double l, double b, Triad& T) {
  const double cl = std::cos(l), sl = std::sin(l), cb = std::cos(b), sb = std::sin(b);
  T.l = l; T.b = b;
  T.n[0] = cb * cl;  T.n[1] = cb * sl;  T.n[2] = sb;
  T.eN[0] = -sb * cl; T.eN[1] = -sb * sl; T.eN[2] = cb;
  T.eE[0] = -sl;     T.eE[1] = cl;      T.eE[2] = 0.0;
}

// ---------------------------------------------------------------------------------------
// One sightline: forward (steps 2-10) and optionally the reverse sweep.
// ---------------------------------------------------------------------------------------
struct Sightline {
  int64_t n_los; double s_max; const double* obs; const double* freqs; int n_freq;
};

// Integration extent of the paper (Fig. 1): from the observer to where the sightline leaves the
// simulation box (centred on the Galactic centre, side lengths box[3]), cut into n_los equal segments, so each
// sightline has its own Delta r_i.  Returns the exit distance, or a negative number if the observer is not
// strictly inside the box.  When a clip box is set (oracle_set_clip_box) it REPLACES the fixed s_max.
bool g_clip = false;
double g_clip_box[3] = {0.0, 0.0, 0.0};
double exit_distance(const double* obs, const double* n, const double* box) {
  double L = std::numeric_limits<double>::infinity();
  for (int k = 0; k < 3; ++k) {
    const double half = 0.5 * box[k];
    if (!(std::fabs(obs[k]) < half)) return -1.0;
    if (n[k] > 0.0) L = std::fmin(L, (half - obs[k]) / n[k]);
    else if (n[k] < 0.0) L = std::fmin(L, (-half - obs[k]) / n[k]);
  }
  return L;
}
double path_length(const double* obs, const Triad& T, double s_max) {
  return g_clip ? exit_distance(obs, T.n, g_clip_box) : s_max;
}

void sightline_forward(const Model& m, const Sightline& S, const Triad& T,
                       double* I, double* Q, double* U /* [n_freq] */) {
  const int64_t N = S.n_los;
  const double Delta = S.s_max / (double)N;     // kpc, step 2
  const double Delta_cm = Delta * KPC_CM;
  const double KF = faraday_K_per_kpc();
  for (int f = 0; f < S.n_freq; ++f) I[f] = Q[f] = U[f] = 0.0;
  double cum = 0.0;  // sum_{m<n} n_e B_LOS
  for (int64_t n = 1; n <= N; ++n) {
    const double s = ((double)n - 0.5) * Delta;
    const double r[3] = {S.obs[0] + s * T.n[0], S.obs[1] + s * T.n[1], S.obs[2] + s * T.n[2]};
    Fields F; eval_fields(m, r, F);                                               // step 3
    const double B_LOS = F.B[0] * T.n[0] + F.B[1] * T.n[1] + F.B[2] * T.n[2];     // step 4
    // Eq.(8) numerator, verbatim:  B_z cos b - B_x cos l sin b - B_y sin l sin b
    const double B_N = F.B[2] * std::cos(T.b) - F.B[0] * std::cos(T.l) * std::sin(T.b) -
                       F.B[1] * std::sin(T.l) * std::sin(T.b);
    // Eq.(8) denominator with the sin/cos swap corrected (S:C-2#4):  B_y cos l - B_x sin l
    const double B_E = F.B[1] * std::cos(T.l) - F.B[0] * std::sin(T.l);
    const double B_trans = std::sqrt(B_N * B_N + B_E * B_E);                       // micro-gauss
    const double chi0 = std::atan2(B_N, B_E);                                     // step 7
    const double nB = F.ne * B_LOS;
    const double RM = KF * Delta * (cum + 0.5 * nB);                              // step 8
    cum += nB;
    for (int f = 0; f < S.n_freq; ++f) {
      const double nu = S.freqs[f];
      const double lambda = C_CMS / nu * 1.0e-2;                                     // metres
      const double jI = emissivity_I(nu, B_trans * 1.0e-6, F.N0, F.alpha);         // step 5
      const double jP = emissivity_P(nu, B_trans * 1.0e-6, F.N0, F.alpha);         // step 6
      const double chi = RM * lambda * lambda + chi0;                             // step 9
      const double TRJ = rayleigh_jeans(nu);
      I[f] += jI * Delta_cm * TRJ;                                                // step 10
      Q[f] += jP * std::cos(2.0 * chi) * Delta_cm * TRJ;
      U[f] += jP * std::sin(2.0 * chi) * Delta_cm * TRJ;
    }
  }
}

// Reverse sweep.  dI,dQ,dU [n_freq] are this pixel's cotangents; grad accumulated (+=).
void sightline_vjp(const Model& m, const Sightline& S, const Triad& T,
                   const double* dI, const double* dQ, const double* dU, double* grad) {
  const int64_t N = S.n_los;
  const double Delta = S.s_max / (double)N;
  const double Delta_cm = Delta * KPC_CM;
  const double KF = faraday_K_per_kpc();
  const double cl = std::cos(T.l), sl = std::sin(T.l), cb = std::cos(T.b), sb = std::sin(T.b);
  // forward sweep, storing what the reverse sweep needs
  std::vector<Fields> F(N);
  std::vector<double> BLOS(N), BN(N), BE(N), RM(N);
  std::vector<double> RMbar(N, 0.0), chi0bar(N, 0.0), Btbar(N, 0.0), N0bar(N, 0.0), alphabar(N, 0.0);
  double cum = 0.0;
  for (int64_t n = 0; n < N; ++n) {
    const double s = ((double)(n + 1) - 0.5) * Delta;
    const double r[3] = {S.obs[0] + s * T.n[0], S.obs[1] + s * T.n[1], S.obs[2] + s * T.n[2]};
    eval_fields(m, r, F[n]);
    BLOS[n] = F[n].B[0] * T.n[0] + F[n].B[1] * T.n[1] + F[n].B[2] * T.n[2];
    BN[n] = F[n].B[2] * cb - F[n].B[0] * cl * sb - F[n].B[1] * sl * sb;
    BE[n] = F[n].B[1] * cl - F[n].B[0] * sl;
    const double nB = F[n].ne * BLOS[n];
    RM[n] = KF * Delta * (cum + 0.5 * nB);
    cum += nB;
  }
  // cotangents of the per-sample quantities (steps 10, 9, 6, 5 transposed)
  for (int64_t n = 0; n < N; ++n) {
    const double Bt = std::sqrt(BN[n] * BN[n] + BE[n] * BE[n]);
    if (Bt <= 0.0) continue;
    const double chi0 = std::atan2(BN[n], BE[n]);
    for (int f = 0; f < S.n_freq; ++f) {
      const double nu = S.freqs[f];
      const double lambda = C_CMS / nu * 1.0e-2;
      const double TRJ = rayleigh_jeans(nu);
      const double jI = emissivity_I(nu, Bt * 1.0e-6, F[n].N0, F[n].alpha);
      const double jP = emissivity_P(nu, Bt * 1.0e-6, F[n].N0, F[n].alpha);
      const double chi = RM[n] * lambda * lambda + chi0;
      const double c2 = std::cos(2.0 * chi), s2 = std::sin(2.0 * chi);
      const double jIbar = dI[f] * Delta_cm * TRJ;
      const double jPbar = (dQ[f] * c2 + dU[f] * s2) * Delta_cm * TRJ;
      const double chibar = jP * (-dQ[f] * s2 + dU[f] * c2) * 2.0 * Delta_cm * TRJ;
      RMbar[n] += chibar * lambda * lambda;
      chi0bar[n] += chibar;
      // j ~ N0 * Bt^((alpha+1)/2) * (alpha-dependent factor)
      const double w = jIbar * jI + jPbar * jP;
      // j is linear in N_0 (Eq. 2, 5): N0bar = jbar * j(N_0 = 1), finite where N_0 = 0
      N0bar[n] += jIbar * emissivity_I(nu, Bt * 1.0e-6, 1.0, F[n].alpha) + jPbar * emissivity_P(nu, Bt * 1.0e-6, 1.0, F[n].alpha);
      Btbar[n] += w * 0.5 * (F[n].alpha + 1.0) / Bt;
      alphabar[n] += jIbar * jI * dln_emissivity_I_dalpha(nu, Bt * 1.0e-6, F[n].alpha) +
                     jPbar * jP * dln_emissivity_P_dalpha(nu, Bt * 1.0e-6, F[n].alpha);
    }
  }
  // transpose of step 8:  (n_e B_LOS)bar_m = K_F Delta ( sum_{n>m} RMbar_n + 1/2 RMbar_m )
  double suffix = 0.0;
  for (int64_t n = N - 1; n >= 0; --n) {
    const double nBbar = KF * Delta * (suffix + 0.5 * RMbar[n]);
    suffix += RMbar[n];
    const double nebar = nBbar * BLOS[n];
    const double BLOSbar = nBbar * F[n].ne;
    double BNbar = 0.0, BEbar = 0.0;
    const double Bt2 = BN[n] * BN[n] + BE[n] * BE[n];
    if (Bt2 > 0.0) {
      const double Bt = std::sqrt(Bt2);
      // chi0 = atan2(B_N, B_E);  B_trans = sqrt(B_N^2 + B_E^2)
      BNbar = chi0bar[n] * BE[n] / Bt2 + Btbar[n] * BN[n] / Bt;
      BEbar = -chi0bar[n] * BN[n] / Bt2 + Btbar[n] * BE[n] / Bt;
    }
    double Bb[3];
    for (int c = 0; c < 3; ++c) Bb[c] = BLOSbar * T.n[c] + BNbar * T.eN[c] + BEbar * T.eE[c];
    const double s = ((double)(n + 1) - 0.5) * Delta;
    const double r[3] = {S.obs[0] + s * T.n[0], S.obs[1] + s * T.n[1], S.obs[2] + s * T.n[2]};
    fields_vjp(m, r, Bb, N0bar[n], nebar, alphabar[n], grad);
  }
}

Model make_model(int kind, const double* params, const double* aux, const int64_t* gdim,
                 const double* gbox, const double* observer) {
  Model m; std::memset(&m, 0, sizeof(m));
  m.kind = kind; m.params = params; m.aux = aux; m.observer = observer;
  if (gdim) { m.nx = gdim[0]; m.ny = gdim[1]; m.nz = gdim[2]; }
  if (gbox) { m.lx = gbox[0]; m.ly = gbox[1]; m.lz = gbox[2]; }
  return m;
}

}  // namespace

// =========================================================================================
// The oracle's own C ABI (host pointers, float64 everywhere).  Return 0 on success.
// =========================================================================================
extern "C" {

int oracle_pix2ang_ring(int64_t nside, int64_t pix, double* z, double* phi) {
  if (nside < 1 || pix < 0 || pix >= 12 * nside * nside) return 1;
  pix2ang_ring(nside, pix, z, phi);
  return 0;
}

// out[0]=K_F per kpc, out[1]=emissivity_I(nu,Btrans[G],N0,alpha), out[2]=emissivity_P(...),
// out[3]=T_RJ(nu), out[4]=digamma(alpha) (alpha reused as the argument), out[5]=dlnjI/dalpha,
// out[6]=dlnjP/dalpha
int oracle_constants(double nu, double Btrans_gauss, double N0, double alpha, double* out) {
  out[0] = faraday_K_per_kpc();
  out[1] = emissivity_I(nu, Btrans_gauss, N0, alpha);
  out[2] = emissivity_P(nu, Btrans_gauss, N0, alpha);
  out[3] = rayleigh_jeans(nu);
  out[4] = digamma(alpha);
  out[5] = dln_emissivity_I_dalpha(nu, Btrans_gauss, alpha);
  out[6] = dln_emissivity_P_dalpha(nu, Btrans_gauss, alpha);
  return 0;
}

// Field values at n_pts points r[n][3]:  B[n][3], N0[n], ne[n], alpha[n].
int oracle_eval_fields(int kind, const double* params, const double* aux, const int64_t* gdim,
                       const double* gbox, const double* observer, int64_t n_pts, const double* r,
                       double* B, double* N0, double* ne, double* alpha) {
  const Model m = make_model(kind, params, aux, gdim, gbox, observer);
  for (int64_t k = 0; k < n_pts; ++k) {
    Fields F; eval_fields(m, r + 3 * k, F);
    B[3 * k] = F.B[0]; B[3 * k + 1] = F.B[1]; B[3 * k + 2] = F.B[2];
    N0[k] = F.N0; ne[k] = F.ne; alpha[k] = F.alpha;
  }
  return 0;
}

// One sightline in an arbitrary direction (l, b) [rad] -- used by the closed-form pins.
int oracle_forward_dir(int kind, const double* params, const double* aux, const int64_t* gdim,
                       const double* gbox, double l, double b, int64_t n_los, double s_max,
                       const double* freqs, int n_freq, const double* observer,
                       double* I, double* Q, double* U) {
  const Model m = make_model(kind, params, aux, gdim, gbox, observer);
  Triad T; make_triad(l, b, T);
  Sightline S{n_los, path_length(observer, T, s_max), observer, freqs, n_freq};
  if (!(S.s_max > 0.0)) return 1;
  sightline_forward(m, S, T, I, Q, U);
  return 0;
}

// Maps.  pix == NULL: all 12 nside^2 pixels (n_pix ignored), else the listed RING pixels.
// params: [batch][n_params] (grid: batch must be 1).  I,Q,U: [batch][n_freq][n_out].
int oracle_forward(int kind, const double* params, int64_t n_params, const double* aux,
                   const int64_t* gdim, const double* gbox, int64_t batch, int64_t nside,
                   int64_t n_los, double s_max, const double* freqs, int n_freq,
                   const double* observer, const int64_t* pix, int64_t n_pix,
                   double* I, double* Q, double* U) {
  if (nside < 1 || n_los < 1 || !(s_max > 0.0) || n_freq < 1 || n_freq > 64 || batch < 1) return 1;
  const int64_t n_out = pix ? n_pix : 12 * nside * nside;
  for (int64_t bi = 0; bi < batch; ++bi) {
    const Model m = make_model(kind, params + bi * n_params, aux, gdim, gbox, observer);
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t k = 0; k < n_out; ++k) {
      const int64_t p = pix ? pix[k] : k;
      double z, phi; pix2ang_ring(nside, p, &z, &phi);
      Triad T; make_triad(phi, 0.5 * PI - std::acos(z), T);  // l = phi, b = pi/2 - theta
      Sightline S{n_los, path_length(observer, T, s_max), observer, freqs, n_freq};
      double Iv[64], Qv[64], Uv[64];
      sightline_forward(m, S, T, Iv, Qv, Uv);
      for (int f = 0; f < n_freq; ++f) {
        const int64_t o = (bi * n_freq + f) * n_out + k;
        I[o] = Iv[f]; Q[o] = Qv[f]; U[o] = Uv[f];
      }
    }
  }
  return 0;
}

// grad[batch][n_params] (grid: [nx][ny][nz][3]) = sum over the listed pixels and frequencies of
// dI dI/dtheta + dQ dQ/dtheta + dU dU/dtheta.  dI,dQ,dU: [batch][n_freq][n_out]; NULL = zeros.
int oracle_vjp(int kind, const double* params, int64_t n_params, const double* aux,
               const int64_t* gdim, const double* gbox, int64_t batch, int64_t nside,
               int64_t n_los, double s_max, const double* freqs, int n_freq,
               const double* observer, const int64_t* pix, int64_t n_pix,
               const double* dI, const double* dQ, const double* dU, double* grad) {
  if (nside < 1 || n_los < 1 || !(s_max > 0.0) || n_freq < 1 || n_freq > 64 || batch < 1) return 1;
  const int64_t n_out = pix ? n_pix : 12 * nside * nside;
  for (int64_t bi = 0; bi < batch; ++bi) {
    const Model m = make_model(kind, params + bi * n_params, aux, gdim, gbox, observer);
    double* g_out = grad + bi * n_params;
    for (int64_t j = 0; j < n_params; ++j) g_out[j] = 0.0;
#pragma omp parallel
    {
      std::vector<double> g_loc((size_t)n_params, 0.0);
#pragma omp for schedule(dynamic, 64)
      for (int64_t k = 0; k < n_out; ++k) {
        const int64_t p = pix ? pix[k] : k;
        double z, phi; pix2ang_ring(nside, p, &z, &phi);
        Triad T; make_triad(phi, 0.5 * PI - std::acos(z), T);
        Sightline S{n_los, path_length(observer, T, s_max), observer, freqs, n_freq};
        double a[64], b[64], c[64];
        for (int f = 0; f < n_freq; ++f) {
          const int64_t o = (bi * n_freq + f) * n_out + k;
          a[f] = dI ? dI[o] : 0.0; b[f] = dQ ? dQ[o] : 0.0; c[f] = dU ? dU[o] : 0.0;
        }
        sightline_vjp(m, S, T, a, b, c, g_loc.data());
      }
#pragma omp critical
      for (int64_t j = 0; j < n_params; ++j) g_out[j] += g_loc[j];
    }
  }
  return 0;
}

// box == NULL: integrate every sightline over [0, s_max] (BASELINE.json configs); else clip at the box faces.
// Returns 1 if the observer is not strictly inside the box.
int oracle_set_clip_box(const double* box, const double* observer) {
  if (!box) { g_clip = false; return 0; }
  for (int k = 0; k < 3; ++k) {
    if (!(box[k] > 0.0) || (observer && !(std::fabs(observer[k]) < 0.5 * box[k]))) return 1;
    g_clip_box[k] = box[k];
  }
  g_clip = true;
  return 0;
}
// exit distance of one direction (for the pins)
double oracle_exit_distance(const double* observer, double l, double b, const double* box) {
  Triad T; make_triad(l, b, T);
  return exit_distance(observer, T.n, box);
}

// which: 0 = n_e, 1 = N_0.  grid == NULL removes it.  The array must stay alive while set.
int oracle_set_scalar_grid(int which, const double* grid, const int64_t* dim, const double* box) {
  ScalarGrid& S = which == 0 ? g_ne_grid : g_n0_grid;
  if (!grid) { S.g = nullptr; return 0; }
  for (int a = 0; a < 3; ++a) {
    if (dim[a] < 2 || !(box[a] > 0.0)) return 1;
    S.n[a] = dim[a]; S.len[a] = box[a];
  }
  S.g = grid;
  return 0;
}

int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void oracle_set_num_threads(int n) {
#ifdef _OPENMP
  omp_set_num_threads(n);
#else
  (void)n;
#endif
}

}  // extern "C"
