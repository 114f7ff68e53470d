// synax_api.cu -- the C ABI of libsynax (include/synax.h): plan object, argument validation, kernel
// dispatch.  Host-side only orchestration; every step of the hot path runs in the kernels of
// synax_forward.cuh / synax_vjp.cuh / synax_grid.cuh.
#include "../../include/synax.h"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

#include "synax_launch.h"
#include "synax_plan_kernels.cuh"

using namespace synax;

// ------------------------------------------------------------------------------------------------
static thread_local char g_err[512] = "";

// Forward, precision 0: sightlines whose Faraday round-off scale exceeds this many radians take the float64 chain.
// Calibrated on B200 against the oracle (profiles/r02_escalate_calibration.md): over seven workloads (cfg-4 model at
// nside 64 / 128, 256 and 1024 samples, n_e x 0.5 .. 4, B x 0.7 .. 1.5, the cfg-1 disc at 408 MHz) the largest map error
// among the sightlines left to the fp32 chain is 2.7e-5 x RMS at 300 rad (bound 1e-4: safety factor 3.7) and
// 0.85-1.8e-4 at 1000 rad (fails); the error grows about linearly with the threshold.
static constexpr double kDefaultEscalateRad = 300.0;

static synax_status fail(synax_status st, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return st;
}
#define CUDA_TRY(expr)                                                                        \
  do {                                                                                        \
    cudaError_t e_ = (expr);                                                                  \
    if (e_ != cudaSuccess)                                                                    \
      return fail(e_ == cudaErrorMemoryAllocation ? SYNAX_ERR_ALLOC : SYNAX_ERR_CUDA,         \
                  "%s failed: %s", #expr, cudaGetErrorString(e_));                            \
  } while (0)

struct synax_plan {
  int nside, n_los, n_freq, device;
  int64_t npix;       // pixels of this plan (a shard holds pixels pix0 + i * pix_stride, i < npix, of the map)
  int64_t pix0, pix_stride;
  double s_max, delta;
  double obs[3];
  double* dirs;       // device [npix][4]
  double* path;       // device [npix] path length / s_max, or null (every sightline integrates [0, s_max])
  double s_max_fixed; // s_max given at creation (restored when the box is removed)
  double freqs[kMaxFreq];
  FreqTab ft;
  int precision;      // 0 auto, 1 fp32 only, 2 float64 chain everywhere
  double escalate_rad;
  int lanes;          // 0 heuristic
  int batch_share;    // parameter vectors per thread in the batched kernels: 0 heuristic, else 1, 2 or 4
  int no_forward_totals;  // 1: the adjoint never uses the Faraday totals of the last forward (always its own pre-pass)
  int* d_vjp_ctrl;    // device control block of the adjoint's pilot (kCtrlWords ints)
  int* d_flag_count;  // device control block, kCtrlWords ints: [flag count, pilot flagged, mode, -]
  int* h_flag_count;  // pinned host mirror (last forward)
  cudaStream_t aux;   // second stream for the float64-angle member of the adjoint's per-CTA pair (fork / join by events)
  cudaEvent_t ev_fork, ev_join;
  // What the last analytic forward left for the next adjoint (which sweeps backwards and needs every sightline's Faraday
  // total first): the totals, the parameters they belong to (device copy, compared on the device) and a host-side stamp
  // of everything else they depend on.
  mutable double* phi_cache; mutable size_t phi_cap;          // [batch][npix]
  mutable double* phi_base; mutable size_t phi_base_cap;      // [ceil(n_los / 32)][batch * npix]: tile bases of the float64-chain sightlines
  mutable unsigned char* phi_has; mutable size_t phi_has_cap; // [batch * npix]
  mutable float* phi_params; mutable size_t phi_params_cap;   // [batch][n_params]
  mutable int* d_phi_ok;
  mutable struct PhiStamp { int valid, code, batch, n_params, precision; double escalate_rad, delta; const double* path; float aux[7]; } phi_stamp;
  mutable int phi_has_bases;   // the last forward also stored tile bases
  mutable Workspace ws;        // per-call scratch, kept between calls (synax_launch.h)
  mutable int64_t launches;
  mutable int64_t last_n_sl;  // sightlines of the last forward (for stats when every one took the float64 chain)
};

static double faraday_K_per_kpc() {
  const double K = SYNAX_QE * SYNAX_QE * SYNAX_QE / (2.0 * SYNAX_PI * SYNAX_ME * SYNAX_ME * SYNAX_C * SYNAX_C * SYNAX_C * SYNAX_C);
  return K * 1.0e4 * 1.0e-6 * SYNAX_KPC;  // rad m^-2 per (cm^-3 uG kpc), Eq.(7)
}

// k_f = 2 lambda_f^2 K_F delta: Faraday angle per unit sum(n_e B_LOS) for the plan's segment length (Eq.(6)-(7))
static void fill_freq_table(synax_plan* p) {
  const double KF = faraday_K_per_kpc();
  p->ft.n_freq = p->n_freq;
  for (int f = 0; f < kMaxFreq; ++f) {
    if (f < p->n_freq) {
      const double lam = SYNAX_C / p->freqs[f] * 1.0e-2;  // m
      const double k = 2.0 * lam * lam * KF * p->delta;   // rad per unit sum(n_e B_LOS)
      p->ft.k_rad[f] = (float)k; p->ft.k_turn[f] = k / (2.0 * SYNAX_PI); p->ft.freq[f] = p->freqs[f];
      p->ft.ln_nu[f] = (float)std::log(p->freqs[f]);
    } else {
      p->ft.k_rad[f] = 0.f; p->ft.k_turn[f] = 0.0; p->ft.freq[f] = 1.0; p->ft.ln_nu[f] = 0.f;
    }
  }
}

extern "C" const char* synax_last_error(void) { return g_err; }
extern "C" const char* synax_version(void) { return "synax-b200 0.1 (sm_100a)"; }

extern "C" synax_status synax_plan_create(int32_t nside, int32_t n_los, double s_max_kpc, const double* freqs_hz,
                                          int32_t n_freq, const double observer_kpc[3], synax_plan** out) {
  if (nside < 1 || nside > 8192) {
    if (out) *out = nullptr;
    return fail(SYNAX_ERR_INVALID_ARG, "nside %d not in 1..8192", nside);
  }
  return synax_plan_create_shard(nside, n_los, s_max_kpc, freqs_hz, n_freq, observer_kpc, 0, 12LL * nside * nside, out);
}

extern "C" synax_status synax_plan_create_shard(int32_t nside, int32_t n_los, double s_max_kpc, const double* freqs_hz,
                                                int32_t n_freq, const double observer_kpc[3], int64_t pix_begin,
                                                int64_t pix_count, synax_plan** out) {
  return synax_plan_create_strided(nside, n_los, s_max_kpc, freqs_hz, n_freq, observer_kpc, pix_begin, 1, pix_count, out);
}

extern "C" synax_status synax_plan_create_strided(int32_t nside, int32_t n_los, double s_max_kpc, const double* freqs_hz,
                                                  int32_t n_freq, const double observer_kpc[3], int64_t pix_begin,
                                                  int64_t pix_stride, int64_t pix_count, synax_plan** out) {
  if (!out) return fail(SYNAX_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  if (nside < 1 || nside > 8192) return fail(SYNAX_ERR_INVALID_ARG, "nside %d not in 1..8192", nside);
  if (pix_begin < 0 || pix_count < 1 || pix_stride < 1 || pix_begin + (pix_count - 1) * pix_stride >= 12LL * nside * nside)
    return fail(SYNAX_ERR_INVALID_ARG, "pixels %lld + i * %lld, i < %lld, not inside the nside=%d map", (long long)pix_begin,
                (long long)pix_stride, (long long)pix_count, nside);
  if (n_los < 1 || n_los > 65536) return fail(SYNAX_ERR_INVALID_ARG, "n_los %d not in 1..65536", n_los);
  if (!(s_max_kpc > 0.0) || !std::isfinite(s_max_kpc)) return fail(SYNAX_ERR_INVALID_ARG, "s_max must be > 0");
  if (!freqs_hz || n_freq < 1 || n_freq > kMaxFreq) return fail(SYNAX_ERR_INVALID_ARG, "n_freq %d not in 1..32 or freqs NULL", n_freq);
  if (!observer_kpc) return fail(SYNAX_ERR_INVALID_ARG, "observer is NULL");
  for (int i = 0; i < 3; ++i)
    if (!std::isfinite(observer_kpc[i])) return fail(SYNAX_ERR_INVALID_ARG, "observer not finite");
  for (int f = 0; f < n_freq; ++f)
    if (!(freqs_hz[f] > 0.0) || !std::isfinite(freqs_hz[f])) return fail(SYNAX_ERR_INVALID_ARG, "freqs[%d] must be > 0", f);

  synax_plan* p = new (std::nothrow) synax_plan();
  if (!p) return fail(SYNAX_ERR_ALLOC, "host allocation failed");
  std::memset(p, 0, sizeof(*p));
  p->nside = nside; p->n_los = n_los; p->n_freq = n_freq;
  p->npix = pix_count; p->pix0 = pix_begin; p->pix_stride = pix_stride;
  p->s_max = s_max_kpc; p->delta = s_max_kpc / (double)n_los; p->s_max_fixed = s_max_kpc; p->path = nullptr;
  for (int f = 0; f < n_freq; ++f) p->freqs[f] = freqs_hz[f];
  for (int i = 0; i < 3; ++i) p->obs[i] = observer_kpc[i];
  p->precision = 0; p->escalate_rad = kDefaultEscalateRad; p->lanes = 0;
  fill_freq_table(p);
  cudaError_t e = cudaGetDevice(&p->device);
  if (e == cudaSuccess) e = cudaMalloc((void**)&p->dirs, (size_t)p->npix * 4 * sizeof(double));
  if (e == cudaSuccess) e = cudaMalloc((void**)&p->d_flag_count, kCtrlWords * sizeof(int));
  if (e == cudaSuccess) e = cudaMalloc((void**)&p->d_vjp_ctrl, kCtrlWords * sizeof(int));
  if (e == cudaSuccess) e = cudaMallocHost((void**)&p->h_flag_count, kCtrlWords * sizeof(int));
  if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&p->aux, cudaStreamNonBlocking);
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming);
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_join, cudaEventDisableTiming);
  if (e == cudaSuccess) {
    for (int i = 0; i < kCtrlWords; ++i) p->h_flag_count[i] = 0;
    e = cudaMemset(p->d_flag_count, 0, kCtrlWords * sizeof(int));
  }
  if (e == cudaSuccess) {
    const int64_t blocks = (p->npix + 255) / 256;
    pix2ang_kernel<<<(unsigned)blocks, 256>>>((int64_t)nside, p->pix0, p->pix_stride, p->npix, p->dirs);
    p->launches++;
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
  }
  if (e != cudaSuccess) {
    synax_status st = fail(e == cudaErrorMemoryAllocation ? SYNAX_ERR_ALLOC : SYNAX_ERR_CUDA, "plan_create: %s", cudaGetErrorString(e));
    if (p->dirs) cudaFree(p->dirs);
    if (p->d_flag_count) cudaFree(p->d_flag_count);
    if (p->d_vjp_ctrl) cudaFree(p->d_vjp_ctrl);
    if (p->h_flag_count) cudaFreeHost(p->h_flag_count);
    if (p->aux) cudaStreamDestroy(p->aux);
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    if (p->ev_join) cudaEventDestroy(p->ev_join);
    delete p;
    return st;
  }
  *out = p;
  return SYNAX_OK;
}

extern "C" synax_status synax_plan_destroy(synax_plan* plan) {
  if (!plan) return SYNAX_OK;
  cudaFree(plan->dirs);
  if (plan->path) cudaFree(plan->path);
  if (plan->phi_cache) cudaFree(plan->phi_cache);
  if (plan->phi_base) cudaFree(plan->phi_base);
  if (plan->phi_has) cudaFree(plan->phi_has);
  if (plan->phi_params) cudaFree(plan->phi_params);
  if (plan->d_phi_ok) cudaFree(plan->d_phi_ok);
  if (plan->ws.base) cudaFree(plan->ws.base);
  cudaFree(plan->d_flag_count);
  cudaFree(plan->d_vjp_ctrl);
  cudaFreeHost(plan->h_flag_count);
  cudaStreamDestroy(plan->aux);
  cudaEventDestroy(plan->ev_fork);
  cudaEventDestroy(plan->ev_join);
  delete plan;
  return SYNAX_OK;
}

extern "C" int64_t synax_plan_npix(const synax_plan* plan) { return plan ? plan->npix : -1; }

extern "C" synax_status synax_plan_set_box(synax_plan* plan, const double box_kpc[3]) {
  if (!plan) return fail(SYNAX_ERR_INVALID_ARG, "plan is NULL");
  // in-flight calls on the caller's (non-blocking) streams may still read plan->path and the frequency table
  CUDA_TRY(cudaDeviceSynchronize());
  plan->phi_stamp.valid = 0;
  if (!box_kpc) {   // back to the fixed [0, s_max]
    if (plan->path) { cudaFree(plan->path); plan->path = nullptr; }
    plan->s_max = plan->s_max_fixed; plan->delta = plan->s_max / (double)plan->n_los;
    fill_freq_table(plan);
    return SYNAX_OK;
  }
  double far2 = 0.0;
  for (int k = 0; k < 3; ++k) {
    if (!(box_kpc[k] > 0.0) || !std::isfinite(box_kpc[k])) return fail(SYNAX_ERR_INVALID_ARG, "box lengths must be > 0");
    if (!(std::fabs(plan->obs[k]) < 0.5 * box_kpc[k])) return fail(SYNAX_ERR_INVALID_ARG, "the observer must be strictly inside the box");
    const double d = 0.5 * box_kpc[k] + std::fabs(plan->obs[k]);
    far2 += d * d;
  }
  if (!plan->path) CUDA_TRY(cudaMalloc((void**)&plan->path, (size_t)plan->npix * sizeof(double)));
  // reference length = distance to the farthest corner, so that every path[i] <= 1 (tile-length bounds stay valid)
  plan->s_max = std::sqrt(far2); plan->delta = plan->s_max / (double)plan->n_los;
  fill_freq_table(plan);
  box_path_kernel<<<(unsigned)((plan->npix + 255) / 256), 256>>>(plan->dirs, plan->npix, plan->obs[0], plan->obs[1], plan->obs[2],
                                                               0.5 * box_kpc[0], 0.5 * box_kpc[1], 0.5 * box_kpc[2],
                                                               1.0 / plan->s_max, plan->path);
  plan->launches++;
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaDeviceSynchronize());
  return SYNAX_OK;
}

extern "C" synax_status synax_plan_set_option(synax_plan* plan, const char* key, double value) {
  if (!plan || !key) return fail(SYNAX_ERR_INVALID_ARG, "plan or key is NULL");
  if (!std::strcmp(key, "precision")) {
    if (value != 0 && value != 1 && value != 2) return fail(SYNAX_ERR_INVALID_ARG, "precision must be 0, 1 or 2");
    plan->precision = (int)value;
  } else if (!std::strcmp(key, "escalate_rad")) {
    if (!(value > 0)) return fail(SYNAX_ERR_INVALID_ARG, "escalate_rad must be > 0");
    plan->escalate_rad = value;
  } else if (!std::strcmp(key, "lanes")) {
    if (value != 0 && value != 1 && value != 8 && value != 32) return fail(SYNAX_ERR_INVALID_ARG, "lanes must be 0, 1, 8 or 32");
    plan->lanes = (int)value;
  } else if (!std::strcmp(key, "use_forward_totals")) {
    if (value != 0 && value != 1) return fail(SYNAX_ERR_INVALID_ARG, "use_forward_totals must be 0 or 1");
    plan->no_forward_totals = value == 0 ? 1 : 0;
    plan->phi_stamp.valid = 0;   // setting the option (to either value) also drops what the plan has stored
  } else if (!std::strcmp(key, "batch_share")) {
    if (value != 0 && value != 1 && value != 2 && value != 4) return fail(SYNAX_ERR_INVALID_ARG, "batch_share must be 0, 1, 2 or 4");
    plan->batch_share = (int)value;
  } else if (!std::strcmp(key, "pool_release_threshold_mb")) {
    // Per-call scratch (constants, flag lists, block partials, the host entry points' staging buffers) comes from the
    // device's stream-ordered pool.  Its default release threshold is 0: every stream synchronisation hands the memory
    // back to the driver and the next call pays for mapping it again (hundreds of MB in the *_host calls: measured
    // outliers of +10 ms per step at cfg 4).  This option raises the threshold of the DEVICE's default pool -- a
    // process-wide setting, hence opt-in; a larger value already set by the application is left alone.
    if (!(value >= 0) || value > 1.0e6) return fail(SYNAX_ERR_INVALID_ARG, "pool_release_threshold_mb must be in 0 .. 1e6");
    cudaMemPool_t pool;
    CUDA_TRY(cudaDeviceGetDefaultMemPool(&pool, plan->device));
    uint64_t thr = 0, want = (uint64_t)value << 20;
    CUDA_TRY(cudaMemPoolGetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr));
    if (thr < want) CUDA_TRY(cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &want));
  } else {
    return fail(SYNAX_ERR_INVALID_ARG, "unknown option '%s'", key);
  }
  return SYNAX_OK;
}

extern "C" synax_status synax_plan_directions(const synax_plan* plan, double* out_device, void* cuda_stream) {
  if (!plan || !out_device) return fail(SYNAX_ERR_INVALID_ARG, "plan or out is NULL");
  CUDA_TRY(cudaMemcpyAsync(out_device, plan->dirs, (size_t)plan->npix * 4 * sizeof(double), cudaMemcpyDeviceToDevice,
                           (cudaStream_t)cuda_stream));
  return SYNAX_OK;
}

extern "C" synax_status synax_plan_stats(const synax_plan* plan, int64_t out[2]) {
  if (!plan || !out) return fail(SYNAX_ERR_INVALID_ARG, "plan or out is NULL");
  out[0] = plan->launches;
  out[1] = plan->h_flag_count[kCtrlMode] == kModeAllF64 ? plan->last_n_sl
                                                             : plan->h_flag_count[kCtrlFlagCount] + plan->h_flag_count[kCtrlCountM];
  return SYNAX_OK;
}

// ------------------------------------------------------------------------------------------------
static synax_status check_model(const synax_plan* plan, const synax_model* m, const void* params, int32_t batch,
                                int* code) {
  if (!plan) return fail(SYNAX_ERR_INVALID_ARG, "plan is NULL");
  if (!m) return fail(SYNAX_ERR_INVALID_ARG, "model is NULL");
  if (!params) return fail(SYNAX_ERR_INVALID_ARG, "params is NULL");
  if (batch < 1) return fail(SYNAX_ERR_INVALID_ARG, "batch %d < 1", batch);
  switch (m->kind) {
    case SYNAX_MODEL_DISC4:
      if (m->n_params != 4) return fail(SYNAX_ERR_INVALID_ARG, "DISC4 needs n_params == 4");
      if (!m->aux) return fail(SYNAX_ERR_INVALID_ARG, "DISC4 needs aux");
      *code = kAnalyticDisc; break;
    case SYNAX_MODEL_FULL16:
      if (m->n_params != 16) return fail(SYNAX_ERR_INVALID_ARG, "FULL16 needs n_params == 16");
      *code = kAnalyticFull; break;
    case SYNAX_MODEL_STACK16:
      if (m->n_params != 16) return fail(SYNAX_ERR_INVALID_ARG, "STACK16 needs n_params == 16");
      if (!m->aux) return fail(SYNAX_ERR_INVALID_ARG, "STACK16 needs aux");
      *code = kStack16; break;
    case SYNAX_MODEL_UNIFORM:
      if (m->n_params != 6) return fail(SYNAX_ERR_INVALID_ARG, "UNIFORM needs n_params == 6");
      *code = kUniform; break;
    case SYNAX_MODEL_GRID_B: {
      if (!m->aux) return fail(SYNAX_ERR_INVALID_ARG, "GRID_B needs aux");
      if (batch != 1) return fail(SYNAX_ERR_INVALID_ARG, "GRID_B needs batch == 1");
      if (m->nx < 2 || m->ny < 2 || m->nz < 2) return fail(SYNAX_ERR_INVALID_ARG, "grid dims must be >= 2");
      if (!(m->lx > 0) || !(m->ly > 0) || !(m->lz > 0)) return fail(SYNAX_ERR_INVALID_ARG, "grid box lengths must be > 0");
      const int64_t n = (int64_t)m->nx * m->ny * m->nz * 3;
      if (n >= (1LL << 31) || m->n_params != (int32_t)n) return fail(SYNAX_ERR_INVALID_ARG, "GRID_B needs n_params == nx*ny*nz*3 < 2^31");
      *code = kGridB; break;
    }
    default: return fail(SYNAX_ERR_INVALID_ARG, "unknown model kind %d", m->kind);
  }
  if ((int64_t)batch * plan->npix >= (1LL << 31)) return fail(SYNAX_ERR_INVALID_ARG, "batch * npix must be < 2^31");
  const float* sg[2] = {m->ne_grid, m->n0_grid};
  const int32_t* sn[2] = {m->ne_n, m->n0_n};
  const double* sl[2] = {m->ne_l, m->n0_l};
  for (int k = 0; k < 2; ++k) {
    if (!sg[k]) continue;
    if (m->kind != SYNAX_MODEL_DISC4 && m->kind != SYNAX_MODEL_GRID_B && m->kind != SYNAX_MODEL_STACK16)
      return fail(SYNAX_ERR_INVALID_ARG, "gridded n_e / N_0 need a DISC4, STACK16 or GRID_B model");
    for (int a = 0; a < 3; ++a)
      if (sn[k][a] < 2 || !(sl[k][a] > 0.0)) return fail(SYNAX_ERR_INVALID_ARG, "scalar grid dims must be >= 2 and box lengths > 0");
  }
  return SYNAX_OK;
}

static ScalarGridDesc make_scalar_desc(const float* g, const int32_t n[3], const double l[3]) {
  ScalarGridDesc d;
  d.g = g; d.nx = g ? n[0] : 2; d.ny = g ? n[1] : 2; d.nz = g ? n[2] : 2;
  d.sx = g ? (double)(n[0] - 1) / l[0] : 0.0; d.sy = g ? (double)(n[1] - 1) / l[1] : 0.0;
  d.sz = g ? (double)(n[2] - 1) / l[2] : 0.0;
  d.bx = 0.5 * (double)(d.nx - 1); d.by = 0.5 * (double)(d.ny - 1); d.bz = 0.5 * (double)(d.nz - 1);
  return d;
}

// Lanes per sightline.  `want`: sightlines from which one thread each is the better choice -- measured on B200 with the cfg-4
// model at 8 frequencies (nside 32 ... 192, 256 ... 4096 samples) and cfg 1: 300,000 for a stand-alone adjoint and the
// float64 entry points (a few waves of 3-CTA-per-SM kernels), 150,000 for the forward, 24,576 for an adjoint that finds the
// Faraday totals of the plan's last forward (no pre-pass, no lane scans: 0.86 against 1.34 ms at nside 64 x 1024 samples).
#ifndef SYNAX_SPLIT_FROM
#define SYNAX_SPLIT_FROM 50000000
#endif
// escalate_rad is tuned for sightlines of >= kFullThresholdFromSamples samples, where the fp32 rounding of the single angles
// averages out over the sum; a sightline of a few samples has nothing to average (parity 1.0 .. 4.2e-4 x RMS at 1 .. 65
// samples with the full threshold), so the threshold shrinks in proportion below that count.
constexpr int kFullThresholdFromSamples = 128;
static double escalate_at(const synax_plan* plan) {
  return plan->escalate_rad * std::min(1.0, (double)plan->n_los / (double)kFullThresholdFromSamples);
}
constexpr double kTileAngleRad = 96.0;   // fp32 chain: largest rotation angle inside a tile before the sightline is redone in float64
constexpr int64_t kSplitFromSamples = SYNAX_SPLIT_FROM;   // forward: LoS samples from which the split mode is worth its extra launches
constexpr int64_t kOneLaneFrom = 300000, kOneLaneFromForward = 150000, kOneLaneFromStored = 24576;
static int pick_lanes(const synax_plan* plan, int64_t n_sl, int64_t want = kOneLaneFrom) {
  if (plan->lanes) return plan->lanes;
  if (n_sl >= want) return 1;
  if (n_sl * 8 >= want) return 8;
  return 32;
}

static int next_freq_block(int remaining) {
  if (remaining >= 8) return 8;
  if (remaining >= 4) return 4;
  return remaining;  // 1, 2, 3
}

namespace synax {
void launch_decide(int* ctrl, int64_t n_pilot, int num, int den, int mode_yes, cudaStream_t st) {
  decide_kernel<<<1, 1, 0, st>>>(ctrl, n_pilot, num, den, mode_yes);
}
}  // namespace synax

static AuxHost make_aux(const synax_model* m) {
  AuxHost a;
  for (int i = 0; i < 7; ++i) a.v[i] = m->aux ? m->aux[i] : 0.0f;
  return a;
}

static Geometry make_geo(const synax_plan* plan) {
  Geometry g;
  g.npix = plan->npix; g.n_los = plan->n_los; g.delta = plan->delta;
  for (int i = 0; i < 3; ++i) { g.obs[i] = plan->obs[i]; g.obsf[i] = (float)plan->obs[i]; }
  g.dirs = plan->dirs; g.path = plan->path;
  return g;
}

static int sm_count(int device) {
  static int cached[64];
  if (device < 0 || device >= 64) return 148;
  if (!cached[device]) {
    int n = 0;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, device) != cudaSuccess || n <= 0) n = 148;
    cached[device] = n;
  }
  return cached[device];
}

// Plan-owned workspace (synax_launch.h).
namespace synax {
void* ws_alloc(Workspace* ws, size_t bytes, cudaStream_t st, bool* pooled) {
  *pooled = false;
  bytes = (bytes + 255) & ~(size_t)255;
  if (bytes == 0) bytes = 256;
  if (ws) {
    const size_t at = ws->used;
    ws->used += bytes;
    if (ws->used > ws->want) ws->want = ws->used;
    if (ws->base && at + bytes <= ws->cap) {
      cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
      if (cudaStreamIsCapturing(st, &cap) != cudaSuccess) cudaGetLastError();
      else if (cap == cudaStreamCaptureStatusNone) return ws->base + at;
    }
  }
  void* q = nullptr;
  if (cudaMallocAsync(&q, bytes, st) != cudaSuccess) return nullptr;
  *pooled = true;
  return q;
}
void ws_enter(Workspace* ws, cudaStream_t st, size_t* mark) {
  *mark = 0;
  if (!ws) return;
  if (ws->depth++ == 0) {
    ws->used = 0;
    const size_t want = std::min(ws->want, kWorkspaceMax);
    if (want > ws->cap) {
      cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
      if (cudaStreamIsCapturing(st, &cap) != cudaSuccess) cudaGetLastError();
      else if (cap == cudaStreamCaptureStatusNone) {
        if (ws->base) cudaFree(ws->base);   // (synchronises the device: earlier calls may still be using it)
        ws->base = nullptr; ws->cap = 0;
        const size_t grow = std::min(kWorkspaceMax, want + want / 4);
        if (cudaMalloc((void**)&ws->base, grow) == cudaSuccess) ws->cap = grow;
        else cudaGetLastError();
      }
    }
  }
  *mark = ws->used;
}
}  // namespace synax

// Per-call scratch in stack order from the plan's workspace (else from the device's stream-ordered pool); everything handed
// out is given back when the guard leaves scope, whatever path the call returns on.
struct StreamScratch {
  cudaStream_t st;
  Workspace* ws;
  size_t mark = 0;
  void* blocks[12];
  int n = 0;
  StreamScratch(const synax_plan* plan, cudaStream_t s);
  StreamScratch(const StreamScratch&) = delete;
  StreamScratch& operator=(const StreamScratch&) = delete;
  ~StreamScratch() {
    for (int i = n - 1; i >= 0; --i) cudaFreeAsync(blocks[i], st);
    ws_leave(ws, mark);
  }
  template <typename T>
  cudaError_t get(T** out, size_t bytes) {
    bool pooled = false;
    if (n >= 12) { *out = nullptr; return cudaErrorMemoryAllocation; }
    void* q = ws_alloc(ws, bytes, st, &pooled);
    if (q && pooled) blocks[n++] = q;
    *out = (T*)q;
    return q ? cudaSuccess : cudaErrorMemoryAllocation;
  }
};
StreamScratch::StreamScratch(const synax_plan* plan, cudaStream_t s) : st(s), ws(&plan->ws) { ws_enter(ws, st, &mark); }

// Per-batch constants of a call (prologue_kernel).  When a gridded n_e replaces the analytic disc, the bound on
// |n_e B_LOS| that sizes the float64 chain's tiles (BatchConsts::tile_d) comes from max |ne_grid|, reduced on the device
// first -- the aux n_e entries are ignored then and say nothing about the grid (synax.h).
static synax_status run_prologue(const synax_plan* plan, const synax_model* model, int code, const float* params, int batch,
                                 StreamScratch& scratch, BatchConsts** bc, BatchConstsD** bd, cudaStream_t st) {
  CUDA_TRY(scratch.get(bc, sizeof(BatchConsts) * (size_t)batch));
  CUDA_TRY(scratch.get(bd, sizeof(BatchConstsD) * (size_t)batch));
  float* ne_max = nullptr;
  if (model->ne_grid) {
    const int64_t n = (int64_t)model->ne_n[0] * model->ne_n[1] * model->ne_n[2];
    CUDA_TRY(scratch.get(&ne_max, sizeof(float)));
    CUDA_TRY(cudaMemsetAsync(ne_max, 0, sizeof(float), st));
    absmax_kernel<<<(unsigned)std::min<int64_t>((n + 1023) / 1024, 1184), 256, 0, st>>>(model->ne_grid, n, ne_max);
    plan->launches++;
  }
  prologue_kernel<<<(batch + 127) / 128, 128, 0, st>>>(code, code == kGridB ? nullptr : params, model->n_params, batch,
                                                      make_aux(model), plan->ft, plan->delta, plan->n_los, ne_max, *bc, *bd);
  plan->launches++;
  CUDA_TRY(cudaGetLastError());
  return SYNAX_OK;
}

static synax_plan::PhiStamp make_phi_stamp(const synax_plan* plan, const synax_model* model, int code, int batch) {
  synax_plan::PhiStamp st;
  std::memset(&st, 0, sizeof(st));
  st.valid = 1; st.code = code; st.batch = batch; st.n_params = model->n_params; st.precision = plan->precision;
  st.escalate_rad = plan->escalate_rad; st.delta = plan->delta; st.path = plan->path;
  for (int i = 0; i < 7; ++i) st.aux[i] = model->aux ? model->aux[i] : 0.f;
  return st;
}

// Buffers for the Faraday totals of an analytic forward of `batch` parameter vectors (grown on demand: the first call
// of a given size allocates, and so synchronises, once).  Gridded n_e is left out: the grid's contents can change
// between the forward and the adjoint without the library seeing it.
static bool phi_buffers(const synax_plan* plan, const synax_model* model, int batch, cudaStream_t st) {
  if (model->ne_grid) return false;
  const size_t need = (size_t)plan->npix * (size_t)batch, needp = (size_t)batch * (size_t)model->n_params;
  // growing a buffer is a cudaMalloc: not inside a stream capture (a captured forward keeps whatever earlier calls allocated)
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(st, &cap) != cudaSuccess) { cudaGetLastError(); return false; }
  if (cap != cudaStreamCaptureStatusNone)
    return plan->phi_cap >= need && plan->phi_params_cap >= needp && plan->d_phi_ok != nullptr;
  if (plan->phi_cap < need) {
    if (plan->phi_cache) cudaFree(plan->phi_cache);
    plan->phi_cache = nullptr; plan->phi_cap = 0;
    if (cudaMalloc((void**)&plan->phi_cache, need * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return false; }
    plan->phi_cap = need;
  }
  if (plan->phi_params_cap < needp) {
    if (plan->phi_params) cudaFree(plan->phi_params);
    plan->phi_params = nullptr; plan->phi_params_cap = 0;
    if (cudaMalloc((void**)&plan->phi_params, needp * sizeof(float)) != cudaSuccess) { cudaGetLastError(); return false; }
    plan->phi_params_cap = needp;
  }
  if (!plan->d_phi_ok && cudaMalloc((void**)&plan->d_phi_ok, sizeof(int)) != cudaSuccess) { cudaGetLastError(); return false; }
  // Tile bases (the Faraday depth before every 32nd sample of the sightlines the float64 chain integrates): 8 bytes per 32
  // samples -- 201 MB at cfg 4.  Optional: when the memory is not there the adjoint keeps its own float64-angle variants.
  const size_t tiles = (size_t)(plan->n_los + 31) / 32;
  if (plan->precision != 1 && tiles > 1) {
    if (plan->phi_base_cap < need * tiles) {
      if (plan->phi_base) cudaFree(plan->phi_base);
      plan->phi_base = nullptr; plan->phi_base_cap = 0;
      if (cudaMalloc((void**)&plan->phi_base, need * tiles * sizeof(double)) == cudaSuccess) plan->phi_base_cap = need * tiles;
      else cudaGetLastError();
    }
    if (plan->phi_has_cap < need) {
      if (plan->phi_has) cudaFree(plan->phi_has);
      plan->phi_has = nullptr; plan->phi_has_cap = 0;
      if (cudaMalloc((void**)&plan->phi_has, need) == cudaSuccess) plan->phi_has_cap = need;
      else cudaGetLastError();
    }
  }
  return true;
}

// The forward.  faraday_only: the pass the adjoint runs when the plan holds no Faraday totals for these parameters -- the
// same strategy (pilot, the two chains, lists) with kernels that integrate the Faraday depth alone (NF = 0 instantiations: no
// emission, no rotation, no maps) and leave every sightline's total, the tile bases of the float64-chain sightlines and the
// stamp behind, exactly as a forward would; *stored says whether they are there afterwards.
static synax_status forward_core(const synax_plan* plan, const synax_model* model, int code, const float* params,
                                 int32_t batch, float* I, float* Q, float* U, cudaStream_t st, bool faraday_only, bool* stored) {
  synax_status stt = SYNAX_OK;
  if (stored) *stored = false;
  const int64_t n_sl = plan->npix * batch;
  if (faraday_only && !(code != kGridB && pick_lanes(plan, n_sl, kOneLaneFromStored) == 1 && phi_buffers(plan, model, batch, st)))
    return SYNAX_OK;   // nowhere to put them (small call, lanes forced, gridded n_e, capture without buffers)
  StreamScratch scratch(plan, st);

  BatchConsts* bc = nullptr;
  BatchConstsD* bd = nullptr;
  stt = run_prologue(plan, model, code, params, batch, scratch, &bc, &bd, st);
  if (stt != SYNAX_OK) return stt;

  ForwardArgs a;
  a.geo = make_geo(plan); a.bc = bc; a.bd = bd; a.batch = batch; a.I = I; a.Q = Q; a.U = U;
  a.n_freq_total = plan->n_freq;
  a.sg_ne = make_scalar_desc(model->ne_grid, model->ne_n, model->ne_l);
  a.sg_n0 = make_scalar_desc(model->n0_grid, model->n0_n, model->n0_l);
  a.flag_count = plan->d_flag_count; a.flag_list = nullptr; a.flag_S = 0.0f; a.flag_T = 0.0f;
  a.append_count = plan->d_flag_count + kCtrlFlagCount; a.append_list = nullptr;
  a.phi = nullptr; a.phi_base = nullptr; a.phi_has = nullptr;
  plan->phi_stamp.valid = 0;

  if (code == kGridB) {
    synax_status gs = grid_forward(plan->ft, a, model, params, plan->precision, escalate_at(plan), sm_count(plan->device),
                                   plan->d_flag_count, plan->h_flag_count, &plan->ws, st, &plan->launches);
    if (gs != SYNAX_OK) return fail(gs, "grid forward failed: %s", cudaGetErrorString(cudaGetLastError()));
    return SYNAX_OK;
  }

  float k_max = 0.f;
  for (int f = 0; f < plan->n_freq; ++f) k_max = fmaxf(k_max, plan->ft.k_rad[f]);
  const bool fast = plan->precision != 2;
  const bool escalate = plan->precision == 0;
  int* ctrl = plan->d_flag_count;
  plan->last_n_sl = n_sl;
  CUDA_TRY(cudaMemsetAsync(ctrl, 0, kCtrlWords * sizeof(int), st));   // mode = fp32 pass then flagged list
  a.mode = nullptr; a.run_when = 0; a.list_u = nullptr; a.count_u = nullptr;
  const int sms = sm_count(plan->device);
  // precision 0: a pilot over ~8k sightlines decides ON THE DEVICE between "fp32 pass + float64 redo of the flagged
  // sightlines" (hardly any flagged), "float64 Faraday chain for every sightline" (nearly all flagged) and "split":
  // classify_kernel sorts the sightlines into one list per chain (decide_forward_kernel).
  bool piloted = false, split_ok = false;
  int* miss_list = nullptr;
  if (escalate) {
    CUDA_TRY(scratch.get(&a.flag_list, sizeof(int) * (size_t)n_sl));
    a.append_list = a.flag_list;
    a.flag_S = (float)(escalate_at(plan) / (double)k_max);
    // ... and when the rotation angle inside one 32-sample tile of the fp32 chain passes kTileAngleRad: that angle is formed
    // and range-reduced in fp32 (error ~2e-7 x angle).  Well-resolved sightlines below the first criterion stay far below
    // it (<~ 20 rad); a run with a few dozen samples per sightline at low frequency does not (parity 1.1e-4 x RMS at 43 samples).
    a.flag_T = (float)(kTileAngleRad / (double)k_max);
    if (n_sl > 16384) {
      const int64_t stride = (n_sl / 8192) | 1;
      const int64_t n_pilot = (n_sl + stride - 1) / stride;
      const unsigned pb = (unsigned)((n_pilot * 32 + kBlock - 1) / kBlock);
      SYNAX_DISPATCH_CODE(code, fwd_launch_pilot, pb, st, a, stride, n_pilot, ctrl);
      // the split mode costs a handful of extra launches: only for calls long enough not to notice (cfg 1: 0.19 ms in all)
      split_ok = n_sl >= 262144 || (n_sl >= 32768 && n_sl * (int64_t)plan->n_los >= kSplitFromSamples);
      if (split_ok) {
        decide_forward_kernel<<<1, 1, 0, st>>>(ctrl, n_pilot);
        CUDA_TRY(scratch.get(&a.list_u, sizeof(int) * (size_t)n_sl));
        CUDA_TRY(scratch.get(&miss_list, sizeof(int) * (size_t)n_sl));
        a.count_u = ctrl + kCtrlCountU;
        const unsigned cb = (unsigned)std::min<int64_t>((n_sl + kBlock - 1) / kBlock, (int64_t)sms * 16);
        SYNAX_DISPATCH_CODE(code, fwd_launch_classify, cb, st, a, ctrl);
        plan->launches += 3;
      } else {
        launch_decide(ctrl, n_pilot, 1, 4, kModeAllF64, st);   // more than a quarter flagged: all-float64
        plan->launches += 2;
      }
      a.mode = ctrl + kCtrlMode;
      piloted = true;
    }
  }
  const int G = pick_lanes(plan, n_sl, kOneLaneFromForward);
  // the adjoint will want the Faraday totals (it has a pre-pass of its own otherwise); whatever the lane count here, it can
  // then run with one thread per sightline
  const bool keep_phi = pick_lanes(plan, n_sl, kOneLaneFromStored) == 1 && phi_buffers(plan, model, batch, st);
  if (keep_phi) a.phi = plan->phi_cache;
  const bool keep_base = keep_phi && plan->precision != 1 && plan->phi_base && plan->phi_has &&
                         plan->phi_base_cap >= (size_t)n_sl * ((size_t)(plan->n_los + 31) / 32) && plan->phi_has_cap >= (size_t)n_sl;
  if (keep_base) { a.phi_base = plan->phi_base; a.phi_has = plan->phi_has; }
  // Every sightline (count known on the host): one group per sightline and the hardware block scheduler balances the
  // CTAs (a persistent grid of 16 CTAs/SM left a 14 % tail at cfg 4: 2.6 sightlines per thread).  Flag list (length
  // known only on the device): persistent grid, groups stride over the list.
  // Split mode: the list is long (2-85 % of the sightlines), so it takes the lane count of the full pass and a grid
  // sized for all sightlines (CTAs past the list's end exit at once).
  const int n_freq_run = faraday_only ? 1 : plan->n_freq;   // Faraday-only: one pass over "zero frequencies"
  auto blocks_for = [&](int lanes, bool use_list, int run_when) {
    const int64_t full = (n_sl * lanes + kBlockD - 1) / kBlockD;
    return (unsigned)(use_list && run_when != 3 ? std::min<int64_t>(full, (int64_t)sms * 16 * 128 / kBlockD) : full);
  };
  auto run_f64 = [&](cudaStream_t on, int lanes, int run_when, int* list, int* count) {
    ForwardArgs pa = a;
    pa.run_when = run_when;
    pa.flag_list = list; pa.flag_count = count;
    for (int f0 = 0; f0 < n_freq_run;) {
      const int nf = faraday_only ? 0 : next_freq_block(plan->n_freq - f0);
      pa.f0 = f0;
      SYNAX_DISPATCH_CODE(code, fwd_launch_f64, lanes, nf, blocks_for(lanes, list != nullptr, run_when), on, pa, plan->ft);
      plan->launches++;
      f0 += faraday_only ? 1 : nf;
    }
  };
  cudaError_t stream_err = cudaSuccess;
  if (fast) {
    if (split_ok) {
      // all-float64 / split: the float64-chain kernel (every sightline, or classify_kernel's flag list) runs on the plan's
      // second stream beside the fp32 kernel over list_u; what the fp32 kernel's exact criterion still flags goes to a
      // separate list (the flag list is being read) and is redone after the join.  Fork after classify_kernel.
      stream_err = cudaEventRecord(plan->ev_fork, st);
      if (stream_err == cudaSuccess) stream_err = cudaStreamWaitEvent(plan->aux, plan->ev_fork, 0);
      if (stream_err != cudaSuccess) return fail(SYNAX_ERR_CUDA, "forward: stream fork failed: %s", cudaGetErrorString(stream_err));
      run_f64(plan->aux, G, 3, a.flag_list, ctrl + kCtrlFlagCount);
    }
    for (int f0 = 0; f0 < n_freq_run;) {
      const int nf = faraday_only ? 0 : next_freq_block(plan->n_freq - f0);
      a.f0 = f0;
      // batches of parameter vectors on modest maps: NB vectors per thread share the sightline geometry (A12)
      const int nb = plan->batch_share ? plan->batch_share : (batch >= 4 ? 4 : (batch >= 2 ? 2 : 1));
      if (nb > 1 && G == 1 && nf == 1 && plan->n_freq == 1 && (code == kAnalyticDisc || code == kAnalyticFull) &&
          !model->ne_grid && !model->n0_grid)
        SYNAX_DISPATCH_CODE(code, fwd_launch_batched, nb, st, a, plan->ft);
      else
        SYNAX_DISPATCH_CODE(code, fwd_launch_fast, false, G, nf, n_sl, st, a, plan->ft);
      plan->launches++;
      if (split_ok) {   // the same pass over list_u (exits at once unless the pilot chose the split mode)
        ForwardArgs al = a;
        al.append_count = ctrl + kCtrlCountM; al.append_list = miss_list;
        SYNAX_DISPATCH_CODE(code, fwd_launch_fast, true, G, nf, n_sl, st, al, plan->ft);
        plan->launches++;
      }
      f0 += faraday_only ? 1 : nf;
    }
    if (escalate) run_f64(st, 8, piloted ? 1 : 0, a.flag_list, ctrl + kCtrlFlagCount);   // fast-then-list: the flagged list, 8 lanes per sightline
    if (split_ok) {
      stream_err = cudaEventRecord(plan->ev_join, plan->aux);
      if (stream_err == cudaSuccess) stream_err = cudaStreamWaitEvent(st, plan->ev_join, 0);
      if (stream_err != cudaSuccess) {
        cudaStreamSynchronize(plan->aux);   // join by hand so that the scratch is not freed under the second stream
        return fail(SYNAX_ERR_CUDA, "forward: stream join failed: %s", cudaGetErrorString(stream_err));
      }
      run_f64(st, 8, 4, miss_list, ctrl + kCtrlCountM);
    } else if (piloted) {
      run_f64(st, G, 2, nullptr, ctrl + kCtrlFlagCount);   // short calls: every sightline when the pilot says all-float64
    }
  } else {
    run_f64(st, G, 0, nullptr, ctrl + kCtrlFlagCount);
  }
  cudaError_t e = cudaGetLastError();
  cudaMemcpyAsync(plan->h_flag_count, ctrl, kCtrlWords * sizeof(int), cudaMemcpyDeviceToHost, st);
  if (e != cudaSuccess) return fail(SYNAX_ERR_CUDA, "forward launch failed: %s", cudaGetErrorString(e));
  if (keep_phi && cudaMemcpyAsync(plan->phi_params, params, sizeof(float) * (size_t)batch * model->n_params,
                                  cudaMemcpyDeviceToDevice, st) == cudaSuccess)
  {
    const synax_plan::PhiStamp now = make_phi_stamp(plan, model, code, batch);
    std::memcpy(&plan->phi_stamp, &now, sizeof(now));   // byte copy: the stamp is compared with memcmp
    plan->phi_has_bases = keep_base ? 1 : 0;
    if (stored) *stored = true;
  }
  return SYNAX_OK;
}

extern "C" synax_status synax_forward(const synax_plan* plan, const synax_model* model, const float* params,
                                      int32_t batch, float* I, float* Q, float* U, void* cuda_stream) {
  int code = 0;
  synax_status stt = check_model(plan, model, params, batch, &code);
  if (stt != SYNAX_OK) return stt;
  if (!I || !Q || !U) return fail(SYNAX_ERR_INVALID_ARG, "I, Q or U is NULL");
  return forward_core(plan, model, code, params, batch, I, Q, U, (cudaStream_t)cuda_stream, false, nullptr);
}

extern "C" synax_status synax_vjp(const synax_plan* plan, const synax_model* model, const float* params,
                                  int32_t batch, const float* dI, const float* dQ, const float* dU, float* grad,
                                  void* cuda_stream) {
  int code = 0;
  synax_status stt = check_model(plan, model, params, batch, &code);
  if (stt != SYNAX_OK) return stt;
  if (!grad) return fail(SYNAX_ERR_INVALID_ARG, "grad is NULL");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  StreamScratch scratch(plan, st);
  BatchConsts* bc = nullptr;
  BatchConstsD* bd = nullptr;
  stt = run_prologue(plan, model, code, params, batch, scratch, &bc, &bd, st);
  if (stt != SYNAX_OK) return stt;
  // Faraday totals of the last forward: usable when everything but the parameter values matches on the host side; the
  // values themselves are compared on the device (no synchronisation)
  const double* phi = nullptr;
  const double* phi_base = nullptr;
  const unsigned char* phi_has = nullptr;
  int G = pick_lanes(plan, plan->npix * batch);
  if (code != kGridB && !plan->no_forward_totals && !model->ne_grid &&
      pick_lanes(plan, plan->npix * batch, kOneLaneFromStored) == 1) {
    synax_plan::PhiStamp now = make_phi_stamp(plan, model, code, batch);
    bool have = plan->phi_stamp.valid && std::memcmp(&now, &plan->phi_stamp, sizeof(now)) == 0;
    // Nothing stored for this plan and these settings (a stand-alone adjoint): a Faraday-only pass with the forward's own
    // strategy leaves the totals and tile bases behind first, and the lean one-thread kernel then does every sightline --
    // instead of a pre-pass inside the adjoint kernel plus its float64-angle variants (cfg 4: 20.9 -> see DESIGN.md section 5).
    // Not where the forward-order kernel runs anyway (one frequency, DISC4 / FULL16, one thread per sightline: no totals needed).
    const bool forward_order = G == 1 && plan->n_freq == 1 && (code == kAnalyticDisc || code == kAnalyticFull) &&
                               !model->n0_grid && batch <= 65535;
    // ... nor for calls so short that the pass's dozen launches show (cfg 1: 0.28 against 0.24 ms)
    const bool long_call = plan->npix * batch * (int64_t)plan->n_los >= kSplitFromSamples;
    if (!have && !forward_order && long_call) {
      bool stored = false;
      stt = forward_core(plan, model, code, params, batch, nullptr, nullptr, nullptr, st, true, &stored);
      if (stt != SYNAX_OK) return stt;
      if (stored) {
        now = make_phi_stamp(plan, model, code, batch);
        have = plan->phi_stamp.valid && std::memcmp(&now, &plan->phi_stamp, sizeof(now)) == 0;
      }
    }
    if (have) {
      G = 1;
      phi_validate_kernel<<<1, 256, 0, st>>>(params, plan->phi_params, (int64_t)batch * model->n_params, plan->d_phi_ok);
      plan->launches++;
      phi = plan->phi_cache;
      if (plan->phi_has_bases) { phi_base = plan->phi_base; phi_has = plan->phi_has; }
    }
  }
  synax_status rs;
  if (code == kGridB)
    rs = grid_vjp(plan->ft, make_geo(plan), bc, bd, model, make_scalar_desc(model->ne_grid, model->ne_n, model->ne_l),
                  make_scalar_desc(model->n0_grid, model->n0_n, model->n0_l), params, dI, dQ, dU, grad, plan->precision, escalate_at(plan),
                  sm_count(plan->device), &plan->ws, st, &plan->launches);
  else
    rs = analytic_vjp(code, plan->ft, make_geo(plan), bc, bd, batch, model->n_params, G,
                      make_scalar_desc(model->ne_grid, model->ne_n, model->ne_l),
                      make_scalar_desc(model->n0_grid, model->n0_n, model->n0_l), plan->precision, escalate_at(plan),
                      plan->batch_share, phi, plan->d_phi_ok, phi_base, phi_has, plan->d_vjp_ctrl, plan->aux, plan->ev_fork, plan->ev_join,
                      dI, dQ, dU, grad, &plan->ws, st, &plan->launches);
  if (rs == SYNAX_ERR_UNSUPPORTED) return fail(rs, "GRID_B vjp: n_los too large for the shared-memory hand-over (see synax.h)");
  if (rs != SYNAX_OK) return fail(rs, "vjp failed: %s", cudaGetErrorString(cudaGetLastError()));
  return SYNAX_OK;
}

// ------------------------------------------------------------------------------------------------
// The paper's arithmetic: everything in float64, float64 buffers at the boundary (synax_dd.cuh).
// ------------------------------------------------------------------------------------------------
static synax_status check_f64_model(const synax_plan* plan, const synax_model* model, const void* params, int32_t batch, int* code) {
  synax_status stt = check_model(plan, model, params, batch, code);
  if (stt != SYNAX_OK) return stt;
  if (*code == kGridB) return fail(SYNAX_ERR_UNSUPPORTED, "the float64 entry points take the analytic models (DISC4, FULL16, STACK16, UNIFORM)");
  return SYNAX_OK;
}

extern "C" synax_status synax_forward_f64(const synax_plan* plan, const synax_model* model, const double* params,
                                          int32_t batch, double* I, double* Q, double* U, void* cuda_stream) {
  int code = 0;
  synax_status stt = check_f64_model(plan, model, params, batch, &code);
  if (stt != SYNAX_OK) return stt;
  if (!I || !Q || !U) return fail(SYNAX_ERR_INVALID_ARG, "I, Q or U is NULL");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  StreamScratch scratch(plan, st);
  void* bc64 = nullptr;
  CUDA_TRY(scratch.get(&bc64, dd_consts_bytes(batch)));
  stt = dd_forward(code, plan->ft, make_geo(plan), params, model->n_params, batch, make_aux(model),
                   make_scalar_desc(model->ne_grid, model->ne_n, model->ne_l), make_scalar_desc(model->n0_grid, model->n0_n, model->n0_l),
                   pick_lanes(plan, plan->npix * batch), bc64, I, Q, U, st, &plan->launches);
  if (stt != SYNAX_OK) return fail(stt, "float64 forward launch failed: %s", cudaGetErrorString(cudaGetLastError()));
  return SYNAX_OK;
}

extern "C" synax_status synax_vjp_f64(const synax_plan* plan, const synax_model* model, const double* params,
                                      int32_t batch, const double* dI, const double* dQ, const double* dU, double* grad,
                                      void* cuda_stream) {
  int code = 0;
  synax_status stt = check_f64_model(plan, model, params, batch, &code);
  if (stt != SYNAX_OK) return stt;
  if (!grad) return fail(SYNAX_ERR_INVALID_ARG, "grad is NULL");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  StreamScratch scratch(plan, st);
  void* bc64 = nullptr;
  double* partial = nullptr;
  const int G = pick_lanes(plan, plan->npix * batch);
  CUDA_TRY(scratch.get(&bc64, dd_consts_bytes(batch)));
  CUDA_TRY(scratch.get(&partial, sizeof(double) * 16 * (size_t)dd_vjp_blocks(plan->npix, G) * (size_t)batch));
  stt = dd_vjp(code, plan->ft, make_geo(plan), params, model->n_params, batch, make_aux(model),
               make_scalar_desc(model->ne_grid, model->ne_n, model->ne_l), make_scalar_desc(model->n0_grid, model->n0_n, model->n0_l),
               G, bc64, partial, dI, dQ, dU, grad, st, &plan->launches);
  if (stt != SYNAX_OK) return fail(stt, "float64 vjp launch failed: %s", cudaGetErrorString(cudaGetLastError()));
  return SYNAX_OK;
}

// synax_vjp_f64 without any allocation: the scratch is a fixed array inside the library (synax_dd.cu).
extern "C" synax_status synax_vjp_f64_noalloc(const synax_plan* plan, const synax_model* model, const double* params,
                                              int32_t batch, const double* dI, const double* dQ, const double* dU,
                                              double* grad, void* cuda_stream) {
  int code = 0;
  synax_status stt = check_f64_model(plan, model, params, batch, &code);
  if (stt != SYNAX_OK) return stt;
  if (!grad) return fail(SYNAX_ERR_INVALID_ARG, "grad is NULL");
  const int G = pick_lanes(plan, plan->npix * batch);
  const size_t need = dd_noalloc_bytes(plan->npix, G, batch), cap = dd_noalloc_capacity();
  if (need > cap)
    return fail(SYNAX_ERR_UNSUPPORTED,
                "synax_vjp_f64_noalloc: this call needs %zu bytes of scratch (npix %lld x %d lanes, batch %d) but the static "
                "array holds %zu; use synax_vjp_f64, a smaller batch or fewer lanes",
                need, (long long)plan->npix, G, (int)batch, cap);
  cudaError_t ce = cudaSuccess;
  stt = dd_vjp_noalloc(plan->device, code, plan->ft, make_geo(plan), params, model->n_params, batch, make_aux(model),
                       make_scalar_desc(model->ne_grid, model->ne_n, model->ne_l),
                       make_scalar_desc(model->n0_grid, model->n0_n, model->n0_l), G, dI, dQ, dU, grad,
                       (cudaStream_t)cuda_stream, &plan->launches, &ce);
  if (stt != SYNAX_OK)
    return fail(stt, "synax_vjp_f64_noalloc failed: %s%s", cudaGetErrorString(ce),
                ce == cudaErrorInvalidDevice ? " (the plan's device must be the current device)" : "");
  return SYNAX_OK;
}

// ------------------------------------------------------------------------------------------------
// Fused Gaussian likelihood (Eq.(15)): forward -> residual cotangents + logL -> VJP.
// ------------------------------------------------------------------------------------------------
// In place: map <- -w (map - obs) (the cotangent of logL), and logL[b] -= w/2 sum (map - obs)^2.
__global__ void __launch_bounds__(256) loglike_residual_kernel(float* __restrict__ map, const float* __restrict__ obs,
                                                               int64_t per_batch, float w, double* __restrict__ logL) {
  const int b = blockIdx.y;
  float* m = map + (int64_t)b * per_batch;
  double acc = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < per_batch; i += (int64_t)gridDim.x * blockDim.x) {
    const float r = m[i] - __ldg(obs + i);
    m[i] = -w * r;
    acc += (double)r * (double)r;
  }
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) {
    int lo = __double2loint(acc), hi = __double2hiint(acc);
    lo = __shfl_xor_sync(0xffffffffu, lo, d); hi = __shfl_xor_sync(0xffffffffu, hi, d);
    acc += __hiloint2double(hi, lo);
  }
  __shared__ double part[8];
  if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int k = 0; k < 8; ++k) t += part[k];
    atomicAdd(logL + b, -0.5 * (double)w * t);
  }
}

extern "C" synax_status synax_loglike_vjp(const synax_plan* plan, const synax_model* model, const float* params,
                                          int32_t batch, const float* I_obs, const float* Q_obs, const float* U_obs,
                                          const double inv_var[3], double* logL, float* grad, void* cuda_stream) {
  int code = 0;
  synax_status stt = check_model(plan, model, params, batch, &code);
  if (stt != SYNAX_OK) return stt;
  if (!inv_var || !logL || !grad) return fail(SYNAX_ERR_INVALID_ARG, "inv_var, logL or grad is NULL");
  for (int k = 0; k < 3; ++k)
    if (!(inv_var[k] >= 0.0) || !std::isfinite(inv_var[k])) return fail(SYNAX_ERR_INVALID_ARG, "inv_var[%d] must be finite and >= 0", k);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int64_t per_batch = (int64_t)plan->n_freq * plan->npix;
  const size_t count = (size_t)batch * (size_t)per_batch;
  StreamScratch scratch(plan, st);
  float* maps = nullptr;
  CUDA_TRY(scratch.get(&maps, 3 * count * sizeof(float)));
  float* m[3] = {maps, maps + count, maps + 2 * count};
  synax_status rs = synax_forward(plan, model, params, batch, m[0], m[1], m[2], cuda_stream);
  if (rs == SYNAX_OK) {
    CUDA_TRY(cudaMemsetAsync(logL, 0, sizeof(double) * (size_t)batch, st));
    const float* obs[3] = {I_obs, Q_obs, U_obs};
    const float* cot[3] = {nullptr, nullptr, nullptr};
    const unsigned bx = (unsigned)std::min<int64_t>((per_batch + 255) / 256, (int64_t)sm_count(plan->device) * 8);
    for (int k = 0; k < 3; ++k) {
      if (!obs[k] || inv_var[k] == 0.0) continue;
      for (int b0 = 0; b0 < batch; b0 += 65535) {   // gridDim.y limit
        loglike_residual_kernel<<<dim3(bx, (unsigned)std::min(65535, batch - b0)), 256, 0, st>>>(
            m[k] + (size_t)b0 * per_batch, obs[k], per_batch, (float)inv_var[k], logL + b0);
        plan->launches++;
      }
      cot[k] = m[k];
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) rs = fail(SYNAX_ERR_CUDA, "loglike residual launch failed: %s", cudaGetErrorString(e));
    else rs = synax_vjp(plan, model, params, batch, cot[0], cot[1], cot[2], grad, cuda_stream);
  }
  return rs;
}

// ADAM (Kingma & Ba 2015, Algorithm 1) -- the paper's field-level optimiser
__global__ void adam_kernel(float* __restrict__ theta, const float* __restrict__ grad, float* __restrict__ m,
                            float* __restrict__ v, int64_t n, float lr, float b1, float b2, float eps, float c1, float c2,
                            float sign) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const float g = sign * grad[i];
  const float mi = fmaf(b1, m[i], (1.0f - b1) * g);
  const float vi = fmaf(b2, v[i], (1.0f - b2) * g * g);
  m[i] = mi; v[i] = vi;
  theta[i] -= lr * (mi * c1) / (sqrtf(vi * c2) + eps);
}

extern "C" synax_status synax_adam_step(float* theta, const float* grad, float* m, float* v, int64_t n, double lr,
                                        double beta1, double beta2, double eps, int32_t t, int32_t maximize,
                                        void* cuda_stream) {
  if (!theta || !grad || !m || !v) return fail(SYNAX_ERR_INVALID_ARG, "theta, grad, m or v is NULL");
  if (n < 1 || t < 1) return fail(SYNAX_ERR_INVALID_ARG, "n and t must be >= 1");
  if (!(beta1 >= 0 && beta1 < 1 && beta2 >= 0 && beta2 < 1) || !(eps >= 0) || !std::isfinite(lr))
    return fail(SYNAX_ERR_INVALID_ARG, "need 0 <= beta < 1, eps >= 0, finite lr");
  const double c1 = 1.0 / (1.0 - std::pow(beta1, (double)t)), c2 = 1.0 / (1.0 - std::pow(beta2, (double)t));
  adam_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(
      theta, grad, m, v, n, (float)lr, (float)beta1, (float)beta2, (float)eps, (float)c1, (float)c2, maximize ? -1.0f : 1.0f);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(SYNAX_ERR_CUDA, "adam launch failed: %s", cudaGetErrorString(e));
  return SYNAX_OK;
}

// ------------------------------------------------------------------------------------------------
// HOST-buffer variants: copies inside the call, stream synchronised on return.
// ------------------------------------------------------------------------------------------------
// Device alias of a page-locked host buffer (cudaHostAlloc, cudaHostRegister, torch pin_memory), or null for
// ordinary pageable memory.
static float* pinned_alias(const void* host) {
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, host) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  return at.type == cudaMemoryTypeHost ? (float*)at.devicePointer : nullptr;
}

extern "C" synax_status synax_forward_host(const synax_plan* plan, const synax_model* model, const float* params,
                                           int32_t batch, float* I, float* Q, float* U, void* cuda_stream) {
  int code = 0;
  synax_status stt = check_model(plan, model, params, batch, &code);
  if (stt != SYNAX_OK) return stt;
  if (!I || !Q || !U) return fail(SYNAX_ERR_INVALID_ARG, "I, Q or U is NULL");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t pbytes = sizeof(float) * (size_t)model->n_params * (size_t)batch;
  const size_t mbytes = sizeof(float) * (size_t)batch * plan->n_freq * (size_t)plan->npix;
  float *dp = nullptr, *dm = nullptr;
  StreamScratch scratch(plan, st);
  CUDA_TRY(scratch.get(&dp, pbytes));
  CUDA_TRY(cudaMemcpyAsync(dp, params, pbytes, cudaMemcpyHostToDevice, st));
  // Page-locked map buffers: the kernels store straight into them.  A map value is written exactly once, by the
  // thread that finishes its sightline, in 128-byte runs of adjacent pixels, and never read back -- posted writes
  // spread over the whole kernel instead of a staging buffer and three copies behind it (A/B on one box, cfg 4:
  // 27.5-29.2 against 29.6-40.7 ms per forward + VJP step; the device-timed forward is unchanged).
  float *zI = pinned_alias(I), *zQ = pinned_alias(Q), *zU = pinned_alias(U);
  if (zI && zQ && zU) {
    synax_status rz = synax_forward(plan, model, dp, batch, zI, zQ, zU, cuda_stream);
    CUDA_TRY(cudaStreamSynchronize(st));
    return rz;
  }
  CUDA_TRY(scratch.get(&dm, 3 * mbytes));
  float* dI = dm; float* dQ = dm + mbytes / sizeof(float); float* dU = dm + 2 * (mbytes / sizeof(float));
  synax_status rs = synax_forward(plan, model, dp, batch, dI, dQ, dU, cuda_stream);
  if (rs == SYNAX_OK) {
    CUDA_TRY(cudaMemcpyAsync(I, dI, mbytes, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(Q, dQ, mbytes, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(U, dU, mbytes, cudaMemcpyDeviceToHost, st));
  }
  CUDA_TRY(cudaStreamSynchronize(st));
  return rs;
}

extern "C" synax_status synax_vjp_host(const synax_plan* plan, const synax_model* model, const float* params,
                                       int32_t batch, const float* dI, const float* dQ, const float* dU, float* grad,
                                       void* cuda_stream) {
  int code = 0;
  synax_status stt = check_model(plan, model, params, batch, &code);
  if (stt != SYNAX_OK) return stt;
  if (!grad) return fail(SYNAX_ERR_INVALID_ARG, "grad is NULL");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t pbytes = sizeof(float) * (size_t)model->n_params * (size_t)batch;
  const size_t mcount = (size_t)batch * plan->n_freq * (size_t)plan->npix;
  float *dp = nullptr, *dg = nullptr, *dc = nullptr;
  StreamScratch scratch(plan, st);
  CUDA_TRY(scratch.get(&dp, pbytes));
  CUDA_TRY(scratch.get(&dg, pbytes));
  CUDA_TRY(scratch.get(&dc, 3 * mcount * sizeof(float)));
  CUDA_TRY(cudaMemcpyAsync(dp, params, pbytes, cudaMemcpyHostToDevice, st));
  const float* src[3] = {dI, dQ, dU};
  const float* dev[3] = {nullptr, nullptr, nullptr};
  for (int k = 0; k < 3; ++k)
    if (src[k]) {
      CUDA_TRY(cudaMemcpyAsync(dc + k * mcount, src[k], mcount * sizeof(float), cudaMemcpyHostToDevice, st));
      dev[k] = dc + k * mcount;
    }
  synax_status rs = synax_vjp(plan, model, dp, batch, dev[0], dev[1], dev[2], dg, cuda_stream);
  if (rs == SYNAX_OK) CUDA_TRY(cudaMemcpyAsync(grad, dg, pbytes, cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  return rs;
}
