/* synax.h -- C ABI of libsynax: line-of-sight integration of Galactic synchrotron Stokes I/Q/U with
 * Faraday rotation on HEALPix sightlines, and its adjoint (VJP) w.r.t. the field-model parameters.
 * Hand-written CUDA for NVIDIA B200 (sm_100a).  No CPU fallback: every call needs a CUDA device.
 *
 * The operation is the hot path of arXiv:2410.01136 ("synax"); citations P:L<n> are line numbers of
 * the paper text (reference PAPER.md), S:<tag> the readings listed in DESIGN.md section 3.
 *
 *   direction of RING pixel i -> (l_i, b_i)                         P:L108 (healpy; Gorski+05 P:L352)
 *   N_int equal segments on [0, s_max], midpoints r_{i,n}            P:L108, observer P:L49
 *   fields B, N_0, n_e, alpha at r_{i,n} (analytic or gridded)       P:L99-110, Eq.12-13
 *   j_I Eq.(2), j_P Eq.(5), chi_0 Eq.(8)
 *   Faraday depth Eq.(7) P:L79 (half-cell midpoint form), chi = RM lambda^2 + chi_0 Eq.(6)
 *   I,Q,U = sum_n j {1, cos 2chi, sin 2chi} Delta_r  Eq.(9), in Kelvin (Rayleigh-Jeans)
 *   reverse-mode gradient of all of the above (the paper uses JAX AD)
 *
 * Units: micro-gauss, kpc, cm^-3, rad, Hz, Kelvin.  HEALPix RING pixel order.  The line of sight n
 * points away from the observer; B_LOS = B.n is signed; +Q is along increasing Galactic longitude
 * (B along e_E gives Q = +P).
 *
 * Pointers: "DEVICE" = device memory of the plan's CUDA device, "HOST" = ordinary host memory.  All
 * buffers are caller-owned; the library never frees or keeps them.  Device calls are asynchronous on
 * `cuda_stream` (a cudaStream_t; NULL = default stream) and the buffers must stay alive until the
 * stream reaches the call; *_host calls return after their results are in the host buffers.
 * Every failure returns a non-zero status and sets synax_last_error(); nothing aborts or throws.
 * Invalid arguments launch no kernel.  Parameter VALUES are not range-checked (NaN in, NaN out).
 */
#ifndef SYNAX_H
#define SYNAX_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct synax_plan synax_plan; /* opaque, library-owned */

typedef enum {
  SYNAX_OK = 0,
  SYNAX_ERR_INVALID_ARG = 1,
  SYNAX_ERR_UNSUPPORTED = 2,
  SYNAX_ERR_CUDA = 3,
  SYNAX_ERR_ALLOC = 4
} synax_status;

typedef enum {
  /* WMAP logarithmic spiral, Eq.(13): params (b0 [uG], psi0, psi1, chi0 [rad]);
   * B = 0 outside 3 < rho < 20 kpc (S:C-2#7).  CR density Eq.(12), alpha and n_e come from `aux`. */
  SYNAX_MODEL_DISC4 = 0,
  /* 16 parameters (BASELINE.json configs 2/4; S:App.C):
   * b0 psi0 psi1 chi0 h_b | B_h z_h0 r_h w_h | n0 h_r h_z alpha | ne0 h_er h_ez
   * disc = DISC4 * exp(-(rho-8)/h_b); halo = B_h /(1+((|z|-z_h0)/w_h)^2) (rho/r_h) exp(1-rho/r_h) phi_hat;
   * N_0 = n0 exp(-rho/h_r) sech^2(z/h_z) Eq.(12); n_e likewise. */
  SYNAX_MODEL_FULL16 = 1,
  /* B on a regular grid [nx][ny][nz][3] (fp32, c fastest), nodes on the faces of a box of lengths
   * (lx,ly,lz) centred on the Galactic centre, trilinear interpolation, zero outside (
   * S:C-2#12).  params IS the grid; CR/alpha/n_e from `aux`.  batch must be 1. */
  SYNAX_MODEL_GRID_B = 2,
  /* homogeneous fields everywhere (toy of P:L123): params (Bx,By,Bz [uG], N0, n_e, alpha). */
  SYNAX_MODEL_UNIFORM = 3,
  /* the paper's own 16-parameter model, Eq.(16) P:L283-289 with Table 3: params (b0 [uG], psi0, psi1,
   * chi0 [rad]) x 4 WMAP spirals B_1..B_4, stacked as
   *   B_x = .6 B1x + .3 B2x + .1 B3z + .3 B4y;  B_y = .6 B1y + .3 B2z + .1 B3y + .3 B4x;  B_z = .6 B1z + .3 B2y + .1 B3x + .3 B4z
   * CR density, alpha and n_e from `aux` (or the optional grids) as for DISC4. */
  SYNAX_MODEL_STACK16 = 4
} synax_model_kind;

typedef struct {
  int32_t kind;     /* synax_model_kind */
  int32_t n_params; /* 4, 16, nx*ny*nz*3 (<2^31), 6, 16 -- must match kind */
  const float* aux; /* HOST. DISC4 / GRID_B / STACK16: {C0, h_r, h_z, alpha, ne0, h_er, h_ez}; else NULL */
  int32_t nx, ny, nz; /* GRID_B only, each >= 2 */
  double lx, ly, lz;  /* GRID_B only, kpc, > 0 (float64: a length rounded to fp32 rescales the grid by up to 6e-8, which
                       * is 1e-3 rad of Faraday rotation at 350 MHz through a strong field) */
  /* Optional gridded scalar fields (the paper's n_e is the YMW16 model on a (256,256,64) grid):
   * DEVICE fp32 [n][n][n] (z fastest), nodes on the faces of a box of lengths *_l centred on the Galactic centre,
   * trilinear, zero outside.  DISC4 and GRID_B only; a non-NULL grid REPLACES the analytic disc built from `aux`
   * (its aux entries are then ignored).  Not differentiated.  NULL (and zeroed sizes) = unused. */
  const float* ne_grid; int32_t ne_n[3]; double ne_l[3];
  const float* n0_grid; int32_t n0_n[3]; double n0_l[3];
} synax_model;

/* Plan = geometry shared by all calls: HEALPix nside (1..8192), samples per sightline n_los
 * (1..65536), path length s_max > 0 (every sightline is integrated over [0, s_max], S:C-2#6),
 * frequencies (HOST, 1..32 values, Hz, > 0) and the observer position (HOST, kpc; P:L49 uses
 * (-8.3, 0, 0.006)).  Created on the current CUDA device; computes and caches the pixel directions
 * there (step A1) and returns after that kernel finished. */
synax_status synax_plan_create(int32_t nside, int32_t n_los, double s_max_kpc, const double* freqs_hz,
                               int32_t n_freq, const double observer_kpc[3], synax_plan** out);
/* The same for a shard of the sky: RING pixels pix_begin .. pix_begin + pix_count - 1 only (sightlines are
 * independent).  Every map / cotangent buffer of this plan then has pix_count pixels
 * per (batch, frequency), and synax_vjp returns the shard's partial gradient (sum over its pixels): summing
 * the partial gradients of disjoint shards that cover the map gives the gradient of the whole map. */
synax_status synax_plan_create_shard(int32_t nside, int32_t n_los, double s_max_kpc, const double* freqs_hz,
                                     int32_t n_freq, const double observer_kpc[3], int64_t pix_begin,
                                     int64_t pix_count, synax_plan** out);
/* The same for every pix_stride-th pixel: RING pixels pix_begin + i * pix_stride, i < pix_count (all inside the map,
 * pix_stride >= 1).  Rank r of N taking (r, N, ceil((npix - r) / N)) gives N disjoint shards that each see every latitude,
 * so their run times are equal -- contiguous RING ranges are latitude bands, and the bands along the Galactic plane take
 * 1.4x as long as the polar ones at 408 MHz.  Buffers and the partial gradient as for a shard. */
synax_status synax_plan_create_strided(int32_t nside, int32_t n_los, double s_max_kpc, const double* freqs_hz,
                                       int32_t n_freq, const double observer_kpc[3], int64_t pix_begin,
                                       int64_t pix_stride, int64_t pix_count, synax_plan** out);
synax_status synax_plan_destroy(synax_plan* plan); /* NULL is allowed */
int64_t synax_plan_npix(const synax_plan* plan);  /* pixels of this plan (12 nside^2 unless a shard), -1 for NULL */

/* Integration extent of the paper (Fig. 1): from the observer to where the sightline leaves a box of
 * side lengths box_kpc[3] centred on the Galactic centre, cut into n_los equal segments -- every sightline then has
 * its own segment length Delta r_i = L_i / n_los.  The observer must be strictly inside the box (else
 * SYNAX_ERR_INVALID_ARG).  Replaces the fixed [0, s_max] for all later calls with this plan; NULL restores it.
 * HOST pointer; synchronises the device. */
synax_status synax_plan_set_box(synax_plan* plan, const double box_kpc[3]);

/* Options.  key "precision": 0 = auto (default), 1 = fp32 only, 2 = float64 Faraday chain for every sightline,
 * (everything in float64, the paper's default precision: synax_forward_f64 / synax_vjp_f64 below).
 * Auto, forward: sightlines whose Faraday round-off scale k_max sum_n |n_e| (|B_LOS|+|B_N|+|B_E|) exceeds
 * "escalate_rad" (default 300 rad, calibrated against the oracle: DESIGN.md section 5) take the float64 Faraday
 * chain -- as a redo of a flagged list after the fp32 pass, for every sightline when a device-side pilot finds most of
 * them flagged, or split between the two chains in between.  Auto, VJP: decided per sightline (per CTA in long calls)
 * -- those above escalate_rad take their Faraday angles from the float64 chain.
 * No mode ever synchronises with the host.  key "escalate_rad": threshold in radians (> 0), for plans with n_los >= 128;
 * below that the threshold in force is escalate_rad x n_los / 128 (a few samples per sightline average no rounding out).
 * key "lanes": lanes per sightline (0 = heuristic, else 1, 8 or 32).  Heuristic: one thread per sightline from 150,000
 * sightlines (npix x batch) in synax_forward, from 300,000 in a stand-alone synax_vjp and the float64 entry points, and from
 * 24,576 in a synax_vjp that finds the Faraday sums of the plan's last forward; 8 lanes down to an eighth of that, else 32.
 * key "use_forward_totals" (setting it, to either value, also drops what the plan has stored): 1 (default) = synax_vjp may
 * take the sightlines' Faraday sums from what the plan's last
 * synax_forward stored (see synax_vjp); 0 = it always recomputes them in its own pre-pass.
 * key "batch_share": parameter vectors integrated per thread when a batch of analytic models is evaluated at one
 * frequency with one thread per sightline -- they share the sightline geometry (0 = heuristic, else 1, 2 or 4).  In
 * synax_vjp values 2 and 4 apply unless the plan's last forward left tile bases (then the kernel that uses those runs).
 * key "pool_release_threshold_mb": raise the release threshold of the device's default stream-ordered memory pool to this
 * many MB.  Per-call scratch comes from a workspace the plan keeps (see "Scratch" below); the pool serves what does not
 * fit into it -- a call that needs more than 256 MB, e.g. the host entry points' staging of large maps -- and every call
 * made inside a stream capture.  With CUDA's default threshold (0) the pool hands everything back at each stream or
 * device synchronisation, and the first pool allocation after one waits ~0.23 ms of host time for memory to be mapped
 * again (measured on B200; while all scratch came from the pool, a cfg-1 forward took 0.38 instead of 0.15 ms in a loop
 * that synchronised every step).  Process-wide for that device, hence opt-in; never lowers a larger threshold set by
 * the application. */
synax_status synax_plan_set_option(synax_plan* plan, const char* key, double value);

/* Pixel directions as cached by the plan: out[4*p..] = (cos l, sin l, cos b, sin b), DEVICE float64
 * [npix][4].  For tests of step A1. */
synax_status synax_plan_directions(const synax_plan* plan, double* out_device, void* cuda_stream);

/* Forward.  params: DEVICE fp32 [batch][n_params] (GRID_B: the grid, batch == 1).
 * I, Q, U: DEVICE fp32 [batch][n_freq][npix], overwritten, Kelvin.
 * Side effect kept inside the plan: a call over >= 24,576 sightlines (or with option "lanes" = 1; analytic models without
 * a gridded n_e; any lane count) also stores each sightline's Faraday sum (one float64, Eq.(7)
 * P:L79 at the far end), for the sightlines its float64 chain integrates the Faraday depth before every 32nd sample (8 bytes
 * per 32 samples and sightline: 201 MB at nside 256 x 1024 samples) and a device copy of `params`, for the next synax_vjp of
 * this plan.  The buffers are plan-owned and grown with cudaMalloc the first time a call of a given size comes (that call
 * synchronises the device once; never inside a stream capture; if the memory is not there the call goes on without them).
 * GRID_B: per-call scratch of 16 bytes per grid node (the grid repacked into 16-byte nodes); synax_vjp takes another 16 bytes
 * per node for the gradient accumulation.
 * Scratch (every entry point but synax_vjp_f64_noalloc): constants, lists, block partials and the buffers above are cut, in
 * stack order, from ONE workspace that stays with the plan (at most 256 MB; grown with cudaFree + cudaMalloc at the start of a
 * call when an earlier call needed more -- that call synchronises the device once; never inside a stream capture).  What
 * does not fit, and all scratch of a call made inside a stream capture (a captured graph must not point into a buffer that
 * may be reallocated), comes from the device's default stream-ordered memory pool (option "pool_release_threshold_mb"). */
synax_status synax_forward(const synax_plan* plan, const synax_model* model, const float* params,
                           int32_t batch, float* I, float* Q, float* U, void* cuda_stream);

/* VJP.  dI, dQ, dU: DEVICE fp32 [batch][n_freq][npix] cotangents (any may be NULL = zeros).
 * grad: DEVICE fp32 [batch][n_params] (GRID_B: [nx][ny][nz][3]); overwritten:
 * grad[b][j] = sum_{f,p} dI dI/dtheta_j + dQ dQ/dtheta_j + dU dU/dtheta_j.
 * DISC4 / GRID_B: `aux` values are constants (not differentiated).
 * The adjoint sweeps every sightline from its far end to the observer and needs the sightline's Faraday sum first: it takes
 * the sums the plan's last synax_forward stored when that call had the same model, batch, options and integration extent and
 * `params` holds bit-identical values (compared on the device, no synchronisation).  With the forward's tile-wise Faraday
 * depths it also needs no float64 Faraday chain of its own.  Otherwise: when the plan holds nothing for this model, batch,
 * options and extent (no forward yet, or settings changed) and the call is long (>= 24,576 sightlines, >= 5e7 LoS samples,
 * several frequencies or STACK16 / UNIFORM), the call first runs a Faraday-only pass of the forward (its strategy and
 * kernels without emission, rotation and maps: about half a forward) and stores the same sums itself -- the plan then holds
 * them for later calls with these parameters; at one frequency (DISC4 / FULL16, one thread per sightline) a forward-order
 * kernel runs that needs no sums; in all other cases (short calls; stored sums that turn out on the device to belong to
 * other parameter values) the sums come from a pre-pass inside the adjoint kernel (+30-70 % work).
 * Results do not depend on the route beyond rounding (both are held to the same bound against the oracle).
 * Ordering: all work is ordered with `cuda_stream` (results are complete when the stream reaches the end of the
 * call).  Long calls (>= 262,144 sightlines) may run part of their kernels on a second stream owned by the plan,
 * forked from and joined back to `cuda_stream` by events inside the call (CUDA-graph capturable); a plan must
 * therefore not be used by two calls that run concurrently -- use one plan per stream.  (synax_forward does the same
 * in its split mode: from 262,144 sightlines, or from 32,768 sightlines with 5e7 or more LoS samples.)
 * GRID_B: n_los <= 4096 (the per-sample hand-over between the two sweeps lives in shared memory); larger n_los
 * returns SYNAX_ERR_UNSUPPORTED. */
synax_status synax_vjp(const synax_plan* plan, const synax_model* model, const float* params,
                       int32_t batch, const float* dI, const float* dQ, const float* dU, float* grad,
                       void* cuda_stream);

/* The paper's own arithmetic (section 2.4: "the default precision is double ... for all examples"): the same two
 * operations with EVERY step in float64 -- positions, fields, emissivity (Eq. 2, 5), Faraday depth (Eq. 7), rotation
 * (Eq. 6), sums (Eq. 9) and the whole adjoint -- on float64 buffers: params DEVICE float64 [batch][n_params]; I, Q, U
 * and the cotangents DEVICE float64 [batch][n_freq][npix]; grad DEVICE float64 [batch][n_params].  Analytic models only
 * (DISC4, FULL16, STACK16, UNIFORM; GRID_B returns SYNAX_ERR_UNSUPPORTED); optional n_e / N_0 grids stay fp32 arrays,
 * interpolated in float64.  The plan's precision / escalate_rad options do not apply.  Asynchronous on `cuda_stream`. */
synax_status synax_forward_f64(const synax_plan* plan, const synax_model* model, const double* params,
                               int32_t batch, double* I, double* Q, double* U, void* cuda_stream);
synax_status synax_vjp_f64(const synax_plan* plan, const synax_model* model, const double* params,
                           int32_t batch, const double* dI, const double* dQ, const double* dU, double* grad,
                           void* cuda_stream);

/* synax_vjp_f64 for callers that cannot allocate (CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): same arguments, same result, but the call's scratch -- the per-batch float64 constants and the per-CTA
 * partial gradients -- lives in a fixed 4 MiB array inside the library image (every GPU that loads the library holds it
 * until the process exits) and the call makes no cudaMalloc, cudaFree or other allocating call.  Limit: a call needs
 * 872 * batch bytes (rounded up to 256) + 128 * batch * ceil(npix * lanes / 128) bytes (lanes = the "lanes" option, else
 * 1, 8 or 32 by size); e.g. nside 64 x batch 10 at 8 lanes, or nside 256 x batch 5 at 1 lane.  More returns SYNAX_ERR_UNSUPPORTED and
 * the message states both numbers; nothing is launched.  The plan's device must be the current device (as for every call).
 * ALL calls on a device share the array: it keeps the last call's contents (a call clears what it reads before use), and
 * two calls that overlap on the GPU -- different streams, or different host threads -- race: keep them on one stream. */
synax_status synax_vjp_f64_noalloc(const synax_plan* plan, const synax_model* model, const double* params,
                                   int32_t batch, const double* dI, const double* dQ, const double* dU, double* grad,
                                   void* cuda_stream);

/* Same operations with HOST buffers of the same shapes: the call copies the inputs to the device,
 * runs, copies the results back and synchronises the stream before returning.  When I, Q and U are all page-locked
 * (cudaHostAlloc / cudaHostRegister) the forward kernels store the maps straight into them and no copy is made.
 * Scratch: the plan's workspace up to 256 MB, beyond that the device's default stream-ordered memory pool (see option
 * "pool_release_threshold_mb": staging cfg 4's maps takes 226 MB). */
synax_status synax_forward_host(const synax_plan* plan, const synax_model* model, const float* params,
                                int32_t batch, float* I, float* Q, float* U, void* cuda_stream);
synax_status synax_vjp_host(const synax_plan* plan, const synax_model* model, const float* params,
                            int32_t batch, const float* dI, const float* dQ, const float* dU,
                            float* grad, void* cuda_stream);

/* Gaussian pixel log-likelihood of Eq.(15) P:L193-197 and its gradient in ONE call (the inner loop of the
 * paper's HMC / ADAM runs): forward, residuals, VJP, with no map leaving the device:
 *   logL[b] = -1/2 sum_{f,p} [ w[0] (I - I_obs)^2 + w[1] (Q - Q_obs)^2 + w[2] (U - U_obs)^2 ]
 *   grad[b][j] = d logL[b] / d theta_j
 * I_obs, Q_obs, U_obs: DEVICE fp32 [n_freq][npix], ONE observation shared by all batch elements; a NULL map takes
 * that Stokes parameter out of the likelihood (the paper uses Q and U only, sigma = 1 mK: w = 1/sigma^2 in K^-2).
 * inv_var: HOST, 3 weights >= 0.  logL: DEVICE float64 [batch], overwritten.  grad: DEVICE fp32 as in synax_vjp.
 * Scratch for the three maps ([batch][n_freq][npix] fp32 each): the plan's workspace (synax_forward), else the pool. */
synax_status synax_loglike_vjp(const synax_plan* plan, const synax_model* model, const float* params,
                               int32_t batch, const float* I_obs, const float* Q_obs, const float* U_obs,
                               const double inv_var[3], double* logL, float* grad, void* cuda_stream);

/* One ADAM update (the optimiser of the paper's field-level fits: Optax ADAM on the 128x128x32 B grid),
 * elementwise on DEVICE buffers of n floats: with g = -grad when `maximize` != 0 (grad of a log-likelihood) else grad,
 *   m <- b1 m + (1-b1) g;  v <- b2 v + (1-b2) g^2;  theta <- theta - lr (m / (1-b1^t)) / (sqrt(v / (1-b2^t)) + eps)
 * (Kingma & Ba 2015, Algorithm 1; t = 1, 2, ... is the step number).  m and v must be zero before the first step. */
synax_status synax_adam_step(float* theta, const float* grad, float* m, float* v, int64_t n, double lr, double beta1,
                             double beta2, double eps, int32_t t, int32_t maximize, void* cuda_stream);

/* Counters since plan creation (for bench.py's gpu_launches): out[0] = kernels launched,
 * out[1] = sightlines redone with the float64 Faraday chain in the last forward (read back lazily:
 * valid after the stream has been synchronised). */
synax_status synax_plan_stats(const synax_plan* plan, int64_t out[2]);

const char* synax_last_error(void); /* thread-local, library-owned, never NULL */
const char* synax_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SYNAX_H */
