/*
 * gprfwi.h -- C-ABI boundary of the B200-native GPR dual-parameter FWI hot path
 * (arxiv/paper_2506_20513): 2-D TM-mode (Ez, Hx, Hy) Yee FDTD in lossy media with CPML, batched
 * over shots, run forward (Algorithm 1) and then as its exact discrete adjoint
 * (Algorithm 2) to give the misfit gradients w.r.t. relative permittivity and
 * conductivity (continuous form: Eqs. (12)-(13)).
 *
 * The paper's own boundary is ctypes -> `void` C functions on raw float pointers
 * (PAPER.md:429-452); this one keeps raw pointers and adds integer error codes.
 *
 * Conventions
 *   - full grid nz x nx Ez nodes INCLUDING the CPML cells; j = z (depth, slow), i = x (fast).
 *     Ez at (j,i), Hx at (j+1/2,i), Hy at (j,i+1/2); eps_r and sigma collocated with Ez
 *     (Eq. (3)); mu = mu0; square cells (the paper's kernel uses one uE1,
 *     PAPER.md:419-424).  The outer ring of Ez nodes is PEC (never updated).
 *   - all arrays fp32.  "device" pointers are CUDA device memory of the current device; "host"
 *     pointers are ordinary host memory.  Model / gradient arrays are [nz][pitch] with row pitch
 *     `pitch` >= nx in floats.  Traces / residuals are [nshots][nt][nrec], receiver fastest
 *     (the paper's rxs[s][comp][iteration][rx]).
 *   - positions are integer full-grid cell indices (z, x) in [1, n-2] (not on the PEC ring).
 *   - wavelet sample n is the line current (A) acting during step n:
 *     Ez[src] -= Cb[src] * w[n] / (dx*dx)  (PAPER.md:364-384 with dl = dz).
 *     trace sample n is Ez at the receiver BEFORE step n (Algorithm 1 stage 1), so sample 0 is 0.
 *   - the library never allocates or frees device memory: every device buffer, including the
 *     workspace that holds fields, CPML psi strips, coefficients, the Ez history or checkpoints,
 *     is caller-owned.  The handle is a small host object.
 *   - all calls only ENQUEUE work on `cuda_stream` (a cudaStream_t passed as void*, NULL = the
 *     legacy default stream); results are valid after the caller synchronises that stream.
 *     Exception: the *_host entry points synchronise the stream before returning.
 *   - return value: 0 (GPRFWI_OK) or a negative gprfwi_status; never throws, never aborts.
 */
#ifndef GPRFWI_H
#define GPRFWI_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  GPRFWI_OK      = 0,
  GPRFWI_EINVAL  = -1, /* null pointer, nz/nx < 2*npml+3, nt <= 0, pitch < nx, dx/dt <= 0, ...   */
  GPRFWI_ECFL    = -2, /* dt > dx / (c0*sqrt(2)): Eq. (11), vacuum c            */
  GPRFWI_EGEOM   = -3, /* a source/receiver index outside [1, n-2]                               */
  GPRFWI_ENOMEM  = -4, /* workspace smaller than gprfwi_workspace_bytes() asks for               */
  GPRFWI_ESTATE  = -5, /* adjoint without a completed forward on this handle                     */
  GPRFWI_ECUDA   = -6, /* a CUDA call or launch failed; text via gprfwi_strerror(GPRFWI_ECUDA)   */
  GPRFWI_ETOOBIG = -7  /* gprfwi_update_noalloc: the model exceeds the library's fixed scratch    */
} gprfwi_status;

typedef struct {
  int32_t nz, nx, pitch;     /* full grid incl. CPML; pitch >= nx, in floats (models, gradients) */
  float   dx, dt;            /* cell size (m), time step (s)                                     */
  int32_t nt;                /* number of time steps                                             */
  int32_t npml, pml_order;   /* CPML thickness in cells (0 = PEC box) and polynomial grading m   */
  float   pml_sigma_max, pml_kappa_max, pml_alpha_max;   /* CPML profile maxima (S/m, -, S/m)    */
  int32_t nshots, nrec;      /* shots batched in one call; receivers per shot                    */
  int32_t wavelet_per_shot;  /* 0: wavelet[nt] shared by all shots; 1: wavelet[nshots][nt]       */
  int32_t checkpoint_stride; /* 0: choose from the workspace size (full history if it fits);
                                K > 0: force checkpoint-and-recompute with stride K              */
} gprfwi_params;

typedef struct gprfwi_handle gprfwi_handle;

/* How the library will lay the problem out in a workspace of at most budget_bytes. */
typedef struct {
  uint64_t workspace_bytes;  /* bytes the plan needs (<= budget)                                 */
  int32_t  full_history;     /* 1: all nt+1 Ez planes held; 0: checkpoint-and-recompute          */
  int32_t  checkpoint_stride;/* K (= nt when full_history)                                       */
  int32_t  shots_per_pass;   /* shots swept together in the adjoint (sub-batch size)             */
  int32_t  time_block;       /* time steps fused per kernel launch                               */
  int32_t  stored_segments;  /* checkpoint segments (the last ones) whose Ez planes the forward pass
                                keeps in spare workspace, so the adjoint does not recompute them    */
  int32_t  reserved;
} gprfwi_plan;

/* Smallest workspace (bytes) with which gprfwi_forward/adjoint can run `p` when allowed to use
 * at most budget_bytes (0 = no limit): the full Ez history if it fits,
 * otherwise checkpoint-and-recompute with a stride and a shot sub-batch chosen to fit; what the
 * budget leaves beyond that plan's minimum then holds the Ez planes of the last checkpoint segments
 * (plan->stored_segments of them), which the adjoint sweeps without recomputing.  The returned size
 * includes those planes and never exceeds budget_bytes.
 * Returns 0 if `p` is invalid or nothing fits.  If plan != NULL it is filled in. */
size_t gprfwi_workspace_bytes(const gprfwi_params* p, size_t budget_bytes, gprfwi_plan* plan);

/* Forward modelling, Algorithm 1: coefficient build, then
 * nt steps of {record receivers, H update + H CPML (Eqs. 4-5), E update + E CPML (Eq. 3 in the
 * Ca/Cb form of PAPER.md:415-424), source injection, save wavefield}.
 *   h        out: *h receives a new handle (release with gprfwi_release).  If *h is non-NULL on
 *            entry it is reused (it must come from an earlier call with identical params).  A reused
 *            handle that meets the same workspace, plan and acquisition again does not rebuild or
 *            re-upload the receiver / CPML tables it keeps in the workspace: between calls on a live
 *            handle the caller must leave the workspace alone.
 *   eps_r, sigma   device [nz][pitch]; must stay unmodified until the last gprfwi_adjoint
 *   wavelet  device [nt] or [nshots][nt]
 *   src_zx   host   [nshots][2]        (z, x) cell indices, copied
 *   rec_zx   host   [nshots][nrec][2]  copied
 *   workspace device, >= gprfwi_workspace_bytes(p, workspace_bytes, NULL) bytes, 256-B aligned;
 *            must stay untouched until the last gprfwi_adjoint for this handle
 *   traces   device [nshots][nt][nrec], overwritten
 * Errors: EINVAL, ECFL, EGEOM, ENOMEM, ECUDA. */
int gprfwi_forward(gprfwi_handle** h, const gprfwi_params* p,
                   const float* eps_r, const float* sigma, const float* wavelet,
                   const int32_t* src_zx, const int32_t* rec_zx,
                   void* workspace, size_t workspace_bytes,
                   float* traces, void* cuda_stream);

/* gprfwi_forward with a relative-permeability model (Table 1 `miu`; the paper's uH4 = 1/HA,
 * HA = m0*mr/dt).  mu_r: device [nz][pitch] fp32, > 0, read during this call only, or
 * NULL (= 1 everywhere, identical to gprfwi_forward).  Reading R22: the H component stored at
 * array index (j, i) -- Hx at (j+1/2, i), Hy at (j, i+1/2) -- takes mu_r[j][i], no averaging.  mu_r is a
 * model input only: gprfwi_adjoint (which uses the same model through the handle) still returns the
 * gradients with respect to eps_r and sigma.  Everything else as gprfwi_forward. */
int gprfwi_forward_mu(gprfwi_handle** h, const gprfwi_params* p,
                      const float* eps_r, const float* sigma, const float* mu_r,
                      const float* wavelet, const int32_t* src_zx, const int32_t* rec_zx,
                      void* workspace, size_t workspace_bytes, float* traces, void* cuda_stream);

/* Adjoint sweep + gradient, Algorithm 2: reverse time loop of {transpose of the
 * E update + E CPML, transpose of the H update + H CPML, adjoint source = residual sample n at the
 * receivers, gradient accumulation}, then the chain rule through Ca/Cb.
 * Result: grad_eps_r[j][i] = d/d eps_r[j][i] of sum_{s,n,r} residual*trace (= J^T residual), same
 * for sigma, on EVERY full-grid cell incl. CPML cells, summed over shots; no masking, no scaling
 * (0.5*||d_syn - d_obs||^2 is obtained with residual = d_syn - d_obs; Eq. (6)).
 * May be called several times (different residuals) after one forward.
 *   residual             device [nshots][nt][nrec]
 *   grad_eps_r, grad_sigma  device [nz][pitch], overwritten (pitch padding untouched)
 * Errors: EINVAL, ESTATE, ECUDA. */
int gprfwi_adjoint(gprfwi_handle* h, const float* residual,
                   float* grad_eps_r, float* grad_sigma, void* cuda_stream);

/* One misfit-gradient evaluation with HOST buffers (what a user without device arrays calls, and
 * what bench.py times as "e2e"): copies the models, wavelet and observed data to the device,
 * runs gprfwi_forward, forms residual = d_syn - d_obs on the device, runs gprfwi_adjoint, copies
 * traces and both gradients back and synchronises the stream.
 *   eps_r, sigma  host [nz][pitch]      wavelet host [nt] or [nshots][nt]
 *   d_obs         host [nshots][nt][nrec]
 *   workspace     device, >= gprfwi_workspace_bytes_host(p, workspace_bytes) bytes
 *   traces        host [nshots][nt][nrec] out (may be NULL)
 *   grad_eps_r, grad_sigma  host [nz][pitch] out
 *   misfit        host out: 0.5 * sum residual^2 (may be NULL)
 * Errors: as gprfwi_forward / gprfwi_adjoint. */
int gprfwi_gradient_host(const gprfwi_params* p,
                         const float* eps_r, const float* sigma, const float* wavelet,
                         const int32_t* src_zx, const int32_t* rec_zx, const float* d_obs,
                         void* workspace, size_t workspace_bytes,
                         float* traces, float* grad_eps_r, float* grad_sigma, double* misfit,
                         void* cuda_stream);

/* Workspace size for gprfwi_gradient_host: gprfwi_workspace_bytes plus room for the device copies
 * of the models, wavelet, traces, residual and gradients.  0 if invalid / nothing fits. */
size_t gprfwi_workspace_bytes_host(const gprfwi_params* p, size_t budget_bytes);

/* residual = d_syn - d_obs on the device (Eq. (6); MSELoss in the paper's script,
 * PAPER.md:226); n elements; if misfit != NULL (device double, must be zeroed by the caller)
 * 0.5*sum residual^2 is added to it. */
int gprfwi_residual(const float* d_syn, const float* d_obs, float* residual, size_t n,
                    double* misfit, void* cuda_stream);

/* Iteration epilogue: what the paper's script does between loss.backward() and
 * the next epoch plus the TV term of Algorithm 3. */
typedef struct {
  int32_t step;                 /* Adam step counter t >= 1 (bias correction 1 - beta^t)                 */
  float   lr_eps_r, lr_sigma;   /* one learning rate per parameter (Eqs. (14)-(15))   */
  float   beta1, beta2, adam_eps;
  int32_t tv_iters;             /* split-variable TV iterations of Algorithm 3; 0 = no TV term          */
  float   tv_rho, tv_lambda, tv_alpha;   /* tv_grad = alpha (X - s U), shrink threshold lambda / rho    */
  int32_t mask_rows;            /* gradient rows j < mask_rows are zeroed (near the sources,
                                   PAPER.md:229-233)                                                     */
  float   eps_r_min, sigma_min; /* clamps after the step                             */
} gprfwi_update_params;

/* Device scratch the epilogue needs for an nz x pitch plane: 7 planes + 256 B. */
size_t gprfwi_update_workspace_bytes(int32_t nz, int32_t pitch);

/* One optimiser step on the device, in place:
 *   for X in (eps_r, sigma):  g = grad_X (+ TV term of X, Algorithm 3; reading R20);
 *   g[j < mask_rows] = 0;  m = b1 m + (1-b1) g;  v = b2 v + (1-b2) g^2;
 *   X -= lr_X (m / (1-b1^t)) / (sqrt(v / (1-b2^t)) + adam_eps);  X = max(X, X_min).
 * eps_r, sigma, m_*, v_*  device [nz][pitch], updated in place (m, v: zero before the first step);
 * grad_eps_r, grad_sigma  device [nz][pitch]; the TV term is added to them in place.
 * Errors: EINVAL (null pointer, nz/nx < 2, pitch < nx, step < 1, tv_rho <= 0 with tv_iters > 0), ECUDA. */
int gprfwi_update(int32_t nz, int32_t nx, int32_t pitch, const gprfwi_update_params* u,
                  float* eps_r, float* sigma, float* grad_eps_r, float* grad_sigma,
                  float* m_eps_r, float* v_eps_r, float* m_sigma, float* v_sigma,
                  void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Multiscale (frequency-staged) inversion: zero-phase FIR along time applied to
 * traces or wavelets before a low-frequency stage.
 *   in, out  device [nseries][nt][nrec] (nrec = 1 for wavelets), out != in
 *   taps     device [ntaps], ntaps odd; out[n] = sum_k taps[k] in[n + k - (ntaps-1)/2], zero outside [0, nt)
 * The filter design (cut-off, window) is the caller's (gprfwi_lowpass_design gives the one of reading R21):
 * any symmetric taps give zero phase.
 * Errors: EINVAL (null pointer, in == out, nt/nrec/nseries < 1, ntaps even or < 1), ECUDA. */
int gprfwi_lowpass(const float* in, float* out, int32_t nseries, int32_t nt, int32_t nrec,
                   const float* taps, int32_t ntaps, void* cuda_stream);

/* gprfwi_update for callers that may not allocate and have no workspace to pass (code under CUDA-graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc): same arguments and result as gprfwi_update
 * minus the workspace.  The TV term's scratch (7 planes + one word) lives in a file-scope device array inside
 * the library, gprfwi_update_noalloc_max_bytes() = 7 * 2^20 * 4 + 256 bytes (29 360 384), which every GPU that
 * loads the library holds until the process exits; its device address is looked up once per device
 * (cudaGetSymbolAddress, with the caller's current device).  The call allocates nothing (no cudaMalloc /
 * cudaFree, no allocating library routine) and only enqueues on the stream.
 *   Limit: gprfwi_update_workspace_bytes(nz, pitch) <= gprfwi_update_noalloc_max_bytes(), i.e. about
 *   nz * pitch <= 2^20 cells (1024 x 1024); larger models return GPRFWI_ETOOBIG -- use gprfwi_update.
 *   All calls on a device share the array, which keeps the last call's contents; every call re-initialises
 *   what it reads.  Calls that OVERLAP on the GPU (different streams, no ordering between them) race on it:
 *   keep them on one stream or order them with events.
 *   The FIRST call on a device performs the address lookup (a runtime query, not a stream operation): callers
 *   that will run under CUDA-graph capture make one call on that device before they begin capturing.
 * Errors: as gprfwi_update, plus ETOOBIG; ECUDA if the symbol lookup fails. */
int gprfwi_update_noalloc(int32_t nz, int32_t nx, int32_t pitch, const gprfwi_update_params* u,
                          float* eps_r, float* sigma, float* grad_eps_r, float* grad_sigma,
                          float* m_eps_r, float* v_eps_r, float* m_sigma, float* v_sigma, void* cuda_stream);
size_t gprfwi_update_noalloc_max_bytes(void);

/* Taps of the stage filter for gprfwi_lowpass (the paper gives no design; DESIGN.md reading
 * R21): Hamming-windowed sinc with corner f_cut (Hz) at sampling interval dt (s), unit gain at DC, computed on
 * the HOST.  ntaps <= 0 picks 4/(f_cut dt) rounded up to odd.  taps: host [ntaps] or NULL (size query).
 * Returns the number of taps (> 0), or GPRFWI_EINVAL (non-positive dt / f_cut, even ntaps). */
int32_t gprfwi_lowpass_design(float dt, float f_cut, int32_t ntaps, float* taps);

/* Coarse grid of the early multiscale stages (reading R23): node-aligned 2:1
 * coarsening, coarse node (J, I) = fine node (2J, 2I), (nz+1)/2 x (nx+1)/2 coarse nodes.
 * gprfwi_restrict: coarse = full weighting of fine (tensor product of (1/4, 1/2, 1/4); a neighbour outside
 * the grid folds onto the centre).  gprfwi_prolong_add: fine += scale * bilinear interpolation of coarse
 * (how a coarse stage's model update returns to the fine model).
 *   fine    device [nz][pitch];  coarse  device [(nz+1)/2][pitch_coarse], pitch_coarse >= (nx+1)/2
 * Both enqueue on the stream.  Errors: EINVAL (null / aliased pointers, nz or nx < 3, pitches too small), ECUDA. */
int gprfwi_restrict(const float* fine, int32_t nz, int32_t nx, int32_t pitch, float* coarse, int32_t pitch_coarse,
                    void* cuda_stream);
int gprfwi_prolong_add(const float* coarse, int32_t pitch_coarse, float scale, float* fine, int32_t nz, int32_t nx,
                       int32_t pitch, void* cuda_stream);

/* Number of kernel launches enqueued by the last forward / adjoint on this handle. */
int64_t gprfwi_launch_count(const gprfwi_handle* h);

/* Plan in use by this handle. */
int gprfwi_get_plan(const gprfwi_handle* h, gprfwi_plan* plan);

/* Frees the host-side handle only (no device memory is owned by the library). */
void gprfwi_release(gprfwi_handle* h);

/* Static text for a status code; for GPRFWI_ECUDA the last CUDA error string seen. */
const char* gprfwi_strerror(int code);

/* Library version (major*10000 + minor*100 + patch). */
int gprfwi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GPRFWI_H */
