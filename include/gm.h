/* gm.h -- C ABI of libgm: the batched galaxy-profile chi^2 + gradient + update
 * hot path of arxiv 2404.07780 (Galmoss) on NVIDIA B200 (sm_100a).
 *
 * Citations "P:<line>" are lines of the paper text; "R:<id>" are the
 * readings of silent / garbled passages listed in DESIGN.md.
 *
 * What the library computes, per galaxy (Fig. 1):
 *   S   = sum of the PSF-convolved components, evaluated at pixel centres
 *         x = j + 0.5, y = H - 0.5 - i (R:G1) from the elliptical
 *         radius of Eq. 2-4 (R:G2) and the radial laws Eq. 1, 7, 9, 11,
 *         12, 13;
 *   M   = PSF (*) S + unconvolved components + sky (Eq. 16), true convolution,
 *         PSF centre (K-1)/2, zero fill outside the cutout, same size (R:C1);
 *   chi2 = sum_ij Omega_ij (D_ij - M_ij)^2 / sigma_ij^2            (Eq. 18);
 *   grad = d chi2 / d p for every entry of the parameter vector (the paper uses
 *         autograd; here the analytic adjoint: flipped-PSF correlation
 *         of G = -2 w (D - M), then a reduction against dS/dp);
 *   fit  = n_iter steps of Adam on u = p or log10 p with projection onto the
 *         parameter ranges (R:O1-O5).
 *
 * Conventions
 *   - Pointers marked "dev" are DEVICE pointers owned by the caller (e.g. torch
 *     allocations); pointers marked "host" are host pointers.  The library never
 *     frees or keeps a caller pointer past the call.
 *   - All images are row-major, [B,H,W] contiguous, float32; row 0 is the TOP row
 *     (largest y).  Angles are radians, lengths pixels, amplitudes intensities.
 *   - Device entry points are asynchronous on `cuda_stream` (a cudaStream_t; NULL =
 *     the legacy default stream), allocate nothing, and never synchronise (gm_init excepted),
 *     from the first call on.  Scratch comes from the caller: `workspace` (dev, 256-byte aligned) of at
 *     least gm_workspace_bytes(model, batch) bytes.
 *   - Process-wide state the library keeps (all of it derived, none of it observable in
 *     results): the nu_n interpolation table, filled once per device by a kernel on the
 *     stream of gm_init or of the first compute call (calls on other streams are made to
 *     wait for that kernel through an event until it has completed; gm_init itself returns
 *     only after the table is complete, so call it before capturing a CUDA graph -- a compute
 *     call that finds the table missing or still in flight on a stream that is being
 *     captured returns GM_EINVAL and enqueues nothing); a 59 KB constant-bank pool per PSF side that holds the
 *     paired taps of a batch-wide PSF (psf_stride == 0) for the duration of a call -- a
 *     region is filled by a device-to-device copy on the call's stream and handed back
 *     through an event on that stream, a later call on the same stream (same
 *     cudaStreamGetId, not merely the same handle) may take it over at once, and when no
 *     region is free (or the PSF is per galaxy) the taps go through shared memory, bit
 *     for bit the same result; gm_set_option(GM_OPT_CONST_TAPS, 0) forces that form.  The
 *     library reads no environment variable.  The *_host entry points take their device
 *     buffers from the device's stream-ordered memory pool and leave up to 8 GB of it
 *     cached for the next call.
 *   - Return value: GM_OK or a negative gm_status; nothing is launched when the
 *     arguments fail validation.  There is no CPU fallback: without a CUDA device
 *     every compute entry point returns GM_ECUDA.
 */
#ifndef GM_H_
#define GM_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GM_VERSION   300     /* major*10000 + minor*100 + patch */
#define GM_MAX_COMP  8       /* components per model                               */
#define GM_MAX_PAR   32      /* entries of the per-galaxy parameter vector          */
#define GM_MAX_K     41      /* PSF side (odd); the paper's PSFs are 41x41   */
#define GM_MAX_BATCHES 64    /* size buckets per gm_fit_multi call                  */

typedef enum {
  GM_OK = 0,
  GM_EINVAL = -1,    /* NULL pointer, even / oversize K, P or C over the maximum,
                        slot index out of range, non-positive size               */
  GM_ENOTSUP = -2,   /* valid request that this build has no kernel for          */
  GM_ECUDA = -3,     /* CUDA launch / runtime error (see gm_last_cuda_error)      */
  GM_EWORKSPACE = -4,/* workspace NULL, misaligned or too small                   */
  GM_ETOOLARGE = -5  /* problem larger than the built-in scratch of a *_static call */
} gm_status;

/* radial laws: Sec. 4.1, 4.2.1 - 4.2.6 */
typedef enum {
  GM_SERSIC = 0, GM_EXPDISK = 1, GM_FERRER = 2, GM_KING = 3,
  GM_GAUSSIAN = 4, GM_MOFFAT = 5, GM_SKY = 6
} gm_kind;

/* index of each quantity inside gm_component.slot[] */
enum { GM_SLOT_XC = 0, GM_SLOT_YC, GM_SLOT_THETA, GM_SLOT_Q, GM_SLOT_AMP,
       GM_SLOT_S0, GM_SLOT_S1, GM_SLOT_S2, GM_SLOT_BOX, GM_SLOT_M0, GM_NSLOT };

/* One summed component (host memory, POD).  slot[k] is the index, inside the
 * galaxy's parameter vector, of the k-th quantity, or -1 when unused:
 *   Sersic   amp=Ie  s0=re    s1=n            Eq. 1
 *   ExpDisk  amp=I0  s0=rs                    Eq. 7
 *   Ferrer   amp=I0  s0=r_out s1=a   s2=b     Eq. 9   (0 for r >= r_out)
 *   King     amp=I0  s0=rc    s1=rt  s2=alpha Eq. 11  (0 for r >= rt, R:K1)
 *   Gaussian amp=I0  s0=FWHM                  Eq. 12  (FWHM = 2 sqrt(2 ln 2) sigma, R:F1)
 *   Moffat   amp=I0  s0=FWHM  s1=n            Eq. 13-14
 *   Sky      amp=I_sky                        Eq. 16  (never convolved)
 * Unused q means 1 (circular), unused theta means 0, unused box means B = 0.
 * Two components naming the same index are TIED: their gradients add.
 * convolve = 1: the component goes through the PSF; 0: added after it.
 * box: the boxiness B of the generalised ellipse, Eq. 2:
 *   r = (|u|^(B+2) + |v/q|^(B+2))^(1/(B+2)), B > -2; its gradient entry is d chi2 / dB.
 * m0: when this slot is used the amplitude slot holds a MAGNITUDE m and the slot itself
 *   the zero point m0 (the paper's gm.p(m, M0=...)); the intensity is
 *     Sersic  Ie = r_box nu^(2n) F / (2 pi q re^2 n Gamma(2n) e^nu)          Eq. 5
 *     ExpDisk I0 = r_box F / (2 pi q rs^2)                                     Eq. 8
 *     Ferrer  I0 = r_box F / (pi q r_out^2 a beta(a, 1 + 2/(2-b)))             Eq. 10
 *     Moffat  I0 = r_box (n-1) F / (pi q rd^2), rd of Eq. 14                   Eq. 15
 *   with F = 10^(-0.4 (m - m0)) and r_box = pi (2+B) / (2 beta(1/(2+B), 1/(2+B))) (Eq. 6),
 *   evaluated in fp64 per galaxy; the gradient is then with respect to m (and m0, q, the
 *   shape slots and B gain the terms through the amplitude).  m0 is normally held fixed
 *   through gm_fit_opts.free_mask.  King, Gaussian and Sky have no magnitude relation in
 *   the paper: a used m0 slot there is GM_EINVAL. */
typedef struct {
  int32_t kind;
  int32_t convolve;
  int32_t slot[GM_NSLOT];
} gm_component;

typedef struct {
  int32_t n_comp;              /* 1..GM_MAX_COMP                                  */
  int32_t n_par;               /* P, 1..GM_MAX_PAR                                */
  const gm_component* comp;    /* host [n_comp]                                   */
} gm_model;

/* One batch of equally sized cutouts.  Mixed sizes = one gm_batch
 * per size, called one after the other (or on different streams). */
typedef struct {
  int32_t B, H, W, K;          /* K odd, 1..GM_MAX_K                               */
  const float*   data;         /* dev [B,H,W]  D_ij          (NULL for gm_render)  */
  const float*   sigma;        /* dev [B,H,W]  sigma_ij > 0 wherever mask != 0     */
  const uint8_t* mask;         /* dev [B,H,W]  Omega: 1 used, 0 ignored (R:X1);
                                  NULL = every pixel used                          */
  const float*   psf;          /* dev [B,K,K] or [K,K]; used as given (R:C1)       */
  int64_t        psf_stride;   /* elements between galaxies; 0 = one shared PSF    */
} gm_batch;

/* Update rule (R:O1-O5).  For every free parameter k, per galaxy, t = 1..n_iter:
 *   u = p or log10 p;  g = dchi2/dp * dp/du
 *   m <- beta1 m + (1-beta1) g ;  s <- beta2 s + (1-beta2) g^2
 *   u <- u - lr[k] lr_decay^(t-1) [m/(1-beta1^t)] / (sqrt(s/(1-beta2^t)) + eps)
 *   u <- min(max(u, T(lo[k])), T(hi[k]))                         (projection)
 * A galaxy stops early once |chi2_t - chi2_(t-1)| <= tol chi2_t held for `patience`
 * consecutive iterations (tol <= 0: never).  All arrays are HOST arrays of n_par. */
typedef struct {
  int32_t n_iter;
  float   beta1, beta2, eps;
  float   lr_decay;
  const float*   lr;
  const float*   lo;
  const float*   hi;           /* +-INFINITY allowed                               */
  const uint8_t* log10_space;  /* 1: optimise u = log10 p; NULL = all 0    */
  const uint8_t* free_mask;    /* 0: parameter held fixed;    NULL = all free      */
  float   tol;
  int32_t patience;
} gm_fit_opts;

/* per-galaxy status written by gm_fit */
enum { GM_FIT_OK = 0, GM_FIT_CONVERGED = 1, GM_FIT_NONFINITE = 2 };

/* ---- device entry points (asynchronous) ---------------------------------- */

/* Optional: build the per-device tables on `cuda_stream` now instead of inside the first
 * compute call.  Idempotent.  The one device entry point that WAITS: it returns after its
 * (microseconds long) table kernel has completed, so a stream capture may begin right after it;
 * needed only before CUDA graph capture.  GM_EINVAL when `cuda_stream` is already capturing. */
int gm_init(void* cuda_stream);

/* Process-wide switches, for tests and measurements (value 0 / 1, default 1 each):
 *   GM_OPT_FUSED       cutouts up to 128 x 128 take the single fused kernel; 0: tile kernels
 *   GM_OPT_CONST_TAPS  a batch-wide PSF is read from the constant bank; 0: shared memory
 *   GM_OPT_TENSOR      with a PSF of more than 9 x 9 taps both convolutions run on the
 *                      tensor cores (fp16 hi/lo split of the fp32 operands, see gm_conv): square cutouts
 *                      of 64 (shared PSF), 96 or 128 pixels in one fused kernel, cutouts above 128 pixels
 *                      with W a multiple of 4 in super-tiles; every other shape and 0: the FP32 (FFMA2)
 *                      convolution
 * The first two give bit for bit the same results; GM_OPT_TENSOR changes the convolution arithmetic:
 * its error is ABSOLUTE, a few 1e-7 of the cutout's brightest pixel (one power-of-two scale per cutout,
 * see gm_conv), i.e. a few 1e-6 relative on pixels within two decades of the maximum and no significant
 * bits below about 1e-7 of it; inside every documented tolerance.  gm_set_option returns
 * GM_EINVAL for an unknown option, gm_get_option -1. */
enum { GM_OPT_FUSED = 0, GM_OPT_CONST_TAPS = 1, GM_OPT_TENSOR = 2, GM_OPT_COUNT_ = 3 };
int gm_set_option(int option, int value);
int gm_get_option(int option);

/* Bytes of device scratch gm_render / gm_loss_grad / gm_fit need for this model
 * and batch shape (B, H, W, K, psf_stride -- one PSF or B of them -- and the model are
 * read; the pointers are not).  0 on invalid input.  Sized by shape alone, for whichever engine may run:
 * with one PSF per galaxy (psf_stride != 0) it holds the tap tables of every galaxy for both engines
 * (forward and adjoint each), which dominates the total -- 0.53 MB per galaxy at K = 41 (0.27 MB at
 * K = 25), 4.4 GB for 8,289 galaxies; a batch-wide PSF costs one set.  A call fills only the tables of the engine it runs. */
size_t gm_workspace_bytes(const gm_model* model, const gm_batch* batch);

/* Render the model image M (App. C "initial_model").
 * params: dev [B,P].  model_out: dev [B,H,W].  batch->data/sigma/mask ignored. */
int gm_render(const gm_model* model, const gm_batch* batch, const float* params,
              float* model_out, void* workspace, size_t workspace_bytes,
              void* cuda_stream);

/* chi^2 (Eq. 18) and its gradient with respect to the PHYSICAL parameters.
 * chi2: dev [B].  grad: dev [B,P] (NULL = not wanted).
 * jtj: dev [B,P,P], jtr: dev [B,P] = J^T W J and J^T W (D-M) with J = dM/dp and
 * W = Omega / sigma^2, or NULL.  jtr costs nothing extra (it is -grad/2);
 * jtj runs P more forward convolutions (one Jacobian column each) and needs a
 * workspace of gm_uncertainty_workspace_bytes(), else GM_EWORKSPACE. */
int gm_loss_grad(const gm_model* model, const gm_batch* batch, const float* params,
                 float* chi2, float* grad, float* jtj, float* jtr,
                 void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Fixed-iteration batched fit.  params: dev [B,P], in/out.
 * chi2_out: dev [B], chi^2 AT the returned parameters.  iters_used: dev [B], the number of
 * the last iteration whose chi^2 was finite and acted upon (= updates applied for
 * GM_FIT_OK and GM_FIT_CONVERGED; for GM_FIT_NONFINITE at iteration t it is t - 1 while
 * the returned parameters are those that entered iteration t - 1, i.e. carry t - 2
 * updates), or NULL.  status: dev [B] GM_FIT_*, or NULL.
 * A galaxy whose chi^2 turns non-finite gets GM_FIT_NONFINITE and keeps the last
 * parameters that had a finite chi^2. */
int gm_fit(const gm_model* model, const gm_batch* batch, float* params,
           const gm_fit_opts* opts, float* chi2_out, int32_t* iters_used,
           int32_t* status, void* workspace, size_t workspace_bytes,
           void* cuda_stream);

/* The same fit for several batches of different cutout size at once (the paper's sample
 * mixes sizes; BASELINE config 2 has five).  Entry i of every array argument
 * belongs to batches[i]: params[i] dev [B_i,P] in/out, opts[i], chi2_out[i] dev [B_i],
 * iters_used[i] / status[i] dev [B_i] (the array or single entries may be NULL),
 * workspaces[i] of workspace_bytes[i] >= gm_workspace_bytes(model, &batches[i]), and
 * cuda_streams[i], the stream batch i is enqueued on.  All arrays are HOST arrays of
 * n_batches (1..GM_MAX_BATCHES).  Iteration t of every batch is enqueued before
 * iteration t+1 of any; with distinct streams the batches run concurrently, so the
 * SMs one batch leaves idle once most of its galaxies stopped early (R:O5) take
 * another batch's galaxies.  Results are identical to calling gm_fit per batch: no
 * batch reads another's data.  Ordering against the caller's other work is the
 * caller's (events on the given streams); nothing is launched if any entry fails
 * validation. */
int gm_fit_multi(const gm_model* model, int32_t n_batches, const gm_batch* batches,
                 float* const* params, const gm_fit_opts* opts, float* const* chi2_out,
                 int32_t* const* iters_used, int32_t* const* status,
                 void* const* workspaces, const size_t* workspace_bytes,
                 void* const* cuda_streams);

/* Covariance-matrix uncertainties (Sec. 5.2):
 *   sigma_p = sqrt(diag[(J^T W J)^-1]),  J = dM/dp at `params`,  W = Omega / sigma^2,
 * over the FREE parameters (free_mask: host [P], 0 = held fixed and left out of the
 * matrix; NULL = all free); fixed parameters get sigma_p = 0.  J^T W J is accumulated and
 * inverted in fp64 (Jacobi scaling + Cholesky).  sigma_p: dev [B,P].  jtj: dev [B,P,P]
 * full matrix as float, or NULL.  status: dev [B], 0 ok, 1 matrix not positive definite
 * or not finite (that galaxy's sigma_p is NaN), or NULL.  batch->data is not read.
 * Workspace: gm_uncertainty_workspace_bytes(model, batch). */
size_t gm_uncertainty_workspace_bytes(const gm_model* model, const gm_batch* batch);
int gm_uncertainty(const gm_model* model, const gm_batch* batch, const float* params,
                   const uint8_t* free_mask, float* sigma_p, float* jtj, int32_t* status,
                   void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Bootstrap uncertainties (Sec. 5.2): "resampling with replacement each galaxy
 * image multiple times (typically 100 iterations) and refitting"; the uncertainty is
 * sigma^2 = (1/M) sum_i (m_i - mean)^2 over the M refits (population variance).
 * Reading B1: one resample draws n_used pixel positions uniformly with replacement from
 * the n_used pixels of the galaxy with mask != 0 (row-major order); c_ij = number of
 * times pixel (i,j) was drawn, and the refit minimises sum c_ij (D-M)^2 / sigma^2.
 * Draws are counter based, so a result does not depend on batching or timing:
 *   mix(z): z = (z ^ z>>30) * 0xBF58476D1CE4E5B9; z = (z ^ z>>27) * 0x94D049BB133111EB;
 *           z ^ z>>31                                    (splitmix64 finaliser, 64-bit wrap)
 *   z(d) = mix(mix(mix(seed ^ (id * 0x9E3779B97F4A7C15)) + r) + d),  d = 0 .. n_used-1
 *   k(d) = ((z >> 32) * n_used) >> 32  = index of the drawn pixel among the used ones
 * with id = id_offset + index of the galaxy in the batch and r the resample index. */
typedef struct {
  int32_t  n_resample;         /* M, 1..GM_MAX_RESAMPLE                              */
  uint64_t seed;
  uint64_t id_offset;          /* identifier of the batch's first galaxy             */
} gm_boot_opts;
#define GM_MAX_RESAMPLE 4096

/* Multiplicities of resample r of every galaxy: counts dev [B,H,W] int32 (0 on masked
 * pixels; sums to n_used per galaxy).  Only B, H, W and mask of `batch` are read.
 * workspace: dev, 256-byte aligned, at least 4*B*(H*W + 1) + 512 bytes. */
int gm_bootstrap_counts(const gm_batch* batch, const gm_boot_opts* boot, int32_t r,
                        int32_t* counts, void* workspace, size_t workspace_bytes,
                        void* cuda_stream);

/* gm_bootstrap_counts for callers that CANNOT ALLOCATE device memory and so have no workspace to
 * pass: code that runs inside a host application which hands it a fixed set of buffers (a plug-in,
 * a pipeline stage), services that fix their memory plan at start-up (real-time, embedded, or
 * running beside a framework that has claimed the whole GPU), and threads for which an allocation
 * could stall or deadlock (another library's callback, a lock the allocator also wants).  Same
 * arguments as gm_bootstrap_counts minus the workspace, same kernels, bit for bit the same counts;
 * the caller still provides the mask (input) and `counts` (output, dev [B,H,W] int32).
 *   - Scratch is an array compiled into the library (`static __device__`, 256-byte aligned,
 *     4 * (GM_STATIC_MAX_PIXELS + GM_STATIC_MAX_B) bytes = about 4.02 MB).  Every GPU on which the
 *     library's device code is loaded holds it until the process exits, used or not.
 *   - Limits: B <= GM_STATIC_MAX_B and B * H * W <= GM_STATIC_MAX_PIXELS (e.g. 64 cutouts of
 *     128 x 128, 16 of 256 x 256).  Anything larger returns GM_ETOOLARGE before any launch or
 *     write; split the batch (id_offset keeps the draws of a galaxy independent of the split) or
 *     call gm_bootstrap_counts with a workspace.
 *   - The call itself makes no cudaMalloc / cudaFree / pool allocation and calls no library routine
 *     that does: two kernels and one cudaMemsetAsync of `counts` on `cuda_stream`, asynchronous.
 *   - The first call on each device looks up the array's device address (cudaGetSymbolAddress, with
 *     that device current; the calling thread's current device is the one used) and keeps it.  Make
 *     that first call during set-up, before any stream capture begins on that device.
 *   - All calls on a device share the one array and it keeps what the last call wrote.  Nothing in it
 *     has to start at zero (each call rewrites every entry it later reads; `counts` is cleared by
 *     the call), but two calls whose kernels may overlap on the GPU -- different streams without an
 *     event between them, or several host threads -- RACE on it and give wrong counts.  Issue
 *     them on one stream, or order them yourself.
 * Errors: GM_EINVAL (NULL pointer, r < 0, non-positive size), GM_ETOOLARGE, GM_ECUDA,
 * GM_ENOTSUP (device ordinal >= 64). */
#define GM_STATIC_MAX_PIXELS (1 << 20)   /* B * H * W of one gm_bootstrap_counts_static call  */
#define GM_STATIC_MAX_B      4096        /* galaxies of one gm_bootstrap_counts_static call    */
int gm_bootstrap_counts_static(const gm_batch* batch, const gm_boot_opts* boot, int32_t r,
                               int32_t* counts, void* cuda_stream);

/* M refits, every one started from `params` (dev [B,P], not modified) with `opts`.
 * sigma_boot: dev [B,P].  mean: dev [B,P] or NULL.  samples: dev [M,B,P] fitted
 * parameters of every refit, or NULL.  Fixed parameters get sigma_boot = 0.
 * The mean and variance are accumulated in fp64 in resample order.
 * Workspace: gm_bootstrap_workspace_bytes(model, batch, M). */
size_t gm_bootstrap_workspace_bytes(const gm_model* model, const gm_batch* batch, int32_t n_resample);
int gm_bootstrap(const gm_model* model, const gm_batch* batch, const float* params,
                 const gm_fit_opts* opts, const gm_boot_opts* boot, float* sigma_boot,
                 float* mean, float* samples, void* workspace, size_t workspace_bytes,
                 void* cuda_stream);

/* The PSF convolution on its own, with a choice of engine (the paper leaves the
 * convolution algorithm open):  out = PSF (*) in, true convolution, PSF centre (K-1)/2, zero
 * fill outside the cutout, same size (R:C1); adjoint != 0: the correlation with the same PSF (R:C2).
 *   GM_CONV_FFMA2   the FP32 direct convolution of the fit path (packed FFMA2 loop); any H, W, odd
 *                   K <= GM_MAX_K
 *   GM_CONV_TENSOR  tcgen05 tensor cores: every fp32 operand is scaled by an exact power of two and
 *                   split into two fp16 halves (22 bits of the SCALED value: one scale per cutout taken
 *                   from its largest |pixel|, so a pixel 2^-k below the maximum keeps 22 - k bits and anything
 *                   below 2^-24 of the scaled range is flushed to zero), three MMAs per product accumulate
 *                   hi*hi + lo*hi + hi*lo in fp32 in tensor memory (the dropped lo*lo term is 2^-22
 *                   relative); Toeplitz band blocks of the PSF stream through shared memory.  H = W = 128
 *                   only (GM_ENOTSUP otherwise); inputs must be finite.  batch->data and out must be
 *                   16-byte aligned (the kernel moves 128-bit rows): GM_EINVAL otherwise, nothing launched;
 *                   GM_CONV_FFMA2 takes any 4-byte aligned view.
 * batch: B, H, W, K, psf, psf_stride are read and batch->data is the INPUT image, dev [B,H,W].
 * out: dev [B,H,W].  workspace: gm_conv_workspace_bytes(engine, batch).  Asynchronous. */
enum { GM_CONV_FFMA2 = 0, GM_CONV_TENSOR = 1 };
size_t gm_conv_workspace_bytes(int engine, const gm_batch* batch);
int gm_conv(int engine, int adjoint, const gm_batch* batch, float* out, void* workspace,
            size_t workspace_bytes, void* cuda_stream);

/* ---- host-buffer entry points (synchronous, end to end) -------------------- */
/* Same operations with every pointer of `batch` and every array argument in HOST
 * memory (pinned memory makes the copies faster, pageable works).  The call
 * allocates device memory, copies the inputs in, runs the device entry point,
 * copies the results out, frees, and returns after the device is idle. */
int gm_render_host(const gm_model* model, const gm_batch* host_batch,
                   const float* params, float* model_out);
int gm_loss_grad_host(const gm_model* model, const gm_batch* host_batch,
                      const float* params, float* chi2, float* grad);
int gm_fit_host(const gm_model* model, const gm_batch* host_batch, float* params,
                const gm_fit_opts* opts, float* chi2_out, int32_t* iters_used,
                int32_t* status);

/* gm_fit_multi with host buffers: every batch is staged on its own stream, fitted
 * concurrently and copied back; returns after all of them are idle. */
int gm_fit_multi_host(const gm_model* model, int32_t n_batches, const gm_batch* host_batches,
                      float* const* params, const gm_fit_opts* opts, float* const* chi2_out,
                      int32_t* const* iters_used, int32_t* const* status);

/* Extended chi^2 log-likelihood, Eq. 17:
 *   ln L = -(k/2) ln 2 - ln Gamma(k/2) + (k/2 - 1) ln chi2 - chi2/2,
 * k = n_used[b] - n_free: "the number of pixels ... not included in the mask" minus "the number of model
 * fit parameters".  A per-galaxy scalar after a fit, so a HOST helper (fp64, no CUDA call):
 * chi2 host [B] (as copied back from gm_fit / gm_loss_grad), n_used host [B], loglike host [B].
 * Entries with k < 1 or chi2 <= 0 or non-finite chi2 get NaN.  GM_EINVAL for NULL / B < 1 / n_free < 0. */
int gm_loglike(int32_t B, const float* chi2, const int32_t* n_used, int32_t n_free, double* loglike);

/* ---- misc ------------------------------------------------------------------ */
const char* gm_strerror(int status);
int         gm_version(void);
/* cudaError_t of the most recent GM_ECUDA on this thread (0 = none) and its text */
int         gm_last_cuda_error(void);
const char* gm_last_cuda_error_string(void);
/* number of kernels launched by this thread's last device entry point; lets a
 * caller (bench.py "gpu_launches") count launches without a profiler */
int64_t     gm_last_launch_count(void);


/* ---- measurement hooks (used by bench.py for the roofline line) ---------------- */
/* While enabled, every launch of the heavy kernels is bracketed by CUDA events
 * recorded on the launching stream (at most 8192 launches are kept):
 *   [GM_PROF_FORWARD]     k_forward   FFMA2 tile kernel (render + PSF convolution + residual)
 *   [GM_PROF_BACKWARD]    k_backward  FFMA2 tile kernel (adjoint convolution + gradient sums)
 *   [GM_PROF_FUSED]       k_fused     FFMA2, all of the above for cutouts that fit one CTA
 *   [GM_PROF_TC_FORWARD]  k_tc_tile   tensor-core forward kernel of cutouts above 128 px
 *   [GM_PROF_TC_BACKWARD] k_tc_tile   tensor-core backward kernel
 *   [GM_PROF_TC_FUSED]    k_tc_fused  tensor cores, 64 / 96 / 128 px cutouts in one launch
 * gm_profile_read waits for them, returns the summed durations in milliseconds and
 * the launch counts per kind, and clears the list.  Off by default; enabling or
 * disabling also clears it. */
int gm_profile_enable(int on);
enum { GM_PROF_FORWARD = 0, GM_PROF_BACKWARD = 1, GM_PROF_FUSED = 2, GM_PROF_TC_FORWARD = 3, GM_PROF_TC_BACKWARD = 4,
       GM_PROF_TC_FUSED = 5, GM_PROF_KINDS = 6 };
int gm_profile_read(double* ms /* host [GM_PROF_KINDS] */, int64_t* count /* host [GM_PROF_KINDS] */);

/* Phase trace of k_tc_fused (the tensor-core kernel of 64 / 96 / 128 px cutouts).  While `device_buf`
 * (device memory, GM_TRACE_ROLES * GM_TRACE_CAP uint64, zeroed by the caller) is set, CTA 0 of every
 * launch appends one record per phase boundary to the list of its role, from the start of the list:
 * record = (tag << 56 | item << 48 | clock64 & (2^48 - 1)); roles: 0 helper warps (render, drain,
 * residual, gradient), 1 MMA issue (first window row ready / last MMA issued, per convolution),
 * 2 unused.  Tags in gm_tc_fused.cuh (TR_*).  nullptr switches it off (default).  Not thread safe
 * against concurrent launches; a measurement hook, one launch at a time. */
#define GM_TRACE_ROLES 3
#define GM_TRACE_CAP   2048
int gm_trace_set(unsigned long long* device_buf);

/* The FP32 peak the roofline is quoted against, MEASURED: a kernel of nothing but
 * independent packed FP32 multiply-adds (fma.rn.f32x2, the instruction of the convolution
 * loops), three 256-thread CTAs per SM in one wave, timed with CUDA events on `cuda_stream` over
 * `repeats` launches after one warm-up launch.  Synchronous (waits for its own events).
 * tflops: host, 2 flop per multiply-add. */
int gm_measure_fp32_peak(int repeats, double* tflops, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* GM_H_ */
