/* pty.h -- C ABI of the B200-native (sm_100a) multislice-ptychography hot path.
 *
 * What it computes: the batched mixed-state multislice forward model of PtyRAD
 * (arxiv 2505.07814; PAPER.md = /root/reference/PAPER.md), an amplitude loss and the
 * exact hand-written adjoint over one minibatch of B scan positions:
 *
 *   r_b = floor(p_b + 0.5),  Delta_b = p_b - r_b                  (footnote 3 :122)
 *   psi_0^(m) = F^-1[ exp(-2 pi i k.Delta_b) F[P^(m)] ]           (shift operator)
 *   for s = 1..Nz:  phi_s = O[s, r_b : r_b+N] * psi_{s-1};
 *                   psi_s = F^-1[ M F[phi_s] ]  for s < Nz         (Eq. 3)
 *   M(k) = exp(-i pi lambda |k|^2 dz + 2 pi i dz (k_x tan th_x + k_y tan th_y))   (Eq. 4, :89)
 *   I_b(k) = sum_m |F[phi_Nz^(m)](k)|^2                           (Eq. 2)
 *   L = sum_b sum_k (sqrt(I_b(k)) - a_b(k))^2                     (Eq. 5 with p = 1/2, :126-131;
 *                                                                  plain sum, R13)
 * F is the unitary 2-D DFT with kernel exp(-2 pi i k.r); k = fftfreq(N)/dx in 1/Angstrom.
 * Gradients use g = dL/dRe + i dL/dIm for complex arrays (what torch.autograd returns);
 * g_positions = dL/dDelta (the integer crop origin is a constant).
 *
 * Layouts.  Every array is dense, row-major, C order, exactly as named below; complex means
 * interleaved (re, im) float32 ("c64").  2-D arrays are (y, x); spectra / detector data have
 * DC at index [0][0] (unshifted FFT order).  positions[b] = (p_y, p_x) in PIXELS = the top-left
 * corner of the N x N crop in object coordinates.  tilt = (theta_y, theta_x) in RADIANS.
 *
 * Alignment.  object, probe and every complex gradient: 8 bytes; meas_amp: 16 bytes; positions,
 * tilt and the real gradients: 4 bytes (violations return PTY_ERR_INVALID_ARG).  The Adam arrays
 * (theta, grad, m, v) may have any 4-byte alignment: the update uses 16-byte vectors when all four
 * are 16-byte aligned and a scalar path otherwise (e.g. a positions[lo:hi] shard view).
 *
 * Devices.  A plan belongs to the device given to pty_create.  Every entry point switches to that
 * device for its own duration and restores the caller's current device before it returns.
 *
 * Memory.  Unless a parameter says "host", every pointer is a DEVICE pointer on the plan's
 * device.  The caller owns every buffer including the workspace and the Adam moments; the
 * library allocates no device memory, frees nothing of the caller's and keeps no caller pointer
 * past a call (except the workspace given to pty_create).
 *
 * Execution.  Everything is enqueued on the given stream; no call synchronises except
 * pty_status, pty_loss_terms, pty_profile_read and the *_host entry points.  The enqueue-only
 * calls make no allocation and no synchronisation, so a sequence of them on fixed pointers can
 * be recorded once with CUDA stream capture and replayed as a graph (launch-bound small
 * configurations; tests/test_gpu_features.py).  One plan per stream; a plan is not thread-safe.
 *
 * Errors.  Every function returns PTY_OK (0) or a negative PTY_ERR_* code; the text of the last
 * error of a plan is available from pty_last_error.  No C++ exception crosses this boundary.
 * Scan positions are device data: a crop that would leave the object is clamped into it and a
 * sticky device flag is raised, reported by pty_status as PTY_ERR_BOUNDS.
 * There is no CPU fallback of any kind.
 */
#ifndef PTY_H
#define PTY_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PTY_OK                 0
#define PTY_ERR_INVALID_ARG   (-1)  /* null pointer, B < 0 or B > Bmax, bad dims            */
#define PTY_ERR_UNSUPPORTED   (-2)  /* N not in {64,128,256}, window larger than the object   */
#define PTY_ERR_WORKSPACE     (-3)  /* workspace null, misaligned (256 B) or too small        */
#define PTY_ERR_CUDA          (-4)  /* a CUDA runtime call failed; see pty_last_error         */
#define PTY_ERR_BOUNDS        (-5)  /* pty_status: some crop left the object and was clamped  */
#define PTY_ERR_ZERO_DATA     (-6)  /* pty_status: a loss-mode-1 call saw a minibatch whose measurements are all
                                       zero; Eq. 5-7 divide by their mean, so the affected terms and their
                                       gradients were set to 0 instead of inf / NaN (sticky flag bit 2)      */

/* pty_dims.flags */
#define PTY_FLAG_SPECTRA       1    /* keep propagated spectra so that g_dz can be produced even
                                       when tilt_mode == 0 (implied by tilt_mode != 0)        */
#define PTY_FLAG_STEP          2    /* reserve gradient buffers in the workspace: pty_step     */
#define PTY_FLAG_HOST          4    /* reserve device staging buffers: pty_grad_host           */
#define PTY_FLAG_AMP_PHASE     8    /* reserve the composed object, its gradient and the patch
                                       coverage map: pty_*_ap (amplitude / phase object)       */
#define PTY_FLAG_TMA_OBJECT   16    /* N = 128, forward kernel: stage the first 12 rows of every role's
                                       object patch column with TMA (cp.async.bulk.tensor into a shared-
                                       memory ring) instead of fetching all rows through registers; same
                                       results.  Needs an even W and a 16-byte aligned `object`, otherwise
                                       the register path runs.  Off by default: measured slower on c4
                                                                                  */
#define PTY_FLAG_PAIR_SUM     32    /* N = 128, adjoint kernel: sum the g_object contributions of the two
                                       probe modes a CTA holds (two groups, one position) in a shared-memory
                                       ring before the one global reduction per pixel -- the on-chip part of
                                       the crop's adjoint: half the atomics,
                                       same results up to the summation order.  Needs an even M
                                       (otherwise a CTA's two items can belong to two positions or two object
                                       states and the per-item reductions run).  Off by default: the ring couples the two
                                       groups' phases and is measured slower      */

/* pty_backward flags */
#define PTY_BWD_ACCUMULATE     1    /* add into the gradient outputs instead of overwriting    */
#define PTY_BWD_REUSE_FORWARD  4    /* the caller asserts that object, probe, positions, tilt and
                                       meas_amp are BIT-UNCHANGED since the pty_forward_loss call
                                       made just before on this plan and stream with the same
                                       pointers and B: its saved waves are reused.  Without this
                                       flag pty_backward always runs the forward itself.        */

typedef struct pty_plan pty_plan;   /* opaque, host side */

typedef struct pty_dims {
    int32_t Nz, H, W;     /* object [Nz][H][W] c64                                            */
    int32_t M, N;         /* probe  [M][N][N] c64; N in {64, 128, 256}; N <= H, N <= W        */
    int32_t Bmax;         /* largest minibatch any call will pass                             */
    float   dz, lambda, dx;   /* slice separation, wavelength, pixel size; Angstrom (Eq. 4)   */
    int32_t tilt_mode;    /* 0: no tilt (tilt pointers ignored); 1: one global tilt [2];
                             2: one tilt per position [B][2]                                  */
    int32_t flags;        /* PTY_FLAG_*                                                       */
    int32_t n_obj;        /* mixed object states N (Eq. 2): object and g_object are
                             [n_obj][Nz][H][W], I = sum_m sum_n |F psi^(m)(n)|^2; 0 or 1 = one state    */
} pty_dims;

/* The paper's loss family (R27-R30).  mode 0 (default): the plain amplitude sum
 *   L = sum_b sum_k (sqrt(I) - a)^2 of the north_star.  mode 1: Eq. 9,
 *   L_total = w_gaussian L_Gaussian(Eq. 5, p = 1/2) + w_poisson L_Poisson(Eq. 6, p = 1, eps) + w_pacbed L_PACBED
 *   (Eq. 7, p = 1/2) + w_sparse L_sparse(Eq. 8, p = 1; only the amplitude / phase entry points know the phase),
 *   every average taken over the detector and the minibatch of the call.  In both modes loss_per_pos[b] is the
 *   plain sum of position b, and every gradient is that of the scalar written to `loss`. */
typedef struct pty_loss {
    int32_t mode;
    float w_gaussian, w_poisson, w_pacbed, w_sparse;
    float eps;            /* Poisson epsilon, 1e-6 in the paper                         */
} pty_loss;

/* Adam for the amplitude / phase parameterisation (separate learning rates). */
typedef struct pty_adam_ap {
    float lr_amp, lr_phase, lr_probe, lr_positions, lr_tilt;
    float beta1, beta2, eps;
    int32_t t;
} pty_adam_ap;
typedef struct pty_adam_state_ap {
    float *m_amp, *v_amp, *m_phase, *v_phase;        /* [n_obj*Nz*H*W] each */
    float *m_probe, *v_probe, *m_positions, *v_positions, *m_tilt, *v_tilt;
} pty_adam_state_ap;

/* Per-iteration constraints of the paper's reconstructions (R31). */
typedef struct pty_constraints {
    int32_t ortho_probe;      /* 1: replace the probe modes by the orthogonal modes of the same mixed state,
                                 ordered by decreasing power (Thibault & Menzel 2013)                  */
    float   sigma_z;          /* > 0: r_z filter, Eq. 13 -- Gaussian blur along depth (in slices) of amp and
                                 phase; taps exp(-j^2 / 2 sigma_z^2), |j| <= max(1, ceil(2 sigma_z)) <= 8,
                                 normalised, end slices replicated                                     */
    int32_t phase_positive;   /* 1: phase = max(phase, 0)                                               */
    int32_t clamp_amp;        /* 1: amp = min(max(amp, amp_min), amp_max)                               */
    float   amp_min, amp_max;
} pty_constraints;

/* Adam hyper-parameters (Kingma & Ba with bias correction; R20).
 * A learning rate of 0 freezes that parameter group (its moments are left untouched). */
typedef struct pty_adam {
    float lr_object, lr_probe, lr_positions, lr_tilt;
    float beta1, beta2, eps;
    int32_t t;            /* 1-based step number used for the bias correction                 */
} pty_adam;

/* Adam moments, device memory owned by the caller, float32, same element order as the
 * parameter viewed as reals (complex = 2 floats).  A group with lr == 0 may pass NULL. */
typedef struct pty_adam_state {
    float *m_object,    *v_object;     /* [Nz*H*W*2] */
    float *m_probe,     *v_probe;      /* [M*N*N*2]  */
    float *m_positions, *v_positions;  /* [B*2]      */
    float *m_tilt,      *v_tilt;       /* [2] (tilt_mode 1) or [B*2] (tilt_mode 2) */
} pty_adam_state;

/* Bytes of device workspace a plan with these dims needs (a multiple of 256). */
int pty_workspace_bytes(const pty_dims* dims, size_t* out_bytes);

/* Create a plan on `device` using the caller's device workspace (256-byte aligned, at least
 * pty_workspace_bytes).  The workspace must stay alive and untouched until pty_destroy. */
int pty_create(pty_plan** out_plan, const pty_dims* dims, void* workspace, size_t workspace_bytes,
               int device);
int pty_destroy(pty_plan* plan);

/* Forward model + loss for one minibatch (PAPER.md:58-90 Eq. 1-4, :126-131 Eq. 5).
 *   object [Nz][H][W] c64, probe [M][N][N] c64, positions [B][2] f32, tilt per tilt_mode
 *   (may be NULL when tilt_mode == 0), meas_amp [B][N][N] f32 = sqrt(counts), DC at [0][0].
 * Outputs (device):
 *   loss          [1] f64      = L                                   (required)
 *   loss_per_pos  [B] f32      = sum_k (sqrt(I_b) - a_b)^2           (may be NULL)
 *   intensity     [B][N][N] f32 = I_b(k)                             (may be NULL)
 * Leaves the incident waves of every slice in the workspace for pty_backward. */
int pty_forward_loss(pty_plan* plan, const void* object, const void* probe,
                     const float* positions, const float* tilt, const float* meas_amp, int32_t B,
                     double* loss, float* loss_per_pos, float* intensity, void* stream);

/* Exact gradient of L for the same minibatch (hand-written adjoint).
 * Runs the forward itself unless flags has PTY_BWD_REUSE_FORWARD, which reuses the waves saved by
 * the immediately preceding pty_forward_loss (same plan, stream, pointers and B).  Reuse is by
 * pointer identity only: with that flag the caller guarantees the arrays were not modified in
 * between (any pty_step / pty_adam_update on the plan cancels the saved state by itself).
 * Outputs (device; any may be NULL = not wanted, except g_object):
 *   g_object    [Nz][H][W] c64  scatter-add over the overlapping patches
 *   g_probe     [M][N][N] c64
 *   g_positions [B][2] f32      = dL/dDelta_b  (y, x)
 *   g_tilt      [2] (tilt_mode 1: summed over b) or [B][2] (tilt_mode 2); ignored for mode 0
 *   g_dz        [1] f32         = dL/d(dz); needs tilt_mode != 0 or PTY_FLAG_SPECTRA
 * flags: PTY_BWD_ACCUMULATE, PTY_BWD_REUSE_FORWARD. */
int pty_backward(pty_plan* plan, const void* object, const void* probe,
                 const float* positions, const float* tilt, const float* meas_amp, int32_t B,
                 void* g_object, void* g_probe, float* g_positions, float* g_tilt, float* g_dz,
                 int32_t flags, void* stream);

/* Select the loss of every later call on this plan (NULL = mode 0).  Host struct, copied. */
int pty_set_loss(pty_plan* plan, const pty_loss* cfg);

/* The four terms (L_Gaussian, L_Poisson, L_PACBED, L_sparse) of the last mode-1 forward on this plan, to host;
 * synchronises the plan's stream.  L_PACBED and L_sparse are evaluated only when they carry a non-zero weight
 * (0 otherwise). */
int pty_loss_terms(pty_plan* plan, double* terms4);

/* Amplitude / phase object: O = amp exp(i phase), both [n_obj][Nz][H][W] f32.  The complex object is
 * composed into the workspace (plan needs PTY_FLAG_AMP_PHASE) and the calls below behave like their complex
 * counterparts; g_amp = Re(conj(g_O) e^{i phase}), g_phase = Im(g_O conj(O)) + w_sparse dL_sparse/dphase.  With loss
 * mode 1 the sparsity term Eq. 8 (mean |phase| over the patches of the minibatch) is part of `loss`. */
int pty_forward_loss_ap(pty_plan* plan, const float* amp, const float* phase, const void* probe,
                        const float* positions, const float* tilt, const float* meas_amp, int32_t B,
                        double* loss, float* loss_per_pos, float* intensity, void* stream);
int pty_backward_ap(pty_plan* plan, const float* amp, const float* phase, const void* probe,
                    const float* positions, const float* tilt, const float* meas_amp, int32_t B,
                    float* g_amp, float* g_phase, void* g_probe, float* g_positions, float* g_tilt, float* g_dz,
                    int32_t flags, void* stream);
/* The paper's minibatch update: forward, Eq. 9 loss, gradients, Adam on amplitude, phase, probe, positions, tilt
 * (plan needs PTY_FLAG_STEP | PTY_FLAG_AMP_PHASE). */
int pty_step_ap(pty_plan* plan, float* amp, float* phase, void* probe, float* positions, float* tilt,
                const float* meas_amp, int32_t B, const pty_adam_ap* hp, const pty_adam_state_ap* st,
                double* loss, void* stream);

/* Apply the constraints in place: amp / phase [n_obj][Nz][H][W] f32 (either may be NULL), probe [M][N][N] c64
 * (may be NULL when ortho_probe == 0; M <= 32 for the orthogonalisation).  Enqueue-only. */
int pty_constrain(pty_plan* plan, float* amp, float* phase, void* probe, const pty_constraints* c, void* stream);
/* Eq. 13 as printed, on a complex object [n_obj][Nz][H][W] c64 in place (real kernel: re and im are blurred). */
int pty_rz_filter_object(pty_plan* plan, void* object, float sigma_z, void* stream);

/* One optimisation step: forward, loss, gradient and an Adam update of object, probe, positions
 * and tilt in place (plan needs PTY_FLAG_STEP).  loss [1] f64 device = L before
 * the update.  hp and st are HOST structs (st holds device pointers). */
int pty_step(pty_plan* plan, void* object, void* probe, float* positions, float* tilt,
             const float* meas_amp, int32_t B, const pty_adam* hp, const pty_adam_state* st,
             double* loss, void* stream);

/* Adam update of one flat float32 parameter array (the kernel pty_step uses), exposed for
 * callers that keep their own gradient buffers.  All device pointers, n floats. */
int pty_adam_update(pty_plan* plan, float* theta, const float* grad, float* m, float* v, size_t n,
                    float lr, float beta1, float beta2, float eps, int32_t t, void* stream);

/* End-to-end variant with HOST buffers (pinned memory recommended; plan needs PTY_FLAG_HOST):
 * copies the inputs host->device, runs pty_forward_loss + pty_backward, copies loss and the
 * gradients device->host and synchronises the stream before returning.  Host outputs that are
 * NULL are skipped.  The measurements (only the loss kernel reads them) travel on a second stream
 * owned by the plan while the forward kernel runs, ordered behind `stream` by events; with pageable
 * host memory the copies serialise and the result is the same. */
int pty_grad_host(pty_plan* plan, const void* h_object, const void* h_probe,
                  const float* h_positions, const float* h_tilt, const float* h_meas_amp, int32_t B,
                  double* h_loss, void* h_g_object, void* h_g_probe, float* h_g_positions,
                  float* h_g_tilt, void* stream);

/* The same call without the final synchronisation: everything is enqueued on `stream` (and the plan's copy
 * stream) and the host outputs are valid after pty_grad_host_wait(plan).  Two plans on two streams fed alternately
 * overlap one minibatch's copies with the other's kernels (bench.py's end-to-end number).  The host buffers must
 * stay untouched, and pinned for any overlap to happen, until the wait returns. */
int pty_grad_host_async(pty_plan* plan, const void* h_object, const void* h_probe,
                  const float* h_positions, const float* h_tilt, const float* h_meas_amp, int32_t B,
                  double* h_loss, void* h_g_object, void* h_g_probe, float* h_g_positions,
                  float* h_g_tilt, void* stream);
int pty_grad_host_wait(pty_plan* plan);

/* Probe-mode orthogonalisation for callers that have no device memory to give (the same operation
 * as pty_constrain with ortho_probe = 1, the same three kernels, the same results).
 *
 * Who needs it.  Every other entry point takes a plan, and a plan lives in a device workspace that the CALLER has to
 * allocate.  Some callers cannot: a host application that handed the whole device to its own memory pool when it
 * started (any further cudaMalloc fails, and the pool hands nothing to plug-ins), a plug-in or post-processing hook
 * that is given the probe pointer and a stream and nothing else, or a control loop that may not stall -- cudaMalloc
 * and cudaFree synchronise the device.  Such a caller still wants the probe modes orthogonalised between iterations.
 *
 * How.  No plan, no workspace, and the call makes no cudaMalloc, cudaFree or other allocating call.  The scratch
 * the operation needs (Gram matrix, eigenvectors, eigenvalues: 33,024 bytes) is a fixed array inside libpty.so's
 * device image, sized for the limit below; every GPU on which the library's kernels get loaded holds those 33 KB
 * until the process exits, whether or not this function is ever called.
 *
 *   probe   [M][N][N] c64 on `device`, 8-byte aligned; replaced in place by the orthogonal modes of the same
 *           mixed state, ordered by decreasing power
 *   M       1 .. PTY_ORTHO_NOALLOC_MAX_MODES; more modes do not fit the fixed scratch: PTY_ERR_UNSUPPORTED, and the
 *           text from pty_last_error(NULL) names the limit (use pty_constrain with a plan for larger M -- which
 *           has the same limit today)
 *   N       1 .. 4096 (any window size, not only 64 / 128 / 256)
 *   device  CUDA device ordinal that owns `probe`; made current for the call, the caller's device is restored
 *   stream  a stream of that device; the three kernels are enqueued on it and the call does not synchronise
 *
 * First call on a device.  It looks up the device address of the scratch array (cudaGetSymbolAddress, which may
 * load the library's kernels onto that device) and remembers it per device.  Make that first call during start-up,
 * outside any stream capture; later calls on that device only launch kernels.
 *
 * Sharing.  There is ONE scratch array per device for the whole process.  Nothing in it has to start at zero:
 * a call overwrites every element it later reads, so the previous call's contents (which stay there) do no
 * harm.  Two calls whose kernels can overlap on the same device -- different streams, different host threads --
 * race on it and give wrong modes: keep all calls for one device on one stream, or order them with events.
 *
 * Errors: PTY_ERR_INVALID_ARG (null or misaligned probe, M < 1, N out of range, bad device), PTY_ERR_UNSUPPORTED
 * (M beyond the limit), PTY_ERR_CUDA; the text is returned by pty_last_error(NULL) on the calling thread. */
#define PTY_ORTHO_NOALLOC_MAX_MODES   32
#define PTY_ORTHO_NOALLOC_SCRATCH_BYTES  (2 * 32 * 32 * 16 + 32 * 8)    /* 33,024 per GPU */
int pty_ortho_probe_noalloc(void* probe, int32_t M, int32_t N, int device, void* stream);

/* Synchronises the plan's last stream and returns PTY_OK, PTY_ERR_BOUNDS (flag bit 1; wins if both are set),
 * PTY_ERR_ZERO_DATA (flag bit 2) or PTY_ERR_CUDA.
 * device_flags (host, may be NULL) receives the raw sticky flag word and clears it. */
int pty_status(pty_plan* plan, int32_t* device_flags);

/* Kernel timing for benchmarks.  pty_profile(plan, 1) makes every later call bracket its forward
 * (a2-a5) and adjoint (a7-a13) kernel launches with CUDA events on the call's own stream (the first
 * 1024 launches after enabling are kept; later ones are not recorded until the next read); pty_profile(plan, 0) stops and forgets them.
 * pty_profile_read synchronises the plan's stream and returns, for the launches recorded since the
 * last read, the summed device time in milliseconds and the launch count of each kernel (host out). */
int pty_profile(pty_plan* plan, int32_t enable);
int pty_profile_read(pty_plan* plan, float* fwd_ms, int32_t* fwd_launches, float* bwd_ms, int32_t* bwd_launches);

/* Number of kernel launches the plan has enqueued so far (for bench accounting). */
int64_t pty_launch_count(const pty_plan* plan);

/* Text of the plan's last error ("" if none).  plan == NULL returns the last creation error. */
const char* pty_last_error(const pty_plan* plan);

/* Library version string, e.g. "pty-b200 0.2 (sm_100a)". */
const char* pty_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PTY_H */
