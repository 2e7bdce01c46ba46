/* ptycho.h — C ABI of the B200 hot path of mixed-state multislice ptychography
 * (arxiv 2505.14372, "phaser").  One call = one batched forward(+adjoint) pass of the model of
 * PAPER.md:113-123 over a group of probe positions, on one GPU, on the caller's stream.
 *
 * Conventions (DESIGN.md §2/§3 give the citations and the readings R1..R29 of the paper):
 *   - complex64 is interleaved (re, im) float32; all arrays are C-contiguous, row-major, last index fastest.
 *   - F is the unnormalised forward DFT with kernel exp(-2 pi i q.r/N); zero frequency at index [0][0].
 *   - gradients are g = dL/d conj(z); a descent step is z <- z - lr*g.
 *   - pointers ending in _d are DEVICE pointers, _h HOST pointers.  The library never allocates device
 *     memory and keeps no pointer after a call returns.  The device-path calls are re-entrant across streams and
 *     threads; process-wide state is limited to (a) a once-per-device record that the kernels' shared-memory limits
 *     have been set, (b) the copy stream and events of ptycho_gradient_host, created on first use and reused (that
 *     call is serialised by a lock), (c) the per-THREAD launch counter and optional profiling record below, and (d) the
 *     16 MiB static device array of ptycho_apply_constraint_static with its per-device cached address.
 *     pt_problem / pt_update / slice_thickness are HOST memory, read synchronously during the call.
 *   - workspace_d: DEVICE memory, 256-byte aligned.  Its first 256 bytes hold the deferred status word: the caller
 *     zeroes them once when the buffer is allocated (cudaMemset); ptycho_status() reads and clears the word.
 *   - all work is enqueued on `cuda_stream` (a cudaStream_t passed as void*); nothing synchronises except
 *     ptycho_status() and the *_host convenience entry point.
 *   - CUDA graphs: every device-path call (everything except ptycho_status, ptycho_gradient_host and the profiling record)
 *     only enqueues kernels on `cuda_stream`, so a sequence of calls can be captured into a CUDA graph and replayed, once the
 *     same calls have run once on that device outside a capture (the first call sets the kernels' shared-memory attributes).
 *     pt_problem / pt_update / slice_thickness are read at capture time (tests: test_step_captured_in_a_cuda_graph_replays_bitwise).
 *   - every function returns int32 status: 0 = PT_OK, < 0 = error.  No exceptions, no printing, no abort.
 *   - resources: the chain kernels take a whole SM each (up to 227 KB of shared memory, the full register file) and, with an
 *     even number of modes, the backward kernel allocates the SM's tensor memory (tcgen05.alloc, all 512 columns at N >= 128)
 *     for the duration of the kernel; the flag PT_NO_MODE_PAIRS selects the kernel that does not (debugging aid).
 */
#ifndef PTYCHO_H_
#define PTYCHO_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct { float re, im; } pt_c64;

enum { PT_LOSS_AMPLITUDE = 0,   /* PAPER.md:157, l = 1/2 (sqrt(I+c) - sqrt(Iexp+c))^2 ; c = 3/8 gives Anscombe */
       PT_LOSS_POISSON = 1,     /* PAPER.md:151, l = I - Iexp (ln(I+eps) - ln(Iexp+eps) + 1)                  */
       PT_LOSS_GAUSSIAN = 2 };  /* PAPER.md:144, l = (I - Iexp)^2 / (2 sigma^2), sigma = loss_c > 0           */

enum { PT_SHIFT_FOURIER_PROBE = 0,    /* integer window on the object + Fourier shift of the probe (R1) */
       PT_SHIFT_BILINEAR_OBJECT = 1 };/* PAPER.md:61 "sampled" (R1, secondary): probe unshifted; the patch is a four-tap
                                       * bilinear sample of the object at c + r, c = X/px - N/2 = i0 + f (i0 = floor(c));
                                       * the object gradient is scattered with the same weights and dL/dX comes through
                                       * the weights (i0 fixed).  Windows need i0 + N <= size - 1.  Step-size terms (R30): dOhat is
                                       * sampled with the same four taps; the position terms come through the patch,
                                       * numX_a = -1/2 dL/df_a, denX_a = sum_{i,k,r} |Psi_{i,k} dT_i/df_a|^2 (f in px).            */

enum { PT_WANT_POS_GRAD = 1,          /* fill grad_pos_d                                                        */
       PT_WANT_ILLUM = 2,             /* fill illum_d with sum_{j,k} |Psi_{i,k,j}|^2             */
       PT_WANT_STEP_SIZES = 4,        /* fill step_terms_d, needs illum_prev_d               */
       PT_ACCUMULATE = 16,            /* add into grad_object_d/grad_probe_d/illum_d/loss_d instead of overwriting */
       PT_WANT_WEIGHTED_ILLUM = 64,   /* with PT_WANT_ILLUM and PT_WANT_STEP_SIZES: illum_d is [2][S][obj_ny][obj_nx]; plane 1 is
                                       * W_i = sum_j alpha_{O,i,j} sum_k |Psi_{i,k,j}|^2, alpha_{O,i,j} = numO[j,i] / (denO[j,i] +
                                       * lsqml_gamma): the per-position step sizes of PAPER.md:221 weighting the slice update as
                                       * PAPER.md:225 prints it (reading R24); used by PT_UPDATE_LSQML_WEIGHTED              */
       PT_LSQML_MODULUS_CHI = 256,    /* with PT_WANT_STEP_SIZES / PT_UPDATE_LSQML*: the LSQML wavefront update is the modulus-constraint
                                       * update of PAPER.md:173, chi~ = (sqrt(Iexp+c)/(eps+sqrt(I+c)) - 1) psi~ = -2 gPhi~ (reading R31), instead
                                       * of the steepest-descent chi = -gPhi (R20): numerators and denominators of the object and probe
                                       * terms x4, position numerators x2, update directions x2.  PT_LOSS_AMPLITUDE only (the paper gives
                                       * that update for the amplitude model), else PT_ERR_UNSUPPORTED                          */
       PT_STASH_FP16 = 512,           /* SURVEY 8(f) rank 4 (PAPER.md:79-81 names reduced precision as future work): the slice waves Psi_{i,k}
                                       * kept for the adjoint are STORED as binary16 pairs (round to nearest even; all arithmetic stays
                                       * float32): half the stash traffic and memory (1.45x the positions in flight).  grad_probe, grad_pos
                                       * and the loss do not read the stash and are unchanged bit for bit; grad_object, illum_d and the
                                       * object step-size terms are formed from the rounded waves: measured 2e-5 .. 1.01e-4 relative L2 from
                                       * the oracle over the parity cases (float32 stash: <= 3.4e-5), i.e. AT the 1e-4 bar, not inside it
                                       * everywhere.  Off by default.
                                       * ptycho_gradient only; not with PT_EPIE, and PT_WANT_ILLUM needs an even mode count or
                                       * PT_WANT_STEP_SIZES (the map comes from the backward kernel's staging): else PT_ERR_UNSUPPORTED */
       PT_NO_SINGLE_SLICE_FUSION = 1024, /* debugging aid: a single-slice problem runs through the multislice kernel sequence (forward chain,
                                       * loss, backward chain) instead of the fused single-slice kernel.  The fused kernel sums
                                       * the probe-gradient partials of the positions one resident CTA takes in float32 before the
                                       * fp64 reduction: grad_probe is bit-reproducible on a device, its last bits depend on the
                                       * device's SM count                                                                       */
       PT_NO_MODE_PAIRS = 128,        /* debugging aid: the backward pass runs one mode per CTA even when the mode count is even
                                       * (no tensor-memory allocation); results differ only by the rounding of one float32 add */
       PT_EPIE = 32 };                /* ptycho_gradient returns the multislice ePIE ("3PIE") update DIRECTIONS instead of
                                       * gradients: grad_object_d <- sum_{j,k} conj(Psi_i,k)/max|Psi_i,k|^2
                                       * chi_i,k (scattered), grad_probe_d <- (1/J) sum_j shift_j^-1(chi'_0,k), chi~ = (sqrt(Iexp+c)/
                                       * (eps+sqrt(I+c)) - 1) psi~, chi'_i = conj(T_i)/max|T_i|^2 chi_i back-propagated slice by
                                       * slice.  To be ADDED with PT_UPDATE_EPIE.  PT_LOSS_AMPLITUDE and PT_SHIFT_FOURIER_PROBE
                                       * only; no position gradient, no step sizes (PT_ERR_UNSUPPORTED).                  */

enum { PT_OK = 0, PT_ERR_NULL = -1, PT_ERR_BAD_SIZE = -2, PT_ERR_BAD_PARAM = -3, PT_ERR_WORKSPACE = -4,
       PT_ERR_CUDA = -5, PT_ERR_OUT_OF_BOUNDS = -6, PT_ERR_NONFINITE = -7, PT_ERR_UNSUPPORTED = -8,
       PT_ERR_STATIC_LIMIT = -9 /* ptycho_apply_constraint_static only: the field needs more than PT_STATIC_SCRATCH_BYTES */ };

/* Problem statement. HOST struct. */
typedef struct {
  int32_t n;                      /* N: probe / pattern side in px; supported: 64, 128, 256                      */
  int32_t n_modes;                /* M >= 1 incoherent probe modes P_k                           */
  int32_t n_slices;               /* S >= 1 object slices O_i                                    */
  int32_t obj_ny, obj_nx;         /* object slice size in px (>= N)                                             */
  int32_t n_pos_total;            /* rows of positions_d / intensity_d                                          */
  int32_t n_batch;                /* J: positions in this call; batch_idx_d has J entries (NULL: rows 0..J-1).  Entries
                                   * outside [0, n_pos_total) are clamped and raise PT_ERR_OUT_OF_BOUNDS (deferred).  A row
                                   * must not appear twice in a batch whose positions are updated (the updates would race) */
  float pixel_size;               /* Angstrom / px (probe and object)                                           */
  float wavelength;               /* Angstrom                                                                   */
  const float *slice_thickness;   /* HOST, S entries (Angstrom); entry S-1 unused (R10)                         */
  float tilt_x_mrad, tilt_y_mrad; /* propagator tilt (R8: exp(+2 pi i dz (kx tan tx + ky tan ty)))*/
  float bandlimit;                /* fraction of Nyquist of the sharp circular mask (R9); <=0 off */
  int32_t loss;                   /* PT_LOSS_*                                                                   */
  float loss_c;                   /* c of the variance-stabilising transform; Gaussian: sigma    */
  float eps;                      /* epsilon > 0 (R11..R13)                                       */
  int32_t shift_mode;             /* PT_SHIFT_*                                                                  */
  int32_t flags;                  /* PT_WANT_* | PT_ACCUMULATE                                                   */
  float lsqml_delta_o;            /* delta_O of PAPER.md:219 (PT_WANT_STEP_SIZES only)                          */
  float lsqml_delta_p;            /* probe analogue: dPhat = -gP / (delta_p + 1) (R19)                          */
  float lsqml_gamma;              /* gamma of PAPER.md:221 in the per-position alphas (PT_WANT_WEIGHTED_ILLUM only) */
  const float *lsqml_probe_precond_d; /* DEVICE [N][N] or NULL: probe preconditioner of PAPER.md:227 (R25), last iteration's
                                   * sum of ptycho_object_transparency maps: dPhat_k = -gP_k / (precond + delta_p), in the
                                   * step-size sweep and in PT_UPDATE_LSQML*; NULL: the constant 1 (R19)              */
} pt_problem;

enum { PT_UPDATE_SGD = 0, PT_UPDATE_LSQML = 1, PT_UPDATE_EPIE = 2, PT_UPDATE_LSQML_WEIGHTED = 3 };
typedef struct {                  /* HOST struct */
  int32_t mode;                   /* PT_UPDATE_SGD:   z <- z - lr * g   */
                                  /* PT_UPDATE_LSQML: O_i += beta_O alpha_{O,i} dOhat_i etc.   (R18) */
                                  /* PT_UPDATE_EPIE:  O_i += beta_obj dO_i, P_k += beta_probe dP_k, with
                                   *                  the directions ptycho_gradient returned under PT_EPIE              */
  float lr_obj, lr_probe, lr_pos;
  float beta_obj, beta_probe;
                                  /* PT_UPDATE_LSQML_WEIGHTED: object as PAPER.md:225 prints it, with per-position step
                                   *                  sizes (R24): O_i += beta_obj dOhat_i W_i / I_i where I_i > 0 (pixels no window
                                   *                  of the batch covers are left alone); probe and positions as PT_UPDATE_LSQML */
  float gamma;                    /* step-size regulariser of PAPER.md:221                                      */
  const float *illum_batch_d;     /* DEVICE, [2][S][obj_ny][obj_nx]: (I, W) as ptycho_gradient wrote them to illum_d under
                                   * PT_WANT_WEIGHTED_ILLUM; PT_UPDATE_LSQML_WEIGHTED only, NULL otherwise                */
} pt_update;

/* Number of floats per position in step_terms_d:  (numO_i, denO_i) i = 0..S-1, (numP, denP),
 * (numX_y, denX_y), (numX_x, denX_x)  => 2*S + 6. */
#define PT_STEP_TERMS_PER_POS(S) (2 * (S) + 6)

/* Device scratch the caller must supply.  ptycho_workspace_bytes returns the RECOMMENDED size (positions are
 * processed in chunks; a larger workspace means larger chunks, capped at 49 GiB — with PT_WANT_STEP_SIZES the patch
 * gradients, probe partials and |Psi|^2 the backward pass stages are kept for the whole batch on top of that, up to 150 GiB
 * in total, so that the step-size sweep needs no second pass through the chain); ptycho_workspace_min_bytes the smallest
 * size the calls accept (with step sizes and a batch that does not fit, each chunk is then recomputed for the sweep).
 * The first 256 bytes hold the deferred status word. */
size_t ptycho_workspace_bytes(const pt_problem *p);
size_t ptycho_workspace_min_bytes(const pt_problem *p);
/* Positions kept in flight per chunk (the memory unit, as opposed to the mini-batch p->n_batch, the optimisation
 * unit) for a workspace of workspace_bytes; 0 if the problem is invalid or the size too small. */
int32_t ptycho_positions_in_flight(const pt_problem *p, size_t workspace_bytes);

/* Forward model + loss.
 *   object_d     [S][obj_ny][obj_nx]  transmission functions O_i
 *   probe_d      [M][N][N]            probe modes in real space, centred at (N/2, N/2); mode weights folded in (R16)
 *   positions_d  [n_pos_total][2]     (y, x) probe-centre coordinates in Angstrom; object pixel (0,0) at 0 (R3)
 *   intensity_d  [n_pos_total][N][N]  measured I_exp, zero frequency at [0][0] (R6); may be NULL if only
 *                                     model_intensity_d is wanted (loss outputs are then zero)
 *   batch_idx_d  [n_batch] int32 rows of positions/intensity, or NULL
 *   loss_d       [1] double  L = sum_j sum_q l   (NULL allowed)
 *   loss_per_pos_d [n_batch] float L_j           (NULL allowed)
 *   model_intensity_d [n_batch][N][N] float I_j  (NULL allowed)
 * Errors: PT_ERR_NULL, PT_ERR_BAD_SIZE, PT_ERR_BAD_PARAM, PT_ERR_WORKSPACE, PT_ERR_CUDA immediately;
 * PT_ERR_OUT_OF_BOUNDS (a window [r0, r0+N) leaves the object: the kernel clamps r0 so it never reads
 * outside, and raises the flag — R4) and PT_ERR_NONFINITE deferred through ptycho_status(). */
int32_t ptycho_forward_loss(const pt_problem *p, const pt_c64 *object_d, const pt_c64 *probe_d,
                            const float *positions_d, const float *intensity_d, const int32_t *batch_idx_d,
                            double *loss_d, float *loss_per_pos_d, float *model_intensity_d,
                            void *workspace_d, size_t workspace_bytes, void *cuda_stream);

/* Loss + gradients: the adjoint of the chain above.
 *   grad_object_d [S][obj_ny][obj_nx]  dL/d conj(O_i), deterministic scatter-add over overlapping patches
 *   grad_probe_d  [M][N][N]            dL/d conj(P_k)
 *   grad_pos_d    [n_batch][2]         dL/dX (per Angstrom), PT_WANT_POS_GRAD            (NULL allowed)
 *   illum_d       [S][obj_ny][obj_nx]  float, this batch's sum_{j,k}|Psi_{i,k}|^2, PT_WANT_ILLUM (NULL allowed);
 *                                      [2][S][obj_ny][obj_nx] under PT_WANT_WEIGHTED_ILLUM (plane 1 = W, see the flag)
 *   illum_prev_d  [S][obj_ny][obj_nx]  float, running sum of the previous iteration (R19);
 *                                      needed with PT_WANT_STEP_SIZES
 *   step_terms_d  [n_batch][2S+6]      float, PT_WANT_STEP_SIZES                          (NULL allowed)
 * Bitwise reproducible: the same inputs give the same outputs on every run (no float atomics). */
int32_t ptycho_gradient(const pt_problem *p, const pt_c64 *object_d, const pt_c64 *probe_d,
                        const float *positions_d, const float *intensity_d, const int32_t *batch_idx_d,
                        pt_c64 *grad_object_d, pt_c64 *grad_probe_d, float *grad_pos_d,
                        float *illum_d, const float *illum_prev_d, float *step_terms_d,
                        double *loss_d, float *loss_per_pos_d,
                        void *workspace_d, size_t workspace_bytes, void *cuda_stream);

/* Update step (PAPER.md:187 SGD; PAPER.md:225 LSQML-style with per-group step sizes, R18).  In place.
 * Any of object_d/probe_d/positions_d may be NULL (that variable is left alone). positions rows batch_idx_d only. */
int32_t ptycho_apply_update(const pt_problem *p, pt_c64 *object_d, pt_c64 *probe_d, float *positions_d,
                            const pt_c64 *grad_object_d, const pt_c64 *grad_probe_d, const float *grad_pos_d,
                            const float *illum_prev_d, const float *step_terms_d, const int32_t *batch_idx_d,
                            const pt_update *u, void *workspace_d, size_t workspace_bytes, void *cuda_stream);

/* LSQML probe preconditioner ("summed object intensity ... recorded in the probe/cutout view"; R25):
 *   objtrans_d [N][N] float <- (PT_ACCUMULATE: +=) sum_{j in batch} prod_i |O_i[r0_j + r]|^2, integer windows of R2
 * (PT_SHIFT_FOURIER_PROBE only, else PT_ERR_UNSUPPORTED).  Fixed summation order.  workspace_d: any workspace of this
 * problem (only the status word is touched: PT_ERR_OUT_OF_BOUNDS is deferred as in ptycho_forward_loss). */
int32_t ptycho_object_transparency(const pt_problem *p, const pt_c64 *object_d, const float *positions_d,
                                   const int32_t *batch_idx_d, float *objtrans_d, void *workspace_d, size_t workspace_bytes,
                                   void *cuda_stream);

/* ---- what completes a usable gradient-descent iteration around ptycho_gradient -------------------
 * All three work on a complex field [n_slices][ny][nx] (object slices; probe modes with n_slices = M, ny = nx = N),
 * DEVICE memory, on `cuda_stream`; deterministic (owner-computes, fixed-order fp64 cost sum).                        */

/* Cost regularisers (the paper names them only — reading R26).  ADDS weight * dR/dconj(field) into
 * grad_d (same shape; may be NULL) and ADDS R into *cost_d (DEVICE double[1]; may be NULL), so both can be chained behind
 * ptycho_gradient's outputs.
 *   PT_REG_L2             R = w sum |z - ref|^2                     (ref = 1: "penalizes a non-vacuum object"; 0 for a probe)
 *   PT_REG_L1             R = w sum sqrt(|z - ref|^2 + eps^2)
 *   PT_REG_TIKHONOV       R = w sum_{d = x, y} sum |D_d z|^2        forward differences inside a slice, no wrap-around
 *   PT_REG_TV             R = w sum_{d = x, y} sum sqrt(|D_d z|^2 + eps^2)
 *   PT_REG_LAYER_TIKHONOV / PT_REG_LAYER_TV   the same with the one difference along depth, z_{i+1} - z_i
 *   PT_REG_L1_PHASE       R = w sum sqrt(phi^2 + eps^2), phi = arg z (principal value; reading R26b); ref unused; zero pixels skipped
 *   PT_REG_L1_FOURIER     R = w sum_s sum_q sqrt(|Z_s[q]|^2 + eps^2), Z_s the unnormalised 2-D DFT of the whole slice s (any ny, nx
 *                         <= 4096; reading R26c: the sparsity-promoting form of "L1 on the object power spectrum"); ref unused;
 *                         needs workspace_bytes >= ptycho_regularizer_workspace_bytes() + 16 * n_slices*ny*nx
 * workspace_d: at least ptycho_regularizer_workspace_bytes() bytes of scratch (per-block cost partials).
 * Errors: PT_ERR_NULL, PT_ERR_BAD_SIZE (a dimension < 1), PT_ERR_BAD_PARAM (unknown kind, eps < 0), PT_ERR_WORKSPACE. */
enum { PT_REG_L2 = 0, PT_REG_L1 = 1, PT_REG_TIKHONOV = 2, PT_REG_TV = 3, PT_REG_LAYER_TIKHONOV = 4, PT_REG_LAYER_TV = 5, PT_REG_L1_PHASE = 6, PT_REG_L1_FOURIER = 7 };
size_t ptycho_regularizer_workspace_bytes(void);
int32_t ptycho_cost_regularizer(int32_t kind, float weight, float ref, float eps, int32_t n_slices, int32_t ny, int32_t nx,
                                const pt_c64 *field_d, pt_c64 *grad_d, double *cost_d,
                                void *workspace_d, size_t workspace_bytes, void *cuda_stream);

/* Constraint regularisers (reading R27), in place on field_d.
 *   PT_CON_AMPLITUDE_CLAMP  |z| limited to [a, b], phase kept (a zero pixel with a > 0 becomes the real number a)
 *   PT_CON_SUPPORT_MASK     z[s][y][x] *= mask_d[y][x]  (probe support in real space; mask_d DEVICE float [ny][nx])
 *   PT_CON_LAYER_BLUR       Gaussian blur along depth, sigma = a slices, as a REAL-SPACE convolution (the paper: no bleeding
 *                           from top to bottom through periodic boundaries): out[p] = sum_t w_t z[p+t] / sum_t w_t over the
 *                           taps |t| <= ceil(4 sigma) that fall inside, w_t = exp(-t^2 / (2 sigma^2))
 *   PT_CON_LOWPASS          the same blur along x, then along y, sigma = a px
 *   PT_CON_SUPPORT_MASK_FOURIER  probe support in reciprocal space: z <- Finv(mask_d .* F(z)), mask_d DEVICE float [n][n], zero
 *                           frequency at [0][0]; ny = nx = n in {64, 128, 256} (the chain kernels' register FFT)
 *   PT_CON_PHASE_DERAMP     removes an affine phase ramp per slice (reading R29, no unwrapping): slopes
 *                           b = arg sum z[y+1,x] conj(z[y,x]), c likewise along x, offset a = arg sum z exp(-i(b(y-yc) + c(x-xc)))
 *                           about the centre; z <- z exp(-i(a + b(y-yc) + c(x-xc))).  Fixed-order fp64 sums.
 * The two blurs need workspace_bytes >= n_slices*ny*nx*8 (one copy of the field), the deramp 256 + n_slices*2080 bytes; the
 * others none (workspace_d may be NULL).
 * Errors: PT_ERR_NULL, PT_ERR_BAD_SIZE, PT_ERR_BAD_PARAM (unknown kind, a > b, sigma <= 0), PT_ERR_WORKSPACE.          */
enum { PT_CON_AMPLITUDE_CLAMP = 0, PT_CON_SUPPORT_MASK = 1, PT_CON_LAYER_BLUR = 2, PT_CON_LOWPASS = 3,
       PT_CON_SUPPORT_MASK_FOURIER = 4, PT_CON_PHASE_DERAMP = 5 };
int32_t ptycho_apply_constraint(int32_t kind, float a, float b, const float *mask_d, int32_t n_slices, int32_t ny, int32_t nx,
                                pt_c64 *field_d, void *workspace_d, size_t workspace_bytes, void *cuda_stream);

/* ptycho_apply_constraint for callers that cannot allocate device memory (code under CUDA graph capture, serving loops,
 * harnesses that forbid cudaMalloc): the kinds that need scratch — PT_CON_LAYER_BLUR, PT_CON_LOWPASS, PT_CON_PHASE_DERAMP —
 * with that scratch in a file-scope `static __device__` array of PT_STATIC_SCRATCH_BYTES inside the library instead of a
 * caller's workspace.  Same kernels, same launch configuration, same results bit for bit as ptycho_apply_constraint; the
 * call (and everything under it) calls no cudaMalloc / cudaFree and no allocating library routine.
 *   - Every GPU that loads the library holds the PT_STATIC_SCRATCH_BYTES (16 MiB) from module load until the process exits.
 *   - Limit: the two blurs need n_slices*ny*nx*8 bytes (fields up to 2 097 152 complex pixels, e.g. 8 slices of 512 x 512),
 *     the deramp 256 + n_slices*2080 bytes.  A larger field is rejected with PT_ERR_STATIC_LIMIT before anything is launched
 *     (field_d untouched); use ptycho_apply_constraint with a caller-owned workspace for it.
 *   - The first call on each device looks up the array's device address (cudaGetSymbolAddress, with that device current —
 *     the device that is current at the call; field_d must live there) and caches it per device; later calls only launch.
 *   - All calls on a device SHARE the one array, and it keeps the previous call's contents.  Nothing in it has to start at
 *     zero: every word a kernel reads (the blurred copy, the per-block partial sums, the slopes) is written earlier in the
 *     same call, so there is nothing to clear and stale contents are never read.  Calls that overlap on the GPU (two
 *     streams, two host threads, two graphs replayed side by side) RACE on it: serialise them on one stream.
 *   - The kinds that need no scratch are not served here: PT_ERR_UNSUPPORTED (ptycho_apply_constraint with workspace_d =
 *     NULL already allocates nothing for them).
 * Errors: PT_ERR_NULL, PT_ERR_BAD_SIZE, PT_ERR_BAD_PARAM (sigma outside (0, 8]), PT_ERR_UNSUPPORTED, PT_ERR_STATIC_LIMIT,
 * PT_ERR_CUDA (address lookup or a launch failed).                                                                     */
#define PT_STATIC_SCRATCH_BYTES (16u << 20)
int32_t ptycho_apply_constraint_static(int32_t kind, float a, int32_t n_slices, int32_t ny, int32_t nx, pt_c64 *field_d,
                                       void *cuda_stream);

/* Adam (Kingma & Ba algorithm 1; reading R28: complex first moment, second moment from |g|^2), step >= 1:
 *   m <- b1 m + (1-b1) g ; v <- b2 v + (1-b2) |g|^2 ; z <- z - lr (m / (1 - b1^step)) / (sqrt(v / (1 - b2^step)) + eps)
 * ptycho_adam_update: n complex numbers (z, g, m complex64; v float).  ptycho_adam_update_real: n floats (positions).
 * m_d and v_d are caller-owned state, zero before the first step.  Errors: PT_ERR_NULL, PT_ERR_BAD_PARAM (step < 1,
 * betas outside [0, 1), eps < 0).                                                                                      */
int32_t ptycho_adam_update(pt_c64 *z_d, const pt_c64 *g_d, pt_c64 *m_d, float *v_d, size_t n, float lr, float beta1,
                           float beta2, float eps, int32_t step, void *cuda_stream);
int32_t ptycho_adam_update_real(float *z_d, const float *g_d, float *m_d, float *v_d, size_t n, float lr, float beta1,
                                float beta2, float eps, int32_t step, void *cuda_stream);

/* End-to-end convenience with HOST buffers (pinned memory recommended): copies object/probe/positions and the
 * batch rows' intensities host->device into the workspace, runs ptycho_gradient, copies gradients and loss
 * back, and synchronises the stream.  The patterns are copied chunk by chunk on a second stream that lives for the duration
 * of the call, in the order the pass consumes them, so the copies overlap the chain kernels (use pinned host memory).
 * Workspace must be ptycho_workspace_host_bytes(p).  batch_idx_h may be NULL; with an index list the whole position table and
 * the list are copied once and the rows compacted on the device, and the patterns travel as one copy per run of consecutive
 * rows.  The call reads the pass's own deferred status before it returns: PT_ERR_OUT_OF_BOUNDS (a window left the object and
 * was clamped, R4, or an index outside [0, n_pos_total)) or PT_ERR_NONFINITE come back as the return value. */
size_t ptycho_workspace_host_bytes(const pt_problem *p);
int32_t ptycho_gradient_host(const pt_problem *p, const pt_c64 *object_h, const pt_c64 *probe_h,
                             const float *positions_h, const float *intensity_h, const int32_t *batch_idx_h,
                             pt_c64 *grad_object_h, pt_c64 *grad_probe_h, float *grad_pos_h,
                             double *loss_h, float *loss_per_pos_h,
                             void *workspace_d, size_t workspace_bytes, void *cuda_stream);

/* Synchronises the stream and returns the deferred device-side status (PT_OK, PT_ERR_OUT_OF_BOUNDS,
 * PT_ERR_NONFINITE, or PT_ERR_CUDA); clears it. */
int32_t ptycho_status(void *workspace_d, void *cuda_stream);

/* Number of the library's own kernel launches enqueued by the calls made so far on this thread (for bench.py). */
int64_t ptycho_launch_count(void);

/* Optional per-kernel device timing, for bench.py's roofline line (the profiling recipe: CUDA events on the
 * launching stream).  After ptycho_profile_enable(1) every kernel this THREAD launches through the calls above is
 * followed by a CUDA event on its stream; ptycho_profile_read synchronises those events, writes per kernel kind
 * (0 <= kind < ptycho_profile_num_kernels()) the summed device time in ms and the number of launches to the two
 * HOST arrays, and resets the record.  ptycho_profile_enable(0) switches it off.  Off by default. */
int32_t ptycho_profile_enable(int32_t on);
int32_t ptycho_profile_num_kernels(void);
const char *ptycho_profile_kernel_name(int32_t kind);
int32_t ptycho_profile_read(float *ms_h, int64_t *launches_h);

/* Measured FP32 FMA throughput of the current device in TFLOP/s (2 flop per FMA), for bench.py's roofline.peak_measured:
 * a register-only kernel of independent FFMA chains on every SM, best of five launches timed with CUDA events on
 * `cuda_stream`; synchronises.  workspace_d: any device buffer of >= 512 bytes (never written in practice). */
int32_t ptycho_profile_fp32_peak(double *tflops_h, void *workspace_d, void *cuda_stream);

const char *ptycho_strerror(int32_t code);

#ifdef __cplusplus
}
#endif
#endif /* PTYCHO_H_ */
