/*
 * afno.h -- C ABI of the B200-native AFNO spectral token-mixing layer.
 *
 * The layer (FourCastNet, arXiv 2208.05419; citations are /root/reference/PAPER.md lines):
 *   step 1  PAPER.md:114  "An FFT spatially mixes the ... grid of tokens"      (rfft2, ortho)
 *   step 2  PAPER.md:115-121  "the channels are mixed using a block-diagonal MLP in the
 *           Fourier space ... MLP weights are shared across tokens"
 *   step 3  PAPER.md:122  "An inverse FFT demixes the tokens"                  (irfft2, ortho)
 *   PAPER.md:136  real-to-complex / complex-to-real FFTs batched over batch and features
 *   PAPER.md:138  weights are real tensors with (re, im) as the fastest index; activations
 *                 act on real and imaginary parts independently
 * Bias, ReLU, softshrink(lambda), hard mode truncation by a kept fraction, ortho
 * normalisation and the residual add are fixed by BASELINE.json:north_star and the
 * readings A1-A20 in DESIGN.md S3.  In formulas (h,r rows; w columns; c column frequency;
 * Wh = W/2+1; channel ch = j*bs + i):
 *
 *   Xh[b,r,c,ch] = (HW)^-1/2 sum_{h,w} x[b,h,w,ch] exp(-2 pi i (r h/H + c w/W))
 *   kept (r,c)  <=>  |kappa(r)| < Kh and c < Kw,  kappa(r) = r if r <= H/2 else r-H,
 *                    Kh = clamp(floor(f (H/2+1)), 1, H/2+1), Kw likewise from W
 *   P1[o] = sum_i Xh[j*bs+i] W1[j,i,o] + b1[j,o];  O1 = relu(Re P1) + i relu(Im P1)
 *   P2[o] = sum_i O1[i] W2[j,i,o] + b2[j,o];       Z = S_l(Re P2) + i S_l(Im P2), 0 if not kept
 *   s[b,h,w,ch] = (HW)^-1/2 sum_{r,c} alpha_c Re(Z[b,r,c,ch] exp(+2 pi i (r h/H + c w/W)))
 *   y = x + s
 *
 * Everything runs on the device in this library's own kernels; there is no CPU fallback.
 * All entry points are plain C: integers, floats, raw pointers.  Unless a parameter says
 * "host", every data pointer is a DEVICE pointer on the current CUDA device, 16-byte
 * aligned, owned by the caller, and must stay valid until the work queued on `cuda_stream`
 * has completed.  fwd/bwd allocate no device memory, never synchronise the host and are
 * CUDA-graph capturable once afno_plan_warmup() has run for the descriptor's (H, W).
 *
 * Errors: every call returns an afno_status_t; nothing aborts or throws.  A human-readable
 * reason for the calling thread's last failure is available from afno_last_error().
 */
#ifndef AFNO_H
#define AFNO_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  AFNO_OK = 0,
  AFNO_ERR_INVALID_ARG = 1, /* null/misaligned/aliased pointer, bad dims, bad lambda/fraction */
  AFNO_ERR_UNSUPPORTED = 2, /* odd W, H or W with a prime factor > 5, size beyond smem limits */
  AFNO_ERR_WORKSPACE = 3,   /* workspace smaller than afno_spectral_workspace_bytes()         */
  AFNO_ERR_CUDA = 4         /* a CUDA runtime call or kernel launch failed                    */
} afno_status_t;

typedef enum { AFNO_F32 = 0, AFNO_BF16 = 1 } afno_dtype_t; /* dtype of x, y, dy, dx */

enum {
  AFNO_FLAG_NO_RESIDUAL = 1,     /* test aid: y = s, dx = branch only (no "+ x", no "+ dy")   */
  AFNO_FLAG_ACCUM_GRADS = 2,     /* dw1, db1, dw2, db2 += instead of =                        */
  AFNO_FLAG_FORCE_FP32_MATH = 4, /* bf16 I/O but fp32 FFT + fp32 FFMA MLP (generic path)      */
  AFNO_FLAG_EXPORT_MASKS = 8,    /* bwd only: write ReLU / softshrink masks, see below        */
  /* Saved context (SURVEY.md S8(a) row B1 "or load saved context"): a training step calls fwd
   * and then bwd on the same x.  fwd with SAVE_CONTEXT needs a workspace of
   * afno_spectral_workspace_bytes(d, 1) bytes and leaves in it the spectrum Xh (rows F1-F2), the
   * hidden activations O1 (F3-F4), the ReLU / softshrink masks (F4, F6; bit-packed) and the bf16
   * operand images of w1, b1, w2, b2; bwd with USE_CONTEXT on the SAME workspace, with the same
   * descriptor (the two context flags aside), the same x and the same parameter values, reads
   * them instead of recomputing rows B1 (F1-F5) and is bit-identical to the stateless bwd.
   * Nothing else may write the workspace in between.  Kernel families that keep no such
   * intermediate (generic-fp32) accept both flags and recompute.  SAVE_CONTEXT is a flag of fwd,
   * USE_CONTEXT of bwd (the other call, or both at once: AFNO_ERR_INVALID_ARG).  fwd records what it
   * saved (geometry, lambda, chunking, EXPORT_MASKS, which moves the layout) in a header; a bwd
   * whose descriptor does not match it, or a workspace that was never saved, yields dx and
   * gradients that are all NaN instead of plausible numbers.  Other parameter VALUES than the
   * ones saved with cannot be detected. */
  AFNO_FLAG_SAVE_CONTEXT = 16,
  AFNO_FLAG_USE_CONTEXT = 32
};

typedef struct {
  int32_t B, H, W, C;     /* x is [B][H][W][C], channel-last, C fastest                      */
  int32_t num_blocks;     /* C % num_blocks == 0; bs = C / num_blocks                        */
  int32_t hidden_factor;  /* hid = bs * hidden_factor, >= 1                                  */
  float lambda;           /* softshrink threshold, >= 0                                      */
  float kept_fraction;    /* f in (0,1]; products with it are evaluated in double            */
  int32_t dtype;          /* afno_dtype_t                                                    */
  uint32_t flags;         /* AFNO_FLAG_*                                                     */
} afno_desc_t;

int afno_version(void);
const char* afno_status_string(int status);
const char* afno_last_error(void); /* thread-local, valid until the thread's next call */

/* Name of the kernel family the descriptor dispatches to: "tcgen05-bf16" (every transform and MLP layer a
 * tensor-core GEMM: bf16, blocks dividing 96, hidden factor 1, H <= 96, W/2+1 <= 96), "hybrid-fft32-tcgen05"
 * (bf16 activations beyond those limits: fp32 FFTs on the CUDA cores, the block MLP, its gradient stages and the
 * parameter gradients on the tensor cores, hidden factors 1..8; the spectra between its kernels are stored as bf16
 * complex when H and W are among 90 / 180 / 360 / 720 / 1,440 and C % 64 == 0, as fp32 complex otherwise)
 * or "generic-fp32".  Returns NULL for an invalid / unsupported descriptor. */
const char* afno_spectral_path(const afno_desc_t* d);

/* Pure host arithmetic; 0 for an invalid descriptor. */
size_t afno_spectral_workspace_bytes(const afno_desc_t* d, int for_backward);

/* Sizes in bytes of the two mask arrays written by AFNO_FLAG_EXPORT_MASKS:
 *   mask1 [B][H][Wh][num_blocks*hid][2] uint8 : 1 where Re/Im P1 > 0      (ReLU passes)
 *   mask2 [B][H][Wh][C][2]              uint8 : 1 where |Re/Im P2| > lambda and (r,c) kept
 * They are written at workspace + 0 and workspace + mask1_bytes (rounded up to 256) and
 * remain valid after afno_spectral_bwd returns (stream order). */
int afno_spectral_mask_bytes(const afno_desc_t* d, size_t* mask1_bytes, size_t* mask2_offset,
                             size_t* mask2_bytes);

/* Builds the per-(device, H, W) constant tables (twiddles, digit permutations, DFT
 * matrices).  Allocates and synchronises: call it outside stream capture.  fwd/bwd call it
 * implicitly on first use when the stream is not capturing. */
int afno_plan_warmup(const afno_desc_t* d);

/* Frees every plan this process has built (all devices).  No call of this library may be in
 * flight; the next fwd / bwd / afno_plan_warmup rebuilds what it needs. */
int afno_plan_destroy_all(void);

/* Forward.  x, y: [B][H][W][C] of d->dtype; y must not alias x.
 * w1 [nb][bs][hid][2], b1 [nb][hid][2], w2 [nb][hid][bs][2], b2 [nb][bs][2]: fp32,
 * out[o] = sum_i in[i] * w[j][i][o] (row vector times matrix), (re, im) fastest. */
int afno_spectral_fwd(const afno_desc_t* d, const void* x, const float* w1, const float* b1,
                      const float* w2, const float* b2, void* y, void* workspace,
                      size_t workspace_bytes, void* cuda_stream);

/* Backward (stateless: recomputes the forward spectrum from x).  dy, dx like x; dx must not
 * alias dy or x.  dw1, db1, dw2, db2: fp32, shapes of the parameters, gradients with respect
 * to the real storage (dW = dL/dRe W + i dL/dIm W = sum conj(in) * g).  Sums over samples
 * and modes are evaluated in a fixed order: two calls give bit-identical results. */
int afno_spectral_bwd(const afno_desc_t* d, const void* x, const void* dy, const float* w1,
                      const float* b1, const float* w2, const float* b2, void* dx, float* dw1,
                      float* db1, float* dw2, float* db2, void* workspace,
                      size_t workspace_bytes, void* cuda_stream);

/* End-to-end variants with HOST buffers (pinned memory recommended).  `arena` is a device
 * scratch buffer of at least afno_spectral_host_arena_bytes(); the calls copy the inputs
 * host->device, run the device path above, copy the results device->host and synchronise
 * before returning.  Every *_host pointer is a host pointer (pinned memory lets the copies
 * overlap).  The work is pipelined over the batch: sample b+1 is copied in on an internal
 * copy stream while sample b computes on `cuda_stream` and sample b-1 is copied out on a
 * second internal stream; y and dx equal the device path's bit for bit, the parameter
 * gradients are the in-order sum of the per-sample gradients (fp32 summation order differs
 * from one batched call).  The context flags and EXPORT_MASKS have no meaning here.
 * afno_spectral_bwd_host accepts x_host == NULL: x is then taken from the arena, where the
 * afno_spectral_fwd_host call that preceded it on the SAME arena and descriptor left it (a
 * training step uploads x once).  Every host call that completes stamps the arena with the
 * B, H, W, C and dtype of the x it leaves there; with x_host == NULL the stamp must match the
 * descriptor, otherwise (fresh or foreign arena, other shape) the call returns
 * AFNO_ERR_INVALID_ARG and computes nothing.  On an error the calls first wait for the copies and
 * kernels they have already enqueued, so the caller may free its buffers at once. */
size_t afno_spectral_host_arena_bytes(const afno_desc_t* d, int for_backward); /* 0 fwd_host, 1 bwd_host, 2 step_host */
int afno_spectral_fwd_host(const afno_desc_t* d, const void* x_host, const float* w1_host,
                           const float* b1_host, const float* w2_host, const float* b2_host,
                           void* y_host, void* arena, size_t arena_bytes, void* cuda_stream);
int afno_spectral_bwd_host(const afno_desc_t* d, const void* x_host, const void* dy_host,
                           const float* w1_host, const float* b1_host, const float* w2_host,
                           const float* b2_host, void* dx_host, float* dw1_host,
                           float* db1_host, float* dw2_host, float* db2_host, void* arena,
                           size_t arena_bytes, void* cuda_stream);

/* A whole training step from HOST buffers in one call: y = fwd(x); dx, dw*, db* = bwd(x, dy) (rows F1-F9, B1-B8).
 * Per sample x and dy travel host->device back to back, the forward (which saves its context) and the backward
 * (which uses it) run as soon as their input has landed, y and dx travel device->host meanwhile: both directions of
 * the link stay busy across the forward / backward boundary.  Results equal afno_spectral_fwd_host followed by
 * afno_spectral_bwd_host bit for bit.  `arena`: at least afno_spectral_host_arena_bytes(d, 2) bytes. */
int afno_spectral_step_host(const afno_desc_t* d, const void* x_host, const void* dy_host,
                            const float* w1_host, const float* b1_host, const float* w2_host,
                            const float* b2_host, void* y_host, void* dx_host, float* dw1_host,
                            float* db1_host, float* dw2_host, float* db2_host, void* arena,
                            size_t arena_bytes, void* cuda_stream);

/* Parameter gradients of one block-diagonal complex linear layer for callers that must not allocate device memory.
 *
 * Who needs this: code that runs where cudaMalloc / cudaFree are off limits and that has no spare device buffer to
 * hand over as a workspace either.  Typical cases are an operator plugged into a framework or serving engine that
 * owns all device memory through its own pool (a raw allocation there escapes the pool's accounting and can fail
 * although the pool has room), a latency-critical loop (cudaMalloc and cudaFree may synchronise the whole device and
 * stall every other stream), and a process confined to a fixed memory reservation that is already handed out.
 * afno_spectral_bwd cannot serve them: it needs a caller workspace of afno_spectral_workspace_bytes() and plan
 * tables that the library allocates on first use.
 *
 * What it computes (rows B4 and B6 of SURVEY.md S8(a); the convention of afno_spectral_bwd above; the layer is
 * PAPER.md:115-121, the gradient reduction PAPER.md:134): for every block j < num_blocks
 *     dw[j][i][o] = sum_{m < M} conj(a[m][j*K + i]) * g[m][j*N + o]      i < K, o < N
 *     db[j][o]    = sum_{m < M} g[m][j*N + o]
 * with a = the layer's input rows (the spectrum Xh for layer 1, the hidden activations O1 for layer 2) and g = the
 * gradient at its output (G1, G2), one row per (sample, mode).  It runs the fp32 kernels the generic-fp32 path of
 * afno_spectral_bwd runs for these rows; sums are taken in a fixed order, so repeated calls agree bit for bit.
 *
 *   a   device, [M][lda] complex fp32 (re, im adjacent), lda >= num_blocks*K complex elements per row
 *   g   device, [M][ldg] complex fp32, ldg >= num_blocks*N
 *   dw  device, [num_blocks][K][N][2] fp32;  db  device, [num_blocks][N][2] fp32; neither may overlap a or g
 *   flags  0 or AFNO_FLAG_ACCUM_GRADS (dw, db += instead of =)
 *   All four pointers 8-byte aligned and owned by the caller.  M == 0 is allowed (a, g are then not read; dw, db
 *   become zero, or stay as they are with ACCUM_GRADS).
 *
 * Scratch memory: the row range is split over thread blocks and each split's partial sums go to a static array of
 * AFNO_STATIC_SCRATCH_BYTES that is part of the library's device code.  Every GPU onto which the library's code gets
 * loaded holds these bytes from then until the process exits, whether or not this function is ever called.  The
 * call itself issues no cudaMalloc, cudaFree or other allocating routine, on the first call or later.
 *   - Limit: one split's partial sums, num_blocks * (K + 1) * N * 8 bytes, must fit the array (8 blocks of 96 x 96: 0.6 MB;
 *     one block of 1,024 x 1,024: 8.4 MB).  Larger shapes return AFNO_ERR_UNSUPPORTED, the message names both sizes;
 *     nothing is launched.  Within the limit the library uses as many splits as fit, up to two per SM per block.
 *   - First call on a device: the function looks up the array's address on the current device once per device
 *     (cudaGetSymbolAddress; the CUDA runtime may load the library's device code at that moment).  Make that first
 *     call with the device current that the stream belongs to, and before any stream capture begins.
 *   - The array is shared by every call on that device and keeps the previous call's partial sums.  That is
 *     harmless for calls that follow each other on one stream: every entry is rewritten before it is read, nothing
 *     needs clearing.  Two calls that can overlap on the GPU (issued to different streams, from one host thread or
 *     several) race on the array and return garbage: serialise them, e.g. keep all calls of a device on one stream
 *     or chain them with events.  Separate processes have separate copies and do not disturb each other.
 * Errors: AFNO_ERR_INVALID_ARG (NULL / misaligned pointer, non-positive num_blocks / K / N, negative M, row stride too
 * small, unknown flag), AFNO_ERR_UNSUPPORTED (beyond the limit above, or num_blocks / tile count beyond the launch grid's 65,535),
 * AFNO_ERR_CUDA (address lookup or launch failed). */
#define AFNO_STATIC_SCRATCH_BYTES (16u << 20)
int afno_block_wgrad_static(const float* a, int32_t lda, const float* g, int32_t ldg, int64_t M, int32_t num_blocks,
                            int32_t K, int32_t N, float* dw, float* db, uint32_t flags, void* cuda_stream);

/* Number of kernel launches the last fwd / bwd call of this thread enqueued (bench.py's
 * "gpu_launches" is counted from this, not guessed). */
int afno_last_launch_count(void);

/* Measurement aid: between start and stop every kernel this thread launches through the
 * library is bracketed by CUDA events on its stream (do not use during stream capture).
 * stop synchronises the device and writes one line per kernel name into `out` (host
 * buffer of `cap` bytes): "<kernel> <launches> <total_ms>\n". */
int afno_profile_start(void);
int afno_profile_stop(char* out, size_t cap);

#ifdef __cplusplus
}
#endif
#endif /* AFNO_H */
