/*
 * afno_oracle.h -- fp64 CPU oracle for the AFNO spectral token-mixing layer.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call this
 * library.  It shares no code, header, table or helper with the CUDA path under
 * paper_2208_05419_b200/csrc/ and never imports it.
 *
 * What it computes (every formula restated from the paper / DESIGN.md reading):
 *   PAPER.md:114  (SIV-A step 1)  "An FFT spatially mixes the ... grid of tokens"
 *   PAPER.md:115-121 (step 2)     block-diagonal MLP in Fourier space, weights
 *                                 shared across tokens
 *   PAPER.md:122  (step 3)        inverse FFT back to the spatial domain
 *   PAPER.md:136  (SIV-C-b)       real-to-complex / complex-to-real FFTs batched
 *                                 over batch and feature dimensions
 *   PAPER.md:138  (SIV-C-b)       complex weights stored as real tensors with
 *                                 (re, im) the fastest index; activations act on
 *                                 real and imaginary parts independently
 * Everything the paper is silent on (ortho normalisation, sign convention, bias,
 * ReLU, softshrink, truncation box, residual, gradient convention) follows the
 * readings A1..A20 listed in DESIGN.md S3.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): brute-force 2-D DFT vs the
 * mixed-radix path, numpy.fft as a library restatement, round trip, Parseval,
 * single cosine / sine closed forms, constant-input closed form, truncation box,
 * kill switch, block/dense equivalence, batch independence, dot-product adjoint
 * identities, central finite differences, affine regime vs plain matrix products.
 * No function here is "parity unpinned".
 *
 * Layouts (host pointers, all double):
 *   x, y, dy, dx : [B][H][W][C]           channel-last, C fastest
 *   w1           : [nb][bs][hid][2]       out[o] = sum_i in[i] * w1[j][i][o]
 *   b1           : [nb][hid][2]
 *   w2           : [nb][hid][bs][2]
 *   b2           : [nb][bs][2]
 *   spectra      : [B][H][Wh][ch][2]      Wh = W/2+1, natural (unshifted) order
 *   masks        : [B][H][Wh][ch][2]      uint8, 1 = derivative passes
 */
#ifndef AFNO_ORACLE_H
#define AFNO_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  int32_t B, H, W, C;
  int32_t num_blocks;     /* C % num_blocks == 0, bs = C / num_blocks            */
  int32_t hidden_factor;  /* hid = bs * hidden_factor                            */
  double lambda;          /* softshrink threshold >= 0                           */
  double kept_fraction;   /* in (0,1]; pass the float32-rounded value the GPU got */
  int32_t no_residual;    /* 1: y = s (branch only), dx = branch only            */
  int32_t naive_dft;      /* 1: literal O(N^2) 2-D sums; 0: simple mixed-radix   */
} afno_oracle_desc;

/* Optional dumps of intermediates (any pointer may be NULL). */
typedef struct {
  double* xhat;  /* [B][H][Wh][C][2]       rfft2_ortho(x)                          */
  double* p1;    /* [B][H][Wh][nb*hid][2]  layer-1 pre-activation (kept modes)     */
  double* p2;    /* [B][H][Wh][C][2]       layer-2 pre-activation (kept modes)     */
  double* z;     /* [B][H][Wh][C][2]       after softshrink, 0 outside kept set    */
} afno_oracle_dump;

/* Kept set of DESIGN.md reading A7/A8: Kh, Kw and membership. */
void afno_oracle_kept(int H, int W, double kept_fraction, int* Kh, int* Kw);

/* rfft2 / irfft2 with "ortho" normalisation on one [H][W] real plane.
 * X: [H][Wh][2].  irfft2 follows reading A4 (C2R on non-Hermitian input). */
void afno_oracle_rfft2(int H, int W, const double* x, double* X, int naive);
void afno_oracle_irfft2(int H, int W, const double* Z, double* s, int naive);

/* 1-D complex DFT, unnormalised, sign = -1 forward / +1 inverse; in/out [n][2]. */
void afno_oracle_dft1(int n, const double* in, double* out, int sign, int naive);

int afno_oracle_fwd(const afno_oracle_desc* d, const double* x, const double* w1,
                    const double* b1, const double* w2, const double* b2, double* y,
                    const afno_oracle_dump* dump);

/* mask1_override: [B][H][Wh][nb*hid][2], mask2_override: [B][H][Wh][C][2]; NULL =
 * derive masks from the oracle's own P1 > 0 and |P2| > lambda (strict). */
int afno_oracle_bwd(const afno_oracle_desc* d, const double* x, const double* dy,
                    const double* w1, const double* b1, const double* w2,
                    const double* b2, double* dx, double* dw1, double* db1,
                    double* dw2, double* db2, const uint8_t* mask1_override,
                    const uint8_t* mask2_override, const afno_oracle_dump* dump);

/* Dense-weight variant used by the block/dense equivalence pin (PAPER.md:115
 * "block-diagonal"): w1d [C][nb*hid][2], w2d [nb*hid][C][2], same biases. */
int afno_oracle_fwd_dense(const afno_oracle_desc* d, const double* x, const double* w1d,
                          const double* b1, const double* w2d, const double* b2,
                          double* y);

int afno_oracle_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
