/*
 * afno_oracle.c -- plain, slow, fp64 CPU oracle for the AFNO spectral layer.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT (see afno_oracle.h for who may call it and for
 * the list of pins).  Written from PAPER.md SIV-A steps 1-3 (lines 112-122) and
 * SIV-C-b (lines 136-138) plus the readings A1..A20 of DESIGN.md S3.  It follows
 * the definition in the order the paper states it: transform, per-mode
 * block-diagonal MLP, inverse transform, residual.  No blocking, no fusion.
 *
 * Index names follow DESIGN.md: h,r in [0,H) (row, row frequency), w in [0,W),
 * c in [0,Wh) (column frequency, Wh = W/2+1), ch = j*bs + i (channel), o (output
 * feature inside a block).
 */
#include "afno_oracle.h"

#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double _Complex cplx;

static const double TWO_PI = 6.283185307179586476925286766559;

int afno_oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------------- */
/* 1-D transforms                                                             */
/* ------------------------------------------------------------------------- */

/* tab[k] = exp(sign * 2 pi i k / n), k = 0..n-1, angles reduced before cexp. */
static cplx* root_table(int n, int sign) {
  cplx* tab = (cplx*)malloc(sizeof(cplx) * (size_t)n);
  for (int k = 0; k < n; ++k) {
    double a = sign * TWO_PI * (double)k / (double)n;
    tab[k] = cos(a) + I * sin(a);
  }
  return tab;
}

/* The DFT by definition: out[k] = sum_j in[j] * exp(sign 2 pi i jk/n). */
static void dft1_by_definition(int n, const cplx* tab, const cplx* in, int istride,
                               cplx* out) {
  for (int k = 0; k < n; ++k) {
    cplx acc = 0.0;
    for (int j = 0; j < n; ++j) acc += in[(size_t)j * istride] * tab[(int)(((long)j * k) % n)];
    out[k] = acc;
  }
}

/* Simple recursive mixed-radix decimation-in-time FFT (radices 2, 3, 5; any other
 * factor falls back to the definition).  tab is the root table of the TOP-level
 * length ntop; the roots of a sub-length n are tab[k * (ntop / n)].
 * out must hold n contiguous values; in is read with stride istride. */
static void fft1_rec(int n, int ntop, const cplx* tab, const cplx* in, int istride,
                     cplx* out) {
  if (n == 1) {
    out[0] = in[0];
    return;
  }
  int p = 0;
  if (n % 2 == 0) p = 2;
  else if (n % 3 == 0) p = 3;
  else if (n % 5 == 0) p = 5;
  if (p == 0) {
    /* roots of length n inside the top-level table */
    int step = ntop / n;
    for (int k = 0; k < n; ++k) {
      cplx acc = 0.0;
      for (int j = 0; j < n; ++j)
        acc += in[(size_t)j * istride] * tab[(int)((((long)j * k) % n) * step)];
      out[k] = acc;
    }
    /* out and in never alias in this file */
    return;
  }
  int m = n / p;
  /* p decimated sub-sequences in[q + p*j], transformed into out[q*m .. q*m+m) */
  for (int q = 0; q < p; ++q)
    fft1_rec(m, ntop, tab, in + (size_t)q * istride, istride * p, out + (size_t)q * m);
  /* X[k + m t] = sum_q  w_n^{q k} Y_q[k] * w_p^{q t},  k in [0,m), t in [0,p) */
  int step_n = ntop / n;
  int step_p = ntop / p;
  for (int k = 0; k < m; ++k) {
    cplx u[5], v[5];
    for (int q = 0; q < p; ++q) u[q] = out[(size_t)q * m + k] * tab[(q * k % n) * step_n];
    for (int t = 0; t < p; ++t) {
      cplx acc = 0.0;
      for (int q = 0; q < p; ++q) acc += u[q] * tab[(q * t % p) * step_p];
      v[t] = acc;
    }
    for (int t = 0; t < p; ++t) out[(size_t)k + (size_t)m * t] = v[t];
  }
}

static void dft1(int n, const cplx* tab, const cplx* in, int istride, cplx* out, int naive) {
  if (naive) dft1_by_definition(n, tab, in, istride, out);
  else fft1_rec(n, n, tab, in, istride, out);
}

void afno_oracle_dft1(int n, const double* in, double* out, int sign, int naive) {
  cplx* tab = root_table(n, sign);
  cplx* a = (cplx*)malloc(sizeof(cplx) * (size_t)n);
  cplx* b = (cplx*)malloc(sizeof(cplx) * (size_t)n);
  for (int k = 0; k < n; ++k) a[k] = in[2 * k] + I * in[2 * k + 1];
  dft1(n, tab, a, 1, b, naive);
  for (int k = 0; k < n; ++k) {
    out[2 * k] = creal(b[k]);
    out[2 * k + 1] = cimag(b[k]);
  }
  free(tab);
  free(a);
  free(b);
}

/* ------------------------------------------------------------------------- */
/* 2-D real transforms, "ortho" normalisation (reading A1), forward sign -,    */
/* inverse sign + (A2), last spatial axis halved (A3).                         */
/* ------------------------------------------------------------------------- */

typedef struct {
  int H, W, Wh;
  cplx *fH, *fW; /* forward roots  exp(-2 pi i k/n) */
  cplx *iH, *iW; /* inverse roots  exp(+2 pi i k/n) */
} plan2;

static void plan2_init(plan2* p, int H, int W) {
  p->H = H;
  p->W = W;
  p->Wh = W / 2 + 1;
  p->fH = root_table(H, -1);
  p->fW = root_table(W, -1);
  p->iH = root_table(H, +1);
  p->iW = root_table(W, +1);
}
static void plan2_free(plan2* p) {
  free(p->fH);
  free(p->fW);
  free(p->iH);
  free(p->iW);
}

/* X[r][c] = (1/sqrt(HW)) sum_h sum_w x[h][w] exp(-2 pi i (r h/H + c w/W))
 * x: [H][W] real with element stride xs; X: [H][Wh] complex, contiguous. */
static void rfft2_plane(const plan2* p, const double* x, size_t xs, cplx* X, int naive) {
  const int H = p->H, W = p->W, Wh = p->Wh;
  const double scale = 1.0 / sqrt((double)H * (double)W);
  if (naive) {
    /* the definition, literally */
    for (int r = 0; r < H; ++r)
      for (int c = 0; c < Wh; ++c) {
        cplx acc = 0.0;
        for (int h = 0; h < H; ++h) {
          cplx eh = p->fH[(int)(((long)r * h) % H)];
          cplx row = 0.0;
          for (int w = 0; w < W; ++w)
            row += x[((size_t)h * W + w) * xs] * p->fW[(int)(((long)c * w) % W)];
          acc += eh * row;
        }
        X[(size_t)r * Wh + c] = scale * acc;
      }
    return;
  }
  cplx* rowin = (cplx*)malloc(sizeof(cplx) * (size_t)W);
  cplx* rowout = (cplx*)malloc(sizeof(cplx) * (size_t)W);
  cplx* colout = (cplx*)malloc(sizeof(cplx) * (size_t)H);
  /* along W: full complex transform of the real row, keep the first Wh bins */
  for (int h = 0; h < H; ++h) {
    for (int w = 0; w < W; ++w) rowin[w] = x[((size_t)h * W + w) * xs];
    fft1_rec(W, W, p->fW, rowin, 1, rowout);
    for (int c = 0; c < Wh; ++c) X[(size_t)h * Wh + c] = rowout[c];
  }
  /* along H for every stored column */
  for (int c = 0; c < Wh; ++c) {
    fft1_rec(H, H, p->fH, X + c, Wh, colout);
    for (int r = 0; r < H; ++r) X[(size_t)r * Wh + c] = scale * colout[r];
  }
  free(rowin);
  free(rowout);
  free(colout);
}

static double alpha_of(int c, int W) {
  /* Hermitian-half weights: 1 for c = 0 and (W even) c = W/2, else 2 */
  if (c == 0) return 1.0;
  if (W % 2 == 0 && c == W / 2) return 1.0;
  return 2.0;
}

/* s[h][w] = (1/sqrt(HW)) sum_r sum_c alpha_c Re( Z[r][c] exp(+2 pi i (r h/H + c w/W)) )
 * (reading A4).  Z: [H][Wh] contiguous; s: [H][W] real with element stride ss. */
static void irfft2_plane(const plan2* p, const cplx* Z, double* s, size_t ss, int naive) {
  const int H = p->H, W = p->W, Wh = p->Wh;
  const double scale = 1.0 / sqrt((double)H * (double)W);
  if (naive) {
    for (int h = 0; h < H; ++h)
      for (int w = 0; w < W; ++w) {
        double acc = 0.0;
        for (int r = 0; r < H; ++r) {
          cplx eh = p->iH[(int)(((long)r * h) % H)];
          for (int c = 0; c < Wh; ++c) {
            cplx ew = p->iW[(int)(((long)c * w) % W)];
            acc += alpha_of(c, W) * creal(Z[(size_t)r * Wh + c] * eh * ew);
          }
        }
        s[((size_t)h * W + w) * ss] = scale * acc;
      }
    return;
  }
  /* Along H first (full complex inverse), T[h][c] = sum_r Z[r][c] e^{+2 pi i r h/H} */
  cplx* T = (cplx*)malloc(sizeof(cplx) * (size_t)H * Wh);
  cplx* colout = (cplx*)malloc(sizeof(cplx) * (size_t)H);
  for (int c = 0; c < Wh; ++c) {
    fft1_rec(H, H, p->iH, Z + c, Wh, colout);
    for (int h = 0; h < H; ++h) T[(size_t)h * Wh + c] = colout[h];
  }
  /* Along W: sum_c alpha_c Re(T[h][c] e^{+2 pi i c w/W}) equals the real part of a
   * full length-W inverse transform of the Hermitian extension U of T[h][.], where
   * the imaginary parts of U[0] and U[W/2] are dropped (they cannot contribute to a
   * real part weighted by alpha = 1). */
  cplx* U = (cplx*)malloc(sizeof(cplx) * (size_t)W);
  cplx* rowout = (cplx*)malloc(sizeof(cplx) * (size_t)W);
  for (int h = 0; h < H; ++h) {
    for (int w = 0; w < W; ++w) U[w] = 0.0;
    for (int c = 0; c < Wh; ++c) {
      cplx t = T[(size_t)h * Wh + c];
      if (alpha_of(c, W) == 1.0) {
        U[c] = creal(t);
      } else {
        U[c] = t;
        U[W - c] = conj(t);
      }
    }
    fft1_rec(W, W, p->iW, U, 1, rowout);
    for (int w = 0; w < W; ++w) s[((size_t)h * W + w) * ss] = scale * creal(rowout[w]);
  }
  free(T);
  free(colout);
  free(U);
  free(rowout);
}

void afno_oracle_rfft2(int H, int W, const double* x, double* X, int naive) {
  plan2 p;
  plan2_init(&p, H, W);
  rfft2_plane(&p, x, 1, (cplx*)X, naive);
  plan2_free(&p);
}

void afno_oracle_irfft2(int H, int W, const double* Z, double* s, int naive) {
  plan2 p;
  plan2_init(&p, H, W);
  irfft2_plane(&p, (const cplx*)Z, s, 1, naive);
  plan2_free(&p);
}

/* ------------------------------------------------------------------------- */
/* Kept set (readings A7, A8)                                                  */
/* ------------------------------------------------------------------------- */

void afno_oracle_kept(int H, int W, double f, int* Kh, int* Kw) {
  int nh = H / 2 + 1, nw = W / 2 + 1;
  int kh = (int)floor(f * (double)nh);
  int kw = (int)floor(f * (double)nw);
  if (kh < 1) kh = 1;
  if (kh > nh) kh = nh;
  if (kw < 1) kw = 1;
  if (kw > nw) kw = nw;
  *Kh = kh;
  *Kw = kw;
}

static int is_kept(int r, int c, int H, int Kh, int Kw) {
  int kappa = (r <= H / 2) ? r : r - H; /* signed row frequency */
  if (kappa < 0) kappa = -kappa;
  return kappa < Kh && c < Kw;
}

/* ------------------------------------------------------------------------- */
/* Per-sample pieces                                                           */
/* ------------------------------------------------------------------------- */

/* spectrum of every channel of one sample: xs [H][W][C] -> S [H][Wh][C] complex;
 * if alpha_weight, S is multiplied by alpha_c (row B2 of the scope table). */
static void sample_rfft2(const plan2* p, int C, const double* xs, cplx* S, int naive,
                         int alpha_weight) {
  const int H = p->H, W = p->W, Wh = p->Wh;
#pragma omp parallel
  {
    cplx* X = (cplx*)malloc(sizeof(cplx) * (size_t)H * Wh);
#pragma omp for schedule(static)
    for (int ch = 0; ch < C; ++ch) {
      rfft2_plane(p, xs + ch, (size_t)C, X, naive);
      for (int r = 0; r < H; ++r)
        for (int c = 0; c < Wh; ++c) {
          double a = alpha_weight ? alpha_of(c, W) : 1.0;
          S[((size_t)r * Wh + c) * C + ch] = a * X[(size_t)r * Wh + c];
        }
    }
    free(X);
  }
}

/* out[h][w][ch] (+)= irfft2 of channel ch of S (optionally divided by alpha_c) */
static void sample_irfft2(const plan2* p, int C, const cplx* S, double* out, int naive,
                          int divide_alpha, int accumulate) {
  const int H = p->H, W = p->W, Wh = p->Wh;
#pragma omp parallel
  {
    cplx* Z = (cplx*)malloc(sizeof(cplx) * (size_t)H * Wh);
    double* s = (double*)malloc(sizeof(double) * (size_t)H * W);
#pragma omp for schedule(static)
    for (int ch = 0; ch < C; ++ch) {
      for (int r = 0; r < H; ++r)
        for (int c = 0; c < Wh; ++c) {
          double a = divide_alpha ? alpha_of(c, W) : 1.0;
          Z[(size_t)r * Wh + c] = S[((size_t)r * Wh + c) * C + ch] / a;
        }
      irfft2_plane(p, Z, s, 1, naive);
      for (size_t t = 0; t < (size_t)H * W; ++t) {
        if (accumulate) out[t * C + ch] += s[t];
        else out[t * C + ch] = s[t];
      }
    }
    free(Z);
    free(s);
  }
}

/* split ReLU ("act on real and imaginary parts independently") */
static cplx relu_split(cplx v) {
  double a = creal(v), b = cimag(v);
  return (a > 0.0 ? a : 0.0) + I * (b > 0.0 ? b : 0.0);
}
/* S_lambda(v) = sign(v) max(|v| - lambda, 0), per component (reading A6) */
static double shrink1(double v, double lam) {
  double m = fabs(v) - lam;
  if (m <= 0.0) return 0.0;
  return v > 0.0 ? m : -m;
}
static cplx shrink_split(cplx v, double lam) {
  return shrink1(creal(v), lam) + I * shrink1(cimag(v), lam);
}

/* ------------------------------------------------------------------------- */
/* Forward                                                                     */
/* ------------------------------------------------------------------------- */

static int check_desc(const afno_oracle_desc* d) {
  if (!d) return 1;
  if (d->B <= 0 || d->H <= 0 || d->W <= 0 || d->C <= 0) return 1;
  if (d->num_blocks <= 0 || d->C % d->num_blocks != 0) return 1;
  if (d->hidden_factor <= 0) return 1;
  if (!(d->lambda >= 0.0)) return 1;
  if (!(d->kept_fraction > 0.0 && d->kept_fraction <= 1.0)) return 1;
  return 0;
}

/* The MLP of one sample on all kept modes.
 *   P1[o] = sum_i Xh[j*bs+i] W1[j,i,o] + b1[j,o];  O1 = relu_split(P1)
 *   P2[o] = sum_i O1[i]     W2[j,i,o] + b2[j,o];   Z  = shrink_split(P2)
 * Outside the kept set Z = 0 exactly (reading A9) and P1 = P2 = O1 = 0.
 * Arrays are [H*Wh][nb*hid] (P1, O1) and [H*Wh][C] (P2, Z). */
static void sample_mlp(const afno_oracle_desc* d, int Kh, int Kw, const cplx* Xh,
                       const cplx* W1, const cplx* B1, const cplx* W2, const cplx* B2,
                       cplx* P1, cplx* O1, cplx* P2, cplx* Z) {
  const int H = d->H, Wh = d->W / 2 + 1, C = d->C, nb = d->num_blocks;
  const int bs = C / nb, hid = bs * d->hidden_factor, CH = nb * hid;
  const long M = (long)H * Wh;
#pragma omp parallel for schedule(static)
  for (long m = 0; m < M; ++m) {
    int r = (int)(m / Wh), c = (int)(m % Wh);
    cplx* p1 = P1 + (size_t)m * CH;
    cplx* o1 = O1 + (size_t)m * CH;
    cplx* p2 = P2 + (size_t)m * C;
    cplx* z = Z + (size_t)m * C;
    if (!is_kept(r, c, H, Kh, Kw)) {
      for (int t = 0; t < CH; ++t) p1[t] = o1[t] = 0.0;
      for (int t = 0; t < C; ++t) p2[t] = z[t] = 0.0;
      continue;
    }
    const cplx* xh = Xh + (size_t)m * C;
    for (int j = 0; j < nb; ++j) {
      for (int o = 0; o < hid; ++o) p1[j * hid + o] = B1[j * hid + o];
      for (int i = 0; i < bs; ++i) {
        cplx a = xh[j * bs + i];
        const cplx* wrow = W1 + ((size_t)j * bs + i) * hid;
        for (int o = 0; o < hid; ++o) p1[j * hid + o] += a * wrow[o];
      }
      for (int o = 0; o < hid; ++o) o1[j * hid + o] = relu_split(p1[j * hid + o]);
      for (int o = 0; o < bs; ++o) p2[j * bs + o] = B2[j * bs + o];
      for (int i = 0; i < hid; ++i) {
        cplx a = o1[j * hid + i];
        const cplx* wrow = W2 + ((size_t)j * hid + i) * bs;
        for (int o = 0; o < bs; ++o) p2[j * bs + o] += a * wrow[o];
      }
      for (int o = 0; o < bs; ++o) z[j * bs + o] = shrink_split(p2[j * bs + o], d->lambda);
    }
  }
}

static void dump_copy(double* dst, const cplx* src, size_t per_sample, int b) {
  if (!dst) return;
  memcpy(dst + (size_t)b * per_sample * 2, src, sizeof(cplx) * per_sample);
}

int afno_oracle_fwd(const afno_oracle_desc* d, const double* x, const double* w1,
                    const double* b1, const double* w2, const double* b2, double* y,
                    const afno_oracle_dump* dump) {
  if (check_desc(d) || !x || !w1 || !b1 || !w2 || !b2 || !y) return 1;
  const int H = d->H, W = d->W, Wh = W / 2 + 1, C = d->C, nb = d->num_blocks;
  const int bs = C / nb, hid = bs * d->hidden_factor, CH = nb * hid;
  const size_t M = (size_t)H * Wh, N = (size_t)H * W * C;
  int Kh, Kw;
  afno_oracle_kept(H, W, d->kept_fraction, &Kh, &Kw);
  plan2 p;
  plan2_init(&p, H, W);
  cplx* Xh = (cplx*)malloc(sizeof(cplx) * M * C);
  cplx* P1 = (cplx*)malloc(sizeof(cplx) * M * CH);
  cplx* O1 = (cplx*)malloc(sizeof(cplx) * M * CH);
  cplx* P2 = (cplx*)malloc(sizeof(cplx) * M * C);
  cplx* Z = (cplx*)malloc(sizeof(cplx) * M * C);
  for (int b = 0; b < d->B; ++b) {
    const double* xs = x + (size_t)b * N;
    double* ys = y + (size_t)b * N;
    /* step 1: FFT over the token grid */
    sample_rfft2(&p, C, xs, Xh, d->naive_dft, 0);
    /* step 2: block-diagonal MLP at every kept mode */
    sample_mlp(d, Kh, Kw, Xh, (const cplx*)w1, (const cplx*)b1, (const cplx*)w2,
               (const cplx*)b2, P1, O1, P2, Z);
    /* step 3: inverse FFT; then the residual (reading A10) */
    sample_irfft2(&p, C, Z, ys, d->naive_dft, 0, 0);
    if (!d->no_residual)
      for (size_t t = 0; t < N; ++t) ys[t] += xs[t];
    if (dump) {
      dump_copy(dump->xhat, Xh, M * C, b);
      dump_copy(dump->p1, P1, M * CH, b);
      dump_copy(dump->p2, P2, M * C, b);
      dump_copy(dump->z, Z, M * C, b);
    }
  }
  free(Xh);
  free(P1);
  free(O1);
  free(P2);
  free(Z);
  plan2_free(&p);
  (void)bs;
  return 0;
}

/* Dense-weight forward: same layer with full [C][CH] and [CH][C] complex matrices. */
int afno_oracle_fwd_dense(const afno_oracle_desc* d, const double* x, const double* w1d,
                          const double* b1, const double* w2d, const double* b2,
                          double* y) {
  if (check_desc(d) || !x || !w1d || !b1 || !w2d || !b2 || !y) return 1;
  const int H = d->H, W = d->W, Wh = W / 2 + 1, C = d->C, nb = d->num_blocks;
  const int bs = C / nb, hid = bs * d->hidden_factor, CH = nb * hid;
  const size_t M = (size_t)H * Wh, N = (size_t)H * W * C;
  const cplx* W1 = (const cplx*)w1d;
  const cplx* W2 = (const cplx*)w2d;
  const cplx* B1 = (const cplx*)b1;
  const cplx* B2 = (const cplx*)b2;
  int Kh, Kw;
  afno_oracle_kept(H, W, d->kept_fraction, &Kh, &Kw);
  plan2 p;
  plan2_init(&p, H, W);
  cplx* Xh = (cplx*)malloc(sizeof(cplx) * M * C);
  cplx* Z = (cplx*)malloc(sizeof(cplx) * M * C);
  for (int b = 0; b < d->B; ++b) {
    const double* xs = x + (size_t)b * N;
    double* ys = y + (size_t)b * N;
    sample_rfft2(&p, C, xs, Xh, d->naive_dft, 0);
#pragma omp parallel
    {
      cplx* o1 = (cplx*)malloc(sizeof(cplx) * (size_t)CH);
#pragma omp for schedule(static)
      for (long m = 0; m < (long)M; ++m) {
        int r = (int)(m / Wh), c = (int)(m % Wh);
        cplx* z = Z + (size_t)m * C;
        if (!is_kept(r, c, H, Kh, Kw)) {
          for (int t = 0; t < C; ++t) z[t] = 0.0;
          continue;
        }
        const cplx* xh = Xh + (size_t)m * C;
        for (int o = 0; o < CH; ++o) {
          cplx acc = B1[o];
          for (int i = 0; i < C; ++i) acc += xh[i] * W1[(size_t)i * CH + o];
          o1[o] = relu_split(acc);
        }
        for (int o = 0; o < C; ++o) {
          cplx acc = B2[o];
          for (int i = 0; i < CH; ++i) acc += o1[i] * W2[(size_t)i * C + o];
          z[o] = shrink_split(acc, d->lambda);
        }
      }
      free(o1);
    }
    sample_irfft2(&p, C, Z, ys, d->naive_dft, 0, 0);
    if (!d->no_residual)
      for (size_t t = 0; t < N; ++t) ys[t] += xs[t];
  }
  free(Xh);
  free(Z);
  plan2_free(&p);
  return 0;
}

/* ------------------------------------------------------------------------- */
/* Backward (rows B1-B8 of the scope table; gradient convention reading A13:   */
/* gradients with respect to the real storage, dP := dL/dRe P + i dL/dIm P).   */
/* ------------------------------------------------------------------------- */

int afno_oracle_bwd(const afno_oracle_desc* d, const double* x, const double* dy,
                    const double* w1, const double* b1, const double* w2,
                    const double* b2, double* dx, double* dw1, double* db1,
                    double* dw2, double* db2, const uint8_t* mask1_override,
                    const uint8_t* mask2_override, const afno_oracle_dump* dump) {
  if (check_desc(d) || !x || !dy || !w1 || !b1 || !w2 || !b2 || !dx || !dw1 || !db1 ||
      !dw2 || !db2)
    return 1;
  const int H = d->H, W = d->W, Wh = W / 2 + 1, C = d->C, nb = d->num_blocks;
  const int bs = C / nb, hid = bs * d->hidden_factor, CH = nb * hid;
  const long M = (long)H * Wh;
  const size_t N = (size_t)H * W * C;
  const cplx* W1 = (const cplx*)w1;
  const cplx* W2 = (const cplx*)w2;
  cplx* DW1 = (cplx*)dw1;
  cplx* DB1 = (cplx*)db1;
  cplx* DW2 = (cplx*)dw2;
  cplx* DB2 = (cplx*)db2;
  int Kh, Kw;
  afno_oracle_kept(H, W, d->kept_fraction, &Kh, &Kw);
  plan2 p;
  plan2_init(&p, H, W);

  cplx* Xh = (cplx*)malloc(sizeof(cplx) * (size_t)M * C);
  cplx* P1 = (cplx*)malloc(sizeof(cplx) * (size_t)M * CH);
  cplx* O1 = (cplx*)malloc(sizeof(cplx) * (size_t)M * CH);
  cplx* P2 = (cplx*)malloc(sizeof(cplx) * (size_t)M * C);
  cplx* Z = (cplx*)malloc(sizeof(cplx) * (size_t)M * C);
  cplx* G = (cplx*)malloc(sizeof(cplx) * (size_t)M * C);   /* dL/dZ, then G2 = dL/dP2 */
  cplx* G1 = (cplx*)malloc(sizeof(cplx) * (size_t)M * CH); /* dL/dP1 */
  cplx* GX = (cplx*)malloc(sizeof(cplx) * (size_t)M * C);  /* dL/dXhat */

  for (size_t t = 0; t < (size_t)nb * bs * hid; ++t) DW1[t] = 0.0;
  for (size_t t = 0; t < (size_t)nb * hid; ++t) DB1[t] = 0.0;
  for (size_t t = 0; t < (size_t)nb * hid * bs; ++t) DW2[t] = 0.0;
  for (size_t t = 0; t < (size_t)nb * bs; ++t) DB2[t] = 0.0;

  for (int b = 0; b < d->B; ++b) {
    const double* xs = x + (size_t)b * N;
    const double* dys = dy + (size_t)b * N;
    double* dxs = dx + (size_t)b * N;
    /* B1: recompute the forward spectrum, P1, O1, P2 */
    sample_rfft2(&p, C, xs, Xh, d->naive_dft, 0);
    sample_mlp(d, Kh, Kw, Xh, W1, (const cplx*)b1, W2, (const cplx*)b2, P1, O1, P2, Z);
    /* B2: G = alpha (.) rfft2_ortho(dY)  (adjoint of the inverse transform) */
    sample_rfft2(&p, C, dys, G, d->naive_dft, 1);

    /* B3, B5, B7: per-mode chain */
#pragma omp parallel for schedule(static)
    for (long m = 0; m < M; ++m) {
      int r = (int)(m / Wh), c = (int)(m % Wh);
      cplx* g2 = G + (size_t)m * C;
      cplx* g1 = G1 + (size_t)m * CH;
      cplx* gx = GX + (size_t)m * C;
      if (!is_kept(r, c, H, Kh, Kw)) {
        for (int t = 0; t < C; ++t) g2[t] = gx[t] = 0.0;
        for (int t = 0; t < CH; ++t) g1[t] = 0.0;
        continue;
      }
      const size_t gm2 = ((size_t)b * M + m) * C;  /* mask index bases */
      const size_t gm1 = ((size_t)b * M + m) * CH;
      /* B3: softshrink mask, strict |v| > lambda per component (A14) */
      for (int t = 0; t < C; ++t) {
        cplx v = P2[(size_t)m * C + t];
        int mr, mi;
        if (mask2_override) {
          mr = mask2_override[(gm2 + t) * 2];
          mi = mask2_override[(gm2 + t) * 2 + 1];
        } else {
          mr = fabs(creal(v)) > d->lambda;
          mi = fabs(cimag(v)) > d->lambda;
        }
        g2[t] = (mr ? creal(g2[t]) : 0.0) + I * (mi ? cimag(g2[t]) : 0.0);
      }
      for (int j = 0; j < nb; ++j) {
        /* B5: G1[i] = mask1 (.) sum_o G2[o] conj(W2[j,i,o]) */
        for (int i = 0; i < hid; ++i) {
          const cplx* wrow = W2 + ((size_t)j * hid + i) * bs;
          cplx acc = 0.0;
          for (int o = 0; o < bs; ++o) acc += g2[j * bs + o] * conj(wrow[o]);
          cplx v = P1[(size_t)m * CH + j * hid + i];
          int mr, mi;
          if (mask1_override) {
            mr = mask1_override[(gm1 + j * hid + i) * 2];
            mi = mask1_override[(gm1 + j * hid + i) * 2 + 1];
          } else {
            mr = creal(v) > 0.0;
            mi = cimag(v) > 0.0;
          }
          g1[j * hid + i] = (mr ? creal(acc) : 0.0) + I * (mi ? cimag(acc) : 0.0);
        }
        /* B7: GX[i] = sum_o G1[o] conj(W1[j,i,o]) */
        for (int i = 0; i < bs; ++i) {
          const cplx* wrow = W1 + ((size_t)j * bs + i) * hid;
          cplx acc = 0.0;
          for (int o = 0; o < hid; ++o) acc += g1[j * hid + o] * conj(wrow[o]);
          gx[j * bs + i] = acc;
        }
      }
    }

    /* B4: db2[j,o] += sum_m G2 ; dW2[j,i,o] += sum_m conj(O1[i]) G2[o]
     * B6: db1[j,o] += sum_m G1 ; dW1[j,i,o] += sum_m conj(Xh[i]) G1[o]
     * one thread owns one (j,i) row of the result, modes summed in order */
#pragma omp parallel for schedule(static)
    for (int ji = 0; ji < nb * hid; ++ji) {
      int j = ji / hid;
      cplx* row = DW2 + (size_t)ji * bs;
      for (long m = 0; m < M; ++m) {
        cplx a = conj(O1[(size_t)m * CH + ji]);
        const cplx* g2 = G + (size_t)m * C + (size_t)j * bs;
        for (int o = 0; o < bs; ++o) row[o] += a * g2[o];
      }
    }
#pragma omp parallel for schedule(static)
    for (int ji = 0; ji < nb * bs; ++ji) {
      int j = ji / bs;
      cplx* row = DW1 + (size_t)ji * hid;
      for (long m = 0; m < M; ++m) {
        cplx a = conj(Xh[(size_t)m * C + ji]);
        const cplx* g1 = G1 + (size_t)m * CH + (size_t)j * hid;
        for (int o = 0; o < hid; ++o) row[o] += a * g1[o];
      }
    }
#pragma omp parallel for schedule(static)
    for (int t = 0; t < C; ++t)
      for (long m = 0; m < M; ++m) DB2[t] += G[(size_t)m * C + t];
#pragma omp parallel for schedule(static)
    for (int t = 0; t < CH; ++t)
      for (long m = 0; m < M; ++m) DB1[t] += G1[(size_t)m * CH + t];

    /* B8: dX = dY + irfft2_ortho(GX / alpha)  (adjoint of rfft2_ortho) */
    if (d->no_residual) {
      sample_irfft2(&p, C, GX, dxs, d->naive_dft, 1, 0);
    } else {
      for (size_t t = 0; t < N; ++t) dxs[t] = dys[t];
      sample_irfft2(&p, C, GX, dxs, d->naive_dft, 1, 1);
    }
    if (dump) {
      dump_copy(dump->xhat, Xh, (size_t)M * C, b);
      dump_copy(dump->p1, P1, (size_t)M * CH, b);
      dump_copy(dump->p2, P2, (size_t)M * C, b);
      dump_copy(dump->z, Z, (size_t)M * C, b);
    }
  }
  free(Xh);
  free(P1);
  free(O1);
  free(P2);
  free(Z);
  free(G);
  free(G1);
  free(GX);
  plan2_free(&p);
  return 0;
}
