// Generic fp32-math path of the AFNO spectral layer: any 2/3/5-smooth H and W (W even), any
// C / num_blocks / hidden_factor, fp32 or bf16 activations.  It is the reference-accuracy
// path (rel-L2 <= 1e-5 against the fp64 oracle) and the fallback for shapes the tcgen05 path
// does not cover.
//
// Kernels (scope-table rows of DESIGN.md S1 in brackets):
//   k_wfft_fwd   [F1, B2]  W-direction real FFT, two real channels packed into one complex
//                          transform, mixed-radix 2/3/4/5 in shared memory, lane = channel pair
//   k_hfft       [F2, F7]  H-direction complex FFT (forward or inverse), lane = channel
//   k_block_gemm [F3-F6, B5, B7]  per-mode block-diagonal complex GEMM with fused
//                          bias / ReLU / softshrink / truncation / mask epilogues
//   k_wfft_inv   [F8, F9, B8]  W-direction complex-to-real inverse FFT + residual + store
//   k_mask_nonzero [B3], k_block_wgrad + k_reduce_parts [B4, B6], k_export_masks
//
// FFT data layout in shared memory: s[index * 32 + lane]; the 32 lanes of a warp hold 32
// different channels (channel-last activations make that the coalesced direction), so every
// butterfly is conflict-free and needs no shuffles; warps split the butterflies of a stage.
#include <cuda_bf16.h>

#include <mutex>
#include <type_traits>
#include <utility>

#include "afno_internal.h"

namespace afno {

namespace {

constexpr int kLanes = 32;
constexpr int kFftWarps = 8;     // H-direction transform (46 KB of shared memory per block at H = 180: 4 blocks per SM)
#ifndef AFNO_WFFT_WARPS
#define AFNO_WFFT_WARPS 16
#endif
constexpr int kWfftWarps = AFNO_WFFT_WARPS;   // W-direction transforms (92 KB per block at W = 360: 2 blocks per SM): measured 8 / 16 warps -> 0.72 / 0.48 ms forward
constexpr int kLoadBatch = 8;   // independent global loads a thread keeps in flight in the FFT kernels' load loops

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
// a + sg * i * b
__device__ __forceinline__ float2 caddi(float2 a, float2 b, float sg) {
  return make_float2(a.x - sg * b.y, a.y + sg * b.x);
}

// ---- radix butterflies: X[q'] = sum_q v[q] exp(sg 2 pi i q q'/R), sg = -1 forward, +1 inverse
template <int R>
__device__ __forceinline__ void small_dft(float2 (&v)[R], float sg);

template <>
__device__ __forceinline__ void small_dft<2>(float2 (&v)[2], float) {
  float2 a = v[0], b = v[1];
  v[0] = cadd(a, b);
  v[1] = csub(a, b);
}
template <>
__device__ __forceinline__ void small_dft<3>(float2 (&v)[3], float sg) {
  const float s3 = 0.86602540378443864676f;
  float2 t = cadd(v[1], v[2]);
  float2 d = csub(v[1], v[2]);
  float2 m = make_float2(v[0].x - 0.5f * t.x, v[0].y - 0.5f * t.y);
  d.x *= s3;
  d.y *= s3;
  v[0] = cadd(v[0], t);
  v[1] = caddi(m, d, sg);
  v[2] = caddi(m, d, -sg);
}
template <>
__device__ __forceinline__ void small_dft<4>(float2 (&v)[4], float sg) {
  float2 a = cadd(v[0], v[2]), b = csub(v[0], v[2]);
  float2 c = cadd(v[1], v[3]), d = csub(v[1], v[3]);
  v[0] = cadd(a, c);
  v[2] = csub(a, c);
  v[1] = caddi(b, d, sg);
  v[3] = caddi(b, d, -sg);
}
template <>
__device__ __forceinline__ void small_dft<5>(float2 (&v)[5], float sg) {
  const float c1 = 0.30901699437494742410f, c2 = -0.80901699437494742410f;
  const float s1 = 0.95105651629515357212f, s2 = 0.58778525229247312917f;
  float2 a1 = cadd(v[1], v[4]), a2 = cadd(v[2], v[3]);
  float2 b1 = csub(v[1], v[4]), b2 = csub(v[2], v[3]);
  float2 p = make_float2(v[0].x + c1 * a1.x + c2 * a2.x, v[0].y + c1 * a1.y + c2 * a2.y);
  float2 q = make_float2(v[0].x + c2 * a1.x + c1 * a2.x, v[0].y + c2 * a1.y + c1 * a2.y);
  float2 u = make_float2(s1 * b1.x + s2 * b2.x, s1 * b1.y + s2 * b2.y);
  float2 w = make_float2(s2 * b1.x - s1 * b2.x, s2 * b1.y - s1 * b2.y);
  v[0] = make_float2(v[0].x + a1.x + a2.x, v[0].y + a1.y + a2.y);
  v[1] = caddi(p, u, sg);
  v[4] = caddi(p, u, -sg);
  v[2] = caddi(q, w, sg);
  v[3] = caddi(q, w, -sg);
}

template <int R>
__device__ __forceinline__ void dif_butterfly(float2* s, int base, int m, int j, int tstep,
                                              const float2* __restrict__ tw, float sg, int lane) {
  float2 v[R];
#pragma unroll
  for (int q = 0; q < R; ++q) v[q] = s[(base + q * m) * kLanes + lane];
  small_dft<R>(v, sg);
  s[base * kLanes + lane] = v[0];
#pragma unroll
  for (int q = 1; q < R; ++q) {
    float2 o = v[q];
    if (j != 0) {
      float2 t = __ldg(tw + j * q * tstep); // exp(-2 pi i j q / L); uniform across the warp
      t.y *= -sg;                           // conjugate for the inverse transform
      o = cmul(o, t);
    }
    s[(base + q * m) * kLanes + lane] = o;
  }
}

// In-place DIF transform of s[n][32]; every thread of the block must call it.
__device__ void fft_inplace(float2* s, const FftPlan& p, float sg, int lane, int warp, int nwarps) {
  const int n = p.n;
  int L = n;
  for (int st = 0; st < p.nstages; ++st) {
    const int r = p.radix[st];
    const int m = L / r;
    const int tstep = n / L;
    const int nbf = n / r;
    for (int t = warp; t < nbf; t += nwarps) {
      const int blk = t / m, j = t - blk * m;
      const int base = blk * L + j;
      if (r == 4) dif_butterfly<4>(s, base, m, j, tstep, p.tw, sg, lane);
      else if (r == 2) dif_butterfly<2>(s, base, m, j, tstep, p.tw, sg, lane);
      else if (r == 3) dif_butterfly<3>(s, base, m, j, tstep, p.tw, sg, lane);
      else dif_butterfly<5>(s, base, m, j, tstep, p.tw, sg, lane);
    }
    __syncthreads();
    L = m;
  }
}

// ---- activation I/O ------------------------------------------------------------------
template <typename T>
struct ActIO;
template <>
struct ActIO<float> {
  typedef float2 raw2;
  static __device__ __forceinline__ raw2 ldraw2(const float* p) { return __ldg((const float2*)p); }
  static __device__ __forceinline__ float2 unraw2(raw2 v) { return v; }
  static __device__ __forceinline__ float ld(const float* p) { return __ldg(p); }
  static __device__ __forceinline__ float2 ld2(const float* p) { return __ldg((const float2*)p); }
  static __device__ __forceinline__ void st(float* p, float v) { *p = v; }
  static __device__ __forceinline__ void st2(float* p, float a, float b) { *(float2*)p = make_float2(a, b); }
};
template <>
struct ActIO<__nv_bfloat16> {
  typedef uint32_t raw2;
  static __device__ __forceinline__ raw2 ldraw2(const __nv_bfloat16* p) { return __ldg((const uint32_t*)p); }
  static __device__ __forceinline__ float2 unraw2(raw2 v) { return make_float2(__uint_as_float(v << 16), __uint_as_float(v & 0xFFFF0000u)); }
  static __device__ __forceinline__ float ld(const __nv_bfloat16* p) { return __bfloat162float(*p); }
  static __device__ __forceinline__ float2 ld2(const __nv_bfloat16* p) {
    return __bfloat1622float2(*(const __nv_bfloat162*)p);
  }
  static __device__ __forceinline__ void st(__nv_bfloat16* p, float v) { *p = __float2bfloat16_rn(v); }
  static __device__ __forceinline__ void st2(__nv_bfloat16* p, float a, float b) {
    *(__nv_bfloat162*)p = __floats2bfloat162_rn(a, b);
  }
};

// ---- F1 / B2: W-direction real FFT ----------------------------------------------------
// grid (ceil(C/64), H, B), block (32, kWfftWarps); smem W*32 float2.
// S[((b*H+h)*Kw + k)*C + ch] = scale * alpha? * sum_w x[b,h,w,ch] exp(-2 pi i k w / W)
template <typename T>
__global__ void __launch_bounds__(kLanes * kWfftWarps)
k_wfft_fwd(const T* __restrict__ x, float2* __restrict__ S, FftPlan pw, int H, int W, int C, int Kw,
           float scale, int alpha_weight) {
  extern __shared__ float2 smem[];
  const int lane = threadIdx.x, warp = threadIdx.y;
  const int h = blockIdx.y, b = blockIdx.z;
  const int c = blockIdx.x * 64 + 2 * lane;
  const bool pair = (c + 1 < C) && ((C & 1) == 0);
  const T* xrow = x + ((size_t)(b * H + h) * W) * C;
  // kLoadBatch independent loads in flight per thread before the first shared-memory store: a warp's loop of one
  // 128-byte load per iteration leaves 2 KB in flight per SM (measured 0.8 TB/s at 180x360)
  for (int w0 = warp; w0 < W; w0 += kWfftWarps * kLoadBatch) {
    float2 v[kLoadBatch];
#pragma unroll
    for (int u = 0; u < kLoadBatch; ++u) {
      const int w = w0 + u * kWfftWarps;
      v[u] = make_float2(0.f, 0.f);
      if (w < W) {
        if (pair) v[u] = ActIO<T>::ld2(xrow + (size_t)w * C + c);
        else {
          if (c < C) v[u].x = ActIO<T>::ld(xrow + (size_t)w * C + c);
          if (c + 1 < C) v[u].y = ActIO<T>::ld(xrow + (size_t)w * C + c + 1);
        }
      }
    }
#pragma unroll
    for (int u = 0; u < kLoadBatch; ++u) {
      const int w = w0 + u * kWfftWarps;
      if (w < W) smem[w * kLanes + lane] = v[u]; // channel c in the real part, channel c+1 in the imaginary part
    }
  }
  __syncthreads();
  fft_inplace(smem, pw, -1.f, lane, warp, kWfftWarps);
  float2* Srow = S + ((size_t)(b * H + h) * Kw) * C;
  for (int k = warp; k < Kw; k += kWfftWarps) {
    const int kn = (k == 0) ? 0 : W - k;
    float2 zk = smem[__ldg(pw.perm + k) * kLanes + lane];
    float2 zn = smem[__ldg(pw.perm + kn) * kLanes + lane];
    float sc = 0.5f * scale;
    if (alpha_weight && k != 0 && 2 * k != W) sc *= 2.f;
    // split the packed transform by Hermitian symmetry
    float2 xa = make_float2(sc * (zk.x + zn.x), sc * (zk.y - zn.y));
    float2 xb = make_float2(sc * (zk.y + zn.y), -sc * (zk.x - zn.x));
    float2* dst = Srow + (size_t)k * C + c;
    if (pair) *(float4*)dst = make_float4(xa.x, xa.y, xb.x, xb.y);
    else {
      if (c < C) dst[0] = xa;
      if (c + 1 < C) dst[1] = xb;
    }
  }
}

// ---- F2 / F7: H-direction complex FFT, in place on S[B][H][Kw][C] --------------------------
// grid (ceil(C/32), Kw, B), block (32, kFftWarps); smem H*32 float2.
__global__ void __launch_bounds__(kLanes * kFftWarps)
k_hfft(float2* __restrict__ S, FftPlan ph, int H, int Kw, int C, float sg) {
  extern __shared__ float2 smem[];
  const int lane = threadIdx.x, warp = threadIdx.y;
  const int kw = blockIdx.y, b = blockIdx.z;
  const int c = blockIdx.x * kLanes + lane;
  float2* base = S + ((size_t)b * H * Kw + kw) * C + c;
  const size_t hstride = (size_t)Kw * C;
  for (int h0 = warp; h0 < H; h0 += kFftWarps * kLoadBatch) {
    float2 v[kLoadBatch];
#pragma unroll
    for (int u = 0; u < kLoadBatch; ++u) {
      const int h = h0 + u * kFftWarps;
      v[u] = (c < C && h < H) ? base[h * hstride] : make_float2(0.f, 0.f);
    }
#pragma unroll
    for (int u = 0; u < kLoadBatch; ++u) {
      const int h = h0 + u * kFftWarps;
      if (h < H) smem[h * kLanes + lane] = v[u];
    }
  }
  __syncthreads();
  fft_inplace(smem, ph, sg, lane, warp, kFftWarps);
  if (c < C)
    for (int k = warp; k < H; k += kFftWarps) base[k * hstride] = smem[__ldg(ph.perm + k) * kLanes + lane];
}

// ---- F8 + F9 / B8: W-direction complex-to-real inverse FFT, residual, store ---------------
// out[b,h,w,ch] = res[b,h,w,ch] + scale * sum_c alpha_c Re(S[b,h,c,ch] exp(+2 pi i c w / W))
// half_interior: divide by alpha (adjoint of the forward real transform, row B8).
template <typename T>
__global__ void __launch_bounds__(kLanes * kWfftWarps)
k_wfft_inv(const float2* __restrict__ S, const T* __restrict__ res, T* __restrict__ out, FftPlan pw,
           int H, int W, int C, int Kw, float scale, int half_interior) {
  extern __shared__ float2 smem[];
  const int lane = threadIdx.x, warp = threadIdx.y;
  const int h = blockIdx.y, b = blockIdx.z;
  const int c = blockIdx.x * 64 + 2 * lane;
  const bool pair = (c + 1 < C) && ((C & 1) == 0);
  const float2* Srow = S + ((size_t)(b * H + h) * Kw) * C;
  for (int k0 = warp; k0 < W; k0 += kWfftWarps * kLoadBatch) {
    float4 t[kLoadBatch];
#pragma unroll
    for (int u = 0; u < kLoadBatch; ++u) {
      const int k = k0 + u * kWfftWarps;
      const int kk = 2 * k > W ? W - k : k;
      t[u] = make_float4(0.f, 0.f, 0.f, 0.f);
      if (k < W && kk < Kw) {
        const float2* src = Srow + (size_t)kk * C + c;
        if (pair) t[u] = __ldg((const float4*)src);
        else {
          if (c < C) { const float2 a = __ldg(src); t[u].x = a.x; t[u].y = a.y; }
          if (c + 1 < C) { const float2 a = __ldg(src + 1); t[u].z = a.x; t[u].w = a.y; }
        }
      }
    }
#pragma unroll
    for (int u = 0; u < kLoadBatch; ++u) {
      const int k = k0 + u * kWfftWarps;
      if (k >= W) continue;
      const bool mirrored = 2 * k > W;
      const int kk = mirrored ? W - k : k;
      float2 z = make_float2(0.f, 0.f);
      if (kk < Kw) {
        float2 ta = make_float2(t[u].x, t[u].y), tb = make_float2(t[u].z, t[u].w);
        if (kk == 0 || 2 * kk == W) {
          ta.y = 0.f; // reading A4: imaginary parts of the c = 0 and c = W/2 columns are discarded
          tb.y = 0.f;
        } else {
          if (half_interior) { ta.x *= 0.5f; ta.y *= 0.5f; tb.x *= 0.5f; tb.y *= 0.5f; }
          if (mirrored) { ta.y = -ta.y; tb.y = -tb.y; } // Hermitian extension
        }
        z = make_float2(ta.x - tb.y, ta.y + tb.x); // Ta + i Tb: channel c -> Re, channel c+1 -> Im
      }
      smem[k * kLanes + lane] = z;
    }
  }
  __syncthreads();
  fft_inplace(smem, pw, +1.f, lane, warp, kWfftWarps);
  const size_t rowoff = ((size_t)(b * H + h) * W) * C;
  for (int w0 = warp; pair && w0 < W; w0 += kWfftWarps * kLoadBatch) {
    float2 r[kLoadBatch];
#pragma unroll
    for (int u = 0; u < kLoadBatch; ++u) {
      const int w = w0 + u * kWfftWarps;
      r[u] = (res && w < W) ? ActIO<T>::ld2(res + rowoff + (size_t)w * C + c) : make_float2(0.f, 0.f);
    }
#pragma unroll
    for (int u = 0; u < kLoadBatch; ++u) {
      const int w = w0 + u * kWfftWarps;
      if (w >= W) continue;
      const float2 z = smem[__ldg(pw.perm + w) * kLanes + lane];
      ActIO<T>::st2(out + rowoff + (size_t)w * C + c, scale * z.x + r[u].x, scale * z.y + r[u].y);
    }
  }
  for (int w = warp; !pair && w < W; w += kWfftWarps) {
    float2 z = smem[__ldg(pw.perm + w) * kLanes + lane];
    float ya = scale * z.x, yb = scale * z.y;
    const size_t off = rowoff + (size_t)w * C + c;
    {
      if (c < C) ActIO<T>::st(out + off, ya + (res ? ActIO<T>::ld(res + off) : 0.f));
      if (c + 1 < C) ActIO<T>::st(out + off + 1, yb + (res ? ActIO<T>::ld(res + off + 1) : 0.f));
    }
  }
}

#include "fft2pass.cuh"

// ---- F3-F6 / B5 / B7: block-diagonal complex GEMM over modes ----------------------------
enum { EPI_RELU = 0, EPI_SHRINK = 1, EPI_MASK = 2, EPI_NONE = 3 };
constexpr int kGemmTM = 64, kGemmRM = 8, kGemmThreads = 256;

__device__ __forceinline__ bool row_is_kept(long long row, int H, int Kw, int Kh) {
  int h = (int)((row / Kw) % H);
  int kappa = (h <= H / 2) ? h : H - h;
  return kappa < Kh;
}
__device__ __forceinline__ float shrink1(float v, float lam) {
  float m = fabsf(v) - lam;
  return m > 0.f ? copysignf(m, v) : 0.f;
}

// out[row][j*N + o] = epi( sum_k in[row][j*K + k] * Wm[j][k][o] + bias[j][o] )
template <int EPI>
__global__ void __launch_bounds__(kGemmThreads)
k_block_gemm(const float2* __restrict__ in, int ldin, const float2* __restrict__ Wm,
             const float2* __restrict__ bias, float2* __restrict__ out, int ldout,
             const float2* __restrict__ aux, int ldaux, long long M, int K, int N, int H, int Kw,
             int Kh, float lambda) {
  extern __shared__ float2 sIn[]; // [kGemmTM][K]
  const int j = blockIdx.y;
  const long long m0 = (long long)blockIdx.x * kGemmTM;
  for (int idx = threadIdx.x; idx < kGemmTM * K; idx += kGemmThreads) {
    int r = idx / K, k = idx - r * K;
    long long row = m0 + r;
    sIn[idx] = (row < M) ? in[(size_t)row * ldin + (size_t)j * K + k] : make_float2(0.f, 0.f);
  }
  __syncthreads();
  const float2* Wj = Wm + (size_t)j * K * N;
  const int total = (kGemmTM / kGemmRM) * N;
  for (int item = threadIdx.x; item < total; item += kGemmThreads) {
    const int rg = item / N, o = item - rg * N;
    float2 acc[kGemmRM];
    const float2 bv = bias ? __ldg(bias + (size_t)j * N + o) : make_float2(0.f, 0.f);
#pragma unroll
    for (int r = 0; r < kGemmRM; ++r) acc[r] = bv;
    const float2* a0 = sIn + (size_t)rg * kGemmRM * K;
#pragma unroll 4
    for (int k = 0; k < K; ++k) {
      const float2 w = __ldg(Wj + (size_t)k * N + o);
#pragma unroll
      for (int r = 0; r < kGemmRM; ++r) {
        const float2 a = a0[r * K + k];
        acc[r].x = fmaf(a.x, w.x, acc[r].x);
        acc[r].x = fmaf(-a.y, w.y, acc[r].x);
        acc[r].y = fmaf(a.x, w.y, acc[r].y);
        acc[r].y = fmaf(a.y, w.x, acc[r].y);
      }
    }
#pragma unroll
    for (int r = 0; r < kGemmRM; ++r) {
      const long long row = m0 + rg * kGemmRM + r;
      if (row >= M) continue;
      float2 v = acc[r];
      if (EPI == EPI_RELU) {
        const bool kept = row_is_kept(row, H, Kw, Kh);
        v.x = kept ? fmaxf(v.x, 0.f) : 0.f;
        v.y = kept ? fmaxf(v.y, 0.f) : 0.f;
      } else if (EPI == EPI_SHRINK) {
        const bool kept = row_is_kept(row, H, Kw, Kh);
        v.x = kept ? shrink1(v.x, lambda) : 0.f;
        v.y = kept ? shrink1(v.y, lambda) : 0.f;
      } else if (EPI == EPI_MASK) {
        const float2 a = aux[(size_t)row * ldaux + (size_t)j * N + o];
        v.x = a.x > 0.f ? v.x : 0.f;
        v.y = a.y > 0.f ? v.y : 0.f;
      }
      out[(size_t)row * ldout + (size_t)j * N + o] = v;
    }
  }
}

// ---- B3: G2 = G (.) [Z != 0] per component (Z != 0 <=> |P2| > lambda and mode kept) --------
__global__ void k_mask_nonzero(float2* __restrict__ G, const float2* __restrict__ Z, size_t n) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (; i < n; i += stride) {
    float2 g = G[i];
    const float2 z = Z[i];
    g.x = (z.x != 0.f) ? g.x : 0.f;
    g.y = (z.y != 0.f) ? g.y : 0.f;
    G[i] = g;
  }
}

// masks in the full [B][H][Wh][ch][2] index space from the stored [B][H][Kw][ch] spectra
__global__ void k_export_masks(const float2* __restrict__ src, uint8_t* __restrict__ dst, int H,
                               int Kw, int Wh, int ch, size_t n, int positive_only) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (; i < n; i += stride) {
    const size_t row = i / ch;
    const int c = (int)(i - row * ch);
    const int kw = (int)(row % Kw);
    const size_t bh = row / Kw;
    const float2 v = src[i];
    uchar2 m;
    m.x = positive_only ? (v.x > 0.f) : (v.x != 0.f);
    m.y = positive_only ? (v.y > 0.f) : (v.y != 0.f);
    ((uchar2*)dst)[(bh * Wh + kw) * ch + c] = m;
  }
}

// Wt[j][o][i] = conj(W[j][i][o])   (W: [nb][K][N] -> Wt: [nb][N][K])
__global__ void k_transpose_conj(const float2* __restrict__ W, float2* __restrict__ Wt, int nb, int K, int N) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t n = (size_t)nb * K * N;
  if (i >= n) return;
  const int o = (int)(i % N);
  const int k = (int)((i / N) % K);
  const int j = (int)(i / ((size_t)N * K));
  float2 w = W[i];
  Wt[((size_t)j * N + o) * K + k] = make_float2(w.x, -w.y);
}

// ---- B4 / B6: parameter gradients, split over row chunks, fixed summation order ------------
// partW[s][j][i][o] = sum_{m in chunk s} conj(A[m][j*K+i]) * G[m][j*N+o];  partB[s][j][o] = sum G
constexpr int kWgTR = 16, kWgTile = 96, kWgReg = 6;
__global__ void __launch_bounds__(256)
k_block_wgrad(const float2* __restrict__ A, int lda, const float2* __restrict__ G, int ldg,
              float2* __restrict__ partW, float2* __restrict__ partB, long long M, int K, int N,
              long long rows_per_split, int ntileN) {
  __shared__ float2 sA[kWgTR][kWgTile];
  __shared__ float2 sG[kWgTR][kWgTile];
  const int s = blockIdx.x, j = blockIdx.y, nb = gridDim.y;
  const int i0 = (blockIdx.z / ntileN) * kWgTile, o0 = (blockIdx.z % ntileN) * kWgTile;
  const int to = threadIdx.x & 15, ti = threadIdx.x >> 4;
  float2 acc[kWgReg][kWgReg];
  float2 accb[kWgReg];
#pragma unroll
  for (int a = 0; a < kWgReg; ++a) {
    accb[a] = make_float2(0.f, 0.f);
#pragma unroll
    for (int c = 0; c < kWgReg; ++c) acc[a][c] = make_float2(0.f, 0.f);
  }
  const long long mbeg = (long long)s * rows_per_split;
  const long long mend = min(M, mbeg + rows_per_split);
  for (long long m0 = mbeg; m0 < mend; m0 += kWgTR) {
    for (int idx = threadIdx.x; idx < kWgTR * kWgTile; idx += 256) {
      const int r = idx / kWgTile, t = idx - r * kWgTile;
      const long long row = m0 + r;
      const bool rv = row < mend;
      sA[r][t] = (rv && i0 + t < K) ? A[(size_t)row * lda + (size_t)j * K + i0 + t] : make_float2(0.f, 0.f);
      sG[r][t] = (rv && o0 + t < N) ? G[(size_t)row * ldg + (size_t)j * N + o0 + t] : make_float2(0.f, 0.f);
    }
    __syncthreads();
#pragma unroll 4
    for (int r = 0; r < kWgTR; ++r) {
      float2 a[kWgReg], g[kWgReg];
#pragma unroll
      for (int q = 0; q < kWgReg; ++q) {
        a[q] = sA[r][ti + 16 * q];
        g[q] = sG[r][to + 16 * q];
      }
#pragma unroll
      for (int q = 0; q < kWgReg; ++q) accb[q] = cadd(accb[q], g[q]);
#pragma unroll
      for (int p = 0; p < kWgReg; ++p)
#pragma unroll
        for (int q = 0; q < kWgReg; ++q) {
          // conj(a) * g
          acc[p][q].x = fmaf(a[p].x, g[q].x, acc[p][q].x);
          acc[p][q].x = fmaf(a[p].y, g[q].y, acc[p][q].x);
          acc[p][q].y = fmaf(a[p].x, g[q].y, acc[p][q].y);
          acc[p][q].y = fmaf(-a[p].y, g[q].x, acc[p][q].y);
        }
    }
    __syncthreads();
  }
#pragma unroll
  for (int p = 0; p < kWgReg; ++p) {
    const int i = i0 + ti + 16 * p;
    if (i >= K) continue;
#pragma unroll
    for (int q = 0; q < kWgReg; ++q) {
      const int o = o0 + to + 16 * q;
      if (o < N) partW[(((size_t)s * nb + j) * K + i) * N + o] = acc[p][q];
    }
  }
  if (ti == 0 && i0 == 0) {
#pragma unroll
    for (int q = 0; q < kWgReg; ++q) {
      const int o = o0 + to + 16 * q;
      if (o < N) partB[((size_t)s * nb + j) * N + o] = accb[q];
    }
  }
}

// out[i] (+)= sum_s part[s][i], s ascending
__global__ void k_reduce_parts(const float2* __restrict__ part, float2* __restrict__ out, size_t n,
                               int S, int accumulate) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float2 acc = accumulate ? out[i] : make_float2(0.f, 0.f);
  for (int s = 0; s < S; ++s) acc = cadd(acc, part[(size_t)s * n + i]);
  out[i] = acc;
}

// ---- host-side launch helpers -----------------------------------------------------------
struct Launcher {
  cudaStream_t st;
  cudaError_t err = cudaSuccess;
  void begin(const char* name) { prof_begin(name, st); }
  void check() {
    if (err == cudaSuccess) err = cudaGetLastError();
    prof_end(st);
    count_launch();
  }
};

template <typename K>
cudaError_t set_smem(K kernel, size_t bytes) {
  if (bytes <= 48 * 1024) return cudaSuccess;
  return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

template <typename T, typename ST = float2>
void launch_wfft_fwd(Launcher& L, const Geometry& g, const Plan& p, const T* x, ST* S, bool alpha) {
  if (L.err != cudaSuccess) return;
  // the long axes (720, 1,440 points; the p -> 1 grid): three passes (N1 x 9 x 10), 16 packed lanes per row
  if (g.C % 64 == 0 && fft3_dispatch(g.W, [&](auto n1) {
        constexpr int N1 = decltype(n1)::value;
        const size_t smem3 = (size_t)g.W * 16 * sizeof(float2);
        L.err = set_smem(k_wfft_fwd3<T, N1, 9, 10, ST>, smem3);
        if (L.err != cudaSuccess) return;
        L.begin("k_wfft_fwd");
        k_wfft_fwd3<T, N1, 9, 10, ST><<<dim3(g.C / 32, g.H, g.B), 1024, smem3, L.st>>>(x, S, p.fw.tw, g.H, g.C, g.Kw, g.scale,
                                                                                      alpha ? 1 : 0);
        L.check();
      }))
    return;
  if (g.C % 64 == 0 && fft2_dispatch(g.W, [&](auto n1, auto n2, auto nw, auto narrow) {
        constexpr int N1 = decltype(n1)::value, N2 = decltype(n2)::value, NW = decltype(nw)::value;
        constexpr int LW = decltype(narrow)::value ? 16 : 32;
        const size_t smem2 = (size_t)g.W * LW * sizeof(float2);
        L.err = set_smem(k_wfft_fwd2<T, N1, N2, NW, LW, ST>, smem2);
        if (L.err != cudaSuccess) return;
        L.begin("k_wfft_fwd");
        k_wfft_fwd2<T, N1, N2, NW, LW, ST><<<dim3(g.C / (2 * LW), g.H, g.B), 32 * NW, smem2, L.st>>>(x, S, p.fw.tw, g.H, g.C, g.Kw,
                                                                                                g.scale, alpha ? 1 : 0);
        L.check();
      }))
    return;
  if constexpr (std::is_same<ST, float2>::value) {
    const size_t smem = (size_t)g.W * kLanes * sizeof(float2);
    L.err = set_smem(k_wfft_fwd<T>, smem);
    if (L.err != cudaSuccess) return;
    dim3 grid((g.C + 63) / 64, g.H, g.B), block(kLanes, kWfftWarps);
    L.begin("k_wfft_fwd");
    k_wfft_fwd<T><<<grid, block, smem, L.st>>>(x, S, p.fw, g.H, g.W, g.C, g.Kw, g.scale, alpha ? 1 : 0);
    L.check();
  } else {
    L.err = cudaErrorInvalidValue;   // the bf16 spectrum exists on the two-pass kernels only (spec16() guarantees them)
  }
}

template <typename ST = float2>
void launch_hfft(Launcher& L, const Geometry& g, const Plan& p, ST* S, int C, bool inverse) {
  if (L.err != cudaSuccess) return;
  if (C % 64 == 0 && g.H == 720) {
    // the long axis of the p -> 1 grid: three passes (8 x 9 x 10), 32 channels per tile
    const size_t smem3 = (size_t)g.H * 32 * sizeof(float2);
    L.err = inverse ? set_smem(k_hfft3<8, 9, 10, +1, ST>, smem3) : set_smem(k_hfft3<8, 9, 10, -1, ST>, smem3);
    if (L.err != cudaSuccess) return;
    L.begin("k_hfft");
    const dim3 grid(C / 32, g.Kw, g.B);
    if (inverse) k_hfft3<8, 9, 10, +1, ST><<<grid, 1024, smem3, L.st>>>(S, p.fh.tw, g.Kw, C);
    else k_hfft3<8, 9, 10, -1, ST><<<grid, 1024, smem3, L.st>>>(S, p.fh.tw, g.Kw, C);
    L.check();
    return;
  }
  if (C % 64 == 0 && fft2_dispatch(g.H, [&](auto n1, auto n2, auto, auto narrow) {
        constexpr int N1 = decltype(n1)::value, N2 = decltype(n2)::value, G = decltype(narrow)::value ? 1 : 2;
        const size_t smem2 = (size_t)g.H * 32 * G * sizeof(float2);
        L.err = inverse ? set_smem(k_hfft2<N1, N2, +1, G, ST>, smem2) : set_smem(k_hfft2<N1, N2, -1, G, ST>, smem2);
        if (L.err != cudaSuccess) return;
        L.begin("k_hfft");
        const dim3 grid(C / (32 * G), g.Kw, g.B);
        if (inverse) k_hfft2<N1, N2, +1, G, ST><<<grid, 32 * hfft2_warps(G), smem2, L.st>>>(S, p.fh.tw, g.Kw, C);
        else k_hfft2<N1, N2, -1, G, ST><<<grid, 32 * hfft2_warps(G), smem2, L.st>>>(S, p.fh.tw, g.Kw, C);
        L.check();
      }))
    return;
  if constexpr (std::is_same<ST, float2>::value) {
    const size_t smem = (size_t)g.H * kLanes * sizeof(float2);
    L.err = set_smem(k_hfft, smem);
    if (L.err != cudaSuccess) return;
    dim3 grid((C + kLanes - 1) / kLanes, g.Kw, g.B), block(kLanes, kFftWarps);
    L.begin("k_hfft");
    k_hfft<<<grid, block, smem, L.st>>>(S, p.fh, g.H, g.Kw, C, inverse ? +1.f : -1.f);
    L.check();
  } else {
    L.err = cudaErrorInvalidValue;
  }
}

template <typename T, typename ST = float2>
void launch_wfft_inv(Launcher& L, const Geometry& g, const Plan& p, const ST* S, const T* res, T* out,
                     bool half_interior) {
  if (L.err != cudaSuccess) return;
  if (g.C % 64 == 0 && fft3_dispatch(g.W, [&](auto n1) {
        constexpr int N1 = decltype(n1)::value;
        const size_t smem3 = (size_t)g.W * 16 * sizeof(float2);
        L.err = set_smem(k_wfft_inv3<T, N1, 9, 10, ST>, smem3);
        if (L.err != cudaSuccess) return;
        L.begin("k_wfft_inv");
        k_wfft_inv3<T, N1, 9, 10, ST><<<dim3(g.C / 32, g.H, g.B), 1024, smem3, L.st>>>(S, res, out, p.fw.tw, g.H, g.C, g.Kw, g.scale,
                                                                                      half_interior ? 1 : 0);
        L.check();
      }))
    return;
  if (g.C % 64 == 0 && fft2_dispatch(g.W, [&](auto n1, auto n2, auto nw, auto narrow) {
        constexpr int N1 = decltype(n1)::value, N2 = decltype(n2)::value, NW = decltype(nw)::value;
        constexpr int LW = decltype(narrow)::value ? 16 : 32;
        const size_t smem2 = (size_t)g.W * LW * sizeof(float2);
        L.err = set_smem(k_wfft_inv2<T, N1, N2, NW, LW, ST>, smem2);
        if (L.err != cudaSuccess) return;
        L.begin("k_wfft_inv");
        k_wfft_inv2<T, N1, N2, NW, LW, ST><<<dim3(g.C / (2 * LW), g.H, g.B), 32 * NW, smem2, L.st>>>(S, res, out, p.fw.tw, g.H, g.C, g.Kw,
                                                                                                g.scale, half_interior ? 1 : 0);
        L.check();
      }))
    return;
  if constexpr (std::is_same<ST, float2>::value) {
    const size_t smem = (size_t)g.W * kLanes * sizeof(float2);
    L.err = set_smem(k_wfft_inv<T>, smem);
    if (L.err != cudaSuccess) return;
    dim3 grid((g.C + 63) / 64, g.H, g.B), block(kLanes, kWfftWarps);
    L.begin("k_wfft_inv");
    k_wfft_inv<T><<<grid, block, smem, L.st>>>(S, res, out, p.fw, g.H, g.W, g.C, g.Kw, g.scale,
                                             half_interior ? 1 : 0);
    L.check();
  } else {
    L.err = cudaErrorInvalidValue;
  }
}

template <int EPI>
void launch_gemm(Launcher& L, const Geometry& g, const float2* in, int ldin, const float2* Wm,
                 const float2* bias, float2* out, int ldout, const float2* aux, int ldaux, int K, int N) {
  if (L.err != cudaSuccess) return;
  const long long M = g.rows();
  const size_t smem = (size_t)kGemmTM * K * sizeof(float2);
  L.err = set_smem(k_block_gemm<EPI>, smem);
  if (L.err != cudaSuccess) return;
  dim3 grid((unsigned)((M + kGemmTM - 1) / kGemmTM), g.nb);
  L.begin("k_block_gemm");
  k_block_gemm<EPI><<<grid, kGemmThreads, smem, L.st>>>(in, ldin, Wm, bias, out, ldout, aux, ldaux, M, K, N,
                                                       g.H, g.Kw, g.Kh, g.lambda);
  L.check();
}

int wgrad_splits(const Geometry& g) {
  const long long M = g.rows();
  long long maxS = (M + kWgTR - 1) / kWgTR;
  long long S = (2 * 148 + g.nb - 1) / g.nb;
  if (S > maxS) S = maxS;
  if (S < 1) S = 1;
  return (int)S;
}

void launch_wgrad(Launcher& L, const Geometry& g, const float2* A, int lda, const float2* G, int ldg,
                  float2* part, float* dW, float* dB, int K, int N) {
  if (L.err != cudaSuccess) return;
  const long long M = g.rows();
  const int S = wgrad_splits(g);
  long long rps = (M + S - 1) / S;
  rps = (rps + kWgTR - 1) / kWgTR * kWgTR;
  const int ntK = (K + kWgTile - 1) / kWgTile, ntN = (N + kWgTile - 1) / kWgTile;
  float2* partW = part;
  float2* partB = part + (size_t)S * g.nb * K * N;
  dim3 grid(S, g.nb, ntK * ntN);
  L.begin("k_block_wgrad");
  k_block_wgrad<<<grid, 256, 0, L.st>>>(A, lda, G, ldg, partW, partB, M, K, N, rps, ntN);
  L.check();
  if (L.err != cudaSuccess) return;
  const size_t nW = (size_t)g.nb * K * N, nB = (size_t)g.nb * N;
  L.begin("k_reduce_parts");
  k_reduce_parts<<<(unsigned)((nW + 255) / 256), 256, 0, L.st>>>(partW, (float2*)dW, nW, S, g.accum ? 1 : 0);
  L.check();
  L.begin("k_reduce_parts");
  k_reduce_parts<<<(unsigned)((nB + 255) / 256), 256, 0, L.st>>>(partB, (float2*)dB, nB, S, g.accum ? 1 : 0);
  L.check();
}

struct GenericWs {
  float2 *Xh, *O1, *Z, *G, *G1, *Wt1, *Wt2, *part;
  void* mlp;   // hybrid forward: weight images of the tensor-core MLP (tc_mlp_forward)
  size_t total;
};

// Hybrid path with every transform on the two-pass kernels: the spectra between the kernels are stored as bf16 complex
// (half the HBM traffic of the path's five round trips; the arithmetic stays fp32, the MLP operands are bf16 anyway).
bool spec16(const Geometry& g) {
  return tc_mlp_supported(g) && fft2_has(g.H) && fft2_has(g.W) && g.C % 64 == 0;
}

GenericWs carve(const Geometry& g, bool backward, char* base, size_t mask_region) {
  GenericWs w{};
  size_t off = mask_region;
  auto take = [&](size_t elems) {
    float2* p = (float2*)(base + off);
    off = align_up(off + elems * sizeof(float2), 256);
    return p;
  };
  const size_t rows = (size_t)g.rows();
  const size_t spec_elems = spec16(g) ? (rows * g.C + 1) / 2 : rows * g.C;   // in units of float2
  w.Xh = take(spec_elems);
  if (backward && tc_mlp_bwd_supported(g)) {
    // hybrid backward: the two spectra and the tensor-core MLP's own region (weight images, operand images, partial sums)
    w.G = take(spec_elems);
    w.mlp = take((tc_mlp_bwd_workspace_bytes(g) + sizeof(float2) - 1) / sizeof(float2));
    w.total = off;
    return w;
  }
  w.O1 = take(rows * g.CH);
  if (!backward && tc_mlp_supported(g)) w.mlp = take((tc_mlp_workspace_bytes(g) + sizeof(float2) - 1) / sizeof(float2));
  if (backward) {
    w.Z = take(rows * g.C);
    w.G = take(rows * g.C);
    w.G1 = take(rows * g.CH);
    w.Wt1 = take((size_t)g.nb * g.bs * g.hid);
    w.Wt2 = take((size_t)g.nb * g.bs * g.hid);
    const size_t S = (size_t)wgrad_splits(g);
    w.part = take(S * ((size_t)g.nb * g.bs * g.hid + (size_t)g.nb * (g.hid > g.bs ? g.hid : g.bs)));
  }
  w.total = off;
  return w;
}

size_t mask_region_bytes(const Geometry& g, size_t* m1, size_t* m2off) {
  const size_t b1 = (size_t)g.modes_all() * g.CH * 2, b2 = (size_t)g.modes_all() * g.C * 2;
  if (m1) *m1 = b1;
  const size_t off2 = align_up(b1, 256);
  if (m2off) *m2off = off2;
  return align_up(off2 + b2, 256);
}

template <typename T>
cudaError_t forward_t(const Geometry& g, const Plan& p, const T* x, const float* w1, const float* b1,
                      const float* w2, const float* b2, T* y, void* ws, cudaStream_t st) {
  GenericWs w = carve(g, false, (char*)ws, 0);
  Launcher L{st};
  if (spec16(g)) {
    // hybrid path, bf16 spectra: F1, F2 (two-pass fp32 FFTs), F3-F6 on the tensor cores in place, F7, F8 + F9
    SpecBf16* S = (SpecBf16*)w.Xh;
    launch_wfft_fwd<T, SpecBf16>(L, g, p, x, S, false);
    launch_hfft<SpecBf16>(L, g, p, S, g.C, false);
    if (L.err == cudaSuccess) L.err = tc_mlp_forward(g, S, true, w1, b1, w2, b2, w.mlp, L.st);
    launch_hfft<SpecBf16>(L, g, p, S, g.C, true);
    launch_wfft_inv<T, SpecBf16>(L, g, p, S, g.no_residual ? nullptr : x, y, false);
    return L.err;
  }
  launch_wfft_fwd<T>(L, g, p, x, w.Xh, false);                                      // F1
  launch_hfft(L, g, p, w.Xh, g.C, false);                                           // F2
  if (w.mlp != nullptr) {
    // hybrid path (bf16 activations): F3-F6 on the tensor cores, in place on the spectrum
    if (L.err == cudaSuccess) L.err = tc_mlp_forward(g, w.Xh, false, w1, b1, w2, b2, w.mlp, L.st);
  } else {
    launch_gemm<EPI_RELU>(L, g, w.Xh, g.C, (const float2*)w1, (const float2*)b1, w.O1, g.CH, nullptr, 0,
                          g.bs, g.hid);                                             // F3, F4
    launch_gemm<EPI_SHRINK>(L, g, w.O1, g.CH, (const float2*)w2, (const float2*)b2, w.Xh, g.C, nullptr, 0,
                            g.hid, g.bs);                                           // F5, F6
  }
  launch_hfft(L, g, p, w.Xh, g.C, true);                                            // F7
  launch_wfft_inv<T>(L, g, p, w.Xh, g.no_residual ? nullptr : x, y, false);         // F8, F9
  return L.err;
}

template <typename T>
cudaError_t backward_t(const Geometry& g, const Plan& p, const T* x, const T* dy, const float* w1,
                       const float* b1, const float* w2, const float* b2, T* dx, float* dw1, float* db1,
                       float* dw2, float* db2, void* ws, size_t mask1_bytes, size_t mask2_offset,
                       cudaStream_t st) {
  size_t m1 = 0, m2off = 0;
  const size_t mask_region = g.export_masks ? mask_region_bytes(g, &m1, &m2off) : 0;
  (void)mask1_bytes;
  (void)mask2_offset;
  GenericWs w = carve(g, true, (char*)ws, mask_region);
  Launcher L{st};
  const size_t rows = (size_t)g.rows();
  if (tc_mlp_bwd_supported(g)) {
    // hybrid path (bf16 activations, hidden factors 1..8): transforms as fp32 FFTs, rows B1 (second half) and B3-B7 on
    // the tensor cores (tc_mlp_bwd, tc_wgrad), GX replaces G in place
    uint8_t* mk1 = g.export_masks ? (uint8_t*)ws : nullptr;
    uint8_t* mk2 = g.export_masks ? (uint8_t*)ws + m2off : nullptr;
    if (spec16(g)) {
      SpecBf16 *SX = (SpecBf16*)w.Xh, *SG = (SpecBf16*)w.G;
      launch_wfft_fwd<T, SpecBf16>(L, g, p, x, SX, false);
      launch_hfft<SpecBf16>(L, g, p, SX, g.C, false);
      launch_wfft_fwd<T, SpecBf16>(L, g, p, dy, SG, true);
      launch_hfft<SpecBf16>(L, g, p, SG, g.C, false);
      if (L.err == cudaSuccess && g.export_masks) L.err = cudaMemsetAsync(ws, 0, mask_region, st);
      if (L.err == cudaSuccess) L.err = tc_mlp_backward(g, SX, SG, true, w1, b1, w2, b2, dw1, db1, dw2, db2, mk1, mk2, w.mlp, st);
      launch_hfft<SpecBf16>(L, g, p, SG, g.C, true);
      launch_wfft_inv<T, SpecBf16>(L, g, p, SG, g.no_residual ? nullptr : dy, dx, true);
      return L.err;
    }
    launch_wfft_fwd<T>(L, g, p, x, w.Xh, false);
    launch_hfft(L, g, p, w.Xh, g.C, false);
    launch_wfft_fwd<T>(L, g, p, dy, w.G, true);
    launch_hfft(L, g, p, w.G, g.C, false);
    if (L.err == cudaSuccess && g.export_masks) L.err = cudaMemsetAsync(ws, 0, mask_region, st);
    if (L.err == cudaSuccess) L.err = tc_mlp_backward(g, w.Xh, w.G, false, w1, b1, w2, b2, dw1, db1, dw2, db2, mk1, mk2, w.mlp, st);
    launch_hfft(L, g, p, w.G, g.C, true);
    launch_wfft_inv<T>(L, g, p, w.G, g.no_residual ? nullptr : dy, dx, true);
    return L.err;
  }
  // B1: recompute the forward up to Z
  launch_wfft_fwd<T>(L, g, p, x, w.Xh, false);
  launch_hfft(L, g, p, w.Xh, g.C, false);
  launch_gemm<EPI_RELU>(L, g, w.Xh, g.C, (const float2*)w1, (const float2*)b1, w.O1, g.CH, nullptr, 0, g.bs,
                        g.hid);
  launch_gemm<EPI_SHRINK>(L, g, w.O1, g.CH, (const float2*)w2, (const float2*)b2, w.Z, g.C, nullptr, 0, g.hid,
                          g.bs);
  // B2: G = alpha (.) rfft2(dy)
  launch_wfft_fwd<T>(L, g, p, dy, w.G, true);
  launch_hfft(L, g, p, w.G, g.C, false);
  if (L.err != cudaSuccess) return L.err;
  // B3: G2 = G (.) mask2
  L.begin("k_mask_nonzero");
  k_mask_nonzero<<<148 * 8, 256, 0, st>>>(w.G, w.Z, rows * g.C);
  L.check();
  if (g.export_masks) {
    if (L.err == cudaSuccess) L.err = cudaMemsetAsync(ws, 0, mask_region, st);
    if (L.err != cudaSuccess) return L.err;
    L.begin("k_export_masks");
    k_export_masks<<<148 * 8, 256, 0, st>>>(w.O1, (uint8_t*)ws, g.H, g.Kw, g.Wh, g.CH, rows * g.CH, 1);
    L.check();
    L.begin("k_export_masks");
    k_export_masks<<<148 * 8, 256, 0, st>>>(w.Z, (uint8_t*)ws + m2off, g.H, g.Kw, g.Wh, g.C, rows * g.C, 0);
    L.check();
  }
  // conjugate-transposed weights for the input-gradient GEMMs
  {
    const size_t n = (size_t)g.nb * g.bs * g.hid;
    L.begin("k_transpose_conj");
    k_transpose_conj<<<(unsigned)((n + 255) / 256), 256, 0, st>>>((const float2*)w1, w.Wt1, g.nb, g.bs, g.hid);
    L.check();
    L.begin("k_transpose_conj");
    k_transpose_conj<<<(unsigned)((n + 255) / 256), 256, 0, st>>>((const float2*)w2, w.Wt2, g.nb, g.hid, g.bs);
    L.check();
  }
  // B4: dW2 = O1^H G2, db2 = sum G2
  launch_wgrad(L, g, w.O1, g.CH, w.G, g.C, w.part, dw2, db2, g.hid, g.bs);
  // B5: G1 = mask1 (.) (G2 W2^H)      Wt2: [nb][bs][hid]
  launch_gemm<EPI_MASK>(L, g, w.G, g.C, w.Wt2, nullptr, w.G1, g.CH, w.O1, g.CH, g.bs, g.hid);
  // B6: dW1 = Xh^H G1, db1 = sum G1
  launch_wgrad(L, g, w.Xh, g.C, w.G1, g.CH, w.part, dw1, db1, g.bs, g.hid);
  // B7: GX = G1 W1^H                   Wt1: [nb][hid][bs]   (into the Z buffer)
  launch_gemm<EPI_NONE>(L, g, w.G1, g.CH, w.Wt1, nullptr, w.Z, g.C, nullptr, 0, g.hid, g.bs);
  // B8: dx = dy + irfft2(GX / alpha)
  launch_hfft(L, g, p, w.Z, g.C, true);
  launch_wfft_inv<T>(L, g, p, w.Z, g.no_residual ? nullptr : dy, dx, true);
  return L.err;
}

} // namespace

bool generic_supported(const Geometry& g, const char** why) {
  const size_t lim = 227 * 1024;
  const bool w_ok = (size_t)g.W * kLanes * sizeof(float2) <= lim || (fft2_has(g.W) && g.C % 64 == 0);
  const bool h_ok = (size_t)g.H * kLanes * sizeof(float2) <= lim;   // (720 points: 184 KB; a column of 1,440 does not fit)
  if (!w_ok || !h_ok) {
    *why = "H or W too large for the shared-memory FFT kernels (max 908; 1,440 with C a multiple of 64)";
    return false;
  }
  const int kmax = g.hid > g.bs ? g.hid : g.bs;
  if ((size_t)kGemmTM * kmax * sizeof(float2) > lim) {
    *why = "block size * hidden_factor too large for the generic GEMM tile (max 443)";
    return false;
  }
  if (g.H > 32767 || g.W > 32767) {
    *why = "H or W exceeds the permutation table range";
    return false;
  }
  return true;
}

size_t generic_workspace_bytes(const Geometry& g, bool backward) {
  const size_t mask_region = (backward && g.export_masks) ? mask_region_bytes(g, nullptr, nullptr) : 0;
  return carve(g, backward, nullptr, mask_region).total;
}

cudaError_t generic_forward(const Geometry& g, const Plan& p, const void* x, const float* w1, const float* b1,
                            const float* w2, const float* b2, void* y, void* ws, cudaStream_t st) {
  if (g.bf16)
    return forward_t<__nv_bfloat16>(g, p, (const __nv_bfloat16*)x, w1, b1, w2, b2, (__nv_bfloat16*)y, ws, st);
  return forward_t<float>(g, p, (const float*)x, w1, b1, w2, b2, (float*)y, ws, st);
}

cudaError_t generic_backward(const Geometry& g, const Plan& p, const void* x, const void* dy, const float* w1,
                             const float* b1, const float* w2, const float* b2, void* dx, float* dw1,
                             float* db1, float* dw2, float* db2, void* ws, size_t mask1_bytes,
                             size_t mask2_offset, cudaStream_t st) {
  if (g.bf16)
    return backward_t<__nv_bfloat16>(g, p, (const __nv_bfloat16*)x, (const __nv_bfloat16*)dy, w1, b1, w2, b2,
                                     (__nv_bfloat16*)dx, dw1, db1, dw2, db2, ws, mask1_bytes, mask2_offset, st);
  return backward_t<float>(g, p, (const float*)x, (const float*)dy, w1, b1, w2, b2, (float*)dx, dw1, db1, dw2,
                           db2, ws, mask1_bytes, mask2_offset, st);
}

// ---- afno_block_wgrad_static: rows B4 / B6 without a workspace -------------------------------------------------
// The same two kernels as launch_wgrad above (k_block_wgrad, then k_reduce_parts in ascending split order); the only
// difference is where the split partial sums live.  They sit in the array below, which is part of the library's
// device image: the driver places it when the module is loaded onto a device and releases it when the process ends,
// so a call needs no cudaMalloc and no caller workspace.  Every call on a device uses the same bytes.  Nothing in
// it has to start at zero: k_block_wgrad writes every (split, block, i < K, o < N) entry it owns, also for a split
// whose row range is empty, before k_reduce_parts reads any of them, so what an earlier call left there is dead.
static __device__ __align__(256) unsigned char s_wgrad_scratch[AFNO_STATIC_SCRATCH_BYTES];

namespace {
// In host code `s_wgrad_scratch` is only a handle for the runtime, not an address a kernel may be given.  The device
// address differs per device and is looked up once per device, with that device current, by cudaGetSymbolAddress
// (which also makes the runtime load this module onto the device if nothing of it has run there yet).
constexpr int kMaxDevices = 64;
std::mutex s_scratch_mutex;
float2* s_scratch_addr[kMaxDevices] = {};

cudaError_t static_scratch(float2** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(s_scratch_mutex);
  if (s_scratch_addr[dev] == nullptr) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, s_wgrad_scratch);
    if (e != cudaSuccess) return e;
    s_scratch_addr[dev] = (float2*)p;
  }
  *out = s_scratch_addr[dev];
  return cudaSuccess;
}
} // namespace

size_t wgrad_static_split_bytes(int nb, int K, int N) {
  return (size_t)nb * ((size_t)K * N + (size_t)N) * sizeof(float2);
}

// The caller (afno_api.cu) has checked the arguments and that one split fits the array.
cudaError_t generic_wgrad_static(const float2* A, int lda, const float2* G, int ldg, long long M, int nb, int K, int N,
                                 float* dW, float* dB, bool accum, cudaStream_t st) {
  float2* part = nullptr;
  cudaError_t e = static_scratch(&part);
  if (e != cudaSuccess) return e;
  // splits: two waves of CTAs over the SMs like wgrad_splits(), at least 16 rows each, and no more than fit the array
  long long S = (2 * 148 + nb - 1) / nb;
  const long long maxS = (M + kWgTR - 1) / kWgTR;
  const long long fit = (long long)(kStaticScratchBytes / wgrad_static_split_bytes(nb, K, N));
  if (S > maxS) S = maxS;
  if (S > fit) S = fit;
  if (S < 1) S = 1;
  long long rps = (M + S - 1) / S;
  rps = (rps + kWgTR - 1) / kWgTR * kWgTR;
  const int ntK = (K + kWgTile - 1) / kWgTile, ntN = (N + kWgTile - 1) / kWgTile;
  float2* partW = part;
  float2* partB = part + (size_t)S * nb * K * N;
  Launcher L{st};
  L.begin("k_block_wgrad");
  k_block_wgrad<<<dim3((unsigned)S, nb, ntK * ntN), 256, 0, L.st>>>(A, lda, G, ldg, partW, partB, M, K, N, rps, ntN);
  L.check();
  if (L.err != cudaSuccess) return L.err;
  const size_t nW = (size_t)nb * K * N, nB = (size_t)nb * N;
  L.begin("k_reduce_parts");
  k_reduce_parts<<<(unsigned)((nW + 255) / 256), 256, 0, L.st>>>(partW, (float2*)dW, nW, (int)S, accum ? 1 : 0);
  L.check();
  L.begin("k_reduce_parts");
  k_reduce_parts<<<(unsigned)((nB + 255) / 256), 256, 0, L.st>>>(partB, (float2*)dB, nB, (int)S, accum ? 1 : 0);
  L.check();
  return L.err;
}

} // namespace afno
