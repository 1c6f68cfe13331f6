// tcgen05 (5th-generation tensor core) path of the AFNO spectral layer for bf16 activations,
// 96-wide channel blocks, H <= 96 (90 in FourCastNet's 8x8 patch grid) and W <= 190 (W/2+1 <= 96 bins).
//
// On B200 the tensor pipe is ~30x the fp32 ALU pipe, while a dense DFT of length 90 / 180 costs
// only ~20x the FLOPs of an FFT, so every transform of the layer is computed as a bf16 GEMM
// with fp32 accumulation against constant DFT matrices (S5 gives the arithmetic and
// the measured error).  The layer becomes three GEMM-chain kernels:
//
//   tc_wdft_fwd2 [F1, B2]   per (b, h, block j):  A1[(ri,kw), c] = Fw[(ri,kw), w] * x[w, c]
//   tc_mix2      [F2-F7]    per (b, kw, block j), everything on chip in tensor memory:
//                            Xh = Fh * A1  ->  relu(Xh W1 + b1)  ->  shrink(. W2 + b2)  ->  Fh^H * Z
//                [B1-B8]    the same chain run for the gradient (modes Bwd / BwdCtx), with
//   tc_wgrad     [B4, B6]   dW, db as a split-K GEMM over the mode rows
//   tc_wdft_inv2 [F8, F9, B8] per (b, h, block j): y[w, c] = x[w, c] + Gw[w, (ri,kw)] * A2[(ri,kw), c]
//
// All global traffic of these kernels moves through the copy engines (tensor-map TMA loads / stores and
// bulk copies, each with an L2 eviction policy); the kernels of a call are chained by programmatic
// dependent launch.
//
// Complex arithmetic runs as real GEMMs on separate (re | im) column halves using the
// instruction descriptor's negate bit for the minus signs, so only W_re and W_im (not the 2x2
// real block form) live in shared memory.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <type_traits>
#include <vector>

#include "afno_internal.h"
#include "tc_common.cuh"

namespace afno {

namespace {

using namespace tc;

// device side, in dependency order
#include "tc_layout.cuh"
#include "tc_wdft.cuh"
#include "tc_mix.cuh"
#include "tc_wgrad.cuh"

// ---- host side: constant operand images ------------------------------------------------------------
uint16_t host_bf16(double v) {
  float f = (float)v;
  uint32_t u;
  memcpy(&u, &f, 4);
  u += 0x7FFFu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}

cudaError_t upload(const std::vector<uint16_t>& h, uint8_t** d) {
  cudaError_t e = cudaMalloc((void**)d, h.size() * 2);
  if (e != cudaSuccess) return e;
  return cudaMemcpy(*d, h.data(), h.size() * 2, cudaMemcpyHostToDevice);
}

template <typename K>
cudaError_t set_smem(K kernel, size_t bytes) {
  return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

// ---- tensor maps (encoded per call on the host: they hold the caller's pointers) -----------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
// bf16 tensor, dims[0] fastest; strides_bytes[i] = byte stride of dims[i + 1]
bool make_tmap(const TcPlan& tp, CUtensorMap* m, const void* base, int rank, const uint64_t* dims,
               const uint64_t* strides_bytes, const uint32_t* box, bool swizzle64) {
  cuuint32_t es[5] = {1, 1, 1, 1, 1};
  cuuint64_t d[5], st[4];
  for (int i = 0; i < rank; ++i) d[i] = dims[i];
  for (int i = 0; i + 1 < rank; ++i) st[i] = strides_bytes[i];
  return ((EncodeTiledFn)tp.encode_tiled)(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, (cuuint32_t)rank, const_cast<void*>(base), d, st,
                                          box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                          swizzle64 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_NONE,
                                          CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
// activation tensor [B*H][W][C] as 64B-swizzled [192 x 32] panels (rows past W: zero-filled / not stored)
bool act_tmap(const TcPlan& tp, CUtensorMap* m, const void* ptr, const Geometry& g) {
  const uint64_t dims[3] = {(uint64_t)g.C, (uint64_t)g.W, (uint64_t)g.B * g.H};
  const uint64_t str[2] = {(uint64_t)g.C * 2, (uint64_t)g.W * g.C * 2};
  const uint32_t box[3] = {32, WP, 1};
  return make_tmap(tp, m, ptr, 3, dims, str, box, true);
}
// half-spectrum [b][kw][j][h][kA2Row] written by tc_wdft_fwd2: one box = rows kw = 0..Kw-1 of (b, j, h)
bool spec_store_tmap(const TcPlan& tp, CUtensorMap* m, const void* ptr, const Geometry& g) {
  const uint64_t row = kOutStride;
  const uint64_t dims[5] = {(uint64_t)kA2Row, (uint64_t)g.H, (uint64_t)g.nb, (uint64_t)g.Kw, (uint64_t)g.B};
  const uint64_t str[4] = {row, row * g.H, row * g.H * g.nb, row * g.H * g.nb * g.Kw};
  const uint32_t box[5] = {(uint32_t)kA2Row, 1, 1, (uint32_t)g.Kw, 1};
  return make_tmap(tp, m, ptr, 5, dims, str, box, false);
}
// the same tensor read by tc_wdft_inv2: one box = 32 channels of one (re | im) part, rows kw = 0..95
// (zero-filled past Kw), 64B-swizzled
bool spec_load_tmap(const TcPlan& tp, CUtensorMap* m, const void* ptr, const Geometry& g) {
  const uint64_t row = kOutStride;
  const uint64_t dims[5] = {32, 6, (uint64_t)g.nb * g.H, (uint64_t)g.Kw, (uint64_t)g.B};
  const uint64_t str[4] = {64, row, row * g.H * g.nb, row * g.H * g.nb * g.Kw};
  const uint32_t box[5] = {32, 1, 1, (uint32_t)BS, 1};
  return make_tmap(tp, m, ptr, 5, dims, str, box, true);
}

// the same tensor read by tc_mix2, one (b, kw, block) tile at a time: six boxes [96 rows h][32 columns]
// (rows past H zero-filled), 64B-swizzled
bool tile_tmap(const TcPlan& tp, CUtensorMap* m, const void* ptr, const Geometry& g) {
  const uint64_t row = kOutStride;
  const uint64_t dims[4] = {32, 6, (uint64_t)g.H, (uint64_t)g.B * g.Kw * g.nb};
  const uint64_t str[3] = {64, row, row * g.H};
  const uint32_t box[4] = {32, 1, (uint32_t)HP, 1};
  return make_tmap(tp, m, ptr, 4, dims, str, box, true);
}

struct TcWs {
  __nv_bfloat16 *A1, *A2, *wprep;
  float* bprep;
  __nv_bfloat16 *A1g, *Xh, *O1, *G2, *G1; // backward only
  float* part;
  uint4* maskbits;   // saved context: bit-packed activation masks, 6 KB per (b, kw, block) tile
  uint8_t *mask1, *mask2;
  size_t mask_region;
  int S;
  size_t total;
};
TcWs tc_carve(const Geometry& g, bool backward, char* base) {
  TcWs w{};
  size_t off = 0;
  auto take = [&](size_t bytes) {
    char* p = base + off;
    off = align_up(off + bytes, 256);
    return p;
  };
  if (backward && g.export_masks) {
    const size_t b1 = (size_t)g.modes_all() * g.CH * 2, b2 = (size_t)g.modes_all() * g.C * 2;
    w.mask1 = (uint8_t*)take(b1);
    w.mask2 = (uint8_t*)take(b2);
    w.mask_region = off;
  }
  const size_t spec = (size_t)g.B * g.Kw * g.nb * g.H * kA2Row * 2;
  w.A1 = (__nv_bfloat16*)take(spec);
  w.A2 = (__nv_bfloat16*)take(spec);
  w.wprep = (__nv_bfloat16*)take((size_t)g.nb * 4 * kWBytes);
  w.bprep = (float*)take((size_t)g.nb * 2 * NT * sizeof(float));
  if (backward) {
    w.A1g = (__nv_bfloat16*)take(spec);
    const size_t img = (size_t)g.B * g.Kw * g.nb * kTileBytes;   // operand-image layout
    w.Xh = (__nv_bfloat16*)take(img);
    w.O1 = (__nv_bfloat16*)take(img);
    w.G2 = (__nv_bfloat16*)take(img);
    w.G1 = (__nv_bfloat16*)take(img);
    w.maskbits = (uint4*)take((size_t)g.B * g.Kw * g.nb * 12 * 32 * sizeof(uint4));
    int S = 148 / (2 * g.nb);   // CTAs per (layer, block) of tc_wgrad
    if (S < 1) S = 1;
    if (S > g.B * g.Kw) S = g.B * g.Kw;
    w.S = S;
    w.part = (float*)take((size_t)2 * g.nb * S * kWgPartFloats * sizeof(float));
  }
  w.total = off;
  return w;
}

} // namespace

bool tc_supported(const Geometry& g) {
  return g.bf16 && g.bs == BS && g.hid == BS && g.H <= HP && g.W <= WP && g.Wh <= BS && g.C % 8 == 0;
}

cudaError_t tc_build_plan(int H, int W, TcPlan* out) {
  const double two_pi = 6.283185307179586476925286766559;
  const int Wh = W / 2 + 1;
  // Ch, Sh: element (r, h) = cos / sin (2 pi r h / H) / sqrt(H); K-major, 96 rows stored, order [k/8][m/8 < 12]
  std::vector<uint16_t> dft2(2 * kDft2Bytes / 2, 0);
  for (int r = 0; r < H; ++r)
    for (int h = 0; h < H; ++h) {
      const double a = two_pi * (double)((long)r * h % H) / (double)H, s = 1.0 / sqrt((double)H);
      const uint32_t off = ((h / 8) * kDft2Lbo + (r / 8) * kDft2Sbo + (r % 8) * 16 + (h % 8) * 2) / 2;
      dft2[off] = host_bf16(cos(a) * s);
      dft2[kDft2Bytes / 2 + off] = host_bf16(sin(a) * s);
    }
  // W-direction constants as tensor-memory A operands: logical [half a][row m < 128][96 words], word q of a
  // row = (k = 2q low half, k = 2q + 1 high half), stored in the order of cimg_word():
  //   Fw half ri: (m = kw, k = w)                  = {cos, -sin}(2 pi kw w / W) / sqrt(W)          [x alpha_kw]
  //   Gw half a : (m = w - 128 a, k = ri * 96 + kw) = alpha_kw {cos, -sin}(...) / sqrt(W)          [or alpha = 1]
  std::vector<uint16_t> fw(2 * kCImgWords, 0), fwa(2 * kCImgWords, 0), gw(2 * kCImgWords, 0), gw1(2 * kCImgWords, 0);
  auto aoff = [](int a, int m, int k) {   // 16-bit element index: word k / 2 of row m, half k % 2
    const int word = k / 2;
    return ((((size_t)a * 6 + word / 16) * 128 + m) * 16 + word % 16) * 2 + k % 2;
  };
  for (int kw = 0; kw < Wh; ++kw)
    for (int w = 0; w < W; ++w) {
      const double a = two_pi * (double)((long)kw * w % W) / (double)W, s = 1.0 / sqrt((double)W);
      const double alpha = (kw == 0 || 2 * kw == W) ? 1.0 : 2.0;
      for (int ri = 0; ri < 2; ++ri) {
        const double v = (ri == 0 ? cos(a) : -sin(a)) * s;
        const size_t of = aoff(ri, kw, w), og = aoff(w / 128, w % 128, ri * BS + kw);
        fw[of] = host_bf16(v);
        fwa[of] = host_bf16(v * alpha);
        gw[og] = host_bf16(v * alpha);
        gw1[og] = host_bf16(v);
      }
    }
  cudaError_t e = upload(dft2, &out->dft2);
  if (e == cudaSuccess) e = upload(fw, &out->fw);
  if (e == cudaSuccess) e = upload(fwa, &out->fw_alpha);
  if (e == cudaSuccess) e = upload(gw, &out->gw);
  if (e == cudaSuccess) e = upload(gw1, &out->gw_noalpha);
  if (e == cudaSuccess) e = set_smem(tc_wdft_fwd2, kWfSmem);
  if (e == cudaSuccess) e = set_smem(tc_wdft_inv2, kWiSmem);
  if (e == cudaSuccess) {
    cudaDriverEntryPointQueryResult q;
    e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &out->encode_tiled, cudaEnableDefault, &q);
    if (e == cudaSuccess && (q != cudaDriverEntryPointSuccess || out->encode_tiled == nullptr)) e = cudaErrorNotSupported;
  }
  if (e == cudaSuccess) e = set_smem(tc_mix2<kMixFwd, false>, kMix2Smem);
  if (e == cudaSuccess) e = set_smem(tc_mix2<kMixFwdSave, false>, kMix2Smem);
  if (e == cudaSuccess) e = set_smem(tc_mix2<kMixBwd, false>, kMix2Smem);
  if (e == cudaSuccess) e = set_smem(tc_mix2<kMixBwd, true>, kMix2Smem);
  if (e == cudaSuccess) e = set_smem(tc_mix2<kMixBwdCtx, false>, kMix2Smem);
  if (e == cudaSuccess) e = set_smem(tc_mix2<kMixBwdCtx, true>, kMix2Smem);
  if (e == cudaSuccess) e = set_smem(tc_wgrad, kWgSmem);
  int dev = 0, sms = 148;
  if (e == cudaSuccess) e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  out->num_sms = sms;
  out->valid = (e == cudaSuccess);
  return e;
}

// CTAs per channel block of tc_mix2 (a regular CTA works on one block)
static int mix2_split(const Geometry& g, const TcPlan& tp) {
  int S = tp.num_sms / g.nb;
  if (S < 1) S = 1;
  if (S > g.B * g.Kw) S = g.B * g.Kw;
  return S;
}
// grid of tc_mix2: nb * S regular CTAs plus, when the (b, kw) pairs do not divide by S and SMs are left
// over, spare CTAs for the remainder (see the kernel)
static int mix2_grid(const Geometry& g, const TcPlan& tp, int S) {
  const int reg = g.nb * S, left = (g.B * g.Kw) % S;
  int spare = tp.num_sms - reg;
  if (spare > g.nb) spare = g.nb;
  if (left == 0 || spare < 0 || (g.B * g.Kw) / S == 0) spare = 0;
  return reg + spare;
}

size_t tc_workspace_bytes(const Geometry& g, bool backward) {
  return tc_carve(g, backward, nullptr).total;
}

// Kernel launch with the programmatic-dependent-launch attribute: `dependent` launches may begin their
// prologue (barrier init, tensor-memory allocation, plan constants) under the tail of the previous kernel
// of the stream; the kernels order themselves with pdl_wait().  The first kernel of an API call is a
// plain launch, so the call as a whole keeps stream order with the caller's work.
static const bool g_use_pdl = getenv("AFNO_NO_PDL") == nullptr;
template <typename... KArgs, typename... Args>
static cudaError_t launch_k(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool dependent,
                            Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = (dependent && g_use_pdl) ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

// W-direction launches: tile = (b, h, block), persistent over the SMs
static cudaError_t launch_wdft_fwd(const Geometry& g, const TcPlan& tp, const void* in, void* spec, const uint8_t* fimg,
                                   cudaStream_t st, bool dependent) {
  CUtensorMap mx, ma;
  if (!act_tmap(tp, &mx, in, g) || !spec_store_tmap(tp, &ma, spec, g)) return cudaErrorInvalidValue;
  const int ntiles = g.B * g.H * g.nb;
  const int grid = ntiles < tp.num_sms ? ntiles : tp.num_sms;
  prof_begin("tc_wdft_fwd", st);
  cudaError_t e = launch_k(tc_wdft_fwd2, grid, kW2Threads, kWfSmem, st, dependent, mx, ma, (const uint32_t*)fimg, ntiles, g.nb,
                           g.H, g.Kw);
  prof_end(st);
  count_launch();
  return e != cudaSuccess ? e : cudaGetLastError();
}
static cudaError_t launch_wdft_inv(const Geometry& g, const TcPlan& tp, const void* spec, const void* res, void* out,
                                   const uint8_t* gimg, cudaStream_t st) {
  CUtensorMap ma, mr, my;
  if (!spec_load_tmap(tp, &ma, spec, g) || !act_tmap(tp, &mr, res ? res : out, g) || !act_tmap(tp, &my, out, g))
    return cudaErrorInvalidValue;
  const int ntiles = g.B * g.H * g.nb;
  const int grid = ntiles < tp.num_sms ? ntiles : tp.num_sms;
  prof_begin("tc_wdft_inv", st);
  cudaError_t e = launch_k(tc_wdft_inv2, grid, kW2Threads, kWiSmem, st, true, ma, mr, my, (const uint32_t*)gimg, ntiles, g.nb,
                           g.H, g.W, res ? 1 : 0);
  prof_end(st);
  count_launch();
  return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t tc_forward(const Geometry& g, const Plan& p, const void* x, const float* w1, const float* b1,
                       const float* w2, const float* b2, void* y, void* ws, cudaStream_t st) {
  // SAVE_CONTEXT: the backward layout, so that tc_backward finds A1 where it expects it
  TcWs w = tc_carve(g, g.save_ctx, (char*)ws);
  const TcPlan& tp = p.tc;
  cudaError_t e;
  const int nW = g.nb * BS * BS;
  prof_begin("k_tc_prep_weights", st);
  k_tc_prep_weights<<<(nW + 255) / 256, 256, 0, st>>>(w1, b1, w2, b2, w.wprep, w.bprep, g.nb);
  prof_end(st);
  count_launch();
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  if ((e = launch_wdft_fwd(g, tp, x, w.A1, tp.fw, st, true)) != cudaSuccess) return e;
  MixParams mp{};
  if (!tile_tmap(tp, &mp.mapA1, w.A1, g)) return cudaErrorInvalidValue;
  mp.mapA1g = mp.mapA1;
  mp.A2 = w.A2; mp.dft = tp.dft2; mp.wprep = (const uint8_t*)w.wprep; mp.bprep = w.bprep;
  mp.B = g.B; mp.H = g.H; mp.Kw = g.Kw; mp.Wh = g.Wh; mp.nb = g.nb; mp.Kh = g.Kh; mp.lambda = g.lambda;
  prof_begin("tc_mix_fwd", st);
  const int S2 = mix2_split(g, tp);
  if (g.save_ctx) {
    // saved context: Xh, O1 (operands of tc_wgrad) and the activation masks stay in the workspace
    mp.Xh = w.Xh; mp.O1 = w.O1; mp.maskbits = w.maskbits;
    e = launch_k(tc_mix2<kMixFwdSave, false>, mix2_grid(g, tp, S2), kMix2Threads, kMix2Smem, st, true, mp, S2);
  } else {
    e = launch_k(tc_mix2<kMixFwd, false>, mix2_grid(g, tp, S2), kMix2Threads, kMix2Smem, st, true, mp, S2);
  }
  if (e != cudaSuccess) return e;
  prof_end(st);
  count_launch();
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  return launch_wdft_inv(g, tp, w.A2, g.no_residual ? nullptr : x, y, tp.gw, st);
}

cudaError_t tc_backward(const Geometry& g, const Plan& p, const void* x, const void* dy, const float* w1,
                        const float* b1, const float* w2, const float* b2, void* dx, float* dw1, float* db1,
                        float* dw2, float* db2, void* ws, cudaStream_t st) {
  TcWs w = tc_carve(g, true, (char*)ws);
  const TcPlan& tp = p.tc;
  cudaError_t e;
  bool dep = false;   // false for the first kernel of the call only
#define TC_LAUNCH(name, ...)                                  \
  prof_begin(name, st);                                       \
  e = launch_k(__VA_ARGS__);                                  \
  prof_end(st);                                               \
  count_launch();                                             \
  dep = true;                                                 \
  if (e != cudaSuccess || (e = cudaGetLastError()) != cudaSuccess) return e;
  const int nW = g.nb * BS * BS;
  if (g.export_masks) {
    if ((e = cudaMemsetAsync(ws, 0, w.mask_region, st)) != cudaSuccess) return e;
  }
  // USE_CONTEXT: the operand images of the weights written by the forward call are still in the
  // workspace (the context belongs to one set of parameters)
  if (!g.use_ctx) {
    TC_LAUNCH("k_tc_prep_weights", k_tc_prep_weights, (nW + 255) / 256, 256, 0, st, dep, w1, b1, w2, b2, w.wprep, w.bprep, g.nb);
  }
  // B1 (first half) and B2: W-direction spectra of x and of dy (alpha-weighted)
  if (!g.use_ctx) {
    if ((e = launch_wdft_fwd(g, tp, x, w.A1, tp.fw, st, dep)) != cudaSuccess) return e;
    dep = true;
  }
  if ((e = launch_wdft_fwd(g, tp, dy, w.A1g, tp.fw_alpha, st, dep)) != cudaSuccess) return e;
  dep = true;
  MixParams mp{};
  if (!tile_tmap(tp, &mp.mapA1, w.A1, g) || !tile_tmap(tp, &mp.mapA1g, w.A1g, g)) return cudaErrorInvalidValue;
  mp.A2 = w.A2;
  mp.Xh = w.Xh; mp.O1 = w.O1; mp.G2 = w.G2; mp.G1 = w.G1;
  mp.dft = tp.dft2; mp.wprep = (const uint8_t*)w.wprep; mp.bprep = w.bprep;
  mp.mask1 = g.export_masks ? w.mask1 : nullptr;
  mp.mask2 = g.export_masks ? w.mask2 : nullptr;
  mp.B = g.B; mp.H = g.H; mp.Kw = g.Kw; mp.Wh = g.Wh; mp.nb = g.nb; mp.Kh = g.Kh; mp.lambda = g.lambda;
  const int S2 = mix2_split(g, tp);
  mp.maskbits = w.maskbits;
  if (g.use_ctx) {
    // gradient stages only: Xh, O1 and the masks were left in the workspace by the forward call
    if (g.export_masks) {
      TC_LAUNCH("tc_mix_bwd", tc_mix2<kMixBwdCtx, true>, mix2_grid(g, tp, S2), kMix2Threads, kMix2Smem, st, dep, mp, S2);
    } else {
      TC_LAUNCH("tc_mix_bwd", tc_mix2<kMixBwdCtx, false>, mix2_grid(g, tp, S2), kMix2Threads, kMix2Smem, st, dep, mp, S2);
    }
  } else if (g.export_masks) {
    TC_LAUNCH("tc_mix_bwd", tc_mix2<kMixBwd, true>, mix2_grid(g, tp, S2), kMix2Threads, kMix2Smem, st, dep, mp, S2);
  } else {
    TC_LAUNCH("tc_mix_bwd", tc_mix2<kMixBwd, false>, mix2_grid(g, tp, S2), kMix2Threads, kMix2Smem, st, dep, mp, S2);
  }
  // B4 / B6: parameter gradients
  const int nred = nW + g.nb * BS;
  TC_LAUNCH("tc_wgrad", tc_wgrad, 2 * g.nb * w.S, 128, kWgSmem, st, dep, w.O1, w.G2, w.Xh, w.G1, w.part, g.B * g.Kw, g.H,
            g.nb, w.S);
  TC_LAUNCH("k_tc_wgrad_reduce", k_tc_wgrad_reduce, dim3((nred + 255) / 256, 2), 256, 0, st, dep, w.part, (float2*)dw2,
            (float2*)db2, (float2*)dw1, (float2*)db1, g.nb, w.S, g.accum ? 1 : 0);
#undef TC_LAUNCH
  // B8: dx = dy + irfft2(GX / alpha)
  return launch_wdft_inv(g, tp, w.A2, g.no_residual ? nullptr : dy, dx, tp.gw_noalpha, st);
}

#ifdef AFNO_TRACE
extern "C" int afno_trace_read(long long* out) {
  return (int)cudaMemcpyFromSymbol(out, g_afno_trace, sizeof(long long) * 64 * 32);
}
#endif
#ifdef AFNO_POLICY_EXPERIMENT
extern "C" int afno_debug_set_policy(int mask) { return (int)cudaMemcpyToSymbol(g_polmask, &mask, sizeof(int)); }
#endif
#ifdef AFNO_TIMING
extern "C" int afno_debug_read_span(long long* out) {
  return (int)cudaMemcpyFromSymbol(out, g_afno_span, sizeof(long long) * 5 * 160 * 2);
}
extern "C" int afno_debug_read(long long* out) {
  return (int)cudaMemcpyFromSymbol(out, g_afno_dbg, sizeof(long long) * 128);
}
#endif

} // namespace afno
