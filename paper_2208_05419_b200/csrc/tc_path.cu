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
#include "tc_mlp.cuh"

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

// the geometry the kernels see: nb = number of 96-channel groups
Geometry tc_geom(const Geometry& g0) {
  Geometry g = g0;
  if (g.nb_blocks != 0) return g;   // already a group geometry
  g.nb_blocks = g0.nb;
  g.bs_block = g0.bs;
  g.nb = (g0.C + BS - 1) / BS;
  g.bs = BS;
  g.hid = BS;
  return g;
}

struct TcWs {
  CtxHeader* header;
  __nv_bfloat16 *A, *wprep;   // A: half-spectrum of ONE chunk of samples, transformed in place by tc_mix2
  float* bprep;
  __nv_bfloat16 *Ax;          // stateless backward only: spectrum of x (A then holds the gradient's)
  __nv_bfloat16 *Xh, *O1;     // whole batch (they are the saved context)
  __nv_bfloat16 *G2, *G1;     // one chunk
  float* part;
  uint4* maskbits;   // saved context: bit-packed activation masks, 6 KB per (b, kw, block) tile; whole batch
  uint8_t *mask1, *mask2;
  size_t mask_region;
  int S;
  int chunk_f, chunk_b;   // samples per chunk in the forward / backward call
  size_t total;
};

// Samples per chunk.  A call walks the batch in chunks of samples: W transform -> per-mode chain (in place)
// -> [parameter gradients ->] inverse W transform, over buffers that hold ONE chunk and are reused by the
// next, so the workspace does not grow with B.  Measured on B200 at 90x180x768, B = 4 fwd+bwd (DESIGN.md
// S5.5): chunks of 1 / 2 / 4 samples -> 0.529 / 0.494 / 0.466 ms per step.  Smaller chunks keep more of the
// half-spectra in the L2 (DRAM traffic 2.07 -> 1.84 GB) but every kernel boundary costs ~4 us of drain and
// ramp-up on these persistent pipelines, which outweighs it: the default is 4.
#ifndef AFNO_CHUNK_FWD
#define AFNO_CHUNK_FWD 4
#endif
#ifndef AFNO_CHUNK_BWD
#define AFNO_CHUNK_BWD 4
#endif
size_t spec_bytes(const Geometry& g, int B) { return (size_t)B * g.Kw * g.nb * g.H * kA2Row * 2; }
size_t img_bytes(const Geometry& g, int B) { return (size_t)B * g.Kw * g.nb * kTileBytes; }
int chunk_samples(const Geometry& g, bool backward) {
  int cb = backward ? AFNO_CHUNK_BWD : AFNO_CHUNK_FWD;
  if (cb < 1) cb = 1;
  if (cb > g.B) cb = g.B;
  return cb;
}

TcWs tc_carve(const Geometry& g0, bool backward, char* base) {
  const Geometry g = tc_geom(g0);
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
  w.header = (CtxHeader*)take(sizeof(CtxHeader));
  w.chunk_f = chunk_samples(g, false);
  w.chunk_b = chunk_samples(g, true);
  const int cmax = w.chunk_f > w.chunk_b ? w.chunk_f : w.chunk_b;
  w.wprep = (__nv_bfloat16*)take((size_t)g.nb * 4 * kWBytes);
  w.bprep = (float*)take((size_t)g.nb * 2 * NT * sizeof(float));
  w.A = (__nv_bfloat16*)take(spec_bytes(g, backward ? cmax : w.chunk_f));
  if (backward) {
    w.Xh = (__nv_bfloat16*)take(img_bytes(g, g.B));
    w.O1 = (__nv_bfloat16*)take(img_bytes(g, g.B));
    w.maskbits = (uint4*)take((size_t)g.B * g.Kw * g.nb * 12 * 32 * sizeof(uint4));
    w.G2 = (__nv_bfloat16*)take(img_bytes(g, w.chunk_b));
    w.G1 = (__nv_bfloat16*)take(img_bytes(g, w.chunk_b));
    int S = 148 / (2 * g.nb);   // CTAs per (layer, block) of tc_wgrad
    if (S < 1) S = 1;
    if (S > w.chunk_b * g.Kw) S = w.chunk_b * g.Kw;
    w.S = S;
    w.part = (float*)take((size_t)2 * g.nb * S * kWgPartFloats * sizeof(float));
    // last, so that the context layout does not depend on it: only the stateless backward uses it
    if (!g.save_ctx && !g.use_ctx) w.Ax = (__nv_bfloat16*)take(spec_bytes(g, w.chunk_b));
  }
  w.total = off;
  return w;
}

} // namespace

bool tc_plan_supported(int H, int W) { return H >= 1 && H <= HP && W >= 2 && W <= WP && W / 2 + 1 <= BS; }

// Blocks of bs channels with bs dividing 96 (96, 48, 32, 24, 16, 12, 8: the paper's own network has 32 blocks
// of 32) run as block-diagonal 96 x 96 weight images inside groups of 96 channels; a last group
// that is only partly filled (C % 96 != 0) is zero-filled / clipped by the tensor-map copies.
bool tc_supported(const Geometry& g) {
  return g.bf16 && g.bs >= 8 && BS % g.bs == 0 && g.hid == g.bs && tc_plan_supported(g.H, g.W) && g.C % 8 == 0;
}



void tc_free_plan(TcPlan* p) {
  uint8_t** tabs[] = {&p->dft2, &p->fw, &p->fw_alpha, &p->gw, &p->gw_noalpha};
  for (uint8_t** t : tabs) {
    cudaFree(*t);
    *t = nullptr;
  }
  p->valid = false;
}

cudaError_t tc_build_plan(int H, int W, TcPlan* out) {
  if (!tc_plan_supported(H, W)) return cudaErrorInvalidValue;   // the images below are sized for H <= 96, W/2+1 <= 96
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
  cfg.numAttrs = dependent ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

// ---- hybrid path: fp32 FFTs on the CUDA cores (generic.cu) + the block MLP on the tensor cores (tc_mlp.cuh) -------
bool tc_mlp_supported(const Geometry& g) {
  if (!g.bf16 || g.force_fp32 || g.C % 8 != 0) return false;
  if (g.hid == g.bs) return g.bs >= 8 && BS % g.bs == 0;
  return g.bs == BS && g.hid % BS == 0 && g.hid / BS <= kMlpMaxHf;   // hidden factor > 1: blocks of 96 only
}
size_t tc_mlp_workspace_bytes(const Geometry& g) {
  if (g.hid != g.bs) {
    const size_t hf = (size_t)g.hid / BS;
    return align_up((size_t)g.nb * hf * 4 * kWBytes, 256) + align_up((size_t)g.nb * (hf + 1) * NT * sizeof(float), 256);
  }
  const size_t groups = (size_t)(g.C + BS - 1) / BS;
  return align_up(groups * 4 * kWBytes, 256) + align_up(groups * 2 * NT * sizeof(float), 256);
}
namespace {
template <typename ST>
cudaError_t mlp_forward_launch(bool multi, int grid, cudaStream_t st, const MlpParams& mp, int S, int hf) {
  // per device and cheap: the attribute is set on every call rather than cached in a static that another device or thread would miss
  cudaError_t e = multi ? set_smem(tc_mlp_fwd_hf<ST>, kMlpHfSmem) : set_smem(tc_mlp_fwd<ST>, mlp_fwd_smem<ST>());
  if (e != cudaSuccess) return e;
  return multi ? launch_k(tc_mlp_fwd_hf<ST>, grid, kMlpThreads, kMlpHfSmem, st, true, mp, S, hf)
               : launch_k(tc_mlp_fwd<ST>, grid, kMlpThreads, mlp_fwd_smem<ST>(), st, true, mp, S);
}
} // namespace
cudaError_t tc_mlp_forward(const Geometry& g, void* X, bool spec16, const float* w1, const float* b1, const float* w2,
                           const float* b2, void* ws, cudaStream_t st) {
  cudaError_t e;
  const bool multi = g.hid != g.bs;
  const int hf = multi ? g.hid / BS : 1;
  const int groups = multi ? g.nb : (g.C + BS - 1) / BS;
  __nv_bfloat16* wprep = (__nv_bfloat16*)ws;
  float* bprep = (float*)((char*)ws + align_up((size_t)groups * hf * 4 * kWBytes, 256));
  const int nW = groups * hf * BS * BS;
  prof_begin("k_tc_prep_weights", st);
  if (multi)
    k_tc_prep_weights_hf<<<(nW + 255) / 256, 256, 0, st>>>(w1, b1, w2, b2, wprep, bprep, g.nb, hf);
  else
    k_tc_prep_weights<<<(nW + 255) / 256, 256, 0, st>>>(w1, b1, w2, b2, wprep, bprep, groups, g.bs, g.C, CtxHeader{},
                                                        (CtxHeader*)nullptr);
  prof_end(st);
  count_launch();
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  int dev = 0, sms = 148;
  if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
  if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
  MlpParams mp{};
  mp.X = X; mp.wprep = (const uint8_t*)wprep; mp.bprep = bprep;
  mp.rows = g.rows(); mp.C = g.C; mp.ngroups = groups; mp.H = g.H; mp.Kw = g.Kw; mp.Kh = g.Kh; mp.lambda = g.lambda;
  const long long ntiles = (mp.rows + kMlpRows - 1) / kMlpRows;
  int S = sms / groups;
  if (S < 1) S = 1;
  if ((long long)S > ntiles) S = (int)ntiles;
  prof_begin(multi ? "tc_mlp_fwd_hf" : "tc_mlp_fwd", st);
  if (spec16 && !multi) {
    // bf16 spectrum, hidden factor 1: the software-pipelined kernel (two operand buffers, two accumulators)
    if ((e = set_smem(tc_mlp_fwd_pipe, kMlpPipeSmem)) != cudaSuccess) return e;
    e = launch_k(tc_mlp_fwd_pipe, groups * S, kMlpThreads, kMlpPipeSmem, st, true, mp, S);
  } else {
    e = spec16 ? mlp_forward_launch<SpecBf16>(multi, groups * S, st, mp, S, hf) : mlp_forward_launch<float2>(multi, groups * S, st, mp, S, hf);
  }
  prof_end(st);
  count_launch();
  return e != cudaSuccess ? e : cudaGetLastError();
}

// hybrid backward (hidden factor 1 here; 2..8, with blocks of 96, through tc_mlp_backward_hf below): rows B1 (second half),
// B3-B7 between the fp32 FFT kernels of generic.cu.
// X = spectrum of x, G = alpha-weighted spectrum of dY (replaced by GX); the parameter gradients go through the same
// tc_wgrad + k_tc_wgrad_reduce launches as the fused path, over tiles of 96 consecutive spectrum rows.
bool tc_mlp_bwd_supported(const Geometry& g) { return tc_mlp_supported(g); }
namespace {
struct MlpBwdWs {
  __nv_bfloat16 *wprep, *Xh, *O1, *G2, *G1;
  float *bprep, *part;
  int groups, S;
  long long ntiles;
  size_t total;
};
MlpBwdWs mlp_bwd_carve(const Geometry& g, char* base) {
  MlpBwdWs w{};
  size_t off = 0;
  auto take = [&](size_t bytes) {
    char* p = base + off;
    off = align_up(off + bytes, 256);
    return p;
  };
  w.groups = (g.C + BS - 1) / BS;
  w.ntiles = (g.rows() + HP - 1) / HP;
  const size_t img = (size_t)w.ntiles * w.groups * kTileBytes;
  w.wprep = (__nv_bfloat16*)take((size_t)w.groups * 4 * kWBytes);
  w.bprep = (float*)take((size_t)w.groups * 2 * NT * sizeof(float));
  w.Xh = (__nv_bfloat16*)take(img);
  w.O1 = (__nv_bfloat16*)take(img);
  w.G2 = (__nv_bfloat16*)take(img);
  w.G1 = (__nv_bfloat16*)take(img);
  int S = 148 / (2 * w.groups);   // CTAs per (layer, group) of tc_wgrad
  if (S < 1) S = 1;
  if ((long long)S > w.ntiles) S = (int)w.ntiles;
  w.S = S;
  w.part = (float*)take((size_t)2 * w.groups * S * kWgPartFloats * sizeof(float));
  w.total = off;
  return w;
}
} // namespace
namespace {
// hidden factor > 1 (blocks of 96): weight images per (block, chunk), O1 / G1 images per chunk, partial sums per chunk
struct MlpBwdHfWs {
  __nv_bfloat16 *wprep, *Xh, *G2, *O1, *G1;
  float *bprep, *part;
  int hf, S;
  long long ntiles;
  size_t chunk_part_floats, total;
};
MlpBwdHfWs mlp_bwd_hf_carve(const Geometry& g, char* base) {
  MlpBwdHfWs w{};
  size_t off = 0;
  auto take = [&](size_t bytes) {
    char* p = base + off;
    off = align_up(off + bytes, 256);
    return p;
  };
  w.hf = g.hid / BS;
  w.ntiles = (g.rows() + HP - 1) / HP;
  const size_t img = (size_t)w.ntiles * g.nb * kTileBytes;
  w.wprep = (__nv_bfloat16*)take((size_t)g.nb * w.hf * 4 * kWBytes);
  w.bprep = (float*)take((size_t)g.nb * (w.hf + 1) * NT * sizeof(float));
  w.Xh = (__nv_bfloat16*)take(img);
  w.G2 = (__nv_bfloat16*)take(img);
  w.O1 = (__nv_bfloat16*)take(img * w.hf);
  w.G1 = (__nv_bfloat16*)take(img * w.hf);
  int S = 148 / (2 * g.nb);
  if (S < 1) S = 1;
  if ((long long)S > w.ntiles) S = (int)w.ntiles;
  w.S = S;
  w.chunk_part_floats = (size_t)2 * g.nb * S * kWgPartFloats;
  w.part = (float*)take(w.chunk_part_floats * w.hf * sizeof(float));
  w.total = off;
  return w;
}

cudaError_t tc_mlp_backward_hf(const Geometry& g, const void* X, void* G, bool spec16, const float* w1, const float* b1,
                               const float* w2, const float* b2, float* dw1, float* db1, float* dw2, float* db2, uint8_t* mask1,
                               uint8_t* mask2, void* ws, cudaStream_t st) {
  cudaError_t e;
  if ((e = spec16 ? set_smem(tc_mlp_bwd_hf<SpecBf16>, kMlpBwdHfSmem) : set_smem(tc_mlp_bwd_hf<float2>, kMlpBwdHfSmem)) != cudaSuccess)
    return e;
  if ((e = set_smem(tc_wgrad, kWgSmem)) != cudaSuccess) return e;
  const MlpBwdHfWs w = mlp_bwd_hf_carve(g, (char*)ws);
  const int hf = w.hf, nW = g.nb * hf * BS * BS;
  prof_begin("k_tc_prep_weights", st);
  k_tc_prep_weights_hf<<<(nW + 255) / 256, 256, 0, st>>>(w1, b1, w2, b2, w.wprep, w.bprep, g.nb, hf);
  prof_end(st);
  count_launch();
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  int dev = 0, sms = 148;
  if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
  if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
  MlpBwdHfParams mp{};
  mp.X = X; mp.G = G; mp.wprep = (const uint8_t*)w.wprep; mp.bprep = w.bprep;
  mp.Xh = w.Xh; mp.G2 = w.G2; mp.O1 = w.O1; mp.G1 = w.G1; mp.mask1 = mask1; mp.mask2 = mask2;
  mp.rows = g.rows(); mp.ntiles = w.ntiles; mp.C = g.C; mp.nb = g.nb; mp.H = g.H; mp.Kw = g.Kw; mp.Wh = g.Wh; mp.Kh = g.Kh;
  mp.hf = hf; mp.lambda = g.lambda;
  int S = sms / g.nb;
  if (S < 1) S = 1;
  if ((long long)S > w.ntiles) S = (int)w.ntiles;
  prof_begin("tc_mlp_bwd_hf", st);
  e = spec16 ? launch_k(tc_mlp_bwd_hf<SpecBf16>, g.nb * S, kMlpThreads, kMlpBwdHfSmem, st, true, mp, S)
             : launch_k(tc_mlp_bwd_hf<float2>, g.nb * S, kMlpThreads, kMlpBwdHfSmem, st, true, mp, S);
  prof_end(st);
  count_launch();
  if (e != cudaSuccess || (e = cudaGetLastError()) != cudaSuccess) return e;
  const size_t img = (size_t)w.ntiles * g.nb * kTileBytes;
  for (int hc = 0; hc < hf; ++hc) {
    // chunk hc: layer 2 = (O1_c, G2) -> dW2[c rows]; layer 1 = (Xh, G1_c) -> dW1[:, c columns]
    prof_begin("tc_wgrad", st);
    e = launch_k(tc_wgrad, 2 * g.nb * w.S, 128, kWgSmem, st, true, (const __nv_bfloat16*)((const char*)w.O1 + hc * img), w.G2, w.Xh,
                 (const __nv_bfloat16*)((const char*)w.G1 + hc * img), w.part + hc * w.chunk_part_floats, (int)w.ntiles, HP, g.nb,
                 w.S, 0);
    prof_end(st);
    count_launch();
    if (e != cudaSuccess || (e = cudaGetLastError()) != cudaSuccess) return e;
  }
  const int nred = nW + g.nb * g.hid;
  prof_begin("k_tc_wgrad_reduce", st);
  e = launch_k(k_tc_wgrad_reduce_hf, dim3((nred + 255) / 256, 2), 256, 0, st, true, w.part, (float2*)dw2, (float2*)db2,
               (float2*)dw1, (float2*)db1, g.nb, w.S, hf, g.accum ? 1 : 0);
  prof_end(st);
  count_launch();
  return e != cudaSuccess ? e : cudaGetLastError();
}
} // namespace
size_t tc_mlp_bwd_workspace_bytes(const Geometry& g) {
  return g.hid != g.bs ? mlp_bwd_hf_carve(g, nullptr).total : mlp_bwd_carve(g, nullptr).total;
}

cudaError_t tc_mlp_backward(const Geometry& g, const void* X, void* G, bool spec16, const float* w1, const float* b1,
                            const float* w2, const float* b2, float* dw1, float* db1, float* dw2, float* db2, uint8_t* mask1,
                            uint8_t* mask2, void* ws, cudaStream_t st) {
  if (g.hid != g.bs) return tc_mlp_backward_hf(g, X, G, spec16, w1, b1, w2, b2, dw1, db1, dw2, db2, mask1, mask2, ws, st);
  cudaError_t e;
  if ((e = spec16 ? set_smem(tc_mlp_bwd<SpecBf16>, kMlpBwdSmem) : set_smem(tc_mlp_bwd<float2>, kMlpBwdSmem)) != cudaSuccess) return e;
  if ((e = set_smem(tc_wgrad, kWgSmem)) != cudaSuccess) return e;
  const MlpBwdWs w = mlp_bwd_carve(g, (char*)ws);
  const int nW = w.groups * BS * BS;
  prof_begin("k_tc_prep_weights", st);
  k_tc_prep_weights<<<(nW + 255) / 256, 256, 0, st>>>(w1, b1, w2, b2, w.wprep, w.bprep, w.groups, g.bs, g.C, CtxHeader{},
                                                      (CtxHeader*)nullptr);
  prof_end(st);
  count_launch();
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  int dev = 0, sms = 148;
  if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
  if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
  MlpBwdParams mp{};
  mp.X = X; mp.G = G; mp.wprep = (const uint8_t*)w.wprep; mp.bprep = w.bprep;
  mp.Xh = w.Xh; mp.O1 = w.O1; mp.G2 = w.G2; mp.G1 = w.G1;
  mp.mask1 = mask1; mp.mask2 = mask2;
  mp.rows = g.rows(); mp.C = g.C; mp.ngroups = w.groups; mp.H = g.H; mp.Kw = g.Kw; mp.Wh = g.Wh; mp.Kh = g.Kh;
  mp.lambda = g.lambda;
  int S = sms / w.groups;
  if (S < 1) S = 1;
  if ((long long)S > w.ntiles) S = (int)w.ntiles;
  prof_begin("tc_mlp_bwd", st);
  e = spec16 ? launch_k(tc_mlp_bwd<SpecBf16>, w.groups * S, kMlpThreads, kMlpBwdSmem, st, true, mp, S)
             : launch_k(tc_mlp_bwd<float2>, w.groups * S, kMlpThreads, kMlpBwdSmem, st, true, mp, S);
  prof_end(st);
  count_launch();
  if (e != cudaSuccess || (e = cudaGetLastError()) != cudaSuccess) return e;
  // B4 / B6: layer 2 = (O1, G2), layer 1 = (Xh, G1); rows past the end of the last tile are zero in G2 / G1
  prof_begin("tc_wgrad", st);
  e = launch_k(tc_wgrad, 2 * w.groups * w.S, 128, kWgSmem, st, true, w.O1, w.G2, w.Xh, w.G1, w.part, (int)w.ntiles, HP, w.groups,
               w.S, 0);
  prof_end(st);
  count_launch();
  if (e != cudaSuccess || (e = cudaGetLastError()) != cudaSuccess) return e;
  const int nred = nW + w.groups * BS;
  prof_begin("k_tc_wgrad_reduce", st);
  e = launch_k(k_tc_wgrad_reduce, dim3((nred + 255) / 256, 2), 256, 0, st, true, w.part, (float2*)dw2, (float2*)db2, (float2*)dw1,
               (float2*)db1, w.groups, w.S, g.bs, g.C, g.accum ? 1 : 0, 0, (const CtxHeader*)nullptr, CtxHeader{}, (uint16_t*)nullptr,
               (size_t)0, 1);
  prof_end(st);
  count_launch();
  return e != cudaSuccess ? e : cudaGetLastError();
}

// W-direction launches: tile = (b, h, block), persistent over the SMs
static cudaError_t launch_wdft_fwd(const Geometry& g, const TcPlan& tp, const void* in, void* spec, const uint8_t* fimg,
                                   cudaStream_t st, bool dependent, bool independent = false) {
  CUtensorMap mx, ma;
  if (!act_tmap(tp, &mx, in, g) || !spec_store_tmap(tp, &ma, spec, g)) return cudaErrorInvalidValue;
  const int ntiles = g.B * g.H * g.nb;
  const int grid = ntiles < tp.num_sms ? ntiles : tp.num_sms;
  prof_begin("tc_wdft_fwd", st);
  cudaError_t e = launch_k(tc_wdft_fwd2, grid, kW2Threads, kWfSmem, st, dependent, mx, ma, (const uint32_t*)fimg, ntiles, g.nb,
                           g.H, g.Kw, independent ? 1 : 0);
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

// context header written by the SAVE_CONTEXT forward / checked by the USE_CONTEXT backward
static CtxHeader make_header(const Geometry& g, const TcWs& w) {
  CtxHeader h{};
  h.magic = kCtxMagic;
  h.B = g.B; h.H = g.H; h.W = g.W; h.C = g.C; h.nb = g.nb_blocks; h.Kh = g.Kh; h.Kw = g.Kw; h.chunk_b = w.chunk_b;
  memcpy(&h.lambda_bits, &g.lambda, 4);
  h.export_masks = g.export_masks ? 1u : 0u;
  return h;
}

// sub-geometry of the samples [b0, b0 + n) and the byte offset of sample b0 in an activation tensor
static Geometry chunk_geometry(const Geometry& g, int n) {
  Geometry c = g;
  c.B = n;
  return c;
}
static size_t act_offset(const Geometry& g, int b0) { return (size_t)b0 * g.H * g.W * g.C * 2; }

cudaError_t tc_forward(const Geometry& g0, const Plan& p, const void* x, const float* w1, const float* b1,
                       const float* w2, const float* b2, void* y, void* ws, cudaStream_t st) {
  const Geometry g = tc_geom(g0);
  // SAVE_CONTEXT: the backward layout, so that tc_backward finds the context where it expects it
  TcWs w = tc_carve(g, g.save_ctx, (char*)ws);
  const TcPlan& tp = p.tc;
  cudaError_t e;
  const int nW = g.nb * BS * BS;
  const CtxHeader hdr = g.save_ctx ? make_header(g, w) : CtxHeader{};
  prof_begin("k_tc_prep_weights", st);
  k_tc_prep_weights<<<(nW + 255) / 256, 256, 0, st>>>(w1, b1, w2, b2, w.wprep, w.bprep, g.nb, g.bs_block, g.C, hdr, w.header);
  prof_end(st);
  count_launch();
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  for (int b0 = 0; b0 < g.B; b0 += w.chunk_f) {
    const Geometry gc = chunk_geometry(g, g.B - b0 < w.chunk_f ? g.B - b0 : w.chunk_f);
    const char* xc = (const char*)x + act_offset(g, b0);
    char* yc = (char*)y + act_offset(g, b0);
    const size_t t0 = (size_t)b0 * g.Kw * g.nb;   // first (b, kw, block) tile of the chunk in whole-batch tensors
    // the first W transform of the call runs beside the weight-image kernel (it reads x and writes A only)
    if ((e = launch_wdft_fwd(gc, tp, xc, w.A, tp.fw, st, true, b0 == 0)) != cudaSuccess) return e;
    MixParams mp{};
    if (!tile_tmap(tp, &mp.mapA1, w.A, gc)) return cudaErrorInvalidValue;
    mp.mapA1g = mp.mapA1;
    mp.A2 = w.A; mp.dft = tp.dft2; mp.wprep = (const uint8_t*)w.wprep; mp.bprep = w.bprep;
    mp.B = gc.B; mp.H = g.H; mp.Kw = g.Kw; mp.Wh = g.Wh; mp.nb = g.nb; mp.C = g.C; mp.Kh = g.Kh; mp.lambda = g.lambda;
    prof_begin("tc_mix_fwd", st);
    const int S2 = mix2_split(gc, tp);
    if (g.save_ctx) {
      // saved context: Xh, O1 (operands of tc_wgrad) and the activation masks stay in the workspace
      mp.Xh = (__nv_bfloat16*)((char*)w.Xh + t0 * kTileBytes);
      mp.O1 = (__nv_bfloat16*)((char*)w.O1 + t0 * kTileBytes);
      mp.maskbits = w.maskbits + t0 * 12 * 32;
      e = launch_k(tc_mix2<kMixFwdSave, false>, mix2_grid(gc, tp, S2), kMix2Threads, kMix2Smem, st, true, mp, S2);
    } else {
      e = launch_k(tc_mix2<kMixFwd, false>, mix2_grid(gc, tp, S2), kMix2Threads, kMix2Smem, st, true, mp, S2);
    }
    prof_end(st);
    if (e != cudaSuccess) return e;
    count_launch();
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if ((e = launch_wdft_inv(gc, tp, w.A, g.no_residual ? nullptr : xc, yc, tp.gw, st)) != cudaSuccess) return e;
  }
  return cudaSuccess;
}

cudaError_t tc_backward(const Geometry& g0, const Plan& p, const void* x, const void* dy, const float* w1,
                        const float* b1, const float* w2, const float* b2, void* dx, float* dw1, float* db1,
                        float* dw2, float* db2, void* ws, cudaStream_t st) {
  const Geometry g = tc_geom(g0);
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
    TC_LAUNCH("k_tc_prep_weights", k_tc_prep_weights, (nW + 255) / 256, 256, 0, st, dep, w1, b1, w2, b2, w.wprep, w.bprep, g.nb,
              g.bs_block, g.C, CtxHeader{}, (CtxHeader*)nullptr);
  }
  const size_t mask1_sample = (size_t)g.H * g.Wh * g.CH * 2, mask2_sample = (size_t)g.H * g.Wh * g.C * 2;
  for (int b0 = 0; b0 < g.B; b0 += w.chunk_b) {
    const Geometry gc = chunk_geometry(g, g.B - b0 < w.chunk_b ? g.B - b0 : w.chunk_b);
    const char* xc = (const char*)x + act_offset(g, b0);
    const char* dyc = (const char*)dy + act_offset(g, b0);
    char* dxc = (char*)dx + act_offset(g, b0);
    const size_t t0 = (size_t)b0 * g.Kw * g.nb;
    __nv_bfloat16* Xh = (__nv_bfloat16*)((char*)w.Xh + t0 * kTileBytes);
    __nv_bfloat16* O1 = (__nv_bfloat16*)((char*)w.O1 + t0 * kTileBytes);
    // B1 (first half) and B2: W-direction spectra of x and of dy (alpha-weighted)
    if (!g.use_ctx) {
      if ((e = launch_wdft_fwd(gc, tp, xc, w.Ax, tp.fw, st, dep)) != cudaSuccess) return e;
      dep = true;
    }
    if ((e = launch_wdft_fwd(gc, tp, dyc, w.A, tp.fw_alpha, st, dep)) != cudaSuccess) return e;
    dep = true;
    MixParams mp{};
    if (!tile_tmap(tp, &mp.mapA1, g.use_ctx ? w.A : w.Ax, gc) || !tile_tmap(tp, &mp.mapA1g, w.A, gc)) return cudaErrorInvalidValue;
    mp.A2 = w.A;   // in place over the gradient's spectrum
    mp.Xh = Xh; mp.O1 = O1; mp.G2 = w.G2; mp.G1 = w.G1;
    mp.dft = tp.dft2; mp.wprep = (const uint8_t*)w.wprep; mp.bprep = w.bprep;
    mp.mask1 = g.export_masks ? w.mask1 + (size_t)b0 * mask1_sample : nullptr;
    mp.mask2 = g.export_masks ? w.mask2 + (size_t)b0 * mask2_sample : nullptr;
    mp.B = gc.B; mp.H = g.H; mp.Kw = g.Kw; mp.Wh = g.Wh; mp.nb = g.nb; mp.C = g.C; mp.Kh = g.Kh; mp.lambda = g.lambda;
    const int S2 = mix2_split(gc, tp);
    mp.maskbits = w.maskbits + t0 * 12 * 32;
    if (g.use_ctx) {
      // gradient stages only: Xh, O1 and the masks were left in the workspace by the forward call
      if (g.export_masks) {
        TC_LAUNCH("tc_mix_bwd", tc_mix2<kMixBwdCtx, true>, mix2_grid(gc, tp, S2), kMix2Threads, kMix2Smem, st, dep, mp, S2);
      } else {
        TC_LAUNCH("tc_mix_bwd", tc_mix2<kMixBwdCtx, false>, mix2_grid(gc, tp, S2), kMix2Threads, kMix2Smem, st, dep, mp, S2);
      }
    } else if (g.export_masks) {
      TC_LAUNCH("tc_mix_bwd", tc_mix2<kMixBwd, true>, mix2_grid(gc, tp, S2), kMix2Threads, kMix2Smem, st, dep, mp, S2);
    } else {
      TC_LAUNCH("tc_mix_bwd", tc_mix2<kMixBwd, false>, mix2_grid(gc, tp, S2), kMix2Threads, kMix2Smem, st, dep, mp, S2);
    }
    // B4 / B6: parameter gradients of the chunk, added to the partial sums of the chunks before it
    TC_LAUNCH("tc_wgrad", tc_wgrad, 2 * g.nb * w.S, 128, kWgSmem, st, dep, O1, w.G2, Xh, w.G1, w.part, gc.B * g.Kw, g.H, g.nb,
              w.S, b0 > 0 ? 1 : 0);
    // B8: dx = dy + irfft2(GX / alpha)
    if ((e = launch_wdft_inv(gc, tp, w.A, g.no_residual ? nullptr : dyc, dxc, tp.gw_noalpha, st)) != cudaSuccess) return e;
  }
  const int nred = nW + g.nb * BS;
  // last kernel of the call: fixed-order sum of the partial sums; with USE_CONTEXT it also checks the context header
  // (a context that does not belong to this call poisons dx and the gradients with NaN)
  TC_LAUNCH("k_tc_wgrad_reduce", k_tc_wgrad_reduce, dim3((nred + 255) / 256, 2), 256, 0, st, dep, w.part, (float2*)dw2,
            (float2*)db2, (float2*)dw1, (float2*)db1, g.nb, w.S, g.bs_block, g.C, g.accum ? 1 : 0, g.use_ctx ? 1 : 0,
            (const CtxHeader*)w.header, make_header(g, w), (uint16_t*)dx, (size_t)g.B * g.H * g.W * g.C, 0);
#undef TC_LAUNCH
  return cudaSuccess;
}

} // namespace afno
