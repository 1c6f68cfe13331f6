// tcgen05 (5th-generation tensor core) path of the AFNO spectral layer for bf16 activations,
// 96-wide channel blocks, H <= 96 (90 in FourCastNet's 8x8 patch grid) and W <= 192.
//
// On B200 the tensor pipe is ~30x the fp32 ALU pipe, while a dense DFT of length 90 / 180 costs
// only ~20x the FLOPs of an FFT, so every transform of the layer is computed as a bf16 GEMM
// with fp32 accumulation against constant DFT matrices (S5 gives the arithmetic and
// the measured error).  The layer becomes three GEMM-chain kernels:
//
//   tc_wdft_fwd  [F1, B2]   per (b, h, 128 channels):  A1[c, (ri,kw)] = x^T[c, w] * Fw[w, (ri,kw)]
//   tc_mix_fwd   [F2-F7]    per (b, kw, block j), everything on chip in tensor memory:
//                            Xh = Fh * A1  ->  relu(Xh W1 + b1)  ->  shrink(. W2 + b2)  ->  Fh^H * Z
//   tc_wdft_inv  [F8, F9, B8] per (b, h, 128 channels): y[c, w] = x + A2^T[c, (ri,kw)] * Gw[(ri,kw), w]
//
// Complex arithmetic runs as real GEMMs on separate (re | im) column halves using the
// instruction descriptor's negate bit for the minus signs, so only W_re and W_im (not the 2x2
// real block form) live in shared memory.
#include <math.h>
#include <string.h>

#include <vector>

#include "afno_internal.h"
#include "tc_common.cuh"

namespace afno {

namespace {

using namespace tc;

constexpr int BS = 96;    // channel block size handled by this path
constexpr int NT = 192;   // (re | im) columns of one block
constexpr int HP = 96;    // H padded to the K extent of the H-direction GEMMs
constexpr int WP = 192;   // W padded to the K / N extent of the W-direction GEMMs
constexpr int CGRP = 128; // channels per W-direction tile (= UMMA M)

// shared-memory operand geometry (bytes), see tc_common.cuh for the layout formulas
constexpr uint32_t kDftLbo = 2048, kDftSbo = 128;   // Ch / Sh: K-major A [128 x 96], order [k/8][m/8]
constexpr uint32_t kDftBytes = 128 * HP * 2;         // 24576
constexpr uint32_t kWLbo = 1536, kWSbo = 128;       // weights: K-major B [96 x 96], order [k/8][n/8]
constexpr uint32_t kWBytes = BS * BS * 2;            // 18432
constexpr uint32_t kTileLbo = 128, kTileSbo = 1536; // mode tile: MN-major B [K=96 rows][N=192]
constexpr uint32_t kTileBytes = HP * NT * 2;         // 36864
constexpr uint32_t kFwLbo = 3072, kFwSbo = 128;     // Fw^T / Gw^T: K-major B [192 x 192]
constexpr uint32_t kFwBytes = WP * NT * 2;           // 73728
constexpr uint32_t kRowLbo = 128, kRowSbo = 3072;   // W-direction data tile: MN-major A [K=192][M=128]
constexpr uint32_t kRowBytes = WP * CGRP * 2;        // 49152

constexpr uint32_t kMixSmem = 2 * kDftBytes + 4 * kWBytes + kTileBytes + 2 * NT * 4; // 161280
constexpr int kTrPitch = 132;                        // fp32 words per row of the epilogue transpose buffer
constexpr uint32_t kTrBytes = 32 * kTrPitch * 4;     // 16896
constexpr int kRowThreads = 256;
constexpr uint32_t kRowSmem = kFwBytes + 2 * kRowBytes + 2 * kTrBytes;               // 205824

// Epilogue transpose of the W-direction kernels: every thread holds 32 consecutive accumulator
// columns of ITS channel (TMEM lane).  The chunk goes through shared memory so that thread
// (q, c4) = (t/32 + 4*pass, t%32) then owns 4 consecutive channels of column q and global
// accesses become 8-byte vectors, 256 contiguous bytes per warp.  t = thread index inside a
// 128-thread warp group; the two groups (column halves) use their own buffer and named barrier.
template <typename F>
__device__ __forceinline__ void transposed_chunk(float* sT, const uint32_t (&v)[32], int t, int bar_id, F&& consume) {
#pragma unroll
  for (int q = 0; q < 32; ++q) sT[q * kTrPitch + t] = __uint_as_float(v[q]);
  asm volatile("bar.sync %0, 128;" ::"r"(bar_id) : "memory");
  const int c4 = (t & 31) * 4;
#pragma unroll
  for (int pass = 0; pass < 8; ++pass) {
    const int q = pass * 4 + (t >> 5);
    consume(pass, q, c4, *(const float4*)&sT[q * kTrPitch + c4]);
  }
  asm volatile("bar.sync %0, 128;" ::"r"(bar_id) : "memory");
}

// ---- weight preparation: fp32 [nb][96][96][2] -> bf16 K-major interleaved operands --------------
// per block, 8 matrices of kWBytes: fwd {W1r, W1i, W2r, W2i} with element (n=o, k=i) = W[i][o];
// bwd {W1r, W1i, W2r, W2i} with element (n=i, k=o) = W[i][o].
__global__ void k_tc_prep_weights(const float* __restrict__ w1, const float* __restrict__ w2,
                                  __nv_bfloat16* __restrict__ out, int nb) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= nb * BS * BS) return;
  const int o = idx % BS, i = (idx / BS) % BS, j = idx / (BS * BS);
  const float2 a = ((const float2*)w1)[idx], b = ((const float2*)w2)[idx];
  __nv_bfloat16* base = out + (size_t)j * 8 * (kWBytes / 2);
  const uint32_t f = ((i / 8) * kWLbo + (o / 8) * kWSbo + (o % 8) * 16 + (i % 8) * 2) / 2; // n=o, k=i
  const uint32_t t = ((o / 8) * kWLbo + (i / 8) * kWSbo + (i % 8) * 16 + (o % 8) * 2) / 2; // n=i, k=o
  const uint32_t m = kWBytes / 2;
  base[0 * m + f] = __float2bfloat16_rn(a.x);
  base[1 * m + f] = __float2bfloat16_rn(a.y);
  base[2 * m + f] = __float2bfloat16_rn(b.x);
  base[3 * m + f] = __float2bfloat16_rn(b.y);
  base[4 * m + t] = __float2bfloat16_rn(a.x);
  base[5 * m + t] = __float2bfloat16_rn(a.y);
  base[6 * m + t] = __float2bfloat16_rn(b.x);
  base[7 * m + t] = __float2bfloat16_rn(b.y);
}

// ---- F1 / B2 and F8 + F9 / B8: the W-direction transforms as GEMMs -------------------------------
// One tile = (b, h, 128 channels): D[c, n] = sum_k A[k, c] * Bconst[k, n], 12 UMMAs of 128x192x16.
//   forward (INVERSE = false): k = w, A = x^T slab, n = (ri, kw); D -> A1[b][kw][j][h][ri][96]
//   inverse (INVERSE = true) : k = (ri, kw), A gathered from A2, n = w; D + residual -> y
// Software pipeline per CTA (persistent over tiles): the operand tile of iteration i+2 is copied
// (cp.async) while the tensor core works on tile i+1 (second TMEM accumulator) and all 8 warps
// run the epilogue of tile i.
template <bool INVERSE>
__global__ void __launch_bounds__(kRowThreads, 1)
tc_wdft(const __nv_bfloat16* __restrict__ in, const __nv_bfloat16* __restrict__ res, __nv_bfloat16* __restrict__ out,
        const uint8_t* __restrict__ Bconst, int B, int H, int W, int C, int Kw, int nb) {
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ __align__(8) uint64_t mbar[2];
  __shared__ uint32_t tmem_slot;
  uint8_t* sF = smem;
  uint8_t* sA0 = smem + kFwBytes;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int grp = warp >> 2, tg = tid & 127;          // column half / thread index inside the warp group
  float* sT = (float*)(smem + kFwBytes + 2 * kRowBytes + grp * kTrBytes);
  for (uint32_t i = tid; i < 2 * kRowBytes / 16; i += kRowThreads) ((uint4*)sA0)[i] = make_uint4(0, 0, 0, 0);
  for (uint32_t i = tid; i < kFwBytes / 16; i += kRowThreads) cp_async16(smem_u32(sF) + i * 16, Bconst + (size_t)i * 16);
  if (tid == 0) {
    mbar_init(&mbar[0], 1);
    mbar_init(&mbar[1], 1);
    mbar_init_fence();
  }
  if (warp == 0) tmem_alloc<512>(&tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
  const int ncg = (C + CGRP - 1) / CGRP;
  const int ntiles = B * H * ncg;
  const int nmine = ntiles > (int)blockIdx.x ? (ntiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
  const uint32_t idesc = idesc_bf16(128, NT, kIdescAMn);
  const int hl = lane & 7, cl4 = lane >> 3;

  auto load_tile = [&](int it) {
    const int t = blockIdx.x + it * gridDim.x;
    const int cg = t % ncg, bh = t / ncg;
    const uint32_t dst = smem_u32(sA0) + (it & 1) * kRowBytes;
    if (!INVERSE) {
      // x[b,h,:,cg*128 .. +128) -> MN-major A operand (K = w, M = channel)
      const __nv_bfloat16* xrow = in + (size_t)bh * W * C;
      const int nunits = ((W + 7) / 8) * 4;
      for (int u = warp; u < nunits; u += kRowThreads / 32) {
        const int w = (u >> 2) * 8 + hl;
        const int mc = (u & 3) * 4 + cl4;
        const int c0 = cg * CGRP + mc * 8;
        if (w < W && c0 < C) cp_async16(dst + mc * kRowSbo + w * 16, xrow + (size_t)w * C + c0);
      }
    } else {
      // A2[b][kw][j][h][ri][cl] gathered into the MN-major A operand (K = (ri,kw), M = channel)
      const int b = bh / H, h = bh - b * H;
      const int kwg = (Kw + 7) / 8;
      const int nunits = 2 * kwg * 4;
      for (int u = warp; u < nunits; u += kRowThreads / 32) {
        const int rg = u >> 2;
        const int ri = rg / kwg, kw = (rg - ri * kwg) * 8 + hl;
        const int mc = (u & 3) * 4 + cl4;
        const int c0 = cg * CGRP + mc * 8;
        if (kw < Kw && c0 < C) {
          const int j = c0 / BS, cl = c0 - j * BS;
          cp_async16(dst + mc * kRowSbo + (ri * BS + kw) * 16,
                     in + ((((size_t)b * Kw + kw) * nb + j) * H + h) * NT + ri * BS + cl);
        }
      }
    }
  };
  auto issue_mma = [&](int it) {
    const uint32_t a = smem_u32(sA0) + (it & 1) * kRowBytes;
    const uint32_t d = tmem + (it & 1) * 256;
#pragma unroll
    for (int ks = 0; ks < WP / 16; ++ks)
      mma_ss(d, smem_desc(a + ks * 2 * kRowLbo, kRowLbo, kRowSbo), smem_desc(smem_u32(sF) + ks * 2 * kFwLbo, kFwLbo, kFwSbo),
             idesc, ks > 0);
    mma_commit(&mbar[it & 1]);
  };

  if (nmine > 0) load_tile(0);
  cp_async_commit();
  if (nmine > 1) load_tile(1);
  cp_async_commit();
  cp_async_wait_group<1>();
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  if (tid == 0 && nmine > 0) issue_mma(0);

  for (int it = 0; it < nmine; ++it) {
    const int t = blockIdx.x + it * gridDim.x;
    const int cg = t % ncg, bh = t / ncg;
    // tile it+1 has landed -> start its MMA into the other accumulator (drained by the epilogue of it-1)
    cp_async_wait_group<0>();
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    if (tid == 0 && it + 1 < nmine) issue_mma(it + 1);
    // accumulator of tile `it`
    mbar_wait(&mbar[it & 1], (uint32_t)((it >> 1) & 1));
    tc_fence_after();
    // its operand buffer is free again: prefetch tile it+2 into it
    if (it + 2 < nmine) load_tile(it + 2);
    cp_async_commit();

    const uint32_t acc = tmem + (it & 1) * 256 + lane_base + grp * BS;
    if (!INVERSE) {
      const int b = bh / H, h = bh - b * H;
#pragma unroll 1
      for (int k = 0; k < 3; ++k) {
        uint32_t v[32];
        tmem_ld32(acc + 32 * k, v);
        tmem_wait_ld();
        transposed_chunk(sT, v, tg, 1 + grp, [&](int, int q, int c4, float4 f) {
          const int kw = 32 * k + q;      // column n = grp*96 + kw  (ri = grp)
          const int c = cg * CGRP + c4;
          if (kw < Kw && c < C) {
            const int j = c / BS, cl = c - j * BS;
            uint2 o = make_uint2(pack_bf16(f.x, f.y), pack_bf16(f.z, f.w));
            *(uint2*)(out + ((((size_t)b * Kw + kw) * nb + j) * H + h) * NT + grp * BS + cl) = o;
          }
        });
      }
    } else {
      const int cbase = cg * CGRP + (tg & 31) * 4;
      const size_t rowoff = (size_t)bh * W * C + cbase;
#pragma unroll 1
      for (int k = 0; k < 3; ++k) {
        const int w0 = grp * BS + 32 * k;
        uint32_t v[32];
        tmem_ld32(acc + 32 * k, v);
        // residual rows of this chunk (8 independent 8-byte loads in flight per thread)
        uint2 rr[8];
#pragma unroll
        for (int pass = 0; pass < 8; ++pass) {
          const int w = w0 + pass * 4 + (tg >> 5);
          rr[pass] = make_uint2(0u, 0u);
          if (res && w < W && cbase < C) rr[pass] = __ldg((const uint2*)(res + rowoff + (size_t)w * C));
        }
        tmem_wait_ld();
        transposed_chunk(sT, v, tg, 1 + grp, [&](int pass, int q, int c4, float4 f) {
          const int w = w0 + q;
          if (w < W && cbase < C) {
            const uint2 r2 = rr[pass];
            const float2 ra = __bfloat1622float2(*(const __nv_bfloat162*)&r2.x);
            const float2 rb = __bfloat1622float2(*(const __nv_bfloat162*)&r2.y);
            uint2 o = make_uint2(pack_bf16(f.x + ra.x, f.y + ra.y), pack_bf16(f.z + rb.x, f.w + rb.y));
            *(uint2*)(out + rowoff + (size_t)w * C) = o;
          }
        });
      }
    }
  }
  cp_async_wait_all();
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc<512>(tmem);
}


// ---- F2-F7: per (b, kw, block) chain  H-DFT -> layer 1 -> layer 2 -> inverse H-DFT ---------------
// 256 threads: warp w owns TMEM lanes 32*(w&3).. (accumulator rows) and the column half w>>2
// (re | im), so every epilogue is split two ways.  Accumulators in tensor memory: region R0 =
// columns [0,192), R1 = [256,448); a layer's bf16 input (A operand) is packed in place over
// the fp32 accumulator it was computed from (all loads, block barrier, then the stores).
struct MixParams {
  const __nv_bfloat16* A1;
  __nv_bfloat16* A2;
  const uint8_t* dft;      // Ch then Sh, kDftBytes each, smem image
  const uint8_t* wprep;    // per block 8 x kWBytes
  const float* b1;         // [nb][96][2]
  const float* b2;
  int B, H, Kw, nb, Kh;
  float lambda;
};

constexpr int kMixThreads = 256;

// D[:, dcol .. dcol+96) (+)= A_smem(K-major [128 x 96]) * tile half (MN-major, 96 columns)
__device__ __forceinline__ void issue_dft(uint32_t d, uint32_t a_base, uint32_t b_base, uint32_t idesc, bool fresh) {
#pragma unroll
  for (int ks = 0; ks < HP / 16; ++ks)
    mma_ss(d, smem_desc(a_base + ks * 2 * kDftLbo, kDftLbo, kDftSbo),
           smem_desc(b_base + ks * 2 * kTileLbo, kTileLbo, kTileSbo), idesc, !(fresh && ks == 0));
}
// D[:, dcol .. dcol+96) (+)= A_tmem(packed bf16, 48 columns = K 96) * W_smem(K-major [96 x 96])
__device__ __forceinline__ void issue_mlp(uint32_t d, uint32_t a_tmem, uint32_t w_base, uint32_t idesc, bool fresh) {
#pragma unroll
  for (int ks = 0; ks < BS / 16; ++ks)
    mma_ts(d, a_tmem + ks * 8, smem_desc(w_base + ks * 2 * kWLbo, kWLbo, kWSbo), idesc, !(fresh && ks == 0));
}
// same with W^H: the forward weight image (n=o, k=i, K-major) read as an MN-major B operand (k=o, n=i)
__device__ __forceinline__ void issue_mlp_t(uint32_t d, uint32_t a_tmem, uint32_t w_base, uint32_t idesc, bool fresh) {
#pragma unroll
  for (int ks = 0; ks < BS / 16; ++ks)
    mma_ts(d, a_tmem + ks * 8, smem_desc(w_base + ks * 2 * kWSbo, kWSbo, kWLbo), idesc, !(fresh && ks == 0));
}

struct MixThread {
  uint32_t lane_base; // TMEM lane offset of this warp's 32 rows
  int colh;           // 0: re columns [0,96), 1: im columns [96,192)
  int r;              // accumulator row of this thread
};

// this thread's 96 accumulator columns of a region -> registers
__device__ __forceinline__ void ld_half(uint32_t region, const MixThread& t, uint32_t (&v)[3][32]) {
#pragma unroll
  for (int k = 0; k < 3; ++k) tmem_ld32(region + t.lane_base + t.colh * BS + 32 * k, v[k]);
  tmem_wait_ld();
}
// packed bf16 A operand of the next GEMM: K index = column, re half -> columns [0,48), im -> [48,96)
__device__ __forceinline__ void st_half_packed(uint32_t region, const MixThread& t, const uint32_t (&pk)[3][16]) {
#pragma unroll
  for (int k = 0; k < 3; ++k) tmem_st16(region + t.lane_base + t.colh * (BS / 2) + 16 * k, pk[k]);
}
__device__ __forceinline__ void store_row_half(__nv_bfloat16* dst, const uint32_t (&pk)[3][16]) {
#pragma unroll
  for (int k = 0; k < 3; ++k)
#pragma unroll
    for (int g = 0; g < 4; ++g)
      *(uint4*)(dst + k * 32 + g * 8) = make_uint4(pk[k][4 * g], pk[k][4 * g + 1], pk[k][4 * g + 2], pk[k][4 * g + 3]);
}
// bf16 rows written as the MN-major B operand of the inverse H-DFT (K = row r)
__device__ __forceinline__ void store_tile_half(uint8_t* tile, const MixThread& t, const uint32_t (&pk)[3][16]) {
#pragma unroll
  for (int k = 0; k < 3; ++k)
#pragma unroll
    for (int g = 0; g < 4; ++g)
      *(uint4*)(tile + (t.colh * 12 + k * 4 + g) * kTileSbo + t.r * 16) =
          make_uint4(pk[k][4 * g], pk[k][4 * g + 1], pk[k][4 * g + 2], pk[k][4 * g + 3]);
}
// rows of a (b,kw,j) tile [H][192] -> MN-major B operand (K = h, N = (ri, c)); 8 warps
__device__ __forceinline__ void load_tile(uint32_t tile_saddr, const __nv_bfloat16* src, int H, int warp, int lane) {
  const int hl = lane & 7, cl4 = lane >> 3;
  const int nunits = ((H + 7) / 8) * 6;
  for (int u = warp; u < nunits; u += kMixThreads / 32) {
    const int h = (u / 6) * 8 + hl;
    const int nc = (u % 6) * 4 + cl4;
    if (h < H) cp_async16(tile_saddr + nc * kTileSbo + h * 16, src + (size_t)h * NT + nc * 8);
  }
}
__device__ __forceinline__ void block_tmem_sync() {
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
}

constexpr uint32_t kMixFwdSmem = kMixSmem + kTileBytes; // two tile buffers (prefetch of the next tile)

__global__ void __launch_bounds__(kMixThreads, 1) tc_mix_fwd(MixParams p) {
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ __align__(8) uint64_t mbar;
  __shared__ uint32_t tmem_slot;
  uint8_t* sCh = smem;
  uint8_t* sSh = smem + kDftBytes;
  uint8_t* sW = smem + 2 * kDftBytes;
  uint8_t* sTile0 = sW + 4 * kWBytes;
  float* sBias = (float*)(sTile0 + kTileBytes); // b1 (re 96 | im 96), b2 (re 96 | im 96)
  uint8_t* sTile1 = sTile0 + kTileBytes + 2 * NT * 4;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  for (uint32_t i = tid; i < kTileBytes / 16; i += kMixThreads) {
    ((uint4*)sTile0)[i] = make_uint4(0, 0, 0, 0);
    ((uint4*)sTile1)[i] = make_uint4(0, 0, 0, 0);
  }
  for (uint32_t i = tid; i < 2 * kDftBytes / 16; i += kMixThreads)
    cp_async16(smem_u32(sCh) + i * 16, p.dft + (size_t)i * 16);
  if (tid == 0) {
    mbar_init(&mbar, 1);
    mbar_init_fence();
  }
  if (warp == 0) tmem_alloc<512>(&tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  MixThread th;
  th.lane_base = (uint32_t)((warp & 3) * 32) << 16;
  th.colh = warp >> 2;
  th.r = (warp & 3) * 32 + lane;
  const uint32_t R0 = tmem, R1 = tmem + 256;
  const uint32_t aCh = smem_u32(sCh), aSh = smem_u32(sSh), aW = smem_u32(sW);
  const uint32_t half = (BS / 8) * kTileSbo;
  const uint32_t id_dft = idesc_bf16(128, BS, kIdescBMn);
  const uint32_t id_mlp = idesc_bf16(128, BS);

  const int ntiles = p.nb * p.B * p.Kw;
  const int per = (ntiles + gridDim.x - 1) / gridDim.x;
  const int t_begin = blockIdx.x * per, t_end = min(ntiles, t_begin + per);
  uint32_t phase = 0;
  int cur_j = -1;
  const int r = th.r;
  const int kappa = (r <= p.H / 2) ? r : p.H - r;
  const bool row_kept = (r < p.H) && (kappa < p.Kh);
  const float* bias1 = sBias + th.colh * BS;
  const float* bias2 = sBias + NT + th.colh * BS;

  auto tile_src = [&](int t) {
    const int j = t / (p.B * p.Kw);
    const int rem = t - j * (p.B * p.Kw);
    return p.A1 + ((size_t)rem * p.nb + j) * p.H * NT;
  };
  if (t_begin < t_end) load_tile(smem_u32(sTile0), tile_src(t_begin), p.H, warp, lane);
  cp_async_commit();

  for (int t = t_begin; t < t_end; ++t) {
    const int j = t / (p.B * p.Kw);
    const int rem = t - j * (p.B * p.Kw);
    uint8_t* sTile = ((t - t_begin) & 1) ? sTile1 : sTile0;
    const uint32_t aTile = smem_u32(sTile);
    const bool new_block = j != cur_j;
    if (new_block) {
      cur_j = j;
      const uint8_t* wsrc = p.wprep + (size_t)j * 8 * kWBytes;
      for (uint32_t i = tid; i < 4 * kWBytes / 16; i += kMixThreads) cp_async16(aW + i * 16, wsrc + (size_t)i * 16);
      for (int i = tid; i < 2 * NT; i += kMixThreads) {
        const int which = i / NT, n = i % NT, ri = n / BS, o = n % BS;
        sBias[i] = (which == 0 ? p.b1 : p.b2)[((size_t)j * BS + o) * 2 + ri];
      }
    }
    // prefetch the next tile into the other buffer (its last reader, the previous inverse DFT, is complete)
    if (t + 1 < t_end) load_tile(smem_u32(((t - t_begin) & 1) ? sTile0 : sTile1), tile_src(t + 1), p.H, warp, lane);
    cp_async_commit();
    if (new_block) cp_async_wait_group<0>();
    else cp_async_wait_group<1>();
    fence_async_smem();
    block_tmem_sync();
    // F2: Xr = Ch Ar + Sh Ai ; Xi = Ch Ai - Sh Ar      (forward kernel exp(-i theta))
    if (tid == 0) {
      issue_dft(R0, aCh, aTile, id_dft, true);
      issue_dft(R0, aSh, aTile + half, id_dft, false);
      issue_dft(R0 + BS, aCh, aTile + half, id_dft, true);
      issue_dft(R0 + BS, aSh, aTile, id_dft | kIdescNegA, false);
      mma_commit(&mbar);
    }
    mbar_wait(&mbar, phase);
    phase ^= 1;
    tc_fence_after();
    {
      uint32_t v[3][32], pk[3][16];
      ld_half(R0, th, v);
      block_tmem_sync();
#pragma unroll
      for (int k = 0; k < 3; ++k)
#pragma unroll
        for (int q = 0; q < 16; ++q) pk[k][q] = pack_bf16(__uint_as_float(v[k][2 * q]), __uint_as_float(v[k][2 * q + 1]));
      st_half_packed(R0, th, pk);
      tmem_wait_st();
    }
    block_tmem_sync();
    // F3: P1 = Xh W1 + b1
    if (tid == 0) {
      issue_mlp(R1, R0, aW + 0 * kWBytes, id_mlp, true);                         // Xr W1r
      issue_mlp(R1, R0 + BS / 2, aW + 1 * kWBytes, id_mlp | kIdescNegB, false);  // - Xi W1i
      issue_mlp(R1 + BS, R0, aW + 1 * kWBytes, id_mlp, true);                    // Xr W1i
      issue_mlp(R1 + BS, R0 + BS / 2, aW + 0 * kWBytes, id_mlp, false);          // + Xi W1r
      mma_commit(&mbar);
    }
    mbar_wait(&mbar, phase);
    phase ^= 1;
    tc_fence_after();
    {
      // F4: bias + split ReLU
      uint32_t v[3][32], pk[3][16];
      ld_half(R1, th, v);
      block_tmem_sync();
#pragma unroll
      for (int k = 0; k < 3; ++k)
#pragma unroll
        for (int q = 0; q < 16; ++q) {
          const float a = fmaxf(__uint_as_float(v[k][2 * q]) + bias1[32 * k + 2 * q], 0.f);
          const float b = fmaxf(__uint_as_float(v[k][2 * q + 1]) + bias1[32 * k + 2 * q + 1], 0.f);
          pk[k][q] = pack_bf16(a, b);
        }
      st_half_packed(R1, th, pk);
      tmem_wait_st();
    }
    block_tmem_sync();
    // F5: P2 = O1 W2 + b2
    if (tid == 0) {
      issue_mlp(R0, R1, aW + 2 * kWBytes, id_mlp, true);
      issue_mlp(R0, R1 + BS / 2, aW + 3 * kWBytes, id_mlp | kIdescNegB, false);
      issue_mlp(R0 + BS, R1, aW + 3 * kWBytes, id_mlp, true);
      issue_mlp(R0 + BS, R1 + BS / 2, aW + 2 * kWBytes, id_mlp, false);
      mma_commit(&mbar);
    }
    mbar_wait(&mbar, phase);
    phase ^= 1;
    tc_fence_after();
    {
      // F6: bias + softshrink + truncation -> bf16 Z as the B operand of the inverse transform
      uint32_t v[3][32], pk[3][16];
      ld_half(R0, th, v);
#pragma unroll
      for (int k = 0; k < 3; ++k)
#pragma unroll
        for (int q = 0; q < 16; ++q) {
          float a = __uint_as_float(v[k][2 * q]) + bias2[32 * k + 2 * q];
          float b = __uint_as_float(v[k][2 * q + 1]) + bias2[32 * k + 2 * q + 1];
          const float ma = fabsf(a) - p.lambda, mb = fabsf(b) - p.lambda;
          a = (row_kept && ma > 0.f) ? copysignf(ma, a) : 0.f;
          b = (row_kept && mb > 0.f) ? copysignf(mb, b) : 0.f;
          pk[k][q] = pack_bf16(a, b);
        }
      if (r < HP) store_tile_half(sTile, th, pk);
    }
    fence_async_smem();
    block_tmem_sync();
    // F7: Tr = Ch Zr - Sh Zi ; Ti = Ch Zi + Sh Zr      (inverse kernel exp(+i theta))
    if (tid == 0) {
      issue_dft(R1, aCh, aTile, id_dft, true);
      issue_dft(R1, aSh, aTile + half, id_dft | kIdescNegA, false);
      issue_dft(R1 + BS, aCh, aTile + half, id_dft, true);
      issue_dft(R1 + BS, aSh, aTile, id_dft, false);
      mma_commit(&mbar);
    }
    mbar_wait(&mbar, phase);
    phase ^= 1;
    tc_fence_after();
    {
      uint32_t v[3][32], pk[3][16];
      ld_half(R1, th, v);
#pragma unroll
      for (int k = 0; k < 3; ++k)
#pragma unroll
        for (int q = 0; q < 16; ++q) pk[k][q] = pack_bf16(__uint_as_float(v[k][2 * q]), __uint_as_float(v[k][2 * q + 1]));
      if (r < p.H) store_row_half(p.A2 + (((size_t)rem * p.nb + j) * p.H + r) * NT + th.colh * BS, pk);
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc<512>(tmem);
}

// ---- B1-B7 (except the parameter sums): per (b, kw, block) backward chain ------------------------
//   recompute  Xh = Fh A1x -> P1 -> O1 -> P2 (masks kept as bit sets in registers)
//   G = Fh A1g ; G2 = G (.) mask2 ; G1 = mask1 (.) (G2 W2^H) ; GX = G1 W1^H ; A2 = Fh^H GX
// Xh, O1, G2, G1 are also written (bf16, tile layout [b*Kw+kw][j][r][192]) for tc_wgrad.
struct MixBwdParams {
  const __nv_bfloat16* A1x;
  const __nv_bfloat16* A1g;
  __nv_bfloat16* A2;
  __nv_bfloat16 *Xh, *O1, *G2, *G1;
  const uint8_t* dft;
  const uint8_t* wprep;
  const float* b1;
  const float* b2;
  uint8_t* mask1; // optional export, [B][H][Wh][C][2]
  uint8_t* mask2;
  int B, H, Kw, Wh, nb, Kh;
  float lambda;
};

constexpr uint32_t kMixBwdSmem = kMixSmem + kTileBytes; // second tile buffer for the gradient spectrum

__global__ void __launch_bounds__(kMixThreads, 1) tc_mix_bwd(MixBwdParams p) {
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ __align__(8) uint64_t mbar;
  __shared__ uint32_t tmem_slot;
  uint8_t* sCh = smem;
  uint8_t* sSh = smem + kDftBytes;
  uint8_t* sW = smem + 2 * kDftBytes;
  uint8_t* sTile = sW + 4 * kWBytes;
  float* sBias = (float*)(sTile + kTileBytes);
  uint8_t* sTileG = sTile + kTileBytes + 2 * NT * 4;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  for (uint32_t i = tid; i < kTileBytes / 16; i += kMixThreads) {
    ((uint4*)sTile)[i] = make_uint4(0, 0, 0, 0);
    ((uint4*)sTileG)[i] = make_uint4(0, 0, 0, 0);
  }
  for (uint32_t i = tid; i < 2 * kDftBytes / 16; i += kMixThreads)
    cp_async16(smem_u32(sCh) + i * 16, p.dft + (size_t)i * 16);
  if (tid == 0) {
    mbar_init(&mbar, 1);
    mbar_init_fence();
  }
  if (warp == 0) tmem_alloc<512>(&tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  MixThread th;
  th.lane_base = (uint32_t)((warp & 3) * 32) << 16;
  th.colh = warp >> 2;
  th.r = (warp & 3) * 32 + lane;
  const uint32_t R0 = tmem, R1 = tmem + 256;
  const uint32_t aCh = smem_u32(sCh), aSh = smem_u32(sSh), aW = smem_u32(sW);
  const uint32_t aTile = smem_u32(sTile), aTileG = smem_u32(sTileG);
  const uint32_t half = (BS / 8) * kTileSbo;
  const uint32_t id_dft = idesc_bf16(128, BS, kIdescBMn);
  const uint32_t id_mlp = idesc_bf16(128, BS);
  const uint32_t id_mlp_t = idesc_bf16(128, BS, kIdescBMn);

  const int ntiles = p.nb * p.B * p.Kw;
  const int per = (ntiles + gridDim.x - 1) / gridDim.x;
  const int t_begin = blockIdx.x * per, t_end = min(ntiles, t_begin + per);
  uint32_t phase = 0;
  int cur_j = -1;
  const int r = th.r;
  const int kappa = (r <= p.H / 2) ? r : p.H - r;
  const bool row_valid = r < p.H;
  const bool row_kept = row_valid && (kappa < p.Kh);
  const float* bias1 = sBias + th.colh * BS;
  const float* bias2 = sBias + NT + th.colh * BS;

  for (int t = t_begin; t < t_end; ++t) {
    const int j = t / (p.B * p.Kw);
    const int rem = t - j * (p.B * p.Kw);
    if (j != cur_j) {
      cur_j = j;
      const uint8_t* wsrc = p.wprep + (size_t)j * 8 * kWBytes;
      for (uint32_t i = tid; i < 4 * kWBytes / 16; i += kMixThreads) cp_async16(aW + i * 16, wsrc + (size_t)i * 16);
      for (int i = tid; i < 2 * NT; i += kMixThreads) {
        const int which = i / NT, n = i % NT, ri = n / BS, o = n % BS;
        sBias[i] = (which == 0 ? p.b1 : p.b2)[((size_t)j * BS + o) * 2 + ri];
      }
    }
    const size_t tile_off = ((size_t)rem * p.nb + j) * p.H * NT;
    load_tile(aTile, p.A1x + tile_off, p.H, warp, lane);
    load_tile(aTileG, p.A1g + tile_off, p.H, warp, lane);
    const size_t row_off = tile_off + (size_t)r * NT + th.colh * BS;
    cp_async_wait_all();
    fence_async_smem();
    block_tmem_sync();
    // ---- Xh = Fh A1x -----------------------------------------------------------------------
    if (tid == 0) {
      issue_dft(R0, aCh, aTile, id_dft, true);
      issue_dft(R0, aSh, aTile + half, id_dft, false);
      issue_dft(R0 + BS, aCh, aTile + half, id_dft, true);
      issue_dft(R0 + BS, aSh, aTile, id_dft | kIdescNegA, false);
      mma_commit(&mbar);
    }
    mbar_wait(&mbar, phase);
    phase ^= 1;
    tc_fence_after();
    {
      uint32_t v[3][32], pk[3][16];
      ld_half(R0, th, v);
      block_tmem_sync();
#pragma unroll
      for (int k = 0; k < 3; ++k)
#pragma unroll
        for (int q = 0; q < 16; ++q) pk[k][q] = pack_bf16(__uint_as_float(v[k][2 * q]), __uint_as_float(v[k][2 * q + 1]));
      st_half_packed(R0, th, pk);
      if (row_valid) store_row_half(p.Xh + row_off, pk);
      tmem_wait_st();
    }
    block_tmem_sync();
    // ---- P1 = Xh W1 + b1 ; O1 = relu ; mask1 -------------------------------------------------
    if (tid == 0) {
      issue_mlp(R1, R0, aW + 0 * kWBytes, id_mlp, true);
      issue_mlp(R1, R0 + BS / 2, aW + 1 * kWBytes, id_mlp | kIdescNegB, false);
      issue_mlp(R1 + BS, R0, aW + 1 * kWBytes, id_mlp, true);
      issue_mlp(R1 + BS, R0 + BS / 2, aW + 0 * kWBytes, id_mlp, false);
      mma_commit(&mbar);
    }
    mbar_wait(&mbar, phase);
    phase ^= 1;
    tc_fence_after();
    uint32_t m1[3], m2[3];
    {
      uint32_t v[3][32], pk[3][16];
      ld_half(R1, th, v);
      block_tmem_sync();
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        uint32_t bits = 0;
#pragma unroll
        for (int q = 0; q < 16; ++q) {
          const float a = __uint_as_float(v[k][2 * q]) + bias1[32 * k + 2 * q];
          const float b = __uint_as_float(v[k][2 * q + 1]) + bias1[32 * k + 2 * q + 1];
          bits |= (a > 0.f ? 1u : 0u) << (2 * q);
          bits |= (b > 0.f ? 1u : 0u) << (2 * q + 1);
          pk[k][q] = pack_bf16(fmaxf(a, 0.f), fmaxf(b, 0.f));
        }
        m1[k] = bits;
      }
      st_half_packed(R1, th, pk);
      if (row_valid) store_row_half(p.O1 + row_off, pk);
      tmem_wait_st();
    }
    block_tmem_sync();
    // ---- P2 = O1 W2 + b2 ; mask2 ----------------------------------------------------------------
    if (tid == 0) {
      issue_mlp(R0, R1, aW + 2 * kWBytes, id_mlp, true);
      issue_mlp(R0, R1 + BS / 2, aW + 3 * kWBytes, id_mlp | kIdescNegB, false);
      issue_mlp(R0 + BS, R1, aW + 3 * kWBytes, id_mlp, true);
      issue_mlp(R0 + BS, R1 + BS / 2, aW + 2 * kWBytes, id_mlp, false);
      mma_commit(&mbar);
    }
    mbar_wait(&mbar, phase);
    phase ^= 1;
    tc_fence_after();
    {
      uint32_t v[3][32];
      ld_half(R0, th, v);
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        uint32_t bits = 0;
#pragma unroll
        for (int q = 0; q < 32; ++q)
          bits |= (fabsf(__uint_as_float(v[k][q]) + bias2[32 * k + q]) > p.lambda ? 1u : 0u) << q;
        m2[k] = row_kept ? bits : 0u;
      }
    }
    block_tmem_sync();
    // ---- G = Fh A1g ; G2 = G (.) mask2 -----------------------------------------------------------
    if (tid == 0) {
      issue_dft(R1, aCh, aTileG, id_dft, true);
      issue_dft(R1, aSh, aTileG + half, id_dft, false);
      issue_dft(R1 + BS, aCh, aTileG + half, id_dft, true);
      issue_dft(R1 + BS, aSh, aTileG, id_dft | kIdescNegA, false);
      mma_commit(&mbar);
    }
    mbar_wait(&mbar, phase);
    phase ^= 1;
    tc_fence_after();
    {
      uint32_t v[3][32], pk[3][16];
      ld_half(R1, th, v);
      block_tmem_sync();
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        const uint32_t bits = m2[k];
#pragma unroll
        for (int q = 0; q < 16; ++q) {
          const float a = (bits >> (2 * q)) & 1u ? __uint_as_float(v[k][2 * q]) : 0.f;
          const float b = (bits >> (2 * q + 1)) & 1u ? __uint_as_float(v[k][2 * q + 1]) : 0.f;
          pk[k][q] = pack_bf16(a, b);
        }
      }
      st_half_packed(R1, th, pk);
      if (row_valid) store_row_half(p.G2 + row_off, pk);
      tmem_wait_st();
    }
    block_tmem_sync();
    // ---- G1 = mask1 (.) (G2 W2^H):  re = G2r W2r^T + G2i W2i^T ; im = G2i W2r^T - G2r W2i^T ----
    if (tid == 0) {
      issue_mlp_t(R0, R1, aW + 2 * kWBytes, id_mlp_t, true);
      issue_mlp_t(R0, R1 + BS / 2, aW + 3 * kWBytes, id_mlp_t, false);
      issue_mlp_t(R0 + BS, R1 + BS / 2, aW + 2 * kWBytes, id_mlp_t, true);
      issue_mlp_t(R0 + BS, R1, aW + 3 * kWBytes, id_mlp_t | kIdescNegB, false);
      mma_commit(&mbar);
    }
    mbar_wait(&mbar, phase);
    phase ^= 1;
    tc_fence_after();
    {
      uint32_t v[3][32], pk[3][16];
      ld_half(R0, th, v);
      block_tmem_sync();
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        const uint32_t bits = m1[k];
#pragma unroll
        for (int q = 0; q < 16; ++q) {
          const float a = (bits >> (2 * q)) & 1u ? __uint_as_float(v[k][2 * q]) : 0.f;
          const float b = (bits >> (2 * q + 1)) & 1u ? __uint_as_float(v[k][2 * q + 1]) : 0.f;
          pk[k][q] = pack_bf16(a, b);
        }
      }
      st_half_packed(R0, th, pk);
      if (row_valid) store_row_half(p.G1 + row_off, pk);
      tmem_wait_st();
    }
    block_tmem_sync();
    // ---- GX = G1 W1^H ----------------------------------------------------------------------------
    if (tid == 0) {
      issue_mlp_t(R1, R0, aW + 0 * kWBytes, id_mlp_t, true);
      issue_mlp_t(R1, R0 + BS / 2, aW + 1 * kWBytes, id_mlp_t, false);
      issue_mlp_t(R1 + BS, R0 + BS / 2, aW + 0 * kWBytes, id_mlp_t, true);
      issue_mlp_t(R1 + BS, R0, aW + 1 * kWBytes, id_mlp_t | kIdescNegB, false);
      mma_commit(&mbar);
    }
    mbar_wait(&mbar, phase);
    phase ^= 1;
    tc_fence_after();
    {
      uint32_t v[3][32], pk[3][16];
      ld_half(R1, th, v);
#pragma unroll
      for (int k = 0; k < 3; ++k)
#pragma unroll
        for (int q = 0; q < 16; ++q)
          pk[k][q] = row_valid ? pack_bf16(__uint_as_float(v[k][2 * q]), __uint_as_float(v[k][2 * q + 1])) : 0u;
      if (r < HP) store_tile_half(sTile, th, pk);
    }
    fence_async_smem();
    block_tmem_sync();
    // ---- A2 = Fh^H GX (inverse kernel) ---------------------------------------------------------
    if (tid == 0) {
      issue_dft(R0, aCh, aTile, id_dft, true);
      issue_dft(R0, aSh, aTile + half, id_dft | kIdescNegA, false);
      issue_dft(R0 + BS, aCh, aTile + half, id_dft, true);
      issue_dft(R0 + BS, aSh, aTile, id_dft, false);
      mma_commit(&mbar);
    }
    // optional mask export (test aid) while the tensor core works: bytes (re, im) interleaved per channel
    if (p.mask1 != nullptr && row_valid) {
      const int b = rem / p.Kw, kw = rem - b * p.Kw;
      const size_t base = ((((size_t)b * p.H + r) * p.Wh + kw) * (size_t)(p.nb * BS) + (size_t)j * BS) * 2 + th.colh;
#pragma unroll
      for (int k = 0; k < 3; ++k)
#pragma unroll 4
        for (int q = 0; q < 32; ++q) {
          p.mask1[base + (size_t)(32 * k + q) * 2] = (uint8_t)((m1[k] >> q) & 1u);
          p.mask2[base + (size_t)(32 * k + q) * 2] = (uint8_t)((m2[k] >> q) & 1u);
        }
    }
    mbar_wait(&mbar, phase);
    phase ^= 1;
    tc_fence_after();
    {
      uint32_t v[3][32], pk[3][16];
      ld_half(R0, th, v);
#pragma unroll
      for (int k = 0; k < 3; ++k)
#pragma unroll
        for (int q = 0; q < 16; ++q) pk[k][q] = pack_bf16(__uint_as_float(v[k][2 * q]), __uint_as_float(v[k][2 * q + 1]));
      if (row_valid) store_row_half(p.A2 + row_off, pk);
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc<512>(tmem);
}


// ---- B4 / B6: parameter gradients as a split-K tensor-core GEMM ------------------------------------
// For block j:  R[(ri_a,i), (ri_g,o)] = sum_rows A[row,(ri_a,i)] * G[row,(ri_g,o)] with K = mode rows.
// Two M=128 accumulators: D_re rows = (re, i) plus a constant-one row 96 (gives sum_rows G = db),
// D_im rows = (im, i).  CTA (j, s) sums tiles rem = s, s+S, ... and writes its partial sums.
constexpr uint32_t kWgABytes = HP * 128 * 2;                           // 24576: MN-major A [K=96][M=128]
constexpr uint32_t kWgStage = 2 * kWgABytes + kTileBytes;              // 86016
constexpr uint32_t kWgSmem = 2 * kWgStage;                             // 172032
constexpr uint32_t kWgALbo = 128, kWgASbo = 1536;

__global__ void __launch_bounds__(128, 1)
tc_wgrad(const __nv_bfloat16* __restrict__ Aws, const __nv_bfloat16* __restrict__ Gws, float* __restrict__ part,
         int BKw, int H, int nb, int S) {
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ __align__(8) uint64_t mbar[2];
  __shared__ uint32_t tmem_slot;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int j = blockIdx.x / S, s = blockIdx.x - j * S;
  for (uint32_t i = tid; i < kWgSmem / 16; i += 128) ((uint4*)smem)[i] = make_uint4(0, 0, 0, 0);
  __syncthreads();
  // constant-one column m = 96 of the "re" A operand, rows r < H, both stages
  for (int i = tid; i < 2 * H; i += 128) {
    const int st = i / H, rr = i - st * H;
    *(uint16_t*)(smem + st * kWgStage + 12 * kWgASbo + rr * 16) = 0x3F80; // bf16 1.0
  }
  if (tid == 0) {
    mbar_init(&mbar[0], 1);
    mbar_init(&mbar[1], 1);
    mbar_init_fence();
  }
  if (warp == 0) tmem_alloc<512>(&tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  const uint32_t lane_base = (uint32_t)(warp * 32) << 16;
  const uint32_t Dre = tmem, Dim = tmem + 256;
  const uint32_t idesc = idesc_bf16(128, NT, kIdescAMn | kIdescBMn);
  const int nt = (BKw - s + S - 1) / S; // tiles of this CTA
  const int hl = lane & 7, cl4 = lane >> 3;
  auto prefetch = [&](int it) {
    const int rem = s + it * S;
    const uint32_t stage = smem_u32(smem) + (it & 1) * kWgStage;
    const size_t off = ((size_t)rem * nb + j) * H * NT;
    const int nunits = ((H + 7) / 8) * 6;
    for (int u = warp; u < nunits; u += 4) {
      const int h = (u / 6) * 8 + hl;
      const int nc = (u % 6) * 4 + cl4;
      if (h < H) {
        const uint32_t adst = stage + (nc < 12 ? 0u : kWgABytes) + (nc % 12) * kWgASbo + h * 16;
        cp_async16(adst, Aws + off + (size_t)h * NT + nc * 8);
        cp_async16(stage + 2 * kWgABytes + nc * kTileSbo + h * 16, Gws + off + (size_t)h * NT + nc * 8);
      }
    }
  };
  if (nt > 0) prefetch(0);
  cp_async_commit();
  for (int it = 0; it < nt; ++it) {
    if (it + 1 < nt) {
      if (it >= 1) mbar_wait(&mbar[(it + 1) & 1], (uint32_t)(((it - 1) >> 1) & 1));
      prefetch(it + 1);
    }
    cp_async_commit();
    cp_async_wait_group<1>();
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    if (tid == 0) {
      tc_fence_after();
      const uint32_t stage = smem_u32(smem) + (it & 1) * kWgStage;
      const uint32_t g = stage + 2 * kWgABytes;
#pragma unroll
      for (int ks = 0; ks < HP / 16; ++ks) {
        const uint64_t bd = smem_desc(g + ks * 2 * kTileLbo, kTileLbo, kTileSbo);
        mma_ss(Dre, smem_desc(stage + ks * 2 * kWgALbo, kWgALbo, kWgASbo), bd, idesc, (it | ks) != 0);
        mma_ss(Dim, smem_desc(stage + kWgABytes + ks * 2 * kWgALbo, kWgALbo, kWgASbo), bd, idesc, (it | ks) != 0);
      }
      mma_commit(&mbar[it & 1]);
    }
  }
  float* dst = part + ((size_t)blockIdx.x * 2) * 128 * NT + (size_t)tid * NT;
  if (nt > 0) {
    mbar_wait(&mbar[(nt - 1) & 1], (uint32_t)(((nt - 1) >> 1) & 1));
    tc_fence_after();
#pragma unroll 1
    for (int acc = 0; acc < 2; ++acc)
#pragma unroll 1
      for (int c0 = 0; c0 < NT; c0 += 32) {
        uint32_t v[32];
        tmem_ld32((acc ? Dim : Dre) + lane_base + c0, v);
        tmem_wait_ld();
#pragma unroll
        for (int q = 0; q < 32; q += 4)
          *(float4*)(dst + (size_t)acc * 128 * NT + c0 + q) =
              make_float4(__uint_as_float(v[q]), __uint_as_float(v[q + 1]), __uint_as_float(v[q + 2]),
                          __uint_as_float(v[q + 3]));
      }
  } else {
    for (int acc = 0; acc < 2; ++acc)
      for (int c0 = 0; c0 < NT; c0 += 4) *(float4*)(dst + (size_t)acc * 128 * NT + c0) = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc<512>(tmem);
}

// dW[j][i][o] = sum_s ( Dre[i][o] + Dim[i][96+o] ,  Dre[i][96+o] - Dim[i][o] ) ;  db[j][o] = sum_s Dre[96][(ri,o)]
__global__ void k_tc_wgrad_reduce(const float* __restrict__ part, float2* __restrict__ dW, float2* __restrict__ dB,
                                  int nb, int S, int accumulate) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  const int nW = nb * BS * BS;
  if (idx < nW) {
    const int o = idx % BS, i = (idx / BS) % BS, j = idx / (BS * BS);
    float2 acc = accumulate ? dW[idx] : make_float2(0.f, 0.f);
    for (int s = 0; s < S; ++s) {
      const float* P = part + ((size_t)(j * S + s) * 2) * 128 * NT;
      const float* Pre = P + (size_t)i * NT;
      const float* Pim = P + (size_t)128 * NT + (size_t)i * NT;
      acc.x += Pre[o] + Pim[BS + o];
      acc.y += Pre[BS + o] - Pim[o];
    }
    dW[idx] = acc;
  } else if (idx < nW + nb * BS) {
    const int k = idx - nW, o = k % BS, j = k / BS;
    float2 acc = accumulate ? dB[k] : make_float2(0.f, 0.f);
    for (int s = 0; s < S; ++s) {
      const float* P = part + ((size_t)(j * S + s) * 2) * 128 * NT + (size_t)96 * NT;
      acc.x += P[o];
      acc.y += P[BS + o];
    }
    dB[k] = acc;
  }
}

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

struct TcWs {
  __nv_bfloat16 *A1, *A2, *wprep;
  __nv_bfloat16 *A1g, *Xh, *O1, *G2, *G1; // backward only
  float* part;
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
  const size_t spec = (size_t)g.B * g.Kw * g.nb * g.H * NT * 2;
  w.A1 = (__nv_bfloat16*)take(spec);
  w.A2 = (__nv_bfloat16*)take(spec);
  w.wprep = (__nv_bfloat16*)take((size_t)g.nb * 8 * kWBytes);
  if (backward) {
    w.A1g = (__nv_bfloat16*)take(spec);
    w.Xh = (__nv_bfloat16*)take(spec);
    w.O1 = (__nv_bfloat16*)take(spec);
    w.G2 = (__nv_bfloat16*)take(spec);
    w.G1 = (__nv_bfloat16*)take(spec);
    int S = 148 / g.nb;
    if (S < 1) S = 1;
    if (S > g.B * g.Kw) S = g.B * g.Kw;
    w.S = S;
    w.part = (float*)take((size_t)g.nb * S * 2 * 128 * NT * sizeof(float));
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
  // Ch, Sh: element (r, h) = cos / sin (2 pi r h / H) / sqrt(H); K-major [k/8][m/8]
  std::vector<uint16_t> dft(2 * kDftBytes / 2, 0);
  for (int r = 0; r < H; ++r)
    for (int h = 0; h < H; ++h) {
      const double a = two_pi * (double)((long)r * h % H) / (double)H, s = 1.0 / sqrt((double)H);
      const uint32_t off = ((h / 8) * kDftLbo + (r / 8) * kDftSbo + (r % 8) * 16 + (h % 8) * 2) / 2;
      dft[off] = host_bf16(cos(a) * s);
      dft[kDftBytes / 2 + off] = host_bf16(sin(a) * s);
    }
  // Fw^T: element (n = ri*96 + kw, k = w) = {cos, -sin}(2 pi kw w / W) / sqrt(W)  [x alpha_kw]
  // Gw^T: element (n = w, k = ri*96 + kw) = alpha_kw {cos, -sin}(2 pi kw w / W) / sqrt(W)  [or alpha = 1]
  std::vector<uint16_t> fw(kFwBytes / 2, 0), fwa(kFwBytes / 2, 0), gw(kFwBytes / 2, 0), gw1(kFwBytes / 2, 0);
  for (int kw = 0; kw < Wh; ++kw)
    for (int w = 0; w < W; ++w) {
      const double a = two_pi * (double)((long)kw * w % W) / (double)W, s = 1.0 / sqrt((double)W);
      const double alpha = (kw == 0 || 2 * kw == W) ? 1.0 : 2.0;
      for (int ri = 0; ri < 2; ++ri) {
        const double v = (ri == 0 ? cos(a) : -sin(a)) * s;
        const int n = ri * BS + kw;
        const uint32_t of = ((w / 8) * kFwLbo + (n / 8) * kFwSbo + (n % 8) * 16 + (w % 8) * 2) / 2;
        const uint32_t og = ((n / 8) * kFwLbo + (w / 8) * kFwSbo + (w % 8) * 16 + (n % 8) * 2) / 2;
        fw[of] = host_bf16(v);
        fwa[of] = host_bf16(v * alpha);
        gw[og] = host_bf16(v * alpha);
        gw1[og] = host_bf16(v);
      }
    }
  cudaError_t e = upload(dft, &out->dft);
  if (e == cudaSuccess) e = upload(fw, &out->fw);
  if (e == cudaSuccess) e = upload(fwa, &out->fw_alpha);
  if (e == cudaSuccess) e = upload(gw, &out->gw);
  if (e == cudaSuccess) e = upload(gw1, &out->gw_noalpha);
  if (e == cudaSuccess) e = set_smem(tc_wdft<false>, kRowSmem);
  if (e == cudaSuccess) e = set_smem(tc_wdft<true>, kRowSmem);
  if (e == cudaSuccess) e = set_smem(tc_mix_fwd, kMixFwdSmem);
  if (e == cudaSuccess) e = set_smem(tc_mix_bwd, kMixBwdSmem);
  if (e == cudaSuccess) e = set_smem(tc_wgrad, kWgSmem);
  int dev = 0, sms = 148;
  if (e == cudaSuccess) e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  out->num_sms = sms;
  out->valid = (e == cudaSuccess);
  return e;
}

size_t tc_workspace_bytes(const Geometry& g, bool backward) {
  return tc_carve(g, backward, nullptr).total;
}

cudaError_t tc_forward(const Geometry& g, const Plan& p, const void* x, const float* w1, const float* b1,
                       const float* w2, const float* b2, void* y, void* ws, cudaStream_t st) {
  TcWs w = tc_carve(g, false, (char*)ws);
  const TcPlan& tp = p.tc;
  cudaError_t e;
  const int nW = g.nb * BS * BS;
  prof_begin("k_tc_prep_weights", st);
  k_tc_prep_weights<<<(nW + 255) / 256, 256, 0, st>>>(w1, w2, w.wprep, g.nb);
  prof_end(st);
  count_launch();
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  const int ncg = (g.C + CGRP - 1) / CGRP;
  const int row_tiles = g.B * g.H * ncg;
  const int grid_row = row_tiles < tp.num_sms ? row_tiles : tp.num_sms;
  prof_begin("tc_wdft_fwd", st);
  tc_wdft<false><<<grid_row, kRowThreads, kRowSmem, st>>>((const __nv_bfloat16*)x, nullptr, w.A1, tp.fw, g.B, g.H, g.W,
                                                          g.C, g.Kw, g.nb);
  prof_end(st);
  count_launch();
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  MixParams mp{w.A1, w.A2, tp.dft, (const uint8_t*)w.wprep, b1, b2, g.B, g.H, g.Kw, g.nb, g.Kh, g.lambda};
  const int mix_tiles = g.nb * g.B * g.Kw;
  const int grid_mix = mix_tiles < tp.num_sms ? mix_tiles : tp.num_sms;
  prof_begin("tc_mix_fwd", st);
  tc_mix_fwd<<<grid_mix, kMixThreads, kMixFwdSmem, st>>>(mp);
  prof_end(st);
  count_launch();
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  prof_begin("tc_wdft_inv", st);
  tc_wdft<true><<<grid_row, kRowThreads, kRowSmem, st>>>(w.A2, g.no_residual ? nullptr : (const __nv_bfloat16*)x,
                                                         (__nv_bfloat16*)y, tp.gw, g.B, g.H, g.W, g.C, g.Kw, g.nb);
  prof_end(st);
  count_launch();
  return cudaGetLastError();
}

cudaError_t tc_backward(const Geometry& g, const Plan& p, const void* x, const void* dy, const float* w1,
                        const float* b1, const float* w2, const float* b2, void* dx, float* dw1, float* db1,
                        float* dw2, float* db2, void* ws, cudaStream_t st) {
  TcWs w = tc_carve(g, true, (char*)ws);
  const TcPlan& tp = p.tc;
  cudaError_t e;
#define TC_LAUNCH(name, ...)                                  \
  prof_begin(name, st);                                       \
  __VA_ARGS__;                                                \
  prof_end(st);                                               \
  count_launch();                                             \
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  const int nW = g.nb * BS * BS;
  if (g.export_masks) {
    if ((e = cudaMemsetAsync(ws, 0, w.mask_region, st)) != cudaSuccess) return e;
  }
  TC_LAUNCH("k_tc_prep_weights", k_tc_prep_weights<<<(nW + 255) / 256, 256, 0, st>>>(w1, w2, w.wprep, g.nb));
  const int ncg = (g.C + CGRP - 1) / CGRP;
  const int row_tiles = g.B * g.H * ncg;
  const int grid_row = row_tiles < tp.num_sms ? row_tiles : tp.num_sms;
  // B1 (first half) and B2: W-direction spectra of x and of dy (alpha-weighted)
  TC_LAUNCH("tc_wdft_fwd", tc_wdft<false><<<grid_row, kRowThreads, kRowSmem, st>>>((const __nv_bfloat16*)x, nullptr, w.A1,
                                                                                  tp.fw, g.B, g.H, g.W, g.C, g.Kw, g.nb));
  TC_LAUNCH("tc_wdft_fwd", tc_wdft<false><<<grid_row, kRowThreads, kRowSmem, st>>>((const __nv_bfloat16*)dy, nullptr, w.A1g,
                                                                                  tp.fw_alpha, g.B, g.H, g.W, g.C, g.Kw, g.nb));
  MixBwdParams mp{};
  mp.A1x = w.A1; mp.A1g = w.A1g; mp.A2 = w.A2;
  mp.Xh = w.Xh; mp.O1 = w.O1; mp.G2 = w.G2; mp.G1 = w.G1;
  mp.dft = tp.dft; mp.wprep = (const uint8_t*)w.wprep; mp.b1 = b1; mp.b2 = b2;
  mp.mask1 = g.export_masks ? w.mask1 : nullptr;
  mp.mask2 = g.export_masks ? w.mask2 : nullptr;
  mp.B = g.B; mp.H = g.H; mp.Kw = g.Kw; mp.Wh = g.Wh; mp.nb = g.nb; mp.Kh = g.Kh; mp.lambda = g.lambda;
  const int mix_tiles = g.nb * g.B * g.Kw;
  const int grid_mix = mix_tiles < tp.num_sms ? mix_tiles : tp.num_sms;
  TC_LAUNCH("tc_mix_bwd", tc_mix_bwd<<<grid_mix, kMixThreads, kMixBwdSmem, st>>>(mp));
  // B4 / B6: parameter gradients
  const int nred = nW + g.nb * BS;
  TC_LAUNCH("tc_wgrad", tc_wgrad<<<g.nb * w.S, 128, kWgSmem, st>>>(w.O1, w.G2, w.part, g.B * g.Kw, g.H, g.nb, w.S));
  TC_LAUNCH("k_tc_wgrad_reduce", k_tc_wgrad_reduce<<<(nred + 255) / 256, 256, 0, st>>>(
                                     w.part, (float2*)dw2, (float2*)db2, g.nb, w.S, g.accum ? 1 : 0));
  TC_LAUNCH("tc_wgrad", tc_wgrad<<<g.nb * w.S, 128, kWgSmem, st>>>(w.Xh, w.G1, w.part, g.B * g.Kw, g.H, g.nb, w.S));
  TC_LAUNCH("k_tc_wgrad_reduce", k_tc_wgrad_reduce<<<(nred + 255) / 256, 256, 0, st>>>(
                                     w.part, (float2*)dw1, (float2*)db1, g.nb, w.S, g.accum ? 1 : 0));
  // B8: dx = dy + irfft2(GX / alpha)
  TC_LAUNCH("tc_wdft_inv", tc_wdft<true><<<grid_row, kRowThreads, kRowSmem, st>>>(
                               w.A2, g.no_residual ? nullptr : (const __nv_bfloat16*)dy, (__nv_bfloat16*)dx,
                               tp.gw_noalpha, g.B, g.H, g.W, g.C, g.Kw, g.nb));
#undef TC_LAUNCH
  return cudaSuccess;
}

} // namespace afno
