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

constexpr int BS = 96;    // channel block size handled by this path
constexpr int NT = 192;   // (re | im) columns of one block
constexpr int HP = 96;    // H padded to the K extent of the H-direction GEMMs
constexpr int WP = 192;   // W padded to the K / N extent of the W-direction GEMMs
constexpr int kA2Row = NT + 8; // elements per stored row of A1 / A2: 192 values + 16 bytes of padding
// Rows of the half-spectra are 400 bytes apart, in shared-memory staging (eight consecutive rows fall
// into distinct 16-byte bank groups) AND in global memory, so that staged rows leave with ONE bulk copy.
constexpr uint32_t kOutStride = 2 * kA2Row;           // 400

// shared-memory operand geometry (bytes), see tc_common.cuh for the layout formulas
constexpr uint32_t kWLbo = 1536, kWSbo = 128;       // weights: K-major B [96 x 96], order [k/8][n/8]
constexpr uint32_t kWBytes = BS * BS * 2;            // 18432
// mode tile (no-swizzle layout of Z / GX and of the operand images): MN-major B [K=96 rows][N=192],
// chunk stride padded by 16 bytes (rows of one chunk are 16 bytes apart: a warp's 32 rows store 512
// contiguous bytes, conflict-free)
constexpr uint32_t kTileLbo = 128, kTileSbo = 1536 + 16;
constexpr uint32_t kTileBytes = (NT / 8) * kTileSbo; // 37248
// ---- weight preparation: fp32 [nb][96][96][2] -> bf16 K-major interleaved operands --------------
// per block 4 matrices of kWBytes {W1r, W1i, W2r, W2i} with element (n=o, k=i) = W[i][o] (the
// backward pass reads the same images as MN-major operands), and the biases regrouped as
// [block][layer][re 96 | im 96] fp32.
__global__ void k_tc_prep_weights(const float* __restrict__ w1, const float* __restrict__ b1,
                                  const float* __restrict__ w2, const float* __restrict__ b2,
                                  __nv_bfloat16* __restrict__ out, float* __restrict__ bout, int nb) {
  pdl_launch_dependents();
  pdl_wait();
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < nb * BS) {
    const int o = idx % BS, j = idx / BS;
    const float2 a = ((const float2*)b1)[idx], b = ((const float2*)b2)[idx];
    float* bb = bout + (size_t)j * 2 * NT;
    bb[o] = a.x;
    bb[BS + o] = a.y;
    bb[NT + o] = b.x;
    bb[NT + BS + o] = b.y;
  }
  if (idx >= nb * BS * BS) return;
  const int o = idx % BS, i = (idx / BS) % BS, j = idx / (BS * BS);
  const float2 a = ((const float2*)w1)[idx], b = ((const float2*)w2)[idx];
  __nv_bfloat16* base = out + (size_t)j * 4 * (kWBytes / 2);
  const uint32_t f = ((i / 8) * kWLbo + (o / 8) * kWSbo + (o % 8) * 16 + (i % 8) * 2) / 2; // n=o, k=i
  const uint32_t m = kWBytes / 2;
  base[0 * m + f] = __float2bfloat16_rn(a.x);
  base[1 * m + f] = __float2bfloat16_rn(a.y);
  base[2 * m + f] = __float2bfloat16_rn(b.x);
  base[3 * m + f] = __float2bfloat16_rn(b.y);
}

__device__ __forceinline__ void pack32(const uint32_t (&v)[32], uint32_t (&pk)[16]) {
#pragma unroll
  for (int q = 0; q < 16; ++q) pk[q] = pack_bf16(__uint_as_float(v[2 * q]), __uint_as_float(v[2 * q + 1]));
}

// Which copies carry a non-default L2 eviction policy (chosen by measurement, S5.3); bit set =
// the policy named in the comment, clear = evict_normal.
enum {
  kPolWfLoad = 1,     // tc_wdft_fwd2: activation loads evict_first
  kPolWfStore = 2,    // tc_wdft_fwd2: A1 stores evict_last
  kPolWiLoad = 4,     // tc_wdft_inv2: A2 and residual loads evict_first
  kPolWiStore = 8,    // tc_wdft_inv2: y stores evict_first
  kPolMixLoad = 16,   // tc_mix2: tile loads evict_first
  kPolMixStore = 32,  // tc_mix2: A2 stores evict_last
  kPolMixImg = 64,    // tc_mix2: Xh, O1 stores evict_first; G2, G1 stores evict_last
  kPolWgLoad = 128    // tc_wgrad: operand loads evict_first
};
#ifdef AFNO_POLICY_EXPERIMENT
__device__ int g_polmask = 255;
#define POLMASK g_polmask
#else
constexpr int kPolMask = kPolWfStore | kPolWgLoad;   // measured: 0 -> 496 us per step, all -> 499, this choice -> 486
#define POLMASK kPolMask
#endif
__device__ __forceinline__ uint64_t pol_first(int bit) { return (POLMASK & bit) ? l2_evict_first() : l2_evict_normal(); }
__device__ __forceinline__ uint64_t pol_last(int bit) { return (POLMASK & bit) ? l2_evict_last() : l2_evict_normal(); }

#ifdef AFNO_TRACE
__device__ long long g_afno_trace[64 * 32];
#define TR(t, slot) do { if (blockIdx.x == 0 && (threadIdx.x & 31) == 0 && (t) >= 40 && (t) < 72) g_afno_trace[((t) - 40) * 64 + (slot)] = clock64(); } while (0)
#else
#define TR(t, slot)
#endif
#ifdef AFNO_TIMING
__device__ long long g_afno_dbg[128];
#define DBG_T0() long long dbg_t = clock64()
#define DBG_ACC(slot) do { long long n_ = clock64(); dbg_acc[slot] += n_ - dbg_t; dbg_t = n_; } while (0)
// per-CTA start / end wall-clock (ns) of the last launch of kernel family k (load balance of the static tile schedule)
__device__ long long g_afno_span[5][160][2];
#define SPAN(k, e) do { if (threadIdx.x == 0 && blockIdx.x < 160) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); g_afno_span[k][blockIdx.x][e] = (long long)t_; } } while (0)
// timeline of CTA 0: wall-clock (ns) at a few points of a kernel
#define TL(slot) do { if (blockIdx.x == 0 && threadIdx.x == 0) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); g_afno_dbg[slot] = (long long)t_; } } while (0)
#else
#define DBG_T0()
#define DBG_ACC(slot)
#define TL(slot)
#define SPAN(k, e)
#endif

// ---- F1 / B2 and F8 + F9 / B8: the W-direction transforms, all global traffic through bulk tensor copies --
// One tile = (b, h, channel block j): N = 96 channels.  The activation tile arrives as three
// 64B-swizzled panels [192 rows (w, zero-filled past W)][32 channels] written by TMA, leaves as rows
// staged in shared memory and sent by one TMA store: no LSU instruction touches global memory, so
// the kernels run at the speed of the copy engines instead of the load/store pipe.
//   forward : D_ri[kw, c] = sum_w Fw_ri[kw, w] x[b,h,w,c]      -> A1 rows [kw][re 96 | im 96 | pad 8]
//   inverse : D_a[w, c]   = sum_(ri,kw) Gw[w, (ri,kw)] A2[..]  -> y[b,h,w,c] = residual + D
// Under load a bulk copy takes ~5 us to land, so bandwidth is bought with bytes in flight: the
// constant DFT matrix (A operand, 2 x [128 x 192] bf16) lives in TENSOR memory (192 columns), which
// leaves all of shared memory to the ring of tiles (6 slots forward, 3 + 3 inverse).  The two
// accumulator halves occupy 192 more columns; a half is handed back as soon as it is in registers.
// 8 warps: warps with (warp % 4) < rows/32 drain the accumulators (TMEM lane quarter = warp % 4),
// one spare warp issues the TMA loads, one the UMMAs.
constexpr int kW2Threads = 256;
constexpr uint32_t kPanel = 192 * 64;                      // 12288: one [192 x 32] bf16 panel
constexpr uint32_t kW2Tile = 3 * kPanel;                   // 36864: a [192 x 96] tile
constexpr uint32_t kCImgWords = 2 * 128 * (WP / 2);        // constant image: [half][6 column groups][row 0..127][16 words = K pairs]
constexpr uint32_t kCCols = WP;                            // TMEM columns of the constant: half a at a * 96
constexpr int kWfSlots = 6;
constexpr uint32_t kWfSmem = kWfSlots * kW2Tile + 1024;    // 222208
constexpr int kWiSlots = 3;
constexpr uint32_t kWiSmem = 2 * kWiSlots * kW2Tile + 1024;

// constant matrix image (global) -> tensor memory columns [0, 192); warps 0..3 load half 0, warps 4..7
// half 1 (lane quarter = warp % 4).  The image is stored [half][column group of 16][row][16 words], so a
// warp's 32 rows of one group are 2 KB contiguous (coalesced: every CTA of the grid reads the same 98 KB at
// the same moment); all of a thread's loads are in flight at once.
__device__ __forceinline__ size_t cimg_word(int a, int row, int word) {
  return (((size_t)a * 6 + word / 16) * 128 + row) * 16 + word % 16;
}
__device__ __forceinline__ void load_const_tmem(uint32_t tmem, const uint32_t* __restrict__ img, int warp, int lane) {
  const int a = warp >> 2, q4 = warp & 3;
  const uint32_t dst = tmem + ((uint32_t)(q4 * 32) << 16) + a * (WP / 2);
  uint4 t[24];
#pragma unroll
  for (int c = 0; c < 6; ++c) {
    const uint4* src = (const uint4*)(img + cimg_word(a, q4 * 32 + lane, 16 * c));
#pragma unroll
    for (int q = 0; q < 4; ++q) t[4 * c + q] = __ldg(src + q);
  }
#pragma unroll
  for (int c = 0; c < 6; ++c) {
    uint32_t v[16];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      v[4 * q] = t[4 * c + q].x; v[4 * q + 1] = t[4 * c + q].y; v[4 * q + 2] = t[4 * c + q].z; v[4 * q + 3] = t[4 * c + q].w;
    }
    tmem_st16(dst + 16 * c, v);
  }
  tmem_wait_st();
}

__global__ void __launch_bounds__(kW2Threads, 1)
tc_wdft_fwd2(const __grid_constant__ CUtensorMap mapX, const __grid_constant__ CUtensorMap mapA1,
             const uint32_t* __restrict__ Fimg, int ntiles, int nb, int H, int Kw) {
  extern __shared__ uint8_t smem_raw[];
  TL(0);
  SPAN(0, 0);
  __shared__ __align__(8) uint64_t full[kWfSlots], sfree[kWfSlots], accfull[2], accempty[2];
  __shared__ uint32_t tmem_slot;
  const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem = smem_raw + (base - smem_u32(smem_raw));
  const uint32_t aS = base;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  if (tid == 0) {
    for (int q = 0; q < kWfSlots; ++q) {
      mbar_init(&full[q], 1);
      mbar_init(&sfree[q], 1);
    }
    for (int q = 0; q < 2; ++q) {
      mbar_init(&accfull[q], 1);
      mbar_init(&accempty[q], 3);
    }
    mbar_init_fence();
    tma_prefetch_desc(&mapX);
    tma_prefetch_desc(&mapA1);
  }
  if (warp == 0) tmem_alloc<512>(&tmem_slot);
  pdl_launch_dependents();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  TL(1);
  load_const_tmem(tmem, Fimg, warp, lane);   // plan constant: loads under the previous kernel's tail
  TL(2);
  pdl_wait();
  TL(3);
  const int nmine = ntiles > (int)blockIdx.x ? (ntiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;

  const uint64_t pol_stream = pol_first(kPolWfLoad), pol_keep = pol_last(kPolWfStore);
  // TMA producer (warp 7): tile it -> slot it % 6
  auto produce = [&](int it) {
    const int s = it % kWfSlots;
    if (it >= kWfSlots) mbar_wait(&sfree[s], (uint32_t)((it / kWfSlots - 1) & 1));
    const int t = blockIdx.x + it * gridDim.x;
    const int j = t % nb, bh = t / nb;
    mbar_expect_tx(&full[s], kW2Tile);
#pragma unroll
    for (int pn = 0; pn < 3; ++pn)
      tma_load3(aS + s * kW2Tile + pn * kPanel, &mapX, j * BS + pn * 32, 0, bh, &full[s], pol_stream);
  };
  if (warp == 7) {
    // the first ring of loads starts at once, under the load of the constant
    if (elect_one())
      for (int it = 0; it < kWfSlots && it < nmine; ++it) produce(it);
    __syncwarp();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();

  if (warp == 7) {
    if (elect_one())
      for (int it = kWfSlots; it < nmine; ++it) produce(it);
    __syncwarp();
  } else if (warp == 3) {
    // ===== MMA issuer: half a = (re | im) rows of the transform, accumulator columns 192 + 96 a =======
    const uint32_t idesc = idesc_bf16(128, BS, kIdescBMn);
    for (int it = 0; it < nmine; ++it) {
      const int s = it % kWfSlots;
      mbar_wait(&full[s], (uint32_t)((it / kWfSlots) & 1));
      const uint32_t bt = aS + s * kW2Tile;
#pragma unroll
      for (int a = 0; a < 2; ++a) {
        if (it >= 1) mbar_wait(&accempty[a], (uint32_t)((it - 1) & 1));
        tc_fence_after();
        if (elect_one()) {
#pragma unroll
          for (int ks = 0; ks < WP / 16; ++ks)
            mma_ts(tmem + kCCols + a * BS, tmem + a * (WP / 2) + ks * 8, smem_desc_sw64(bt + ks * 1024, kPanel, 512), idesc,
                   ks > 0);
          mma_commit(&accfull[a]);
        }
        __syncwarp();
      }
    }
  } else {
    // ===== epilogue warps 0,1,2 (re) and 4,5,6 (im): row kw = 32 * (warp % 4) + lane ==================
    const int a = warp >> 2, q4 = warp & 3;
    const int kw = q4 * 32 + lane;
    const uint32_t lane_base = (uint32_t)(q4 * 32) << 16;
    const uint32_t acc = tmem + kCCols + a * BS + lane_base;
    for (int it = 0; it < nmine; ++it) {
      const int s = it % kWfSlots;
      const int t = blockIdx.x + it * gridDim.x;
      const int j = t % nb, bh = t / nb, b = bh / H, h = bh - b * H;
      mbar_wait(&accfull[a], (uint32_t)(it & 1));
      tc_fence_after();
      uint32_t v0[32], v1[32], v2[32];
      tmem_ld32(acc, v0);
      tmem_ld32(acc + 32, v1);
      tmem_ld32(acc + 64, v2);
      tmem_wait_ld();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&accempty[a]);
      // the tile's own operand slot is free once BOTH halves' MMAs have read it: stage the output rows there
      if (a == 0) mbar_wait(&accfull[1], (uint32_t)(it & 1));
      uint8_t* row = smem + s * kW2Tile + kw * kOutStride + a * (BS * 2);
      if (kw < Kw) {
        uint32_t pk[16];
        pack32(v0, pk);
#pragma unroll
        for (int g = 0; g < 4; ++g) *(uint4*)(row + g * 16) = make_uint4(pk[4 * g], pk[4 * g + 1], pk[4 * g + 2], pk[4 * g + 3]);
        pack32(v1, pk);
#pragma unroll
        for (int g = 0; g < 4; ++g) *(uint4*)(row + 64 + g * 16) = make_uint4(pk[4 * g], pk[4 * g + 1], pk[4 * g + 2], pk[4 * g + 3]);
        pack32(v2, pk);
#pragma unroll
        for (int g = 0; g < 4; ++g) *(uint4*)(row + 128 + g * 16) = make_uint4(pk[4 * g], pk[4 * g + 1], pk[4 * g + 2], pk[4 * g + 3]);
      }
      fence_async_smem();
      asm volatile("bar.sync 1, 192;" ::: "memory");
      if (warp == 0 && elect_one()) {
        tma_store5(&mapA1, 0, h, j, 0, b, aS + s * kW2Tile, pol_keep);   // the next kernel reads A1
        bulk_commit();
        if (it > 0) {
          bulk_wait_read<1>();   // the previous tile's store has read its slot
          mbar_arrive(&sfree[(it - 1) % kWfSlots]);
        }
      }
      __syncwarp();
    }
    if (warp == 0 && elect_one()) bulk_wait<0>();
    __syncwarp();
  }
  tc_fence_before();
  __syncthreads();
  TL(4);
  SPAN(0, 1);
  if (warp == 0) tmem_dealloc<512>(tmem);
}

// inverse: a ring of 3 operand tiles (A2 rows as K = ri * 96 + kw) and a ring of 3 residual / output tiles
__global__ void __launch_bounds__(kW2Threads, 1)
tc_wdft_inv2(const __grid_constant__ CUtensorMap mapA2, const __grid_constant__ CUtensorMap mapRes,
             const __grid_constant__ CUtensorMap mapY, const uint32_t* __restrict__ Gimg, int ntiles, int nb, int H, int W,
             int has_res) {
  extern __shared__ uint8_t smem_raw[];
  TL(8);
  SPAN(1, 0);
  __shared__ __align__(8) uint64_t ofull[kWiSlots], ofree[kWiSlots], rfull[kWiSlots], rfree[kWiSlots], accfull[2], accempty[2];
  __shared__ uint32_t tmem_slot;
  const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem = smem_raw + (base - smem_u32(smem_raw));
  const uint32_t aO = base, aR = aO + kWiSlots * kW2Tile;
  uint8_t* sR = smem + kWiSlots * kW2Tile;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  if (tid == 0) {
    for (int q = 0; q < kWiSlots; ++q) {
      mbar_init(&ofull[q], 1);
      mbar_init(&ofree[q], 1);
      mbar_init(&rfull[q], 1);
      mbar_init(&rfree[q], 1);
    }
    mbar_init(&accfull[0], 1);
    mbar_init(&accfull[1], 1);
    mbar_init(&accempty[0], 4);
    mbar_init(&accempty[1], 2);
    mbar_init_fence();
    tma_prefetch_desc(&mapA2);
    tma_prefetch_desc(&mapRes);
    tma_prefetch_desc(&mapY);
  }
  if (warp == 0) tmem_alloc<512>(&tmem_slot);
  pdl_launch_dependents();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  TL(9);
  load_const_tmem(tmem, Gimg, warp, lane);   // plan constant: loads under the previous kernel's tail
  TL(10);
  pdl_wait();
  TL(11);
  const int nmine = ntiles > (int)blockIdx.x ? (ntiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;

  const uint64_t pol_stream = pol_first(kPolWiLoad), pol_out = pol_first(kPolWiStore);
  // TMA producer (warp 6)
  auto produce = [&](int it) {
    const int s = it % kWiSlots;
    const uint32_t par = (uint32_t)((it / kWiSlots - 1) & 1);
    const int t = blockIdx.x + it * gridDim.x;
    const int j = t % nb, bh = t / nb, b = bh / H, h = bh - b * H;
    if (it >= kWiSlots) mbar_wait(&ofree[s], par);   // the slot's previous MMAs have completed
    mbar_expect_tx(&ofull[s], kW2Tile);
#pragma unroll
    for (int pn = 0; pn < 6; ++pn)   // panel pn = ri * 3 + n -> K rows ri * 96.., N panel n
      tma_load5(aO + s * kW2Tile + (pn % 3) * kPanel + (pn / 3) * (BS * 64), &mapA2, 0, pn, j * H + h, 0, b, &ofull[s], pol_stream);
    if (has_res) {
      if (it >= kWiSlots) mbar_wait(&rfree[s], par);  // the slot's previous store has read it
      mbar_expect_tx(&rfull[s], kW2Tile);
#pragma unroll
      for (int pn = 0; pn < 3; ++pn)
        tma_load3(aR + s * kW2Tile + pn * kPanel, &mapRes, j * BS + pn * 32, 0, bh, &rfull[s], pol_stream);
    }
  };
  if (warp == 6) {
    // the first ring of loads starts at once, under the load of the constant
    if (elect_one())
      for (int it = 0; it < kWiSlots && it < nmine; ++it) produce(it);
    __syncwarp();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();

  if (warp == 6) {
    if (elect_one())
      for (int it = kWiSlots; it < nmine; ++it) produce(it);
    __syncwarp();
  } else if (warp == 7) {
    // ===== MMA issuer: half a = rows w = 128 a .. of the transform, accumulator columns 192 + 96 a =====
    const uint32_t idesc = idesc_bf16(128, BS, kIdescBMn);
    for (int it = 0; it < nmine; ++it) {
      const int s = it % kWiSlots;
      mbar_wait(&ofull[s], (uint32_t)((it / kWiSlots) & 1));
      const uint32_t bt = aO + s * kW2Tile;
#pragma unroll
      for (int a = 0; a < 2; ++a) {
        if (it >= 1) mbar_wait(&accempty[a], (uint32_t)((it - 1) & 1));
        tc_fence_after();
        if (elect_one()) {
#pragma unroll
          for (int ks = 0; ks < WP / 16; ++ks)
            mma_ts(tmem + kCCols + a * BS, tmem + a * (WP / 2) + ks * 8, smem_desc_sw64(bt + ks * 1024, kPanel, 512), idesc,
                   ks > 0);
          mma_commit(&accfull[a]);
          if (a == 1) mma_commit(&ofree[s]);
        }
        __syncwarp();
      }
    }
  } else {
    // ===== epilogue warps 0..3 (w < 128) and 4, 5 (w = 128..191): row w = 128 a + 32 (warp % 4) + lane ==
    const int a = warp >> 2, q4 = warp & 3;
    const int w = a * 128 + q4 * 32 + lane;
    const uint32_t lane_base = (uint32_t)(q4 * 32) << 16;
    const uint32_t acc = tmem + kCCols + a * BS + lane_base;
    for (int it = 0; it < nmine; ++it) {
      const int s = it % kWiSlots;
      const uint32_t par = (uint32_t)((it / kWiSlots) & 1);
      const int t = blockIdx.x + it * gridDim.x;
      const int j = t % nb, bh = t / nb;
      uint8_t* rt = sR + s * kW2Tile;
      mbar_wait(&accfull[a], (uint32_t)(it & 1));
      tc_fence_after();
      uint32_t v[3][32];
      tmem_ld32(acc, v[0]);
      tmem_ld32(acc + 32, v[1]);
      tmem_ld32(acc + 64, v[2]);
      tmem_wait_ld();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&accempty[a]);
      if (has_res) {
        mbar_wait(&rfull[s], par);
      } else if (it >= kWiSlots) {
        // no residual load to wait for: the slot's previous store must have read it
        mbar_wait(&rfree[s], par ^ 1u);
      }
      if (w < W) {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          uint8_t* pan = rt + k * kPanel;
#pragma unroll
          for (int g = 0; g < 4; ++g) {
            uint4* ptr = (uint4*)(pan + sw64_off(w, g));
            uint4 r = make_uint4(0, 0, 0, 0);
            if (has_res) r = *ptr;
            // bf16 -> fp32 is a 16-bit shift; one rounding of (residual + branch)
            uint4 o;
            o.x = pack_bf16(__uint_as_float(v[k][8 * g + 0]) + __uint_as_float(r.x << 16),
                            __uint_as_float(v[k][8 * g + 1]) + __uint_as_float(r.x & 0xFFFF0000u));
            o.y = pack_bf16(__uint_as_float(v[k][8 * g + 2]) + __uint_as_float(r.y << 16),
                            __uint_as_float(v[k][8 * g + 3]) + __uint_as_float(r.y & 0xFFFF0000u));
            o.z = pack_bf16(__uint_as_float(v[k][8 * g + 4]) + __uint_as_float(r.z << 16),
                            __uint_as_float(v[k][8 * g + 5]) + __uint_as_float(r.z & 0xFFFF0000u));
            o.w = pack_bf16(__uint_as_float(v[k][8 * g + 6]) + __uint_as_float(r.w << 16),
                            __uint_as_float(v[k][8 * g + 7]) + __uint_as_float(r.w & 0xFFFF0000u));
            *ptr = o;
          }
        }
      }
      fence_async_smem();
      asm volatile("bar.sync 1, 192;" ::: "memory");
      if (warp == 0 && elect_one()) {
#pragma unroll
        for (int pn = 0; pn < 3; ++pn) tma_store3(&mapY, j * BS + pn * 32, 0, bh, aR + s * kW2Tile + pn * kPanel, pol_out);
        bulk_commit();
        if (it > 0) {
          bulk_wait_read<1>();
          mbar_arrive(&rfree[(it - 1) % kWiSlots]);
        }
      }
      __syncwarp();
    }
    if (warp == 0 && elect_one()) bulk_wait<0>();
    __syncwarp();
  }
  tc_fence_before();
  __syncthreads();
  TL(12);
  SPAN(1, 1);
  if (warp == 0) tmem_dealloc<512>(tmem);
}

// ---- F2-F7 / B1-B7: per (b, kw, block) GEMM chains in tensor memory (kernel tc_mix2 below) ----------

struct MixParams {
  CUtensorMap mapA1;         // input tiles (forward: spectrum of x; stateless backward: the same), see tile_tmap
  CUtensorMap mapA1g;        // backward: gradient tiles
  __nv_bfloat16* A2;
  __nv_bfloat16 *Xh, *O1, *G2, *G1; // backward: operands of tc_wgrad
  const uint8_t* dft;        // Ch then Sh, kDft2Bytes each, smem image
  const uint8_t* wprep;      // per block 4 x kWBytes: W1r, W1i, W2r, W2i (n=o, k=i, K-major)
  const float* bprep;        // per block [2 layers][192]: (re 96 | im 96)
  uint8_t* mask1;            // optional export, [B][H][Wh][C][2]
  uint8_t* mask2;
  uint4* maskbits;           // saved context: [tile][12 epilogue warps][32 lanes] {m1[0], m1[1], m2[0], m2[1]}
  int B, H, Kw, Wh, nb, Kh;
  float lambda;
};

// ---- tc_mix2: two mode tiles in flight per CTA (ping-pong), 12 epilogue warps ------------------------
// Same arithmetic and the same stages as tc_mix, rescheduled so that the tensor core and the
// epilogue warps never wait for each other:
//   * the CTA runs two tile streams X and Y; "phase" t belongs to stream t & 1 and is stage
//     (t >> 1) % NS of that stream's current tile.  The control warp issues the GEMMs S_0, S_1, ..
//     in phase order, the epilogue warps drain E_0, E_1, .. in phase order; S_t only waits for
//     E_(t-2) (the same stream's previous stage) and E_t for S_t, so S_(t+1) runs under E_t.
//   * tensor memory is five 96-column slots; phase t accumulates (re | im) into slots 3t, 3t+1
//     (mod 5), its epilogue compacts the bf16 A operand of the next GEMM into slot 3t, which
//     frees slot 3t+1; by the time S_(t+2) needs its two slots, 3t+1 and 3t+2 (the A operand of
//     S_(t+1), read by the in-order tensor pipe before S_(t+2) writes) are free: 480 columns.
//   * accumulator rows >= 96 hold nothing (H <= 96), so the warps of TMEM lane quarter 3
//     (warp % 4 == 3) are the control warp (3), the copy warp (7), the image warp (11) and a spare;
//     each of lane quarters 0..2 has four epilogue warps, one per 48-column quarter (re lo, re hi,
//     im lo, im hi).
//   * three tile buffers: tile i lives in buffer i % 3: the input tile (six 64B-swizzled TMA panels),
//     then staged operand images (FwdSave / BwdCtx), then the B operand of the inverse transform, then
//     the staged output rows; stateless backward: x tile, then the gradient tile, then GX.
// Every CTA works on ONE channel block j (grid = nb * S), so the weights are loaded once.
constexpr int kMix2Threads = 512;
constexpr uint32_t kDft2Lbo = 1536, kDft2Sbo = 128;  // Ch / Sh: K-major A, 96 stored rows, order [k/8][m/8 < 12]
constexpr uint32_t kDft2Bytes = 12 * kDft2Lbo;        // 18432 (rows 96..127 alias the next k-chunk: finite, unused)
// A tile buffer is also the staging area of the tile's output rows (kOutStride apart).
constexpr uint32_t kTileBuf = 96 * kOutStride;        // 38400 >= kTileBytes
constexpr uint32_t kMix2Smem = 2 * kDft2Bytes + 4 * kWBytes + 3 * kTileBuf; // 225792
constexpr uint32_t kSlot = 96;

// bulk (async-proxy) store of a thread's own staged bytes: shared -> global, tracked by bulk groups
__device__ __forceinline__ void bulk_store(void* dst, uint32_t src_smem, uint32_t bytes, uint64_t pol) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;" ::"l"(dst), "r"(src_smem),
               "r"(bytes), "l"(pol)
               : "memory");
  bulk_commit();
}

struct Mix2Bars {
  uint64_t dfull[2];  // stream's current stage accumulated (tcgen05.commit)
  uint64_t edone[2];  // stream's current stage drained by the 12 epilogue warps
  uint64_t xfull[3];  // buffer holds the input tile (forward: spectrum; backward: x spectrum)
  uint64_t gfull[3];  // backward: buffer holds the gradient tile
  uint64_t xfree[3];  // backward: stage 0 has consumed the x tile (tcgen05.commit)
  uint64_t sdone[3];  // the 12 epilogue warps have staged the tile's output rows in the buffer
  uint64_t imgfull[2]; // stream: the 12 epilogue warps have staged an operand image (Xh, O1, G2, G1) in the tile buffer
  uint64_t imgfree[2]; // stream: the image's bulk store has read the buffer
};

// One transform product pair: the same A (DFT matrix K-step) times two B tile halves
__device__ __forceinline__ void issue_dft2_pair(uint32_t d0, uint32_t d1, uint32_t a_base, uint32_t b0, uint32_t b1,
                                                uint32_t id0, uint32_t id1, bool fresh) {
#pragma unroll
  for (int ks = 0; ks < HP / 16; ++ks) {
    const uint64_t ad = smem_desc(a_base + ks * 2 * kDft2Lbo, kDft2Lbo, kDft2Sbo);
    const uint32_t acc = !(fresh && ks == 0);
    mma_ss(d0, ad, smem_desc(b0 + ks * 2 * kTileLbo, kTileLbo, kTileSbo), id0, acc);
    mma_ss(d1, ad, smem_desc(b1 + ks * 2 * kTileLbo, kTileLbo, kTileSbo), id1, acc);
  }
}
// forward transform (exp(-i theta)):  Xr = Ch Ar + Sh Ai ; Xi = Ch Ai - Sh Ar
// The input tile is six 64B-swizzled panels [96 rows (h, zero-filled past H)][32 columns] written by TMA:
// panels 0..2 = re, 3..5 = im.
constexpr uint32_t kInPanel = HP * 64;   // 6144
__device__ __forceinline__ void issue_dft2_pair_sw(uint32_t d0, uint32_t d1, uint32_t a_base, uint32_t b0, uint32_t b1,
                                                   uint32_t id0, uint32_t id1, bool fresh) {
#pragma unroll
  for (int ks = 0; ks < HP / 16; ++ks) {
    const uint64_t ad = smem_desc(a_base + ks * 2 * kDft2Lbo, kDft2Lbo, kDft2Sbo);
    const uint32_t acc = !(fresh && ks == 0);
    mma_ss(d0, ad, smem_desc_sw64(b0 + ks * 1024, kInPanel, 512), id0, acc);
    mma_ss(d1, ad, smem_desc_sw64(b1 + ks * 1024, kInPanel, 512), id1, acc);
  }
}
__device__ __forceinline__ void issue_fwd_dft2(uint32_t Dre, uint32_t Dim, uint32_t aCh, uint32_t aSh, uint32_t tile) {
  const uint32_t id = idesc_bf16(128, BS, kIdescBMn), half = 3 * kInPanel;
  issue_dft2_pair_sw(Dre, Dim, aCh, tile, tile + half, id, id, true);
  issue_dft2_pair_sw(Dre, Dim, aSh, tile + half, tile, id, id | kIdescNegB, false);
}
// inverse transform (exp(+i theta)):  Tr = Ch Zr - Sh Zi ; Ti = Ch Zi + Sh Zr
__device__ __forceinline__ void issue_inv_dft2(uint32_t Dre, uint32_t Dim, uint32_t aCh, uint32_t aSh, uint32_t tile) {
  const uint32_t id = idesc_bf16(128, BS, kIdescBMn), half = (BS / 8) * kTileSbo;
  issue_dft2_pair(Dre, Dim, aCh, tile, tile + half, id, id, true);
  issue_dft2_pair(Dre, Dim, aSh, tile + half, tile, id | kIdescNegB, id, false);
}
// T = S W (TRANSPOSED = false) or S W^H (true); S = compact bf16 A operand: re at columns
// [S, S+48), im at [S+48, S+96) (two bf16 per column)
template <bool TRANSPOSED>
__device__ __forceinline__ void issue_mlp2(uint32_t Tre, uint32_t Tim, uint32_t S, uint32_t wr, uint32_t wi) {
  const uint32_t id = idesc_bf16(128, BS, TRANSPOSED ? kIdescBMn : 0u);
  const uint32_t lbo = TRANSPOSED ? kWSbo : kWLbo, sbo = TRANSPOSED ? kWLbo : kWSbo;
#pragma unroll
  for (int ks = 0; ks < BS / 16; ++ks) {
    const uint32_t acc = ks != 0;
    mma_ts(Tre, S + ks * 8, smem_desc(wr + ks * 2 * lbo, lbo, sbo), id, acc);
    mma_ts(Tim, S + ks * 8, smem_desc(wi + ks * 2 * lbo, lbo, sbo), TRANSPOSED ? (id | kIdescNegB) : id, acc);
  }
#pragma unroll
  for (int ks = 0; ks < BS / 16; ++ks) {
    mma_ts(Tre, S + 48 + ks * 8, smem_desc(wi + ks * 2 * lbo, lbo, sbo), TRANSPOSED ? id : (id | kIdescNegB), 1u);
    mma_ts(Tim, S + 48 + ks * 8, smem_desc(wr + ks * 2 * lbo, lbo, sbo), id, 1u);
  }
}

__device__ __forceinline__ void ld48(uint32_t taddr, uint32_t (&v)[48]) {
  tmem_ld16<0>(taddr, v);
  tmem_ld16<16>(taddr + 16, v);
  tmem_ld16<32>(taddr + 32, v);
  tmem_wait_ld();
}
__device__ __forceinline__ void st24(uint32_t taddr, const uint32_t (&pk)[24]) {
  tmem_st8<0>(taddr, pk);
  tmem_st8<8>(taddr + 8, pk);
  tmem_st8<16>(taddr + 16, pk);
}
__device__ __forceinline__ void pack48(const uint32_t (&v)[48], uint32_t (&pk)[24]) {
#pragma unroll
  for (int q = 0; q < 24; ++q) pk[q] = pack_bf16(__uint_as_float(v[2 * q]), __uint_as_float(v[2 * q + 1]));
}
// 48 columns of this thread's row -> six 16-byte pieces of an operand image / operand tile
__device__ __forceinline__ void store_chunks6(uint8_t* base, int chunk0, int r, const uint32_t (&pk)[24]) {
#pragma unroll
  for (int g = 0; g < 6; ++g)
    *(uint4*)(base + (chunk0 + g) * kTileSbo + r * 16) = make_uint4(pk[4 * g], pk[4 * g + 1], pk[4 * g + 2], pk[4 * g + 3]);
}

// softshrink of a packed bf16 pair: a - min(max(a, -lambda), lambda)
__device__ __forceinline__ uint32_t shrink_bf16x2(uint32_t a, uint32_t lam2, uint32_t nlam2) {
  uint32_t c, r;
  asm("max.bf16x2 %0, %1, %2;" : "=r"(c) : "r"(a), "r"(nlam2));
  asm("min.bf16x2 %0, %1, %2;" : "=r"(c) : "r"(c), "r"(lam2));
  asm("sub.rn.bf16x2 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(c));
  return r;
}
// Z = S_lambda(a + b) on a packed pair: the sum is rounded to bf16 once, then shrunk (exact zeros inside
// the threshold; lambda at bf16 precision).  Forward value and backward mask (Z != 0) come from this one
// function, so the gradient is the gradient of the function the forward pass evaluates.
__device__ __forceinline__ uint32_t shrink_sum(float v0, float v1, float b0, float b1, uint32_t lam2, uint32_t nlam2) {
  return shrink_bf16x2(pack_bf16(v0 + b0, v1 + b1), lam2, nlam2);
}
// relu + one rounding of two fp32 values to a packed bf16 pair (lo, hi)
__device__ __forceinline__ uint32_t pack_relu_bf16(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.relu.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
// Activation masks of a thread's 48 columns: pair p (columns 2p, 2p+1) -> word p / 12, bits
// 15 - p % 12 (even column) and 31 - p % 12 (odd column).  `q` is a packed pair of NON-NEGATIVE
// bf16 values; a value is "on" iff it is non-zero (adding 0x7fff carries into the sign bit).
template <int P>
__device__ __forceinline__ void mask_collect(uint32_t (&m)[2], uint32_t q) {
  constexpr int s = P % 12;
  m[P / 12] |= ((q + 0x7FFF7FFFu) >> s) & (0x80008000u >> s);
}
// the same for signed values
template <int P>
__device__ __forceinline__ void mask_collect_signed(uint32_t (&m)[2], uint32_t q) {
  mask_collect<P>(m, q & 0x7FFF7FFFu);
}
// packed bf16 pair with the halves whose mask bit is clear zeroed
template <int P>
__device__ __forceinline__ uint32_t mask_apply(const uint32_t (&m)[2], uint32_t val) {
  constexpr int s = P % 12;
  uint32_t mk;
  // prmt default mode: selector nibble 8 + k = sign of byte k replicated; bytes 1, 3 -> (0,1), (2,3)
  asm("prmt.b32 %0, %1, %2, 0xBB99;" : "=r"(mk) : "r"(m[P / 12] << s), "r"(0u));
  return val & mk;
}
template <int P>
__device__ __forceinline__ uint32_t mask_bit(const uint32_t (&m)[2], int odd) {
  return (m[P / 12] >> (15 - P % 12 + 16 * odd)) & 1u;
}
template <int P>
struct MaskLoop {
  template <typename F>
  static __device__ __forceinline__ void run(F&& f) {
    f(std::integral_constant<int, P>{});
    if constexpr (P + 1 < 24) MaskLoop<P + 1>::run(f);
  }
};
// mbarrier wait without the nanosleep back-off (the ping-pong hand-offs are latency critical)
__device__ __forceinline__ void mbar_wait_fast(uint64_t* mbar, uint32_t parity) {
  while (!mbar_try_wait(mbar, parity)) {
  }
}

// MODE: kMixFwd (4 stages), kMixBwd (stateless backward: recompute + gradient, 7 stages), kMixFwdSave
// (forward that also leaves Xh, O1 and the activation masks in the workspace: the saved context),
// kMixBwdCtx (gradient stages only, 4 stages, reads the saved context).
constexpr int kMixFwd = 0, kMixBwd = 1, kMixFwdSave = 2, kMixBwdCtx = 3;
template <int MODE, bool EXPORT>
__global__ void __launch_bounds__(kMix2Threads, 1) tc_mix2(const __grid_constant__ MixParams p, int S) {
  constexpr bool BACKWARD = MODE == kMixBwd || MODE == kMixBwdCtx;   // has the gradient stages
  constexpr bool RECOMP = MODE == kMixBwd, SAVE = MODE == kMixFwdSave, CTXB = MODE == kMixBwdCtx;
  constexpr int kStage0 = CTXB ? 3 : 0;                               // stage number of a tile's first phase
  // FwdSave / BwdCtx: the operand images for tc_wgrad are staged in the tile's buffer (idle between its
  // first GEMM and the write of the inverse transform's operand) and leave by bulk copies issued by
  // warp 11, so no epilogue warp ever stalls on the global store path.  The stateless backward reloads
  // that buffer with the gradient tile meanwhile and stores the images with plain vector stores.
  constexpr bool STAGED = SAVE || CTXB;
  extern __shared__ __align__(1024) uint8_t smem[];
  TL(BACKWARD ? 24 : 16);
  SPAN(BACKWARD ? 3 : 2, 0);
  __shared__ Mix2Bars bars;
  __shared__ uint32_t tmem_slot;
  __shared__ __align__(16) float sBias[2 * NT];
  constexpr int NS = RECOMP ? 7 : 4;
  uint8_t* sCh = smem;
  uint8_t* sSh = smem + kDft2Bytes;
  uint8_t* sW = smem + 2 * kDft2Bytes;
  uint8_t* sT = sW + 4 * kWBytes;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int BKw = p.B * p.Kw;
  // Work split.  The first nb * S CTAs are "regular": CTA (j, s0) of block j takes the (b, kw) pairs
  // s0, s0 + S, ...  If the grid has spare CTAs beyond those (148 SMs against 8 x 18), the regular CTAs
  // stop at the largest multiple of S, so that each has the SAME, even number of tiles (tiles run in
  // pairs), and spare CTA k takes the few left-over pairs of blocks k, k + nspare, ..., one block
  // ("segment") after the other, reloading the weights in between.
  const int nreg = p.nb * S, nspare = (int)gridDim.x - nreg;
  const bool spare = (int)blockIdx.x >= nreg;
  const int main_tiles = nspare > 0 ? (BKw / S) * S : BKw;
  const int nseg = spare ? (p.nb - ((int)blockIdx.x - nreg) + nspare - 1) / nspare : 1;
  pdl_launch_dependents();
  for (uint32_t i = tid; i < 3 * kTileBuf / 16; i += kMix2Threads) ((uint4*)sT)[i] = make_uint4(0, 0, 0, 0);
  for (uint32_t i = tid; i < 2 * kDft2Bytes / 16; i += kMix2Threads) cp_async16(smem_u32(sCh) + i * 16, p.dft + (size_t)i * 16);
  TL(BACKWARD ? 25 : 17);
  pdl_wait();   // the weight images below are written by an earlier kernel of the chain
  TL(BACKWARD ? 26 : 18);
  if (warp == 0) tmem_alloc<512>(&tmem_slot);
#pragma unroll 1
  for (int seg = 0; seg < nseg; ++seg) {
  const int j = spare ? ((int)blockIdx.x - nreg) + seg * nspare : (int)blockIdx.x / S;
  const int s0 = spare ? main_tiles : (int)blockIdx.x - j * S;
  const int step = spare ? 1 : S;
  const int n = s0 < (spare ? BKw : main_tiles) ? ((spare ? BKw : main_tiles) - s0 + step - 1) / step : 0;   // tiles of this segment
  // Tile i is (b, kw) pair rem = BKw - 1 - (s0 + i * step): the tiles run from the LAST sample to the
  // first.  The W-direction kernels run from the first sample to the last, so this kernel starts on the
  // part of A1 its producer wrote last (still in the 126 MB L2) and finishes with the part of A2 its
  // consumer reads first.
  const int rtop = BKw - 1 - s0;
  {
    const uint8_t* wsrc = p.wprep + (size_t)j * 4 * kWBytes;
    for (uint32_t i = tid; i < 4 * kWBytes / 16; i += kMix2Threads) cp_async16(smem_u32(sW) + i * 16, wsrc + (size_t)i * 16);
  }
  for (int i = tid; i < 2 * NT; i += kMix2Threads) sBias[i] = p.bprep[(size_t)j * 2 * NT + i];
  if (tid == 0) {
    if (seg > 0) {   // every barrier is idle (the segment ended with a CTA-wide sync): start over
      uint64_t* all = (uint64_t*)&bars;
      for (uint32_t q = 0; q < sizeof(Mix2Bars) / 8; ++q)
        asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(smem_u32(all + q)) : "memory");
    }
    for (int q = 0; q < 2; ++q) {
      mbar_init(&bars.dfull[q], 1);
      mbar_init(&bars.edone[q], 12);
      mbar_init(&bars.imgfull[q], 12);
      mbar_init(&bars.imgfree[q], 1);
    }
    for (int q = 0; q < 3; ++q) {
      mbar_init(&bars.xfull[q], 1);
      mbar_init(&bars.gfull[q], 1);
      mbar_init(&bars.xfree[q], 1);
      mbar_init(&bars.sdone[q], 12);
    }
    mbar_init_fence();
  }
  cp_async_wait_all();
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  TL(BACKWARD ? 27 : 19);
  // Stream 1 runs kLag stages behind stream 0, so tiles finish (and buffers become free) at
  // regular intervals and a transform stage of one stream overlaps an MLP stage of the other.
  constexpr int kLag = NS / 2;
  const int T = 2 * (NS * ((n + 1) / 2) + kLag);   // phases
  const int lq = warp & 3;

  if (lq == 3 && warp != 3) {
    // ================================ copy warp (7; 11 and 15 idle) ============================
    // warp 7 lane 0 issues every copy (TMA tile loads in, bulk stores of the staged rows out); the other
    // two warps of this lane quarter have nothing to do
    const uint32_t aT = smem_u32(sT);
    const uint64_t pol_stream = pol_first(kPolMixLoad), pol_keep = pol_last(kPolMixStore);
    const uint64_t pol_img = SAVE ? pol_first(kPolMixImg) : pol_last(kPolMixImg);
    if (warp == 7 && lane == 0) {
      auto load = [&](int buf, const CUtensorMap* m, int i, uint64_t* full) {
        const int tile_id = (rtop - i * step) * p.nb + j;
        mbar_expect_tx(full, 6 * kInPanel);
#pragma unroll
        for (int pn = 0; pn < 6; ++pn) tma_load4(aT + buf * kTileBuf + pn * kInPanel, m, 0, pn, 0, tile_id, full, pol_stream);
      };
      // tile k's output rows are staged in its buffer by the epilogue warps; they leave with one bulk copy
      // and the buffer is free once the copy has read it
      auto drain = [&](int k) {
        const int buf = k % 3;
        mbar_wait(&bars.sdone[buf], (uint32_t)((k / 3) & 1));
        bulk_store(p.A2 + ((size_t)(rtop - k * step) * p.nb + j) * p.H * kA2Row, aT + buf * kTileBuf, (uint32_t)p.H * kOutStride,
                   pol_keep);   // the next kernel reads A2
        bulk_wait_read<0>();
      };
      if (!RECOMP) {
        const CUtensorMap* src = CTXB ? &p.mapA1g : &p.mapA1;
        for (int i = 0; i < n; ++i) {
          if (i >= 3) drain(i - 3);
          load(i % 3, src, i, &bars.xfull[i % 3]);
        }
        for (int k = n > 3 ? n - 3 : 0; k < n; ++k) drain(k);
      } else {
        // x(0) x(1) x(2) | g(0) g(1) | then for k = 0, 1, ..: x(k+3) after the last stage of tile k,
        // g(k+2) after stage 0 of tile k+2 -- the order in which the buffers become free
        for (int i = 0; i < 3 && i < n; ++i) load(i, &p.mapA1, i, &bars.xfull[i]);
        for (int i = 0; i < 2 && i < n; ++i) {
          mbar_wait(&bars.xfree[i], 0u);
          load(i, &p.mapA1g, i, &bars.gfull[i]);
        }
        for (int k = 0; k < n; ++k) {
          const int ix = k + 3, ig = k + 2;
          drain(k);
          if (ix < n) load(ix % 3, &p.mapA1, ix, &bars.xfull[ix % 3]);
          if (ig < n) {
            mbar_wait(&bars.xfree[ig % 3], (uint32_t)((ig / 3) & 1));
            load(ig % 3, &p.mapA1g, ig, &bars.gfull[ig % 3]);
          }
        }
      }
      bulk_wait<0>();
    }
    if (STAGED && warp == 11 && lane == 0) {
      // ---- image warp: the phases in order; an image phase = wait for the staged image, send it ----
      uint32_t cnt[2] = {0, 0};
      for (int t = 0; t < T; ++t) {
        const int stream = t & 1, u = (t >> 1) - (stream ? kLag : 0);
        if (u < 0) continue;
        const int pair = u / NS, stg = u - pair * NS;
        const int i = 2 * pair + stream;
        if (i >= n) continue;
        const int se = stg + kStage0;
        if (!(SAVE ? (se == 0 || se == 1) : (se == 3 || se == 4))) continue;
        __nv_bfloat16* img = se == 0 ? p.Xh : se == 1 ? p.O1 : se == 3 ? p.G2 : p.G1;
        mbar_wait(&bars.imgfull[stream], cnt[stream] & 1u);
        ++cnt[stream];
        // Xh, O1 are read a whole kernel later: stream them out; G2, G1 are read by the next kernel
        bulk_store((uint8_t*)img + ((size_t)(rtop - i * step) * p.nb + j) * kTileBytes, aT + (i % 3) * kTileBuf, kTileBytes,
                   pol_img);
        bulk_wait_read<0>();
        mbar_arrive(&bars.imgfree[stream]);
      }
      bulk_wait<0>();
    }
    __syncwarp();
  } else if (warp == 3) {
    // ================================ control warp ===========================================
    const uint32_t aCh = smem_u32(sCh), aSh = smem_u32(sSh), aW = smem_u32(sW), aT = smem_u32(sT);
    const uint32_t w1r = aW, w1i = aW + kWBytes, w2r = aW + 2 * kWBytes, w2i = aW + 3 * kWBytes;
    uint32_t cs0 = 0, cs1 = 0;   // phases issued so far per stream
#ifdef AFNO_TIMING
    long long dbg_acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
#endif
    DBG_T0();
    for (int t = 0; t < T; ++t) {
      const int stream = t & 1, u = (t >> 1) - (stream ? kLag : 0);
      if (u < 0) continue;
      const int pair = u / NS, stg = u - pair * NS;
      const int i = 2 * pair + stream;
      if (i >= n) continue;
      const uint32_t Dre = tmem + kSlot * (uint32_t)((3 * t) % 5), Dim = tmem + kSlot * (uint32_t)((3 * t + 1) % 5);
      const uint32_t SA = tmem + kSlot * (uint32_t)((3 * t + 4) % 5);   // slot of phase t - 2
      const uint32_t cs = stream ? cs1 : cs0;
      if (cs > 0) mbar_wait_fast(&bars.edone[stream], (cs - 1) & 1u);
      TR(t, 0);
      DBG_ACC(0);
      const int buf = i % 3;
      const uint32_t use = (uint32_t)(i / 3);
      const uint32_t tile = aT + buf * kTileBuf;
      const int se = stg + kStage0;
      const bool first = stg == 0, dftg = RECOMP && stg == 3, last = stg == NS - 1;
      if (first) mbar_wait(&bars.xfull[buf], use & 1u);
      if (dftg) mbar_wait(&bars.gfull[buf], use & 1u);
      DBG_ACC(1);
      if (elect_one()) {
        tc_fence_after();
        if (first || dftg) {
          issue_fwd_dft2(Dre, Dim, aCh, aSh, tile);
        } else if (last) {
          issue_inv_dft2(Dre, Dim, aCh, aSh, tile);
        } else if (se == 1) {
          issue_mlp2<false>(Dre, Dim, SA, w1r, w1i);
        } else if (se == 2) {
          issue_mlp2<false>(Dre, Dim, SA, w2r, w2i);
        } else if (se == 4) {
          issue_mlp2<true>(Dre, Dim, SA, w2r, w2i);    // G1 = G2 W2^H
        } else {
          issue_mlp2<true>(Dre, Dim, SA, w1r, w1i);    // GX = G1 W1^H
        }
        mma_commit(&bars.dfull[stream]);
        if (RECOMP && first) mma_commit(&bars.xfree[buf]);
      }
      __syncwarp();
      TR(t, 2);
      DBG_ACC(2);
      if (stream) ++cs1; else ++cs0;
    }
#ifdef AFNO_TIMING
    if (blockIdx.x == 0 && lane == 0) {
      for (int q = 0; q < 8; ++q) g_afno_dbg[(BACKWARD ? 80 : 64) + q] = dbg_acc[q];
      g_afno_dbg[(BACKWARD ? 80 : 64) + 7] = n;
    }
#endif
  } else {
    // ================================ epilogue warps =========================================
    const int cq = warp >> 2;              // column quarter: 0 re lo, 1 re hi, 2 im lo, 3 im hi
    const int half = cq >> 1, chalf = cq & 1;
    const int r = lq * 32 + lane;
    const uint32_t lane_sel = (uint32_t)(lq * 32) << 16;
    const int kappa = (r <= p.H / 2) ? r : p.H - r;
    const bool row_valid = r < p.H;
    const bool row_kept = row_valid && (kappa < p.Kh);
    const int chunk0 = half * 12 + chalf * 6;            // first 16-byte chunk (8 columns) of this warp's 48 columns
    const float* bias1 = sBias + half * BS + chalf * 48;
    const float* bias2 = bias1 + NT;
    const uint32_t bar_id = 1 + lq;
    uint32_t m1[2][2] = {{0, 0}, {0, 0}}, m2[2][2] = {{0, 0}, {0, 0}};   // [stream][word]
    uint32_t ce[2] = {0, 0};
    uint32_t ci[2] = {0, 0};   // images staged so far per stream
    // the tile buffer may be overwritten once the stream's last image store has read it
    auto wait_img_read = [&](int stream) {
      if (STAGED && ci[stream] > 0) mbar_wait(&bars.imgfree[stream], (ci[stream] - 1) & 1u);
    };
#ifdef AFNO_TIMING
    long long dbg_acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    long long dbg_m[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    long long dbg_f[8] = {0, 0, 0, 0, 0, 0, 0, 0};
#endif
    DBG_T0();
    for (int u0 = 0; u0 < T / 2; ++u0) {
#pragma unroll
      for (int stream = 0; stream < 2; ++stream) {
        const int t = 2 * u0 + stream;
        const int u = u0 - (stream ? kLag : 0);
        if (u < 0) continue;
        const int pair = u / NS, stg = u - pair * NS;
        const int i = 2 * pair + stream;
        if (i >= n) continue;
        const int rem = rtop - i * step;
        const uint32_t src = tmem + lane_sel + kSlot * (uint32_t)((3 * t + half) % 5) + chalf * 48;
        const uint32_t dstA = tmem + lane_sel + kSlot * (uint32_t)((3 * t) % 5) + 24 * cq;
        uint8_t* tile = sT + (i % 3) * kTileBuf;
        const size_t img_off = ((size_t)rem * p.nb + j) * kTileBytes;
        const int se = stg + kStage0;
        const size_t mask_idx = (((size_t)rem * p.nb + j) * 12 + (size_t)(cq * 3 + lq)) * 32 + lane;
        uint4 mk = make_uint4(0, 0, 0, 0);
        if (CTXB && stg == 0) mk = p.maskbits[mask_idx];   // issued before the wait: its latency hides under the GEMM
        mbar_wait_fast(&bars.dfull[stream], ce[stream] & 1u);
        ++ce[stream];
        TR(t, 4 + warp * 3);
        DBG_ACC(0);
        tc_fence_after();
        uint32_t v[48], pk[24];
        ld48(src, v);
        DBG_ACC(2);
        bool writes_a = false, early_arrive = false;
        // backward: operand image (Xh, O1, G2, G1) this stage also writes for tc_wgrad; stored AFTER the
        // hand-off to the next GEMM, so the global stores run in the shadow of the tensor core
        uint8_t* gimg = nullptr;
        if (CTXB && stg == 0) {
          m1[stream][0] = mk.x; m1[stream][1] = mk.y;
          m2[stream][0] = mk.z; m2[stream][1] = mk.w;
        }
        if (se == 0) {
          // ---- spectrum Xh ----
          pack48(v, pk);
          writes_a = true;
          if (RECOMP || SAVE) gimg = (uint8_t*)p.Xh + img_off;
        } else if (se == 1) {
          // ---- O1 = relu(P1 + b1) ----
#pragma unroll
          for (int q = 0; q < 12; ++q) {
            const float4 bq = *(const float4*)(bias1 + 4 * q);
            pk[2 * q] = pack_relu_bf16(__uint_as_float(v[4 * q]) + bq.x, __uint_as_float(v[4 * q + 1]) + bq.y);
            pk[2 * q + 1] = pack_relu_bf16(__uint_as_float(v[4 * q + 2]) + bq.z, __uint_as_float(v[4 * q + 3]) + bq.w);
          }
          if (RECOMP || SAVE) {
            m1[stream][0] = m1[stream][1] = 0;
            MaskLoop<0>::run([&](auto P) { mask_collect<decltype(P)::value>(m1[stream], pk[decltype(P)::value]); });
            gimg = (uint8_t*)p.O1 + img_off;
          }
          writes_a = true;
        } else if (se == 2) {
          // ---- P2 + b2: forward Z = softshrink (truncated) -> B operand of the inverse transform;
          //      backward: only the mask ----
          // Z = softshrink(P2 + b2), zero on truncated rows (shrink_sum)
          const float lam = p.lambda;
          const uint32_t lam2 = pack_bf16(lam, lam), nlam2 = lam2 ^ 0x80008000u;
#pragma unroll
          for (int q = 0; q < 12; ++q) {
            const float4 bq = *(const float4*)(bias2 + 4 * q);
            pk[2 * q] = shrink_sum(__uint_as_float(v[4 * q]), __uint_as_float(v[4 * q + 1]), bq.x, bq.y, lam2, nlam2);
            pk[2 * q + 1] = shrink_sum(__uint_as_float(v[4 * q + 2]), __uint_as_float(v[4 * q + 3]), bq.z, bq.w, lam2, nlam2);
          }
          if (!row_kept) {
#pragma unroll
            for (int q = 0; q < 24; ++q) pk[q] = 0u;
          }
          if (RECOMP || SAVE) {
            // softshrink mask: Z != 0
            m2[stream][0] = m2[stream][1] = 0;
            MaskLoop<0>::run([&](auto P) { mask_collect_signed<decltype(P)::value>(m2[stream], pk[decltype(P)::value]); });
          }
          if (!BACKWARD) {
            // forward: Z is the B operand of the inverse transform
            wait_img_read(stream);
            store_chunks6(tile, chunk0, r, pk);
            fence_async_smem();
            if (SAVE) p.maskbits[mask_idx] = make_uint4(m1[stream][0], m1[stream][1], m2[stream][0], m2[stream][1]);
          }
        } else if (se == (BACKWARD ? 6 : 3)) {
          // ---- last stage: rows of A2.  The accumulator is in registers: release the tensor-memory
          //      slots now, so the next tile's first GEMM never waits for the global stores ----
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(&bars.edone[stream]);
          early_arrive = true;
          pack48(v, pk);
          if (row_valid) {
            // staged in the tile's own buffer (its last GEMM has completed)
            uint8_t* srow = tile + r * kOutStride + cq * 96;
#pragma unroll
            for (int g = 0; g < 6; ++g)
              *(uint4*)(srow + 16 * g) = make_uint4(pk[4 * g], pk[4 * g + 1], pk[4 * g + 2], pk[4 * g + 3]);
          }
          fence_async_smem();
          __syncwarp();
          if (lane == 0) mbar_arrive(&bars.sdone[i % 3]);
        } else if (se == 3 || se == 4) {
          // ---- G2 = G (.) mask2 ; G1 = mask1 (.) (G2 W2^H) ----
          pack48(v, pk);
          if (se == 3) {
            MaskLoop<0>::run([&](auto P) { pk[decltype(P)::value] = mask_apply<decltype(P)::value>(m2[stream], pk[decltype(P)::value]); });
          } else {
            MaskLoop<0>::run([&](auto P) { pk[decltype(P)::value] = mask_apply<decltype(P)::value>(m1[stream], pk[decltype(P)::value]); });
          }
          writes_a = true;
          gimg = (uint8_t*)(se == 3 ? p.G2 : p.G1) + img_off;
        } else {
          // ---- stage 5: GX -> B operand of the inverse transform (the tile's own buffer) ----
#pragma unroll
          for (int q = 0; q < 24; ++q)
            pk[q] = row_valid ? pack_bf16(__uint_as_float(v[2 * q]), __uint_as_float(v[2 * q + 1])) : 0u;
          wait_img_read(stream);
          store_chunks6(tile, chunk0, r, pk);
          fence_async_smem();
          if (EXPORT && row_valid) {
            const int b = rem / p.Kw, kw = rem - b * p.Kw;
            const size_t base = ((((size_t)b * p.H + r) * p.Wh + kw) * (size_t)(p.nb * BS) + (size_t)j * BS + chalf * 48) * 2 + half;
            MaskLoop<0>::run([&](auto P) {
              constexpr int pp = decltype(P)::value;
              p.mask1[base + (size_t)(2 * pp) * 2] = (uint8_t)mask_bit<pp>(m1[stream], 0);
              p.mask1[base + (size_t)(2 * pp + 1) * 2] = (uint8_t)mask_bit<pp>(m1[stream], 1);
              p.mask2[base + (size_t)(2 * pp) * 2] = (uint8_t)mask_bit<pp>(m2[stream], 0);
              p.mask2[base + (size_t)(2 * pp + 1) * 2] = (uint8_t)mask_bit<pp>(m2[stream], 1);
            });
          }
        }
#ifdef AFNO_TIMING
        { long long n_ = clock64(); dbg_m[se] += n_ - dbg_t; dbg_t = n_; }
#endif
        TR(t, 5 + warp * 3);
        if (writes_a) {
          // the four warps of this lane quarter have their accumulator columns in registers:
          // compact the bf16 operand into the first slot (columns of the other warps' sources)
          asm volatile("bar.sync %0, 128;" ::"r"(bar_id) : "memory");
          DBG_ACC(4);
          st24(dstA, pk);
          tmem_wait_st();
          DBG_ACC(5);
        }
        if (!early_arrive) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(&bars.edone[stream]);
        }
        if (gimg != nullptr) {
          if (STAGED) {
            wait_img_read(stream);
            store_chunks6(tile, chunk0, r, pk);
            fence_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars.imgfull[stream]);
            ++ci[stream];
          } else {
            store_chunks6(gimg, chunk0, r, pk);
          }
        }
        TR(t, 6 + warp * 3);
        DBG_ACC(1);
      }
    }
#ifdef AFNO_TIMING
    if (blockIdx.x == 0 && tid == 0)
      for (int q = 0; q < 8; ++q) {
        g_afno_dbg[(BACKWARD ? 88 : 72) + q] = dbg_acc[q];
        g_afno_dbg[(BACKWARD ? 104 : 96) + q] = dbg_m[q];
        g_afno_dbg[(BACKWARD ? 120 : 112) + q] = dbg_f[q];
      }
#endif
  }
  tc_fence_before();
  __syncthreads();   // end of the segment: every role is done, every copy has landed
  }
  TL(BACKWARD ? 28 : 20);
  SPAN(BACKWARD ? 3 : 2, 1);
  tc_fence_after();
  if (warp == 0) tmem_dealloc<512>(tmem_slot);
}

// ---- B4 / B6: parameter gradients as a split-K tensor-core GEMM ------------------------------------
// For block j:  R[(ri_a,i), (ri_g,o)] = sum_rows A[row,(ri_a,i)] * G[row,(ri_g,o)] with K = mode rows.
// Two M=128 accumulators: D_re rows = (re, i) plus a constant-one row 96 (gives sum_rows G = db),
// D_im rows = (im, i).  CTA (j, s) sums tiles rem = s, s+S, ... and writes its partial sums.
constexpr uint32_t kWgALbo = 128, kWgASbo = 1536 + 16;                  // MN-major A [K=96][M=128], padded chunk stride
constexpr uint32_t kWgABytes = 16 * kWgASbo;                            // 24832
constexpr uint32_t kWgStage = 2 * kWgABytes + kTileBytes;              // 86016
constexpr uint32_t kWgSmem = 2 * kWgStage;                             // 172032
// partial sums of one CTA: rows 0..96 of D_re (96 channels + the db row) then rows 0..95 of D_im, fp32,
// row pitch 196 floats (784 bytes: a warp's 32 rows staged in shared memory hit distinct bank groups)
constexpr int kWgPitch = NT + 4;
constexpr int kWgRowsRe = BS + 1, kWgRowsIm = BS;
constexpr uint32_t kWgPartFloats = (kWgRowsRe + kWgRowsIm) * kWgPitch;   // 37828 floats = 151312 bytes
static_assert(kWgPartFloats * 4 <= kWgSmem, "partial sums are staged in the operand stages");

__device__ __forceinline__ void bulk_copy(uint32_t dst_smem, const void* src, uint32_t bytes, uint64_t* bar, uint64_t pol) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
                   dst_smem),
               "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol)
               : "memory");
}

// Operand-image tensors written by tc_mix2<true> ([tile][24 chunks][kTileSbo bytes]).  ONE launch covers
// both layers: CTAs [0, nb*S) form layer 2 (A = O1, G = G2), CTAs [nb*S, 2*nb*S) layer 1 (A = Xh, G = G1).
__global__ void __launch_bounds__(128, 1)
tc_wgrad(const __nv_bfloat16* __restrict__ A_l2, const __nv_bfloat16* __restrict__ G_l2,
         const __nv_bfloat16* __restrict__ A_l1, const __nv_bfloat16* __restrict__ G_l1, float* __restrict__ part,
         int BKw, int H, int nb, int S) {
  extern __shared__ __align__(1024) uint8_t smem[];
  TL(32);
  SPAN(4, 0);
  __shared__ __align__(8) uint64_t full[2], empty[2], done;
  __shared__ uint32_t tmem_slot;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int layer = blockIdx.x / (nb * S), cta = blockIdx.x - layer * nb * S;
  const int j = cta / S, s = cta - j * S;
  const __nv_bfloat16* Aws = layer ? A_l1 : A_l2;
  const __nv_bfloat16* Gws = layer ? G_l1 : G_l2;
  pdl_launch_dependents();
  for (uint32_t i = tid; i < kWgSmem / 16; i += 128) ((uint4*)smem)[i] = make_uint4(0, 0, 0, 0);
  __syncthreads();
  // constant-one column m = 96 of the "re" A operand, rows r < H, both stages
  for (int i = tid; i < 2 * H; i += 128) {
    const int st = i / H, rr = i - st * H;
    *(uint16_t*)(smem + st * kWgStage + 12 * kWgASbo + rr * 16) = 0x3F80; // bf16 1.0
  }
  if (tid == 0) {
    for (int b = 0; b < 2; ++b) {
      mbar_init(&full[b], 1);
      mbar_init(&empty[b], 1);
    }
    mbar_init(&done, 1);
    mbar_init_fence();
  }
  if (warp == 0) tmem_alloc<512>(&tmem_slot);
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  TL(33);
  pdl_wait();
  TL(34);
  const uint32_t tmem = tmem_slot;
  const uint32_t lane_base = (uint32_t)(warp * 32) << 16;
  const uint32_t Dre = tmem, Dim = tmem + 256;
  const uint32_t idesc = idesc_bf16(128, NT, kIdescAMn | kIdescBMn);
  const int nt = (BKw - s + S - 1) / S; // tiles of this CTA
  (void)lane;
  if (warp == 0 && elect_one()) {
    // ---- producer: three bulk copies per tile (A re half, A im half, G), async proxy, no LSU ----
    constexpr uint32_t kHalfImg = 12 * kTileSbo;
    const uint64_t pol_stream = pol_first(kPolWgLoad);
    for (int it = 0; it < nt; ++it) {
      const int b = it & 1, use = it >> 1;
      if (use > 0) mbar_wait(&empty[b], (uint32_t)((use - 1) & 1));
      const size_t off = ((size_t)(s + it * S) * nb + j) * kTileBytes;
      const uint32_t stage = smem_u32(smem) + b * kWgStage;
      mbar_expect_tx(&full[b], 2 * kHalfImg + kTileBytes);
      bulk_copy(stage, (const uint8_t*)Aws + off, kHalfImg, &full[b], pol_stream);
      bulk_copy(stage + kWgABytes, (const uint8_t*)Aws + off + kHalfImg, kHalfImg, &full[b], pol_stream);
      bulk_copy(stage + 2 * kWgABytes, (const uint8_t*)Gws + off, kTileBytes, &full[b], pol_stream);
    }
  } else if (warp == 1 && elect_one()) {
    // ---- MMA issuer ----
    for (int it = 0; it < nt; ++it) {
      const int b = it & 1;
      mbar_wait(&full[b], (uint32_t)((it >> 1) & 1));
      tc_fence_after();
      const uint32_t stage = smem_u32(smem) + b * kWgStage;
      const uint32_t g = stage + 2 * kWgABytes;
#pragma unroll
      for (int ks = 0; ks < HP / 16; ++ks) {
        const uint64_t bd = smem_desc(g + ks * 2 * kTileLbo, kTileLbo, kTileSbo);
        mma_ss(Dre, smem_desc(stage + ks * 2 * kWgALbo, kWgALbo, kWgASbo), bd, idesc, (it | ks) != 0);
        mma_ss(Dim, smem_desc(stage + kWgABytes + ks * 2 * kWgALbo, kWgALbo, kWgASbo), bd, idesc, (it | ks) != 0);
      }
      mma_commit(&empty[b]);
    }
    mma_commit(&done);
  }
  __syncwarp();
  // Partial sums: accumulator rows -> shared memory (the operand stages are free: every MMA has
  // completed) -> ONE bulk store per CTA.  Row-strided vector stores straight to global memory took 11 us.
  float* stage = (float*)smem;
  if (nt > 0) {
    mbar_wait(&done, 0u);
    TL(35);
    tc_fence_after();
#pragma unroll 1
    for (int acc = 0; acc < 2; ++acc) {
      const int rows = acc ? kWgRowsIm : kWgRowsRe;
      if (warp * 32 < rows) {   // warp-uniform: tcgen05.ld is a warp-wide instruction
        float* srow = stage + (size_t)(acc * kWgRowsRe + tid) * kWgPitch;
#pragma unroll 1
        for (int c0 = 0; c0 < NT; c0 += 32) {
          uint32_t v[32];
          tmem_ld32((acc ? Dim : Dre) + lane_base + c0, v);
          tmem_wait_ld();
          if (tid < rows) {
#pragma unroll
            for (int q = 0; q < 32; q += 4)
              *(float4*)(srow + c0 + q) = make_float4(__uint_as_float(v[q]), __uint_as_float(v[q + 1]),
                                                      __uint_as_float(v[q + 2]), __uint_as_float(v[q + 3]));
          }
        }
      }
    }
  } else {
    for (uint32_t i = tid; i < kWgPartFloats / 4; i += 128) ((float4*)stage)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  fence_async_smem();
  __syncthreads();
  if (tid == 0) {
    bulk_store(part + (size_t)blockIdx.x * kWgPartFloats, smem_u32(smem), kWgPartFloats * 4, l2_evict_normal());
    bulk_wait<0>();
  }
  tc_fence_before();
  __syncthreads();
  TL(36);
  SPAN(4, 1);
  if (warp == 0) tmem_dealloc<512>(tmem);
}

// dW[j][i][o] = sum_s ( Dre[i][o] + Dim[i][96+o] ,  Dre[i][96+o] - Dim[i][o] ) ;  db[j][o] = sum_s Dre[96][(ri,o)]
// blockIdx.y = 0: layer 2 partial sums (first nb*S CTAs of tc_wgrad), 1: layer 1
__global__ void k_tc_wgrad_reduce(const float* __restrict__ part, float2* __restrict__ dW2, float2* __restrict__ dB2,
                                  float2* __restrict__ dW1, float2* __restrict__ dB1, int nb, int S, int accumulate) {
  pdl_launch_dependents();
  pdl_wait();
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  const int nW = nb * BS * BS;
  const int layer = blockIdx.y;
  part += (size_t)layer * nb * S * kWgPartFloats;
  float2* dW = layer ? dW1 : dW2;
  float2* dB = layer ? dB1 : dB2;
  if (idx < nW) {
    const int o = idx % BS, i = (idx / BS) % BS, j = idx / (BS * BS);
    float2 acc = accumulate ? dW[idx] : make_float2(0.f, 0.f);
    for (int s = 0; s < S; ++s) {
      const float* P = part + (size_t)(j * S + s) * kWgPartFloats;
      const float* Pre = P + (size_t)i * kWgPitch;
      const float* Pim = P + (size_t)(kWgRowsRe + i) * kWgPitch;
      acc.x += Pre[o] + Pim[BS + o];
      acc.y += Pre[BS + o] - Pim[o];
    }
    dW[idx] = acc;
  } else if (idx < nW + nb * BS) {
    const int k = idx - nW, o = k % BS, j = k / BS;
    float2 acc = accumulate ? dB[k] : make_float2(0.f, 0.f);
    for (int s = 0; s < S; ++s) {
      const float* P = part + (size_t)(j * S + s) * kWgPartFloats + (size_t)BS * kWgPitch;
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
