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
constexpr int CGRP = 128; // channels per W-direction tile (= UMMA M)
constexpr int kA2Row = NT + 8; // elements per stored row of A2: 192 values + 16 bytes (see kOutStride)

// shared-memory operand geometry (bytes), see tc_common.cuh for the layout formulas
constexpr uint32_t kWLbo = 1536, kWSbo = 128;       // weights: K-major B [96 x 96], order [k/8][n/8]
constexpr uint32_t kWBytes = BS * BS * 2;            // 18432
// mode tile: MN-major B [K=96 rows][N=192]; the 16-byte pad on the chunk stride keeps cp.async
// writes of consecutive chunks of one row (the coalesced global order) bank-conflict-free
constexpr uint32_t kTileLbo = 128, kTileSbo = 1536 + 16;
constexpr uint32_t kTileBytes = (NT / 8) * kTileSbo; // 37248
constexpr uint32_t kFwLbo = 2048, kFwSbo = 128;     // Fw / Gw halves: K-major A [128 x 192], order [k/8][m/8]
constexpr uint32_t kFwHalf = 128 * WP * 2;           // 49152 per 128-row half
constexpr uint32_t kFwBytes = 2 * kFwHalf;           // 98304
constexpr uint32_t kRowLbo = 128, kRowSbo = 3072 + 16; // W-direction data tile: MN-major B [K=192][N=128], padded
constexpr uint32_t kRowBytes = (CGRP / 8) * kRowSbo; // 49408

constexpr int kRowEpiThreads = 256;                 // 8 epilogue warps
constexpr int kRowProdWarps = 4;                     // producer warps per operand buffer
constexpr int kRowThreads = kRowEpiThreads + 2 * kRowProdWarps * 32;
constexpr uint32_t kRowSmem = kFwBytes + 2 * kRowBytes;                              // 196608

// ---- weight preparation: fp32 [nb][96][96][2] -> bf16 K-major interleaved operands --------------
// per block 4 matrices of kWBytes {W1r, W1i, W2r, W2i} with element (n=o, k=i) = W[i][o] (the
// backward pass reads the same images as MN-major operands), and the biases regrouped as
// [block][layer][re 96 | im 96] fp32.
__global__ void k_tc_prep_weights(const float* __restrict__ w1, const float* __restrict__ b1,
                                  const float* __restrict__ w2, const float* __restrict__ b2,
                                  __nv_bfloat16* __restrict__ out, float* __restrict__ bout, int nb) {
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

// ---- F1 / B2 and F8 + F9 / B8: the W-direction transforms as GEMMs -------------------------------
// One tile = (b, h, 128 channels).  The constant DFT matrix is the A operand (accumulator
// rows = output index), the activation tile the MN-major B operand (columns = channels):
//   forward (INVERSE = false): D_ri[kw, c] = sum_w  Fw_ri[kw, w] * x[b,h,w,c]      ri = re, im
//   inverse (INVERSE = true) : D_a[w, c]   = sum_(ri,kw) Gw[w, (ri,kw)] * A2[..]    a = w / 128
// so every thread's accumulator row is 128 CONTIGUOUS channels of one output row and the
// epilogue is plain 32-byte vector I/O (no transpose).  Two 128x128x192 GEMMs per tile.
// Warp-specialised and persistent: producer warp p copies tiles it = p, p+2, .. (cp.async)
// into operand buffer p and issues their MMAs into accumulator pair p; the 8 epilogue warps
// (accumulator a = warp/4, TMEM lanes 32*(warp%4)..) drain tile it while tile it+1 computes.
__device__ __forceinline__ void pack32(const uint32_t (&v)[32], uint32_t (&pk)[16]) {
#pragma unroll
  for (int q = 0; q < 16; ++q) pk[q] = pack_bf16(__uint_as_float(v[2 * q]), __uint_as_float(v[2 * q + 1]));
}
__device__ __forceinline__ void ldg256(const void* p, uint32_t (&r)[8]) {
  asm volatile("ld.global.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
               : "l"(p));
}
__device__ __forceinline__ void stg256(void* p, const uint32_t* r) {
  asm volatile("st.global.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]),
               "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7])
               : "memory");
}

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
#else
#define DBG_T0()
#define DBG_ACC(slot)
#endif

template <bool INVERSE>
__global__ void __launch_bounds__(kRowThreads, 1)
tc_wdft(const __nv_bfloat16* __restrict__ in, const __nv_bfloat16* __restrict__ res, __nv_bfloat16* __restrict__ out,
        const uint8_t* __restrict__ Aconst, int B, int H, int W, int C, int Kw, int nb) {
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ __align__(8) uint64_t full[2], empty[2];
  __shared__ uint32_t tmem_slot;
  uint8_t* sF = smem;
  uint8_t* sB0 = smem + kFwBytes;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  for (uint32_t i = tid; i < 2 * kRowBytes / 16; i += kRowThreads) ((uint4*)sB0)[i] = make_uint4(0, 0, 0, 0);
  for (uint32_t i = tid; i < kFwBytes / 16; i += kRowThreads) cp_async16(smem_u32(sF) + i * 16, Aconst + (size_t)i * 16);
  if (tid == 0) {
    mbar_init(&full[0], 1);
    mbar_init(&full[1], 1);
    mbar_init(&empty[0], kRowEpiThreads);
    mbar_init(&empty[1], kRowEpiThreads);
    mbar_init_fence();
  }
  if (warp == 0) tmem_alloc<512>(&tmem_slot);
  cp_async_wait_all();
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  const int ncg = (C + CGRP - 1) / CGRP;
  const int ntiles = B * H * ncg;
  const int nmine = ntiles > (int)blockIdx.x ? (ntiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;

  if (warp >= kRowEpiThreads / 32) {
    // ===== producer group p (4 warps): tiles it = p, p+2, ... -> operand buffer p, accumulator pair p ==
    // (a single warp sustains only ~1 cp.async instruction per 200 cycles, so the copy is spread)
    const int pw = warp - kRowEpiThreads / 32;
    const int p = pw / kRowProdWarps, sub = pw % kRowProdWarps;
    const uint32_t dst = smem_u32(sB0) + p * kRowBytes;
    const uint32_t idesc = idesc_bf16(128, CGRP, kIdescBMn);
#ifdef AFNO_TIMING
    long long dbg_acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
#endif
    DBG_T0();
    for (int it = p; it < nmine; it += 2) {
      const int use = it >> 1;
      // the previous MMAs on this buffer have completed (their commit also frees the operand tile)
      if (use > 0) mbar_wait(&full[p], (uint32_t)((use - 1) & 1));
      DBG_ACC(0);
      const int t = blockIdx.x + it * gridDim.x;
      const int cg = t % ncg, bh = t / ncg;
      if (!INVERSE) {
        // x[b,h,:,cg*128 .. +128) -> MN-major B operand (K = w, N = channel).  One cp.async
        // instruction = 2 rows x 16 consecutive 16-byte chunks: full sectors on the global side
        const __nv_bfloat16* xrow = in + (size_t)bh * W * C + cg * CGRP;
        const int mc = lane & 15;
        const bool cok = cg * CGRP + mc * 8 < C;
        for (int w = 2 * sub + (lane >> 4); w < W; w += 2 * kRowProdWarps)
          if (cok) cp_async16(dst + mc * kRowSbo + w * 16, xrow + (size_t)w * C + mc * 8);
      } else {
        // A2[b][kw][j][h][ri][cl] (rows kA2Row elements apart) gathered into the MN-major B operand
        // (K = (ri,kw), N = channel)
        const int b = bh / H, h = bh - b * H;
        const size_t kwstride = (size_t)nb * H * kA2Row;
        const __nv_bfloat16* base = in + ((size_t)b * Kw * nb * H + h) * kA2Row;
        const int mc = lane & 15;
        const int c0 = cg * CGRP + mc * 8;
        const int j = c0 / BS, cl = c0 - j * BS;
        const __nv_bfloat16* cbase = base + (size_t)j * H * kA2Row + cl;
        for (int rr = 2 * sub + (lane >> 4); rr < 2 * Kw; rr += 2 * kRowProdWarps) {
          const int ri = rr >= Kw ? 1 : 0, kw = rr - ri * Kw;
          if (c0 < C) cp_async16(dst + mc * kRowSbo + (ri * BS + kw) * 16, cbase + (size_t)kw * kwstride + ri * BS);
        }
      }
      DBG_ACC(1);
      cp_async_wait_all();
      DBG_ACC(2);
      fence_async_smem();
      asm volatile("bar.sync %0, %1;" ::"r"(1 + p), "n"(kRowProdWarps * 32) : "memory");
      DBG_ACC(3);
      if (sub == 0 && elect_one()) {
        // the epilogue has drained this accumulator pair's previous contents
        if (use > 0) mbar_wait(&empty[p], (uint32_t)((use - 1) & 1));
        DBG_ACC(4);
        tc_fence_after();
#pragma unroll
        for (int a = 0; a < 2; ++a) {
          const uint32_t d = tmem + p * 256 + a * CGRP;
          const uint32_t am = smem_u32(sF) + a * kFwHalf;
#pragma unroll
          for (int ks = 0; ks < WP / 16; ++ks)
            mma_ss(d, smem_desc(am + ks * 2 * kFwLbo, kFwLbo, kFwSbo), smem_desc(dst + ks * 2 * kRowLbo, kRowLbo, kRowSbo),
                   idesc, ks > 0);
        }
        mma_commit(&full[p]);
        DBG_ACC(5);
      }
      __syncwarp();
    }
#ifdef AFNO_TIMING
    if (blockIdx.x == 0 && p == 0 && sub == 0 && lane == 0)
      for (int q = 0; q < 8; ++q) g_afno_dbg[(INVERSE ? 16 : 0) + q] = dbg_acc[q];
#endif
  } else {
    // ===== epilogue warps: accumulator a = warp / 4, row m = 32 * (warp % 4) + lane ====================
    const int a = warp >> 2;
    const int m = (warp & 3) * 32 + lane;
    const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
#ifdef AFNO_TIMING
    long long dbg_acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
#endif
    DBG_T0();
    for (int it = 0; it < nmine; ++it) {
      const int t = blockIdx.x + it * gridDim.x;
      const int cg = t % ncg, bh = t / ncg;
      // forward: row = frequency kw of part ri = a ; inverse: row = w = 128 a + m
      const int row = INVERSE ? a * 128 + m : m;
      const bool rvalid = INVERSE ? (row < W) : (row < Kw);
      const bool warp_has_rows = INVERSE ? (a * 128 + (warp & 3) * 32 < W) : ((warp & 3) * 32 < Kw);
      const int b = bh / H, h = bh - b * H;
      mbar_wait(&full[it & 1], (uint32_t)((it >> 1) & 1));
      DBG_ACC(0);
      tc_fence_after();
      const uint32_t acc = tmem + (it & 1) * 256 + a * CGRP + lane_base;
      if (warp_has_rows) {
#pragma unroll 1
        for (int k = 0; k < 4; ++k) {
          const int c = cg * CGRP + 32 * k;   // 32 channels of one block (96 = 3 * 32)
          uint32_t v[32], pk[16];
          tmem_ld32(acc + 32 * k, v);
          if (!INVERSE) {
            tmem_wait_ld();
            if (k == 3) {
              tc_fence_before();
              mbar_arrive(&empty[it & 1]);
            }
            pack32(v, pk);
            if (rvalid && c < C) {
              const int j = c / BS, cl = c - j * BS;
              __nv_bfloat16* dstp = out + ((((size_t)b * Kw + row) * nb + j) * H + h) * NT + a * BS + cl;
#ifndef AFNO_DBG_NO_STORE
              stg256(dstp, pk);
              stg256(dstp + 16, pk + 8);
#else
              if (pk[0] == 0x12345u) stg256(dstp, pk);
#endif
            }
          } else {
            uint32_t r0[8] = {0, 0, 0, 0, 0, 0, 0, 0}, r1[8] = {0, 0, 0, 0, 0, 0, 0, 0};
            const size_t off = ((size_t)bh * W + row) * C + c;
            const bool ok = rvalid && c < C;
            if (ok && res) {
              ldg256(res + off, r0);
              ldg256(res + off + 16, r1);
            }
            tmem_wait_ld();
            if (k == 3) {
              tc_fence_before();
              mbar_arrive(&empty[it & 1]);
            }
#pragma unroll
            for (int q = 0; q < 8; ++q) {
              // bf16 -> fp32 is a 16-bit shift; one rounding of (residual + branch)
              pk[q] = pack_bf16(__uint_as_float(v[2 * q]) + __uint_as_float(r0[q] << 16),
                                __uint_as_float(v[2 * q + 1]) + __uint_as_float(r0[q] & 0xFFFF0000u));
              pk[8 + q] = pack_bf16(__uint_as_float(v[16 + 2 * q]) + __uint_as_float(r1[q] << 16),
                                    __uint_as_float(v[16 + 2 * q + 1]) + __uint_as_float(r1[q] & 0xFFFF0000u));
            }
            if (ok) {
              stg256(out + off, pk);
              stg256(out + off + 16, pk + 8);
            }
          }
        }
      } else {
        tc_fence_before();
        mbar_arrive(&empty[it & 1]);
      }
      DBG_ACC(1);
    }
#ifdef AFNO_TIMING
    if (blockIdx.x == 0 && warp == 0 && lane == 0) {
      g_afno_dbg[(INVERSE ? 16 : 0) + 8] = dbg_acc[0];
      g_afno_dbg[(INVERSE ? 16 : 0) + 9] = dbg_acc[1];
      g_afno_dbg[(INVERSE ? 16 : 0) + 10] = nmine;
    }
#endif
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc<512>(tmem);
}

// ---- F2-F7 / B1-B7: per (b, kw, block) GEMM chains in tensor memory (kernel tc_mix2 below) ----------
constexpr int kMixLoadWarps = 3;

struct MixParams {
  const __nv_bfloat16* A1;   // forward: spectrum tiles; backward: x tiles
  const __nv_bfloat16* A1g;  // backward: gradient tiles
  __nv_bfloat16* A2;
  __nv_bfloat16 *Xh, *O1, *G2, *G1; // backward: operands of tc_wgrad
  const uint8_t* dft;        // Ch then Sh, kDft2Bytes each, smem image
  const uint8_t* wprep;      // per block 4 x kWBytes: W1r, W1i, W2r, W2i (n=o, k=i, K-major)
  const float* bprep;        // per block [2 layers][192]: (re 96 | im 96)
  uint8_t* mask1;            // optional export, [B][H][Wh][C][2]
  uint8_t* mask2;
  int B, H, Kw, Wh, nb, Kh;
  float lambda;
};

// rows of a (b,kw,j) tile [H][192] -> MN-major B operand (K = h, N = (ri, c)); loader warp `sub`
__device__ __forceinline__ void load_tile_warp(uint32_t tile_saddr, const __nv_bfloat16* src, int H, int lane, int sub) {
  // the tile is contiguous in global memory: chunk q = 16 bytes at src + 8 q, row h = q / 24
  const int nchunks = H * (NT / 8);
  for (int q = sub * 32 + lane; q < nchunks; q += kMixLoadWarps * 32) {
    const int h = q / (NT / 8), nc = q - h * (NT / 8);
    cp_async16(tile_saddr + nc * kTileSbo + h * 16, src + (size_t)q * 8);
  }
}

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
//     (warp % 4 == 3) are the control warp and the three loader warps; each of lane quarters 0..2
//     has four epilogue warps, one per 48-column quarter (re lo, re hi, im lo, im hi).
//   * three tile buffers: tile i lives in buffer i % 3 (input tile, then the B operand of the
//     inverse transform); backward: x tile, then the gradient tile, then GX.
// Every CTA works on ONE channel block j (grid = nb * S), so the weights are loaded once.
constexpr int kMix2Threads = 512;
constexpr uint32_t kDft2Lbo = 1536, kDft2Sbo = 128;  // Ch / Sh: K-major A, 96 stored rows, order [k/8][m/8 < 12]
constexpr uint32_t kDft2Bytes = 12 * kDft2Lbo;        // 18432 (rows 96..127 alias the next k-chunk: finite, unused)
// A tile buffer is also the staging area of the tile's output rows.  Rows are 400 bytes apart, in
// shared memory (eight consecutive rows fall into distinct 16-byte bank groups) AND in the global
// A2 tensor, so that a whole tile leaves with ONE bulk copy (async proxy, no L1 traffic).
constexpr uint32_t kOutStride = 2 * kA2Row;           // 400
constexpr uint32_t kTileBuf = 96 * kOutStride;        // 38400 >= kTileBytes
constexpr uint32_t kMix2Smem = 2 * kDft2Bytes + 4 * kWBytes + 3 * kTileBuf; // 225792
constexpr uint32_t kSlot = 96;

// bulk (async-proxy) store of a thread's own staged bytes: shared -> global, tracked by bulk groups
__device__ __forceinline__ void bulk_store(void* dst, uint32_t src_smem, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src_smem), "r"(bytes)
               : "memory");
  asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

struct Mix2Bars {
  uint64_t dfull[2];  // stream's current stage accumulated (tcgen05.commit)
  uint64_t edone[2];  // stream's current stage drained by the 12 epilogue warps
  uint64_t xfull[3];  // buffer holds the input tile (forward: spectrum; backward: x spectrum)
  uint64_t gfull[3];  // backward: buffer holds the gradient tile
  uint64_t xfree[3];  // backward: stage 0 has consumed the x tile (tcgen05.commit)
  uint64_t sdone[3];  // the 12 epilogue warps have staged the tile's output rows in the buffer
  uint64_t tfree[3];  // the staged rows have left the buffer (loader warp 0, after its bulk store has read them)
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
__device__ __forceinline__ void issue_fwd_dft2(uint32_t Dre, uint32_t Dim, uint32_t aCh, uint32_t aSh, uint32_t tile) {
  const uint32_t id = idesc_bf16(128, BS, kIdescBMn), half = (BS / 8) * kTileSbo;
  issue_dft2_pair(Dre, Dim, aCh, tile, tile + half, id, id, true);
  issue_dft2_pair(Dre, Dim, aSh, tile + half, tile, id, id | kIdescNegB, false);
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

template <bool BACKWARD, bool EXPORT>
__global__ void __launch_bounds__(kMix2Threads, 1) tc_mix2(MixParams p, int S) {
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ Mix2Bars bars;
  __shared__ uint32_t tmem_slot;
  __shared__ __align__(16) float sBias[2 * NT];
  constexpr int NS = BACKWARD ? 7 : 4;
  uint8_t* sCh = smem;
  uint8_t* sSh = smem + kDft2Bytes;
  uint8_t* sW = smem + 2 * kDft2Bytes;
  uint8_t* sT = sW + 4 * kWBytes;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int j = blockIdx.x / S, s0 = blockIdx.x - j * S;
  const int BKw = p.B * p.Kw;
  const int n = s0 < BKw ? (BKw - s0 + S - 1) / S : 0;   // tiles of this CTA: rem = s0 + i * S
  for (uint32_t i = tid; i < 3 * kTileBuf / 16; i += kMix2Threads) ((uint4*)sT)[i] = make_uint4(0, 0, 0, 0);
  for (uint32_t i = tid; i < 2 * kDft2Bytes / 16; i += kMix2Threads) cp_async16(smem_u32(sCh) + i * 16, p.dft + (size_t)i * 16);
  {
    const uint8_t* wsrc = p.wprep + (size_t)j * 4 * kWBytes;
    for (uint32_t i = tid; i < 4 * kWBytes / 16; i += kMix2Threads) cp_async16(smem_u32(sW) + i * 16, wsrc + (size_t)i * 16);
  }
  for (int i = tid; i < 2 * NT; i += kMix2Threads) sBias[i] = p.bprep[(size_t)j * 2 * NT + i];
  if (tid == 0) {
    for (int q = 0; q < 2; ++q) {
      mbar_init(&bars.dfull[q], 1);
      mbar_init(&bars.edone[q], 12);
    }
    for (int q = 0; q < 3; ++q) {
      mbar_init(&bars.xfull[q], kMixLoadWarps * 32);
      mbar_init(&bars.gfull[q], kMixLoadWarps * 32);
      mbar_init(&bars.xfree[q], 1);
      mbar_init(&bars.sdone[q], 12);
      mbar_init(&bars.tfree[q], 1);
    }
    mbar_init_fence();
  }
  if (warp == 0) tmem_alloc<512>(&tmem_slot);
  cp_async_wait_all();
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  // Stream 1 runs kLag stages behind stream 0, so tiles finish (and buffers become free) at
  // regular intervals and a transform stage of one stream overlaps an MLP stage of the other.
  constexpr int kLag = NS / 2;
  const int T = 2 * (NS * ((n + 1) / 2) + kLag);   // phases
  const int lq = warp & 3;

  if (lq == 3 && warp != 3) {
    // ================================ loader warps (7, 11, 15) ================================
    const int sub = (warp >> 2) - 1;
    const uint32_t aT = smem_u32(sT);
    auto tile_off = [&](int i) { return ((size_t)(s0 + i * S) * p.nb + j) * p.H * NT; };
    auto load = [&](int buf, const __nv_bfloat16* src, uint64_t* full) {
      // rows H..95 of the operand are K padding: the output staging of the buffer's previous tile
      // overlaps them, so they are cleared again
      for (int q = sub * 32 + lane; q < (HP - p.H) * (NT / 8); q += kMixLoadWarps * 32) {
        const int nc = q / (HP - p.H), h = p.H + q - nc * (HP - p.H);
        *(uint4*)(sT + buf * kTileBuf + nc * kTileSbo + h * 16) = make_uint4(0, 0, 0, 0);
      }
      load_tile_warp(aT + buf * kTileBuf, src, p.H, lane, sub);
      cp_async_wait_all();
      fence_async_smem();
      mbar_arrive(full);
    };
    // tile k's output rows are staged in its buffer by the epilogue warps; loader warp 0 sends them
    // to A2 with one bulk copy and frees the buffer once the copy has read it
    auto drain = [&](int k) {
      const int buf = k % 3;
      const uint32_t par = (uint32_t)((k / 3) & 1);
      if (sub == 0) {
        if (lane == 0) {
          mbar_wait(&bars.sdone[buf], par);
          bulk_store(p.A2 + ((size_t)(s0 + k * S) * p.nb + j) * p.H * kA2Row, aT + buf * kTileBuf,
                     (uint32_t)p.H * kOutStride);
          bulk_wait_read();
          mbar_arrive(&bars.tfree[buf]);
        }
        __syncwarp();
      }
      mbar_wait(&bars.tfree[buf], par);
    };
    if (!BACKWARD) {
      for (int i = 0; i < n; ++i) {
        if (i >= 3) drain(i - 3);
        load(i % 3, p.A1 + tile_off(i), &bars.xfull[i % 3]);
      }
      for (int k = n > 3 ? n - 3 : 0; k < n; ++k) drain(k);
    } else {
      // x(0) x(1) x(2) | g(0) g(1) | then for k = 0, 1, ..: x(k+3) after the last stage of tile k,
      // g(k+2) after stage 0 of tile k+2 -- the order in which the buffers become free
      for (int i = 0; i < 3 && i < n; ++i) load(i, p.A1 + tile_off(i), &bars.xfull[i]);
      for (int i = 0; i < 2 && i < n; ++i) {
        mbar_wait(&bars.xfree[i], 0u);
        load(i, p.A1g + tile_off(i), &bars.gfull[i]);
      }
      for (int k = 0; k < n; ++k) {
        const int ix = k + 3, ig = k + 2;
        drain(k);
        if (ix < n) load(ix % 3, p.A1 + tile_off(ix), &bars.xfull[ix % 3]);
        if (ig < n) {
          mbar_wait(&bars.xfree[ig % 3], (uint32_t)((ig / 3) & 1));
          load(ig % 3, p.A1g + tile_off(ig), &bars.gfull[ig % 3]);
        }
      }
    }
    if (sub == 0 && lane == 0) bulk_wait_all();
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
      const bool first = stg == 0, dftg = BACKWARD && stg == 3, last = stg == NS - 1;
      if (first) mbar_wait(&bars.xfull[buf], use & 1u);
      if (dftg) mbar_wait(&bars.gfull[buf], use & 1u);
      DBG_ACC(1);
      if (elect_one()) {
        tc_fence_after();
        if (first || dftg) {
          issue_fwd_dft2(Dre, Dim, aCh, aSh, tile);
        } else if (last) {
          issue_inv_dft2(Dre, Dim, aCh, aSh, tile);
        } else if (stg == 1) {
          issue_mlp2<false>(Dre, Dim, SA, w1r, w1i);
        } else if (stg == 2) {
          issue_mlp2<false>(Dre, Dim, SA, w2r, w2i);
        } else if (stg == 4) {
          issue_mlp2<true>(Dre, Dim, SA, w2r, w2i);    // G1 = G2 W2^H
        } else {
          issue_mlp2<true>(Dre, Dim, SA, w1r, w1i);    // GX = G1 W1^H
        }
        mma_commit(&bars.dfull[stream]);
        if (BACKWARD && first) mma_commit(&bars.xfree[buf]);
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
        const int rem = s0 + i * S;
        const uint32_t src = tmem + lane_sel + kSlot * (uint32_t)((3 * t + half) % 5) + chalf * 48;
        const uint32_t dstA = tmem + lane_sel + kSlot * (uint32_t)((3 * t) % 5) + 24 * cq;
        uint8_t* tile = sT + (i % 3) * kTileBuf;
        const size_t img_off = ((size_t)rem * p.nb + j) * kTileBytes;
        mbar_wait_fast(&bars.dfull[stream], ce[stream] & 1u);
        ++ce[stream];
        TR(t, 4 + warp * 3);
        DBG_ACC(0);
        tc_fence_after();
        uint32_t v[48], pk[24];
        ld48(src, v);
        DBG_ACC(2);
        bool writes_a = false, early_arrive = false;
        if (stg == 0) {
          // ---- spectrum Xh ----
          pack48(v, pk);
          writes_a = true;
          if (BACKWARD) store_chunks6((uint8_t*)p.Xh + img_off, chunk0, r, pk);
        } else if (stg == 1) {
          // ---- O1 = relu(P1 + b1) ----
#pragma unroll
          for (int q = 0; q < 12; ++q) {
            const float4 bq = *(const float4*)(bias1 + 4 * q);
            pk[2 * q] = pack_relu_bf16(__uint_as_float(v[4 * q]) + bq.x, __uint_as_float(v[4 * q + 1]) + bq.y);
            pk[2 * q + 1] = pack_relu_bf16(__uint_as_float(v[4 * q + 2]) + bq.z, __uint_as_float(v[4 * q + 3]) + bq.w);
          }
          if (BACKWARD) {
            m1[stream][0] = m1[stream][1] = 0;
            MaskLoop<0>::run([&](auto P) { mask_collect<decltype(P)::value>(m1[stream], pk[decltype(P)::value]); });
          }
          writes_a = true;
          if (BACKWARD) store_chunks6((uint8_t*)p.O1 + img_off, chunk0, r, pk);
        } else if (stg == 2) {
          // ---- P2 + b2: forward Z = softshrink (truncated) -> B operand of the inverse transform;
          //      backward: only the mask ----
          const float lam = p.lambda;
          if (!BACKWARD) {
            // Z = S_lambda(P2 + b2): the sum is rounded to bf16 once, then a - clamp(a, -lambda, lambda)
            // on packed pairs (exact zeros inside the threshold; lambda at bf16 precision)
            const uint32_t lam2 = pack_bf16(lam, lam), nlam2 = lam2 ^ 0x80008000u;
#pragma unroll
            for (int q = 0; q < 12; ++q) {
              const float4 bq = *(const float4*)(bias2 + 4 * q);
              pk[2 * q] = shrink_bf16x2(pack_bf16(__uint_as_float(v[4 * q]) + bq.x, __uint_as_float(v[4 * q + 1]) + bq.y),
                                        lam2, nlam2);
              pk[2 * q + 1] = shrink_bf16x2(
                  pack_bf16(__uint_as_float(v[4 * q + 2]) + bq.z, __uint_as_float(v[4 * q + 3]) + bq.w), lam2, nlam2);
            }
            if (!row_kept) {
#pragma unroll
              for (int q = 0; q < 24; ++q) pk[q] = 0u;
            }
            store_chunks6(tile, chunk0, r, pk);
            fence_async_smem();
          } else {
#pragma unroll
            for (int q = 0; q < 12; ++q) {
              const float4 bq = *(const float4*)(bias2 + 4 * q);
              // |P2 + b2| - lambda > 0  <=>  the rounded, relu-ed difference is non-zero
              pk[2 * q] = pack_relu_bf16(fabsf(__uint_as_float(v[4 * q]) + bq.x) - lam,
                                         fabsf(__uint_as_float(v[4 * q + 1]) + bq.y) - lam);
              pk[2 * q + 1] = pack_relu_bf16(fabsf(__uint_as_float(v[4 * q + 2]) + bq.z) - lam,
                                             fabsf(__uint_as_float(v[4 * q + 3]) + bq.w) - lam);
            }
            m2[stream][0] = m2[stream][1] = 0;
            if (row_kept)
              MaskLoop<0>::run([&](auto P) { mask_collect<decltype(P)::value>(m2[stream], pk[decltype(P)::value]); });
          }
        } else if (!BACKWARD || stg == 6) {
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
        } else if (stg == 3 || stg == 4) {
          // ---- G2 = G (.) mask2 ; G1 = mask1 (.) (G2 W2^H) ----
          pack48(v, pk);
          if (stg == 3) {
            MaskLoop<0>::run([&](auto P) { pk[decltype(P)::value] = mask_apply<decltype(P)::value>(m2[stream], pk[decltype(P)::value]); });
          } else {
            MaskLoop<0>::run([&](auto P) { pk[decltype(P)::value] = mask_apply<decltype(P)::value>(m1[stream], pk[decltype(P)::value]); });
          }
          writes_a = true;
          store_chunks6((uint8_t*)(stg == 3 ? p.G2 : p.G1) + img_off, chunk0, r, pk);
        } else {
          // ---- stage 5: GX -> B operand of the inverse transform (the tile's own buffer) ----
#pragma unroll
          for (int q = 0; q < 24; ++q)
            pk[q] = row_valid ? pack_bf16(__uint_as_float(v[2 * q]), __uint_as_float(v[2 * q + 1])) : 0u;
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
        { long long n_ = clock64(); dbg_m[stg] += n_ - dbg_t; dbg_t = n_; }
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
  __syncthreads();
  if (warp == 0) tmem_dealloc<512>(tmem);
}

// ---- B4 / B6: parameter gradients as a split-K tensor-core GEMM ------------------------------------
// For block j:  R[(ri_a,i), (ri_g,o)] = sum_rows A[row,(ri_a,i)] * G[row,(ri_g,o)] with K = mode rows.
// Two M=128 accumulators: D_re rows = (re, i) plus a constant-one row 96 (gives sum_rows G = db),
// D_im rows = (im, i).  CTA (j, s) sums tiles rem = s, s+S, ... and writes its partial sums.
constexpr uint32_t kWgALbo = 128, kWgASbo = 1536 + 16;                  // MN-major A [K=96][M=128], padded chunk stride
constexpr uint32_t kWgABytes = 16 * kWgASbo;                            // 24832
constexpr uint32_t kWgStage = 2 * kWgABytes + kTileBytes;              // 86016
constexpr uint32_t kWgSmem = 2 * kWgStage;                             // 172032

__device__ __forceinline__ void bulk_copy(uint32_t dst_smem, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst_smem),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}

// Aws / Gws: operand-image tensors written by tc_mix<true> ([tile][24 chunks][kTileSbo bytes]).
__global__ void __launch_bounds__(128, 1)
tc_wgrad(const __nv_bfloat16* __restrict__ Aws, const __nv_bfloat16* __restrict__ Gws, float* __restrict__ part,
         int BKw, int H, int nb, int S) {
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ __align__(8) uint64_t full[2], empty[2], done;
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
  const uint32_t tmem = tmem_slot;
  const uint32_t lane_base = (uint32_t)(warp * 32) << 16;
  const uint32_t Dre = tmem, Dim = tmem + 256;
  const uint32_t idesc = idesc_bf16(128, NT, kIdescAMn | kIdescBMn);
  const int nt = (BKw - s + S - 1) / S; // tiles of this CTA
  (void)lane;
  if (warp == 0 && elect_one()) {
    // ---- producer: three bulk copies per tile (A re half, A im half, G), async proxy, no LSU ----
    constexpr uint32_t kHalfImg = 12 * kTileSbo;
    for (int it = 0; it < nt; ++it) {
      const int b = it & 1, use = it >> 1;
      if (use > 0) mbar_wait(&empty[b], (uint32_t)((use - 1) & 1));
      const size_t off = ((size_t)(s + it * S) * nb + j) * kTileBytes;
      const uint32_t stage = smem_u32(smem) + b * kWgStage;
      mbar_expect_tx(&full[b], 2 * kHalfImg + kTileBytes);
      bulk_copy(stage, (const uint8_t*)Aws + off, kHalfImg, &full[b]);
      bulk_copy(stage + kWgABytes, (const uint8_t*)Aws + off + kHalfImg, kHalfImg, &full[b]);
      bulk_copy(stage + 2 * kWgABytes, (const uint8_t*)Gws + off, kTileBytes, &full[b]);
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
  float* dst = part + ((size_t)blockIdx.x * 2) * 128 * NT + (size_t)tid * NT;
  if (nt > 0) {
    mbar_wait(&done, 0u);
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
  float* bprep;
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
  w.A2 = (__nv_bfloat16*)take((size_t)g.B * g.Kw * g.nb * g.H * kA2Row * 2);
  w.wprep = (__nv_bfloat16*)take((size_t)g.nb * 4 * kWBytes);
  w.bprep = (float*)take((size_t)g.nb * 2 * NT * sizeof(float));
  if (backward) {
    w.A1g = (__nv_bfloat16*)take(spec);
    const size_t img = (size_t)g.B * g.Kw * g.nb * kTileBytes;   // operand-image layout
    w.Xh = (__nv_bfloat16*)take(img);
    w.O1 = (__nv_bfloat16*)take(img);
    w.G2 = (__nv_bfloat16*)take(img);
    w.G1 = (__nv_bfloat16*)take(img);
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
  // Ch, Sh: element (r, h) = cos / sin (2 pi r h / H) / sqrt(H); K-major, 96 rows stored, order [k/8][m/8 < 12]
  std::vector<uint16_t> dft2(2 * kDft2Bytes / 2, 0);
  for (int r = 0; r < H; ++r)
    for (int h = 0; h < H; ++h) {
      const double a = two_pi * (double)((long)r * h % H) / (double)H, s = 1.0 / sqrt((double)H);
      const uint32_t off = ((h / 8) * kDft2Lbo + (r / 8) * kDft2Sbo + (r % 8) * 16 + (h % 8) * 2) / 2;
      dft2[off] = host_bf16(cos(a) * s);
      dft2[kDft2Bytes / 2 + off] = host_bf16(sin(a) * s);
    }
  // W-direction constants as K-major A operands, two 128-row halves each (kFwHalf bytes):
  //   Fw  half ri : element (m = kw, k = w)          = {cos, -sin}(2 pi kw w / W) / sqrt(W)   [x alpha_kw]
  //   Gw  half a  : element (m = w - 128 a, k = ri*96 + kw) = alpha_kw {cos, -sin}(...) / sqrt(W)  [or alpha = 1]
  std::vector<uint16_t> fw(kFwBytes / 2, 0), fwa(kFwBytes / 2, 0), gw(kFwBytes / 2, 0), gw1(kFwBytes / 2, 0);
  auto aoff = [](int m, int k) { return ((k / 8) * kFwLbo + (m / 8) * kFwSbo + (m % 8) * 16 + (k % 8) * 2) / 2; };
  for (int kw = 0; kw < Wh; ++kw)
    for (int w = 0; w < W; ++w) {
      const double a = two_pi * (double)((long)kw * w % W) / (double)W, s = 1.0 / sqrt((double)W);
      const double alpha = (kw == 0 || 2 * kw == W) ? 1.0 : 2.0;
      for (int ri = 0; ri < 2; ++ri) {
        const double v = (ri == 0 ? cos(a) : -sin(a)) * s;
        const uint32_t of = ri * (kFwHalf / 2) + aoff(kw, w);
        const uint32_t og = (w / 128) * (kFwHalf / 2) + aoff(w % 128, ri * BS + kw);
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
  if (e == cudaSuccess) e = set_smem(tc_wdft<false>, kRowSmem);
  if (e == cudaSuccess) e = set_smem(tc_wdft<true>, kRowSmem);
  if (e == cudaSuccess) e = set_smem(tc_mix2<false, false>, kMix2Smem);
  if (e == cudaSuccess) e = set_smem(tc_mix2<true, false>, kMix2Smem);
  if (e == cudaSuccess) e = set_smem(tc_mix2<true, true>, kMix2Smem);
  if (e == cudaSuccess) e = set_smem(tc_wgrad, kWgSmem);
  int dev = 0, sms = 148;
  if (e == cudaSuccess) e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  out->num_sms = sms;
  out->valid = (e == cudaSuccess);
  return e;
}

// CTAs per channel block of tc_mix2 (every CTA works on one block)
static int mix2_split(const Geometry& g, const TcPlan& tp) {
  int S = tp.num_sms / g.nb;
  if (S < 1) S = 1;
  if (S > g.B * g.Kw) S = g.B * g.Kw;
  return S;
}

size_t tc_workspace_bytes(const Geometry& g, bool backward) {
  return tc_carve(g, backward, nullptr).total;
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
  const int ncg = (g.C + CGRP - 1) / CGRP;
  const int row_tiles = g.B * g.H * ncg;
  const int grid_row = row_tiles < tp.num_sms ? row_tiles : tp.num_sms;
  prof_begin("tc_wdft_fwd", st);
  tc_wdft<false><<<grid_row, kRowThreads, kRowSmem, st>>>((const __nv_bfloat16*)x, nullptr, w.A1, tp.fw, g.B, g.H, g.W,
                                                          g.C, g.Kw, g.nb);
  prof_end(st);
  count_launch();
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  MixParams mp{};
  mp.A1 = w.A1; mp.A2 = w.A2; mp.dft = tp.dft2; mp.wprep = (const uint8_t*)w.wprep; mp.bprep = w.bprep;
  mp.B = g.B; mp.H = g.H; mp.Kw = g.Kw; mp.Wh = g.Wh; mp.nb = g.nb; mp.Kh = g.Kh; mp.lambda = g.lambda;
  prof_begin("tc_mix_fwd", st);
  const int S2 = mix2_split(g, tp);
  tc_mix2<false, false><<<g.nb * S2, kMix2Threads, kMix2Smem, st>>>(mp, S2);
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
  TC_LAUNCH("k_tc_prep_weights", k_tc_prep_weights<<<(nW + 255) / 256, 256, 0, st>>>(w1, b1, w2, b2, w.wprep, w.bprep, g.nb));
  const int ncg = (g.C + CGRP - 1) / CGRP;
  const int row_tiles = g.B * g.H * ncg;
  const int grid_row = row_tiles < tp.num_sms ? row_tiles : tp.num_sms;
  // B1 (first half) and B2: W-direction spectra of x and of dy (alpha-weighted)
  if (!g.use_ctx) {
    TC_LAUNCH("tc_wdft_fwd", tc_wdft<false><<<grid_row, kRowThreads, kRowSmem, st>>>((const __nv_bfloat16*)x, nullptr, w.A1,
                                                                                    tp.fw, g.B, g.H, g.W, g.C, g.Kw, g.nb));
  }
  TC_LAUNCH("tc_wdft_fwd", tc_wdft<false><<<grid_row, kRowThreads, kRowSmem, st>>>((const __nv_bfloat16*)dy, nullptr, w.A1g,
                                                                                  tp.fw_alpha, g.B, g.H, g.W, g.C, g.Kw, g.nb));
  MixParams mp{};
  mp.A1 = w.A1; mp.A1g = w.A1g; mp.A2 = w.A2;
  mp.Xh = w.Xh; mp.O1 = w.O1; mp.G2 = w.G2; mp.G1 = w.G1;
  mp.dft = tp.dft2; mp.wprep = (const uint8_t*)w.wprep; mp.bprep = w.bprep;
  mp.mask1 = g.export_masks ? w.mask1 : nullptr;
  mp.mask2 = g.export_masks ? w.mask2 : nullptr;
  mp.B = g.B; mp.H = g.H; mp.Kw = g.Kw; mp.Wh = g.Wh; mp.nb = g.nb; mp.Kh = g.Kh; mp.lambda = g.lambda;
  const int S2 = mix2_split(g, tp);
  if (g.export_masks) {
    TC_LAUNCH("tc_mix_bwd", tc_mix2<true, true><<<g.nb * S2, kMix2Threads, kMix2Smem, st>>>(mp, S2));
  } else {
    TC_LAUNCH("tc_mix_bwd", tc_mix2<true, false><<<g.nb * S2, kMix2Threads, kMix2Smem, st>>>(mp, S2));
  }
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

#ifdef AFNO_TRACE
extern "C" int afno_trace_read(long long* out) {
  return (int)cudaMemcpyFromSymbol(out, g_afno_trace, sizeof(long long) * 64 * 32);
}
#endif
#ifdef AFNO_TIMING
extern "C" int afno_debug_read(long long* out) {
  return (int)cudaMemcpyFromSymbol(out, g_afno_dbg, sizeof(long long) * 128);
}
#endif

} // namespace afno
