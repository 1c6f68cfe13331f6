// Part of the tcgen05 path (tc_path.cu includes the parts in order, inside namespace afno { namespace { ):
// tc_mix2, the per-mode GEMM chain in tensor memory (rows F2-F7, B1-B3, B5, B7, H part of B8).
// Not a standalone header: it relies on tc_common.cuh and on the parts included before it.
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
  int B, H, Kw, Wh, nb, C, Kh;   // nb = groups of 96 channels, C = channels (the last group may be partly filled)
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

// Z = S_lambda(v + b) evaluated on the fp32 accumulator (reading A15): z = t - min(max(t, -lambda), lambda)
// with t = v + b in fp32, exact zeros inside the threshold, then ONE rounding of the pair to bf16.  Forward
// value and backward mask (Z != 0, i.e. |t| > lambda in fp32) come from this one function, so the gradient
// is the gradient of the function the forward pass evaluates.
__device__ __forceinline__ uint32_t shrink_sum(float v0, float v1, float b0, float b1, float lam) {
  const float t0 = v0 + b0, t1 = v1 + b1;
  return pack_bf16(t0 - fminf(fmaxf(t0, -lam), lam), t1 - fminf(fmaxf(t1, -lam), lam));
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
  pdl_wait();   // the weight images below are written by an earlier kernel of the chain
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
    const uint64_t pol_stream = pol(kPolMixLoadA), pol_keep = pol(kPolMixStoreA);
    const uint64_t pol_img = SAVE ? pol(kPolMixStoreCtx) : pol(kPolMixStoreG);
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
      const int buf = i % 3;
      const uint32_t use = (uint32_t)(i / 3);
      const uint32_t tile = aT + buf * kTileBuf;
      const int se = stg + kStage0;
      const bool first = stg == 0, dftg = RECOMP && stg == 3, last = stg == NS - 1;
      if (first) mbar_wait(&bars.xfull[buf], use & 1u);
      if (dftg) mbar_wait(&bars.gfull[buf], use & 1u);
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
      if (stream) ++cs1; else ++cs0;
    }
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
    // BwdCtx: the mask bits of a stream's NEXT tile are loaded a whole tile ahead (a load issued just before
    // the first epilogue of the tile exposed ~1,000 cycles of its latency)
    auto mask_index = [&](int i) {
      return (((size_t)(rtop - i * step) * p.nb + j) * 12 + (size_t)(cq * 3 + lq)) * 32 + lane;
    };
    uint4 mkn[2] = {make_uint4(0, 0, 0, 0), make_uint4(0, 0, 0, 0)};
    if (CTXB) {
      if (0 < n) mkn[0] = p.maskbits[mask_index(0)];
      if (1 < n) mkn[1] = p.maskbits[mask_index(1)];
    }
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
        const size_t mask_idx = mask_index(i);
        uint4 mk = make_uint4(0, 0, 0, 0);
        if (CTXB && stg == 0) {
          mk = mkn[stream];
          if (i + 2 < n) mkn[stream] = p.maskbits[mask_index(i + 2)];
        }
        mbar_wait_fast(&bars.dfull[stream], ce[stream] & 1u);
        ++ce[stream];
        tc_fence_after();
        uint32_t v[48], pk[24];
        ld48(src, v);
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
#pragma unroll
          for (int q = 0; q < 12; ++q) {
            const float4 bq = *(const float4*)(bias2 + 4 * q);
            pk[2 * q] = shrink_sum(__uint_as_float(v[4 * q]), __uint_as_float(v[4 * q + 1]), bq.x, bq.y, lam);
            pk[2 * q + 1] = shrink_sum(__uint_as_float(v[4 * q + 2]), __uint_as_float(v[4 * q + 3]), bq.z, bq.w, lam);
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
            const int ch0 = j * BS + chalf * 48;   // first channel of this thread's 48 columns
            const size_t base = ((((size_t)b * p.H + r) * p.Wh + kw) * (size_t)p.C + (size_t)ch0) * 2 + half;
            MaskLoop<0>::run([&](auto P) {
              constexpr int pp = decltype(P)::value;
              if (ch0 + 2 * pp < p.C) {   // C is even: both channels of the pair exist or neither does
                p.mask1[base + (size_t)(2 * pp) * 2] = (uint8_t)mask_bit<pp>(m1[stream], 0);
                p.mask1[base + (size_t)(2 * pp + 1) * 2] = (uint8_t)mask_bit<pp>(m1[stream], 1);
                p.mask2[base + (size_t)(2 * pp) * 2] = (uint8_t)mask_bit<pp>(m2[stream], 0);
                p.mask2[base + (size_t)(2 * pp + 1) * 2] = (uint8_t)mask_bit<pp>(m2[stream], 1);
              }
            });
          }
        }
        if (writes_a) {
          // the four warps of this lane quarter have their accumulator columns in registers:
          // compact the bf16 operand into the first slot (columns of the other warps' sources)
          asm volatile("bar.sync %0, 128;" ::"r"(bar_id) : "memory");
          st24(dstA, pk);
          tmem_wait_st();
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
      }
    }
  }
  tc_fence_before();
  __syncthreads();   // end of the segment: every role is done, every copy has landed
  }
  tc_fence_after();
  if (warp == 0) tmem_dealloc<512>(tmem_slot);
}
