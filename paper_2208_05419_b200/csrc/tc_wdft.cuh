// Part of the tcgen05 path (tc_path.cu includes the parts in order, inside namespace afno { namespace { ):
// tc_wdft_fwd2 / tc_wdft_inv2, the W-direction transforms (rows F1, B2, F8 + F9, B8).
// Not a standalone header: it relies on tc_common.cuh and on the parts included before it.
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
             const uint32_t* __restrict__ Fimg, int ntiles, int nb, int H, int Kw, int independent) {
  extern __shared__ uint8_t smem_raw[];
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
  load_const_tmem(tmem, Fimg, warp, lane);   // plan constant: loads under the previous kernel's tail
  // `independent`: the previous kernel of the call (the weight-image kernel, the call's first and a plain launch)
  // touches nothing this kernel reads or writes, so the two run side by side; the wait moves to the end of this
  // kernel, which keeps completion transitive for the kernels behind it.
  if (!independent) pdl_wait();
  const int nmine = ntiles > (int)blockIdx.x ? (ntiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;

  const uint64_t pol_stream = pol(kPolWfLoadX), pol_keep = pol(kPolWfStoreA);
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
  if (independent) pdl_wait();
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc<512>(tmem);
}

// inverse: a ring of 3 operand tiles (A2 rows as K = ri * 96 + kw) and a ring of 3 residual / output tiles
__global__ void __launch_bounds__(kW2Threads, 1)
tc_wdft_inv2(const __grid_constant__ CUtensorMap mapA2, const __grid_constant__ CUtensorMap mapRes,
             const __grid_constant__ CUtensorMap mapY, const uint32_t* __restrict__ Gimg, int ntiles, int nb, int H, int W,
             int has_res) {
  extern __shared__ uint8_t smem_raw[];
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
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  load_const_tmem(tmem, Gimg, warp, lane);   // plan constant: loads under the previous kernel's tail
  pdl_wait();
  // AFTER the wait: a dependent kernel that becomes resident beside this one (k_tc_wgrad_reduce: no shared memory)
  // may then rely on everything before this kernel in the stream having completed, and does its sums under this
  // kernel instead of after it
  pdl_launch_dependents();
  const int nmine = ntiles > (int)blockIdx.x ? (ntiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;

  const uint64_t pol_spec = pol(kPolWiLoadA), pol_res = pol(kPolWiLoadRes), pol_out = pol(kPolWiStoreY);
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
      tma_load5(aO + s * kW2Tile + (pn % 3) * kPanel + (pn / 3) * (BS * 64), &mapA2, 0, pn, j * H + h, 0, b, &ofull[s], pol_spec);
    if (has_res) {
      if (it >= kWiSlots) mbar_wait(&rfree[s], par);  // the slot's previous store has read it
      mbar_expect_tx(&rfull[s], kW2Tile);
#pragma unroll
      for (int pn = 0; pn < 3; ++pn)
        tma_load3(aR + s * kW2Tile + pn * kPanel, &mapRes, j * BS + pn * 32, 0, bh, &rfull[s], pol_res);
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
  if (warp == 0) tmem_dealloc<512>(tmem);
}
