// Part of the tcgen05 path (tc_path.cu includes the parts in order, inside namespace afno { namespace { ):
// tc_wgrad and k_tc_wgrad_reduce, the parameter gradients (rows B4, B6).
// Not a standalone header: it relies on tc_common.cuh and on the parts included before it.
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

// shared -> global bulk reduction (fp32 add), tracked by bulk groups
__device__ __forceinline__ void bulk_reduce_add_f32(void* dst, uint32_t src_smem, uint32_t bytes) {
  asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f32 [%0], [%1], %2;" ::"l"(dst), "r"(src_smem), "r"(bytes)
               : "memory");
  bulk_commit();
}

// Operand-image tensors written by tc_mix2<true> ([tile][24 chunks][kTileSbo bytes]).  ONE launch covers
// both layers: CTAs [0, nb*S) form layer 2 (A = O1, G = G2), CTAs [nb*S, 2*nb*S) layer 1 (A = Xh, G = G1).
__global__ void __launch_bounds__(128, 1)
tc_wgrad(const __nv_bfloat16* __restrict__ A_l2, const __nv_bfloat16* __restrict__ G_l2,
         const __nv_bfloat16* __restrict__ A_l1, const __nv_bfloat16* __restrict__ G_l1, float* __restrict__ part,
         int BKw, int H, int nb, int S, int accumulate) {
  extern __shared__ __align__(1024) uint8_t smem[];
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
  pdl_wait();
  const uint32_t tmem = tmem_slot;
  const uint32_t lane_base = (uint32_t)(warp * 32) << 16;
  const uint32_t Dre = tmem, Dim = tmem + 256;
  const uint32_t idesc = idesc_bf16(128, NT, kIdescAMn | kIdescBMn);
  const int nt = (BKw - s + S - 1) / S; // tiles of this CTA
  (void)lane;
  if (warp == 0 && elect_one()) {
    // ---- producer: three bulk copies per tile (A re half, A im half, G), async proxy, no LSU ----
    constexpr uint32_t kHalfImg = 12 * kTileSbo;
    const uint64_t pol_ctx = pol(kPolWgLoadCtx), pol_g = pol(kPolWgLoadG);
    for (int it = 0; it < nt; ++it) {
      const int b = it & 1, use = it >> 1;
      if (use > 0) mbar_wait(&empty[b], (uint32_t)((use - 1) & 1));
      const size_t off = ((size_t)(s + it * S) * nb + j) * kTileBytes;
      const uint32_t stage = smem_u32(smem) + b * kWgStage;
      mbar_expect_tx(&full[b], 2 * kHalfImg + kTileBytes);
      bulk_copy(stage, (const uint8_t*)Aws + off, kHalfImg, &full[b], pol_ctx);
      bulk_copy(stage + kWgABytes, (const uint8_t*)Aws + off + kHalfImg, kHalfImg, &full[b], pol_ctx);
      bulk_copy(stage + 2 * kWgABytes, (const uint8_t*)Gws + off, kTileBytes, &full[b], pol_g);
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
    // the first chunk of a call stores its partial sums, every later chunk adds to them (one CTA per
    // slot, launches in stream order: the summation order is fixed)
    if (accumulate) bulk_reduce_add_f32(part + (size_t)blockIdx.x * kWgPartFloats, smem_u32(smem), kWgPartFloats * 4);
    else bulk_store(part + (size_t)blockIdx.x * kWgPartFloats, smem_u32(smem), kWgPartFloats * 4, l2_evict_normal());
    bulk_wait<0>();
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc<512>(tmem);
}

// dW[blk][ii][oo] = sum_s ( Dre[i][o] + Dim[i][96+o] ,  Dre[i][96+o] - Dim[i][o] ) ;  db[ch] = sum_s Dre[96][(ri,o)]
// with (i, o) the positions of the block's channels inside their group of 96 (the off-diagonal blocks of the
// group's 96 x 96 product are not parameters and are dropped).
// blockIdx.y = 0: layer 2 partial sums (first ngroups*S CTAs of tc_wgrad), 1: layer 1
// USE_CONTEXT (`guard`): the last kernel of the call also checks the context header the forward call left against
// this call's descriptor; on a mismatch (context never saved, other geometry / flag set) the gradients become NaN
// here and the grid overwrites dx with NaN (a foreign context must not return plausible numbers).
__global__ void k_tc_wgrad_reduce(const float* part, float2* __restrict__ dW2, float2* __restrict__ dB2,
                                  float2* __restrict__ dW1, float2* __restrict__ dB1, int ngroups, int S, int bs, int C,
                                  int accumulate, int guard, const CtxHeader* __restrict__ got, const CtxHeader want,
                                  uint16_t* __restrict__ dx, size_t n_act, int wait_first) {
  pdl_launch_dependents();
  // wait_first = 0 (fused path): the kernel before this one in the stream is tc_wdft_inv2, which lets its dependents
  // start only after ITS prerequisites (tc_wgrad among them) have completed: the partial sums are final, and the
  // sums below run under the inverse transform; only the guard's overwrite of dx has to wait for it.
  // PTX promises visibility of a prerequisite grid's writes only to the grid that executes griddepcontrol.wait, and
  // this grid reads `part` BEFORE its own wait: the reads therefore go to L2 (ld.global.cg, __ldcg below), where
  // tc_wgrad's bulk stores / bulk reductions land, never through the non-coherent path or a stale L1 line, and
  // `part` is not declared __restrict__ (S5.3 states the reliance).
  if (wait_first) pdl_wait();
  bool ok = true;
  if (guard) {
    const uint32_t* a = (const uint32_t*)got;
    const uint32_t* b = (const uint32_t*)&want;
    for (uint32_t q = 0; q < sizeof(CtxHeader) / 4; ++q) ok = ok && (a[q] == b[q]);
  }
  const float poison = __int_as_float(0x7FC00000);
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  const int nW = C * bs;          // nb * bs * bs complex weights
  const int layer = blockIdx.y;
  const float* lpart = part + (size_t)layer * ngroups * S * kWgPartFloats;
  float2* dW = layer ? dW1 : dW2;
  float2* dB = layer ? dB1 : dB2;
  if (idx < nW) {
    const int oo = idx % bs, ci = idx / bs;            // input channel ci = blk * bs + ii, output blk * bs + oo
    const int co = (ci / bs) * bs + oo;
    const int j = ci / BS, i = ci - j * BS, o = co - j * BS;
    float2 acc = accumulate ? dW[idx] : make_float2(0.f, 0.f);
    for (int s = 0; s < S; ++s) {
      const float* P = lpart + (size_t)(j * S + s) * kWgPartFloats;
      const float* Pre = P + (size_t)i * kWgPitch;
      const float* Pim = P + (size_t)(kWgRowsRe + i) * kWgPitch;
      acc.x += __ldcg(Pre + o) + __ldcg(Pim + BS + o);
      acc.y += __ldcg(Pre + BS + o) - __ldcg(Pim + o);
    }
    dW[idx] = ok ? acc : make_float2(poison, poison);
  } else if (idx < nW + C) {
    const int k = idx - nW, j = k / BS, o = k - j * BS;
    float2 acc = accumulate ? dB[k] : make_float2(0.f, 0.f);
    for (int s = 0; s < S; ++s) {
      const float* P = lpart + (size_t)(j * S + s) * kWgPartFloats + (size_t)BS * kWgPitch;
      acc.x += __ldcg(P + o);
      acc.y += __ldcg(P + BS + o);
    }
    dB[k] = ok ? acc : make_float2(poison, poison);
  }
  if (!wait_first) pdl_wait();   // dx is complete (and this call's completion stays transitive)
  if (guard && !ok) {
    const size_t nthreads = (size_t)gridDim.x * gridDim.y * blockDim.x;
    const size_t t0 = ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * blockDim.x + threadIdx.x;
    for (size_t i = t0; i < n_act; i += nthreads) dx[i] = 0x7FC0;   // bf16 NaN
  }
}
