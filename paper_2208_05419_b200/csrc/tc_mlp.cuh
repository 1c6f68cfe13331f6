// Part of the tcgen05 path (tc_path.cu includes the parts in order, inside namespace afno { namespace { ):
// tc_mlp_fwd, rows F3-F6 for grids the fused chain (tc_mix2) does not reach (H > 96 or W/2+1 > 96, e.g. the 180x360
// grid of BASELINE.json configs[3]): the transforms run as fp32 mixed-radix FFTs on the CUDA cores (generic.cu,
// the design BASELINE.json:north_star describes), the block-diagonal complex MLP on the tensor cores.
// Not a standalone header: it relies on tc_common.cuh and on the parts included before it.
//
// The spectrum is the generic path's X[row][C] (fp32 complex, row = (b, h, kw < Kw)); the kernel works IN PLACE on
// tiles of 128 rows x one group of 96 channels:
//   fp32 tile --cp.async--> staging --convert--> bf16 A operand [128 x (re 96 | im 96)] (K-major, shared memory)
//   D1 = A W1 (tensor memory) -> + b1, split ReLU -> bf16 A operand (the same buffer) -> D2 = O1 W2
//   -> + b2, softshrink on the fp32 sum, truncation -> fp32 complex back to X.
// Weights are the images k_tc_prep_weights builds (block-diagonal for blocks narrower than 96).  Every CTA works
// on one group, so the weights load once; the next tile streams into the staging buffer while this one computes.
constexpr int kMlpThreads = 256;
constexpr int kMlpRows = 128;
constexpr uint32_t kMlpALbo = kMlpRows * 16 + 16, kMlpASbo = 128;   // K-major A [128 x 192]: k-chunk stride padded by 16 B
constexpr uint32_t kMlpABytes = (NT / 8) * kMlpALbo;                // 49,536
template <typename ST>
constexpr uint32_t mlp_stage_bytes() { return kMlpRows * BS * (uint32_t)sizeof(ST); }   // 98,304 (fp32) / 49,152 (bf16): [128 rows][96 complex]
template <typename ST>
constexpr uint32_t mlp_fwd_smem() { return 4 * kWBytes + kMlpABytes + mlp_stage_bytes<ST>(); }   // 221,568 / 172,416

struct MlpParams {
  void* X;                   // [rows][C] complex (fp32 or bf16: the kernel's ST), transformed in place
  const uint8_t* wprep;      // per group 4 x kWBytes: W1r, W1i, W2r, W2i
  const float* bprep;        // per group [2 layers][192]
  long long rows;
  int C, ngroups, H, Kw, Kh;
  float lambda;
};

// ---- pieces shared by the kernels of the hybrid path -------------------------------------------------------------------------
// ST = storage type of the spectrum (afno_internal.h): float2 (fp32 complex) or SpecBf16 (bf16 complex, used when every
// transform of the call runs through the two-pass FFT kernels).

// 8 adjacent complex channels (at `src`, global or shared memory) -> bf16 (re x 8, im x 8)
template <typename ST>
__device__ __forceinline__ void mlp_pack8(const ST* src, uint4& re, uint4& im);
template <>
__device__ __forceinline__ void mlp_pack8<float2>(const float2* src, uint4& re, uint4& im) {
  const float4* s4 = (const float4*)src;
  const float4 a = s4[0], b = s4[1], c = s4[2], d = s4[3];
  re = make_uint4(pack_bf16(a.x, a.z), pack_bf16(b.x, b.z), pack_bf16(c.x, c.z), pack_bf16(d.x, d.z));
  im = make_uint4(pack_bf16(a.y, a.w), pack_bf16(b.y, b.w), pack_bf16(c.y, c.w), pack_bf16(d.y, d.w));
}
template <>
__device__ __forceinline__ void mlp_pack8<SpecBf16>(const SpecBf16* src, uint4& re, uint4& im) {
  const uint4* s4 = (const uint4*)src;   // a word = (re, im) of one channel: de-interleave by byte permutes
  const uint4 a = s4[0], b = s4[1];
  re = make_uint4(__byte_perm(a.x, a.y, 0x5410), __byte_perm(a.z, a.w, 0x5410), __byte_perm(b.x, b.y, 0x5410), __byte_perm(b.z, b.w, 0x5410));
  im = make_uint4(__byte_perm(a.x, a.y, 0x7632), __byte_perm(a.z, a.w, 0x7632), __byte_perm(b.x, b.y, 0x7632), __byte_perm(b.z, b.w, 0x7632));
}

// T (+)= A W (transposed = false) or A W^H (true) as real GEMMs on the (re | im) halves; A = bf16 K-major
// [96 rows][re 96 | im 96] in shared memory (chunk of 8 columns = kTileSbo bytes), W = the images of one 96 x 96 block
// (read as MN-major operands with the negate bit for the conjugate transpose); acc0 = 1 keeps what D holds.
__device__ __forceinline__ void mlp_issue_gemm(uint32_t D, uint32_t aA, uint32_t wr, uint32_t wi, bool transposed, uint32_t acc0,
                                               uint64_t* bar) {
  const uint32_t id = idesc_bf16(128, BS, transposed ? kIdescBMn : 0u);
  const uint32_t lbo = transposed ? kWSbo : kWLbo, sbo = transposed ? kWLbo : kWSbo;
#pragma unroll
  for (int ks = 0; ks < BS / 16; ++ks) {
    const uint64_t ad = smem_desc(aA + ks * 2 * kTileSbo, kTileSbo, kTileLbo);
    mma_ss(D, ad, smem_desc(wr + ks * 2 * lbo, lbo, sbo), id, acc0 | (uint32_t)(ks != 0));
    mma_ss(D + BS, ad, smem_desc(wi + ks * 2 * lbo, lbo, sbo), transposed ? (id | kIdescNegB) : id, acc0 | (uint32_t)(ks != 0));
  }
#pragma unroll
  for (int ks = 0; ks < BS / 16; ++ks) {
    const uint64_t ad = smem_desc(aA + (BS / 8 + ks * 2) * kTileSbo, kTileSbo, kTileLbo);
    mma_ss(D, ad, smem_desc(wi + ks * 2 * lbo, lbo, sbo), transposed ? id : (id | kIdescNegB), 1u);
    mma_ss(D + BS, ad, smem_desc(wr + ks * 2 * lbo, lbo, sbo), id, 1u);
  }
  mma_commit(bar);
}
// ROWS complex rows of one channel group -> bf16 K-major operand buffer (chunk of 8 columns = STRIDE bytes); lanes run
// over the 8-channel chunks of a row.  Rows past `rows` and channels past `nch` become zero.  mask2 != nullptr: the
// softshrink mask of the row ({re bits 0..31, re 32..47, im 0..31, im 32..47} per row and 48-channel half) is applied.
template <int ROWS, uint32_t STRIDE, typename ST>
__device__ __forceinline__ void mlp_load_operand(const ST* __restrict__ src_rows, long long r0, long long rows, int C, int ch0, int nch,
                                                 uint8_t* dstbuf, const uint4 (*mask2)[2], int tid) {
  for (uint32_t u = tid; u < ROWS * (BS / 8); u += kMlpThreads) {
    const int rr = u / (BS / 8), c8 = u - rr * (BS / 8);
    uint4 re = make_uint4(0, 0, 0, 0), im = re;
    if (r0 + rr < rows && 8 * c8 < nch) mlp_pack8<ST>(src_rows + (size_t)(r0 + rr) * C + ch0 + 8 * c8, re, im);
    if (mask2 != nullptr) {
      const uint4 mk = mask2[rr][c8 / 6];
      const int sh = (c8 % 6) * 8;
      const uint32_t mre = (uint32_t)((((uint64_t)mk.y << 32) | mk.x) >> sh) & 0xFFu;
      const uint32_t mim = (uint32_t)((((uint64_t)mk.w << 32) | mk.z) >> sh) & 0xFFu;
      auto sel = [](uint32_t v, uint32_t bits) {   // bits: bit 0 -> low half, bit 1 -> high half
        return v & ((bits & 1u ? 0x0000FFFFu : 0u) | (bits & 2u ? 0xFFFF0000u : 0u));
      };
      re = make_uint4(sel(re.x, mre), sel(re.y, mre >> 2), sel(re.z, mre >> 4), sel(re.w, mre >> 6));
      im = make_uint4(sel(im.x, mim), sel(im.y, mim >> 2), sel(im.z, mim >> 4), sel(im.w, mim >> 6));
    }
    uint8_t* dst = dstbuf + (size_t)rr * 16;
    *(uint4*)(dst + (size_t)c8 * STRIDE) = re;
    *(uint4*)(dst + (size_t)(BS / 8 + c8) * STRIDE) = im;
  }
}
// The same in two halves, for the bf16 spectrum (32 bytes per unit): fetch keeps a thread's units in registers, so that
// the loads of the NEXT operand are in flight under a GEMM and its epilogue; commit de-interleaves, masks and stores.
constexpr int kMlpFetchUnits = (HP * (BS / 8) + kMlpThreads - 1) / kMlpThreads;   // 5
struct MlpFetch { uint4 a[kMlpFetchUnits], b[kMlpFetchUnits]; };
__device__ __forceinline__ void mlp_fetch_operand(const SpecBf16* __restrict__ src_rows, long long r0, long long rows, int C, int ch0,
                                                  int nch, int tid, MlpFetch& f) {
#pragma unroll
  for (int k = 0; k < kMlpFetchUnits; ++k) {
    const uint32_t u = tid + k * kMlpThreads;
    const int rr = u / (BS / 8), c8 = u - rr * (BS / 8);
    f.a[k] = f.b[k] = make_uint4(0, 0, 0, 0);
    if (u < HP * (BS / 8) && r0 + rr < rows && 8 * c8 < nch) {
      const uint4* src = (const uint4*)(src_rows + (size_t)(r0 + rr) * C + ch0 + 8 * c8);
      f.a[k] = __ldg(src);
      f.b[k] = __ldg(src + 1);
    }
  }
}
__device__ __forceinline__ void mlp_commit_operand(const MlpFetch& f, uint8_t* dstbuf, const uint4 (*mask2)[2], int tid) {
#pragma unroll
  for (int k = 0; k < kMlpFetchUnits; ++k) {
    const uint32_t u = tid + k * kMlpThreads;
    if (u >= HP * (BS / 8)) continue;
    const int rr = u / (BS / 8), c8 = u - rr * (BS / 8);
    const uint4 a = f.a[k], b = f.b[k];
    uint4 re = make_uint4(__byte_perm(a.x, a.y, 0x5410), __byte_perm(a.z, a.w, 0x5410), __byte_perm(b.x, b.y, 0x5410), __byte_perm(b.z, b.w, 0x5410));
    uint4 im = make_uint4(__byte_perm(a.x, a.y, 0x7632), __byte_perm(a.z, a.w, 0x7632), __byte_perm(b.x, b.y, 0x7632), __byte_perm(b.z, b.w, 0x7632));
    if (mask2 != nullptr) {
      const uint4 mk = mask2[rr][c8 / 6];
      const int sh = (c8 % 6) * 8;
      const uint32_t mre = (uint32_t)((((uint64_t)mk.y << 32) | mk.x) >> sh) & 0xFFu;
      const uint32_t mim = (uint32_t)((((uint64_t)mk.w << 32) | mk.z) >> sh) & 0xFFu;
      auto sel = [](uint32_t v, uint32_t bits) { return v & ((bits & 1u ? 0x0000FFFFu : 0u) | (bits & 2u ? 0xFFFF0000u : 0u)); };
      re = make_uint4(sel(re.x, mre), sel(re.y, mre >> 2), sel(re.z, mre >> 4), sel(re.w, mre >> 6));
      im = make_uint4(sel(im.x, mim), sel(im.y, mim >> 2), sel(im.z, mim >> 4), sel(im.w, mim >> 6));
    }
    uint8_t* dst = dstbuf + (size_t)rr * 16;
    *(uint4*)(dst + (size_t)c8 * kTileSbo) = re;
    *(uint4*)(dst + (size_t)(BS / 8 + c8) * kTileSbo) = im;
  }
}
// 48 accumulator columns of this thread's row (the caller waits with tmem_wait_ld)
__device__ __forceinline__ void mlp_ld48(uint32_t taddr, uint32_t (&v)[48]) {
  tmem_ld16<0>(taddr, v);
  tmem_ld16<16>(taddr + 16, v);
  tmem_ld16<32>(taddr + 32, v);
}
// O1 = relu(v + bias) of 48 columns -> six 16-byte pieces of the operand buffer; returns the ReLU mask bits
__device__ __forceinline__ uint64_t mlp_relu_store(const uint32_t (&v)[48], const float* bias, uint8_t* dst) {
  uint64_t m = 0;
#pragma unroll
  for (int g = 0; g < 6; ++g) {
    uint32_t pk[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const float lo = __uint_as_float(v[8 * g + 2 * e]) + bias[8 * g + 2 * e];
      const float hi = __uint_as_float(v[8 * g + 2 * e + 1]) + bias[8 * g + 2 * e + 1];
      m |= (uint64_t)(lo > 0.f) << (8 * g + 2 * e);
      m |= (uint64_t)(hi > 0.f) << (8 * g + 2 * e + 1);
      pk[e] = pack_relu_bf16(lo, hi);
    }
    *(uint4*)(dst + (size_t)g * kTileSbo) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
  }
  return m;
}
// G1 = mask (.) v of 48 columns -> operand buffer
__device__ __forceinline__ void mlp_masked_store(const uint32_t (&v)[48], uint64_t m, uint8_t* dst) {
#pragma unroll
  for (int g = 0; g < 6; ++g) {
    uint32_t pk[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const int c = 8 * g + 2 * e;
      const float lo = ((m >> c) & 1u) ? __uint_as_float(v[c]) : 0.f;
      const float hi = ((m >> (c + 1)) & 1u) ? __uint_as_float(v[c + 1]) : 0.f;
      pk[e] = pack_bf16(lo, hi);
    }
    *(uint4*)(dst + (size_t)g * kTileSbo) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
  }
}
// softshrink mask bits of 48 columns: |v + bias| > lambda on kept rows
__device__ __forceinline__ uint64_t mlp_shrink_mask(const uint32_t (&v)[48], const float* bias, float lam, bool kept) {
  uint64_t m = 0;
#pragma unroll
  for (int c = 0; c < 48; ++c) m |= (uint64_t)(kept && fabsf(__uint_as_float(v[c]) + bias[c]) > lam) << c;
  return m;
}
// complex values (re in vr, im in vi: 48 channels of this thread's row, fp32 bits) -> rows of the spectrum G: each warp
// transposes its 32 rows through a private slice of an idle operand buffer (16 channels per pass, padded row pitch) and
// stores 128 (fp32) / 64 (bf16) contiguous bytes per row
template <typename ST>
__device__ __forceinline__ void mlp_store_rows(const uint32_t (&vr)[48], const uint32_t (&vi)[48], uint8_t* scratch, ST* G,
                                               long long wrow0, long long rows, int C, int chg, int nch, int lane) {
  constexpr uint32_t kRow = 16 * sizeof(ST), kPitch = kRow + 16, kPieces = kRow / 16, kCpp = 16 / sizeof(ST);   // channels per 16-byte piece
#pragma unroll
  for (int pass = 0; pass < 3; ++pass) {
#pragma unroll
    for (int c = 0; c < 16; c += 2) {
      const int cc = pass * 16 + c;
      SpecIO<ST>::stpair((ST*)(scratch + lane * kPitch) + c, make_float2(__uint_as_float(vr[cc]), __uint_as_float(vi[cc])),
                         make_float2(__uint_as_float(vr[cc + 1]), __uint_as_float(vi[cc + 1])));
    }
    __syncwarp();
    const int chp = pass * 16;   // first channel of this pass within the thread's 48
#pragma unroll
    for (int it = 0; it < (int)kPieces; ++it) {
      const int id = it * 32 + lane, rr = id / (int)kPieces, piece = id % (int)kPieces;
      const uint4 o = *(const uint4*)(scratch + rr * kPitch + piece * 16);
      if (wrow0 + rr < rows && chg + chp + (int)kCpp * piece < nch)
        *(uint4*)(G + (size_t)(wrow0 + rr) * C + chg + chp + kCpp * piece) = o;
    }
    __syncwarp();
  }
}
// Z = softshrink(P2 + b2) on the fp32 sum (reading A15), zero on truncated rows, in place in the accumulator registers
__device__ __forceinline__ void mlp_shrink48(uint32_t (&vr)[48], uint32_t (&vi)[48], const float* bre, const float* bim, float lam,
                                             bool kept) {
#pragma unroll
  for (int c = 0; c < 48; ++c) {
    const float t0 = __uint_as_float(vr[c]) + bre[c], t1 = __uint_as_float(vi[c]) + bim[c];
    vr[c] = __float_as_uint(kept ? t0 - fminf(fmaxf(t0, -lam), lam) : 0.f);
    vi[c] = __float_as_uint(kept ? t1 - fminf(fmaxf(t1, -lam), lam) : 0.f);
  }
}
// activation masks of this thread's 48 channels -> [..][C'][2] bytes (parity tests)
__device__ __forceinline__ void mlp_export_mask(uint8_t* dst, uint64_t mre, uint64_t mim, int nvalid) {
  for (int c = 0; c < 48; ++c)
    if (c < nvalid) *(uchar2*)(dst + 2 * c) = make_uchar2((unsigned char)((mre >> c) & 1u), (unsigned char)((mim >> c) & 1u));
}

template <typename ST>
__global__ void __launch_bounds__(kMlpThreads, 1) tc_mlp_fwd(const MlpParams p, int S) {
  extern __shared__ __align__(1024) uint8_t smem[];
  ST* const X = (ST*)p.X;
  __shared__ __align__(8) uint64_t done[2];
  __shared__ uint32_t tmem_slot;
  __shared__ __align__(16) float sBias[2 * NT];
  uint8_t* sW = smem;
  uint8_t* sA = smem + 4 * kWBytes;
  uint8_t* sStage = sA + kMlpABytes;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int j = blockIdx.x / S, s0 = blockIdx.x - j * S;
  const long long ntiles = (p.rows + kMlpRows - 1) / kMlpRows;
  const int ch0 = j * BS;                       // first channel of the group
  const int nch = min(BS, p.C - ch0);           // channels of the group that exist (a multiple of 8)
  pdl_launch_dependents();
  for (uint32_t i = tid; i < kMlpABytes / 16; i += kMlpThreads) ((uint4*)sA)[i] = make_uint4(0, 0, 0, 0);
  if (tid == 0) {
    mbar_init(&done[0], 1);
    mbar_init(&done[1], 1);
    mbar_init_fence();
  }
  if (warp == 0) tmem_alloc<512>(&tmem_slot);
  pdl_wait();   // the spectrum and the weight images are written by earlier kernels of the call
  {
    const uint8_t* wsrc = p.wprep + (size_t)j * 4 * kWBytes;
    for (uint32_t i = tid; i < 4 * kWBytes / 16; i += kMlpThreads) cp_async16(smem_u32(sW) + i * 16, wsrc + (size_t)i * 16);
  }
  for (int i = tid; i < 2 * NT; i += kMlpThreads) sBias[i] = p.bprep[(size_t)j * 2 * NT + i];
  // staging loads of one tile: 16-byte pieces, a row of the group is nch * sizeof(ST) contiguous bytes; pieces past the
  // last row or the last channel are zero-filled (cp.async with src-size 0)
  constexpr int kCpp = 16 / sizeof(ST), kPpr = BS / kCpp;   // channels per piece, pieces per row
  auto stage_tile = [&](long long t) {
    const long long r0 = t * kMlpRows;
    for (uint32_t i = tid; i < mlp_stage_bytes<ST>() / 16; i += kMlpThreads) {
      const int r = i / kPpr, c2 = i - r * kPpr;
      const bool ok = (r0 + r < p.rows) && (kCpp * c2 < nch);
      const ST* src = X + (size_t)(ok ? r0 + r : 0) * p.C + ch0 + (ok ? kCpp * c2 : 0);
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_u32(sStage) + i * 16), "l"(src), "r"(ok ? 16 : 0)
                   : "memory");
    }
    cp_async_commit();
  };
  if (s0 < ntiles) stage_tile(s0);
  cp_async_wait_all();
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  const uint32_t aW = smem_u32(sW), aA = smem_u32(sA);
  const uint32_t w1r = aW, w1i = aW + kWBytes, w2r = aW + 2 * kWBytes, w2i = aW + 3 * kWBytes;
  const uint32_t D1 = tmem, D2 = tmem + NT;   // (re 96 | im 96) each
  const int q = warp & 3, chalf = warp >> 2;  // TMEM lane quarter, column half (48 of the 96 channels)
  const int r = q * 32 + lane;
  const uint32_t lane_sel = (uint32_t)(q * 32) << 16;
  uint32_t ph = 0;
  // T = A W as real GEMMs on the (re | im) halves: T_re = A_re W_re - A_im W_im ; T_im = A_re W_im + A_im W_re
  auto issue_layer = [&](uint32_t D, uint32_t wr, uint32_t wi, uint64_t* bar) {
    const uint32_t id = idesc_bf16(128, BS, 0u);
#pragma unroll
    for (int ks = 0; ks < BS / 16; ++ks) {
      const uint64_t ad = smem_desc(aA + ks * 2 * kMlpALbo, kMlpALbo, kMlpASbo);
      mma_ss(D, ad, smem_desc(wr + ks * 2 * kWLbo, kWLbo, kWSbo), id, ks != 0);
      mma_ss(D + BS, ad, smem_desc(wi + ks * 2 * kWLbo, kWLbo, kWSbo), id, ks != 0);
    }
#pragma unroll
    for (int ks = 0; ks < BS / 16; ++ks) {
      const uint64_t ad = smem_desc(aA + (BS / 8 + ks * 2) * kMlpALbo, kMlpALbo, kMlpASbo);
      mma_ss(D, ad, smem_desc(wi + ks * 2 * kWLbo, kWLbo, kWSbo), id | kIdescNegB, 1u);
      mma_ss(D + BS, ad, smem_desc(wr + ks * 2 * kWLbo, kWLbo, kWSbo), id, 1u);
    }
    mma_commit(bar);
  };
  for (long long t = s0; t < ntiles; t += S) {
    const long long r0 = t * kMlpRows;
    // ---- staging -> bf16 A operand: unit = (row, 8 channels); lanes run over the channel chunks ----
    for (uint32_t u = tid; u < kMlpRows * (BS / 8); u += kMlpThreads) {
      const int rr = u / (BS / 8), c8 = u - rr * (BS / 8);
      uint4 re, im;
      mlp_pack8<ST>((const ST*)sStage + (size_t)rr * BS + 8 * c8, re, im);
      uint8_t* dst = sA + (size_t)rr * 16;
      *(uint4*)(dst + (size_t)c8 * kMlpALbo) = re;
      *(uint4*)(dst + (size_t)(BS / 8 + c8) * kMlpALbo) = im;
    }
    fence_async_smem();
    __syncthreads();
    if (t + S < ntiles) stage_tile(t + S);   // the next tile streams in while this one computes
    if (warp == 0 && elect_one()) {
      tc_fence_after();
      issue_layer(D1, w1r, w1i, &done[0]);
    }
    __syncwarp();
    mbar_wait(&done[0], ph);
    tc_fence_after();
    // ---- O1 = relu(P1 + b1) -> bf16 A operand of layer 2 (the A buffer is free: layer 1 has completed) ----
#pragma unroll
    for (int half = 0; half < 2; ++half) {
      uint32_t v[48];
      tmem_ld16<0>(D1 + lane_sel + half * BS + chalf * 48, v);
      tmem_ld16<16>(D1 + lane_sel + half * BS + chalf * 48 + 16, v);
      tmem_ld16<32>(D1 + lane_sel + half * BS + chalf * 48 + 32, v);
      tmem_wait_ld();
      const float* bias = sBias + half * BS + chalf * 48;
      uint8_t* dst = sA + (size_t)(r >> 3) * kMlpASbo + (r & 7) * 16 + (size_t)(half * (BS / 8) + chalf * 6) * kMlpALbo;
#pragma unroll
      for (int g = 0; g < 6; ++g) {
        uint32_t pk[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const float lo = fmaxf(__uint_as_float(v[8 * g + 2 * e]) + bias[8 * g + 2 * e], 0.f);
          const float hi = fmaxf(__uint_as_float(v[8 * g + 2 * e + 1]) + bias[8 * g + 2 * e + 1], 0.f);
          pk[e] = pack_bf16(lo, hi);
        }
        *(uint4*)(dst + (size_t)g * kMlpALbo) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
      }
    }
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    if (warp == 0 && elect_one()) {
      tc_fence_after();
      issue_layer(D2, w2r, w2i, &done[1]);
    }
    __syncwarp();
    mbar_wait(&done[1], ph);
    tc_fence_after();
    // ---- Z = softshrink(P2 + b2) on the fp32 sum, zero on truncated rows -> spectrum rows, in place ----
    {
      uint32_t vr[48], vi[48];
      mlp_ld48(D2 + lane_sel + chalf * 48, vr);
      mlp_ld48(D2 + lane_sel + BS + chalf * 48, vi);
      tmem_wait_ld();
      const long long row = r0 + r;
      const int h = (int)((row / p.Kw) % p.H);
      const bool kept = row < p.rows && ((h <= p.H / 2) ? h : p.H - h) < p.Kh;
      const float* bre = sBias + NT + chalf * 48;
      mlp_shrink48(vr, vi, bre, bre + BS, p.lambda, kept);
      // a thread holds one ROW (48 channels): the warp transposes through its private slice of the (now idle) operand
      // buffer and stores contiguous row segments (mlp_store_rows)
      mlp_store_rows<ST>(vr, vi, sA + (size_t)warp * (kMlpABytes / 8 / 16 * 16), X + ch0, r0 + q * 32, p.rows, p.C, chalf * 48, nch, lane);
    }
    ph ^= 1u;
    cp_async_wait_all();   // the next tile has landed in the staging buffer
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc<512>(tmem);
}

// ---- hidden factor > 1 (hid = hf * 96, blocks of 96 channels): SURVEY.md S8(f) item 2 -------------------------------
// P2 = sum over the hf hidden chunks of relu(X W1[:, chunk] + b1[chunk]) W2[chunk, :]: per tile the bf16 operand of X
// stays in shared memory, the chunk's weight images (74 KB, from L2) are reloaded per chunk, layer 2 accumulates over
// the chunks in tensor memory.  Simpler than tc_mlp_fwd (no staging buffer: the tile is converted straight from
// global memory); no BASELINE.json configuration uses hf > 1.
constexpr int kMlpMaxHf = 8;
constexpr uint32_t kMlpHfSmem = 4 * kWBytes + 2 * kMlpABytes;   // 172,800

// weight images per (block, chunk): {W1r, W1i}[in 96][out = chunk's 96 hidden], {W2r, W2i}[in = chunk's 96 hidden][out 96];
// biases per block: b1 [hf][re 96 | im 96], then b2 [re 96 | im 96]
__global__ void k_tc_prep_weights_hf(const float* __restrict__ w1, const float* __restrict__ b1, const float* __restrict__ w2,
                                     const float* __restrict__ b2, __nv_bfloat16* __restrict__ out, float* __restrict__ bout,
                                     int nb, int hf) {
  pdl_launch_dependents();   // the MLP kernel behind it sets itself up meanwhile; it waits (pdl_wait) before it reads the images
  const int hid = hf * BS;
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < nb * hid) {           // b1 is [nb][hid][2]
    const int j = idx / hid, o = idx - j * hid, hc = o / BS, oo = o - hc * BS;
    const float2 a = ((const float2*)b1)[idx];
    float* bb = bout + (size_t)j * (hf + 1) * NT + (size_t)hc * NT;
    bb[oo] = a.x;
    bb[BS + oo] = a.y;
  }
  if (idx < nb * BS) {            // b2 is [nb][96][2]
    const int j = idx / BS, o = idx - j * BS;
    const float2 b = ((const float2*)b2)[idx];
    float* bb = bout + (size_t)j * (hf + 1) * NT + (size_t)hf * NT;
    bb[o] = b.x;
    bb[BS + o] = b.y;
  }
  if (idx >= nb * hf * BS * BS) return;
  const int o = idx % BS, i = (idx / BS) % BS, hc = (idx / (BS * BS)) % hf, j = idx / (BS * BS * hf);
  const float2 a = ((const float2*)w1)[((size_t)j * BS + i) * hid + hc * BS + o];          // W1[j][i][hc*96 + o]
  const float2 b = ((const float2*)w2)[((size_t)j * hid + hc * BS + i) * BS + o];          // W2[j][hc*96 + i][o]
  __nv_bfloat16* base = out + ((size_t)j * hf + hc) * 4 * (kWBytes / 2);
  const uint32_t f = ((i / 8) * kWLbo + (o / 8) * kWSbo + (o % 8) * 16 + (i % 8) * 2) / 2; // n=o, k=i
  const uint32_t m = kWBytes / 2;
  base[0 * m + f] = __float2bfloat16_rn(a.x);
  base[1 * m + f] = __float2bfloat16_rn(a.y);
  base[2 * m + f] = __float2bfloat16_rn(b.x);
  base[3 * m + f] = __float2bfloat16_rn(b.y);
}

template <typename ST>
__global__ void __launch_bounds__(kMlpThreads, 1) tc_mlp_fwd_hf(const MlpParams p, int S, int hf) {
  extern __shared__ __align__(1024) uint8_t smem[];
  ST* const X = (ST*)p.X;
  __shared__ __align__(8) uint64_t done[2];
  __shared__ uint32_t tmem_slot;
  __shared__ __align__(16) float sBias[(kMlpMaxHf + 1) * NT];
  uint8_t* sW = smem;
  uint8_t* sAX = smem + 4 * kWBytes;
  uint8_t* sAO = sAX + kMlpABytes;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int j = blockIdx.x / S, s0 = blockIdx.x - j * S;
  const long long ntiles = (p.rows + kMlpRows - 1) / kMlpRows;
  const int ch0 = j * BS;
  pdl_launch_dependents();
  for (uint32_t i = tid; i < 2 * kMlpABytes / 16; i += kMlpThreads) ((uint4*)sAX)[i] = make_uint4(0, 0, 0, 0);
  if (tid == 0) {
    mbar_init(&done[0], 1);
    mbar_init(&done[1], 1);
    mbar_init_fence();
  }
  if (warp == 0) tmem_alloc<512>(&tmem_slot);
  pdl_wait();
  for (int i = tid; i < (hf + 1) * NT; i += kMlpThreads) sBias[i] = p.bprep[(size_t)j * (hf + 1) * NT + i];
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  const uint32_t aW = smem_u32(sW), aX = smem_u32(sAX), aO = smem_u32(sAO);
  const uint32_t D1 = tmem, D2 = tmem + NT;
  const int q = warp & 3, chalf = warp >> 2;
  const int r = q * 32 + lane;
  const uint32_t lane_sel = (uint32_t)(q * 32) << 16;
  uint32_t ph = 0;
  auto issue_layer = [&](uint32_t D, uint32_t aA, uint32_t wr, uint32_t wi, uint32_t acc0, uint64_t* bar) {
    const uint32_t id = idesc_bf16(128, BS, 0u);
#pragma unroll
    for (int ks = 0; ks < BS / 16; ++ks) {
      const uint64_t ad = smem_desc(aA + ks * 2 * kMlpALbo, kMlpALbo, kMlpASbo);
      mma_ss(D, ad, smem_desc(wr + ks * 2 * kWLbo, kWLbo, kWSbo), id, acc0 | (uint32_t)(ks != 0));
      mma_ss(D + BS, ad, smem_desc(wi + ks * 2 * kWLbo, kWLbo, kWSbo), id, acc0 | (uint32_t)(ks != 0));
    }
#pragma unroll
    for (int ks = 0; ks < BS / 16; ++ks) {
      const uint64_t ad = smem_desc(aA + (BS / 8 + ks * 2) * kMlpALbo, kMlpALbo, kMlpASbo);
      mma_ss(D, ad, smem_desc(wi + ks * 2 * kWLbo, kWLbo, kWSbo), id | kIdescNegB, 1u);
      mma_ss(D + BS, ad, smem_desc(wr + ks * 2 * kWLbo, kWLbo, kWSbo), id, 1u);
    }
    mma_commit(bar);
  };
  for (long long t = s0; t < ntiles; t += S) {
    const long long r0 = t * kMlpRows;
    // ---- spectrum rows -> bf16 A operand (lanes run over the 8-channel chunks of a row) ----
    mlp_load_operand<kMlpRows, kMlpALbo, ST>(X, r0, p.rows, p.C, ch0, BS, sAX, nullptr, tid);
    for (int hc = 0; hc < hf; ++hc) {
      // the chunk's weight images (the previous chunk's GEMMs have completed: done[1] was awaited)
      const uint8_t* wsrc = p.wprep + ((size_t)j * hf + hc) * 4 * kWBytes;
      for (uint32_t i = tid; i < 4 * kWBytes / 16; i += kMlpThreads) cp_async16(aW + i * 16, wsrc + (size_t)i * 16);
      cp_async_wait_all();
      fence_async_smem();
      tc_fence_before();
      __syncthreads();
      if (warp == 0 && elect_one()) {
        tc_fence_after();
        issue_layer(D1, aX, aW, aW + kWBytes, 0u, &done[0]);
      }
      __syncwarp();
      mbar_wait(&done[0], ph);
      tc_fence_after();
#pragma unroll
      for (int half = 0; half < 2; ++half) {
        uint32_t v[48];
        tmem_ld16<0>(D1 + lane_sel + half * BS + chalf * 48, v);
        tmem_ld16<16>(D1 + lane_sel + half * BS + chalf * 48 + 16, v);
        tmem_ld16<32>(D1 + lane_sel + half * BS + chalf * 48 + 32, v);
        tmem_wait_ld();
        const float* bias = sBias + (size_t)hc * NT + half * BS + chalf * 48;
        uint8_t* dst = sAO + (size_t)(r >> 3) * kMlpASbo + (r & 7) * 16 + (size_t)(half * (BS / 8) + chalf * 6) * kMlpALbo;
#pragma unroll
        for (int g = 0; g < 6; ++g) {
          uint32_t pk[4];
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const float lo = fmaxf(__uint_as_float(v[8 * g + 2 * e]) + bias[8 * g + 2 * e], 0.f);
            const float hi = fmaxf(__uint_as_float(v[8 * g + 2 * e + 1]) + bias[8 * g + 2 * e + 1], 0.f);
            pk[e] = pack_bf16(lo, hi);
          }
          *(uint4*)(dst + (size_t)g * kMlpALbo) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
        }
      }
      fence_async_smem();
      tc_fence_before();
      __syncthreads();
      if (warp == 0 && elect_one()) {
        tc_fence_after();
        issue_layer(D2, aO, aW + 2 * kWBytes, aW + 3 * kWBytes, hc > 0 ? 1u : 0u, &done[1]);
      }
      __syncwarp();
      mbar_wait(&done[1], ph);
      tc_fence_after();
      ph ^= 1u;
    }
    // ---- Z = softshrink(P2 + b2) on the fp32 sum, zero on truncated rows -> spectrum rows, in place ----
    {
      uint32_t vr[48], vi[48];
      mlp_ld48(D2 + lane_sel + chalf * 48, vr);
      mlp_ld48(D2 + lane_sel + BS + chalf * 48, vi);
      tmem_wait_ld();
      const long long row = r0 + r;
      const int h = (int)((row / p.Kw) % p.H);
      const bool kept = row < p.rows && ((h <= p.H / 2) ? h : p.H - h) < p.Kh;
      const float* bre = sBias + (size_t)hf * NT + chalf * 48;
      mlp_shrink48(vr, vi, bre, bre + BS, p.lambda, kept);
      // a thread holds one ROW (48 channels): the warp transposes through its private slice of the (now idle) operand
      // buffer and stores contiguous row segments (mlp_store_rows)
      mlp_store_rows<ST>(vr, vi, sAO + (size_t)warp * (kMlpABytes / 8 / 16 * 16), X + ch0, r0 + q * 32, p.rows, p.C, chalf * 48, BS, lane);
    }
    tc_fence_before();
    __syncthreads();   // every warp has read its accumulators and left the scratch area: next tile
    tc_fence_after();
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc<512>(tmem);
}

// ---- hybrid BACKWARD (rows B1 second half, B3-B7) on the tensor cores, hidden factor 1 ---------------------------------
// For grids the fused chain does not reach the backward call runs the transforms as fp32 FFTs (generic.cu) and this
// kernel in between: per tile of 96 spectrum rows x one group of 96 channels
//   X (fp32 spectrum of x) -> bf16 operand -> P1 = X W1 -> O1 = relu(P1 + b1), mask1 = (P1 + b1 > 0)
//   -> P2 = O1 W2 -> mask2 = (|P2 + b2| > lambda, kept row)                       [recompute, row B1]
//   G (fp32 alpha-weighted spectrum of dY) -> G2 = mask2 (.) G (bf16)              [B3]
//   -> G1 = mask1 (.) (G2 W2^H) -> GX = G1 W1^H -> fp32, in place over G           [B5, B7]
// The four bf16 operands X, O1, G2, G1 live in shared memory in the K-major layout of a 96-row A operand, which is
// byte for byte the operand-image format of tc_wgrad (tc_layout.cuh: chunk of 8 columns = 96 rows x 16 B + 16 B):
// each leaves with one bulk copy as soon as it is complete, and the parameter gradients (rows B4, B6) are then the
// SAME tc_wgrad + k_tc_wgrad_reduce launches the fused path uses, over tiles of 96 consecutive spectrum rows.
// Activation masks live as bit sets in registers (thread = row x 48 channels); mask2 crosses to the coalesced
// load mapping of G through a 3 KB shared-memory table.
constexpr uint32_t kMlpBwdSmem = 4 * kWBytes + 4 * kTileBytes + 512;   // 223,232 (+512: rows 96..127 of the last chunk alias past the buffer)

struct MlpBwdParams {
  const void* X;             // [rows][C] spectrum of x (the kernel's ST), read only
  void* G;                   // [rows][C] alpha-weighted spectrum of dY, replaced by GX
  const uint8_t* wprep;      // per group 4 x kWBytes: W1r, W1i, W2r, W2i
  const float* bprep;        // per group [2 layers][192]
  __nv_bfloat16 *Xh, *O1, *G2, *G1;   // operand images for tc_wgrad: [tile][group][kTileBytes]
  uint8_t *mask1, *mask2;    // optional export, [B][H][Wh][C][2]
  long long rows;
  int C, ngroups, H, Kw, Wh, Kh;
  float lambda;
};

template <typename ST>
__global__ void __launch_bounds__(kMlpThreads, 1) tc_mlp_bwd(const MlpBwdParams p, int S) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const ST* const X = (const ST*)p.X;
  ST* const G = (ST*)p.G;
  __shared__ __align__(8) uint64_t done;
  __shared__ uint32_t tmem_slot;
  __shared__ __align__(16) float sBias[2 * NT];
  __shared__ __align__(16) uint4 sMask2[HP][2];   // per row and 48-channel half: {re bits 0..31, re 32..47, im 0..31, im 32..47}
  uint8_t* sW = smem;
  uint8_t* bX = smem + 4 * kWBytes;
  uint8_t* bO = bX + kTileBytes;
  uint8_t* bG2 = bO + kTileBytes;
  uint8_t* bG1 = bG2 + kTileBytes;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int j = blockIdx.x / S, s0 = blockIdx.x - j * S;
  const long long ntiles = (p.rows + HP - 1) / HP;
  const int ch0 = j * BS;
  const int nch = min(BS, p.C - ch0);           // channels of the group that exist (a multiple of 8)
  pdl_launch_dependents();
  for (uint32_t i = tid; i < (4 * kTileBytes + 512) / 16; i += kMlpThreads) ((uint4*)bX)[i] = make_uint4(0, 0, 0, 0);
  if (tid == 0) {
    mbar_init(&done, 1);
    mbar_init_fence();
  }
  if (warp == 0) tmem_alloc<256>(&tmem_slot);
  pdl_wait();   // the spectra and the weight images are written by earlier kernels of the call
  {
    const uint8_t* wsrc = p.wprep + (size_t)j * 4 * kWBytes;
    for (uint32_t i = tid; i < 4 * kWBytes / 16; i += kMlpThreads) cp_async16(smem_u32(sW) + i * 16, wsrc + (size_t)i * 16);
  }
  for (int i = tid; i < 2 * NT; i += kMlpThreads) sBias[i] = p.bprep[(size_t)j * 2 * NT + i];
  cp_async_wait_all();
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t D = tmem_slot;   // (re 96 | im 96) fp32 accumulator
  const uint32_t aW = smem_u32(sW);
  const uint32_t w1r = aW, w1i = aW + kWBytes, w2r = aW + 2 * kWBytes, w2i = aW + 3 * kWBytes;
  const int q = warp & 3, chalf = warp >> 2;    // TMEM lane quarter (rows 32 q ..), 48-channel half of the group
  const int r = q * 32 + lane;                  // row of the tile (quarter 3 holds no rows: HP = 96)
  const bool epi = q < 3;
  const uint32_t acc = D + ((uint32_t)(q * 32) << 16) + chalf * 48;   // this thread's re columns; im at + BS
  const bool storer = tid == 3 * 32;            // lane 0 of an otherwise idle warp issues the image copies
  const uint64_t pol_img = l2_evict_normal();
  const size_t chunk_off = (size_t)chalf * 6 * kTileSbo, im_off = (size_t)(BS / 8) * kTileSbo;
  uint32_t ph = 0;
  // every thread has written its part of operand `buf`: hand it to the tensor core (and to the copy engine as an image)
  auto start_gemm = [&](const uint8_t* buf, uint32_t wr, uint32_t wi, bool transposed, __nv_bfloat16* img, size_t img_off) {
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    if (warp == 0 && elect_one()) {
      tc_fence_after();
      mlp_issue_gemm(D, smem_u32(buf), wr, wi, transposed, 0u, &done);
    }
    if (storer) bulk_store((uint8_t*)img + img_off, smem_u32(buf), kTileBytes, pol_img);
    __syncwarp();
  };
  auto finish_gemm = [&]() {
    mbar_wait(&done, ph);
    tc_fence_after();
    ph ^= 1u;
  };
  // bf16 spectrum: the next operand's rows travel global -> registers under the GEMM before it (G under layer 2 and
  // its epilogue, the next tile's X under GX and its store); fp32 spectrum: loaded where it is needed
  constexpr bool kPrefetch = std::is_same<ST, SpecBf16>::value;
  MlpFetch fx, fg;
  if constexpr (kPrefetch) {
    if (s0 < ntiles) mlp_fetch_operand((const SpecBf16*)X, s0 * HP, p.rows, p.C, ch0, nch, tid, fx);
  }
  for (long long t = s0; t < ntiles; t += S) {
    const long long r0 = t * HP;
    const size_t img_off = ((size_t)t * p.ngroups + j) * kTileBytes;
    const long long row = r0 + r;
    const int h = (int)((row / p.Kw) % p.H);
    const bool row_valid = epi && row < p.rows;
    const bool kept = row_valid && ((h <= p.H / 2) ? h : p.H - h) < p.Kh;
    uint64_t m1[2] = {0, 0}, m2[2] = {0, 0};   // [re, im] bits of this thread's 48 channels
    // ---- X -> bf16 operand; P1 = X W1 ----
    if constexpr (kPrefetch) mlp_commit_operand(fx, bX, nullptr, tid);
    else mlp_load_operand<HP, kTileSbo, ST>(X, r0, p.rows, p.C, ch0, nch, bX, nullptr, tid);
    start_gemm(bX, w1r, w1i, false, p.Xh, img_off);
    finish_gemm();
    // ---- O1 = relu(P1 + b1), mask1 ----
    if (epi) {
#pragma unroll
      for (int half = 0; half < 2; ++half) {
        uint32_t v[48];
        mlp_ld48(acc + half * BS, v);
        tmem_wait_ld();
        m1[half] = mlp_relu_store(v, sBias + half * BS + chalf * 48, bO + (size_t)r * 16 + half * im_off + chunk_off);
      }
    }
    start_gemm(bO, w2r, w2i, false, p.O1, img_off);
    if constexpr (kPrefetch) mlp_fetch_operand((const SpecBf16*)G, r0, p.rows, p.C, ch0, nch, tid, fg);
    finish_gemm();
    // ---- mask2 = (|P2 + b2| > lambda) on kept rows ----
    if (epi) {
#pragma unroll
      for (int half = 0; half < 2; ++half) {
        uint32_t v[48];
        mlp_ld48(acc + half * BS, v);
        tmem_wait_ld();
        m2[half] = mlp_shrink_mask(v, sBias + NT + half * BS + chalf * 48, p.lambda, kept);
      }
      sMask2[r][chalf] = make_uint4((uint32_t)m2[0], (uint32_t)(m2[0] >> 32), (uint32_t)m2[1], (uint32_t)(m2[1] >> 32));
    }
    if (storer) bulk_wait_read<1>();   // the Xh image has left bX (the scratch area of the last epilogue)
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    // ---- G2 = mask2 (.) G -> bf16 operand; G1pre = G2 W2^H ----
    if constexpr (kPrefetch) mlp_commit_operand(fg, bG2, sMask2, tid);
    else mlp_load_operand<HP, kTileSbo, ST>((const ST*)G, r0, p.rows, p.C, ch0, nch, bG2, sMask2, tid);
    start_gemm(bG2, w2r, w2i, true, p.G2, img_off);
    finish_gemm();
    // ---- G1 = mask1 (.) G1pre ----
    if (epi) {
#pragma unroll
      for (int half = 0; half < 2; ++half) {
        uint32_t v[48];
        mlp_ld48(acc + half * BS, v);
        tmem_wait_ld();
        mlp_masked_store(v, m1[half], bG1 + (size_t)r * 16 + half * im_off + chunk_off);
      }
    }
    start_gemm(bG1, w1r, w1i, true, p.G1, img_off);
    if constexpr (kPrefetch) {
      if (t + S < ntiles) mlp_fetch_operand((const SpecBf16*)X, (t + S) * HP, p.rows, p.C, ch0, nch, tid, fx);
    }
    finish_gemm();
    // ---- GX -> fp32 complex, in place over G ----
    if (epi) {
      uint32_t vr[48], vi[48];
      mlp_ld48(acc, vr);
      mlp_ld48(acc + BS, vi);
      tmem_wait_ld();
      mlp_store_rows<ST>(vr, vi, bX + (size_t)warp * (kTileBytes / 8 / 16 * 16), G + ch0, r0 + q * 32, p.rows, p.C, chalf * 48, nch, lane);
      if (p.mask1 != nullptr && row_valid) {
        // export for the mask-consistent parity tests: [B][H][Wh][C][2] bytes, this thread's 48 channels
        const long long bh = row / p.Kw;
        const int kw = (int)(row - bh * p.Kw);
        const size_t base = ((size_t)(bh * p.Wh + kw) * p.C + ch0 + chalf * 48) * 2;
        mlp_export_mask(p.mask1 + base, m1[0], m1[1], nch - chalf * 48);
        mlp_export_mask(p.mask2 + base, m2[0], m2[1], nch - chalf * 48);
      }
    }
    if (storer) bulk_wait_read<0>();   // every image of this tile has left its buffer
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
  }
  if (storer) bulk_wait<0>();
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc<256>(D);
}

// ---- hybrid backward, hidden factor 2..8 (blocks of 96): SURVEY.md S8(f) item 2 -----------------------------------------
// Two passes over the hf hidden chunks of 96 per tile of 96 spectrum rows, the chunk's weight images (74 KB) reloaded
// from L2 each time (as tc_mlp_fwd_hf does):
//   pass 1 (recompute): P1_c = X W1[:, c] -> O1_c = relu(P1_c + b1_c), mask1_c (bits kept in shared memory);
//                       P2 += O1_c W2[c, :] accumulated over the chunks in tensor memory -> mask2
//   pass 2 (gradient):  G2 = mask2 (.) G;  G1_c = mask1_c (.) (G2 W2[c, :]^H);  GX += G1_c W1[:, c]^H accumulated over
//                       the chunks in tensor memory -> fp32, in place over G
// Operand buffers: X, G2 (one each per tile) and ONE buffer shared by O1_c (pass 1) and G1_c (pass 2); all four kinds
// leave as tc_wgrad operand images (O1 and G1 per chunk), the parameter gradients are one tc_wgrad launch per chunk
// (layer 2: O1_c, G2 -> dW2[c rows]; layer 1: Xh, G1_c -> dW1[:, c columns]) and k_tc_wgrad_reduce_hf.
constexpr uint32_t kMlpBwdHfSmem = 4 * kWBytes + 3 * kTileBytes + 512 + kMlpMaxHf * HP * 2 * 16;   // 210,560

struct MlpBwdHfParams {
  const void* X;
  void* G;
  const uint8_t* wprep;      // per (block, chunk) 4 x kWBytes (k_tc_prep_weights_hf)
  const float* bprep;        // per block: b1 [hf][192], then b2 [192]
  __nv_bfloat16 *Xh, *G2;    // images [tile][block]
  __nv_bfloat16 *O1, *G1;    // images [chunk][tile][block]
  uint8_t *mask1, *mask2;    // optional export: mask1 [B][H][Wh][nb * hid][2], mask2 [B][H][Wh][C][2]
  long long rows, ntiles;
  int C, nb, H, Kw, Wh, Kh, hf;
  float lambda;
};

template <typename ST>
__global__ void __launch_bounds__(kMlpThreads, 1) tc_mlp_bwd_hf(const MlpBwdHfParams p, int S) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const ST* const X = (const ST*)p.X;
  ST* const G = (ST*)p.G;
  __shared__ __align__(8) uint64_t done;
  __shared__ uint32_t tmem_slot;
  __shared__ __align__(16) float sBias[(kMlpMaxHf + 1) * NT];
  __shared__ __align__(16) uint4 sMask2[HP][2];
  uint8_t* sW = smem;
  uint8_t* bX = smem + 4 * kWBytes;
  uint8_t* bG2 = bX + kTileBytes;
  uint8_t* bH = bG2 + kTileBytes;                       // O1_c in pass 1, G1_c in pass 2
  uint4* sMask1 = (uint4*)(bH + kTileBytes + 512);      // [chunk][row][48-channel half]
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int j = blockIdx.x / S, s0 = blockIdx.x - j * S;
  const int hf = p.hf, hid = hf * BS;
  const int ch0 = j * BS;
  pdl_launch_dependents();
  for (uint32_t i = tid; i < (3 * kTileBytes + 512) / 16; i += kMlpThreads) ((uint4*)bX)[i] = make_uint4(0, 0, 0, 0);
  if (tid == 0) {
    mbar_init(&done, 1);
    mbar_init_fence();
  }
  if (warp == 0) tmem_alloc<512>(&tmem_slot);
  pdl_wait();
  for (int i = tid; i < (hf + 1) * NT; i += kMlpThreads) sBias[i] = p.bprep[(size_t)j * (hf + 1) * NT + i];
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t D1 = tmem_slot, D2 = tmem_slot + NT;   // per-chunk accumulator, accumulator over the chunks
  const uint32_t aW = smem_u32(sW);
  const uint32_t wAr = aW, wAi = aW + kWBytes, wBr = aW + 2 * kWBytes, wBi = aW + 3 * kWBytes;   // W1 chunk, W2 chunk
  const int q = warp & 3, chalf = warp >> 2;
  const int r = q * 32 + lane;
  const bool epi = q < 3;
  const uint32_t lane_col = ((uint32_t)(q * 32) << 16) + chalf * 48;   // this thread's re columns of an accumulator; im at + BS
  const bool storer = tid == 3 * 32;
  const uint64_t pol_img = l2_evict_normal();
  const size_t chunk_off = (size_t)chalf * 6 * kTileSbo, im_off = (size_t)(BS / 8) * kTileSbo;
  uint32_t ph = 0;
  constexpr bool kPrefetch = std::is_same<ST, SpecBf16>::value;
  MlpFetch fq;
  const SpecBf16* fetch_src = nullptr;   // set before a run_gemm call: what to fetch under that GEMM
  long long fetch_r0 = 0;
  if constexpr (kPrefetch) {
    if (s0 < p.ntiles) mlp_fetch_operand((const SpecBf16*)X, s0 * HP, p.rows, p.C, ch0, BS, tid, fq);
  }
  // operand `buf` is complete: GEMM into D (and the image copy); returns when the GEMM has completed
  auto run_gemm = [&](uint32_t D, const uint8_t* buf, uint32_t wr, uint32_t wi, bool transposed, uint32_t acc0,
                      __nv_bfloat16* img, size_t img_off) {
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    if (warp == 0 && elect_one()) {
      tc_fence_after();
      mlp_issue_gemm(D, smem_u32(buf), wr, wi, transposed, acc0, &done);
    }
    if (storer && img != nullptr) bulk_store((uint8_t*)img + img_off, smem_u32(buf), kTileBytes, pol_img);
    __syncwarp();
    // bf16 spectrum: the next operand's rows travel global -> registers under this GEMM (G under the last layer-2 GEMM of
    // pass 1, the next tile's X under the last GEMM of pass 2)
    if constexpr (kPrefetch) {
      if (fetch_src != nullptr) mlp_fetch_operand(fetch_src, fetch_r0, p.rows, p.C, ch0, BS, tid, fq);
      fetch_src = nullptr;
    }
    mbar_wait(&done, ph);
    tc_fence_after();
    ph ^= 1u;
  };
  // the chunk's weight images; the GEMMs that read the previous chunk's have completed (run_gemm waits)
  auto load_weights = [&](int hc) {
    const uint8_t* wsrc = p.wprep + ((size_t)j * hf + hc) * 4 * kWBytes;
    for (uint32_t i = tid; i < 4 * kWBytes / 16; i += kMlpThreads) cp_async16(aW + i * 16, wsrc + (size_t)i * 16);
    cp_async_wait_all();
  };
  // the previous image copy has left the buffer the next epilogue overwrites
  auto buffers_free = [&]() {
    if (storer) bulk_wait_read<0>();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
  };
  const size_t chunk_imgs = (size_t)p.ntiles * p.nb * kTileBytes;   // bytes of one chunk's image tensor
  for (long long t = s0; t < p.ntiles; t += S) {
    const long long r0 = t * HP;
    const size_t img_off = ((size_t)t * p.nb + j) * kTileBytes;
    const long long row = r0 + r;
    const int h = (int)((row / p.Kw) % p.H);
    const bool row_valid = epi && row < p.rows;
    const bool kept = row_valid && ((h <= p.H / 2) ? h : p.H - h) < p.Kh;
    const long long bh = row / p.Kw;
    const int kw = (int)(row - bh * p.Kw);
    if constexpr (kPrefetch) mlp_commit_operand(fq, bX, nullptr, tid);
    else mlp_load_operand<HP, kTileSbo, ST>(X, r0, p.rows, p.C, ch0, BS, bX, nullptr, tid);
    // ---- pass 1 ----
    for (int hc = 0; hc < hf; ++hc) {
      load_weights(hc);
      run_gemm(D1, bX, wAr, wAi, false, 0u, hc == 0 ? p.Xh : nullptr, img_off);
      buffers_free();   // the previous chunk's O1 image has left bH
      if (epi) {
        uint64_t m1[2];
#pragma unroll
        for (int half = 0; half < 2; ++half) {
          uint32_t v[48];
          mlp_ld48(D1 + lane_col + half * BS, v);
          tmem_wait_ld();
          m1[half] = mlp_relu_store(v, sBias + (size_t)hc * NT + half * BS + chalf * 48, bH + (size_t)r * 16 + half * im_off + chunk_off);
        }
        sMask1[((size_t)hc * HP + r) * 2 + chalf] = make_uint4((uint32_t)m1[0], (uint32_t)(m1[0] >> 32), (uint32_t)m1[1], (uint32_t)(m1[1] >> 32));
        if (p.mask1 != nullptr && row_valid)
          mlp_export_mask(p.mask1 + ((size_t)(bh * p.Wh + kw) * ((size_t)p.nb * hid) + (size_t)j * hid + hc * BS + chalf * 48) * 2, m1[0],
                          m1[1], 48);
      }
      if (kPrefetch && hc == hf - 1) { fetch_src = (const SpecBf16*)G; fetch_r0 = r0; }
      run_gemm(D2, bH, wBr, wBi, false, hc > 0 ? 1u : 0u, p.O1, (size_t)hc * chunk_imgs + img_off);
    }
    // ---- mask2 = (|P2 + b2| > lambda) on kept rows ----
    if (epi) {
      uint64_t m2[2];
#pragma unroll
      for (int half = 0; half < 2; ++half) {
        uint32_t v[48];
        mlp_ld48(D2 + lane_col + half * BS, v);
        tmem_wait_ld();
        m2[half] = mlp_shrink_mask(v, sBias + (size_t)hf * NT + half * BS + chalf * 48, p.lambda, kept);
      }
      sMask2[r][chalf] = make_uint4((uint32_t)m2[0], (uint32_t)(m2[0] >> 32), (uint32_t)m2[1], (uint32_t)(m2[1] >> 32));
      if (p.mask2 != nullptr && row_valid)
        mlp_export_mask(p.mask2 + ((size_t)(bh * p.Wh + kw) * p.C + ch0 + chalf * 48) * 2, m2[0], m2[1], 48);
    }
    buffers_free();
    // ---- pass 2 ----
    if constexpr (kPrefetch) mlp_commit_operand(fq, bG2, sMask2, tid);
    else mlp_load_operand<HP, kTileSbo, ST>((const ST*)G, r0, p.rows, p.C, ch0, BS, bG2, sMask2, tid);
    for (int hc = 0; hc < hf; ++hc) {
      load_weights(hc);
      run_gemm(D1, bG2, wBr, wBi, true, 0u, hc == 0 ? p.G2 : nullptr, img_off);   // G2 W2[c, :]^H
      buffers_free();
      if (epi) {
        const uint4 mk = sMask1[((size_t)hc * HP + r) * 2 + chalf];
        const uint64_t m1[2] = {((uint64_t)mk.y << 32) | mk.x, ((uint64_t)mk.w << 32) | mk.z};
#pragma unroll
        for (int half = 0; half < 2; ++half) {
          uint32_t v[48];
          mlp_ld48(D1 + lane_col + half * BS, v);
          tmem_wait_ld();
          mlp_masked_store(v, m1[half], bH + (size_t)r * 16 + half * im_off + chunk_off);
        }
      }
      if (kPrefetch && hc == hf - 1 && t + S < p.ntiles) { fetch_src = (const SpecBf16*)X; fetch_r0 = (t + S) * HP; }
      run_gemm(D2, bH, wAr, wAi, true, hc > 0 ? 1u : 0u, p.G1, (size_t)hc * chunk_imgs + img_off);   // GX += G1_c W1[:, c]^H
    }
    buffers_free();   // bX is the scratch area of the store below
    // ---- GX -> fp32 complex, in place over G ----
    if (epi) {
      uint32_t vr[48], vi[48];
      mlp_ld48(D2 + lane_col, vr);
      mlp_ld48(D2 + lane_col + BS, vi);
      tmem_wait_ld();
      mlp_store_rows<ST>(vr, vi, bX + (size_t)warp * (kTileBytes / 8 / 16 * 16), G + ch0, r0 + q * 32, p.rows, p.C, chalf * 48, BS, lane);
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
  }
  if (storer) bulk_wait<0>();
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc<512>(D1);
}

// dW1[j][i][c*96 + o], db1[j][c*96 + o] from chunk c's layer-1 partial sums; dW2[j][c*96 + i][o] from its layer-2 partial
// sums, db2[j][o] from chunk 0's (sum of G2 rows, the same for every chunk).  part: [chunk][layer 2 | layer 1][block][S].
__global__ void k_tc_wgrad_reduce_hf(const float* __restrict__ part, float2* __restrict__ dW2, float2* __restrict__ dB2,
                                     float2* __restrict__ dW1, float2* __restrict__ dB1, int nb, int S, int hf, int accumulate) {
  pdl_launch_dependents();
  pdl_wait();
  const int hid = hf * BS;
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  const int layer = blockIdx.y;                 // 0: layer 2, 1: layer 1 (the order of tc_wgrad's CTAs)
  const int nW = nb * hf * BS * BS;
  const size_t chunk_part = (size_t)2 * nb * S * kWgPartFloats;
  if (idx < nW) {
    const int o = idx % BS, i = (idx / BS) % BS, hc = (idx / (BS * BS)) % hf, j = idx / (BS * BS * hf);
    const float* P0 = part + (size_t)hc * chunk_part + (size_t)layer * nb * S * kWgPartFloats + (size_t)j * S * kWgPartFloats;
    float2 acc = make_float2(0.f, 0.f);
    for (int s = 0; s < S; ++s) {
      const float* Pre = P0 + (size_t)s * kWgPartFloats + (size_t)i * kWgPitch;
      const float* Pim = P0 + (size_t)s * kWgPartFloats + (size_t)(kWgRowsRe + i) * kWgPitch;
      acc.x += Pre[o] + Pim[BS + o];
      acc.y += Pre[BS + o] - Pim[o];
    }
    float2* dst = layer ? dW1 + ((size_t)j * BS + i) * hid + hc * BS + o       // W1[j][i][c*96 + o]
                        : dW2 + ((size_t)j * hid + hc * BS + i) * BS + o;      // W2[j][c*96 + i][o]
    if (accumulate) { acc.x += dst->x; acc.y += dst->y; }
    *dst = acc;
  } else if (idx < nW + nb * hid) {
    const int k = idx - nW, o = k % BS, hc = (k / BS) % hf, j = k / hid;
    if (layer == 0 && hc != 0) return;          // db2 comes from chunk 0 only
    const float* P0 = part + (size_t)hc * chunk_part + (size_t)layer * nb * S * kWgPartFloats + (size_t)j * S * kWgPartFloats +
                      (size_t)BS * kWgPitch;
    float2 acc = make_float2(0.f, 0.f);
    for (int s = 0; s < S; ++s) {
      acc.x += P0[(size_t)s * kWgPartFloats + o];
      acc.y += P0[(size_t)s * kWgPartFloats + BS + o];
    }
    float2* dst = layer ? dB1 + (size_t)j * hid + hc * BS + o : dB2 + (size_t)j * BS + o;
    if (accumulate) { acc.x += dst->x; acc.y += dst->y; }
    *dst = acc;
  }
}

// ---- hybrid forward, bf16 spectrum, hidden factor 1: software-pipelined over two tiles ------------------------------------
// tc_mlp_fwd runs load | GEMM | epilogue | GEMM | epilogue + store in sequence; both GEMM latencies are exposed.  With a
// bf16 spectrum the staging buffer is 48 KB, which leaves room for TWO operand buffers, and two accumulators fit
// tensor memory (2 x 192 columns): layer 2 of tile t runs under the conversion of tile t + 1, layer 1 of tile t + 1
// under the softshrink epilogue and store of tile t.  Same arithmetic and layouts as tc_mlp_fwd.
constexpr uint32_t kMlpPipeSmem = 4 * kWBytes + 2 * kMlpABytes + kMlpRows * BS * 4;   // 221,952

__global__ void __launch_bounds__(kMlpThreads, 1) tc_mlp_fwd_pipe(const MlpParams p, int S) {
  typedef SpecBf16 ST;
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ __align__(8) uint64_t done[2];
  __shared__ uint32_t tmem_slot;
  __shared__ __align__(16) float sBias[2 * NT];
  ST* const X = (ST*)p.X;
  uint8_t* sW = smem;
  uint8_t* sA0 = smem + 4 * kWBytes;
  uint8_t* sStage = sA0 + 2 * kMlpABytes;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int j = blockIdx.x / S, s0 = blockIdx.x - j * S;
  const long long ntiles = (p.rows + kMlpRows - 1) / kMlpRows;
  const int ch0 = j * BS;
  const int nch = min(BS, p.C - ch0);
  pdl_launch_dependents();
  for (uint32_t i = tid; i < 2 * kMlpABytes / 16; i += kMlpThreads) ((uint4*)sA0)[i] = make_uint4(0, 0, 0, 0);
  if (tid == 0) {
    mbar_init(&done[0], 1);
    mbar_init(&done[1], 1);
    mbar_init_fence();
  }
  if (warp == 0) tmem_alloc<512>(&tmem_slot);
  pdl_wait();
  {
    const uint8_t* wsrc = p.wprep + (size_t)j * 4 * kWBytes;
    for (uint32_t i = tid; i < 4 * kWBytes / 16; i += kMlpThreads) cp_async16(smem_u32(sW) + i * 16, wsrc + (size_t)i * 16);
  }
  for (int i = tid; i < 2 * NT; i += kMlpThreads) sBias[i] = p.bprep[(size_t)j * 2 * NT + i];
  // staging loads of one tile: 16-byte pieces (4 channels); pieces past the last row or channel are zero-filled
  auto stage_tile = [&](long long t) {
    const long long r0 = t * kMlpRows;
    for (uint32_t i = tid; i < kMlpRows * BS * 4 / 16; i += kMlpThreads) {
      const int rr = i / (BS / 4), c4 = i - rr * (BS / 4);
      const bool ok = (r0 + rr < p.rows) && (4 * c4 < nch);
      const ST* src = X + (size_t)(ok ? r0 + rr : 0) * p.C + ch0 + (ok ? 4 * c4 : 0);
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_u32(sStage) + i * 16), "l"(src), "r"(ok ? 16 : 0) : "memory");
    }
  };
  // staging -> bf16 K-major operand buffer: unit = (row, 8 channels)
  auto convert = [&](uint8_t* sA) {
    for (uint32_t u = tid; u < kMlpRows * (BS / 8); u += kMlpThreads) {
      const int rr = u / (BS / 8), c8 = u - rr * (BS / 8);
      uint4 re, im;
      mlp_pack8<ST>((const ST*)sStage + (size_t)rr * BS + 8 * c8, re, im);
      uint8_t* dst = sA + (size_t)rr * 16;
      *(uint4*)(dst + (size_t)c8 * kMlpALbo) = re;
      *(uint4*)(dst + (size_t)(BS / 8 + c8) * kMlpALbo) = im;
    }
  };
  if (s0 < ntiles) stage_tile(s0);
  cp_async_wait_all();
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  const uint32_t aW = smem_u32(sW);
  const uint32_t w1r = aW, w1i = aW + kWBytes, w2r = aW + 2 * kWBytes, w2i = aW + 3 * kWBytes;
  const int q = warp & 3, chalf = warp >> 2;
  const int r = q * 32 + lane;
  const uint32_t lane_sel = (uint32_t)(q * 32) << 16;
  uint32_t ph[2] = {0, 0};
  auto issue_layer = [&](uint32_t D, uint32_t aA, uint32_t wr, uint32_t wi, uint64_t* bar) {
    const uint32_t id = idesc_bf16(128, BS, 0u);
#pragma unroll
    for (int ks = 0; ks < BS / 16; ++ks) {
      const uint64_t ad = smem_desc(aA + ks * 2 * kMlpALbo, kMlpALbo, kMlpASbo);
      mma_ss(D, ad, smem_desc(wr + ks * 2 * kWLbo, kWLbo, kWSbo), id, ks != 0);
      mma_ss(D + BS, ad, smem_desc(wi + ks * 2 * kWLbo, kWLbo, kWSbo), id, ks != 0);
    }
#pragma unroll
    for (int ks = 0; ks < BS / 16; ++ks) {
      const uint64_t ad = smem_desc(aA + (BS / 8 + ks * 2) * kMlpALbo, kMlpALbo, kMlpASbo);
      mma_ss(D, ad, smem_desc(wi + ks * 2 * kWLbo, kWLbo, kWSbo), id | kIdescNegB, 1u);
      mma_ss(D + BS, ad, smem_desc(wr + ks * 2 * kWLbo, kWLbo, kWSbo), id, 1u);
    }
    mma_commit(bar);
  };
  // prime the pipeline: tile s0 -> buffer 0, layer 1 issued
  if (s0 < ntiles) {
    convert(sA0);
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    if (s0 + S < ntiles) stage_tile(s0 + S);
    if (warp == 0 && elect_one()) {
      tc_fence_after();
      issue_layer(tmem, smem_u32(sA0), w1r, w1i, &done[0]);
    }
    __syncwarp();
  }
  int cur = 0;
  for (long long t = s0; t < ntiles; t += S, cur ^= 1) {
    const long long r0 = t * kMlpRows;
    const int nxt = cur ^ 1;
    uint8_t* sA = sA0 + (size_t)cur * kMlpABytes;
    uint8_t* sAn = sA0 + (size_t)nxt * kMlpABytes;
    const uint32_t D = tmem + (uint32_t)cur * NT, Dn = tmem + (uint32_t)nxt * NT;
    const bool has_next = t + S < ntiles;
    // ---- layer 1 of this tile has been issued: O1 = relu(P1 + b1) -> operand of layer 2, over X ----
    mbar_wait(&done[cur], ph[cur]);
    ph[cur] ^= 1u;
    tc_fence_after();
#pragma unroll
    for (int half = 0; half < 2; ++half) {
      uint32_t v[48];
      mlp_ld48(D + lane_sel + half * BS + chalf * 48, v);
      tmem_wait_ld();
      const float* bias = sBias + half * BS + chalf * 48;
      uint8_t* dst = sA + (size_t)r * 16 + (size_t)(half * (BS / 8) + chalf * 6) * kMlpALbo;
#pragma unroll
      for (int g = 0; g < 6; ++g) {
        uint32_t pk[4];
#pragma unroll
        for (int e = 0; e < 4; ++e)
          pk[e] = pack_relu_bf16(__uint_as_float(v[8 * g + 2 * e]) + bias[8 * g + 2 * e], __uint_as_float(v[8 * g + 2 * e + 1]) + bias[8 * g + 2 * e + 1]);
        *(uint4*)(dst + (size_t)g * kMlpALbo) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
      }
    }
    cp_async_wait_all();   // (the next tile, requested an iteration ago, has landed in the staging buffer)
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    if (warp == 0 && elect_one()) {
      tc_fence_after();
      issue_layer(D, smem_u32(sA), w2r, w2i, &done[cur]);
    }
    __syncwarp();
    // ---- under layer 2: the next tile staging -> other buffer, its layer 1 queued behind ----
    if (has_next) {
      convert(sAn);
      fence_async_smem();
      tc_fence_before();
      __syncthreads();
      if (t + 2LL * S < ntiles) stage_tile(t + 2LL * S);
      if (warp == 0 && elect_one()) {
        tc_fence_after();
        issue_layer(Dn, smem_u32(sAn), w1r, w1i, &done[nxt]);
      }
      __syncwarp();
    }
    // ---- Z = softshrink(P2 + b2), zero on truncated rows -> spectrum rows, in place (under the next tile's layer 1) ----
    mbar_wait(&done[cur], ph[cur]);
    ph[cur] ^= 1u;
    tc_fence_after();
    {
      uint32_t vr[48], vi[48];
      mlp_ld48(D + lane_sel + chalf * 48, vr);
      mlp_ld48(D + lane_sel + BS + chalf * 48, vi);
      tmem_wait_ld();
      const long long row = r0 + r;
      const int h = (int)((row / p.Kw) % p.H);
      const bool kept = row < p.rows && ((h <= p.H / 2) ? h : p.H - h) < p.Kh;
      const float* bre = sBias + NT + chalf * 48;
      mlp_shrink48(vr, vi, bre, bre + BS, p.lambda, kept);
      mlp_store_rows<ST>(vr, vi, sA + (size_t)warp * (kMlpABytes / 8 / 16 * 16), X + ch0, r0 + q * 32, p.rows, p.C, chalf * 48, nch, lane);
    }
    tc_fence_before();
    __syncthreads();   // buffer `cur` (scratch) and its accumulator are free for the tile after next
    tc_fence_after();
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc<512>(tmem);
}
