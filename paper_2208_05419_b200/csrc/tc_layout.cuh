// Part of the tcgen05 path (tc_path.cu includes the parts in order, inside namespace afno { namespace { ):
// sizes and operand geometry, measurement macros, L2 policy choice, weight-image kernel.
// Not a standalone header: it relies on tc_common.cuh and on the parts included before it.
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
// Context header (AFNO_FLAG_SAVE_CONTEXT -> AFNO_FLAG_USE_CONTEXT): the forward call records what it saved,
// the backward call's guard kernel compares and poisons dx and the gradients with NaN on a mismatch.
struct CtxHeader {
  uint32_t magic;
  int32_t B, H, W, C, nb, Kh, Kw, chunk_b;
  uint32_t lambda_bits, export_masks;
  uint32_t pad[5];
};
constexpr uint32_t kCtxMagic = 0xAF90C7E5u;

// ---- weight preparation: fp32 [nb][bs][bs][2] -> bf16 K-major interleaved operands --------------
// per GROUP of 96 channels 4 matrices of kWBytes {W1r, W1i, W2r, W2i} with element (n=o, k=i) = W[i][o] (the
// backward pass reads the same images as MN-major operands): the blocks of the group sit on the diagonal,
// everything else (other blocks, channels past C in a partly filled last group) is zero.  The biases are
// regrouped as [group][layer][re 96 | im 96] fp32.
__global__ void k_tc_prep_weights(const float* __restrict__ w1, const float* __restrict__ b1,
                                  const float* __restrict__ w2, const float* __restrict__ b2,
                                  __nv_bfloat16* __restrict__ out, float* __restrict__ bout, int ngroups, int bs, int C,
                                  const CtxHeader hdr, CtxHeader* __restrict__ hdr_out) {
  pdl_launch_dependents();
  pdl_wait();
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx == 0 && hdr_out != nullptr) *hdr_out = hdr;   // SAVE_CONTEXT: what this call leaves in the workspace
  if (idx < ngroups * BS) {
    const int o = idx % BS, j = idx / BS;
    float2 a = make_float2(0.f, 0.f), b = make_float2(0.f, 0.f);
    if (idx < C) {   // biases are [C][2] whatever the block size
      a = ((const float2*)b1)[idx];
      b = ((const float2*)b2)[idx];
    }
    float* bb = bout + (size_t)j * 2 * NT;
    bb[o] = a.x;
    bb[BS + o] = a.y;
    bb[NT + o] = b.x;
    bb[NT + BS + o] = b.y;
  }
  if (idx >= ngroups * BS * BS) return;
  const int o = idx % BS, i = (idx / BS) % BS, j = idx / (BS * BS);
  const int ci = j * BS + i, co = j * BS + o;        // channels
  float2 a = make_float2(0.f, 0.f), b = make_float2(0.f, 0.f);
  if (ci < C && co < C && ci / bs == co / bs) {
    const size_t src = ((size_t)(ci / bs) * bs + ci % bs) * bs + co % bs;
    a = ((const float2*)w1)[src];
    b = ((const float2*)w2)[src];
  }
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

// L2 eviction policy of every bulk-copy site (2 bits each: 0 evict_normal, 1 evict_first, 2 evict_last).
// The chunk buffers (half-spectrum A, gradient images G2 / G1) are rewritten by every chunk and should
// never leave the L2; everything else streams through once.
enum PolSite {
  kPolWfLoadX = 0,     // tc_wdft_fwd2: activation loads (x, dy)
  kPolWfStoreA = 1,    // tc_wdft_fwd2: half-spectrum stores
  kPolWiLoadA = 2,     // tc_wdft_inv2: half-spectrum loads
  kPolWiLoadRes = 3,   // tc_wdft_inv2: residual loads (x, dy)
  kPolWiStoreY = 4,    // tc_wdft_inv2: output stores (y, dx)
  kPolMixLoadA = 5,    // tc_mix2: tile loads
  kPolMixStoreA = 6,   // tc_mix2: tile stores (in place)
  kPolMixStoreCtx = 7, // tc_mix2<FwdSave>: Xh, O1 stores (read a whole pass later)
  kPolMixStoreG = 8,   // tc_mix2<Bwd*>: G2, G1 (and Xh, O1 of the stateless backward) stores, read by the next kernel
  kPolWgLoadCtx = 9,   // tc_wgrad: Xh, O1 loads
  kPolWgLoadG = 10     // tc_wgrad: G2, G1 loads
};
// Chosen by a measured sweep on the headline step (B = 4 fwd+bwd, whole-batch chunks): all evict_normal 0.469 ms,
// the round-1 choice (A stores evict_last, wgrad loads evict_first) 0.456, this table 0.453: half-spectrum and
// G2 / G1 stores evict_last (the next kernel reads them), their loads evict_first (read exactly once), the
// activations and the saved context left at evict_normal (evict_first on them costs 3 %).
#ifndef AFNO_POLICIES
#define AFNO_POLICIES ((0u << 0) | (2u << 2) | (1u << 4) | (0u << 6) | (0u << 8) | (1u << 10) | (2u << 12) | (0u << 14) | (2u << 16) | (1u << 18) | (1u << 20))
#endif
__device__ __forceinline__ uint64_t pol(PolSite site) {
  const uint32_t v = ((uint32_t)(AFNO_POLICIES) >> (2 * (int)site)) & 3u;
  return v == 1 ? l2_evict_first() : v == 2 ? l2_evict_last() : l2_evict_normal();
}
