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
