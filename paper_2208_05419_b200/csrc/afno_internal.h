// Internal declarations shared by the translation units of libafno_b200.so.
// Nothing here is part of the C ABI (include/afno.h) and nothing here is shared with oracle/.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/afno.h"

namespace afno {

constexpr int kMaxStages = 16;

// One 1-D FFT plan: in-place decimation-in-frequency, output bin k lands at perm[k].
struct FftPlan {
  int n;
  int nstages;
  int radix[kMaxStages];
  const float2* tw;    // device: tw[k] = exp(-2 pi i k / n), rounded from fp64
  const int16_t* perm; // device: position of output bin k after the last stage
};

// Resolved problem geometry (host side), derived once per call from afno_desc_t.
struct Geometry {
  int B, H, W, C, nb, bs, hid, CH; // CH = nb * hid
  int Wh, Kh, Kw;
  // tcgen05 path only (tc_path.cu): the kernels work on GROUPS of 96 channels; with blocks narrower than 96
  // (bs divides 96) a group holds 96 / bs blocks and nb / bs above describe the groups, nb_blocks / bs_block
  // the caller's blocks
  int nb_blocks = 0, bs_block = 0;
  float lambda;
  float scale; // 1/sqrt(H*W)
  bool bf16, no_residual, accum, export_masks, force_fp32, save_ctx, use_ctx;
  long long modes_all() const { return (long long)B * H * Wh; }
  long long rows() const { return (long long)B * H * Kw; } // rows of the stored spectra
};

// constant operand images of the tcgen05 path (device pointers, shared-memory layout order)
struct TcPlan {
  bool valid = false;
  int num_sms = 148;
  uint8_t* dft2 = nullptr;
  uint8_t *fw = nullptr, *fw_alpha = nullptr, *gw = nullptr, *gw_noalpha = nullptr;
  void* encode_tiled = nullptr; // cuTensorMapEncodeTiled, resolved through the runtime (no link to libcuda)
};

struct Plan {
  int device, H, W;
  FftPlan fh, fw;
  TcPlan tc;
};

// launch accounting (thread-local, reported through afno_last_launch_count) and the optional
// per-kernel CUDA-event profiler behind afno_profile_start / afno_profile_stop
void count_launch(int n = 1);
void prof_begin(const char* kernel_name, cudaStream_t st);
void prof_end(cudaStream_t st);

// ---- generic fp32-math path (generic.cu) -------------------------------------------
size_t generic_workspace_bytes(const Geometry& g, bool backward);
cudaError_t generic_forward(const Geometry& g, const Plan& p, const void* x, const float* w1,
                            const float* b1, const float* w2, const float* b2, void* y,
                            void* ws, cudaStream_t st);
cudaError_t generic_backward(const Geometry& g, const Plan& p, const void* x, const void* dy,
                             const float* w1, const float* b1, const float* w2, const float* b2,
                             void* dx, float* dw1, float* db1, float* dw2, float* db2, void* ws,
                             size_t mask1_bytes, size_t mask2_offset, cudaStream_t st);
bool generic_supported(const Geometry& g, const char** why);

// ---- tcgen05 bf16 path (tc_path.cu) --------------------------------------------------
bool tc_supported(const Geometry& g);
bool tc_plan_supported(int H, int W);   // grid sizes the constant operand images can be built for
void tc_free_plan(TcPlan* p);
cudaError_t tc_build_plan(int H, int W, TcPlan* out);
size_t tc_workspace_bytes(const Geometry& g, bool backward);
cudaError_t tc_forward(const Geometry& g, const Plan& p, const void* x, const float* w1, const float* b1,
                       const float* w2, const float* b2, void* y, void* ws, cudaStream_t st);

cudaError_t tc_backward(const Geometry& g, const Plan& p, const void* x, const void* dy, const float* w1,
                        const float* b1, const float* w2, const float* b2, void* dx, float* dw1, float* db1,
                        float* dw2, float* db2, void* ws, cudaStream_t st);

// hybrid path (bf16 activations on grids beyond the fused chain): generic fp32 FFTs + tensor-core block MLP, forward
bool tc_mlp_supported(const Geometry& g);
size_t tc_mlp_workspace_bytes(const Geometry& g);
// X (and G below): the spectrum in the generic path's [row][C] layout, fp32 complex or (spec16) bf16 complex
cudaError_t tc_mlp_forward(const Geometry& g, void* X, bool spec16, const float* w1, const float* b1, const float* w2,
                           const float* b2, void* ws, cudaStream_t st);

// hybrid backward, hidden factors 1..8 (blocks of 96 for hf > 1; tc_mlp_backward dispatches hf > 1 to tc_mlp_backward_hf):
// block MLP gradient stages and parameter gradients on the tensor cores
bool tc_mlp_bwd_supported(const Geometry& g);
size_t tc_mlp_bwd_workspace_bytes(const Geometry& g);
cudaError_t tc_mlp_backward(const Geometry& g, const void* X, void* G, bool spec16, const float* w1, const float* b1,
                            const float* w2, const float* b2, float* dw1, float* db1, float* dw2, float* db2, uint8_t* mask1,
                            uint8_t* mask2, void* ws, cudaStream_t st);

// afno_block_wgrad_static (generic.cu): rows B4 / B6 on caller-supplied operands, the split partial sums kept in the
// library's static device array instead of a workspace.  wgrad_static_split_bytes: bytes one split occupies there.
constexpr size_t kStaticScratchBytes = AFNO_STATIC_SCRATCH_BYTES;
size_t wgrad_static_split_bytes(int nb, int K, int N);
cudaError_t generic_wgrad_static(const float2* A, int lda, const float2* G, int ldg, long long M, int nb, int K, int N,
                                 float* dW, float* dB, bool accum, cudaStream_t st);

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

#ifdef __CUDACC__
// Storage type of the half-spectra between the kernels of the generic / hybrid paths: fp32 complex (float2) or, on the
// hybrid path when every transform runs through the two-pass kernels, bf16 complex (SpecBf16: re in the low half).
// The arithmetic is fp32 either way; pairs = two adjacent channels.
struct SpecBf16 { uint32_t v; };
template <typename ST> struct SpecIO;
template <> struct SpecIO<float2> {
  typedef float4 pair_t;
  static __device__ __forceinline__ pair_t ldpair(const float2* p) { return __ldg((const float4*)p); }
  static __device__ __forceinline__ void unpair(pair_t v, float2& a, float2& b) { a = make_float2(v.x, v.y); b = make_float2(v.z, v.w); }
  static __device__ __forceinline__ void stpair(float2* p, float2 a, float2 b) { *(float4*)p = make_float4(a.x, a.y, b.x, b.y); }
  static __device__ __forceinline__ float2 ld(const float2* p) { return *p; }
  static __device__ __forceinline__ void st(float2* p, float2 v) { *p = v; }
};
template <> struct SpecIO<SpecBf16> {
  typedef uint2 pair_t;
  static __device__ __forceinline__ float2 up(uint32_t u) { return make_float2(__uint_as_float(u << 16), __uint_as_float(u & 0xFFFF0000u)); }
  static __device__ __forceinline__ uint32_t down(float2 v) {
    __nv_bfloat162 t = __floats2bfloat162_rn(v.x, v.y);
    return *reinterpret_cast<uint32_t*>(&t);
  }
  static __device__ __forceinline__ pair_t ldpair(const SpecBf16* p) { return __ldg((const uint2*)p); }
  static __device__ __forceinline__ void unpair(pair_t v, float2& a, float2& b) { a = up(v.x); b = up(v.y); }
  static __device__ __forceinline__ void stpair(SpecBf16* p, float2 a, float2 b) { *(uint2*)p = make_uint2(down(a), down(b)); }
  static __device__ __forceinline__ float2 ld(const SpecBf16* p) { return up(p->v); }
  static __device__ __forceinline__ void st(SpecBf16* p, float2 v) { p->v = down(v); }
};
#endif

} // namespace afno
