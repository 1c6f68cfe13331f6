// C ABI of libafno_b200.so (include/afno.h): descriptor validation, plan cache, dispatch.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <mutex>
#include <string>
#include <vector>

#include "afno_internal.h"

namespace afno {

namespace {

thread_local std::string t_error;
thread_local int t_launches = 0;

int fail(int status, const std::string& msg) {
  t_error = msg;
  return status;
}

bool smooth235(int n, std::vector<int>* radices) {
  if (n < 1) return false;
  std::vector<int> r;
  while (n % 4 == 0) { r.push_back(4); n /= 4; }
  while (n % 2 == 0) { r.push_back(2); n /= 2; }
  while (n % 3 == 0) { r.push_back(3); n /= 3; }
  while (n % 5 == 0) { r.push_back(5); n /= 5; }
  if (n != 1) return false;
  if (radices) *radices = r;
  return true;
}

// Validates d and fills g.  Returns AFNO_OK or an error status (message set).
int resolve(const afno_desc_t* d, Geometry* g) {
  if (!d) return fail(AFNO_ERR_INVALID_ARG, "descriptor is NULL");
  if (d->B <= 0 || d->H <= 0 || d->W <= 0 || d->C <= 0)
    return fail(AFNO_ERR_INVALID_ARG, "B, H, W, C must be positive");
  if (d->num_blocks <= 0 || d->C % d->num_blocks != 0)
    return fail(AFNO_ERR_INVALID_ARG, "num_blocks must be positive and divide C");
  if (d->hidden_factor < 1) return fail(AFNO_ERR_INVALID_ARG, "hidden_factor must be >= 1");
  if (!(d->lambda >= 0.f) || isinf(d->lambda)) return fail(AFNO_ERR_INVALID_ARG, "lambda must be finite and >= 0");
  if (!(d->kept_fraction > 0.f && d->kept_fraction <= 1.f))
    return fail(AFNO_ERR_INVALID_ARG, "kept_fraction must be in (0, 1]");
  if (d->dtype != AFNO_F32 && d->dtype != AFNO_BF16) return fail(AFNO_ERR_INVALID_ARG, "unknown dtype");
  if (d->flags & ~(uint32_t)(AFNO_FLAG_NO_RESIDUAL | AFNO_FLAG_ACCUM_GRADS | AFNO_FLAG_FORCE_FP32_MATH |
                             AFNO_FLAG_EXPORT_MASKS | AFNO_FLAG_SAVE_CONTEXT | AFNO_FLAG_USE_CONTEXT))
    return fail(AFNO_ERR_INVALID_ARG, "unknown flag bits");
  if ((d->flags & AFNO_FLAG_SAVE_CONTEXT) && (d->flags & AFNO_FLAG_USE_CONTEXT))
    return fail(AFNO_ERR_INVALID_ARG, "AFNO_FLAG_SAVE_CONTEXT (forward) and AFNO_FLAG_USE_CONTEXT (backward) exclude each other");
  if ((long long)d->B * d->H * d->W >= (1LL << 31) / 4)
    return fail(AFNO_ERR_UNSUPPORTED, "B*H*W too large for 32-bit token indexing");
  if (d->W % 2 != 0) return fail(AFNO_ERR_UNSUPPORTED, "odd W is not supported on the GPU path");
  if (!smooth235(d->H, nullptr) || !smooth235(d->W, nullptr))
    return fail(AFNO_ERR_UNSUPPORTED, "H and W must have no prime factor larger than 5");
  g->B = d->B; g->H = d->H; g->W = d->W; g->C = d->C;
  g->nb = d->num_blocks;
  g->bs = d->C / d->num_blocks;
  g->hid = g->bs * d->hidden_factor;
  g->CH = g->nb * g->hid;
  g->Wh = d->W / 2 + 1;
  // readings A7/A8: box of low |wavenumber|, floor, clamped to >= 1; product in double
  const double f = (double)d->kept_fraction;
  const int nh = d->H / 2 + 1;
  int kh = (int)floor(f * (double)nh), kw = (int)floor(f * (double)g->Wh);
  g->Kh = kh < 1 ? 1 : (kh > nh ? nh : kh);
  g->Kw = kw < 1 ? 1 : (kw > g->Wh ? g->Wh : kw);
  g->lambda = d->lambda;
  g->scale = (float)(1.0 / sqrt((double)d->H * (double)d->W));
  g->bf16 = d->dtype == AFNO_BF16;
  g->no_residual = (d->flags & AFNO_FLAG_NO_RESIDUAL) != 0;
  g->accum = (d->flags & AFNO_FLAG_ACCUM_GRADS) != 0;
  g->export_masks = (d->flags & AFNO_FLAG_EXPORT_MASKS) != 0;
  g->force_fp32 = (d->flags & AFNO_FLAG_FORCE_FP32_MATH) != 0;
  g->save_ctx = (d->flags & AFNO_FLAG_SAVE_CONTEXT) != 0;
  g->use_ctx = (d->flags & AFNO_FLAG_USE_CONTEXT) != 0;
  const char* why = nullptr;
  if (!generic_supported(*g, &why)) return fail(AFNO_ERR_UNSUPPORTED, why);
  return AFNO_OK;
}

// which kernel family serves the descriptor
bool use_tc_fwd(const Geometry& g) { return !g.force_fp32 && tc_supported(g); }
bool use_tc_bwd(const Geometry& g) { return use_tc_fwd(g); }
size_t workspace_bytes(const Geometry& g, bool backward) {
  if (backward) return use_tc_bwd(g) ? tc_workspace_bytes(g, true) : generic_workspace_bytes(g, true);
  return use_tc_fwd(g) ? tc_workspace_bytes(g, false) : generic_workspace_bytes(g, false);
}

// ---- plan cache ------------------------------------------------------------------------
std::mutex g_plan_mutex;
std::vector<Plan*> g_plans;

cudaError_t build_fft_plan(int n, FftPlan* out) {
  std::vector<int> radices;
  smooth235(n, &radices);
  if ((int)radices.size() > kMaxStages) return cudaErrorInvalidValue;
  memset(out, 0, sizeof(*out));
  out->n = n;
  out->nstages = (int)radices.size();
  for (size_t i = 0; i < radices.size(); ++i) out->radix[i] = radices[i];
  std::vector<float2> tw(n);
  const double two_pi = 6.283185307179586476925286766559;
  for (int k = 0; k < n; ++k) {
    const double a = -two_pi * (double)k / (double)n;
    tw[k] = make_float2((float)cos(a), (float)sin(a));
  }
  // DIF output order: bin k sits at sum_s (k_s * n / (r_1 ... r_s)), k = k_1 + r_1 (k_2 + r_2 (...))
  std::vector<int16_t> perm(n);
  for (int k = 0; k < n; ++k) {
    int kk = k, L = n, pos = 0;
    for (int r : radices) {
      const int m = L / r;
      pos += (kk % r) * m;
      kk /= r;
      L = m;
    }
    perm[k] = (int16_t)pos;
  }
  float2* dtw = nullptr;
  int16_t* dperm = nullptr;
  cudaError_t e = cudaMalloc(&dtw, sizeof(float2) * n);
  if (e == cudaSuccess) e = cudaMalloc(&dperm, sizeof(int16_t) * n);
  if (e == cudaSuccess) e = cudaMemcpy(dtw, tw.data(), sizeof(float2) * n, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(dperm, perm.data(), sizeof(int16_t) * n, cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {   // nothing of a failed plan stays allocated
    cudaFree(dtw);
    cudaFree(dperm);
    return e;
  }
  out->tw = dtw;
  out->perm = dperm;
  return cudaSuccess;
}

void free_fft_plan(FftPlan* p) {
  cudaFree(const_cast<float2*>(p->tw));
  cudaFree(const_cast<int16_t*>(p->perm));
  p->tw = nullptr;
  p->perm = nullptr;
}

// Returns the plan for (current device, H, W); builds it when allowed.
int get_plan(const Geometry& g, bool may_build, const Plan** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(AFNO_ERR_CUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
  std::lock_guard<std::mutex> lock(g_plan_mutex);
  for (Plan* p : g_plans)
    if (p->device == dev && p->H == g.H && p->W == g.W) {
      *out = p;
      return AFNO_OK;
    }
  if (!may_build)
    return fail(AFNO_ERR_INVALID_ARG, "stream is capturing and no plan exists: call afno_plan_warmup first");
  Plan* p = new Plan();
  p->device = dev;
  p->H = g.H;
  p->W = g.W;
  e = build_fft_plan(g.H, &p->fh);
  if (e == cudaSuccess) e = build_fft_plan(g.W, &p->fw);
  if (e == cudaSuccess && tc_plan_supported(g.H, g.W)) e = tc_build_plan(g.H, g.W, &p->tc);
  if (e != cudaSuccess) {
    free_fft_plan(&p->fh);
    free_fft_plan(&p->fw);
    tc_free_plan(&p->tc);
    delete p;
    return fail(AFNO_ERR_CUDA, std::string("plan creation: ") + cudaGetErrorString(e));
  }
  g_plans.push_back(p);
  *out = p;
  return AFNO_OK;
}

bool aligned16(const void* p) { return ((uintptr_t)p & 15u) == 0; }

bool overlaps(const void* a, const void* b, size_t bytes) {
  const char* pa = (const char*)a;
  const char* pb = (const char*)b;
  return pa < pb + bytes && pb < pa + bytes;
}

int stream_may_build(cudaStream_t st, bool* may_build) {
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  cudaError_t e = cudaStreamIsCapturing(st, &cs);
  if (e != cudaSuccess) return fail(AFNO_ERR_CUDA, std::string("cudaStreamIsCapturing: ") + cudaGetErrorString(e));
  *may_build = cs == cudaStreamCaptureStatusNone;
  return AFNO_OK;
}

size_t act_bytes(const Geometry& g) {
  return (size_t)g.B * g.H * g.W * g.C * (g.bf16 ? 2 : 4);
}

} // namespace

void count_launch(int n) { t_launches += n; }

// ---- optional per-kernel profiler (CUDA events around every launch) -----------------------
namespace {
struct ProfRec {
  const char* name;
  cudaEvent_t a, b;
};
thread_local bool t_prof_on = false;
thread_local std::vector<ProfRec> t_prof;
} // namespace

void prof_begin(const char* name, cudaStream_t st) {
  if (!t_prof_on) return;
  ProfRec r{name, nullptr, nullptr};
  if (cudaEventCreate(&r.a) != cudaSuccess || cudaEventCreate(&r.b) != cudaSuccess) return;
  cudaEventRecord(r.a, st);
  t_prof.push_back(r);
}
void prof_end(cudaStream_t st) {
  if (!t_prof_on || t_prof.empty()) return;
  cudaEventRecord(t_prof.back().b, st);
}

} // namespace afno

using namespace afno;

extern "C" {

int afno_version(void) { return 100; }

const char* afno_status_string(int status) {
  switch (status) {
    case AFNO_OK: return "ok";
    case AFNO_ERR_INVALID_ARG: return "invalid argument";
    case AFNO_ERR_UNSUPPORTED: return "unsupported configuration";
    case AFNO_ERR_WORKSPACE: return "workspace too small";
    case AFNO_ERR_CUDA: return "CUDA error";
    default: return "unknown status";
  }
}

const char* afno_last_error(void) { return t_error.c_str(); }

int afno_last_launch_count(void) { return t_launches; }

int afno_profile_start(void) {
  for (auto& r : t_prof) {
    cudaEventDestroy(r.a);
    cudaEventDestroy(r.b);
  }
  t_prof.clear();
  t_prof_on = true;
  return AFNO_OK;
}

int afno_profile_stop(char* out, size_t cap) {
  t_prof_on = false;
  cudaError_t e = cudaDeviceSynchronize();
  if (e != cudaSuccess) return fail(AFNO_ERR_CUDA, std::string("profile sync: ") + cudaGetErrorString(e));
  struct Agg { const char* name; int n; double ms; };
  std::vector<Agg> agg;
  for (auto& r : t_prof) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, r.a, r.b) != cudaSuccess) ms = 0.f;
    bool found = false;
    for (auto& a : agg)
      if (strcmp(a.name, r.name) == 0) { a.n++; a.ms += ms; found = true; break; }
    if (!found) agg.push_back({r.name, 1, (double)ms});
    cudaEventDestroy(r.a);
    cudaEventDestroy(r.b);
  }
  t_prof.clear();
  std::string text;
  char line[256];
  for (auto& a : agg) {
    snprintf(line, sizeof(line), "%s %d %.6f\n", a.name, a.n, a.ms);
    text += line;
  }
  if (out && cap > 0) {
    const size_t n = text.size() < cap - 1 ? text.size() : cap - 1;
    memcpy(out, text.data(), n);
    out[n] = 0;
  }
  return AFNO_OK;
}

const char* afno_spectral_path(const afno_desc_t* d) {
  Geometry g;
  if (resolve(d, &g) != AFNO_OK) return nullptr;
  // "hybrid": fp32 FFTs on the CUDA cores + the block MLP (forward, and, for hidden factors 1..8, also the gradient stages and
  // the parameter gradients) on the tensor cores
  return use_tc_fwd(g) ? "tcgen05-bf16" : (tc_mlp_supported(g) ? "hybrid-fft32-tcgen05" : "generic-fp32");
}

size_t afno_spectral_workspace_bytes(const afno_desc_t* d, int for_backward) {
  Geometry g;
  if (resolve(d, &g) != AFNO_OK) return 0;
  return workspace_bytes(g, for_backward != 0);
}

int afno_spectral_mask_bytes(const afno_desc_t* d, size_t* mask1_bytes, size_t* mask2_offset,
                             size_t* mask2_bytes) {
  Geometry g;
  int rc = resolve(d, &g);
  if (rc != AFNO_OK) return rc;
  const size_t b1 = (size_t)g.modes_all() * g.CH * 2, b2 = (size_t)g.modes_all() * g.C * 2;
  if (mask1_bytes) *mask1_bytes = b1;
  if (mask2_offset) *mask2_offset = align_up(b1, 256);
  if (mask2_bytes) *mask2_bytes = b2;
  return AFNO_OK;
}

int afno_plan_warmup(const afno_desc_t* d) {
  Geometry g;
  int rc = resolve(d, &g);
  if (rc != AFNO_OK) return rc;
  const Plan* p = nullptr;
  return get_plan(g, true, &p);
}

int afno_spectral_fwd(const afno_desc_t* d, const void* x, const float* w1, const float* b1,
                      const float* w2, const float* b2, void* y, void* workspace,
                      size_t workspace_bytes, void* cuda_stream) {
  t_launches = 0;
  Geometry g;
  int rc = resolve(d, &g);
  if (rc != AFNO_OK) return rc;
  if (!x || !w1 || !b1 || !w2 || !b2 || !y || !workspace) return fail(AFNO_ERR_INVALID_ARG, "NULL pointer argument");
  if (g.use_ctx) return fail(AFNO_ERR_INVALID_ARG, "AFNO_FLAG_USE_CONTEXT is a flag of afno_spectral_bwd");
  const void* ptrs[] = {x, w1, b1, w2, b2, y, workspace};
  for (const void* p : ptrs)
    if (!aligned16(p)) return fail(AFNO_ERR_INVALID_ARG, "pointers must be 16-byte aligned");
  if (overlaps(x, y, act_bytes(g))) return fail(AFNO_ERR_INVALID_ARG, "y must not alias x");
  if (workspace_bytes < afno::workspace_bytes(g, g.save_ctx))
    return fail(AFNO_ERR_WORKSPACE, g.save_ctx ? "AFNO_FLAG_SAVE_CONTEXT needs a workspace of afno_spectral_workspace_bytes(d, 1)"
                                               : "workspace smaller than afno_spectral_workspace_bytes(d, 0)");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  bool may_build = false;
  rc = stream_may_build(st, &may_build);
  if (rc != AFNO_OK) return rc;
  const Plan* p = nullptr;
  rc = get_plan(g, may_build, &p);
  if (rc != AFNO_OK) return rc;
  cudaError_t e = (use_tc_fwd(g) && p->tc.valid) ? tc_forward(g, *p, x, w1, b1, w2, b2, y, workspace, st)
                                                 : generic_forward(g, *p, x, w1, b1, w2, b2, y, workspace, st);
  if (e != cudaSuccess) return fail(AFNO_ERR_CUDA, std::string("forward launch: ") + cudaGetErrorString(e));
  return AFNO_OK;
}

int afno_spectral_bwd(const afno_desc_t* d, const void* x, const void* dy, const float* w1,
                      const float* b1, const float* w2, const float* b2, void* dx, float* dw1,
                      float* db1, float* dw2, float* db2, void* workspace,
                      size_t workspace_bytes, void* cuda_stream) {
  t_launches = 0;
  Geometry g;
  int rc = resolve(d, &g);
  if (rc != AFNO_OK) return rc;
  if (!x || !dy || !w1 || !b1 || !w2 || !b2 || !dx || !dw1 || !db1 || !dw2 || !db2 || !workspace)
    return fail(AFNO_ERR_INVALID_ARG, "NULL pointer argument");
  if (g.save_ctx) return fail(AFNO_ERR_INVALID_ARG, "AFNO_FLAG_SAVE_CONTEXT is a flag of afno_spectral_fwd");
  const void* ptrs[] = {x, dy, w1, b1, w2, b2, dx, dw1, db1, dw2, db2, workspace};
  for (const void* p : ptrs)
    if (!aligned16(p)) return fail(AFNO_ERR_INVALID_ARG, "pointers must be 16-byte aligned");
  if (overlaps(dx, dy, act_bytes(g)) || overlaps(dx, x, act_bytes(g)))
    return fail(AFNO_ERR_INVALID_ARG, "dx must not alias dy or x");
  if (workspace_bytes < afno::workspace_bytes(g, true))
    return fail(AFNO_ERR_WORKSPACE, "workspace smaller than afno_spectral_workspace_bytes(d, 1)");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  bool may_build = false;
  rc = stream_may_build(st, &may_build);
  if (rc != AFNO_OK) return rc;
  const Plan* p = nullptr;
  rc = get_plan(g, may_build, &p);
  if (rc != AFNO_OK) return rc;
  size_t m1 = 0, m2off = 0, m2 = 0;
  afno_spectral_mask_bytes(d, &m1, &m2off, &m2);
  cudaError_t e = (use_tc_bwd(g) && p->tc.valid)
                      ? tc_backward(g, *p, x, dy, w1, b1, w2, b2, dx, dw1, db1, dw2, db2, workspace, st)
                      : generic_backward(g, *p, x, dy, w1, b1, w2, b2, dx, dw1, db1, dw2, db2, workspace, m1, m2off, st);
  if (e != cudaSuccess) return fail(AFNO_ERR_CUDA, std::string("backward launch: ") + cudaGetErrorString(e));
  return AFNO_OK;
}

// ---- host-buffer (end-to-end) variants ---------------------------------------------------
namespace {
struct Arena {
  char* base;
  size_t off = 0;
  void* take(size_t bytes) {
    void* p = base ? base + off : nullptr;
    off = align_up(off + bytes, 256);
    return p;
  }
};
// What the x at the head of an arena belongs to: written by every host call that leaves a complete x there, checked by
// afno_spectral_bwd_host when it is asked to reuse that x (x_host == NULL).
struct ArenaStamp {
  uint32_t magic;
  int32_t B, H, W, C, dtype;
  uint32_t pad[2];
};
constexpr uint32_t kArenaMagic = 0x41464E4Fu;   // "AFNO"
ArenaStamp stamp_of(const Geometry& g) { return ArenaStamp{kArenaMagic, g.B, g.H, g.W, g.C, g.bf16 ? 1 : 0, {0u, 0u}}; }

struct HostLayout {
  void* stamp;   // ArenaStamp, same offset in the three layouts (x and the parameters come first in all of them)
  void *x, *dy, *y, *dx;
  float *w1, *b1, *w2, *b2, *dw1, *db1, *dw2, *db2;
  void* ws;
  size_t ws_bytes, total, act, nw, nb1, nb2;
};
HostLayout host_layout(const afno_desc_t* d, const Geometry& g, int mode, char* base) {
  const bool backward = mode != 0;
  HostLayout h{};
  Arena a{base};
  h.act = act_bytes(g);
  h.nw = (size_t)g.nb * g.bs * g.hid * 2 * sizeof(float);
  h.nb1 = (size_t)g.nb * g.hid * 2 * sizeof(float);
  h.nb2 = (size_t)g.nb * g.bs * 2 * sizeof(float);
  h.x = a.take(h.act);
  h.w1 = (float*)a.take(h.nw);
  h.b1 = (float*)a.take(h.nb1);
  h.w2 = (float*)a.take(h.nw);
  h.b2 = (float*)a.take(h.nb2);
  h.stamp = a.take(sizeof(ArenaStamp));
  if (backward) {
    h.dy = a.take(h.act);
    h.dx = a.take(h.act);
    h.dw1 = (float*)a.take(h.nw);
    h.db1 = (float*)a.take(h.nb1);
    h.dw2 = (float*)a.take(h.nw);
    h.db2 = (float*)a.take(h.nb2);
  }
  if (mode != 1) h.y = a.take(h.act);
  h.ws_bytes = afno_spectral_workspace_bytes(d, backward ? 1 : 0);
  h.ws = a.take(h.ws_bytes);
  h.total = a.off;
  return h;
}
} // namespace

size_t afno_spectral_host_arena_bytes(const afno_desc_t* d, int for_backward) {
  Geometry g;
  if (resolve(d, &g) != AFNO_OK) return 0;
  return host_layout(d, g, for_backward == 2 ? 2 : (for_backward != 0 ? 1 : 0), nullptr).total;
}

#define AFNO_CUDA_TRY(expr)                                                                     \
  do {                                                                                          \
    cudaError_t e_ = (expr);                                                                    \
    if (e_ != cudaSuccess) return fail(AFNO_ERR_CUDA, std::string(#expr ": ") + cudaGetErrorString(e_)); \
  } while (0)

// The host variants are PCIe-bound (0.5 GB per fwd+bwd step at B = 4 against 0.5 ms of kernels), so they
// pipeline over the batch: sample b+1 travels host->device on one copy stream while sample b computes on
// the caller's stream and sample b-1 travels device->host on a second copy stream (the link is full
// duplex).  Samples are independent ("batched"); the parameter gradients of the samples
// are accumulated in order with AFNO_FLAG_ACCUM_GRADS.
namespace {
// Internal copy streams and reusable events of the host variants, one set per device (created on first use,
// kept for the life of the process).
struct HostPipe {
  int device = -1;
  cudaStream_t h2d = nullptr, d2h = nullptr;
  std::vector<cudaEvent_t> ev;
  size_t next = 0;
  // records an event on `on` and makes `waiter` wait for it; events are recycled round-robin (a recycled
  // event's earlier wait has long been enqueued: re-recording does not disturb it)
  cudaError_t mark(cudaStream_t on, cudaStream_t waiter) {
    if (ev.size() < 64) {
      cudaEvent_t e;
      cudaError_t rc = cudaEventCreateWithFlags(&e, cudaEventDisableTiming);
      if (rc != cudaSuccess) return rc;
      ev.push_back(e);
      next = ev.size() - 1;
    } else {
      next = (next + 1) % ev.size();
    }
    cudaError_t rc = cudaEventRecord(ev[next], on);
    if (rc != cudaSuccess) return rc;
    return cudaStreamWaitEvent(waiter, ev[next], 0);
  }
  // quiesce everything the call has enqueued (also on the error paths: the caller may free its buffers)
  void drain(cudaStream_t st) {
    cudaStreamSynchronize(h2d);
    cudaStreamSynchronize(st);
    cudaStreamSynchronize(d2h);
  }
};
// one set per (thread, device); released when the thread ends (errors ignored: at process exit the runtime may be gone)
struct HostPipes {
  std::vector<HostPipe*> v;
  ~HostPipes() {
    for (HostPipe* p : v) {
      for (cudaEvent_t e : p->ev) cudaEventDestroy(e);
      if (p->h2d) cudaStreamDestroy(p->h2d);
      if (p->d2h) cudaStreamDestroy(p->d2h);
      delete p;
    }
  }
};
thread_local HostPipes t_pipes;
cudaError_t host_pipe(HostPipe** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  for (HostPipe* p : t_pipes.v)
    if (p->device == dev) {
      *out = p;
      return cudaSuccess;
    }
  HostPipe* p = new HostPipe();
  if ((e = cudaStreamCreateWithFlags(&p->h2d, cudaStreamNonBlocking)) != cudaSuccess ||
      (e = cudaStreamCreateWithFlags(&p->d2h, cudaStreamNonBlocking)) != cudaSuccess) {
    if (p->h2d) cudaStreamDestroy(p->h2d);
    delete p;
    return e;
  }
  p->device = dev;
  t_pipes.v.push_back(p);
  *out = p;
  return cudaSuccess;
}
// like AFNO_CUDA_TRY, but lets the copies and kernels already in flight finish before returning
#define AFNO_PIPE_TRY(expr)                                                                     \
  do {                                                                                          \
    cudaError_t e_ = (expr);                                                                    \
    if (e_ != cudaSuccess) {                                                                    \
      hp->drain(st);                                                                            \
      return fail(AFNO_ERR_CUDA, std::string(#expr ": ") + cudaGetErrorString(e_));             \
    }                                                                                           \
  } while (0)
} // namespace

int afno_spectral_fwd_host(const afno_desc_t* d, const void* x_host, const float* w1_host,
                           const float* b1_host, const float* w2_host, const float* b2_host,
                           void* y_host, void* arena, size_t arena_bytes, void* cuda_stream) {
  Geometry g;
  int rc = resolve(d, &g);
  if (rc != AFNO_OK) return rc;
  if (!x_host || !w1_host || !b1_host || !w2_host || !b2_host || !y_host || !arena)
    return fail(AFNO_ERR_INVALID_ARG, "NULL pointer argument");
  if (!aligned16(arena)) return fail(AFNO_ERR_INVALID_ARG, "arena must be 16-byte aligned");
  HostLayout h = host_layout(d, g, 0, (char*)arena);
  if (arena_bytes < h.total) return fail(AFNO_ERR_WORKSPACE, "arena smaller than afno_spectral_host_arena_bytes(d, 0)");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  HostPipe* hp = nullptr;
  AFNO_CUDA_TRY(host_pipe(&hp));
  afno_desc_t d1 = *d;
  d1.B = 1;
  d1.flags &= ~(uint32_t)(AFNO_FLAG_SAVE_CONTEXT | AFNO_FLAG_USE_CONTEXT);
  const size_t sample = h.act / (size_t)g.B;
  AFNO_PIPE_TRY(hp->mark(st, hp->h2d));   // the copies start after the caller's earlier work on the stream
  AFNO_PIPE_TRY(cudaMemcpyAsync(h.w1, w1_host, h.nw, cudaMemcpyHostToDevice, hp->h2d));
  AFNO_PIPE_TRY(cudaMemcpyAsync(h.b1, b1_host, h.nb1, cudaMemcpyHostToDevice, hp->h2d));
  AFNO_PIPE_TRY(cudaMemcpyAsync(h.w2, w2_host, h.nw, cudaMemcpyHostToDevice, hp->h2d));
  AFNO_PIPE_TRY(cudaMemcpyAsync(h.b2, b2_host, h.nb2, cudaMemcpyHostToDevice, hp->h2d));
  for (int b = 0; b < g.B; ++b) {
    const size_t off = (size_t)b * sample;
    AFNO_PIPE_TRY(cudaMemcpyAsync((char*)h.x + off, (const char*)x_host + off, sample, cudaMemcpyHostToDevice, hp->h2d));
    AFNO_PIPE_TRY(hp->mark(hp->h2d, st));
    rc = afno_spectral_fwd(&d1, (char*)h.x + off, h.w1, h.b1, h.w2, h.b2, (char*)h.y + off, h.ws, h.ws_bytes, cuda_stream);
    if (rc != AFNO_OK) {
      hp->drain(st);
      return rc;
    }
    AFNO_PIPE_TRY(hp->mark(st, hp->d2h));
    AFNO_PIPE_TRY(cudaMemcpyAsync((char*)y_host + off, (char*)h.y + off, sample, cudaMemcpyDeviceToHost, hp->d2h));
  }
  AFNO_PIPE_TRY(cudaStreamSynchronize(hp->d2h));
  const ArenaStamp stamp = stamp_of(g);   // x of this descriptor now sits complete at the head of the arena
  AFNO_PIPE_TRY(cudaMemcpyAsync(h.stamp, &stamp, sizeof(stamp), cudaMemcpyHostToDevice, st));
  AFNO_PIPE_TRY(cudaStreamSynchronize(st));
  return AFNO_OK;
}

int afno_spectral_bwd_host(const afno_desc_t* d, const void* x_host, const void* dy_host,
                           const float* w1_host, const float* b1_host, const float* w2_host,
                           const float* b2_host, void* dx_host, float* dw1_host,
                           float* db1_host, float* dw2_host, float* db2_host, void* arena,
                           size_t arena_bytes, void* cuda_stream) {
  Geometry g;
  int rc = resolve(d, &g);
  if (rc != AFNO_OK) return rc;
  // x_host == NULL: x is still in the arena from the afno_spectral_fwd_host call that preceded this one on the
  // same arena and descriptor (a training step uploads x once)
  if (!dy_host || !w1_host || !b1_host || !w2_host || !b2_host || !dx_host || !dw1_host ||
      !db1_host || !dw2_host || !db2_host || !arena)
    return fail(AFNO_ERR_INVALID_ARG, "NULL pointer argument");
  if (d->flags & AFNO_FLAG_ACCUM_GRADS)
    return fail(AFNO_ERR_INVALID_ARG, "AFNO_FLAG_ACCUM_GRADS is not meaningful for the host variant");
  if (d->flags & AFNO_FLAG_EXPORT_MASKS)
    return fail(AFNO_ERR_INVALID_ARG, "AFNO_FLAG_EXPORT_MASKS is not meaningful for the host variant");
  if (!aligned16(arena)) return fail(AFNO_ERR_INVALID_ARG, "arena must be 16-byte aligned");
  HostLayout h = host_layout(d, g, 1, (char*)arena);
  if (arena_bytes < h.total) return fail(AFNO_ERR_WORKSPACE, "arena smaller than afno_spectral_host_arena_bytes(d, 1)");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (!x_host) {
    // the arena must say that a host call left x of exactly this shape and dtype there: a fresh or foreign arena would
    // otherwise yield plausible-looking dx and gradients of whatever bytes it holds
    ArenaStamp got{};
    AFNO_CUDA_TRY(cudaMemcpyAsync(&got, h.stamp, sizeof(got), cudaMemcpyDeviceToHost, st));
    AFNO_CUDA_TRY(cudaStreamSynchronize(st));
    const ArenaStamp want = stamp_of(g);
    if (memcmp(&got, &want, sizeof(want)) != 0)
      return fail(AFNO_ERR_INVALID_ARG,
                  "x_host is NULL, but no afno_spectral_fwd_host / _step_host / _bwd_host call with the same B, H, W, C "
                  "and dtype has left x in this arena");
  }
  HostPipe* hp = nullptr;
  AFNO_CUDA_TRY(host_pipe(&hp));
  afno_desc_t d1 = *d;
  d1.B = 1;
  d1.flags &= ~(uint32_t)(AFNO_FLAG_SAVE_CONTEXT | AFNO_FLAG_USE_CONTEXT);
  const size_t sample = h.act / (size_t)g.B;
  AFNO_PIPE_TRY(hp->mark(st, hp->h2d));
  AFNO_PIPE_TRY(cudaMemcpyAsync(h.w1, w1_host, h.nw, cudaMemcpyHostToDevice, hp->h2d));
  AFNO_PIPE_TRY(cudaMemcpyAsync(h.b1, b1_host, h.nb1, cudaMemcpyHostToDevice, hp->h2d));
  AFNO_PIPE_TRY(cudaMemcpyAsync(h.w2, w2_host, h.nw, cudaMemcpyHostToDevice, hp->h2d));
  AFNO_PIPE_TRY(cudaMemcpyAsync(h.b2, b2_host, h.nb2, cudaMemcpyHostToDevice, hp->h2d));
  for (int b = 0; b < g.B; ++b) {
    const size_t off = (size_t)b * sample;
    if (x_host)
      AFNO_PIPE_TRY(cudaMemcpyAsync((char*)h.x + off, (const char*)x_host + off, sample, cudaMemcpyHostToDevice, hp->h2d));
    AFNO_PIPE_TRY(cudaMemcpyAsync((char*)h.dy + off, (const char*)dy_host + off, sample, cudaMemcpyHostToDevice, hp->h2d));
    AFNO_PIPE_TRY(hp->mark(hp->h2d, st));
    d1.flags = b == 0 ? (d1.flags & ~(uint32_t)AFNO_FLAG_ACCUM_GRADS) : (d1.flags | AFNO_FLAG_ACCUM_GRADS);
    rc = afno_spectral_bwd(&d1, (char*)h.x + off, (char*)h.dy + off, h.w1, h.b1, h.w2, h.b2, (char*)h.dx + off, h.dw1, h.db1,
                           h.dw2, h.db2, h.ws, h.ws_bytes, cuda_stream);
    if (rc != AFNO_OK) {
      hp->drain(st);
      return rc;
    }
    AFNO_PIPE_TRY(hp->mark(st, hp->d2h));
    AFNO_PIPE_TRY(cudaMemcpyAsync((char*)dx_host + off, (char*)h.dx + off, sample, cudaMemcpyDeviceToHost, hp->d2h));
  }
  AFNO_PIPE_TRY(cudaMemcpyAsync(dw1_host, h.dw1, h.nw, cudaMemcpyDeviceToHost, hp->d2h));
  AFNO_PIPE_TRY(cudaMemcpyAsync(db1_host, h.db1, h.nb1, cudaMemcpyDeviceToHost, hp->d2h));
  AFNO_PIPE_TRY(cudaMemcpyAsync(dw2_host, h.dw2, h.nw, cudaMemcpyDeviceToHost, hp->d2h));
  AFNO_PIPE_TRY(cudaMemcpyAsync(db2_host, h.db2, h.nb2, cudaMemcpyDeviceToHost, hp->d2h));
  AFNO_PIPE_TRY(cudaStreamSynchronize(hp->d2h));
  const ArenaStamp stamp = stamp_of(g);   // x of this descriptor now sits complete at the head of the arena
  AFNO_PIPE_TRY(cudaMemcpyAsync(h.stamp, &stamp, sizeof(stamp), cudaMemcpyHostToDevice, st));
  AFNO_PIPE_TRY(cudaStreamSynchronize(st));
  return AFNO_OK;
}

// One training step from host buffers: per sample x and dy travel host->device back to back on one copy stream, the
// forward (saving its context) and the backward (using it) run on the caller's stream as soon as their input has
// landed, y and dx travel device->host on the second copy stream: the two directions of the link stay busy across
// the forward / backward boundary, which the two separate calls cannot do (each synchronises before it returns).
int afno_spectral_step_host(const afno_desc_t* d, const void* x_host, const void* dy_host, const float* w1_host,
                            const float* b1_host, const float* w2_host, const float* b2_host, void* y_host,
                            void* dx_host, float* dw1_host, float* db1_host, float* dw2_host, float* db2_host,
                            void* arena, size_t arena_bytes, void* cuda_stream) {
  Geometry g;
  int rc = resolve(d, &g);
  if (rc != AFNO_OK) return rc;
  if (!x_host || !dy_host || !w1_host || !b1_host || !w2_host || !b2_host || !y_host || !dx_host || !dw1_host ||
      !db1_host || !dw2_host || !db2_host || !arena)
    return fail(AFNO_ERR_INVALID_ARG, "NULL pointer argument");
  if (d->flags & (AFNO_FLAG_ACCUM_GRADS | AFNO_FLAG_EXPORT_MASKS))
    return fail(AFNO_ERR_INVALID_ARG, "AFNO_FLAG_ACCUM_GRADS / AFNO_FLAG_EXPORT_MASKS are not meaningful for the host variant");
  if (!aligned16(arena)) return fail(AFNO_ERR_INVALID_ARG, "arena must be 16-byte aligned");
  afno_desc_t d1 = *d;
  d1.B = 1;
  d1.flags &= ~(uint32_t)(AFNO_FLAG_SAVE_CONTEXT | AFNO_FLAG_USE_CONTEXT);
  HostLayout h = host_layout(d, g, 2, (char*)arena);
  if (arena_bytes < h.total) return fail(AFNO_ERR_WORKSPACE, "arena smaller than afno_spectral_host_arena_bytes(d, 2)");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  HostPipe* hp = nullptr;
  AFNO_CUDA_TRY(host_pipe(&hp));
  afno_desc_t df = d1, db = d1;
  df.flags |= AFNO_FLAG_SAVE_CONTEXT;
  const size_t sample = h.act / (size_t)g.B;
  AFNO_PIPE_TRY(hp->mark(st, hp->h2d));
  AFNO_PIPE_TRY(cudaMemcpyAsync(h.w1, w1_host, h.nw, cudaMemcpyHostToDevice, hp->h2d));
  AFNO_PIPE_TRY(cudaMemcpyAsync(h.b1, b1_host, h.nb1, cudaMemcpyHostToDevice, hp->h2d));
  AFNO_PIPE_TRY(cudaMemcpyAsync(h.w2, w2_host, h.nw, cudaMemcpyHostToDevice, hp->h2d));
  AFNO_PIPE_TRY(cudaMemcpyAsync(h.b2, b2_host, h.nb2, cudaMemcpyHostToDevice, hp->h2d));
  for (int b = 0; b < g.B; ++b) {
    const size_t off = (size_t)b * sample;
    AFNO_PIPE_TRY(cudaMemcpyAsync((char*)h.x + off, (const char*)x_host + off, sample, cudaMemcpyHostToDevice, hp->h2d));
    AFNO_PIPE_TRY(hp->mark(hp->h2d, st));
    rc = afno_spectral_fwd(&df, (char*)h.x + off, h.w1, h.b1, h.w2, h.b2, (char*)h.y + off, h.ws, h.ws_bytes, cuda_stream);
    if (rc != AFNO_OK) {
      hp->drain(st);
      return rc;
    }
    AFNO_PIPE_TRY(hp->mark(st, hp->d2h));
    AFNO_PIPE_TRY(cudaMemcpyAsync((char*)y_host + off, (char*)h.y + off, sample, cudaMemcpyDeviceToHost, hp->d2h));
    AFNO_PIPE_TRY(cudaMemcpyAsync((char*)h.dy + off, (const char*)dy_host + off, sample, cudaMemcpyHostToDevice, hp->h2d));
    AFNO_PIPE_TRY(hp->mark(hp->h2d, st));
    db.flags = (d1.flags | AFNO_FLAG_USE_CONTEXT) | (b == 0 ? 0u : (uint32_t)AFNO_FLAG_ACCUM_GRADS);
    rc = afno_spectral_bwd(&db, (char*)h.x + off, (char*)h.dy + off, h.w1, h.b1, h.w2, h.b2, (char*)h.dx + off, h.dw1, h.db1,
                           h.dw2, h.db2, h.ws, h.ws_bytes, cuda_stream);
    if (rc != AFNO_OK) {
      hp->drain(st);
      return rc;
    }
    AFNO_PIPE_TRY(hp->mark(st, hp->d2h));
    AFNO_PIPE_TRY(cudaMemcpyAsync((char*)dx_host + off, (char*)h.dx + off, sample, cudaMemcpyDeviceToHost, hp->d2h));
  }
  AFNO_PIPE_TRY(cudaMemcpyAsync(dw1_host, h.dw1, h.nw, cudaMemcpyDeviceToHost, hp->d2h));
  AFNO_PIPE_TRY(cudaMemcpyAsync(db1_host, h.db1, h.nb1, cudaMemcpyDeviceToHost, hp->d2h));
  AFNO_PIPE_TRY(cudaMemcpyAsync(dw2_host, h.dw2, h.nw, cudaMemcpyDeviceToHost, hp->d2h));
  AFNO_PIPE_TRY(cudaMemcpyAsync(db2_host, h.db2, h.nb2, cudaMemcpyDeviceToHost, hp->d2h));
  AFNO_PIPE_TRY(cudaStreamSynchronize(hp->d2h));
  const ArenaStamp stamp = stamp_of(g);   // x of this descriptor now sits complete at the head of the arena
  AFNO_PIPE_TRY(cudaMemcpyAsync(h.stamp, &stamp, sizeof(stamp), cudaMemcpyHostToDevice, st));
  AFNO_PIPE_TRY(cudaStreamSynchronize(st));
  return AFNO_OK;
}

// Rows B4 / B6 on caller-supplied operands with the split partial sums in the library's static device array: see
// include/afno.h.  Nothing on this path allocates: argument checks here, then the address lookup and three launches
// in generic.cu.  (The per-kernel profiler creates CUDA events; it is off unless afno_profile_start was called.)
int afno_block_wgrad_static(const float* a, int32_t lda, const float* g, int32_t ldg, int64_t M, int32_t num_blocks,
                            int32_t K, int32_t N, float* dw, float* db, uint32_t flags, void* cuda_stream) {
  t_launches = 0;
  if (num_blocks <= 0 || K <= 0 || N <= 0) return fail(AFNO_ERR_INVALID_ARG, "num_blocks, K and N must be positive");
  if (M < 0) return fail(AFNO_ERR_INVALID_ARG, "M must be >= 0");
  if (flags & ~(uint32_t)AFNO_FLAG_ACCUM_GRADS)
    return fail(AFNO_ERR_INVALID_ARG, "afno_block_wgrad_static takes no flag other than AFNO_FLAG_ACCUM_GRADS");
  if ((long long)num_blocks * K > lda || (long long)num_blocks * N > ldg)
    return fail(AFNO_ERR_INVALID_ARG, "row stride smaller than num_blocks*K (lda) or num_blocks*N (ldg) complex elements");
  if (!dw || !db || (M > 0 && (!a || !g))) return fail(AFNO_ERR_INVALID_ARG, "NULL pointer argument");
  const void* ptrs[] = {a, g, dw, db};
  for (const void* p : ptrs)
    if (((uintptr_t)p & 7u) != 0) return fail(AFNO_ERR_INVALID_ARG, "pointers must be 8-byte aligned (complex fp32)");
  const long long tiles = (long long)((K + 95) / 96) * ((N + 95) / 96);
  if (num_blocks > 65535 || tiles > 65535)
    return fail(AFNO_ERR_UNSUPPORTED, "num_blocks or ceil(K/96)*ceil(N/96) exceeds 65,535 (launch grid)");
  const size_t need = wgrad_static_split_bytes(num_blocks, K, N);
  if (need > kStaticScratchBytes)
    return fail(AFNO_ERR_UNSUPPORTED,
                "afno_block_wgrad_static: num_blocks*(K+1)*N*8 = " + std::to_string(need) +
                    " bytes of partial sums exceed the static scratch array of " + std::to_string(kStaticScratchBytes) +
                    " bytes (AFNO_STATIC_SCRATCH_BYTES); use afno_spectral_bwd with a caller workspace for this shape");
  cudaError_t e = generic_wgrad_static((const float2*)a, lda, (const float2*)g, ldg, (long long)M, num_blocks, K, N, dw, db,
                                       (flags & AFNO_FLAG_ACCUM_GRADS) != 0, (cudaStream_t)cuda_stream);
  if (e != cudaSuccess) return fail(AFNO_ERR_CUDA, std::string("afno_block_wgrad_static: ") + cudaGetErrorString(e));
  return AFNO_OK;
}

// Frees every plan of the calling process (constant tables on all devices).  No call of this library may
// be in flight; the next fwd / bwd / afno_plan_warmup rebuilds what it needs.
int afno_plan_destroy_all(void) {
  std::lock_guard<std::mutex> lock(g_plan_mutex);
  int dev = 0;
  cudaGetDevice(&dev);
  for (Plan* p : g_plans) {
    cudaSetDevice(p->device);
    free_fft_plan(&p->fh);
    free_fft_plan(&p->fw);
    tc_free_plan(&p->tc);
    delete p;
  }
  g_plans.clear();
  cudaSetDevice(dev);
  return AFNO_OK;
}

} // extern "C"
