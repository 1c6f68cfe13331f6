// Part of generic.cu (included inside namespace afno { namespace { after the radix butterflies): two-pass FFT kernels
// for the grid sizes of BASELINE.json and of the paper (90, 180, 360 points per axis).
//
// The generic kernels above run one radix-2/3/4/5 stage per pass over shared memory; ncu shows them bound by the
// instruction issue rate (index arithmetic, twiddle loads, one butterfly per warp iteration: 27 k warp instructions per
// 180-point x 32-channel tile where the arithmetic needs ~6 k).  Here N = N1 x N2 and each of the two passes is a
// complete length-N1 (length-N2) transform held in REGISTERS by one thread (lane = channel), fully unrolled, every
// inner twiddle a compile-time constant:
//   n = N2 n1 + n2, k = k1 + N1 k2:
//   pass A (per n2): y[k1] = w_N^(n2 k1) sum_n1 x[N2 n1 + n2] w_N1^(n1 k1)       -> shared memory row k1 N2 + n2
//   pass B (per k1): X[k1 + N1 k2] = sum_n2 y[k1 N2 + n2] w_N2^(n2 k2)           -> natural order, straight to global memory
// Two shared-memory passes instead of four or five, no output permutation.  Same arithmetic (fp32), same results to
// rounding; used when the size is in the table below and C is a multiple of 64, the generic kernels otherwise.
constexpr double cx_pi = 3.14159265358979323846264338327950288;
constexpr double cx_sin(double x) {   // |x| <= pi
  double x2 = x * x, term = x, sum = x;
  for (int i = 1; i <= 16; ++i) {
    term *= -x2 / (double)((2 * i) * (2 * i + 1));
    sum += term;
  }
  return sum;
}
constexpr double cx_cos(double x) {
  double x2 = x * x, term = 1.0, sum = 1.0;
  for (int i = 1; i <= 16; ++i) {
    term *= -x2 / (double)((2 * i - 1) * (2 * i));
    sum += term;
  }
  return sum;
}

template <int N>
struct FirstRadix {
  static constexpr int value = (N <= 5) ? N : (N % 4 == 0) ? 4 : (N % 2 == 0) ? 2 : (N % 3 == 0) ? 3 : 5;
};

// natural-order in, natural-order out; SG = -1 forward (exp(-i..)), +1 inverse
template <int N, int SG>
struct RegFFT {
  static constexpr int R = FirstRadix<N>::value, M = N / R;
  template <int E>
  static __device__ __forceinline__ float2 twiddle(float2 t) {
    constexpr int e = E % N;
    if constexpr (e == 0) {
      return t;
    } else {
      constexpr double ang = 2.0 * cx_pi * (double)(e > N / 2 ? e - N : e) / (double)N;
      constexpr float c = (float)cx_cos(ang), s = (float)((double)SG * cx_sin(ang));
      return make_float2(fmaf(t.x, c, -t.y * s), fmaf(t.x, s, t.y * c));
    }
  }
  template <int J, int... P>
  static __device__ __forceinline__ void column(const float2 (&v)[N], float2 (&y)[R][M], std::integer_sequence<int, P...>) {
    float2 t[R];
    ((t[P] = v[P * M + J]), ...);
    small_dft<R>(t, (float)SG);
    ((y[P][J] = twiddle<J * P>(t[P])), ...);
  }
  template <int... J>
  static __device__ __forceinline__ void columns(const float2 (&v)[N], float2 (&y)[R][M], std::integer_sequence<int, J...>) {
    (column<J>(v, y, std::make_integer_sequence<int, R>{}), ...);
  }
  static __device__ __forceinline__ void run(float2 (&v)[N]) {
    if constexpr (N <= 5) {
      small_dft<N>(v, (float)SG);
    } else {
      float2 y[R][M];
      columns(v, y, std::make_integer_sequence<int, M>{});
#pragma unroll
      for (int p = 0; p < R; ++p) RegFFT<M, SG>::run(y[p]);
#pragma unroll
      for (int p = 0; p < R; ++p)
#pragma unroll
        for (int k = 0; k < M; ++k) v[R * k + p] = y[p][k];
    }
  }
};

// pass A of one (n2, lane): rows n1 N2 + n2 -> rows k1 N2 + n2, in place.  tw[k] = exp(-2 pi i k / N).
// (tws: stride of the twiddle table, for a sub-transform of length N / tws inside a three-pass transform)
template <int N1, int N2, int SG>
__device__ __forceinline__ void pass_a(float2* s, int lw, int l, int n2, const float2* __restrict__ tw, int tws = 1) {
  float2 v[N1];
#pragma unroll
  for (int n1 = 0; n1 < N1; ++n1) v[n1] = s[(n1 * N2 + n2) * lw + l];
  RegFFT<N1, SG>::run(v);
  s[n2 * lw + l] = v[0];
#pragma unroll
  for (int k1 = 1; k1 < N1; ++k1) {
    float2 o = v[k1];
    if (n2 != 0) {
      float2 t = __ldg(tw + tws * n2 * k1);   // uniform across the warp
      if (SG > 0) t.y = -t.y;
      o = cmul(o, t);
    }
    s[(k1 * N2 + n2) * lw + l] = o;
  }
}
// pass B of one (k1, lane): rows k1 N2 + n2 -> v[k2] = X[k1 + N1 k2]
template <int N1, int N2, int SG>
__device__ __forceinline__ void pass_b(const float2* s, int lw, int l, int k1, float2 (&v)[N2]) {
#pragma unroll
  for (int n2 = 0; n2 < N2; ++n2) v[n2] = s[(k1 * N2 + n2) * lw + l];
  RegFFT<N2, SG>::run(v);
}

constexpr int kF2Warps = 8;
constexpr int kF2MaxBatch = 24;   // rows a thread keeps in flight before its first shared-memory store

// ---- F2 / F7: H-direction complex FFT, in place on S[B][H][Kw][C]; tile = 32 G channels of one (b, kw) column ---------
// grid (C / (32 G), Kw, B), block 256; smem H * 32 G float2 (G = 2 up to 360 points, 1 beyond: 184 KB at 720)
constexpr int hfft2_warps(int) { return kF2Warps; }
template <int N1, int N2, int SG, int G, typename ST>
__global__ void __launch_bounds__(32 * hfft2_warps(G)) k_hfft2(ST* __restrict__ S, const float2* __restrict__ tw, int Kw, int C) {
  constexpr int H = N1 * N2, LW = 32 * G, NW = hfft2_warps(G);
  extern __shared__ float2 smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int kw = blockIdx.y, b = blockIdx.z;
  ST* base = S + ((size_t)b * H * Kw + kw) * C + (size_t)blockIdx.x * LW;
  const size_t hstride = (size_t)Kw * C;
  // a row of the tile is 256 G contiguous bytes: one float2 (G = 1) or float4 (G = 2) per lane; up to kF2MaxBatch
  // rows of the warp are in flight before the first shared-memory store
  typedef typename std::conditional<G == 2, typename SpecIO<ST>::pair_t, ST>::type vec_t;
  constexpr int PER = (H + NW - 1) / NW, LB = PER < kF2MaxBatch ? PER : kF2MaxBatch;
  for (int h0 = warp; h0 < H; h0 += NW * LB) {
    vec_t v[LB];
#pragma unroll
    for (int u = 0; u < LB; ++u) {
      const int h = h0 + u * NW;
      if (h < H) v[u] = *(const vec_t*)(base + (size_t)h * hstride + G * lane);
    }
#pragma unroll
    for (int u = 0; u < LB; ++u) {
      const int h = h0 + u * NW;
      if (h < H) {
        if constexpr (G == 2) {
          float2 a, b2;
          SpecIO<ST>::unpair(v[u], a, b2);
          *(float4*)(smem + h * LW + 2 * lane) = make_float4(a.x, a.y, b2.x, b2.y);
        } else {
          smem[h * LW + lane] = SpecIO<ST>::ld(&v[u]);
        }
      }
    }
  }
  __syncthreads();
  for (int task = warp; task < G * N2; task += NW) {
    const int g = task / N2, n2 = task - g * N2;
    pass_a<N1, N2, SG>(smem, LW, g * 32 + lane, n2, tw);
  }
  __syncthreads();
  for (int task = warp; task < G * N1; task += NW) {
    const int g = task / N1, k1 = task - g * N1;
    float2 v[N2];
    pass_b<N1, N2, SG>(smem, LW, g * 32 + lane, k1, v);
    ST* dst = base + g * 32 + lane;
#pragma unroll
    for (int k2 = 0; k2 < N2; ++k2) SpecIO<ST>::st(dst + (size_t)(k1 + N1 * k2) * hstride, v[k2]);
  }
}

// ---- the same for the long axis of the p -> 1 grid (720 = 8 x 9 x 10): three passes with short codelets -----------------
// N = N1 x Q, Q = N2 x N3: pass 1 is pass A of (N1, Q); every block k1 of Q rows then is a two-pass transform of length Q
// (twiddle table read with stride N1), whose result X[k1 + N1 (k2 + N2 k3)] leaves from registers.  The 24- and 30-point
// codelets of the two-pass split need ~190 registers (one 8-warp block per SM with a 184 KB tile); 8- to 10-point
// codelets fit 64, so one block runs 32 warps.  grid (C / 32, Kw, B), block 1024; smem H * 32 float2.
template <int N1, int N2, int N3, int SG, typename ST>
__global__ void __launch_bounds__(1024) k_hfft3(ST* __restrict__ S, const float2* __restrict__ tw, int Kw, int C) {
  constexpr int Q = N2 * N3, H = N1 * Q, NW = 32;
  extern __shared__ float2 smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int kw = blockIdx.y, b = blockIdx.z;
  ST* base = S + ((size_t)b * H * Kw + kw) * C + (size_t)blockIdx.x * 32 + lane;
  const size_t hstride = (size_t)Kw * C;
  constexpr int PER = (H + NW - 1) / NW, LB = PER < 12 ? PER : 12;
  for (int h0 = warp; h0 < H; h0 += NW * LB) {
    ST v[LB];
#pragma unroll
    for (int u = 0; u < LB; ++u) {
      const int h = h0 + u * NW;
      if (h < H) v[u] = base[(size_t)h * hstride];
    }
#pragma unroll
    for (int u = 0; u < LB; ++u) {
      const int h = h0 + u * NW;
      if (h < H) smem[h * 32 + lane] = SpecIO<ST>::ld(&v[u]);
    }
  }
  __syncthreads();
  for (int m = warp; m < Q; m += NW) pass_a<N1, Q, SG>(smem, 32, lane, m, tw);
  __syncthreads();
  for (int t = warp; t < N1 * N3; t += NW) {
    const int k1 = t / N3, n3 = t - k1 * N3;
    pass_a<N2, N3, SG>(smem + k1 * Q * 32, 32, lane, n3, tw, N1);
  }
  __syncthreads();
  for (int t = warp; t < N1 * N2; t += NW) {
    const int k1 = t / N2, k2 = t - k1 * N2;
    float2 v[N3];
    pass_b<N2, N3, SG>(smem + k1 * Q * 32, 32, lane, k2, v);
#pragma unroll
    for (int k3 = 0; k3 < N3; ++k3) SpecIO<ST>::st(base + (size_t)(k1 + N1 * (k2 + N2 * k3)) * hstride, v[k3]);
  }
}

// ---- F1 / B2: W-direction real FFT, two real channels packed into one complex transform ---------------------------------
// grid (C / (2 LW), H, B), block 32 NW; smem W * LW float2.  LW = 32 packed channels per row (one task per warp
// iteration) up to 360 points; LW = 16 beyond (184 KB at 1,440 points): a warp then runs two tasks side by side, one
// per half-warp.  Pass B runs the tasks k1 and N1 - k1 together: the Hermitian split of bin k needs Z[k] and Z[W - k],
// which live in exactly those two tasks, so the half-spectrum leaves from registers.
template <typename T, int N1, int N2, int NW, int LW, typename ST>
__global__ void __launch_bounds__(32 * NW, LW == 32 ? 2 : 1)
k_wfft_fwd2(const T* __restrict__ x, ST* __restrict__ S, const float2* __restrict__ tw, int H, int C, int Kw, float scale,
            int alpha_weight) {
  constexpr int W = N1 * N2, TPW = 32 / LW, NSLOT = NW * TPW;
  extern __shared__ float2 smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int l = lane % LW, slot = warp * TPW + lane / LW;
  const int h = blockIdx.y, b = blockIdx.z;
  const int c = blockIdx.x * (2 * LW) + 2 * l;
  const T* xrow = x + ((size_t)(b * H + h) * W) * C + c;
  {
    // rows in flight kept in the storage type (bf16 pairs: one register each)
    constexpr int PER = (W + NSLOT - 1) / NSLOT, LB = PER < 2 * kF2MaxBatch ? PER : 2 * kF2MaxBatch;
    for (int w0 = slot; w0 < W; w0 += NSLOT * LB) {
      typename ActIO<T>::raw2 v[LB];
#pragma unroll
      for (int u = 0; u < LB; ++u) {
        const int w = w0 + u * NSLOT;
        if (w < W) v[u] = ActIO<T>::ldraw2(xrow + (size_t)w * C);
      }
#pragma unroll
      for (int u = 0; u < LB; ++u) {
        const int w = w0 + u * NSLOT;
        if (w < W) smem[w * LW + l] = ActIO<T>::unraw2(v[u]);   // channel c in the real part, channel c + 1 in the imaginary part
      }
    }
  }
  __syncthreads();
  for (int n2 = slot; n2 < N2; n2 += NSLOT) pass_a<N1, N2, -1>(smem, LW, l, n2, tw);
  __syncthreads();
  ST* Srow = S + ((size_t)(b * H + h) * Kw) * C + c;
  // bin k from Z[k] = zk and Z[W - k] = zn (both channels of the pair)
  auto emit = [&](int k, float2 zk, float2 zn) {
    if (k >= Kw) return;
    float sc = 0.5f * scale;
    if (alpha_weight && k != 0 && 2 * k != W) sc *= 2.f;
    SpecIO<ST>::stpair(Srow + (size_t)k * C, make_float2(sc * (zk.x + zn.x), sc * (zk.y - zn.y)),
                       make_float2(sc * (zk.y + zn.y), -sc * (zk.x - zn.x)));
  };
  // work items: k1 = 0 alone, k1 = N1 / 2 alone (N1 even), pairs (k1, N1 - k1)
  constexpr int kItems = N1 / 2 + 1;
  for (int item = slot; item < kItems; item += NSLOT) {
    const int ka = item, kb = (N1 - item) % N1;
    float2 va[N2];
    pass_b<N1, N2, -1>(smem, LW, l, ka, va);
    if (ka == kb) {
      if (ka == 0) {
        // k = N1 k2, W - k = N1 (N2 - k2)
#pragma unroll
        for (int k2 = 0; k2 < N2; ++k2) emit(N1 * k2, va[k2], va[(N2 - k2) % N2]);
      } else {
        // k1 = N1 / 2: W - k = k1 + N1 (N2 - 1 - k2)
#pragma unroll
        for (int k2 = 0; k2 < N2; ++k2) emit(ka + N1 * k2, va[k2], va[N2 - 1 - k2]);
      }
    } else {
      float2 vb[N2];
      pass_b<N1, N2, -1>(smem, LW, l, kb, vb);
#pragma unroll
      for (int k2 = 0; k2 < N2; ++k2) {
        emit(ka + N1 * k2, va[k2], vb[N2 - 1 - k2]);
        emit(kb + N1 * k2, vb[k2], va[N2 - 1 - k2]);
      }
    }
  }
}

// ---- F8 + F9 / B8: W-direction complex-to-real inverse FFT, residual, store ------------------------------------------
// grid (C / (2 LW), H, B), block 32 NW; smem W * LW float2
template <typename T, int N1, int N2, int NW, int LW, typename ST>
__global__ void __launch_bounds__(32 * NW, LW == 32 ? 2 : 1)
k_wfft_inv2(const ST* __restrict__ S, const T* __restrict__ res, T* __restrict__ out, const float2* __restrict__ tw, int H,
            int C, int Kw, float scale, int half_interior) {
  constexpr int W = N1 * N2, TPW = 32 / LW, NSLOT = NW * TPW;
  extern __shared__ float2 smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int l = lane % LW, slot = warp * TPW + lane / LW;
  const int h = blockIdx.y, b = blockIdx.z;
  const int c = blockIdx.x * (2 * LW) + 2 * l;
  const ST* Srow = S + ((size_t)(b * H + h) * Kw) * C + c;
  // every stored bin kk <= W/2 feeds the transform twice: as z[kk] and, conjugated (Hermitian extension), as z[W - kk]
  {
    constexpr int PER = (W / 2 + NSLOT) / NSLOT, LB = PER < kF2MaxBatch ? PER : kF2MaxBatch;
    for (int k0 = slot; k0 <= W / 2; k0 += NSLOT * LB) {
      typename SpecIO<ST>::pair_t t[LB];
#pragma unroll
      for (int u = 0; u < LB; ++u) {
        const int kk = k0 + u * NSLOT;
        t[u] = typename SpecIO<ST>::pair_t{};
        if (kk < Kw) t[u] = SpecIO<ST>::ldpair(Srow + (size_t)kk * C);
      }
#pragma unroll
      for (int u = 0; u < LB; ++u) {
        const int kk = k0 + u * NSLOT;
        if (kk > W / 2) continue;
        float2 ta, tb;
        SpecIO<ST>::unpair(t[u], ta, tb);
        if (kk == 0 || 2 * kk == W) {
          ta.y = 0.f;   // reading A4: imaginary parts of the c = 0 and c = W/2 columns are discarded
          tb.y = 0.f;
        } else if (half_interior) {
          ta.x *= 0.5f; ta.y *= 0.5f; tb.x *= 0.5f; tb.y *= 0.5f;
        }
        // Ta + i Tb: channel c -> Re, channel c + 1 -> Im
        smem[kk * LW + l] = make_float2(ta.x - tb.y, ta.y + tb.x);
        if (kk != 0 && 2 * kk != W) smem[(W - kk) * LW + l] = make_float2(ta.x + tb.y, -ta.y + tb.x);   // conj(Ta) + i conj(Tb)
      }
    }
  }
  __syncthreads();
  for (int n2 = slot; n2 < N2; n2 += NSLOT) pass_a<N1, N2, +1>(smem, LW, l, n2, tw);
  __syncthreads();
  const size_t rowoff = ((size_t)(b * H + h) * W) * C + c;
  for (int k1 = slot; k1 < N1; k1 += NSLOT) {
    typename ActIO<T>::raw2 r[N2];
#pragma unroll
    for (int k2 = 0; k2 < N2; ++k2)
      if (res) r[k2] = ActIO<T>::ldraw2(res + rowoff + (size_t)(k1 + N1 * k2) * C);
    float2 v[N2];
    pass_b<N1, N2, +1>(smem, LW, l, k1, v);
#pragma unroll
    for (int k2 = 0; k2 < N2; ++k2) {
      const float2 rr = res ? ActIO<T>::unraw2(r[k2]) : make_float2(0.f, 0.f);
      ActIO<T>::st2(out + rowoff + (size_t)(k1 + N1 * k2) * C, scale * v[k2].x + rr.x, scale * v[k2].y + rr.y);
    }
  }
}

// ---- the W-direction transforms of the p -> 1 grid (1,440 = 16 x 9 x 10 points): three passes, 16 packed lanes per row ----
// (see k_hfft3; grid (C / 32, H, B), block 1024 = 64 half-warp task slots; smem W * 16 float2 = 184 KB)
template <int N1, int N2, int N3, int SG>
__device__ __forceinline__ void three_pass_ab(float2* smem, int l, int slot, const float2* __restrict__ tw) {
  constexpr int Q = N2 * N3, NSLOT = 64;
  for (int m = slot; m < Q; m += NSLOT) pass_a<N1, Q, SG>(smem, 16, l, m, tw);
  __syncthreads();
  for (int t = slot; t < N1 * N3; t += NSLOT) {
    const int k1 = t / N3, n3 = t - k1 * N3;
    pass_a<N2, N3, SG>(smem + k1 * Q * 16, 16, l, n3, tw, N1);
  }
  __syncthreads();
}

template <typename T, int N1, int N2, int N3, typename ST>
__global__ void __launch_bounds__(1024)
k_wfft_fwd3(const T* __restrict__ x, ST* __restrict__ S, const float2* __restrict__ tw, int H, int C, int Kw, float scale,
            int alpha_weight) {
  constexpr int Q = N2 * N3, W = N1 * Q, NSLOT = 64;
  extern __shared__ float2 smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int l = lane & 15, slot = warp * 2 + (lane >> 4);
  const int h = blockIdx.y, b = blockIdx.z;
  const int c = blockIdx.x * 32 + 2 * l;
  const T* xrow = x + ((size_t)(b * H + h) * W) * C + c;
  {
    constexpr int PER = (W + NSLOT - 1) / NSLOT, LB = PER < 12 ? PER : 12;
    for (int w0 = slot; w0 < W; w0 += NSLOT * LB) {
      typename ActIO<T>::raw2 v[LB];
#pragma unroll
      for (int u = 0; u < LB; ++u) {
        const int w = w0 + u * NSLOT;
        if (w < W) v[u] = ActIO<T>::ldraw2(xrow + (size_t)w * C);
      }
#pragma unroll
      for (int u = 0; u < LB; ++u) {
        const int w = w0 + u * NSLOT;
        if (w < W) smem[w * 16 + l] = ActIO<T>::unraw2(v[u]);
      }
    }
  }
  __syncthreads();
  three_pass_ab<N1, N2, N3, -1>(smem, l, slot, tw);
  ST* Srow = S + ((size_t)(b * H + h) * Kw) * C + c;
  auto emit = [&](int k, float2 zk, float2 zn) {   // bin k from Z[k] and Z[W - k]
    if (k >= Kw) return;
    float sc = 0.5f * scale;
    if (alpha_weight && k != 0 && 2 * k != W) sc *= 2.f;
    SpecIO<ST>::stpair(Srow + (size_t)k * C, make_float2(sc * (zk.x + zn.x), sc * (zk.y - zn.y)),
                       make_float2(sc * (zk.y + zn.y), -sc * (zk.x - zn.x)));
  };
  // last pass: task (k1, k2) yields Z[k1 + N1 (k2 + N2 k3)], k3 < N3.  Z[W - k] lives in the partner task
  //   k1 >= 1:        (N1 - k1, N2 - 1 - k2), element N3 - 1 - k3
  //   k1 = 0, k2 >= 1: (0, N2 - k2),           element N3 - 1 - k3
  //   k1 = k2 = 0:     itself,                 element (N3 - k3) mod N3
  // a slot runs a task together with its partner (the one with the smaller index takes the pair)
  for (int ti = slot; ti < N1 * N2; ti += NSLOT) {
    const int k1 = ti / N2, k2 = ti - k1 * N2;
    const int p1 = (N1 - k1) % N1, p2 = k1 ? N2 - 1 - k2 : (N2 - k2) % N2;
    const int pti = p1 * N2 + p2;
    if (ti > pti) continue;
    float2 va[N3];
    pass_b<N2, N3, -1>(smem + k1 * Q * 16, 16, l, k2, va);
    if (ti == pti) {
      const bool origin = (k1 | k2) == 0;
#pragma unroll
      for (int k3 = 0; k3 < N3; ++k3) emit(k1 + N1 * (k2 + N2 * k3), va[k3], origin ? va[(N3 - k3) % N3] : va[N3 - 1 - k3]);
    } else {
      float2 vb[N3];
      pass_b<N2, N3, -1>(smem + p1 * Q * 16, 16, l, p2, vb);
#pragma unroll
      for (int k3 = 0; k3 < N3; ++k3) {
        emit(k1 + N1 * (k2 + N2 * k3), va[k3], vb[N3 - 1 - k3]);
        emit(p1 + N1 * (p2 + N2 * k3), vb[k3], va[N3 - 1 - k3]);
      }
    }
  }
}

template <typename T, int N1, int N2, int N3, typename ST>
__global__ void __launch_bounds__(1024)
k_wfft_inv3(const ST* __restrict__ S, const T* __restrict__ res, T* __restrict__ out, const float2* __restrict__ tw, int H, int C,
            int Kw, float scale, int half_interior) {
  constexpr int Q = N2 * N3, W = N1 * Q, NSLOT = 64;
  extern __shared__ float2 smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int l = lane & 15, slot = warp * 2 + (lane >> 4);
  const int h = blockIdx.y, b = blockIdx.z;
  const int c = blockIdx.x * 32 + 2 * l;
  const ST* Srow = S + ((size_t)(b * H + h) * Kw) * C + c;
  {
    constexpr int PER = (W / 2 + NSLOT) / NSLOT, LB = PER < 8 ? PER : 8;
    for (int k0 = slot; k0 <= W / 2; k0 += NSLOT * LB) {
      typename SpecIO<ST>::pair_t t[LB];
#pragma unroll
      for (int u = 0; u < LB; ++u) {
        const int kk = k0 + u * NSLOT;
        t[u] = typename SpecIO<ST>::pair_t{};
        if (kk < Kw) t[u] = SpecIO<ST>::ldpair(Srow + (size_t)kk * C);
      }
#pragma unroll
      for (int u = 0; u < LB; ++u) {
        const int kk = k0 + u * NSLOT;
        if (kk > W / 2) continue;
        float2 ta, tb;
        SpecIO<ST>::unpair(t[u], ta, tb);
        if (kk == 0 || 2 * kk == W) {
          ta.y = 0.f;   // reading A4
          tb.y = 0.f;
        } else if (half_interior) {
          ta.x *= 0.5f; ta.y *= 0.5f; tb.x *= 0.5f; tb.y *= 0.5f;
        }
        smem[kk * 16 + l] = make_float2(ta.x - tb.y, ta.y + tb.x);
        if (kk != 0 && 2 * kk != W) smem[(W - kk) * 16 + l] = make_float2(ta.x + tb.y, -ta.y + tb.x);
      }
    }
  }
  __syncthreads();
  three_pass_ab<N1, N2, N3, +1>(smem, l, slot, tw);
  const size_t rowoff = ((size_t)(b * H + h) * W) * C + c;
  for (int t = slot; t < N1 * N2; t += NSLOT) {
    const int k1 = t / N2, k2 = t - k1 * N2;
    typename ActIO<T>::raw2 r[N3];
#pragma unroll
    for (int k3 = 0; k3 < N3; ++k3)
      if (res) r[k3] = ActIO<T>::ldraw2(res + rowoff + (size_t)(k1 + N1 * (k2 + N2 * k3)) * C);
    float2 v[N3];
    pass_b<N2, N3, +1>(smem + k1 * Q * 16, 16, l, k2, v);
#pragma unroll
    for (int k3 = 0; k3 < N3; ++k3) {
      const float2 rr = res ? ActIO<T>::unraw2(r[k3]) : make_float2(0.f, 0.f);
      ActIO<T>::st2(out + rowoff + (size_t)(k1 + N1 * (k2 + N2 * k3)) * C, scale * v[k3].x + rr.x, scale * v[k3].y + rr.y);
    }
  }
}

// size table of the two-pass kernels: N -> (N1, N2), the warps per block of the W-direction kernels (pass A has N2 tasks,
// pass B N1 / 2 + 1 paired items forward, N1 tasks inverse); `narrow` stays 0 (64 channels per H tile, 32 packed lanes per
// W tile).  720 and 1,440 points go to the three-pass kernels (fft3_dispatch); fft2_has() lists every size one of the
// register kernels serves.
template <typename F>
bool fft2_dispatch(int n, F&& f) {
  using std::integral_constant;
  if (n == 90) { f(integral_constant<int, 9>{}, integral_constant<int, 10>{}, integral_constant<int, 5>{}, integral_constant<int, 0>{}); return true; }
  if (n == 180) { f(integral_constant<int, 12>{}, integral_constant<int, 15>{}, integral_constant<int, 8>{}, integral_constant<int, 0>{}); return true; }
  if (n == 360) { f(integral_constant<int, 18>{}, integral_constant<int, 20>{}, integral_constant<int, 10>{}, integral_constant<int, 0>{}); return true; }
  return false;
}
// three-pass sizes: N -> N1 (N = N1 x 9 x 10)
template <typename F>
bool fft3_dispatch(int n, F&& f) {
  using std::integral_constant;
  if (n == 720) { f(integral_constant<int, 8>{}); return true; }
  if (n == 1440) { f(integral_constant<int, 16>{}); return true; }
  return false;
}
inline bool fft2_has(int n) { return n == 90 || n == 180 || n == 360 || n == 720 || n == 1440; }
