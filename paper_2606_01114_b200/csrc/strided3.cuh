// Stage functions of the three-stage strided passes of L = 1024 (demag_fast.cu: LDG / STG tiles; demag_tma3.cu:
// tiles moved by the TMA engine).  A tile is 2L rows x 64 B in shared memory: rows [0, L) hold the even-output
// half, rows [L, 2L) the odd-output half of the pruned length-2L transform; L = R1 R2 R3.
#pragma once
#include "fft_core.cuh"

namespace mm {

constexpr int kStrideThreads = 256;

constexpr int ilog2c(int v) { return v <= 1 ? 0 : 1 + ilog2c(v / 2); }

// Radix plan of the length-L sub-transforms of the three-stage strided passes: L = R1 R2 R3.  Only L = 1024
// runs them: every L <= 512 runs the two-stage kernels of demag_fast2.cu (fast_two_stage).
template <int L> struct FastPlan;
template <> struct FastPlan<1024> { static constexpr int R1 = 16, R2 = 8, R3 = 8; };

template <typename T, int L> struct Tile {
  using P = FastPlan<L>;
  static constexpr int R1 = P::R1, R2 = P::R2, R3 = P::R3;
  static constexpr int q1 = R2 * R3, q2 = R3;
  static constexpr int B = 64 / (int)sizeof(Cx<T>);   // lanes along the batch (64-byte rows)
  static constexpr int smem_bytes_ = 2 * L * 64;
  // threads per CTA: the 128 KB tile of L = 1024 admits one CTA per SM, which then gets 16 warps (fp32)
  static constexpr int NT = (smem_bytes_ > 110 * 1024 && sizeof(T) == 4) ? 2 * kStrideThreads : kStrideThreads;
  static constexpr int NS = NT / B;                   // task slots
  static constexpr int LOG3 = ilog2c(R3);
  static constexpr int smem_bytes = 2 * L * 64;
  // resident CTAs per SM the kernels are compiled for (shared memory and registers)
  static constexpr int min_blocks =
      smem_bytes <= 72 * 1024 ? (sizeof(T) == 4 ? 3 : 2) : (smem_bytes <= 110 * 1024 ? 2 : 1);
};

// ------------------------------------------------------------------ strided-pass stages
// Shared-memory element (logical row r, lane): sm[(r ^ ((r >> LOG3) & 1)) * B + lane].

// Forward first stage for butterfly bf: v[s] holds input row bf + q1 s.  Writes the even half
// (rows u1 q1 + bf) and the odd half (+L) after the inter-stage twiddle w_L^(bf u1).
template <typename T, int L>
__device__ __forceinline__ void fwd_first(Cx<T>* sm, const Cx<T>* __restrict__ W, int lane,
                                          int bf, Cx<T>* v) {
  using TL = Tile<T, L>;
  constexpr int R1 = TL::R1, q1 = TL::q1, B = TL::B;
  const int rb = bf ^ ((bf >> TL::LOG3) & 1);
  Cx<T> tw[R1];
#pragma unroll
  for (int u = 1; u < R1; ++u) tw[u] = __ldg(W + 2 * bf * u);
  Cx<T> e[R1];
#pragma unroll
  for (int s = 0; s < R1; ++s) e[s] = v[s];
  Dft<T, R1, false>::run(e);
#pragma unroll
  for (int u = 0; u < R1; ++u)
    sm[(u * q1 + rb) * B + lane] = u ? cmul(e[u], tw[u]) : e[0];
#pragma unroll
  for (int s = 0; s < R1; ++s) v[s] = cmul(v[s], __ldg(W + bf + q1 * s));
  Dft<T, R1, false>::run(v);
#pragma unroll
  for (int u = 0; u < R1; ++u)
    sm[(L + u * q1 + rb) * B + lane] = u ? cmul(v[u], tw[u]) : v[0];
}

// Forward middle stage over both halves, in place.
template <typename T, int L>
__device__ __forceinline__ void fwd_middle(Cx<T>* sm, const Cx<T>* __restrict__ W, int lane,
                                           int slot) {
  using TL = Tile<T, L>;
  constexpr int R1 = TL::R1, R2 = TL::R2, q1 = TL::q1, q2 = TL::q2, B = TL::B, NS = TL::NS;
  constexpr int NTASK = 2 * R1 * q2;
#pragma unroll
  for (int i0 = 0; i0 < NTASK; i0 += NS) {
    const int i = i0 + slot;
    if (NTASK % NS != 0 && i >= NTASK) break;
    const int t2 = i % q2, hu = i / q2;
    const int b0 = hu * q1 + t2, b1 = b0 ^ 1;
    Cx<T> v[R2];
#pragma unroll
    for (int s = 0; s < R2; ++s) v[s] = sm[(((s & 1) ? b1 : b0) + q2 * s) * B + lane];
    Dft<T, R2, false>::run(v);
#pragma unroll
    for (int u = 1; u < R2; ++u) v[u] = cmul(v[u], __ldg(W + 2 * R1 * t2 * u));
#pragma unroll
    for (int u = 0; u < R2; ++u) sm[(((u & 1) ? b1 : b0) + q2 * u) * B + lane] = v[u];
  }
}

// Forward last stage of task i (rows i R3 .. i R3 + R3 - 1): loads and transforms; v[u3] is
// the value of logical row i R3 + u3.
template <typename T, int L>
__device__ __forceinline__ void fwd_last(const Cx<T>* sm, int lane, int i, Cx<T>* v) {
  using TL = Tile<T, L>;
  constexpr int R3 = TL::R3, B = TL::B;
  const int g = i & 1, base = i * R3;
  const int pe = base + g, po = base - g;
#pragma unroll
  for (int s = 0; s < R3; ++s) v[s] = sm[(((s & 1) ? po : pe) + s) * B + lane];
  Dft<T, R3, false>::run(v);
}

// Inverse first stage (mirror of fwd_last): v[u3] = value of logical row i R3 + u3 on entry;
// the inverse butterfly's outputs are stored at rows i R3 + s.
template <typename T, int L>
__device__ __forceinline__ void inv_first(Cx<T>* sm, int lane, int i, Cx<T>* v) {
  using TL = Tile<T, L>;
  constexpr int R3 = TL::R3, B = TL::B;
  const int g = i & 1, base = i * R3;
  const int pe = base + g, po = base - g;
  Dft<T, R3, true>::run(v);
#pragma unroll
  for (int s = 0; s < R3; ++s) sm[(((s & 1) ? po : pe) + s) * B + lane] = v[s];
}

// Inverse middle stage (mirror of fwd_middle).
template <typename T, int L>
__device__ __forceinline__ void inv_middle(Cx<T>* sm, const Cx<T>* __restrict__ W, int lane,
                                           int slot) {
  using TL = Tile<T, L>;
  constexpr int R1 = TL::R1, R2 = TL::R2, q1 = TL::q1, q2 = TL::q2, B = TL::B, NS = TL::NS;
  constexpr int NTASK = 2 * R1 * q2;
#pragma unroll
  for (int i0 = 0; i0 < NTASK; i0 += NS) {
    const int i = i0 + slot;
    if (NTASK % NS != 0 && i >= NTASK) break;
    const int t2 = i % q2, hu = i / q2;
    const int b0 = hu * q1 + t2, b1 = b0 ^ 1;
    Cx<T> v[R2];
#pragma unroll
    for (int u = 0; u < R2; ++u) v[u] = sm[(((u & 1) ? b1 : b0) + q2 * u) * B + lane];
#pragma unroll
    for (int u = 1; u < R2; ++u) v[u] = cmulc(v[u], __ldg(W + 2 * R1 * t2 * u));
    Dft<T, R2, true>::run(v);
#pragma unroll
    for (int s = 0; s < R2; ++s) sm[(((s & 1) ? b1 : b0) + q2 * s) * B + lane] = v[s];
  }
}

// Inverse last stage for butterfly bf (mirror of fwd_first) with the truncation combine:
// v[s] = e_s + conj(w_2L^(bf + q1 s)) o_s = output sample bf + q1 s.
template <typename T, int L>
__device__ __forceinline__ void inv_last(const Cx<T>* sm, const Cx<T>* __restrict__ W, int lane,
                                         int bf, Cx<T>* v) {
  using TL = Tile<T, L>;
  constexpr int R1 = TL::R1, q1 = TL::q1, B = TL::B;
  const int rb = bf ^ ((bf >> TL::LOG3) & 1);
  Cx<T> tw[R1];
#pragma unroll
  for (int u = 1; u < R1; ++u) tw[u] = __ldg(W + 2 * bf * u);
  Cx<T> o[R1];
#pragma unroll
  for (int u = 0; u < R1; ++u) {
    const Cx<T> a = sm[(u * q1 + rb) * B + lane], b = sm[(L + u * q1 + rb) * B + lane];
    v[u] = u ? cmulc(a, tw[u]) : a;
    o[u] = u ? cmulc(b, tw[u]) : b;
  }
  Dft<T, R1, true>::run(v);
  Dft<T, R1, true>::run(o);
#pragma unroll
  for (int s = 0; s < R1; ++s) v[s] = cadd(v[s], cmulc(o[s], __ldg(W + bf + q1 * s)));
}

// two adjacent complex values as one vector access where the type allows it
template <typename T> struct Pair2;
template <> struct Pair2<float> {
  static __device__ __forceinline__ void st(float2* p, float2 a, float2 b) {
    *reinterpret_cast<float4*>(p) = make_float4(a.x, a.y, b.x, b.y);
  }
  static __device__ __forceinline__ void ld(const float2* p, float2& a, float2& b) {
    const float4 t = *reinterpret_cast<const float4*>(p);
    a = make_float2(t.x, t.y);
    b = make_float2(t.z, t.w);
  }
};
template <> struct Pair2<double> {
  static __device__ __forceinline__ void st(double2* p, double2 a, double2 b) { p[0] = a; p[1] = b; }
  static __device__ __forceinline__ void ld(const double2* p, double2& a, double2& b) { a = p[0]; b = p[1]; }
};


}  // namespace mm
