// Stage functions of the two-register-stage strided passes (demag_fast2.cu: LDG / STG tiles; demag_tma.cu:
// tiles moved by the TMA engine).  P = 2L = K1 K2 (plan2.cuh): stage A = pruned radix-K1 butterfly of K1/2
// inputs + twiddle -> shared memory; stage B = radix-K2 butterfly; A', B' the mirror images.
#pragma once
#include "fft_core.cuh"
#include "plan2.cuh"

namespace mm {

template <typename T, int L> struct Tile2 {
  using P = Plan2<L>;
  static constexpr int K1 = P::K1, K2 = P::K2, A = K1 / 2;
  static constexpr int K2P = (K2 + 1) / 2 * 2;       // row pitch of a k1 block: even, so that bf ^ 1 stays inside it
  static constexpr int JN = K2 / 2 + 1;              // k2 values of a stage-B thread that can hold a k <= L
  static constexpr int B = 64 / (int)sizeof(Cx<T>);  // lanes along the batch (64-byte rows)
  static constexpr int tasksA = K2 * B, tasksB = K1 * B;
  static constexpr int NT = ((tasksA > tasksB ? tasksA : tasksB) + 31) / 32 * 32;
  static constexpr int slotsB = (tasksB + 31) / 32 * 32 / B;   // stage-B slots rounded up to whole warps
  // Does the stage-B thread of slot (pair0, odd) hold a row k = k1 + K1 j <= L in its slot j < JN?  Even K2:
  // every j < K2/2 (the slot j = K2/2 is k = L of k1 = 0, handled apart).  Odd K2: k1 <= K1/2 (even slots and
  // the self-paired k1 = K1/2) holds j <= (K2-1)/2, k1 > K1/2 (odd slots of the other pairs) one row less.
  static __device__ __forceinline__ bool has_row(int j, bool pair0, bool odd) {
    if (K2 % 2 == 0) return j < K2 / 2;
    return j < K2 / 2 || (j == K2 / 2 && (pair0 || !odd));
  }
  static constexpr int smem_bytes = K1 * K2P * 64;
  // root table staged in shared memory: [K2][TWP], TWP = K1 + 16 bytes: the rows of a warp's slots 16 bytes apart in the banks
  static constexpr int TWP = K1 + 32 / (int)sizeof(Cx<T>) / 2, tw_bytes = (K2 * TWP * (int)sizeof(Cx<T>) + 127) / 128 * 128;
  static constexpr int min_blocks = sizeof(T) == 8 ? 2 : (smem_bytes >= 32 * 1024 ? 3 : 4);
  static_assert(K1 * K2 == 2 * L && K1 % 2 == 0 && NT <= 256, "plan");
};

// Shared-memory element (k1, bf, lane): sm[(k1 K2P + (bf ^ odd(k1))) B + lane], odd(k1) = k1 >= K1/2:
// the two k1 of a stage-B half warp (slots 2p, 2p + 1) read rows of opposite parity, i.e.
// different 64-byte halves of the banks.
template <int K1> __device__ __forceinline__ int slot_k1(int slot) {
  const int p = slot >> 1, odd = slot & 1;
  return p == 0 ? (odd ? K1 / 2 : 0) : (odd ? K1 - p : p);
}

template <typename T, int K1, int... I>
__device__ __forceinline__ void rot_fwd(const Cx<T>* v, Cx<T>* o, std::integer_sequence<int, I...>) {
  ((o[I] = mul_root<T, K1, I, false>(v[I])), ...);
}
template <typename T, int K1, int... I>
__device__ __forceinline__ void rot_inv_add(Cx<T>* e, const Cx<T>* o, std::integer_sequence<int, I...>) {
  ((e[I] = add_root<T, K1, I, true>(e[I], o[I])), ...);
}

// two adjacent complex values as one vector access where the type allows it
template <typename T> struct Vec2;
template <> struct Vec2<float> {
  static __device__ __forceinline__ void st(float2* p, float2 a, float2 b) {
    *reinterpret_cast<float4*>(p) = make_float4(a.x, a.y, b.x, b.y);
  }
  static __device__ __forceinline__ void ld(const float2* p, float2& a, float2& b) {
    const float4 t = *reinterpret_cast<const float4*>(p);
    a = make_float2(t.x, t.y);
    b = make_float2(t.z, t.w);
  }
  static __device__ __forceinline__ void ldg(const float2* p, float2& a, float2& b) {
    const float4 t = __ldg(reinterpret_cast<const float4*>(p));
    a = make_float2(t.x, t.y);
    b = make_float2(t.z, t.w);
  }
};
template <> struct Vec2<double> {
  static __device__ __forceinline__ void st(double2* p, double2 a, double2 b) { p[0] = a; p[1] = b; }
  static __device__ __forceinline__ void ld(const double2* p, double2& a, double2& b) { a = p[0]; b = p[1]; }
  static __device__ __forceinline__ void ldg(const double2* p, double2& a, double2& b) {
    a = __ldg(p); b = __ldg(p + 1);
  }
};

// ---- stage A, forward: v[s] = a[bf + K2 s] (s < K1/2) -> shared memory
// TWS: the root table has been staged in shared memory with row pitch K1 + 2 (Tile2::TWP; the persistent box
// kernels of demag_tma.cu), else it is read from global memory (row pitch K1).
template <typename T, int L, bool TWS = false>
__device__ __forceinline__ void fwdA(Cx<T>* sm, const Cx<T>* __restrict__ Wt, int lane, int bf, Cx<T>* v) {
  using TL = Tile2<T, L>;
  constexpr int K1 = TL::K1, K2P = TL::K2P, A = TL::A, B = TL::B;
  Cx<T> o[A];
  rot_fwd<T, K1>(v, o, std::make_integer_sequence<int, A>{});
  Dft<T, A, false>::run(v);   // even outputs k1 = 2u
  Dft<T, A, false>::run(o);   // odd outputs  k1 = 2u + 1
  const Cx<T>* tw = Wt + bf * (TWS ? TL::TWP : K1);
  Cx<T>* lo = sm + bf * B + lane;          // rows of k1 <  K1/2: (k1 K2P + bf)
  Cx<T>* hi = sm + (bf ^ 1) * B + lane;    // rows of k1 >= K1/2: (k1 K2P + (bf ^ 1))
#pragma unroll
  for (int u = 0; u < A; ++u) {
    Cx<T> w0, w1;
    if constexpr (TWS) Vec2<T>::ld(tw + 2 * u, w0, w1); else Vec2<T>::ldg(tw + 2 * u, w0, w1);
    (2 * u >= K1 / 2 ? hi : lo)[(2 * u) * K2P * B] = u ? cmul(v[u], w0) : v[0];
    (2 * u + 1 >= K1 / 2 ? hi : lo)[(2 * u + 1) * K2P * B] = cmul(o[u], w1);
  }
}

// ---- stage B, forward: t[k2] = X[k1 + K1 k2]
template <typename T, int L>
__device__ __forceinline__ void fwdB(const Cx<T>* sm, int lane, int k1, Cx<T>* t) {
  using TL = Tile2<T, L>;
  constexpr int K1 = TL::K1, K2 = TL::K2, K2P = TL::K2P, B = TL::B;
  const int odd = k1 >= K1 / 2 ? 1 : 0;
  const Cx<T>* base = sm + k1 * K2P * B + lane;
  const Cx<T>* pe = base + odd * B;   // even bf: row bf + odd
  const Cx<T>* po = base - odd * B;   // odd bf:  row bf - odd
#pragma unroll
  for (int bf = 0; bf < K2; ++bf) t[bf] = ((bf & 1) ? po : pe)[bf * B];
  Dft<T, K2, false>::run(t);
}

// ---- stage B', inverse: t[k2] = X[k1 + K1 k2] on entry
template <typename T, int L>
__device__ __forceinline__ void invB(Cx<T>* sm, int lane, int k1, Cx<T>* t) {
  using TL = Tile2<T, L>;
  constexpr int K1 = TL::K1, K2 = TL::K2, K2P = TL::K2P, B = TL::B;
  Dft<T, K2, true>::run(t);
  const int odd = k1 >= K1 / 2 ? 1 : 0;
  Cx<T>* base = sm + k1 * K2P * B + lane;
  Cx<T>* pe = base + odd * B;
  Cx<T>* po = base - odd * B;
#pragma unroll
  for (int bf = 0; bf < K2; ++bf) ((bf & 1) ? po : pe)[bf * B] = t[bf];
}

// ---- stage A', inverse with truncation: v[s] = x[bf + K2 s], s < K1/2
template <typename T, int L, bool TWS = false>
__device__ __forceinline__ void invA(const Cx<T>* sm, const Cx<T>* __restrict__ Wt, int lane, int bf, Cx<T>* v) {
  using TL = Tile2<T, L>;
  constexpr int K1 = TL::K1, K2P = TL::K2P, A = TL::A, B = TL::B;
  Cx<T> o[A];
  const Cx<T>* tw = Wt + bf * (TWS ? TL::TWP : K1);
  const Cx<T>* lo = sm + bf * B + lane;
  const Cx<T>* hi = sm + (bf ^ 1) * B + lane;
#pragma unroll
  for (int u = 0; u < A; ++u) {
    Cx<T> w0, w1;
    if constexpr (TWS) Vec2<T>::ld(tw + 2 * u, w0, w1); else Vec2<T>::ldg(tw + 2 * u, w0, w1);
    const Cx<T> a = (2 * u >= K1 / 2 ? hi : lo)[(2 * u) * K2P * B];
    const Cx<T> b = (2 * u + 1 >= K1 / 2 ? hi : lo)[(2 * u + 1) * K2P * B];
    v[u] = u ? cmulc(a, w0) : a;
    o[u] = cmulc(b, w1);
  }
  Dft<T, A, true>::run(v);
  Dft<T, A, true>::run(o);
  rot_inv_add<T, K1>(v, o, std::make_integer_sequence<int, A>{});
}

}  // namespace mm
