// Two-stage plans P = 2L = K1 x K2 (K1 even) of the register-stage kernels: the strided passes of
// demag_fast2.cu (x and y axes) and the tile pass of demag_ztile.cu (z axis).  K1/2 inputs per stage-A
// thread, K2 per stage-B thread; both radices run fully in registers (fft_core.cuh).
#pragma once

namespace mm {

template <int L> struct Plan2;
template <> struct Plan2<64> { static constexpr int K1 = 16, K2 = 8; };
template <> struct Plan2<128> { static constexpr int K1 = 16, K2 = 16; };
template <> struct Plan2<256> { static constexpr int K1 = 32, K2 = 16; };
template <> struct Plan2<512> { static constexpr int K1 = 32, K2 = 32; };
// the paper's own sides: 200 = 20 x 10, 700 = 28 x 25 (5 x 5), 800 = 32 x 25
template <> struct Plan2<100> { static constexpr int K1 = 20, K2 = 10; };
template <> struct Plan2<350> { static constexpr int K1 = 28, K2 = 25; };
template <> struct Plan2<400> { static constexpr int K1 = 32, K2 = 25; };

#define MM_PLAN2_LENGTHS(X) X(64) X(128) X(256) X(512) X(100) X(350) X(400)   // strided passes (x, y)
#define MM_ZTILE_LENGTHS(X) X(350) X(400)                                     // tile pass (z), nz > 256

// run-time view of the table above; false if L has no plan
inline bool plan2_of(int L, int* K1, int* K2) {
  switch (L) {
#define MM_PLAN2_ROW(LL) case LL: *K1 = Plan2<LL>::K1; *K2 = Plan2<LL>::K2; return true;
    MM_PLAN2_LENGTHS(MM_PLAN2_ROW)
#undef MM_PLAN2_ROW
    default: return false;
  }
}

}  // namespace mm
