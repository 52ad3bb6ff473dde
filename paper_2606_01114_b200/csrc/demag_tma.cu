// K1, K2, K4, K5, the strided passes of the x-first demag path (S1, S2, S4, S5; "zero-padding and ...
// FFT ... in the y- and z-directions", "the output is then truncated"), with their tiles moved by the TMA
// engine: 2D cp.async.bulk.tensor boxes of {64 or 128 bytes x up to 256 rows} instead of LDG / STG from every
// lane (BASELINE.json north_star: "TMA or cp.async staging of pencil tiles for the strided y/z passes").
// Same plans and stage arithmetic as demag_fast2.cu (strided2.cuh), bit-identical results.  A persistent CTA
// walks tiles (column block of 64 bytes; K2 / K4: of one kx plane); the box loads of the next tile are issued as
// soon as the input buffer has been read, so they overlap the arithmetic and the stores of the current one.
//   K2: input tile [L rows] -> stage A -> exchange tile -> stage B -> the same buffer in natural row order
//       -> box stores.
//   K4: input tile [2L rows] -> stage B' reads its rows k1 + K1 k2, the tile itself becomes the exchange
//       tile (value bf of thread k1 at row (k1 ^ (bf & 1)) + K1 bf: the four bf of a warp then read rows of
//       both parities, i.e. both 64-byte halves of the banks) -> stage A' -> output tile [L rows] -> box stores.
//   K1: input tile of m [L rows x 64 B] -> stage A -> exchange tile -> stage B + Hermitian separation by warp
//       shuffles -> the same buffer as [L + 1 rows x 128 B] (A[k], B[k] side by side) -> box stores.
//   K5: the mirror image: input tile [L + 1 rows x 128 B] becomes the exchange tile -> output tile of H.
// Columns beyond the end of a row are zero-filled on load and clipped on store by the tensor map.
// Every place where threads have READ a buffer that the next box load will overwrite carries a
// fence.proxy.async before the barrier (see xf2_tma_kernel).
// Measured against the LDG / STG kernels in profiles/r02_tma_strided.md; MM_B200_TMA=0 selects the latter.
#define MM_NO_PACKED_F32
#include <cuda.h>

#include <cstdlib>

#include "bulk_copy.cuh"
#include "demag_fast.cuh"
#include "strided2.cuh"
#include "strided3.cuh"

namespace mm {

namespace {

__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
               ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* map, int c0, int c1, const void* src) {
  asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];" ::"l"(map), "r"(c0),
               "r"(c1), "r"(smem_u32(src))
               : "memory");
}

// rows per box: the largest even divisor of L up to 256 (a box holds at most 256 rows, and a box of 64-byte
// rows must start on a 128-byte boundary of shared memory)
constexpr int box_rows(int L) {
  int r = 2;
  for (int d = 2; d <= 256 && d <= L; d += 2)
    if (L % d == 0) r = d;
  return r;
}

// the root table of the plan, Wt[bf K1 + k1], into shared memory with row pitch TWP (every thread of the CTA; the
// first __syncthreads of the kernel publishes it): a persistent CTA reads it for every tile, and an LDS is not
// behind the global-load path that `long_scoreboard` showed on top in these kernels (profiles/r02_tma_strided.md)
template <typename T, int L> __device__ __forceinline__ void stage_roots(Cx<T>* tws, const Cx<T>* __restrict__ Wt) {
  using TL = Tile2<T, L>;
  for (int i = threadIdx.x; i < TL::K1 * TL::K2; i += blockDim.x) tws[(i / TL::K1) * TL::TWP + i % TL::K1] = __ldg(Wt + i);
}

// dynamic shared memory per CTA that still lets two CTAs share an SM (228 KB per SM, 1 KB reserved per CTA)
constexpr int kTwoCtaSmem = (228 * 1024 - 2 * 1024) / 2;

template <typename T, int L> struct TmaTile {
  using TL = Tile2<T, L>;
  static constexpr int R = box_rows(L);
  static_assert(L % R == 0 && (R * 64) % 128 == 0 && (L * 64) % 128 == 0, "box alignment");
  static constexpr int EW = 64 / (int)sizeof(T);                    // elements of the map's type per 64-byte row
  static constexpr int in2_bytes = L * 64;                          // K2 input tile
  static constexpr int ex_bytes = TL::K1 * TL::K2P * 64;            // exchange tile (>= 2L rows)
  // the root table rides in shared memory where two CTAs still fit with it
  static constexpr bool tws2 = in2_bytes + ex_bytes + 64 + TL::tw_bytes <= kTwoCtaSmem;
  static constexpr int smem2 = in2_bytes + ex_bytes + 64 + (tws2 ? TL::tw_bytes : 0);
  static constexpr int in4_bytes = 2 * L * 64, out4_bytes = L * 64; // K4: input = exchange tile, output tile
  static constexpr bool tws4 = in4_bytes + out4_bytes + 64 + TL::tw_bytes <= kTwoCtaSmem;
  static constexpr int smem4 = in4_bytes + out4_bytes + 64 + (tws4 ? TL::tw_bytes : 0);
  static constexpr int NT = TL::NT;
  // resident CTAs the kernels are compiled for: fp32 three where the tile leaves room (<= 72 KB), else two
  static constexpr int mb2 = sizeof(T) == 8 ? (NT <= 128 ? 2 : 1) : (smem2 <= 72 * 1024 ? 3 : 2);
  static constexpr int mb4 = sizeof(T) == 8 ? (NT <= 128 ? 2 : 1) : (smem4 <= 72 * 1024 ? 3 : 2);
};

// ---------------------------------------------------------------- K2: forward y
// mapIn: A1 as [(nx + 1) ny rows][2 Q reals], box {EW, R}; mapOut: A2 as [(nx + 1) Py rows][2 Q reals].
// STG: rows that do not start on a 32-byte sector (fp32 with nz = 2 mod 4): box stores would be partial-sector
// writes, so the output goes to global memory straight from the registers (outp, Q) as in yf2_kernel; the loads,
// which are what the LDG / STG kernel waits for, still come by boxes one tile ahead.
template <typename T, int L, bool STG>
__global__ void __launch_bounds__(TmaTile<T, L>::NT, TmaTile<T, L>::mb2)
yf2_tma_kernel(const __grid_constant__ CUtensorMap mapIn, const __grid_constant__ CUtensorMap mapOut,
               const Cx<T>* __restrict__ Wt, int colblocks, int ntile, Cx<T>* __restrict__ outp, int Q) {
  using TT = TmaTile<T, L>;
  using TL = Tile2<T, L>;
  constexpr int K1 = TL::K1, K2 = TL::K2, A = TL::A, B = TL::B, R = TT::R;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Cx<T>* in = reinterpret_cast<Cx<T>*>(smem_raw);                        // [L][B]
  Cx<T>* ex = reinterpret_cast<Cx<T>*>(smem_raw + TT::in2_bytes);        // exchange tile, then output [2L][B]
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + TT::in2_bytes + TT::ex_bytes);
  Cx<T>* tws = reinterpret_cast<Cx<T>*>(smem_raw + TT::in2_bytes + TT::ex_bytes + 64);
  const int lane = threadIdx.x % B, slot = threadIdx.x / B;
  if constexpr (TT::tws2) stage_roots<T, L>(tws, Wt);
  auto issue = [&](int tile) {
    const int cb = tile % colblocks, plane = tile / colblocks;
    mbar_expect_tx(bar, TT::in2_bytes);
#pragma unroll
    for (int q = 0; q < L / R; ++q) tma_load_2d(in + q * R * B, &mapIn, cb * TT::EW, plane * L + q * R, bar);
  };
  if (threadIdx.x == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if ((int)blockIdx.x < ntile) issue(blockIdx.x);
  }
  __syncthreads();
  int it = 0;
  for (int tile = blockIdx.x; tile < ntile; tile += gridDim.x, ++it) {
    const int cb = tile % colblocks, plane = tile / colblocks;
    mbar_wait(bar, it & 1);
    Cx<T> v[A];
    if (slot < K2) {
#pragma unroll
      for (int s = 0; s < A; ++s) v[s] = in[(slot + K2 * s) * B + lane];
    }
    // the previous tile's stores must have read the exchange / output buffer before it is overwritten
    if (!STG && threadIdx.x == 0) bulk_wait_read0();
    fence_async_smem();   // the reads above are performed before the next box loads (async proxy) may overwrite the tile
    __syncthreads();   // every thread holds its inputs: the input buffer is free, and so is the output buffer
    if (threadIdx.x == 0 && tile + (int)gridDim.x < ntile) issue(tile + gridDim.x);
    if (slot < K2) fwdA<T, L, TT::tws2>(ex, TT::tws2 ? tws : Wt, lane, slot, v);
    __syncthreads();
    {
      const int k1 = slot < K1 ? slot_k1<K1>(slot) : 0;
      Cx<T> t[K2];
      if (slot < K1) fwdB<T, L>(ex, lane, k1, t);
      __syncthreads();   // the exchange tile has been read: it becomes the output tile, rows in natural order
      if constexpr (STG) {
        const int colq = cb * B + lane;
        if (slot < K1 && colq < Q) {
          Cx<T>* out = outp + (size_t)plane * 2 * L * Q + colq;
#pragma unroll
          for (int k2 = 0; k2 < K2; ++k2) out[(size_t)(k1 + K1 * k2) * Q] = t[k2];
        }
      } else if (slot < K1) {
#pragma unroll
        for (int k2 = 0; k2 < K2; ++k2) ex[(k1 + K1 * k2) * B + lane] = t[k2];
      }
    }
    if constexpr (!STG) {
      fence_async_smem();
      __syncthreads();
      if (threadIdx.x == 0) {
#pragma unroll
        for (int q = 0; q < 2 * L / R; ++q)
          tma_store_2d(&mapOut, cb * TT::EW, plane * 2 * L + q * R, ex + q * R * B);
        bulk_commit();
      }
    }
  }
  if (!STG && threadIdx.x == 0) bulk_wait0();
}

// ---------------------------------------------------------------- K4: inverse y, truncated
// mapIn: A2 as [(nx + 1) Py rows][2 Q reals]; mapOut: A1 as [(nx + 1) ny rows][2 Q reals].
template <typename T, int L, bool STG>
__global__ void __launch_bounds__(TmaTile<T, L>::NT, TmaTile<T, L>::mb4)
yi2_tma_kernel(const __grid_constant__ CUtensorMap mapIn, const __grid_constant__ CUtensorMap mapOut,
               const Cx<T>* __restrict__ Wt, int colblocks, int ntile, Cx<T>* __restrict__ outp, int Q) {
  using TT = TmaTile<T, L>;
  using TL = Tile2<T, L>;
  constexpr int K1 = TL::K1, K2 = TL::K2, A = TL::A, B = TL::B, R = TT::R;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Cx<T>* in = reinterpret_cast<Cx<T>*>(smem_raw);                        // [2L][B], then the exchange tile
  Cx<T>* outb = reinterpret_cast<Cx<T>*>(smem_raw + TT::in4_bytes);      // [L][B]
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + TT::in4_bytes + TT::out4_bytes);
  Cx<T>* tws = reinterpret_cast<Cx<T>*>(smem_raw + TT::in4_bytes + TT::out4_bytes + 64);
  const int lane = threadIdx.x % B, slot = threadIdx.x / B;
  if constexpr (TT::tws4) stage_roots<T, L>(tws, Wt);
  auto issue = [&](int tile) {
    const int cb = tile % colblocks, plane = tile / colblocks;
    mbar_expect_tx(bar, TT::in4_bytes);
#pragma unroll
    for (int q = 0; q < 2 * L / R; ++q) tma_load_2d(in + q * R * B, &mapIn, cb * TT::EW, plane * 2 * L + q * R, bar);
  };
  if (threadIdx.x == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if ((int)blockIdx.x < ntile) issue(blockIdx.x);
  }
  __syncthreads();
  int it = 0;
  for (int tile = blockIdx.x; tile < ntile; tile += gridDim.x, ++it) {
    const int cb = tile % colblocks, plane = tile / colblocks;
    mbar_wait(bar, it & 1);
    {   // stage B': thread k1 = slot
      Cx<T> t[K2];
      if (slot < K1) {
#pragma unroll
        for (int k2 = 0; k2 < K2; ++k2) t[k2] = in[(slot + K1 * k2) * B + lane];
        Dft<T, K2, true>::run(t);
      }
      __syncthreads();   // every input row is in registers: the tile becomes the exchange tile
      if (slot < K1) {
#pragma unroll
        for (int bf = 0; bf < K2; ++bf) in[((slot ^ (bf & 1)) + K1 * bf) * B + lane] = t[bf];
      }
    }
    __syncthreads();
    Cx<T> v[A];
    if (slot < K2) {   // stage A' of bf = slot, truncated to the L wanted samples
      const int bf = slot, sw = bf & 1;
      Cx<T> o[A];
      const Cx<T>* tw = TT::tws4 ? tws + bf * TL::TWP : Wt + bf * K1;
      const Cx<T>* row = in + (K1 * bf) * B + lane;
#pragma unroll
      for (int u = 0; u < A; ++u) {
        Cx<T> w0, w1;
        if constexpr (TT::tws4) Vec2<T>::ld(tw + 2 * u, w0, w1); else Vec2<T>::ldg(tw + 2 * u, w0, w1);
        const Cx<T> a = row[((2 * u) ^ sw) * B], b = row[((2 * u + 1) ^ sw) * B];
        v[u] = u ? cmulc(a, w0) : a;
        o[u] = cmulc(b, w1);
      }
      Dft<T, A, true>::run(v);
      Dft<T, A, true>::run(o);
      rot_inv_add<T, K1>(v, o, std::make_integer_sequence<int, A>{});
    }
    // the previous tile's stores must have read the output buffer before it is overwritten
    if (!STG && threadIdx.x == 0) bulk_wait_read0();
    fence_async_smem();   // reads of the exchange tile performed before the async proxy overwrites it
    __syncthreads();   // the exchange tile has been read: the loads of the next tile may land in it
    if (threadIdx.x == 0 && tile + (int)gridDim.x < ntile) issue(tile + gridDim.x);
    if constexpr (STG) {
      const int colq = cb * B + lane;
      if (slot < K2 && colq < Q) {
        Cx<T>* out = outp + (size_t)plane * L * Q + colq;
#pragma unroll
        for (int s = 0; s < A; ++s) out[(size_t)(slot + K2 * s) * Q] = v[s];
      }
    } else {
      if (slot < K2) {
#pragma unroll
        for (int s = 0; s < A; ++s) outb[(slot + K2 * s) * B + lane] = v[s];
      }
      fence_async_smem();
      __syncthreads();
      if (threadIdx.x == 0) {
#pragma unroll
        for (int q = 0; q < L / R; ++q) tma_store_2d(&mapOut, cb * TT::EW, plane * L + q * R, outb + q * R * B);
        bulk_commit();
      }
    }
  }
  if (!STG && threadIdx.x == 0) bulk_wait0();
}

// ---------------------------------------------------------------- K1: forward x, r2c
// Same arithmetic as xf2_kernel (demag_fast2.cu: two real columns ride as one complex column and are separated by
// Hermitian symmetry with warp shuffles).  mapIn: m as [nx rows][ny Q reals], box {EW, R}; mapOut: A1 as
// [(nx + 1) rows][2 ny Q reals], box {2 EW, R}; mapRow: the same array with a box of one row, for the row k = L.
// The exchange tile becomes the output tile [L + 1 rows][2 B complex] once stage B has read it.
template <typename T, int L> struct TmaTileX {
  using TL = Tile2<T, L>;
  using TT = TmaTile<T, L>;
  static constexpr int io_bytes = (L + 1) * 128;                    // the tile of A1: rows k <= L of 128 bytes
  static constexpr int ex_bytes = (TT::ex_bytes > io_bytes ? TT::ex_bytes : io_bytes + 127) / 128 * 128;
  static constexpr bool tws1 = TT::in2_bytes + ex_bytes + 64 + TL::tw_bytes <= kTwoCtaSmem;   // root table in shared memory
  static constexpr bool tws5 = ex_bytes + TT::out4_bytes + 64 + TL::tw_bytes <= kTwoCtaSmem;
  static constexpr int smem1 = TT::in2_bytes + ex_bytes + 64 + (tws1 ? TL::tw_bytes : 0);   // K1: input tile of m, exchange / output tile
  static constexpr int smem5 = ex_bytes + TT::out4_bytes + 64 + (tws5 ? TL::tw_bytes : 0);  // K5: input / exchange tile, output tile of H
  static constexpr int NT = TL::NT;
  static constexpr int mb1 = sizeof(T) == 8 ? (NT <= 128 ? 2 : 1) : (smem1 <= 72 * 1024 ? 3 : 2);
  static constexpr int mb5 = sizeof(T) == 8 ? (NT <= 128 ? 2 : 1) : (smem5 <= 72 * 1024 ? 3 : 2);
};

template <typename T> __device__ __forceinline__ Cx<T> shfl_xor_cx(Cx<T> v, int m) {
  Cx<T> r;
  r.x = __shfl_xor_sync(0xffffffffu, v.x, m);
  r.y = __shfl_xor_sync(0xffffffffu, v.y, m);
  return r;
}

template <typename T, int L>
__global__ void __launch_bounds__(TmaTileX<T, L>::NT, TmaTileX<T, L>::mb1)
xf2_tma_kernel(const __grid_constant__ CUtensorMap mapIn, const __grid_constant__ CUtensorMap mapOut,
               const __grid_constant__ CUtensorMap mapRow, const Cx<T>* __restrict__ Wt, int ntile) {
  using TT = TmaTile<T, L>;
  using TX = TmaTileX<T, L>;
  using TL = Tile2<T, L>;
  constexpr int K1 = TL::K1, K2 = TL::K2, A = TL::A, B = TL::B, R = TT::R, JN = TL::JN;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Cx<T>* in = reinterpret_cast<Cx<T>*>(smem_raw);                        // [L][B]
  Cx<T>* ex = reinterpret_cast<Cx<T>*>(smem_raw + TT::in2_bytes);        // exchange tile, then output [L + 1][2 B]
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + TT::in2_bytes + TX::ex_bytes);
  Cx<T>* tws = reinterpret_cast<Cx<T>*>(smem_raw + TT::in2_bytes + TX::ex_bytes + 64);
  const int lane = threadIdx.x % B, slot = threadIdx.x / B;
  if constexpr (TX::tws1) stage_roots<T, L>(tws, Wt);
  auto issue = [&](int tile) {
    mbar_expect_tx(bar, TT::in2_bytes);
#pragma unroll
    for (int q = 0; q < L / R; ++q) tma_load_2d(in + q * R * B, &mapIn, tile * TT::EW, q * R, bar);
  };
  if (threadIdx.x == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if ((int)blockIdx.x < ntile) issue(blockIdx.x);
  }
  __syncthreads();
  int it = 0;
  for (int tile = blockIdx.x; tile < ntile; tile += gridDim.x, ++it) {
    mbar_wait(bar, it & 1);
    Cx<T> v[A];
    if (slot < K2) {
#pragma unroll
      for (int s = 0; s < A; ++s) v[s] = in[(slot + K2 * s) * B + lane];
    }
    if (threadIdx.x == 0) bulk_wait_read0();   // the previous tile's stores have read the output tile
    // Generic-proxy reads followed by an async-proxy write of the same shared memory need a proxy fence: the
    // barrier alone does not wait for loads that have been issued but not performed.  Without it the box load
    // of the next tile was seen to overwrite a row before its LDS executed (about one tile in 1e5, fp64).
    fence_async_smem();
    __syncthreads();                           // the input tile is in registers
    if (threadIdx.x == 0 && tile + (int)gridDim.x < ntile) issue(tile + gridDim.x);
    if (slot < K2) fwdA<T, L, TX::tws1>(ex, TX::tws1 ? tws : Wt, lane, slot, v);
    __syncthreads();
    const bool live = slot < K1;
    const int k1 = slot_k1<K1>(live ? slot : 0);
    Cx<T> t[K2];
    if (slot < TL::slotsB) fwdB<T, L>(ex, lane, k1, t);
    __syncthreads();   // the exchange tile has been read: it becomes the output tile
    if (slot < TL::slotsB) {   // whole warps: every lane takes part in the shuffles
      const bool pair0 = (slot >> 1) == 0, odd = slot & 1;
      Cx<T>* orow = ex + 2 * lane;
#pragma unroll
      for (int j = 0; j < JN; ++j) {
        if (K2 % 2 == 0 && j == K2 / 2) {   // even K2: the last j holds only k = L (k1 = 0), its own mirror
          if (live && k1 == 0) {
            const Cx<T> z = t[j % K2];
            Vec2<T>::st(orow + (size_t)L * 2 * B, mk<T>(2 * z.x, (T)0), mk<T>(2 * z.y, (T)0));
          }
          continue;
        }
        const Cx<T> r = shfl_xor_cx<T>(t[(2 * K2 - 1 - j) % K2], B);
        const Cx<T> own = odd ? t[(2 * K2 - 1 - j) % K2] : t[(K2 - j) % K2];
        if (live && TL::has_row(j, pair0, odd)) {
          const Cx<T> z = t[j % K2], zm = cconj(pair0 ? own : r);
          const Cx<T> s = cadd(z, zm), d = csub(z, zm);
          Vec2<T>::st(orow + (size_t)(k1 + K1 * j) * 2 * B, s, mk<T>(d.y, -d.x));
        }
      }
    }
    fence_async_smem();
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
      for (int q = 0; q < L / R; ++q) tma_store_2d(&mapOut, tile * 2 * TT::EW, q * R, ex + q * R * 2 * B);
      tma_store_2d(&mapRow, tile * 2 * TT::EW, L, ex + L * 2 * B);
      bulk_commit();
    }
  }
  if (threadIdx.x == 0) bulk_wait0();
}

// ---------------------------------------------------------------- K5: inverse x, c2r, truncated
// Same arithmetic as xi2_kernel.  mapIn / mapRow: A1 as for K1; mapOut: H as [nx rows][ny Q reals], box {EW, R}.
// The input tile [L + 1][2 B] becomes the exchange tile once every stage-B' thread holds its rows.
template <typename T, int L>
__global__ void __launch_bounds__(TmaTileX<T, L>::NT, TmaTileX<T, L>::mb5)
xi2_tma_kernel(const __grid_constant__ CUtensorMap mapIn, const __grid_constant__ CUtensorMap mapRow,
               const __grid_constant__ CUtensorMap mapOut, const Cx<T>* __restrict__ Wt, T scale, int ntile) {
  using TT = TmaTile<T, L>;
  using TX = TmaTileX<T, L>;
  using TL = Tile2<T, L>;
  constexpr int K1 = TL::K1, K2 = TL::K2, A = TL::A, B = TL::B, R = TT::R, JN = TL::JN;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Cx<T>* in = reinterpret_cast<Cx<T>*>(smem_raw);                        // [L + 1][2 B], then the exchange tile
  Cx<T>* outb = reinterpret_cast<Cx<T>*>(smem_raw + TX::ex_bytes);       // [L][B]
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + TX::ex_bytes + TT::out4_bytes);
  Cx<T>* tws = reinterpret_cast<Cx<T>*>(smem_raw + TX::ex_bytes + TT::out4_bytes + 64);
  const int lane = threadIdx.x % B, slot = threadIdx.x / B;
  if constexpr (TX::tws5) stage_roots<T, L>(tws, Wt);
  auto issue = [&](int tile) {
    mbar_expect_tx(bar, TX::io_bytes);
#pragma unroll
    for (int q = 0; q < L / R; ++q) tma_load_2d(in + q * R * 2 * B, &mapIn, tile * 2 * TT::EW, q * R, bar);
    tma_load_2d(in + L * 2 * B, &mapRow, tile * 2 * TT::EW, L, bar);
  };
  if (threadIdx.x == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if ((int)blockIdx.x < ntile) issue(blockIdx.x);
  }
  __syncthreads();
  int it = 0;
  for (int tile = blockIdx.x; tile < ntile; tile += gridDim.x, ++it) {
    mbar_wait(bar, it & 1);
    const bool live = slot < K1;
    const int k1 = slot_k1<K1>(live ? slot : 0);
    Cx<T> t[K2];
    if (slot < TL::slotsB) {   // whole warps: every lane takes part in the shuffles
      const bool pair0 = (slot >> 1) == 0, odd = slot & 1;
      const Cx<T>* irow = in + 2 * lane;
      Cx<T> a[JN], b[JN];
#pragma unroll
      for (int j = 0; j < JN; ++j) {
        const bool last_even = K2 % 2 == 0 && j == K2 / 2;   // only k = L of k1 = 0
        if (live && (last_even ? k1 == 0 : TL::has_row(j, pair0, odd)))
          Vec2<T>::ld(irow + (size_t)(k1 + K1 * j) * 2 * B, a[j], b[j]);
        else a[j] = b[j] = mk<T>((T)0, (T)0);
      }
#pragma unroll
      for (int k2 = 0; k2 < K2; ++k2) t[k2] = mk<T>((T)0, (T)0);
#pragma unroll
      for (int j = 0; j < JN; ++j) {
        if (K2 % 2 == 0 && j == K2 / 2) {   // k = L (k1 = 0): its own mirror
          if (k1 == 0) t[j % K2] = mk<T>(a[j].x - b[j].y, a[j].y + b[j].x);
          continue;
        }
        const Cx<T> S = mk<T>(a[j].x + b[j].y, b[j].x - a[j].y);
        const Cx<T> r = shfl_xor_cx<T>(S, B);
        if (!pair0) { if (TL::has_row(j, false, !odd)) t[(2 * K2 - 1 - j) % K2] = r; }
        else if (odd) { if (!(K2 % 2 == 1 && j == K2 / 2)) t[(2 * K2 - 1 - j) % K2] = S; }
        else if (j >= 1) t[(K2 - j) % K2] = S;
        if (TL::has_row(j, pair0, odd)) t[j % K2] = mk<T>(a[j].x - b[j].y, a[j].y + b[j].x);
      }
    }
    __syncthreads();   // every input row is in registers: the tile becomes the exchange tile
    if (live) invB<T, L>(in, lane, k1, t);
    __syncthreads();
    Cx<T> v[A];
    if (slot < K2) invA<T, L, TX::tws5>(in, TX::tws5 ? tws : Wt, lane, slot, v);
    if (threadIdx.x == 0) bulk_wait_read0();   // the previous tile's stores have read the output buffer
    fence_async_smem();                        // reads of the exchange tile performed before the async proxy overwrites it
    __syncthreads();                           // the exchange tile has been read: the next tile may land in it
    if (threadIdx.x == 0 && tile + (int)gridDim.x < ntile) issue(tile + gridDim.x);
    if (slot < K2) {
#pragma unroll
      for (int s = 0; s < A; ++s) outb[(slot + K2 * s) * B + lane] = mk<T>(scale * v[s].x, scale * v[s].y);
    }
    fence_async_smem();
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
      for (int q = 0; q < L / R; ++q) tma_store_2d(&mapOut, tile * TT::EW, q * R, outb + q * R * B);
      bulk_commit();
    }
  }
  if (threadIdx.x == 0) bulk_wait0();
}

// ---------------------------------------------------------------- L = 1024: three-stage passes by boxes
// The tile of the three-stage kernels (demag_fast.cu) is 2L rows x 64 B = 128 KB: one CTA per SM, whose global
// loads, transform and stores then run one after the other (0.43-0.57 of the roofline, profiles/r01_*).  Here a
// persistent CTA keeps a separate 64 KB input tile that the box loads of the NEXT tile fill while the current one
// is transformed, and the result leaves by box stores from the transform tile.  Rows of a tile that the boxes
// move are in global order (no XOR swizzle): the accesses of the last / first stage, whose four (fp32) or eight
// (fp64) tasks of a warp touch rows of equal parity, swap the order of each row pair in odd slots instead.
// shared-memory row (swizzled) of frequency k < 2L in the three-stage tile: what the host tables posx / posy hold
// (demag_fast.cu: fast_swizzle(fast_pos_logical(k))), as arithmetic instead of a dependent table load
template <int L> __device__ __forceinline__ int pos3(int k) {
  using P = FastPlan<L>;
  constexpr int l1 = ilog2c(P::R1), l2 = ilog2c(P::R2), l3 = ilog2c(P::R3);
  const int h = k & 1, kk = k >> 1;
  const int u1 = kk & (P::R1 - 1), u2 = (kk >> l1) & (P::R2 - 1), u3 = kk >> (l1 + l2);
  const int row = h * L + (u1 << (l2 + l3)) + (u2 << l3) + u3;
  return row ^ ((row >> l3) & 1);
}

template <typename T, int L> struct Tma3 {
  using TL = Tile<T, L>;
  static constexpr int R = 256;                                   // rows per box
  static constexpr int EW = 64 / (int)sizeof(T);
  static constexpr int in_bytes = L * 64, sm_bytes = 2 * L * 64;
  static constexpr int smem2 = in_bytes + sm_bytes + 64;
  static constexpr int NT = TL::NT;
  static_assert(L % R == 0, "box rows");
};

// K2: forward y.  mapIn: A1 as [(nx + 1) L rows][2 Q reals], mapOut: A2 as [(nx + 1) 2L rows][2 Q reals]; box {EW, R}.
template <typename T, int L>
__global__ void __launch_bounds__(Tma3<T, L>::NT, 1)
yf3_tma_kernel(const __grid_constant__ CUtensorMap mapIn, const __grid_constant__ CUtensorMap mapOut,
               const Cx<T>* __restrict__ W, int colblocks, int ntile) {
  using TT = Tma3<T, L>;
  using TL = Tile<T, L>;
  constexpr int R1 = TL::R1, R2 = TL::R2, R3 = TL::R3, q1 = TL::q1, B = TL::B, NS = TL::NS, R = TT::R;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Cx<T>* in = reinterpret_cast<Cx<T>*>(smem_raw);                        // [L][B], global row order
  Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw + TT::in_bytes);         // [2L][B], swizzled; global order at the end
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + TT::in_bytes + TT::sm_bytes);
  const int lane = threadIdx.x % B, slot = threadIdx.x / B, sp = slot & 1;
  auto issue = [&](int tile) {
    const int cb = tile % colblocks, plane = tile / colblocks;
    mbar_expect_tx(bar, TT::in_bytes);
#pragma unroll
    for (int q = 0; q < L / R; ++q) tma_load_2d(in + q * R * B, &mapIn, cb * TT::EW, plane * L + q * R, bar);
  };
  if (threadIdx.x == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if ((int)blockIdx.x < ntile) issue(blockIdx.x);
  }
  __syncthreads();
  int it = 0;
  for (int tile = blockIdx.x; tile < ntile; tile += gridDim.x, ++it) {
    const int cb = tile % colblocks, plane = tile / colblocks;
    if (threadIdx.x == 0) bulk_wait_read0();   // the previous tile's stores have read the transform tile
    mbar_wait(bar, it & 1);
    __syncthreads();
#pragma unroll 1
    for (int bf = slot; bf < q1; bf += NS) {
      Cx<T> v[R1];
#pragma unroll
      for (int s = 0; s < R1; ++s) v[s] = in[(bf + q1 * s) * B + lane];
      fwd_first<T, L>(sm, W, lane, bf, v);
    }
    fence_async_smem();   // the reads of the input tile are performed before the next box loads overwrite it
    __syncthreads();
    if (threadIdx.x == 0 && tile + (int)gridDim.x < ntile) issue(tile + gridDim.x);
    fwd_middle<T, L>(sm, W, lane, slot);
    __syncthreads();
#pragma unroll 1
    for (int i = slot; i < 2 * R1 * R2; i += NS) {   // NS is even: the parity of a thread's tasks is that of its slot
      Cx<T> v[R3];
      fwd_last<T, L>(sm, lane, i, v);
      // rows i R3 + u in global order; odd slots write each row pair in swapped order (both bank halves busy)
      Cx<T>* o = sm + (size_t)i * R3 * B + lane;
#pragma unroll
      for (int u = 0; u < R3; u += 2) {
        const Cx<T> a = sp ? v[u + 1] : v[u], b = sp ? v[u] : v[u + 1];
        o[(u + sp) * B] = a;
        o[(u + 1 - sp) * B] = b;
      }
    }
    fence_async_smem();
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
      for (int q = 0; q < 2 * L / R; ++q) tma_store_2d(&mapOut, cb * TT::EW, plane * 2 * L + q * R, sm + q * R * B);
      bulk_commit();
    }
  }
  if (threadIdx.x == 0) bulk_wait0();
}

// K4 at L = 1024: inverse y, truncated.  The 2L spectrum rows of a tile land in the transform tile itself by box
// loads (global row order), in two halves with a barrier each: the first stage works in place on the even-output
// half while the odd half is still in flight.  The L output rows leave from a separate 64 KB tile by box stores
// that overlap the loads of the next tile, which are issued as soon as the last stage has read the transform tile.
// Against yi_fast_kernel (LDG / STG): the loads are all in flight at once instead of 16 per thread in four
// rounds (`long_scoreboard` was 45 % of its stall samples, profiles/r02_l1024.md).
template <typename T, int L>
__global__ void __launch_bounds__(Tma3<T, L>::NT, 1)
yi3_tma_kernel(const __grid_constant__ CUtensorMap mapIn, const __grid_constant__ CUtensorMap mapOut,
               const Cx<T>* __restrict__ W, int colblocks, int ntile) {
  using TT = Tma3<T, L>;
  using TL = Tile<T, L>;
  constexpr int R1 = TL::R1, R2 = TL::R2, R3 = TL::R3, q1 = TL::q1, B = TL::B, NS = TL::NS, R = TT::R;
  static_assert((R1 * R2) % NS == 0 && NS % 2 == 0, "a thread's first-stage tasks keep the parity of its slot and split evenly over the halves");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw);                        // [2L][B]: global order on arrival, then swizzled
  Cx<T>* outb = reinterpret_cast<Cx<T>*>(smem_raw + TT::sm_bytes);       // [L][B]
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + TT::sm_bytes + TT::in_bytes);   // even half, odd half
  const int lane = threadIdx.x % B, slot = threadIdx.x / B, sp = slot & 1;
  auto issue = [&](int tile) {
    const int cb = tile % colblocks, plane = tile / colblocks;
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      mbar_expect_tx(bars + h, TT::in_bytes);
#pragma unroll
      for (int q = 0; q < L / R; ++q)
        tma_load_2d(sm + (h * L + q * R) * B, &mapIn, cb * TT::EW, plane * 2 * L + h * L + q * R, bars + h);
    }
  };
  if (threadIdx.x == 0) {
    mbar_init(bars, 1);
    mbar_init(bars + 1, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if ((int)blockIdx.x < ntile) issue(blockIdx.x);
  }
  __syncthreads();
  int it = 0;
  for (int tile = blockIdx.x; tile < ntile; tile += gridDim.x, ++it) {
    const int cb = tile % colblocks, plane = tile / colblocks;
#pragma unroll 1
    for (int h = 0; h < 2; ++h) {
      mbar_wait(bars + h, it & 1);
#pragma unroll 1
      for (int i = h * R1 * R2 + slot; i < (h + 1) * R1 * R2; i += NS) {
        // rows i R3 + u in global order; odd slots read each row pair in swapped order (both bank halves busy)
        Cx<T> v[R3];
        const Cx<T>* r = sm + (size_t)i * R3 * B + lane;
#pragma unroll
        for (int u = 0; u < R3; u += 2) {
          const Cx<T> a = r[(u + sp) * B], b = r[(u + 1 - sp) * B];
          v[u] = sp ? b : a;
          v[u + 1] = sp ? a : b;
        }
        inv_first<T, L>(sm, lane, i, v);   // in place: the task's own eight rows, now swizzled
      }
    }
    if (threadIdx.x == 0) bulk_wait_read0();   // the previous tile's stores have read the output tile
    __syncthreads();
    inv_middle<T, L>(sm, W, lane, slot);
    __syncthreads();
#pragma unroll 1
    for (int bf = slot; bf < q1; bf += NS) {
      Cx<T> v[R1];
      inv_last<T, L>(sm, W, lane, bf, v);
#pragma unroll
      for (int s = 0; s < R1; ++s) outb[(bf + q1 * s) * B + lane] = v[s];
    }
    fence_async_smem();   // reads of the transform tile performed before the next loads; output tile visible to the stores
    __syncthreads();
    if (threadIdx.x == 0) {
      if (tile + (int)gridDim.x < ntile) issue(tile + gridDim.x);
#pragma unroll
      for (int q = 0; q < L / R; ++q) tma_store_2d(&mapOut, cb * TT::EW, plane * L + q * R, outb + q * R * B);
      bulk_commit();
    }
  }
  if (threadIdx.x == 0) bulk_wait0();
}

// K5 at L = 1024: inverse x, c2r, truncated.  The spectrum rows k <= L of a tile (128 bytes each: A[k], B[k] side by
// side) arrive by box loads in two halves through one 64 KB landing buffer: the rows of even k (513 of them; a
// tensor map over every second row of A1) are scattered into the even-output half of the transform tile as
// Z[k] = A + i B and Z[2L - k] = conj A + i conj B, and the first two stages run on that half while the rows of
// odd k land; the second half likewise overlaps the loads of the next tile's first half.  The L output rows go
// straight to global memory (no room for an output tile).  Against xi_fast_kernel: 0.42 -> see profiles/r02_l1024.md.
template <typename T, int L> struct Tma3X {
  using TL = Tile<T, L>;
  static constexpr int land_bytes = ((L / 2 + 1) * 128 + 127) / 128 * 128;   // rows of even k: L / 2 + 1
  static constexpr int smem5 = land_bytes + 2 * L * 64 + 64;
};

// inverse middle stage of the tasks [lo, hi) (strided3.cuh: inv_middle runs all 2 R1 q2 of them)
template <typename T, int L>
__device__ __forceinline__ void inv_middle_range(Cx<T>* sm, const Cx<T>* __restrict__ W, int lane, int slot, int lo, int hi) {
  using TL = Tile<T, L>;
  constexpr int R1 = TL::R1, R2 = TL::R2, q1 = TL::q1, q2 = TL::q2, B = TL::B, NS = TL::NS;
#pragma unroll 1
  for (int i = lo + slot; i < hi; i += NS) {
    const int t2 = i % q2, hu = i / q2;
    const int b0 = hu * q1 + t2, b1 = b0 ^ 1;
    Cx<T> v[R2];
#pragma unroll
    for (int u = 0; u < R2; ++u) v[u] = sm[(((u & 1) ? b1 : b0) + q2 * u) * B + lane];
#pragma unroll
    for (int u = 1; u < R2; ++u) v[u] = cmulc(v[u], __ldg(W + 2 * R1 * t2 * u));
    Dft<T, R2, true>::run(v);
#pragma unroll
    for (int s2 = 0; s2 < R2; ++s2) sm[(((s2 & 1) ? b1 : b0) + q2 * s2) * B + lane] = v[s2];
  }
}

template <typename T, int L>
__global__ void __launch_bounds__(Tma3<T, L>::NT, 1)
xi3_tma_kernel(const __grid_constant__ CUtensorMap mapEven, const __grid_constant__ CUtensorMap mapEvenLast,
               const __grid_constant__ CUtensorMap mapOdd, Cx<T>* __restrict__ Hp, const Cx<T>* __restrict__ W,
               size_t npairs, T scale, int ntile) {
  using TT = Tma3<T, L>;
  using TX = Tma3X<T, L>;
  using TL = Tile<T, L>;
  constexpr int R1 = TL::R1, R2 = TL::R2, R3 = TL::R3, q1 = TL::q1, q2 = TL::q2, B = TL::B, NS = TL::NS, R = TT::R;
  constexpr int H = L / 2;   // rows per half (+ the row k = L in the even half)
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Cx<T>* land = reinterpret_cast<Cx<T>*>(smem_raw);                      // [H + 1][2 B]
  Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw + TX::land_bytes);       // [2L][B], swizzled
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + TX::land_bytes + TT::sm_bytes);
  const int lane = threadIdx.x % B, slot = threadIdx.x / B;
  auto issue = [&](int tile, int odd) {
    mbar_expect_tx(bar, (H + (odd ? 0 : 1)) * 128);
#pragma unroll
    for (int q = 0; q < H / R; ++q) tma_load_2d(land + q * R * 2 * B, odd ? &mapOdd : &mapEven, tile * 2 * TT::EW, q * R, bar);
    if (!odd) tma_load_2d(land + H * 2 * B, &mapEvenLast, tile * 2 * TT::EW, H, bar);
  };
  // rows j of the landing buffer hold k = 2 j + odd: Z[k] and its mirror Z[2L - k] into the transform tile
  auto scatter = [&](int odd) {
#pragma unroll 2
    for (int j = slot; j < H + (odd ? 0 : 1); j += NS) {
      const int k = 2 * j + odd;
      Cx<T> a, b;
      Vec2<T>::ld(land + (size_t)j * 2 * B + 2 * lane, a, b);
      sm[pos3<L>(k) * B + lane] = mk<T>(a.x - b.y, a.y + b.x);
      if (k != 0 && k != L) sm[pos3<L>(2 * L - k) * B + lane] = mk<T>(a.x + b.y, b.x - a.y);
    }
  };
  if (threadIdx.x == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if ((int)blockIdx.x < ntile) issue(blockIdx.x, 0);
  }
  __syncthreads();
  for (int tile = blockIdx.x; tile < ntile; tile += gridDim.x) {
    const bool ok = (size_t)tile * B + lane < npairs;
    const size_t pair = ok ? (size_t)tile * B + lane : 0;
#pragma unroll 1
    for (int h = 0; h < 2; ++h) {
      mbar_wait(bar, h);   // two phases per tile: even rows (parity 0), odd rows (parity 1)
      scatter(h);
      fence_async_smem();   // the landing buffer has been read before the next loads overwrite it
      __syncthreads();
      if (threadIdx.x == 0) {
        if (h == 0) issue(tile, 1);
        else if (tile + (int)gridDim.x < ntile) issue(tile + gridDim.x, 0);
      }
#pragma unroll 1
      for (int i = h * R1 * R2 + slot; i < (h + 1) * R1 * R2; i += NS) {
        Cx<T> v[R3];
        const int g = i & 1, base = i * R3, pe = base + g, po = base - g;
#pragma unroll
        for (int u = 0; u < R3; ++u) v[u] = sm[(((u & 1) ? po : pe) + u) * B + lane];
        inv_first<T, L>(sm, lane, i, v);
      }
      __syncthreads();
      inv_middle_range<T, L>(sm, W, lane, slot, h * R1 * q2, (h + 1) * R1 * q2);
    }
    __syncthreads();
    Cx<T>* out = Hp + pair;
#pragma unroll 1
    for (int bf = slot; bf < q1; bf += NS) {
      Cx<T> v[R1];
      inv_last<T, L>(sm, W, lane, bf, v);
      if (ok) {
#pragma unroll
        for (int s2 = 0; s2 < R1; ++s2) out[(size_t)(bf + q1 * s2) * npairs] = mk<T>(scale * v[s2].x, scale * v[s2].y);
      }
    }
    __syncthreads();   // the transform tile has been read: the next tile's scatter may overwrite it
  }
}

// K1 at L = 1024: forward x, r2c.  The input tile of m arrives by box loads one tile ahead (mapIn: m as [nx rows]
// [ny Q reals], box {EW, R}); the Hermitian separation reads the transform tile through `pos` and stores straight
// to global memory, 128 bytes per row and tile, as xf_fast_kernel does (an output tile of (L + 1) x 128 bytes
// does not fit beside the two others).
template <typename T, int L>
__global__ void __launch_bounds__(Tma3<T, L>::NT, 1)
xf3_tma_kernel(const __grid_constant__ CUtensorMap mapIn, Cx<T>* __restrict__ A1, const Cx<T>* __restrict__ W,
               size_t npairs, int ntile) {
  using TT = Tma3<T, L>;
  using TL = Tile<T, L>;
  constexpr int R1 = TL::R1, R2 = TL::R2, R3 = TL::R3, q1 = TL::q1, B = TL::B, NS = TL::NS, R = TT::R;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Cx<T>* in = reinterpret_cast<Cx<T>*>(smem_raw);                        // [L][B], global row order
  Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw + TT::in_bytes);         // [2L][B], swizzled
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + TT::in_bytes + TT::sm_bytes);
  const int lane = threadIdx.x % B, slot = threadIdx.x / B;
  auto issue = [&](int tile) {
    mbar_expect_tx(bar, TT::in_bytes);
#pragma unroll
    for (int q = 0; q < L / R; ++q) tma_load_2d(in + q * R * B, &mapIn, tile * TT::EW, q * R, bar);
  };
  if (threadIdx.x == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if ((int)blockIdx.x < ntile) issue(blockIdx.x);
  }
  __syncthreads();
  int it = 0;
  for (int tile = blockIdx.x; tile < ntile; tile += gridDim.x, ++it) {
    const bool ok = (size_t)tile * B + lane < npairs;
    const size_t pair = ok ? (size_t)tile * B + lane : 0;
    mbar_wait(bar, it & 1);
#pragma unroll 1
    for (int bf = slot; bf < q1; bf += NS) {
      Cx<T> v[R1];
#pragma unroll
      for (int s = 0; s < R1; ++s) v[s] = in[(bf + q1 * s) * B + lane];
      fwd_first<T, L>(sm, W, lane, bf, v);
    }
    fence_async_smem();   // the reads of the input tile are performed before the next box loads overwrite it
    __syncthreads();
    if (threadIdx.x == 0 && tile + (int)gridDim.x < ntile) issue(tile + gridDim.x);
    fwd_middle<T, L>(sm, W, lane, slot);
    __syncthreads();
#pragma unroll 1
    for (int i = slot; i < 2 * R1 * R2; i += NS) {
      Cx<T> v[R3];
      fwd_last<T, L>(sm, lane, i, v);
      const int g = i & 1, base = i * R3, pe = base + g, po = base - g;
#pragma unroll
      for (int u = 0; u < R3; ++u) sm[(((u & 1) ? po : pe) + u) * B + lane] = v[u];
    }
    __syncthreads();
    Cx<T>* out = A1 + 2 * pair;
    const size_t rowc = 2 * npairs;
#pragma unroll 4
    for (int k = slot; k <= L; k += NS) {
      const int p1 = pos3<L>(k), p2 = pos3<L>((2 * L - k) & (2 * L - 1));
      const Cx<T> z1 = sm[p1 * B + lane], z2 = cconj(sm[p2 * B + lane]);
      const Cx<T> s = cadd(z1, z2), d = csub(z1, z2);
      if (ok)
        Vec2<T>::st(out + (size_t)k * rowc, mk<T>((T)0.5 * s.x, (T)0.5 * s.y), mk<T>((T)0.5 * d.y, (T)-0.5 * d.x));
    }
    __syncthreads();   // the transform tile has been read: the next tile's first stage may overwrite it
  }
}

// ---------------------------------------------------------------- host side

typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                             const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                             CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeFn encode_fn() {
  static EncodeFn fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeFn>(p);
  }
  return fn;
}

// [rows][row_reals] reals; box {box_bytes, R rows}
template <typename T> bool make_map_rows(CUtensorMap* map, const void* base, size_t rows, size_t row_reals, int box_bytes,
                                         int R) {
  EncodeFn fn = encode_fn();
  if (!fn) return false;
  const cuuint64_t dims[2] = {(cuuint64_t)row_reals, (cuuint64_t)rows};
  const cuuint64_t strides[1] = {(cuuint64_t)row_reals * sizeof(T)};
  const cuuint32_t box[2] = {(cuuint32_t)(box_bytes / sizeof(T)), (cuuint32_t)R}, estr[2] = {1, 1};
  return fn(map, sizeof(T) == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2,
            const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
            CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
// [rows][Q complex] viewed as rows of 2 Q reals; box {64 bytes, R rows}
template <typename T> bool make_map(CUtensorMap* map, void* base, size_t rows, int Q, int R) {
  return make_map_rows<T>(map, base, rows, (size_t)2 * Q, 64, R);
}

int sm_count_tma() {
  static int sms = 0;
  if (!sms) {
    int dev = 0;
    cudaGetDevice(&dev);
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) sms = 148;
  }
  return sms;
}

template <typename T, int L, bool STG>
cudaError_t launch_tma_y(int which, const FastGeom& g, const FastBufs<T>& b, const CUtensorMap& mapA1, const CUtensorMap& mapA2,
                         cudaStream_t st) {
  using TT = TmaTile<T, L>;
  using TL = Tile2<T, L>;
  const int colblocks = (g.Q + TL::B - 1) / TL::B, ntile = colblocks * (g.nx + 1);
  cudaError_t e;
  int per_sm = 1;   // persistent grid = what is resident at once (registers and shared memory)
  if (which == 1) {
    if ((e = cudaFuncSetAttribute(yf2_tma_kernel<T, L, STG>, cudaFuncAttributeMaxDynamicSharedMemorySize, TT::smem2)) != cudaSuccess) return e;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, yf2_tma_kernel<T, L, STG>, TT::NT, TT::smem2) != cudaSuccess || per_sm < 1) per_sm = 1;
    int grid = per_sm * sm_count_tma();
    if (grid > ntile) grid = ntile;
    yf2_tma_kernel<T, L, STG><<<grid, TT::NT, TT::smem2, st>>>(mapA1, mapA2, b.T2y, colblocks, ntile, b.A2, g.Q);
  } else {
    if ((e = cudaFuncSetAttribute(yi2_tma_kernel<T, L, STG>, cudaFuncAttributeMaxDynamicSharedMemorySize, TT::smem4)) != cudaSuccess) return e;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, yi2_tma_kernel<T, L, STG>, TT::NT, TT::smem4) != cudaSuccess || per_sm < 1) per_sm = 1;
    int grid = per_sm * sm_count_tma();
    if (grid > ntile) grid = ntile;
    yi2_tma_kernel<T, L, STG><<<grid, TT::NT, TT::smem4, st>>>(mapA2, mapA1, b.T2y, colblocks, ntile, b.A1, g.Q);
  }
  return cudaSuccess;
}

template <typename T, int L>
cudaError_t launch_tma(int which, const FastGeom& g, const FastBufs<T>& b, cudaStream_t st) {
  using TT = TmaTile<T, L>;
  alignas(64) CUtensorMap mapA1, mapA2;
  if (!make_map<T>(&mapA1, b.A1, (size_t)(g.nx + 1) * g.ny, g.Q, TT::R) ||
      !make_map<T>(&mapA2, b.A2, (size_t)(g.nx + 1) * g.Py, g.Q, TT::R))
    return cudaErrorNotSupported;
  // rows must start on a 32-byte sector for box STORES: with rows 16 bytes off (fp32, nz = 2 mod 4) they turn into
  // partial-sector writes and the pass runs 1.5-2.4 x slower than the LDG / STG kernel (350^3 fp32: K2 0.70 ->
  // 1.02 ms with two, 1.71 ms with three resident CTAs; profiles/r02_tma_strided.md).
  if (((size_t)g.Q * 2 * sizeof(T)) % 32) {
    // measured (fp32): K4 at 512x512x90 0.399 -> 0.323 ms, but K2 (twice the stores) 0.400 -> 0.657 ms, and at L = 350
    // both lose (K2 0.70 -> 1.07, K4 0.65 -> 0.94 ms): only K4 of the power-of-two lengths takes this variant
    if constexpr ((L & (L - 1)) == 0) {
      if (which == 3) return launch_tma_y<T, L, true>(which, g, b, mapA1, mapA2, st);
    }
    return cudaErrorNotSupported;
  }
  return launch_tma_y<T, L, false>(which, g, b, mapA1, mapA2, st);
}

// L = 1024 (three-stage plan): which = 1 (K2), 3 (K4).  Persistent, one CTA per SM.
template <typename T>
cudaError_t launch_tma3(int which, const FastGeom& g, const FastBufs<T>& b, cudaStream_t st) {
  constexpr int L = 1024;
  using TT = Tma3<T, L>;
  using TL = Tile<T, L>;
  if (((size_t)g.Q * 2 * sizeof(T)) % 32) return cudaErrorNotSupported;
  alignas(64) CUtensorMap mapA1, mapA2;
  if (!make_map<T>(&mapA1, b.A1, (size_t)(g.nx + 1) * g.ny, g.Q, TT::R) ||
      !make_map<T>(&mapA2, b.A2, (size_t)(g.nx + 1) * g.Py, g.Q, TT::R))
    return cudaErrorNotSupported;
  const int colblocks = (g.Q + TL::B - 1) / TL::B, ntile = colblocks * (g.nx + 1);
  int grid = sm_count_tma();
  if (grid > ntile) grid = ntile;
  cudaError_t e;
  if (which == 1) {
    if ((e = cudaFuncSetAttribute(yf3_tma_kernel<T, L>, cudaFuncAttributeMaxDynamicSharedMemorySize, TT::smem2)) != cudaSuccess) return e;
    yf3_tma_kernel<T, L><<<grid, TT::NT, TT::smem2, st>>>(mapA1, mapA2, b.Wy, colblocks, ntile);
  } else {
    if ((e = cudaFuncSetAttribute(yi3_tma_kernel<T, L>, cudaFuncAttributeMaxDynamicSharedMemorySize, TT::smem2)) != cudaSuccess) return e;
    yi3_tma_kernel<T, L><<<grid, TT::NT, TT::smem2, st>>>(mapA2, mapA1, b.Wy, colblocks, ntile);
  }
  return cudaSuccess;
}

// [rows][row_reals] reals with a row pitch of its own (every second row of an array); box {box_bytes, R rows}
template <typename T> bool make_map_pitch(CUtensorMap* map, const void* base, size_t rows, size_t row_reals, size_t pitch_reals,
                                          int box_bytes, int R) {
  EncodeFn fn = encode_fn();
  if (!fn) return false;
  const cuuint64_t dims[2] = {(cuuint64_t)row_reals, (cuuint64_t)rows};
  const cuuint64_t strides[1] = {(cuuint64_t)pitch_reals * sizeof(T)};
  const cuuint32_t box[2] = {(cuuint32_t)(box_bytes / sizeof(T)), (cuuint32_t)R}, estr[2] = {1, 1};
  return fn(map, sizeof(T) == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2,
            const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
            CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// K5 at L = 1024: the rows of even and of odd k of A1 as two tensors
template <typename T>
cudaError_t launch_tma3_xi(const FastGeom& g, const FastBufs<T>& b, T* H, T scale, cudaStream_t st) {
  constexpr int L = 1024;
  using TT = Tma3<T, L>;
  using TX = Tma3X<T, L>;
  using TL = Tile<T, L>;
  const size_t row_reals = (size_t)g.ny * g.Q;        // reals of one x row of H; a row of A1 holds twice as many
  if ((row_reals * sizeof(T)) % 32) return cudaErrorNotSupported;
  const T* a1 = reinterpret_cast<const T*>(b.A1);
  alignas(64) CUtensorMap mapE, mapEl, mapO;
  if (!make_map_pitch<T>(&mapE, a1, L / 2 + 1, 2 * row_reals, 4 * row_reals, 128, TT::R) ||
      !make_map_pitch<T>(&mapEl, a1, L / 2 + 1, 2 * row_reals, 4 * row_reals, 128, 1) ||
      !make_map_pitch<T>(&mapO, a1 + 2 * row_reals, L / 2, 2 * row_reals, 4 * row_reals, 128, TT::R))
    return cudaErrorNotSupported;
  const size_t npairs = row_reals / 2;
  const int ntile = (int)((npairs + TL::B - 1) / TL::B);
  int grid = sm_count_tma();
  if (grid > ntile) grid = ntile;
  cudaError_t e = cudaFuncSetAttribute(xi3_tma_kernel<T, L>, cudaFuncAttributeMaxDynamicSharedMemorySize, TX::smem5);
  if (e != cudaSuccess) return e;
  xi3_tma_kernel<T, L><<<grid, TT::NT, TX::smem5, st>>>(mapE, mapEl, mapO, reinterpret_cast<Cx<T>*>(H), b.Wx, npairs, scale, ntile);
  return cudaSuccess;
}

// K1 at L = 1024 with its input tile by boxes
template <typename T>
cudaError_t launch_tma3_x(const FastGeom& g, const FastBufs<T>& b, const T* m, cudaStream_t st) {
  constexpr int L = 1024;
  using TT = Tma3<T, L>;
  using TL = Tile<T, L>;
  const size_t row_reals = (size_t)g.ny * g.Q;
  if ((row_reals * sizeof(T)) % 32) return cudaErrorNotSupported;
  alignas(64) CUtensorMap mapF;
  if (!make_map_rows<T>(&mapF, m, g.nx, row_reals, 64, TT::R)) return cudaErrorNotSupported;
  const size_t npairs = row_reals / 2;
  const int ntile = (int)((npairs + TL::B - 1) / TL::B);
  int grid = sm_count_tma();
  if (grid > ntile) grid = ntile;
  cudaError_t e = cudaFuncSetAttribute(xf3_tma_kernel<T, L>, cudaFuncAttributeMaxDynamicSharedMemorySize, TT::smem2);
  if (e != cudaSuccess) return e;
  xf3_tma_kernel<T, L><<<grid, TT::NT, TT::smem2, st>>>(mapF, b.A1, b.Wx, npairs, ntile);
  return cudaSuccess;
}

// K1 / K5 by boxes: the x axis is the row axis of m, A1 and H as they lie in memory
template <typename T, int L>
cudaError_t launch_tma_x(int which, const FastGeom& g, const FastBufs<T>& b, const T* m, T* H, T scale, cudaStream_t st) {
  using TT = TmaTile<T, L>;
  using TX = TmaTileX<T, L>;
  using TL = Tile2<T, L>;
  const size_t row_reals = (size_t)g.ny * g.Q;   // reals of one x row of m / H; a row of A1 holds twice as many
  if ((row_reals * sizeof(T)) % 32) return cudaErrorNotSupported;   // rows must start on a sector (see launch_tma)
  alignas(64) CUtensorMap mapF, mapA, mapRow;
  if (!make_map_rows<T>(&mapF, which == 0 ? (const void*)m : (const void*)H, g.nx, row_reals, 64, TT::R) ||
      !make_map_rows<T>(&mapA, b.A1, (size_t)g.nx + 1, 2 * row_reals, 128, TT::R) ||
      !make_map_rows<T>(&mapRow, b.A1, (size_t)g.nx + 1, 2 * row_reals, 128, 1))
    return cudaErrorNotSupported;
  const size_t npairs = row_reals / 2;
  const int ntile = (int)((npairs + TL::B - 1) / TL::B);
  cudaError_t e;
  int per_sm = 1;
  if (which == 0) {
    if ((e = cudaFuncSetAttribute(xf2_tma_kernel<T, L>, cudaFuncAttributeMaxDynamicSharedMemorySize, TX::smem1)) != cudaSuccess) return e;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, xf2_tma_kernel<T, L>, TX::NT, TX::smem1) != cudaSuccess || per_sm < 1) per_sm = 1;
    int grid = per_sm * sm_count_tma();
    if (grid > ntile) grid = ntile;
    xf2_tma_kernel<T, L><<<grid, TX::NT, TX::smem1, st>>>(mapF, mapA, mapRow, b.T2x, ntile);
  } else {
    if ((e = cudaFuncSetAttribute(xi2_tma_kernel<T, L>, cudaFuncAttributeMaxDynamicSharedMemorySize, TX::smem5)) != cudaSuccess) return e;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, xi2_tma_kernel<T, L>, TX::NT, TX::smem5) != cudaSuccess || per_sm < 1) per_sm = 1;
    int grid = per_sm * sm_count_tma();
    if (grid > ntile) grid = ntile;
    xi2_tma_kernel<T, L><<<grid, TX::NT, TX::smem5, st>>>(mapA, mapRow, mapF, b.T2x, (T)0.5 * scale, ntile);
  }
  return cudaSuccess;
}

}  // namespace

bool tma_enabled() {
  static int on = -1;
  if (on < 0) {
    const char* e = std::getenv("MM_B200_TMA");
    on = (e && e[0] == '0') ? 0 : 1;
  }
  return on == 1;
}

// true when strided_tma_launch will run the box kernels for this transform length, row length and precision
// which: 1 = K2, 3 = K4
bool strided_tma_usable(int L, int Q, size_t real_bytes, int which) {
  if (!tma_enabled() || !encode_fn()) return false;
  const bool aligned = ((size_t)Q * 2 * real_bytes) % 32 == 0;
  if (fast_two_stage(L)) return aligned || (which == 3 && (L & (L - 1)) == 0);   // see launch_tma
  return L == 1024 && aligned;
}

// which: 1 = K2 (forward y), 3 = K4 (inverse y).  cudaErrorNotSupported: the caller runs the LDG / STG kernel.
template <typename T>
cudaError_t strided_tma_launch(int which, const FastGeom& g, const FastBufs<T>& b, cudaStream_t st) {
  if (!tma_enabled() || !encode_fn()) return cudaErrorNotSupported;
  if (g.ny == 1024) return launch_tma3<T>(which, g, b, st);
  switch (g.ny) {
#define MM_TMA_CASE(LL) case LL: return launch_tma<T, LL>(which, g, b, st);
    MM_PLAN2_LENGTHS(MM_TMA_CASE)
#undef MM_TMA_CASE
    default: return cudaErrorNotSupported;
  }
}

template cudaError_t strided_tma_launch<float>(int, const FastGeom&, const FastBufs<float>&, cudaStream_t);
template cudaError_t strided_tma_launch<double>(int, const FastGeom&, const FastBufs<double>&, cudaStream_t);

// The x passes by boxes win or tie for the powers of two and L = 100 and lose for L = 350, 400 (350^3 fp64: K1
// 0.81 -> 0.90 ms, K5 0.70 -> 0.89 ms; the (L + 1) x 128-byte tile leaves one 224-thread CTA per SM there;
// profiles/r02_tma_strided.md): those lengths keep the LDG / STG kernels.
constexpr bool tma_x_wins(int L) { return L != 350 && L != 400; }

bool strided_tma_x_usable(int L, int ny, int Q, size_t real_bytes) {
  return tma_enabled() && encode_fn() && fast_two_stage(L) && tma_x_wins(L) && ((size_t)ny * Q * real_bytes) % 32 == 0;
}
bool strided_tma3_x_usable(int ny, int Q, size_t real_bytes) {   // K1 at L = 1024
  return tma_enabled() && encode_fn() && ((size_t)ny * Q * real_bytes) % 32 == 0;
}

// which: 0 = K1 (forward x, r2c), 4 = K5 (inverse x, c2r).  cudaErrorNotSupported: the caller runs the LDG / STG kernel.
template <typename T>
cudaError_t strided_tma_x_launch(int which, const FastGeom& g, const FastBufs<T>& b, const T* m, T* H, T scale,
                                 cudaStream_t st) {
  if (!tma_enabled() || !encode_fn()) return cudaErrorNotSupported;
  if (g.nx == 1024) return which == 0 ? launch_tma3_x<T>(g, b, m, st) : launch_tma3_xi<T>(g, b, H, scale, st);
  switch (g.nx) {
#define MM_TMA_CASE(LL) case LL: if constexpr (tma_x_wins(LL)) return launch_tma_x<T, LL>(which, g, b, m, H, scale, st); else return cudaErrorNotSupported;
    MM_PLAN2_LENGTHS(MM_TMA_CASE)
#undef MM_TMA_CASE
    default: return cudaErrorNotSupported;
  }
}

template cudaError_t strided_tma_x_launch<float>(int, const FastGeom&, const FastBufs<float>&, const float*, float*, float,
                                                 cudaStream_t);
template cudaError_t strided_tma_x_launch<double>(int, const FastGeom&, const FastBufs<double>&, const double*, double*,
                                                  double, cudaStream_t);

}  // namespace mm
