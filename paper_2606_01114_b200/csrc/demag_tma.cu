// K2 and K4, the y passes of the x-first demag path (S2 / S4, "zero-padding and ... FFT ... in
// the y- and z-directions", "the output is then truncated"), with their tiles moved by the TMA engine: 2D
// cp.async.bulk.tensor boxes of {64 bytes x up to 256 rows} instead of LDG / STG from every lane
// (BASELINE.json north_star: "TMA or cp.async staging of pencil tiles for the strided y/z passes").
// Same plans and stage arithmetic as demag_fast2.cu (strided2.cuh), bit-identical results.  A persistent CTA
// walks tiles (column block of 64 bytes, kx plane); the box loads of the next tile are issued as soon as the
// input buffer has been read, so they overlap the arithmetic and the stores of the current one.
//   K2: input tile [L rows] -> stage A -> exchange tile -> stage B -> the same buffer in natural row order
//       -> box stores.
//   K4: input tile [2L rows] -> stage B' reads its rows k1 + K1 k2, the tile itself becomes the exchange
//       tile (value bf of thread k1 at row (k1 ^ (bf & 1)) + K1 bf: the four bf of a warp then read rows of
//       both parities, i.e. both 64-byte halves of the banks) -> stage A' -> output tile [L rows] -> box stores.
// Columns beyond the end of a row are zero-filled on load and clipped on store by the tensor map.
// Measured against the LDG / STG kernels in profiles/r02_tma_strided.md; MM_B200_TMA=0 selects the latter.
#define MM_NO_PACKED_F32
#include <cuda.h>

#include <cstdlib>

#include "bulk_copy.cuh"
#include "demag_fast.cuh"
#include "strided2.cuh"

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

template <typename T, int L> struct TmaTile {
  using TL = Tile2<T, L>;
  static constexpr int R = box_rows(L);
  static_assert(L % R == 0 && (R * 64) % 128 == 0 && (L * 64) % 128 == 0, "box alignment");
  static constexpr int EW = 64 / (int)sizeof(T);                    // elements of the map's type per 64-byte row
  static constexpr int in2_bytes = L * 64;                          // K2 input tile
  static constexpr int ex_bytes = TL::K1 * TL::K2P * 64;            // exchange tile (>= 2L rows)
  static constexpr int smem2 = in2_bytes + ex_bytes + 64;
  static constexpr int in4_bytes = 2 * L * 64, out4_bytes = L * 64; // K4: input = exchange tile, output tile
  static constexpr int smem4 = in4_bytes + out4_bytes + 64;
  static constexpr int NT = TL::NT;
  // resident CTAs the kernels are compiled for: fp32 three where the tile leaves room (<= 72 KB), else two
  static constexpr int mb2 = sizeof(T) == 8 ? (NT <= 128 ? 2 : 1) : (smem2 <= 72 * 1024 ? 3 : 2);
  static constexpr int mb4 = sizeof(T) == 8 ? (NT <= 128 ? 2 : 1) : (smem4 <= 72 * 1024 ? 3 : 2);
};

// ---------------------------------------------------------------- K2: forward y
// mapIn: A1 as [(nx + 1) ny rows][2 Q reals], box {EW, R}; mapOut: A2 as [(nx + 1) Py rows][2 Q reals].
template <typename T, int L>
__global__ void __launch_bounds__(TmaTile<T, L>::NT, TmaTile<T, L>::mb2)
yf2_tma_kernel(const __grid_constant__ CUtensorMap mapIn, const __grid_constant__ CUtensorMap mapOut,
               const Cx<T>* __restrict__ Wt, int colblocks, int ntile) {
  using TT = TmaTile<T, L>;
  using TL = Tile2<T, L>;
  constexpr int K1 = TL::K1, K2 = TL::K2, A = TL::A, B = TL::B, R = TT::R;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Cx<T>* in = reinterpret_cast<Cx<T>*>(smem_raw);                        // [L][B]
  Cx<T>* ex = reinterpret_cast<Cx<T>*>(smem_raw + TT::in2_bytes);        // exchange tile, then output [2L][B]
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + TT::in2_bytes + TT::ex_bytes);
  const int lane = threadIdx.x % B, slot = threadIdx.x / B;
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
    if (threadIdx.x == 0) bulk_wait_read0();
    __syncthreads();   // every thread holds its inputs: the input buffer is free, and so is the output buffer
    if (threadIdx.x == 0 && tile + (int)gridDim.x < ntile) issue(tile + gridDim.x);
    if (slot < K2) fwdA<T, L>(ex, Wt, lane, slot, v);
    __syncthreads();
    {
      const int k1 = slot < K1 ? slot_k1<K1>(slot) : 0;
      Cx<T> t[K2];
      if (slot < K1) fwdB<T, L>(ex, lane, k1, t);
      __syncthreads();   // the exchange tile has been read: it becomes the output tile, rows in natural order
      if (slot < K1) {
#pragma unroll
        for (int k2 = 0; k2 < K2; ++k2) ex[(k1 + K1 * k2) * B + lane] = t[k2];
      }
    }
    fence_async_smem();
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
      for (int q = 0; q < 2 * L / R; ++q)
        tma_store_2d(&mapOut, cb * TT::EW, plane * 2 * L + q * R, ex + q * R * B);
      bulk_commit();
    }
  }
  if (threadIdx.x == 0) bulk_wait0();
}

// ---------------------------------------------------------------- K4: inverse y, truncated
// mapIn: A2 as [(nx + 1) Py rows][2 Q reals]; mapOut: A1 as [(nx + 1) ny rows][2 Q reals].
template <typename T, int L>
__global__ void __launch_bounds__(TmaTile<T, L>::NT, TmaTile<T, L>::mb4)
yi2_tma_kernel(const __grid_constant__ CUtensorMap mapIn, const __grid_constant__ CUtensorMap mapOut,
               const Cx<T>* __restrict__ Wt, int colblocks, int ntile) {
  using TT = TmaTile<T, L>;
  using TL = Tile2<T, L>;
  constexpr int K1 = TL::K1, K2 = TL::K2, A = TL::A, B = TL::B, R = TT::R;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Cx<T>* in = reinterpret_cast<Cx<T>*>(smem_raw);                        // [2L][B], then the exchange tile
  Cx<T>* outb = reinterpret_cast<Cx<T>*>(smem_raw + TT::in4_bytes);      // [L][B]
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + TT::in4_bytes + TT::out4_bytes);
  const int lane = threadIdx.x % B, slot = threadIdx.x / B;
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
      const Cx<T>* tw = Wt + bf * K1;
      const Cx<T>* row = in + (K1 * bf) * B + lane;
#pragma unroll
      for (int u = 0; u < A; ++u) {
        Cx<T> w0, w1;
        Vec2<T>::ldg(tw + 2 * u, w0, w1);
        const Cx<T> a = row[((2 * u) ^ sw) * B], b = row[((2 * u + 1) ^ sw) * B];
        v[u] = u ? cmulc(a, w0) : a;
        o[u] = cmulc(b, w1);
      }
      Dft<T, A, true>::run(v);
      Dft<T, A, true>::run(o);
      rot_inv_add<T, K1>(v, o, std::make_integer_sequence<int, A>{});
    }
    // the previous tile's stores must have read the output buffer before it is overwritten
    if (threadIdx.x == 0) bulk_wait_read0();
    __syncthreads();   // the exchange tile has been read: the loads of the next tile may land in it
    if (threadIdx.x == 0 && tile + (int)gridDim.x < ntile) issue(tile + gridDim.x);
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
  if (threadIdx.x == 0) bulk_wait0();
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

// [rows][Q complex] viewed as rows of 2 Q reals; box {64 bytes, R rows}
template <typename T> bool make_map(CUtensorMap* map, void* base, size_t rows, int Q, int R) {
  EncodeFn fn = encode_fn();
  if (!fn) return false;
  const cuuint64_t dims[2] = {(cuuint64_t)2 * Q, (cuuint64_t)rows};
  const cuuint64_t strides[1] = {(cuuint64_t)Q * 2 * sizeof(T)};
  const cuuint32_t box[2] = {(cuuint32_t)(64 / sizeof(T)), (cuuint32_t)R}, estr[2] = {1, 1};
  return fn(map, sizeof(T) == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, base, dims,
            strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
            CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
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

template <typename T, int L>
cudaError_t launch_tma(int which, const FastGeom& g, const FastBufs<T>& b, cudaStream_t st) {
  using TT = TmaTile<T, L>;
  using TL = Tile2<T, L>;
  alignas(64) CUtensorMap mapA1, mapA2;
  // rows must start on a 32-byte sector: with rows 16 bytes off (fp32, nz = 2 mod 4) the box stores turn into
  // partial-sector writes and the pass runs 1.5-2.4 x slower than the LDG / STG kernel (350^3 fp32: K2 0.70 ->
  // 1.02 ms with two, 1.71 ms with three resident CTAs; profiles/r02_tma_strided.md)
  if (((size_t)g.Q * 2 * sizeof(T)) % 32) return cudaErrorNotSupported;
  if (!make_map<T>(&mapA1, b.A1, (size_t)(g.nx + 1) * g.ny, g.Q, TT::R) ||
      !make_map<T>(&mapA2, b.A2, (size_t)(g.nx + 1) * g.Py, g.Q, TT::R))
    return cudaErrorNotSupported;
  const int colblocks = (g.Q + TL::B - 1) / TL::B, ntile = colblocks * (g.nx + 1);
  cudaError_t e;
  if (which == 1) {
    if ((e = cudaFuncSetAttribute(yf2_tma_kernel<T, L>, cudaFuncAttributeMaxDynamicSharedMemorySize, TT::smem2)) != cudaSuccess) return e;
    int per_sm = 1;   // persistent grid = what is resident at once (registers and shared memory)
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, yf2_tma_kernel<T, L>, TT::NT, TT::smem2) != cudaSuccess || per_sm < 1) per_sm = 1;
    int grid = per_sm * sm_count_tma();
    if (grid > ntile) grid = ntile;
    yf2_tma_kernel<T, L><<<grid, TT::NT, TT::smem2, st>>>(mapA1, mapA2, b.T2y, colblocks, ntile);
  } else {
    if ((e = cudaFuncSetAttribute(yi2_tma_kernel<T, L>, cudaFuncAttributeMaxDynamicSharedMemorySize, TT::smem4)) != cudaSuccess) return e;
    int per_sm = 1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, yi2_tma_kernel<T, L>, TT::NT, TT::smem4) != cudaSuccess || per_sm < 1) per_sm = 1;
    int grid = per_sm * sm_count_tma();
    if (grid > ntile) grid = ntile;
    yi2_tma_kernel<T, L><<<grid, TT::NT, TT::smem4, st>>>(mapA2, mapA1, b.T2y, colblocks, ntile);
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
bool strided_tma_usable(int L, int Q, size_t real_bytes) {
  return tma_enabled() && encode_fn() && fast_two_stage(L) && ((size_t)Q * 2 * real_bytes) % 32 == 0;
}

// which: 1 = K2 (forward y), 3 = K4 (inverse y).  cudaErrorNotSupported: the caller runs the LDG / STG kernel.
template <typename T>
cudaError_t strided_tma_launch(int which, const FastGeom& g, const FastBufs<T>& b, cudaStream_t st) {
  if (!tma_enabled() || !encode_fn()) return cudaErrorNotSupported;
  switch (g.ny) {
#define MM_TMA_CASE(LL) case LL: return launch_tma<T, LL>(which, g, b, st);
    MM_PLAN2_LENGTHS(MM_TMA_CASE)
#undef MM_TMA_CASE
    default: return cudaErrorNotSupported;
  }
}

template cudaError_t strided_tma_launch<float>(int, const FastGeom&, const FastBufs<float>&, cudaStream_t);
template cudaError_t strided_tma_launch<double>(int, const FastGeom&, const FastBufs<double>&, cudaStream_t);

}  // namespace mm
