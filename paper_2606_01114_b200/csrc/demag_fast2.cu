// Two-stage strided passes of the x-first demag path (K1, K2, K4, K5) for every
// transform length with a plan in plan2.cuh: the powers of two 64 .. 512 and the paper's own sides
// L = 100, 350, 400, whose padded lengths are 200 = 20 x 10, 700 = 28 x 25
// and 800 = 32 x 25.
//
// The pruned length-P transform (P = 2L = K1 K2, K1 even, L non-zero inputs; "zero-padding
// and ... FFT") is split as
//     X[k1 + K1 k2] = sum_bf w_K2^(bf k2) . w_P^(bf k1) . sum_{s < K1/2} a[bf + K2 s] w_K1^(s k1)
// stage A: one thread per (bf, column): K1/2 inputs straight from global memory, pruned
//          radix-K1 butterfly with compile-time roots, twiddle w_P^(bf k1), to shared memory;
// stage B: one thread per (k1, column): radix-K2 butterfly, K2 outputs straight to global
//          memory in NATURAL frequency order (row k1 + K1 k2).
// The inverse is the mirror image with the truncation folded into stage A' (only the L wanted
// samples are computed).  One exchange through shared memory per transform instead of two:
// the passes are bound by L1/shared-memory wavefronts, not by HBM (profiles/r01_v2_fast_path.md).
// Radix 25 runs as 5 x 5, radix 14 / 10 as 2 x 7 / 2 x 5 in registers (fft_core.cuh).
//
// K1/K5 (x axis, r2c / c2r): two real columns (q, q+1) ride as one complex column Z = a + i b.
// The Hermitian separation A[k] = (Z[k] + conj Z[-k]) / 2, B[k] = (Z[k] - conj Z[-k]) / 2i needs
// Z[-k], which sits in the stage-B thread of k1' = K1 - k1 at k2' = K2 - 1 - k2.  Stage-B slots
// are ordered so that k1 and K1 - k1 are neighbours (slots 2p, 2p + 1) and hence B lanes apart
// in the same warp: the halves are swapped with warp shuffles, no extra pass through shared
// memory.  (The factor 1/2 is applied in K5's output scale.)
//
// Columns beyond the end of a row (3 nz and ny 3 nz / 2 need not be multiples of the 64-byte row of a
// tile) are loaded from column 0 and never stored.
// scalar fp32 complex add/subtract here: the two-wide form (mm_common.cuh) measured slower in these
// memory-latency-bound passes (K2 0.497 -> 0.528 ms at config 4) and faster only in K3
#define MM_NO_PACKED_F32
#include "demag_fast.cuh"
#include "strided2.cuh"

namespace mm {

// fp32 and fp64 (fp64: K1 0.79 -> 0.69 ms, K5 0.96 -> 0.57 ms at config 4 against the three-stage kernels)
bool fast_two_stage(int L) {
  switch (L) {
#define MM_PLAN2_CASE(LL) case LL: return true;
    MM_PLAN2_LENGTHS(MM_PLAN2_CASE)
#undef MM_PLAN2_CASE
    default: return false;
  }
}

#define MM_T2_PROLOGUE                                                     \
  extern __shared__ __align__(16) unsigned char smem_raw[];                \
  Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw);                          \
  using TL = Tile2<T, L>;                                                  \
  constexpr int K1 = TL::K1, K2 = TL::K2, A = TL::A, JN = TL::JN, B = TL::B; \
  const int lane = threadIdx.x % B, slot = threadIdx.x / B;                \
  (void)JN; (void)A;

// ---------------------------------------------------------------- K2: forward y
// grid (ceil(Q / B), planes)
template <typename T, int L>
__global__ void __launch_bounds__(Tile2<T, L>::NT, Tile2<T, L>::min_blocks)
yf2_kernel(const Cx<T>* __restrict__ A1, Cx<T>* __restrict__ A2, const Cx<T>* __restrict__ Wt, int Q) {
  MM_T2_PROLOGUE
  const int colq = blockIdx.x * B + lane;
  const bool ok = colq < Q;
  const size_t col = ok ? colq : 0;
  const Cx<T>* in = A1 + (size_t)blockIdx.y * L * Q + col;
  Cx<T>* out = A2 + (size_t)blockIdx.y * 2 * L * Q + col;
  if (slot < K2) {
    Cx<T> v[A];
#pragma unroll
    for (int s = 0; s < A; ++s) v[s] = in[(size_t)(slot + K2 * s) * Q];
    fwdA<T, L>(sm, Wt, lane, slot, v);
  }
  __syncthreads();
  if (slot < K1) {
    const int k1 = slot_k1<K1>(slot);
    Cx<T> t[K2];
    fwdB<T, L>(sm, lane, k1, t);
    if (ok) {
#pragma unroll
      for (int k2 = 0; k2 < K2; ++k2) out[(size_t)(k1 + K1 * k2) * Q] = t[k2];
    }
  }
}

// ---------------------------------------------------------------- K4: inverse y
template <typename T, int L>
__global__ void __launch_bounds__(Tile2<T, L>::NT, Tile2<T, L>::min_blocks)
yi2_kernel(const Cx<T>* __restrict__ A2, Cx<T>* __restrict__ A1, const Cx<T>* __restrict__ Wt, int Q) {
  MM_T2_PROLOGUE
  const int colq = blockIdx.x * B + lane;
  const bool ok = colq < Q;
  const size_t col = ok ? colq : 0;
  const Cx<T>* in = A2 + (size_t)blockIdx.y * 2 * L * Q + col;
  Cx<T>* out = A1 + (size_t)blockIdx.y * L * Q + col;
  if (slot < K1) {
    const int k1 = slot_k1<K1>(slot);
    Cx<T> t[K2];
#pragma unroll
    for (int k2 = 0; k2 < K2; ++k2) t[k2] = in[(size_t)(k1 + K1 * k2) * Q];
    invB<T, L>(sm, lane, k1, t);
  }
  __syncthreads();
  if (slot < K2 && ok) {
    Cx<T> v[A];
    invA<T, L>(sm, Wt, lane, slot, v);
#pragma unroll
    for (int s = 0; s < A; ++s) out[(size_t)(slot + K2 * s) * Q] = v[s];
  }
}

template <typename T> __device__ __forceinline__ Cx<T> shfl_xor_cx(Cx<T> v, int m) {
  Cx<T> r;
  r.x = __shfl_xor_sync(0xffffffffu, v.x, m);
  r.y = __shfl_xor_sync(0xffffffffu, v.y, m);
  return r;
}

// ---------------------------------------------------------------- K1: forward x, r2c
// m [x][y][q] real, read as complex pairs (q, q+1); npairs = ny Q / 2 pairs per x row; the
// spectrum rows k <= nx of A1 hold (A[k], B[k]) at complex columns (2 pair, 2 pair + 1).
// Stage-B thread k1 holds Z[k1 + K1 j] and stores the rows k = k1 + K1 j <= L.  Z[-k] is the partner
// thread's t[K2 - 1 - j] (k1' = K1 - k1), the thread's own t[K2 - 1 - j] for the self-paired k1 = K1/2
// and its own t[(K2 - j) % K2] for k1 = 0.  Every lane of a warp takes part in the shuffles (threads
// past the last slot with dummy values).
// SLAB (demag_slab.cuh): the transform axis is y of the x plane sv.x0 + blockIdx.y (npairs = pairs of one
// (x, y) row), and spectrum row ky goes to the rank that owns it: sv.p[ky / rpr] + ((ky % rpr) nx + x) rowc.
template <typename T, int L, bool SLAB>
__global__ void __launch_bounds__(Tile2<T, L>::NT, Tile2<T, L>::min_blocks)
xf2_kernel(const Cx<T>* __restrict__ mp, Cx<T>* __restrict__ A1, const Cx<T>* __restrict__ Wt, size_t npairs,
           SlabView<T> sv) {
  MM_T2_PROLOGUE
  const size_t pairq = (size_t)blockIdx.x * B + lane;
  const bool ok = pairq < npairs;
  const size_t pair = ok ? pairq : 0;
  const int xg = SLAB ? sv.x0 + (int)blockIdx.y : 0;
  const Cx<T>* in = mp + (SLAB ? (size_t)xg * L * npairs : (size_t)0) + pair;
  if (slot < K2) {
    Cx<T> v[A];
#pragma unroll
    for (int s = 0; s < A; ++s) v[s] = in[(size_t)(slot + K2 * s) * npairs];
    fwdA<T, L>(sm, Wt, lane, slot, v);
  }
  __syncthreads();
  if (slot < TL::slotsB) {   // whole warps: every lane takes part in the shuffles
    const bool live = TL::slotsB == K1 || slot < K1;
    const int k1 = slot_k1<K1>(live ? slot : 0);
    const bool pair0 = (slot >> 1) == 0, odd = slot & 1;
    Cx<T> t[K2];
    fwdB<T, L>(sm, lane, k1, t);
    const size_t rowc = 2 * npairs;
    auto row = [&](int k) -> Cx<T>* {
      if constexpr (SLAB) return sv.p[k / sv.rpr] + ((size_t)(k % sv.rpr) * sv.nx + xg) * rowc + 2 * pair;
      else return A1 + (size_t)k * rowc + 2 * pair;
    };
#pragma unroll
    for (int j = 0; j < JN; ++j) {
      if (K2 % 2 == 0 && j == K2 / 2) {   // even K2: the last j holds only k = L (k1 = 0), its own mirror
        if (live && ok && k1 == 0) {
          const Cx<T> z = t[j % K2];
          Vec2<T>::st(row(L), mk<T>(2 * z.x, (T)0), mk<T>(2 * z.y, (T)0));
        }
        continue;
      }
      const Cx<T> r = shfl_xor_cx<T>(t[(2 * K2 - 1 - j) % K2], B);
      const Cx<T> own = odd ? t[(2 * K2 - 1 - j) % K2] : t[(K2 - j) % K2];
      if (live && ok && TL::has_row(j, pair0, odd)) {
        const Cx<T> z = t[j % K2], zm = cconj(pair0 ? own : r);
        const Cx<T> s = cadd(z, zm), d = csub(z, zm);
        Vec2<T>::st(row(k1 + K1 * j), s, mk<T>(d.y, -d.x));
      }
    }
  }
}

// ---------------------------------------------------------------- K5: inverse x, c2r
// Z[k] = A[k] + i B[k], Z[P - k] = conj A[k] + i conj B[k]; the truncated inverse gives
// h_q(x) + i h_{q+1}(x), written as the real pair (q, q+1) of H, times scale.  A stage-B' thread loads
// its rows k = k1 + K1 j <= L, keeps Z[k] in t[j] and hands S = conj A + i conj B = Z[P - k] to the
// thread that owns P - k: the partner's (or, for k1 = K1/2, its own) slot K2 - 1 - j, for k1 = 0 its own
// slot (K2 - j) % K2.  The self-mirrored rows k = 0 and k = L keep Z[k].
template <typename T, int L, bool SLAB>
__global__ void __launch_bounds__(Tile2<T, L>::NT, Tile2<T, L>::min_blocks)
xi2_kernel(const Cx<T>* __restrict__ A1, Cx<T>* __restrict__ Hp, const Cx<T>* __restrict__ Wt, size_t npairs,
           T scale, SlabView<T> sv) {
  MM_T2_PROLOGUE
  const size_t pairq = (size_t)blockIdx.x * B + lane;
  const bool ok = pairq < npairs;
  const size_t pair = ok ? pairq : 0;
  const int xg = SLAB ? sv.x0 + (int)blockIdx.y : 0;
  if (slot < TL::slotsB) {   // whole warps: every lane takes part in the shuffles
    const bool live = TL::slotsB == K1 || slot < K1;
    const int k1 = slot_k1<K1>(live ? slot : 0);
    const bool pair0 = (slot >> 1) == 0, odd = slot & 1;
    const size_t rowc = 2 * npairs;
    auto row = [&](int k) -> const Cx<T>* {
      if constexpr (SLAB) return sv.p[k / sv.rpr] + ((size_t)(k % sv.rpr) * sv.nx + xg) * rowc + 2 * pair;
      else return A1 + (size_t)k * rowc + 2 * pair;
    };
    Cx<T> t[K2];
    Cx<T> a[JN], b[JN];
#pragma unroll
    for (int j = 0; j < JN; ++j) {
      const bool last_even = K2 % 2 == 0 && j == K2 / 2;   // only k = L of k1 = 0
      if (live && (last_even ? k1 == 0 : TL::has_row(j, pair0, odd)))
        Vec2<T>::ld(row(k1 + K1 * j), a[j], b[j]);
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
      // the mirror Z[P - k] of row k goes to the partner's (k1 = K1/2: the thread's own) slot K2 - 1 - j, for
      // k1 = 0 to its own slot (K2 - j) % K2; the self-mirrored rows k = 0 and k = L keep Z[k]
      if (!pair0) { if (TL::has_row(j, false, !odd)) t[(2 * K2 - 1 - j) % K2] = r; }
      else if (odd) { if (!(K2 % 2 == 1 && j == K2 / 2)) t[(2 * K2 - 1 - j) % K2] = S; }
      else if (j >= 1) t[(K2 - j) % K2] = S;
      if (TL::has_row(j, pair0, odd)) t[j % K2] = mk<T>(a[j].x - b[j].y, a[j].y + b[j].x);
    }
    if (live) invB<T, L>(sm, lane, k1, t);
  }
  __syncthreads();
  if (slot < K2 && ok) {
    Cx<T> v[A];
    invA<T, L>(sm, Wt, lane, slot, v);
    Cx<T>* out = Hp + (SLAB ? (size_t)xg * L * npairs : (size_t)0) + pair;
#pragma unroll
    for (int s = 0; s < A; ++s)
      out[(size_t)(slot + K2 * s) * npairs] = mk<T>(scale * v[s].x, scale * v[s].y);
  }
}

// ---------------------------------------------------------------- host side

template <typename K> static cudaError_t opt_in(K kernel, int bytes) {
  if (bytes <= 48 * 1024) return cudaSuccess;
  return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}

template <typename T, int L>
static cudaError_t launch2(int which, const FastGeom& g, const FastBufs<T>& b, const T* m, T* H, T scale,
                           cudaStream_t st) {
  using TL = Tile2<T, L>;
  const size_t npairs = (size_t)g.ny * g.Q / 2;
  const unsigned gx = (unsigned)((npairs + TL::B - 1) / TL::B), gq = (unsigned)((g.Q + TL::B - 1) / TL::B);
  const int nk = g.nx + 1;
  cudaError_t e;
  switch (which) {
    case 0:
      if ((e = opt_in(xf2_kernel<T, L, false>, TL::smem_bytes)) != cudaSuccess) return e;
      xf2_kernel<T, L, false><<<gx, TL::NT, TL::smem_bytes, st>>>(reinterpret_cast<const Cx<T>*>(m), b.A1, b.T2x, npairs,
                                                                 SlabView<T>{});
      break;
    case 1:
      if ((e = opt_in(yf2_kernel<T, L>, TL::smem_bytes)) != cudaSuccess) return e;
      yf2_kernel<T, L><<<dim3(gq, nk), TL::NT, TL::smem_bytes, st>>>(b.A1, b.A2, b.T2y, g.Q);
      break;
    case 3:
      if ((e = opt_in(yi2_kernel<T, L>, TL::smem_bytes)) != cudaSuccess) return e;
      yi2_kernel<T, L><<<dim3(gq, nk), TL::NT, TL::smem_bytes, st>>>(b.A2, b.A1, b.T2y, g.Q);
      break;
    default:
      if ((e = opt_in(xi2_kernel<T, L, false>, TL::smem_bytes)) != cudaSuccess) return e;
      xi2_kernel<T, L, false><<<gx, TL::NT, TL::smem_bytes, st>>>(b.A1, reinterpret_cast<Cx<T>*>(H), b.T2x, npairs,
                                                                 (T)0.5 * scale, SlabView<T>{});
      break;
  }
  return cudaSuccess;
}

template <typename T>
cudaError_t strided2_launch(int which, const FastGeom& g, const FastBufs<T>& b, const T* m, T* H, T scale,
                            cudaStream_t st) {
  const int L = (which == 0 || which == 4) ? g.nx : g.ny;
  switch (L) {
#define MM_PLAN2_CASE(LL) case LL: return launch2<T, LL>(which, g, b, m, H, scale, st);
    MM_PLAN2_LENGTHS(MM_PLAN2_CASE)
#undef MM_PLAN2_CASE
    default: return cudaErrorInvalidValue;
  }
}

template cudaError_t strided2_launch<float>(int, const FastGeom&, const FastBufs<float>&, const float*,
                                            float*, float, cudaStream_t);
template cudaError_t strided2_launch<double>(int, const FastGeom&, const FastBufs<double>&, const double*,
                                             double*, double, cudaStream_t);

// ---- slab layout (demag_slab.cuh): y is the first transformed axis, x planes [sv.x0, sv.x0 + nxl) of one rank
template <typename T, int L>
static cudaError_t launch_slab(int which, int nxl, int Q, const Cx<T>* Wt, const SlabView<T>& sv, const T* m, T* H,
                               T scale, cudaStream_t st) {
  using TL = Tile2<T, L>;
  const size_t npairs = (size_t)Q / 2;
  const dim3 grid((unsigned)((npairs + TL::B - 1) / TL::B), nxl);
  cudaError_t e;
  if (which == 0) {
    if ((e = opt_in(xf2_kernel<T, L, true>, TL::smem_bytes)) != cudaSuccess) return e;
    xf2_kernel<T, L, true><<<grid, TL::NT, TL::smem_bytes, st>>>(reinterpret_cast<const Cx<T>*>(m), nullptr, Wt, npairs, sv);
  } else {
    if ((e = opt_in(xi2_kernel<T, L, true>, TL::smem_bytes)) != cudaSuccess) return e;
    xi2_kernel<T, L, true><<<grid, TL::NT, TL::smem_bytes, st>>>(nullptr, reinterpret_cast<Cx<T>*>(H), Wt, npairs,
                                                                 (T)0.5 * scale, sv);
  }
  return cudaSuccess;
}

template <typename T>
cudaError_t slab_y_launch(int which, int ny, int nxl, int Q, const Cx<T>* Wt, const SlabView<T>& sv, const T* m, T* H,
                          T scale, cudaStream_t st) {
  switch (ny) {
#define MM_PLAN2_CASE(LL) case LL: return launch_slab<T, LL>(which, nxl, Q, Wt, sv, m, H, scale, st);
    MM_PLAN2_LENGTHS(MM_PLAN2_CASE)
#undef MM_PLAN2_CASE
    default: return cudaErrorInvalidValue;
  }
}
template cudaError_t slab_y_launch<float>(int, int, int, int, const float2*, const SlabView<float>&, const float*, float*,
                                          float, cudaStream_t);
template cudaError_t slab_y_launch<double>(int, int, int, int, const double2*, const SlabView<double>&, const double*,
                                           double*, double, cudaStream_t);

void fast2_plan(int L, int* K1, int* K2) {
  if (!plan2_of(L, K1, K2)) { *K1 = 0; *K2 = 0; }
}

}  // namespace mm
