// K3 of the x-first demag path for z lengths outside demag_fast.cu's warp-per-pencil kernels: the
// paper's own nz = 100, 350, 400 and nz = 90.
//
//   S3: A2[kx][ky'][q = 3 z + c] in place:  z forward (pruned) . Nhat multiply . z inverse (truncated)
//       (last forward FFT, "pointwise multiplication with the ... demagnetisation kernel",
//       first inverse FFT; the innermost spectrum never reaches HBM).
//
// A CTA owns NPAIR mirror pairs of pencils (ky, Py - ky) of one kx plane -- a pair shares its Nhat row up to
// the sign of the entries odd in ky -- as a tile of Pz rows in shared memory.  The pencil keeps the layout
// it has in HBM, [z][c] with c fastest, so the load and the store are straight copies; the tile's columns
// are the (pencil, component) pairs and a thread owns one task of one column:
//   stage A   (bf, col):  K1/2 samples z = bf + K2 s -> pruned radix-K1 butterfly in registers, root
//                         w_Pz^(bf k1) -> rows k1 K2 + bf               (its own rows: in place, no hazard)
//   stage B   (k1, col):  radix-K2 butterfly over bf -> X[kz = k1 + K1 k2] at row k1 K2 + k2      (in place)
//   multiply  (kz, pair): Hhat = Nhat mhat for both pencils of the pair; the Nhat row is read from global
//                         memory with kz along the lanes (coalesced, every entry exactly once)
//   stage B', A': the mirror images, A' computing only the nz wanted samples.
// Pz = K1 K2 with the plans of plan2.cuh (700 = 28 x 25, 800 = 32 x 25, 200 = 20 x 10, 180 = 20 x 9): two
// register stages and one exchange per direction, against the run-time radix stages of demag_mixed.cu
// (about 18 shared-memory passes per element, profiles/r01_v4_paper_meshes.md).
// With K2 = 1 (mod 8) consecutive k1 blocks of a column start 3 K2 = 3 (mod 8) elements apart, so a warp's
// accesses of stages B / B' fall on consecutive bank groups in fp64.
#define MM_NO_PACKED_F32
#include "demag_ztile.cuh"

#include "fft_core.cuh"
#include "plan2.cuh"

namespace mm {

template <typename T, int NZ> struct ZTile {
  using P = Plan2<NZ>;
  static constexpr int K1 = P::K1, K2 = P::K2, A = K1 / 2, Pz = 2 * NZ, Q = 3 * NZ;
  // pairs per CTA: the tile of one pair is 2 x 3 Pz complex (fp32 350: 33.6 KB, fp64: 67.2 KB)
  static constexpr int NPAIR = sizeof(T) == 4 ? 2 : 1;
  static constexpr int NP = 2 * NPAIR, C = 3 * NP;
  static constexpr int PITCH = 3 * Pz + (sizeof(T) == 4 ? 2 : 1);   // elements per pencil buffer
  static constexpr int tasksA = K2 * C, tasksB = K1 * C;
  static constexpr int NT = ((tasksA > tasksB ? tasksA : tasksB) + 31) / 32 * 32;
  static constexpr int smem_bytes = NP * PITCH * (int)sizeof(Cx<T>);
  // resident CTAs the kernel is compiled for: shared memory, and registers (fp64 stages hold ~170: two CTAs)
  static constexpr int by_smem = (200 * 1024) / (smem_bytes + 1024);
  static constexpr int min_blocks = by_smem >= 3 && sizeof(T) == 4 && NT <= 256 ? 3 : (by_smem >= 2 ? 2 : 1);
  static_assert(K1 * K2 == Pz && K1 % 2 == 0 && NT <= 512, "plan");
};

template <typename T, int K1, int... I>
__device__ __forceinline__ void zt_rot_fwd(const Cx<T>* v, Cx<T>* o, std::integer_sequence<int, I...>) {
  ((o[I] = mul_root<T, K1, I, false>(v[I])), ...);
}
template <typename T, int K1, int... I>
__device__ __forceinline__ void zt_rot_inv_add(Cx<T>* e, const Cx<T>* o, std::integer_sequence<int, I...>) {
  ((e[I] = add_root<T, K1, I, true>(e[I], o[I])), ...);
}

// grid (ceil(ny / NPAIR), nx + 1).  Wt[bf K1 + k1] = exp(-2 pi i bf k1 / Pz).  tab: Nhat octant rows
// [kx][ky <= ny][6][ozp].  posy: row of y frequency ky in a plane of A2.
template <typename T, int NZ>
__global__ void __launch_bounds__(ZTile<T, NZ>::NT, ZTile<T, NZ>::min_blocks)
zt_kernel(Cx<T>* __restrict__ A2, const T* __restrict__ tab, const Cx<T>* __restrict__ Wt,
          const uint16_t* __restrict__ posy, int ny, int ozp) {
  using Z = ZTile<T, NZ>;
  constexpr int K1 = Z::K1, K2 = Z::K2, A = Z::A, Pz = Z::Pz, Q = Z::Q, NP = Z::NP, C = Z::C, PITCH = Z::PITCH,
                NT = Z::NT, NPAIR = Z::NPAIR;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Cx<T>* tile = reinterpret_cast<Cx<T>*>(smem_raw);
  __shared__ size_t rowoff[NP];
  const int tid = threadIdx.x;
  const int plane = blockIdx.y, i0 = blockIdx.x * NPAIR, Py = 2 * ny;
  if (tid < NP) {
    const int i = i0 + (tid >> 1);
    const int ky = (tid & 1) ? (i == 0 ? ny : Py - i) : i;
    rowoff[tid] = i < ny ? ((size_t)plane * Py + posy[ky]) * Q : (size_t)0;
  }
  __syncthreads();
  // ---- load: pencil p -> tile[p PITCH + q], q < Q (rows z < nz; the rows of the padding are written by stage A)
  for (int e = tid; e < NP * Q; e += NT) {
    const int p = e / Q, q = e - p * Q;
    tile[p * PITCH + q] = (i0 + (p >> 1) < ny) ? A2[rowoff[p] + q] : mk<T>((T)0, (T)0);
  }
  __syncthreads();
  const int col = tid % C, task = tid / C;
  Cx<T>* cbase = tile + (col / 3) * PITCH + (col % 3);   // element (row, col) at cbase[3 row]
  // ---- stage A
  if (task < K2) {
    const int bf = task;
    Cx<T> v[A], o[A];
#pragma unroll
    for (int s = 0; s < A; ++s) v[s] = cbase[3 * (bf + K2 * s)];
    zt_rot_fwd<T, K1>(v, o, std::make_integer_sequence<int, A>{});
    Dft<T, A, false>::run(v);   // even k1
    Dft<T, A, false>::run(o);   // odd k1
    const Cx<T>* tw = Wt + bf * K1;
#pragma unroll
    for (int u = 0; u < A; ++u) {
      const Cx<T> w0 = __ldg(tw + 2 * u), w1 = __ldg(tw + 2 * u + 1);
      cbase[3 * ((2 * u) * K2 + bf)] = u ? cmul(v[u], w0) : v[0];
      cbase[3 * ((2 * u + 1) * K2 + bf)] = cmul(o[u], w1);
    }
  }
  __syncthreads();
  // ---- stage B: X[k1 + K1 k2] -> row k1 K2 + k2
  if (task < K1) {
    Cx<T> t[K2];
    Cx<T>* r = cbase + 3 * task * K2;
#pragma unroll
    for (int bf = 0; bf < K2; ++bf) t[bf] = r[3 * bf];
    Dft<T, K2, false>::run(t);
#pragma unroll
    for (int k2 = 0; k2 < K2; ++k2) r[3 * k2] = t[k2];
  }
  __syncthreads();
  // ---- Hhat = Nhat mhat.  kz runs along the lanes: the octant row is read coalesced, once.  The mirrored
  // halves (kz > nz, ky > ny) reuse the octant entry with the sign of the components odd along that axis.
  for (int e = tid; e < NPAIR * Pz; e += NT) {
    const int pp = e / Pz, kz = e - pp * Pz;
    const int i = i0 + pp;
    if (i >= ny) break;
    const int row = (kz % K1) * K2 + kz / K1;
    const bool mir = kz > NZ;
    const int idx = mir ? Pz - kz : kz;
    const T* trow = tab + ((size_t)plane * (ny + 1) + i) * 6 * ozp;
    T n[6];
#pragma unroll
    for (int c = 0; c < 6; ++c) n[c] = __ldg(trow + c * ozp + idx);
    if (mir) { n[4] = -n[4]; n[5] = -n[5]; }
    Cx<T>* s0 = tile + (2 * pp) * PITCH + 3 * row;
    {
      const Cx<T> a = s0[0], b = s0[1], c = s0[2];
      s0[0] = mk<T>(n[0] * a.x + n[3] * b.x + n[4] * c.x, n[0] * a.y + n[3] * b.y + n[4] * c.y);
      s0[1] = mk<T>(n[3] * a.x + n[1] * b.x + n[5] * c.x, n[3] * a.y + n[1] * b.y + n[5] * c.y);
      s0[2] = mk<T>(n[4] * a.x + n[5] * b.x + n[2] * c.x, n[4] * a.y + n[5] * b.y + n[2] * c.y);
    }
    // the partner pencil: ky = Py - i (same row, N_xy and N_yz negated), for the pair i = 0 the row ky = ny
    if (i == 0) {
      const T* t2 = trow + (size_t)ny * 6 * ozp;
#pragma unroll
      for (int c = 0; c < 6; ++c) n[c] = __ldg(t2 + c * ozp + idx);
      if (mir) { n[4] = -n[4]; n[5] = -n[5]; }
    } else {
      n[3] = -n[3]; n[5] = -n[5];
    }
    Cx<T>* s1 = s0 + PITCH;
    {
      const Cx<T> a = s1[0], b = s1[1], c = s1[2];
      s1[0] = mk<T>(n[0] * a.x + n[3] * b.x + n[4] * c.x, n[0] * a.y + n[3] * b.y + n[4] * c.y);
      s1[1] = mk<T>(n[3] * a.x + n[1] * b.x + n[5] * c.x, n[3] * a.y + n[1] * b.y + n[5] * c.y);
      s1[2] = mk<T>(n[4] * a.x + n[5] * b.x + n[2] * c.x, n[4] * a.y + n[5] * b.y + n[2] * c.y);
    }
  }
  __syncthreads();
  // ---- stage B'
  if (task < K1) {
    Cx<T> t[K2];
    Cx<T>* r = cbase + 3 * task * K2;
#pragma unroll
    for (int k2 = 0; k2 < K2; ++k2) t[k2] = r[3 * k2];
    Dft<T, K2, true>::run(t);
#pragma unroll
    for (int bf = 0; bf < K2; ++bf) r[3 * bf] = t[bf];
  }
  __syncthreads();
  // ---- stage A' with the truncation: samples z = bf + K2 s, s < K1/2, back to rows z
  if (task < K2) {
    const int bf = task;
    Cx<T> v[A], o[A];
    const Cx<T>* tw = Wt + bf * K1;
#pragma unroll
    for (int u = 0; u < A; ++u) {
      const Cx<T> w0 = __ldg(tw + 2 * u), w1 = __ldg(tw + 2 * u + 1);
      const Cx<T> a = cbase[3 * ((2 * u) * K2 + bf)], b = cbase[3 * ((2 * u + 1) * K2 + bf)];
      v[u] = u ? cmulc(a, w0) : a;
      o[u] = cmulc(b, w1);
    }
    Dft<T, A, true>::run(v);
    Dft<T, A, true>::run(o);
    zt_rot_inv_add<T, K1>(v, o, std::make_integer_sequence<int, A>{});
#pragma unroll
    for (int s = 0; s < A; ++s) cbase[3 * (bf + K2 * s)] = v[s];
  }
  __syncthreads();
  for (int e = tid; e < NP * Q; e += NT) {
    const int p = e / Q, q = e - p * Q;
    if (i0 + (p >> 1) < ny) A2[rowoff[p] + q] = tile[p * PITCH + q];
  }
}

bool ztile_supported(int nz) {
  switch (nz) {
#define MM_ZT_CASE(LL) case LL: return true;
    MM_ZTILE_LENGTHS(MM_ZT_CASE)
#undef MM_ZT_CASE
    default: return false;
  }
}

template <typename T, int NZ>
static cudaError_t launch_zt(const FastGeom& g, const FastBufs<T>& b, cudaStream_t st) {
  using Z = ZTile<T, NZ>;
  if (Z::smem_bytes > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(zt_kernel<T, NZ>, cudaFuncAttributeMaxDynamicSharedMemorySize, Z::smem_bytes);
    if (e != cudaSuccess) return e;
  }
  const int ozp = (g.nz + 2) / 2 * 2;   // InitGeom::ozp: nz + 1 rounded up to even
  zt_kernel<T, NZ><<<dim3((g.ny + Z::NPAIR - 1) / Z::NPAIR, g.nx + 1), Z::NT, Z::smem_bytes, st>>>(
      b.A2, b.table, b.T2z, b.posy, g.ny, ozp);
  return cudaSuccess;
}

template <typename T> cudaError_t ztile_launch(const FastGeom& g, const FastBufs<T>& b, cudaStream_t st) {
  switch (g.nz) {
#define MM_ZT_CASE(LL) case LL: return launch_zt<T, LL>(g, b, st);
    MM_ZTILE_LENGTHS(MM_ZT_CASE)
#undef MM_ZT_CASE
    default: return cudaErrorInvalidValue;
  }
}

template cudaError_t ztile_launch<float>(const FastGeom&, const FastBufs<float>&, cudaStream_t);
template cudaError_t ztile_launch<double>(const FastGeom&, const FastBufs<double>&, cudaStream_t);

}  // namespace mm
