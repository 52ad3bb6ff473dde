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
//   stage B   (k1, col):  radix-K2 butterfly over bf -> X[kz = k1 + K1 k2], k2 < K2, in registers; the three
//                         components of a (k1, pencil) sit in neighbouring lanes, so the multiply
//                         Hhat = Nhat mhat takes the other two by warp shuffle (Nhat row staged in shared
//                         memory by a bulk copy); stage B' follows in the same registers -> rows k1 K2 + bf
//   stage A'  the mirror image of A, computing only the nz wanted samples.
// Pencils and table rows arrive by bulk asynchronous copies (cp.async.bulk + mbarrier), the result leaves
// by a bulk store; three __syncthreads per tile.
// Pz = K1 K2 with the plans of plan2.cuh (700 = 28 x 25, 800 = 32 x 25, 200 = 20 x 10, 180 = 20 x 9): two
// register stages and one exchange per direction, against the run-time radix stages of demag_mixed.cu
// (about 18 shared-memory passes per element, profiles/r01_v4_paper_meshes.md).
// With K2 = 1 (mod 8) consecutive k1 blocks of a column start 3 K2 = 3 (mod 8) elements apart, so a warp's
// accesses of stages B / B' fall on consecutive bank groups in fp64.
#define MM_NO_PACKED_F32
#include "demag_ztile.cuh"

#include "bulk_copy.cuh"
#include "fft_core.cuh"
#include "plan2.cuh"

namespace mm {

template <typename T, int NZ> struct ZTile {
  using P = Plan2<NZ>;
  static constexpr int K1 = P::K1, K2 = P::K2, A = K1 / 2, Pz = 2 * NZ, Q = 3 * NZ;
  static constexpr int OZP = (NZ + 2) / 2 * 2;        // kz pitch of a table row (InitGeom::ozp)
  // pairs per CTA: the tile of one pair is 2 x 3 Pz complex (fp32 350: 33.6 KB, fp64: 67.2 KB)
  static constexpr int NPAIR = sizeof(T) == 4 ? 2 : 1;
  static constexpr int NP = 2 * NPAIR, C = 3 * NP;
  // elements per pencil buffer: 3 Pz plus a pad that spreads the pencils of a warp over the banks
  // (fp32: = 4 mod 16 and even, so that a pencil starts on a 16-byte boundary; fp64: = 7 mod 8)
  static constexpr int PITCH = sizeof(T) == 4 ? 3 * Pz + ((4 - 3 * Pz % 16) + 16) % 16 : 3 * Pz + ((7 - 3 * Pz % 8) + 8) % 8;
  // stage B runs on lane triples (the three components of one (k1, pencil)): 10 triples per warp
  static constexpr int NTRI = K1 * NP, tasksA = K2 * C;
  static constexpr int warpsB = (NTRI + 9) / 10, warpsA = (tasksA + 31) / 32;
  static constexpr int NT = 32 * (warpsA > warpsB ? warpsA : warpsB);
  static constexpr int pencil_bytes = Q * (int)sizeof(Cx<T>);
  static constexpr int tile_bytes = NP * PITCH * (int)sizeof(Cx<T>);
  // one staged table row per pair, plus the row ky = ny of the partner of ky = 0 (one pencil per plane).  In shared memory the six components of a row are OZS apart and the rows of
  // the pairs SLOT apart, chosen so that the three components a lane triple reads, for the neighbouring kz of
  // a warp and for both pairs, fall on different banks (OZS = 8 mod 32 words, SLOT = 4 mod 32 words in fp32;
  // OZS = 4 mod 16 double words in fp64).
  static constexpr int OZS = sizeof(T) == 4 ? OZP + ((8 - OZP % 32) + 32) % 32 : OZP + ((4 - OZP % 16) + 16) % 16;
  static constexpr int SLOT = sizeof(T) == 4 ? 6 * OZS + ((4 - 6 * OZS % 32) + 32) % 32 : 6 * OZS;
  // NPAIR slots for the rows of the pairs + one for the row ky = ny (the partner of ky = 0, one pencil per plane)
  // where two CTAs per SM still fit with it (not fp64 at nz = 400: that pencil then reads its row from global memory)
  static constexpr bool NYSLOT = 2 * (tile_bytes + (NPAIR + 1) * SLOT * (int)sizeof(T) + 16 + 1024) <= 228 * 1024;
  static constexpr int NSLOT = NPAIR + (NYSLOT ? 1 : 0);
  static constexpr int smem_bytes = tile_bytes + NSLOT * SLOT * (int)sizeof(T) + 16;
  // resident CTAs the kernel is compiled for: what shared memory admits and what the register file admits at
  // ~80 (fp32) / ~144 (fp64) registers per thread (fp64, K1 = 32: a few hundred bytes of spills beat one CTA per SM)
  static constexpr int by_smem = (220 * 1024) / (smem_bytes + 1024);
  static constexpr int by_regs = 65536 / ((sizeof(T) == 4 ? 72 : 144) * NT);
  static constexpr int min_blocks = by_smem < by_regs ? (by_smem < 1 ? 1 : by_smem) : (by_regs < 1 ? 1 : by_regs);
  static_assert(K1 * K2 == Pz && K1 % 2 == 0 && NT <= 512 && NZ % 2 == 0, "plan");
  static_assert(pencil_bytes % 16 == 0 && tile_bytes % 16 == 0, "bulk copies move 16-byte multiples");
};

template <typename T, int K1, int... I>
__device__ __forceinline__ void zt_rot_fwd(const Cx<T>* v, Cx<T>* o, std::integer_sequence<int, I...>) {
  ((o[I] = mul_root<T, K1, I, false>(v[I])), ...);
}
template <typename T, int K1, int... I>
__device__ __forceinline__ void zt_rot_inv_add(Cx<T>* e, const Cx<T>* o, std::integer_sequence<int, I...>) {
  ((e[I] = add_root<T, K1, I, true>(e[I], o[I])), ...);
}
// two adjacent roots of the stage table as one 16-byte load where the type allows it
template <typename T> __device__ __forceinline__ void ldg2(const Cx<T>* p, Cx<T>& a, Cx<T>& b);
template <> __device__ __forceinline__ void ldg2<float>(const float2* p, float2& a, float2& b) {
  const float4 t = __ldg(reinterpret_cast<const float4*>(p));
  a = make_float2(t.x, t.y);
  b = make_float2(t.z, t.w);
}
template <> __device__ __forceinline__ void ldg2<double>(const double2* p, double2& a, double2& b) {
  a = __ldg(p);
  b = __ldg(p + 1);
}
// one table element global -> shared without passing through registers
template <typename T> __device__ __forceinline__ void cp_async_elem(T* dst_smem, const T* src) {
  if constexpr (sizeof(T) == 4)
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(dst_smem)), "l"(src) : "memory");
  else
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(dst_smem)), "l"(src) : "memory");
}
template <typename T> __device__ __forceinline__ Cx<T> shfl_cx(Cx<T> v, int src) {
  Cx<T> r;
  r.x = __shfl_sync(0xffffffffu, v.x, src);
  r.y = __shfl_sync(0xffffffffu, v.y, src);
  return r;
}

// grid (ceil(ny / NPAIR), planes); the table plane of blockIdx.y is k0 + blockIdx.y; xm: the rows of a plane
// are kx, not ky (slab layout: N_xy, N_xz instead of N_xy, N_yz change sign on the mirrored half).  Wt[bf K1 + k1] = exp(-2 pi i bf k1 / Pz).  tab: Nhat octant rows
// [kx][ky <= ny][6][OZP].  posy: row of y frequency ky in a plane of A2.
template <typename T, int NZ>
__global__ void __launch_bounds__(ZTile<T, NZ>::NT, ZTile<T, NZ>::min_blocks)
zt_kernel(Cx<T>* __restrict__ A2, const T* __restrict__ tab, const Cx<T>* __restrict__ Wt,
          const uint16_t* __restrict__ posy, int ny, int k0, int xm) {
  using Z = ZTile<T, NZ>;
  constexpr int K1 = Z::K1, K2 = Z::K2, A = Z::A, Pz = Z::Pz, Q = Z::Q, NP = Z::NP, C = Z::C, PITCH = Z::PITCH,
                NPAIR = Z::NPAIR, OZP = Z::OZP, OZS = Z::OZS, SLOT = Z::SLOT;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Cx<T>* tile = reinterpret_cast<Cx<T>*>(smem_raw);
  T* tabs = reinterpret_cast<T*>(smem_raw + Z::tile_bytes);                       // [NPAIR] x SLOT: [6] x OZS
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + Z::tile_bytes + Z::NSLOT * SLOT * sizeof(T));
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int plane = blockIdx.y, i0 = blockIdx.x * NPAIR, Py = 2 * ny;
  const int npair = ny - i0 < NPAIR ? ny - i0 : NPAIR;   // pairs of this CTA that exist
  auto pencil = [&](int p) -> Cx<T>* {
    const int i = i0 + (p >> 1);
    const int ky = (p & 1) ? (i == 0 ? ny : Py - i) : i;
    return A2 + ((size_t)plane * Py + posy[ky]) * Q;
  };
  // ---- bulk asynchronous loads: the pencils (barrier 0), then the table rows (barrier 1)
  if (tid == 0) {
    mbar_init(bars, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    mbar_expect_tx(bars, 2 * npair * Z::pencil_bytes);
    for (int p = 0; p < 2 * npair; ++p) bulk_load(tile + p * PITCH, pencil(p), Z::pencil_bytes, bars);
  }
  // the table rows of the pairs, element by element into the padded layout (asynchronous copies, waited for
  // before stage B)
  {
    // (one component row per step: no index division in the copy loop, which the issue-bound pass would pay for)
    const T* rows = tab + ((size_t)(k0 + plane) * (ny + 1) + i0) * 6 * OZP;
#pragma unroll
    for (int pp = 0; pp < NPAIR; ++pp) {
      if (pp < npair) {
#pragma unroll
        for (int cc = 0; cc < 6; ++cc)
          for (int e = tid; e < OZP; e += Z::NT)
            cp_async_elem<T>(tabs + pp * SLOT + cc * OZS + e, rows + (pp * 6 + cc) * OZP + e);
      }
    }
    if (Z::NYSLOT && i0 == 0) {   // the CTA that holds the pair (0, ny): the row ky = ny into the extra slot
      const T* rown = tab + ((size_t)(k0 + plane) * (ny + 1) + ny) * 6 * OZP;
#pragma unroll
      for (int cc = 0; cc < 6; ++cc)
        for (int e = tid; e < OZP; e += Z::NT) cp_async_elem<T>(tabs + NPAIR * SLOT + cc * OZS + e, rown + cc * OZP + e);
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  }
  // pencils of pairs beyond the last one (odd ny): zero, so that their columns stay finite
  for (int e = tid; e < (NP - 2 * npair) * Q; e += Z::NT) tile[2 * npair * PITCH + (e / Q) * PITCH + e % Q] = mk<T>((T)0, (T)0);
  __syncthreads();   // the barriers are initialised
  mbar_wait(bars, 0);
  // ---- stage A: thread = (bf, column), column = (pencil, component), element (row, col) at cbase[3 row]
  {
    const int col = tid % C, bf = tid / C;
    Cx<T>* cbase = tile + (col / 3) * PITCH + (col % 3);
    if (bf < K2) {
      Cx<T> v[A], o[A];
#pragma unroll
      for (int s = 0; s < A; ++s) v[s] = cbase[3 * (bf + K2 * s)];
      zt_rot_fwd<T, K1>(v, o, std::make_integer_sequence<int, A>{});
      Dft<T, A, false>::run(v);   // even k1
      Dft<T, A, false>::run(o);   // odd k1
      const Cx<T>* tw = Wt + bf * K1;
#pragma unroll
      for (int u = 0; u < A; ++u) {
        Cx<T> w0, w1;
        ldg2<T>(tw + 2 * u, w0, w1);
        cbase[3 * ((2 * u) * K2 + bf)] = u ? cmul(v[u], w0) : v[0];
        cbase[3 * ((2 * u + 1) * K2 + bf)] = cmul(o[u], w1);
      }
    }
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  __syncthreads();
  // ---- stage B . Nhat . stage B': lane triple = the three components of one (k1, pencil); the multiply
  // Hhat_c = sum_c' Nhat_cc' mhat_c' takes the other two components from the neighbouring lanes by shuffle.
  // X[kz = k1 + K1 k2] of the thread's component sits in t[k2].
  {
    const int tri = warp * 10 + lane / 3, c = lane % 3;
    const bool act = lane < 30 && tri < Z::NTRI;
    const int trc = act ? tri : 0;
    const int p = trc % NP, k1 = trc / NP;
    Cx<T>* r = tile + p * PITCH + 3 * k1 * K2 + c;
    Cx<T> t[K2];
#pragma unroll
    for (int bf = 0; bf < K2; ++bf) t[bf] = r[3 * bf];
    Dft<T, K2, false>::run(t);
    // table components of row c of the symmetric tensor: xx yy zz xy xz yz = 0 .. 5
    const int ca = c == 0 ? 3 : (c == 1 ? 5 : 4), cb = c == 0 ? 4 : (c == 1 ? 3 : 5);   // N[c][(c+1)%3], N[c][(c+2)%3]
    const int la = lane - c + (c + 1) % 3, lb = lane - c + (c + 2) % 3;
    const int pair = p >> 1, i = i0 + pair;
    const bool odd = p & 1;
    // the odd pencil of pair i is ky = Py - i: row i with the entries odd in ky (xy, yz) negated; the odd
    // pencil of pair 0 is ky = ny, whose own row is read from global memory (one pencil per plane)
    const bool nyq = odd && i == 0;
    const T* ts = tabs + ((Z::NYSLOT && nyq) ? NPAIR : pair) * SLOT;
    const T* tg = tab + ((size_t)(k0 + plane) * (ny + 1) + ny) * 6 * OZP;
    const T sy = (odd && i != 0) ? (T)-1 : (T)1;
    const int co = xm ? 4 : 5;   // with xy, the component that is odd along the row axis
    const T fya = (ca == 3 || ca == co) ? sy : (T)1, fyb = (cb == 3 || cb == co) ? sy : (T)1;
    const bool za = ca == 4 || ca == 5, zb = cb == 4 || cb == 5;     // odd in kz
#pragma unroll
    for (int k2 = 0; k2 < K2; ++k2) {
      const int kz = k1 + K1 * k2;
      // mirrored half along kz: known at compile time except for the one k2 whose block straddles kz = nz
      const bool mir = K1 * k2 + K1 - 1 <= NZ ? false : (K1 * k2 > NZ ? true : kz > NZ);
      const int idx = mir ? Pz - kz : kz;
      T ns = ts[c * OZS + idx], na = ts[ca * OZS + idx], nb = ts[cb * OZS + idx];
      if constexpr (!Z::NYSLOT) {
        if (nyq) { ns = __ldg(tg + c * OZP + idx); na = __ldg(tg + ca * OZP + idx); nb = __ldg(tg + cb * OZP + idx); }
      }
      na *= (za && mir) ? -fya : fya;
      nb *= (zb && mir) ? -fyb : fyb;
      const Cx<T> x = t[k2], xa = shfl_cx<T>(x, la), xb = shfl_cx<T>(x, lb);
      t[k2] = mk<T>(ns * x.x + na * xa.x + nb * xb.x, ns * x.y + na * xa.y + nb * xb.y);
    }
    Dft<T, K2, true>::run(t);
    if (act) {
#pragma unroll
      for (int bf = 0; bf < K2; ++bf) r[3 * bf] = t[bf];
    }
  }
  __syncthreads();
  // ---- stage A' with the truncation: samples z = bf + K2 s, s < K1/2, back to rows z
  {
    const int col = tid % C, bf = tid / C;
    Cx<T>* cbase = tile + (col / 3) * PITCH + (col % 3);
    if (bf < K2) {
      Cx<T> v[A], o[A];
      const Cx<T>* tw = Wt + bf * K1;
#pragma unroll
      for (int u = 0; u < A; ++u) {
        Cx<T> w0, w1;
        ldg2<T>(tw + 2 * u, w0, w1);
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
  }
  fence_async_smem();
  __syncthreads();
  if (tid == 0) {
    for (int p = 0; p < 2 * npair; ++p) bulk_store(pencil(p), tile + p * PITCH, Z::pencil_bytes);
    bulk_commit();
    bulk_wait_read0();   // the tile may be released once the copy engine has read it
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
static cudaError_t launch_zt(const FastGeom& g, const FastBufs<T>& b, int k0, int nk, int xm, cudaStream_t st) {
  using Z = ZTile<T, NZ>;
  if (Z::smem_bytes > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(zt_kernel<T, NZ>, cudaFuncAttributeMaxDynamicSharedMemorySize, Z::smem_bytes);
    if (e != cudaSuccess) return e;
  }
  zt_kernel<T, NZ><<<dim3((g.ny + Z::NPAIR - 1) / Z::NPAIR, nk), Z::NT, Z::smem_bytes, st>>>(
      b.A2, b.table, b.T2z, b.posy, g.ny, k0, xm);
  return cudaSuccess;
}

template <typename T>
cudaError_t ztile_launch(const FastGeom& g, const FastBufs<T>& b, int k0, int nk, int xm, cudaStream_t st) {
  switch (g.nz) {
#define MM_ZT_CASE(LL) case LL: return launch_zt<T, LL>(g, b, k0, nk, xm, st);
    MM_ZTILE_LENGTHS(MM_ZT_CASE)
#undef MM_ZT_CASE
    default: return cudaErrorInvalidValue;
  }
}

template cudaError_t ztile_launch<float>(const FastGeom&, const FastBufs<float>&, int, int, int, cudaStream_t);
template cudaError_t ztile_launch<double>(const FastGeom&, const FastBufs<double>&, int, int, int, cudaStream_t);

}  // namespace mm
