// K1..K5 of the fast demag path.
//
//   K1 xf : m [x][y][z][c] real      -> A1[kx<=nx][y][q]      x forward, r2c, pruned   (S1)
//   K2 yf : A1                       -> A2[kx][ky'][q]        y forward, pruned        (S2)
//   K3 zp : A2 in place, x Nhat                               z forward, tensor
//                                                             multiply, z inverse      (S3)
//   K4 yi : A2                       -> A1[kx][y][q]          y inverse, truncated     (S4)
//   K5 xi : A1                       -> H [x][y][z][c] real   x inverse, c2r, truncated(S5)
// q = 3 z + c is the flattened (z, component) index, the fastest axis everywhere.
//
// K1, K2, K4, K5 ("strided passes"): the transform axis is strided, 64 bytes of q are the
// batch.  A CTA owns a tile of 2L rows x 64 B in shared memory (L = n_d; rows [0, L) hold the
// even-output half, rows [L, 2L) the odd-output half of the pruned length-2L transform); lanes
// run along the batch so every global access is a run of 64-byte row segments and every shared
// access of a quarter/half warp is conflict-free (rows of a warp's neighbouring tasks differ
// in bit 0; the last stage's rows are made to differ by the XOR swizzle below).  Three radix
// stages: the first straight from global memory in registers, the middle one in shared
// memory, the last one straight to global memory.
//
// K3 ("contiguous pass"): the z pencil of one (kx, ky') is 3 nz contiguous complex values.  A
// group of G = Pz/16 lanes owns a pencil, each lane 16 values of each component in registers:
// pruned radix-16 stage, one exchange through shared memory, radix-G stage, 3x3 real-symmetric
// multiply in registers, and the mirror image back.  Pencils move by bulk async copies.
#include "demag_fast.cuh"

#include <cuda/std/cstdint>

#include "bulk_copy.cuh"
#include "demag_ztile.cuh"

#include "fft_core.cuh"
#include "strided3.cuh"

namespace mm {

// k = h + 2 (u1 + R1 (u2 + R2 u3))  ->  row h L + u1 R2 R3 + u2 R3 + u3   (L = 1024)
int fast_pos_logical(int L, int k) {
  using P = FastPlan<1024>;
  const int h = k & 1;
  int kk = k >> 1;
  const int u1 = kk % P::R1; kk /= P::R1;
  const int u2 = kk % P::R2; kk /= P::R2;
  return h * L + u1 * P::R2 * P::R3 + u2 * P::R3 + kk;
}
int fast_swizzle(int L, int row) {
  (void)L;
  return row ^ ((row >> ilog2c(FastPlan<1024>::R3)) & 1);
}

#define MM_TILE_PROLOGUE                                                   \
  extern __shared__ __align__(16) unsigned char smem_raw[];                \
  Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw);                          \
  using TL = Tile<T, L>;                                                   \
  constexpr int R1 = TL::R1, R2 = TL::R2, R3 = TL::R3, q1 = TL::q1, B = TL::B, NS = TL::NS; \
  const int lane = threadIdx.x % B, slot = threadIdx.x / B;                \
  (void)R2; (void)R3;

// ---------------------------------------------------------------- K2: forward y (S2)
// grid (Q / B, planes).  A1, A2 point at the first plane of the launch.
template <typename T, int L>
__global__ void __launch_bounds__(Tile<T, L>::NT, Tile<T, L>::min_blocks)
yf_fast_kernel(const Cx<T>* __restrict__ A1, Cx<T>* __restrict__ A2, const Cx<T>* __restrict__ W, int Q) {
  MM_TILE_PROLOGUE
  // columns beyond the end of a row (3 nz need not be a multiple of the 64-byte row of a tile) are loaded from
  // column 0 and never stored
  const bool ok = blockIdx.x * B + lane < Q;
  const size_t col = ok ? (size_t)blockIdx.x * B + lane : 0;
  const Cx<T>* in = A1 + (size_t)blockIdx.y * L * Q + col;
  Cx<T>* out = A2 + (size_t)blockIdx.y * 2 * L * Q + col;
#pragma unroll 1
  for (int bf = slot; bf < q1; bf += NS) {
    Cx<T> v[R1];
#pragma unroll
    for (int s = 0; s < R1; ++s) v[s] = in[(size_t)(bf + q1 * s) * Q];
    fwd_first<T, L>(sm, W, lane, bf, v);
  }
  __syncthreads();
  fwd_middle<T, L>(sm, W, lane, slot);
  __syncthreads();
#pragma unroll 1
  for (int i = slot; i < 2 * R1 * R2; i += NS) {
    Cx<T> v[R3];
    fwd_last<T, L>(sm, lane, i, v);
    if (ok) {
#pragma unroll
      for (int u = 0; u < R3; ++u) out[(size_t)(i * R3 + u) * Q] = v[u];
    }
  }
}

// ---------------------------------------------------------------- K4: inverse y (S4)
template <typename T, int L>
__global__ void __launch_bounds__(Tile<T, L>::NT, Tile<T, L>::min_blocks)
yi_fast_kernel(const Cx<T>* __restrict__ A2, Cx<T>* __restrict__ A1, const Cx<T>* __restrict__ W, int Q) {
  MM_TILE_PROLOGUE
  const bool ok = blockIdx.x * B + lane < Q;
  const size_t col = ok ? (size_t)blockIdx.x * B + lane : 0;
  const Cx<T>* in = A2 + (size_t)blockIdx.y * 2 * L * Q + col;
  Cx<T>* out = A1 + (size_t)blockIdx.y * L * Q + col;
#pragma unroll 2
  for (int i = slot; i < 2 * R1 * R2; i += NS) {
    Cx<T> v[R3];
#pragma unroll
    for (int u = 0; u < R3; ++u) v[u] = in[(size_t)(i * R3 + u) * Q];
    inv_first<T, L>(sm, lane, i, v);
  }
  __syncthreads();
  inv_middle<T, L>(sm, W, lane, slot);
  __syncthreads();
#pragma unroll 1
  for (int bf = slot; bf < q1; bf += NS) {
    Cx<T> v[R1];
    inv_last<T, L>(sm, W, lane, bf, v);
    if (ok) {
#pragma unroll
      for (int s = 0; s < R1; ++s) out[(size_t)(bf + q1 * s) * Q] = v[s];
    }
  }
}

// ---------------------------------------------------------------- K1: forward x, r2c (S1)
// The real array m[x][y][q] is read as complex pairs (q, q+1): Z = FFT(a + i b) of two real
// signals, separated afterwards with A[k] = (Z[k] + conj Z[-k])/2, B[k] = (Z[k] - conj Z[-k])/(2i)
// for k <= nx.  grid (ny Q / 2 / B).  npairs = ny Q / 2 (pairs per x row); rowc = ny Q.
template <typename T, int L>
__global__ void __launch_bounds__(Tile<T, L>::NT, Tile<T, L>::min_blocks)
xf_fast_kernel(const Cx<T>* __restrict__ mp, Cx<T>* __restrict__ A1, const Cx<T>* __restrict__ W,
               const uint16_t* __restrict__ pos, size_t npairs) {
  MM_TILE_PROLOGUE
  const bool ok = (size_t)blockIdx.x * B + lane < npairs;
  const size_t pair = ok ? (size_t)blockIdx.x * B + lane : 0;
  const Cx<T>* in = mp + pair;
#pragma unroll 1
  for (int bf = slot; bf < q1; bf += NS) {
    Cx<T> v[R1];
#pragma unroll
    for (int s = 0; s < R1; ++s) v[s] = in[(size_t)(bf + q1 * s) * npairs];
    fwd_first<T, L>(sm, W, lane, bf, v);
  }
  __syncthreads();
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
    const int p1 = pos[k], p2 = pos[(2 * L - k) & (2 * L - 1)];
    const Cx<T> z1 = sm[p1 * B + lane], z2 = cconj(sm[p2 * B + lane]);
    const Cx<T> s = cadd(z1, z2), d = csub(z1, z2);
    if (ok)
      Pair2<T>::st(out + (size_t)k * rowc, mk<T>((T)0.5 * s.x, (T)0.5 * s.y),
                   mk<T>((T)0.5 * d.y, (T)-0.5 * d.x));
  }
}

// ---------------------------------------------------------------- K5: inverse x, c2r (S5)
// Z[k] = A[k] + i B[k], Z[Px - k] = conj A[k] + i conj B[k]; the truncated inverse gives
// h_q(x) + i h_{q+1}(x), written as the real pair (q, q+1) of H, times scale (-Ms).
template <typename T, int L>
__global__ void __launch_bounds__(Tile<T, L>::NT, Tile<T, L>::min_blocks)
xi_fast_kernel(const Cx<T>* __restrict__ A1, Cx<T>* __restrict__ Hp, const Cx<T>* __restrict__ W,
               const uint16_t* __restrict__ pos, size_t npairs, T scale) {
  MM_TILE_PROLOGUE
  const bool ok = (size_t)blockIdx.x * B + lane < npairs;
  const size_t pair = ok ? (size_t)blockIdx.x * B + lane : 0;
  const Cx<T>* in = A1 + 2 * pair;
  const size_t rowc = 2 * npairs;
  // four independent row loads in flight per thread (one at a time left this pass latency-bound: 0.26 of the
  // roofline at L = 1024)
#pragma unroll 4
  for (int k = slot; k <= L; k += NS) {
    Cx<T> a, b;
    Pair2<T>::ld(in + (size_t)k * rowc, a, b);
    sm[pos[k] * B + lane] = mk<T>(a.x - b.y, a.y + b.x);
    if (k != 0 && k != L) sm[pos[2 * L - k] * B + lane] = mk<T>(a.x + b.y, b.x - a.y);
  }
  __syncthreads();
#pragma unroll 1
  for (int i = slot; i < 2 * R1 * R2; i += NS) {
    Cx<T> v[R3];
    const int g = i & 1, base = i * R3, pe = base + g, po = base - g;
#pragma unroll
    for (int u = 0; u < R3; ++u) v[u] = sm[(((u & 1) ? po : pe) + u) * B + lane];
    inv_first<T, L>(sm, lane, i, v);
  }
  __syncthreads();
  inv_middle<T, L>(sm, W, lane, slot);
  __syncthreads();
  Cx<T>* out = Hp + pair;
#pragma unroll 1
  for (int bf = slot; bf < q1; bf += NS) {
    Cx<T> v[R1];
    inv_last<T, L>(sm, W, lane, bf, v);
    if (ok) {
#pragma unroll
      for (int s = 0; s < R1; ++s)
        out[(size_t)(bf + q1 * s) * npairs] = mk<T>(scale * v[s].x, scale * v[s].y);
    }
  }
}

// ---------------------------------------------------------------- K3: fused z pass (S3)
template <typename T, int G> struct ZpCfg {
  static constexpr int nz = 8 * G, Pz = 16 * G, Q = 3 * nz;
  static constexpr int OZP = nz + 2;        // kz pitch of a table row (InitGeom::ozp)
  static constexpr int NPW = 32 / G;        // pencils per warp task
  static constexpr int NSUB = 16 / G;       // second-stage sub-transforms per lane
  static constexpr int PITCH = G + 1;       // exchange row pitch (conflict-free transposition)
  static constexpr int XB = 16 * PITCH;     // exchange elements per pencil (aliases the pencil)
  // One persistent CTA per SM holding every warp the register file and shared memory admit
  // (fp32: 12 x 164 registers, 12 x 18.1 KB): warps of one CTA start together and stay close
  // in the 70 KB instruction stream, which three independent 4-warp CTAs did not (1.06 -> 0.93 ms
  // at config 4, profiles/r01_v3_*.md).  fp64: 6 warps (36.3 KB per warp, 255 registers).
  static constexpr int WARPS = sizeof(T) == 4 ? 12 : 7;
  static constexpr int MINB = 1;
  // fp64: the 15 inter-stage roots of a lane (60 registers) live in shared memory, [u][t]
  static constexpr int TWS = sizeof(T) == 4 ? 1 : G;
  static constexpr int tw_bytes = sizeof(T) == 4 ? 0 : 16 * G * (int)sizeof(Cx<T>);
  static constexpr int pencil_bytes = Q * (int)sizeof(Cx<T>);
  // Pencil pitch in shared memory.  With G < 16 a half warp (fp32) holds 16 / G pencils whose lanes touch the same
  // relative positions; Q = 24 G is a multiple of 16 complex values, so dense pencils would share their banks (G = 8:
  // 43 % of the wavefronts were conflicts and the pass ran at 92 % L1/shared throughput, profiles/r02_k3_thin.md).
  // A pitch of Q + G shifts the pencils of a half warp by G banks: with each lane taking the first-stage outputs
  // k1 = t + G i every access pattern of the kernel then covers all 16 banks once.
  static constexpr int PQ = Q + (G < 16 ? G : 0);
  static constexpr int slot_bytes = PQ * (int)sizeof(Cx<T>);
  static constexpr int table_bytes = 6 * OZP * (int)sizeof(T);  // one (kx, ky) row, 16 B multiple
  // per warp: two stages of NPW pencils + the table rows of the NPW / 2 mirror pairs.  The row ky = ny (the
  // partner of ky = 0, the only pair that does not share its row) is needed by one task per plane: it lands in
  // the pencil area of the OTHER stage, whose prefetch that task defers until its multiply is done, instead of
  // in a slot of its own (fp64: 37.1 -> 30.8 KB per warp, 7 warps instead of 6).
  static constexpr int warp_bytes = 2 * NPW * slot_bytes + (NPW / 2) * table_bytes;
  static constexpr int hdr_for(int warps) { return (4 * warps * 8 + 127) / 128 * 128; }  // mbarriers
  static constexpr int smem_for(int warps) { return hdr_for(warps) + warps * warp_bytes + tw_bytes; }
  static constexpr int smem_bytes = smem_for(WARPS);
  static_assert(XB <= Q, "exchange buffer must fit in the pencil it aliases");
  static_assert(table_bytes <= NPW * slot_bytes, "the row ky = ny must fit in a stage's pencil area");
  static_assert(table_bytes % 16 == 0 && pencil_bytes % 16 == 0 && slot_bytes % 16 == 0, "bulk copies need 16 B multiples");
};

// Forward z transform of one component of one pencil.  a[j] = sample z = t + G j (j < 8; the
// samples j >= 8 are the zero padding).  X[i G + v] = spectrum at kz = t + G i + 16 v.
template <typename T, int G>
__device__ __forceinline__ void zp_forward(const Cx<T>* a, Cx<T>* xb, const Cx<T>* tw, int t,
                                           Cx<T>* X) {
  using C = ZpCfg<T, G>;
  Cx<T> e[8], o[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) e[j] = a[j];
  // pruned radix 16: even outputs = DFT8(a), odd outputs = DFT8(a w16^j)
  o[0] = e[0];
  o[1] = mul_root<T, 16, 1, false>(e[1]);
  o[2] = mul_root<T, 16, 2, false>(e[2]);
  o[3] = mul_root<T, 16, 3, false>(e[3]);
  o[4] = mul_root<T, 16, 4, false>(e[4]);
  o[5] = mul_root<T, 16, 5, false>(e[5]);
  o[6] = mul_root<T, 16, 6, false>(e[6]);
  o[7] = mul_root<T, 16, 7, false>(e[7]);
  Dft<T, 8, false>::run(e);
  Dft<T, 8, false>::run(o);
  xb[t] = e[0];
#pragma unroll
  for (int v = 0; v < 8; ++v) {
    if (v) xb[(2 * v) * C::PITCH + t] = cmul(e[v], tw[(2 * v) * C::TWS]);
    xb[(2 * v + 1) * C::PITCH + t] = cmul(o[v], tw[(2 * v + 1) * C::TWS]);
  }
  __syncwarp();
#pragma unroll
  for (int i = 0; i < C::NSUB; ++i) {
    Cx<T> b[G];
#pragma unroll
    for (int tp = 0; tp < G; ++tp) b[tp] = xb[(t + G * i) * C::PITCH + tp];
    Dft<T, G, false>::run(b);
#pragma unroll
    for (int v = 0; v < G; ++v) X[i * G + v] = b[v];
  }
  __syncwarp();
}

// Mirror image: X -> the 8 truncated samples z = t + G j of this lane, in r[j].
template <typename T, int G>
__device__ __forceinline__ void zp_inverse(Cx<T>* r, Cx<T>* xb, const Cx<T>* tw, int t,
                                           const Cx<T>* X) {
  using C = ZpCfg<T, G>;
#pragma unroll
  for (int i = 0; i < C::NSUB; ++i) {
    Cx<T> b[G];
#pragma unroll
    for (int v = 0; v < G; ++v) b[v] = X[i * G + v];
    Dft<T, G, true>::run(b);
#pragma unroll
    for (int tp = 0; tp < G; ++tp) xb[(t + G * i) * C::PITCH + tp] = b[tp];
  }
  __syncwarp();
  Cx<T> e[8], o[8];
  e[0] = xb[t];
#pragma unroll
  for (int v = 0; v < 8; ++v) {
    if (v) e[v] = cmulc(xb[(2 * v) * C::PITCH + t], tw[(2 * v) * C::TWS]);
    o[v] = cmulc(xb[(2 * v + 1) * C::PITCH + t], tw[(2 * v + 1) * C::TWS]);
  }
  __syncwarp();
  Dft<T, 8, true>::run(e);
  Dft<T, 8, true>::run(o);
  r[0] = cadd(e[0], o[0]);
  r[1] = add_root<T, 16, 1, true>(e[1], o[1]);
  r[2] = add_root<T, 16, 2, true>(e[2], o[2]);
  r[3] = add_root<T, 16, 3, true>(e[3], o[3]);
  r[4] = add_root<T, 16, 4, true>(e[4], o[4]);
  r[5] = add_root<T, 16, 5, true>(e[5], o[5]);
  r[6] = add_root<T, 16, 6, true>(e[6], o[6]);
  r[7] = add_root<T, 16, 7, true>(e[7], o[7]);
}

// Hhat = Nhat mhat at the 16 frequencies of this lane.  trow: the (kx, ky) table row in shared
// memory, [6][OZP]; s3, s4, s5: signs of N_xy, N_xz, N_yz on the mirrored half of the row axis (ky rows:
// N_xy, N_yz are odd in ky, so (s, 1, s); kx rows of the slab layout: N_xy, N_xz odd in kx, (s, s, 1)); the kz
// mirror (N_xz, N_yz odd in kz) is resolved per frequency.
template <typename T, int G>
__device__ __forceinline__ void zp_multiply(const T* trow, int t, T s3, T s4, T s5, Cx<T>* X0, Cx<T>* X1,
                                            Cx<T>* X2) {
  using C = ZpCfg<T, G>;
#pragma unroll
  for (int f = 0; f < 16; ++f) {
    const int kz = t + G * (f / G) + 16 * (f % G);
    // kz > nz (the mirrored half, where N_xz and N_yz change sign) is known at compile time
    // except for the one block of frequencies that straddles kz = nz
    bool mir;
    if ((f % G) < G / 2) mir = false;
    else if ((f % G) > G / 2) mir = true;
    else mir = kz > C::nz;
    const int idx = mir ? C::Pz - kz : kz;
    const T nxx = trow[idx], nyy = trow[C::OZP + idx], nzz = trow[2 * C::OZP + idx],
            nxy = s3 * trow[3 * C::OZP + idx];
    T nxz = s4 * trow[4 * C::OZP + idx], nyz = s5 * trow[5 * C::OZP + idx];
    if (mir) { nxz = -nxz; nyz = -nyz; }
    const Cx<T> a = X0[f], b = X1[f], c = X2[f];
    X0[f] = mk<T>(nxx * a.x + nxy * b.x + nxz * c.x, nxx * a.y + nxy * b.y + nxz * c.y);
    X1[f] = mk<T>(nxy * a.x + nyy * b.x + nyz * c.x, nxy * a.y + nyy * b.y + nyz * c.y);
    X2[f] = mk<T>(nxz * a.x + nyz * b.x + nzz * c.x, nxz * a.y + nyz * b.y + nzz * c.y);
  }
}

// A2 points at the first plane of the launch, whose kx is kx0.  One warp task = NPW pencils =
// NPW/2 mirror pairs (ky, Py - ky) of one plane, which share their Nhat rows.  Pencils and
// table rows arrive by bulk asynchronous copies one task ahead; the pencil's own buffer is
// the exchange buffer of its transforms once its samples sit in registers.
// xm != 0 (MASK variant only): the rows of a plane are kx, not ky (slab layout, demag_slab.cuh).
// MASK: the mesh has nzd < 8 G layers (any period Pz >= 2 nzd - 1 gives the same linear convolution, reading
// Q27): pencils in HBM hold 3 nzd values, the samples z >= nzd read as zero and only 3 nzd values go back.
// CONTIG (only without MASK): the rows of a plane lie in natural ky order (two-stage y pass), so the table rows of
// the NPW/2 mirror pairs of a task are one contiguous run: one bulk copy instead of NPW/2.
template <typename T, int G, int WARPS, int MINB, bool MASK, bool CONTIG = false>
__global__ void __launch_bounds__(WARPS * 32, MINB)
zp_fast_kernel(Cx<T>* __restrict__ A2, const T* __restrict__ tab, const Cx<T>* __restrict__ Wz,
               const uint16_t* __restrict__ posy, int ny, int kx0, int ntask, int nzd, int xm) {
  using C = ZpCfg<T, G>;
  constexpr int Q = C::Q, NPW = C::NPW;
  const int qd = MASK ? 3 * nzd : Q;                                    // values of a pencil in HBM
  const uint32_t pbytes = MASK ? (uint32_t)(qd * sizeof(Cx<T>)) : (uint32_t)C::pencil_bytes;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw) + 4 * warp;  // stage 0, stage 1, table, row ky = ny
  unsigned char* wraw = smem_raw + C::hdr_for(WARPS) + (size_t)warp * C::warp_bytes;
  Cx<T>* pbase = reinterpret_cast<Cx<T>*>(wraw);
  T* tbase = reinterpret_cast<T*>(wraw + 2 * NPW * C::slot_bytes);
  const int t = lane % G, pw = lane / G;
  const int Py = 2 * ny;
  if (threadIdx.x == 0) {
    for (int i = 0; i < 4 * WARPS; ++i) mbar_init(reinterpret_cast<uint64_t*>(smem_raw) + i, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if constexpr (sizeof(T) == 8) {
    Cx<T>* tws = reinterpret_cast<Cx<T>*>(smem_raw + C::hdr_for(WARPS) + (size_t)WARPS * C::warp_bytes);
    for (int i = threadIdx.x; i < 16 * G; i += WARPS * 32) tws[i] = __ldg(Wz + (i % G) * (i / G));
  }
  __syncthreads();
  Cx<T> twr[sizeof(T) == 4 ? 16 : 1];
  const Cx<T>* tw = twr;
  if constexpr (sizeof(T) == 4) {
#pragma unroll
    for (int u = 1; u < 16; ++u) twr[u] = __ldg(Wz + t * u);
    twr[0] = mk<T>(1, 0);
  } else {
    tw = reinterpret_cast<const Cx<T>*>(smem_raw + C::hdr_for(WARPS) + (size_t)WARPS * C::warp_bytes) + t;
  }

  const int gw = blockIdx.x * WARPS + warp, stride = gridDim.x * WARPS;
  auto pencil_ptr = [&](int task, int p) -> Cx<T>* {
    const int pair = task * (NPW / 2) + (p >> 1);
    const int plane = pair / ny, i = pair - plane * ny;
    const int ky = (p & 1) ? (i == 0 ? ny : Py - i) : i;
    return A2 + ((size_t)plane * Py + posy[ky]) * qd;
  };
  auto issue = [&](int task, int stage) {
    mbar_expect_tx(bars + stage, NPW * pbytes);
    for (int p = 0; p < NPW; ++p)
      bulk_load(pbase + (stage * NPW + p) * C::PQ, pencil_ptr(task, p), pbytes, bars + stage);
  };
  // table rows of a task: ky = i for mirror pair i; the pair i = 0 (always the first of its
  // task) is (ky = 0, ky = ny) and needs the row ky = ny as well (issue_nyq)
  auto issue_table = [&](int task) {
    const int pair0 = task * (NPW / 2);
    const int plane = pair0 / ny, i0 = pair0 - plane * ny;
    const T* rows = tab + ((size_t)(kx0 + plane) * (ny + 1)) * 6 * C::OZP;
    mbar_expect_tx(bars + 2, (NPW / 2) * C::table_bytes);
    if constexpr (CONTIG) {   // the rows ky = i0 .. i0 + NPW/2 - 1 are one run of the table
      bulk_load(tbase, rows + (size_t)i0 * 6 * C::OZP, (NPW / 2) * C::table_bytes, bars + 2);
    } else {
      for (int pp = 0; pp < NPW / 2; ++pp)
        bulk_load(tbase + pp * 6 * C::OZP, rows + (size_t)(i0 + pp) * 6 * C::OZP, C::table_bytes, bars + 2);
    }
  };
  // the row ky = ny of a task that holds pair 0, into the pencil area of the stage the task does not use
  auto issue_nyq = [&](int task, int other) {
    const int plane = task * (NPW / 2) / ny;
    const T* rows = tab + ((size_t)(kx0 + plane) * (ny + 1)) * 6 * C::OZP;
    mbar_expect_tx(bars + 3, C::table_bytes);
    bulk_load(pbase + other * NPW * C::PQ, rows + (size_t)ny * 6 * C::OZP, C::table_bytes, bars + 3);
  };
  if (lane == 0 && gw < ntask) { issue(gw, 0); issue_table(gw); }
  int it = 0, nq = 0;
  // not unrolled: the body is ~2,300 instructions and two copies of it (the compiler's choice,
  // to make `stage` a constant) overflow the instruction cache
#pragma unroll 1
  for (int task = gw; task < ntask; task += stride, ++it) {
    const int stage = it & 1;
    const bool more = task + stride < ntask;
    const bool has0 = (task * (NPW / 2)) % ny == 0;   // this task holds the pair (ky = 0, ky = ny)
    if (lane == 0) {
      bulk_wait_read0();  // the previous task's store has finished reading the other stage
      if (has0) issue_nyq(task, stage ^ 1);
      else if (more) issue(task + stride, stage ^ 1);
    }
    __syncwarp();
    mbar_wait(bars + stage, (it >> 1) & 1);
    Cx<T>* pen = pbase + (stage * NPW + pw) * C::PQ;
    Cx<T> X[3][16];
    {
      Cx<T> a[3][8];
#pragma unroll
      for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int j = 0; j < 8; ++j)
          a[c][j] = (!MASK || t + G * j < nzd) ? pen[(t + G * j) * 3 + c] : mk<T>((T)0, (T)0);
      __syncwarp();  // every sample is in registers: the pencil buffer becomes the exchange buffer
#pragma unroll
      for (int c = 0; c < 3; ++c) zp_forward<T, G>(a[c], pen, tw, t, X[c]);
    }
    // ---- tensor multiply
    {
      const int pair = task * (NPW / 2) + (pw >> 1);
      const int i = pair % ny;
      // the odd pencil of pair i is ky = Py - i (row i, odd components negated), of pair 0 ky = ny
      const bool nyq = (pw & 1) && i == 0;
      const T sy = ((pw & 1) && i != 0) ? (T)-1 : (T)1;
      const T s4 = (MASK && xm) ? sy : (T)1, s5 = (MASK && xm) ? (T)1 : sy;
      mbar_wait(bars + 2, it & 1);
      if (has0) { mbar_wait(bars + 3, nq & 1); ++nq; }
      const T* trow = nyq ? reinterpret_cast<const T*>(pbase + (stage ^ 1) * NPW * C::PQ)
                          : tbase + (pw >> 1) * 6 * C::OZP;
      zp_multiply<T, G>(trow, t, sy, s4, s5, X[0], X[1], X[2]);
      if (has0) fence_async_smem();   // the row was read through the generic proxy; pencils land there next
      __syncwarp();
      if (lane == 0 && more) {
        issue_table(task + stride);
        if (has0) issue(task + stride, stage ^ 1);   // the prefetch this task deferred
      }
    }
    // ---- inverse; the truncated samples go back into the staged pencil
    {
      Cx<T> r[3][8];
#pragma unroll
      for (int c = 0; c < 3; ++c) zp_inverse<T, G>(r[c], pen, tw, t, X[c]);
      __syncwarp();  // the last exchange has been read
#pragma unroll
      for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int j = 0; j < 8; ++j) pen[(t + G * j) * 3 + c] = r[c][j];
    }
    fence_async_smem();
    __syncwarp();
    if (lane == 0) {
      for (int p = 0; p < NPW; ++p)
        bulk_store(pencil_ptr(task, p), pbase + (stage * NPW + p) * C::PQ, pbytes);
      bulk_commit();
    }
  }
  if (lane == 0) bulk_wait0();
}

// ---------------------------------------------------------------- K3 for nz = 256 (fp32)
// Pz = 512 = 16 x 32: all 32 lanes of a warp own ONE pencil, 16 frequencies x 3 components per
// lane as above.  The second stage is a radix-32 transform per first-stage output k1 (16 of
// them): it is split over the lane pair (k1, h): h = 0 computes its even outputs (radix 16 of
// b[s] + b[s + 16]), h = 1 its odd outputs (radix 16 of (b[s] - b[s + 16]) w32^s), both reading
// all 32 exchanged values.  Lane t = k1 + 16 h then holds the spectrum at kz = t + 32 u, u < 16.
// The way back mirrors it: each lane writes g[s] = IDFT16(X)[s] (h = 1: times conj w32^s) to slot
// s + 16 h, and the first-stage reader combines b[tp] = g[tp & 15] +- g[(tp & 15) + 16].
// Pencils are processed one at a time (the two pencils of a mirror pair (ky, Py - ky) in turn,
// sharing one staged Nhat row), double buffered by bulk copies as in zp_fast_kernel.
template <typename T> struct ZwCfg {
  static constexpr int nz = 256, Pz = 512, Q = 3 * nz, OZP = nz + 2, PITCH = 33;
  static constexpr int WARPS = sizeof(T) == 4 ? 12 : 6;
  static constexpr int pencil_bytes = Q * (int)sizeof(Cx<T>);
  static constexpr int table_bytes = 6 * OZP * (int)sizeof(T);
  static constexpr int warp_bytes = 2 * pencil_bytes + table_bytes;
  static constexpr int hdr_bytes = (3 * WARPS * 8 + 127) / 128 * 128;
  // fp64: the 15 inter-stage roots of a lane live in shared memory, [u][t] (as in zp_fast_kernel)
  static constexpr int TWS = sizeof(T) == 4 ? 1 : 32;
  static constexpr int tw_bytes = sizeof(T) == 4 ? 0 : 16 * 32 * (int)sizeof(Cx<T>);
  static constexpr int smem_bytes = hdr_bytes + WARPS * warp_bytes + tw_bytes;
  static_assert(smem_bytes <= 227 * 1024, "one CTA per SM");
  static_assert(16 * PITCH <= Q, "exchange buffer must fit in the pencil it aliases");
  static_assert(table_bytes % 16 == 0 && pencil_bytes % 16 == 0, "bulk copies need 16 B multiples");
};

template <typename T, int... S>
__device__ __forceinline__ void zw_half_fwd(const Cx<T>* row, T sgn, bool h, Cx<T>* c,
                                            std::integer_sequence<int, S...>) {
  ((c[S] = [&] {
     const Cx<T> lo = row[S], hi = row[S + 16];
     const Cx<T> d = mk<T>(fma(sgn, hi.x, lo.x), fma(sgn, hi.y, lo.y));
     const Cx<T> r = mul_root<T, 32, S, false>(d);
     return h ? r : d;
   }()),
   ...);
}
template <typename T, int... S>
__device__ __forceinline__ void zw_half_inv(Cx<T>* row, bool h, const Cx<T>* c,
                                            std::integer_sequence<int, S...>) {
  ((row[S] = h ? mul_root<T, 32, S, true>(c[S]) : c[S]), ...);
}

// a[j] = sample z = t + 32 j (j < 8)  ->  X[u] = spectrum at kz = t + 32 u
template <typename T>
__device__ __forceinline__ void zw_forward(const Cx<T>* a, Cx<T>* xb, const Cx<T>* tw, int t, Cx<T>* X) {
  using C = ZwCfg<T>;
  Cx<T> e[8], o[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) e[j] = a[j];
  o[0] = e[0];
  o[1] = mul_root<T, 16, 1, false>(e[1]);
  o[2] = mul_root<T, 16, 2, false>(e[2]);
  o[3] = mul_root<T, 16, 3, false>(e[3]);
  o[4] = mul_root<T, 16, 4, false>(e[4]);
  o[5] = mul_root<T, 16, 5, false>(e[5]);
  o[6] = mul_root<T, 16, 6, false>(e[6]);
  o[7] = mul_root<T, 16, 7, false>(e[7]);
  Dft<T, 8, false>::run(e);
  Dft<T, 8, false>::run(o);
  xb[t] = e[0];
#pragma unroll
  for (int v = 0; v < 8; ++v) {
    if (v) xb[(2 * v) * C::PITCH + t] = cmul(e[v], tw[(2 * v) * C::TWS]);
    xb[(2 * v + 1) * C::PITCH + t] = cmul(o[v], tw[(2 * v + 1) * C::TWS]);
  }
  __syncwarp();
  const bool h = t >= 16;
  zw_half_fwd<T>(xb + (t & 15) * C::PITCH, h ? (T)-1 : (T)1, h, X, std::make_integer_sequence<int, 16>{});
  Dft<T, 16, false>::run(X);
  __syncwarp();
}

template <typename T>
__device__ __forceinline__ void zw_inverse(Cx<T>* r, Cx<T>* xb, const Cx<T>* tw, int t, const Cx<T>* X) {
  using C = ZwCfg<T>;
  const bool h = t >= 16;
  {
    Cx<T> c[16];
#pragma unroll
    for (int u = 0; u < 16; ++u) c[u] = X[u];
    Dft<T, 16, true>::run(c);
    zw_half_inv<T>(xb + (t & 15) * C::PITCH + (h ? 16 : 0), h, c, std::make_integer_sequence<int, 16>{});
  }
  __syncwarp();
  const T sgn = h ? (T)-1 : (T)1;
  const Cx<T>* col = xb + (t & 15);
  Cx<T> e[8], o[8];
#pragma unroll
  for (int v = 0; v < 8; ++v) {
    const Cx<T> l0 = col[(2 * v) * C::PITCH], h0 = col[(2 * v) * C::PITCH + 16];
    const Cx<T> l1 = col[(2 * v + 1) * C::PITCH], h1 = col[(2 * v + 1) * C::PITCH + 16];
    const Cx<T> b0 = mk<T>(fma(sgn, h0.x, l0.x), fma(sgn, h0.y, l0.y));
    const Cx<T> b1 = mk<T>(fma(sgn, h1.x, l1.x), fma(sgn, h1.y, l1.y));
    e[v] = v ? cmulc(b0, tw[(2 * v) * C::TWS]) : b0;
    o[v] = cmulc(b1, tw[(2 * v + 1) * C::TWS]);
  }
  __syncwarp();
  Dft<T, 8, true>::run(e);
  Dft<T, 8, true>::run(o);
  r[0] = cadd(e[0], o[0]);
  r[1] = add_root<T, 16, 1, true>(e[1], o[1]);
  r[2] = add_root<T, 16, 2, true>(e[2], o[2]);
  r[3] = add_root<T, 16, 3, true>(e[3], o[3]);
  r[4] = add_root<T, 16, 4, true>(e[4], o[4]);
  r[5] = add_root<T, 16, 5, true>(e[5], o[5]);
  r[6] = add_root<T, 16, 6, true>(e[6], o[6]);
  r[7] = add_root<T, 16, 7, true>(e[7], o[7]);
}

template <typename T>
__device__ __forceinline__ void zw_multiply(const T* trow, int t, T s3, T s4, T s5, Cx<T>* X0, Cx<T>* X1, Cx<T>* X2) {
  using C = ZwCfg<T>;
#pragma unroll
  for (int u = 0; u < 16; ++u) {
    const int kz = t + 32 * u;
    bool mir;
    if (u < 8) mir = false;
    else if (u > 8) mir = true;
    else mir = t > 0;
    const int idx = mir ? C::Pz - kz : kz;
    const T nxx = trow[idx], nyy = trow[C::OZP + idx], nzz = trow[2 * C::OZP + idx],
            nxy = s3 * trow[3 * C::OZP + idx];
    T nxz = s4 * trow[4 * C::OZP + idx], nyz = s5 * trow[5 * C::OZP + idx];
    if (mir) { nxz = -nxz; nyz = -nyz; }
    const Cx<T> a = X0[u], b = X1[u], c = X2[u];
    X0[u] = mk<T>(nxx * a.x + nxy * b.x + nxz * c.x, nxx * a.y + nxy * b.y + nxz * c.y);
    X1[u] = mk<T>(nxy * a.x + nyy * b.x + nyz * c.x, nxy * a.y + nyy * b.y + nyz * c.y);
    X2[u] = mk<T>(nxz * a.x + nyz * b.x + nzz * c.x, nxz * a.y + nyz * b.y + nzz * c.y);
  }
}

// A2 points at the first plane of the launch (kx = kx0).  A warp walks mirror pairs
// pair = plane ny + i -> pencils ky = i and ky = (i == 0 ? ny : Py - i), one pencil per step.
template <typename T, bool MASK>
__global__ void __launch_bounds__(ZwCfg<T>::WARPS * 32, 1)
zw_fast_kernel(Cx<T>* __restrict__ A2, const T* __restrict__ tab, const Cx<T>* __restrict__ Wz,
               const uint16_t* __restrict__ posy, int ny, int kx0, int npair, int nzd, int xm) {
  using C = ZwCfg<T>;
  constexpr int Q = C::Q;
  const int qd = MASK ? 3 * nzd : Q;                                    // values of a pencil in HBM (see zp_fast_kernel)
  const uint32_t pbytes = MASK ? (uint32_t)(qd * sizeof(Cx<T>)) : (uint32_t)C::pencil_bytes;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, t = threadIdx.x & 31;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw) + 3 * warp;  // pencil buffer 0, 1, table
  unsigned char* wraw = smem_raw + C::hdr_bytes + (size_t)warp * C::warp_bytes;
  Cx<T>* pbase = reinterpret_cast<Cx<T>*>(wraw);
  T* trow = reinterpret_cast<T*>(wraw + 2 * C::pencil_bytes);
  const int Py = 2 * ny;
  if (threadIdx.x == 0) {
    for (int i = 0; i < 3 * C::WARPS; ++i) mbar_init(reinterpret_cast<uint64_t*>(smem_raw) + i, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if constexpr (sizeof(T) == 8) {
    Cx<T>* tws = reinterpret_cast<Cx<T>*>(smem_raw + C::hdr_bytes + (size_t)C::WARPS * C::warp_bytes);
    for (int i = threadIdx.x; i < 16 * 32; i += C::WARPS * 32) tws[i] = __ldg(Wz + (i % 32) * (i / 32));
  }
  __syncthreads();
  Cx<T> twr[sizeof(T) == 4 ? 16 : 1];
  const Cx<T>* tw = twr;
  if constexpr (sizeof(T) == 4) {
#pragma unroll
    for (int u = 1; u < 16; ++u) twr[u] = __ldg(Wz + t * u);
    twr[0] = mk<T>(1, 0);
  } else {
    tw = reinterpret_cast<const Cx<T>*>(smem_raw + C::hdr_bytes + (size_t)C::WARPS * C::warp_bytes) + t;
  }

  const int gw = blockIdx.x * C::WARPS + warp, stride = gridDim.x * C::WARPS;
  const int mine = gw < npair ? (npair - gw + stride - 1) / stride : 0;  // pairs of this warp
  const int nsteps = 2 * mine;
  auto pencil_ptr = [&](int step) -> Cx<T>* {
    const int pair = gw + (step >> 1) * stride;
    const int plane = pair / ny, i = pair - plane * ny;
    const int ky = (step & 1) ? (i == 0 ? ny : Py - i) : i;
    return A2 + ((size_t)plane * Py + posy[ky]) * qd;
  };
  // Nhat row of a step; -1 if it is the row already staged (second pencil of a pair i != 0)
  auto table_row = [&](int step) -> long long {
    const int pair = gw + (step >> 1) * stride;
    const int plane = pair / ny, i = pair - plane * ny;
    if ((step & 1) && i != 0) return -1;
    return ((long long)(kx0 + plane) * (ny + 1) + ((step & 1) ? ny : i));
  };
  if (t == 0 && nsteps > 0) {
    mbar_expect_tx(bars + 0, pbytes);
    bulk_load(pbase, pencil_ptr(0), pbytes, bars + 0);
    mbar_expect_tx(bars + 2, C::table_bytes);
    bulk_load(trow, tab + (size_t)table_row(0) * 6 * C::OZP, C::table_bytes, bars + 2);
  }
  int tphase = 0;
#pragma unroll 1
  for (int step = 0; step < nsteps; ++step) {
    const int buf = step & 1;
    if (t == 0) {
      bulk_wait_read0();  // the previous step's store has finished reading the other buffer
      if (step + 1 < nsteps) {
        mbar_expect_tx(bars + (buf ^ 1), pbytes);
        bulk_load(pbase + (buf ^ 1) * Q, pencil_ptr(step + 1), pbytes, bars + (buf ^ 1));
      }
    }
    __syncwarp();
    mbar_wait(bars + buf, (step >> 1) & 1);
    Cx<T>* pen = pbase + buf * Q;
    Cx<T> X[3][16];
    {
      Cx<T> a[3][8];
#pragma unroll
      for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int j = 0; j < 8; ++j)
          a[c][j] = (!MASK || t + 32 * j < nzd) ? pen[(t + 32 * j) * 3 + c] : mk<T>((T)0, (T)0);
      __syncwarp();  // every sample is in registers: the pencil buffer becomes the exchange buffer
#pragma unroll
      for (int c = 0; c < 3; ++c) zw_forward<T>(a[c], pen, tw, t, X[c]);
    }
    {
      const int pair = gw + (step >> 1) * stride;
      const int i = pair % ny;
      const T sy = ((step & 1) && i != 0) ? (T)-1 : (T)1;
      const T s4 = (MASK && xm) ? sy : (T)1, s5 = (MASK && xm) ? (T)1 : sy;
      if (table_row(step) >= 0) { mbar_wait(bars + 2, tphase); tphase ^= 1; }
      zw_multiply<T>(trow, t, sy, s4, s5, X[0], X[1], X[2]);
      __syncwarp();
      if (t == 0 && step + 1 < nsteps) {
        const long long row = table_row(step + 1);
        if (row >= 0) {
          mbar_expect_tx(bars + 2, C::table_bytes);
          bulk_load(trow, tab + (size_t)row * 6 * C::OZP, C::table_bytes, bars + 2);
        }
      }
    }
    {
      Cx<T> r[3][8];
#pragma unroll
      for (int c = 0; c < 3; ++c) zw_inverse<T>(r[c], pen, tw, t, X[c]);
      __syncwarp();  // the last exchange has been read
#pragma unroll
      for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int j = 0; j < 8; ++j) pen[(t + 32 * j) * 3 + c] = r[c][j];
    }
    fence_async_smem();
    __syncwarp();
    if (t == 0) {
      bulk_store(pencil_ptr(step), pen, pbytes);
      bulk_commit();
    }
  }
  if (t == 0) bulk_wait0();
}

// ---------------------------------------------------------------- host side

// z: the warp-per-pencil kernels hold nzt = 64, 128 or 256 layers and take any 16 <= nz <= nzt (at most four
// times the layers: K3 is a third of the work) whose pencils are multiples of 16 bytes (bulk copies); above
// 256 layers the tile pass of demag_ztile.cu with a plan of its own.
int fast_z_transform(int nz, size_t real_bytes, int ny) {
  if (nz >= 16 && nz <= 256 && ((size_t)3 * nz * 2 * real_bytes) % 16 == 0)
    return (nz <= 32 && ny % 4 == 0) ? 32 : (nz <= 64 ? 64 : (nz <= 128 ? 128 : 256));
  return ztile_supported(nz) ? nz : 0;
}
// x, y: a two-stage plan (plan2.cuh) or the three-stage L = 1024 kernels.  K1 / K5 move the real arrays as
// complex pairs.
bool fast_supported(int nx, int ny, int nz, size_t real_bytes) {
  auto okxy = [](int n) { return fast_two_stage(n) || n == 1024; };
  const int nzt = fast_z_transform(nz, real_bytes, ny);
  // the nzt = 64 / 32 kernels walk two / four mirror pairs of ky per task (nzt = 32 only where ny is a multiple of 4)
  return okxy(nx) && okxy(ny) && nzt != 0 && ((size_t)ny * 3 * nz) % 2 == 0 && !(nzt <= 64 && ny % 2);
}

template <typename K> static cudaError_t opt_in_smem(K kernel, int bytes) {
  if (bytes <= 48 * 1024) return cudaSuccess;
  return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}

static int g_sm_count = 0;
static int sm_count() {
  if (!g_sm_count) {
    int dev = 0;
    cudaGetDevice(&dev);
    if (cudaDeviceGetAttribute(&g_sm_count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        g_sm_count <= 0)
      g_sm_count = 148;
  }
  return g_sm_count;
}

template <typename T, int L>
static cudaError_t launch_xf(const FastGeom& g, const FastBufs<T>& b, const T* m, cudaStream_t st) {
  using TL = Tile<T, L>;
  cudaError_t e = opt_in_smem(xf_fast_kernel<T, L>, TL::smem_bytes);
  if (e != cudaSuccess) return e;
  const size_t npairs = (size_t)g.ny * g.Q / 2;
  xf_fast_kernel<T, L><<<(unsigned)((npairs + TL::B - 1) / TL::B), TL::NT, TL::smem_bytes, st>>>(
      reinterpret_cast<const Cx<T>*>(m), b.A1, b.Wx, b.posx, npairs);
  return cudaSuccess;
}
template <typename T, int L>
static cudaError_t launch_xi(const FastGeom& g, const FastBufs<T>& b, T* H, T scale, cudaStream_t st) {
  using TL = Tile<T, L>;
  cudaError_t e = opt_in_smem(xi_fast_kernel<T, L>, TL::smem_bytes);
  if (e != cudaSuccess) return e;
  const size_t npairs = (size_t)g.ny * g.Q / 2;
  xi_fast_kernel<T, L><<<(unsigned)((npairs + TL::B - 1) / TL::B), TL::NT, TL::smem_bytes, st>>>(
      b.A1, reinterpret_cast<Cx<T>*>(H), b.Wx, b.posx, npairs, scale);
  return cudaSuccess;
}
template <typename T, int L>
static cudaError_t launch_yf(const FastGeom& g, const FastBufs<T>& b, int k0, int nk, cudaStream_t st) {
  using TL = Tile<T, L>;
  cudaError_t e = opt_in_smem(yf_fast_kernel<T, L>, TL::smem_bytes);
  if (e != cudaSuccess) return e;
  dim3 grid((g.Q + TL::B - 1) / TL::B, nk);
  yf_fast_kernel<T, L><<<grid, TL::NT, TL::smem_bytes, st>>>(
      b.A1 + (size_t)k0 * g.ny * g.Q, b.A2, b.Wy, g.Q);
  return cudaSuccess;
}
template <typename T, int L>
static cudaError_t launch_yi(const FastGeom& g, const FastBufs<T>& b, int k0, int nk, cudaStream_t st) {
  using TL = Tile<T, L>;
  cudaError_t e = opt_in_smem(yi_fast_kernel<T, L>, TL::smem_bytes);
  if (e != cudaSuccess) return e;
  dim3 grid((g.Q + TL::B - 1) / TL::B, nk);
  yi_fast_kernel<T, L><<<grid, TL::NT, TL::smem_bytes, st>>>(
      b.A2, b.A1 + (size_t)k0 * g.ny * g.Q, b.Wy, g.Q);
  return cudaSuccess;
}
template <typename T, int G>
static cudaError_t launch_zp(const FastGeom& g, const FastBufs<T>& b, int k0, int nk, int xm, cudaStream_t st) {
  using C = ZpCfg<T, G>;
  constexpr int WARPS = C::WARPS, MINB = C::MINB;
  const int ntask = (int)((size_t)nk * g.ny * 2 / C::NPW);
  int grid = sm_count() * MINB;
  if (grid * WARPS > ntask) grid = (ntask + WARPS - 1) / WARPS;
  cudaError_t e;
  if (g.nz == C::nz && !xm && b.two_y && C::NPW > 2) {   // rows in natural ky order: one copy per run of pencils
    if ((e = opt_in_smem(zp_fast_kernel<T, G, WARPS, MINB, false, true>, C::smem_bytes)) != cudaSuccess) return e;
    zp_fast_kernel<T, G, WARPS, MINB, false, true><<<grid, WARPS * 32, C::smem_bytes, st>>>(
        b.A2, b.table, b.Wz, b.posy, g.ny, k0, ntask, g.nz, 0);
  } else if (g.nz == C::nz && !xm) {
    if ((e = opt_in_smem(zp_fast_kernel<T, G, WARPS, MINB, false>, C::smem_bytes)) != cudaSuccess) return e;
    zp_fast_kernel<T, G, WARPS, MINB, false><<<grid, WARPS * 32, C::smem_bytes, st>>>(
        b.A2, b.table, b.Wz, b.posy, g.ny, k0, ntask, g.nz, 0);
  } else {   // fewer layers than the transform holds: masked reads, shorter copies
    if ((e = opt_in_smem(zp_fast_kernel<T, G, WARPS, MINB, true>, C::smem_bytes)) != cudaSuccess) return e;
    zp_fast_kernel<T, G, WARPS, MINB, true><<<grid, WARPS * 32, C::smem_bytes, st>>>(
        b.A2, b.table, b.Wz, b.posy, g.ny, k0, ntask, g.nz, xm);
  }
  return cudaPeekAtLastError();   // a K3 that did not launch must not pass for a field
}

template <typename T>
static cudaError_t launch_zw(const FastGeom& g, const FastBufs<T>& b, int k0, int nk, int xm, cudaStream_t st) {
  using C = ZwCfg<T>;
  const int npair = nk * g.ny;
  int grid = sm_count();
  if (grid * C::WARPS > npair) grid = (npair + C::WARPS - 1) / C::WARPS;
  cudaError_t e;
  if (g.nz == C::nz && !xm) {
    if ((e = opt_in_smem(zw_fast_kernel<T, false>, C::smem_bytes)) != cudaSuccess) return e;
    zw_fast_kernel<T, false><<<grid, C::WARPS * 32, C::smem_bytes, st>>>(b.A2, b.table, b.Wz, b.posy, g.ny, k0, npair, g.nz, 0);
  } else {
    if ((e = opt_in_smem(zw_fast_kernel<T, true>, C::smem_bytes)) != cudaSuccess) return e;
    zw_fast_kernel<T, true><<<grid, C::WARPS * 32, C::smem_bytes, st>>>(b.A2, b.table, b.Wz, b.posy, g.ny, k0, npair, g.nz, xm);
  }
  return cudaSuccess;
}

// K3 on nk planes of b.A2 starting at table plane k0; xm: the rows of a plane are kx (slab layout)
template <typename T>
cudaError_t k3_launch(const FastGeom& g, const FastBufs<T>& b, int k0, int nk, int xm, cudaStream_t st) {
  if (g.nzt == 256) return launch_zw<T>(g, b, k0, nk, xm, st);
  if (g.nzt == 128) return launch_zp<T, 16>(g, b, k0, nk, xm, st);
  if (g.nzt == 64) return launch_zp<T, 8>(g, b, k0, nk, xm, st);
  if (g.nzt == 32) return launch_zp<T, 4>(g, b, k0, nk, xm, st);
  return ztile_launch<T>(g, b, k0, nk, xm, st);
}
template cudaError_t k3_launch<float>(const FastGeom&, const FastBufs<float>&, int, int, int, cudaStream_t);
template cudaError_t k3_launch<double>(const FastGeom&, const FastBufs<double>&, int, int, int, cudaStream_t);

template <typename T>
cudaError_t demag_fast_launch(const FastGeom& g, const FastBufs<T>& b, const T* m, T* H, T scale,
                              cudaStream_t st, unsigned long long* launches, Prof* prof) {
  cudaError_t e = cudaSuccess;
  const int nplanes = g.nx + 1;
  prof->mark(0, st);
  e = strided_tma_x_launch<T>(0, g, b, m, H, scale, st);
  if (e == cudaErrorNotSupported)
    e = b.two_x ? strided2_launch<T>(0, g, b, m, H, scale, st) : launch_xf<T, 1024>(g, b, m, st);
  if (e != cudaSuccess) return e;
  prof->mark(1, st);
  e = strided_tma_launch<T>(1, g, b, st);
  if (e == cudaErrorNotSupported)
    e = b.two_y ? strided2_launch<T>(1, g, b, m, H, scale, st) : launch_yf<T, 1024>(g, b, 0, nplanes, st);
  if (e != cudaSuccess) return e;
  prof->mark(2, st);
  e = k3_launch<T>(g, b, 0, nplanes, 0, st);
  if (e != cudaSuccess) return e;
  prof->mark(3, st);
  e = strided_tma_launch<T>(3, g, b, st);
  if (e == cudaErrorNotSupported)
    e = b.two_y ? strided2_launch<T>(3, g, b, m, H, scale, st) : launch_yi<T, 1024>(g, b, 0, nplanes, st);
  if (e != cudaSuccess) return e;
  prof->mark(4, st);
  e = strided_tma_x_launch<T>(4, g, b, m, H, scale, st);
  if (e == cudaErrorNotSupported)
    e = b.two_x ? strided2_launch<T>(4, g, b, m, H, scale, st) : launch_xi<T, 1024>(g, b, H, scale, st);
  if (e != cudaSuccess) return e;
  *launches += 5;
  prof->mark(-1, st);
  return cudaGetLastError();
}

template cudaError_t demag_fast_launch<float>(const FastGeom&, const FastBufs<float>&, const float*,
                                              float*, float, cudaStream_t, unsigned long long*, Prof*);
template cudaError_t demag_fast_launch<double>(const FastGeom&, const FastBufs<double>&,
                                               const double*, double*, double, cudaStream_t,
                                               unsigned long long*, Prof*);

}  // namespace mm
