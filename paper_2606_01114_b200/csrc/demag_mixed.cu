// Mixed-radix x-first demag passes (see demag_mixed.cuh).
//
//   K1 xf : m [x][y][q] real      -> A1[kx<=nx][y][q]    x forward, r2c, pruned          (S1)
//   K2 yf : A1                    -> A2[kx][ky'][q]      y forward, pruned               (S2)
//   K3 zp : A2 in place, x Nhat                           z forward . Nhat . z inverse    (S3)
//   K4 yi : A2                    -> A1[kx][y][q]        y inverse, truncated            (S4)
//   K5 xi : A1                    -> H [x][y][q] real    x inverse, c2r, truncated       (S5)
// q = 3 z + c.  Strided passes (K1, K2, K4, K5): a CTA owns all P = 2L rows of 64 bytes of q in
// shared memory, lanes along the batch, in-place run-time radix stages (fft_core.cuh); the pruned
// transform is the pair of length-L transforms of a_j and a_j w_P^j (rows [0, L) and [L, 2L)).
// K3: a CTA owns NPAIR mirror pairs (ky, Py - ky) of one kx plane, which share their Nhat rows;
// the tile is Pz rows x (3 components x pencils) columns, so the contiguous pencil q = 3 z + c
// lands in rows z, three adjacent columns, and the stages again run with lanes along the batch.
#define MM_NO_PACKED_F32
#include "demag_mixed.cuh"

#include "fft_core.cuh"

namespace mm {

template <typename T> struct MixB { static constexpr int value = 64 / (int)sizeof(Cx<T>); };

#define MM_MIXED_PROLOGUE                                              \
  extern __shared__ __align__(16) unsigned char smem_raw[];           \
  Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw);                     \
  constexpr int B = MixB<T>::value;                                   \
  const int lane = threadIdx.x % B, slot = threadIdx.x / B, NS = blockDim.x / B; \
  const int L = pl.L, P = pl.P;

// ---------------------------------------------------------------- K2: forward y
// grid (ceil(Q / B), planes)
template <typename T>
__global__ void __launch_bounds__(256, 2) yf_mixed_kernel(const Cx<T>* __restrict__ A1, Cx<T>* __restrict__ A2,
                                                       const Cx<T>* __restrict__ W, FftPlan pl, int Q) {
  MM_MIXED_PROLOGUE
  const int col = blockIdx.x * B + lane;
  const bool ok = col < Q;
  const Cx<T>* in = A1 + (size_t)blockIdx.y * L * Q + col;
  Cx<T>* out = A2 + (size_t)blockIdx.y * P * Q + col;
  for (int y = slot; y < L; y += NS) {
    const Cx<T> v = ok ? in[(size_t)y * Q] : mk<T>(0, 0);
    sm[y * B + lane] = v;
    sm[(L + y) * B + lane] = cmul(v, __ldg(W + y));
  }
  __syncthreads();
  run_stages_fwd<T>(sm, B, lane, slot, NS, P, pl, W);
  if (ok)
    for (int r = slot; r < P; r += NS) out[(size_t)r * Q] = sm[r * B + lane];
}

// ---------------------------------------------------------------- K4: inverse y
template <typename T>
__global__ void __launch_bounds__(256, 2) yi_mixed_kernel(const Cx<T>* __restrict__ A2, Cx<T>* __restrict__ A1,
                                                       const Cx<T>* __restrict__ W, FftPlan pl, int Q) {
  MM_MIXED_PROLOGUE
  const int col = blockIdx.x * B + lane;
  const bool ok = col < Q;
  const Cx<T>* in = A2 + (size_t)blockIdx.y * P * Q + col;
  Cx<T>* out = A1 + (size_t)blockIdx.y * L * Q + col;
  for (int r = slot; r < P; r += NS) sm[r * B + lane] = ok ? in[(size_t)r * Q] : mk<T>(0, 0);
  __syncthreads();
  run_stages_inv<T>(sm, B, lane, slot, NS, P, pl, W);
  if (ok)
    for (int y = slot; y < L; y += NS)
      out[(size_t)y * Q] = cadd(sm[y * B + lane], cmulc(sm[(L + y) * B + lane], __ldg(W + y)));
}

// ---------------------------------------------------------------- K1: forward x, r2c
// m[x][y][q] real is read as complex pairs (q, q + 1): Z = FFT(a + i b) of two real columns,
// separated with A[k] = (Z[k] + conj Z[-k]) / 2, B[k] = (Z[k] - conj Z[-k]) / 2i for k <= nx.
// grid ceil(npairs / B); npairs = ny Q / 2 pairs per x row.
template <typename T>
__global__ void __launch_bounds__(256, 2) xf_mixed_kernel(const Cx<T>* __restrict__ mp, Cx<T>* __restrict__ A1,
                                                       const Cx<T>* __restrict__ W, const uint16_t* __restrict__ pos,
                                                       FftPlan pl, size_t npairs) {
  MM_MIXED_PROLOGUE
  const size_t pair = (size_t)blockIdx.x * B + lane;
  const bool ok = pair < npairs;
  const Cx<T>* in = mp + pair;
  for (int x = slot; x < L; x += NS) {
    const Cx<T> v = ok ? in[(size_t)x * npairs] : mk<T>(0, 0);
    sm[x * B + lane] = v;
    sm[(L + x) * B + lane] = cmul(v, __ldg(W + x));
  }
  __syncthreads();
  run_stages_fwd<T>(sm, B, lane, slot, NS, P, pl, W);
  if (!ok) return;
  Cx<T>* out = A1 + 2 * pair;
  const size_t rowc = 2 * npairs;
  for (int k = slot; k <= L; k += NS) {
    const int p1 = pos[k], p2 = pos[k ? P - k : 0];
    const Cx<T> z1 = sm[p1 * B + lane], z2 = cconj(sm[p2 * B + lane]);
    const Cx<T> s = cadd(z1, z2), d = csub(z1, z2);
    out[(size_t)k * rowc] = mk<T>((T)0.5 * s.x, (T)0.5 * s.y);
    out[(size_t)k * rowc + 1] = mk<T>((T)0.5 * d.y, (T)-0.5 * d.x);
  }
}

// ---------------------------------------------------------------- K5: inverse x, c2r
// Z[k] = A[k] + i B[k], Z[P - k] = conj A[k] + i conj B[k]; the truncated inverse gives
// h_q(x) + i h_{q+1}(x), written as the real pair (q, q + 1) of H, times scale.
template <typename T>
__global__ void __launch_bounds__(256, 2) xi_mixed_kernel(const Cx<T>* __restrict__ A1, Cx<T>* __restrict__ Hp,
                                                       const Cx<T>* __restrict__ W, const uint16_t* __restrict__ pos,
                                                       FftPlan pl, size_t npairs, T scale) {
  MM_MIXED_PROLOGUE
  const size_t pair = (size_t)blockIdx.x * B + lane;
  const bool ok = pair < npairs;
  const Cx<T>* in = A1 + 2 * pair;
  const size_t rowc = 2 * npairs;
  for (int k = slot; k <= L; k += NS) {
    const Cx<T> a = ok ? in[(size_t)k * rowc] : mk<T>(0, 0), b = ok ? in[(size_t)k * rowc + 1] : mk<T>(0, 0);
    sm[pos[k] * B + lane] = mk<T>(a.x - b.y, a.y + b.x);
    if (k != 0 && k != L) sm[pos[P - k] * B + lane] = mk<T>(a.x + b.y, b.x - a.y);
  }
  __syncthreads();
  run_stages_inv<T>(sm, B, lane, slot, NS, P, pl, W);
  if (!ok) return;
  Cx<T>* out = Hp + pair;
  for (int x = slot; x < L; x += NS) {
    const Cx<T> v = cadd(sm[x * B + lane], cmulc(sm[(L + x) * B + lane], __ldg(W + x)));
    out[(size_t)x * npairs] = mk<T>(scale * v.x, scale * v.y);
  }
}

// ---------------------------------------------------------------- K3: fused z pass
// grid (ceil(ny / NPAIR), planes); block = C * NT threads, C = 6 NPAIR columns (3 components of
// the 2 NPAIR pencils); shared memory Pz rows of pitch C + 1.
template <typename T>
__global__ void __launch_bounds__(256, 2) zp_mixed_kernel(Cx<T>* __restrict__ A2, const T* __restrict__ tab,
                                                       const Cx<T>* __restrict__ Wz,
                                                       const uint16_t* __restrict__ posy,
                                                       const uint16_t* __restrict__ fz, FftPlan pl, int ny, int Q,
                                                       int ozp, int NPAIR) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw);
  __shared__ size_t rowoff[32];
  const int nz = pl.L, Pz = pl.P, Py = 2 * ny;
  const int NP = 2 * NPAIR, C = 3 * NP, pitch = C + 1;
  const int plane = blockIdx.y, i0 = blockIdx.x * NPAIR;
  const int tid = threadIdx.x, NTHR = blockDim.x;
  if (tid < NP) {
    const int i = i0 + (tid >> 1);
    const int ky = (tid & 1) ? (i == 0 ? ny : Py - i) : i;
    rowoff[tid] = i < ny ? ((size_t)plane * Py + posy[ky]) * Q : (size_t)0;
  }
  __syncthreads();
  for (int e = tid; e < NP * Q; e += NTHR) {
    const int p = e / Q, q = e - p * Q;
    const bool valid = i0 + (p >> 1) < ny;
    const Cx<T> v = valid ? A2[rowoff[p] + q] : mk<T>(0, 0);
    const int z = q / 3, c = q - 3 * z;
    sm[z * pitch + 3 * p + c] = v;
    sm[(nz + z) * pitch + 3 * p + c] = cmul(v, __ldg(Wz + z));
  }
  __syncthreads();
  run_stages_fwd<T>(sm, pitch, tid % C, tid / C, NTHR / C, Pz, pl, Wz);
  // Hhat = Nhat mhat; row r holds frequency kz = fz[r]; the mirrored halves (kz > nz, ky > ny) reuse
  // the octant entry with the sign of the components that are odd along the mirrored axis
  for (int e = tid; e < Pz * NP; e += NTHR) {
    const int p = e % NP, r = e / NP;
    const int i = i0 + (p >> 1);
    if (i >= ny) continue;
    const int kz = fz[r];
    const bool mir = kz > nz;
    const int idx = mir ? Pz - kz : kz;
    const bool odd = p & 1;
    const T sy = (odd && i != 0) ? (T)-1 : (T)1;
    const T* trow = tab + ((size_t)plane * (ny + 1) + ((odd && i == 0) ? ny : i)) * 6 * ozp;
    const T nxx = __ldg(trow + idx), nyy = __ldg(trow + ozp + idx), nzz = __ldg(trow + 2 * ozp + idx),
            nxy = sy * __ldg(trow + 3 * ozp + idx);
    T nxz = __ldg(trow + 4 * ozp + idx), nyz = sy * __ldg(trow + 5 * ozp + idx);
    if (mir) { nxz = -nxz; nyz = -nyz; }
    Cx<T>* s = sm + r * pitch + 3 * p;
    const Cx<T> a = s[0], b = s[1], c = s[2];
    s[0] = mk<T>(nxx * a.x + nxy * b.x + nxz * c.x, nxx * a.y + nxy * b.y + nxz * c.y);
    s[1] = mk<T>(nxy * a.x + nyy * b.x + nyz * c.x, nxy * a.y + nyy * b.y + nyz * c.y);
    s[2] = mk<T>(nxz * a.x + nyz * b.x + nzz * c.x, nxz * a.y + nyz * b.y + nzz * c.y);
  }
  __syncthreads();
  run_stages_inv<T>(sm, pitch, tid % C, tid / C, NTHR / C, Pz, pl, Wz);
  for (int e = tid; e < NP * Q; e += NTHR) {
    const int p = e / Q, q = e - p * Q;
    if (i0 + (p >> 1) >= ny) continue;
    const int z = q / 3, c = q - 3 * z;
    A2[rowoff[p] + q] =
        cadd(sm[z * pitch + 3 * p + c], cmulc(sm[(nz + z) * pitch + 3 * p + c], __ldg(Wz + z)));
  }
}

// ---------------------------------------------------------------- host side

static const size_t kSmemLimit = 227 * 1024;

static int zp_pairs(int nz, size_t cs, int ny) {
  // mirror pairs per CTA: within ~100 KB of shared memory (two CTAs per SM), at most 5 (32 row offsets)
  int best = 1;
  for (int np = 1; np <= 5 && np <= ny; ++np)
    if ((size_t)(2 * nz) * (6 * np + 1) * cs <= 100 * 1024) best = np;
  return best;
}

bool mixed_supported(int nx, int ny, int nz, size_t real_bytes) {
  if (nx < 2 || ny < 2 || nz < 2) return false;
  if (((size_t)ny * 3 * nz) % 2) return false;              // K1 / K5 move the real arrays as complex pairs
  const size_t cs = 2 * real_bytes;
  if ((size_t)(2 * nx) * 64 > kSmemLimit || (size_t)(2 * ny) * 64 > kSmemLimit) return false;
  return (size_t)(2 * nz) * 7 * cs <= kSmemLimit;           // one mirror pair of z pencils
}

template <typename K> static cudaError_t opt_in(K kernel, size_t bytes) {
  if (bytes <= 48 * 1024) return cudaSuccess;
  return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

// threads of a strided pass: a whole number of slots of B lanes, about one slot per 4 rows
static int strided_threads(int P, int B) {
  int t = P / 4 * B;
  t = (t + 31) / 32 * 32;
  if (t < 64) t = 64;
  if (t > 256) t = 256;
  return t / B * B;
}

template <typename T>
cudaError_t demag_mixed_launch(const FastGeom& g, const MixedPlans& pl, const MixedBufs<T>& b, const T* m, T* H,
                               T scale, cudaStream_t st, unsigned long long* launches, Prof* prof) {
  constexpr int B = MixB<T>::value;
  const size_t cs = sizeof(Cx<T>);
  const size_t npairs = (size_t)g.ny * g.Q / 2;
  const int nplanes = g.nx + 1;
  cudaError_t e;
  const size_t sx = (size_t)g.Px * 64, sy = (size_t)g.Py * 64;
  const unsigned gx = (unsigned)((npairs + B - 1) / B), gq = (unsigned)((g.Q + B - 1) / B);
  prof->mark(0, st);
  if ((e = opt_in(xf_mixed_kernel<T>, sx)) != cudaSuccess) return e;
  xf_mixed_kernel<T><<<gx, strided_threads(g.Px, B), sx, st>>>(reinterpret_cast<const Cx<T>*>(m), b.A1, b.Wx, b.posx,
                                                             pl.px, npairs);
  prof->mark(1, st);
  if ((e = opt_in(yf_mixed_kernel<T>, sy)) != cudaSuccess) return e;
  yf_mixed_kernel<T><<<dim3(gq, nplanes), strided_threads(g.Py, B), sy, st>>>(b.A1, b.A2, b.Wy, pl.py, g.Q);
  prof->mark(2, st);
  {
    const int np = zp_pairs(g.nz, cs, g.ny);
    const int C = 6 * np;
    const size_t sz = (size_t)g.Pz * (C + 1) * cs;
    int nt = 256 / C;
    if (nt < 1) nt = 1;
    if ((e = opt_in(zp_mixed_kernel<T>, sz)) != cudaSuccess) return e;
    const int ozp = (g.nz + 2) / 2 * 2;   // InitGeom::ozp: oz = nz + 1 rounded up to even
    zp_mixed_kernel<T><<<dim3((g.ny + np - 1) / np, nplanes), C * nt, sz, st>>>(b.A2, b.table, b.Wz, b.posy, b.fz,
                                                                               pl.pz, g.ny, g.Q, ozp, np);
  }
  prof->mark(3, st);
  if ((e = opt_in(yi_mixed_kernel<T>, sy)) != cudaSuccess) return e;
  yi_mixed_kernel<T><<<dim3(gq, nplanes), strided_threads(g.Py, B), sy, st>>>(b.A2, b.A1, b.Wy, pl.py, g.Q);
  prof->mark(4, st);
  if ((e = opt_in(xi_mixed_kernel<T>, sx)) != cudaSuccess) return e;
  xi_mixed_kernel<T><<<gx, strided_threads(g.Px, B), sx, st>>>(b.A1, reinterpret_cast<Cx<T>*>(H), b.Wx, b.posx,
                                                             pl.px, npairs, scale);
  prof->mark(-1, st);
  *launches += 5;
  return cudaGetLastError();
}

template cudaError_t demag_mixed_launch<float>(const FastGeom&, const MixedPlans&, const MixedBufs<float>&,
                                               const float*, float*, float, cudaStream_t, unsigned long long*, Prof*);
template cudaError_t demag_mixed_launch<double>(const FastGeom&, const MixedPlans&, const MixedBufs<double>&,
                                                const double*, double*, double, cudaStream_t, unsigned long long*,
                                                Prof*);

}  // namespace mm
