// S1..S5 of the demag hot path: pruned forward z (r2c) and y passes, the fused
// x pass (forward, tensor multiply, inverse; the 2nx-point x spectrum never leaves shared
// memory), truncated inverse y and z (c2r) passes.  PAPER.md:47, :53 describe the sequence
// (pad+FFT y,z -> pad+FFT x -> pointwise multiply with the demag kernel -> inverse x ->
// truncate -> inverse y,z); the all-to-all transposes of the paper's multi-device version
// are not part of this single-GPU path.
//
// Spectral layout in HBM (x fastest, so every pass reads and writes runs contiguous in x):
//   A1[c][kz][y ][x]   c<3, kz<Kz=nz+1, y<ny,   x<nx      after S1 / before S5
//   A2[c][kz][ky'][x]  ky' = position in the digit-reversed length-Py transform
// Pruning: a length-2L transform with only L non-zero inputs is two length-L transforms
// (even outputs: a_j; odd outputs: a_j w_2L^j); the zero half is never read or stored.
// Truncation on the way back is the mirror image.
// scalar fp32 complex add/subtract here: the two-wide form (mm_common.cuh) measured slower in these
// memory-latency-bound passes (K2 0.497 -> 0.528 ms at config 4) and faster only in K3
#define MM_NO_PACKED_F32
#include "demag_passes.cuh"

#include "fft_core.cuh"

namespace mm {

// ---------------------------------------------------------------- S1: forward z, r2c
// Tile: B consecutive x, the line pair (y0, y0+1), all z, 3 components.  The two real lines
// are packed as one complex line (re = y0, im = y0+1) and separated after the transform
// with A[k] = (Z[k] + conj Z[-k])/2, B[k] = (Z[k] - conj Z[-k])/(2i).
template <typename T>
__global__ void __launch_bounds__(512) zf_kernel(DemagGeom g, const T* __restrict__ m,
                                                 Cx<T>* __restrict__ A1,
                                                 const Cx<T>* __restrict__ Wz,
                                                 const uint16_t* __restrict__ posz) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw);
  const int B = g.Bz, tid = threadIdx.x, NTHR = blockDim.x;
  const int x0 = blockIdx.x * B, y0 = blockIdx.y * 2;
  const bool has1 = (y0 + 1) < g.ny;
  const int nz = g.nz, Pz = g.Pz, Kz = g.Kz;
  const int line = nz * 3;
#pragma unroll 4
  for (int e = tid; e < B * line; e += NTHR) {
    const int xl = e / line, rem = e - xl * line;
    const int z = rem / 3, c = rem - z * 3;
    const size_t gi = ((size_t)(x0 + xl) * g.ny + y0) * line + rem;
    const Cx<T> v = mk<T>(m[gi], has1 ? m[gi + line] : (T)0);
    sm[(size_t)(c * Pz + z) * B + xl] = v;
    if (Pz > 1) sm[(size_t)(c * Pz + nz + z) * B + xl] = cmul(v, __ldg(Wz + z));
  }
  __syncthreads();
  run_stages_fwd<T>(sm, B, tid % B, tid / B, NTHR / B, 3 * Pz, g.pz, Wz);
#pragma unroll 4
  for (int e = tid; e < 3 * Kz * B; e += NTHR) {
    const int xl = e % B, kz = (e / B) % Kz, c = e / (B * Kz);
    Cx<T> a, b;
    if (Pz == 1) {
      const Cx<T> z1 = sm[(size_t)(c * Pz) * B + xl];
      a = mk<T>(z1.x, 0);
      b = mk<T>(z1.y, 0);
    } else {
      const int p1 = posz[kz], p2 = posz[kz ? Pz - kz : 0];
      const Cx<T> z1 = sm[(size_t)(c * Pz + p1) * B + xl];
      const Cx<T> z2 = cconj(sm[(size_t)(c * Pz + p2) * B + xl]);
      const Cx<T> s = cadd(z1, z2), d = csub(z1, z2);
      a = mk<T>((T)0.5 * s.x, (T)0.5 * s.y);
      b = mk<T>((T)0.5 * d.y, (T)-0.5 * d.x);
    }
    const size_t o = (((size_t)c * Kz + kz) * g.ny + y0) * g.nx + x0 + xl;
    A1[o] = a;
    if (has1) A1[o + g.nx] = b;
  }
}

// ---------------------------------------------------------------- S2: forward y
template <typename T>
__global__ void __launch_bounds__(512) yf_kernel(DemagGeom g, const Cx<T>* __restrict__ A1,
                                                 Cx<T>* __restrict__ A2,
                                                 const Cx<T>* __restrict__ Wy) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw);
  const int B = g.By, tid = threadIdx.x, NTHR = blockDim.x;
  const int x0 = blockIdx.x * B, kz = blockIdx.y, c = blockIdx.z;
  const int ny = g.ny, Py = g.Py;
  const Cx<T>* in = A1 + ((size_t)c * g.Kz + kz) * ny * g.nx + x0;
  Cx<T>* out = A2 + ((size_t)c * g.Kz + kz) * Py * g.nx + x0;
#pragma unroll 4
  for (int e = tid; e < ny * B; e += NTHR) {
    const int xl = e % B, y = e / B;
    const Cx<T> v = in[(size_t)y * g.nx + xl];
    sm[(size_t)y * B + xl] = v;
    sm[(size_t)(ny + y) * B + xl] = cmul(v, __ldg(Wy + y));
  }
  __syncthreads();
  run_stages_fwd<T>(sm, B, tid % B, tid / B, NTHR / B, Py, g.py, Wy);
#pragma unroll 4
  for (int e = tid; e < Py * B; e += NTHR) {
    const int xl = e % B, r = e / B;
    out[(size_t)r * g.nx + xl] = sm[(size_t)r * B + xl];
  }
}

// ---------------------------------------------------------------- S3: fused x pass
// Tile: Bk consecutive ky' rows of one kz plane, 3 components, all x.  Forward pruned x
// transform, H_r = sum_c Nhat_rc m_c per spectral point (Nhat real symmetric, 6 values),
// inverse truncated x transform, written back in place.
// Table layout: T[kz][ky' block][kx'][6][Bk], already scaled by 1/(Px Py Pz).
template <typename T>
__global__ void __launch_bounds__(512) xp_kernel(DemagGeom g, Cx<T>* __restrict__ A,
                                                 const T* __restrict__ table,
                                                 const Cx<T>* __restrict__ Wx) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw);
  const int B = g.Bk, tid = threadIdx.x, NTHR = blockDim.x;
  const int blk = blockIdx.x, kz = blockIdx.y;
  const int nx = g.nx, Px = g.Px, Py = g.Py, Kz = g.Kz;
  const int ky0 = blk * B;
#pragma unroll(sizeof(T) == 8 ? 8 : 4)
  for (int e = tid; e < 3 * B * nx; e += NTHR) {
    const int x = e % nx, p = (e / nx) % B, c = e / (nx * B);
    const Cx<T> v = A[(((size_t)c * Kz + kz) * Py + ky0 + p) * nx + x];
    sm[(size_t)(c * Px + x) * B + p] = v;
    if (Px > 1) sm[(size_t)(c * Px + nx + x) * B + p] = cmul(v, __ldg(Wx + x));
  }
  __syncthreads();
  run_stages_fwd<T>(sm, B, tid % B, tid / B, NTHR / B, 3 * Px, g.px, Wx);
  const T* tb = table + ((size_t)kz * (Py / B) + blk) * Px * 6 * B;
#pragma unroll(sizeof(T) == 8 ? 8 : 4)
  for (int e = tid; e < Px * B; e += NTHR) {
    const int p = e % B, r = e / B;
    const T* t6 = tb + (size_t)r * 6 * B + p;
    const T nxx = t6[0], nyy = t6[B], nzz = t6[2 * B], nxy = t6[3 * B], nxz = t6[4 * B],
            nyz = t6[5 * B];
    Cx<T>* s0 = sm + (size_t)r * B + p;
    Cx<T>* s1 = s0 + (size_t)Px * B;
    Cx<T>* s2 = s1 + (size_t)Px * B;
    const Cx<T> a = *s0, b = *s1, c = *s2;
    *s0 = mk<T>(nxx * a.x + nxy * b.x + nxz * c.x, nxx * a.y + nxy * b.y + nxz * c.y);
    *s1 = mk<T>(nxy * a.x + nyy * b.x + nyz * c.x, nxy * a.y + nyy * b.y + nyz * c.y);
    *s2 = mk<T>(nxz * a.x + nyz * b.x + nzz * c.x, nxz * a.y + nyz * b.y + nzz * c.y);
  }
  __syncthreads();
  run_stages_inv<T>(sm, B, tid % B, tid / B, NTHR / B, 3 * Px, g.px, Wx);
#pragma unroll(sizeof(T) == 8 ? 8 : 4)
  for (int e = tid; e < 3 * B * nx; e += NTHR) {
    const int x = e % nx, p = (e / nx) % B, c = e / (nx * B);
    Cx<T> v = sm[(size_t)(c * Px + x) * B + p];
    if (Px > 1) v = cadd(v, cmulc(sm[(size_t)(c * Px + nx + x) * B + p], __ldg(Wx + x)));
    A[(((size_t)c * Kz + kz) * Py + ky0 + p) * nx + x] = v;
  }
}

// ---------------------------------------------------------------- S4: inverse y
template <typename T>
__global__ void __launch_bounds__(512) yi_kernel(DemagGeom g, const Cx<T>* __restrict__ A2,
                                                 Cx<T>* __restrict__ A1,
                                                 const Cx<T>* __restrict__ Wy) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw);
  const int B = g.By, tid = threadIdx.x, NTHR = blockDim.x;
  const int x0 = blockIdx.x * B, kz = blockIdx.y, c = blockIdx.z;
  const int ny = g.ny, Py = g.Py;
  const Cx<T>* in = A2 + ((size_t)c * g.Kz + kz) * Py * g.nx + x0;
  Cx<T>* out = A1 + ((size_t)c * g.Kz + kz) * ny * g.nx + x0;
#pragma unroll 4
  for (int e = tid; e < Py * B; e += NTHR) {
    const int xl = e % B, r = e / B;
    sm[(size_t)r * B + xl] = in[(size_t)r * g.nx + xl];
  }
  __syncthreads();
  run_stages_inv<T>(sm, B, tid % B, tid / B, NTHR / B, Py, g.py, Wy);
#pragma unroll 4
  for (int e = tid; e < ny * B; e += NTHR) {
    const int xl = e % B, y = e / B;
    const Cx<T> v =
        cadd(sm[(size_t)y * B + xl], cmulc(sm[(size_t)(ny + y) * B + xl], __ldg(Wy + y)));
    out[(size_t)y * g.nx + xl] = v;
  }
}

// ---------------------------------------------------------------- S5: inverse z, c2r
// Rebuilds the Hermitian length-Pz spectrum of the packed line pair, Z[k] = A[k] + i B[k],
// Z[Pz-k] = conj A[k] + i conj B[k], inverts, keeps z < nz; re -> line y0, im -> line y0+1.
template <typename T>
__global__ void __launch_bounds__(512) zi_kernel(DemagGeom g, const Cx<T>* __restrict__ A1,
                                                 T* __restrict__ H, const Cx<T>* __restrict__ Wz,
                                                 const uint16_t* __restrict__ posz, T scale) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw);
  const int B = g.Bz, tid = threadIdx.x, NTHR = blockDim.x;
  const int x0 = blockIdx.x * B, y0 = blockIdx.y * 2;
  const bool has1 = (y0 + 1) < g.ny;
  const int nz = g.nz, Pz = g.Pz, Kz = g.Kz;
  for (int e = tid; e < 3 * Kz * B; e += NTHR) {
    const int xl = e % B, kz = (e / B) % Kz, c = e / (B * Kz);
    const size_t o = (((size_t)c * Kz + kz) * g.ny + y0) * g.nx + x0 + xl;
    const Cx<T> a = A1[o];
    const Cx<T> b = has1 ? A1[o + g.nx] : mk<T>(0, 0);
    if (Pz == 1) {
      sm[(size_t)(c * Pz) * B + xl] = mk<T>(a.x, b.x);
    } else if (kz == 0 || kz == nz) {
      sm[(size_t)(c * Pz + posz[kz]) * B + xl] = mk<T>(a.x, b.x);
    } else {
      sm[(size_t)(c * Pz + posz[kz]) * B + xl] = mk<T>(a.x - b.y, a.y + b.x);
      sm[(size_t)(c * Pz + posz[Pz - kz]) * B + xl] = mk<T>(a.x + b.y, b.x - a.y);
    }
  }
  __syncthreads();
  run_stages_inv<T>(sm, B, tid % B, tid / B, NTHR / B, 3 * Pz, g.pz, Wz);
  const int line = nz * 3;
  for (int e = tid; e < B * line; e += NTHR) {
    const int xl = e / line, rem = e - xl * line;
    const int z = rem / 3, c = rem - z * 3;
    Cx<T> v = sm[(size_t)(c * Pz + z) * B + xl];
    if (Pz > 1) v = cadd(v, cmulc(sm[(size_t)(c * Pz + nz + z) * B + xl], __ldg(Wz + z)));
    const size_t gi = ((size_t)(x0 + xl) * g.ny + y0) * line + rem;
    H[gi] = scale * v.x;
    if (has1) H[gi + line] = scale * v.y;
  }
}

// ---------------------------------------------------------------- host launchers

template <typename K> static cudaError_t set_smem(K kernel, size_t bytes) {
  if (bytes <= 48 * 1024) return cudaSuccess;
  return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

// Threads per CTA: a whole number of threads per column (the in-place stages give thread
// (col, tt) the butterflies tt, tt + NT, ... of its column).
// The kernels hold up to 128 registers per thread, so 512 threads fill an SM's register file: when
// the tile leaves room for several CTAs per SM the CTA shrinks accordingly (two or three CTAs whose
// load, transform and store phases overlap instead of one that runs them back to back).
static int pick_threads(int B, int rows, size_t smem_bytes) {
  int ctas = (int)((size_t)(227 * 1024) / (smem_bytes + 1024));
  if (ctas < 1) ctas = 1;
  if (ctas > 4) ctas = 4;
  const int cap = 512 / ctas;
  int want = B * (rows / 8 > 0 ? rows / 8 : 1);
  if ((B & (B - 1)) == 0) {
    int t = 64;
    while (t < want && t * 2 <= cap) t *= 2;
    if (t < B) t = B;
    return t;
  }
  int nt = want / B;
  if (nt > cap / B) nt = cap / B;
  return B * (nt > 0 ? nt : 1);
}

template <typename T>
cudaError_t demag_field_launch(const DemagGeom& g, const DemagBufs<T>& b, const T* m, T* H,
                               T scale, cudaStream_t st, unsigned long long* launches, Prof* prof) {
  cudaError_t err;
  const size_t cs = sizeof(Cx<T>);
  Cx<T>* A2 = g.Py > 1 ? b.A2 : b.A1;  // ny == 1: the y pass is the identity
  {
    const size_t sb = (size_t)3 * g.Pz * g.Bz * cs;
    if ((err = set_smem(zf_kernel<T>, sb)) != cudaSuccess) return err;
    dim3 grid(g.nx / g.Bz, (g.ny + 1) / 2);
    prof->mark(0, st);
    zf_kernel<T><<<grid, pick_threads(g.Bz, 3 * g.Pz, sb), sb, st>>>(g, m, b.A1, b.Wz, b.posz);
    ++*launches;
  }
  if (g.Py > 1) {
    const size_t sb = (size_t)g.Py * g.By * cs;
    if ((err = set_smem(yf_kernel<T>, sb)) != cudaSuccess) return err;
    dim3 grid(g.nx / g.By, g.Kz, 3);
    prof->mark(1, st);
    yf_kernel<T><<<grid, pick_threads(g.By, g.Py, sb), sb, st>>>(g, b.A1, b.A2, b.Wy);
    ++*launches;
  }
  {
    const size_t sb = (size_t)3 * g.Px * g.Bk * cs;
    if ((err = set_smem(xp_kernel<T>, sb)) != cudaSuccess) return err;
    dim3 grid(g.Py / g.Bk, g.Kz);
    prof->mark(2, st);
    xp_kernel<T><<<grid, pick_threads(g.Bk, 3 * g.Px, sb), sb, st>>>(g, A2, b.table, b.Wx);
    ++*launches;
  }
  if (g.Py > 1) {
    const size_t sb = (size_t)g.Py * g.By * cs;
    if ((err = set_smem(yi_kernel<T>, sb)) != cudaSuccess) return err;
    dim3 grid(g.nx / g.By, g.Kz, 3);
    prof->mark(3, st);
    yi_kernel<T><<<grid, pick_threads(g.By, g.Py, sb), sb, st>>>(g, b.A2, b.A1, b.Wy);
    ++*launches;
  }
  {
    const size_t sb = (size_t)3 * g.Pz * g.Bz * cs;
    if ((err = set_smem(zi_kernel<T>, sb)) != cudaSuccess) return err;
    dim3 grid(g.nx / g.Bz, (g.ny + 1) / 2);
    prof->mark(4, st);
    zi_kernel<T><<<grid, pick_threads(g.Bz, 3 * g.Pz, sb), sb, st>>>(g, b.A1, H, b.Wz, b.posz, scale);
    ++*launches;
  }
  prof->mark(-1, st);
  return cudaGetLastError();
}

template cudaError_t demag_field_launch<float>(const DemagGeom&, const DemagBufs<float>&,
                                               const float*, float*, float, cudaStream_t,
                                               unsigned long long*, Prof*);
template cudaError_t demag_field_launch<double>(const DemagGeom&, const DemagBufs<double>&,
                                                const double*, double*, double, cudaStream_t,
                                                unsigned long long*, Prof*);

}  // namespace mm
