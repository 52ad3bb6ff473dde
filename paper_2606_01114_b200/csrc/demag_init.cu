// S0: the Fourier-space demag tensor.
//
// PAPER.md:43 names "Newell's formula" (ref. 23) for the kernel N of eq. 4 without
// printing it; SURVEY.md 8(c) O1 restates it.  Plain fp64 evaluation loses all digits at
// large offsets (error ~ 6e-17 R^3 against a value ~ R^-3), so the generating functions are
// evaluated in __float128 on the device (CUDA 12.9 compiles fp128 for sm_100), only for
// offsets i,j,k >= 0.  Instead of mirroring the table onto the padded grid and running an
// FFT, the exact even/odd parity is used: per axis, the DFT of an even (odd) real sequence
// of period P is a cosine (sine) sum over the half range, so Nhat on the octant
// kx<=nx, ky<=ny, kz<=nz is three separable real dense transforms in fp64:
//    even: Nhat(q) = N(0) + 2 sum_{k>=1} N(k) cos(2 pi k q / P)
//    odd : Nhat(q) = -2 i sum_{k>=1} N(k) sin(2 pi k q / P)      (two odd axes -> factor -1)
// The octant is then packed into the layout the x pass consumes (digit-reversed kx', ky'
// positions, sign flips for mirrored odd axes, 1/(Px Py Pz) folded in).
#include <crt/device_fp128_functions.h>

#include "demag_init.cuh"

namespace mm {

typedef __float128 q128;

__device__ __forceinline__ q128 qabs(q128 v) { return v < 0 ? -v : v; }

// Newell's f for non-negative arguments; terms with vanishing prefactor are skipped.
__device__ q128 newell_f_pos(q128 x, q128 y, q128 z) {
  const q128 xx = x * x, yy = y * y, zz = z * z;
  const q128 R = __nv_fp128_sqrt(xx + yy + zz);
  q128 acc = (2 * xx - yy - zz) * R / 6;
  if (y > 0 && xx + zz > 0) acc += (y / 2) * (zz - xx) * __nv_fp128_asinh(y / __nv_fp128_sqrt(xx + zz));
  if (z > 0 && xx + yy > 0) acc += (z / 2) * (yy - xx) * __nv_fp128_asinh(z / __nv_fp128_sqrt(xx + yy));
  if (x > 0 && y > 0 && z > 0) acc -= x * y * z * __nv_fp128_atan(y * z / (x * R));
  return acc;
}

// Newell's g for non-negative arguments (g vanishes when x or y vanishes).
__device__ q128 newell_g_pos(q128 x, q128 y, q128 z) {
  if (!(x > 0) || !(y > 0)) return 0;
  const q128 xx = x * x, yy = y * y, zz = z * z;
  const q128 R = __nv_fp128_sqrt(xx + yy + zz);
  q128 acc = -x * y * R / 3;
  acc += (y / 6) * (3 * zz - yy) * __nv_fp128_asinh(x / __nv_fp128_sqrt(yy + zz));
  acc += (x / 6) * (3 * zz - xx) * __nv_fp128_asinh(y / __nv_fp128_sqrt(xx + zz));
  if (z > 0) {
    acc += x * y * z * __nv_fp128_asinh(z / __nv_fp128_sqrt(xx + yy));
    acc -= (z * zz / 6) * __nv_fp128_atan(x * y / (z * R));
    acc -= (z * yy / 2) * __nv_fp128_atan(x * z / (y * R));
    acc -= (z * xx / 2) * __nv_fp128_atan(y * z / (x * R));
  }
  return acc;
}

// Generating function of tensor component comp (xx yy zz xy xz yz) at lattice point
// (i,j,k) * (dx,dy,dz), i,j,k >= -1.  f is even in all arguments; g is odd in its first two.
__global__ void newell_lattice_kernel(int comp, int nx, int ny, int nz, double dx, double dy,
                                      double dz, q128* __restrict__ F) {
  const size_t sx = nx + 2, sy = ny + 2, sz = nz + 2;
  const size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= sx * sy * sz) return;
  const int k = (int)(g % sz) - 1, j = (int)((g / sz) % sy) - 1, i = (int)(g / (sz * sy)) - 1;
  const q128 X = (q128)dx * (i < 0 ? -i : i), Y = (q128)dy * (j < 0 ? -j : j),
             Z = (q128)dz * (k < 0 ? -k : k);
  const int si = i < 0 ? -1 : 1, sj = j < 0 ? -1 : 1, sk = k < 0 ? -1 : 1;
  q128 v;
  switch (comp) {
    case 0: v = newell_f_pos(X, Y, Z); break;
    case 1: v = newell_f_pos(Y, Z, X); break;
    case 2: v = newell_f_pos(Z, X, Y); break;
    case 3: v = (si * sj) * newell_g_pos(X, Y, Z); break;
    case 4: v = (si * sk) * newell_g_pos(X, Z, Y); break;
    default: v = (sj * sk) * newell_g_pos(Y, Z, X); break;
  }
  F[g] = v;
}

// N(i,j,k) = -1/(4 pi V) * (second difference in x, y and z of F), rounded to fp64 once.
__global__ void newell_diff_kernel(int comp, int nx, int ny, int nz, double dx, double dy,
                                   double dz, const q128* __restrict__ F, double* __restrict__ N) {
  const size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= (size_t)nx * ny * nz) return;
  const int k = (int)(g % nz), j = (int)((g / nz) % ny), i = (int)(g / ((size_t)nz * ny));
  const bool zero = (comp == 3 && (i == 0 || j == 0)) || (comp == 4 && (i == 0 || k == 0)) ||
                    (comp == 5 && (j == 0 || k == 0));
  if (zero) { N[g] = 0.0; return; }
  const size_t sy = ny + 2, sz = nz + 2;
  q128 acc = 0;
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b)
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const int w = (a == 1 ? -2 : 1) * (b == 1 ? -2 : 1) * (c == 1 ? -2 : 1);
        acc += (q128)w * F[((size_t)(i + a) * sy + (j + b)) * sz + (k + c)];
      }
  const q128 pi = 3.14159265358979323846264338327950288Q;
  const q128 V = (q128)dx * (q128)dy * (q128)dz;
  N[g] = (double)(-acc / (4 * pi * V));
}

// cos/sin(2 pi r / P), r < P, in fp64 with exact argument reduction.
__global__ void trig_table_kernel(int P, double* __restrict__ c, double* __restrict__ s) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= P) return;
  double sv, cv;
  sincospi(2.0 * (double)r / (double)P, &sv, &cv);
  c[r] = cv;
  s[r] = sv;
}

// out[o][q][i] = sum_k M(q,k) in[o][k][i], q < nout, k < nin; M from the parity (see header).
__global__ void parity_transform_kernel(const double* __restrict__ in, double* __restrict__ out,
                                        size_t outer, int nin, int nout, size_t inner, int P,
                                        int odd, const double* __restrict__ c,
                                        const double* __restrict__ s) {
  const size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= outer * nout * inner) return;
  const size_t i = g % inner;
  const int q = (int)((g / inner) % nout);
  const size_t o = g / (inner * nout);
  const double* src = in + o * nin * inner + i;
  double acc = 0.0;
  if (P == 1) {
    acc = odd ? 0.0 : src[0];
  } else if (odd) {
    for (int k = 1; k < nin; ++k) acc += src[(size_t)k * inner] * s[(int)(((long long)k * q) % P)];
    acc *= 2.0;
  } else {
    for (int k = 1; k < nin; ++k) acc += src[(size_t)k * inner] * c[(int)(((long long)k * q) % P)];
    acc = src[0] + 2.0 * acc;
  }
  out[g] = acc;
}

// Packs the natural-order octant Nhat[kx<=nx][ky<=ny][kz<=nz] of one component into the
// x-pass table T[kz][ky' block][kx'][6][Bk].
template <typename T>
__global__ void pack_table_kernel(int comp, InitGeom g, const double* __restrict__ oct,
                                  const uint16_t* __restrict__ fx, const uint16_t* __restrict__ fy,
                                  T* __restrict__ table, double scale) {
  const size_t total = (size_t)g.Kz * g.Py * g.Px;
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= total) return;
  const int px = (int)(e % g.Px), py = (int)((e / g.Px) % g.Py), kz = (int)(e / ((size_t)g.Px * g.Py));
  int kx = fx[px], ky = fy[py];
  int flipx = 0, flipy = 0;
  if (kx > g.nx) { kx = g.Px - kx; flipx = 1; }
  if (ky > g.ny) { ky = g.Py - ky; flipy = 1; }
  double v = oct[((size_t)kx * g.oy + ky) * g.oz + kz];
  // parity under a mirror: xy odd in x and y; xz odd in x (and z, never mirrored); yz odd in y
  int flip = 0;
  if (comp == 3) flip = flipx ^ flipy;
  if (comp == 4) flip = flipx;
  if (comp == 5) flip = flipy;
  if (comp >= 3) v = -v;  // (-i)^2 of the two odd axes
  if (flip) v = -v;
  const int blk = py / g.Bk, p = py % g.Bk;
  table[((((size_t)kz * (g.Py / g.Bk) + blk) * g.Px + px) * 6 + comp) * g.Bk + p] = (T)(v * scale);
}

// Inverse of the packing for one component (tests): out[kx][ky][kz], unscaled.
template <typename T>
__global__ void unpack_table_kernel(int comp, InitGeom g, const T* __restrict__ table,
                                    const uint16_t* __restrict__ posx,
                                    const uint16_t* __restrict__ posy, T* __restrict__ out,
                                    double unscale) {
  const size_t total = (size_t)g.ox * g.oy * g.oz;
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= total) return;
  const int kz = (int)(e % g.oz), ky = (int)((e / g.oz) % g.oy), kx = (int)(e / ((size_t)g.oz * g.oy));
  const int px = posx[kx], py = posy[ky];
  const int blk = py / g.Bk, p = py % g.Bk;
  const T v = table[((((size_t)kz * (g.Py / g.Bk) + blk) * g.Px + px) * 6 + comp) * g.Bk + p];
  out[e] = (T)((double)v * unscale);
}

// Fast path (demag_fast.cu): the natural-order octant itself, T[kx][ky][6][ozp] (kz < oz used,
// the pitch ozp keeps every (kx, ky) row a multiple of 16 bytes for bulk copies), with the
// (-i)^2 of the two odd axes and the normalisation folded in; the mirror signs are applied
// by the z pass.
// transpose != 0 (slab layout, demag_fast.cuh SlabView): rows ordered T[ky][kx] instead of T[kx][ky].
template <typename T>
__global__ void pack_fast_kernel(int comp, InitGeom g, const double* __restrict__ oct,
                                 T* __restrict__ table, double scale, int transpose) {
  const size_t total = (size_t)g.ox * g.oy * g.oz;
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= total) return;
  const int kz = (int)(e % g.oz);
  size_t xy = e / g.oz;
  if (transpose) xy = (xy % g.oy) * g.ox + xy / g.oy;
  const double v = comp >= 3 ? -oct[e] : oct[e];
  table[(xy * 6 + comp) * g.ozp + kz] = (T)(v * scale);
  if (kz == g.oz - 1)
    for (int z = g.oz; z < g.ozp; ++z) table[(xy * 6 + comp) * g.ozp + z] = (T)0;  // pitch padding
}
template <typename T>
__global__ void unpack_fast_kernel(int comp, InitGeom g, const T* __restrict__ table,
                                   T* __restrict__ out, double unscale) {
  const size_t total = (size_t)g.ox * g.oy * g.oz;
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= total) return;
  const int kz = (int)(e % g.oz);
  const size_t xy = e / g.oz;
  out[e] = (T)((double)table[(xy * 6 + comp) * g.ozp + kz] * unscale);
}

static unsigned blocks_for(size_t n, int t) { return (unsigned)((n + t - 1) / t); }

template <typename T>
cudaError_t demag_init_launch(const InitGeom& g, double dx, double dy, double dz, void* scratch,
                              const uint16_t* fx, const uint16_t* fy, T* table, int fast,
                              cudaStream_t st, unsigned long long* launches) {
  // scratch carve-up: F lattice (fp128) | octant ping | octant pong | trig tables
  unsigned char* p = static_cast<unsigned char*>(scratch);
  const size_t nF = (size_t)(g.nx + 2) * (g.ny + 2) * (g.nz + 2);
  const size_t nO = (size_t)g.ox * g.oy * g.oz;
  q128* F = reinterpret_cast<q128*>(p);
  p += ((nF * sizeof(q128) + 255) / 256) * 256;
  double* ping = reinterpret_cast<double*>(p);
  p += ((nO * sizeof(double) + 255) / 256) * 256;
  double* pong = reinterpret_cast<double*>(p);
  p += ((nO * sizeof(double) + 255) / 256) * 256;
  double* trig = reinterpret_cast<double*>(p);  // 2 * max(P) doubles per axis, reused
  const double scale = 1.0 / ((double)g.Px * (double)g.Py * (double)g.Pz);
  // parity of component comp along x, y, z (1 = odd)
  static const int odd[6][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}, {1, 1, 0}, {1, 0, 1}, {0, 1, 1}};
  for (int comp = 0; comp < 6; ++comp) {
    newell_lattice_kernel<<<blocks_for(nF, 128), 128, 0, st>>>(comp, g.nx, g.ny, g.nz, dx, dy, dz, F);
    newell_diff_kernel<<<blocks_for((size_t)g.nx * g.ny * g.nz, 128), 128, 0, st>>>(
        comp, g.nx, g.ny, g.nz, dx, dy, dz, F, ping);
    *launches += 2;
    // x: [1][nx][ny*nz] -> [1][ox][ny*nz]
    double* c = trig;
    double* s = trig + 4096;
    trig_table_kernel<<<blocks_for(g.Px, 128), 128, 0, st>>>(g.Px, c, s);
    parity_transform_kernel<<<blocks_for((size_t)g.ox * g.ny * g.nz, 256), 256, 0, st>>>(
        ping, pong, 1, g.nx, g.ox, (size_t)g.ny * g.nz, g.Px, odd[comp][0], c, s);
    // y: [ox][ny][nz] -> [ox][oy][nz]
    trig_table_kernel<<<blocks_for(g.Py, 128), 128, 0, st>>>(g.Py, c, s);
    parity_transform_kernel<<<blocks_for((size_t)g.ox * g.oy * g.nz, 256), 256, 0, st>>>(
        pong, ping, g.ox, g.ny, g.oy, (size_t)g.nz, g.Py, odd[comp][1], c, s);
    // z: [ox*oy][nz][1] -> [ox*oy][oz][1]
    trig_table_kernel<<<blocks_for(g.Pz, 128), 128, 0, st>>>(g.Pz, c, s);
    parity_transform_kernel<<<blocks_for(nO, 256), 256, 0, st>>>(
        ping, pong, (size_t)g.ox * g.oy, g.nz, g.oz, 1, g.Pz, odd[comp][2], c, s);
    if (fast)
      pack_fast_kernel<T><<<blocks_for(nO, 256), 256, 0, st>>>(comp, g, pong, table, scale, fast == 2);
    else
      pack_table_kernel<T><<<blocks_for((size_t)g.Kz * g.Py * g.Px, 256), 256, 0, st>>>(
          comp, g, pong, fx, fy, table, scale);
    *launches += 7;
  }
  return cudaGetLastError();
}

size_t demag_init_scratch_bytes(const InitGeom& g) {
  const size_t nF = (size_t)(g.nx + 2) * (g.ny + 2) * (g.nz + 2);
  const size_t nO = (size_t)g.ox * g.oy * g.oz;
  return ((nF * 16 + 255) / 256) * 256 + 2 * (((nO * 8 + 255) / 256) * 256) + 2 * 4096 * 8;
}

template <typename T>
cudaError_t demag_export_launch(const InitGeom& g, const T* table, const uint16_t* posx,
                                const uint16_t* posy, T* out, int fast, cudaStream_t st,
                                unsigned long long* launches) {
  const size_t nO = (size_t)g.ox * g.oy * g.oz;
  const double unscale = (double)g.Px * (double)g.Py * (double)g.Pz;
  for (int comp = 0; comp < 6; ++comp) {
    if (fast)
      unpack_fast_kernel<T><<<blocks_for(nO, 256), 256, 0, st>>>(comp, g, table, out + comp * nO,
                                                                 unscale);
    else
      unpack_table_kernel<T><<<blocks_for(nO, 256), 256, 0, st>>>(comp, g, table, posx, posy,
                                                                   out + comp * nO, unscale);
    ++*launches;
  }
  return cudaGetLastError();
}

template cudaError_t demag_init_launch<float>(const InitGeom&, double, double, double, void*,
                                              const uint16_t*, const uint16_t*, float*, int,
                                              cudaStream_t, unsigned long long*);
template cudaError_t demag_init_launch<double>(const InitGeom&, double, double, double, void*,
                                               const uint16_t*, const uint16_t*, double*, int,
                                               cudaStream_t, unsigned long long*);
template cudaError_t demag_export_launch<float>(const InitGeom&, const float*, const uint16_t*,
                                                const uint16_t*, float*, int, cudaStream_t,
                                                unsigned long long*);
template cudaError_t demag_export_launch<double>(const InitGeom&, const double*, const uint16_t*,
                                                 const uint16_t*, double*, int, cudaStream_t,
                                                 unsigned long long*);

}  // namespace mm
