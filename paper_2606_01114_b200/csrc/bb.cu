// Barzilai-Borwein minimiser iteration; see bb.cuh.
#include "bb.cuh"

namespace mm {

static unsigned bb_grid(size_t n) {
  size_t b = (n + 255) / 256;
  return (unsigned)(b < 1 ? 1 : (b > (size_t)kBbMaxBlocks ? (size_t)kBbMaxBlocks : b));
}

// fixed-order tree: the result depends on the grid only, not on scheduling
__device__ __forceinline__ void block_sum3(double& a, double& b, double& c, double* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    a += __shfl_xor_sync(0xffffffffu, a, o);
    b += __shfl_xor_sync(0xffffffffu, b, o);
    c += __shfl_xor_sync(0xffffffffu, c, o);
  }
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0) { red[3 * w] = a; red[3 * w + 1] = b; red[3 * w + 2] = c; }
  __syncthreads();
  if (threadIdx.x == 0) {
    a = b = c = 0.0;
    for (int i = 0; i < (int)(blockDim.x >> 5); ++i) { a += red[3 * i]; b += red[3 * i + 1]; c += red[3 * i + 2]; }
  }
}

// partial[block] = (s.s, s.y, y.y) over the block's elements, s = m - m_prev, y = g - g_prev
template <typename T>
__global__ void __launch_bounds__(256) bb_sums_kernel(const BbState* __restrict__ s, const T* __restrict__ m,
                                                      const T* __restrict__ g, const T* __restrict__ mp,
                                                      const T* __restrict__ gp, size_t n3,
                                                      double* __restrict__ partial) {
  __shared__ double red[24];
  if (s->converged || s->n == 0) return;
  double ss = 0.0, sy = 0.0, yy = 0.0;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n3; q += stride) {
    const double sv = (double)m[q] - (double)mp[q], yv = (double)g[q] - (double)gp[q];
    ss += sv * sv; sy += sv * yv; yy += yv * yv;
  }
  block_sum3(ss, sy, yy, red);
  if (threadIdx.x == 0) {
    partial[3 * blockIdx.x] = ss; partial[3 * blockIdx.x + 1] = sy; partial[3 * blockIdx.x + 2] = yy;
  }
}

// one CTA: total of the partials, then the step length (reading Q30)
__global__ void __launch_bounds__(256) bb_tau_kernel(BbState* __restrict__ s, const double* __restrict__ partial,
                                                     int nblocks) {
  __shared__ double red[24];
  if (s->converged) return;
  double tau = s->tau0;
  if (s->n > 0) {
    double ss = 0.0, sy = 0.0, yy = 0.0;
    for (int i = threadIdx.x; i < nblocks; i += blockDim.x) {
      ss += partial[3 * i]; sy += partial[3 * i + 1]; yy += partial[3 * i + 2];
    }
    block_sum3(ss, sy, yy, red);
    if (threadIdx.x != 0) return;
    s->ss = ss; s->sy = sy; s->yy = yy;
    const double q = (s->n & 1ull) ? ss / sy : sy / yy;
    tau = (sy > 0.0 && isfinite(q)) ? q : s->tau0;
  } else if (threadIdx.x != 0) {
    return;
  }
  tau = fmin(s->tau_max, fmax(s->tau_min, tau));
  s->tau = tau;
}

template <typename T> __device__ __forceinline__ unsigned long long bb_bits(T v);
template <> __device__ __forceinline__ unsigned long long bb_bits<float>(float v) { return __float_as_uint(v); }
template <> __device__ __forceinline__ unsigned long long bb_bits<double>(double v) {
  return (unsigned long long)__double_as_longlong(v);
}

// m <- [(1 - tau^2 g^2 / 4) m - tau g] / (1 + tau^2 g^2 / 4); keeps the old iterate and gradient
template <typename T>
__global__ void __launch_bounds__(256) bb_update_kernel(BbState* __restrict__ s, T* __restrict__ m,
                                                        const T* __restrict__ g, T* __restrict__ mp,
                                                        T* __restrict__ gp, size_t ncell) {
  if (s->converged) return;
  const T tau = (T)s->tau;
  T dmax = 0;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < ncell; i += stride) {
    const T m0 = m[3 * i], m1 = m[3 * i + 1], m2 = m[3 * i + 2];
    const T g0 = g[3 * i], g1 = g[3 * i + 1], g2 = g[3 * i + 2];
    const T a = (T)0.25 * tau * tau * (g0 * g0 + g1 * g1 + g2 * g2);
    const T inv = (T)1 / ((T)1 + a);
    const T n0 = (((T)1 - a) * m0 - tau * g0) * inv;
    const T n1 = (((T)1 - a) * m1 - tau * g1) * inv;
    const T n2 = (((T)1 - a) * m2 - tau * g2) * inv;
    // a non-finite change (blown-up state) counts as +inf: never reported as converged
    const T d0 = fabs(n0 - m0), d1 = fabs(n1 - m1), d2 = fabs(n2 - m2);
    const T dd = (d0 == d0 && d1 == d1 && d2 == d2) ? fmax(d0, fmax(d1, d2)) : (T)INFINITY;
    dmax = fmax(dmax, dd);
    mp[3 * i] = m0; mp[3 * i + 1] = m1; mp[3 * i + 2] = m2;
    gp[3 * i] = g0; gp[3 * i + 1] = g1; gp[3 * i + 2] = g2;
    m[3 * i] = n0; m[3 * i + 1] = n1; m[3 * i + 2] = n2;
  }
  // the maximum is order-independent: the atomic keeps the result deterministic
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) dmax = fmax(dmax, __shfl_xor_sync(0xffffffffu, dmax, o));
  if ((threadIdx.x & 31) == 0 && dmax > 0) atomicMax(&s->dmbits, bb_bits<T>(dmax));
}

template <typename T> __global__ void bb_finish_kernel(BbState* s) {
  if (s->converged) return;
  double dm;
  if (sizeof(T) == 4) dm = (double)__uint_as_float((unsigned)s->dmbits);
  else dm = __longlong_as_double((long long)s->dmbits);
  s->dm_max = dm;
  s->converged = dm <= s->tol ? 1 : 0;
  s->n += 1;
  s->dmbits = 0;
}

template <typename T>
cudaError_t bb_iterate_launch(BbState* sd, T* m, const T* g, T* mp, T* gp, double* partial, size_t n3,
                              cudaStream_t st, unsigned long long* launches) {
  const unsigned nb = bb_grid(n3);
  bb_sums_kernel<T><<<nb, 256, 0, st>>>(sd, m, g, mp, gp, n3, partial);
  bb_tau_kernel<<<1, 256, 0, st>>>(sd, partial, (int)nb);
  bb_update_kernel<T><<<bb_grid(n3 / 3), 256, 0, st>>>(sd, m, g, mp, gp, n3 / 3);
  bb_finish_kernel<T><<<1, 1, 0, st>>>(sd);
  *launches += 4;
  return cudaGetLastError();
}

template cudaError_t bb_iterate_launch<float>(BbState*, float*, const float*, float*, float*, double*, size_t,
                                              cudaStream_t, unsigned long long*);
template cudaError_t bb_iterate_launch<double>(BbState*, double*, const double*, double*, double*, double*, size_t,
                                               cudaStream_t, unsigned long long*);

}  // namespace mm
