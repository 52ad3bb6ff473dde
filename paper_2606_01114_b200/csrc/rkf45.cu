// RKF45 stage combinations, error maximum, device-side step controller and commit
// (rkf45.cuh).  All four kernels are plain streaming passes: HBM-bound,
// 3 s B/real read per K_j used plus 3 s written, small next to the six H_eff evaluations.
#include "rkf45.cuh"

namespace mm {

// Fehlberg 1969, RK4(5): a_ij, and the two weight rows.
static const double kA[5][5] = {
    {1.0 / 4.0, 0, 0, 0, 0},
    {3.0 / 32.0, 9.0 / 32.0, 0, 0, 0},
    {1932.0 / 2197.0, -7200.0 / 2197.0, 7296.0 / 2197.0, 0, 0},
    {439.0 / 216.0, -8.0, 3680.0 / 513.0, -845.0 / 4104.0, 0},
    {-8.0 / 27.0, 2.0, -3544.0 / 2565.0, 1859.0 / 4104.0, -11.0 / 40.0}};
static const double kB4[6] = {25.0 / 216.0, 0, 1408.0 / 2565.0, 2197.0 / 4104.0, -1.0 / 5.0, 0};
static const double kB5[6] = {16.0 / 135.0, 0, 6656.0 / 12825.0, 28561.0 / 56430.0, -9.0 / 50.0, 2.0 / 55.0};

const double* rkf_row(int i) { return kA[i - 1]; }

template <typename T> struct Coef { T c[6]; };

template <typename T, int NK>
__global__ void __launch_bounds__(256) rkf_combine_kernel(const RkfState* __restrict__ s, const T* __restrict__ m0,
                                                          const T* __restrict__ K, size_t n3, Coef<T> a,
                                                          T* __restrict__ out) {
  const T dt = (T)s->dt;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n3; q += stride) {
    T acc = 0;
#pragma unroll
    for (int j = 0; j < NK; ++j) acc += a.c[j] * K[(size_t)j * n3 + q];
    out[q] = m0[q] + dt * acc;
  }
}

template <typename T> __device__ __forceinline__ unsigned long long real_bits(T v);
template <> __device__ __forceinline__ unsigned long long real_bits<float>(float v) { return __float_as_uint(v); }
template <> __device__ __forceinline__ unsigned long long real_bits<double>(double v) {
  return (unsigned long long)__double_as_longlong(v);
}

template <typename T>
__global__ void __launch_bounds__(256) rkf_final_kernel(RkfState* __restrict__ s, const T* __restrict__ m0,
                                                        const T* __restrict__ K, size_t n3, Coef<T> b5,
                                                        Coef<T> d, T* __restrict__ cand) {
  const T dt = (T)s->dt;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  T emax = 0;
  for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n3; q += stride) {
    T s5 = 0, e = 0;
#pragma unroll
    for (int j = 0; j < 6; ++j) {
      const T k = K[(size_t)j * n3 + q];
      s5 += b5.c[j] * k;
      e += d.c[j] * k;
    }
    cand[q] = m0[q] + dt * s5;
    // a non-finite estimate (blown-up state) must not vanish in fmax: it counts as +inf, which the
    // controller rejects (err <= tol fails) and mm_rkf45_state reports
    const T ae = fabs(dt * e);
    emax = fmax(emax, ae == ae ? ae : (T)INFINITY);
  }
  // maximum is order-independent: the atomic keeps the result deterministic
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) emax = fmax(emax, __shfl_xor_sync(0xffffffffu, emax, o));
  if ((threadIdx.x & 31) == 0 && emax > 0) atomicMax(&s->errbits, real_bits<T>(emax));
}

template <typename T> __global__ void rkf_control_kernel(RkfState* s) {
  double err;
  if (sizeof(T) == 4) err = (double)__uint_as_float((unsigned)s->errbits);
  else err = __longlong_as_double((long long)s->errbits);
  const double dt = s->dt;
  const int accept = err <= s->tol ? 1 : 0;
  double fac = err > 0.0 ? 0.9 * pow(s->tol / err, 0.2) : 5.0;
  fac = fmin(5.0, fmax(0.2, fac));
  const double dn = fmin(s->dt_max, fmax(s->dt_min, dt * fac));
  s->err = err;
  s->dt_last = dt;
  s->accept = accept;
  if (accept) { s->t += dt; s->n_acc += 1; } else { s->n_rej += 1; }
  s->dt = dn;
  s->errbits = 0;
}

template <typename T>
__global__ void __launch_bounds__(256) rkf_commit_kernel(const RkfState* __restrict__ s, T* __restrict__ m,
                                                         const T* __restrict__ cand, size_t ncell) {
  if (!s->accept) return;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < ncell; i += stride) {
    const T x = cand[3 * i], y = cand[3 * i + 1], z = cand[3 * i + 2];
    const T nrm = sqrt(x * x + y * y + z * z);
    if (nrm > (T)0) { m[3 * i] = x / nrm; m[3 * i + 1] = y / nrm; m[3 * i + 2] = z / nrm; }   // a vacuum cell stays zero
  }
}

static unsigned grid_for(size_t n) {
  size_t b = (n + 255) / 256;
  const size_t cap = 148 * 16;
  return (unsigned)(b < 1 ? 1 : (b > cap ? cap : b));
}

template <typename T>
cudaError_t rkf_combine_launch(const RkfState* sd, const T* m0, const T* K, size_t n3, int nk, const double* a,
                               T* out, cudaStream_t st) {
  Coef<T> c{};
  for (int j = 0; j < nk; ++j) c.c[j] = (T)a[j];
  const unsigned g = grid_for(n3);
  switch (nk) {
    case 1: rkf_combine_kernel<T, 1><<<g, 256, 0, st>>>(sd, m0, K, n3, c, out); break;
    case 2: rkf_combine_kernel<T, 2><<<g, 256, 0, st>>>(sd, m0, K, n3, c, out); break;
    case 3: rkf_combine_kernel<T, 3><<<g, 256, 0, st>>>(sd, m0, K, n3, c, out); break;
    case 4: rkf_combine_kernel<T, 4><<<g, 256, 0, st>>>(sd, m0, K, n3, c, out); break;
    case 5: rkf_combine_kernel<T, 5><<<g, 256, 0, st>>>(sd, m0, K, n3, c, out); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

template <typename T>
cudaError_t rkf_finish_launch(RkfState* sd, T* m0, const T* K, size_t n3, T* cand, cudaStream_t st,
                              unsigned long long* launches) {
  Coef<T> b5{}, d{};
  for (int j = 0; j < 6; ++j) { b5.c[j] = (T)kB5[j]; d.c[j] = (T)(kB5[j] - kB4[j]); }
  rkf_final_kernel<T><<<grid_for(n3), 256, 0, st>>>(sd, m0, K, n3, b5, d, cand);
  rkf_control_kernel<T><<<1, 1, 0, st>>>(sd);
  rkf_commit_kernel<T><<<grid_for(n3 / 3), 256, 0, st>>>(sd, m0, cand, n3 / 3);
  *launches += 3;
  return cudaGetLastError();
}

template cudaError_t rkf_combine_launch<float>(const RkfState*, const float*, const float*, size_t, int,
                                               const double*, float*, cudaStream_t);
template cudaError_t rkf_combine_launch<double>(const RkfState*, const double*, const double*, size_t, int,
                                                const double*, double*, cudaStream_t);
template cudaError_t rkf_finish_launch<float>(RkfState*, float*, const float*, size_t, float*, cudaStream_t,
                                              unsigned long long*);
template cudaError_t rkf_finish_launch<double>(RkfState*, double*, const double*, size_t, double*, cudaStream_t,
                                               unsigned long long*);

}  // namespace mm
