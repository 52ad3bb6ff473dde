// Shared device helpers of the CUDA path: complex arithmetic on float2/double2, plan
// descriptors.  (No code is shared with oracle/.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mm {

template <typename T> struct cx_of;
template <> struct cx_of<float> { using type = float2; };
template <> struct cx_of<double> { using type = double2; };
template <typename T> using Cx = typename cx_of<T>::type;

template <typename T> __host__ __device__ __forceinline__ Cx<T> mk(T a, T b) {
  Cx<T> r; r.x = a; r.y = b; return r;
}
template <typename C> __device__ __forceinline__ C cadd(C a, C b) { a.x += b.x; a.y += b.y; return a; }
template <typename C> __device__ __forceinline__ C csub(C a, C b) { a.x -= b.x; a.y -= b.y; return a; }
#if defined(__CUDA_ARCH__) && !defined(MM_NO_PACKED_F32)
// fp32 complex add / subtract as ONE two-wide instruction (sm_100 FADD2 on the register pair
// holding (re, im)): same lanes, same rounding, half the issue slots.  The FFT kernels are bound
// by instruction issue, not by the FP32 pipe (profiles/r01_v2_fast_path.md).
__device__ __forceinline__ unsigned long long f2_pack(float2 a) {
  unsigned long long r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a.x), "f"(a.y));
  return r;
}
__device__ __forceinline__ float2 f2_unpack(unsigned long long a) {
  float2 r;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(a));
  return r;
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) {
  unsigned long long r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_pack(a)), "l"(f2_pack(b)));
  return f2_unpack(r);
}
__device__ __forceinline__ float2 csub(float2 a, float2 b) {
  unsigned long long r;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_pack(a)), "l"(f2_pack(b)));
  return f2_unpack(r);
}
#endif
// Complex products with the rounding pinned (one rounded product, one fused multiply-add per component): which
// product the compiler fuses otherwise depends on the surrounding code, and the LDG / STG and the box kernels
// must agree bit for bit (tests/test_gpu_fast.py).
__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }
// a * b
template <typename C> __device__ __forceinline__ C cmul(C a, C b) {
  C r; r.x = fma(a.x, b.x, -mul_rn(a.y, b.y)); r.y = fma(a.x, b.y, mul_rn(a.y, b.x)); return r;
}
// a * conj(b)
template <typename C> __device__ __forceinline__ C cmulc(C a, C b) {
  C r; r.x = fma(a.x, b.x, mul_rn(a.y, b.y)); r.y = fma(a.y, b.x, -mul_rn(a.x, b.y)); return r;
}
template <typename C> __device__ __forceinline__ C cconj(C a) { a.y = -a.y; return a; }

constexpr int MM_MAX_STAGES = 8;

// Radix plan of one in-place transform of length L = prod radix[i], radix[i] in {2, 3, 4, 5, 6, 7, 8, 10, 14, 16}.
struct FftPlan {
  int L;        // sub-transform length (n_d); the padded length is P = 2L (or 1)
  int P;
  int nstages;
  int radix[MM_MAX_STAGES];
};


// Optional per-kernel timing with CUDA events on the launching stream (bench.py's roofline
// leg).  mark(id) is called immediately before kernel `id` is enqueued, mark(-1) after the
// last kernel of a call; the time between two consecutive marks belongs to the first.
struct Prof {
  static constexpr int kKinds = 8;
  static constexpr int kMaxMarks = 8192;
  bool on = false;
  cudaEvent_t* ev = nullptr;
  int* kind = nullptr;
  int n = 0, cap = 0;
  void mark(int id, cudaStream_t st) {
    if (!on || n >= kMaxMarks) return;
    if (n == cap) {
      const int ncap = cap ? cap * 2 : 64;
      cudaEvent_t* e2 = new cudaEvent_t[ncap];
      int* k2 = new int[ncap];
      for (int i = 0; i < cap; ++i) { e2[i] = ev[i]; k2[i] = kind[i]; }
      for (int i = cap; i < ncap; ++i) cudaEventCreate(&e2[i]);
      delete[] ev; delete[] kind;
      ev = e2; kind = k2; cap = ncap;
    }
    kind[n] = id;
    cudaEventRecord(ev[n], st);
    ++n;
  }
  ~Prof() {
    for (int i = 0; i < cap; ++i) cudaEventDestroy(ev[i]);
    delete[] ev; delete[] kind;
  }
};

}  // namespace mm
