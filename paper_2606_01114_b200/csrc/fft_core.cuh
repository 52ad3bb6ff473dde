// In-register radix-R DFT butterflies and in-place shared-memory FFT stages.
//
// Scheme: a tile holds N rows x B columns of complex
// values, column = one independent pencil ("lanes along batch": consecutive threads own
// consecutive columns, so every shared-memory access of a warp is a contiguous run and
// twiddles are warp-uniform).  Forward = decimation in frequency, in place, natural order
// in -> digit-reversed order out; inverse = the exact mirror image (decimation in time,
// digit-reversed in -> natural out).  The pointwise multiply with the demag tensor happens
// in digit-reversed order, so no reordering pass is ever executed (FFT,
// pointwise multiplication, inverse FFT).
#pragma once
#include <utility>

#include "mm_common.cuh"

namespace mm {

// cos(2 pi k / 32), k = 0..8
constexpr double kCos32[9] = {1.0,
                                         0.98078528040323044913,
                                         0.92387953251128675613,
                                         0.83146961230254523708,
                                         0.70710678118654752440,
                                         0.55557023301960222474,
                                         0.38268343236508977173,
                                         0.19509032201612826785,
                                         0.0};

// cos / sin of 2 pi num / den at compile time for any den (the radices of the mixed-radix plans: 28, 25,
// 20, 18, ...).  The angle is reduced to the first octant in exact integer arithmetic, then a Taylor
// series in double (|x| <= pi / 4: 13 terms leave < 1e-17); the result is within a few 1e-16 of the
// correctly rounded value, far inside the 1e-12 parity bar.
constexpr double kPi = 3.14159265358979323846264338327950288;
constexpr double small_sin(double x) {
  double term = x, sum = x;
  for (int i = 1; i <= 13; ++i) { term *= -x * x / ((2.0 * i) * (2.0 * i + 1.0)); sum += term; }
  return sum;
}
constexpr double small_cos(double x) {
  double term = 1.0, sum = 1.0;
  for (int i = 1; i <= 13; ++i) { term *= -x * x / ((2.0 * i - 1.0) * (2.0 * i)); sum += term; }
  return sum;
}
constexpr double sin_turn(long long num, long long den);
constexpr double cos_turn(long long num, long long den) {   // cos(2 pi num / den), 0 <= num < den
  if (2 * num > den) return cos_turn(den - num, den);
  if (4 * num > den) return -cos_turn(den - 2 * num, 2 * den);
  if (8 * num > den) return sin_turn(den - 4 * num, 4 * den);
  return small_cos(2.0 * kPi * (double)num / (double)den);
}
constexpr double sin_turn(long long num, long long den) {   // sin(2 pi num / den), 0 <= num < den
  if (2 * num > den) return -sin_turn(den - num, den);
  if (4 * num > den) return sin_turn(den - 2 * num, 2 * den);
  if (8 * num > den) return cos_turn(den - 4 * num, 4 * den);
  return small_sin(2.0 * kPi * (double)num / (double)den);
}

constexpr bool near_enough(double a, double b) { return a - b < 4e-16 && b - a < 4e-16; }
static_assert(near_enough(cos_turn(1, 5), 0.30901699437494742410) && near_enough(sin_turn(1, 7), 0.78183148246802980871) &&
                  near_enough(cos_turn(3, 8), -0.70710678118654752440) && near_enough(sin_turn(11, 25), 0.36812455268467795916) &&
                  near_enough(cos_turn(13, 28), -0.97492791218182360702) && near_enough(sin_turn(27, 28), -0.22252093395631440429),
              "compile-time trigonometry");

template <int R, int S> constexpr double root_cos() {
  if constexpr (32 % R != 0) {
    return cos_turn(S % R, R);
  } else {
    constexpr int a = (S % R) * (32 / R);  // angle in 1/32 turns, 0..31
    if (a <= 8) return kCos32[a];
    if (a <= 16) return -kCos32[16 - a];
    if (a <= 24) return -kCos32[a - 16];
    return kCos32[32 - a];
  }
}
template <int R, int S> constexpr double root_sin() {
  if constexpr (32 % R != 0) {
    return sin_turn(S % R, R);
  } else {
    constexpr int a = (S % R) * (32 / R);
    if (a <= 8) return kCos32[8 - a];
    if (a <= 16) return kCos32[a - 8];
    if (a <= 24) return -kCos32[24 - a];
    return -kCos32[a - 24];
  }
}

// v * w_R^S with w_R = exp(-2 pi i / R) (forward) or its conjugate (INV).
template <typename T, int R, int S, bool INV> __device__ __forceinline__ Cx<T> mul_root(Cx<T> v) {
  constexpr int s = S % R;
  if constexpr (s == 0) {
    return v;
  } else if constexpr (4 * s == R) {  // -i (forward)
    return INV ? mk<T>(-v.y, v.x) : mk<T>(v.y, -v.x);
  } else if constexpr (2 * s == R) {
    return mk<T>(-v.x, -v.y);
  } else if constexpr (4 * s == 3 * R) {  // +i (forward)
    return INV ? mk<T>(v.y, -v.x) : mk<T>(-v.y, v.x);
  } else if constexpr (8 * s == R) {  // (1 - i)/sqrt2 (forward); one multiply + two fused multiply-adds
    constexpr T h = (T)0.70710678118654752440;
    if constexpr (INV) { const T t = v.x * h; return mk<T>(fma(-v.y, h, t), fma(v.y, h, t)); }
    else { const T t = v.y * h; return mk<T>(fma(v.x, h, t), fma(-v.x, h, t)); }
  } else if constexpr (8 * s == 3 * R) {  // (-1 - i)/sqrt2 (forward)
    constexpr T h = (T)0.70710678118654752440;
    if constexpr (INV) { const T t = v.x * h; return mk<T>(fma(-v.y, h, -t), fma(-v.y, h, t)); }
    else { const T t = v.y * h; return mk<T>(fma(-v.x, h, t), fma(-v.x, h, -t)); }
  } else {
    constexpr T c = (T)root_cos<R, s>();
    constexpr T sn = (T)root_sin<R, s>();
    // forward: (c - i sn); inverse: (c + i sn)
    return INV ? mk<T>(v.x * c - v.y * sn, v.y * c + v.x * sn)
               : mk<T>(v.x * c + v.y * sn, v.y * c - v.x * sn);
  }
}

// e + o * w_R^S with the products contracted into the sums (two fused multiply-adds per real).
template <typename T, int R, int S, bool INV> __device__ __forceinline__ Cx<T> add_root(Cx<T> e, Cx<T> o) {
  constexpr int s = S % R;
  if constexpr (s == 0) {
    return cadd(e, o);
  } else if constexpr (4 * s == R) {  // -i (forward)
    return INV ? mk<T>(e.x - o.y, e.y + o.x) : mk<T>(e.x + o.y, e.y - o.x);
  } else if constexpr (2 * s == R) {
    return csub(e, o);
  } else if constexpr (4 * s == 3 * R) {  // +i (forward)
    return INV ? mk<T>(e.x + o.y, e.y - o.x) : mk<T>(e.x - o.y, e.y + o.x);
  } else {
    constexpr T c = (T)root_cos<R, s>();
    constexpr T sn = (T)root_sin<R, s>();
    return INV ? mk<T>(fma(o.x, c, fma(-o.y, sn, e.x)), fma(o.y, c, fma(o.x, sn, e.y)))
               : mk<T>(fma(o.x, c, fma(o.y, sn, e.x)), fma(o.y, c, fma(-o.x, sn, e.y)));
  }
}

// (a - b) * w_R^S.  The quarter-turn roots swap the two halves of the complex value: the
// difference is then taken half by half into the swapped positions, so the packed two-wide
// arithmetic of cadd/csub downstream never needs a register shuffle.
template <typename T, int R, int S, bool INV> __device__ __forceinline__ Cx<T> sub_root(Cx<T> a, Cx<T> b) {
  constexpr int s = S % R;
  if constexpr (4 * s == R) {  // -i (forward): (d.y, -d.x)
    return INV ? mk<T>(b.y - a.y, a.x - b.x) : mk<T>(a.y - b.y, b.x - a.x);
  } else if constexpr (4 * s == 3 * R) {  // +i (forward): (-d.y, d.x)
    return INV ? mk<T>(a.y - b.y, b.x - a.x) : mk<T>(b.y - a.y, a.x - b.x);
  } else {
    return mul_root<T, R, S, INV>(csub(a, b));
  }
}

// Radix-R DFT of v[0..R) in registers, natural order in and out, unnormalised.
// Decimation in frequency: sums -> even outputs, twiddled differences -> odd outputs.
template <typename T, int R, bool INV> struct Dft {
  template <int... I>
  static __device__ __forceinline__ void split(const Cx<T>* v, Cx<T>* a, Cx<T>* b,
                                               std::integer_sequence<int, I...>) {
    ((a[I] = cadd(v[I], v[I + R / 2])), ...);
    ((b[I] = sub_root<T, R, I, INV>(v[I], v[I + R / 2])), ...);
  }
  static __device__ __forceinline__ void run(Cx<T>* v) {
    Cx<T> a[R / 2], b[R / 2];
    split(v, a, b, std::make_integer_sequence<int, R / 2>{});
    Dft<T, R / 2, INV>::run(a);
    Dft<T, R / 2, INV>::run(b);
#pragma unroll
    for (int k = 0; k < R / 2; ++k) {
      v[2 * k] = a[k];
      v[2 * k + 1] = b[k];
    }
  }
};
template <typename T, bool INV> struct Dft<T, 1, INV> {
  static __device__ __forceinline__ void run(Cx<T>*) {}
};

// Odd prime radices 3, 5, 7 (meshes that are not powers of two: the paper's own workloads are
// 100 x 25 x 1, N = 100, 350, 400 and 512 x 512 x 90 cells).  With
// a_k = v_k + v_{R-k}, b_k = v_k - v_{R-k}:
//   X_j, X_{R-j} = v_0 + sum_k cos(2 pi j k / R) a_k  -/+  i sum_k sin(2 pi j k / R) b_k   (forward).
template <int R> constexpr double odd_cos(int m) {  // cos(2 pi m / R), m < R
  const int h = m <= R / 2 ? m : R - m;
  if (h == 0) return 1.0;
  if (R == 3) return -0.5;
  if (R == 5) return h == 1 ? 0.30901699437494742410 : -0.80901699437494742410;
  return h == 1 ? 0.62348980185873353053 : (h == 2 ? -0.22252093395631440429 : -0.90096886790241912624);
}
template <int R> constexpr double odd_sin(int m) {  // sin(2 pi m / R), m < R
  const int h = m <= R / 2 ? m : R - m;
  const double sg = m <= R / 2 ? 1.0 : -1.0;
  if (h == 0) return 0.0;
  if (R == 3) return sg * 0.86602540378443864676;
  if (R == 5) return sg * (h == 1 ? 0.95105651629515357212 : 0.58778525229247312917);
  return sg * (h == 1 ? 0.78183148246802980871 : (h == 2 ? 0.97492791218182360702 : 0.43388373911755812048));
}
template <typename T, int R, bool INV> struct DftOdd {
  static __device__ __forceinline__ void run(Cx<T>* v) {
    constexpr int H = R / 2;
    Cx<T> a[H], b[H], out[R];
#pragma unroll
    for (int k = 1; k <= H; ++k) {
      a[k - 1] = mk<T>(v[k].x + v[R - k].x, v[k].y + v[R - k].y);
      b[k - 1] = mk<T>(v[k].x - v[R - k].x, v[k].y - v[R - k].y);
    }
    out[0] = v[0];
#pragma unroll
    for (int k = 0; k < H; ++k) { out[0].x += a[k].x; out[0].y += a[k].y; }
#pragma unroll
    for (int j = 1; j <= H; ++j) {
      Cx<T> r = v[0], s = mk<T>((T)0, (T)0);
#pragma unroll
      for (int k = 1; k <= H; ++k) {
        const T c = (T)odd_cos<R>((j * k) % R), sn = (T)odd_sin<R>((j * k) % R);
        r.x = fma(c, a[k - 1].x, r.x); r.y = fma(c, a[k - 1].y, r.y);
        s.x = fma(sn, b[k - 1].x, s.x); s.y = fma(sn, b[k - 1].y, s.y);
      }
      const Cx<T> lo = mk<T>(r.x + s.y, r.y - s.x), hi = mk<T>(r.x - s.y, r.y + s.x);  // r - i s, r + i s
      out[j] = INV ? hi : lo;
      out[R - j] = INV ? lo : hi;
    }
#pragma unroll
    for (int k = 0; k < R; ++k) v[k] = out[k];
  }
};
template <typename T, bool INV> struct Dft<T, 3, INV> : DftOdd<T, 3, INV> {};
template <typename T, bool INV> struct Dft<T, 5, INV> : DftOdd<T, 5, INV> {};
template <typename T, bool INV> struct Dft<T, 7, INV> : DftOdd<T, 7, INV> {};

// Radix 2 x Q (Q = 3, 5, 7) in registers, decimation in frequency: sums and differences of the
// halves, the differences turned by w_R^n (compile-time roots), then two radix-Q transforms;
// even outputs from the sums, odd outputs from the differences.
template <int R> constexpr double comp_cos(int m) {   // cos(2 pi m / R), R = 6, 10, 14, m < R / 2
  constexpr double c6[3] = {1.0, 0.5, -0.5};
  constexpr double c10[5] = {1.0, 0.80901699437494742410, 0.30901699437494742410, -0.30901699437494742410,
                             -0.80901699437494742410};
  constexpr double c14[7] = {1.0, 0.90096886790241912624, 0.62348980185873353053, 0.22252093395631440429,
                             -0.22252093395631440429, -0.62348980185873353053, -0.90096886790241912624};
  return R == 6 ? c6[m] : (R == 10 ? c10[m] : c14[m]);
}
template <int R> constexpr double comp_sin(int m) {   // sin(2 pi m / R)
  constexpr double s6[3] = {0.0, 0.86602540378443864676, 0.86602540378443864676};
  constexpr double s10[5] = {0.0, 0.58778525229247312917, 0.95105651629515357212, 0.95105651629515357212,
                             0.58778525229247312917};
  constexpr double s14[7] = {0.0, 0.43388373911755812048, 0.78183148246802980871, 0.97492791218182360702,
                             0.97492791218182360702, 0.78183148246802980871, 0.43388373911755812048};
  return R == 6 ? s6[m] : (R == 10 ? s10[m] : s14[m]);
}
template <typename T, int R, bool INV> struct DftTwoOdd {
  static __device__ __forceinline__ void run(Cx<T>* v) {
    constexpr int Q = R / 2;
    Cx<T> a[Q], b[Q];
#pragma unroll
    for (int n = 0; n < Q; ++n) {
      a[n] = mk<T>(v[n].x + v[n + Q].x, v[n].y + v[n + Q].y);
      const Cx<T> d = mk<T>(v[n].x - v[n + Q].x, v[n].y - v[n + Q].y);
      const T c = (T)comp_cos<R>(n), sn = (T)comp_sin<R>(n);
      // forward: d (c - i sn); inverse: d (c + i sn)
      b[n] = n == 0 ? d
                    : (INV ? mk<T>(d.x * c - d.y * sn, d.y * c + d.x * sn) : mk<T>(d.x * c + d.y * sn, d.y * c - d.x * sn));
    }
    Dft<T, Q, INV>::run(a);
    Dft<T, Q, INV>::run(b);
#pragma unroll
    for (int k = 0; k < Q; ++k) {
      v[2 * k] = a[k];
      v[2 * k + 1] = b[k];
    }
  }
};
template <typename T, bool INV> struct Dft<T, 6, INV> : DftTwoOdd<T, 6, INV> {};
template <typename T, bool INV> struct Dft<T, 10, INV> : DftTwoOdd<T, 10, INV> {};
template <typename T, bool INV> struct Dft<T, 14, INV> : DftTwoOdd<T, 14, INV> {};

// Composite radix N = RA x RB in registers (Cooley-Tukey, compile-time roots): with n = RB n1 + n2 and
// k = k1 + RA k2,  X[k] = sum_n2 w_RB^(n2 k2) . w_N^(n2 k1) . sum_n1 w_RA^(n1 k1) x[RB n1 + n2].
// Used for 25 = 5 x 5, 9 = 3 x 3, 15 = 5 x 3, 12 = 4 x 3 of the two-stage mixed-radix plans.
template <typename T, int RA, int RB, bool INV> struct DftCT {
  static constexpr int N = RA * RB;
  template <int N2, int... K1>
  static __device__ __forceinline__ void inner(const Cx<T>* v, Cx<T>* t, std::integer_sequence<int, K1...>) {
    Cx<T> y[RA];
#pragma unroll
    for (int n1 = 0; n1 < RA; ++n1) y[n1] = v[RB * n1 + N2];
    Dft<T, RA, INV>::run(y);
    ((t[N2 * RA + K1] = mul_root<T, N, N2 * K1, INV>(y[K1])), ...);
  }
  template <int... N2>
  static __device__ __forceinline__ void first(const Cx<T>* v, Cx<T>* t, std::integer_sequence<int, N2...>) {
    (inner<N2>(v, t, std::make_integer_sequence<int, RA>{}), ...);
  }
  static __device__ __forceinline__ void run(Cx<T>* v) {
    Cx<T> t[N];
    first(v, t, std::make_integer_sequence<int, RB>{});
#pragma unroll
    for (int k1 = 0; k1 < RA; ++k1) {
      Cx<T> z[RB];
#pragma unroll
      for (int n2 = 0; n2 < RB; ++n2) z[n2] = t[n2 * RA + k1];
      Dft<T, RB, INV>::run(z);
#pragma unroll
      for (int k2 = 0; k2 < RB; ++k2) v[k1 + RA * k2] = z[k2];
    }
  }
};
template <typename T, bool INV> struct Dft<T, 25, INV> : DftCT<T, 5, 5, INV> {};
template <typename T, bool INV> struct Dft<T, 9, INV> : DftCT<T, 3, 3, INV> {};
template <typename T, bool INV> struct Dft<T, 15, INV> : DftCT<T, 5, 3, INV> {};
template <typename T, bool INV> struct Dft<T, 12, INV> : DftCT<T, 4, 3, INV> {};

// One forward stage of span S (radix R) over a tile of N rows x B columns in shared memory,
// row r of column c at sm[r * B + c].  Thread (col, tt) with NT threads per column.
// W[q] = exp(-2 pi i q / P); wstep = P / S so that w_S^(t u) = W[t u wstep].
template <typename T, int R>
__device__ __forceinline__ void stage_fwd(Cx<T>* sm, int B, int col, int tt, int NT, int N, int S,
                                          const Cx<T>* __restrict__ W, int wstep) {
  const unsigned q = S / R, qB = q * B, nb = N / R;
  for (unsigned b = tt; b < nb; b += NT) {
    const unsigned blk = b / q, t = b - blk * q;
    Cx<T>* p = sm + (blk * S + t) * B + col;
    Cx<T> v[R];
#pragma unroll
    for (int s = 0; s < R; ++s) v[s] = p[s * qB];
    Dft<T, R, false>::run(v);
    if (q > 1) {
      // w_S^(t u), u = 1 .. R - 1: the first from the table, the rest by successive products
      // (R - 2 roundings: well inside the 1e-12 / 2e-5 bars) instead of R - 1 table loads
      const Cx<T> w1 = __ldg(W + t * wstep);
      Cx<T> w = w1;
      v[1] = cmul(v[1], w);
#pragma unroll
      for (int u = 2; u < R; ++u) { w = cmul(w, w1); v[u] = cmul(v[u], w); }
    }
#pragma unroll
    for (int u = 0; u < R; ++u) p[u * qB] = v[u];
  }
}

// Exact mirror of stage_fwd: conj twiddle, inverse butterfly (unnormalised).
template <typename T, int R>
__device__ __forceinline__ void stage_inv(Cx<T>* sm, int B, int col, int tt, int NT, int N, int S,
                                          const Cx<T>* __restrict__ W, int wstep) {
  const unsigned q = S / R, qB = q * B, nb = N / R;
  for (unsigned b = tt; b < nb; b += NT) {
    const unsigned blk = b / q, t = b - blk * q;
    Cx<T>* p = sm + (blk * S + t) * B + col;
    Cx<T> v[R];
#pragma unroll
    for (int u = 0; u < R; ++u) v[u] = p[u * qB];
    if (q > 1) {
      const Cx<T> w1 = __ldg(W + t * wstep);
      Cx<T> w = w1;
      v[1] = cmulc(v[1], w);
#pragma unroll
      for (int u = 2; u < R; ++u) { w = cmul(w, w1); v[u] = cmulc(v[u], w); }
    }
    Dft<T, R, true>::run(v);
#pragma unroll
    for (int s = 0; s < R; ++s) p[s * qB] = v[s];
  }
}

// All forward stages of the length-L sub-transforms tiling the N rows (N multiple of L).
template <typename T>
__device__ __forceinline__ void run_stages_fwd(Cx<T>* sm, int B, int col, int tt, int NT, int N,
                                               const FftPlan& pl, const Cx<T>* __restrict__ W) {
  int S = pl.L;
  for (int i = 0; i < pl.nstages; ++i) {
    const int R = pl.radix[i];
    const int wstep = pl.P / S;
    switch (R) {
      case 16: stage_fwd<T, 16>(sm, B, col, tt, NT, N, S, W, wstep); break;
      case 14: stage_fwd<T, 14>(sm, B, col, tt, NT, N, S, W, wstep); break;
      case 10: stage_fwd<T, 10>(sm, B, col, tt, NT, N, S, W, wstep); break;
      case 6: stage_fwd<T, 6>(sm, B, col, tt, NT, N, S, W, wstep); break;
      case 8: stage_fwd<T, 8>(sm, B, col, tt, NT, N, S, W, wstep); break;
      case 7: stage_fwd<T, 7>(sm, B, col, tt, NT, N, S, W, wstep); break;
      case 5: stage_fwd<T, 5>(sm, B, col, tt, NT, N, S, W, wstep); break;
      case 3: stage_fwd<T, 3>(sm, B, col, tt, NT, N, S, W, wstep); break;
      case 4: stage_fwd<T, 4>(sm, B, col, tt, NT, N, S, W, wstep); break;
      default: stage_fwd<T, 2>(sm, B, col, tt, NT, N, S, W, wstep); break;
    }
    S /= R;
    __syncthreads();
  }
}

template <typename T>
__device__ __forceinline__ void run_stages_inv(Cx<T>* sm, int B, int col, int tt, int NT, int N,
                                               const FftPlan& pl, const Cx<T>* __restrict__ W) {
  int S = 1;
  for (int i = pl.nstages - 1; i >= 0; --i) {
    const int R = pl.radix[i];
    S *= R;
    const int wstep = pl.P / S;
    switch (R) {
      case 16: stage_inv<T, 16>(sm, B, col, tt, NT, N, S, W, wstep); break;
      case 14: stage_inv<T, 14>(sm, B, col, tt, NT, N, S, W, wstep); break;
      case 10: stage_inv<T, 10>(sm, B, col, tt, NT, N, S, W, wstep); break;
      case 6: stage_inv<T, 6>(sm, B, col, tt, NT, N, S, W, wstep); break;
      case 8: stage_inv<T, 8>(sm, B, col, tt, NT, N, S, W, wstep); break;
      case 7: stage_inv<T, 7>(sm, B, col, tt, NT, N, S, W, wstep); break;
      case 5: stage_inv<T, 5>(sm, B, col, tt, NT, N, S, W, wstep); break;
      case 3: stage_inv<T, 3>(sm, B, col, tt, NT, N, S, W, wstep); break;
      case 4: stage_inv<T, 4>(sm, B, col, tt, NT, N, S, W, wstep); break;
      default: stage_inv<T, 2>(sm, B, col, tt, NT, N, S, W, wstep); break;
    }
    __syncthreads();
  }
}

// Host side: position of frequency k in the digit-reversed output of the pruned length-P
// transform (first a radix-2 split into even/odd outputs, then the plan's stages on L).
//   k = u0 + 2 (u1 + R1 (u2 + R2 (...)))  ->  pos = u0 L + u1 L/R1 + u2 L/(R1 R2) + ...
inline int pos_of_freq(const FftPlan& pl, int k) {
  if (pl.P == 1) return 0;
  int pos = (k & 1) * pl.L;
  int kk = k >> 1, span = pl.L;
  for (int i = 0; i < pl.nstages; ++i) {
    const int R = pl.radix[i];
    span /= R;
    pos += (kk % R) * span;
    kk /= R;
  }
  return pos;
}

// n = 2^a 3^b 5^c 7^d: radix-8 stages (then 4 or 2) for the power of two, then the odd primes.
// nstages = -1 if n has another prime factor or needs more than MM_MAX_STAGES stages.
inline FftPlan make_plan(int n) {
  FftPlan pl{};
  pl.L = n;
  pl.P = n == 1 ? 1 : 2 * n;
  pl.nstages = 0;
  int p2 = 1, odd = n;
  bool full = false;   // more than MM_MAX_STAGES stages: unsupported, never written past radix[]
  auto push = [&](int r) {
    if (pl.nstages == MM_MAX_STAGES) { full = true; return; }
    pl.radix[pl.nstages++] = r;
  };
  while (odd % 2 == 0) { odd /= 2; p2 *= 2; }
  while (p2 >= 8) { push(8); p2 /= 8; }
  const int primes[3] = {7, 5, 3};
  // a remaining factor 2 (or each 2 of a remaining 4) joins an odd prime: radix 14, 10 or 6
  for (int f : primes)
    while (p2 > 1 && odd % f == 0) {
      push(2 * f);
      odd /= f;
      p2 /= 2;
    }
  if (p2 > 1) push(p2);
  for (int f : primes)
    while (odd % f == 0) {
      push(f);
      odd /= f;
    }
  if (full) { pl.nstages = -1; return pl; }
  if (odd != 1) pl.nstages = -1;
  return pl;
}

}  // namespace mm
