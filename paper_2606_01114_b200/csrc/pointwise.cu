// S6/S7: one pass over the mesh computes the 6-point exchange stencil
// (eq. 2, Neumann boundary), the DMI field from the same six neighbours
// (eq. 3, central differences), uniaxial anisotropy and the spin-torque field
// (PAPER.md:30), Zeeman, adds H_demag, forms the LLG right-hand side
// (eq. 1) and
// applies the RK4 stage arithmetic, so H_eff and k_i are never written to HBM.
// HBM-bound: 128-bit loads/stores, 4 (fp32) or 2 (fp64) consecutive z cells per thread; the six
// neighbours come from L1/L2.
#include "pointwise.cuh"

#include "../../include/mm_b200.h"

namespace mm {

// NR consecutive reals, 16-byte aligned, moved by 128-bit accesses.  A thread owns CPT consecutive
// z cells: 4 in fp32 (12 reals = 3 float4), 2 in fp64 (6 reals = 3 double2; with 4 cells the
// fp64 kernel held 60 doubles per thread and ran at 56 % of the HBM rate).
template <typename T> struct Cpt { static constexpr int value = sizeof(T) == 4 ? 4 : 2; };
template <typename T, int NR> struct VN;
template <int NR> struct VN<float, NR> {
  // NR = 12 (four cells): three 128-bit accesses; NR = 6 (two cells, nz = 2 mod 4: rows are only 8-byte
  // aligned): three 64-bit accesses
  static __device__ __forceinline__ void ld(const float* p, float (&v)[NR]) {
    if constexpr (NR % 4 == 0) {
      const float4* q = reinterpret_cast<const float4*>(p);
#pragma unroll
      for (int i = 0; i < NR / 4; ++i) {
        const float4 t = q[i];
        v[4 * i] = t.x; v[4 * i + 1] = t.y; v[4 * i + 2] = t.z; v[4 * i + 3] = t.w;
      }
    } else {
      const float2* q = reinterpret_cast<const float2*>(p);
#pragma unroll
      for (int i = 0; i < NR / 2; ++i) {
        const float2 t = q[i];
        v[2 * i] = t.x; v[2 * i + 1] = t.y;
      }
    }
  }
  static __device__ __forceinline__ void st(float* p, const float (&v)[NR]) {
    if constexpr (NR % 4 == 0) {
      float4* q = reinterpret_cast<float4*>(p);
#pragma unroll
      for (int i = 0; i < NR / 4; ++i) q[i] = make_float4(v[4 * i], v[4 * i + 1], v[4 * i + 2], v[4 * i + 3]);
    } else {
      float2* q = reinterpret_cast<float2*>(p);
#pragma unroll
      for (int i = 0; i < NR / 2; ++i) q[i] = make_float2(v[2 * i], v[2 * i + 1]);
    }
  }
};
template <int NR> struct VN<double, NR> {
  static __device__ __forceinline__ void ld(const double* p, double (&v)[NR]) {
    const double2* q = reinterpret_cast<const double2*>(p);
#pragma unroll
    for (int i = 0; i < NR / 2; ++i) {
      const double2 t = q[i];
      v[2 * i] = t.x; v[2 * i + 1] = t.y;
    }
  }
  static __device__ __forceinline__ void st(double* p, const double (&v)[NR]) {
    double2* q = reinterpret_cast<double2*>(p);
#pragma unroll
    for (int i = 0; i < NR / 2; ++i) q[i] = make_double2(v[2 * i], v[2 * i + 1]);
  }
};

// Everything that happens in one cell once its neighbours are known.
// mc: m at the cell; lap: exchange field already summed; hd: demag field (or 0);
// m0v / accv: RK4 step-start state and running sum (only read in RK modes).
// Returns through o[3] the value to store in `out` (or m0 for PW_RK_FINAL); accv is updated.
// hx += E x d  (one DMI direction: E = scaled DMI vector, d = m(i + e_k) - m(i - e_k))
template <typename T> __device__ __forceinline__ void dmi_add(const T* E, const T* d, T* hx) {
  hx[0] += E[1] * d[2] - E[2] * d[1];
  hx[1] += E[2] * d[0] - E[0] * d[2];
  hx[2] += E[0] * d[1] - E[1] * d[0];
}

template <typename T, int MODE, bool DMI>
__device__ __forceinline__ void cell_update(const PwParams<T>& p, const T* mc, const T* lap,
                                            const T* hx, const T* hd, const T* m0v, T* accv, T* o) {
  T h[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) h[c] = (p.terms & MM_TERM_EXCHANGE) ? lap[c] : (T)0;
  if (MODE == PW_EXCHANGE) {
#pragma unroll
    for (int c = 0; c < 3; ++c) o[c] = lap[c];
    return;
  }
  if (p.terms & MM_TERM_DEMAG) {
#pragma unroll
    for (int c = 0; c < 3; ++c) h[c] += hd[c];
  }
  if (p.terms & MM_TERM_ANISOTROPY) {
    const T d = p.kan * (mc[0] * p.u[0] + mc[1] * p.u[1] + mc[2] * p.u[2]);
#pragma unroll
    for (int c = 0; c < 3; ++c) h[c] += d * p.u[c];
  }
  if (p.terms & MM_TERM_ZEEMAN) {
#pragma unroll
    for (int c = 0; c < 3; ++c) h[c] += p.hext[c];
  }
  if (DMI) {
#pragma unroll
    for (int c = 0; c < 3; ++c) h[c] += hx[c];
  }
  if (p.terms & MM_TERM_STT) {
    h[0] += p.sdamp * (mc[1] * p.sp[2] - mc[2] * p.sp[1]) + p.sfield * p.sp[0];
    h[1] += p.sdamp * (mc[2] * p.sp[0] - mc[0] * p.sp[2]) + p.sfield * p.sp[1];
    h[2] += p.sdamp * (mc[0] * p.sp[1] - mc[1] * p.sp[0]) + p.sfield * p.sp[2];
  }
  if (MODE == PW_HEFF) {
#pragma unroll
    for (int c = 0; c < 3; ++c) o[c] = h[c];
    return;
  }
  // m x H, then m x (m x H) as a genuine double cross product (keeps m . dm/dt = 0)
  const T t0 = mc[1] * h[2] - mc[2] * h[1];
  const T t1 = mc[2] * h[0] - mc[0] * h[2];
  const T t2 = mc[0] * h[1] - mc[1] * h[0];
  const T d0 = mc[1] * t2 - mc[2] * t1;
  const T d1 = mc[2] * t0 - mc[0] * t2;
  const T d2 = mc[0] * t1 - mc[1] * t0;
  if (MODE == PW_MIN_G) {
    o[0] = d0; o[1] = d1; o[2] = d2;
    return;
  }
  T k[3] = {p.pref * (t0 + p.alpha * d0), p.pref * (t1 + p.alpha * d1),
            p.pref * (t2 + p.alpha * d2)};
  if (MODE == PW_RHS) {
#pragma unroll
    for (int c = 0; c < 3; ++c) o[c] = k[c];
  } else if (MODE == PW_RK_STAGE) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      accv[c] = p.first ? k[c] : accv[c] + p.wk * k[c];
      o[c] = m0v[c] + p.a * k[c];
    }
  } else {  // PW_RK_FINAL
    T v[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) v[c] = m0v[c] + p.a * (accv[c] + k[c]);
    const T inv = (T)1 / sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
#pragma unroll
    for (int c = 0; c < 3; ++c) o[c] = v[c] * inv;
  }
}

// Vector path: nz % CPT == 0.  Thread = CPT consecutive z cells of one (x, y) line.
template <typename T, int MODE, bool DMI, int CPT>
__global__ void __launch_bounds__(256) pw_vec_kernel(PwParams<T> p, const T* __restrict__ m,
                                                     const T* __restrict__ Hd, T* __restrict__ out,
                                                     T* __restrict__ m0, T* __restrict__ acc) {
  constexpr int NR = 3 * CPT;
  using V = VN<T, NR>;
  const int nzq = p.nz / CPT;
  const size_t total = (size_t)p.nx * p.ny * nzq;
  const size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= total) return;
  const int zq = (int)(g % nzq);
  const int y = (int)((g / nzq) % p.ny);
  const int x = (int)(g / ((size_t)nzq * p.ny));
  const size_t sy = (size_t)p.nz * 3, sx = sy * p.ny;
  const size_t base = (size_t)x * sx + (size_t)y * sy + (size_t)zq * NR;
  const bool need_lap = (p.terms & MM_TERM_EXCHANGE) || MODE == PW_EXCHANGE || DMI;

  T mc[NR], lap[NR], hx[DMI ? NR : 1];
  V::ld(m + base, mc);
#pragma unroll
  for (int i = 0; i < NR; ++i) lap[i] = 0;
#pragma unroll
  for (int i = 0; i < (DMI ? NR : 1); ++i) hx[i] = 0;
  if (need_lap) {
    T nb[NR], dd[DMI ? NR : 1];
    if (p.nx > 1) {
      V::ld(m + (x > 0 ? base - sx : base), nb);
#pragma unroll
      for (int i = 0; i < NR; ++i) {
        lap[i] += p.ex[0] * (nb[i] - mc[i]);
        if (DMI) dd[i] = -nb[i];
      }
      V::ld(m + (x + 1 < p.nx ? base + sx : base), nb);
#pragma unroll
      for (int i = 0; i < NR; ++i) {
        lap[i] += p.ex[0] * (nb[i] - mc[i]);
        if (DMI) dd[i] += nb[i];
      }
      if (DMI) {
#pragma unroll
        for (int j = 0; j < CPT; ++j) dmi_add<T>(p.dmi[0], dd + 3 * j, hx + 3 * j);
      }
    }
    if (p.ny > 1) {
      V::ld(m + (y > 0 ? base - sy : base), nb);
#pragma unroll
      for (int i = 0; i < NR; ++i) {
        lap[i] += p.ex[1] * (nb[i] - mc[i]);
        if (DMI) dd[i] = -nb[i];
      }
      V::ld(m + (y + 1 < p.ny ? base + sy : base), nb);
#pragma unroll
      for (int i = 0; i < NR; ++i) {
        lap[i] += p.ex[1] * (nb[i] - mc[i]);
        if (DMI) dd[i] += nb[i];
      }
      if (DMI) {
#pragma unroll
        for (int j = 0; j < CPT; ++j) dmi_add<T>(p.dmi[1], dd + 3 * j, hx + 3 * j);
      }
    }
    {
      T lo[3], hi[3];
      const bool has_lo = zq > 0, has_hi = zq + 1 < nzq;
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        lo[c] = has_lo ? m[base - 3 + c] : mc[c];
        hi[c] = has_hi ? m[base + NR + c] : mc[NR - 3 + c];
      }
#pragma unroll
      for (int j = 0; j < CPT; ++j)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const T below = j == 0 ? lo[c] : mc[3 * (j - 1) + c];
          const T above = j == CPT - 1 ? hi[c] : mc[3 * (j + 1) + c];
          lap[3 * j + c] += p.ex[2] * ((below - mc[3 * j + c]) + (above - mc[3 * j + c]));
          if (DMI) dd[3 * j + c] = above - below;
        }
      if (DMI) {
#pragma unroll
        for (int j = 0; j < CPT; ++j) dmi_add<T>(p.dmi[2], dd + 3 * j, hx + 3 * j);
      }
    }
  }
  T hd[NR], m0v[NR], accv[NR], o[NR];
#pragma unroll
  for (int i = 0; i < NR; ++i) hd[i] = m0v[i] = accv[i] = 0;
  if (MODE != PW_EXCHANGE && (p.terms & MM_TERM_DEMAG)) V::ld(Hd + base, hd);
  if (MODE == PW_RK_STAGE || MODE == PW_RK_FINAL) {
    V::ld(m0 + base, m0v);
    if (!(MODE == PW_RK_STAGE && p.first)) V::ld(acc + base, accv);
  }
#pragma unroll
  for (int j = 0; j < CPT; ++j)
    cell_update<T, MODE, DMI>(p, mc + 3 * j, lap + 3 * j, hx + (DMI ? 3 * j : 0), hd + 3 * j, m0v + 3 * j,
                              accv + 3 * j, o + 3 * j);
  if (MODE == PW_RK_STAGE) V::st(acc + base, accv);
  V::st((MODE == PW_RK_FINAL ? m0 : out) + base, o);
}

// Scalar path for the other nz (thin films, odd nz): thread = one cell.
template <typename T, int MODE, bool DMI>
__global__ void __launch_bounds__(256) pw_cell_kernel(PwParams<T> p, const T* __restrict__ m,
                                                      const T* __restrict__ Hd, T* __restrict__ out,
                                                      T* __restrict__ m0, T* __restrict__ acc) {
  const size_t total = (size_t)p.nx * p.ny * p.nz;
  const size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= total) return;
  const int z = (int)(g % p.nz);
  const int y = (int)((g / p.nz) % p.ny);
  const int x = (int)(g / ((size_t)p.nz * p.ny));
  const size_t sy = (size_t)p.nz * 3, sx = sy * p.ny;
  const size_t base = g * 3;
  const bool need_lap = (p.terms & MM_TERM_EXCHANGE) || MODE == PW_EXCHANGE || DMI;
  T mc[3], lap[3] = {0, 0, 0}, hx[3] = {0, 0, 0};
#pragma unroll
  for (int c = 0; c < 3; ++c) mc[c] = m[base + c];
  if (need_lap) {
    const size_t off[3] = {sx, sy, 3};
    const int idx[3] = {x, y, z}, n[3] = {p.nx, p.ny, p.nz};
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const size_t lo = idx[d] > 0 ? base - off[d] : base;
      const size_t hi = idx[d] + 1 < n[d] ? base + off[d] : base;
#pragma unroll
      for (int c = 0; c < 3; ++c) lap[c] += p.ex[d] * ((m[lo + c] - mc[c]) + (m[hi + c] - mc[c]));
      if (DMI) {
        const T dd[3] = {m[hi] - m[lo], m[hi + 1] - m[lo + 1], m[hi + 2] - m[lo + 2]};
        dmi_add<T>(p.dmi[d], dd, hx);
      }
    }
  }
  T hd[3] = {0, 0, 0}, m0v[3] = {0, 0, 0}, accv[3] = {0, 0, 0}, o[3];
  if (MODE != PW_EXCHANGE && (p.terms & MM_TERM_DEMAG)) {
#pragma unroll
    for (int c = 0; c < 3; ++c) hd[c] = Hd[base + c];
  }
  if (MODE == PW_RK_STAGE || MODE == PW_RK_FINAL) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      m0v[c] = m0[base + c];
      if (!(MODE == PW_RK_STAGE && p.first)) accv[c] = acc[base + c];
    }
  }
  cell_update<T, MODE, DMI>(p, mc, lap, hx, hd, m0v, accv, o);
  T* dst = MODE == PW_RK_FINAL ? m0 : out;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    if (MODE == PW_RK_STAGE) acc[base + c] = accv[c];
    dst[base + c] = o[c];
  }
}

// Per-cell Ms and A (eq. 2 as div(A grad M); reading Q31): thread = one cell.
//   exchange  2/(mu0 Ms_i) sum A_ij (m_j - m_i)/d^2, A_ij = 2 A_i A_j/(A_i + A_j); a neighbour outside the
//             mesh or in vacuum (Ms_j = 0): no term
//   DMI, anisotropy with Ms_i; for DMI a neighbour outside the mesh or with Ms_j = 0 is the cell itself
//   Ms_i = 0: vacuum -- those terms vanish, dm/dt = 0, a zero vector is not renormalised
template <typename T, int MODE>
__global__ void __launch_bounds__(256) pw_inhom_kernel(PwParams<T> p, const T* __restrict__ m,
                                                       const T* __restrict__ Hd, T* __restrict__ out,
                                                       T* __restrict__ m0, T* __restrict__ acc) {
  const size_t total = (size_t)p.nx * p.ny * p.nz;
  const size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= total) return;
  const int z = (int)(g % p.nz);
  const int y = (int)((g / p.nz) % p.ny);
  const int x = (int)(g / ((size_t)p.nz * p.ny));
  const size_t off[3] = {(size_t)p.nz * p.ny, (size_t)p.nz, 1};   // in cells
  const int idx[3] = {x, y, z}, n[3] = {p.nx, p.ny, p.nz};
  const size_t base = g * 3;
  const T Msi = p.ms_cells ? p.ms_cells[g] : p.ms_ref, Ai = p.a_cells ? p.a_cells[g] : p.a_ref;
  const bool mag = Msi > (T)0;
  T mc[3] = {m[base], m[base + 1], m[base + 2]};
  T lap[3] = {0, 0, 0}, hx[3] = {0, 0, 0};
  const bool want_ex = (p.terms & MM_TERM_EXCHANGE) || MODE == PW_EXCHANGE;
  const bool want_dmi = (p.terms & MM_TERM_DMI) && MODE != PW_EXCHANGE;
  if (mag && (want_ex || want_dmi)) {
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      T dm[3] = {0, 0, 0};
#pragma unroll
      for (int sg = -1; sg <= 1; sg += 2) {
        const bool inside = sg < 0 ? idx[d] > 0 : idx[d] + 1 < n[d];
        const size_t cj = inside ? (sg < 0 ? g - off[d] : g + off[d]) : g;
        const T Msj = p.ms_cells ? p.ms_cells[cj] : p.ms_ref, Aj = p.a_cells ? p.a_cells[cj] : p.a_ref;
        const T mj[3] = {m[3 * cj], m[3 * cj + 1], m[3 * cj + 2]};
        if (want_ex && inside && Msj > (T)0 && Ai + Aj > (T)0) {   // a vacuum neighbour is no exchange partner
          const T w = p.exq[d] * ((T)2 * Ai * Aj / (Ai + Aj));
#pragma unroll
          for (int c = 0; c < 3; ++c) lap[c] += w * (mj[c] - mc[c]);
        }
        const bool use = inside && Msj > (T)0;
#pragma unroll
        for (int c = 0; c < 3; ++c) dm[c] += (T)sg * (use ? mj[c] : mc[c]);
      }
      if (want_dmi) dmi_add<T>(p.dmiq[d], dm, hx);
    }
  }
  const T inv_ms = mag ? (T)1 / Msi : (T)0;
  T h[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) h[c] = lap[c] * inv_ms;
  T* dst = MODE == PW_RK_FINAL ? m0 : out;
  if (MODE == PW_EXCHANGE) {
#pragma unroll
    for (int c = 0; c < 3; ++c) dst[base + c] = h[c];
    return;
  }
  if (!(p.terms & MM_TERM_EXCHANGE)) h[0] = h[1] = h[2] = (T)0;
#pragma unroll
  for (int c = 0; c < 3; ++c) h[c] += hx[c] * inv_ms;
  if (p.terms & MM_TERM_ANISOTROPY) {
    const T dot = p.kanq * inv_ms * (mc[0] * p.u[0] + mc[1] * p.u[1] + mc[2] * p.u[2]);
#pragma unroll
    for (int c = 0; c < 3; ++c) h[c] += dot * p.u[c];
  }
  if (p.terms & MM_TERM_DEMAG) {
#pragma unroll
    for (int c = 0; c < 3; ++c) h[c] += Hd[base + c];
  }
  if (p.terms & MM_TERM_ZEEMAN) {
#pragma unroll
    for (int c = 0; c < 3; ++c) h[c] += p.hext[c];
  }
  if (p.terms & MM_TERM_STT) {
    h[0] += p.sdamp * (mc[1] * p.sp[2] - mc[2] * p.sp[1]) + p.sfield * p.sp[0];
    h[1] += p.sdamp * (mc[2] * p.sp[0] - mc[0] * p.sp[2]) + p.sfield * p.sp[1];
    h[2] += p.sdamp * (mc[0] * p.sp[1] - mc[1] * p.sp[0]) + p.sfield * p.sp[2];
  }
  if (MODE == PW_HEFF) {
#pragma unroll
    for (int c = 0; c < 3; ++c) dst[base + c] = h[c];
    return;
  }
  const T t0 = mc[1] * h[2] - mc[2] * h[1];
  const T t1 = mc[2] * h[0] - mc[0] * h[2];
  const T t2 = mc[0] * h[1] - mc[1] * h[0];
  T dd[3] = {mc[1] * t2 - mc[2] * t1, mc[2] * t0 - mc[0] * t2, mc[0] * t1 - mc[1] * t0};
  T k[3] = {p.pref * (t0 + p.alpha * dd[0]), p.pref * (t1 + p.alpha * dd[1]), p.pref * (t2 + p.alpha * dd[2])};
  if (!mag) { k[0] = k[1] = k[2] = (T)0; dd[0] = dd[1] = dd[2] = (T)0; }
  if (MODE == PW_MIN_G) {
#pragma unroll
    for (int c = 0; c < 3; ++c) dst[base + c] = dd[c];
  } else if (MODE == PW_RHS) {
#pragma unroll
    for (int c = 0; c < 3; ++c) dst[base + c] = k[c];
  } else if (MODE == PW_RK_STAGE) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      acc[base + c] = p.first ? k[c] : acc[base + c] + p.wk * k[c];
      dst[base + c] = m0[base + c] + p.a * k[c];
    }
  } else {  // PW_RK_FINAL
    T v[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) v[c] = m0[base + c] + p.a * (acc[base + c] + k[c]);
    const T nrm = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    const T inv = nrm > (T)0 ? (T)1 / nrm : (T)0;
#pragma unroll
    for (int c = 0; c < 3; ++c) dst[base + c] = v[c] * inv;
  }
}

template <typename T>
__global__ void __launch_bounds__(256) scale_by_ms_kernel(const T* __restrict__ m, const T* __restrict__ ms,
                                                          T* __restrict__ out, size_t ncell) {
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < 3 * ncell; q += stride) out[q] = ms[q / 3] * m[q];
}
template <typename T>
cudaError_t scale_by_ms_launch(const T* m, const T* ms_cells, T* out, size_t ncell, cudaStream_t st) {
  size_t b = (3 * ncell + 255) / 256;
  if (b > 148 * 32) b = 148 * 32;
  scale_by_ms_kernel<T><<<(unsigned)b, 256, 0, st>>>(m, ms_cells, out, ncell);
  return cudaGetLastError();
}
template cudaError_t scale_by_ms_launch<float>(const float*, const float*, float*, size_t, cudaStream_t);
template cudaError_t scale_by_ms_launch<double>(const double*, const double*, double*, size_t, cudaStream_t);

template <typename T, int MODE, bool DMI>
static void launch_mode_dmi(const PwParams<T>& p, const T* m, const T* Hd, T* out, T* m0, T* acc,
                            cudaStream_t st) {
  if (p.nz % Cpt<T>::value == 0) {
    const size_t total = (size_t)p.nx * p.ny * (p.nz / Cpt<T>::value);
    pw_vec_kernel<T, MODE, DMI, Cpt<T>::value><<<(unsigned)((total + 255) / 256), 256, 0, st>>>(p, m, Hd, out, m0, acc);
  } else if (p.nz % 2 == 0) {   // fp32 with nz = 2 mod 4 (the paper's nz = 350, 90): two cells per thread, 64-bit accesses
    const size_t total = (size_t)p.nx * p.ny * (p.nz / 2);
    pw_vec_kernel<T, MODE, DMI, 2><<<(unsigned)((total + 255) / 256), 256, 0, st>>>(p, m, Hd, out, m0, acc);
  } else {
    const size_t total = (size_t)p.nx * p.ny * p.nz;
    pw_cell_kernel<T, MODE, DMI><<<(unsigned)((total + 255) / 256), 256, 0, st>>>(p, m, Hd, out, m0, acc);
  }
}
template <typename T, int MODE>
static void launch_mode(const PwParams<T>& p, const T* m, const T* Hd, T* out, T* m0, T* acc,
                        cudaStream_t st) {
  if (p.ms_cells || p.a_cells) {
    const size_t total = (size_t)p.nx * p.ny * p.nz;
    pw_inhom_kernel<T, MODE><<<(unsigned)((total + 255) / 256), 256, 0, st>>>(p, m, Hd, out, m0, acc);
    return;
  }
  if (MODE != PW_EXCHANGE && (p.terms & MM_TERM_DMI)) launch_mode_dmi<T, MODE, true>(p, m, Hd, out, m0, acc, st);
  else launch_mode_dmi<T, MODE, false>(p, m, Hd, out, m0, acc, st);
}

template <typename T>
cudaError_t pointwise_launch(int mode, const PwParams<T>& p, const T* m, const T* Hd, T* out,
                             T* m0, T* acc, cudaStream_t st, unsigned long long* launches,
                             Prof* prof) {
  prof->mark(5, st);
  switch (mode) {
    case PW_EXCHANGE: launch_mode<T, PW_EXCHANGE>(p, m, Hd, out, m0, acc, st); break;
    case PW_HEFF: launch_mode<T, PW_HEFF>(p, m, Hd, out, m0, acc, st); break;
    case PW_RHS: launch_mode<T, PW_RHS>(p, m, Hd, out, m0, acc, st); break;
    case PW_RK_STAGE: launch_mode<T, PW_RK_STAGE>(p, m, Hd, out, m0, acc, st); break;
    case PW_MIN_G: launch_mode<T, PW_MIN_G>(p, m, Hd, out, m0, acc, st); break;
    default: launch_mode<T, PW_RK_FINAL>(p, m, Hd, out, m0, acc, st); break;
  }
  ++*launches;
  prof->mark(-1, st);
  return cudaGetLastError();
}

// embed != 0: one CTA per (x, y) row of the EMBEDDED array; cells outside the mesh are written as zero on
// every call, so the scratch array needs no state between calls.  embed == 0: one CTA per mesh row.
template <typename T>
__global__ void __launch_bounds__(128) embed_copy_kernel(const T* __restrict__ src, T* __restrict__ dst, int nx, int ny,
                                                         int nz, int eny, int enz, int embed) {
  const int rows = embed ? eny : ny;
  const int x = blockIdx.x / rows, y = blockIdx.x - x * rows;
  const size_t small = ((size_t)x * ny + y) * nz * 3, big = ((size_t)x * eny + y) * enz * 3;
  if (embed) {
    const bool in = x < nx && y < ny;
    for (int q = threadIdx.x; q < 3 * enz; q += blockDim.x) dst[big + q] = (in && q < 3 * nz) ? src[small + q] : (T)0;
  } else {
    for (int q = threadIdx.x; q < 3 * nz; q += blockDim.x) dst[small + q] = src[big + q];
  }
}

template <typename T>
cudaError_t embed_copy_launch(const T* src, T* dst, int nx, int ny, int nz, int enx, int eny, int enz, int embed,
                              cudaStream_t st) {
  const unsigned grid = embed ? (unsigned)(enx * eny) : (unsigned)(nx * ny);
  embed_copy_kernel<T><<<grid, 128, 0, st>>>(src, dst, nx, ny, nz, eny, enz, embed);
  return cudaGetLastError();
}
template cudaError_t embed_copy_launch<float>(const float*, float*, int, int, int, int, int, int, int, cudaStream_t);
template cudaError_t embed_copy_launch<double>(const double*, double*, int, int, int, int, int, int, int, cudaStream_t);

template cudaError_t pointwise_launch<float>(int, const PwParams<float>&, const float*,
                                             const float*, float*, float*, float*, cudaStream_t,
                                             unsigned long long*, Prof*);
template cudaError_t pointwise_launch<double>(int, const PwParams<double>&, const double*,
                                              const double*, double*, double*, double*,
                                              cudaStream_t, unsigned long long*, Prof*);

}  // namespace mm
