// Adaptive Runge-Kutta-Fehlberg 4(5) stepping (the integrator the paper supports;
// "globally reduces the maximum error before computing the next step size").  The six right-hand
// sides are the ordinary S1..S6 evaluations; this file adds the stage combinations, the error
// maximum and a DEVICE-resident step controller, so an attempted step needs no host round trip
// and can be captured in a CUDA graph.  Readings Q23-Q26 of DESIGN.md.
#pragma once
#include "mm_common.cuh"

namespace mm {

// Controller state, resident in the persistent workspace (one 128-byte record).
struct RkfState {
  double t;        // simulated time reached by accepted steps [s]
  double dt;       // size of the NEXT attempt [s]
  double tol;      // accept iff err <= tol
  double dt_min, dt_max;
  double err;      // max |m5 - m4| of the last attempt
  double dt_last;  // size of the last attempt
  unsigned long long errbits;  // running maximum of the attempt in flight (bit pattern of a non-negative real)
  unsigned long long n_acc, n_rej;
  int accept;      // last attempt accepted
  int pad;
};

// out := m0 + dt * sum_{j < nk} a[j] K_j  (K_j = K + j * n3; dt read from the device state)
template <typename T>
cudaError_t rkf_combine_launch(const RkfState* st_dev, const T* m0, const T* K, size_t n3, int nk,
                               const double* a, T* out, cudaStream_t st);

// cand := m0 + dt * sum b5[j] K_j;  errbits := max |dt * sum (b5[j] - b4[j]) K_j|;  then the
// controller (accept / next dt / counters) and the commit (m0 := cand / |cand| per cell if accepted).
template <typename T>
cudaError_t rkf_finish_launch(RkfState* st_dev, T* m0, const T* K, size_t n3, T* cand, cudaStream_t st,
                              unsigned long long* launches);

// Fehlberg's tableau (row i, i = 1..5: coefficients of k_1..k_i in the input of stage i + 1)
const double* rkf_row(int i);

}  // namespace mm
