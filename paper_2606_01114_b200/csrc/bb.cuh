// Barzilai-Borwein energy minimiser ("The Barzikai-Borwein algorithm for minimising
// the system energy ... all ranks terminate together after the convergence criteria are met";
// PAPER.md:146-148 minimizer.minimize(state)).  The paper names the algorithm only; the scheme is
// reading Q30 of DESIGN.md.  One iteration = one ordinary S1..S6 evaluation producing
// g = m x (m x H_eff), three mesh-wide sums in a fixed order, a one-CTA controller, the
// norm-preserving update with the maximum change of m, and a one-thread finish.  The state lives
// on the DEVICE: an iteration needs no host round trip (the paper's distributed version needs
// global reductions here) and a converged state turns further iterations into no-ops.
#pragma once
#include "mm_common.cuh"

namespace mm {

struct BbState {
  unsigned long long n;        // iterations done
  double tau0, tau_min, tau_max, tol;
  double tau;                  // step length of the last iteration [m/A]
  double dm_max;               // max |m_{n+1} - m_n| of the last iteration
  double ss, sy, yy;           // the three sums of the last iteration (n > 0)
  unsigned long long dmbits;   // running maximum of the iteration in flight (bit pattern, non-negative real)
  int converged;
  int pad;
};

constexpr int kBbMaxBlocks = 148 * 16;   // partial-sum slots (3 doubles each)

// g: the evaluated m x (m x H_eff); m_prev, g_prev: the previous iterate (written here);
// partial: kBbMaxBlocks * 3 doubles.
template <typename T>
cudaError_t bb_iterate_launch(BbState* st_dev, T* m, const T* g, T* m_prev, T* g_prev, double* partial,
                              size_t n3, cudaStream_t st, unsigned long long* launches);

}  // namespace mm
