// S6/S7: fused local field terms + LLG right-hand side + RK4 stage arithmetic.
#pragma once
#include "mm_common.cuh"

namespace mm {

enum PwMode {
  PW_EXCHANGE = 0,  // out := H_exchange(m)
  PW_HEFF = 1,      // out := sum of enabled terms (Hd added when the demag term is on)
  PW_RHS = 2,       // out := LLG right-hand side at H_eff
  PW_RK_STAGE = 3,  // k := RHS; acc := (first ? k : acc + wk k); out := m0 + a k
  PW_RK_FINAL = 4,  // k := RHS; m0 := normalise(m0 + b (acc + k))
  PW_MIN_G = 5      // out := m x (m x H_eff), the minimiser's tangential gradient (bb.cuh)
};

template <typename T> struct PwParams {
  int nx, ny, nz;
  unsigned terms;     // MM_TERM_* mask actually applied
  T ex[3];            // 2A/(mu0 Ms) / d_d^2
  T kan, u[3];        // 2Ku/(mu0 Ms), unit axis
  T hext[3];          // A/m
  T dmi[3][3];        // DMI vectors e_k^DMI times 2D/(mu0 Ms) / (2 d_k); row k = 0 if n_k = 1
  T sp[3], sdamp, sfield;  // spin-torque field a_damp (m x p) + a_field p: unit p, amplitudes in A/m
  // per-cell material parameters (reading Q31); both NULL = uniform (the fields above)
  const T* ms_cells;  // Ms_i [nx][ny][nz] in A/m, or NULL (ms_ref everywhere)
  const T* a_cells;   // A_i in J/m, or NULL (a_ref everywhere)
  T ms_ref, a_ref;
  T exq[3];           // 2/(mu0 d_d^2)
  T kanq;             // 2 Ku / mu0
  T dmiq[3][3];       // DMI vectors times (2D/mu0) / (2 d_k); row k = 0 if n_k = 1
  T pref, alpha;      // -gamma/(1+alpha^2), alpha
  // RK4 bookkeeping
  int first;          // stage 1: acc is written, not accumulated
  T wk;               // weight of k in acc (1 or 2)
  T a;                // stage step a_i * dt  (PW_RK_STAGE)  /  dt/6 (PW_RK_FINAL)
};

template <typename T>
cudaError_t pointwise_launch(int mode, const PwParams<T>& p, const T* m, const T* Hd, T* out,
                             T* m0, T* acc, cudaStream_t st, unsigned long long* launches,
                             Prof* prof);

// out[i][c] = Ms_i m[i][c]: the magnetisation M = Ms m the demag passes transform when Ms varies per cell.
template <typename T>
cudaError_t scale_by_ms_launch(const T* m, const T* ms_cells, T* out, size_t ncell, cudaStream_t st);

// Copies between the mesh [nx][ny][nz][3] and its embedding in the corner of [..][eny][enz][3]
// (mm_api.cu "Embedding") of enx x eny x enz cells.  embed != 0: mesh -> embedded array, the cells
// outside the mesh written as zero; embed == 0: embedded array -> mesh.
template <typename T>
cudaError_t embed_copy_launch(const T* src, T* dst, int nx, int ny, int nz, int enx, int eny, int enz, int embed,
                              cudaStream_t st);

}  // namespace mm
