// Mixed-radix x-first demag path: the layout and pass order of demag_fast.cu (x r2c -> y ->
// z . Nhat . z^-1 -> y^-1 -> x^-1 c2r on the [x][y][3 z + c] arrays, octant Nhat table) for every
// mesh n_d = 2^a 3^b 5^c 7^d >= 2 that the power-of-two kernels do not cover: the paper's own
// workloads (N = 100, 350, 400 cubes, 512 x 512 x 90) and power-of-two
// sizes outside demag_fast.cu's plans.  Transforms are the run-time radix stages of fft_core.cuh
// in shared memory (zero-padding, FFT, pointwise multiplication, inverse, truncation).
#pragma once
#include "demag_fast.cuh"

namespace mm {

struct MixedPlans {
  FftPlan px, py, pz;   // plans of the length-n_d sub-transforms (P_d = 2 n_d)
};

template <typename T> struct MixedBufs {
  const Cx<T>* Wx;        // W[q] = exp(-2 pi i q / P_d)
  const Cx<T>* Wy;
  const Cx<T>* Wz;
  const uint16_t* posx;   // position of frequency k in the digit-reversed transform of the axis
  const uint16_t* posy;
  const uint16_t* fz;     // frequency held at position r of the z transform
  const T* table;         // Nhat[kx <= nx][ky <= ny][6][ozp]
  Cx<T>* A1;              // [nx + 1][ny][Q]
  Cx<T>* A2;              // [nx + 1][Py][Q], ky rows in digit-reversed order
};

// true if this path covers the mesh (every n_d >= 2, ny * 3 nz even, tiles fit shared memory)
bool mixed_supported(int nx, int ny, int nz, size_t real_bytes);

template <typename T>
cudaError_t demag_mixed_launch(const FastGeom& g, const MixedPlans& pl, const MixedBufs<T>& b, const T* m, T* H,
                               T scale, cudaStream_t st, unsigned long long* launches, Prof* prof);

}  // namespace mm
