// Geometry / buffer descriptors of the demag passes and their host launcher.
#pragma once
#include "mm_common.cuh"

namespace mm {

struct DemagGeom {
  int nx, ny, nz;  // cells
  int Px, Py, Pz;  // padded lengths (2n, or 1 when n == 1)
  int Kz;          // kz planes kept after the r2c z pass: Pz/2 + 1
  FftPlan px, py, pz;
  int Bz, By, Bk;  // tile widths: x columns of the z passes, x columns of the y passes,
                   // ky' rows of the x pass
};

template <typename T> struct DemagBufs {
  const Cx<T>* Wx;       // Wx[q] = exp(-2 pi i q / Px), q < Px
  const Cx<T>* Wy;
  const Cx<T>* Wz;
  const uint16_t* posz;  // position of frequency kz in the digit-reversed z transform
  const T* table;        // packed Fourier-space tensor, see xp_kernel
  Cx<T>* A1;             // [3][Kz][ny][nx]
  Cx<T>* A2;             // [3][Kz][Py][nx]
};

// Enqueues S1..S5: H := scale * crop(IFFT(table . FFT(pad(m)))).
template <typename T>
cudaError_t demag_field_launch(const DemagGeom& g, const DemagBufs<T>& b, const T* m, T* H,
                               T scale, cudaStream_t st, unsigned long long* launches, Prof* prof);

}  // namespace mm
