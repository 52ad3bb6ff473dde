// S0 launcher: Newell tensor -> packed Fourier-space table (see demag_init.cu).
#pragma once
#include "mm_common.cuh"

namespace mm {

struct InitGeom {
  int nx, ny, nz;
  int Px, Py, Pz;
  int Kz;
  int ox, oy, oz;  // octant extents: n_d + 1, or 1 when n_d == 1
  int ozp;         // fast path: kz pitch of a table row (oz rounded up to even: 16-byte bulk copies)
  int Bk;          // ky' rows per x-pass tile (table blocking)
};

size_t demag_init_scratch_bytes(const InitGeom& g);

// fx[pos] / fy[pos]: frequency held at position pos of the digit-reversed x / y transform.
// fast == 1: pack the natural-order octant T[kx][ky][6][ozp] for demag_fast.cu instead; fast == 2: T[ky][kx][6][ozp]
// (slab layout).
template <typename T>
cudaError_t demag_init_launch(const InitGeom& g, double dx, double dy, double dz, void* scratch,
                              const uint16_t* fx, const uint16_t* fy, T* table, int fast,
                              cudaStream_t st, unsigned long long* launches);

// posx[k] / posy[k]: position of frequency k.  out: [6][ox][oy][oz], unscaled.
template <typename T>
cudaError_t demag_export_launch(const InitGeom& g, const T* table, const uint16_t* posx,
                                const uint16_t* posy, T* out, int fast, cudaStream_t st,
                                unsigned long long* launches);

}  // namespace mm
