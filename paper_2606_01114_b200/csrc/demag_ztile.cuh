// K3 (S3: last axis forward . Nhat multiply . inverse) of the x-first demag path as a
// shared-memory tile with two register stages per direction, for the z lengths of plan2.cuh's
// MM_ZTILE_LENGTHS (the paper's nz = 100, 350, 400 and 90).  See demag_ztile.cu.
#pragma once
#include "demag_fast.cuh"

namespace mm {

bool ztile_supported(int nz);

// In place on nk planes of b.A2 whose table planes start at k0; b.T2z is the plan's stage twiddle table;
// xm: the rows of a plane are kx (slab layout).
template <typename T>
cudaError_t ztile_launch(const FastGeom& g, const FastBufs<T>& b, int k0, int nk, int xm, cudaStream_t st);

}  // namespace mm
