// K3 (S3: last axis forward . Nhat multiply . inverse) of the x-first demag path as a
// shared-memory tile with two register stages per direction, for the z lengths of plan2.cuh's
// MM_ZTILE_LENGTHS (the paper's nz = 100, 350, 400 and 90).  See demag_ztile.cu.
#pragma once
#include "demag_fast.cuh"

namespace mm {

bool ztile_supported(int nz);

// In place on b.A2 (all nx + 1 planes); b.T2z is the plan's stage twiddle table.
template <typename T> cudaError_t ztile_launch(const FastGeom& g, const FastBufs<T>& b, cudaStream_t st);

}  // namespace mm
