// Fast demag path ("x-first"): geometry, buffers and the host launcher.
//
// Same operation as demag_passes.cu (PAPER.md:45 eq. 4, :47, :53: zero-padded FFT of m, pointwise
// multiply with the Fourier-space demag tensor, inverse FFT, crop) but with the axes visited in
// the order x (r2c) -> y -> z.Nhat.z^-1 -> y^-1 -> x^-1 (c2r), which on the [x][y][z][3] state
// layout makes every pass coalesced without any transposition and puts the
// shortest transforms on the largest (fully padded) data.  See DESIGN.md section 5.
#pragma once
#include "mm_common.cuh"

namespace mm {

struct FastGeom {
  int nx, ny, nz;
  int nzt;         // the z transform runs at period Pz = 2 nzt, nzt >= nz (fast_z_transform)
  int Px, Py, Pz;  // 2 nx, 2 ny, 2 nzt
  int Q;           // complex columns per (kx, y) row: 3 nz
};

// true if the fast kernels cover this mesh (otherwise the generic path of demag_passes.cu runs)
bool fast_supported(int nx, int ny, int nz, size_t real_bytes);
// nzt of the K3 kernel that serves nz (0: none): 32 (ny a multiple of 4), 64, 128, 256 for the warp-per-pencil kernels of demag_fast.cu,
// which take any nz up to their capacity with the missing layers read as zero (the period 2 nzt >= 2 nz - 1
// gives the same linear convolution, reading Q27), or nz itself for the tile pass of demag_ztile.cu.
int fast_z_transform(int nz, size_t real_bytes, int ny);

template <typename T> struct FastBufs {
  const Cx<T>* Wx;        // Wx[q] = exp(-2 pi i q / Px), q < Px
  const Cx<T>* Wy;        // ... / Py
  const Cx<T>* Wz;        // ... / Pz
  const uint16_t* posx;   // shared-memory row (swizzled) of x frequency k in the K1/K5 tile, k < Px
  const uint16_t* posy;   // row of y frequency k in A2, k < Py
  const Cx<T>* T2x;       // two-stage plan of the x axis: T2x[bf K1 + k1] = exp(-2 pi i bf k1 / Px) (or unused)
  const Cx<T>* T2y;       // ... of the y axis
  const Cx<T>* T2z;       // ... of the z axis (tile pass of demag_ztile.cu; unused by the warp-per-pencil kernels)
  bool two_x, two_y;      // the axis runs the two-stage kernels of demag_fast2.cu (natural frequency order)
  const T* table;         // Nhat[kx <= nx][ky <= ny][6][ozp] (kz <= nz used), scaled by 1/(Px Py Pz), parity sign folded
  Cx<T>* A1;              // [nx + 1][ny][Q]
  Cx<T>* A2;              // [nx + 1][Py][Q]; ky rows in natural order (two-stage y pass) or in the three-stage
                          // plan's order (L = 1024; K3 finds row ky through posy)
};

// Enqueues K1..K5: H := scale * crop(IFFT(table . FFT(pad(m)))).
template <typename T>
cudaError_t demag_fast_launch(const FastGeom& g, const FastBufs<T>& b, const T* m, T* H, T scale,
                              cudaStream_t st, unsigned long long* launches, Prof* prof);

// Slab layout ("sharded into contiguous slabs along the x-axis", "all-to-all
// transpose"): R ranks, rank r owns the x planes [r nx/R, (r+1) nx/R) of m and H and the rows ky in [r rpr, (r+1) rpr)
// of the half spectrum, rpr = ceil((ny + 1) / R), held as S_r[ky - r rpr][x < nx][Q].  The y pass of a rank
// writes every spectrum row straight into the buffer of the rank that owns it, p[ky / rpr] (the transpose is the
// store; between GPUs these are peer pointers over NVLink), the inverse y pass gathers them the same way.
template <typename T> struct SlabView {
  Cx<T>* p[8];   // S_r of every rank
  int rpr;       // ky rows per rank
  int nx;        // x planes of the whole mesh
  int x0;        // first x plane of the launching rank
};
// which: 0 = forward y (r2c, pruned) of the x planes [sv.x0, sv.x0 + nxl) of m into the S buffers,
// 4 = inverse y (c2r, truncated) from the S buffers into the same planes of H.  Wt: two-stage table of length ny.
template <typename T>
cudaError_t slab_y_launch(int which, int ny, int nxl, int Q, const Cx<T>* Wt, const SlabView<T>& sv, const T* m, T* H,
                          T scale, cudaStream_t st);

// K3 (S3) on nk planes of b.A2 (g.ny mirror pairs of rows each) whose table planes start at k0; xm != 0: the
// rows of a plane are kx instead of ky (slab layout of demag_slab.cu).
template <typename T>
cudaError_t k3_launch(const FastGeom& g, const FastBufs<T>& b, int k0, int nk, int xm, cudaStream_t st);

// Two-stage strided passes (demag_fast2.cu).  which: 0 = K1 (x forward), 1 = K2 (y forward),
// 3 = K4 (y inverse), 4 = K5 (x inverse).
template <typename T>
cudaError_t strided2_launch(int which, const FastGeom& g, const FastBufs<T>& b, const T* m, T* H, T scale,
                            cudaStream_t st);
bool fast_two_stage(int L);                      // the two-stage kernels cover length L (both precisions)
void fast2_plan(int L, int* K1, int* K2);        // P = 2L = K1 K2 (plan2.cuh; 0, 0 if L has no plan)

// K2 / K4 with their tiles moved by 2D TMA boxes (demag_tma.cu); which: 1 = K2, 3 = K4.  Returns
// cudaErrorNotSupported when the driver entry point, the plan or the alignment is missing or MM_B200_TMA=0 is
// set: the caller then runs the LDG / STG kernels of demag_fast2.cu.
template <typename T>
cudaError_t strided_tma_launch(int which, const FastGeom& g, const FastBufs<T>& b, cudaStream_t st);
bool strided_tma_usable(int L, int Q, size_t real_bytes, int which);   // the box kernel of pass `which` will run for this length / row / precision
// K1 / K5 the same way; which: 0 = K1, 4 = K5 (m, H, scale as for strided2_launch).
template <typename T>
cudaError_t strided_tma_x_launch(int which, const FastGeom& g, const FastBufs<T>& b, const T* m, T* H, T scale,
                                 cudaStream_t st);
bool strided_tma_x_usable(int L, int ny, int Q, size_t real_bytes);
bool strided_tma3_x_usable(int ny, int Q, size_t real_bytes);   // K1 at L = 1024 (xf3_tma_kernel)

// Host helpers for the tables above (plan order of the fast kernels).
int fast_pos_logical(int L, int k);   // row of frequency k < 2L in the [even half | odd half] layout
int fast_swizzle(int L, int row);     // shared-memory row of logical row

}  // namespace mm
