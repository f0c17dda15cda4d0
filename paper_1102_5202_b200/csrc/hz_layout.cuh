// hz_layout.cuh -- how the resident fields sit in HBM.
//
// Structure of arrays: one padded 3D array per grid function, x fastest, with
// NG ghost layers on every active side.  Rows are `pitch` elements long with the first INTERIOR
// element of every row on a 128-byte boundary, so a warp reading 32 consecutive interior cells
// touches the minimum number of sectors.  All fields of one set (9 primitives, 10 metric
// components, ...) share one allocation and are `fs` elements apart.
#pragma once
#include <cstddef>

namespace hz {

// Boundary kind of one side of an axis (side 0 = low, 1 = high) from the per-axis code of hz_grid.bc:
// 0 periodic, 1 outflow (zero gradient), 2 external (ghost layers are supplied through hz_halo_unpack;
// only the z axis may be external).  Codes 3 / 4: external on the low / high side only, outflow on the other.
__host__ __device__ inline int bc_side(int bc, int side) {
  if (bc <= 2) return bc;
  if (bc == 3) return side == 0 ? 2 : 1;
  return side == 0 ? 1 : 2;
}

struct Layout {
  int n[3];        // interior cells per axis
  int ng;          // ghost layers of an active axis: 2 (MC) or 3 (PPM)
  int g[3];        // ghost layers per side (ng on active axes, 0 on one-cell axes)
  int N[3];        // padded logical extent n + 2g
  int ox;          // x offset of interior cell 0 inside a row
  int pitch;       // row length in elements
  long long sz;    // plane stride = pitch*N[1]
  long long fs;    // field stride (elements)
  double h[3];     // spacings
  int bc[3];

  __host__ __device__ long long idx(int i, int j, int k) const {
    return (long long)(k + g[2]) * sz + (long long)(j + g[1]) * pitch + (i + ox);
  }
  __host__ __device__ long long stride(int d) const { return d == 0 ? 1 : (d == 1 ? (long long)pitch : sz); }
  __host__ __device__ long long ncell() const { return (long long)n[0] * n[1] * n[2]; }
};

}  // namespace hz
