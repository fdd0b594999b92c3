// =============================================================================================
// tpc_search.cuh -- per-row geometry staged in shared memory and the grid window lookup shared by
// the neighbour finder (R9) and the follower's extrapolation search (R16).
//
// R8: the grid is only an acceleration structure.  bin_window() returns a SUPERSET of the bins
// that cover a cm window; every candidate is re-tested against the exact window by the caller,
// so results do not depend on the cell size.
// =============================================================================================
#pragma once
#include "tpc_common.cuh"

namespace tpc {

struct SmRow {
  float X[kMaxRows];
  float ymax[kMaxRows];
  int32_t ny[kMaxRows];
  int32_t rowbase[kMaxRows];
};

__device__ __forceinline__ void load_rows(SmRow& sm, const Geo& g) {
  for (int r = threadIdx.x; r < g.s.nrows; r += blockDim.x) {
    sm.X[r] = g.row.X[r];
    sm.ymax[r] = g.row.ymax[r];
    sm.ny[r] = g.row.ny[r];
    sm.rowbase[r] = g.row.rowbase[r];
  }
}

// Bins of (sector s, row r) that cover the cm window [ya,yb] x [za,zb] (raw z).  The pads dominate
// fp32 rounding of the window edges (|y| < 50 cm: ulp 4e-6; |z| <= 3.3e4 cm: ulp 4e-3).
struct BinWin {
  int first;  // bin index of (zb0, yb0)
  int ny, ybspan, nzb;
};

__device__ __forceinline__ BinWin bin_window(const SmRow& sm, const Scalars& sc, int s, int r, float ya, float yb,
                                             float za, float zb) {
  const float py = 0.002f;
  const float pz = 0.02f + 1e-6f * fmaxf(fabsf(za), fabsf(zb));
  float z0, z1;
  if (s < 18) {
    z0 = za - pz;
    z1 = zb + pz;
  } else {
    z0 = -(zb + pz);
    z1 = -(za - pz);
  }
  const int ny = sm.ny[r];
  const int zb0 = clampbin((z0 - sc.z_lo) * sc.inv_cz, sc.nz);
  const int zb1 = clampbin((z1 - sc.z_lo) * sc.inv_cz, sc.nz);
  const int yb0 = clampbin(((ya - py) + sm.ymax[r]) * sc.inv_cy, ny);
  const int yb1 = clampbin(((yb + py) + sm.ymax[r]) * sc.inv_cy, ny);
  BinWin w;
  w.ny = ny;
  w.first = s * sc.bins_per_sector + sm.rowbase[r] + zb0 * ny + yb0;
  w.ybspan = yb1 - yb0 + 1;
  w.nzb = zb1 - zb0 + 1;
  return w;
}

}  // namespace tpc
