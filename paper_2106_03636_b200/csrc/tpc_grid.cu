// =============================================================================================
// tpc_grid.cu -- step 1 of the hot path (BASELINE.json north_star (1)):
// sort the clusters of every (sector, pad row) into a (y, zeta) grid.
//
//   k_bin_count   one thread per cluster: bin id (R7 formula, fp32), rank = atomicAdd(count[bin])
//   exclusive scan of the counts -> bin_first   (tpc_scan.cuh)
//   k_scatter     cluster -> 16-byte record at bin_first[bin] + rank
//   k_canon       bins holding >= 2 clusters are re-ordered by original index, which turns the
//                 arrival-order ranks of the atomics into the STABLE order R7 asks for, so the
//                 grid is bit-identical from run to run and equal to a stable sort by bin.
//
// Roofline: HBM-bound streaming + one random 4-byte atomic and one random 16-byte store per
// cluster.
// =============================================================================================
#include "tpc_common.cuh"
#include "tpc_scan.cuh"

namespace tpc {

namespace {

constexpr int kThreads = 256;

struct GridSmem {
  float ymax[kMaxRows];
  int32_t ny[kMaxRows];
  int32_t rowbase[kMaxRows];
};

__global__ void __launch_bounds__(kThreads)
k_bin_count(const __grid_constant__ Geo g, int64_t n, const float* __restrict__ y, const float* __restrict__ z,
            const int32_t* __restrict__ sector_row, int32_t* __restrict__ key, int32_t* __restrict__ rank,
            int32_t* __restrict__ count, int32_t* __restrict__ ws_counters) {
  __shared__ GridSmem sm;
  for (int r = threadIdx.x; r < g.s.nrows; r += kThreads) {
    sm.ymax[r] = g.row.ymax[r];
    sm.ny[r] = g.row.ny[r];
    sm.rowbase[r] = g.row.rowbase[r];
  }
  __syncthreads();
  const int nrows = g.s.nrows;
  const float inv_cy = g.s.inv_cy, inv_cz = g.s.inv_cz, z_lo = g.s.z_lo, z_hi = g.s.z_hi;
  const int nz = g.s.nz, bps = g.s.bins_per_sector;
  bool clamped = false;
  for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < n; i += (int64_t)gridDim.x * kThreads) {
    const int sr = sector_row[i];
    const int s = sr / nrows, r = sr - s * nrows;
    const float yy = y[i];
    const float zeta = (s < 18) ? z[i] : -z[i];  // R2/R7: mirrored drift coordinate
    const int yb = clampbin((yy + sm.ymax[r]) * inv_cy, sm.ny[r]);
    const int zb = clampbin((zeta - z_lo) * inv_cz, nz);
    clamped |= !(zeta >= z_lo && zeta <= z_hi);
    const int b = s * bps + sm.rowbase[r] + zb * sm.ny[r] + yb;
    key[i] = b;
    rank[i] = atomicAdd(count + b, 1);
  }
  if (__any_sync(0xffffffffu, clamped) && (threadIdx.x & 31) == 0) atomicOr(ws_counters + WC_STATUS, TPC_ST_Z_CLAMPED);
}

__global__ void __launch_bounds__(kThreads)
k_scatter(int64_t n, const float* __restrict__ y, const float* __restrict__ z, const int32_t* __restrict__ sector_row,
          const int32_t* __restrict__ key, const int32_t* __restrict__ rank, const int32_t* __restrict__ bin_first,
          Rec* __restrict__ rec) {
  for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < n; i += (int64_t)gridDim.x * kThreads) {
    const int pos = __ldg(bin_first + key[i]) + rank[i];
    rec[pos] = make_float4(y[i], z[i], __int_as_float((int)i), __int_as_float(sector_row[i]));
  }
}

// One thread per bin; bins with fewer than two clusters (the vast majority, mean occupancy ~1) cost two
// coalesced loads.  Insertion sort by original index (max occupancy seen on the configs: 17).
__global__ void __launch_bounds__(kThreads)
k_canon(int64_t nb, const int32_t* __restrict__ bin_first, Rec* __restrict__ rec) {
  for (int64_t b = (int64_t)blockIdx.x * kThreads + threadIdx.x; b < nb; b += (int64_t)gridDim.x * kThreads) {
    const int a = bin_first[b], e = bin_first[b + 1];
    for (int i = a + 1; i < e; i++) {
      const Rec v = rec[i];
      const int vi = rec_idx(v);
      int j = i - 1;
      while (j >= a) {
        const Rec u = rec[j];
        if (rec_idx(u) <= vi) break;
        rec[j + 1] = u;
        j--;
      }
      rec[j + 1] = v;
    }
  }
}

__global__ void __launch_bounds__(kThreads)
k_export_sorted(int64_t n, const Rec* __restrict__ rec, int32_t* __restrict__ sorted_idx) {
  for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < n; i += (int64_t)gridDim.x * kThreads)
    sorted_idx[i] = rec_idx(rec[i]);
}

}  // namespace

cudaError_t launch_grid_build(const Geo& g, const Ws& w, const float* y, const float* z, const int32_t* sector_row,
                              cudaStream_t st) {
  const int64_t n = w.L.n, nb = w.L.nb;
  cudaError_t e;
  if ((e = cudaMemsetAsync(w.counters, 0, sizeof(int32_t) * WC_N, st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(w.bin_first, 0, sizeof(int32_t) * (size_t)(nb + 2), st)) != cudaSuccess) return e;
  if (n > 0) {
    TPC_LAUNCH(KID_BIN_COUNT, st,
               (k_bin_count<<<blocks_for(n, kThreads), kThreads, 0, st>>>(g, n, y, z, sector_row, w.key, w.rank,
                                                                         w.bin_first, w.counters)));
  }
  if ((e = exclusive_scan<int32_t>(w.bin_first, w.bin_first, nb + 1, (int32_t*)w.scan_tmp, st)) != cudaSuccess) return e;
  if (n > 0) {
    TPC_LAUNCH(KID_SCATTER, st,
               (k_scatter<<<blocks_for(n, kThreads), kThreads, 0, st>>>(n, y, z, sector_row, w.key, w.rank, w.bin_first,
                                                                       w.rec)));
    TPC_LAUNCH(KID_CANON, st, (k_canon<<<blocks_for(nb, kThreads), kThreads, 0, st>>>(nb, w.bin_first, w.rec)));
  }
  return cudaGetLastError();
}

cudaError_t launch_grid_export(const Ws& w, int32_t* sorted_idx, int32_t* bin_first, cudaStream_t st) {
  cudaError_t e;
  if (sorted_idx && w.L.n > 0)
    TPC_LAUNCH(KID_EXPORT, st,
               (k_export_sorted<<<blocks_for(w.L.n, kThreads), kThreads, 0, st>>>(w.L.n, w.rec, sorted_idx)));
  if (bin_first)
    if ((e = cudaMemcpyAsync(bin_first, w.bin_first, sizeof(int32_t) * (size_t)(w.L.nb + 1), cudaMemcpyDeviceToDevice,
                             st)) != cudaSuccess)
      return e;
  return cudaGetLastError();
}

}  // namespace tpc
