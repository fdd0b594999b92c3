// =============================================================================================
// tpc_grid.cu -- step 1 of the hot path (BASELINE.json north_star (1)):
// sort the clusters of every (sector, pad row) into a (y, zeta) grid.
//
// A two-level counting sort whose random accesses all stay inside the L2:
//   k_bucket_hist     bin id of every cluster (R7 formula, fp32); a BUCKET is kBucketBins...
//                     consecutive bins (a few thousand clusters).  Per-block shared-memory
//                     histogram over the buckets, flushed with one atomic per non-empty bucket.
//   scan              bucket offsets.
//   k_part_scatter    cluster -> 16-byte record moved into the range of its PART (~sqrt(#buckets)
//                     consecutive buckets) of one temporary array; a tile of 4096 clusters is
//                     ranked in shared memory, staged there in destination order and written out
//                     as whole runs: one global atomic per (tile, part) instead of one per cluster.
//   k_bucket_scatter  the same step inside the parts: records of a part -> their buckets' ranges of
//                     the second temporary array.
//   k_bucket_sort     one block per bucket: counts the bucket's bins in shared memory, scans them
//                     (-> bin_first), places the records, and re-orders every bin holding >= 2
//                     clusters by original index, which turns the arrival order of the atomics
//                     into the STABLE order R7 asks for: the grid is bit-identical from run to
//                     run and equal to a stable sort by bin.  The bucket (~100 KB) stays in L2
//                     between the passes.
//
// Roofline: HBM streaming, 104 B per cluster + 4 B per bin.
// =============================================================================================
#include "tpc_common.cuh"
#include "tpc_scan.cuh"

namespace tpc {

namespace {

constexpr int kThreads = 256;
constexpr unsigned kFull = 0xffffffffu;
constexpr int64_t kSortCap = kMaxBuckets;    // one block per bucket: measured 2.62 -> 2.37 ms
constexpr int kHistThreads = 1024;  // the bucket histogram takes up to 192 KB of shared memory: one or two big blocks per SM
constexpr int kUnroll = 4;  // independent loads in flight per thread in the streaming passes

struct GridSmem {
  float ymax[kMaxRows];
  int32_t ny[kMaxRows];
  int32_t rowbase[kMaxRows];
};

__device__ __forceinline__ void load_grid_rows(GridSmem& sm, const Geo& g) {
  for (int r = threadIdx.x; r < g.s.nrows; r += blockDim.x) {
    sm.ymax[r] = g.row.ymax[r];
    sm.ny[r] = g.row.ny[r];
    sm.rowbase[r] = g.row.rowbase[r];
  }
}

// R7 bin id, fp32, one rounding per operation; *clamped is raised for zeta outside [z_lo, z_hi].
__device__ __forceinline__ int bin_of(const GridSmem& sm, const Scalars& sc, int sr, float yy, float zz, bool* clamped) {
  const int s = sector_of(sc, sr), r = sr - s * sc.nrows;  // callers pass valid sector_rows only
  const float zeta = (s < 18) ? zz : -zz;  // R2/R7: mirrored drift coordinate
  const int yb = clampbin((yy + sm.ymax[r]) * sc.inv_cy, sm.ny[r]);
  const int zb = clampbin((zeta - sc.z_lo) * sc.inv_cz, sc.nz);
  if (clamped) *clamped |= !(zeta >= sc.z_lo && zeta <= sc.z_hi);
  return s * sc.bins_per_sector + sm.rowbase[r] + zb * sm.ny[r] + yb;
}

// shared-memory index with one pad word per 32: conflict-free both for t*32+k and for random access
__device__ __forceinline__ int pad32(int j) { return j + (j >> 5); }

__global__ void __launch_bounds__(kHistThreads)
k_bucket_hist(const __grid_constant__ Geo g, int64_t n, int bucket_shift, int nbuckets, const float* __restrict__ y,
              const float* __restrict__ z, const int32_t* __restrict__ sector_row, int32_t* __restrict__ bucket_cnt,
              int32_t* __restrict__ ws_counters) {
  extern __shared__ int32_t hist[];  // [nbuckets + 1]
  __shared__ GridSmem sm;
  load_grid_rows(sm, g);
  for (int j = threadIdx.x; j <= nbuckets; j += kHistThreads) hist[j] = 0;
  __syncthreads();
  const Scalars& sc = g.s;
  const int sr_end = sc.nsec * sc.nrows;
  bool clamped = false, bad = false;
  // every block takes one contiguous slice of the input (the tail of the loop keeps the warp whole for match_any)
  const int64_t per = ((n + gridDim.x - 1) / gridDim.x + kHistThreads * kUnroll - 1) / (kHistThreads * kUnroll) * (kHistThreads * kUnroll);
  const int64_t lo = (int64_t)blockIdx.x * per, hi = lo + per < n ? lo + per : n;
  // a warp takes kUnroll x 32 consecutive clusters per iteration: all loads are issued before the first use
  for (int64_t i0 = lo + (int64_t)(threadIdx.x >> 5) * (32 * kUnroll); i0 < hi; i0 += (int64_t)kHistThreads * kUnroll) {
    int srv[kUnroll];
    float yv[kUnroll], zv[kUnroll];
#pragma unroll
    for (int j = 0; j < kUnroll; j++) {
      const int64_t i = i0 + j * 32 + (threadIdx.x & 31);
      srv[j] = i < hi ? __ldcs(sector_row + i) : 0;
      yv[j] = i < hi ? __ldcs(y + i) : 0.0f;
      zv[j] = i < hi ? __ldcs(z + i) : 0.0f;
    }
#pragma unroll
    for (int j = 0; j < kUnroll; j++) {
      // a sector_row outside [0, n_sectors * n_rows) names no grid bin: the cluster goes to the extra bucket
      // `nbuckets` behind the grid (no search ever reaches it) and a status bit is raised
      int bk = -1;
      if (i0 + j * 32 + (threadIdx.x & 31) < hi) {
        if ((unsigned)srv[j] < (unsigned)sr_end) bk = bin_of(sm, sc, srv[j], yv[j], zv[j], &clamped) >> bucket_shift;
        else { bk = nbuckets; bad = true; }
      }
      // inputs ordered by row put a whole warp in one bucket: one add of 32; otherwise shared-memory atomics
      // (same-address lanes are merged by the hardware)
      const int bk0 = __shfl_sync(kFull, bk, 0);
      if (__all_sync(kFull, bk == bk0)) {
        if (bk >= 0 && (threadIdx.x & 31) == 0) atomicAdd(hist + bk, 32);
      } else if (bk >= 0) {
        atomicAdd(hist + bk, 1);
      }
    }
  }
  __syncthreads();
  for (int j = threadIdx.x; j <= nbuckets; j += kHistThreads) {
    const int c = hist[j];
    if (c) atomicAdd(bucket_cnt + j, c);
  }
  if (__any_sync(kFull, clamped) && (threadIdx.x & 31) == 0) atomicOr(ws_counters + WC_STATUS, TPC_ST_Z_CLAMPED);
  if (__any_sync(kFull, bad) && (threadIdx.x & 31) == 0) atomicOr(ws_counters + WC_STATUS, TPC_ST_BAD_ROW);
}

// ---- two-pass scatter: global cursor atomics replaced by shared-memory ranks ----------------------------------------
// A PART is 2^part_shift consecutive buckets (about the square root of the bucket count).  k_part_scatter moves every
// cluster, as a 16-byte record, into its part's range; k_bucket_scatter moves the records of a part into their
// buckets' ranges.  Both rank the records of a 4096-element tile in shared memory and reserve one run per (tile,
// destination) with a single global atomic, so the global atomics drop from one per cluster to one per ~20 clusters and
// every run is written as consecutive records.  The order inside a bucket is arbitrary either way; k_bucket_sort's
// re-ordering by original index makes the grid the stable sort R7 asks for.
constexpr int kPartThreads = 512, kPartItems = 8, kPartTile = kPartThreads * kPartItems;
constexpr int kMaxParts = 1024;   // parts of the first pass (+ 1 for the bad-row bucket)
constexpr int kLocalCap = 2048;   // buckets a tile of the second pass can rank in shared memory (a tile straddling parts)

__device__ __forceinline__ int part_of(int bk, int part_shift, int nbuckets, int nparts) {
  return bk == nbuckets ? nparts : bk >> part_shift;
}

// shared-memory rank of a key inside the tile; a warp whose lanes all hold the same key (inputs ordered by row) takes
// one atomic for all of them
__device__ __forceinline__ int tile_rank(int32_t* cnt, int key, bool valid, int lane) {
  const int k0 = __shfl_sync(kFull, key, 0);
  if (__all_sync(kFull, valid && key == k0)) {
    int base = 0;
    if (lane == 0) base = atomicAdd(cnt + key, 32);
    return __shfl_sync(kFull, base, 0) + lane;
  }
  return valid ? atomicAdd(cnt + key, 1) : 0;
}

__global__ void k_scan_cursors(int nbuckets, int part_shift, int nparts, const int32_t* __restrict__ bucket_first,
                              int32_t* __restrict__ bucket_cursor, int32_t* __restrict__ part_cursor) {
  for (int j = blockIdx.x * blockDim.x + threadIdx.x; j <= nbuckets + 1; j += gridDim.x * blockDim.x) {
    bucket_cursor[j] = bucket_first[j];
    if (j <= nparts) {
      const int64_t b = (int64_t)j << part_shift;
      part_cursor[j] = bucket_first[b < nbuckets ? b : nbuckets];
    }
  }
}

// Shared state of one tile: counts per destination, their exclusive offsets inside the tile, and (global base of the
// run - offset inside the tile) so that staged position p goes to delta[dest] + p.
template <int NDEST>
struct TileSmem {
  GridSmem grid;
  int32_t cnt[NDEST];
  int32_t loc[NDEST];
  int32_t delta[NDEST];
  uint16_t dest[kPartTile];  // destination of every staged position
  int32_t scan[kPartThreads / 32 + 1];
};

// counts -> offsets inside the tile, one global atomic per non-empty destination; ndest <= NDEST (a multiple of kPartThreads)
template <int NDEST>
__device__ __forceinline__ void tile_reserve(TileSmem<NDEST>& sm, int ndest, int32_t* __restrict__ cursor) {
  constexpr int PER = NDEST / kPartThreads;
  const int tid = threadIdx.x;
  int c[PER], acc = 0;
#pragma unroll
  for (int k = 0; k < PER; k++) {
    const int j = tid * PER + k;
    c[k] = j < ndest ? sm.cnt[j] : 0;
    acc += c[k];
  }
  int total;
  int ex = block_excl_scan<int, kPartThreads>(acc, &total, sm.scan);
#pragma unroll
  for (int k = 0; k < PER; k++) {
    const int j = tid * PER + k;
    if (j < ndest) {
      sm.loc[j] = ex;
      if (c[k]) sm.delta[j] = atomicAdd(cursor + j, c[k]) - ex;
      ex += c[k];
    }
  }
}

__global__ void __launch_bounds__(kPartThreads, 2)
k_part_scatter(const __grid_constant__ Geo g, int64_t n, int bucket_shift, int part_shift, int nbuckets, int nparts,
               const float* __restrict__ y, const float* __restrict__ z, const int32_t* __restrict__ sector_row,
               int32_t* __restrict__ part_cursor, Rec* __restrict__ out) {
  extern __shared__ float4 stage[];  // [kPartTile]: the tile's records in destination order
  __shared__ TileSmem<kMaxParts + kPartThreads> sm;
  load_grid_rows(sm.grid, g);
  const Scalars& sc = g.s;
  const int sr_end = sc.nsec * sc.nrows;
  const int tid = threadIdx.x, lane = tid & 31;
  for (int64_t t0 = (int64_t)blockIdx.x * kPartTile; t0 < n; t0 += (int64_t)gridDim.x * kPartTile) {
    for (int j = tid; j <= nparts; j += kPartThreads) sm.cnt[j] = 0;
    __syncthreads();
    int srv[kPartItems];
    float yv[kPartItems], zv[kPartItems];
#pragma unroll
    for (int j = 0; j < kPartItems; j++) {
      const int64_t i = t0 + j * kPartThreads + tid;
      srv[j] = i < n ? __ldcs(sector_row + i) : 0;
      yv[j] = i < n ? __ldcs(y + i) : 0.0f;
      zv[j] = i < n ? __ldcs(z + i) : 0.0f;
    }
    int where[kPartItems];  // part << 13 | rank inside the tile (< 4096)
#pragma unroll
    for (int j = 0; j < kPartItems; j++) {
      const bool valid = t0 + j * kPartThreads + tid < n;
      int pt = 0;
      if (valid) {
        if ((unsigned)srv[j] < (unsigned)sr_end) {
          pt = part_of(bin_of(sm.grid, sc, srv[j], yv[j], zv[j], nullptr) >> bucket_shift, part_shift, nbuckets, nparts);
        } else {  // no such (sector, row): parked behind the grid with an impossible sector_row (see k_bucket_hist)
          pt = nparts;
          srv[j] = kBadRow;
        }
      }
      where[j] = (pt << 13) | tile_rank(sm.cnt, pt, valid, lane);
    }
    __syncthreads();
    tile_reserve(sm, nparts + 1, part_cursor);
    __syncthreads();
#pragma unroll
    for (int j = 0; j < kPartItems; j++) {
      const int64_t i = t0 + j * kPartThreads + tid;
      if (i < n) {
        const int pt = where[j] >> 13, p = sm.loc[pt] + (where[j] & 8191);
        stage[p] = make_float4(yv[j], zv[j], __int_as_float((int)i), __int_as_float(srv[j]));
        sm.dest[p] = (uint16_t)pt;
      }
    }
    __syncthreads();
    const int count = (int)(n - t0 < kPartTile ? n - t0 : kPartTile);
    for (int p = tid; p < count; p += kPartThreads) out[sm.delta[sm.dest[p]] + p] = stage[p];  // consecutive lanes, consecutive records
    __syncthreads();
  }
}

// Second pass: the runs of a tile all lie inside one part (a few MB, a handful of pages), so they are written straight
// from the registers (staging them as in the first pass was measured slower: 1.25 -> 1.45 ms).
__global__ void __launch_bounds__(kPartThreads, 2)
k_bucket_scatter(const __grid_constant__ Geo g, int64_t n, int bucket_shift, int part_shift, int nbuckets,
                  const Rec* __restrict__ in, int32_t* __restrict__ cursor, Rec* __restrict__ out) {
  __shared__ GridSmem sm;
  __shared__ int32_t cnt[kLocalCap];
  __shared__ int32_t s_min;
  load_grid_rows(sm, g);
  const Scalars& sc = g.s;
  const int tid = threadIdx.x, lane = tid & 31;
  for (int64_t t0 = (int64_t)blockIdx.x * kPartTile; t0 < n; t0 += (int64_t)gridDim.x * kPartTile) {
    for (int j = tid; j < kLocalCap; j += kPartThreads) cnt[j] = 0;
    if (tid == 0) s_min = 0x7fffffff;
    __syncthreads();
    Rec r[kPartItems];
    int bk[kPartItems];
    int mn = 0x7fffffff;
#pragma unroll
    for (int j = 0; j < kPartItems; j++) {
      const int64_t i = t0 + j * kPartThreads + tid;
      r[j] = in[i < n ? i : n - 1];
    }
#pragma unroll
    for (int j = 0; j < kPartItems; j++) {
      const int sr = rec_sr(r[j]);
      bk[j] = sr == kBadRow ? nbuckets : bin_of(sm, sc, sr, r[j].x, r[j].y, nullptr) >> bucket_shift;
      if (t0 + j * kPartThreads + tid < n && bk[j] < mn) mn = bk[j];
    }
    mn = __reduce_min_sync(kFull, mn);
    if (lane == 0) atomicMin(&s_min, mn);
    __syncthreads();
    const int b0 = (s_min >> part_shift) << part_shift;  // the records are ordered by part: the tile starts in this one
    int where[kPartItems];  // rank inside the tile; -1 - slot for a bucket beyond the tile's reach (a tile that straddles
                            // many small parts): that record takes a cursor atomic of its own
#pragma unroll
    for (int j = 0; j < kPartItems; j++) {
      const bool valid = t0 + j * kPartThreads + tid < n;
      const int loc = bk[j] - b0;
      const bool local = loc < kLocalCap;
      const int rk = tile_rank(cnt, local ? loc : 0, valid && local, lane);
      where[j] = (valid && !local) ? -1 - atomicAdd(cursor + bk[j], 1) : rk;
    }
    __syncthreads();
    for (int j = tid; j < kLocalCap; j += kPartThreads) {
      const int c = cnt[j];
      if (c) cnt[j] = atomicAdd(cursor + b0 + j, c);
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < kPartItems; j++)
      if (t0 + j * kPartThreads + tid < n) out[where[j] < 0 ? -1 - where[j] : cnt[bk[j] - b0] + where[j]] = r[j];
    __syncthreads();
  }
}

// One block per bucket (grid-stride).  cnt[] holds, in turn: bin counts, exclusive offsets, running cursors
// (= end offsets once every record is placed).
constexpr int kSortThreads = 512;

__global__ void __launch_bounds__(kSortThreads)
k_bucket_sort(const __grid_constant__ Geo g, int64_t n, int64_t nb, int bucket_shift, int nbuckets,
              const int32_t* __restrict__ bucket_first, const Rec* __restrict__ tmp, Rec* rec, int32_t* __restrict__ bin_first) {
  extern __shared__ int32_t cnt[];  // [pad32(bucket bins)]
  __shared__ GridSmem sm;
  __shared__ int32_t scan_sm[kSortThreads / 32 + 1];
  load_grid_rows(sm, g);
  const Scalars& sc = g.s;
  const int bbins = 1 << bucket_shift;
  const int per_thread = bbins / kSortThreads;  // bucket bins are a power of two >= 8192
  const int tid = threadIdx.x;
  for (int b = blockIdx.x; b < nbuckets; b += gridDim.x) {
    const int start = bucket_first[b], end = bucket_first[b + 1];
    const int64_t bin0 = (int64_t)b << bucket_shift;
    const int nbins = (int)((nb - bin0) < bbins ? (nb - bin0) : bbins);
    __syncthreads();  // previous bucket's re-ordering pass is done with cnt[]
    for (int j = tid; j < bbins; j += kSortThreads) cnt[pad32(j)] = 0;
    __syncthreads();
    for (int i0 = start + tid; i0 < end; i0 += kSortThreads * kUnroll) {
      Rec r[kUnroll];
#pragma unroll
      for (int j = 0; j < kUnroll; j++) {
        const int i = i0 + j * kSortThreads;
        r[j] = tmp[i < end ? i : end - 1];
      }
#pragma unroll
      for (int j = 0; j < kUnroll; j++)
        if (i0 + j * kSortThreads < end)
          atomicAdd(cnt + pad32(bin_of(sm, sc, rec_sr(r[j]), r[j].x, r[j].y, nullptr) - (int)bin0), 1);
    }
    __syncthreads();
    // exclusive scan over the bucket's bins, thread t owns bins [t*per_thread, (t+1)*per_thread)
    int acc = 0;
    for (int k = 0; k < per_thread; k++) acc += cnt[pad32(tid * per_thread + k)];
    int total;
    int ex = block_excl_scan<int, kSortThreads>(acc, &total, scan_sm);
    for (int k = 0; k < per_thread; k++) {
      const int j = tid * per_thread + k;
      const int c = cnt[pad32(j)];
      cnt[pad32(j)] = ex;
      ex += c;
    }
    __syncthreads();
    for (int j = tid; j < nbins; j += kSortThreads) bin_first[bin0 + j] = start + cnt[pad32(j)];  // coalesced
    if (b == nbuckets - 1 && tid == 0) bin_first[nb] = bucket_first[nbuckets];  // clusters of the grid (n minus the bad rows)
    __syncthreads();
    for (int i0 = start + tid; i0 < end; i0 += kSortThreads * kUnroll) {
      Rec r[kUnroll];
#pragma unroll
      for (int j = 0; j < kUnroll; j++) {
        const int i = i0 + j * kSortThreads;
        r[j] = tmp[i < end ? i : end - 1];
      }
#pragma unroll
      for (int j = 0; j < kUnroll; j++)
        if (i0 + j * kSortThreads < end) {
          const int pos = atomicAdd(cnt + pad32(bin_of(sm, sc, rec_sr(r[j]), r[j].x, r[j].y, nullptr) - (int)bin0), 1);
          rec[start + pos] = r[j];
        }
    }
    __syncthreads();  // the block's own global writes are visible to it from here on
    // bins with >= 2 clusters: insertion sort by original index (max occupancy seen on the configs: 17)
    for (int j = tid; j < nbins; j += kSortThreads) {
      const int a = start + (j ? cnt[pad32(j - 1)] : 0), e = start + cnt[pad32(j)];
      for (int i = a + 1; i < e; i++) {
        const Rec v = rec[i];
        const int vi = rec_idx(v);
        int q = i - 1;
        while (q >= a) {
          const Rec u = rec[q];
          if (rec_idx(u) <= vi) break;
          rec[q + 1] = u;
          q--;
        }
        rec[q + 1] = v;
      }
    }
  }
  // clusters without a valid (sector, row) keep their place behind the grid (order unspecified; no bin covers them)
  if (blockIdx.x == 0)
    for (int i = bucket_first[nbuckets] + tid; i < bucket_first[nbuckets + 1]; i += kSortThreads) rec[i] = tmp[i];
}

__global__ void __launch_bounds__(kThreads)
k_export_sorted(int64_t n, const Rec* __restrict__ rec, int32_t* __restrict__ sorted_idx) {
  for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < n; i += (int64_t)gridDim.x * kThreads)
    sorted_idx[i] = rec_idx(rec[i]);
}

}  // namespace

// bucket geometry: 8192 bins per bucket, doubled until at most kMaxBuckets buckets remain (nb <= 2^30)
static inline int bucket_shift_for(int64_t nb) {
  int sh = kBucketShift0;
  while (((nb + ((int64_t)1 << sh) - 1) >> sh) > kMaxBuckets) sh++;
  return sh;
}

cudaError_t launch_grid_build(const Geo& g, const Ws& w, const float* y, const float* z, const int32_t* sector_row,
                              cudaStream_t st) {
  const int64_t n = w.L.n, nb = w.L.nb;
  cudaError_t e;
  const int sh = bucket_shift_for(nb);
  const int nbuckets = (int)((nb + ((int64_t)1 << sh) - 1) >> sh);
  const size_t hist_smem = sizeof(int32_t) * (size_t)(nbuckets + 1);
  const size_t sort_smem = sizeof(int32_t) * (size_t)(((size_t)1 << sh) + ((size_t)1 << (sh - 5)) + 32);
  static bool attr_done_dev[kMaxDevices] = {false};  // function attributes are per device
  int dev = 0;
  if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
  bool& attr_done = attr_done_dev[dev < kMaxDevices ? dev : kMaxDevices - 1];
  if (!attr_done || dev >= kMaxDevices) {
    if ((e = cudaFuncSetAttribute(k_bucket_hist, cudaFuncAttributeMaxDynamicSharedMemorySize, (kMaxBuckets + 1) * 4)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_bucket_sort, cudaFuncAttributeMaxDynamicSharedMemorySize, (32768 + 1024 + 32) * 4)) != cudaSuccess)
      return e;
    if ((e = cudaFuncSetAttribute(k_part_scatter, cudaFuncAttributeMaxDynamicSharedMemorySize, kPartTile * 16)) != cudaSuccess) return e;
    attr_done = true;
  }
  if ((e = cudaMemsetAsync(w.counters, 0, sizeof(int32_t) * WC_N, st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(w.bucket_first, 0, sizeof(int32_t) * (size_t)(kMaxBuckets + 2), st)) != cudaSuccess) return e;
  if (n > 0)
    TPC_LAUNCH(KID_BUCKET_HIST, st,
               (k_bucket_hist<<<blocks_for(n, kHistThreads * 64, 148 * (hist_smem + 2048 <= 110000 ? 2 : 1)), kHistThreads,
                               hist_smem, st>>>(
                   g, n, sh, nbuckets, y, z, sector_row, w.bucket_first, w.counters)));
  // nbuckets grid buckets + the bucket of clusters without a valid (sector, row) + the total
  if ((e = exclusive_scan<int32_t>(w.bucket_first, w.bucket_first, nbuckets + 2, (int32_t*)w.scan_tmp, st)) != cudaSuccess) return e;
  // parts of 2^ps buckets: about the square root of the bucket count, at most kMaxParts
  int ps = 0;
  while (((int64_t)1 << (2 * ps)) < nbuckets || ((nbuckets + (1 << ps) - 1) >> ps) > kMaxParts) ps++;
  const int nparts = (nbuckets + (1 << ps) - 1) >> ps;
  int32_t* part_cursor = w.bucket_cursor + kMaxBuckets + 2;
  TPC_LAUNCH(KID_SCAN, st,
             (k_scan_cursors<<<blocks_for(nbuckets + 2, 256, 64), 256, 0, st>>>(nbuckets, ps, nparts, w.bucket_first, w.bucket_cursor,
                                                                                part_cursor)));
  if (n > 0) {
    TPC_LAUNCH(KID_PART_SCATTER, st,
               (k_part_scatter<<<blocks_for(n, kPartTile, 148 * 64), kPartThreads, kPartTile * 16, st>>>(g, n, sh, ps, nbuckets, nparts, y, z, sector_row,
                                                                                            part_cursor, w.rec)));
    TPC_LAUNCH(KID_BUCKET_SCATTER, st,
               (k_bucket_scatter<<<blocks_for(n, kPartTile, 148 * 64), kPartThreads, 0, st>>>(g, n, sh, ps, nbuckets, w.rec, w.bucket_cursor,
                                                                                               (Rec*)w.hit_rec)));
  }
  TPC_LAUNCH(KID_BUCKET_SORT, st,
             (k_bucket_sort<<<blocks_for(nbuckets, 1, kSortCap), kSortThreads, sort_smem, st>>>(
                 g, n, nb, sh, nbuckets, w.bucket_first, (const Rec*)w.hit_rec, w.rec, w.bin_first)));
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
