// =============================================================================================
// tpc_common.cuh -- device-side geometry tables, workspace layout and small helpers shared by the
// kernels of libtpc_b200.so (grid, find, fit).  Product code: shares nothing with oracle/.
//
// Geometry and conventions follow SURVEY.md §8(c) R1-R7 (restated in DESIGN.md "Readings"):
//   R1 rows at sector-local x = row_x[r], |y| <= row_x[r]*tan_half
//   R2 sectors 0..17 side +1, 18..35 side -1; the grid's drift axis is zeta = side*z
//   R7 per (sector,row): ny_r = max(1, ceil(2 ymax_r / cell_y)), nz = ceil((z_hi-z_lo)/cell_z),
//      bin = zbin*ny_r + ybin (z-major), all fp32, one rounding per operation
// =============================================================================================
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tpc_b200.h"

namespace tpc {

constexpr int kMaxRows = TPC_MAX_ROWS;

// Per-row geometry needed by every search (R1, R7).  Passed to kernels by value (__grid_constant__)
// and staged into shared memory by each block, because rows differ across the lanes of a warp.
struct RowGeo {
  float X[kMaxRows];       // pad-row x
  float ymax[kMaxRows];    // X*tan_half
  int32_t ny[kMaxRows];    // y bins of the row
  int32_t rowbase[kMaxRows + 1];  // first bin of row r inside a sector; [n_rows] = bins per sector
};

// Per-row constants of the cellular-automaton neighbour finder (R9).
struct CaGeo {
  float wu[kMaxRows];    // weight of the upper neighbour in the 3-point interpolation
  float iy[kMaxRows];    // 1/(sigma_y^2 (1+wu^2+wd^2))
  float iz[kMaxRows];    // 1/(sigma_z^2 (1+wu^2+wd^2))
  float wyu[kMaxRows], wzu[kMaxRows];  // search half-window towards row r+1
  float wyd[kMaxRows], wzd[kMaxRows];  // search half-window towards row r-1
};

// Scalars (R4, R6, R7, R9-R22).
struct Scalars {
  int32_t nsec, nrows, nz, bins_per_sector;
  uint32_t rows_magic;  // ceil(2^32 / nrows): sector = umulhi(sector_row, rows_magic), exact for sector_row < 2^24
  int32_t slab_w, nslab;  // tracklet ordering: z slabs of slab_w bins, nslab = ceil(nz / slab_w)
  float inv_cy, inv_cz, z_lo, z_hi;
  float kB, sy2, sz2, sig_y, sig_z;
  float ca_cut, chi2_cut, chi2_chain_cut, win_max, max_sinphi, edge_margin;
  int32_t max_gap, min_hits, n_fit_passes;
  float cov0[5];
};

struct Geo {
  Scalars s;
  RowGeo row;
  CaGeo ca;
};

// Internal device counters (int32) at the head of the workspace.
enum {
  WC_N_STARTS = 0,     // tracklets to follow (clamped)
  WC_QUEUE = 1,        // work-queue head of the follower
  WC_STATUS = 2,       // TPC_ST_* bits
  WC_STARTS_FOUND = 3, // before clamping
  WC_FIT_QUEUE = 4,    // work-queue head of the cached refit
  WC_QUEUE_B = 5,      // work-queue head of the follower's phase B
  WC_N_SURV = 6,       // tracklets that go on to phase B (start hit not picked up by an upward leg, R17)
  WC_N_WAVE = 7,       // tracklets of the current phase-A wave (R17)
  WC_PROP64 = 8,       // unsigned long long at [8,9]: follower transports
  WC_UPD64 = 10,       // unsigned long long at [10,11]: follower updates
  WC_CAND64 = 12,      // unsigned long long at [12,13]: candidates tested
  WC_CLAIMS64 = 14,    // unsigned long long at [14,15]: hits recorded by the tracklets that finished phase B
  WC_N = 16
};

// Sorted 16-byte cluster record: one LDG.128 brings everything a candidate test needs.
//   .x = y, .y = z (raw, not mirrored), .z = original index (int bits), .w = sector_row (int bits)
using Rec = float4;

// Workspace layout: a pure function of (n, max_tracklets, n_bins).  All offsets 256-byte aligned.
struct Layout {
  int64_t n, scap, scap_pad, nb, nchunks;
  int64_t scan_tiles;  // capacity (elements) of the scan scratch
  size_t off_counters, off_rec, off_key, off_bucket_first, off_bucket_cursor, off_bin_first, off_link_up, off_link_dn, off_up_c,
      off_owner, off_hit_rec, off_tl_init, off_tl_info, off_tl_key, off_tl_mask, off_tl_scan, off_row_hit,
      off_tl_state, off_surv, off_surv_scan, off_picked, off_chunk_base, off_chunk_scan0, off_scan_tmp, total;
};

// R20 selection key, 64 bits: [63:56] nHits | [55:25] 0x7FFFFFFF - original index of the start hit |
// [24:0] tracklet number t.  (nHits, start index) is unique per tracklet, so the low field never
// decides a comparison: max(key) = most hits, ties to the lowest original start index, as R20 asks;
// t makes the key of a tracklet unique even among tracklets dropped for capacity and names the owner in a dump.
constexpr int kKeyTBits = 25;
constexpr int64_t kMaxTracklets = (int64_t)1 << kKeyTBits;  // 33,554,432
constexpr int kMaxBuckets = 49152;   // grid build: first-level buckets of the counting sort (their histogram fits shared memory)
constexpr int kBucketShift0 = 13;    // ... of at least 2^13 bins each  // grid build: first-level buckets of the counting sort
constexpr int kStateVec = 6;    // float4 per tracklet of follower state carried from phase A to phase B (24 words)
constexpr int kStartBit = 1 << 30;  // rec.w: set on start hits by k_compact_starts (read by the upward legs, R17)
constexpr int kBadRow = kStartBit - 1;  // rec.w of a cluster whose sector_row names no (sector, row): parked behind the grid
constexpr int kMaxDevices = 64;     // per-device caches of function attributes / occupancy (one entry per CUDA device)
constexpr int kMaskWords = 5;  // kept-row mask per tracklet (rows 0..159)

// Start record of a tracklet (R14 inputs), written by k_compact_starts: one 32-byte load in the follower.
struct TlInit {
  float y0, z0, y1, z1;       // start hit and its cleaned up-neighbour
  int32_t p0, p1, sr0, orig0; // grid positions, sector_row and original index of the start hit
};

constexpr int kScanTile = 4096;  // elements per scan tile (256 threads x 16)

inline size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }

inline Layout make_layout(int64_t n, int64_t scap, int64_t nb, int nrows, int64_t nchunks) {
  Layout L{};
  L.n = n;
  L.scap = scap;
  L.scap_pad = (scap + 31) & ~(int64_t)31;
  L.nb = nb;
  L.nchunks = nchunks;
  int64_t longest = nb + 1;
  if (nchunks + 1 > longest) longest = nchunks + 1;
  if (n + 1 > longest) longest = n + 1;
  if (scap + 1 > longest) longest = scap + 1;
  L.scan_tiles = (longest + kScanTile - 1) / kScanTile + 2;
  size_t o = 0;
  auto take = [&](size_t bytes) {
    size_t at = o;
    o = align256(o + bytes);
    return at;
  };
  L.off_counters = take(sizeof(int32_t) * WC_N);
  L.off_rec = take(sizeof(Rec) * (size_t)(n + 1));
  L.off_key = take(sizeof(int32_t) * (size_t)(n + 1));      // start-hit flags and their scan (R10)
  L.off_bucket_first = take(sizeof(int32_t) * (size_t)(kMaxBuckets + 2));
  L.off_bucket_cursor = take(sizeof(int32_t) * (size_t)(kMaxBuckets + 2 + 1024 + 2));  // + the part cursors of the grid build
  L.off_bin_first = take(sizeof(int32_t) * (size_t)(nb + 2));
  L.off_link_up = take(sizeof(int32_t) * (size_t)(n + 1));
  L.off_link_dn = take(sizeof(int32_t) * (size_t)(n + 1));
  L.off_up_c = take(sizeof(int32_t) * (size_t)(n + 1));
  L.off_owner = take(sizeof(uint64_t) * (size_t)(n + 1));
  L.off_hit_rec = take(sizeof(float4) * (size_t)(n + 1));   // (y, z, row, orig) in hit-list order for the refit
  L.off_tl_init = take(sizeof(TlInit) * (size_t)(L.scap_pad + 1));
  L.off_tl_info = take(sizeof(int32_t) * (size_t)(L.scap_pad + 1));
  L.off_tl_key = take(sizeof(uint64_t) * (size_t)(L.scap_pad + 1));
  L.off_tl_mask = take(sizeof(uint32_t) * kMaskWords * (size_t)(L.scap_pad + 1));
  L.off_tl_scan = take(sizeof(int64_t) * (size_t)(L.scap_pad + 2));
  L.off_row_hit = take(sizeof(int32_t) * (size_t)L.scap_pad * (size_t)nrows);  // [t][row], tracklet-major
  L.off_tl_state = take(sizeof(float4) * kStateVec * (size_t)(L.scap_pad + 1));  // follower state between phases A and B
  L.off_surv = take(sizeof(int32_t) * (size_t)(L.scap_pad + 2));
  L.off_surv_scan = take(sizeof(int32_t) * (size_t)(L.scap_pad + 2));
  L.off_picked = take((size_t)(n + 256));  // one byte per cluster: attached by some upward leg (R17)
  L.off_chunk_base = take(sizeof(int32_t) * (size_t)(nchunks + 2));   // tracklets before chunk (sector, slab, row)
  L.off_chunk_scan0 = take(sizeof(int32_t) * (size_t)(nchunks + 2));  // grid-order start count at the chunk's first cluster
  L.off_scan_tmp = take(sizeof(int64_t) * (size_t)L.scan_tiles);
  L.total = o;
  return L;
}


// Typed view of a workspace.
struct Ws {
  Layout L;
  int32_t* counters;
  Rec* rec;
  int32_t *key, *bucket_first, *bucket_cursor, *bin_first, *link_up, *link_dn, *up_c;
  unsigned long long* owner;
  float4* hit_rec;
  TlInit* tl_init;
  int32_t* tl_info;
  unsigned long long* tl_key;
  uint32_t* tl_mask;
  long long* tl_scan;
  int32_t* row_hit;
  int32_t *chunk_base, *chunk_scan0;
  float4* tl_state;
  int32_t *surv, *surv_scan;
  uint8_t* picked;
  long long* scan_tmp;
};

inline Ws bind_ws(const Layout& L, void* workspace) {
  char* b = (char*)workspace;
  Ws w;
  w.L = L;
  w.counters = (int32_t*)(b + L.off_counters);
  w.rec = (Rec*)(b + L.off_rec);
  w.key = (int32_t*)(b + L.off_key);
  w.bucket_first = (int32_t*)(b + L.off_bucket_first);
  w.bucket_cursor = (int32_t*)(b + L.off_bucket_cursor);
  w.bin_first = (int32_t*)(b + L.off_bin_first);
  w.link_up = (int32_t*)(b + L.off_link_up);
  w.link_dn = (int32_t*)(b + L.off_link_dn);
  w.up_c = (int32_t*)(b + L.off_up_c);
  w.owner = (unsigned long long*)(b + L.off_owner);
  w.hit_rec = (float4*)(b + L.off_hit_rec);
  w.tl_init = (TlInit*)(b + L.off_tl_init);
  w.tl_info = (int32_t*)(b + L.off_tl_info);
  w.tl_key = (unsigned long long*)(b + L.off_tl_key);
  w.tl_mask = (uint32_t*)(b + L.off_tl_mask);
  w.tl_scan = (long long*)(b + L.off_tl_scan);
  w.row_hit = (int32_t*)(b + L.off_row_hit);
  w.tl_state = (float4*)(b + L.off_tl_state);
  w.surv = (int32_t*)(b + L.off_surv);
  w.surv_scan = (int32_t*)(b + L.off_surv_scan);
  w.picked = (uint8_t*)(b + L.off_picked);
  w.chunk_base = (int32_t*)(b + L.off_chunk_base);
  w.chunk_scan0 = (int32_t*)(b + L.off_chunk_scan0);
  w.scan_tmp = (long long*)(b + L.off_scan_tmp);
  return w;
}

// Host launchers implemented in tpc_grid.cu / tpc_find.cu / tpc_fit.cu (each only enqueues).
cudaError_t launch_grid_build(const Geo& g, const Ws& w, const float* y, const float* z, const int32_t* sector_row,
                              cudaStream_t st);
cudaError_t launch_grid_export(const Ws& w, int32_t* sorted_idx, int32_t* bin_first, cudaStream_t st);
cudaError_t launch_find(const Geo& g, const Ws& w, int32_t* cluster_track, int64_t max_tracks, int32_t* trk_seed,
                        int32_t* trk_sector, int32_t* trk_nhits, int64_t* trk_first_hit, int32_t* trk_hits,
                        int32_t* counters, cudaStream_t st);
cudaError_t launch_find_export(const Geo& g, const Ws& w, int32_t* link_up, int32_t* link_dn, int32_t* up_c,
                               int32_t* dn_c, int32_t* starts, int32_t* tl_nhits, int32_t* row_hit, cudaStream_t st);
// follower (tpc_follow.cu) and selection (tpc_select.cu) stages of launch_find
cudaError_t launch_follow(const Geo& g, const Ws& w, cudaStream_t st);
cudaError_t launch_select(const Geo& g, const Ws& w, int32_t* cluster_track, int64_t max_tracks, int32_t* trk_seed,
                          int32_t* trk_sector, int32_t* trk_nhits, int64_t* trk_first_hit, int32_t* trk_hits,
                          int32_t* counters, cudaStream_t st);
// w == nullptr: gather the hits through y / z / sector_row; else read the records tpc_find_tracks cached in w
cudaError_t launch_fit(const Geo& g, const Ws* w, int64_t n, const float* y, const float* z, const int32_t* sector_row,
                       const int32_t* counters, int64_t max_tracks, const int32_t* trk_nhits,
                       const int64_t* trk_first_hit, const int32_t* trk_hits, float* par, float* cov, float* xref,
                       float* zref, float* chi2, int32_t* ndf, cudaStream_t st);

cudaError_t launch_track_time(const Geo& g, double v_drift, const int32_t* counters, int64_t max_tracks,
                              const int32_t* trk_sector, const float* par, const float* xref, const float* zref, float* phi0,
                              float* z0, float* dca, float* t0, cudaStream_t st);

// tpc_merge.cu (R26)
size_t merge_ws_bytes(const Geo& g, int64_t max_tracks);
cudaError_t launch_merge(const Geo& g, const Ws& fw, float chi2_cut, float dz_max, float ce_tol, int max_rows,
                         const int32_t* counters, int64_t max_tracks, const int32_t* trk_seed, const int32_t* trk_sector,
                         const int32_t* trk_nhits, const int64_t* trk_first_hit, const float* par, const float* cov,
                         const float* xref, const float* zref, const float* chi2, const int32_t* ndf, void* merge_ws,
                         int32_t* trk_succ, int32_t* trk_pred, float* trk_succ_chi2, int32_t* trk_global, int32_t* n_global,
                         int32_t* g_head, int32_t* g_nseg, int32_t* g_nhits, float* gpar, float* gcov, float* gxref,
                         float* gzref, float* gchi2, int32_t* gndf, cudaStream_t st);

// tpc_api.cu: records the text of a failed CUDA call for tpc_last_cuda_error and returns TPC_ECUDA
int report_cuda_error(cudaError_t e);

size_t pair_sides_ws_bytes(int64_t max_collisions);
cudaError_t launch_pair_sides(const int32_t* n_a, const float* t_a, const int32_t* c_a, const int32_t* n_c, const float* t_c,
                              const int32_t* c_c, int64_t max_collisions, double dt_max, double sigma_t, double v_drift,
                              void* workspace, int32_t* pair_of_a, int32_t* pair_of_c, float* t_out, float* zv_out,
                              int32_t* n_pairs, cudaStream_t st);

// tpc_fit.cu (R28)
cudaError_t launch_fit_physics(const Geo& g, const tpc_fit_options_t& opt, const Ws* w, const float* y, const float* z,
                               const int32_t* sector_row, const int32_t* counters, int64_t max_tracks, const int32_t* trk_nhits,
                               const int64_t* trk_first_hit, const int32_t* trk_hits, const float* trk_t0, float* par, float* cov,
                               float* xref, float* zref, float* chi2, int32_t* ndf, uint8_t* hit_flag, cudaStream_t st);
cudaError_t launch_tag_clusters(int64_t n, const int32_t* cluster_track, const int32_t* counters, int64_t max_tracks,
                                const float* par, const int32_t* ndf, const int32_t* trk_hits, const uint8_t* hit_flag,
                                double qpt_max, uint8_t* tag, cudaStream_t st);

// tpc_cluster.cu (R27)
size_t cluster_ws_bytes(int64_t n_digits);
cudaError_t launch_clusterize(const Geo& g, int64_t n, const int32_t* sr, const int32_t* pad, const int32_t* tim,
                              const int32_t* adc, float pad_width, float time_width, int peak_min, void* workspace,
                              int64_t max_clusters, float* y, float* z, float* q, int32_t* out_sr, int32_t* out_pad,
                              int32_t* out_time, int32_t* n_clusters, cudaStream_t st);

size_t collisions_ws_bytes(int64_t nb, int64_t max_tracks);
cudaError_t launch_collisions(const int32_t* counters, int64_t max_tracks, const float* t0, const float* dca,
                              const int32_t* trk_sector, int side_sel, double t_lo,
                              double w, int64_t nb, double dca_max, int32_t n_min, void* workspace, int64_t max_collisions,
                              float* coll_time, int32_t* coll_ntracks, int32_t* coll_bin, int32_t* trk_collision,
                              int32_t* n_collisions, cudaStream_t st);

// ---- device helpers -------------------------------------------------------------------------
// R7: clamp-to-range binning; NaN and negatives go to bin 0.
__device__ __forceinline__ int clampbin(float v, int n) {
  if (!(v > 0.0f)) return 0;
  if (v >= (float)n) return n - 1;
  return (int)v;
}

__device__ __forceinline__ Rec ld_rec(const Rec* __restrict__ recs, int k) { return __ldg(recs + k); }
__device__ __forceinline__ int rec_idx(const Rec& r) { return __float_as_int(r.z); }
__device__ __forceinline__ int rec_sr(const Rec& r) { return __float_as_int(r.w) & (kStartBit - 1); }
// sector of a VALID sector_row (0 <= sr < nsec * nrows <= 2^24): sr / nrows without the integer division
// (rows_magic * nrows - 2^32 < nrows <= 152, so the quotient is exact while sr * 152 < 2^32)
__device__ __forceinline__ int sector_of(const Scalars& sc, int sr) { return (int)__umulhi((unsigned)sr, sc.rows_magic); }
__device__ __forceinline__ bool rec_is_start(const Rec& r) { return (__float_as_int(r.w) & kStartBit) != 0; }

// R20 selection key (layout above)
__device__ __forceinline__ unsigned long long sel_key(int nh, int start_orig, int t) {
  return ((unsigned long long)(unsigned)nh << 56) | ((unsigned long long)(0x7FFFFFFFu - (unsigned)start_orig) << kKeyTBits) |
         (unsigned long long)(unsigned)t;
}

constexpr int64_t kBlockCap = 148 * 64;  // grid-stride kernels: blocks per launch (per-block table set-up is amortised; measured optimum)
inline unsigned blocks_for(int64_t n, int threads, int64_t cap = kBlockCap) {
  int64_t b = (n + threads - 1) / threads;
  if (b > cap) b = cap;
  if (b < 1) b = 1;
  return (unsigned)b;
}

}  // namespace tpc
