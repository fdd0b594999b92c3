// =============================================================================================
// tpc_select.cu -- step 4 of the hot path (BASELINE.json north_star (4) "sector-local track
// selection with cluster-to-track assignment"), integer work only.
// One WARP per tracklet, lanes = pad rows, over the tracklet-major row_hit[t][row] table:
//
//   k_push_keys     atomicMax of the tracklet's 64-bit key onto every cluster it recorded
//   k_count_kept    kept rows = rows whose cluster is still owned by this key (ballot -> 160-bit
//                   mask per tracklet); accept iff kept >= min_hits; value (1<<32 | kept) for the
//                   int64 scan that numbers the tracks and their hit-list offsets
//   k_write_tracks  accepted tracklets write their hit list (row-ascending, original indices),
//                   the (y, z, row) record of every hit for the refit, and the per-track arrays; the
//                   counters block.  cluster_track[orig] = track is a scatter by ORIGINAL index, i.e.
//                   (input order is arbitrary) 1.3e8 random 4-byte writes on configs[4]: written
//                   directly they cost a DRAM read-modify-write of a 32-byte sector each and 4.5 of
//                   the kernel's 5.9 ms.  So above one window of 2^22 clusters the kernel only
//                   PARTITIONS (orig, track) pairs by window -- block-local ranks from shared-memory
//                   counters, one global cursor add per block and window -- and
//   k_assign        scatters window after window, each a 16 MB slice of cluster_track that stays in
//                   L2 until its sectors are complete.
//
// Only the tracklets that went through phase B of the follower (`surv`, R17) take part.  Tracklets are numbered by
// (sector, z slab, row) (tpc_find.cu), so the few thousand warps in
// flight work on one z slab of one sector: the owner / record gathers and the atomics stay in L2.
// =============================================================================================
#include "tpc_common.cuh"
#include "tpc_prof.cuh"
#include "tpc_scan.cuh"

namespace tpc {

namespace {

constexpr int kThreads = 256;

__global__ void __launch_bounds__(kThreads)
k_push_keys(int nrows, const int32_t* __restrict__ row_hit, const int32_t* __restrict__ tl_info,
            const unsigned long long* __restrict__ tl_key, unsigned long long* __restrict__ owner,
            const int32_t* __restrict__ surv, const int32_t* __restrict__ ws_counters) {
  const int n_surv = ws_counters[WC_N_SURV];
  const int lane = threadIdx.x & 31;
  const int64_t nwarps = (int64_t)gridDim.x * (kThreads / 32);
  for (int64_t i = (int64_t)blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5); i < n_surv; i += nwarps) {
    const int64_t t = __ldg(surv + i);
    const int info = __ldg(tl_info + t);
    const int lo = (info >> 8) & 0xff, hi = (info >> 16) & 0xff;
    const unsigned long long key = __ldg(tl_key + t);
    const int32_t* hits = row_hit + t * nrows;
    int c[kMaskWords];
    unsigned long long own[kMaskWords];
#pragma unroll
    for (int w = 0; w < kMaskWords; w++) {
      const int r = 32 * w + lane;
      c[w] = (r >= lo && r <= hi) ? __ldg(hits + r) : -1;
    }
    // a plain read first: a claim that already lost (on average about half of them) needs no atomic
#pragma unroll
    for (int w = 0; w < kMaskWords; w++) own[w] = c[w] >= 0 ? __ldcg(owner + c[w]) : ~0ull;
#pragma unroll
    for (int w = 0; w < kMaskWords; w++)
      if (own[w] < key) atomicMax(owner + c[w], key);
  }
}

__global__ void __launch_bounds__(kThreads)
k_count_kept(int nrows, int min_hits, const int32_t* __restrict__ row_hit, const int32_t* __restrict__ tl_info,
             const unsigned long long* __restrict__ tl_key, const unsigned long long* __restrict__ owner,
             uint32_t* __restrict__ tl_mask, long long* __restrict__ tl_val, const int32_t* __restrict__ surv,
             const int32_t* __restrict__ ws_counters) {
  const int n_surv = ws_counters[WC_N_SURV];
  const int lane = threadIdx.x & 31;
  const int64_t nwarps = (int64_t)gridDim.x * (kThreads / 32);
  for (int64_t i = (int64_t)blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5); i < n_surv; i += nwarps) {
    const int64_t t = __ldg(surv + i);
    const int info = __ldg(tl_info + t);
    const int lo = (info >> 8) & 0xff, hi = (info >> 16) & 0xff;
    const unsigned long long key = __ldg(tl_key + t);
    const int32_t* hits = row_hit + t * nrows;
    // all of the tracklet's rows are requested before the first use, then all owner gathers (5 loads in flight per
    // lane instead of 1: these kernels are latency-bound, not bandwidth-bound)
    int c[kMaskWords];
    unsigned long long own[kMaskWords];
#pragma unroll
    for (int w = 0; w < kMaskWords; w++) {
      const int r = 32 * w + lane;
      c[w] = (r >= lo && r <= hi) ? __ldg(hits + r) : -1;
    }
#pragma unroll
    for (int w = 0; w < kMaskWords; w++) own[w] = c[w] >= 0 ? __ldcg(owner + c[w]) : 0ull;
    int kept = 0;
    unsigned mine = 0u;  // lane w keeps mask word w
#pragma unroll
    for (int w = 0; w < kMaskWords; w++) {
      const unsigned m = __ballot_sync(0xffffffffu, c[w] >= 0 && own[w] == key);
      kept += __popc(m);
      if (lane == w) mine = m;
    }
    if (lane < kMaskWords) tl_mask[t * kMaskWords + lane] = mine;
    if (lane == 0) tl_val[t] = kept >= min_hits ? ((1ll << 32) | (long long)kept) : 0ll;
  }
}

constexpr int kMaxPart = 128;  // windows of cluster_track (2^shift clusters each) the scatter is partitioned into

// PART = false: cluster_track written directly (n <= one window: it stays in L2 anyway).
// PART = true: (orig, track) pairs appended to window orig >> shift of `pairs`; window b owns the slots
// [b << shift, (b + 1) << shift) -- it can never hold more pairs than it has clusters.
template <bool PART>
__global__ void __launch_bounds__(kThreads)
k_write_tracks(int nrows, const Rec* __restrict__ rec, const TlInit* __restrict__ tl_init,
               const int32_t* __restrict__ row_hit, const uint32_t* __restrict__ tl_mask,
               const long long* __restrict__ tl_scan, int64_t scap_pad, int64_t max_tracks,
               int32_t* __restrict__ cluster_track, int32_t* __restrict__ trk_seed, int32_t* __restrict__ trk_sector,
               int32_t* __restrict__ trk_nhits, int64_t* __restrict__ trk_first_hit, int32_t* __restrict__ trk_hits,
               float4* __restrict__ hit_rec, int32_t* __restrict__ counters, const int32_t* __restrict__ surv,
               const int32_t* __restrict__ ws_counters, int shift, int nparts, unsigned long long* __restrict__ pairs,
               int32_t* __restrict__ part_cursor) {
  __shared__ int s_cnt[kMaxPart], s_base[kMaxPart];
  const int n_starts = ws_counters[WC_N_STARTS], n_surv = ws_counters[WC_N_SURV];
  const int lane = threadIdx.x & 31;
  constexpr int kWarps = kThreads / 32;
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    const long long total = tl_scan[scap_pad];
    const long long K = total >> 32;
    counters[TPC_CNT_TRACKS_FOUND] = (int)K;
    counters[TPC_CNT_TRACKS] = (int)(K < max_tracks ? K : max_tracks);
    counters[TPC_CNT_TRACKLETS] = n_starts;
    counters[TPC_CNT_STARTS_FOUND] = ws_counters[WC_STARTS_FOUND];
    if (K <= max_tracks) counters[TPC_CNT_HITS] = (int)(total & 0xffffffffll);
    counters[TPC_CNT_STATUS] = ws_counters[WC_STATUS] | (K > max_tracks ? TPC_ST_TRACK_OVERFLOW : 0);
    counters[TPC_CNT_FOLLOWED_DOWN] = n_surv;
    counters[TPC_CNT_RESERVED7] = 0;
    for (int k = 0; k < 8; k++) counters[TPC_CNT_PROP_LO + k] = ws_counters[WC_PROP64 + k];
  }
  // one warp per surviving tracklet; the trip count is the same for all warps of a block (block barriers inside)
  for (int64_t i0 = (int64_t)blockIdx.x * kWarps; i0 < n_surv; i0 += (int64_t)gridDim.x * kWarps) {
    const int64_t i = i0 + (threadIdx.x >> 5);
    if (PART) {
      for (int j = threadIdx.x; j < nparts; j += kThreads) s_cnt[j] = 0;
      __syncthreads();
    }
    long long k = -1, first = 0;
    int64_t t = 0;
    if (i < n_surv) {
      t = __ldg(surv + i);
      const long long ex = __ldg(tl_scan + t), nx = __ldg(tl_scan + t + 1);
      first = ex & 0xffffffffll;
      if ((nx >> 32) != (ex >> 32)) {  // accepted (R20)
        k = ex >> 32;
        if (k == max_tracks && lane == 0) counters[TPC_CNT_HITS] = (int)first;  // first dropped track: hits used so far
        if (k >= max_tracks) k = -1;
        if (k >= 0 && lane == 0) {
          const float4 b = __ldg(reinterpret_cast<const float4*>(tl_init + t) + 1);
          trk_seed[k] = __float_as_int(b.w);
          trk_sector[k] = __float_as_int(b.z) / nrows;
          trk_nhits[k] = (int)((nx & 0xffffffffll) - first);
          trk_first_hit[k] = first;
        }
      }
    }
    unsigned m[kMaskWords];
    int c[kMaskWords], rank[kMaskWords];
    Rec h[kMaskWords];
    const int32_t* hits = row_hit + t * nrows;
#pragma unroll
    for (int w = 0; w < kMaskWords; w++) m[w] = k >= 0 ? __ldg(tl_mask + t * kMaskWords + w) : 0u;
#pragma unroll
    for (int w = 0; w < kMaskWords; w++) c[w] = ((m[w] >> lane) & 1u) ? __ldg(hits + 32 * w + lane) : -1;
#pragma unroll
    for (int w = 0; w < kMaskWords; w++) h[w] = c[w] >= 0 ? ld_rec(rec, c[w]) : make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    long long at = first;
#pragma unroll
    for (int w = 0; w < kMaskWords; w++) {
      rank[w] = 0;
      if (c[w] >= 0) {
        const long long o = at + __popc(m[w] & ((1u << lane) - 1u));
        trk_hits[o] = rec_idx(h[w]);
        hit_rec[o] = make_float4(h[w].x, h[w].y, __int_as_float(32 * w + lane), h[w].z);
        if (PART) rank[w] = atomicAdd(&s_cnt[rec_idx(h[w]) >> shift], 1);
        else cluster_track[rec_idx(h[w])] = (int)k;
      }
      at += __popc(m[w]);
    }
    if (PART) {
      __syncthreads();
      for (int j = threadIdx.x; j < nparts; j += kThreads) {
        const int cnt = s_cnt[j];
        s_base[j] = cnt ? atomicAdd(part_cursor + j, cnt) : 0;
      }
      __syncthreads();
#pragma unroll
      for (int w = 0; w < kMaskWords; w++) {
        if (c[w] >= 0) {
          const int orig = rec_idx(h[w]);
          const int b = orig >> shift;
          pairs[((int64_t)b << shift) + s_base[b] + rank[w]] = (unsigned long long)(unsigned)orig | ((unsigned long long)(unsigned)k << 32);
        }
      }
    }
  }
}

// cluster_track[orig] = track for the pairs of one window after the other: block (b, j) takes every kAssignBlocks-th
// tile of window b, and blocks start in index order, so at any time the blocks in flight write into one or two windows.
constexpr int kAssignBlocks = 148 * 8;

__global__ void __launch_bounds__(kThreads)
k_assign(int shift, const unsigned long long* __restrict__ pairs, const int32_t* __restrict__ part_cursor,
         int32_t* __restrict__ cluster_track) {
  const int b = blockIdx.x / kAssignBlocks, j = blockIdx.x % kAssignBlocks;
  const int cnt = part_cursor[b];
  const unsigned long long* src = pairs + ((int64_t)b << shift);
  for (int i = j * kThreads + threadIdx.x; i < cnt; i += kAssignBlocks * kThreads) {
    const unsigned long long pr = __ldcs(src + i);
    cluster_track[(unsigned)(pr & 0xffffffffull)] = (int)(pr >> 32);
  }
}

}  // namespace

cudaError_t launch_select(const Geo& g, const Ws& w, int32_t* cluster_track, int64_t max_tracks, int32_t* trk_seed,
                          int32_t* trk_sector, int32_t* trk_nhits, int64_t* trk_first_hit, int32_t* trk_hits,
                          int32_t* counters, cudaStream_t st) {
  const int64_t n = w.L.n, scap_pad = w.L.scap_pad;
  const int nrows = g.s.nrows;
  // One warp per surviving tracklet.  Grid sizes are measured, not derived (configs[4], 2.0e6 survivors): push and
  // write run fastest with (nearly) one warp per tracklet and no grid-stride loop -- consecutive tracklets in flight
  // share z slab and cache lines (push 1.72 -> 1.20 ms, write 7.4 -> 6.1 ms against a 9472-block grid); count is
  // fastest on the 9472-block grid-stride grid.  (Before R17, with 3 tracklets per track claiming the same clusters,
  // consecutive tracklets in flight meant same-line atomic contention and push was 2.5x slower that way.)
  const unsigned wblocks = blocks_for(w.L.scap * 32, kThreads);
  const unsigned wblocks_wide = blocks_for(w.L.scap * 32, kThreads, 148 * 2048);
  cudaError_t e;
  if ((e = cudaMemsetAsync(w.owner, 0, sizeof(uint64_t) * (size_t)(n + 1), st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(w.tl_scan, 0, sizeof(long long) * (size_t)(scap_pad + 2), st)) != cudaSuccess) return e;
  if (n > 0) {
    if ((e = cudaMemsetAsync(cluster_track, 0xFF, sizeof(int32_t) * (size_t)n, st)) != cudaSuccess) return e;
    TPC_LAUNCH(KID_PUSH_KEYS, st,
               (k_push_keys<<<wblocks_wide, kThreads, 0, st>>>(nrows, w.row_hit, w.tl_info, w.tl_key, w.owner, w.surv, w.counters)));
    TPC_LAUNCH(KID_COUNT_KEPT, st,
               (k_count_kept<<<wblocks, kThreads, 0, st>>>(nrows, g.s.min_hits, w.row_hit, w.tl_info, w.tl_key, w.owner,
                                                          w.tl_mask, w.tl_scan, w.surv, w.counters)));
  }
  if ((e = exclusive_scan<long long>(w.tl_scan, w.tl_scan, scap_pad + 1, w.scan_tmp, st)) != cudaSuccess) return e;
  // windows of the cluster_track scatter: 2^22 clusters (16 MB), more only if that would give more than kMaxPart
  int shift = 22;
  while (n > 0 && ((n - 1) >> shift) >= kMaxPart) shift++;
  const int nparts = n > 0 ? (int)(((n - 1) >> shift) + 1) : 1;
  unsigned long long* pairs = w.owner;     // the R20 keys are dead once k_count_kept has run
  int32_t* part_cursor = w.bucket_cursor;  // the grid build's cursors are dead since tpc_grid_build
  if (nparts > 1) {
    if ((e = cudaMemsetAsync(part_cursor, 0, sizeof(int32_t) * (size_t)nparts, st)) != cudaSuccess) return e;
    TPC_LAUNCH(KID_WRITE_TRACKS, st,
               (k_write_tracks<true><<<wblocks_wide, kThreads, 0, st>>>(
                   nrows, w.rec, w.tl_init, w.row_hit, w.tl_mask, w.tl_scan, scap_pad, max_tracks, cluster_track, trk_seed,
                   trk_sector, trk_nhits, trk_first_hit, trk_hits, w.hit_rec, counters, w.surv, w.counters, shift, nparts, pairs,
                   part_cursor)));
    TPC_LAUNCH(KID_ASSIGN, st,
               (k_assign<<<(unsigned)(nparts * kAssignBlocks), kThreads, 0, st>>>(shift, pairs, part_cursor, cluster_track)));
  } else {
    TPC_LAUNCH(KID_WRITE_TRACKS, st,
               (k_write_tracks<false><<<wblocks_wide, kThreads, 0, st>>>(
                   nrows, w.rec, w.tl_init, w.row_hit, w.tl_mask, w.tl_scan, scap_pad, max_tracks, cluster_track, trk_seed,
                   trk_sector, trk_nhits, trk_first_hit, trk_hits, w.hit_rec, counters, w.surv, w.counters, shift, nparts, pairs,
                   part_cursor)));
  }
  return cudaGetLastError();
}

}  // namespace tpc
