// =============================================================================================
// tpc_select.cu -- step 4 of the hot path (BASELINE.json north_star (4) "sector-local track
// selection with cluster-to-track assignment"), integer work only.
//
//   k_push_keys    one warp per tracklet: atomicMax of its 64-bit key onto every recorded cluster
//   k_mark         one thread per CLUSTER: the winning key names its tracklet t (low key bits);
//                  set bit `row` in t's 160-bit kept-row mask
//   k_count_kept   one thread per tracklet: kept = popcount(mask); accept iff kept >= min_hits;
//                  value (1<<32 | kept) for the int64 scan that numbers tracks and hit offsets
//   k_assign       one thread per CLUSTER: owner accepted -> cluster_track, and the hit goes to
//                  trk_hits[first + rank], rank = kept rows below its own (a tracklet holds at
//                  most one cluster per row, so the hit list comes out row-ascending);
//                  the (y, z, row) of the hit is stored beside it for the refit
//   k_track_info   one thread per tracklet: trk_seed / trk_sector / trk_nhits / trk_first_hit,
//                  and the counters block
//
// The per-cluster passes touch N clusters instead of the ~3.6 N (tracklet,row) claims, stream the
// owner array in grid order, and need no row_hit table.
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
            const int32_t* __restrict__ ws_counters) {
  const int n_starts = ws_counters[WC_N_STARTS];
  const int lane = threadIdx.x & 31;
  const int64_t nwarps = (int64_t)gridDim.x * (kThreads / 32);
  for (int64_t t = (int64_t)blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5); t < n_starts; t += nwarps) {
    const int info = __ldg(tl_info + t);
    const int lo = (info >> 8) & 0xff, hi = (info >> 16) & 0xff;
    const unsigned long long key = __ldg(tl_key + t);
    const int32_t* hits = row_hit + t * nrows;
    for (int r = lo + lane; r <= hi; r += 32) {
      const int c = __ldg(hits + r);
      if (c >= 0) atomicMax(owner + c, key);
    }
  }
}

__global__ void __launch_bounds__(kThreads)
k_mark(int nrows, int64_t n, const Rec* __restrict__ rec, const unsigned long long* __restrict__ owner,
       uint32_t* __restrict__ tl_mask) {
  for (int64_t p = (int64_t)blockIdx.x * kThreads + threadIdx.x; p < n; p += (int64_t)gridDim.x * kThreads) {
    const unsigned long long key = owner[p];
    if (key == 0ull) continue;
    const int t = key_tracklet(key);
    const int row = rec_sr(ld_rec(rec, (int)p)) % nrows;
    atomicOr(tl_mask + (int64_t)t * kMaskWords + (row >> 5), 1u << (row & 31));
  }
}

__global__ void __launch_bounds__(kThreads)
k_count_kept(int min_hits, int64_t scap_pad, const uint32_t* __restrict__ tl_mask, long long* __restrict__ tl_val,
             const int32_t* __restrict__ ws_counters) {
  const int n_starts = ws_counters[WC_N_STARTS];
  for (int64_t t = (int64_t)blockIdx.x * kThreads + threadIdx.x; t <= scap_pad; t += (int64_t)gridDim.x * kThreads) {
    long long val = 0;
    if (t < n_starts) {
      const uint4* m = reinterpret_cast<const uint4*>(tl_mask + t * kMaskWords);
      const uint4 a = __ldg(m), b = __ldg(m + 1);
      const int kept = __popc(a.x) + __popc(a.y) + __popc(a.z) + __popc(a.w) + __popc(b.x);
      if (kept >= min_hits) val = (1ll << 32) | (long long)kept;
    }
    tl_val[t] = val;
  }
}

__global__ void __launch_bounds__(kThreads)
k_assign(int nrows, int64_t n, const Rec* __restrict__ rec, const unsigned long long* __restrict__ owner,
         const uint32_t* __restrict__ tl_mask, const long long* __restrict__ tl_scan, int64_t max_tracks,
         int32_t* __restrict__ cluster_track, int32_t* __restrict__ trk_hits, float4* __restrict__ hit_rec) {
  for (int64_t p = (int64_t)blockIdx.x * kThreads + threadIdx.x; p < n; p += (int64_t)gridDim.x * kThreads) {
    const Rec h = ld_rec(rec, (int)p);
    const int orig = rec_idx(h);
    const unsigned long long key = owner[p];
    int trk = -1;
    if (key != 0ull) {
      const int t = key_tracklet(key);
      const long long ex = __ldg(tl_scan + t), nx = __ldg(tl_scan + t + 1);
      const long long k = ex >> 32;
      if ((nx >> 32) != k && k < max_tracks) {  // owner accepted (R20) and inside the caller's capacity
        const int row = rec_sr(h) % nrows;
        const uint32_t* m = tl_mask + (int64_t)t * kMaskWords;
        const int w = row >> 5;
        int rank = __popc(__ldg(m + w) & ((1u << (row & 31)) - 1u));
        for (int j = 0; j < w; j++) rank += __popc(__ldg(m + j));
        const long long at = (ex & 0xffffffffll) + rank;
        trk_hits[at] = orig;
        hit_rec[at] = make_float4(h.x, h.y, __int_as_float(row), h.z);
        trk = (int)k;
      }
    }
    cluster_track[orig] = trk;
  }
}

__global__ void __launch_bounds__(kThreads)
k_track_info(int nrows, int64_t scap_pad, const TlInit* __restrict__ tl_init, const long long* __restrict__ tl_scan,
             int64_t max_tracks, int32_t* __restrict__ trk_seed, int32_t* __restrict__ trk_sector,
             int32_t* __restrict__ trk_nhits, int64_t* __restrict__ trk_first_hit, int32_t* __restrict__ counters,
             const int32_t* __restrict__ ws_counters) {
  const int n_starts = ws_counters[WC_N_STARTS];
  for (int64_t t = (int64_t)blockIdx.x * kThreads + threadIdx.x; t < scap_pad; t += (int64_t)gridDim.x * kThreads) {
    if (t == 0) {
      const long long total = tl_scan[scap_pad];
      const long long K = total >> 32;
      counters[TPC_CNT_TRACKS_FOUND] = (int)K;
      counters[TPC_CNT_TRACKS] = (int)(K < max_tracks ? K : max_tracks);
      counters[TPC_CNT_TRACKLETS] = n_starts;
      counters[TPC_CNT_STARTS_FOUND] = ws_counters[WC_STARTS_FOUND];
      if (K <= max_tracks) counters[TPC_CNT_HITS] = (int)(total & 0xffffffffll);
      counters[TPC_CNT_STATUS] = ws_counters[WC_STATUS] | (K > max_tracks ? TPC_ST_TRACK_OVERFLOW : 0);
      counters[TPC_CNT_RESERVED6] = 0;
      counters[TPC_CNT_RESERVED7] = 0;
      for (int k = 0; k < 6; k++) counters[TPC_CNT_PROP_LO + k] = ws_counters[WC_PROP64 + k];
      counters[14] = 0;
      counters[15] = 0;
    }
    if (t >= n_starts) continue;
    const long long ex = tl_scan[t], nx = tl_scan[t + 1];
    if ((nx >> 32) == (ex >> 32)) continue;  // not accepted
    const long long k = ex >> 32;
    const long long first = ex & 0xffffffffll;
    if (k == max_tracks) counters[TPC_CNT_HITS] = (int)first;  // first dropped track: hits used so far
    if (k >= max_tracks) continue;
    const float4 b = __ldg(reinterpret_cast<const float4*>(tl_init + t) + 1);
    trk_seed[k] = __float_as_int(b.w);
    trk_sector[k] = __float_as_int(b.z) / nrows;
    trk_nhits[k] = (int)((nx & 0xffffffffll) - first);
    trk_first_hit[k] = first;
  }
}

}  // namespace

cudaError_t launch_select(const Geo& g, const Ws& w, int32_t* cluster_track, int64_t max_tracks, int32_t* trk_seed,
                          int32_t* trk_sector, int32_t* trk_nhits, int64_t* trk_first_hit, int32_t* trk_hits,
                          int32_t* counters, cudaStream_t st) {
  const int64_t n = w.L.n, scap_pad = w.L.scap_pad;
  const int nrows = g.s.nrows;
  cudaError_t e;
  if ((e = cudaMemsetAsync(w.owner, 0, sizeof(uint64_t) * (size_t)(n + 1), st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(w.tl_mask, 0, sizeof(uint32_t) * kMaskWords * (size_t)(scap_pad + 1), st)) != cudaSuccess) return e;
  if (n > 0) {
    TPC_LAUNCH(KID_PUSH_KEYS, st,
               (k_push_keys<<<blocks_for(w.L.scap * 32, kThreads), kThreads, 0, st>>>(nrows, w.row_hit, w.tl_info, w.tl_key,
                                                                                     w.owner, w.counters)));
    TPC_LAUNCH(KID_MARK, st, (k_mark<<<blocks_for(n, kThreads), kThreads, 0, st>>>(nrows, n, w.rec, w.owner, w.tl_mask)));
  }
  TPC_LAUNCH(KID_COUNT_KEPT, st,
             (k_count_kept<<<blocks_for(scap_pad + 1, kThreads), kThreads, 0, st>>>(g.s.min_hits, scap_pad, w.tl_mask,
                                                                                  w.tl_scan, w.counters)));
  if ((e = exclusive_scan<long long>(w.tl_scan, w.tl_scan, scap_pad + 1, w.scan_tmp, st)) != cudaSuccess) return e;
  if (n > 0)
    TPC_LAUNCH(KID_ASSIGN, st,
               (k_assign<<<blocks_for(n, kThreads), kThreads, 0, st>>>(nrows, n, w.rec, w.owner, w.tl_mask, w.tl_scan,
                                                                      max_tracks, cluster_track, trk_hits, w.hit_rec)));
  TPC_LAUNCH(KID_TRACK_INFO, st,
             (k_track_info<<<blocks_for(scap_pad > 0 ? scap_pad : 1, kThreads), kThreads, 0, st>>>(
                 nrows, scap_pad, w.tl_init, w.tl_scan, max_tracks, trk_seed, trk_sector, trk_nhits, trk_first_hit, counters,
                 w.counters)));
  return cudaGetLastError();
}

}  // namespace tpc
