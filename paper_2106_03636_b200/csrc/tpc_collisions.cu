// =============================================================================================
// tpc_collisions.cu -- collisions from the per-track time offsets (second
// half; R25).  Integer work on a 1-D time histogram:
//
//   k_t0_hist     one thread per track (of the selected TPC side): bin of its t0 (R24), h[bin]++ and q[bin] += round(1024 (t0 - t_lo))
//   k_t0_peaks    one thread per bin: 5-bin sums s[b]; peak iff s >= n_min, s > s[b-j], s >= s[b+j], j = 1..3
//   scan          numbers the peaks in time order
//   k_t0_collect  one thread per bin: a peak writes its collision (mean time of its 5 bins, track count)
//   k_t0_assign   one thread per track: nearest peak within 5 bins (ties: the earlier one)
//
// Sizes are tiny next to the hot path (1.8e6 tracks, ~1e4 bins per Time Frame): clarity over speed.
// =============================================================================================
#include "tpc_common.cuh"
#include "tpc_prof.cuh"
#include "tpc_scan.cuh"

namespace tpc {

namespace {

constexpr int kThreads = 256;

__global__ void __launch_bounds__(kThreads)
k_t0_hist(const int32_t* __restrict__ counters, int64_t max_tracks, const float* __restrict__ t0,
          const float* __restrict__ dca, const int32_t* __restrict__ trk_sector, int side_sel, double t_lo, double w, int64_t nb, double dca_max, int32_t* __restrict__ trk_bin,
          int32_t* __restrict__ h, unsigned long long* __restrict__ q) {
  int64_t K = counters[TPC_CNT_TRACKS];
  if (K > max_tracks) K = max_tracks;
  for (int64_t k = (int64_t)blockIdx.x * kThreads + threadIdx.x; k < K; k += (int64_t)gridDim.x * kThreads) {
    const double t = t0[k];
    int b = -1;
    const bool side_ok = side_sel == 0 || ((side_sel > 0) == (trk_sector[k] < 18));
    if (t == t && (double)dca[k] <= dca_max && side_ok) {
      const double u = (t - t_lo) / w;
      if (u >= 0.0 && u < (double)nb) {
        b = (int)floor(u);
        atomicAdd(h + b, 1);
        atomicAdd(q + b, (unsigned long long)llround((t - t_lo) * 1024.0));
      }
    }
    trk_bin[k] = b;
  }
}

__device__ __forceinline__ int h_at(const int32_t* __restrict__ h, int64_t nb, int64_t b) {
  return (b >= 0 && b < nb) ? h[b] : 0;
}
__device__ __forceinline__ int s_at(const int32_t* __restrict__ h, int64_t nb, int64_t b) {
  return h_at(h, nb, b - 2) + h_at(h, nb, b - 1) + h_at(h, nb, b) + h_at(h, nb, b + 1) + h_at(h, nb, b + 2);
}

__global__ void __launch_bounds__(kThreads)
k_t0_peaks(int64_t nb, int32_t n_min, const int32_t* __restrict__ h, int32_t* __restrict__ flag, int32_t* __restrict__ scan_in) {
  for (int64_t b = (int64_t)blockIdx.x * kThreads + threadIdx.x; b <= nb; b += (int64_t)gridDim.x * kThreads) {
    int f = 0;
    if (b < nb) {
      const int s = s_at(h, nb, b);
      if (s >= n_min) {
        f = 1;
        for (int j = 1; j <= 3; j++)
          if (!(s > s_at(h, nb, b - j) && s >= s_at(h, nb, b + j))) f = 0;
      }
    }
    flag[b] = f;
    scan_in[b] = f;
  }
}

__global__ void __launch_bounds__(kThreads)
k_t0_collect(int64_t nb, double t_lo, const int32_t* __restrict__ h, const unsigned long long* __restrict__ q,
             const int32_t* __restrict__ flag, const int32_t* __restrict__ scan, int64_t max_collisions,
             float* __restrict__ coll_time, int32_t* __restrict__ coll_ntracks, int32_t* __restrict__ coll_bin,
             int32_t* __restrict__ n_collisions) {
  for (int64_t b = (int64_t)blockIdx.x * kThreads + threadIdx.x; b < nb; b += (int64_t)gridDim.x * kThreads) {
    if (b == 0) {
      const int total = scan[nb];
      n_collisions[0] = total;
      n_collisions[1] = total < max_collisions ? total : (int)max_collisions;
    }
    if (!flag[b]) continue;
    const int c = scan[b];
    if (c >= max_collisions) continue;
    long long cnt = 0, sum = 0;
    for (int64_t bb = b - 2; bb <= b + 2; bb++)
      if (bb >= 0 && bb < nb) {
        cnt += h[bb];
        sum += (long long)q[bb];
      }
    coll_time[c] = (float)(t_lo + ((double)sum / (double)cnt) / 1024.0);
    coll_ntracks[c] = (int)cnt;
    coll_bin[c] = (int)b;
  }
}

__global__ void __launch_bounds__(kThreads)
k_t0_assign(const int32_t* __restrict__ counters, int64_t max_tracks, int64_t nb, const int32_t* __restrict__ trk_bin,
            const int32_t* __restrict__ flag, const int32_t* __restrict__ scan, int64_t max_collisions,
            int32_t* __restrict__ trk_collision) {
  int64_t K = counters[TPC_CNT_TRACKS];
  if (K > max_tracks) K = max_tracks;
  for (int64_t k = (int64_t)blockIdx.x * kThreads + threadIdx.x; k < K; k += (int64_t)gridDim.x * kThreads) {
    const int b = trk_bin[k];
    int c = -1;
    if (b >= 0) {
      for (int d = 0; d <= 5 && c < 0; d++) {  // nearest peak; at equal distance the earlier one
        if (b - d >= 0 && flag[b - d]) c = scan[b - d];
        else if (b + d < nb && flag[b + d]) c = scan[b + d];
      }
    }
    trk_collision[k] = (c >= 0 && c < max_collisions) ? c : -1;
  }
}

}  // namespace

size_t collisions_ws_bytes(int64_t nb, int64_t max_tracks) {
  size_t o = 0;
  o += align256(sizeof(int32_t) * (size_t)(nb + 1));             // h
  o += align256(sizeof(unsigned long long) * (size_t)(nb + 1));  // q
  o += align256(sizeof(int32_t) * (size_t)(nb + 2));             // flag
  o += align256(sizeof(int32_t) * (size_t)(nb + 2));             // scan
  o += align256(sizeof(int32_t) * (size_t)(max_tracks + 1));     // trk_bin
  o += align256(sizeof(int32_t) * (size_t)((nb + 1 + kScanTile - 1) / kScanTile + 4));  // scan scratch
  return o;
}

cudaError_t launch_collisions(const int32_t* counters, int64_t max_tracks, const float* t0, const float* dca,
                              const int32_t* trk_sector, int side_sel, double t_lo,
                              double w, int64_t nb, double dca_max, int32_t n_min, void* workspace, int64_t max_collisions,
                              float* coll_time, int32_t* coll_ntracks, int32_t* coll_bin, int32_t* trk_collision,
                              int32_t* n_collisions, cudaStream_t st) {
  char* p = (char*)workspace;
  int32_t* h = (int32_t*)p;
  p += align256(sizeof(int32_t) * (size_t)(nb + 1));
  unsigned long long* q = (unsigned long long*)p;
  p += align256(sizeof(unsigned long long) * (size_t)(nb + 1));
  int32_t* flag = (int32_t*)p;
  p += align256(sizeof(int32_t) * (size_t)(nb + 2));
  int32_t* scan = (int32_t*)p;
  p += align256(sizeof(int32_t) * (size_t)(nb + 2));
  int32_t* trk_bin = (int32_t*)p;
  p += align256(sizeof(int32_t) * (size_t)(max_tracks + 1));
  int32_t* scan_tmp = (int32_t*)p;
  cudaError_t e;
  if ((e = cudaMemsetAsync(h, 0, (size_t)((char*)flag - (char*)h), st)) != cudaSuccess) return e;  // h and q
  TPC_LAUNCH(KID_COLLISIONS, st,
             (k_t0_hist<<<blocks_for(max_tracks, kThreads, 148 * 8), kThreads, 0, st>>>(counters, max_tracks, t0, dca, trk_sector, side_sel,
                                                                                       t_lo, w, nb, dca_max, trk_bin, h, q)));
  TPC_LAUNCH(KID_COLLISIONS, st, (k_t0_peaks<<<blocks_for(nb + 1, kThreads, 148 * 8), kThreads, 0, st>>>(nb, n_min, h, flag, scan)));
  if ((e = exclusive_scan<int32_t>(scan, scan, nb + 1, scan_tmp, st)) != cudaSuccess) return e;
  TPC_LAUNCH(KID_COLLISIONS, st,
             (k_t0_collect<<<blocks_for(nb, kThreads, 148 * 8), kThreads, 0, st>>>(nb, t_lo, h, q, flag, scan, max_collisions,
                                                                                  coll_time, coll_ntracks, coll_bin, n_collisions)));
  TPC_LAUNCH(KID_COLLISIONS, st,
             (k_t0_assign<<<blocks_for(max_tracks, kThreads, 148 * 8), kThreads, 0, st>>>(counters, max_tracks, nb, trk_bin, flag,
                                                                                         scan, max_collisions, trk_collision)));
  return cudaGetLastError();
}

}  // namespace tpc
