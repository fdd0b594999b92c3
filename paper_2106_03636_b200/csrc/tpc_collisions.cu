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
#include <mutex>

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

// R29: pairing of the two sides' collisions.  which = 0: thread i of side A looks for its best partner on side C;
// which = 1: thread j of side C for its best partner on side A.  The cost is formed in double in R29's operation
// order; ties go to the lower index (strict < while the partner index ascends).
__global__ void __launch_bounds__(kThreads)
k_pair_best(int which, const int32_t* __restrict__ n_a, const float* __restrict__ t_a, const int32_t* __restrict__ c_a,
            const int32_t* __restrict__ n_c, const float* __restrict__ t_c, const int32_t* __restrict__ c_c, int max_coll,
            double dt_max, double sigma_t, int32_t* __restrict__ best) {
  // the counts come from device memory: never beyond the capacity the tables and outputs were sized for
  const int nA = min(max(n_a[1], 0), max_coll), nC = min(max(n_c[1], 0), max_coll);
  const int n_own = which == 0 ? nA : nC, n_oth = which == 0 ? nC : nA;
  for (int i = blockIdx.x * kThreads + threadIdx.x; i < n_own; i += gridDim.x * kThreads) {
    int b = -1;
    double bc = 0.0;
    for (int j = 0; j < n_oth; j++) {
      const int ia = which == 0 ? i : j, ic = which == 0 ? j : i;
      const double dt = (double)t_c[ic] - (double)t_a[ia];
      if (!(fabs(dt) <= dt_max)) continue;
      const double u = dt / sigma_t, dn = (double)c_a[ia] - (double)c_c[ic];
      const double cost = u * u + (dn * dn) / ((double)c_a[ia] + (double)c_c[ic] + 1.0);
      if (b < 0 || cost < bc) {
        b = j;
        bc = cost;
      }
    }
    best[i] = b;
  }
}

// reciprocal pairs in ascending order of the side-A index (a Time Frame holds a few hundred collisions: one thread)
__global__ void k_pair_emit(const int32_t* __restrict__ n_a, const float* __restrict__ t_a, const int32_t* __restrict__ n_c,
                            const float* __restrict__ t_c, const int32_t* __restrict__ best_c, const int32_t* __restrict__ best_a,
                            int max_coll, double v_drift, int32_t* __restrict__ pair_of_a, int32_t* __restrict__ pair_of_c,
                            float* __restrict__ t_out, float* __restrict__ zv_out, int32_t* __restrict__ n_pairs) {
  const int nA = min(max(n_a[1], 0), max_coll), nC = min(max(n_c[1], 0), max_coll);
  for (int j = 0; j < nC; j++) pair_of_c[j] = -1;
  int np = 0;
  for (int i = 0; i < nA; i++) {
    const int j = best_c[i];
    if (j >= 0 && best_a[j] == i) {
      pair_of_a[i] = j;
      pair_of_c[j] = i;
      t_out[np] = (float)(((double)t_a[i] + (double)t_c[j]) * 0.5);
      zv_out[np] = (float)((v_drift * ((double)t_c[j] - (double)t_a[i])) * 0.5);
      np++;
    } else {
      pair_of_a[i] = -1;
    }
  }
  n_pairs[0] = np;
}

}  // namespace

size_t pair_sides_ws_bytes(int64_t max_collisions) { return 2 * align256(sizeof(int32_t) * (size_t)(max_collisions + 1)); }

cudaError_t launch_pair_sides(const int32_t* n_a, const float* t_a, const int32_t* c_a, const int32_t* n_c, const float* t_c,
                              const int32_t* c_c, int64_t max_collisions, double dt_max, double sigma_t, double v_drift,
                              void* workspace, int32_t* pair_of_a, int32_t* pair_of_c, float* t_out, float* zv_out,
                              int32_t* n_pairs, cudaStream_t st) {
  int32_t* best_c = (int32_t*)workspace;
  int32_t* best_a = (int32_t*)((char*)workspace + align256(sizeof(int32_t) * (size_t)(max_collisions + 1)));
  const unsigned blocks = blocks_for(max_collisions, kThreads, 148 * 4);
  const int cap = (int)max_collisions;
  TPC_LAUNCH(KID_COLLISIONS, st, (k_pair_best<<<blocks, kThreads, 0, st>>>(0, n_a, t_a, c_a, n_c, t_c, c_c, cap, dt_max, sigma_t, best_c)));
  TPC_LAUNCH(KID_COLLISIONS, st, (k_pair_best<<<blocks, kThreads, 0, st>>>(1, n_a, t_a, c_a, n_c, t_c, c_c, cap, dt_max, sigma_t, best_a)));
  TPC_LAUNCH(KID_COLLISIONS, st,
             (k_pair_emit<<<1, 1, 0, st>>>(n_a, t_a, n_c, t_c, best_c, best_a, cap, v_drift, pair_of_a, pair_of_c, t_out, zv_out, n_pairs)));
  return cudaGetLastError();
}

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

// =============================================================================================
// tpc_pair_sides_static -- tpc_pair_sides for callers that cannot allocate device memory (include/tpc_b200.h has the
// user's view: who such callers are, the limit, the first-call rule, the sharing rule).
//
// The two arg-min tables of R29 (best_c: side A's choice per side-A collision, best_a: side C's choice) are the only
// scratch memory the pairing needs.  Here they live in a file-scope __device__ array, i.e. in the device image of
// this library: the driver reserves it on a GPU when the library's module is loaded there and keeps it until the
// process ends.  Nothing is allocated at call time.
//
// g_pair_scratch below is only a handle on the host side.  Host code cannot use `g_pair_scratch` as a pointer: that
// expression is the address of a host shadow variable, and a kernel handed it would fault (or, on a system where the
// GPU can read host memory, scribble over the shadow instead of the real array).  The device address is asked for once
// per device with cudaGetSymbolAddress while that device is current, checked, cached in g_pair_scratch_dev[device], and
// that pointer is what the kernels get -- the very kernels tpc_pair_sides runs, through the same launch sequence.
// =============================================================================================
namespace {

constexpr size_t kPairStaticHalf = (sizeof(int32_t) * (size_t)(TPC_PAIR_SIDES_STATIC_MAX + 1) + 255) & ~(size_t)255;  // one table
static __device__ __align__(256) unsigned char g_pair_scratch[2 * kPairStaticHalf];  // best_c | best_a, 131 584 bytes

constexpr int kPairMaxDevices = 64;
void* g_pair_scratch_dev[kPairMaxDevices] = {nullptr};  // device address of g_pair_scratch on device d; NULL = not looked up yet
std::mutex g_pair_scratch_mutex;

// Device address of the scratch array on the CURRENT device.  The first call per device does the look-up (and with it
// whatever module loading the runtime still owes on that device); later calls read the cache.
cudaError_t pair_scratch_address(void** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  const bool cached = dev >= 0 && dev < kPairMaxDevices;
  std::lock_guard<std::mutex> lock(g_pair_scratch_mutex);
  if (cached && g_pair_scratch_dev[dev]) {
    *out = g_pair_scratch_dev[dev];
    return cudaSuccess;
  }
  void* p = nullptr;
  e = cudaGetSymbolAddress(&p, g_pair_scratch);
  if (e != cudaSuccess) return e;
  if (!p || ((uintptr_t)p & 255) != 0) return cudaErrorInvalidSymbol;
  if (cached) g_pair_scratch_dev[dev] = p;
  *out = p;
  return cudaSuccess;
}

}  // namespace

extern "C" int tpc_pair_sides_static(const int32_t* n_collisions_a, const float* coll_time_a, const int32_t* coll_ntracks_a,
                                     const int32_t* n_collisions_c, const float* coll_time_c, const int32_t* coll_ntracks_c,
                                     int64_t max_collisions, double dt_max, double sigma_t, double v_drift, int32_t* pair_of_a,
                                     int32_t* pair_of_c, float* t, float* z_vertex, int32_t* n_pairs, void* stream) {
  if (max_collisions < 1 || !(dt_max > 0.0) || !(sigma_t > 0.0) || !(v_drift > 0.0) || !n_collisions_a || !coll_time_a ||
      !coll_ntracks_a || !n_collisions_c || !coll_time_c || !coll_ntracks_c || !pair_of_a || !pair_of_c || !t || !z_vertex ||
      !n_pairs)
    return TPC_EINVAL;
  if (max_collisions > TPC_PAIR_SIDES_STATIC_MAX) return TPC_ELIMIT;  // the tables would not fit the fixed array
  void* scratch = nullptr;
  cudaError_t e = pair_scratch_address(&scratch);
  if (e != cudaSuccess) return tpc::report_cuda_error(e);
  // Same layout as launch_pair_sides gives a caller's workspace: best_c first, best_a one 256-byte-rounded table
  // later.  max_collisions <= the static maximum, so both tables end inside the array.
  int32_t* best_c = (int32_t*)scratch;
  int32_t* best_a = (int32_t*)((char*)scratch + tpc::align256(sizeof(int32_t) * (size_t)(max_collisions + 1)));
  cudaStream_t st = (cudaStream_t)stream;
  const unsigned blocks = tpc::blocks_for(max_collisions, tpc::kThreads, 148 * 4);
  // plain launches: counted, never bracketed by events (creating an event is an allocation)
  tpc::prof_count(tpc::KID_COLLISIONS);
  const int cap = (int)max_collisions;
  tpc::k_pair_best<<<blocks, tpc::kThreads, 0, st>>>(0, n_collisions_a, coll_time_a, coll_ntracks_a, n_collisions_c, coll_time_c,
                                                     coll_ntracks_c, cap, dt_max, sigma_t, best_c);
  tpc::prof_count(tpc::KID_COLLISIONS);
  tpc::k_pair_best<<<blocks, tpc::kThreads, 0, st>>>(1, n_collisions_a, coll_time_a, coll_ntracks_a, n_collisions_c, coll_time_c,
                                                     coll_ntracks_c, cap, dt_max, sigma_t, best_a);
  tpc::prof_count(tpc::KID_COLLISIONS);
  tpc::k_pair_emit<<<1, 1, 0, st>>>(n_collisions_a, coll_time_a, n_collisions_c, coll_time_c, best_c, best_a, cap, v_drift, pair_of_a,
                                    pair_of_c, t, z_vertex, n_pairs);
  e = cudaGetLastError();
  return e == cudaSuccess ? TPC_OK : tpc::report_cuda_error(e);
}
