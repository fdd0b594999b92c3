// =============================================================================================
// tpc_cluster.cu -- the step in front of the hot path ("TPC
// clusterizer"; R27): clusters from zero-suppressed digits (sector_row, pad, time bin, ADC).
//
// Digits arrive in any order and are sparse in (row, pad, time): a dense charge map of a 128-orbit Time Frame
// would take ~200 GB, so the cells go into an open-addressing hash table (key = sector_row | time | pad, linear
// probing, load <= 0.5) -- insertion and the eight neighbour look-ups of the peak test are one or two probes each.
//
//   k_digit_insert  one thread per digit: claim the cell's slot (atomicCAS on the key), add the ADC (two digits of
//                   one cell add up)
//   k_digit_peaks   one thread per table slot: an occupied cell with ADC >= peak_min reads its 8 neighbours; R27
//                   peak rule (strictly above the four earlier neighbours, at least equal to the four later ones);
//                   a peak writes its 3 x 3 centre of gravity (integer sums, fp32 position in R27's operation order)
//                   to the next free output slot (atomic counter: the output order is unspecified)
// =============================================================================================
#include "tpc_common.cuh"
#include "tpc_prof.cuh"

namespace tpc {

namespace {

constexpr int kThreads = 256;
constexpr unsigned long long kEmpty = ~0ull;

__device__ __forceinline__ unsigned long long cell_key(int s, int t, int p) {
  return ((unsigned long long)(unsigned)s << 40) | ((unsigned long long)(unsigned)t << 16) | (unsigned long long)(unsigned)p;
}

__device__ __forceinline__ unsigned long long mix64(unsigned long long x) {  // splitmix64 finaliser
  x ^= x >> 30;
  x *= 0xbf58476d1ce4e5b9ull;
  x ^= x >> 27;
  x *= 0x94d049bb133111ebull;
  x ^= x >> 31;
  return x;
}

__global__ void __launch_bounds__(kThreads)
k_digit_insert(int64_t n, int sr_end, const int32_t* __restrict__ sr, const int32_t* __restrict__ pad,
               const int32_t* __restrict__ tim, const int32_t* __restrict__ adc, unsigned long long* keys,
               int32_t* __restrict__ vals, unsigned long long mask) {
  for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < n; i += (int64_t)gridDim.x * kThreads) {
    const int s = sr[i], p = pad[i], t = tim[i];
    if ((unsigned)s >= (unsigned)sr_end || (unsigned)p > 65535u || (unsigned)t >= (1u << 24)) continue;  // no such cell
    if (adc[i] <= 0) continue;  // R27: not a zero-suppressed digit (keeps every cell sum, and so S at a peak, positive)
    const unsigned long long k = cell_key(s, t, p);
    unsigned long long h = mix64(k) & mask;
    for (;;) {
      const unsigned long long prev = atomicCAS(keys + h, kEmpty, k);
      if (prev == kEmpty || prev == k) {
        atomicAdd(vals + h, adc[i]);
        break;
      }
      h = (h + 1) & mask;
    }
  }
}

__device__ __forceinline__ int cell_value(const unsigned long long* __restrict__ keys, const int32_t* __restrict__ vals,
                                          unsigned long long mask, int s, int t, int p) {
  if (t < 0 || p < 0 || p > 65535 || t >= (1 << 24)) return 0;
  const unsigned long long k = cell_key(s, t, p);
  unsigned long long h = mix64(k) & mask;
  for (;;) {
    const unsigned long long kk = keys[h];
    if (kk == k) return vals[h];
    if (kk == kEmpty) return 0;
    h = (h + 1) & mask;
  }
}

__global__ void __launch_bounds__(kThreads)
k_digit_peaks(const __grid_constant__ Geo g, const unsigned long long* __restrict__ keys, const int32_t* __restrict__ vals,
              unsigned long long mask, float pad_width, float time_width, int peak_min, int64_t max_clusters,
              float* __restrict__ y, float* __restrict__ z, float* __restrict__ q, int32_t* __restrict__ out_sr,
              int32_t* __restrict__ out_pad, int32_t* __restrict__ out_time, int32_t* __restrict__ n_clusters) {
  const int nrows = g.s.nrows;
  for (unsigned long long h = (unsigned long long)blockIdx.x * kThreads + threadIdx.x; h <= mask;
       h += (unsigned long long)gridDim.x * kThreads) {
    const unsigned long long k = keys[h];
    if (k == kEmpty) continue;
    const int a = vals[h];
    if (a < peak_min) continue;
    const int s = (int)(k >> 40), t0 = (int)((k >> 16) & 0xFFFFFF), p0 = (int)(k & 0xFFFF);
    int b[9];
#pragma unroll
    for (int j = 0; j < 9; j++) {
      const int dt = j / 3 - 1, dp = j % 3 - 1;
      b[j] = (j == 4) ? a : cell_value(keys, vals, mask, s, t0 + dt, p0 + dp);
    }
    bool peak = true;
    int S = 0, Sp = 0, St = 0;
#pragma unroll
    for (int j = 0; j < 9; j++) {
      const int dt = j / 3 - 1, dp = j % 3 - 1;
      if (j < 4) peak = peak && (a > b[j]);   // time - 1 (any pad), and pad - 1 at the same time
      if (j > 4) peak = peak && (a >= b[j]);
      S += b[j];
      Sp += b[j] * dp;
      St += b[j] * dt;
    }
    if (!peak) continue;
    const int idx = atomicAdd(n_clusters, 1);
    if (idx >= max_clusters) continue;
    const int sector = s / nrows, r = s - sector * nrows;
    const float fp = (float)Sp / (float)S, ft = (float)St / (float)S;
    const float yc = (((float)p0 + 0.5f) + fp) * pad_width - g.row.ymax[r];
    const float zeta = (((float)t0 + 0.5f) + ft) * time_width + g.s.z_lo;
    y[idx] = yc;
    z[idx] = sector < 18 ? zeta : -zeta;
    q[idx] = (float)S;
    out_sr[idx] = s;
    out_pad[idx] = p0;
    out_time[idx] = t0;
  }
}

__global__ void k_cluster_count(int64_t max_clusters, int32_t* __restrict__ n_clusters) {
  const int found = n_clusters[0];
  n_clusters[1] = found < max_clusters ? found : (int)max_clusters;
}

inline unsigned long long table_slots(int64_t n) {
  unsigned long long s = 1024;
  while (s < 2ull * (unsigned long long)(n > 0 ? n : 0)) s <<= 1;
  return s;
}

}  // namespace

size_t cluster_ws_bytes(int64_t n_digits) {
  const unsigned long long slots = table_slots(n_digits);
  return align256(sizeof(unsigned long long) * slots) + align256(sizeof(int32_t) * slots);
}

cudaError_t launch_clusterize(const Geo& g, int64_t n, const int32_t* sr, const int32_t* pad, const int32_t* tim,
                              const int32_t* adc, float pad_width, float time_width, int peak_min, void* workspace,
                              int64_t max_clusters, float* y, float* z, float* q, int32_t* out_sr, int32_t* out_pad,
                              int32_t* out_time, int32_t* n_clusters, cudaStream_t st) {
  const unsigned long long slots = table_slots(n);
  unsigned long long* keys = (unsigned long long*)workspace;
  int32_t* vals = (int32_t*)((char*)workspace + align256(sizeof(unsigned long long) * slots));
  cudaError_t e;
  if ((e = cudaMemsetAsync(keys, 0xFF, sizeof(unsigned long long) * slots, st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(vals, 0, sizeof(int32_t) * slots, st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(n_clusters, 0, sizeof(int32_t) * 2, st)) != cudaSuccess) return e;
  if (n > 0)
    TPC_LAUNCH(KID_CLUSTERIZE, st,
               (k_digit_insert<<<blocks_for(n, kThreads), kThreads, 0, st>>>(n, g.s.nsec * g.s.nrows, sr, pad, tim, adc, keys, vals,
                                                                            slots - 1)));
  TPC_LAUNCH(KID_CLUSTERIZE, st,
             (k_digit_peaks<<<blocks_for((int64_t)slots, kThreads), kThreads, 0, st>>>(g, keys, vals, slots - 1, pad_width, time_width,
                                                                                      peak_min, max_clusters, y, z, q, out_sr,
                                                                                      out_pad, out_time, n_clusters)));
  TPC_LAUNCH(KID_CLUSTERIZE, st, (k_cluster_count<<<1, 1, 0, st>>>(max_clusters, n_clusters)));
  return cudaGetLastError();
}

}  // namespace tpc
