// =============================================================================================
// tpc_merge.cu -- the step right after the hot path ("full tracking in
// the TPC", l.60; R26): merging of the sector-local tracks across the 20-degree sector edges,
// across the central electrode and across holes longer than max_gap, and the refit of the merged hit lists.
//
//   k_merge_ends     per track: rows of its first / last hit (from the hit records tpc_find_tracks cached), z of
//                    its inner end, bucket (sector, z slab, group of 8 first rows) of that end; bucket histogram
//   k_merge_scatter  end records into bucket order (the order inside a bucket is irrelevant: every arg-min below
//                    breaks ties by seed)
//   k_merge_scan     one thread per track A: every track B whose inner end lies in the buckets the R26 windows can
//                    reach is put to the tests that need no arithmetic on the states -- row window, z window,
//                    (tanlambda, q/pT) gate -- on its 32-byte end record; the survivors (nearly always the true
//                    continuation and nobody else) are appended to a pair list
//   k_merge_eval     one thread per pair: A's outer state by R12, rotation into B's frame, transport to B's first
//                    hit, Cholesky chi2; a pair under the cut offers (chi2, seed of B) to A and (chi2, seed of A) to
//                    B by 64-bit atomicMin: the best successor / predecessor (ties: lowest seed)
//   k_merge_link     one thread per pair: it is A's best successor iff A's key is its own; A -> B is a link iff B's
//                    key is the pair's too (reciprocal arg-mins)
//   k_merge_chains   heads (no predecessor) are numbered by a scan; each walks its chain: trk_global, pieces, hits;
//                    a track without links keeps its sector-local fit
//   k_merge_refit    one thread per merged chain: R22's two passes over the concatenated hit records, with the
//                    frame rotation at a change of sector and the zRef re-basing at a change of side
//
// The arithmetic restates R26 operator by operator in fp32 (the library is compiled with -fmad=false; R26 has no
// mad), so the integer decisions (links) and the merged parameters equal the CPU oracle's bit for bit.
// =============================================================================================
#include "tpc_common.cuh"
#include "tpc_kalman.cuh"
#include "tpc_prof.cuh"
#include "tpc_scan.cuh"

#include <cstring>

namespace tpc {

namespace {

constexpr int kThreads = 128;
constexpr float kSlabCm = 128.0f;  // z slab of the end buckets (>= dz_max is not required: the lookup covers a range)
constexpr int kRowGroups = 19;     // first rows in groups of 8: a bucket is (sector, z slab, row group)
constexpr float kSlabEps = 0.01f;  // cm; widens a z lookup beyond any rounding of its fp32 window test
constexpr float kCos20 = 0.93969262078590838405f, kSin20 = 0.34202014332566873304f;
enum { REL_NONE = 0, REL_SAME = 1, REL_NEXT = 2, REL_PREV = 3, REL_CE = 4 };

struct MergeP {
  float chi2_cut, dz_max, ce_tol;
  int max_rows;
  int nslab;  // z slabs per sector
};

// inner end of a track, in bucket order: all the R26 windows need before the states are touched
struct EndRec {
  float z_in;   // zRef + dz at the innermost hit
  int rows;     // first row | last row << 8 | sector << 16
  int seed;     // original index of the start hit: tie-break
  int track;    // index of the track
  float tanl, qpt, c33, c44;  // the gate of R26: tanlambda, q/pT and their variances
};

struct MergeWs {
  EndRec* ends;       // [K] bucket order
  int32_t* bucket;    // [K] bucket of track k
  int32_t* bfirst;    // [nbuckets + 2]
  int32_t* bcursor;   // [nbuckets + 2]
  int32_t* rows;      // [K] first | last << 8 | sector << 16, track order
  float* z_in;        // [K]
  unsigned long long* succ_key;  // [K] (chi2 bits << 32 | seed of the best successor)
  unsigned long long* pred_key;  // [K] (chi2 bits << 32 | seed of the best predecessor)
  int32_t* pair_a;    // [pair_cap] pairs that passed the windows and the gate: track A,
  int32_t* pair_b;    //            track B | relation << 28,
  float* pair_chi2;   //            chi2 (-1: impossible or above the cut)
  int32_t* n_pairs;   // [1]
  int64_t pair_cap;
  int32_t* flag;      // [K + 1] head flags and their scan
  int32_t* mlist;     // [K] global tracks of more than one piece (any order); mlist[K] = their number
  int32_t* scan_tmp;
};

__device__ __forceinline__ int sector_relation(int sa, int sb) {
  if (sa == sb) return REL_SAME;
  const int aa = sa % 18, ab = sb % 18;
  if ((sa < 18) != (sb < 18)) return aa == ab ? REL_CE : REL_NONE;
  if (ab == (aa + 1) % 18) return REL_NEXT;
  if (aa == (ab + 1) % 18) return REL_PREV;
  return REL_NONE;
}

__device__ __forceinline__ int slab_of(float zeta, float z_lo, int nslab) {
  const float v = (zeta - z_lo) * (1.0f / kSlabCm);
  if (!(v > 0.0f)) return 0;
  if (v >= (float)nslab) return nslab - 1;
  return (int)v;
}

__device__ __forceinline__ void load_state(KState& st, const float* __restrict__ par, const float* __restrict__ cov, int64_t ld,
                                           int64_t k) {
#pragma unroll
  for (int i = 0; i < 5; i++) st.p[i] = __ldg(par + i * ld + k);
#pragma unroll
  for (int i = 0; i < 15; i++) st.C[i] = __ldg(cov + i * ld + k);
}

// R26 rotation of a state at x into the frame turned by D (cd = cos D, sd = sin D)
__device__ __forceinline__ bool rotate_state(KState& st, float& x, float cd, float sd, float max_sinphi) {
  const float y = st.p[0], s = st.p[2];
  const float c = sqrtf(1.0f - s * s);
  const float xn = x * cd + y * sd;
  const float yn = y * cd - x * sd;
  const float sn = s * cd - c * sd;
  const float cn = c * cd + s * sd;
  if (!(cn > 0.0f) || !(fabsf(sn) <= max_sinphi)) return false;
  const float j0 = c / cn, j2 = cn / c;
  // C'_ij = (J_i C_ij) J_j with J = (j0, 1, j2, 1, 1); a factor 1 changes nothing
  st.C[TPC_CI(0, 0)] = (j0 * st.C[TPC_CI(0, 0)]) * j0;
  st.C[TPC_CI(1, 0)] = st.C[TPC_CI(1, 0)] * j0;
  st.C[TPC_CI(2, 0)] = (j2 * st.C[TPC_CI(2, 0)]) * j0;
  st.C[TPC_CI(2, 1)] = j2 * st.C[TPC_CI(2, 1)];
  st.C[TPC_CI(2, 2)] = (j2 * st.C[TPC_CI(2, 2)]) * j2;
  st.C[TPC_CI(3, 0)] = st.C[TPC_CI(3, 0)] * j0;
  st.C[TPC_CI(3, 2)] = st.C[TPC_CI(3, 2)] * j2;
  st.C[TPC_CI(4, 0)] = st.C[TPC_CI(4, 0)] * j0;
  st.C[TPC_CI(4, 2)] = st.C[TPC_CI(4, 2)] * j2;
  st.p[0] = yn;
  st.p[2] = sn;
  x = xn;
  return true;
}

// chi2 = d^T S^-1 d over N of the 5 parameters (index map idx), S = lower triangle of a + lower triangle of b
template <int N>
__device__ __forceinline__ float chi2_cholesky(const float (&Sa)[15], const float (&Sb)[15], const float (&d)[5], const int (&idx)[N]) {
  float L[N][N], yv[N];
#pragma unroll
  for (int i = 0; i < N; i++) {
#pragma unroll
    for (int j = 0; j <= i; j++) {
      float sum = Sa[TPC_CI(idx[i], idx[j])] + Sb[TPC_CI(idx[i], idx[j])];
#pragma unroll
      for (int k = 0; k < j; k++) sum = sum - L[i][k] * L[j][k];
      if (i == j) {
        if (!(sum > 0.0f)) return -1.0f;
        L[i][i] = sqrtf(sum);
      } else {
        L[i][j] = sum / L[j][j];
      }
    }
  }
  float chi2 = 0.0f;
#pragma unroll
  for (int i = 0; i < N; i++) {
    float sum = d[idx[i]];
#pragma unroll
    for (int k = 0; k < i; k++) sum = sum - L[i][k] * yv[k];
    yv[i] = sum / L[i][i];
    chi2 = chi2 + yv[i] * yv[i];
  }
  return chi2;
}

__global__ void __launch_bounds__(kThreads)
k_merge_ends(const __grid_constant__ Geo g, MergeP mp, const int32_t* __restrict__ counters, int64_t max_tracks,
             const int32_t* __restrict__ trk_seed, const int32_t* __restrict__ trk_sector, const int32_t* __restrict__ trk_nhits,
             const int64_t* __restrict__ trk_first_hit, const float4* __restrict__ hit_rec, const float* __restrict__ par,
             const float* __restrict__ zref, MergeWs w) {
  int64_t K = counters[TPC_CNT_TRACKS];
  if (K > max_tracks) K = max_tracks;
  for (int64_t k = (int64_t)blockIdx.x * kThreads + threadIdx.x; k < K; k += (int64_t)gridDim.x * kThreads) {
    const int64_t f = trk_first_hit[k];
    const int n = trk_nhits[k], s = trk_sector[k];
    const int rf = __float_as_int(__ldg(hit_rec + f).z), rl = __float_as_int(__ldg(hit_rec + f + n - 1).z);
    const float z = zref[k] + par[1 * max_tracks + k];
    const float zeta = s < 18 ? z : -z;
    const int b = (s * mp.nslab + slab_of(zeta, g.s.z_lo, mp.nslab)) * kRowGroups + (rf >> 3);
    w.rows[k] = rf | (rl << 8) | (s << 16);
    w.z_in[k] = z;
    w.bucket[k] = b;
    w.succ_key[k] = ~0ull;
    w.pred_key[k] = ~0ull;
    atomicAdd(w.bfirst + b, 1);
  }
}

__global__ void __launch_bounds__(kThreads)
k_merge_scatter(const int32_t* __restrict__ counters, int64_t max_tracks, const int32_t* __restrict__ trk_seed,
                const float* __restrict__ par, const float* __restrict__ cov, MergeWs w) {
  int64_t K = counters[TPC_CNT_TRACKS];
  if (K > max_tracks) K = max_tracks;
  for (int64_t k = (int64_t)blockIdx.x * kThreads + threadIdx.x; k < K; k += (int64_t)gridDim.x * kThreads) {
    const int slot = atomicAdd(w.bcursor + w.bucket[k], 1);
    EndRec e;
    e.z_in = w.z_in[k];
    e.rows = w.rows[k];
    e.seed = trk_seed[k];
    e.track = (int)k;
    float4* dst = reinterpret_cast<float4*>(w.ends + slot);
    dst[0] = make_float4(e.z_in, __int_as_float(e.rows), __int_as_float(e.seed), __int_as_float(e.track));
    dst[1] = make_float4(par[3 * max_tracks + k], par[4 * max_tracks + k], cov[TPC_CI(3, 3) * max_tracks + k],
                         cov[TPC_CI(4, 4) * max_tracks + k]);
  }
}

// chi2 of "B follows A" for a pair that passed the windows and the gate (R26); -1 = impossible
__device__ __forceinline__ float pair_chi2(const KState& out, float x_a, float zref_a, int rel, int b, int rf_b, const float* sX,
                                           const float* __restrict__ par, const float* __restrict__ cov,
                                           const float* __restrict__ zref, int64_t max_tracks, float kB, float ms, float ce_tol) {
  KState r = out;
  float x = x_a;
  if (rel == REL_NEXT || rel == REL_PREV) {
    const float sd = rel == REL_NEXT ? kSin20 : -kSin20;
    if (!rotate_state(r, x, kCos20, sd, ms)) return -1.0f;
  }
  const float xb = sX[rf_b];
  if (!propagate(r, xb - x, kB, ms)) return -1.0f;
  KState sbst;
  load_state(sbst, par, cov, max_tracks, b);
  const float zref_b = zref[b];
  float d[5];
  d[0] = r.p[0] - sbst.p[0];
  d[1] = (zref_a - zref_b) + (r.p[1] - sbst.p[1]);
  d[2] = r.p[2] - sbst.p[2];
  d[3] = r.p[3] - sbst.p[3];
  d[4] = r.p[4] - sbst.p[4];
  if (rel == REL_CE) {
    const float zsum = (zref_a + r.p[1]) + (zref_b + sbst.p[1]);
    const float cb = sqrtf(1.0f - sbst.p[2] * sbst.p[2]);
    const float lim = ce_tol + ((2.0f * fabsf(sbst.p[3])) * (xb - x_a)) / cb;
    if (!(fabsf(zsum) <= lim)) return -1.0f;
    const int idx[4] = {0, 2, 3, 4};
    return chi2_cholesky<4>(r.C, sbst.C, d, idx);
  }
  const int idx[5] = {0, 1, 2, 3, 4};
  return chi2_cholesky<5>(r.C, sbst.C, d, idx);
}

__device__ __forceinline__ unsigned long long chi2_key(float chi2, int seed) {
  return ((unsigned long long)__float_as_uint(chi2) << 32) | (unsigned long long)(unsigned)seed;  // chi2 >= 0: ordered as uint
}

// chi2 of one pair and its offers to both ends (R26 arbitration)
__device__ __forceinline__ float eval_pair(const MergeP& mp, const float* sX, int a, int b, int rel, int rows_a, int rf_b,
                                           const int32_t* __restrict__ trk_seed, const float* __restrict__ par,
                                           const float* __restrict__ cov, const float* __restrict__ zref, int64_t max_tracks,
                                           float kB, float ms, const MergeWs& w) {
  const int rf_a = rows_a & 0xff, rl_a = (rows_a >> 8) & 0xff;
  KState out;
  load_state(out, par, cov, max_tracks, a);
  if (rl_a != rf_a && !propagate(out, sX[rl_a] - sX[rf_a], kB, ms)) return -1.0f;
  const float chi2 = pair_chi2(out, sX[rl_a], zref[a], rel, b, rf_b, sX, par, cov, zref, max_tracks, kB, ms, mp.ce_tol);
  if (!(chi2 >= 0.0f) || !(chi2 < mp.chi2_cut)) return -1.0f;
  atomicMin(w.succ_key + a, chi2_key(chi2, trk_seed[b]));
  atomicMin(w.pred_key + b, chi2_key(chi2, trk_seed[a]));
  return chi2;
}

__global__ void __launch_bounds__(kThreads)
k_merge_scan(const __grid_constant__ Geo g, MergeP mp, const int32_t* __restrict__ counters, int64_t max_tracks,
             const int32_t* __restrict__ trk_seed, const float* __restrict__ par, const float* __restrict__ cov, const float* __restrict__ zref, MergeWs w) {
  __shared__ float sX[kMaxRows];
  const Scalars& sc = g.s;
  for (int r = threadIdx.x; r < sc.nrows; r += blockDim.x) sX[r] = g.row.X[r];
  __syncthreads();
  int64_t K = counters[TPC_CNT_TRACKS];
  if (K > max_tracks) K = max_tracks;
  const float kB = sc.kB, ms = sc.max_sinphi;
  const float gate = 4.0f * mp.chi2_cut;
  for (int64_t a = (int64_t)blockIdx.x * kThreads + threadIdx.x; a < K; a += (int64_t)gridDim.x * kThreads) {
    const int rows_a = w.rows[a];
    const int rf_a = rows_a & 0xff, rl_a = (rows_a >> 8) & 0xff, s_a = rows_a >> 16;
    // what the tests need of A's outer state: dz (transported), tanlambda and q/pT with their variances (unchanged by R12)
    float dz_out = par[1 * max_tracks + a];
    const float tl_a = par[3 * max_tracks + a], q_a = par[4 * max_tracks + a];
    const float c33_a = cov[TPC_CI(3, 3) * max_tracks + a], c44_a = cov[TPC_CI(4, 4) * max_tracks + a];
    if (rl_a != rf_a) {
      KState st;
      load_state(st, par, cov, max_tracks, a);
      Transport T;
      if (!transport_state(st, sX[rl_a] - sX[rf_a], kB, ms, T)) continue;  // no outer state: A has no successor
      dz_out = T.dz;
    }
    const float zA = zref[a] + dz_out;
    const int g0 = (rl_a + 1) >> 3;
    int g1 = (rl_a + mp.max_rows) >> 3;
    if (g1 > kRowGroups - 1) g1 = kRowGroups - 1;
    if (g0 > g1) continue;
    for (int sb = 0; sb < sc.nsec; sb++) {
      const int rel = sector_relation(s_a, sb);
      if (rel == REL_NONE) continue;
      // z of B's inner end: within dz_max of zA (same side) or of -zA (across the electrode); as zeta of B's side
      const float zc = rel == REL_CE ? -zA : zA;
      const float side_b = sb < 18 ? 1.0f : -1.0f;
      const float za = (zc - (mp.dz_max + kSlabEps)) * side_b, zb = (zc + (mp.dz_max + kSlabEps)) * side_b;
      const int s0 = slab_of(fminf(za, zb), sc.z_lo, mp.nslab), s1 = slab_of(fmaxf(za, zb), sc.z_lo, mp.nslab);
      for (int sl = s0; sl <= s1; sl++) {
        // first rows rl_a + 1 .. rl_a + max_rows: a contiguous run of row groups inside every (sector, slab)
        const int bb = (sb * mp.nslab + sl) * kRowGroups;
        const int e0 = w.bfirst[bb + g0], e1 = w.bfirst[bb + g1 + 1];
        for (int e = e0; e < e1; e++) {
          const float4 er = __ldg(reinterpret_cast<const float4*>(w.ends + e));
          const int rows_b = __float_as_int(er.y), b = __float_as_int(er.w);
          const int rf_b = rows_b & 0xff;
          const int dr = rf_b - rl_a;
          if (dr < 1 || dr > mp.max_rows || b == (int)a) continue;
          const float zB = er.x;
          if (rel == REL_CE ? !(fabsf(zB + zA) <= mp.dz_max) : !(fabsf(zB - zA) <= mp.dz_max)) continue;
          const float4 gt = __ldg(reinterpret_cast<const float4*>(w.ends + e) + 1);
          const float d3 = tl_a - gt.x, d4 = q_a - gt.y;
          if (!(d3 * d3 <= gate * (c33_a + gt.z)) || !(d4 * d4 <= gate * (c44_a + gt.w))) continue;
          const int slot = atomicAdd(w.n_pairs, 1);
          if (slot < w.pair_cap) {
            w.pair_a[slot] = (int)a;
            w.pair_b[slot] = b | (rel << 28);
          }  // else: list full (4 survivors per track on average: never seen); counted in n_global[3]
        }
      }
    }
  }
}

__global__ void __launch_bounds__(kThreads)
k_merge_eval(const __grid_constant__ Geo g, MergeP mp, int64_t max_tracks, const int32_t* __restrict__ trk_seed,
             const float* __restrict__ par, const float* __restrict__ cov, const float* __restrict__ zref, MergeWs w) {
  __shared__ float sX[kMaxRows];
  const Scalars& sc = g.s;
  for (int r = threadIdx.x; r < sc.nrows; r += blockDim.x) sX[r] = g.row.X[r];
  __syncthreads();
  int64_t np = w.n_pairs[0];
  if (np > w.pair_cap) np = w.pair_cap;
  for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < np; i += (int64_t)gridDim.x * kThreads) {
    const int a = w.pair_a[i], pb = w.pair_b[i];
    const int b = pb & 0x0fffffff, rel = pb >> 28;
    w.pair_chi2[i] = eval_pair(mp, sX, a, b, rel, w.rows[a], w.rows[b] & 0xff, trk_seed, par, cov, zref, max_tracks, sc.kB,
                               sc.max_sinphi, w);
  }
}

__global__ void __launch_bounds__(kThreads)
k_merge_link(const int32_t* __restrict__ trk_seed, MergeWs w, float* __restrict__ succ_chi2, int32_t* __restrict__ succ,
             int32_t* __restrict__ pred) {
  int64_t np = w.n_pairs[0];
  if (np > w.pair_cap) np = w.pair_cap;
  for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < np; i += (int64_t)gridDim.x * kThreads) {
    const float chi2 = w.pair_chi2[i];
    if (!(chi2 >= 0.0f)) continue;
    const int a = w.pair_a[i], b = w.pair_b[i] & 0x0fffffff;
    if (w.succ_key[a] != chi2_key(chi2, trk_seed[b])) continue;
    succ_chi2[a] = chi2;  // B is A's best candidate successor ...
    if (w.pred_key[b] == chi2_key(chi2, trk_seed[a])) {  // ... and A is B's best candidate predecessor: a link
      succ[a] = b;
      pred[b] = a;
    }
  }
}

__global__ void __launch_bounds__(kThreads)
k_merge_heads(const int32_t* __restrict__ counters, int64_t max_tracks, const int32_t* __restrict__ pred, int32_t* __restrict__ flag) {
  int64_t K = counters[TPC_CNT_TRACKS];
  if (K > max_tracks) K = max_tracks;
  for (int64_t k = (int64_t)blockIdx.x * kThreads + threadIdx.x; k <= max_tracks; k += (int64_t)gridDim.x * kThreads)
    flag[k] = (k < K && pred[k] < 0) ? 1 : 0;
}

__global__ void __launch_bounds__(kThreads)
k_merge_chains(const int32_t* __restrict__ counters, int64_t max_tracks, const int32_t* __restrict__ trk_nhits,
               const float* __restrict__ par, const float* __restrict__ cov, const float* __restrict__ xref,
               const float* __restrict__ zref, const float* __restrict__ chi2, const int32_t* __restrict__ ndf,
               const int32_t* __restrict__ succ, const int32_t* __restrict__ pred, const int32_t* __restrict__ scan,
               int32_t* __restrict__ trk_global, int32_t* __restrict__ n_global, int32_t* __restrict__ g_head,
               int32_t* __restrict__ g_nseg, int32_t* __restrict__ g_nhits, float* __restrict__ gpar, float* __restrict__ gcov,
               float* __restrict__ gxref, float* __restrict__ gzref, float* __restrict__ gchi2, int32_t* __restrict__ gndf,
               int32_t* __restrict__ mlist, const int32_t* __restrict__ n_pairs, int64_t pair_cap) {
  int64_t K = counters[TPC_CNT_TRACKS];
  if (K > max_tracks) K = max_tracks;
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    n_global[0] = scan[max_tracks];
    n_global[1] = (int)K - scan[max_tracks];  // links
    n_global[2] = n_pairs[0];                 // pairs that passed the windows and the gate
    n_global[3] = n_pairs[0] > pair_cap ? (int)(n_pairs[0] - pair_cap) : 0;  // ... of which not tested (list full)
  }
  for (int64_t h = (int64_t)blockIdx.x * kThreads + threadIdx.x; h < K; h += (int64_t)gridDim.x * kThreads) {
    if (pred[h] >= 0) continue;
    const int gi = scan[h];
    int nseg = 0, nh = 0;
    for (int k = (int)h; k >= 0; k = succ[k]) {
      trk_global[k] = gi;
      nseg++;
      nh += trk_nhits[k];
    }
    g_head[gi] = (int)h;
    g_nseg[gi] = nseg;
    g_nhits[gi] = nh;
    if (nseg == 1) {  // no links: the sector-local fit stands
#pragma unroll
      for (int i = 0; i < 5; i++) gpar[i * max_tracks + gi] = par[i * max_tracks + h];
#pragma unroll
      for (int i = 0; i < 15; i++) gcov[i * max_tracks + gi] = cov[i * max_tracks + h];
      gxref[gi] = xref[h];
      gzref[gi] = zref[h];
      gchi2[gi] = chi2[h];
      gndf[gi] = ndf[h];
    } else {
      mlist[atomicAdd(mlist + max_tracks, 1)] = gi;
    }
  }
}

// R26 refit of one chain per thread.  The hits of a chain are walked piece by piece in the direction of the pass: `k` / `i`
// address the current hit, succ[] leads to the next piece on the way out and pred[] on the way in, so a chain may have
// any number of pieces (holes longer than max_gap inside one sector give one piece each; with a small min_hits that is
// dozens).

__global__ void __launch_bounds__(kThreads)
k_merge_refit(const __grid_constant__ Geo g, const int32_t* __restrict__ n_global, int64_t max_tracks,
              const int32_t* __restrict__ trk_sector, const int32_t* __restrict__ trk_nhits,
              const int64_t* __restrict__ trk_first_hit, const float4* __restrict__ hit_rec, const float* __restrict__ par,
              const float* __restrict__ zref, const int32_t* __restrict__ succ, const int32_t* __restrict__ pred,
              const int32_t* __restrict__ g_head,
              const int32_t* __restrict__ g_nseg, const int32_t* __restrict__ g_nhits, float* __restrict__ gpar,
              float* __restrict__ gcov, float* __restrict__ gxref, float* __restrict__ gzref, float* __restrict__ gchi2,
              int32_t* __restrict__ gndf, const int32_t* __restrict__ mlist) {
  __shared__ float sX[kMaxRows];
  const Scalars& sc = g.s;
  for (int r = threadIdx.x; r < sc.nrows; r += blockDim.x) sX[r] = g.row.X[r];
  __syncthreads();
  (void)n_global;
  const int M = mlist[max_tracks];
  const float kB = sc.kB, ms = sc.max_sinphi, sy2 = sc.sy2, sz2 = sc.sz2;
  for (int64_t li = (int64_t)blockIdx.x * kThreads + threadIdx.x; li < M; li += (int64_t)gridDim.x * kThreads) {
    const int gi = mlist[li];
    const int h = g_head[gi];
    int tail = h;
    for (int k = succ[h]; k >= 0; k = succ[k]) tail = k;
    bool ok = true;
    KState st;
#pragma unroll
    for (int i = 0; i < 5; i++) st.p[i] = par[i * max_tracks + h];
#pragma unroll
    for (int i = 0; i < 15; i++) st.C[i] = 0.0f;
    float zr = zref[h];
    int cur_sec = trk_sector[h];
    float x_at = sX[__float_as_int(__ldg(hit_rec + trk_first_hit[h]).z)];
    float c2 = 0.0f;
    int lost = 0;
    const int N = g_nhits[gi];
    for (int pass = 0; pass < sc.n_fit_passes && ok; pass++) {
      reset_cov(st, sc.cov0);
      c2 = 0.0f;
      lost = 0;
      const int dir = (pass & 1) ? -1 : 1;
      int k = dir > 0 ? h : tail;
      int i = dir > 0 ? 0 : trk_nhits[k] - 1;
      for (int cnt = 0; cnt < N && ok; cnt++) {
        const float4 hit = __ldg(hit_rec + trk_first_hit[k] + i);
        const int hs = trk_sector[k];
        const float xh = sX[__float_as_int(hit.z)];
        bool rebase = false;
        if (hs != cur_sec) {
          const int rel = sector_relation(cur_sec, hs);
          if (rel == REL_NEXT || rel == REL_PREV) {
            const float cd = kCos20, sd = rel == REL_NEXT ? kSin20 : -kSin20;
            if (dir < 0) {  // inward: stay in the old frame up to the plane of the next hit (R26)
              const float xc = xh * cd - hit.x * sd;
              if (!propagate(st, xc - x_at, kB, ms)) { ok = false; break; }
              x_at = xc;
            }
            if (!rotate_state(st, x_at, cd, sd, ms)) { ok = false; break; }
          } else if (rel == REL_CE) {
            rebase = true;
          }
          cur_sec = hs;
        }
        if (cnt > 0) {
          if (!propagate(st, xh - x_at, kB, ms)) { ok = false; break; }
          x_at = xh;
        }
        if (rebase) {
          zr = hit.y - st.p[1];
          lost++;
        }
        const Innov I = innovation(st, sy2, sz2);
        c2 = c2 + update(st, I, hit.x, hit.y - zr);
        // next hit in the direction of the pass
        i += dir;
        if (i < 0 || i >= trk_nhits[k]) {
          const int nk = dir > 0 ? succ[k] : pred[k];
          if (nk >= 0) {
            k = nk;
            i = dir > 0 ? 0 : trk_nhits[k] - 1;
          }
        }
      }
    }
#pragma unroll
    for (int i = 0; i < 5; i++) gpar[i * max_tracks + gi] = st.p[i];
#pragma unroll
    for (int i = 0; i < 15; i++) gcov[i * max_tracks + gi] = st.C[i];
    gxref[gi] = x_at;
    gzref[gi] = zr;
    gchi2[gi] = ok ? c2 : -1.0f;
    gndf[gi] = ok ? 2 * N - 5 - lost : -1;
  }
}

__global__ void __launch_bounds__(256) k_fill_u32(unsigned* p, unsigned v, size_t n) {
  for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (size_t)gridDim.x * 256) p[i] = v;
}
inline cudaError_t cudaMemsetD32Async_compat(void* p, unsigned v, size_t n, cudaStream_t st) {
  k_fill_u32<<<blocks_for((int64_t)n, 256, 148 * 8), 256, 0, st>>>((unsigned*)p, v, n);
  return cudaGetLastError();
}

inline int merge_nslab(const Geo& g) {
  int n = (int)ceilf((g.s.z_hi - g.s.z_lo) / kSlabCm) + 1;
  if (n < 1) n = 1;
  if (n > 4096) n = 4096;
  return n;
}

struct MergeLayout {
  size_t off_ends, off_bucket, off_bfirst, off_bcursor, off_rows, off_z, off_skey, off_key, off_flag, off_mlist, off_pa, off_pb, off_pc, off_np, off_tmp, total;
  int64_t pair_cap;
  int64_t nbuckets;
};

inline MergeLayout merge_layout(int nsec, int nslab, int64_t max_tracks) {
  MergeLayout L{};
  L.nbuckets = (int64_t)nsec * nslab * kRowGroups;
  size_t o = 0;
  auto take = [&](size_t bytes) {
    size_t at = o;
    o = align256(o + bytes);
    return at;
  };
  const size_t K = (size_t)max_tracks + 1;
  L.off_ends = take(sizeof(EndRec) * K);
  L.off_bucket = take(sizeof(int32_t) * K);
  L.off_bfirst = take(sizeof(int32_t) * (size_t)(L.nbuckets + 2));
  L.off_bcursor = take(sizeof(int32_t) * (size_t)(L.nbuckets + 2));
  L.off_rows = take(sizeof(int32_t) * K);
  L.off_z = take(sizeof(float) * K);
  L.off_skey = take(sizeof(unsigned long long) * K);
  L.off_key = take(sizeof(unsigned long long) * K);
  L.off_flag = take(sizeof(int32_t) * (K + 1));
  L.off_mlist = take(sizeof(int32_t) * (K + 1));
  L.pair_cap = 4 * max_tracks;  // pairs that pass the windows and the gate: one or two per track that has any
  L.off_pa = take(sizeof(int32_t) * (size_t)L.pair_cap);
  L.off_pb = take(sizeof(int32_t) * (size_t)L.pair_cap);
  L.off_pc = take(sizeof(float) * (size_t)L.pair_cap);
  L.off_np = take(sizeof(int32_t) * 4);
  const int64_t longest = (int64_t)K + 1 > L.nbuckets + 2 ? (int64_t)K + 1 : L.nbuckets + 2;
  L.off_tmp = take(sizeof(int64_t) * (size_t)((longest + kScanTile - 1) / kScanTile + 2));
  L.total = o;
  return L;
}

}  // namespace

size_t merge_ws_bytes(const Geo& g, int64_t max_tracks) { return merge_layout(g.s.nsec, merge_nslab(g), max_tracks).total; }

cudaError_t launch_merge(const Geo& g, const Ws& fw, float chi2_cut, float dz_max, float ce_tol, int max_rows,
                         const int32_t* counters, int64_t max_tracks, const int32_t* trk_seed, const int32_t* trk_sector,
                         const int32_t* trk_nhits, const int64_t* trk_first_hit, const float* par, const float* cov,
                         const float* xref, const float* zref, const float* chi2, const int32_t* ndf, void* merge_ws,
                         int32_t* trk_succ, int32_t* trk_pred, float* trk_succ_chi2, int32_t* trk_global, int32_t* n_global,
                         int32_t* g_head, int32_t* g_nseg, int32_t* g_nhits, float* gpar, float* gcov, float* gxref,
                         float* gzref, float* gchi2, int32_t* gndf, cudaStream_t st) {
  MergeP mp;
  mp.chi2_cut = chi2_cut;
  mp.dz_max = dz_max;
  mp.ce_tol = ce_tol;
  mp.max_rows = max_rows;
  mp.nslab = merge_nslab(g);
  const MergeLayout L = merge_layout(g.s.nsec, mp.nslab, max_tracks);
  char* b = (char*)merge_ws;
  MergeWs w;
  w.ends = (EndRec*)(b + L.off_ends);
  w.bucket = (int32_t*)(b + L.off_bucket);
  w.bfirst = (int32_t*)(b + L.off_bfirst);
  w.bcursor = (int32_t*)(b + L.off_bcursor);
  w.rows = (int32_t*)(b + L.off_rows);
  w.z_in = (float*)(b + L.off_z);
  w.succ_key = (unsigned long long*)(b + L.off_skey);
  w.pair_a = (int32_t*)(b + L.off_pa);
  w.pair_b = (int32_t*)(b + L.off_pb);
  w.pair_chi2 = (float*)(b + L.off_pc);
  w.n_pairs = (int32_t*)(b + L.off_np);
  w.pair_cap = L.pair_cap;
  w.pred_key = (unsigned long long*)(b + L.off_key);
  w.flag = (int32_t*)(b + L.off_flag);
  w.mlist = (int32_t*)(b + L.off_mlist);
  w.scan_tmp = (int32_t*)(b + L.off_tmp);
  cudaError_t e;
  const unsigned blocks = blocks_for(max_tracks, kThreads, 148 * 16);
  if ((e = cudaMemsetAsync(w.bfirst, 0, sizeof(int32_t) * (size_t)(L.nbuckets + 2), st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(trk_pred, 0xFF, sizeof(int32_t) * (size_t)max_tracks, st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(w.mlist + max_tracks, 0, sizeof(int32_t), st)) != cudaSuccess) return e;
  TPC_LAUNCH(KID_MERGE, st,
             (k_merge_ends<<<blocks, kThreads, 0, st>>>(g, mp, counters, max_tracks, trk_seed, trk_sector, trk_nhits, trk_first_hit,
                                                       fw.hit_rec, par, zref, w)));
  if ((e = exclusive_scan<int32_t>(w.bfirst, w.bfirst, L.nbuckets + 1, w.scan_tmp, st)) != cudaSuccess) return e;
  if ((e = cudaMemcpyAsync(w.bcursor, w.bfirst, sizeof(int32_t) * (size_t)(L.nbuckets + 1), cudaMemcpyDeviceToDevice, st)) !=
      cudaSuccess)
    return e;
  TPC_LAUNCH(KID_MERGE, st, (k_merge_scatter<<<blocks, kThreads, 0, st>>>(counters, max_tracks, trk_seed, par, cov, w)));
  if ((e = cudaMemsetAsync(w.n_pairs, 0, sizeof(int32_t), st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(trk_succ, 0xFF, sizeof(int32_t) * (size_t)max_tracks, st)) != cudaSuccess) return e;
  {
    const float minus1 = -1.0f;
    unsigned bits;
    memcpy(&bits, &minus1, sizeof(bits));
    if ((e = cudaMemsetD32Async_compat(trk_succ_chi2, bits, (size_t)max_tracks, st)) != cudaSuccess) return e;
  }
  TPC_LAUNCH(KID_MERGE, st, (k_merge_scan<<<blocks, kThreads, 0, st>>>(g, mp, counters, max_tracks, trk_seed, par, cov, zref, w)));
  const unsigned pblocks = blocks_for(L.pair_cap, kThreads, 148 * 16);
  TPC_LAUNCH(KID_MERGE, st, (k_merge_eval<<<pblocks, kThreads, 0, st>>>(g, mp, max_tracks, trk_seed, par, cov, zref, w)));
  TPC_LAUNCH(KID_MERGE, st, (k_merge_link<<<pblocks, kThreads, 0, st>>>(trk_seed, w, trk_succ_chi2, trk_succ, trk_pred)));
  TPC_LAUNCH(KID_MERGE, st, (k_merge_heads<<<blocks, kThreads, 0, st>>>(counters, max_tracks, trk_pred, w.flag)));
  if ((e = exclusive_scan<int32_t>(w.flag, w.flag, max_tracks + 1, w.scan_tmp, st)) != cudaSuccess) return e;
  TPC_LAUNCH(KID_MERGE, st,
             (k_merge_chains<<<blocks, kThreads, 0, st>>>(counters, max_tracks, trk_nhits, par, cov, xref, zref, chi2, ndf, trk_succ,
                                                         trk_pred, w.flag, trk_global, n_global, g_head, g_nseg, g_nhits, gpar,
                                                         gcov, gxref, gzref, gchi2, gndf, w.mlist, w.n_pairs, w.pair_cap)));
  TPC_LAUNCH(KID_MERGE, st,
             (k_merge_refit<<<blocks, kThreads, 0, st>>>(g, n_global, max_tracks, trk_sector, trk_nhits, trk_first_hit, fw.hit_rec,
                                                        par, zref, trk_succ, trk_pred, g_head, g_nseg, g_nhits, gpar, gcov, gxref, gzref,
                                                        gchi2, gndf, w.mlist)));
  return cudaGetLastError();
}

}  // namespace tpc
