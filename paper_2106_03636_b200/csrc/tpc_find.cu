// =============================================================================================
// tpc_find.cu -- steps 2, 3a and 4 of the hot path (BASELINE.json north_star (2)-(4); SURVEY.md
// §8(c) R9-R20) on the grid built by tpc_grid.cu.  All internal indices are GRID POSITIONS (index
// into the sorted record array); original indices are only used for tie-breaks (R9, R16, R20) and
// in the outputs.
//
//   k_neighbours     R9   one thread per cluster: best (up,down) pair on rows r+1 / r-1
//   k_clean          R10  reciprocal links, start-hit flags            (+ scan, k_compact_starts)
//   k_follow         R11-R18 one thread per start hit: Kalman chain phase, up leg, jump back,
//                    down leg; row_hit table; pushes its 64-bit selection key (R20) onto every
//                    cluster it recorded with atomicMax
//   k_count_kept     R20  hits still owned by the tracklet, accept if >= min_hits (+ int64 scan)
//   k_write_tracks   R20  track list, hit lists (original indices), cluster_track
// =============================================================================================
#include "tpc_common.cuh"
#include "tpc_kalman.cuh"
#include "tpc_scan.cuh"

namespace tpc {

namespace {

constexpr int kThreads = 256;
constexpr int kFollowThreads = 128;

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

// Bins of (sector s, row r) that cover the cm window [ya,yb] x [za,zb] (raw z).  A superset is
// enough (R8): every candidate is re-tested against the exact window by the caller.  The pads
// dominate fp32 rounding of the window edges (|y| < 50 cm: ulp 4e-6; |z| <= 3.3e4 cm: ulp 4e-3).
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

// ---------------------------------------------------------------------------------------------
// R9: cellular-automaton neighbour finder.
// ---------------------------------------------------------------------------------------------
struct SmCa {
  float wu[kMaxRows], iy[kMaxRows], iz[kMaxRows], wyu[kMaxRows], wzu[kMaxRows], wyd[kMaxRows], wzd[kMaxRows];
};

__global__ void __launch_bounds__(kThreads)
k_neighbours(const __grid_constant__ Geo g, int64_t n, const Rec* __restrict__ rec, const int32_t* __restrict__ bin_first,
             int32_t* __restrict__ link_up, int32_t* __restrict__ link_dn) {
  __shared__ SmRow sm;
  __shared__ SmCa ca;
  load_rows(sm, g);
  for (int r = threadIdx.x; r < g.s.nrows; r += blockDim.x) {
    ca.wu[r] = g.ca.wu[r];
    ca.iy[r] = g.ca.iy[r];
    ca.iz[r] = g.ca.iz[r];
    ca.wyu[r] = g.ca.wyu[r];
    ca.wzu[r] = g.ca.wzu[r];
    ca.wyd[r] = g.ca.wyd[r];
    ca.wzd[r] = g.ca.wzd[r];
  }
  __syncthreads();
  const Scalars& sc = g.s;
  const int nrows = sc.nrows;
  for (int64_t p = (int64_t)blockIdx.x * kThreads + threadIdx.x; p < n; p += (int64_t)gridDim.x * kThreads) {
    const Rec h = ld_rec(rec, (int)p);
    const int sr = rec_sr(h);
    const int s = sr / nrows, r = sr - s * nrows;
    int bu = -1, bd = -1;
    if (r >= 1 && r <= nrows - 2) {
      const float yh = h.x, zh = h.y;
      const float wu = ca.wu[r], iy = ca.iy[r], iz = ca.iz[r];
      const float wyu = ca.wyu[r], wzu = ca.wzu[r], wyd = ca.wyd[r], wzd = ca.wzd[r];
      const BinWin WU = bin_window(sm, sc, s, r + 1, yh - wyu, yh + wyu, zh - wzu, zh + wzu);
      const BinWin WD = bin_window(sm, sc, s, r - 1, yh - wyd, yh + wyd, zh - wzd, zh + wzd);
      bool have = false;
      float best = 0.0f;
      int bui = 0, bdi = 0;  // original indices of the best pair (tie-break)
      for (int zu = 0; zu < WU.nzb; zu++) {
        const int b0 = WU.first + zu * WU.ny;
        const int ka = __ldg(bin_first + b0), ke = __ldg(bin_first + b0 + WU.ybspan);
        for (int k = ka; k < ke; k++) {
          const Rec u = ld_rec(rec, k);
          if (!(fabsf(u.x - yh) <= wyu && fabsf(u.y - zh) <= wzu)) continue;
          const int ui = rec_idx(u);
          for (int zd = 0; zd < WD.nzb; zd++) {
            const int c0 = WD.first + zd * WD.ny;
            const int ja = __ldg(bin_first + c0), je = __ldg(bin_first + c0 + WD.ybspan);
            for (int j = ja; j < je; j++) {
              const Rec d = ld_rec(rec, j);
              if (!(fabsf(d.x - yh) <= wyd && fabsf(d.y - zh) <= wzd)) continue;
              const int di = rec_idx(d);
              const float ry = (yh - d.x) - wu * (u.x - d.x);
              const float rz = (zh - d.y) - wu * (u.y - d.y);
              const float D2 = (ry * ry) * iy + (rz * rz) * iz;
              // minimal D2; ties: lowest original u index, then lowest original d index (R9)
              if (!have || D2 < best || (D2 == best && (ui < bui || (ui == bui && di < bdi)))) {
                have = true;
                best = D2;
                bui = ui;
                bdi = di;
                bu = k;
                bd = j;
              }
            }
          }
        }
      }
      if (!(have && best < sc.ca_cut)) bu = bd = -1;
    }
    link_up[p] = bu;
    link_dn[p] = bd;
  }
}

// ---------------------------------------------------------------------------------------------
// R10: reciprocal links and start hits.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads)
k_clean(int64_t n, const int32_t* __restrict__ link_up, const int32_t* __restrict__ link_dn, int32_t* __restrict__ up_c,
        int32_t* __restrict__ flag) {
  for (int64_t p = (int64_t)blockIdx.x * kThreads + threadIdx.x; p <= n; p += (int64_t)gridDim.x * kThreads) {
    if (p == n) {
      flag[p] = 0;  // sentinel so that the exclusive scan leaves the total at [n]
      continue;
    }
    const int u = link_up[p], d = link_dn[p];
    const int uc = (u >= 0 && __ldg(link_dn + u) == (int)p) ? u : -1;
    const int dc = (d >= 0 && __ldg(link_up + d) == (int)p) ? d : -1;
    up_c[p] = uc;
    flag[p] = (uc >= 0 && dc < 0) ? 1 : 0;
  }
}

__global__ void __launch_bounds__(kThreads)
k_compact_starts(int64_t n, int64_t scap, const int32_t* __restrict__ scan, int32_t* __restrict__ starts,
                 int32_t* __restrict__ ws_counters) {
  for (int64_t p = (int64_t)blockIdx.x * kThreads + threadIdx.x; p < n; p += (int64_t)gridDim.x * kThreads) {
    const int t = scan[p];
    if (scan[p + 1] != t && t < scap) starts[t] = (int)p;
    if (p == 0) {
      const int total = scan[n];
      ws_counters[WC_STARTS_FOUND] = total;
      ws_counters[WC_N_STARTS] = total < scap ? total : (int)scap;
      if (total > scap) atomicOr(ws_counters + WC_STATUS, TPC_ST_TRACKLET_OVERFLOW);
    }
  }
}

// ---------------------------------------------------------------------------------------------
// R11-R18: Kalman following, one thread per start hit; R20 key push at the end.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long sel_key(int nh, int start_orig) {
  return ((unsigned long long)(unsigned)nh << 32) | (unsigned long long)(0xFFFFFFFFu - (unsigned)start_orig);
}

__global__ void __launch_bounds__(kFollowThreads)
k_follow(const __grid_constant__ Geo g, const Rec* __restrict__ rec, const int32_t* __restrict__ bin_first,
         const int32_t* __restrict__ up_c, const int32_t* __restrict__ starts, int64_t scap_pad, int32_t* row_hit,
         int32_t* __restrict__ tl_info, unsigned long long* __restrict__ owner, int32_t* __restrict__ ws_counters) {
  __shared__ SmRow sm;
  load_rows(sm, g);
  __syncthreads();
  const Scalars& sc = g.s;
  const int nrows = sc.nrows;
  const int n_starts = ws_counters[WC_N_STARTS];
  const int lane = threadIdx.x & 31;
  const float kB = sc.kB, ms = sc.max_sinphi, sy2 = sc.sy2, sz2 = sc.sz2;
  unsigned long long work[3] = {0ull, 0ull, 0ull};
  for (;;) {
    int base = 0;
    if (lane == 0) base = atomicAdd(ws_counters + WC_QUEUE, 32);
    base = __shfl_sync(0xffffffffu, base, 0);
    if (base >= n_starts) break;
    const int t = base + lane;
    if (t >= n_starts) continue;
    int32_t* my_hits = row_hit + t;  // row r at my_hits[r * scap_pad]
    const int p0 = starts[t];
    const Rec h0 = ld_rec(rec, p0);
    const int sr0 = rec_sr(h0);
    const int s = sr0 / nrows, r0 = sr0 - s * nrows;
    const int p1 = up_c[p0];
    const Rec h1 = ld_rec(rec, p1);
    const int r1 = rec_sr(h1) - s * nrows;
    // R14: initial state from the start hit and its up-neighbour
    KState st;
    const float zref = h0.y;
    {
      const float dx = sm.X[r1] - sm.X[r0], dy = h1.x - h0.x;
      const float ch = sqrtf(dx * dx + dy * dy);
      st.p[0] = h0.x;
      st.p[1] = 0.0f;
      st.p[2] = dy / ch;
      st.p[3] = (h1.y - h0.y) / ch;
      st.p[4] = 0.0f;
      reset_cov(st, sc.cov0);
      const Innov I = innovation(st, sy2, sz2);
      update(st, I, h0.x, 0.0f);
    }
    my_hits[(int64_t)r0 * scap_pad] = p0;
    int nh = 1, lo = r0, hi = r0, r_at = r0;
    unsigned nprop = 0, nupd = 1, ncand = 0;  // work counters (TPC_CNT_PROP/UPD/CAND)
    // R15: chain phase along the cleaned up-links
    for (int hn = p1; hn >= 0;) {
      const Rec c = ld_rec(rec, hn);
      const int rn = rec_sr(c) - s * nrows;
      KState trial = st;
      if (!propagate(trial, sm.X[rn] - sm.X[r_at], kB, ms)) break;
      nprop++;
      const Innov I = innovation(trial, sy2, sz2);
      const float chi2 = chi2_of(I, c.x - trial.p[0], (c.y - zref) - trial.p[1]);
      if (chi2 > sc.chi2_chain_cut) break;  // discard the prediction: state stays at the previous hit
      update(trial, I, c.x, c.y - zref);
      nupd++;
      st = trial;
      my_hits[(int64_t)rn * scap_pad] = hn;
      nh++;
      hi = rn;
      r_at = rn;
      hn = up_c[hn];
    }
    // R16 upward from the last chain hit, R17 jump back to the start row, R16 downward
    for (int leg = 0; leg < 2; leg++) {
      const int dir = leg == 0 ? 1 : -1;
      int r = leg == 0 ? r_at + 1 : r0 - 1;
      if (leg == 1) {
        if (!propagate(st, sm.X[r0] - sm.X[r_at], kB, ms)) break;
        nprop++;
        r_at = r0;
      }
      int misses = 0;
      for (; r >= 0 && r < nrows; r += dir) {
        if (!propagate(st, sm.X[r] - sm.X[r_at], kB, ms)) break;
        nprop++;
        r_at = r;
        if (fabsf(st.p[0]) > sm.ymax[r] + sc.edge_margin) break;  // left the sector
        const Innov I = innovation(st, sy2, sz2);
        const float wy = fminf(sqrtf(sc.chi2_cut * I.S00), sc.win_max);
        const float wz = fminf(sqrtf(sc.chi2_cut * I.S11), sc.win_max);
        const float yp = st.p[0], dzp = st.p[1];
        const float zc = zref + dzp;
        const BinWin W = bin_window(sm, sc, s, r, yp - wy, yp + wy, zc - wz, zc + wz);
        bool have = false;
        float best = 0.0f, by = 0.0f, bz = 0.0f;
        int bi = 0, bk = -1;
        for (int zi = 0; zi < W.nzb; zi++) {
          const int b0 = W.first + zi * W.ny;
          const int ka = __ldg(bin_first + b0), ke = __ldg(bin_first + b0 + W.ybspan);
          for (int k = ka; k < ke; k++) {
            const Rec c = ld_rec(rec, k);
            const float q0 = c.x - yp, q1 = (c.y - zref) - dzp;
            if (!(fabsf(q0) <= wy && fabsf(q1) <= wz)) continue;
            const float chi2 = chi2_of(I, q0, q1);
            ncand++;
            const int ci = rec_idx(c);
            if (!have || chi2 < best || (chi2 == best && ci < bi)) {  // ties: lowest original index
              have = true;
              best = chi2;
              bi = ci;
              bk = k;
              by = c.x;
              bz = c.y;
            }
          }
        }
        if (have && best < sc.chi2_cut) {
          update(st, I, by, bz - zref);
          nupd++;
          my_hits[(int64_t)r * scap_pad] = bk;
          nh++;
          lo = min(lo, r);
          hi = max(hi, r);
          misses = 0;
        } else {
          my_hits[(int64_t)r * scap_pad] = -1;
          misses++;
          if (misses > sc.max_gap) break;
        }
      }
    }
    // R18 record + R20 key push.  Rows lo..hi were each written exactly once above.
    tl_info[t] = nh | (lo << 8) | (hi << 16);
    const unsigned long long key = sel_key(nh, rec_idx(h0));
    for (int r = lo; r <= hi; r++) {
      const int c = my_hits[(int64_t)r * scap_pad];
      if (c >= 0) atomicMax(owner + c, key);
    }
    work[0] += nprop;
    work[1] += nupd;
    work[2] += ncand;
  }
  // one 64-bit atomic per warp and counter
#pragma unroll
  for (int k = 0; k < 3; k++) {
    unsigned long long v = work[k];
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    if (lane == 0 && v) atomicAdd((unsigned long long*)(ws_counters + WC_PROP64) + k, v);
  }
}

// ---------------------------------------------------------------------------------------------
// R20: selection.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads)
k_count_kept(int min_hits, const Rec* __restrict__ rec, const int32_t* __restrict__ starts, int64_t scap_pad,
             const int32_t* __restrict__ row_hit, const int32_t* __restrict__ tl_info,
             const unsigned long long* __restrict__ owner, long long* __restrict__ tl_val,
             const int32_t* __restrict__ ws_counters) {
  const int n_starts = ws_counters[WC_N_STARTS];
  for (int64_t t = (int64_t)blockIdx.x * kThreads + threadIdx.x; t <= scap_pad; t += (int64_t)gridDim.x * kThreads) {
    long long val = 0;
    if (t < n_starts) {
      const int info = tl_info[t];
      const int nh = info & 0xff, lo = (info >> 8) & 0xff, hi = (info >> 16) & 0xff;
      const unsigned long long key = sel_key(nh, rec_idx(ld_rec(rec, starts[t])));
      int kept = 0;
      for (int r = lo; r <= hi; r++) {
        const int c = row_hit[(int64_t)r * scap_pad + t];
        if (c >= 0 && owner[c] == key) kept++;
      }
      if (kept >= min_hits) val = (1ll << 32) | (long long)kept;
    }
    tl_val[t] = val;
  }
}

__global__ void __launch_bounds__(kThreads)
k_write_tracks(int nrows, const Rec* __restrict__ rec, const int32_t* __restrict__ starts, int64_t scap_pad,
               const int32_t* __restrict__ row_hit, const int32_t* __restrict__ tl_info,
               const unsigned long long* __restrict__ owner, const long long* __restrict__ tl_scan, int64_t max_tracks,
               int32_t* __restrict__ cluster_track, int32_t* __restrict__ trk_seed, int32_t* __restrict__ trk_sector,
               int32_t* __restrict__ trk_nhits, int64_t* __restrict__ trk_first_hit, int32_t* __restrict__ trk_hits,
               int32_t* __restrict__ counters, const int32_t* __restrict__ ws_counters) {
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
    const int info = tl_info[t];
    const int nh = info & 0xff, lo = (info >> 8) & 0xff, hi = (info >> 16) & 0xff;
    const Rec h0 = ld_rec(rec, starts[t]);
    const unsigned long long key = sel_key(nh, rec_idx(h0));
    trk_seed[k] = rec_idx(h0);
    trk_sector[k] = rec_sr(h0) / nrows;
    trk_nhits[k] = (int)((nx & 0xffffffffll) - first);
    trk_first_hit[k] = first;
    long long w = first;
    for (int r = lo; r <= hi; r++) {
      const int c = row_hit[(int64_t)r * scap_pad + t];
      if (c >= 0 && owner[c] == key) {
        const int orig = rec_idx(ld_rec(rec, c));
        trk_hits[w++] = orig;
        cluster_track[orig] = (int)k;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// parity/debug export in original indices
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ int to_orig(const Rec* rec, int pos) { return pos >= 0 ? rec_idx(rec[pos]) : -1; }

__global__ void __launch_bounds__(kThreads)
k_export_links(int64_t n, const Rec* __restrict__ rec, const int32_t* __restrict__ link_up,
               const int32_t* __restrict__ link_dn, const int32_t* __restrict__ up_c, int32_t* o_up, int32_t* o_dn,
               int32_t* o_upc, int32_t* o_dnc) {
  for (int64_t p = (int64_t)blockIdx.x * kThreads + threadIdx.x; p < n; p += (int64_t)gridDim.x * kThreads) {
    const int me = rec_idx(rec[p]);
    const int u = link_up[p], d = link_dn[p];
    if (o_up) o_up[me] = to_orig(rec, u);
    if (o_dn) o_dn[me] = to_orig(rec, d);
    if (o_upc) o_upc[me] = to_orig(rec, up_c[p]);
    if (o_dnc) o_dnc[me] = (d >= 0 && link_up[d] == (int)p) ? to_orig(rec, d) : -1;
  }
}

__global__ void __launch_bounds__(kThreads)
k_export_tracklets(int nrows, const Rec* __restrict__ rec, const int32_t* __restrict__ starts, int64_t scap_pad,
                   const int32_t* __restrict__ row_hit, const int32_t* __restrict__ tl_info, int32_t* o_starts,
                   int32_t* o_nhits, int32_t* o_row_hit, const int32_t* __restrict__ ws_counters) {
  const int n_starts = ws_counters[WC_N_STARTS];
  for (int64_t t = (int64_t)blockIdx.x * kThreads + threadIdx.x; t < n_starts; t += (int64_t)gridDim.x * kThreads) {
    const int info = tl_info[t];
    const int nh = info & 0xff, lo = (info >> 8) & 0xff, hi = (info >> 16) & 0xff;
    if (o_starts) o_starts[t] = to_orig(rec, starts[t]);
    if (o_nhits) o_nhits[t] = nh;
    if (o_row_hit)
      for (int r = 0; r < nrows; r++)
        o_row_hit[t * nrows + r] = (r >= lo && r <= hi) ? to_orig(rec, row_hit[(int64_t)r * scap_pad + t]) : -1;
  }
}

inline unsigned blocks_for(int64_t n, int threads, int64_t cap = 148 * 64) {
  int64_t b = (n + threads - 1) / threads;
  if (b > cap) b = cap;
  if (b < 1) b = 1;
  return (unsigned)b;
}

int g_follow_blocks = 0;

}  // namespace

cudaError_t launch_find(const Geo& g, const Ws& w, int32_t* cluster_track, int64_t max_tracks, int32_t* trk_seed,
                        int32_t* trk_sector, int32_t* trk_nhits, int64_t* trk_first_hit, int32_t* trk_hits,
                        int32_t* counters, cudaStream_t st) {
  const int64_t n = w.L.n, scap = w.L.scap, scap_pad = w.L.scap_pad;
  cudaError_t e;
  if (g_follow_blocks == 0) {
    int dev = 0, sms = 0, per_sm = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_follow, kFollowThreads, 0)) != cudaSuccess) return e;
    g_follow_blocks = sms * (per_sm > 0 ? per_sm : 1);
  }
  // queue heads restart; status bits from the grid build are kept
  if ((e = cudaMemsetAsync(w.counters + WC_QUEUE, 0, sizeof(int32_t), st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(w.counters + WC_N_STARTS, 0, sizeof(int32_t), st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(w.counters + WC_PROP64, 0, sizeof(int32_t) * 6, st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(w.owner, 0, sizeof(uint64_t) * (size_t)(n + 1), st)) != cudaSuccess) return e;
  if (n > 0 && (e = cudaMemsetAsync(cluster_track, 0xFF, sizeof(int32_t) * (size_t)n, st)) != cudaSuccess) return e;
  int32_t* flag = w.key;  // the bin ids of the grid build are dead by now
  if (n > 0)
    TPC_LAUNCH(KID_NEIGHBOURS, st,
               (k_neighbours<<<blocks_for(n, kThreads), kThreads, 0, st>>>(g, n, w.rec, w.bin_first, w.link_up, w.link_dn)));
  TPC_LAUNCH(KID_CLEAN, st, (k_clean<<<blocks_for(n + 1, kThreads), kThreads, 0, st>>>(n, w.link_up, w.link_dn, w.up_c, flag)));
  if ((e = exclusive_scan<int32_t>(flag, flag, n + 1, (int32_t*)w.scan_tmp, st)) != cudaSuccess) return e;
  if (n > 0) {
    TPC_LAUNCH(KID_COMPACT_STARTS, st,
               (k_compact_starts<<<blocks_for(n, kThreads), kThreads, 0, st>>>(n, scap, flag, w.starts, w.counters)));
    TPC_LAUNCH(KID_FOLLOW, st,
               (k_follow<<<g_follow_blocks, kFollowThreads, 0, st>>>(g, w.rec, w.bin_first, w.up_c, w.starts, scap_pad,
                                                                    w.row_hit, w.tl_info, w.owner, w.counters)));
  }
  TPC_LAUNCH(KID_COUNT_KEPT, st,
             (k_count_kept<<<blocks_for(scap_pad + 1, kThreads), kThreads, 0, st>>>(
                 g.s.min_hits, w.rec, w.starts, scap_pad, w.row_hit, w.tl_info, w.owner, w.tl_scan, w.counters)));
  if ((e = exclusive_scan<long long>(w.tl_scan, w.tl_scan, scap_pad + 1, w.scan_tmp, st)) != cudaSuccess) return e;
  TPC_LAUNCH(KID_WRITE_TRACKS, st,
             (k_write_tracks<<<blocks_for(scap_pad > 0 ? scap_pad : 1, kThreads), kThreads, 0, st>>>(
                 g.s.nrows, w.rec, w.starts, scap_pad, w.row_hit, w.tl_info, w.owner, w.tl_scan, max_tracks,
                 cluster_track, trk_seed, trk_sector, trk_nhits, trk_first_hit, trk_hits, counters, w.counters)));
  return cudaGetLastError();
}

cudaError_t launch_find_export(const Geo& g, const Ws& w, int32_t* link_up, int32_t* link_dn, int32_t* up_c,
                               int32_t* dn_c, int32_t* starts, int32_t* tl_nhits, int32_t* row_hit, cudaStream_t st) {
  const int64_t n = w.L.n;
  if (n > 0 && (link_up || link_dn || up_c || dn_c))
    TPC_LAUNCH(KID_EXPORT, st,
               (k_export_links<<<blocks_for(n, kThreads), kThreads, 0, st>>>(n, w.rec, w.link_up, w.link_dn, w.up_c,
                                                                            link_up, link_dn, up_c, dn_c)));
  if (w.L.scap > 0 && (starts || tl_nhits || row_hit))
    TPC_LAUNCH(KID_EXPORT, st,
               (k_export_tracklets<<<blocks_for(w.L.scap, kThreads), kThreads, 0, st>>>(
                   g.s.nrows, w.rec, w.starts, w.L.scap_pad, w.row_hit, w.tl_info, starts, tl_nhits, row_hit, w.counters)));
  return cudaGetLastError();
}

}  // namespace tpc
