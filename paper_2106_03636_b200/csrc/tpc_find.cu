// =============================================================================================
// tpc_find.cu -- step 2 of the hot path (BASELINE.json north_star (2)) on
// the grid built by tpc_grid.cu, and the launch sequence of tpc_find_tracks.  All internal
// indices are GRID POSITIONS (index into the sorted record array); original indices are only
// used for tie-breaks (R9, R16, R20) and in the outputs.
//
//   k_neighbours      R9   one thread per cluster: best (up,down) pair on rows r+1 / r-1
//   k_clean           R10  reciprocal links, start-hit flags                     (+ scan)
//   k_compact_starts  R10/R14  start list: one 32-byte start record per tracklet
//   launch_follow     R11-R18  tpc_follow.cu
//   launch_select     R20      tpc_select.cu
// =============================================================================================
#include "tpc_common.cuh"
#include "tpc_scan.cuh"
#include "tpc_search.cuh"

namespace tpc {

namespace {

constexpr int kThreads = 256;
constexpr int kMaxCand = 8;  // up-candidates staged per thread; more (dense toy inputs) take the slow path

struct SmCa {
  float wu[kMaxRows], iy[kMaxRows], iz[kMaxRows], wyu[kMaxRows], wzu[kMaxRows], wyd[kMaxRows], wzd[kMaxRows];
};

// Running arg-min of R9: minimal D2; ties: lowest original u index, then lowest original d index.  best starts at
// +inf and the indices at INT_MAX, so the first pair offered is always taken (as "!have ||" would).
struct BestPair {
  float best;
  int bui, bdi, bu, bd;
  __device__ __forceinline__ void reset() {
    best = __int_as_float(0x7f800000);
    bui = bdi = 0x7fffffff;
    bu = bd = -1;
  }
  __device__ __forceinline__ bool have() const { return bu >= 0; }
  __device__ __forceinline__ void offer(float D2, int ui, int di, int k, int j) {
    if (D2 < best || (D2 == best && (ui < bui || (ui == bui && di < bdi)))) {
      best = D2;
      bui = ui;
      bdi = di;
      bu = k;
      bd = j;
    }
  }
};

__device__ __forceinline__ float pair_d2(float yh, float zh, float wu, float iy, float iz, float uy, float uz, float dy,
                                         float dz) {
  const float ry = (yh - dy) - wu * (uy - dy);
  const float rz = (zh - dz) - wu * (uz - dz);
  return (ry * ry) * iy + (rz * rz) * iz;
}

// Slow path (more than kMaxCand up-candidates in the window): plain nested loops over both windows.
__device__ __noinline__ void neighbours_nested(const Rec* __restrict__ rec, const int32_t* __restrict__ bin_first,
                                               const BinWin WU, const BinWin WD, float yh, float zh, float wu, float iy,
                                               float iz, float wyu, float wzu, float wyd, float wzd, BestPair& B) {
  for (int zu = 0; zu < WU.nzb; zu++) {
    const int b0 = WU.first + zu * WU.ny;
    const int ka = __ldg(bin_first + b0), ke = __ldg(bin_first + b0 + WU.ybspan);
    for (int k = ka; k < ke; k++) {
      const Rec u = ld_rec(rec, k);
      if (!(fabsf(u.x - yh) <= wyu && fabsf(u.y - zh) <= wzu)) continue;
      for (int zd = 0; zd < WD.nzb; zd++) {
        const int c0 = WD.first + zd * WD.ny;
        const int ja = __ldg(bin_first + c0), je = __ldg(bin_first + c0 + WD.ybspan);
        for (int j = ja; j < je; j++) {
          const Rec d = ld_rec(rec, j);
          if (!(fabsf(d.x - yh) <= wyd && fabsf(d.y - zh) <= wzd)) continue;
          B.offer(pair_d2(yh, zh, wu, iy, iz, u.x, u.y, d.x, d.y), rec_idx(u), rec_idx(d), k, j);
        }
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// R9: cellular-automaton neighbour finder.  A window covers at most two z-bin rows when the cell is
// not smaller than the window (the normal case), so both sides' bin ranges are fetched up front in one
// round trip; candidates are then requested kCaBatch at a time and tested branch-free.  The up-window
// candidates are staged in shared memory (slot-major: a warp's 16-byte accesses are conflict-free) and
// every down-window candidate is paired with the staged ones.  The arg-min is order-independent because
// the tie-break is explicit.  Windows over more than two z-bin rows, or more than kMaxCand staged
// candidates, take the plain nested loops.
// ---------------------------------------------------------------------------------------------
constexpr int kCaBatch = 4;  // candidate records in flight per thread and side (measured optimum)

struct Ranges {
  int ka0, n0, ka1, n1;
};

__device__ __forceinline__ Ranges load_ranges(const int32_t* __restrict__ bin_first, const BinWin& W) {
  Ranges R;
  R.ka1 = R.n1 = 0;
  const int e0 = __ldg(bin_first + W.first + W.ybspan);
  R.ka0 = __ldg(bin_first + W.first);
  if (W.nzb > 1) {
    const int e1 = __ldg(bin_first + W.first + W.ny + W.ybspan);
    R.ka1 = __ldg(bin_first + W.first + W.ny);
    R.n1 = e1 - R.ka1;
  }
  R.n0 = e0 - R.ka0;
  return R;
}

__global__ void __launch_bounds__(kThreads, 4)
k_neighbours(const __grid_constant__ Geo g, int64_t n, const Rec* __restrict__ rec, const int32_t* __restrict__ bin_first,
             int32_t* __restrict__ link_up, int32_t* __restrict__ link_dn) {
  __shared__ SmRow sm;
  __shared__ SmCa ca;
  __shared__ float4 cand[kMaxCand][kThreads];  // (y, z, orig idx, grid pos) of the up-candidates
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
  const int tid = threadIdx.x;
  for (int64_t p = (int64_t)blockIdx.x * kThreads + tid; p < n; p += (int64_t)gridDim.x * kThreads) {
    const Rec h = ld_rec(rec, (int)p);
    const int sr = rec_sr(h);
    const bool on_grid = sr < sc.nsec * nrows;  // (a cluster parked behind the grid has an impossible sector_row)
    const int s = on_grid ? sector_of(sc, sr) : 0, r = sr - s * nrows;
    int bu = -1, bd = -1;
    if (on_grid && r >= 1 && r <= nrows - 2) {
      const float yh = h.x, zh = h.y;
      const float wu = ca.wu[r], iy = ca.iy[r], iz = ca.iz[r];
      const float wyu = ca.wyu[r], wzu = ca.wzu[r], wyd = ca.wyd[r], wzd = ca.wzd[r];
      const BinWin WU = bin_window(sm, sc, s, r + 1, yh - wyu, yh + wyu, zh - wzu, zh + wzu);
      const BinWin WD = bin_window(sm, sc, s, r - 1, yh - wyd, yh + wyd, zh - wzd, zh + wzd);
      BestPair B;
      B.reset();
      bool slow = WU.nzb > 2 || WD.nzb > 2;
      if (!slow) {
        const Ranges RU = load_ranges(bin_first, WU), RD = load_ranges(bin_first, WD);
        int nu = 0;
        const int ntu = RU.n0 + RU.n1;
        for (int i0 = 0; i0 < ntu; i0 += kCaBatch) {
          Rec c[kCaBatch];
          int kk[kCaBatch];
#pragma unroll
          for (int j = 0; j < kCaBatch; j++) {
            const int i = min(i0 + j, ntu - 1);
            kk[j] = i < RU.n0 ? RU.ka0 + i : RU.ka1 + (i - RU.n0);
            c[j] = ld_rec(rec, kk[j]);
          }
#pragma unroll
          for (int j = 0; j < kCaBatch; j++) {
            if (i0 + j < ntu && fabsf(c[j].x - yh) <= wyu && fabsf(c[j].y - zh) <= wzu) {
              if (nu < kMaxCand) cand[nu][tid] = make_float4(c[j].x, c[j].y, c[j].z, __int_as_float(kk[j]));
              nu++;
            }
          }
        }
        slow = nu > kMaxCand;
        const int ntd = (nu > 0 && !slow) ? RD.n0 + RD.n1 : 0;
        for (int i0 = 0; i0 < ntd; i0 += kCaBatch) {
          Rec c[kCaBatch];
          int kk[kCaBatch];
#pragma unroll
          for (int j = 0; j < kCaBatch; j++) {
            const int i = min(i0 + j, ntd - 1);
            kk[j] = i < RD.n0 ? RD.ka0 + i : RD.ka1 + (i - RD.n0);
            c[j] = ld_rec(rec, kk[j]);
          }
          // window test per slot; the pair arithmetic runs once, for the first slot inside the window (nearly
          // always the only one), and a rare second round takes the others
          unsigned inmask = 0u;
          int first_in = kCaBatch;
#pragma unroll
          for (int j = kCaBatch - 1; j >= 0; j--) {
            if (i0 + j < ntd && fabsf(c[j].x - yh) <= wyd && fabsf(c[j].y - zh) <= wzd) {
              inmask |= 1u << j;
              first_in = j;
            }
          }
          Rec ds = c[0];
          int ks = kk[0];
#pragma unroll
          for (int j = 1; j < kCaBatch; j++)
            if (first_in == j) {
              ds = c[j];
              ks = kk[j];
            }
          if (inmask) {
            const int di = rec_idx(ds);
            for (int a = 0; a < nu; a++) {
              const float4 u = cand[a][tid];
              B.offer(pair_d2(yh, zh, wu, iy, iz, u.x, u.y, ds.x, ds.y), __float_as_int(u.z), di, __float_as_int(u.w), ks);
            }
          }
          if (inmask & (inmask - 1u)) {
#pragma unroll
            for (int j = 1; j < kCaBatch; j++) {
              if (((inmask >> j) & 1u) && j != first_in) {
                const int di = rec_idx(c[j]);
                for (int a = 0; a < nu; a++) {
                  const float4 u = cand[a][tid];
                  B.offer(pair_d2(yh, zh, wu, iy, iz, u.x, u.y, c[j].x, c[j].y), __float_as_int(u.z), di,
                          __float_as_int(u.w), kk[j]);
                }
              }
            }
          }
        }
      }
      if (slow) {
        B.reset();
        neighbours_nested(rec, bin_first, WU, WD, yh, zh, wu, iy, iz, wyu, wzu, wyd, wzd, B);
      }
      if (B.have() && B.best < sc.ca_cut) {
        bu = B.bu;
        bd = B.bd;
      }
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
    up_c[p] = (uc < 0 && dc >= 0) ? -2 : uc;  // -2: top of a chain (linked downward only); read by the R17 wave test
    flag[p] = (uc >= 0 && dc < 0) ? 1 : 0;
  }
}

// Tracklet order.  Tracklets are numbered by (sector, z slab, row, grid order inside): a slab is slab_w z-bins
// (about one drift length), so tracklets with neighbouring numbers are tracks of the same few collisions
// and touch the same few percent of a sector.  The passes that run one WARP per tracklet (selection) then
// have a working set far below the L2 size.  The numbering needs no sort: a chunk (sector, slab, row) is a
// contiguous range of grid positions, its number of start hits is a difference of the grid-order flag scan,
// and an exclusive scan over the chunks in (sector, slab, row) order gives each chunk's first tracklet.
__global__ void __launch_bounds__(kThreads)
k_chunk_counts(const __grid_constant__ Geo g, int64_t nchunks, const int32_t* __restrict__ bin_first,
               const int32_t* __restrict__ scan, int32_t* __restrict__ chunk_cnt, int32_t* __restrict__ chunk_scan0) {
  const Scalars& sc = g.s;
  for (int64_t q = (int64_t)blockIdx.x * kThreads + threadIdx.x; q <= nchunks; q += (int64_t)gridDim.x * kThreads) {
    if (q == nchunks) {
      chunk_cnt[q] = 0;  // sentinel: the exclusive scan leaves the total here
      continue;
    }
    const int r = (int)(q % sc.nrows);
    const int sj = (int)(q / sc.nrows);
    const int j = sj % sc.nslab, s = sj / sc.nslab;
    const int ny = g.row.ny[r];
    const int base = s * sc.bins_per_sector + g.row.rowbase[r];
    const int zb0 = j * sc.slab_w;
    int zb1 = zb0 + sc.slab_w;
    if (zb1 > sc.nz) zb1 = sc.nz;
    const int s0 = scan[bin_first[base + zb0 * ny]], s1 = scan[bin_first[base + zb1 * ny]];
    chunk_cnt[q] = s1 - s0;
    chunk_scan0[q] = s0;
  }
}

// Start list.  Everything R14 needs from memory goes into one 32-byte record per tracklet, gathered here
// with full memory-level parallelism instead of as a dependent chain inside the follower.
__global__ void __launch_bounds__(kThreads)
k_compact_starts(const __grid_constant__ Geo g, int64_t n, int64_t scap, const int32_t* __restrict__ scan,
                 Rec* rec, const int32_t* __restrict__ up_c, const int32_t* __restrict__ chunk_base,
                 const int32_t* __restrict__ chunk_scan0, TlInit* __restrict__ tl_init, int32_t* __restrict__ ws_counters) {
  const Scalars& sc = g.s;
  for (int64_t p = (int64_t)blockIdx.x * kThreads + threadIdx.x; p < n; p += (int64_t)gridDim.x * kThreads) {
    const int ex = scan[p];
    if (scan[p + 1] != ex) {
      const Rec h0 = rec[p];
      const int sr0 = rec_sr(h0);
      const int s = sr0 / sc.nrows, r = sr0 - s * sc.nrows;
      const float zeta = (s < 18) ? h0.y : -h0.y;  // R2/R7, the same expression the grid build bins with
      const int zb = clampbin((zeta - sc.z_lo) * sc.inv_cz, sc.nz);
      const int64_t q = ((int64_t)s * sc.nslab + zb / sc.slab_w) * sc.nrows + r;
      const int t = chunk_base[q] + (ex - chunk_scan0[q]);
      if (t < scap) {
        // mark the record as a start hit: the upward legs of the follower look at this bit (R17).  Only this thread
        // writes this word; other threads read at most y and z of this record.  (k_clear_start_bits undoes it.)
        reinterpret_cast<int*>(rec + p)[3] = sr0 | kStartBit;
        const int p1 = up_c[p];
        const Rec h1 = rec[p1];
        float4* o = reinterpret_cast<float4*>(tl_init + t);
        o[0] = make_float4(h0.x, h0.y, h1.x, h1.y);
        o[1] = make_float4(__int_as_float((int)p), __int_as_float(p1), __int_as_float(sr0), h0.z);
      }
    }
    if (p == 0) {
      const int total = scan[n];
      ws_counters[WC_STARTS_FOUND] = total;
      ws_counters[WC_N_STARTS] = total < scap ? total : (int)scap;
      if (total > scap) atomicOr(ws_counters + WC_STATUS, TPC_ST_TRACKLET_OVERFLOW);
    }
  }
}

// The start bits of the PREVIOUS tpc_find_tracks on this grid (another set of cuts gives other start hits): the old
// start list is still in tl_init.  After tpc_grid_build the list is empty and this is a no-op.
__global__ void __launch_bounds__(kThreads)
k_clear_start_bits(Rec* rec, const TlInit* __restrict__ tl_init, const int32_t* __restrict__ ws_counters) {
  const int n_starts = ws_counters[WC_N_STARTS];
  for (int64_t t = (int64_t)blockIdx.x * kThreads + threadIdx.x; t < n_starts; t += (int64_t)gridDim.x * kThreads)
    reinterpret_cast<int*>(rec + tl_init[t].p0)[3] &= ~kStartBit;
}

// ---------------------------------------------------------------------------------------------
// parity/debug export in original indices
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ int to_orig(const Rec* rec, int pos) { return pos >= 0 ? rec_idx(rec[pos]) : pos; }

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
k_export_tracklets(int nrows, const Rec* __restrict__ rec, const TlInit* __restrict__ tl_init,
                   const int32_t* __restrict__ row_hit, const int32_t* __restrict__ tl_info, int32_t* o_starts,
                   int32_t* o_nhits, int32_t* o_row_hit, const int32_t* __restrict__ ws_counters) {
  const int n_starts = ws_counters[WC_N_STARTS];
  for (int64_t t = (int64_t)blockIdx.x * kThreads + threadIdx.x; t < n_starts; t += (int64_t)gridDim.x * kThreads) {
    const int info = tl_info[t];
    const int nh = info & 0xff, lo = (info >> 8) & 0xff, hi = (info >> 16) & 0xff;
    if (o_starts) o_starts[t] = tl_init[t].orig0;
    if (o_nhits) o_nhits[t] = nh;
    if (o_row_hit)
      for (int r = 0; r < nrows; r++)
        o_row_hit[t * nrows + r] = (r >= lo && r <= hi) ? to_orig(rec, row_hit[t * nrows + r]) : -1;
  }
}

}  // namespace

cudaError_t launch_find(const Geo& g, const Ws& w, int32_t* cluster_track, int64_t max_tracks, int32_t* trk_seed,
                        int32_t* trk_sector, int32_t* trk_nhits, int64_t* trk_first_hit, int32_t* trk_hits,
                        int32_t* counters, cudaStream_t st) {
  const int64_t n = w.L.n, scap = w.L.scap;
  cudaError_t e;
  if (n > 0 && scap > 0)
    TPC_LAUNCH(KID_COMPACT_STARTS, st,
               (k_clear_start_bits<<<blocks_for(scap, kThreads, 148 * 8), kThreads, 0, st>>>(w.rec, w.tl_init, w.counters)));
  // queue heads restart; status bits from the grid build are kept
  if ((e = cudaMemsetAsync(w.counters + WC_QUEUE, 0, sizeof(int32_t), st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(w.counters + WC_N_STARTS, 0, sizeof(int32_t), st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(w.counters + WC_PROP64, 0, sizeof(int32_t) * 8, st)) != cudaSuccess) return e;
  int32_t* flag = w.key;  // the bin ids of the grid build are dead by now
  if (n > 0)
    TPC_LAUNCH(KID_NEIGHBOURS, st,
               (k_neighbours<<<blocks_for(n, kThreads), kThreads, 0, st>>>(g, n, w.rec, w.bin_first, w.link_up, w.link_dn)));
  TPC_LAUNCH(KID_CLEAN, st, (k_clean<<<blocks_for(n + 1, kThreads), kThreads, 0, st>>>(n, w.link_up, w.link_dn, w.up_c, flag)));
  if ((e = exclusive_scan<int32_t>(flag, flag, n + 1, (int32_t*)w.scan_tmp, st)) != cudaSuccess) return e;
  if (n > 0) {
    const int64_t nchunks = w.L.nchunks;
    TPC_LAUNCH(KID_COMPACT_STARTS, st,
               (k_chunk_counts<<<blocks_for(nchunks + 1, kThreads), kThreads, 0, st>>>(g, nchunks, w.bin_first, flag,
                                                                                      w.chunk_base, w.chunk_scan0)));
    if ((e = exclusive_scan<int32_t>(w.chunk_base, w.chunk_base, nchunks + 1, (int32_t*)w.scan_tmp, st)) != cudaSuccess)
      return e;
    TPC_LAUNCH(KID_COMPACT_STARTS, st,
               (k_compact_starts<<<blocks_for(n, kThreads), kThreads, 0, st>>>(g, n, scap, flag, w.rec, w.up_c, w.chunk_base,
                                                                              w.chunk_scan0, w.tl_init, w.counters)));
    if ((e = launch_follow(g, w, st)) != cudaSuccess) return e;
  }
  return launch_select(g, w, cluster_track, max_tracks, trk_seed, trk_sector, trk_nhits, trk_first_hit, trk_hits, counters,
                       st);
}

cudaError_t launch_find_export(const Geo& g, const Ws& w, int32_t* link_up, int32_t* link_dn, int32_t* up_c,
                               int32_t* dn_c, int32_t* starts, int32_t* tl_nhits, int32_t* row_hit, cudaStream_t st) {
  const int64_t n = w.L.n;
  if (n > 0 && (link_up || link_dn || up_c || dn_c))
    TPC_LAUNCH(KID_EXPORT, st,
               (k_export_links<<<blocks_for(n, kThreads), kThreads, 0, st>>>(n, w.rec, w.link_up, w.link_dn, w.up_c,
                                                                            link_up, link_dn, up_c, dn_c)));
  if (n > 0 && w.L.scap > 0 && (starts || tl_nhits || row_hit))
    TPC_LAUNCH(KID_EXPORT, st,
               (k_export_tracklets<<<blocks_for(w.L.scap, kThreads), kThreads, 0, st>>>(
                   g.s.nrows, w.rec, w.tl_init, w.row_hit, w.tl_info, starts, tl_nhits, row_hit, w.counters)));
  return cudaGetLastError();
}

}  // namespace tpc
