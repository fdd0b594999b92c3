// =============================================================================================
// tpc_follow.cu -- step 3a of the hot path (BASELINE.json north_star (3) "Kalman-filter track
// following"): one LANE per tracklet with the fp32 5-parameter state and
// its 15 covariance elements in registers.
//
// Execution shape.  A tracklet is a sequence of row steps of four kinds -- chain step along the
// cleaned links (R15), extrapolation step up or down with a windowed search (R16), the one-step
// jump back to the start row (R17) -- and all of them are "transport (R12), pick a measurement,
// update (R13)".  The kernel is ONE loop whose body holds a single copy of the transport and of
// the update, so the lanes of a warp execute them together whatever phase each lane is in, and a
// lane that finishes its tracklet pulls the next one from the queue inside the same loop (no
// waiting for the longest tracklet of a batch).  Tracklets are queued in (sector, z slab, row) order
// (tpc_find.cu), so concurrently running lanes walk neighbouring bins (L2 locality of the lookups).
//
// Output: row_hit[t][row] (grid positions, -1 = no hit), tl_info[t] = nHits | lo<<8 | hi<<16,
// tl_key[t] = R20 selection key.  The key is pushed onto the clusters by k_push_keys
// (tpc_select.cu) once nHits is final.
// =============================================================================================
#include "tpc_common.cuh"
#include "tpc_kalman.cuh"
#include "tpc_prof.cuh"
#include "tpc_search.cuh"

namespace tpc {

namespace {

#ifndef TPC_FOLLOW_THREADS
#define TPC_FOLLOW_THREADS 64
#endif
// 64-thread blocks, 10 per SM: 96 registers per thread without spills and 20 resident warps per SM (measured on
// configs[4]: 128 x 4 blocks at 112 registers = 16 warps: 28.0 ms; 64 x 10 at 96 registers, batch 3: 25.3 ms)
constexpr int kFollowThreads = TPC_FOLLOW_THREADS;
constexpr unsigned kFull = 0xffffffffu;
#ifndef TPC_FOLLOW_BATCH
#define TPC_FOLLOW_BATCH 3
#endif
#ifndef TPC_FOLLOW_MIN_BLOCKS
#define TPC_FOLLOW_MIN_BLOCKS 10
#endif
#ifndef TPC_FOLLOW_PREFETCH
#define TPC_FOLLOW_PREFETCH 1
#endif
constexpr int kBatch = TPC_FOLLOW_BATCH;  // candidate records in flight per lane in the R15/R16 search

// L1 prefetch of one line: the follower knows one step ahead roughly where it will look.
__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }

enum Phase { PH_FETCH = 0, PH_INIT, PH_CHAIN, PH_UP, PH_JUMP, PH_DOWN, PH_DONE };

__global__ void __launch_bounds__(kFollowThreads, TPC_FOLLOW_MIN_BLOCKS)
k_follow(const __grid_constant__ Geo g, const Rec* __restrict__ rec, const int32_t* __restrict__ bin_first,
         const int32_t* __restrict__ up_c, const TlInit* __restrict__ tl_init, int32_t* __restrict__ row_hit,
         int32_t* __restrict__ tl_info, unsigned long long* __restrict__ tl_key, int32_t* __restrict__ ws_counters) {
  __shared__ SmRow sm;
  load_rows(sm, g);
  __syncthreads();
  const Scalars& sc = g.s;
  const int nrows = sc.nrows;
  const int n_starts = ws_counters[WC_N_STARTS];
  const int lane = threadIdx.x & 31;
  const float kB = sc.kB, ms = sc.max_sinphi, sy2 = sc.sy2, sz2 = sc.sz2;

  // per-lane tracklet state
  int phase = PH_FETCH;
  KState st;
  float zref = 0.0f;
  int t = 0, s = 0, r0 = 0, r_at = 0, r = 0, hn = -1, p0 = 0, orig0 = 0;
  int misses = 0, nh = 0, lo = 0, hi = 0;
  unsigned nprop = 0, nupd = 0, ncand = 0;  // work counters of this lane over all its tracklets (TPC_CNT_PROP/UPD/CAND)
  int pf_ka = -1;  // first grid position of the bin the NEXT step is expected to search (-1: no prediction)
#pragma unroll
  for (int k = 0; k < 5; k++) st.p[k] = 0.0f;
#pragma unroll
  for (int k = 0; k < 15; k++) st.C[k] = 0.0f;

  for (;;) {
    // ---- lanes without a tracklet take the next ones from the queue (one atomic per warp) --------
    const unsigned need = __ballot_sync(kFull, phase == PH_FETCH);
    if (need) {
      const int leader = __ffs(need) - 1;
      int base = 0;
      if (lane == leader) base = atomicAdd(ws_counters + WC_QUEUE, __popc(need));
      base = __shfl_sync(kFull, base, leader);
      if (phase == PH_FETCH) {
        t = base + __popc(need & ((1u << lane) - 1u));
        if (t >= n_starts) {
          phase = PH_DONE;
        } else {
          const float4* ip = reinterpret_cast<const float4*>(tl_init + t);
          const float4 a = __ldg(ip), b = __ldg(ip + 1);
          p0 = __float_as_int(b.x);
          hn = __float_as_int(b.y);
          prefetch_l1(rec + hn);
          const int sr0 = __float_as_int(b.z);
          orig0 = __float_as_int(b.w);
          s = sr0 / nrows;
          r0 = sr0 - s * nrows;
          // R14: initial state from the start hit and its up-neighbour (always on row r0 + 1, R9)
          const float dx = sm.X[r0 + 1] - sm.X[r0], dy = a.z - a.x;
          const float ch = sqrtf(dx * dx + dy * dy);
          zref = a.y;
          st.p[0] = a.x;
          st.p[1] = 0.0f;
          st.p[2] = dy / ch;
          st.p[3] = (a.w - a.y) / ch;
          st.p[4] = 0.0f;
          reset_cov(st, sc.cov0);
          nh = 0;
          lo = hi = r_at = r0;
          phase = PH_INIT;
        }
      }
    }
    if (__all_sync(kFull, phase == PH_DONE)) break;

    // ---- target row of this step; chain steps prefetch their next link --------------------------
    const bool isI = phase == PH_INIT, chain = phase == PH_CHAIN, isJ = phase == PH_JUMP;
    const bool leg = phase == PH_UP || phase == PH_DOWN;
    int rn = r0;                      // PH_INIT, PH_JUMP
    if (chain) rn = r_at + 1;         // links join adjacent rows (R9)
    if (leg) rn = r;
    int nxt = -1;
    if (chain) nxt = __ldg(up_c + hn);
    // the bin offset requested during the previous step has arrived by now: pull the records it points to
    // into L1 while the transport below is computed
    if (pf_ka >= 0) prefetch_l1(rec + pf_ka);
    pf_ka = -1;
    // ---- R12 transport (one copy for every phase; __syncwarp keeps the compiler from cloning it
    //      into the phase branches, which would serialise the lanes again) --------------------------
    __syncwarp();
    bool ok = phase != PH_DONE;
    const bool moved = ok && !isI;
    Transport T;
    float yp = st.p[0], dzp = st.p[1];
    float C00n = st.C[TPC_CI(0, 0)], C10n = st.C[TPC_CI(1, 0)], C11n = st.C[TPC_CI(1, 1)];
    if (moved) {
      ok = transport_state(st, sm.X[rn] - sm.X[r_at], kB, ms, T);
      if (ok) {
        nprop++;
        yp = T.y;
        dzp = T.dz;
        transport_cov_diag(st, T, C00n, C11n);
        C10n = transport_cov_10(st, T);
      }
    }
    // ---- candidates of this step: up to two contiguous ranges of grid positions -------------------
    //   chain step (R15): the linked cluster alone, no window;  leg step (R16): the bins covering the
    //   chi2 window (a superset, every candidate is re-tested in cm);  init / jump: none.
    // The bin offsets are requested here, as soon as the predicted position and its two variances are
    // known; the rest of F C F^T below runs while they are in flight.
    float wy = 3.0e38f, wz = 3.0e38f;
    int ka0 = 0, e0 = 0, ka1 = 0, e1 = 0;  // [ka, e) per range; the differences are taken after the covariance math
    bool edge_out = false, many = false;
    BinWin W;
    W.first = W.ny = W.ybspan = W.nzb = 0;
    if (chain && ok) {
      ka0 = hn;
      e0 = hn + 1;
    } else if (leg && ok) {
      edge_out = fabsf(yp) > sm.ymax[rn] + sc.edge_margin;
      if (!edge_out) {
        wy = fminf(sqrtf(sc.chi2_cut * (C00n + sy2)), sc.win_max);
        wz = fminf(sqrtf(sc.chi2_cut * (C11n + sz2)), sc.win_max);
        const float zc = zref + dzp;
        W = bin_window(sm, sc, s, rn, yp - wy, yp + wy, zc - wz, zc + wz);
        e0 = __ldg(bin_first + W.first + W.ybspan);
        ka0 = __ldg(bin_first + W.first);
        if (W.nzb > 1) {
          e1 = __ldg(bin_first + W.first + W.ny + W.ybspan);
          ka1 = __ldg(bin_first + W.first + W.ny);
        }
        many = W.nzb > 2;
      }
    }
    // innovation covariance of the PREDICTED state from the three elements of C' it depends on: the search
    // and the chain cut are decided before the transport is committed, so a rejected chain step (R15) simply
    // never commits and no copy of the state is kept
    const Innov I = innovation3(C00n, C10n, C11n, sy2, sz2);
    const int n0 = e0 - ka0, n1 = e1 - ka1;
    // ---- arg-min chi2 over the candidates (ties: lowest original index) ----------------------------
    __syncwarp();
    bool have = false;
    float best = 0.0f, by = 0.0f, bz = 0.0f;
    int bi = 0, bk = -1;
    const int ntot = n0 + n1;
    // kBatch records are requested together (one memory round trip per batch instead of one per candidate)
    // and tested branch-free; slots past the end re-read the last candidate and are masked out.
    for (int i0 = 0; i0 < ntot; i0 += kBatch) {
      Rec c[kBatch];
      int kk[kBatch];
#pragma unroll
      for (int j = 0; j < kBatch; j++) {
        const int i = min(i0 + j, ntot - 1);
        kk[j] = i < n0 ? ka0 + i : ka1 + (i - n0);
        c[j] = ld_rec(rec, kk[j]);
      }
      // window test per slot (cheap); the chi2 arithmetic runs once, on the first slot inside the window --
      // nearly always the only one -- and a rare second round takes the others.
      unsigned inmask = 0u;
      int first_in = kBatch;
#pragma unroll
      for (int j = kBatch - 1; j >= 0; j--) {
        const float q0 = c[j].x - yp, q1 = (c[j].y - zref) - dzp;
        if ((i0 + j < ntot) && fabsf(q0) <= wy && fabsf(q1) <= wz) {
          inmask |= 1u << j;
          first_in = j;
        }
      }
      if (leg) ncand += __popc(inmask);
      Rec cs = c[0];
      int ks = kk[0];
#pragma unroll
      for (int j = 1; j < kBatch; j++)
        if (first_in == j) {
          cs = c[j];
          ks = kk[j];
        }
      if (inmask) {
        const float chi2 = chi2_of(I, cs.x - yp, (cs.y - zref) - dzp);
        const int ci = rec_idx(cs);
        if (!have || chi2 < best || (chi2 == best && ci < bi)) {
          have = true;
          best = chi2;
          bi = ci;
          bk = ks;
          by = cs.x;
          bz = cs.y;
        }
      }
      if (inmask & (inmask - 1u)) {  // more than one slot inside the window
#pragma unroll
        for (int j = 1; j < kBatch; j++) {
          if (((inmask >> j) & 1u) && j != first_in) {
            const float chi2 = chi2_of(I, c[j].x - yp, (c[j].y - zref) - dzp);
            const int ci = rec_idx(c[j]);
            if (!have || chi2 < best || (chi2 == best && ci < bi)) {
              have = true;
              best = chi2;
              bi = ci;
              bk = kk[j];
              by = c[j].x;
              bz = c[j].y;
            }
          }
        }
      }
    }
    if (many) {  // windows of more than two z-bin rows (cells much smaller than the window): generic loop
      for (int zi = 2; zi < W.nzb; zi++) {
        const int b0 = W.first + zi * W.ny;
        const int ka = __ldg(bin_first + b0), ke = __ldg(bin_first + b0 + W.ybspan);
        for (int k = ka; k < ke; k++) {
          const Rec c = ld_rec(rec, k);
          const float q0 = c.x - yp, q1 = (c.y - zref) - dzp;
          if (!(fabsf(q0) <= wy && fabsf(q1) <= wz)) continue;
          const float chi2 = chi2_of(I, q0, q1);
          ncand++;
          const int ci = rec_idx(c);
          if (!have || chi2 < best || (chi2 == best && ci < bi)) {
            have = true;
            best = chi2;
            bi = ci;
            bk = k;
            by = c.x;
            bz = c.y;
          }
        }
      }
    }
    // ---- decision: R14 start hit / R15 chain cut (a bad chi2 discards the prediction) / R16 cut ----
    bool upd = isI;
    float my = yp, mz = 0.0f;  // R14: update with the start hit itself (yp == y0, dz == 0)
    int mk = p0;
    if (chain && ok) {
      if (!have || best > sc.chi2_chain_cut) ok = false;
      else upd = true;
    }
    if (leg && have && best < sc.chi2_cut) upd = true;
    if (!isI && upd) {
      my = by;
      mz = bz - zref;
      mk = bk;
    }
    // ---- look one step ahead (prefetch only: nothing below depends on it) ---------------------------
    //   next chain cluster: its record;  next row of a leg (or the first row after the chain): the bin at the
    //   linearly extrapolated position -- its offset is loaded now (in flight during the update) and the
    //   records behind it are prefetched at the top of the next iteration.  st still holds the state at the
    //   previous row here, so the slope costs two subtractions.
    if (TPC_FOLLOW_PREFETCH && chain && upd && nxt >= 0) prefetch_l1(rec + nxt);
    if (TPC_FOLLOW_PREFETCH && moved && ok && !isJ) {
      const int r2 = rn + ((phase == PH_DOWN) ? -1 : 1);
      if (r2 >= 0 && r2 < nrows) {
        const float y2 = yp + (yp - st.p[0]);
        const float z2 = zref + (dzp + (dzp - st.p[1]));
        const float zeta = (s < 18) ? z2 : -z2;
        const int ny2 = sm.ny[r2];
        const int zb = clampbin((zeta - sc.z_lo) * sc.inv_cz, sc.nz);
        const int yb = clampbin((y2 + sm.ymax[r2]) * sc.inv_cy, ny2);
        pf_ka = __ldg(bin_first + (s * sc.bins_per_sector + sm.rowbase[r2] + zb * ny2 + yb));
      }
    }
    // ---- commit the transport, R13 update (one copy for every phase) --------------------------------
    __syncwarp();
    if (moved && ok) transport_apply(st, T);
    if (ok) r_at = rn;
    if (upd) {
      update(st, I, my, mz);
      nupd++;
      nh++;
      lo = min(lo, rn);
      hi = max(hi, rn);
    }
    // ---- bookkeeping and phase transitions ---------------------------------------------------------------
    __syncwarp();
    const bool searched = leg && ok && !edge_out;
    if (upd || searched) row_hit[(int64_t)t * nrows + rn] = upd ? mk : -1;
    bool finish = false;
    if (isI) {
      phase = PH_CHAIN;
    } else if (chain) {
      if (upd) hn = nxt;
      if (!upd || hn < 0) {  // end of the chain phase: R16 upward from the last chain hit
        phase = PH_UP;
        r = r_at + 1;
        misses = 0;
        if (r >= nrows) phase = PH_JUMP;
      }
    } else if (leg) {
      misses = upd ? 0 : misses + 1;
      r += (phase == PH_UP) ? 1 : -1;
      if (!searched || misses > sc.max_gap || r < 0 || r >= nrows) {  // end of the leg
        if (phase == PH_UP) phase = PH_JUMP;  // R17
        else finish = true;
      }
    } else if (isJ) {
      phase = PH_DOWN;
      r = r0 - 1;
      misses = 0;
      if (!ok || r < 0) finish = true;
    }
    if (finish) {  // R18 record; the R20 key is pushed by k_push_keys
      tl_info[t] = nh | (lo << 8) | (hi << 16);
      tl_key[t] = sel_key(nh, orig0, t);
      phase = PH_FETCH;
    }
  }
  // one 64-bit atomic per warp and counter
#pragma unroll
  for (int k = 0; k < 3; k++) {
    unsigned long long v = k == 0 ? nprop : (k == 1 ? nupd : ncand);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(kFull, v, d);
    if (lane == 0 && v) atomicAdd((unsigned long long*)(ws_counters + WC_PROP64) + k, v);
  }
}

int g_follow_blocks = 0;

}  // namespace

cudaError_t launch_follow(const Geo& g, const Ws& w, cudaStream_t st) {
  cudaError_t e;
  if (g_follow_blocks == 0) {
    int dev = 0, sms = 0, per_sm = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_follow, kFollowThreads, 0)) != cudaSuccess) return e;
    g_follow_blocks = sms * (per_sm > 0 ? per_sm : 1);
  }
  TPC_LAUNCH(KID_FOLLOW, st,
             (k_follow<<<g_follow_blocks, kFollowThreads, 0, st>>>(g, w.rec, w.bin_first, w.up_c, w.tl_init, w.row_hit,
                                                                  w.tl_info, w.tl_key, w.counters)));
  return cudaGetLastError();
}

}  // namespace tpc
