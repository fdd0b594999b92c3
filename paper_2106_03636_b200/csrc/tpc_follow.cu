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
// waiting for the longest tracklet of a batch).  Tracklets are queued in grid order, so
// concurrently running lanes walk neighbouring bins (L2 locality of the R16 lookups).
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

constexpr int kFollowThreads = 128;
constexpr unsigned kFull = 0xffffffffu;

enum Phase { PH_FETCH = 0, PH_INIT, PH_CHAIN, PH_UP, PH_JUMP, PH_DOWN, PH_DONE };

__global__ void __launch_bounds__(kFollowThreads)
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
  unsigned long long work[3] = {0ull, 0ull, 0ull};

  // per-lane tracklet state
  int phase = PH_FETCH;
  KState st;
  float zref = 0.0f;
  int t = 0, s = 0, r0 = 0, r_at = 0, r = 0, hn = -1, p0 = 0, orig0 = 0;
  int misses = 0, nh = 0, lo = 0, hi = 0;
  unsigned nprop = 0, nupd = 0, ncand = 0;
  int32_t* my_hits = row_hit;
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
          my_hits = row_hit + (int64_t)t * nrows;
          nh = 0;
          lo = hi = r_at = r0;
          nprop = nupd = ncand = 0;
          phase = PH_INIT;
        }
      }
    }
    if (__all_sync(kFull, phase == PH_DONE)) break;

    // ---- target row of this step; chain steps prefetch their cluster and the next link ---------
    const bool chain = phase == PH_CHAIN;
    const bool leg = phase == PH_UP || phase == PH_DOWN;
    int rn = r0;                      // PH_INIT, PH_JUMP
    if (chain) rn = r_at + 1;         // links join adjacent rows (R9)
    if (leg) rn = r;
    Rec cpre = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    int nxt = -1;
    if (chain) {
      cpre = ld_rec(rec, hn);
      nxt = __ldg(up_c + hn);
    }
    // ---- R12 transport (one copy for every phase) -----------------------------------------------
    KState nx = st;
    bool ok = phase != PH_DONE;
    if (ok && phase != PH_INIT) {
      ok = propagate(nx, sm.X[rn] - sm.X[r_at], kB, ms);
      if (ok) nprop++;
    }
    const Innov I = innovation(nx, sy2, sz2);
    // ---- measurement for this step ----------------------------------------------------------------
    bool upd = false, edge_out = false;
    float my = 0.0f, mz = 0.0f;
    int mk = -1;
    if (phase == PH_INIT) {  // R14: update with the start hit itself
      upd = true;
      my = nx.p[0];
      mz = 0.0f;
      mk = p0;
    } else if (chain && ok) {  // R15: the linked cluster, no window; a bad chi2 discards the prediction
      const float chi2 = chi2_of(I, cpre.x - nx.p[0], (cpre.y - zref) - nx.p[1]);
      if (chi2 > sc.chi2_chain_cut) {
        ok = false;
      } else {
        upd = true;
        my = cpre.x;
        mz = cpre.y - zref;
        mk = hn;
      }
    } else if (leg && ok) {  // R16: windowed arg-min chi2 over the row
      edge_out = fabsf(nx.p[0]) > sm.ymax[rn] + sc.edge_margin;
      if (!edge_out) {
        const float wy = fminf(sqrtf(sc.chi2_cut * I.S00), sc.win_max);
        const float wz = fminf(sqrtf(sc.chi2_cut * I.S11), sc.win_max);
        const float yp = nx.p[0], dzp = nx.p[1];
        const float zc = zref + dzp;
        const BinWin W = bin_window(sm, sc, s, rn, yp - wy, yp + wy, zc - wz, zc + wz);
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
          upd = true;
          my = by;
          mz = bz - zref;
          mk = bk;
        }
      }
    }
    // commit the transport (a failed one leaves the state where it was, R15)
    if (ok) st = nx;
    // ---- R13 update (one copy for every phase) -----------------------------------------------------
    if (upd) {
      update(st, I, my, mz);
      nupd++;
    }
    // ---- bookkeeping and phase transitions ------------------------------------------------------------
    bool finish = false, end_leg = false;
    switch (phase) {
      case PH_INIT:
        my_hits[r0] = p0;
        nh = 1;
        phase = PH_CHAIN;
        break;
      case PH_CHAIN:
        if (upd) {
          my_hits[rn] = mk;
          nh++;
          hi = rn;
          r_at = rn;
          hn = nxt;
        }
        if (!upd || hn < 0) {  // end of the chain phase: R16 upward from the last chain hit
          phase = PH_UP;
          r = r_at + 1;
          misses = 0;
          if (r >= nrows) phase = PH_JUMP;
        }
        break;
      case PH_UP:
      case PH_DOWN:
        if (!ok) {
          end_leg = true;
        } else {
          r_at = rn;
          if (edge_out) {
            end_leg = true;  // left the sector
          } else {
            if (upd) {
              my_hits[rn] = mk;
              nh++;
              lo = min(lo, rn);
              hi = max(hi, rn);
              misses = 0;
            } else {
              my_hits[rn] = -1;
              misses++;
              if (misses > sc.max_gap) end_leg = true;
            }
            if (!end_leg) {
              r += (phase == PH_UP) ? 1 : -1;
              if (r < 0 || r >= nrows) end_leg = true;
            }
          }
        }
        if (end_leg) {
          if (phase == PH_UP) phase = PH_JUMP;  // R17
          else finish = true;
        }
        break;
      case PH_JUMP:
        if (!ok) {
          finish = true;
        } else {
          r_at = r0;
          phase = PH_DOWN;
          r = r0 - 1;
          misses = 0;
          if (r < 0) finish = true;
        }
        break;
      default:
        break;
    }
    if (finish) {  // R18 record; the R20 key is pushed by k_push_keys
      tl_info[t] = nh | (lo << 8) | (hi << 16);
      tl_key[t] = sel_key(nh, orig0, t);
      work[0] += nprop;
      work[1] += nupd;
      work[2] += ncand;
      phase = PH_FETCH;
    }
  }
  // one 64-bit atomic per warp and counter
#pragma unroll
  for (int k = 0; k < 3; k++) {
    unsigned long long v = work[k];
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
