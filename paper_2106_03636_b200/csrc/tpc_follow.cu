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
#include "tpc_scan.cuh"
#include "tpc_search.cuh"

namespace tpc {

namespace {

// 64-thread blocks, 10 per SM: 96 registers per thread without spills and 20 resident warps per SM (measured on
// configs[4], before R17: 128 x 4 blocks at 112 registers = 16 warps: 28.0 ms; 64 x 10 at 96 registers: 25.3 ms;
// with the R17 waves a batch of 2 candidate records is the optimum: 11.0 ms against 11.3 with 3 and 12.3 with 4)
constexpr int kFollowThreads = 64;
constexpr int kFollowMinBlocks = 10;
constexpr unsigned kFull = 0xffffffffu;
constexpr int kBatch = 2;  // candidate records in flight per lane in the R15/R16 search

enum Phase { PH_FETCH = 0, PH_INIT, PH_CHAIN, PH_UP, PH_JUMP, PH_DOWN, PH_DONE };

// PHASE_B = false: phase A (R14 init, R15 chain, R16 upward leg) for the tracklets of one wave, listed in `surv`
// (R17: first the start hits without a plausible predecessor, then those of the rest that nobody picked up); the
// state at the end of the upward leg goes to tl_state, and every START hit an upward leg attaches is marked in `picked` (R17).
// PHASE_B = true: the tracklets listed in `surv` (start hit not picked up) resume from tl_state with the R17 jump
// and the R16 downward leg, and write their R18 record and R20 key.
template <bool PHASE_B>
__global__ void __launch_bounds__(kFollowThreads, kFollowMinBlocks)
k_follow(const __grid_constant__ Geo g, const Rec* __restrict__ rec, const int32_t* __restrict__ bin_first,
         const int32_t* __restrict__ up_c, const TlInit* __restrict__ tl_init, int32_t* __restrict__ row_hit,
         int32_t* __restrict__ tl_info, unsigned long long* __restrict__ tl_key, float4* __restrict__ tl_state,
         const int32_t* __restrict__ surv, uint8_t* __restrict__ picked, int32_t* __restrict__ ws_counters) {
  __shared__ SmRow sm;
  load_rows(sm, g);
  __syncthreads();
  const Scalars& sc = g.s;
  const int nrows = sc.nrows;
  const int n_starts = PHASE_B ? ws_counters[WC_N_SURV] : ws_counters[WC_N_WAVE];  // entries of `surv` to work on
  const int lane = threadIdx.x & 31;
  const float kB = sc.kB, ms = sc.max_sinphi, sy2 = sc.sy2, sz2 = sc.sz2;

  // per-lane tracklet state
  int phase = PH_FETCH;
  KState st;
  float zref = 0.0f;
  int t = 0, s = 0, r0 = 0, r_at = 0, r = 0, hn = -1, p0 = 0, orig0 = 0;
  int misses = 0, nh = 0, lo = 0, hi = 0;
  unsigned nprop = 0, nupd = 0, ncand = 0, nclaims = 0;  // work counters of this lane over all its tracklets
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
      if (lane == leader) base = atomicAdd(ws_counters + (PHASE_B ? WC_QUEUE_B : WC_QUEUE), __popc(need));
      base = __shfl_sync(kFull, base, leader);
      if (phase == PH_FETCH) {
        const int q = base + __popc(need & ((1u << lane) - 1u));
        if (q >= n_starts) {
          phase = PH_DONE;
        } else if (PHASE_B) {
          t = __ldg(surv + q);
          const float4 b = __ldg(reinterpret_cast<const float4*>(tl_init + t) + 1);
          const float4* sp = tl_state + (int64_t)t * kStateVec;
          const float4 v0 = sp[0], v1 = sp[1], v2 = sp[2], v3 = sp[3], v4 = sp[4], v5 = sp[5];
          p0 = __float_as_int(b.x);
          const int sr0 = __float_as_int(b.z);
          orig0 = __float_as_int(b.w);
          s = sr0 / nrows;
          r0 = sr0 - s * nrows;
          st.p[0] = v0.x; st.p[1] = v0.y; st.p[2] = v0.z; st.p[3] = v0.w; st.p[4] = v1.x;
          st.C[0] = v1.y; st.C[1] = v1.z; st.C[2] = v1.w;
          st.C[3] = v2.x; st.C[4] = v2.y; st.C[5] = v2.z; st.C[6] = v2.w;
          st.C[7] = v3.x; st.C[8] = v3.y; st.C[9] = v3.z; st.C[10] = v3.w;
          st.C[11] = v4.x; st.C[12] = v4.y; st.C[13] = v4.z; st.C[14] = v4.w;
          zref = v5.x;
          r_at = __float_as_int(v5.y);
          const int info = __float_as_int(v5.z);
          nh = info & 0xff;
          lo = (info >> 8) & 0xff;
          hi = (info >> 16) & 0xff;
          phase = PH_JUMP;
        } else {
          t = __ldg(surv + q);
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
          nh = 0;
          lo = hi = r_at = r0;
          phase = PH_INIT;
        }
      }
    }
    if (__all_sync(kFull, phase == PH_DONE)) break;

    // ---- target row of this step; chain steps prefetch their next link --------------------------
    // phase A never sees PH_JUMP / PH_DOWN, phase B never PH_INIT / PH_CHAIN / PH_UP: the template prunes them
    const bool isI = !PHASE_B && phase == PH_INIT, chain = !PHASE_B && phase == PH_CHAIN, isJ = PHASE_B && phase == PH_JUMP;
    const bool leg = PHASE_B ? phase == PH_DOWN : phase == PH_UP;
    int rn = r0;                      // PH_INIT, PH_JUMP
    if (chain) rn = r_at + 1;         // links join adjacent rows (R9)
    if (leg) rn = r;
    int nxt = -1;
    if (chain) nxt = __ldg(up_c + hn);
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
    bool have = false, bstart = false;  // bstart: the best candidate is a start hit (R17 marking)
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
          bstart = rec_is_start(cs);
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
              bstart = rec_is_start(c[j]);
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
            bstart = rec_is_start(c);
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
    if (!PHASE_B && leg && upd && bstart) picked[mk] = 1;  // R17: an upward leg attached another tracklet's start hit
    bool finish = false;  // phase A: end of the upward leg; phase B: end of the tracklet
    if (isI) {
      phase = PH_CHAIN;
    } else if (chain) {
      if (upd) hn = nxt;
      if (!upd || hn < 0) {  // end of the chain phase: R16 upward from the last chain hit
        phase = PH_UP;
        r = r_at + 1;
        misses = 0;
        if (r >= nrows) finish = true;
      }
    } else if (leg) {
      misses = upd ? 0 : misses + 1;
      r += PHASE_B ? -1 : 1;
      if (!searched || misses > sc.max_gap || r < 0 || r >= nrows) finish = true;  // end of the leg
    } else if (isJ) {  // R17
      phase = PH_DOWN;
      r = r0 - 1;
      misses = 0;
      if (!ok || r < 0) finish = true;
    }
    if (finish) {
      if (PHASE_B) {  // R18 record; the R20 key is pushed by k_push_keys
        tl_info[t] = nh | (lo << 8) | (hi << 16);
        tl_key[t] = sel_key(nh, orig0, t);
        nclaims += nh;
      } else {  // park the state: phase B resumes it if no upward leg picked this tracklet's start hit up
        float4* sp = tl_state + (int64_t)t * kStateVec;
        sp[0] = make_float4(st.p[0], st.p[1], st.p[2], st.p[3]);
        sp[1] = make_float4(st.p[4], st.C[0], st.C[1], st.C[2]);
        sp[2] = make_float4(st.C[3], st.C[4], st.C[5], st.C[6]);
        sp[3] = make_float4(st.C[7], st.C[8], st.C[9], st.C[10]);
        sp[4] = make_float4(st.C[11], st.C[12], st.C[13], st.C[14]);
        sp[5] = make_float4(zref, __int_as_float(r_at), __int_as_float(nh | (lo << 8) | (hi << 16)), 0.0f);
      }
      phase = PH_FETCH;
    }
  }
  // one 64-bit atomic per warp and counter
#pragma unroll
  for (int k = 0; k < 4; k++) {
    unsigned long long v = k == 0 ? nprop : (k == 1 ? nupd : (k == 2 ? ncand : nclaims));
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(kFull, v, d);
    if (lane == 0 && v) atomicAdd((unsigned long long*)(ws_counters + WC_PROP64) + k, v);
  }
}

int g_follow_blocks[kMaxDevices] = {0};  // resident blocks of k_follow per device

}  // namespace

namespace {

constexpr int kThreads = 256;

// R17 wave test, one thread per tracklet: does the backward straight line through the start hit and its up-neighbour
// meet, within max_gap + 3 rows below, the top of a lower chain (up' == -2)?  Tolerance 4 sigma per (rows + 1).
// Such a start hit waits for the first wave.  The answer is kept in tl_info[t] until phase B overwrites it.
__global__ void __launch_bounds__(kThreads)
k_wave_test(const __grid_constant__ Geo g, const Rec* __restrict__ rec, const int32_t* __restrict__ bin_first,
            const int32_t* __restrict__ up_c, const TlInit* __restrict__ tl_init, int32_t* __restrict__ tl_info,
            const int32_t* __restrict__ ws_counters) {
  __shared__ SmRow sm;
  load_rows(sm, g);
  __syncthreads();
  const Scalars& sc = g.s;
  const int nrows = sc.nrows;
  const int n_starts = ws_counters[WC_N_STARTS];
  const float sig_y = sc.sig_y, sig_z = sc.sig_z;
  for (int64_t t = (int64_t)blockIdx.x * kThreads + threadIdx.x; t < n_starts; t += (int64_t)gridDim.x * kThreads) {
    const float4* ip = reinterpret_cast<const float4*>(tl_init + t);
    const float4 a = __ldg(ip), b = __ldg(ip + 1);
    const int sr0 = __float_as_int(b.z);
    const int s = sr0 / nrows, r0 = sr0 - s * nrows;
    const float dxu = sm.X[r0 + 1] - sm.X[r0];
    const float my = (a.z - a.x) / dxu, mz = (a.w - a.y) / dxu;
    bool found = false;
    for (int k = 1; k <= sc.max_gap + 3 && !found; k++) {
      const int r = r0 - k;
      if (r < 0) break;
      const float dxk = sm.X[r0] - sm.X[r];
      const float yp = a.x - my * dxk, zp = a.y - mz * dxk;
      const float ty = (4.0f * sig_y) * (float)(k + 1), tz = (4.0f * sig_z) * (float)(k + 1);
      const BinWin W = bin_window(sm, sc, s, r, yp - ty, yp + ty, zp - tz, zp + tz);
      for (int zi = 0; zi < W.nzb && !found; zi++) {
        const int b0 = W.first + zi * W.ny;
        const int ka = __ldg(bin_first + b0), ke = __ldg(bin_first + b0 + W.ybspan);
        for (int c = ka; c < ke; c++) {
          const Rec h = ld_rec(rec, c);
          if (fabsf(h.x - yp) <= ty && fabsf(h.y - zp) <= tz && __ldg(up_c + c) == -2) found = true;
        }
      }
    }
    tl_info[t] = found ? 1 : 0;
  }
}

// R17 lists.  mode 0: first wave = start hits that do not wait;  mode 1: second wave = waiting start hits that no
// upward leg of the first wave picked up;  mode 2: phase B = tracklets whose start hit nobody picked up -- all
// others (absorbed, or never run) get an empty R18 record (nHits = 0, empty row range) that selection and export skip.
__global__ void __launch_bounds__(kThreads)
k_list_flags(int mode, int64_t scap_pad, const TlInit* __restrict__ tl_init, const uint8_t* __restrict__ picked,
             int32_t* __restrict__ tl_info, int32_t* __restrict__ flag, const int32_t* __restrict__ ws_counters) {
  const int n_starts = ws_counters[WC_N_STARTS];  // flag[] beyond it was zeroed by the caller (memset)
  (void)scap_pad;
  for (int64_t t = (int64_t)blockIdx.x * kThreads + threadIdx.x; t < n_starts; t += (int64_t)gridDim.x * kThreads) {
    int f = 0;
    {
      if (mode == 0) {
        f = tl_info[t] ? 0 : 1;
      } else {
        const bool pk = picked[tl_init[t].p0] != 0;
        if (mode == 1) {
          f = (tl_info[t] && !pk) ? 1 : 0;
        } else {
          f = pk ? 0 : 1;
          if (!f) tl_info[t] = 0 | (1 << 8) | (0 << 16);
        }
      }
    }
    flag[t] = f;
  }
}

__global__ void __launch_bounds__(kThreads)
k_list_build(int count_index, int64_t scap_pad, const int32_t* __restrict__ scan, int32_t* __restrict__ list,
             int32_t* __restrict__ ws_counters) {
  const int n_starts = ws_counters[WC_N_STARTS];
  if (blockIdx.x == 0 && threadIdx.x == 0) ws_counters[count_index] = scan[scap_pad];
  for (int64_t t = (int64_t)blockIdx.x * kThreads + threadIdx.x; t < n_starts; t += (int64_t)gridDim.x * kThreads) {
    const int i = scan[t];
    if (scan[t + 1] != i) list[i] = (int)t;
  }
}

}  // namespace

cudaError_t launch_follow(const Geo& g, const Ws& w, cudaStream_t st) {
  cudaError_t e;
  const int64_t scap_pad = w.L.scap_pad;
  int dev = 0;
  if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
  int& follow_blocks = g_follow_blocks[dev < kMaxDevices ? dev : kMaxDevices - 1];
  if (follow_blocks == 0 || dev >= kMaxDevices) {
    int sms = 0, per_sm = 0;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_follow<false>, kFollowThreads, 0)) != cudaSuccess) return e;
    follow_blocks = sms * (per_sm > 0 ? per_sm : 1);
  }
  if ((e = cudaMemsetAsync(w.picked, 0, (size_t)(w.L.n + 1), st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(w.counters + WC_QUEUE_B, 0, sizeof(int32_t) * 3, st)) != cudaSuccess) return e;  // + N_SURV, N_WAVE
  TPC_LAUNCH(KID_SURVIVORS, st,
             (k_wave_test<<<blocks_for(w.L.scap, kThreads), kThreads, 0, st>>>(g, w.rec, w.bin_first, w.up_c, w.tl_init, w.tl_info,
                                                                              w.counters)));
  for (int mode = 0; mode < 3; mode++) {  // two waves of phase A, then phase B
    if ((e = cudaMemsetAsync(w.surv_scan, 0, sizeof(int32_t) * (size_t)(scap_pad + 2), st)) != cudaSuccess) return e;
    TPC_LAUNCH(KID_SURVIVORS, st,
               (k_list_flags<<<blocks_for(scap_pad + 1, kThreads), kThreads, 0, st>>>(mode, scap_pad, w.tl_init, w.picked, w.tl_info,
                                                                                      w.surv_scan, w.counters)));
    if ((e = exclusive_scan<int32_t>(w.surv_scan, w.surv_scan, scap_pad + 1, (int32_t*)w.scan_tmp, st)) != cudaSuccess) return e;
    TPC_LAUNCH(KID_SURVIVORS, st,
               (k_list_build<<<blocks_for(scap_pad, kThreads), kThreads, 0, st>>>(mode == 2 ? WC_N_SURV : WC_N_WAVE, scap_pad,
                                                                                  w.surv_scan, w.surv, w.counters)));
    if (mode < 2) {
      if ((e = cudaMemsetAsync(w.counters + WC_QUEUE, 0, sizeof(int32_t), st)) != cudaSuccess) return e;
      TPC_LAUNCH(KID_FOLLOW, st,
                 (k_follow<false><<<follow_blocks, kFollowThreads, 0, st>>>(g, w.rec, w.bin_first, w.up_c, w.tl_init, w.row_hit,
                                                                             w.tl_info, w.tl_key, w.tl_state, w.surv, w.picked,
                                                                             w.counters)));
    } else {
      TPC_LAUNCH(KID_FOLLOW_B, st,
                 (k_follow<true><<<follow_blocks, kFollowThreads, 0, st>>>(g, w.rec, w.bin_first, w.up_c, w.tl_init, w.row_hit,
                                                                            w.tl_info, w.tl_key, w.tl_state, w.surv, w.picked,
                                                                            w.counters)));
    }
  }
  return cudaGetLastError();
}

}  // namespace tpc
