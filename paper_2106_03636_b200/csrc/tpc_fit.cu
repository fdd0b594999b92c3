// =============================================================================================
// tpc_fit.cu -- step 3b of the hot path (BASELINE.json north_star (3) "refit of helices ... with
// the time offset left free"): per accepted track, a 3-point circle seed
// followed by an outward and an inward fp32 Kalman pass over its hit list.
//
//   k_fit         one LANE per track, 5-parameter state + 15 covariance elements in registers.  Reads
//                 the (y, z, row) records that tpc_find_tracks stored in hit-list order (one
//                 sequential 16-byte stream per track).  Like the follower it is one loop with a
//                 single copy of transport + update; a lane that finishes its track pulls the next
//                 one from a queue, so the lanes of a warp stay busy whatever the track lengths.
//   k_fit_gather  same arithmetic, hits gathered through the caller's y / z / sector_row arrays
//                 (original indices): self-contained, refits any hit lists (e.g. truth hits).
// The track count K is read from counters[TPC_CNT_TRACKS] on the device (no host sync).
// =============================================================================================
#include "tpc_common.cuh"
#include "tpc_kalman.cuh"
#include "tpc_prof.cuh"

namespace tpc {

namespace {

constexpr int kFitThreads = 128;

__global__ void __launch_bounds__(kFitThreads)
k_fit_gather(const __grid_constant__ Geo g, const float* __restrict__ y, const float* __restrict__ z,
      const int32_t* __restrict__ sector_row, const int32_t* __restrict__ counters, int64_t max_tracks,
      const int32_t* __restrict__ trk_nhits, const int64_t* __restrict__ trk_first_hit,
      const int32_t* __restrict__ trk_hits, float* __restrict__ par, float* __restrict__ cov, float* __restrict__ xref,
      float* __restrict__ zref_out, float* __restrict__ chi2_out, int32_t* __restrict__ ndf) {
  __shared__ float sX[kMaxRows];
  const Scalars& sc = g.s;
  const int nrows = sc.nrows;
  for (int r = threadIdx.x; r < nrows; r += blockDim.x) sX[r] = g.row.X[r];
  __syncthreads();
  int64_t K = counters[TPC_CNT_TRACKS];
  if (K > max_tracks) K = max_tracks;
  const float kB = sc.kB, ms = sc.max_sinphi, sy2 = sc.sy2, sz2 = sc.sz2;
  for (int64_t k = (int64_t)blockIdx.x * kFitThreads + threadIdx.x; k < K; k += (int64_t)gridDim.x * kFitThreads) {
    const int n = trk_nhits[k];
    const int32_t* hits = trk_hits + trk_first_hit[k];
    auto rowx = [&](int h) { return sX[__ldg(sector_row + h) % nrows]; };
    // R21: seed from the first, middle and last hit
    const int a = hits[0], b = hits[n / 2], c = hits[n - 1], h1 = hits[n > 1 ? 1 : 0];
    const float x1 = rowx(a), y1 = __ldg(y + a), x2 = rowx(b), y2 = __ldg(y + b), x3 = rowx(c), y3 = __ldg(y + c);
    const float cross = (x2 - x1) * (y3 - y1) - (x3 - x1) * (y2 - y1);
    const float d12 = sqrtf((x2 - x1) * (x2 - x1) + (y2 - y1) * (y2 - y1));
    const float d23 = sqrtf((x3 - x2) * (x3 - x2) + (y3 - y2) * (y3 - y2));
    const float d13 = sqrtf((x3 - x1) * (x3 - x1) + (y3 - y1) * (y3 - y1));
    const float kappa = (2.0f * cross) / ((d12 * d23) * d13);  // signed curvature of the circumcircle
    const float dx = rowx(h1) - x1, dy = __ldg(y + h1) - y1;
    const float ch = sqrtf(dx * dx + dy * dy);
    float sphi = dy / ch - ((kappa * ch) * 0.5f) * (dx / ch);  // chord direction rotated back by half the turn
    if (sphi > ms) sphi = ms;
    if (sphi < -ms) sphi = -ms;
    const float zref = __ldg(z + a);
    KState st;
    st.p[0] = y1;
    st.p[1] = 0.0f;
    st.p[2] = sphi;
    st.p[3] = (__ldg(z + h1) - zref) / ch;
    st.p[4] = -(kappa / kB);
    // R22: pass 1 inner -> outer, pass 2 outer -> inner, ...; covariance reset at the start of every pass
    float chi2 = 0.0f;
    float x_at = x1;
    bool ok = true;
    for (int pass = 0; pass < sc.n_fit_passes && ok; pass++) {
      reset_cov(st, sc.cov0);
      chi2 = 0.0f;
      const int dir = (pass & 1) ? -1 : 1;
      int i = dir > 0 ? 0 : n - 1;
      for (int cnt = 0; cnt < n; cnt++, i += dir) {
        const int h = hits[i];
        const float xh = rowx(h);
        if (cnt > 0) {  // the first hit of a pass is the one the state already sits at (no transport)
          if (!propagate(st, xh - x_at, kB, ms)) {
            ok = false;
            break;
          }
          x_at = xh;
        }
        const Innov I = innovation(st, sy2, sz2);
        chi2 = chi2 + update(st, I, __ldg(y + h), __ldg(z + h) - zref);
      }
    }
#pragma unroll
    for (int i = 0; i < 5; i++) par[(int64_t)i * max_tracks + k] = st.p[i];
#pragma unroll
    for (int i = 0; i < 15; i++) cov[(int64_t)i * max_tracks + k] = st.C[i];
    xref[k] = x_at;
    zref_out[k] = zref;
    chi2_out[k] = ok ? chi2 : -1.0f;
    ndf[k] = ok ? 2 * n - 5 : -1;
  }
}

// R28: k_fit_gather with process noise after every transport (R28a) and outlier
// rejection in the last pass (R28b).  x0inv = 0 and outlier_cut <= 0 give k_fit_gather's results bit for bit.
__device__ __forceinline__ void add_scattering(KState& st, float arc, float x0inv) {
  if (!(x0inv > 0.0f)) return;
  const float s = st.p[2], tl = st.p[3], q = st.p[4];
  const float one_tl2 = 1.0f + tl * tl;
  const float L = fabsf(arc) * sqrtf(one_tl2);
  const float th2 = (((0.0136f * 0.0136f) * (q * q)) / one_tl2) * (L * x0inv);
  st.C[TPC_CI(2, 2)] = st.C[TPC_CI(2, 2)] + (th2 * (1.0f - s * s)) * one_tl2;
  st.C[TPC_CI(3, 3)] = st.C[TPC_CI(3, 3)] + (th2 * one_tl2) * one_tl2;
  st.C[TPC_CI(4, 3)] = st.C[TPC_CI(4, 3)] + ((th2 * tl) * q) * one_tl2;
  st.C[TPC_CI(4, 4)] = st.C[TPC_CI(4, 4)] + ((th2 * tl) * tl) * (q * q);
}

// R28d: mean energy loss over |arc| (dir > 0 outward: momentum is lost; inward: gained back) and its straggling
__device__ __forceinline__ void add_energy_loss(KState& st, float arc, int dir, float dedx, float eloss_sigma) {
  if (!(dedx > 0.0f)) return;
  const float q = st.p[4];
  const float rel = (dedx * fabsf(arc)) * fabsf(q);
  const float dq = rel * q;
  st.p[4] = dir > 0 ? q + dq : q - dq;
  st.C[TPC_CI(4, 4)] = st.C[TPC_CI(4, 4)] + (eloss_sigma * dq) * (eloss_sigma * dq);
}

// R28e: the two measurement variances at a hit of raw z for the predicted state; zs = side v_drift t0
__device__ __forceinline__ void cluster_errors(const KState& st, const tpc_fit_options_t& o, float sy2, float sz2, bool have_d,
                                               float z_raw, float zs, float& ey, float& ez) {
  ey = sy2;
  ez = sz2;
  if (o.err_ang_y > 0.0f) {
    const float s = st.p[2];
    const float tan2 = (s * s) / (1.0f - s * s);
    ey = ey * (1.0f + o.err_ang_y * tan2);
  }
  if (o.err_ang_z > 0.0f) {
    const float tl = st.p[3];
    ez = ez * (1.0f + o.err_ang_z * (tl * tl));
  }
  if (have_d) {
    float d = o.z_len - fabsf(z_raw + zs);
    if (d < 0.0f) d = 0.0f;
    if (o.err_drift_y > 0.0f) ey = ey + o.err_drift_y * d;
    if (o.err_drift_z > 0.0f) ez = ez + o.err_drift_z * d;
  }
}

// REC: hits streamed from the workspace's track-ordered records (y, z, row, orig) that tpc_find_tracks wrote (one
// sequential 16-byte stream per track, as in k_fit); else gathered through y / z / sector_row and trk_hits.
template <bool REC>
__global__ void __launch_bounds__(kFitThreads)
k_fit_physics(const __grid_constant__ Geo g, const __grid_constant__ tpc_fit_options_t opt, const float4* __restrict__ hit_rec,
              const float* __restrict__ y, const float* __restrict__ z, const int32_t* __restrict__ sector_row,
              const int32_t* __restrict__ counters, int64_t max_tracks, const int32_t* __restrict__ trk_nhits,
              const int64_t* __restrict__ trk_first_hit, const int32_t* __restrict__ trk_hits, const float* __restrict__ trk_t0,
              float* __restrict__ par, float* __restrict__ cov, float* __restrict__ xref, float* __restrict__ zref_out,
              float* __restrict__ chi2_out, int32_t* __restrict__ ndf, uint8_t* __restrict__ hit_flag) {
  __shared__ float sX[kMaxRows];
  const Scalars& sc = g.s;
  const int nrows = sc.nrows;
  for (int r = threadIdx.x; r < nrows; r += blockDim.x) sX[r] = g.row.X[r];
  __syncthreads();
  int64_t K = counters[TPC_CNT_TRACKS];
  if (K > max_tracks) K = max_tracks;
  const float kB = sc.kB, ms = sc.max_sinphi, sy2 = sc.sy2, sz2 = sc.sz2;
  for (int64_t k = (int64_t)blockIdx.x * kFitThreads + threadIdx.x; k < K; k += (int64_t)gridDim.x * kFitThreads) {
    const int n = trk_nhits[k];
    const int64_t first = trk_first_hit[k];
    // hit i of the list as (y, raw z, x of its row, original cluster index)
    auto hit_at = [&](int i) {
      if (REC) {
        const float4 r = __ldg(hit_rec + first + i);
        return make_float4(r.x, r.y, sX[__float_as_int(r.z)], r.w);
      }
      const int h = trk_hits[first + i];
      return make_float4(__ldg(y + h), __ldg(z + h), sX[__ldg(sector_row + h) % nrows], __int_as_float(h));
    };
    const float4 ha = hit_at(0), hb = hit_at(n / 2), hc = hit_at(n - 1), hh1 = hit_at(n > 1 ? 1 : 0);
    const float x1 = ha.z, y1 = ha.x, x2 = hb.z, y2 = hb.x, x3 = hc.z, y3 = hc.x;
    const float cross = (x2 - x1) * (y3 - y1) - (x3 - x1) * (y2 - y1);
    const float d12 = sqrtf((x2 - x1) * (x2 - x1) + (y2 - y1) * (y2 - y1));
    const float d23 = sqrtf((x3 - x2) * (x3 - x2) + (y3 - y2) * (y3 - y2));
    const float d13 = sqrtf((x3 - x1) * (x3 - x1) + (y3 - y1) * (y3 - y1));
    const float kappa = (2.0f * cross) / ((d12 * d23) * d13);
    const float dx = hh1.z - x1, dy = hh1.x - y1;
    const float ch = sqrtf(dx * dx + dy * dy);
    float sphi = dy / ch - ((kappa * ch) * 0.5f) * (dx / ch);
    if (sphi > ms) sphi = ms;
    if (sphi < -ms) sphi = -ms;
    const float zref = ha.y;
    KState st;
    st.p[0] = y1;
    st.p[1] = 0.0f;
    st.p[2] = sphi;
    st.p[3] = (hh1.y - zref) / ch;
    st.p[4] = -(kappa / kB);
    float chi2 = 0.0f;
    float x_at = x1;
    int nrej = 0;
    bool ok = true;
    for (int i = 0; i < n; i++) hit_flag[first + i] = 0;
    const float t0 = trk_t0 ? trk_t0[k] : 0.0f;
    const bool have_d = trk_t0 && t0 == t0;
    const float side = (__ldg(sector_row + __float_as_int(ha.w)) / nrows) < 18 ? 1.0f : -1.0f;
    const float zs = have_d ? side * (opt.v_drift * t0) : 0.0f;
    const float x0inv = opt.x0inv, outlier_cut = opt.outlier_cut;
    for (int pass = 0; pass < sc.n_fit_passes && ok; pass++) {
      reset_cov(st, sc.cov0);
      chi2 = 0.0f;
      const bool last = pass == sc.n_fit_passes - 1;
      const int dir = (pass & 1) ? -1 : 1;
      int i = dir > 0 ? 0 : n - 1;
      for (int cnt = 0; cnt < n; cnt++, i += dir) {
        const float4 hit = hit_at(i);
        const float xh = hit.z;
        if (cnt > 0) {  // the first hit of a pass is the one the state already sits at (no transport)
          const float dxk = xh - x_at;
          const float s1 = st.p[2], kap = -(kB * st.p[4]);
          if (!propagate(st, dxk, kB, ms)) {
            ok = false;
            break;
          }
          const float s2 = st.p[2];
          const float c1 = sqrtf(mad(-s1, s1, 1.0f)), c2 = sqrtf(mad(-s2, s2, 1.0f));
          const float t = (s1 + s2) / (c1 + c2);
          const float Lc = dxk * sqrtf(mad(t, t, 1.0f));
          const float arc = Lc * asin_ratio((kap * Lc) * 0.5f);
          add_scattering(st, arc, x0inv);
          add_energy_loss(st, arc, dir, opt.dedx, opt.eloss_sigma);
          x_at = xh;
        }
        const float zraw = hit.y;
        float sy2h, sz2h;
        cluster_errors(st, opt, sy2, sz2, have_d, zraw, zs, sy2h, sz2h);
        const Innov I = innovation(st, sy2h, sz2h);
        const float yh = hit.x, zh = zraw - zref;
        if (last && outlier_cut > 0.0f && chi2_of(I, yh - st.p[0], zh - st.p[1]) > outlier_cut) {
          hit_flag[first + i] = 1;
          nrej++;
          continue;
        }
        chi2 = chi2 + update(st, I, yh, zh);
      }
    }
#pragma unroll
    for (int i = 0; i < 5; i++) par[(int64_t)i * max_tracks + k] = st.p[i];
#pragma unroll
    for (int i = 0; i < 15; i++) cov[(int64_t)i * max_tracks + k] = st.C[i];
    xref[k] = x_at;
    zref_out[k] = zref;
    chi2_out[k] = ok ? chi2 : -1.0f;
    ndf[k] = ok ? 2 * (n - nrej) - 5 : -1;
  }
}

// R28c cluster tags: bit 0 attached, bit 1 track not used for physics (refit failed or |q/pT| > qpt_max), bit 2 hit
// rejected by R28b
__global__ void __launch_bounds__(256)
k_tag_tracks(int64_t n, const int32_t* __restrict__ cluster_track, int64_t max_tracks, const float* __restrict__ par,
             const int32_t* __restrict__ ndf, double qpt_max, uint8_t* __restrict__ tag) {
  for (int64_t c = (int64_t)blockIdx.x * 256 + threadIdx.x; c < n; c += (int64_t)gridDim.x * 256) {
    const int k = cluster_track[c];
    uint8_t t = 0;
    if (k >= 0) {
      t = 1;
      if (__ldg(ndf + k) < 0 || (double)fabsf(__ldg(par + 4 * max_tracks + k)) > qpt_max) t |= 2;
    }
    tag[c] = t;
  }
}

__global__ void __launch_bounds__(256)
k_tag_hits(const int32_t* __restrict__ counters, const int32_t* __restrict__ trk_hits, const uint8_t* __restrict__ hit_flag,
           uint8_t* __restrict__ tag) {
  const int64_t H = counters[TPC_CNT_HITS];
  for (int64_t j = (int64_t)blockIdx.x * 256 + threadIdx.x; j < H; j += (int64_t)gridDim.x * 256)
    if (hit_flag[j]) tag[trk_hits[j]] |= 4;  // a cluster is in one hit list at most: no other thread touches this byte
}

// R21 seeds for the cached refit, one thread per track (full memory parallelism for the four hit gathers and no
// divergence, instead of a few lanes of a warp doing it inside the fit loop).  seed[k] = two float4:
// (y1, sinphi, tanlambda, q/pT), (zRef, x1, first hit's y/z are re-read by the fit loop, -, -).
__global__ void __launch_bounds__(256)
k_fit_seed(const __grid_constant__ Geo g, const float4* __restrict__ hit_rec, const int32_t* __restrict__ counters,
           int64_t max_tracks, int64_t k_cap, const int32_t* __restrict__ trk_nhits, const int64_t* __restrict__ trk_first_hit,
           float4* __restrict__ seed) {
  __shared__ float sX[kMaxRows];
  const Scalars& sc = g.s;
  for (int r = threadIdx.x; r < sc.nrows; r += blockDim.x) sX[r] = g.row.X[r];
  __syncthreads();
  int64_t K = counters[TPC_CNT_TRACKS];
  if (K > max_tracks) K = max_tracks;
  if (K > k_cap) K = k_cap;
  const float kB = sc.kB, ms = sc.max_sinphi;
  for (int64_t k = (int64_t)blockIdx.x * 256 + threadIdx.x; k < K; k += (int64_t)gridDim.x * 256) {
    const int n = trk_nhits[k];
    const float4* hits = hit_rec + trk_first_hit[k];
    // R21: seed from the first, middle and last hit
    const float4 a = __ldg(hits), b = __ldg(hits + n / 2), c = __ldg(hits + (n - 1)), h1 = __ldg(hits + (n > 1 ? 1 : 0));
    const float x1 = sX[__float_as_int(a.z)], y1 = a.x, x2 = sX[__float_as_int(b.z)], y2 = b.x,
                x3 = sX[__float_as_int(c.z)], y3 = c.x;
    const float cross = (x2 - x1) * (y3 - y1) - (x3 - x1) * (y2 - y1);
    const float d12 = sqrtf((x2 - x1) * (x2 - x1) + (y2 - y1) * (y2 - y1));
    const float d23 = sqrtf((x3 - x2) * (x3 - x2) + (y3 - y2) * (y3 - y2));
    const float d13 = sqrtf((x3 - x1) * (x3 - x1) + (y3 - y1) * (y3 - y1));
    const float kappa = (2.0f * cross) / ((d12 * d23) * d13);  // signed curvature of the circumcircle
    const float dx = sX[__float_as_int(h1.z)] - x1, dy = h1.x - y1;
    const float ch = sqrtf(dx * dx + dy * dy);
    float sphi = dy / ch - ((kappa * ch) * 0.5f) * (dx / ch);  // chord direction rotated back by half the turn
    if (sphi > ms) sphi = ms;
    if (sphi < -ms) sphi = -ms;
    const float zref = a.y;
    seed[2 * k] = make_float4(y1, sphi, (h1.y - zref) / ch, -(kappa / kB));
    seed[2 * k + 1] = make_float4(zref, x1, 0.0f, 0.0f);
  }
}

constexpr unsigned kFull = 0xffffffffu;
enum FitPhase { F_FETCH = 0, F_RUN, F_DONE };

__global__ void __launch_bounds__(kFitThreads)
k_fit(const __grid_constant__ Geo g, const float4* __restrict__ hit_rec, const int32_t* __restrict__ counters,
      int64_t max_tracks, int64_t k_cap, const int32_t* __restrict__ trk_nhits, const int64_t* __restrict__ trk_first_hit,
      float* __restrict__ par, float* __restrict__ cov, float* __restrict__ xref, float* __restrict__ zref_out,
      float* __restrict__ chi2_out, int32_t* __restrict__ ndf, const float4* __restrict__ seed,
      int32_t* __restrict__ ws_counters) {
  __shared__ float sX[kMaxRows];
  const Scalars& sc = g.s;
  for (int r = threadIdx.x; r < sc.nrows; r += blockDim.x) sX[r] = g.row.X[r];
  __syncthreads();
  int64_t K64 = counters[TPC_CNT_TRACKS];
  if (K64 > max_tracks) K64 = max_tracks;
  if (K64 > k_cap) K64 = k_cap;
  const int K = (int)K64;
  const int lane = threadIdx.x & 31;
  const float kB = sc.kB, ms = sc.max_sinphi, sy2 = sc.sy2, sz2 = sc.sz2;
  const int npass = sc.n_fit_passes;

  int phase = F_FETCH;
  KState st;
#pragma unroll
  for (int k = 0; k < 5; k++) st.p[k] = 0.0f;
#pragma unroll
  for (int k = 0; k < 15; k++) st.C[k] = 0.0f;
  const float4* hits = hit_rec;
  float4 pre = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
  int k = 0, n = 0, i = 0, cnt = 0, pass = 0, dir = 1;
  float x_at = 0.0f, chi2 = 0.0f, zref = 0.0f;

  for (;;) {
    const unsigned need = __ballot_sync(kFull, phase == F_FETCH);
    if (need) {
      const int leader = __ffs(need) - 1;
      int base = 0;
      if (lane == leader) base = atomicAdd(ws_counters + WC_FIT_QUEUE, __popc(need));
      base = __shfl_sync(kFull, base, leader);
      if (phase == F_FETCH) {
        k = base + __popc(need & ((1u << lane) - 1u));
        if (k >= K) {
          phase = F_DONE;
        } else {
          n = trk_nhits[k];
          hits = hit_rec + trk_first_hit[k];
          // R21 seed, prepared by k_fit_seed
          const float4 s0 = __ldg(seed + 2 * (int64_t)k), s1 = __ldg(seed + 2 * (int64_t)k + 1);
          const float4 a = __ldg(hits);
          zref = s1.x;
          const float x1 = s1.y;
          st.p[0] = s0.x;
          st.p[1] = 0.0f;
          st.p[2] = s0.y;
          st.p[3] = s0.z;
          st.p[4] = s0.w;
          reset_cov(st, sc.cov0);  // R22: covariance reset at the start of every pass
          x_at = x1;
          chi2 = 0.0f;
          pass = 0;
          dir = 1;
          i = 0;
          cnt = 0;
          pre = a;
          phase = F_RUN;
        }
      }
    }
    if (__all_sync(kFull, phase == F_DONE)) break;
    const bool run = phase == F_RUN;
    // this step's hit was loaded one step ahead; issue the next one now
    const float4 h = pre;
    int i_next = i + dir;
    if (cnt + 1 >= n) i_next = ((pass + 1) & 1) ? n - 1 : 0;  // first hit of the next pass
    if (run) pre = __ldg(hits + i_next);
    const float xh = sX[__float_as_int(h.z)];
    bool ok = true;
    __syncwarp();  // one copy of transport + update for all lanes (see tpc_follow.cu)
    if (run && cnt > 0) {  // the first hit of a pass is the one the state already sits at (no transport)
      ok = propagate(st, xh - x_at, kB, ms);
      if (ok) x_at = xh;
    }
    if (run && ok) {
      const Innov I = innovation(st, sy2, sz2);
      chi2 = chi2 + update(st, I, h.x, h.y - zref);
    }
    if (run) {
      bool finish = !ok;
      if (ok) {
        cnt++;
        i = i_next;
        if (cnt >= n) {  // end of a pass: R22 pass 1 inner -> outer, pass 2 outer -> inner, ...
          pass++;
          if (pass >= npass) {
            finish = true;
          } else {
            reset_cov(st, sc.cov0);
            chi2 = 0.0f;
            dir = (pass & 1) ? -1 : 1;
            cnt = 0;
          }
        }
      }
      if (finish) {
#pragma unroll
        for (int q = 0; q < 5; q++) par[(int64_t)q * max_tracks + k] = st.p[q];
#pragma unroll
        for (int q = 0; q < 15; q++) cov[(int64_t)q * max_tracks + k] = st.C[q];
        xref[k] = x_at;
        zref_out[k] = zref;
        chi2_out[k] = ok ? chi2 : -1.0f;
        ndf[k] = ok ? 2 * n - 5 : -1;
        phase = F_FETCH;
      }
    }
  }
}

int g_fit_blocks[kMaxDevices] = {0};  // resident blocks of k_fit per device

}  // namespace

cudaError_t launch_fit(const Geo& g, const Ws* w, int64_t n, const float* y, const float* z, const int32_t* sector_row,
                       const int32_t* counters, int64_t max_tracks, const int32_t* trk_nhits,
                       const int64_t* trk_first_hit, const int32_t* trk_hits, float* par, float* cov, float* xref,
                       float* zref, float* chi2, int32_t* ndf, cudaStream_t st) {
  (void)n;
  if (max_tracks <= 0) return cudaSuccess;
  cudaError_t e;
  int64_t max_tracks_fit = max_tracks;  // tracks the cached path can hold seeds for (see below)
  if (w) {
    int dev = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    int& fit_blocks = g_fit_blocks[dev < kMaxDevices ? dev : kMaxDevices - 1];
    if (fit_blocks == 0 || dev >= kMaxDevices) {
      int sms = 0, per_sm = 0;
      if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
      if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_fit, kFitThreads, 0)) != cudaSuccess) return e;
      fit_blocks = sms * (per_sm > 0 ? per_sm : 1);
    }
    // the hit lists come from the tpc_find_tracks call on this workspace, so K <= its tracklets <= scap_pad; the seed
    // scratch (the follower's parked states, dead by now) holds kStateVec / 2 seeds per tracklet
    const int64_t seed_cap = w->L.scap_pad * (int64_t)(kStateVec / 2);
    if (max_tracks > seed_cap) max_tracks_fit = seed_cap;
    int64_t blocks = (max_tracks_fit + kFitThreads - 1) / kFitThreads;
    if (blocks > fit_blocks) blocks = fit_blocks;
    if ((e = cudaMemsetAsync(w->counters + WC_FIT_QUEUE, 0, sizeof(int32_t), st)) != cudaSuccess) return e;
    // seeds go where the follower parked its states (dead by now; at least 96 bytes per tracklet >= 32 per track)
    float4* seed = w->tl_state;
    int64_t sblocks = (max_tracks_fit + 255) / 256;
    if (sblocks > 148 * 64) sblocks = 148 * 64;
    TPC_LAUNCH(KID_FIT, st,
               (k_fit_seed<<<(unsigned)sblocks, 256, 0, st>>>(g, w->hit_rec, counters, max_tracks, max_tracks_fit, trk_nhits, trk_first_hit, seed)));
    TPC_LAUNCH(KID_FIT, st,
               (k_fit<<<(unsigned)blocks, kFitThreads, 0, st>>>(g, w->hit_rec, counters, max_tracks, max_tracks_fit, trk_nhits, trk_first_hit,
                                                               par, cov, xref, zref, chi2, ndf, seed, w->counters)));
    return cudaGetLastError();
  }
  int64_t blocks = (max_tracks + kFitThreads - 1) / kFitThreads;
  if (blocks > 148 * 16) blocks = 148 * 16;
  TPC_LAUNCH(KID_FIT, st,
             (k_fit_gather<<<(unsigned)blocks, kFitThreads, 0, st>>>(g, y, z, sector_row, counters, max_tracks, trk_nhits,
                                                                    trk_first_hit, trk_hits, par, cov, xref, zref, chi2, ndf)));
  return cudaGetLastError();
}

cudaError_t launch_fit_physics(const Geo& g, const tpc_fit_options_t& opt, const Ws* w, const float* y, const float* z,
                               const int32_t* sector_row, const int32_t* counters, int64_t max_tracks, const int32_t* trk_nhits,
                               const int64_t* trk_first_hit, const int32_t* trk_hits, const float* trk_t0, float* par, float* cov,
                               float* xref, float* zref, float* chi2, int32_t* ndf, uint8_t* hit_flag, cudaStream_t st) {
  if (max_tracks <= 0) return cudaSuccess;
  int64_t blocks = (max_tracks + kFitThreads - 1) / kFitThreads;
  if (blocks > 148 * 16) blocks = 148 * 16;
  if (w) {
    TPC_LAUNCH(KID_FIT_PHYSICS, st,
               (k_fit_physics<true><<<(unsigned)blocks, kFitThreads, 0, st>>>(g, opt, w->hit_rec, y, z, sector_row, counters, max_tracks,
                                                                             trk_nhits, trk_first_hit, trk_hits, trk_t0, par, cov,
                                                                             xref, zref, chi2, ndf, hit_flag)));
  } else {
    TPC_LAUNCH(KID_FIT_PHYSICS, st,
               (k_fit_physics<false><<<(unsigned)blocks, kFitThreads, 0, st>>>(g, opt, nullptr, y, z, sector_row, counters, max_tracks,
                                                                              trk_nhits, trk_first_hit, trk_hits, trk_t0, par, cov,
                                                                              xref, zref, chi2, ndf, hit_flag)));
  }
  return cudaGetLastError();
}

cudaError_t launch_tag_clusters(int64_t n, const int32_t* cluster_track, const int32_t* counters, int64_t max_tracks,
                                const float* par, const int32_t* ndf, const int32_t* trk_hits, const uint8_t* hit_flag,
                                double qpt_max, uint8_t* tag, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  TPC_LAUNCH(KID_FIT_PHYSICS, st,
             (k_tag_tracks<<<blocks_for(n, 256), 256, 0, st>>>(n, cluster_track, max_tracks, par, ndf, qpt_max, tag)));
  if (hit_flag)
    TPC_LAUNCH(KID_FIT_PHYSICS, st, (k_tag_hits<<<blocks_for(n, 256), 256, 0, st>>>(counters, trk_hits, hit_flag, tag)));
  return cudaGetLastError();
}

}  // namespace tpc
