// =============================================================================================
// tpc_vertex.cu -- first step after the hot path ("assignment of
// tracks to collisions happens only after the track reconstruction"; R24): per fitted
// track, the point of closest approach of its helix to the beam line (the origin of every
// sector-local frame), the z there and the time offset it implies.
//
//   k_track_time  one thread per track; reads the SoA fp32 state written by tpc_fit_tracks
//                 (coalesced), textbook circle geometry in fp64 (1.8e6 tracks per Time Frame:
//                 nothing to optimise, the kernel streams 28 B in and 16 B out per track).
// The track count K is read from counters[TPC_CNT_TRACKS] on the device (no host sync).
// =============================================================================================
#include "tpc_common.cuh"
#include "tpc_prof.cuh"

namespace tpc {

namespace {

constexpr int kThreads = 256;

__global__ void __launch_bounds__(kThreads)
k_track_time(double kB, double v_drift, const int32_t* __restrict__ counters, int64_t max_tracks,
             const int32_t* __restrict__ trk_sector, const float* __restrict__ par, const float* __restrict__ xref,
             const float* __restrict__ zref, float* __restrict__ phi0, float* __restrict__ z0, float* __restrict__ dca,
             float* __restrict__ t0) {
  const double kPi = 3.14159265358979323846;
  int64_t K = counters[TPC_CNT_TRACKS];
  if (K > max_tracks) K = max_tracks;
  for (int64_t k = (int64_t)blockIdx.x * kThreads + threadIdx.x; k < K; k += (int64_t)gridDim.x * kThreads) {
    const double x = xref[k], y = par[0 * max_tracks + k], dz = par[1 * max_tracks + k], s = par[2 * max_tracks + k],
                 tl = par[3 * max_tracks + k], q = par[4 * max_tracks + k];
    const double c = sqrt(1.0 - s * s);
    const double kap = -(kB * q);  // R4
    const double zabs = (double)zref[k] + dz;
    double phip, zb, d;
    if (fabs(kap) < 1e-9) {  // straight line
      const double ts = -(x * c + y * s);
      const double px = x + ts * c, py = y + ts * s;
      d = sqrt(px * px + py * py);
      phip = atan2(s, c);
      zb = zabs + tl * ts;
    } else {
      const double xc = x - s / kap, yc = y + c / kap;  // circle centre
      const double rc = sqrt(xc * xc + yc * yc);
      const double R = 1.0 / fabs(kap);
      const double px = xc * (1.0 - R / rc), py = yc * (1.0 - R / rc);  // closest point of the circle to the origin
      d = fabs(rc - R);
      phip = atan2(-((xc - px) * kap), (yc - py) * kap);  // direction of flight there
      double dphi = asin(s) - phip;                       // turning angle from there to the state
      dphi = dphi - 2.0 * kPi * floor((dphi + kPi) / (2.0 * kPi));
      zb = zabs - (tl * dphi) / kap;
    }
    const int sec = trk_sector[k];
    const double alpha = ((sec % 18) + 0.5) * (20.0 * kPi / 180.0);  // R2
    double ph = phip + alpha;
    ph = ph - 2.0 * kPi * floor(ph / (2.0 * kPi));
    const double side = sec < 18 ? 1.0 : -1.0;
    phi0[k] = (float)ph;
    z0[k] = (float)zb;
    dca[k] = (float)d;
    t0[k] = (float)(-(side * zb) / v_drift);  // R5
  }
}

}  // namespace

cudaError_t launch_track_time(const Geo& g, double v_drift, const int32_t* counters, int64_t max_tracks,
                              const int32_t* trk_sector, const float* par, const float* xref, const float* zref, float* phi0,
                              float* z0, float* dca, float* t0, cudaStream_t st) {
  if (max_tracks <= 0) return cudaSuccess;
  TPC_LAUNCH(KID_TRACK_TIME, st,
             (k_track_time<<<blocks_for(max_tracks, kThreads, 148 * 8), kThreads, 0, st>>>(
                 (double)g.s.kB, v_drift, counters, max_tracks, trk_sector, par, xref, zref, phi0, z0, dca, t0)));
  return cudaGetLastError();
}

}  // namespace tpc
