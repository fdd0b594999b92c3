// =============================================================================================
// tpc_oracle.cpp -- plain, slow, single-threaded CPU ORACLE of the TPC tracking hot path.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
// code, header, table or helper with the CUDA path under paper_2106_03636_b200/csrc/.
//
// What it computes (BASELINE.json north_star steps 1-4; PAPER.md is a system overview that
// names TPC tracking as the dominant synchronous workload but does not
// spell the algorithm out, so every rule is a *reading* fixed in SURVEY.md §8(c) R1-R23 and
// restated in DESIGN.md "Readings"):
//   orc_grid        R7      per-(sector,row) (y, zeta) grid: stable sort by bin, bin_first
//   orc_neighbours  R9      cellular-automaton best (up,down) pair per cluster
//   orc_links       R10     reciprocal-link cleaning, start hits
//   orc_follow      R11-R18 Kalman following of the start hits in the order R17 fixes: wave test, two waves of
//                           phase A (init, chain, up leg), phase B (jump, down leg) for the start hits that no
//                           upward leg picked up; the others are absorbed
//   orc_select      R20     one-shot arbitration by 64-bit key, exclusive assignment
//   orc_fit         R21-R22 3-point seed + outward/inward Kalman refit
//   orc_propagate / orc_update   the R12 / R13 primitives, exported for the pins (I7)
//   orc_beamline    R24     closest approach of a fitted helix to the beam line, z there, time offset
//   orc_collisions  R25     collisions as peaks of the per-track time offsets; track -> collision
//   orc_merge_match / orc_merge_fit  R26  links between sector-local tracks (sector edges, central electrode, long
//                           holes) by a 5-parameter chi2, reciprocal arg-mins; refit of the merged hit lists
//   orc_clusterize  R27     clusters from zero-suppressed digits: peaks in (pad, time), 3 x 3 centre of gravity
//   orc_fit_physics / orc_tag_clusters  R28  refit with multiple-scattering process noise, outlier rejection, mean
//                           energy loss, angle- and drift-dependent cluster errors; per-cluster tags for a compression step
//   orc_pair_sides  R29     pairing of the two TPC sides' collisions into (t, z_vertex)
//   orc_set_arith, orc_decisions_begin/end   arithmetic contract switch and the follower's decision log (near-tie report)
//
// Every function exists for real_t = float (suffix _f32: reproduces the GPU's arithmetic: one IEEE
// operation per written operation -- build with -ffp-contract=off -- where mad(a, b, c) is the IEEE
// fusedMultiplyAdd, ONE rounding, in the sums of products of R12 / R13)
// and for real_t = double (suffix _f64: analytic pins I1, I7, I8).  orc_set_arith(0) evaluates every mad
// as a multiplication followed by an addition (two roundings), so that the tests can measure one
// rounding sequence against the other under north_star's tolerances (tests/test_oracle_arith.py).  The step order and notation follow
// R1-R23 so the file can be checked against DESIGN.md by eye; nothing is blocked, fused or
// reordered.  The grid is only an acceleration structure (R8): every search is defined over all
// clusters of a row, and `use_grid = 0` runs exactly that brute force.
//
// Pins (-m "not gpu"): tests/test_oracle_pins.py (I1-I10 of SURVEY.md §8(c)), tests/test_oracle_r17.py (R17: the
// wave test line by line, the wave loop, the three R17 modes measured against one another, configs[0] against the
// stored summary), tests/test_oracle_arith.py (the fused arithmetic term by term, one rounding against the other, the
// near-tie report), tests/test_oracle_beamline.py (R24), tests/test_oracle_collisions.py (R25, R29),
// tests/test_oracle_merge.py (R26), tests/test_oracle_clusterizer.py (R27), tests/test_oracle_physics.py (R28).  Track count,
// efficiency and fake rate themselves are "parity unpinned" by the paper (it publishes no number
// for any synthetic workload); they are fixed only by oracle == GPU.
// =============================================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

namespace {

constexpr int kMaxRows = 152;

// Arithmetic contract: g_fused = 1 (default): mad(a,b,c) = fma(a,b,c), one rounding;
// g_fused = 0: a*b rounded, then + c rounded (the file is compiled with -ffp-contract=off, so the compiler
// never fuses on its own).  fma(-a, b, c) = c - a*b with one rounding (the negation is exact).
int g_fused = 1;
template <class T>
inline T mad(T a, T b, T c) {
  if (g_fused) return std::fma(a, b, c);
  const T ab = a * b;
  return ab + c;
}

// Decision log (tests/parity.py near-tie report): one record per decision the follower takes, in the order it
// takes them.  kind 0: R16 search (chosen = attached cluster or -1; best / second = the two lowest chi2 inside the
// window, +inf if absent; cut = chi2_cut);  kind 1: R15 chain step (chosen = linked cluster if accepted else -1;
// best = its chi2; cut = chi2_chain_cut);  kind 2: a transport refused by |sinphi| > max_sinphi (best = the
// larger |sinphi|, cut = max_sinphi);  kind 3: R16 edge test (best = |y'|, cut = ymax + edge_margin; chosen = 0
// if the leg goes on, -1 if it stops).
struct DecRec {
  int32_t tracklet, row, kind, chosen;
  double best, second, cut;
};
DecRec* g_dec = nullptr;
int64_t g_dec_cap = 0, g_dec_n = 0;
inline void log_decision(int tracklet, int row, int kind, int32_t chosen, double best, double second, double cut) {
  if (!g_dec) return;
  if (g_dec_n < g_dec_cap) g_dec[g_dec_n] = DecRec{tracklet, row, kind, chosen, best, second, cut};
  g_dec_n++;
}

// Host POD filled by oracle/tpc_oracle.py (its own definition; not the CUDA library's header).
struct OrcParams {
  int32_t n_sectors, n_rows;
  double row_x[kMaxRows];
  double tan_half, kB, sigma_y, sigma_z, z_lo, z_hi, cell_y, cell_z;
  double ca_max_dydx, ca_max_dzdx, ca_cut;
  double chi2_cut, chi2_chain_cut, win_max, max_sinphi, edge_margin;
  int32_t max_gap, min_hits, n_fit_passes, reserved;
  double cov0[5];
};

// ---------------------------------------------------------------------------------------------
// Geometry tables (R1, R2, R7), all in real_t T so that float mode rounds exactly like the GPU.
// ---------------------------------------------------------------------------------------------
template <class T>
struct Geo {
  int nsec, nrows, nz;
  T X[kMaxRows], ymax[kMaxRows];
  int ny[kMaxRows];
  int64_t rowbase[kMaxRows + 1];  // first bin of row r inside a sector; rowbase[nrows] = bins per sector
  T inv_cy, inv_cz, z_lo;
  T kB, sy2, sz2;

  explicit Geo(const OrcParams& P) {
    nsec = P.n_sectors;
    nrows = P.n_rows;
    const T tan_half = (T)P.tan_half, cell_y = (T)P.cell_y, cell_z = (T)P.cell_z;
    z_lo = (T)P.z_lo;
    nz = std::max(1, (int)std::ceil(((T)P.z_hi - z_lo) / cell_z));
    inv_cy = (T)1 / cell_y;
    inv_cz = (T)1 / cell_z;
    rowbase[0] = 0;
    for (int r = 0; r < nrows; r++) {
      X[r] = (T)P.row_x[r];
      ymax[r] = X[r] * tan_half;                                         // R1: |y| <= X_r tan 10deg
      ny[r] = std::max(1, (int)std::ceil(((T)2 * ymax[r]) / cell_y));     // R7
      rowbase[r + 1] = rowbase[r] + (int64_t)ny[r] * nz;
    }
    kB = (T)P.kB;
    sy2 = (T)P.sigma_y * (T)P.sigma_y;
    sz2 = (T)P.sigma_z * (T)P.sigma_z;
  }
  // R2/R7: mirrored drift coordinate zeta = side*z, side = +1 for sectors 0..17, -1 for 18..35.
  T side(int sector) const { return sector < 18 ? (T)1 : (T)-1; }
  static int clampbin(T v, int n) {
    if (!(v > (T)0)) return 0;
    if (v >= (T)n) return n - 1;
    return (int)v;
  }
  int ybin(int r, T y) const { return clampbin((y + ymax[r]) * inv_cy, ny[r]); }
  int zbin(int sector, T z) const { return clampbin((side(sector) * z - z_lo) * inv_cz, nz); }
  int64_t bins_per_sector() const { return rowbase[nrows]; }
  int64_t bin_of(int sector, int r, T y, T z) const {
    return (int64_t)sector * bins_per_sector() + rowbase[r] + (int64_t)zbin(sector, z) * ny[r] + ybin(r, y);
  }
};

// ---------------------------------------------------------------------------------------------
// Cluster container + the two search back ends (R8): brute force over the row, or the R7 grid.
// ---------------------------------------------------------------------------------------------
template <class T>
struct Clusters {
  int64_t n;
  const T* y;
  const T* z;
  const int32_t* sector_row;
  int nrows;
  int sector(int64_t i) const { return sector_row[i] / nrows; }
  int row(int64_t i) const { return sector_row[i] % nrows; }
};

template <class T>
struct Index {
  const Geo<T>& G;
  const Clusters<T>& cl;
  bool use_grid;
  std::vector<int32_t> sorted;      // original indices in (sector,row,bin) order, ties by index (R7)
  std::vector<int32_t> bin_first;   // exclusive prefix sum over all bins, +1 sentinel
  std::vector<int64_t> row_first;   // first sorted position of every (sector,row), +1 sentinel

  Index(const Geo<T>& g, const Clusters<T>& c, bool grid) : G(g), cl(c), use_grid(grid) {
    const int64_t nb = (int64_t)G.nsec * G.bins_per_sector();
    std::vector<int64_t> key(cl.n);
    for (int64_t i = 0; i < cl.n; i++) key[i] = G.bin_of(cl.sector(i), cl.row(i), cl.y[i], cl.z[i]);
    sorted.resize(cl.n);
    for (int64_t i = 0; i < cl.n; i++) sorted[i] = (int32_t)i;
    std::stable_sort(sorted.begin(), sorted.end(), [&](int32_t a, int32_t b) { return key[a] < key[b]; });
    bin_first.assign(nb + 1, 0);
    for (int64_t i = 0; i < cl.n; i++) bin_first[key[i] + 1]++;
    for (int64_t b = 0; b < nb; b++) bin_first[b + 1] += bin_first[b];
    row_first.assign((int64_t)G.nsec * G.nrows + 1, 0);
    for (int s = 0; s < G.nsec; s++)
      for (int r = 0; r < G.nrows; r++)
        row_first[(int64_t)s * G.nrows + r] = bin_first[(int64_t)s * G.bins_per_sector() + G.rowbase[r]];
    row_first[(int64_t)G.nsec * G.nrows] = cl.n;
  }

  // Visit every cluster of (sector,row) that could lie in [ya,yb] x [za,zb] (cm).  The visitor
  // re-checks the exact window itself, so the grid only has to return a superset (R8).
  template <class F>
  void visit(int sector, int r, T ya, T yb, T za, T zb, F&& f) const {
    const int64_t sr = (int64_t)sector * G.nrows + r;
    if (!use_grid) {
      for (int64_t k = row_first[sr]; k < row_first[sr + 1]; k++) f(sorted[k]);
      return;
    }
    // widen by a few ulps of the largest |z| so rounding of window edges can never drop a bin
    const T pz = (T)0.01 + ((T)4.8e-7) * std::max(std::fabs(za), std::fabs(zb));
    const T py = (T)0.001;
    const T s = G.side(sector);
    T z0 = s > 0 ? za - pz : -(zb + pz);
    T z1 = s > 0 ? zb + pz : -(za - pz);
    const int zb0 = Geo<T>::clampbin((z0 - G.z_lo) * G.inv_cz, G.nz);
    const int zb1 = Geo<T>::clampbin((z1 - G.z_lo) * G.inv_cz, G.nz);
    const int yb0 = G.ybin(r, ya - py), yb1 = G.ybin(r, yb + py);
    const int64_t base = (int64_t)sector * G.bins_per_sector() + G.rowbase[r];
    for (int zb_ = zb0; zb_ <= zb1; zb_++) {
      const int64_t b0 = base + (int64_t)zb_ * G.ny[r] + yb0, b1 = base + (int64_t)zb_ * G.ny[r] + yb1;
      for (int64_t k = bin_first[b0]; k < bin_first[b1 + 1]; k++) f(sorted[k]);
    }
  }
};

// ---------------------------------------------------------------------------------------------
// R11-R13: state p = (y, dz, sinphi, tanlambda, q/pT) at local x, full symmetric covariance.
// ---------------------------------------------------------------------------------------------
template <class T> struct Thr;
template <> struct Thr<float>  { static constexpr float  asin_u = 0.05f, e_kdx = 1e-3f; };
template <> struct Thr<double> { static constexpr double asin_u = 1e-3,  e_kdx = 1e-5;  };

template <class T>
struct State {
  T p[5];
  T C[5][5];
};

// asin(u)/u: series for small |u| (next term 35 u^8/1152), otherwise the double-precision library
// asin rounded once to T (the GPU does the same, so float mode agrees to the last bit in practice).
template <class T>
T asin_ratio(T u) {
  if (std::fabs(u) < Thr<T>::asin_u) {
    const T u2 = u * u;
    return mad(u2, mad(u2, mad(u2, (T)0.044642857, (T)0.075), (T)0.16666667), (T)1);
  }
  const double ud = (double)u;
  return (T)(std::asin(ud) / ud);
}

// R12: exact helix transport x -> x + dx.  Returns false (state untouched) if |sinphi'| > max_sinphi.
// If F_out != nullptr the 5x5 Jacobian is written there.
template <class T>
bool propagate(State<T>& st, T dx, T kB, T max_sinphi, T (*F_out)[5] = nullptr) {
  const T y = st.p[0], dz = st.p[1], s1 = st.p[2], tl = st.p[3], q = st.p[4];
  const T kappa = -(kB * q);                       // R4: dphi/ds = -kB q/pT
  const T s2 = mad(kappa, dx, s1);
  if (!(std::fabs(s1) <= max_sinphi) || !(std::fabs(s2) <= max_sinphi)) return false;
  const T c1 = std::sqrt(mad(-s1, s1, (T)1)), c2 = std::sqrt(mad(-s2, s2, (T)1));
  const T cc = c1 + c2;
  const T t = (s1 + s2) / cc;                      // tan of the mean direction
  const T L = dx * std::sqrt(mad(t, t, (T)1));     // signed chord
  const T u = (kappa * L) * (T)0.5;
  const T arc = L * asin_ratio(u);                 // signed arc length in the bending plane
  // Jacobian (non-trivial terms), g = 1 + c1 c2 + s1 s2
  const T g = mad(s1, s2, mad(c1, c2, (T)1));
  const T c1c2 = c1 * c2;
  const T f02 = (dx * g) / (cc * c1c2);                       // dy'/dsinphi
  const T f04 = -((kB * (dx * dx)) * g) / (c2 * (cc * cc));   // dy'/dq
  const T f12 = ((tl * dx) * t) / c1c2;                       // ddz'/dsinphi
  const T f13 = arc;                                          // ddz'/dtanl
  const T f24 = -(kB * dx);                                   // dsinphi'/dq
  T E;                                                        // d(arc)/d(kappa)
  if (std::fabs(kappa * dx) < Thr<T>::e_kdx) {
    const T c1_2 = c1 * c1, c1_3 = c1_2 * c1, c1_5 = c1_3 * c1_2;
    E = ((dx * dx) * s1) / ((T)2 * c1_3) + ((kappa * ((dx * dx) * dx)) * ((T)1 + (T)2 * (s1 * s1))) / ((T)3 * c1_5);
  } else {
    E = (dx / c2 - arc) / kappa;
  }
  const T f14 = -((kB * tl) * E);                             // ddz'/dq
  T F[5][5] = {{1, 0, f02, 0, f04}, {0, 1, f12, f13, f14}, {0, 0, 1, 0, f24}, {0, 0, 0, 1, 0}, {0, 0, 0, 0, 1}};
  // state
  st.p[0] = mad(dx, t, y);
  st.p[1] = mad(tl, arc, dz);
  st.p[2] = s2;
  // C' = F C F^T (Q = 0, R6): dense products, sums over k ascending, every term one mad; lower triangle kept, mirrored.
  T M[5][5], N[5][5];
  for (int i = 0; i < 5; i++)
    for (int j = 0; j < 5; j++) {
      T acc = 0;
      for (int k = 0; k < 5; k++) acc = mad(F[i][k], st.C[k][j], acc);
      M[i][j] = acc;
    }
  for (int i = 0; i < 5; i++)
    for (int j = 0; j <= i; j++) {
      T acc = 0;
      for (int k = 0; k < 5; k++) acc = mad(M[i][k], F[j][k], acc);
      N[i][j] = acc;
    }
  for (int i = 0; i < 5; i++)
    for (int j = 0; j <= i; j++) st.C[i][j] = st.C[j][i] = N[i][j];
  if (F_out)
    for (int i = 0; i < 5; i++)
      for (int j = 0; j < 5; j++) F_out[i][j] = F[i][j];
  return true;
}

// R13: innovation covariance S = C[0:2,0:2] + R and its inverse (full 2x2).
template <class T>
struct Innov {
  T S00, S01, S11, Si00, Si01, Si11;
};
template <class T>
Innov<T> innovation(const State<T>& st, T sy2, T sz2) {
  Innov<T> I;
  I.S00 = st.C[0][0] + sy2;
  I.S01 = st.C[1][0];
  I.S11 = st.C[1][1] + sz2;
  const T det = mad(-I.S01, I.S01, I.S00 * I.S11);
  const T idet = (T)1 / det;
  I.Si00 = I.S11 * idet;
  I.Si01 = -(I.S01 * idet);
  I.Si11 = I.S00 * idet;
  return I;
}
template <class T>
T chi2_of(const Innov<T>& I, T r0, T r1) {
  return mad(r1 * r1, I.Si11, mad((T)2 * (r0 * r1), I.Si01, (r0 * r0) * I.Si00));
}
// R13: Kalman update with measurement (ym, zm) (zm already relative to zRef); returns chi2.
template <class T>
T update(State<T>& st, T ym, T zm, T sy2, T sz2) {
  const Innov<T> I = innovation(st, sy2, sz2);
  const T r0 = ym - st.p[0], r1 = zm - st.p[1];
  const T chi2 = chi2_of(I, r0, r1);
  T K[5][2];
  for (int i = 0; i < 5; i++) {
    K[i][0] = mad(st.C[i][1], I.Si01, st.C[i][0] * I.Si00);
    K[i][1] = mad(st.C[i][1], I.Si11, st.C[i][0] * I.Si01);
  }
  T N[5][5];
  for (int i = 0; i < 5; i++)
    for (int j = 0; j <= i; j++) N[i][j] = mad(-K[i][1], st.C[1][j], mad(-K[i][0], st.C[0][j], st.C[i][j]));
  for (int i = 0; i < 5; i++) st.p[i] = mad(K[i][1], r1, mad(K[i][0], r0, st.p[i]));
  for (int i = 0; i < 5; i++)
    for (int j = 0; j <= i; j++) st.C[i][j] = st.C[j][i] = N[i][j];
  return chi2;
}

template <class T>
void reset_cov(State<T>& st, const OrcParams& P) {
  for (int i = 0; i < 5; i++)
    for (int j = 0; j < 5; j++) st.C[i][j] = (i == j) ? (T)P.cov0[i] : (T)0;
}

// ---------------------------------------------------------------------------------------------
// Step 2 -- R9: cellular-automaton neighbour finder.
// ---------------------------------------------------------------------------------------------
template <class T>
void neighbours(const OrcParams& P, const Geo<T>& G, const Clusters<T>& cl, const Index<T>& ix,
                int32_t* link_up, int32_t* link_dn) {
  for (int64_t h = 0; h < cl.n; h++) {
    link_up[h] = link_dn[h] = -1;
    const int r = cl.row(h), s = cl.sector(h);
    if (r < 1 || r > G.nrows - 2) continue;
    const T dxu = G.X[r + 1] - G.X[r], dxd = G.X[r] - G.X[r - 1];
    const T wu = dxd / (dxu + dxd), wd = (T)1 - wu;
    const T den = ((T)1 + wu * wu) + wd * wd;
    const T iy = (T)1 / (G.sy2 * den), iz = (T)1 / (G.sz2 * den);
    const T wyu = (T)P.ca_max_dydx * dxu, wzu = (T)P.ca_max_dzdx * dxu;
    const T wyd = (T)P.ca_max_dydx * dxd, wzd = (T)P.ca_max_dzdx * dxd;
    const T yh = cl.y[h], zh = cl.z[h];
    std::vector<int32_t> U, D;
    ix.visit(s, r + 1, yh - wyu, yh + wyu, zh - wzu, zh + wzu, [&](int32_t u) {
      if (std::fabs(cl.y[u] - yh) <= wyu && std::fabs(cl.z[u] - zh) <= wzu) U.push_back(u);
    });
    ix.visit(s, r - 1, yh - wyd, yh + wyd, zh - wzd, zh + wzd, [&](int32_t d) {
      if (std::fabs(cl.y[d] - yh) <= wyd && std::fabs(cl.z[d] - zh) <= wzd) D.push_back(d);
    });
    std::sort(U.begin(), U.end());
    std::sort(D.begin(), D.end());
    bool have = false;
    T best = 0;
    int32_t bu = -1, bd = -1;
    for (int32_t u : U)
      for (int32_t d : D) {
        const T ry = (yh - cl.y[d]) - wu * (cl.y[u] - cl.y[d]);
        const T rz = (zh - cl.z[d]) - wu * (cl.z[u] - cl.z[d]);
        const T D2 = (ry * ry) * iy + (rz * rz) * iz;
        if (!have || D2 < best) { have = true; best = D2; bu = u; bd = d; }   // ties: lowest u, then lowest d
      }
    if (have && best < (T)P.ca_cut) { link_up[h] = bu; link_dn[h] = bd; }
  }
}

// R10: keep reciprocal links only; start hit = cleaned up-link present and cleaned down-link absent.
void clean_links(int64_t n, const int32_t* link_up, const int32_t* link_dn, int32_t* up_c, int32_t* dn_c,
                 std::vector<int32_t>& starts) {
  for (int64_t h = 0; h < n; h++) {
    up_c[h] = (link_up[h] >= 0 && link_dn[link_up[h]] == (int32_t)h) ? link_up[h] : -1;
    dn_c[h] = (link_dn[h] >= 0 && link_up[link_dn[h]] == (int32_t)h) ? link_dn[h] : -1;
    if (up_c[h] < 0 && dn_c[h] >= 0) up_c[h] = -2;   // R10: top of a chain (linked downward only); read by R17
  }
  starts.clear();
  for (int64_t h = 0; h < n; h++)
    if (up_c[h] >= 0 && dn_c[h] < 0) starts.push_back((int32_t)h);
}

// ---------------------------------------------------------------------------------------------
// Step 3a -- R14-R18: Kalman following of one start hit.
// ---------------------------------------------------------------------------------------------
struct TraceRec {   // one record per hit attached in an R16 search (pin I6)
  int32_t tracklet, row, chosen, pad;
  double y_pred, dz_pred, zref, S00, S01, S11, chi2;
};

template <class T>
struct Follower {
  const OrcParams& P;
  const Geo<T>& G;
  const Clusters<T>& cl;
  const Index<T>& ix;
  TraceRec* trace;
  int64_t trace_cap, trace_n;

  // R16: extrapolate row by row in direction dir (+1/-1) starting after row r_at (state is at X[r_at]).
  // Returns the row the state is at when the leg ends.
  uint8_t* picked_up = nullptr;  // R17: set for every cluster an UPWARD leg attaches (phase A)
  void log_sinphi(const State<T>& st, T dx, int tracklet, int r) const {   // decision log only
    if (!g_dec) return;
    const T s2 = mad(-(G.kB * st.p[4]), dx, st.p[2]);
    log_decision(tracklet, r, 2, -1, std::max(std::fabs((double)st.p[2]), std::fabs((double)s2)), 0.0, P.max_sinphi);
  }
  int extrapolate(State<T>& st, T zref, int sector, int r_at, int r_first, int dir, int32_t* row_hit, int tracklet) {
    int misses = 0;
    for (int r = r_first; r >= 0 && r < G.nrows; r += dir) {
      if (!propagate(st, G.X[r] - G.X[r_at], G.kB, (T)P.max_sinphi)) {         // |sinphi'| > max: stop
        log_sinphi(st, G.X[r] - G.X[r_at], tracklet, r);
        break;
      }
      r_at = r;
      const bool out = std::fabs(st.p[0]) > G.ymax[r] + (T)P.edge_margin;
      log_decision(tracklet, r, 3, out ? -1 : 0, std::fabs(st.p[0]), 0.0, G.ymax[r] + (T)P.edge_margin);
      if (out) break;                                                          // left the sector
      const Innov<T> I = innovation(st, G.sy2, G.sz2);
      const T wy = std::min(std::sqrt((T)P.chi2_cut * I.S00), (T)P.win_max);
      const T wz = std::min(std::sqrt((T)P.chi2_cut * I.S11), (T)P.win_max);
      const T yp = st.p[0], dzp = st.p[1];
      const T zc = zref + dzp;
      bool have = false;
      T best = 0;
      int32_t bi = -1;
      double second = HUGE_VAL;   // decision log only: runner-up chi2
      ix.visit(sector, r, yp - wy, yp + wy, zc - wz, zc + wz, [&](int32_t c) {
        const T r0 = cl.y[c] - yp, r1 = (cl.z[c] - zref) - dzp;
        if (!(std::fabs(r0) <= wy && std::fabs(r1) <= wz)) return;
        const T chi2 = chi2_of(I, r0, r1);
        if (!have || chi2 < best || (chi2 == best && c < bi)) {
          if (have) second = std::min(second, (double)best);
          have = true; best = chi2; bi = c;
        } else {
          second = std::min(second, (double)chi2);
        }
      });
      log_decision(tracklet, r, 0, (have && best < (T)P.chi2_cut) ? bi : -1, have ? (double)best : HUGE_VAL, second,
                   (double)P.chi2_cut);
      if (have && best < (T)P.chi2_cut) {
        if (trace && trace_n < trace_cap) {
          TraceRec& t = trace[trace_n++];
          t.tracklet = tracklet; t.row = r; t.chosen = bi; t.pad = 0;
          t.y_pred = yp; t.dz_pred = dzp; t.zref = zref; t.S00 = I.S00; t.S01 = I.S01; t.S11 = I.S11; t.chi2 = best;
        }
        update(st, cl.y[bi], cl.z[bi] - zref, G.sy2, G.sz2);
        row_hit[r] = bi;
        if (picked_up && dir > 0) picked_up[bi] = 1;
        misses = 0;
      } else {
        misses++;
        if (misses > P.max_gap) break;
      }
    }
    return r_at;
  }

  // R17 wave test: does the backward straight line through the start hit h0 and its up-neighbour meet, within
  // max_gap + 3 rows below, the top of a lower chain (up' = -2)?  (A chain's last cluster and a fragment's first
  // cluster carry no links by R9, so a gap of g missing rows puts the lower chain top g + 3 rows below h0.)
  // Tolerance 4 sigma per row of distance plus one.  Such a start hit waits for the first wave: the tracklet of the lower
  // fragment will most likely pick it up.
  bool has_predecessor(int32_t h0, const int32_t* up_c) const {
    const int sector = cl.sector(h0), r0 = cl.row(h0);
    const int32_t h1 = up_c[h0];
    const T dxu = G.X[cl.row(h1)] - G.X[r0];
    const T my = (cl.y[h1] - cl.y[h0]) / dxu, mz = (cl.z[h1] - cl.z[h0]) / dxu;
    bool found = false;
    for (int k = 1; k <= P.max_gap + 3 && !found; k++) {
      const int r = r0 - k;
      if (r < 0) break;
      const T dxk = G.X[r0] - G.X[r];
      const T yp = cl.y[h0] - my * dxk, zp = cl.z[h0] - mz * dxk;
      const T ty = ((T)4 * (T)P.sigma_y) * (T)(k + 1), tz = ((T)4 * (T)P.sigma_z) * (T)(k + 1);
      ix.visit(sector, r, yp - ty, yp + ty, zp - tz, zp + tz, [&](int32_t c) {
        if (std::fabs(cl.y[c] - yp) <= ty && std::fabs(cl.z[c] - zp) <= tz && up_c[c] == -2) found = true;
      });
    }
    return found;
  }

  // Phase A of following start hit h0 (R14 init, R15 chain, R16 upward leg); row_hit[nrows] receives original
  // indices (-1 = none).  Leaves the state where the upward leg ended (at X[*r_at_out]).
  void follow_up(int32_t h0, const int32_t* up_c, int32_t* row_hit, int tracklet, State<T>* st_out, T* zref_out, int* r_at_out) {
    for (int r = 0; r < G.nrows; r++) row_hit[r] = -1;
    const int sector = cl.sector(h0), r0 = cl.row(h0);
    const int32_t h1 = up_c[h0];
    // R14: initial state from the start hit and its up-neighbour
    const T dx = G.X[cl.row(h1)] - G.X[r0], dy = cl.y[h1] - cl.y[h0];
    const T ch = std::sqrt(dx * dx + dy * dy);
    const T zref = cl.z[h0];
    State<T> st;
    st.p[0] = cl.y[h0];
    st.p[1] = 0;
    st.p[2] = dy / ch;
    st.p[3] = (cl.z[h1] - cl.z[h0]) / ch;
    st.p[4] = 0;
    reset_cov(st, P);
    update(st, cl.y[h0], (T)0, G.sy2, G.sz2);
    row_hit[r0] = h0;
    // R15: chain phase along the cleaned up-links
    int r_at = r0;
    for (int32_t h = h0; up_c[h] >= 0;) {
      const int32_t hn = up_c[h];
      const int rn = cl.row(hn);
      State<T> trial = st;
      if (!propagate(trial, G.X[rn] - G.X[r_at], G.kB, (T)P.max_sinphi)) {
        log_sinphi(st, G.X[rn] - G.X[r_at], tracklet, rn);
        break;
      }
      const Innov<T> I = innovation(trial, G.sy2, G.sz2);
      const T chi2 = chi2_of(I, cl.y[hn] - trial.p[0], (cl.z[hn] - zref) - trial.p[1]);
      log_decision(tracklet, rn, 1, chi2 > (T)P.chi2_chain_cut ? -1 : hn, (double)chi2, HUGE_VAL, (double)P.chi2_chain_cut);
      if (chi2 > (T)P.chi2_chain_cut) break;       // discard the prediction; state stays at the previous hit
      update(trial, cl.y[hn], cl.z[hn] - zref, G.sy2, G.sz2);
      st = trial;
      row_hit[rn] = hn;
      r_at = rn;
      h = hn;
    }
    // R16 upward from the last chain hit
    r_at = extrapolate(st, zref, sector, r_at, r_at + 1, +1, row_hit, tracklet);
    *st_out = st;
    *zref_out = zref;
    *r_at_out = r_at;
  }

  // Phase B (only for tracklets whose start hit no upward leg picked up, R17): one step back to the start row
  // (no update), then R16 downward.  Returns nHits of the whole tracklet.
  int follow_down(int32_t h0, int32_t* row_hit, int tracklet, State<T>* st_io, T zref, int r_at) {
    const int sector = cl.sector(h0), r0 = cl.row(h0);
    State<T> st = *st_io;
    if (propagate(st, G.X[r0] - G.X[r_at], G.kB, (T)P.max_sinphi))
      extrapolate(st, zref, sector, r0, r0 - 1, -1, row_hit, tracklet);
    else
      log_sinphi(st, G.X[r0] - G.X[r_at], tracklet, r0);
    int nh = 0;
    for (int r = 0; r < G.nrows; r++) nh += row_hit[r] >= 0;
    *st_io = st;
    return nh;
  }
};

// ---------------------------------------------------------------------------------------------
// Step 3b -- R21-R22: refit of one hit list (row-ascending original indices).
// out: par[5], cov[15] (lower triangle row-major: 00,10,11,20,21,22,...), xref, zref, chi2, ndf
// ---------------------------------------------------------------------------------------------
template <class T>
bool fit_one(const OrcParams& P, const Geo<T>& G, const Clusters<T>& cl, const int32_t* hits, int n, T* par, T* cov,
             T* xref, T* zref_out, T* chi2_out, int32_t* ndf) {
  const int32_t a = hits[0], b = hits[n / 2], c = hits[n - 1];
  const T x1 = G.X[cl.row(a)], y1 = cl.y[a], x2 = G.X[cl.row(b)], y2 = cl.y[b], x3 = G.X[cl.row(c)], y3 = cl.y[c];
  // R21: signed curvature of the circle through the three points, kappa = 2*cross/(d12 d23 d13)
  const T cross = (x2 - x1) * (y3 - y1) - (x3 - x1) * (y2 - y1);
  const T d12 = std::sqrt((x2 - x1) * (x2 - x1) + (y2 - y1) * (y2 - y1));
  const T d23 = std::sqrt((x3 - x2) * (x3 - x2) + (y3 - y2) * (y3 - y2));
  const T d13 = std::sqrt((x3 - x1) * (x3 - x1) + (y3 - y1) * (y3 - y1));
  const T kappa = ((T)2 * cross) / ((d12 * d23) * d13);
  const int32_t h1 = hits[1];
  const T dx = G.X[cl.row(h1)] - x1, dy = cl.y[h1] - y1;
  const T ch = std::sqrt(dx * dx + dy * dy);
  T sphi = dy / ch - ((kappa * ch) * (T)0.5) * (dx / ch);
  const T ms = (T)P.max_sinphi;
  if (sphi > ms) sphi = ms;
  if (sphi < -ms) sphi = -ms;
  const T zref = cl.z[a];
  State<T> st;
  st.p[0] = y1;
  st.p[1] = 0;
  st.p[2] = sphi;
  st.p[3] = (cl.z[h1] - zref) / ch;
  st.p[4] = -(kappa / G.kB);
  // R22: pass 1 inner -> outer, pass 2 outer -> inner, ...; C reset at the start of every pass
  T chi2 = 0;
  int at = 0;   // index into hits[] of the hit the state sits at
  bool ok = true;
  for (int pass = 0; pass < P.n_fit_passes && ok; pass++) {
    reset_cov(st, P);
    chi2 = 0;
    const int dir = (pass % 2 == 0) ? +1 : -1;
    const int first = (dir > 0) ? 0 : n - 1;
    for (int k = first; k >= 0 && k < n; k += dir) {
      const int32_t h = hits[k];
      if (k != at) {
        if (!propagate(st, G.X[cl.row(h)] - G.X[cl.row(hits[at])], G.kB, (T)P.max_sinphi)) { ok = false; break; }
        at = k;
      }
      chi2 += update(st, cl.y[h], cl.z[h] - zref, G.sy2, G.sz2);
    }
  }
  for (int i = 0; i < 5; i++) par[i] = st.p[i];
  for (int i = 0, m = 0; i < 5; i++)
    for (int j = 0; j <= i; j++) cov[m++] = st.C[i][j];
  *xref = G.X[cl.row(hits[at])];
  *zref_out = zref;
  *chi2_out = ok ? chi2 : (T)-1;
  *ndf = ok ? 2 * n - 5 : -1;
  return ok;
}

// ---------------------------------------------------------------------------------------------
// Whole-stage drivers behind the extern "C" surface.
// ---------------------------------------------------------------------------------------------
template <class T>
struct Ctx {
  OrcParams P;
  Geo<T> G;
  Clusters<T> cl;
  Index<T> ix;
  Ctx(const OrcParams& p, int64_t n, const T* y, const T* z, const int32_t* sr, int use_grid)
      : P(p), G(p), cl{n, y, z, sr, p.n_rows}, ix(G, cl, use_grid != 0) {}
};

template <class T>
int64_t grid_impl(const OrcParams* P, int64_t n, const T* y, const T* z, const int32_t* sr, int32_t* sorted_idx,
                  int32_t* bin_first, int64_t bin_cap) {
  Ctx<T> c(*P, n, y, z, sr, 1);
  const int64_t nb = (int64_t)c.G.nsec * c.G.bins_per_sector();
  if (sorted_idx) std::memcpy(sorted_idx, c.ix.sorted.data(), sizeof(int32_t) * n);
  if (bin_first && bin_cap >= nb + 1) std::memcpy(bin_first, c.ix.bin_first.data(), sizeof(int32_t) * (nb + 1));
  return nb;
}

template <class T>
void neighbours_impl(const OrcParams* P, int64_t n, const T* y, const T* z, const int32_t* sr, int use_grid,
                     int32_t* link_up, int32_t* link_dn) {
  Ctx<T> c(*P, n, y, z, sr, use_grid);
  neighbours(c.P, c.G, c.cl, c.ix, link_up, link_dn);
}

// R17 modes (R17).  The paper fixes none of this (PAPER.md l.47 only says the tracker derives from the
// Run-2 HLT tracker), so the reading is stated three ways and the tests measure one against the other:
//   mode 0  SURVEY.md §8(c) R17 as first written: every start hit is followed in full (R14 init, R15 chain, R16
//           upward leg, one-step jump back, R16 downward leg); nothing is marked, nobody is absorbed
//   mode 1  phases: phase A (R14, R15, R16 upward) for every start hit, every cluster an upward leg attaches is
//           marked; a tracklet whose start hit is marked is absorbed (records nothing, claims nothing); the others
//           run phase B (jump + R16 downward)
//   mode 2  phases + waves (the method the CUDA path implements; the default): phase A runs in two waves -- first
//           the start hits for which wave_test() is false, then those of the rest that no first-wave leg marked
enum { R17_NAIVE = 0, R17_PHASES = 1, R17_WAVES = 2 };

template <class T>
void wave_test_impl(const OrcParams* P, int64_t n, const T* y, const T* z, const int32_t* sr, int use_grid,
                    const int32_t* up_c, int64_t n_starts, const int32_t* starts, uint8_t* waits) {
  Ctx<T> c(*P, n, y, z, sr, use_grid);
  Follower<T> f{c.P, c.G, c.cl, c.ix, nullptr, 0, 0};
  for (int64_t t = 0; t < n_starts; t++) waits[t] = f.has_predecessor(starts[t], up_c) ? 1 : 0;
}

template <class T>
int64_t follow_impl(const OrcParams* P, int64_t n, const T* y, const T* z, const int32_t* sr, int use_grid,
                    const int32_t* up_c, int64_t n_starts, const int32_t* starts, int32_t* row_hit, int32_t* n_hits,
                    T* state_out, TraceRec* trace, int64_t trace_cap, int r17_mode, uint8_t* ran_out) {
  Ctx<T> c(*P, n, y, z, sr, use_grid);
  Follower<T> f{c.P, c.G, c.cl, c.ix, trace, trace_cap, 0};
  std::vector<uint8_t> picked_up((size_t)n, 0);
  std::vector<State<T>> sts((size_t)n_starts);
  std::vector<T> zrefs((size_t)n_starts);
  std::vector<int> r_ats((size_t)n_starts);
  std::vector<uint8_t> waits((size_t)n_starts, 0), ran((size_t)n_starts, 0);
  // (i) wave test (mode 2 only): start hits with a plausible predecessor below them wait for the first wave
  if (r17_mode == R17_WAVES)
    for (int64_t t = 0; t < n_starts; t++) waits[(size_t)t] = f.has_predecessor(starts[t], up_c) ? 1 : 0;
  // marks are only made in modes 1 and 2
  f.picked_up = (r17_mode == R17_NAIVE) ? nullptr : picked_up.data();
  // (ii) first wave: the start hits that do not wait (all of them in modes 0 and 1);
  // (iii) second wave: the waiting start hits that no upward leg of the first wave marked.
  // The list of a wave is fixed BEFORE the wave runs (whole-wave barrier): marks made during a wave do not change it.
  for (int wave = 0; wave < 2; wave++) {
    std::vector<int64_t> todo;
    for (int64_t t = 0; t < n_starts; t++)
      if (wave == 0 ? !waits[(size_t)t] : (waits[(size_t)t] && !picked_up[(size_t)starts[t]])) todo.push_back(t);
    for (int64_t t : todo) {
      f.follow_up(starts[t], up_c, row_hit + t * c.G.nrows, (int)t, &sts[(size_t)t], &zrefs[(size_t)t], &r_ats[(size_t)t]);
      ran[(size_t)t] = 1;
    }
  }
  f.picked_up = nullptr;
  if (std::getenv("ORC_VERBOSE")) {
    int64_t nw = 0, nr = 0;
    for (int64_t t = 0; t < n_starts; t++) { nw += waits[(size_t)t]; nr += ran[(size_t)t]; }
    std::fprintf(stderr, "R17 mode %d: %lld start hits, %lld wait, %lld ran phase A\n", r17_mode, (long long)n_starts, (long long)nw, (long long)nr);
  }
  // (iv) a tracklet whose start hit is marked after both waves -- whether it ran or not -- is absorbed: it records
  // nothing and claims nothing (R18: nHits = 0, empty table); all others run phase B.
  for (int64_t t = 0; t < n_starts; t++) {
    if (!ran[(size_t)t]) sts[(size_t)t] = State<T>();
    if (!ran[(size_t)t] || picked_up[(size_t)starts[t]]) {
      n_hits[t] = 0;
      for (int r = 0; r < c.G.nrows; r++) row_hit[t * c.G.nrows + r] = -1;
    } else {
      n_hits[t] = f.follow_down(starts[t], row_hit + t * c.G.nrows, (int)t, &sts[(size_t)t], zrefs[(size_t)t], r_ats[(size_t)t]);
    }
    if (ran_out) ran_out[t] = ran[(size_t)t];
    if (state_out) {   // 5 params, 15 cov (lower), zref : 21 values per tracklet
      const State<T>& fs = sts[(size_t)t];
      T* o = state_out + t * 21;
      for (int i = 0; i < 5; i++) o[i] = fs.p[i];
      for (int i = 0, m = 5; i < 5; i++)
        for (int j = 0; j <= i; j++) o[m++] = fs.C[i][j];
      o[20] = zrefs[(size_t)t];
    }
  }
  return f.trace_n;
}

// R20: selection.  key(t) = nHits << 32 | (0xFFFFFFFF - start index); owner = max key per cluster.
int64_t select_impl(int64_t n, int n_rows, int64_t n_starts, const int32_t* starts, const int32_t* row_hit,
                    const int32_t* n_hits, int min_hits, int32_t* cluster_track, int32_t* trk_seed, int32_t* trk_nhits,
                    int64_t* trk_first_hit, int32_t* trk_hits) {
  std::vector<uint64_t> owner(n, 0);
  auto key = [&](int64_t t) { return ((uint64_t)(uint32_t)n_hits[t] << 32) | (uint64_t)(0xFFFFFFFFu - (uint32_t)starts[t]); };
  for (int64_t t = 0; t < n_starts; t++)
    for (int r = 0; r < n_rows; r++) {
      const int32_t c = row_hit[t * n_rows + r];
      if (c >= 0) owner[c] = std::max(owner[c], key(t));
    }
  for (int64_t i = 0; i < n; i++) cluster_track[i] = -1;
  int64_t K = 0, nh = 0;
  for (int64_t t = 0; t < n_starts; t++) {
    int kept = 0;
    for (int r = 0; r < n_rows; r++) {
      const int32_t c = row_hit[t * n_rows + r];
      if (c >= 0 && owner[c] == key(t)) kept++;
    }
    if (kept < min_hits) continue;
    trk_seed[K] = starts[t];
    trk_nhits[K] = kept;
    trk_first_hit[K] = nh;
    for (int r = 0; r < n_rows; r++) {
      const int32_t c = row_hit[t * n_rows + r];
      if (c >= 0 && owner[c] == key(t)) { trk_hits[nh++] = c; cluster_track[c] = (int32_t)K; }
    }
    K++;
  }
  return K;
}

template <class T>
void fit_impl(const OrcParams* P, int64_t n, const T* y, const T* z, const int32_t* sr, int64_t K,
              const int32_t* trk_nhits, const int64_t* trk_first_hit, const int32_t* trk_hits, T* par, T* cov, T* xref,
              T* zref, T* chi2, int32_t* ndf) {
  OrcParams Pp = *P;
  Geo<T> G(Pp);
  Clusters<T> cl{n, y, z, sr, Pp.n_rows};
  for (int64_t k = 0; k < K; k++) {
    T p5[5], c15[15];
    fit_one(Pp, G, cl, trk_hits + trk_first_hit[k], trk_nhits[k], p5, c15, xref + k, zref + k, chi2 + k, ndf + k);
    for (int i = 0; i < 5; i++) par[i * K + k] = p5[i];     // SoA [5][K]
    for (int i = 0; i < 15; i++) cov[i * K + k] = c15[i];   // SoA [15][K]
  }
}

template <class T>
int propagate_impl(const OrcParams* P, T* p5, T* c15, T dx, T* F25) {
  State<T> st;
  for (int i = 0; i < 5; i++) st.p[i] = p5[i];
  for (int i = 0, m = 0; i < 5; i++)
    for (int j = 0; j <= i; j++) st.C[i][j] = st.C[j][i] = c15[m++];
  T F[5][5];
  const bool ok = propagate(st, dx, (T)P->kB, (T)P->max_sinphi, F);
  if (!ok) return 0;
  for (int i = 0; i < 5; i++) p5[i] = st.p[i];
  for (int i = 0, m = 0; i < 5; i++)
    for (int j = 0; j <= i; j++) c15[m++] = st.C[i][j];
  if (F25)
    for (int i = 0; i < 5; i++)
      for (int j = 0; j < 5; j++) F25[i * 5 + j] = F[i][j];
  return 1;
}

template <class T>
T update_impl(const OrcParams* P, T* p5, T* c15, T ym, T zm) {
  State<T> st;
  for (int i = 0; i < 5; i++) st.p[i] = p5[i];
  for (int i = 0, m = 0; i < 5; i++)
    for (int j = 0; j <= i; j++) st.C[i][j] = st.C[j][i] = c15[m++];
  const T sy2 = (T)P->sigma_y * (T)P->sigma_y, sz2 = (T)P->sigma_z * (T)P->sigma_z;
  const T chi2 = update(st, ym, zm, sy2, sz2);
  for (int i = 0; i < 5; i++) p5[i] = st.p[i];
  for (int i = 0, m = 0; i < 5; i++)
    for (int j = 0; j <= i; j++) c15[m++] = st.C[i][j];
  return chi2;
}


// ---------------------------------------------------------------------------------------------
// R26 ("full tracking in the TPC", l.60): merging of the sector-local
// tracks of R20-R22 across the 20-degree sector edges, across the central electrode (A side <-> C side) and across
// holes longer than max_gap, then a refit of the merged hit list.  The paper fixes none of it: this is a reading.
//
//   outer state of track A  = its fitted state (R22, at the innermost hit) transported by R12 to the row of its
//                             outermost hit, covariance included (Q = 0: the fit is one helix)
//   relation of (A, B)      : same sector | azimuthal neighbours on one side (B's frame is rotated by D = +-20 deg) |
//                             mirror sectors across the central electrode (same azimuth, other side)
//   B can follow A iff        1 <= first row of B - last row of A <= max_rows, the ends are close in z
//                             (same side: |z_B - z_A| <= dz_max; across the electrode the two sides measure
//                             z_true -+ v_d t, so |z_B + z_A| <= dz_max), tanlambda and q/pT are not hopelessly
//                             apart (d_i^2 <= 4 chi2_cut (C_A,ii + C_B,ii), i = tanlambda, q/pT: a gate that only
//                             removes pairs the chi2 cut would remove, since chi2 >= d_i^2 / S_ii), and
//                             chi2 < chi2_cut, where
//   chi2                    : A's outer state rotated into B's frame (x' = x cosD + y sinD, y' = -x sinD + y cosD,
//                             sinphi' = sinphi cosD - cosphi sinD, cosphi' > 0; covariance C'_ij = J_i C_ij J_j with
//                             J = (cosphi/cosphi', 1, cosphi'/cosphi, 1, 1)), transported by R12 to the x of B's
//                             innermost hit, d = that state - B's fitted state (z through zRef_A - zRef_B),
//                             S = C_A' + C_B, chi2 = d^T S^-1 d by Cholesky, over (y, z, sinphi, tanlambda, q/pT);
//                             across the electrode z is not compared (the time offset is free: 4 parameters) but
//                             |z_A' + z_B| <= ce_tol + 2 |tanlambda_B| dx / cosphi_B must hold (z_true = 0 somewhere
//                             on the dx = x_B - x_A between the two ends)
//   arbitration             : succ[A] = arg-min chi2 over B, pred[B] = arg-min chi2 over A (ties: lowest seed);
//                             A -> B is a link iff succ[A] = B and pred[B] = A (reciprocal, as R10)
//   global tracks           = the chains of links (first rows strictly increase along a chain, so there is no cycle)
// ---------------------------------------------------------------------------------------------
struct OrcMergeParams {
  double chi2_cut, dz_max, ce_tol;
  int32_t max_rows, reserved;
};

enum { REL_NONE = 0, REL_SAME = 1, REL_NEXT = 2, REL_PREV = 3, REL_CE = 4 };  // B's sector relative to A's

inline int sector_relation(int sa, int sb) {
  if (sa == sb) return REL_SAME;
  const int aa = sa % 18, ab = sb % 18;
  if ((sa < 18) != (sb < 18)) return aa == ab ? REL_CE : REL_NONE;
  if (ab == (aa + 1) % 18) return REL_NEXT;   // B's frame = A's rotated by +20 degrees
  if (aa == (ab + 1) % 18) return REL_PREV;   // ... by -20 degrees
  return REL_NONE;
}

// Rotation of a state at x into the frame turned by D (cd = cos D, sd = sin D).  Returns false if the track does not
// point into the +x half of the new frame (cosphi' <= 0) or |sinphi'| > max_sinphi.
// Covariance: the rotated state is a state at the FIXED plane x' = xn of the new frame.  A shift dy along the old plane
// moves the point to (xn + dy sd, yn + dy cd); brought back to x' = xn along the track (slope sn / cn) that is
// dy' = dy (cd - sd sn / cn) = dy c / cn, and a change ds at the same point turns the direction by ds' = ds cn / c: the
// diagonal J below.  The same step back over dx' = -dy sd also changes z by -dy sd tanl / cn and sinphi by -dy sd kappa
// (kappa = -kB q/pT): these two cross terms (dz'/dy, dsinphi'/dy) are DROPPED -- R26 keeps the diagonal form, an
// approximation stated in DESIGN.md R26 and measured by the pin (at 20 degrees: |dz'/dy| = 0.34 |tanl| / cn).
template <class T>
bool rotate_state(State<T>& st, T& x, T cd, T sd, T max_sinphi) {
  const T y = st.p[0], s = st.p[2];
  const T c = std::sqrt((T)1 - s * s);
  const T xn = x * cd + y * sd;
  const T yn = y * cd - x * sd;
  const T sn = s * cd - c * sd;
  const T cn = c * cd + s * sd;
  if (!(cn > (T)0) || !(std::fabs(sn) <= max_sinphi)) return false;
  T J[5] = {c / cn, (T)1, cn / c, (T)1, (T)1};
  for (int i = 0; i < 5; i++)
    for (int j = 0; j <= i; j++) st.C[i][j] = st.C[j][i] = (J[i] * st.C[i][j]) * J[j];
  st.p[0] = yn;
  st.p[2] = sn;
  x = xn;
  return true;
}

// chi2 = d^T S^-1 d over the parameters idx[0..n), S symmetric positive definite, by Cholesky; -1 if S is not.
template <class T>
T chi2_cholesky(const T S[5][5], const T d[5], const int* idx, int n) {
  T L[5][5], yv[5];
  for (int i = 0; i < n; i++)
    for (int j = 0; j <= i; j++) {
      T sum = S[idx[i]][idx[j]];
      for (int k = 0; k < j; k++) sum = sum - L[i][k] * L[j][k];
      if (i == j) {
        if (!(sum > (T)0)) return (T)-1;
        L[i][i] = std::sqrt(sum);
      } else {
        L[i][j] = sum / L[j][j];
      }
    }
  T chi2 = 0;
  for (int i = 0; i < n; i++) {
    T sum = d[idx[i]];
    for (int k = 0; k < i; k++) sum = sum - L[i][k] * yv[k];
    yv[i] = sum / L[i][i];
    chi2 = chi2 + yv[i] * yv[i];
  }
  return chi2;
}

template <class T>
struct TrackView {   // the fitted sector-local tracks, SoA with leading dimension ld
  int64_t K, ld;
  const T *par, *cov, *zref;
  const int32_t *sector, *row_first, *row_last, *seed;
  State<T> state(int64_t k) const {
    State<T> st;
    for (int i = 0; i < 5; i++) st.p[i] = par[i * ld + k];
    for (int i = 0, m = 0; i < 5; i++)
      for (int j = 0; j <= i; j++, m++) st.C[i][j] = st.C[j][i] = cov[m * ld + k];
    return st;
  }
};

constexpr double kCos20 = 0.93969262078590838405, kSin20 = 0.34202014332566873304;

// chi2 of "B follows A" (see the header of this section), -1 if the pair is impossible.  `out` is A's outer state at
// the x of A's outermost hit.
template <class T>
T match_chi2(const OrcParams& P, const OrcMergeParams& M, const Geo<T>& G, const TrackView<T>& tv, int64_t a, int64_t b,
             const State<T>& out, int rel) {
  const int dr = tv.row_first[b] - tv.row_last[a];
  if (dr < 1 || dr > M.max_rows) return (T)-1;
  const T zA = tv.zref[a] + out.p[1], zB = tv.zref[b] + tv.par[1 * tv.ld + b];
  if (rel == REL_CE ? !(std::fabs(zB + zA) <= (T)M.dz_max) : !(std::fabs(zB - zA) <= (T)M.dz_max)) return (T)-1;
  // gate: tanlambda and q/pT are untouched by rotation and transport, and so are their variances; chi2 >= d_i^2 / S_ii
  // for every single parameter (S positive definite), so a pair four times beyond the cut in one of them cannot pass
  for (int i = 3; i < 5; i++) {
    const T di = out.p[i] - tv.par[i * tv.ld + b];
    const T sii = out.C[i][i] + tv.cov[(i * (i + 1) / 2 + i) * tv.ld + b];
    if (!(di * di <= ((T)4 * (T)M.chi2_cut) * sii)) return (T)-1;
  }
  State<T> r = out;
  T x = G.X[tv.row_last[a]];
  if (rel == REL_NEXT || rel == REL_PREV) {
    const T sd = rel == REL_NEXT ? (T)kSin20 : -(T)kSin20;
    if (!rotate_state(r, x, (T)kCos20, sd, (T)P.max_sinphi)) return (T)-1;
  }
  const T xb = G.X[tv.row_first[b]];
  if (!propagate(r, xb - x, G.kB, (T)P.max_sinphi)) return (T)-1;
  const State<T> sb = tv.state(b);
  T d[5], S[5][5];
  d[0] = r.p[0] - sb.p[0];
  d[1] = (tv.zref[a] - tv.zref[b]) + (r.p[1] - sb.p[1]);
  for (int i = 2; i < 5; i++) d[i] = r.p[i] - sb.p[i];
  for (int i = 0; i < 5; i++)
    for (int j = 0; j < 5; j++) S[i][j] = r.C[i][j] + sb.C[i][j];
  if (rel == REL_CE) {
    const T zsum = (tv.zref[a] + r.p[1]) + (tv.zref[b] + sb.p[1]);
    const T cb = std::sqrt((T)1 - sb.p[2] * sb.p[2]);
    const T lim = (T)M.ce_tol + (((T)2 * std::fabs(sb.p[3])) * (xb - G.X[tv.row_last[a]])) / cb;
    if (!(std::fabs(zsum) <= lim)) return (T)-1;
    const int idx[4] = {0, 2, 3, 4};
    return chi2_cholesky(S, d, idx, 4);
  }
  const int idx[5] = {0, 1, 2, 3, 4};
  return chi2_cholesky(S, d, idx, 5);
}

template <class T>
void merge_match_impl(const OrcParams* P, const OrcMergeParams* M, int64_t K, const T* par, const T* cov, const T* zref,
                      const int32_t* sector, const int32_t* row_first, const int32_t* row_last, const int32_t* seed,
                      int32_t* succ, int32_t* pred, T* succ_chi2, T* pair_chi2 /* [K*K] or NULL: every pair, for the pins */) {
  Geo<T> G(*P);
  TrackView<T> tv{K, K, par, cov, zref, sector, row_first, row_last, seed};
  std::vector<T> best_s((size_t)K), best_p((size_t)K);
  for (int64_t k = 0; k < K; k++) succ[k] = pred[k] = -1;
  if (pair_chi2)
    for (int64_t i = 0; i < K * K; i++) pair_chi2[i] = (T)-1;
  std::vector<std::vector<int32_t>> by_sector((size_t)G.nsec);
  for (int64_t k = 0; k < K; k++) by_sector[(size_t)sector[k]].push_back((int32_t)k);
  for (int64_t a = 0; a < K; a++) {
    State<T> out = tv.state(a);
    if (row_last[a] != row_first[a] &&
        !propagate(out, G.X[row_last[a]] - G.X[row_first[a]], G.kB, (T)P->max_sinphi))
      continue;   // no outer state: A has no successor
    for (int sb = 0; sb < G.nsec; sb++) {
      const int rel = sector_relation(sector[a], sb);
      if (rel == REL_NONE) continue;
      for (int32_t b : by_sector[(size_t)sb]) {
        if (b == a) continue;
        const T chi2 = match_chi2(*P, *M, G, tv, a, b, out, rel);
        if (pair_chi2) pair_chi2[a * K + b] = chi2;
        if (!(chi2 >= (T)0) || !(chi2 < (T)M->chi2_cut)) continue;
        if (succ[a] < 0 || chi2 < best_s[(size_t)a] || (chi2 == best_s[(size_t)a] && seed[b] < seed[succ[a]])) {
          succ[a] = b;
          best_s[(size_t)a] = chi2;
        }
        if (pred[b] < 0 || chi2 < best_p[(size_t)b] || (chi2 == best_p[(size_t)b] && seed[a] < seed[pred[b]])) {
          pred[b] = (int32_t)a;
          best_p[(size_t)b] = chi2;
        }
      }
    }
  }
  // reciprocal links only
  for (int64_t a = 0; a < K; a++) {
    succ_chi2[a] = succ[a] >= 0 ? best_s[(size_t)a] : (T)-1;
    if (succ[a] >= 0 && pred[succ[a]] != (int32_t)a) succ[a] = -1;
  }
  for (int64_t b = 0; b < K; b++)
    if (pred[b] >= 0 && succ[pred[b]] != (int32_t)b) pred[b] = -1;
}

// Refit of the global tracks (chains of links).  A chain's hits are taken segment by segment, rows ascending; the
// filter is R22's (pass 1 inner -> outer, pass 2 outer -> inner, covariance reset to cov0 at the start of a pass, all
// hits used) started from the head segment's own fitted state, with two additions at a change of segment:
//   other sector : the state is rotated into the new frame (rotate_state, D = +-20 degrees) -- outward at once (as in
//                  the matching), inward only after a transport, in the old frame, to the plane of the next hit
//   other side   : the time offset is free, so zRef is re-based on the first hit of the new side
//                  (zRef <- z_hit - dz predicted there: that hit's z residual is zero, and ndf loses 1)
// A track without links keeps its sector-local fit.  Output per global track (in ascending order of the head's
// sector-local index): head, segments, hits, state at the innermost hit in the head's frame.
template <class T>
int64_t merge_fit_impl(const OrcParams* P, int64_t n, const T* y, const T* z, const int32_t* sr, int64_t K, const T* par,
                       const T* cov, const T* xref, const T* zref, const T* chi2, const int32_t* ndf, const int32_t* sector,
                       const int32_t* trk_nhits, const int64_t* trk_first_hit, const int32_t* trk_hits, const int32_t* succ,
                       const int32_t* pred, int32_t* trk_global, int32_t* g_head, int32_t* g_nseg, int32_t* g_nhits, T* gpar,
                       T* gcov, T* gxref, T* gzref, T* gchi2, int32_t* gndf) {
  Geo<T> G(*P);
  Clusters<T> cl{n, y, z, sr, P->n_rows};
  int64_t Mg = 0;
  for (int64_t h = 0; h < K; h++)
    if (pred[h] < 0) Mg++;
  int64_t g = 0;
  for (int64_t h = 0; h < K; h++) {
    if (pred[h] >= 0) continue;
    std::vector<int32_t> seg;
    for (int32_t k = (int32_t)h; k >= 0; k = succ[k]) seg.push_back(k);
    int nh = 0;
    for (int32_t k : seg) {
      trk_global[k] = (int32_t)g;
      nh += trk_nhits[k];
    }
    g_head[g] = (int32_t)h;
    g_nseg[g] = (int32_t)seg.size();
    g_nhits[g] = nh;
    if (seg.size() == 1) {
      for (int i = 0; i < 5; i++) gpar[i * Mg + g] = par[i * K + h];
      for (int i = 0; i < 15; i++) gcov[i * Mg + g] = cov[i * K + h];
      gxref[g] = xref[h]; gzref[g] = zref[h]; gchi2[g] = chi2[h]; gndf[g] = ndf[h];
      g++;
      continue;
    }
    // hits of the chain in order, with the sector of each
    std::vector<int32_t> hits, hsec;
    for (int32_t k : seg)
      for (int i = 0; i < trk_nhits[k]; i++) {
        hits.push_back(trk_hits[trk_first_hit[k] + i]);
        hsec.push_back(sector[k]);
      }
    State<T> st;
    for (int i = 0; i < 5; i++) st.p[i] = par[i * K + h];
    T zr = zref[h];
    T x_at = G.X[cl.row(hits[0])];
    int cur_sec = sector[h];
    T c2 = 0;
    int lost = 0;
    bool ok = true;
    const int N = (int)hits.size();
    for (int pass = 0; pass < P->n_fit_passes && ok; pass++) {
      reset_cov(st, *P);
      c2 = 0;
      lost = 0;
      const int dir = (pass % 2 == 0) ? +1 : -1;
      int k = dir > 0 ? 0 : N - 1;
      for (int cnt = 0; cnt < N && ok; cnt++, k += dir) {
        const int32_t hit = hits[k];
        const int hs = hsec[k];
        bool rebase = false;
        if (hs != cur_sec) {
          const int rel = sector_relation(cur_sec, hs);
          if (rel == REL_NEXT || rel == REL_PREV) {
            const T cd = (T)kCos20, sd = rel == REL_NEXT ? (T)kSin20 : -(T)kSin20;
            if (dir < 0) {
              // inward, |sinphi| grows in the frame being entered (a track leaves a sector through the edge it bends
              // towards): stay in the current frame up to the plane of the next hit, x = X_h cosD - y_h sinD there
              const T xc = G.X[cl.row(hit)] * cd - cl.y[hit] * sd;
              if (!propagate(st, xc - x_at, G.kB, (T)P->max_sinphi)) { ok = false; break; }
              x_at = xc;
            }
            if (!rotate_state(st, x_at, cd, sd, (T)P->max_sinphi)) { ok = false; break; }
          } else if (rel == REL_CE) {
            rebase = true;
          }
          cur_sec = hs;
        }
        const T xh = G.X[cl.row(hit)];
        if (cnt > 0) {   // the first hit of a pass is the one the state sits at
          if (!propagate(st, xh - x_at, G.kB, (T)P->max_sinphi)) { ok = false; break; }
          x_at = xh;
        }
        if (rebase) {
          zr = cl.z[hit] - st.p[1];
          lost++;
        }
        c2 += update(st, cl.y[hit], cl.z[hit] - zr, G.sy2, G.sz2);
      }
    }
    for (int i = 0; i < 5; i++) gpar[i * Mg + g] = st.p[i];
    for (int i = 0, m = 0; i < 5; i++)
      for (int j = 0; j <= i; j++) gcov[(m++) * Mg + g] = st.C[i][j];
    gxref[g] = x_at;
    gzref[g] = zr;
    gchi2[g] = ok ? c2 : (T)-1;
    gndf[g] = ok ? 2 * N - 5 - lost : -1;
    g++;
  }
  return Mg;
}

}  // namespace

// =============================================================================================
// C surface (loaded with ctypes by oracle/tpc_oracle.py)
// =============================================================================================
#define ORC_API extern "C" __attribute__((visibility("default")))

ORC_API int64_t orc_sizeof_params() { return (int64_t)sizeof(OrcParams); }
ORC_API int64_t orc_sizeof_decision() { return (int64_t)sizeof(DecRec); }
// arithmetic contract: 1 (default) = mad is a fused multiply-add, 0 = multiplication then addition
ORC_API void orc_set_arith(int fused) { g_fused = fused ? 1 : 0; }
ORC_API int orc_get_arith() { return g_fused; }
// decision log of the follower (see DecRec): records go to buf[cap] until orc_decisions_end(), which returns how
// many decisions were taken (may exceed cap: the rest were dropped)
ORC_API void orc_decisions_begin(DecRec* buf, int64_t cap) { g_dec = buf; g_dec_cap = cap; g_dec_n = 0; }
ORC_API int64_t orc_decisions_end() { g_dec = nullptr; return g_dec_n; }
ORC_API int64_t orc_sizeof_trace() { return (int64_t)sizeof(TraceRec); }

ORC_API int64_t orc_grid_f32(const OrcParams* P, int64_t n, const float* y, const float* z, const int32_t* sr,
                             int32_t* sorted_idx, int32_t* bin_first, int64_t bin_cap) {
  return grid_impl<float>(P, n, y, z, sr, sorted_idx, bin_first, bin_cap);
}
ORC_API int64_t orc_grid_f64(const OrcParams* P, int64_t n, const double* y, const double* z, const int32_t* sr,
                             int32_t* sorted_idx, int32_t* bin_first, int64_t bin_cap) {
  return grid_impl<double>(P, n, y, z, sr, sorted_idx, bin_first, bin_cap);
}
ORC_API void orc_neighbours_f32(const OrcParams* P, int64_t n, const float* y, const float* z, const int32_t* sr,
                                int use_grid, int32_t* link_up, int32_t* link_dn) {
  neighbours_impl<float>(P, n, y, z, sr, use_grid, link_up, link_dn);
}
ORC_API void orc_neighbours_f64(const OrcParams* P, int64_t n, const double* y, const double* z, const int32_t* sr,
                                int use_grid, int32_t* link_up, int32_t* link_dn) {
  neighbours_impl<double>(P, n, y, z, sr, use_grid, link_up, link_dn);
}
// returns the number of start hits written to starts[] (capacity n)
ORC_API int64_t orc_links(int64_t n, const int32_t* link_up, const int32_t* link_dn, int32_t* up_c, int32_t* dn_c,
                          int32_t* starts) {
  std::vector<int32_t> s;
  clean_links(n, link_up, link_dn, up_c, dn_c, s);
  std::memcpy(starts, s.data(), sizeof(int32_t) * s.size());
  return (int64_t)s.size();
}
// r17_mode: 0 naive, 1 phases, 2 phases + waves (see follow_impl); ran_out[n_starts] (may be NULL): 1 if the start
// hit ran phase A
ORC_API int64_t orc_follow_f32(const OrcParams* P, int64_t n, const float* y, const float* z, const int32_t* sr,
                               int use_grid, const int32_t* up_c, int64_t n_starts, const int32_t* starts,
                               int32_t* row_hit, int32_t* n_hits, float* state_out, TraceRec* trace, int64_t trace_cap,
                               int r17_mode, uint8_t* ran_out) {
  return follow_impl<float>(P, n, y, z, sr, use_grid, up_c, n_starts, starts, row_hit, n_hits, state_out, trace, trace_cap,
                            r17_mode, ran_out);
}
ORC_API int64_t orc_follow_f64(const OrcParams* P, int64_t n, const double* y, const double* z, const int32_t* sr,
                               int use_grid, const int32_t* up_c, int64_t n_starts, const int32_t* starts,
                               int32_t* row_hit, int32_t* n_hits, double* state_out, TraceRec* trace, int64_t trace_cap,
                               int r17_mode, uint8_t* ran_out) {
  return follow_impl<double>(P, n, y, z, sr, use_grid, up_c, n_starts, starts, row_hit, n_hits, state_out, trace, trace_cap,
                             r17_mode, ran_out);
}
// R17 (i): waits[t] = 1 if start hit t has a plausible predecessor below it (Follower::has_predecessor)
ORC_API void orc_wave_test_f32(const OrcParams* P, int64_t n, const float* y, const float* z, const int32_t* sr,
                               int use_grid, const int32_t* up_c, int64_t n_starts, const int32_t* starts, uint8_t* waits) {
  wave_test_impl<float>(P, n, y, z, sr, use_grid, up_c, n_starts, starts, waits);
}
ORC_API void orc_wave_test_f64(const OrcParams* P, int64_t n, const double* y, const double* z, const int32_t* sr,
                               int use_grid, const int32_t* up_c, int64_t n_starts, const int32_t* starts, uint8_t* waits) {
  wave_test_impl<double>(P, n, y, z, sr, use_grid, up_c, n_starts, starts, waits);
}
ORC_API int64_t orc_select(int64_t n, int n_rows, int64_t n_starts, const int32_t* starts, const int32_t* row_hit,
                           const int32_t* n_hits, int min_hits, int32_t* cluster_track, int32_t* trk_seed,
                           int32_t* trk_nhits, int64_t* trk_first_hit, int32_t* trk_hits) {
  return select_impl(n, n_rows, n_starts, starts, row_hit, n_hits, min_hits, cluster_track, trk_seed, trk_nhits,
                     trk_first_hit, trk_hits);
}
ORC_API void orc_fit_f32(const OrcParams* P, int64_t n, const float* y, const float* z, const int32_t* sr, int64_t K,
                         const int32_t* trk_nhits, const int64_t* trk_first_hit, const int32_t* trk_hits, float* par,
                         float* cov, float* xref, float* zref, float* chi2, int32_t* ndf) {
  fit_impl<float>(P, n, y, z, sr, K, trk_nhits, trk_first_hit, trk_hits, par, cov, xref, zref, chi2, ndf);
}
ORC_API void orc_fit_f64(const OrcParams* P, int64_t n, const double* y, const double* z, const int32_t* sr, int64_t K,
                         const int32_t* trk_nhits, const int64_t* trk_first_hit, const int32_t* trk_hits, double* par,
                         double* cov, double* xref, double* zref, double* chi2, int32_t* ndf) {
  fit_impl<double>(P, n, y, z, sr, K, trk_nhits, trk_first_hit, trk_hits, par, cov, xref, zref, chi2, ndf);
}
ORC_API int orc_propagate_f32(const OrcParams* P, float* p5, float* c15, float dx, float* F25) {
  return propagate_impl<float>(P, p5, c15, dx, F25);
}
ORC_API int orc_propagate_f64(const OrcParams* P, double* p5, double* c15, double dx, double* F25) {
  return propagate_impl<double>(P, p5, c15, dx, F25);
}
// R26 rotation primitive, exported for its pin (tests/test_oracle_merge.py: every entry of J against finite differences
// of the exact map built from the pinned R12).  p5 / c15 (lower triangle, row-major) / x are updated in place.
template <class T>
int rotate_impl(const OrcParams* P, T* p5, T* c15, T* x, T cd, T sd) {
  State<T> st;
  for (int i = 0; i < 5; i++) st.p[i] = p5[i];
  for (int i = 0, m = 0; i < 5; i++)
    for (int j = 0; j <= i; j++, m++) st.C[i][j] = st.C[j][i] = c15[m];
  T xx = *x;
  if (!rotate_state(st, xx, cd, sd, (T)P->max_sinphi)) return 0;
  for (int i = 0; i < 5; i++) p5[i] = st.p[i];
  for (int i = 0, m = 0; i < 5; i++)
    for (int j = 0; j <= i; j++, m++) c15[m] = st.C[i][j];
  *x = xx;
  return 1;
}
ORC_API int orc_rotate_f32(const OrcParams* P, float* p5, float* c15, float* x, float cd, float sd) {
  return rotate_impl<float>(P, p5, c15, x, cd, sd);
}
ORC_API int orc_rotate_f64(const OrcParams* P, double* p5, double* c15, double* x, double cd, double sd) {
  return rotate_impl<double>(P, p5, c15, x, cd, sd);
}
ORC_API float orc_update_f32(const OrcParams* P, float* p5, float* c15, float ym, float zm) {
  return update_impl<float>(P, p5, c15, ym, zm);
}
ORC_API double orc_update_f64(const OrcParams* P, double* p5, double* c15, double ym, double zm) {
  return update_impl<double>(P, p5, c15, ym, zm);
}

// ---------------------------------------------------------------------------------------------
// R24 ("assignment of tracks to collisions happens only after
// the track reconstruction"): point of closest approach of a fitted helix to the beam line -- the origin of
// every sector-local frame -- the z there, and the time offset it implies.  Plain double arithmetic on the
// fp32 track state; textbook circle geometry:
//   curvature kappa = -kB q/pT, cos(phi) = sqrt(1 - sin^2), circle centre C = (x - sin/kappa, y + cos/kappa),
//   r_C = |C|, R = 1/|kappa|;  dca = |r_C - R|;  closest point P = C (1 - R/r_C);
//   direction at P: phi_P = atan2(-(C_x - P_x) kappa, (C_y - P_y) kappa);
//   turning angle P -> state: dphi = asin(sin phi) - phi_P wrapped to (-pi, pi];  z0 = z - tanl dphi / kappa;
//   straight line (|kappa| < 1e-9 / cm): path t* = -(x cos + y sin), P = (x, y) + t* (cos, sin), z0 = z + tanl t*.
//   global azimuth phi0 = phi_P + alpha_sector (R2) in [0, 2 pi);  time offset t0 = -side z0 / v_drift (R5: a
//   primary from a vertex at z = 0 is measured at z = -side v_d t at the beam line).
// ---------------------------------------------------------------------------------------------
ORC_API void orc_beamline(const OrcParams* P, int64_t K, const float* par, int64_t ldp, const float* xref,
                          const float* zref, const int32_t* sector, double v_drift, float* phi0, float* z0, float* dca,
                          float* t0) {
  const double kPi = 3.14159265358979323846;
  for (int64_t k = 0; k < K; k++) {
    const double x = xref[k], y = par[0 * ldp + k], dz = par[1 * ldp + k], s = par[2 * ldp + k], tl = par[3 * ldp + k],
                 q = par[4 * ldp + k];
    const double c = std::sqrt(1.0 - s * s);
    const double kap = -(P->kB * q);
    const double zabs = (double)zref[k] + dz;
    double phip, zb, d;
    if (std::fabs(kap) < 1e-9) {
      const double ts = -(x * c + y * s);
      const double px = x + ts * c, py = y + ts * s;
      d = std::sqrt(px * px + py * py);
      phip = std::atan2(s, c);
      zb = zabs + tl * ts;
    } else {
      const double xc = x - s / kap, yc = y + c / kap;
      const double rc = std::sqrt(xc * xc + yc * yc);
      const double R = 1.0 / std::fabs(kap);
      const double px = xc * (1.0 - R / rc), py = yc * (1.0 - R / rc);
      d = std::fabs(rc - R);
      phip = std::atan2(-((xc - px) * kap), (yc - py) * kap);
      double dphi = std::asin(s) - phip;
      dphi = dphi - 2.0 * kPi * std::floor((dphi + kPi) / (2.0 * kPi));  // into [-pi, pi)
      zb = zabs - (tl * dphi) / kap;
    }
    const int sec = sector[k];
    const double alpha = ((sec % 18) + 0.5) * (20.0 * kPi / 180.0);
    double ph = phip + alpha;
    ph = ph - 2.0 * kPi * std::floor(ph / (2.0 * kPi));
    const double side = sec < 18 ? 1.0 : -1.0;
    phi0[k] = (float)ph;
    z0[k] = (float)zb;
    dca[k] = (float)d;
    t0[k] = (float)(-(side * zb) / v_drift);
  }
}

// ---------------------------------------------------------------------------------------------
// R25 (second half): collisions from the per-track time offsets of R24.
// Integer work throughout (times are accumulated as round(t0 * 1024) in int64), so the result is unique:
//   1. tracks used: finite t0, dca <= dca_max, t_lo <= t0 < t_lo + nb*w, and on the selected TPC side (side_sel = +1:
//      sectors < 18, -1: sectors >= 18, 0: both -- the two sides see a collision at t -/+ z_vertex / v_d, so they are
//      clustered separately and paired afterwards);  bin b = floor((t0 - t_lo) / w)
//   2. h[b] = tracks in bin b;  s[b] = h[b-2] + ... + h[b+2]  (out-of-range bins count 0)
//   3. bin b is a peak iff s[b] >= n_min, s[b] > s[b-j] and s[b] >= s[b+j] for j = 1..3
//   4. collisions = peaks in ascending b;  time = t_lo + (sum of q over the peak's 5 bins / tracks there) / 1024
//      with q = round((t0 - t_lo) * 1024);  n_tracks = tracks in those 5 bins
//   5. a used track belongs to the peak nearest to its bin (ties: the earlier peak) if within 5 bins, else -1;
//      unused tracks get -1
// Returns the number of collisions; coll_* hold at most coll_cap entries.
// ---------------------------------------------------------------------------------------------
ORC_API int64_t orc_collisions(int64_t K, const float* t0, const float* dca, const int32_t* sector, int32_t side_sel, double t_lo, double w, int64_t nb, double dca_max,
                               int32_t n_min, int64_t coll_cap, float* coll_time, int32_t* coll_ntracks, int32_t* coll_bin,
                               int32_t* trk_collision) {
  std::vector<int32_t> h((size_t)nb, 0), bin((size_t)K, -1);
  std::vector<int64_t> q((size_t)nb, 0);
  for (int64_t k = 0; k < K; k++) {
    const double t = t0[k];
    if (!(t == t) || !((double)dca[k] <= dca_max)) continue;   // NaN or displaced
    if (side_sel != 0 && (side_sel > 0) != (sector[k] < 18)) continue;
    const double u = (t - t_lo) / w;
    if (!(u >= 0.0) || !(u < (double)nb)) continue;
    const int64_t b = (int64_t)std::floor(u);
    bin[(size_t)k] = (int32_t)b;
    h[(size_t)b] += 1;
    q[(size_t)b] += (int64_t)std::llround((t - t_lo) * 1024.0);
  }
  auto H = [&](int64_t b) -> int64_t { return (b >= 0 && b < nb) ? h[(size_t)b] : 0; };
  auto S = [&](int64_t b) -> int64_t { return H(b - 2) + H(b - 1) + H(b) + H(b + 1) + H(b + 2); };
  std::vector<int32_t> peaks;
  for (int64_t b = 0; b < nb; b++) {
    const int64_t s = S(b);
    if (s < n_min) continue;
    bool peak = true;
    for (int j = 1; j <= 3; j++) peak = peak && s > S(b - j) && s >= S(b + j);
    if (peak) peaks.push_back((int32_t)b);
  }
  const int64_t C = (int64_t)peaks.size();
  for (int64_t c = 0; c < C && c < coll_cap; c++) {
    const int64_t b = peaks[(size_t)c];
    int64_t cnt = 0, sum = 0;
    for (int64_t bb = b - 2; bb <= b + 2; bb++)
      if (bb >= 0 && bb < nb) {
        cnt += h[(size_t)bb];
        sum += q[(size_t)bb];
      }
    coll_time[c] = (float)(t_lo + ((double)sum / (double)cnt) / 1024.0);
    coll_ntracks[c] = (int32_t)cnt;
    coll_bin[c] = (int32_t)b;
  }
  for (int64_t k = 0; k < K; k++) {
    int32_t best = -1;
    int64_t bestd = 6;
    if (bin[(size_t)k] >= 0)
      for (int64_t c = 0; c < C; c++) {   // plain scan: the oracle is allowed to be slow
        int64_t d = (int64_t)peaks[(size_t)c] - bin[(size_t)k];
        if (d < 0) d = -d;
        if (d < bestd) {
          bestd = d;
          best = (int32_t)c;
        }
      }
    trk_collision[k] = (best >= 0 && best < coll_cap) ? best : -1;
  }
  return C;
}

// ---------------------------------------------------------------------------------------------
// R26 C surface (see the section above): track matching across sector edges / the central electrode / long holes,
// and the refit of the merged hit lists.  pair_chi2 (may be NULL): [K*K], chi2 of "b follows a" at [a*K + b], -1 = impossible.
// ---------------------------------------------------------------------------------------------
ORC_API int64_t orc_sizeof_merge_params() { return (int64_t)sizeof(OrcMergeParams); }
ORC_API void orc_merge_match_f32(const OrcParams* P, const OrcMergeParams* M, int64_t K, const float* par, const float* cov,
                                 const float* zref, const int32_t* sector, const int32_t* row_first, const int32_t* row_last,
                                 const int32_t* seed, int32_t* succ, int32_t* pred, float* succ_chi2, float* pair_chi2) {
  merge_match_impl<float>(P, M, K, par, cov, zref, sector, row_first, row_last, seed, succ, pred, succ_chi2, pair_chi2);
}
ORC_API void orc_merge_match_f64(const OrcParams* P, const OrcMergeParams* M, int64_t K, const double* par, const double* cov,
                                 const double* zref, const int32_t* sector, const int32_t* row_first, const int32_t* row_last,
                                 const int32_t* seed, int32_t* succ, int32_t* pred, double* succ_chi2, double* pair_chi2) {
  merge_match_impl<double>(P, M, K, par, cov, zref, sector, row_first, row_last, seed, succ, pred, succ_chi2, pair_chi2);
}
ORC_API int64_t orc_merge_fit_f32(const OrcParams* P, int64_t n, const float* y, const float* z, const int32_t* sr, int64_t K,
                                  const float* par, const float* cov, const float* xref, const float* zref, const float* chi2,
                                  const int32_t* ndf, const int32_t* sector, const int32_t* trk_nhits,
                                  const int64_t* trk_first_hit, const int32_t* trk_hits, const int32_t* succ, const int32_t* pred,
                                  int32_t* trk_global, int32_t* g_head, int32_t* g_nseg, int32_t* g_nhits, float* gpar,
                                  float* gcov, float* gxref, float* gzref, float* gchi2, int32_t* gndf) {
  return merge_fit_impl<float>(P, n, y, z, sr, K, par, cov, xref, zref, chi2, ndf, sector, trk_nhits, trk_first_hit, trk_hits,
                               succ, pred, trk_global, g_head, g_nseg, g_nhits, gpar, gcov, gxref, gzref, gchi2, gndf);
}
ORC_API int64_t orc_merge_fit_f64(const OrcParams* P, int64_t n, const double* y, const double* z, const int32_t* sr, int64_t K,
                                  const double* par, const double* cov, const double* xref, const double* zref,
                                  const double* chi2, const int32_t* ndf, const int32_t* sector, const int32_t* trk_nhits,
                                  const int64_t* trk_first_hit, const int32_t* trk_hits, const int32_t* succ, const int32_t* pred,
                                  int32_t* trk_global, int32_t* g_head, int32_t* g_nseg, int32_t* g_nhits, double* gpar,
                                  double* gcov, double* gxref, double* gzref, double* gchi2, int32_t* gndf) {
  return merge_fit_impl<double>(P, n, y, z, sr, K, par, cov, xref, zref, chi2, ndf, sector, trk_nhits, trk_first_hit, trk_hits,
                                succ, pred, trk_global, g_head, g_nseg, g_nhits, gpar, gcov, gxref, gzref, gchi2, gndf);
}

// ---------------------------------------------------------------------------------------------
// R27 (the TPC clusterizer is the step that feeds the tracker).
// Input: zero-suppressed digits (sector_row, pad, time bin, ADC), any order; two digits of the same cell add up.  A
// digit of ADC <= 0 is not a zero-suppressed digit and is ignored (so every cell holds a positive sum and S > 0).
// The paper gives no algorithm; this is the textbook reading:
//   peak    : a digit of ADC a >= peak_min that beats its 8 neighbours in (pad, time) -- strictly the four "earlier"
//             ones (time - 1 at any pad, and pad - 1 at the same time), at least equal to the four "later" ones, so a
//             plateau yields exactly one peak; a missing neighbour counts as 0
//   cluster : centre of gravity of the 3 x 3 cells around a peak (p0, t0), integer sums S = sum a, Sp = sum a dp,
//             St = sum a dt; in fp32, one operation per operator:
//               y    = ((p0 + 0.5) + Sp / S) * pad_width - ymax_row            (pad p covers [p, p + 1) pad widths)
//               zeta = ((t0 + 0.5) + St / S) * time_width + z_lo,  z = side * zeta   (R2)
//               q    = S
// Output: clusters in ascending (sector_row, time, pad) order of their peaks, with the peak cell of each.
// Returns the number of clusters found (at most `cap` are written).
// ---------------------------------------------------------------------------------------------
ORC_API int64_t orc_clusterize(const OrcParams* P, int64_t n, const int32_t* sr, const int32_t* pad, const int32_t* tim,
                               const int32_t* adc, double pad_width, double time_width, int32_t peak_min, int64_t cap,
                               float* y, float* z, float* q, int32_t* out_sr, int32_t* out_pad, int32_t* out_time) {
  Geo<float> G(*P);
  std::vector<std::pair<uint64_t, int64_t>> cells;
  cells.reserve((size_t)n);
  auto key = [](int64_t s, int64_t t, int64_t p) { return ((uint64_t)s << 40) | ((uint64_t)t << 16) | (uint64_t)p; };
  for (int64_t i = 0; i < n; i++)
    if (adc[i] > 0) cells.push_back({key(sr[i], tim[i], pad[i]), (int64_t)adc[i]});
  std::sort(cells.begin(), cells.end());
  size_t m = 0;   // cells of the same key add up
  for (size_t i = 0; i < cells.size(); i++) {
    if (m > 0 && cells[m - 1].first == cells[i].first) cells[m - 1].second += cells[i].second;
    else cells[m++] = cells[i];
  }
  cells.resize(m);
  auto value = [&](int64_t s, int64_t t, int64_t p) -> int64_t {
    if (t < 0 || p < 0 || p > 65535) return 0;
    const uint64_t k = key(s, t, p);
    auto it = std::lower_bound(cells.begin(), cells.end(), std::make_pair(k, (int64_t)INT64_MIN));
    return (it != cells.end() && it->first == k) ? it->second : 0;
  };
  const float pw = (float)pad_width, tw = (float)time_width;
  int64_t found = 0;
  for (const auto& c : cells) {
    const int64_t s = (int64_t)(c.first >> 40), t0 = (int64_t)((c.first >> 16) & 0xFFFFFF), p0 = (int64_t)(c.first & 0xFFFF);
    const int64_t a = c.second;
    if (a < peak_min) continue;
    bool peak = true;
    int64_t S = 0, Sp = 0, St = 0;
    for (int dt = -1; dt <= 1; dt++)
      for (int dp = -1; dp <= 1; dp++) {
        const int64_t b = (dt == 0 && dp == 0) ? a : value(s, t0 + dt, p0 + dp);
        if (dt != 0 || dp != 0) {
          const bool earlier = dt < 0 || (dt == 0 && dp < 0);
          if (earlier ? !(a > b) : !(a >= b)) peak = false;
        }
        S += b;
        Sp += b * dp;
        St += b * dt;
      }
    if (!peak) continue;
    if (found < cap) {
      const int sector = (int)(s / G.nrows), r = (int)(s % G.nrows);
      const float fp = (float)Sp / (float)S, ft = (float)St / (float)S;
      const float yc = (((float)p0 + 0.5f) + fp) * pw - G.ymax[r];
      const float zeta = (((float)t0 + 0.5f) + ft) * tw + G.z_lo;
      y[found] = yc;
      z[found] = G.side(sector) * zeta;
      q[found] = (float)S;
      out_sr[found] = (int32_t)s;
      out_pad[found] = (int32_t)p0;
      out_time[found] = (int32_t)t0;
    }
    found++;
  }
  return found;
}


// ---------------------------------------------------------------------------------------------
// R28 (synchronous tracking exists for the "removal of hits of tracks
// not used for physics", l.47).  The paper gives no formula; the reading is the textbook one:
//   R28a process noise.  After every transport of the refit over a path of L = |arc| sqrt(1 + tanl^2) cm through
//        material of radiation length X0 (x0inv = 1/X0 per cm), multiple scattering with the Highland width without
//        its logarithm, beta = 1:  theta0^2 = (0.0136 GeV)^2 (q/pT)^2 / (1 + tanl^2) * L * x0inv   (p = pT sqrt(1+tanl^2))
//        is added to the covariance of the directions:  C22 += theta0^2 (1 - s^2)(1 + tl^2),  C33 += theta0^2 (1 + tl^2)^2,
//        C43 += theta0^2 tl q (1 + tl^2),  C44 += theta0^2 tl^2 q^2   (s = sinphi, tl = tanl, q = q/pT).
//        x0inv = 0 (the synthetic events have no material) reproduces R22 bit for bit.
//   R28b outlier rejection.  In the LAST pass a hit whose chi2 against the predicted state exceeds outlier_cut is not
//        used: no update, hit_flag = 1, ndf loses 2.  outlier_cut <= 0 switches it off.
//   R28d energy loss.  After every transport (after R28a) the momentum changes by the mean loss dedx (GeV / cm of path,
//        beta = 1) over the path L:  dp/p = -dedx L / p = -dedx |arc| |q|  (p = sqrt(1 + tl^2) / |q|, L = |arc| sqrt(1 + tl^2)),
//        to first order  dq = (dedx |arc| |q|) q;  a track is taken to fly outward, so the outward passes lose momentum,
//        q' = q + dq, and the inward passes gain it back, q' = q - dq.  Straggling: C44 += (eloss_sigma dq)^2.
//        dedx = 0 reproduces R28a bit for bit.
//   R28e cluster errors.  At every hit, from the PREDICTED state (s, tl) and the hit's drift length d:
//        sigma_y^2 = sy2 (1 + err_ang_y s^2 / (1 - s^2)) + err_drift_y d,   sigma_z^2 = sz2 (1 + err_ang_z tl^2) + err_drift_z d
//        d = max(0, z_len - |z + side v_drift t0|) with the track's time offset t0 of R24 (R5: z_true = z + side v_d t);
//        without trk_t0 (NULL, or a NaN entry) the drift terms are left out.  Used by the outlier test and the update alike.
//        All four coefficients 0 reproduce R28a/b bit for bit.
//   R28c cluster tags (what a compression step would drop): per cluster, bit 0 = attached to a track; bit 1 = that
//        track is not used for physics: its refit failed (ndf < 0) or |q/pT| > qpt_max (low-pT loopers);
//        bit 2 = the hit was rejected by R28b.  An unattached cluster has tag 0.
// ---------------------------------------------------------------------------------------------
struct OrcFitOptions {
  double x0inv, outlier_cut;
  double dedx, eloss_sigma;
  double err_ang_y, err_ang_z, err_drift_y, err_drift_z;
  double v_drift, z_len;
};

template <class T>
void add_scattering(State<T>& st, T arc, T x0inv) {
  if (!(x0inv > (T)0)) return;
  const T s = st.p[2], tl = st.p[3], q = st.p[4];
  const T one_tl2 = (T)1 + tl * tl;
  const T L = std::fabs(arc) * std::sqrt(one_tl2);
  const T th2 = ((((T)0.0136 * (T)0.0136) * (q * q)) / one_tl2) * (L * x0inv);
  st.C[2][2] = st.C[2][2] + (th2 * ((T)1 - s * s)) * one_tl2;
  st.C[3][3] = st.C[3][3] + (th2 * one_tl2) * one_tl2;
  const T c43 = ((th2 * tl) * q) * one_tl2;
  st.C[4][3] = st.C[4][3] + c43;
  st.C[3][4] = st.C[4][3];
  st.C[4][4] = st.C[4][4] + ((th2 * tl) * tl) * (q * q);
}

// R28d: mean energy loss over |arc| (dir = +1 outward: momentum is lost; -1 inward: gained back) and its straggling
template <class T>
void add_energy_loss(State<T>& st, T arc, int dir, T dedx, T eloss_sigma) {
  if (!(dedx > (T)0)) return;
  const T q = st.p[4];
  const T rel = (dedx * std::fabs(arc)) * std::fabs(q);
  const T dq = rel * q;
  st.p[4] = dir > 0 ? q + dq : q - dq;
  st.C[4][4] = st.C[4][4] + (eloss_sigma * dq) * (eloss_sigma * dq);
}

// R28e: the two measurement variances at a hit of raw z, for the predicted state st; zs = side v_drift t0
template <class T>
void cluster_errors(const State<T>& st, const OrcFitOptions& O, T sy2, T sz2, bool have_d, T z_raw, T zs, T* sy2h, T* sz2h) {
  T ey = sy2, ez = sz2;
  if (O.err_ang_y > 0) {
    const T s = st.p[2];
    const T tan2 = (s * s) / ((T)1 - s * s);
    ey = ey * ((T)1 + (T)O.err_ang_y * tan2);
  }
  if (O.err_ang_z > 0) {
    const T tl = st.p[3];
    ez = ez * ((T)1 + (T)O.err_ang_z * (tl * tl));
  }
  if (have_d) {
    T d = (T)O.z_len - std::fabs(z_raw + zs);
    if (d < (T)0) d = 0;
    if (O.err_drift_y > 0) ey = ey + (T)O.err_drift_y * d;
    if (O.err_drift_z > 0) ez = ez + (T)O.err_drift_z * d;
  }
  *sy2h = ey;
  *sz2h = ez;
}

// fit_one (R21-R22) with the R28 options; hit_flag[n] receives 1 for hits rejected in the last pass; t0 = the track's
// time offset (R24) or NaN
template <class T>
bool fit_one_physics(const OrcParams& P, const OrcFitOptions& O, const Geo<T>& G, const Clusters<T>& cl, const int32_t* hits,
                     int n, T t0, T* par, T* cov, T* xref, T* zref_out, T* chi2_out, int32_t* ndf, uint8_t* hit_flag) {
  const int32_t a = hits[0], b = hits[n / 2], c = hits[n - 1];
  const T x1 = G.X[cl.row(a)], y1 = cl.y[a], x2 = G.X[cl.row(b)], y2 = cl.y[b], x3 = G.X[cl.row(c)], y3 = cl.y[c];
  const T cross = (x2 - x1) * (y3 - y1) - (x3 - x1) * (y2 - y1);
  const T d12 = std::sqrt((x2 - x1) * (x2 - x1) + (y2 - y1) * (y2 - y1));
  const T d23 = std::sqrt((x3 - x2) * (x3 - x2) + (y3 - y2) * (y3 - y2));
  const T d13 = std::sqrt((x3 - x1) * (x3 - x1) + (y3 - y1) * (y3 - y1));
  const T kappa = ((T)2 * cross) / ((d12 * d23) * d13);
  const int32_t h1 = hits[1];
  const T dx = G.X[cl.row(h1)] - x1, dy = cl.y[h1] - y1;
  const T ch = std::sqrt(dx * dx + dy * dy);
  T sphi = dy / ch - ((kappa * ch) * (T)0.5) * (dx / ch);
  const T ms = (T)P.max_sinphi;
  if (sphi > ms) sphi = ms;
  if (sphi < -ms) sphi = -ms;
  const T zref = cl.z[a];
  State<T> st;
  st.p[0] = y1; st.p[1] = 0; st.p[2] = sphi; st.p[3] = (cl.z[h1] - zref) / ch; st.p[4] = -(kappa / G.kB);
  T chi2 = 0;
  int at = 0, nrej = 0;
  bool ok = true;
  for (int i = 0; i < n; i++) hit_flag[i] = 0;
  const bool have_d = t0 == t0;
  const T side = cl.sector(a) < 18 ? (T)1 : (T)-1;
  const T zs = have_d ? side * ((T)O.v_drift * t0) : (T)0;
  for (int pass = 0; pass < P.n_fit_passes && ok; pass++) {
    reset_cov(st, P);
    chi2 = 0;
    const bool last = pass == P.n_fit_passes - 1;
    const int dir = (pass % 2 == 0) ? +1 : -1;
    const int first = (dir > 0) ? 0 : n - 1;
    for (int k = first; k >= 0 && k < n; k += dir) {
      const int32_t h = hits[k];
      if (k != at) {
        const T dxk = G.X[cl.row(h)] - G.X[cl.row(hits[at])];
        // arc length of this step (the same expression R12 forms), for the scattering width
        const T s1 = st.p[2], kap = -(G.kB * st.p[4]);
        if (!propagate(st, dxk, G.kB, (T)P.max_sinphi)) { ok = false; break; }
        const T s2 = st.p[2];
        const T c1 = std::sqrt(mad(-s1, s1, (T)1)), c2 = std::sqrt(mad(-s2, s2, (T)1));
        const T t = (s1 + s2) / (c1 + c2);
        const T Lc = dxk * std::sqrt(mad(t, t, (T)1));
        const T arc = Lc * asin_ratio((kap * Lc) * (T)0.5);
        add_scattering(st, arc, (T)O.x0inv);
        add_energy_loss(st, arc, dir, (T)O.dedx, (T)O.eloss_sigma);
        at = k;
      }
      T sy2h, sz2h;
      cluster_errors(st, O, G.sy2, G.sz2, have_d, cl.z[h], zs, &sy2h, &sz2h);
      if (last && O.outlier_cut > 0) {
        const Innov<T> I = innovation(st, sy2h, sz2h);
        const T c2h = chi2_of(I, cl.y[h] - st.p[0], (cl.z[h] - zref) - st.p[1]);
        if (c2h > (T)O.outlier_cut) {
          hit_flag[k] = 1;
          nrej++;
          continue;
        }
      }
      chi2 += update(st, cl.y[h], cl.z[h] - zref, sy2h, sz2h);
    }
  }
  for (int i = 0; i < 5; i++) par[i] = st.p[i];
  for (int i = 0, m = 0; i < 5; i++)
    for (int j = 0; j <= i; j++) cov[m++] = st.C[i][j];
  *xref = G.X[cl.row(hits[at])];
  *zref_out = zref;
  *chi2_out = ok ? chi2 : (T)-1;
  *ndf = ok ? 2 * (n - nrej) - 5 : -1;
  return ok;
}

template <class T>
void fit_physics_impl(const OrcParams* P, const OrcFitOptions* O, int64_t n, const T* y, const T* z, const int32_t* sr, int64_t K,
                      const int32_t* trk_nhits, const int64_t* trk_first_hit, const int32_t* trk_hits, const T* trk_t0, T* par,
                      T* cov, T* xref, T* zref, T* chi2, int32_t* ndf, uint8_t* hit_flag) {
  OrcParams Pp = *P;
  Geo<T> G(Pp);
  Clusters<T> cl{n, y, z, sr, Pp.n_rows};
  const T nan = std::nan("");
  for (int64_t k = 0; k < K; k++) {
    T p5[5], c15[15];
    fit_one_physics(Pp, *O, G, cl, trk_hits + trk_first_hit[k], trk_nhits[k], trk_t0 ? trk_t0[k] : nan, p5, c15, xref + k, zref + k, chi2 + k, ndf + k,
                    hit_flag + trk_first_hit[k]);
    for (int i = 0; i < 5; i++) par[i * K + k] = p5[i];
    for (int i = 0; i < 15; i++) cov[i * K + k] = c15[i];
  }
}

ORC_API void orc_fit_physics_f32(const OrcParams* P, const OrcFitOptions* O, int64_t n, const float* y, const float* z,
                                 const int32_t* sr, int64_t K, const int32_t* trk_nhits, const int64_t* trk_first_hit,
                                 const int32_t* trk_hits, const float* trk_t0, float* par, float* cov, float* xref, float* zref,
                                 float* chi2, int32_t* ndf, uint8_t* hit_flag) {
  fit_physics_impl<float>(P, O, n, y, z, sr, K, trk_nhits, trk_first_hit, trk_hits, trk_t0, par, cov, xref, zref, chi2, ndf, hit_flag);
}
ORC_API void orc_fit_physics_f64(const OrcParams* P, const OrcFitOptions* O, int64_t n, const double* y, const double* z,
                                 const int32_t* sr, int64_t K, const int32_t* trk_nhits, const int64_t* trk_first_hit,
                                 const int32_t* trk_hits, const double* trk_t0, double* par, double* cov, double* xref,
                                 double* zref, double* chi2, int32_t* ndf, uint8_t* hit_flag) {
  fit_physics_impl<double>(P, O, n, y, z, sr, K, trk_nhits, trk_first_hit, trk_hits, trk_t0, par, cov, xref, zref, chi2, ndf, hit_flag);
}
// R28c: tag[n] from cluster_track[n], the per-track q/pT (par row 4, leading dimension ldp) and ndf, and hit_flag in
// hit-list order (may be NULL)
ORC_API void orc_tag_clusters(int64_t n, const int32_t* cluster_track, int64_t K, const float* qpt, const int32_t* ndf,
                              const int32_t* trk_nhits, const int64_t* trk_first_hit, const int32_t* trk_hits,
                              const uint8_t* hit_flag, double qpt_max, uint8_t* tag) {
  for (int64_t c = 0; c < n; c++) {
    const int32_t k = cluster_track[c];
    uint8_t t = 0;
    if (k >= 0) {
      t = 1;
      if (ndf[k] < 0 || std::fabs((double)qpt[k]) > qpt_max) t |= 2;
    }
    tag[c] = t;
  }
  if (hit_flag)
    for (int64_t k = 0; k < K; k++)
      for (int i = 0; i < trk_nhits[k]; i++)
        if (hit_flag[trk_first_hit[k] + i]) tag[trk_hits[trk_first_hit[k] + i]] |= 4;
}

// ---------------------------------------------------------------------------------------------
// R29 (last part): pairing of the collisions found on the two TPC sides (R25 with
// side_sel = +1 and -1).  By R5 a collision at time t with vertex z_v is seen at t - z_v/v_d by side A and at
// t + z_v/v_d by side C, with about the same number of tracks on either side.
//   admissible : |t_C - t_A| <= dt_max (= 2 z_max / v_d)
//   cost       : ((t_C - t_A) / sigma_t)^2 + (n_A - n_C)^2 / (n_A + n_C + 1)     (double, in this order)
//   pairs      : best_C[i] = arg-min cost over admissible j, best_A[j] = arg-min over admissible i (ties: the lower
//                index); (i, j) is a pair iff best_C[i] = j and best_A[j] = i -- reciprocal, as R10 and R26
//   result     : t = (t_A + t_C) / 2,  z_v = v_d (t_C - t_A) / 2,  per pair, in ascending i
// pair_of_a[nA], pair_of_c[nC] receive the partner's index or -1.  Returns the number of pairs.
// ---------------------------------------------------------------------------------------------
ORC_API int64_t orc_pair_sides(int64_t nA, const float* tA, const int32_t* cntA, int64_t nC, const float* tC, const int32_t* cntC,
                               double dt_max, double sigma_t, double v_drift, int32_t* pair_of_a, int32_t* pair_of_c,
                               float* t_out, float* zv_out) {
  std::vector<int32_t> bestC((size_t)nA, -1), bestA((size_t)nC, -1);
  std::vector<double> costA((size_t)nA, 0.0), costC((size_t)nC, 0.0);
  for (int64_t i = 0; i < nA; i++)
    for (int64_t j = 0; j < nC; j++) {
      const double dt = (double)tC[j] - (double)tA[i];
      if (!(std::fabs(dt) <= dt_max)) continue;
      const double u = dt / sigma_t, dn = (double)cntA[i] - (double)cntC[j];
      const double cost = u * u + (dn * dn) / ((double)cntA[i] + (double)cntC[j] + 1.0);
      if (bestC[(size_t)i] < 0 || cost < costA[(size_t)i]) { bestC[(size_t)i] = (int32_t)j; costA[(size_t)i] = cost; }
      if (bestA[(size_t)j] < 0 || cost < costC[(size_t)j]) { bestA[(size_t)j] = (int32_t)i; costC[(size_t)j] = cost; }
    }
  for (int64_t j = 0; j < nC; j++) pair_of_c[j] = -1;
  int64_t np = 0;
  for (int64_t i = 0; i < nA; i++) {
    const int32_t j = bestC[(size_t)i];
    if (j >= 0 && bestA[(size_t)j] == (int32_t)i) {
      pair_of_a[i] = j;
      pair_of_c[j] = (int32_t)i;
      t_out[np] = (float)(((double)tA[i] + (double)tC[j]) * 0.5);
      zv_out[np] = (float)((v_drift * ((double)tC[j] - (double)tA[i])) * 0.5);
      np++;
    } else {
      pair_of_a[i] = -1;
    }
  }
  return np;
}
