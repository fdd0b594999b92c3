// =============================================================================================
// tpc_kalman.cuh -- fp32 5-parameter Kalman state in registers: helix transport (R12),
// measurement update (R13).  SURVEY.md §8(c) R11-R13; DESIGN.md "Kernels / follower".
//
//   state p = (y, dz = z - zRef, sinphi, tanlambda, q/pT) at sector-local x, cosphi > 0   (R11)
//   covariance: 15 lower-triangle elements C(i,j), j <= i, index i*(i+1)/2 + j
//
// Every expression is written as one IEEE operation per operator and the library is compiled
// with -fmad=false, so the rounding sequence is fixed by the source text (DESIGN.md "Arithmetic
// contract"): mad(a, b, c) is the fused multiply-add (FFMA, one rounding) and stands exactly where
// the contract names one -- the sums of products of R12 / R13.  The sparse F C F^T below adds the
// non-zero terms of the dense product in ascending-k order, one mad per term, which gives the same
// fp32 result as the dense triple loop (fma(0, x, acc) = acc, fma(1, x, acc) = x + acc).
// =============================================================================================
#pragma once
#include "tpc_common.cuh"

namespace tpc {

#define TPC_CI(i, j) ((i) * ((i) + 1) / 2 + (j))

__device__ __forceinline__ float mad(float a, float b, float c) { return __fmaf_rn(a, b, c); }

struct KState {
  float p[5];
  float C[15];
};

// symmetric read: element (i,j) of the full matrix
__device__ __forceinline__ float csym(const float (&C)[15], int i, int j) {
  return (j <= i) ? C[TPC_CI(i, j)] : C[TPC_CI(j, i)];
}

__device__ __forceinline__ void reset_cov(KState& st, const float (&cov0)[5]) {
#pragma unroll
  for (int k = 0; k < 15; k++) st.C[k] = 0.0f;
  st.C[TPC_CI(0, 0)] = cov0[0];
  st.C[TPC_CI(1, 1)] = cov0[1];
  st.C[TPC_CI(2, 2)] = cov0[2];
  st.C[TPC_CI(3, 3)] = cov0[3];
  st.C[TPC_CI(4, 4)] = cov0[4];
}

// asin(u)/u.  Series below |u| = 0.05 (row-to-row steps always land here); the long R17 jump
// back to the start row can exceed it and takes the double-precision asin rounded once to fp32.
__device__ __forceinline__ float asin_ratio(float u) {
  if (fabsf(u) < 0.05f) {
    const float u2 = u * u;
    return mad(u2, mad(u2, mad(u2, 0.044642857f, 0.075f), 0.16666667f), 1.0f);
  }
  const double ud = (double)u;
  return (float)(asin(ud) / ud);
}

// R12: exact helix transport x -> x + dx, in three pieces so that a caller can start its memory lookups
// as soon as the predicted position and its variances are known and do the rest of F C F^T while they fly:
//   transport_state     new (y, dz, sinphi) and the non-trivial Jacobian terms; false (nothing usable) when
//                       |sinphi| would exceed max_sinphi
//   transport_cov_diag  the (0,0) and (1,1) elements of C' = F C F^T (what the R16 search window needs)
//   transport_apply     commits the state and the full C' (no process noise, R6)
// propagate() = the three in sequence.  The expressions are the same in every piece, so a value computed
// twice is the same value (and the compiler merges them).
struct Transport {
  float y, dz, s2;
  float f02, f04, f12, f13, f14, f24;
};

__device__ __forceinline__ bool transport_state(const KState& st, float dx, float kB, float max_sinphi, Transport& T) {
  const float y = st.p[0], dz = st.p[1], s1 = st.p[2], tl = st.p[3], q = st.p[4];
  const float kappa = -(kB * q);  // R4
  const float s2 = mad(kappa, dx, s1);
  if (!(fabsf(s1) <= max_sinphi) || !(fabsf(s2) <= max_sinphi)) return false;
  const float c1 = sqrtf(mad(-s1, s1, 1.0f)), c2 = sqrtf(mad(-s2, s2, 1.0f));
  const float cc = c1 + c2;
  const float t = (s1 + s2) / cc;             // tangent of the mean direction
  const float L = dx * sqrtf(mad(t, t, 1.0f));  // signed chord
  const float u = (kappa * L) * 0.5f;
  const float arc = L * asin_ratio(u);        // signed arc length in the bending plane
  const float g = mad(s1, s2, mad(c1, c2, 1.0f));
  const float c1c2 = c1 * c2;
  T.f02 = (dx * g) / (cc * c1c2);                    // dy'/dsinphi
  T.f04 = -((kB * (dx * dx)) * g) / (c2 * (cc * cc));  // dy'/dq
  T.f12 = ((tl * dx) * t) / c1c2;                    // ddz'/dsinphi
  T.f13 = arc;                                       // ddz'/dtanl
  T.f24 = -(kB * dx);                                // dsinphi'/dq
  float E;                                           // d(arc)/d(kappa), series near 0
  if (fabsf(kappa * dx) < 1e-3f) {
    const float c1_2 = c1 * c1, c1_3 = c1_2 * c1, c1_5 = c1_3 * c1_2;
    E = ((dx * dx) * s1) / (2.0f * c1_3) +
        ((kappa * ((dx * dx) * dx)) * (1.0f + 2.0f * (s1 * s1))) / (3.0f * c1_5);
  } else {
    E = (dx / c2 - arc) / kappa;
  }
  T.f14 = -((kB * tl) * E);  // ddz'/dq
  T.y = mad(dx, t, y);
  T.dz = mad(tl, arc, dz);
  T.s2 = s2;
  return true;
}

// row 0 and row 1 of M = F C
__device__ __forceinline__ float tr_m0(const KState& st, const Transport& T, int j) {
  return mad(T.f04, csym(st.C, 4, j), mad(T.f02, csym(st.C, 2, j), csym(st.C, 0, j)));
}
__device__ __forceinline__ float tr_m1(const KState& st, const Transport& T, int j) {
  return mad(T.f14, csym(st.C, 4, j), mad(T.f13, csym(st.C, 3, j), mad(T.f12, csym(st.C, 2, j), csym(st.C, 1, j))));
}

__device__ __forceinline__ void transport_cov_diag(const KState& st, const Transport& T, float& C00, float& C11) {
  C00 = mad(tr_m0(st, T, 4), T.f04, mad(tr_m0(st, T, 2), T.f02, tr_m0(st, T, 0)));
  C11 = mad(tr_m1(st, T, 4), T.f14, mad(tr_m1(st, T, 3), T.f13, mad(tr_m1(st, T, 2), T.f12, tr_m1(st, T, 1))));
}
// ... and the (1,0) element: with the two above, everything the innovation covariance S (R13) needs
__device__ __forceinline__ float transport_cov_10(const KState& st, const Transport& T) {
  return mad(tr_m1(st, T, 4), T.f04, mad(tr_m1(st, T, 2), T.f02, tr_m1(st, T, 0)));
}

__device__ __forceinline__ void transport_apply(KState& st, const Transport& T) {
  const float f02 = T.f02, f04 = T.f04, f12 = T.f12, f13 = T.f13, f14 = T.f14, f24 = T.f24;
  // M = F C (rows 0,1,2 differ from C), then N = M F^T, lower triangle.
  float M0[5], M1[5], M2[5];
#pragma unroll
  for (int j = 0; j < 5; j++) {
    M0[j] = tr_m0(st, T, j);
    M1[j] = tr_m1(st, T, j);
    M2[j] = mad(f24, csym(st.C, 4, j), csym(st.C, 2, j));
  }
  // rows 3 and 4 of M are rows 3 and 4 of C
  const float M30 = st.C[TPC_CI(3, 0)], M31 = st.C[TPC_CI(3, 1)], M32 = st.C[TPC_CI(3, 2)], M33 = st.C[TPC_CI(3, 3)],
              M34 = st.C[TPC_CI(4, 3)];
  const float M40 = st.C[TPC_CI(4, 0)], M41 = st.C[TPC_CI(4, 1)], M42 = st.C[TPC_CI(4, 2)], M43 = st.C[TPC_CI(4, 3)],
              M44 = st.C[TPC_CI(4, 4)];
  st.p[0] = T.y;
  st.p[1] = T.dz;
  st.p[2] = T.s2;
  st.C[TPC_CI(0, 0)] = mad(M0[4], f04, mad(M0[2], f02, M0[0]));
  st.C[TPC_CI(1, 0)] = mad(M1[4], f04, mad(M1[2], f02, M1[0]));
  st.C[TPC_CI(1, 1)] = mad(M1[4], f14, mad(M1[3], f13, mad(M1[2], f12, M1[1])));
  st.C[TPC_CI(2, 0)] = mad(M2[4], f04, mad(M2[2], f02, M2[0]));
  st.C[TPC_CI(2, 1)] = mad(M2[4], f14, mad(M2[3], f13, mad(M2[2], f12, M2[1])));
  st.C[TPC_CI(2, 2)] = mad(M2[4], f24, M2[2]);
  st.C[TPC_CI(3, 0)] = mad(M34, f04, mad(M32, f02, M30));
  st.C[TPC_CI(3, 1)] = mad(M34, f14, mad(M33, f13, mad(M32, f12, M31)));
  st.C[TPC_CI(3, 2)] = mad(M34, f24, M32);
  st.C[TPC_CI(3, 3)] = M33;
  st.C[TPC_CI(4, 0)] = mad(M44, f04, mad(M42, f02, M40));
  st.C[TPC_CI(4, 1)] = mad(M44, f14, mad(M43, f13, mad(M42, f12, M41)));
  st.C[TPC_CI(4, 2)] = mad(M44, f24, M42);
  st.C[TPC_CI(4, 3)] = M43;
  st.C[TPC_CI(4, 4)] = M44;
}

// Returns false and leaves the state untouched when |sinphi| would exceed max_sinphi.
__device__ __forceinline__ bool propagate(KState& st, float dx, float kB, float max_sinphi) {
  Transport T;
  if (!transport_state(st, dx, kB, max_sinphi, T)) return false;
  transport_apply(st, T);
  return true;
}

// R13: innovation covariance S = C[0:2,0:2] + diag(sigma_y^2, sigma_z^2) and its inverse.
struct Innov {
  float S00, S01, S11, Si00, Si01, Si11;
};

// from the three covariance elements it depends on (so that it can be formed before C' is committed)
__device__ __forceinline__ Innov innovation3(float C00, float C10, float C11, float sy2, float sz2) {
  Innov I;
  I.S00 = C00 + sy2;
  I.S01 = C10;
  I.S11 = C11 + sz2;
  const float det = mad(-I.S01, I.S01, I.S00 * I.S11);
  const float idet = 1.0f / det;
  I.Si00 = I.S11 * idet;
  I.Si01 = -(I.S01 * idet);
  I.Si11 = I.S00 * idet;
  return I;
}

__device__ __forceinline__ Innov innovation(const KState& st, float sy2, float sz2) {
  return innovation3(st.C[TPC_CI(0, 0)], st.C[TPC_CI(1, 0)], st.C[TPC_CI(1, 1)], sy2, sz2);
}

__device__ __forceinline__ float chi2_of(const Innov& I, float r0, float r1) {
  return mad(r1 * r1, I.Si11, mad(2.0f * (r0 * r1), I.Si01, (r0 * r0) * I.Si00));
}

// R13: Kalman update with measurement (ym, zm) (zm relative to zRef), gain K = C H^T S^-1.
__device__ __forceinline__ float update(KState& st, const Innov& I, float ym, float zm) {
  const float r0 = ym - st.p[0], r1 = zm - st.p[1];
  const float chi2 = chi2_of(I, r0, r1);
  float K0[5], K1[5];
#pragma unroll
  for (int i = 0; i < 5; i++) {
    const float Ci0 = csym(st.C, i, 0), Ci1 = csym(st.C, i, 1);
    K0[i] = mad(Ci1, I.Si01, Ci0 * I.Si00);
    K1[i] = mad(Ci1, I.Si11, Ci0 * I.Si01);
  }
  float N[15];
#pragma unroll
  for (int i = 0; i < 5; i++)
#pragma unroll
    for (int j = 0; j <= i; j++)
      N[TPC_CI(i, j)] = mad(-K1[i], csym(st.C, 1, j), mad(-K0[i], csym(st.C, 0, j), st.C[TPC_CI(i, j)]));
#pragma unroll
  for (int i = 0; i < 5; i++) st.p[i] = mad(K1[i], r1, mad(K0[i], r0, st.p[i]));
#pragma unroll
  for (int k = 0; k < 15; k++) st.C[k] = N[k];
  return chi2;
}

}  // namespace tpc
