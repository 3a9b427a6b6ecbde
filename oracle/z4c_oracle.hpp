// =====================================================================================
// oracle/z4c_oracle.hpp -- TEST INFRASTRUCTURE, NOT PRODUCT.
//
// Plain, slow, block-free CPU statement of the Z4c + RK4 hot path of arXiv 2409.10383
// ("Performance-Portable Numerical Relativity with AthenaK"), written from the paper
// and from the readings O1-O8 / Q1-Q19 recorded in SURVEY.md section 8(c) and
// DESIGN.md.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may call into it.  It shares NO code with the CUDA path
// (paper_2409_10383_b200/csrc) and neither includes the other.
//
// This header holds the per-cell arithmetic as templates over the scalar type so the
// same statements can be run with `double` (the oracle proper) and with an operation
// counting scalar (the flop census that DESIGN.md's roofline uses).
//
// Pins (tests/test_oracle_pins.py): P1 Minkowski, P2 polynomial exactness, P3 Ricci
// identity vs sympy, P4 isotropic Schwarzschild, P5 Kerr-Schild Schwarzschild, P6 linear
// wave convergence, P7 Theta/kappa decay, P8 robust stability, P9 invariances.
// Parity unpinned: the evolved state of puncture data (configs 3-4) has no closed form;
// it is pinned only through P4 at t=0 and bounded constraint norms.
// =====================================================================================
#pragma once
#include <cstdint>

namespace oz4c {

// Field order fixed by BASELINE.json north_star (a) / SURVEY.md section 8(b).
enum Field {
  CHI = 0, GXX = 1, GXY = 2, GXZ = 3, GYY = 4, GYZ = 5, GZZ = 6, KHAT = 7,
  AXX = 8, AXY = 9, AXZ = 10, AYY = 11, AYZ = 12, AZZ = 13,
  GAMX = 14, GAMY = 15, GAMZ = 16, THETA = 17, ALPHA = 18,
  BETAX = 19, BETAY = 20, BETAZ = 21, NF = 22
};

// symmetric-pair -> packed index (xx,xy,xz,yy,yz,zz)
static const int SYM[3][3] = {{0, 1, 2}, {1, 3, 4}, {2, 4, 5}};

struct Params {
  int32_t N[3];         // global interior cells per axis (x,y,z); x fastest in memory
  int32_t bc;           // 0 periodic, 1 outflow-copy (clamp)  -- O2
  double dx;            // same spacing on all axes; cell centres xmin+(i+1/2)dx
  double cfl;           // dt = cfl*dx (CFL 0.25)
  double kappa1, kappa2;                          // PAPER.md:203 (0.02, 0)
  double lapse_oplog, lapse_harmonic, lapse_advect;
  double shift_gamma, shift_eta, shift_advect;
  double ko_eps;        // PAPER.md:203 (0.5)
  double chi_floor;     // Q8
  int32_t ng;           // ghost zones of the GPU layout = stencil half-width: 3 (or 0) -> 4th order (Q1),
                        // 4 -> 6th order, the paper's production scheme ("6th order with 4 ghosts", 279)
};
inline bool sixth_order(const Params& P) { return P.ng == 4; }

// ---------------------------------------------------------------------------------
// O3 stencils, all in difference-from-centre form (Q14).  `l` points at the centre of
// a 7-value line u_{i-3..i+3} along one axis: l[s], s in [-3,3].  h = dx.
// ---------------------------------------------------------------------------------
template <class T>
inline T d1_centred(const T* l, double h) {
  // [8(u+1 - u-1) - (u+2 - u-2)] / (12h)
  return (T(8.0) * (l[1] - l[-1]) - (l[2] - l[-2])) / T(12.0 * h);
}
template <class T>
inline T d2_centred(const T* l, double h) {
  // [16(d+1 + d-1) - (d+2 + d-2)] / (12 h^2),  d_s = u_{i+s}-u_i
  T dp1 = l[1] - l[0], dm1 = l[-1] - l[0], dp2 = l[2] - l[0], dm2 = l[-2] - l[0];
  return (T(16.0) * (dp1 + dm1) - (dp2 + dm2)) / T(12.0 * h * h);
}
template <class T>
inline T d1_upwind(const T* l, double h, bool positive) {
  // beta>=0: [-3 d-1 + 18 d+1 - 6 d+2 + d+3]/(12h);  beta<0: mirrored with sign flip (Q9)
  T dm1 = l[-1] - l[0], dp1 = l[1] - l[0];
  if (positive) {
    T dp2 = l[2] - l[0], dp3 = l[3] - l[0];
    return (T(-3.0) * dm1 + T(18.0) * dp1 - T(6.0) * dp2 + dp3) / T(12.0 * h);
  } else {
    T dm2 = l[-2] - l[0], dm3 = l[-3] - l[0];
    return (T(-1.0) * dm3 + T(6.0) * dm2 - T(18.0) * dm1 + T(3.0) * dp1) / T(12.0 * h);
  }
}
template <class T>
inline T ko_axis(const T* l) {
  // (d+3 + d-3) - 6(d+2 + d-2) + 15(d+1 + d-1); caller multiplies by eps/(64h)  (Q11)
  T s1 = (l[1] - l[0]) + (l[-1] - l[0]);
  T s2 = (l[2] - l[0]) + (l[-2] - l[0]);
  T s3 = (l[3] - l[0]) + (l[-3] - l[0]);
  return s3 - T(6.0) * s2 + T(15.0) * s1;
}
// mixed second derivative: centred-1st along b applied to centred-1st along a.
// `v(sa,sb)` returns u at offsets sa along a, sb along b, for sa,sb in {-2,-1,1,2}.
template <class T, class V>
inline T d2_mixed(V v, double h) {
  T inner[5];
  for (int sb = -2; sb <= 2; ++sb) {
    if (sb == 0) { inner[2] = T(0.0); continue; }
    inner[sb + 2] = T(8.0) * (v(1, sb) - v(-1, sb)) - (v(2, sb) - v(-2, sb));
  }
  return (T(8.0) * (inner[3] - inner[1]) - (inner[4] - inner[0])) / T(144.0 * h * h);
}

// ---------------------------------------------------------------------------------
// NEXT-1: the 6th-order set for 4 ghost zones (PAPER.md:124 footnote: "6th order with 4 ghosts";
// the scheme of every performance run). Coefficients are the unique ones of their
// support and order (pinned by polynomial exactness to degree 6 in tests/test_oracle_pins.py):
//   centred 1st  (-1, 9, -45, 0, 45, -9, 1)/60;  centred 2nd (2, -27, 270, -490, 270, -27, 2)/180;
//   lopsided 1st on offsets -2..+4: (2, -24, -35, 80, -30, 8, -1)/60 (mirror, sign flipped, for beta < 0);
//   Kreiss-Oliger: -eps h^7/256 d^8 (9 points), i.e. (eps/256h)(56 s1 - 28 s2 + 8 s3 - s4), s_k = d_k + d_-k.
// Same difference-from-centre form as above (Q14).
// ---------------------------------------------------------------------------------
template <class T>
inline T d1_centred6(const T* l, double h) {
  return (T(45.0) * (l[1] - l[-1]) - T(9.0) * (l[2] - l[-2]) + (l[3] - l[-3])) / T(60.0 * h);
}
template <class T>
inline T d2_centred6(const T* l, double h) {
  T s1 = (l[1] - l[0]) + (l[-1] - l[0]), s2 = (l[2] - l[0]) + (l[-2] - l[0]), s3 = (l[3] - l[0]) + (l[-3] - l[0]);
  return (T(270.0) * s1 - T(27.0) * s2 + T(2.0) * s3) / T(180.0 * h * h);
}
template <class T>
inline T d1_upwind6(const T* l, double h, bool positive) {
  const int g = positive ? 1 : -1;   // mirror the offsets for beta < 0 and flip the sign
  T dm2 = l[-2 * g] - l[0], dm1 = l[-g] - l[0], dp1 = l[g] - l[0], dp2 = l[2 * g] - l[0], dp3 = l[3 * g] - l[0],
    dp4 = l[4 * g] - l[0];
  T num = T(2.0) * dm2 - T(24.0) * dm1 + T(80.0) * dp1 - T(30.0) * dp2 + T(8.0) * dp3 - dp4;
  return positive ? num / T(60.0 * h) : num / T(-60.0 * h);
}
template <class T>
inline T ko_axis6(const T* l) {
  // 56 s1 - 28 s2 + 8 s3 - s4; caller multiplies by eps/(256h)
  T s1 = (l[1] - l[0]) + (l[-1] - l[0]), s2 = (l[2] - l[0]) + (l[-2] - l[0]);
  T s3 = (l[3] - l[0]) + (l[-3] - l[0]), s4 = (l[4] - l[0]) + (l[-4] - l[0]);
  return T(56.0) * s1 - T(28.0) * s2 + T(8.0) * s3 - s4;
}
template <class T, class V>
inline T d2_mixed6(V v, double h) {
  // centred-1st (6th order) along b of centred-1st along a; v(sa,sb) for sa,sb in {-3..3}\{0}
  T inner[7];
  for (int sb = -3; sb <= 3; ++sb) {
    if (sb == 0) { inner[3] = T(0.0); continue; }
    inner[sb + 3] = T(45.0) * (v(1, sb) - v(-1, sb)) - T(9.0) * (v(2, sb) - v(-2, sb)) + (v(3, sb) - v(-3, sb));
  }
  return (T(45.0) * (inner[4] - inner[2]) - T(9.0) * (inner[5] - inner[1]) + (inner[6] - inner[0])) / T(3600.0 * h * h);
}

// ---------------------------------------------------------------------------------
// 3x3 symmetric helpers
// ---------------------------------------------------------------------------------
template <class T>
inline T det_sym(const T* g) {
  // fixed evaluation order (reading R-E1 in DESIGN.md: the enforcement is bit-specified)
  return g[0] * (g[3] * g[5] - g[4] * g[4]) - g[1] * (g[1] * g[5] - g[4] * g[2]) +
         g[2] * (g[1] * g[4] - g[3] * g[2]);
}
template <class T>
inline void inv_sym(const T* g, T det, T* gi) {
  gi[0] = (g[3] * g[5] - g[4] * g[4]) / det;
  gi[1] = (g[2] * g[4] - g[1] * g[5]) / det;
  gi[2] = (g[1] * g[4] - g[2] * g[3]) / det;
  gi[3] = (g[0] * g[5] - g[2] * g[2]) / det;
  gi[4] = (g[1] * g[2] - g[0] * g[4]) / det;
  gi[5] = (g[0] * g[3] - g[1] * g[1]) / det;
}

// Per-cell derivative bundle handed to the source-term routine (S2 -> S3).
template <class T>
struct Derivs {
  T d1[NF][3];    // centred first derivatives d_k u_f
  T d2[NF][6];    // centred second derivatives d_k d_l u_f (packed sym); only 11 fields used
  T adv[NF];      // sum_k beta^k D^{+-}_k u_f (upwinded)
  T ko[NF];       // (eps/64h) sum_axes ko_axis
};

// Intermediates exposed for pins P3-P5.
template <class T>
struct Geometry {
  T ginv[6];      // conformal inverse metric
  T Gl[3][6];     // Gamma~_{l ij}  (first index lowered), packed (ij)
  T Gu[3][6];     // Gamma~^k_{ij}
  T Gd[3];        // Gamma~_d^k = ginv^{ij} Gamma~^k_{ij}
  T Rt[6];        // R~_ij
  T Rchi[6];      // R^chi_ij
  T Ric[6];       // R_ij = R~ + R^chi
  T Rscal;        // R = chi ginv^{ij} R_ij
  T DDalpha[6];   // D_i D_j alpha
  T Aup[6];       // A~^{ij}
  T AA;           // A~_ij A~^ij
  T K;            // Khat + 2 Theta
};

}  // namespace oz4c
