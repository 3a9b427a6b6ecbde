// Device-side building blocks of the Z4c hot path (sm_100a): finite-difference stencils in
// difference-from-centre form and the 3x3 tensor algebra shared by the RHS kernel (K2) and the
// constraint kernel (K4). Equations: DESIGN.md "The method" (= SURVEY.md section 8(c) O3-O5; the paper
// defers them to Daszuta et al. 2021 at PAPER.md:51, 57).
#pragma once
#include <cstdint>

namespace z4c {

constexpr int NF = 22;
enum : int {
  CHI = 0, GXX = 1, GXY = 2, GXZ = 3, GYY = 4, GYZ = 5, GZZ = 6, KHAT = 7,
  AXX = 8, AXY = 9, AXZ = 10, AYY = 11, AYZ = 12, AZZ = 13,
  GAMX = 14, GAMY = 15, GAMZ = 16, THETA = 17, ALPHA = 18, BETAX = 19, BETAY = 20, BETAZ = 21
};
// Ghost zones per side = stencil half-width, fixed at compile time: 3 -> 4th-order stencils (BASELINE configs),
// 4 -> 6th-order stencils, the paper's production scheme (NEXT-1). The library is built once
// per value (libz4c.so, libz4c_ng4.so).
#ifndef Z4C_NG
#define Z4C_NG 3
#endif
constexpr int NG = Z4C_NG;
static_assert(NG == 3 || NG == 4, "supported ghost counts");

// packed index of a symmetric pair: xx,xy,xz,yy,yz,zz
__host__ __device__ constexpr int sym(int i, int j) {
  return i <= j ? (i * 3 - (i * (i - 1)) / 2 + (j - i)) : (j * 3 - (j * (j - 1)) / 2 + (i - j));
}

// Per-launch constants of the finite-difference operators.
// (NG = 3 values; NG = 4 in brackets)
struct FdConst {
  double inv12h;     // 1/(12 h)      [1/(60 h)]    centred 1st; half of it weights the upwinded term
  double inv12h2;    // 1/(12 h^2)    [1/(180 h^2)] centred 2nd
  double inv144h2;   // 1/(144 h^2)   [1/(3600 h^2)] mixed 2nd
  double ko;         // eps/(64 h)    [eps/(256 h)] Kreiss-Oliger
};

// One axis of one field: 6 neighbour loads feed the centred 1st/2nd derivative, the upwinded
// derivative and the Kreiss-Oliger sum (O3). `p` points at the cell, `s` is the element stride of the
// axis. Returns raw (unscaled) stencil sums.
struct AxisRaw { double d1, d2, up, ko; };

template <bool WANT_D1, bool WANT_D2>
__device__ __forceinline__ AxisRaw axis_raw(const double* __restrict__ p, const int s, const double c,
                                            const bool pos) {
  AxisRaw r;
#if Z4C_NG == 3
  const double lm3 = __ldg(p - 3 * s), lm2 = __ldg(p - 2 * s), lm1 = __ldg(p - s);
  const double lp1 = __ldg(p + s), lp2 = __ldg(p + 2 * s), lp3 = __ldg(p + 3 * s);
  const double dm1 = lm1 - c, dp1 = lp1 - c, dm2 = lm2 - c, dp2 = lp2 - c, dm3 = lm3 - c, dp3 = lp3 - c;
  const double s1 = dp1 + dm1, s2 = dp2 + dm2, s3 = dp3 + dm3;
  r.d1 = WANT_D1 ? (8.0 * (lp1 - lm1) - (lp2 - lm2)) : 0.0;
  r.d2 = WANT_D2 ? (16.0 * s1 - s2) : 0.0;
  r.ko = s3 - 6.0 * s2 + 15.0 * s1;
  // upwind: beta >= 0 uses (-1,+1,+2,+3); beta < 0 is the mirror image with the sign flipped, so
  // beta * D^- u = |beta| * D^+ (mirrored u)
  const double a1 = pos ? dp1 : dm1, b1 = pos ? dm1 : dp1;
  const double a2 = pos ? dp2 : dm2, a3 = pos ? dp3 : dm3;
  r.up = -3.0 * b1 + 18.0 * a1 - 6.0 * a2 + a3;
#else
  // 6th order: centred (45 e1 - 9 e2 + e3)/60h, (270 s1 - 27 s2 + 2 s3)/180h^2; KO (56 s1 - 28 s2 + 8 s3 - s4);
  // lopsided numerator on the upwind side, offsets -2..+4: 2 d-2 - 24 d-1 + 80 d+1 - 30 d+2 + 8 d+3 - d+4
  const double lm4 = __ldg(p - 4 * s), lm3 = __ldg(p - 3 * s), lm2 = __ldg(p - 2 * s), lm1 = __ldg(p - s);
  const double lp1 = __ldg(p + s), lp2 = __ldg(p + 2 * s), lp3 = __ldg(p + 3 * s), lp4 = __ldg(p + 4 * s);
  const double dm1 = lm1 - c, dp1 = lp1 - c, dm2 = lm2 - c, dp2 = lp2 - c, dm3 = lm3 - c, dp3 = lp3 - c,
               dm4 = lm4 - c, dp4 = lp4 - c;
  const double s1 = dp1 + dm1, s2 = dp2 + dm2, s3 = dp3 + dm3, s4 = dp4 + dm4;
  r.d1 = WANT_D1 ? (45.0 * (lp1 - lm1) - 9.0 * (lp2 - lm2) + (lp3 - lm3)) : 0.0;
  r.d2 = WANT_D2 ? (270.0 * s1 - 27.0 * s2 + 2.0 * s3) : 0.0;
  r.ko = 56.0 * s1 - 28.0 * s2 + 8.0 * s3 - s4;
  const double b2 = pos ? dm2 : dp2, b1 = pos ? dm1 : dp1;
  const double a1 = pos ? dp1 : dm1, a2 = pos ? dp2 : dm2, a3 = pos ? dp3 : dm3, a4 = pos ? dp4 : dm4;
  r.up = 2.0 * b2 - 24.0 * b1 + 80.0 * a1 - 30.0 * a2 + 8.0 * a3 - a4;
#endif
  return r;
}

// centred 1st derivative only (fields/axes where nothing else is needed: K4's d_k At_ij)
__device__ __forceinline__ double d1_raw(const double* __restrict__ p, const int s) {
#if Z4C_NG == 3
  return 8.0 * (__ldg(p + s) - __ldg(p - s)) - (__ldg(p + 2 * s) - __ldg(p - 2 * s));
#else
  return 45.0 * (__ldg(p + s) - __ldg(p - s)) - 9.0 * (__ldg(p + 2 * s) - __ldg(p - 2 * s)) +
         (__ldg(p + 3 * s) - __ldg(p - 3 * s));
#endif
}

// mixed second derivative D_b(D_a u), raw (scale 1/(144 h^2) [1/(3600 h^2)]); 16 [36] loads
__device__ __forceinline__ double mixed_raw(const double* __restrict__ p, const int sa, const int sb) {
  auto inner = [&](const double* q) { return d1_raw(q, sa); };
#if Z4C_NG == 3
  return 8.0 * (inner(p + sb) - inner(p - sb)) - (inner(p + 2 * sb) - inner(p - 2 * sb));
#else
  return 45.0 * (inner(p + sb) - inner(p - sb)) - 9.0 * (inner(p + 2 * sb) - inner(p - 2 * sb)) +
         (inner(p + 3 * sb) - inner(p - 3 * sb));
#endif
}

// ---- 3x3 symmetric algebra ------------------------------------------------------------------
__device__ __forceinline__ double det3(const double* g) {
  return g[0] * (g[3] * g[5] - g[4] * g[4]) - g[1] * (g[1] * g[5] - g[4] * g[2]) +
         g[2] * (g[1] * g[4] - g[3] * g[2]);
}
__device__ __forceinline__ void inv3(const double* g, double* gi) {
  const double idet = 1.0 / det3(g);
  gi[0] = (g[3] * g[5] - g[4] * g[4]) * idet;
  gi[1] = (g[2] * g[4] - g[1] * g[5]) * idet;
  gi[2] = (g[1] * g[4] - g[2] * g[3]) * idet;
  gi[3] = (g[0] * g[5] - g[2] * g[2]) * idet;
  gi[4] = (g[1] * g[2] - g[0] * g[4]) * idet;
  gi[5] = (g[0] * g[3] - g[1] * g[1]) * idet;
}
// full contraction of two symmetric tensors given in packed form: a^{ij} b_{ij}
__device__ __forceinline__ double contract(const double* a, const double* b) {
  return a[0] * b[0] + a[3] * b[3] + a[5] * b[5] + 2.0 * (a[1] * b[1] + a[2] * b[2] + a[4] * b[4]);
}

// Christoffel symbols of the conformal metric from dg[p][k] = d_k gt_p.
//   Gl[l][p] = Gamma~_{l ij},  Gu[k][p] = Gamma~^k_{ij},  Gd[k] = gi^{ij} Gamma~^k_{ij}
__device__ __forceinline__ void christoffel(const double (&dg)[6][3], const double* gi,
                                            double (&Gl)[3][6], double (&Gu)[3][6], double* Gd) {
#pragma unroll
  for (int l = 0; l < 3; ++l)
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = i; j < 3; ++j)
        Gl[l][sym(i, j)] = 0.5 * (dg[sym(j, l)][i] + dg[sym(i, l)][j] - dg[sym(i, j)][l]);
#pragma unroll
  for (int k = 0; k < 3; ++k) {
#pragma unroll
    for (int p = 0; p < 6; ++p)
      Gu[k][p] = gi[sym(k, 0)] * Gl[0][p] + gi[sym(k, 1)] * Gl[1][p] + gi[sym(k, 2)] * Gl[2][p];
    Gd[k] = contract(gi, Gu[k]);
  }
}

// R~_ij (O4) from: g, gi, lapg[p] = gi^{lm} d_l d_m gt_p, dGam[k][j] = d_j Gamt^k, Gl, Gu, Gd.
__device__ __forceinline__ void ricci_conformal(const double* g, const double* gi, const double* lapg,
                                                const double (&dGam)[3][3], const double (&Gl)[3][6],
                                                const double (&Gu)[3][6], const double* Gd, double* Rt) {
  // T[k][m][i] = gi^{lm} Gamma~^k_{l i}   (second index raised)
  double T[3][3][3];
#pragma unroll
  for (int k = 0; k < 3; ++k)
#pragma unroll
    for (int m = 0; m < 3; ++m)
#pragma unroll
      for (int i = 0; i < 3; ++i)
        T[k][m][i] = gi[sym(0, m)] * Gu[k][sym(0, i)] + gi[sym(1, m)] * Gu[k][sym(1, i)] +
                     gi[sym(2, m)] * Gu[k][sym(2, i)];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = i; j < 3; ++j) {
      const int p = sym(i, j);
      double r = -0.5 * lapg[p];
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        r += 0.5 * (g[sym(k, i)] * dGam[k][j] + g[sym(k, j)] * dGam[k][i]);
        r += 0.5 * Gd[k] * (Gl[i][sym(j, k)] + Gl[j][sym(i, k)]);
#pragma unroll
        for (int m = 0; m < 3; ++m) {
          // gi^{lm}( Gu^k_{li} Gl_{jkm} + Gu^k_{lj} Gl_{ikm} + Gu^k_{im} Gl_{klj} ) with T[k][m][.] = gi^{lm} Gu^k_{l .};
          // third term: gi^{lm} Gu^q_{im} Gl_{qlj} = gi^{lm} Gl_{q im} Gu^q_{lj} = Gl_{k im} T[k][m][j]  (lower q on the
          // first factor instead of the second: 3 FMAs per (k, m) instead of 6)
          r += T[k][m][i] * Gl[j][sym(k, m)] + T[k][m][j] * Gl[i][sym(k, m)] + T[k][m][j] * Gl[k][sym(i, m)];
        }
      }
      Rt[p] = r;
    }
}

// R^chi_ij (O4) and the conformal second covariant derivative of chi.
__device__ __forceinline__ void ricci_chi(const double chi, const double* dchi, const double* ddchi,
                                          const double* g, const double* gi, const double (&Gu)[3][6],
                                          double* Rchi) {
  double DD[6];
#pragma unroll
  for (int p = 0; p < 6; ++p) DD[p] = ddchi[p] - (Gu[0][p] * dchi[0] + Gu[1][p] * dchi[1] + Gu[2][p] * dchi[2]);
  const double lap = contract(gi, DD);
  double dd[6];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = i; j < 3; ++j) dd[sym(i, j)] = dchi[i] * dchi[j];
  const double d2 = contract(gi, dd);
  const double ichi = 1.0 / chi;
  const double h = 0.5 * ichi, q = 0.25 * ichi * ichi;
  const double tr = h * lap - 3.0 * q * d2;
#pragma unroll
  for (int p = 0; p < 6; ++p) Rchi[p] = h * DD[p] - q * dd[p] + g[p] * tr;
}

// x^(-1/3) by a fully specified sequence of IEEE operations (reading R-E1): bit-level seed
// K - bits(x)/3 with K = floor(4/3 (1023 - 0.045) 2^52), then five Newton steps
// y <- y + (y (1 - x y y y)) (1/3), every operation rounded separately (no FMA contraction).
__device__ __forceinline__ double inv_cbrt_spec(const double x) {
  const unsigned long long K = 0x553F0A3D70A3D70AULL;
  double y = __longlong_as_double((long long)(K - (unsigned long long)__double_as_longlong(x) / 3ULL));
  const double third = 1.0 / 3.0;
#pragma unroll
  for (int it = 0; it < 5; ++it) {
    double r = __dmul_rn(x, y);
    r = __dmul_rn(r, y);
    r = __dmul_rn(r, y);
    const double e = __dsub_rn(1.0, r);
    y = __dadd_rn(y, __dmul_rn(__dmul_rn(y, e), third));
  }
  return y;
}

}  // namespace z4c
