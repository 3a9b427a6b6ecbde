// Per-cell Z4c source terms on the device (S3 of SURVEY.md section 8(a); equations O4-O5 of section 8(c),
// restated in DESIGN.md "The method"; the paper defers them to Daszuta et al. 2021 at PAPER.md:51, 57).
// Everything here works on registers: the derivative bundle of one cell comes in, 22 time derivatives
// (or the constraint monitors) go out. Used by the RHS kernels (K2) and the constraint kernel (K4).
#pragma once
#include "z4c_math.cuh"

namespace z4c {

// Gauge / damping parameters of one launch (subset of z4c_params).
struct SrcParams {
  double kappa1, kappa2;
  double lapse_oplog, lapse_harmonic, lapse_advect;
  double shift_gamma, shift_eta, shift_advect;
};

__host__ __device__ constexpr bool need_d1(int f) { return !(f >= AXX && f <= AZZ); }
__host__ __device__ constexpr bool need_d2(int f) { return f <= GZZ || f >= ALPHA; }

// Derivative bundle of one cell (S2 -> S3). Second derivatives are contracted with gt^{ij} as soon as a field's
// stencils are done (the inverse metric needs only centre values), so only those of chi and alpha are kept:
// 66 -> 24 live doubles. Entries of fields that need no such derivative are never read, so after unrolling
// they do not occupy registers.
struct Derivs {
  double gi[6];      // gt^{ij}, filled before the first field is differentiated
  double d1[NF][3];  // centred d_k u_f
  double d2chi[6];   // centred d_k d_l chi, packed (xx,xy,xz,yy,yz,zz)
  double d2alpha[6]; // centred d_k d_l alpha
  double lapg[6];    // gt^{lm} d_l d_m gt_p
  double lapb[3];    // gt^{jk} d_j d_k beta^i
  double ddivb[3];   // d_j d_k beta^k   (must be zeroed before the shift is differentiated)
};

__device__ __forceinline__ void derivs_begin(const double* g, Derivs& D) {
  inv3(g, D.gi);
  D.ddivb[0] = D.ddivb[1] = D.ddivb[2] = 0.0;
}

// Hand the six second derivatives of field F to the bundle.
template <int F>
__device__ __forceinline__ void consume_d2(const double* d2, Derivs& D) {
  if (F == CHI) {
#pragma unroll
    for (int p = 0; p < 6; ++p) D.d2chi[p] = d2[p];
  } else if (F == ALPHA) {
#pragma unroll
    for (int p = 0; p < 6; ++p) D.d2alpha[p] = d2[p];
  } else if (F >= GXX && F <= GZZ) {
    D.lapg[F - GXX] = contract(D.gi, d2);
  } else if (F >= BETAX) {
    constexpr int i = F - BETAX;
    D.lapb[i] = contract(D.gi, d2);
#pragma unroll
    for (int j = 0; j < 3; ++j) D.ddivb[j] += d2[sym(j, i)];
  }
}

// Geometry shared by the RHS and the constraints.
struct Geom {
  double gi[6];      // gt^{ij}
  double Gu[3][6];   // Gamt^k_{ij}
  double Gd[3];      // gt^{ij} Gamt^k_{ij}
  double Ric[6];     // R_ij = Rt_ij + Rchi_ij
  double Rscal;      // chi gt^{ij} R_ij
  double Aup[6];     // At^{ij}
  double Am[3][3];   // At^i_j = gt^{ik} At_kj
  double AA;         // At_ij At^ij
  double K;          // Khat + 2 Theta
};

__device__ __forceinline__ void geometry(const double* u, const Derivs& D, Geom& G) {
  const double* g = u + GXX;
  const double* A = u + AXX;
#pragma unroll
  for (int p = 0; p < 6; ++p) G.gi[p] = D.gi[p];
  double dg[6][3];
#pragma unroll
  for (int p = 0; p < 6; ++p)
#pragma unroll
    for (int k = 0; k < 3; ++k) dg[p][k] = D.d1[GXX + p][k];
  double Gl[3][6];
  christoffel(dg, G.gi, Gl, G.Gu, G.Gd);
  double dGam[3][3];
#pragma unroll
  for (int k = 0; k < 3; ++k)
#pragma unroll
    for (int j = 0; j < 3; ++j) dGam[k][j] = D.d1[GAMX + k][j];
  double Rt[6], Rchi[6];
  ricci_conformal(g, G.gi, D.lapg, dGam, Gl, G.Gu, G.Gd, Rt);
  ricci_chi(u[CHI], D.d1[CHI], D.d2chi, g, G.gi, G.Gu, Rchi);
#pragma unroll
  for (int p = 0; p < 6; ++p) G.Ric[p] = Rt[p] + Rchi[p];
  G.Rscal = u[CHI] * contract(G.gi, G.Ric);
  // At^i_j and At^{ij}
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j)
      G.Am[i][j] = G.gi[sym(i, 0)] * A[sym(0, j)] + G.gi[sym(i, 1)] * A[sym(1, j)] + G.gi[sym(i, 2)] * A[sym(2, j)];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = i; j < 3; ++j)
      G.Aup[sym(i, j)] = G.Am[i][0] * G.gi[sym(0, j)] + G.Am[i][1] * G.gi[sym(1, j)] + G.Am[i][2] * G.gi[sym(2, j)];
  G.AA = contract(G.Aup, A);
  G.K = u[KHAT] + 2.0 * u[THETA];
}

// O5: out[f] += F_f(y).  `out` must already hold the upwinded advection and Kreiss-Oliger terms
// (with the gauge advection switches applied), which the derivative gather produces.
__device__ __forceinline__ void z4c_sources_post(const SrcParams& P, const double* u, const Derivs& D, const Geom& G,
                                                 double* out);
__device__ __forceinline__ void z4c_sources(const SrcParams& P, const double* u, const Derivs& D, double* out) {
  Geom G;
  geometry(u, D, G);
  z4c_sources_post(P, u, D, G, out);
}

// The derivatives that only the assembly after geometry() reads: 30 doubles. A kernel may park them in shared
// memory across geometry(), where the Christoffel / Ricci temporaries peak (STORE = true before, false after).
constexpr int NPARK = 30;
template <bool STORE>
__device__ __forceinline__ void park_late_derivs(Derivs& D, double* slot, const int stride) {
  int q = 0;
  auto io = [&](double& x) {
    if (STORE) slot[q * stride] = x; else x = slot[q * stride];
    ++q;
  };
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    io(D.d1[BETAX][a]); io(D.d1[BETAY][a]); io(D.d1[BETAZ][a]);
    io(D.d1[KHAT][a]); io(D.d1[THETA][a]); io(D.d1[ALPHA][a]);
    io(D.lapb[a]); io(D.ddivb[a]);
  }
#pragma unroll
  for (int p = 0; p < 6; ++p) io(D.d2alpha[p]);
}

// The same slots, written as soon as field F's stencils are done (a kernel with a dedicated parking area can keep
// these values out of registers through the whole field stream, not only through geometry()).
template <int F>
__device__ __forceinline__ void park_field_early(const Derivs& D, double* slot, const int stride) {
  constexpr int col = F == BETAX ? 0 : F == BETAY ? 1 : F == BETAZ ? 2 : F == KHAT ? 3 : F == THETA ? 4 : F == ALPHA ? 5 : -1;
  if (col >= 0) {
#pragma unroll
    for (int a = 0; a < 3; ++a) slot[(a * 8 + col) * stride] = D.d1[F][a];
  }
  if (F >= BETAX) slot[((F - BETAX) * 8 + 6) * stride] = D.lapb[F - BETAX];
  if (F == BETAZ) {
#pragma unroll
    for (int a = 0; a < 3; ++a) slot[(a * 8 + 7) * stride] = D.ddivb[a];
  }
  if (F == ALPHA) {
#pragma unroll
    for (int p = 0; p < 6; ++p) slot[(24 + p) * stride] = D.d2alpha[p];
  }
}

__device__ __forceinline__ void z4c_sources_post(const SrcParams& P, const double* u, const Derivs& D, const Geom& G,
                                                 double* out) {
  const double* g = u + GXX;
  const double* A = u + AXX;
  const double chi = u[CHI], alpha = u[ALPHA], Theta = u[THETA], K = G.K;
  const double* gi = G.gi;
  const double* dchi = D.d1[CHI];
  const double* da = D.d1[ALPHA];
  // d_i beta^k = D.d1[BETAX + k][i]
  const double divb = D.d1[BETAX][0] + D.d1[BETAY][1] + D.d1[BETAZ][2];
  const double ichi = 1.0 / chi;

  // D_iD_j alpha
  double DDa[6];
  {
    double dd[6];
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = i; j < 3; ++j) dd[sym(i, j)] = da[i] * dchi[j] + da[j] * dchi[i];
    // gi^{kl} da_k dchi_l = 1/2 gi^{kl} (da_k dchi_l + da_l dchi_k)
    const double dadchi = 0.5 * contract(gi, dd);
#pragma unroll
    for (int p = 0; p < 6; ++p)
      DDa[p] = D.d2alpha[p] - (G.Gu[0][p] * da[0] + G.Gu[1][p] * da[1] + G.Gu[2][p] * da[2]) +
               0.5 * ichi * (dd[p] - g[p] * dadchi);
  }

  out[CHI] += (2.0 / 3.0) * chi * (alpha * K - divb);

#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = i; j < 3; ++j) {
      const int p = sym(i, j);
      double s = -2.0 * alpha * A[p];
#pragma unroll
      for (int k = 0; k < 3; ++k) s += g[sym(i, k)] * D.d1[BETAX + k][j] + g[sym(k, j)] * D.d1[BETAX + k][i];
      out[GXX + p] += s - (2.0 / 3.0) * g[p] * divb;
    }

  out[KHAT] += -chi * contract(gi, DDa) + alpha * (G.AA + K * K * (1.0 / 3.0)) +
               alpha * (P.kappa1 * (1.0 - P.kappa2)) * Theta;

  {
    double X[6];
#pragma unroll
    for (int p = 0; p < 6; ++p) X[p] = alpha * G.Ric[p] - DDa[p];
    const double Xtr3 = contract(gi, X) * (1.0 / 3.0);
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = i; j < 3; ++j) {
        const int p = sym(i, j);
        // At_ik gt^{kl} At_lj = At_ik At^k_j
        const double AgA = A[sym(i, 0)] * G.Am[0][j] + A[sym(i, 1)] * G.Am[1][j] + A[sym(i, 2)] * G.Am[2][j];
        double s = chi * (X[p] - g[p] * Xtr3) + alpha * (K * A[p] - 2.0 * AgA);
#pragma unroll
        for (int k = 0; k < 3; ++k) s += A[sym(i, k)] * D.d1[BETAX + k][j] + A[sym(k, j)] * D.d1[BETAX + k][i];
        out[AXX + p] += s - (2.0 / 3.0) * A[p] * divb;
      }
  }

  {
    const double* ddivb = D.ddivb;   // d_j (d_k beta^k)
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      double s = 0.0, b = 0.0;
#pragma unroll
      for (int j = 0; j < 3; ++j) {
        s -= 2.0 * G.Aup[sym(i, j)] * da[j];
        b -= 1.5 * G.Aup[sym(i, j)] * dchi[j] * ichi;
        b -= gi[sym(i, j)] * (2.0 * D.d1[KHAT][j] + D.d1[THETA][j]) * (1.0 / 3.0);
        s += gi[sym(i, j)] * ddivb[j] * (1.0 / 3.0);
        s -= G.Gd[j] * D.d1[BETAX + i][j];
      }
      b += contract(G.Gu[i], G.Aup);
      s += 2.0 * alpha * b;
      s += D.lapb[i];
      s += (2.0 / 3.0) * G.Gd[i] * divb;
      s -= 2.0 * P.kappa1 * alpha * (u[GAMX + i] - G.Gd[i]);
      out[GAMX + i] += s;
    }
  }

  out[THETA] += 0.5 * alpha * (G.Rscal - G.AA + (2.0 / 3.0) * K * K) - alpha * (P.kappa1 * (2.0 + P.kappa2)) * Theta;

  out[ALPHA] += -(P.lapse_oplog * alpha + P.lapse_harmonic * alpha * alpha) * u[KHAT];
#pragma unroll
  for (int i = 0; i < 3; ++i) out[BETAX + i] += P.shift_gamma * u[GAMX + i] - P.shift_eta * u[BETAX + i];
}

// O5 constraints: c = {H, M_x, M_y, M_z, |M|^2, |Z|^2}. dAt(i, q) returns the centred d_i At_p, p = 0..5, of axis i in
// q[6]: the 18 derivatives of At_ij are asked for one axis at a time (6 live values instead of 18, which together with
// the geometry did not fit the register file: 552 bytes of spill in round 1).
template <class DA>
__device__ __forceinline__ void z4c_constraints_point(const double* u, const Derivs& D, DA dAt, double* c) {
  Geom G;
  geometry(u, D, G);
  const double* g = u + GXX;
  const double* A = u + AXX;
  const double* gi = G.gi;
  const double ichi = 1.0 / u[CHI];
  c[0] = G.Rscal - G.AA + (2.0 / 3.0) * G.K * G.K;
  double M[3];
#pragma unroll
  for (int j = 0; j < 3; ++j) M[j] = -(2.0 / 3.0) * (D.d1[KHAT][j] + 2.0 * D.d1[THETA][j]);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    double dAi[6];
    dAt(i, dAi);
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      double s = 0.0;
      // d_i At^i_j = (d_i gt^{ik}) At_kj + gt^{ik} d_i At_kj,  d_i gt^{ik} = - gt^{ic} d_i gt_cd gt^{dk}
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        double dginv = 0.0;
#pragma unroll
        for (int cc = 0; cc < 3; ++cc)
#pragma unroll
          for (int d = 0; d < 3; ++d) dginv -= gi[sym(i, cc)] * D.d1[GXX + sym(cc, d)][i] * gi[sym(d, k)];
        s += dginv * A[sym(k, j)] + gi[sym(i, k)] * dAi[sym(k, j)];
        s += G.Gu[i][sym(i, k)] * G.Am[k][j] - G.Gu[k][sym(i, j)] * G.Am[i][k];
      }
      s -= 1.5 * G.Am[i][j] * D.d1[CHI][i] * ichi;
      M[j] += s;
    }
  }
#pragma unroll
  for (int j = 0; j < 3; ++j) c[1 + j] = M[j];
  double Z[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) Z[i] = u[GAMX + i] - G.Gd[i];
  double m2 = 0.0, z2 = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      m2 += gi[sym(i, j)] * M[i] * M[j];
      z2 += g[sym(i, j)] * Z[i] * Z[j];
    }
  c[4] = m2;
  c[5] = z2;
}

}  // namespace z4c
