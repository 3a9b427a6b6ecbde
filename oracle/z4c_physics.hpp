// =====================================================================================
// oracle/z4c_physics.hpp -- TEST INFRASTRUCTURE, NOT PRODUCT (see z4c_oracle.hpp).
//
// Per-cell Z4c algebra: O4 (derived quantities), O5 (evolution equations + constraints)
// of SURVEY.md section 8(c).  PAPER.md:51 and PAPER.md:57 (section 2) defer the continuum
// equations to Daszuta et al. 2021 Eq. 8-13, 22, which are not printed in the paper; the
// system written here is the standard Z4c system of Bernuzzi & Hilditch 2010 / Hilditch
// et al. 2013 (cited at PAPER.md:51) -- reading Q2 -- and is pinned by P3-P7.
// Statements follow the notation of O4/O5 line by line; sums are written out as loops.
// =====================================================================================
#pragma once
#include "z4c_oracle.hpp"

namespace oz4c {

// O4: gamma~^ij, Christoffels, Ricci, D_iD_j alpha, A~^ij, traces.
template <class T>
inline void geometry(const T* u, const Derivs<T>& D, Geometry<T>& G) {
  const T* g = u + GXX;
  const T* A = u + AXX;
  const T chi = u[CHI];
  T det = det_sym(g);
  inv_sym(g, det, G.ginv);
  auto gi = [&](int i, int j) -> T { return G.ginv[SYM[i][j]]; };
  auto gl = [&](int i, int j) -> T { return g[SYM[i][j]]; };
  auto dg = [&](int k, int i, int j) -> T { return D.d1[GXX + SYM[i][j]][k]; };  // d_k g_ij

  // Gamma~_{l ij} = 1/2 (d_i g_jl + d_j g_il - d_l g_ij)
  for (int l = 0; l < 3; ++l)
    for (int i = 0; i < 3; ++i)
      for (int j = i; j < 3; ++j)
        G.Gl[l][SYM[i][j]] = T(0.5) * (dg(i, j, l) + dg(j, i, l) - dg(l, i, j));
  // Gamma~^k_{ij} = ginv^{kl} Gamma~_{l ij}
  for (int k = 0; k < 3; ++k)
    for (int p = 0; p < 6; ++p) {
      T s = T(0.0);
      for (int l = 0; l < 3; ++l) s = s + gi(k, l) * G.Gl[l][p];
      G.Gu[k][p] = s;
    }
  // Gamma~_d^k = ginv^{ij} Gamma~^k_{ij}
  for (int k = 0; k < 3; ++k) {
    T s = T(0.0);
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 3; ++j) s = s + gi(i, j) * G.Gu[k][SYM[i][j]];
    G.Gd[k] = s;
  }
  auto Gl3 = [&](int a, int b, int c) -> T { return G.Gl[a][SYM[b][c]]; };  // Gamma~_{a bc}
  auto Gu3 = [&](int a, int b, int c) -> T { return G.Gu[a][SYM[b][c]]; };  // Gamma~^a_{bc}

  // R~_ij = -1/2 ginv^{lm} d_l d_m g_ij + 1/2 (g_ki d_j Gam^k + g_kj d_i Gam^k)
  //         + 1/2 Gd^k (Gamma~_{ijk} + Gamma~_{jik})
  //         + ginv^{lm} ( Gu^k_{li} Gl_{jkm} + Gu^k_{lj} Gl_{ikm} + Gu^k_{im} Gl_{klj} )
  for (int i = 0; i < 3; ++i)
    for (int j = i; j < 3; ++j) {
      const int p = SYM[i][j];
      T lap = T(0.0);
      for (int l = 0; l < 3; ++l)
        for (int m = 0; m < 3; ++m) lap = lap + gi(l, m) * D.d2[GXX + p][SYM[l][m]];
      T r = T(-0.5) * lap;
      for (int k = 0; k < 3; ++k) {
        r = r + T(0.5) * (gl(k, i) * D.d1[GAMX + k][j] + gl(k, j) * D.d1[GAMX + k][i]);
        r = r + T(0.5) * G.Gd[k] * (Gl3(i, j, k) + Gl3(j, i, k));
      }
      for (int l = 0; l < 3; ++l)
        for (int m = 0; m < 3; ++m) {
          T s = T(0.0);
          for (int k = 0; k < 3; ++k)
            s = s + Gu3(k, l, i) * Gl3(j, k, m) + Gu3(k, l, j) * Gl3(i, k, m) +
                Gu3(k, i, m) * Gl3(k, l, j);
          r = r + gi(l, m) * s;
        }
      G.Rt[p] = r;
    }

  // D~_i D~_j chi = d_i d_j chi - Gu^k_{ij} d_k chi
  T DDchi[6];
  for (int p = 0; p < 6; ++p) {
    T s = D.d2[CHI][p];
    for (int k = 0; k < 3; ++k) s = s - G.Gu[k][p] * D.d1[CHI][k];
    DDchi[p] = s;
  }
  T lapchi = T(0.0), dchi2 = T(0.0);
  for (int l = 0; l < 3; ++l)
    for (int m = 0; m < 3; ++m) {
      lapchi = lapchi + gi(l, m) * DDchi[SYM[l][m]];
      dchi2 = dchi2 + gi(l, m) * D.d1[CHI][l] * D.d1[CHI][m];
    }
  // R^chi_ij = (1/2chi) DDchi_ij + (1/2chi) g_ij lapchi - (1/4chi^2) dchi_i dchi_j
  //            - (3/4chi^2) g_ij dchi2
  for (int i = 0; i < 3; ++i)
    for (int j = i; j < 3; ++j) {
      const int p = SYM[i][j];
      G.Rchi[p] = DDchi[p] / (T(2.0) * chi) + g[p] * lapchi / (T(2.0) * chi) -
                  D.d1[CHI][i] * D.d1[CHI][j] / (T(4.0) * chi * chi) -
                  T(3.0) * g[p] * dchi2 / (T(4.0) * chi * chi);
      G.Ric[p] = G.Rt[p] + G.Rchi[p];
    }
  T tr = T(0.0);
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) tr = tr + gi(i, j) * G.Ric[SYM[i][j]];
  G.Rscal = chi * tr;

  // D_iD_j alpha = d_i d_j alpha - Gu^k_{ij} d_k alpha
  //   + (1/2chi)(d_i alpha d_j chi + d_j alpha d_i chi - g_ij ginv^{kl} d_k alpha d_l chi)
  T dadchi = T(0.0);
  for (int k = 0; k < 3; ++k)
    for (int l = 0; l < 3; ++l) dadchi = dadchi + gi(k, l) * D.d1[ALPHA][k] * D.d1[CHI][l];
  for (int i = 0; i < 3; ++i)
    for (int j = i; j < 3; ++j) {
      const int p = SYM[i][j];
      T s = D.d2[ALPHA][p];
      for (int k = 0; k < 3; ++k) s = s - G.Gu[k][p] * D.d1[ALPHA][k];
      s = s + (D.d1[ALPHA][i] * D.d1[CHI][j] + D.d1[ALPHA][j] * D.d1[CHI][i] - g[p] * dadchi) /
                  (T(2.0) * chi);
      G.DDalpha[p] = s;
    }

  // A~^{ij} = ginv^{ik} ginv^{jl} A~_kl ;  A~_ij A~^ij ;  K = Khat + 2 Theta
  for (int i = 0; i < 3; ++i)
    for (int j = i; j < 3; ++j) {
      T s = T(0.0);
      for (int k = 0; k < 3; ++k)
        for (int l = 0; l < 3; ++l) s = s + gi(i, k) * gi(j, l) * A[SYM[k][l]];
      G.Aup[SYM[i][j]] = s;
    }
  T aa = T(0.0);
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) aa = aa + A[SYM[i][j]] * G.Aup[SYM[i][j]];
  G.AA = aa;
  G.K = u[KHAT] + T(2.0) * u[THETA];
}

// O5: the 22 time derivatives F(y) + Q_KO(y) at one cell.
template <class T>
inline void rhs_point(const Params& P, const T* u, const Derivs<T>& D, T* out) {
  Geometry<T> G;
  geometry(u, D, G);
  const T* g = u + GXX;
  const T* A = u + AXX;
  const T chi = u[CHI], alpha = u[ALPHA], Theta = u[THETA];
  const T K = G.K;
  auto gi = [&](int i, int j) -> T { return G.ginv[SYM[i][j]]; };
  auto dbeta = [&](int i, int k) -> T { return D.d1[BETAX + k][i]; };  // d_i beta^k
  const T divb = dbeta(0, 0) + dbeta(1, 1) + dbeta(2, 2);
  const double k1 = P.kappa1, k2 = P.kappa2;

  // d_t chi = 2/3 chi [alpha K - d_k beta^k] + beta^k d_k chi
  out[CHI] = T(2.0 / 3.0) * chi * (alpha * K - divb) + D.adv[CHI];

  // d_t g_ij = -2 alpha A_ij + adv + g_ik d_j beta^k + g_kj d_i beta^k - 2/3 g_ij divb
  for (int i = 0; i < 3; ++i)
    for (int j = i; j < 3; ++j) {
      const int p = SYM[i][j];
      T s = T(-2.0) * alpha * A[p] + D.adv[GXX + p];
      for (int k = 0; k < 3; ++k) s = s + g[SYM[i][k]] * dbeta(j, k) + g[SYM[k][j]] * dbeta(i, k);
      out[GXX + p] = s - T(2.0 / 3.0) * g[p] * divb;
    }

  // d_t Khat = -D^iD_i alpha + alpha [AA + K^2/3] + alpha k1 (1-k2) Theta + adv
  T DDa_tr = T(0.0);
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) DDa_tr = DDa_tr + gi(i, j) * G.DDalpha[SYM[i][j]];
  out[KHAT] = T(-1.0) * chi * DDa_tr + alpha * (G.AA + K * K / T(3.0)) +
              alpha * T(k1 * (1.0 - k2)) * Theta + D.adv[KHAT];

  // d_t A_ij = chi [ -D_iD_j alpha + alpha R_ij ]^TF + alpha [ K A_ij - 2 A_ik ginv^{kl} A_lj ]
  //            + adv + A_ik d_j beta^k + A_kj d_i beta^k - 2/3 A_ij divb
  T X[6];
  T Xtr = T(0.0);
  for (int p = 0; p < 6; ++p) X[p] = alpha * G.Ric[p] - G.DDalpha[p];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) Xtr = Xtr + gi(i, j) * X[SYM[i][j]];
  for (int i = 0; i < 3; ++i)
    for (int j = i; j < 3; ++j) {
      const int p = SYM[i][j];
      T AgA = T(0.0);
      for (int k = 0; k < 3; ++k)
        for (int l = 0; l < 3; ++l) AgA = AgA + A[SYM[i][k]] * gi(k, l) * A[SYM[l][j]];
      T s = chi * (X[p] - g[p] * Xtr / T(3.0)) + alpha * (K * A[p] - T(2.0) * AgA) +
            D.adv[AXX + p];
      for (int k = 0; k < 3; ++k) s = s + A[SYM[i][k]] * dbeta(j, k) + A[SYM[k][j]] * dbeta(i, k);
      out[AXX + p] = s - T(2.0 / 3.0) * A[p] * divb;
    }

  // d_t Gam^i = -2 Aup^{ij} d_j alpha
  //   + 2 alpha [ Gu^i_{jk} Aup^{jk} - 3/2 Aup^{ij} d_j chi / chi - 1/3 ginv^{ij} d_j (2 Khat + Theta) ]
  //   + ginv^{jk} d_j d_k beta^i + 1/3 ginv^{ij} d_j d_k beta^k
  //   + adv - Gd^j d_j beta^i + 2/3 Gd^i divb - 2 alpha k1 (Gam^i - Gd^i)
  for (int i = 0; i < 3; ++i) {
    T s = T(0.0);
    for (int j = 0; j < 3; ++j) s = s - T(2.0) * G.Aup[SYM[i][j]] * D.d1[ALPHA][j];
    T b = T(0.0);
    for (int j = 0; j < 3; ++j) {
      for (int k = 0; k < 3; ++k) b = b + G.Gu[i][SYM[j][k]] * G.Aup[SYM[j][k]];
      b = b - T(1.5) * G.Aup[SYM[i][j]] * D.d1[CHI][j] / chi;
      b = b - gi(i, j) * (T(2.0) * D.d1[KHAT][j] + D.d1[THETA][j]) / T(3.0);
    }
    s = s + T(2.0) * alpha * b;
    for (int j = 0; j < 3; ++j)
      for (int k = 0; k < 3; ++k) {
        s = s + gi(j, k) * D.d2[BETAX + i][SYM[j][k]];
        s = s + gi(i, j) * D.d2[BETAX + k][SYM[j][k]] / T(3.0);
      }
    s = s + D.adv[GAMX + i];
    for (int j = 0; j < 3; ++j) s = s - G.Gd[j] * dbeta(j, i);
    s = s + T(2.0 / 3.0) * G.Gd[i] * divb;
    s = s - T(2.0 * k1) * alpha * (u[GAMX + i] - G.Gd[i]);
    out[GAMX + i] = s;
  }

  // d_t Theta = 1/2 alpha [ R - AA + 2/3 K^2 ] - alpha k1 (2+k2) Theta + adv
  out[THETA] = T(0.5) * alpha * (G.Rscal - G.AA + T(2.0 / 3.0) * K * K) -
               alpha * T(k1 * (2.0 + k2)) * Theta + D.adv[THETA];

  // d_t alpha = -(c_log alpha + c_harm alpha^2) Khat + c_adv adv      (Q7: Khat, not K)
  out[ALPHA] = T(-1.0) * (T(P.lapse_oplog) * alpha + T(P.lapse_harmonic) * alpha * alpha) * u[KHAT] +
               T(P.lapse_advect) * D.adv[ALPHA];

  // d_t beta^i = c_Gam Gam^i - eta beta^i + c_adv adv                 (Q6)
  for (int i = 0; i < 3; ++i)
    out[BETAX + i] = T(P.shift_gamma) * u[GAMX + i] - T(P.shift_eta) * u[BETAX + i] +
                     T(P.shift_advect) * D.adv[BETAX + i];

  // Kreiss-Oliger dissipation on all 22 fields (O3)
  for (int f = 0; f < NF; ++f) out[f] = out[f] + D.ko[f];
}

// O5 constraints at one cell: out = {H, M_x, M_y, M_z, |M|^2, |Z|^2}.
// dA[k][p] = centred d_k A~_p (the 18 extra derivatives S5 needs).
template <class T>
inline void constraints_point(const T* u, const Derivs<T>& D, const T dA[3][6], T* out) {
  Geometry<T> G;
  geometry(u, D, G);
  const T* g = u + GXX;
  const T* A = u + AXX;
  const T chi = u[CHI];
  const T K = G.K;
  auto gi = [&](int i, int j) -> T { return G.ginv[SYM[i][j]]; };
  // H = R - AA + 2/3 K^2
  out[0] = G.Rscal - G.AA + T(2.0 / 3.0) * K * K;
  // mixed A^i_j = ginv^{ik} A_kj
  T Am[3][3];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      T s = T(0.0);
      for (int k = 0; k < 3; ++k) s = s + gi(i, k) * A[SYM[k][j]];
      Am[i][j] = s;
    }
  // d_i ginv^{ab} = - ginv^{ac} d_i g_cd ginv^{db}
  T M[3];
  for (int j = 0; j < 3; ++j) {
    T s = T(0.0);
    for (int i = 0; i < 3; ++i) {
      // d_i A^i_j = (d_i ginv^{ik}) A_kj + ginv^{ik} d_i A_kj
      for (int k = 0; k < 3; ++k) {
        T dginv = T(0.0);
        for (int c = 0; c < 3; ++c)
          for (int d = 0; d < 3; ++d)
            dginv = dginv - gi(i, c) * D.d1[GXX + SYM[c][d]][i] * gi(d, k);
        s = s + dginv * A[SYM[k][j]] + gi(i, k) * dA[i][SYM[k][j]];
      }
      // + Gu^i_{ik} A^k_j - Gu^k_{ij} A^i_k
      for (int k = 0; k < 3; ++k)
        s = s + G.Gu[i][SYM[i][k]] * Am[k][j] - G.Gu[k][SYM[i][j]] * Am[i][k];
      // - 3/2 A^i_j d_i chi / chi
      s = s - T(1.5) * Am[i][j] * D.d1[CHI][i] / chi;
    }
    // - 2/3 d_j K
    s = s - T(2.0 / 3.0) * (D.d1[KHAT][j] + T(2.0) * D.d1[THETA][j]);
    M[j] = s;
    out[1 + j] = s;
  }
  T m2 = T(0.0), z2 = T(0.0);
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      m2 = m2 + gi(i, j) * M[i] * M[j];
      z2 = z2 + g[SYM[i][j]] * (u[GAMX + i] - G.Gd[i]) * (u[GAMX + j] - G.Gd[j]);
    }
  out[4] = m2;
  out[5] = z2;
}

}  // namespace oz4c
