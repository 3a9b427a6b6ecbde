// =====================================================================================
// oracle/z4c_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT (see z4c_oracle.hpp).
//
// Block-free global-array driver: O1 grid, O2 neighbour access by wrap/clamp (which is
// also the definition the GPU ghost fill K1 must reproduce: PAPER.md:65, 75-76, 84),
// O6 classical RK4 in the 3-register recurrence, O7 enforcement.
// Compiled with -O2 -ffp-contract=off (no FMA contraction: every * and + below is one
// IEEE-754 binary64 operation, in the order written).  Optional OpenMP over z-planes.
// =====================================================================================
#include "z4c_physics.hpp"
#include "z4c_amr.hpp"

#include <cmath>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace oz4c {

// ---- operation-counting scalar (flop census for DESIGN.md's roofline) -----------------
struct Counts { long long add, mul, div; };
static thread_local Counts g_counts = {0, 0, 0};
struct CScalar {
  double v;
  CScalar() : v(0) {}
  explicit CScalar(double x) : v(x) {}
};
inline CScalar operator+(CScalar a, CScalar b) { ++g_counts.add; return CScalar(a.v + b.v); }
inline CScalar operator-(CScalar a, CScalar b) { ++g_counts.add; return CScalar(a.v - b.v); }
inline CScalar operator*(CScalar a, CScalar b) { ++g_counts.mul; return CScalar(a.v * b.v); }
inline CScalar operator/(CScalar a, CScalar b) { ++g_counts.div; return CScalar(a.v / b.v); }
inline double value(double x) { return x; }
inline double value(CScalar x) { return x.v; }

// ---- O2 neighbour access ---------------------------------------------------------------
static inline int map_index(int i, int N, int bc) {
  if (bc == 0) { i %= N; if (i < 0) i += N; return i; }
  return i < 0 ? 0 : (i >= N ? N - 1 : i);
}

struct View {
  const Params& P;
  const double* u;       // [NF][Nz][Ny][Nx]; with pad > 0: [NF][Nz+2pad][Ny+2pad][Nx+2pad]
  size_t ncell;
  int pad;               // 0: neighbours by wrap/clamp (O2); > 0: the array carries `pad` filled ghost layers (NEXT-3:
                         // the fine level of a refinement boundary, whose ghosts come from prolongation)
  View(const Params& p, const double* uu, int pad_ = 0) : P(p), u(uu),
      ncell((size_t)(p.N[0] + 2 * pad_) * (p.N[1] + 2 * pad_) * (p.N[2] + 2 * pad_)), pad(pad_) {}
  inline double at(int f, int i, int j, int k) const {
    if (pad > 0)
      return u[(size_t)f * ncell + ((size_t)(k + pad) * (P.N[1] + 2 * pad) + (j + pad)) * (P.N[0] + 2 * pad) + (i + pad)];
    i = map_index(i, P.N[0], P.bc); j = map_index(j, P.N[1], P.bc); k = map_index(k, P.N[2], P.bc);
    return u[(size_t)f * ncell + ((size_t)k * P.N[1] + j) * P.N[0] + i];
  }
};

// ---- S2: gather all derivatives of one cell -------------------------------------------
static const bool NEEDS_D1[NF] = {1, 1,1,1,1,1,1, 1, 0,0,0,0,0,0, 1,1,1, 1, 1, 1,1,1};
static const bool NEEDS_D2[NF] = {1, 1,1,1,1,1,1, 0, 0,0,0,0,0,0, 0,0,0, 0, 1, 1,1,1};

template <class T>
static void gather(const View& V, int i, int j, int k, bool all_d1, T* u, Derivs<T>& D) {
  const double h = V.P.dx;
  const int c[3] = {i, j, k};
  for (int f = 0; f < NF; ++f) u[f] = T(V.at(f, i, j, k));
  for (int f = 0; f < NF; ++f) {
    const bool o6 = sixth_order(V.P);
    const int width = o6 ? 4 : 3;
    T line[3][9];
    for (int a = 0; a < 3; ++a)
      for (int s = -4; s <= 4; ++s) {
        int q[3] = {c[0], c[1], c[2]};
        q[a] += s;
        // offsets beyond the stencil half-width are never used (and do not exist in a padded array)
        line[a][s + 4] = (s < -width || s > width) ? T(0.0) : T(V.at(f, q[0], q[1], q[2]));
      }
    T adv = T(0.0), ko = T(0.0);
    for (int a = 0; a < 3; ++a) {
      const T* l = &line[a][4];
      if (NEEDS_D1[f] || all_d1) D.d1[f][a] = o6 ? d1_centred6(l, h) : d1_centred(l, h); else D.d1[f][a] = T(0.0);
      if (NEEDS_D2[f]) D.d2[f][SYM[a][a]] = o6 ? d2_centred6(l, h) : d2_centred(l, h);
      const T beta = u[BETAX + a];
      adv = adv + beta * (o6 ? d1_upwind6(l, h, value(beta) >= 0.0) : d1_upwind(l, h, value(beta) >= 0.0));
      ko = ko + (o6 ? ko_axis6(l) : ko_axis(l));
    }
    D.adv[f] = adv;
    D.ko[f] = T(V.P.ko_eps / ((o6 ? 256.0 : 64.0) * h)) * ko;
    if (NEEDS_D2[f]) {
      for (int a = 0; a < 3; ++a)
        for (int b = a + 1; b < 3; ++b) {
          auto v = [&](int sa, int sb) -> T {
            int q[3] = {c[0], c[1], c[2]};
            q[a] += sa; q[b] += sb;
            return T(V.at(f, q[0], q[1], q[2]));
          };
          D.d2[f][SYM[a][b]] = o6 ? d2_mixed6<T>(v, h) : d2_mixed<T>(v, h);
        }
    } else {
      for (int p = 0; p < 6; ++p) D.d2[f][p] = T(0.0);
    }
  }
}

// ---- S2+S3 over the grid: rhs = F(y) + Q_KO(y) ------------------------------------------
static void rhs_global(const Params& P, const double* u, double* rhs, int pad = 0) {
  View V(P, u, pad);
  const size_t nc = (size_t)P.N[0] * P.N[1] * P.N[2];   // rhs holds interior cells only
#pragma omp parallel for schedule(static)
  for (int k = 0; k < P.N[2]; ++k)
    for (int j = 0; j < P.N[1]; ++j)
      for (int i = 0; i < P.N[0]; ++i) {
        double uc[NF], out[NF];
        Derivs<double> D;
        gather<double>(V, i, j, k, false, uc, D);
        rhs_point<double>(P, uc, D, out);
        const size_t c = ((size_t)k * P.N[1] + j) * P.N[0] + i;
        for (int f = 0; f < NF; ++f) rhs[(size_t)f * nc + c] = out[f];
      }
}

// ---- O7 enforcement --------------------------------------------------------------------
// Reading R-E1: x^(-1/3) is evaluated by a fully specified sequence of IEEE
// operations (bit-level seed, five Newton steps) so that two independent implementations
// agree bit for bit; libm cbrt is only specified to ~1 ulp and an ulp of gamma~_ii ~ 1 is
// amplified by dt/h^2 into A~_ij.
static inline double inv_cbrt_spec(double x) {
  uint64_t b;
  std::memcpy(&b, &x, 8);
  // seed: bits(y) = K - bits(x)/3, K = floor(4/3 * (1023 - 0.045) * 2^52)
  const uint64_t K = 0x553F0A3D70A3D70AULL;   // = 6142639675755714314
  b = K - b / 3ULL;
  double y;
  std::memcpy(&y, &b, 8);
  const double third = 1.0 / 3.0;
  for (int it = 0; it < 5; ++it) {
    double r = x * y;
    r = r * y;
    r = r * y;
    double e = 1.0 - r;
    y = y + (y * e) * third;
  }
  return y;
}

// returns 0 if fine, 1 if det<=0 or non-finite was seen in this cell
static inline int enforce_point(double* u, double chi_floor) {
  double* g = u + GXX;
  double* A = u + AXX;
  double det = det_sym(g);
  int bad = !(det > 0.0) || !std::isfinite(det);
  if (bad) return 1;
  double s = inv_cbrt_spec(det);
  for (int p = 0; p < 6; ++p) g[p] = s * g[p];
  double det2 = det_sym(g);
  double gi[6];
  inv_sym(g, det2, gi);
  double t = gi[0] * A[0] + gi[3] * A[3] + gi[5] * A[5] +
             2.0 * (gi[1] * A[1] + gi[2] * A[2] + gi[4] * A[4]);
  const double third = 1.0 / 3.0;
  for (int p = 0; p < 6; ++p) A[p] = A[p] - third * (g[p] * t);
  if (!std::isfinite(u[CHI])) return 1;
  if (u[CHI] < chi_floor) u[CHI] = chi_floor;
  return 0;
}

static int enforce_global(const Params& P, double* u, int do_enforce) {
  if (!do_enforce) return 0;
  const size_t nc = (size_t)P.N[0] * P.N[1] * P.N[2];
  int bad = 0;
#pragma omp parallel for schedule(static) reduction(| : bad)
  for (long long c = 0; c < (long long)nc; ++c) {
    double uc[NF];
    for (int f = 0; f < NF; ++f) uc[f] = u[(size_t)f * nc + c];
    bad |= enforce_point(uc, P.chi_floor);
    for (int f = 0; f < NF; ++f) {
      if (!std::isfinite(uc[f])) bad |= 1;
      u[(size_t)f * nc + c] = uc[f];
    }
  }
  return bad;
}

// ---- O6 RK4, 3-register recurrence -------------------------------------------------------
// One stage of the recurrence on n values: L = F(y) + Q_KO(y) of the current y. (One function so that the
// single-level and the two-level drivers run the very same statements.)
// Reading O6 (amended in round 2): the two factors 1/6 of the recurrence are applied as a multiplication by the
// correctly rounded double 1/6, not as a division. The paper prints no recurrence at all ("a family of
// explicit Runge-Kutta methods"; RK4 at PAPER.md:169, 203, 279), so which of the two equal real-number forms is used is
// ours to fix; the product costs the GPU one instruction where the IEEE division costs ~15 in each of 44 places, in
// kernels that are instruction-fetch bound. Oracle and kernels use the same form, each rounding product and sum separately.
static const double SIXTH = 1.0 / 6.0;
static void rk_stage_update(int stage, size_t n, double dt, const double* L, double* y, double* Pr, double* Q) {
  if (stage == 1) {
    // stage 1: P = L(y); Q = P; y = E(y + P/2)
#pragma omp parallel for schedule(static)
    for (long long q = 0; q < (long long)n; ++q) {
      Pr[q] = dt * L[q];
      Q[q] = Pr[q];
      y[q] = y[q] + 0.5 * Pr[q];
    }
  } else if (stage == 2) {
    // stage 2: P = L(y); y = E(y + (P-Q)/2); Q = Q * (1/6)
#pragma omp parallel for schedule(static)
    for (long long q = 0; q < (long long)n; ++q) {
      Pr[q] = dt * L[q];
      y[q] = y[q] + 0.5 * (Pr[q] - Q[q]);
      Q[q] = Q[q] * SIXTH;
    }
  } else if (stage == 3) {
    // stage 3: P = L(y) - P/2; y = E(y + P); Q = Q - P
#pragma omp parallel for schedule(static)
    for (long long q = 0; q < (long long)n; ++q) {
      Pr[q] = dt * L[q] - 0.5 * Pr[q];
      y[q] = y[q] + Pr[q];
      Q[q] = Q[q] - Pr[q];
    }
  } else {
    // stage 4: P = L(y) + 2P; y = E(y + (Q + P * (1/6)))
#pragma omp parallel for schedule(static)
    for (long long q = 0; q < (long long)n; ++q) {
      Pr[q] = dt * L[q] + 2.0 * Pr[q];
      y[q] = y[q] + (Q[q] + Pr[q] * SIXTH);
    }
  }
}

static int step_global(const Params& P, double* y, int nsteps, int do_enforce) {
  const size_t n = (size_t)NF * P.N[0] * P.N[1] * P.N[2];
  std::vector<double> Pr(n), Q(n), L(n);
  const double dt = P.cfl * P.dx;
  int bad = 0;
  for (int st = 0; st < nsteps; ++st)
    for (int stage = 1; stage <= 4; ++stage) {
      rhs_global(P, y, L.data());
      rk_stage_update(stage, n, dt, L.data(), y, Pr.data(), Q.data());
      bad |= enforce_global(P, y, do_enforce);
    }
  return bad;
}

// ---- NEXT-3: restriction / prolongation at a factor-2 refinement boundary (z4c_amr.hpp) -----------
// Restriction, step 1 of MeshBlock B's protocol ("Restrict the data in the active region to fill the
// coarse buffer"). fine: [nfields][Nf_z][Nf_y][Nf_x], the active cells of the fine region in global fine order,
// tiled by MeshBlocks of nf^3 cells; coarse: [nfields][Nf_z/2][Nf_y/2][Nf_x/2]. Eq. (2) with the outer product
// of the three 1-D weight sets, summed z-outermost, x-innermost.
static void restrict_region(int ng, int nf, const int32_t* Nf, const double* fine, double* coarse, int nfields) {
  const int n = ng + 1;
  const int Mc[3] = {Nf[0] / 2, Nf[1] / 2, Nf[2] / 2};
  const size_t nfc = (size_t)Nf[0] * Nf[1] * Nf[2], ncc = (size_t)Mc[0] * Mc[1] * Mc[2];
#pragma omp parallel for schedule(static)
  for (int K = 0; K < Mc[2]; ++K)
    for (int J = 0; J < Mc[1]; ++J)
      for (int I = 0; I < Mc[0]; ++I) {
        const int C[3] = {I, J, K};
        double w[3][8];
        int s[3], r[3];
        for (int a = 0; a < 3; ++a) {
          const int blk = (2 * C[a]) / nf;                 // the fine MeshBlock that owns the children
          const int Il = C[a] - blk * (nf / 2);            // coarse index local to that block
          s[a] = blk * nf + restrict_weights(Il, n, nf, w[a]);
          r[a] = restrict_ref(Il, n, nf);
        }
        for (int f = 0; f < nfields; ++f) {
          const double* F = fine + (size_t)f * nfc;
          const double fr = F[((size_t)(s[2] + r[2]) * Nf[1] + (s[1] + r[1])) * Nf[0] + (s[0] + r[0])];
          double sum = 0.0;                                // R-I1: f_r + sum W (f - f_r)
          for (int c = 0; c < n; ++c)
            for (int b = 0; b < n; ++b)
              for (int a = 0; a < n; ++a)
                sum = sum + ((w[2][c] * w[1][b]) * w[0][a]) *
                                (F[((size_t)(s[2] + c) * Nf[1] + (s[1] + b)) * Nf[0] + (s[0] + a)] - fr);
          coarse[(size_t)f * ncc + ((size_t)K * Mc[1] + J) * Mc[0] + I] = fr + sum;
        }
      }
}

// Prolongation, step 5 ("Prolongate the coarse buffer to fill the fine ghost zones"): the value at the
// fine node (i, j, k) -- fine indices relative to the corner of the fine region, any sign -- from the coarse level
// coarse[nfields][Nc_z][Nc_y][Nc_x] (global array, neighbours by wrap/clamp as in O2); the fine region's corner is
// the coarse cell `origin`.
static double prolong_point(int ng, const int32_t* Nc, int bc, const int32_t* origin, const double* coarse, int f,
                            int i, int j, int k) {
  const int n = ng + 1;
  const int q[3] = {i, j, k};
  double w[3][8];
  int s[3], r[3];
  for (int a = 0; a < 3; ++a) {
    s[a] = origin[a] + prolong_weights(q[a], n, w[a]);
    r[a] = prolong_ref(q[a], n);
  }
  const size_t ncc = (size_t)Nc[0] * Nc[1] * Nc[2];
  auto at = [&](int a, int b, int c) {
    const int ii = map_index(s[0] + a, Nc[0], bc), jj = map_index(s[1] + b, Nc[1], bc),
              kk = map_index(s[2] + c, Nc[2], bc);
    return coarse[(size_t)f * ncc + ((size_t)kk * Nc[1] + jj) * Nc[0] + ii];
  };
  const double fr = at(r[0], r[1], r[2]);
  double sum = 0.0;                                        // R-I1: f_r + sum W (f - f_r)
  for (int c = 0; c < n; ++c)
    for (int b = 0; b < n; ++b)
      for (int a = 0; a < n; ++a) sum = sum + ((w[2][c] * w[1][b]) * w[0][a]) * (at(a, b, c) - fr);
  return fr + sum;
}

// Two-level state helpers: covered coarse cells <- restriction of the fine level; padded fine array <- fine
// interior + ghost layers by prolongation (all faces, edges and corners of the fine region).
static void two_level_sync(const Params& Pc, const Params& Pf, int nf, const int32_t* origin, double* uc,
                           const double* uf, double* ufp) {
  const int g = Pf.ng;
  const int Mc[3] = {Pf.N[0] / 2, Pf.N[1] / 2, Pf.N[2] / 2};
  std::vector<double> R((size_t)NF * Mc[0] * Mc[1] * Mc[2]);
  restrict_region(g, nf, Pf.N, uf, R.data(), NF);
  const size_t ncc = (size_t)Pc.N[0] * Pc.N[1] * Pc.N[2], nrc = (size_t)Mc[0] * Mc[1] * Mc[2];
  for (int f = 0; f < NF; ++f)
    for (int K = 0; K < Mc[2]; ++K)
      for (int J = 0; J < Mc[1]; ++J)
        for (int I = 0; I < Mc[0]; ++I)
          uc[(size_t)f * ncc + ((size_t)(origin[2] + K) * Pc.N[1] + (origin[1] + J)) * Pc.N[0] + (origin[0] + I)] =
              R[(size_t)f * nrc + ((size_t)K * Mc[1] + J) * Mc[0] + I];
  const int mx = Pf.N[0] + 2 * g, my = Pf.N[1] + 2 * g, mz = Pf.N[2] + 2 * g;
  const size_t npf = (size_t)mx * my * mz, nif = (size_t)Pf.N[0] * Pf.N[1] * Pf.N[2];
#pragma omp parallel for schedule(static)
  for (int k = -g; k < Pf.N[2] + g; ++k)
    for (int j = -g; j < Pf.N[1] + g; ++j)
      for (int i = -g; i < Pf.N[0] + g; ++i) {
        const bool inside = i >= 0 && i < Pf.N[0] && j >= 0 && j < Pf.N[1] && k >= 0 && k < Pf.N[2];
        for (int f = 0; f < NF; ++f)
          ufp[(size_t)f * npf + ((size_t)(k + g) * my + (j + g)) * mx + (i + g)] =
              inside ? uf[(size_t)f * nif + ((size_t)k * Pf.N[1] + j) * Pf.N[0] + i]
                     : prolong_point(g, Pc.N, Pc.bc, origin, uc, f, i, j, k);
      }
}

// Two-level static refinement (the set-up of the test at PAPER.md:171): the coarse level covers the
// whole mesh, the fine level a box whose corner is the coarse cell `origin`; both advance with the same dt (no
// subcycling), and after every RK stage the protocol of section 3.1 runs: restrict the fine active region into the
// coarse nodes it covers (step B.1; those nodes are what the coarse neighbours receive, steps A.2 / B.2), then
// prolongate the coarse level into the fine ghost zones (step B.5). Returns 1 if a bad cell was seen, -1 if the two
// parameter sets do not describe one time step.
static int step_two_level(const Params& Pc, const Params& Pf, int nf, const int32_t* origin, double* uc, double* uf,
                          int nsteps) {
  const double dt = Pc.cfl * Pc.dx;
  if (std::fabs(dt - Pf.cfl * Pf.dx) > 1e-14 * dt || Pf.ng != Pc.ng) return -1;
  const int g = Pf.ng;
  const size_t ncn = (size_t)NF * Pc.N[0] * Pc.N[1] * Pc.N[2], nfn = (size_t)NF * Pf.N[0] * Pf.N[1] * Pf.N[2];
  const size_t npf = (size_t)NF * (Pf.N[0] + 2 * g) * (Pf.N[1] + 2 * g) * (Pf.N[2] + 2 * g);
  std::vector<double> Prc(ncn), Qc(ncn), Lc(ncn), Prf(nfn), Qf(nfn), Lf(nfn), ufp(npf);
  int bad = 0;
  two_level_sync(Pc, Pf, nf, origin, uc, uf, ufp.data());
  for (int st = 0; st < nsteps; ++st)
    for (int stage = 1; stage <= 4; ++stage) {
      rhs_global(Pc, uc, Lc.data());
      rhs_global(Pf, ufp.data(), Lf.data(), g);
      rk_stage_update(stage, ncn, dt, Lc.data(), uc, Prc.data(), Qc.data());
      bad |= enforce_global(Pc, uc, 1);
      rk_stage_update(stage, nfn, dt, Lf.data(), uf, Prf.data(), Qf.data());
      bad |= enforce_global(Pf, uf, 1);
      two_level_sync(Pc, Pf, nf, origin, uc, uf, ufp.data());
    }
  return bad;
}

// textbook 4-array RK4 without enforcement (pin P9: the recurrence equals this)
static void step_textbook(const Params& P, double* y, int nsteps) {
  const size_t n = (size_t)NF * P.N[0] * P.N[1] * P.N[2];
  std::vector<double> k1(n), k2(n), k3(n), k4(n), t(n);
  const double dt = P.cfl * P.dx;
  for (int st = 0; st < nsteps; ++st) {
    rhs_global(P, y, k1.data());
    for (size_t q = 0; q < n; ++q) t[q] = y[q] + 0.5 * dt * k1[q];
    rhs_global(P, t.data(), k2.data());
    for (size_t q = 0; q < n; ++q) t[q] = y[q] + 0.5 * dt * k2[q];
    rhs_global(P, t.data(), k3.data());
    for (size_t q = 0; q < n; ++q) t[q] = y[q] + dt * k3[q];
    rhs_global(P, t.data(), k4.data());
    for (size_t q = 0; q < n; ++q)
      y[q] = y[q] + dt / 6.0 * (k1[q] + 2.0 * k2[q] + 2.0 * k3[q] + k4[q]);
  }
}

}  // namespace oz4c

// =====================================================================================
// extern "C" surface (ctypes from tests/, bench.py cpu_baseline, smoke()).
// All arrays are host double[NF][Nz][Ny][Nx] (x fastest) unless stated.
// =====================================================================================
using namespace oz4c;

extern "C" {

int oz4c_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void oz4c_set_num_threads(int n) {
#ifdef _OPENMP
  omp_set_num_threads(n);
#else
  (void)n;
#endif
}

// rhs = F(u) + Q_KO(u) (not multiplied by dt)
void oz4c_rhs(const Params* P, const double* u, double* rhs) { rhs_global(*P, u, rhs); }

// O7 in place; returns 1 if a bad cell was seen
int oz4c_enforce(const Params* P, double* u) { return enforce_global(*P, u, 1); }

// O6; do_enforce=0 replaces E by the identity (pin P9). returns 1 if a bad cell was seen
int oz4c_step(const Params* P, double* u, int nsteps, int do_enforce) {
  return step_global(*P, u, nsteps, do_enforce);
}
void oz4c_step_textbook(const Params* P, double* u, int nsteps) { step_textbook(*P, u, nsteps); }

double oz4c_inv_cbrt(double x) { return inv_cbrt_spec(x); }

// NEXT-3. Eq. (1) weights; restriction / prolongation stencil positions and weights along one
// axis (readings Q21, Q22); the two operators on arrays; the two-level RK4 step.
void oz4c_lagrange_weights(int n, const double* xs, double x, double* w) { lagrange_weights(n, xs, x, w); }
int oz4c_restrict_weights(int Il, int ng, int nf, double* w) { return restrict_weights(Il, ng + 1, nf, w); }
int oz4c_prolong_weights(int i, int ng, double* w) { return prolong_weights(i, ng + 1, w); }
void oz4c_restrict(int ng, int nf, const int32_t* Nf, const double* fine, double* coarse, int nfields) {
  restrict_region(ng, nf, Nf, fine, coarse, nfields);
}
// out[nfields][hi2-lo2][hi1-lo1][hi0-lo0]: prolonged values on the fine index box [lo, hi) (relative to the region)
void oz4c_prolong(int ng, const int32_t* Nc, int bc, const int32_t* origin, const double* coarse, const int32_t* lo,
                  const int32_t* hi, double* out, int nfields) {
  const size_t nx = hi[0] - lo[0], ny = hi[1] - lo[1], nz = hi[2] - lo[2];
  for (int f = 0; f < nfields; ++f)
    for (int k = lo[2]; k < hi[2]; ++k)
      for (int j = lo[1]; j < hi[1]; ++j)
        for (int i = lo[0]; i < hi[0]; ++i)
          out[(size_t)f * nx * ny * nz + ((size_t)(k - lo[2]) * ny + (j - lo[1])) * nx + (i - lo[0])] =
              prolong_point(ng, Nc, bc, origin, coarse, f, i, j, k);
}
int oz4c_step_two_level(const Params* Pc, const Params* Pf, int nf, const int32_t* origin, double* uc, double* uf,
                        int nsteps) {
  return step_two_level(*Pc, *Pf, nf, origin, uc, uf, nsteps);
}

// S5: out = {H_rms,H_max,M_rms,M_max,Theta_rms,Theta_max,Z_rms,Z_max};
// percell nullable: [4][Nz][Ny][Nx] = H, Mx, My, Mz
void oz4c_constraints(const Params* P, const double* u, double* out, double* percell) {
  View V(*P, u);
  const size_t nc = V.ncell;
  double sH = 0, sM = 0, sT = 0, sZ = 0, mH = 0, mM = 0, mT = 0, mZ = 0;
  for (int k = 0; k < P->N[2]; ++k)
    for (int j = 0; j < P->N[1]; ++j)
      for (int i = 0; i < P->N[0]; ++i) {
        double uc[NF], c6[6];
        Derivs<double> D;
        gather<double>(V, i, j, k, true, uc, D);
        double dA[3][6];
        for (int a = 0; a < 3; ++a)
          for (int p = 0; p < 6; ++p) dA[a][p] = D.d1[AXX + p][a];
        constraints_point<double>(uc, D, dA, c6);
        const size_t c = ((size_t)k * P->N[1] + j) * P->N[0] + i;
        if (percell) for (int q = 0; q < 4; ++q) percell[(size_t)q * nc + c] = c6[q];
        const double H = c6[0], M = std::sqrt(c6[4]), Z = std::sqrt(c6[5]), T = uc[THETA];
        sH += H * H; sM += c6[4]; sT += T * T; sZ += c6[5];
        mH = std::fmax(mH, std::fabs(H)); mM = std::fmax(mM, M);
        mT = std::fmax(mT, std::fabs(T)); mZ = std::fmax(mZ, Z);
      }
  out[0] = std::sqrt(sH / nc); out[1] = mH; out[2] = std::sqrt(sM / nc); out[3] = mM;
  out[4] = std::sqrt(sT / nc); out[5] = mT; out[6] = std::sqrt(sZ / nc); out[7] = mZ;
}

// NEXT-4 (sections 3.3.1-3.3.2): per-MeshBlock refinement indicators. Blocks of n^3 cells tile
// the global array (block id = (bz*nby + by)*nbx + bx). minchi[b] = min over the block of chi (chi-min criterion:
// refine if it falls below a threshold); maxdchi[b] = max over the block of |grad chi| (d-chi-max criterion: refine if it
// exceeds a threshold), with grad = the scheme's centred first derivative and |.| the Euclidean norm (reading Q20).
void oz4c_refine_indicators(const Params* P, const double* u, int n, double* minchi, double* maxdchi) {
  View V(*P, u);
  const int nbx = P->N[0] / n, nby = P->N[1] / n, nbz = P->N[2] / n;
  const bool o6 = sixth_order(*P);
  for (int bz = 0; bz < nbz; ++bz)
    for (int by = 0; by < nby; ++by)
      for (int bx = 0; bx < nbx; ++bx) {
        double mn = INFINITY, mx = 0.0;
        for (int k = bz * n; k < (bz + 1) * n; ++k)
          for (int j = by * n; j < (by + 1) * n; ++j)
            for (int i = bx * n; i < (bx + 1) * n; ++i) {
              const int c[3] = {i, j, k};
              double g2 = 0.0;
              for (int a = 0; a < 3; ++a) {
                double l[9];
                for (int s = -4; s <= 4; ++s) {
                  int q[3] = {c[0], c[1], c[2]};
                  q[a] += s;
                  l[s + 4] = V.at(CHI, q[0], q[1], q[2]);
                }
                const double d = o6 ? d1_centred6(&l[4], P->dx) : d1_centred(&l[4], P->dx);
                g2 += d * d;
              }
              mn = std::fmin(mn, V.at(CHI, i, j, k));
              mx = std::fmax(mx, std::sqrt(g2));
            }
        const int b = (bz * nby + by) * nbx + bx;
        minchi[b] = mn;
        maxdchi[b] = mx;
      }
}

// Pins P2: apply one stencil of O3 to a single scalar array f[Nz][Ny][Nx].
// kind: 0 centred-1st(axis a), 1 centred-2nd(axis a), 2 mixed(a,b), 3 upwind+ (a), 4 upwind- (a),
//       5 KO summed over the three axes including the eps/(64h) factor
void oz4c_stencil(const Params* P, const double* f, int kind, int a, int b, double* out) {
  Params P1 = *P;
  std::vector<double> tmp;  // View indexes field 0 only
  View V(P1, f);
  const double h = P->dx;
  for (int k = 0; k < P->N[2]; ++k)
    for (int j = 0; j < P->N[1]; ++j)
      for (int i = 0; i < P->N[0]; ++i) {
        const int c[3] = {i, j, k};
        const bool o6 = sixth_order(*P);
        auto line = [&](int ax, double* l) {
          for (int s = -4; s <= 4; ++s) {
            int q[3] = {c[0], c[1], c[2]};
            q[ax] += s;
            l[s + 4] = V.at(0, q[0], q[1], q[2]);
          }
        };
        double lbuf[9], r = 0.0;
        double* l = lbuf + 1;   // so that &l[3] is the centre in both layouts
        if (kind == 0) { line(a, lbuf); r = o6 ? d1_centred6(&l[3], h) : d1_centred(&l[3], h); }
        else if (kind == 1) { line(a, lbuf); r = o6 ? d2_centred6(&l[3], h) : d2_centred(&l[3], h); }
        else if (kind == 2) {
          auto v = [&](int sa, int sb) -> double {
            int q[3] = {c[0], c[1], c[2]};
            q[a] += sa; q[b] += sb;
            return V.at(0, q[0], q[1], q[2]);
          };
          r = o6 ? d2_mixed6<double>(v, h) : d2_mixed<double>(v, h);
        } else if (kind == 3 || kind == 4) {
          line(a, lbuf);
          r = o6 ? d1_upwind6(&l[3], h, kind == 3) : d1_upwind(&l[3], h, kind == 3);
        } else {
          for (int ax = 0; ax < 3; ++ax) { line(ax, lbuf); r += o6 ? ko_axis6(&l[3]) : ko_axis(&l[3]); }
          r *= P->ko_eps / ((o6 ? 256.0 : 64.0) * h);
        }
        out[((size_t)k * P->N[1] + j) * P->N[0] + i] = r;
      }
}

// Pins P3-P5: per-cell intermediates. out[NQ][Nz][Ny][Nx] with
// 0-5 R~_ij, 6-11 R^chi_ij, 12-17 D_iD_j alpha, 18 R, 19 AA, 20-22 Gd^k, 23-28 ginv
enum { NQ = 29 };
int oz4c_num_intermediates(void) { return NQ; }
void oz4c_intermediates(const Params* P, const double* u, double* out) {
  View V(*P, u);
  const size_t nc = V.ncell;
#pragma omp parallel for schedule(static)
  for (int k = 0; k < P->N[2]; ++k)
    for (int j = 0; j < P->N[1]; ++j)
      for (int i = 0; i < P->N[0]; ++i) {
        double uc[NF];
        Derivs<double> D;
        Geometry<double> G;
        gather<double>(V, i, j, k, false, uc, D);
        geometry<double>(uc, D, G);
        const size_t c = ((size_t)k * P->N[1] + j) * P->N[0] + i;
        for (int p = 0; p < 6; ++p) {
          out[(size_t)(0 + p) * nc + c] = G.Rt[p];
          out[(size_t)(6 + p) * nc + c] = G.Rchi[p];
          out[(size_t)(12 + p) * nc + c] = G.DDalpha[p];
          out[(size_t)(23 + p) * nc + c] = G.ginv[p];
        }
        out[(size_t)18 * nc + c] = G.Rscal;
        out[(size_t)19 * nc + c] = G.AA;
        for (int q = 0; q < 3; ++q) out[(size_t)(20 + q) * nc + c] = G.Gd[q];
      }
}

// Flop census at one cell (i,j,k) of u: counts[0..2] = add, mul, div for S2+S3 (one RHS
// evaluation, derivatives included), counts[3..5] likewise for S5.  Uses the operation
// counting scalar; FMA fusion is not assumed (a fused pair counts as 1 add + 1 mul).
void oz4c_count_flops(const Params* P, const double* u, int i, int j, int k, long long* counts) {
  View V(*P, u);
  {
    g_counts = {0, 0, 0};
    CScalar uc[NF], out[NF];
    Derivs<CScalar> D;
    gather<CScalar>(V, i, j, k, false, uc, D);
    rhs_point<CScalar>(*P, uc, D, out);
    counts[0] = g_counts.add; counts[1] = g_counts.mul; counts[2] = g_counts.div;
  }
  {
    g_counts = {0, 0, 0};
    CScalar uc[NF], c6[6];
    Derivs<CScalar> D;
    gather<CScalar>(V, i, j, k, true, uc, D);
    CScalar dA[3][6];
    for (int a = 0; a < 3; ++a)
      for (int p = 0; p < 6; ++p) dA[a][p] = D.d1[AXX + p][a];
    constraints_point<CScalar>(uc, D, dA, c6);
    counts[3] = g_counts.add; counts[4] = g_counts.mul; counts[5] = g_counts.div;
  }
}

}  // extern "C"
