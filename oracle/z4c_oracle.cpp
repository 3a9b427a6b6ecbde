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
  const double* u;       // [NF][Nz][Ny][Nx]
  size_t ncell;
  View(const Params& p, const double* uu) : P(p), u(uu),
      ncell((size_t)p.N[0] * p.N[1] * p.N[2]) {}
  inline double at(int f, int i, int j, int k) const {
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
    T line[3][9];
    for (int a = 0; a < 3; ++a)
      for (int s = -4; s <= 4; ++s) {
        int q[3] = {c[0], c[1], c[2]};
        q[a] += s;
        line[a][s + 4] = T(V.at(f, q[0], q[1], q[2]));
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
static void rhs_global(const Params& P, const double* u, double* rhs) {
  View V(P, u);
  const size_t nc = V.ncell;
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
static int step_global(const Params& P, double* y, int nsteps, int do_enforce) {
  const size_t n = (size_t)NF * P.N[0] * P.N[1] * P.N[2];
  std::vector<double> Pr(n), Q(n), L(n);
  const double dt = P.cfl * P.dx;
  int bad = 0;
  for (int st = 0; st < nsteps; ++st) {
    // stage 1: P = L(y); Q = P; y = E(y + P/2)
    rhs_global(P, y, L.data());
#pragma omp parallel for schedule(static)
    for (long long q = 0; q < (long long)n; ++q) {
      Pr[q] = dt * L[q];
      Q[q] = Pr[q];
      y[q] = y[q] + 0.5 * Pr[q];
    }
    bad |= enforce_global(P, y, do_enforce);
    // stage 2: P = L(y); y = E(y + (P-Q)/2); Q = Q/6
    rhs_global(P, y, L.data());
#pragma omp parallel for schedule(static)
    for (long long q = 0; q < (long long)n; ++q) {
      Pr[q] = dt * L[q];
      y[q] = y[q] + 0.5 * (Pr[q] - Q[q]);
      Q[q] = Q[q] / 6.0;
    }
    bad |= enforce_global(P, y, do_enforce);
    // stage 3: P = L(y) - P/2; y = E(y + P); Q = Q - P
    rhs_global(P, y, L.data());
#pragma omp parallel for schedule(static)
    for (long long q = 0; q < (long long)n; ++q) {
      Pr[q] = dt * L[q] - 0.5 * Pr[q];
      y[q] = y[q] + Pr[q];
      Q[q] = Q[q] - Pr[q];
    }
    bad |= enforce_global(P, y, do_enforce);
    // stage 4: P = L(y) + 2P; y = E(y + (Q + P/6))
    rhs_global(P, y, L.data());
#pragma omp parallel for schedule(static)
    for (long long q = 0; q < (long long)n; ++q) {
      Pr[q] = dt * L[q] + 2.0 * Pr[q];
      y[q] = y[q] + (Q[q] + Pr[q] / 6.0);
    }
    bad |= enforce_global(P, y, do_enforce);
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
