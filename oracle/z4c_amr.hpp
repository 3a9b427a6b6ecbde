// =====================================================================================
// oracle/z4c_amr.hpp -- TEST INFRASTRUCTURE, NOT PRODUCT (see z4c_oracle.hpp).
//
// NEXT-3: the restriction and prolongation operators of a factor-2 refinement boundary for
// cell-centred finite differences (section 3.1), written out from the text:
//
//   Eq. (1), PAPER.md:104   l_i(x) = prod_{0<=m<=k, m != i} (x - x_m)/(x_i - x_m)
//                           (the paper's subscript reads "m != j"; with l_i on the left it must
//                            be m != i -- SURVEY.md Q17)
//   Eq. (2), PAPER.md:108   f(x) = sum_i l_i(x) f(x_i)
//   "generalized to two and three spatial dimensions by taking the outer-product between the
//    interpolation weights for each dimension"
//   stencil size n = N_g + 1 points per dimension
//   restriction: "the stencil is always within the active region" of the fine MeshBlock
//                (PAPER.md:114), hence lopsided next to a block face
//   prolongation: Lagrange interpolation from coarse-buffer nodes to the fine ghost nodes
//
//
// Geometry (cell-centred nodes). Along one axis, fine node i sits at (i + 1/2) h,
// coarse node I at (I + 1/2) 2h. In fine-index units the coarse node is at x = 2I + 1/2 (midway
// between fine nodes 2I and 2I+1); in coarse-index units fine node i = 2I + p (p = 0, 1) is at
// X = I - 1/4 + p/2.
//
// Readings (the paper fixes n and the "inside the active region" rule, not the stencil position):
//   Q21 restriction stencil = the n consecutive fine nodes nearest the coarse node, a tie (n odd)
//       resolved towards the lower index, then shifted by the least amount that puts it inside
//       the active region [0, nf) of the fine MeshBlock that owns fine cells 2I, 2I+1.
//   Q22 prolongation stencil = the n consecutive coarse nodes nearest the fine node (unique for
//       even n because the fine node is off-centre by 1/4; centred on the parent cell for odd n).
//   Q23 the 22 fields are interpolated as they are; the algebraic constraints are not re-imposed
//       on interpolated values (the paper does not mention it).
//   R-I1 floating-point form of Eq. (1)-(2). Because sum_i l_i = 1, Eq. (2) is evaluated as
//       f(x) = f_r + sum_i l_i (f(x_i) - f_r), r = the stencil node nearest the target (the lower child for
//       restriction, the parent node for prolongation): on a nearly flat background the differences are exact and
//       the rounding error is relative to the perturbation, not to the O(1) field -- the same reason as the
//       difference-from-centre stencils (Q14); an ulp of chi or gt_ii in a ghost node is otherwise amplified by
//       dt/h^2 into At_ij. Eq. (1) is evaluated as one product of numerators over one product of denominators (all
//       exact multiples of 1/4), so every weight is the exact dyadic rational. The 3-D weight is (l_z l_y) l_x and
//       the sum runs z outermost, x innermost, every operation rounded separately: oracle and GPU agree bit for bit.
// =====================================================================================
#pragma once
#include <cmath>

namespace oz4c {

// Eq. (1): weights of the n nodes xs[0..n) at the point x.
inline void lagrange_weights(int n, const double* xs, double x, double* w) {
  for (int i = 0; i < n; ++i) {
    double num = 1.0, den = 1.0;
    for (int m = 0; m < n; ++m) {
      if (m == i) continue;
      num = num * (x - xs[m]);
      den = den * (xs[i] - xs[m]);
    }
    w[i] = num / den;
  }
}

inline int floor_div2(int i) { return i >= 0 ? i / 2 : -((-i + 1) / 2); }

// Q21: first fine node (index local to the fine block, active cells [0, nf)) of the restriction stencil of the
// coarse node whose children are the local fine cells 2Il, 2Il+1.
inline int restrict_start(int Il, int n, int nf) {
  int s = 2 * Il + 1 - (n + 1) / 2;   // n even: 2Il + 1 - n/2 (symmetric); n odd: the extra node on the low side
  if (s < 0) s = 0;
  if (s > nf - n) s = nf - n;
  return s;
}
// restriction weights along one axis for local coarse index Il: nodes s..s+n-1, target x = 2 Il + 1/2
inline int restrict_weights(int Il, int n, int nf, double* w) {
  const int s = restrict_start(Il, n, nf);
  double xs[8];
  for (int q = 0; q < n; ++q) xs[q] = (double)(s + q);
  lagrange_weights(n, xs, 2.0 * Il + 0.5, w);
  return s;
}

// R-I1 reference node, as an index into the stencil: the lower child 2 Il (restriction), the parent I (prolongation)
inline int restrict_ref(int Il, int n, int nf) { return 2 * Il - restrict_start(Il, n, nf); }

// Q22: first coarse node of the prolongation stencil of fine node i (any sign), and its weights.
inline int prolong_weights(int i, int n, double* w) {
  const int I = floor_div2(i);
  const int p = i - 2 * I;            // 0: the fine node lies at I - 1/4, 1: at I + 1/4
  int s;
  if (n % 2 == 0) s = I - n / 2 + p;  // even n: {I-n/2 .. I+n/2-1} for p = 0, shifted up by one for p = 1
  else s = I - (n - 1) / 2;           // odd n: centred on the parent cell
  double xs[8];
  for (int q = 0; q < n; ++q) xs[q] = (double)(s + q);
  lagrange_weights(n, xs, (double)I - 0.25 + 0.5 * p, w);
  return s;
}
inline int prolong_ref(int i, int n) {
  const int I = floor_div2(i);
  const int p = i - 2 * I;
  return (n % 2 == 0) ? n / 2 - p : (n - 1) / 2;
}

}  // namespace oz4c
