// NEXT-3: restriction and prolongation at a factor-2 refinement boundary between two MeshBlockPacks (sm_100a).
// PAPER.md:69-118 (section 3.1): Lagrange interpolation, Eq. (1) at PAPER.md:104 (product over m != i), Eq. (2) at
// PAPER.md:108, outer product of the per-axis weights, n = N_g + 1 nodes per axis, the
// restriction stencil "always within the active region" of the fine MeshBlock, prolongation from the
// coarse buffer into the fine ghost nodes. Stencil positions: readings Q21 / Q22 of DESIGN.md.
//
// Geometry (cell-centred): along an axis the coarse node I sits midway between the fine nodes 2I and
// 2I+1; the fine node i = 2I + p (p = 0, 1) sits a quarter of a coarse cell below / above the coarse node I. All node
// distances are therefore multiples of a quarter cell, and every weight is a ratio of two small integers:
//   w_q = prod_{m != q} (4X - 4x_m) / prod_{m != q} (4x_q - 4x_m)      (X, x in the units of the source level)
// evaluated here in integer arithmetic with one exact division (the quotients are dyadic rationals for n <= 5).
//
// Floating-point form (reading R-I1): since the weights sum to one, Eq. (2) is evaluated as
//   f(x) = f_r + sum_{abc} ((l_z l_y) l_x) (f_abc - f_r),   r = the stencil node nearest the target,
// summed z outermost, x innermost, every product and sum rounded separately (no FMA contraction). On the nearly flat
// backgrounds of BASELINE's configs the differences are exact, so an interpolated chi or gt_ii is reproducible to the
// last bit -- an ulp there would be amplified by dt/h^2 into At_ij, as with the stencils (Q14) and the enforcement (R-E1).
#pragma once
#include <cuda_runtime.h>

#include "z4c_kernels.cuh"
#include "z4c_pack.cuh"

namespace z4c {

constexpr int AMR_N = NG + 1;   // nodes per axis

// weights of the nodes s, s+1, .., s+n-1 at the position X4/4 (all in the index units of the source level)
__host__ __device__ inline void lagrange_quarters(const int s, const int X4, double* w) {
  for (int q = 0; q < AMR_N; ++q) {
    long long num = 1, den = 1;
    for (int m = 0; m < AMR_N; ++m) {
      if (m == q) continue;
      num *= (long long)(X4 - 4 * (s + m));
      den *= (long long)(4 * (q - m));
    }
    w[q] = (double)num / (double)den;
  }
}

// The weights depend only on where the target sits relative to its stencil, which takes three values per axis for the
// restriction (stencil shifted up at the block's lower edge, centred, shifted down at its upper edge) and two for the
// prolongation (lower / upper child): the launcher evaluates the integer formula once on the host and hands the kernels
// the table (same expression, same exact dyadic doubles).
struct AmrWeights {
  double r[3][AMR_N];   // restriction: case 0 = first coarse cell of a fine block, 1 = regular, 2 = last
  double p[2][AMR_N];   // prolongation: child 0 / 1
};
inline AmrWeights make_amr_weights(const int nf) {
  AmrWeights t;
  const int half = nf / 2;
  const int Il[3] = {0, half > 2 ? 1 : 0, half - 1};
  for (int c = 0; c < 3; ++c) {
    int s = 2 * Il[c] + 1 - (AMR_N + 1) / 2;
    s = s < 0 ? 0 : (s > nf - AMR_N ? nf - AMR_N : s);
    lagrange_quarters(s, 8 * Il[c] + 2, t.r[c]);
  }
  for (int c = 0; c < 2; ++c) {
    const int s = (AMR_N % 2 == 0) ? -AMR_N / 2 + c : -(AMR_N - 1) / 2;
    lagrange_quarters(s, -1 + 2 * c, t.p[c]);
  }
  return t;
}

__device__ __forceinline__ int floor_half(const int i) { return i >= 0 ? i >> 1 : -((1 - i) >> 1); }

// Restriction stencil of the coarse node whose children are the LOCAL fine cells 2*Il, 2*Il+1 of a block with nf
// active cells: the n nearest fine nodes (tie towards the lower index), shifted into [0, nf). Returns the first node.
__device__ __forceinline__ int restrict_axis(const int Il, const int nf, const AmrWeights& t, double* w, int& ref) {
  const int s0 = 2 * Il + 1 - (AMR_N + 1) / 2;      // target 2 Il + 1/2
  const int s = max(0, min(s0, nf - AMR_N));
  const int c = s0 < 0 ? 0 : (s0 > nf - AMR_N ? 2 : 1);
#pragma unroll
  for (int q = 0; q < AMR_N; ++q) w[q] = c == 0 ? t.r[0][q] : (c == 1 ? t.r[1][q] : t.r[2][q]);
  ref = 2 * Il - s;                         // the lower child, as an index into the stencil
  return s;
}

// Prolongation stencil of the fine node i (relative to the corner of the fine region, any sign): the n nearest
// coarse nodes. Returns the first coarse node, relative to the region's corner cell.
__device__ __forceinline__ int prolong_axis(const int i, const AmrWeights& t, double* w, int& ref) {
  const int I = floor_half(i), p = i - 2 * I;
  const int s = (AMR_N % 2 == 0) ? I - AMR_N / 2 + p : I - (AMR_N - 1) / 2;   // target I - 1/4 + p/2
#pragma unroll
  for (int q = 0; q < AMR_N; ++q) w[q] = p ? t.p[1][q] : t.p[0][q];
  ref = I - s;                                  // the parent node, as an index into the stencil
  return s;
}

struct AmrGeom {
  int origin[3];   // coarse global cell index of the fine region's corner
  int Mc[3];       // coarse cells covered per axis = fine cells / 2
  int layer = -1;  // k_restrict: >= 0 = only the covered cells within `layer` cells of the region's faces (what the
                   // coarse neighbours and the prolongation read); -1 = every covered cell
};

// Step B.1: covered coarse interior cells <- restriction of the fine active cells, and steps A.2 / B.2
// for those cells: the thread also writes the ghost images of its coarse cell (same wrap / clamp rule as O2, the
// target list of the stage update's push), so the coarse level needs no whole-pack ghost fill after a restriction.
// One thread per (covered coarse cell, field).
// cells within a.layer of the region's faces (the launcher only sets a layer with 2 * layer <= every extent)
__host__ __device__ inline long long restrict_layer_cells(const AmrGeom& a) {
  const long long Mx = a.Mc[0], My = a.Mc[1], Mz = a.Mc[2], L2 = 2 * a.layer;
  return Mx * My * Mz - (Mx - L2) * (My - L2) * (Mz - L2);
}
constexpr int RB_X = 16, RB_Y = 4, RB_Z = 2;   // k_restrict's brick of coarse cells per CTA (128 threads)
__global__ void __launch_bounds__(RB_X * RB_Y * RB_Z) k_restrict(Pack gf, const double* __restrict__ yf, Pack gc,
                                                  double* __restrict__ yc, AmrGeom a, AmrWeights wt) {
  // a CTA takes a 16 x 4 x 2 brick of coarse cells of one field, so that the fine rows and planes its threads share
  // (half of each stencil overlaps the neighbour's) are found in this SM's L1
  const int bricks_x = (a.Mc[0] + RB_X - 1) / RB_X, bricks_y = (a.Mc[1] + RB_Y - 1) / RB_Y;
  const int f = blockIdx.y;
  const int bx = blockIdx.x % bricks_x, by = (blockIdx.x / bricks_x) % bricks_y, bz = blockIdx.x / (bricks_x * bricks_y);
  int C[3] = {bx * RB_X + (int)(threadIdx.x % RB_X), by * RB_Y + (int)((threadIdx.x / RB_X) % RB_Y),
              bz * RB_Z + (int)(threadIdx.x / (RB_X * RB_Y))};
  if (a.layer >= 0) {
    // only the `layer` cells under each face of the region, enumerated directly: z-slabs, y-slabs, x-slabs
    const int L2 = 2 * a.layer, Mx = a.Mc[0], My = a.Mc[1], Mz = a.Mc[2];
    const long long nZ = (long long)L2 * My * Mx, nY = (long long)(Mz - L2) * L2 * Mx;
    long long r = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (r >= restrict_layer_cells(a)) return;
    if (r < nZ) {
      const int zz = (int)(r / ((long long)My * Mx));
      C[0] = (int)(r % Mx); C[1] = (int)((r / Mx) % My); C[2] = zz < a.layer ? zz : Mz - L2 + zz;
    } else if (r < nZ + nY) {
      r -= nZ;
      const int q = (int)((r / Mx) % L2);
      C[0] = (int)(r % Mx); C[1] = q < a.layer ? q : My - L2 + q; C[2] = a.layer + (int)(r / ((long long)L2 * Mx));
    } else {
      r -= nZ + nY;
      const int q = (int)(r % L2);
      C[0] = q < a.layer ? q : Mx - L2 + q; C[1] = a.layer + (int)((r / L2) % (My - L2));
      C[2] = a.layer + (int)(r / ((long long)L2 * (My - L2)));
    }
  } else if (C[0] >= a.Mc[0] || C[1] >= a.Mc[1] || C[2] >= a.Mc[2]) {
    return;
  }
  double w[3][AMR_N];
  int s[3], fb[3], ref[3];
  const int half = gf.n / 2;
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    fb[d] = C[d] / half;                                               // fine block that owns the two children
    s[d] = restrict_axis(C[d] - fb[d] * half, gf.n, wt, w[d], ref[d]) + NG;   // padded index of the first stencil node
  }
  const double* src0 = yf + (((long long)fb[2] * gf.nb[1] + fb[1]) * gf.nb[0] + fb[0]) * gf.m3 +
                       ((long long)s[2] * gf.m + s[1]) * gf.m + s[0];
  const long long roff = ((long long)ref[2] * gf.m + ref[1]) * gf.m + ref[0];
  // destination: the coarse interior cell (origin + C) and its ghost images
  int cb[3], cl[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const int G = a.origin[d] + C[d];
    cb[d] = G / gc.n;
    cl[d] = G - cb[d] * gc.n + NG;
  }
  int tbx[NG + 1], tlx[NG + 1], tby[NG + 1], tly[NG + 1], tbz[NG + 1], tlz[NG + 1];
  const int cx = push_targets(cl[0] - NG, cb[0], gc.n, gc.nb[0], gc.bc, tbx, tlx);
  const int cy = push_targets(cl[1] - NG, cb[1], gc.n, gc.nb[1], gc.bc, tby, tly);
  const int cz = push_targets(cl[2] - NG, cb[2], gc.n, gc.nb[2], gc.bc, tbz, tlz);
  {
    const double* src = src0 + f * gf.fs;
    const double fr = __ldg(src + roff);
    double sum = 0.0;
#pragma unroll
    for (int kk = 0; kk < AMR_N; ++kk)
#pragma unroll
      for (int jj = 0; jj < AMR_N; ++jj) {
        const double* row = src + ((long long)kk * gf.m + jj) * gf.m;
        const double wzy = __dmul_rn(w[2][kk], w[1][jj]);
#pragma unroll
        for (int ii = 0; ii < AMR_N; ++ii)
          sum = __dadd_rn(sum, __dmul_rn(__dmul_rn(wzy, w[0][ii]), __dsub_rn(__ldg(row + ii), fr)));
      }
    const double sz = __dadd_rn(fr, sum);
    double* yf_c = yc + f * gc.fs;
#pragma unroll 1
    for (int q = 0; q < cz; ++q)       // target (0, 0, 0) is the cell itself
#pragma unroll 1
      for (int r = 0; r < cy; ++r)
#pragma unroll 1
        for (int p = 0; p < cx; ++p)
          yf_c[(((long long)tbz[q] * gc.nb[1] + tby[r]) * gc.nb[0] + tbx[p]) * gc.m3 +
               ((long long)tlz[q] * gc.m + tly[r]) * gc.m + tlx[p]] = sz;
  }
}

// Step B.5: every ghost cell of every fine block that lies OUTSIDE the fine region <- prolongation of
// the coarse level (its interior cells, reached by the same wrap / clamp rule as O2, so coarse ghosts need not be
// current). Ghost cells inside the region belong to the same-level exchange and are left alone.
// One thread per cell of the shell around the fine region (stencil, weights and targets once, then the 22 fields in
// turn): the shell -- the padded region minus the region,
// 2 N_g layers per axis -- is enumerated directly (z-slabs, then y-slabs, then x-slabs), the value is interpolated
// once and stored into every fine block whose padded box holds the cell (up to two per axis near block boundaries).
__device__ __forceinline__ int prolong_targets(const int c, const int n, const int nbl, int* tb, int* tl) {
  if (c < 0) { tb[0] = 0; tl[0] = c + NG; return 1; }
  if (c >= n * nbl) { tb[0] = nbl - 1; tl[0] = c - (nbl - 1) * n + NG; return 1; }
  const int b = c / n, l = c - b * n;
  int k = 0;
  tb[k] = b; tl[k] = l + NG; ++k;
  if (l < NG && b > 0) { tb[k] = b - 1; tl[k] = l + n + NG; ++k; }
  if (l >= n - NG && b < nbl - 1) { tb[k] = b + 1; tl[k] = l - n + NG; ++k; }
  return k;
}

__host__ __device__ inline long long prolong_shell_cells(const int n, const int* nb) {
  const long long Nx = (long long)n * nb[0], Ny = (long long)n * nb[1], Nz = (long long)n * nb[2];
  return (Nx + 2 * NG) * (Ny + 2 * NG) * (Nz + 2 * NG) - Nx * Ny * Nz;
}

__global__ void __launch_bounds__(128) k_prolong(Pack gc, const double* __restrict__ yc, Pack gf,
                                                 double* __restrict__ yf, AmrGeom a, AmrWeights wt) {
  const int n = gf.n;
  constexpr int G2 = 2 * NG;
  const int Nx = n * gf.nb[0], Ny = n * gf.nb[1], Nz = n * gf.nb[2];
  const int Mx = Nx + G2, My = Ny + G2;
  const long long nZ = (long long)G2 * My * Mx, nY = (long long)Nz * G2 * Mx, nX = (long long)Nz * Ny * G2;
  const long long cells = nZ + nY + nX;
  long long r = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (r >= cells) return;
  int gi[3];                                   // fine index relative to the region's corner, outside it on >= 1 axis
  if (r < nZ) {
    const int zz = (int)(r / ((long long)My * Mx));
    gi[0] = (int)(r % Mx) - NG; gi[1] = (int)((r / Mx) % My) - NG; gi[2] = zz < NG ? zz - NG : Nz + zz - NG;
  } else if (r < nZ + nY) {
    r -= nZ;
    const int q = (int)((r / Mx) % G2);
    gi[0] = (int)(r % Mx) - NG; gi[1] = q < NG ? q - NG : Ny + q - NG; gi[2] = (int)(r / ((long long)G2 * Mx));
  } else {
    r -= nZ + nY;
    const int q = (int)(r % G2);
    gi[0] = q < NG ? q - NG : Nx + q - NG; gi[1] = (int)((r / G2) % Ny); gi[2] = (int)(r / ((long long)G2 * Ny));
  }
  double w[3][AMR_N];
  int off[3][AMR_N];         // per axis: offset contribution of every stencil node inside one field of the coarse pack
                             // (32 bits: the launcher refuses a coarse field of 2^31 doubles or more)
  int ref[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const int s = a.origin[d] + prolong_axis(gi[d], wt, w[d], ref[d]);
    const int N = gc.n * gc.nb[d];
    const long long bstride = d == 0 ? gc.m3 : (d == 1 ? (long long)gc.nb[0] * gc.m3 : (long long)gc.nb[0] * gc.nb[1] * gc.m3);
    const long long lstride = d == 0 ? 1 : (d == 1 ? gc.m : gc.m2);
#pragma unroll
    for (int q = 0; q < AMR_N; ++q) {
      int G = s + q;
      if (gc.bc == 0) { G %= N; if (G < 0) G += N; } else { G = G < 0 ? 0 : (G >= N ? N - 1 : G); }
      const int cb = G / gc.n;
      off[d][q] = (int)(cb * bstride + (long long)(G - cb * gc.n + NG) * lstride);
    }
  }
  int roff = 0;
#pragma unroll
  for (int q = 0; q < AMR_N; ++q)          // ref[] is a run-time index: select instead of indexing the register array
    if (q == ref[2])
#pragma unroll
      for (int r2 = 0; r2 < AMR_N; ++r2)
        if (r2 == ref[1])
#pragma unroll
          for (int r1 = 0; r1 < AMR_N; ++r1)
            if (r1 == ref[0]) roff = off[2][q] + off[1][r2] + off[0][r1];
  int tbx[3], tlx[3], tby[3], tly[3], tbz[3], tlz[3];
  const int cx = prolong_targets(gi[0], n, gf.nb[0], tbx, tlx);
  const int cy = prolong_targets(gi[1], n, gf.nb[1], tby, tly);
  const int cz = prolong_targets(gi[2], n, gf.nb[2], tbz, tlz);
#pragma unroll 1
  for (int f = 0; f < NF; ++f) {
    const double* src = yc + f * gc.fs;
    const double fr = __ldg(src + roff);
    double sum = 0.0;
#pragma unroll
    for (int kk = 0; kk < AMR_N; ++kk)
#pragma unroll
      for (int jj = 0; jj < AMR_N; ++jj) {
        const double wzy = __dmul_rn(w[2][kk], w[1][jj]);
#pragma unroll
        for (int ii = 0; ii < AMR_N; ++ii)
          sum = __dadd_rn(sum, __dmul_rn(__dmul_rn(wzy, w[0][ii]),
                                         __dsub_rn(__ldg(src + off[2][kk] + off[1][jj] + off[0][ii]), fr)));
      }
    const double sz = __dadd_rn(fr, sum);
    double* dst = yf + f * gf.fs;
#pragma unroll 1
    for (int q = 0; q < cz; ++q)
#pragma unroll 1
      for (int r2 = 0; r2 < cy; ++r2)
#pragma unroll 1
        for (int p = 0; p < cx; ++p)
          dst[(((long long)tbz[q] * gf.nb[1] + tby[r2]) * gf.nb[0] + tbx[p]) * gf.m3 +
              ((long long)tlz[q] * gf.m + tly[r2]) * gf.m + tlx[p]] = sz;
  }
}

}  // namespace z4c
