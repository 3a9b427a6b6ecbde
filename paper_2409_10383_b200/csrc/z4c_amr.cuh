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

#include "z4c_pack.cuh"

namespace z4c {

constexpr int AMR_N = NG + 1;   // nodes per axis

// weights of the nodes s, s+1, .., s+n-1 at the position X4/4 (all in the index units of the source level)
__device__ __forceinline__ void lagrange_quarters(const int s, const int X4, double* w) {
#pragma unroll
  for (int q = 0; q < AMR_N; ++q) {
    long long num = 1, den = 1;
#pragma unroll
    for (int m = 0; m < AMR_N; ++m) {
      if (m == q) continue;
      num *= (long long)(X4 - 4 * (s + m));
      den *= (long long)(4 * (q - m));
    }
    w[q] = (double)num / (double)den;
  }
}

__device__ __forceinline__ int floor_half(const int i) { return i >= 0 ? i >> 1 : -((1 - i) >> 1); }

// Restriction stencil of the coarse node whose children are the LOCAL fine cells 2*Il, 2*Il+1 of a block with nf
// active cells: the n nearest fine nodes (tie towards the lower index), shifted into [0, nf). Returns the first node.
__device__ __forceinline__ int restrict_axis(const int Il, const int nf, double* w, int& ref) {
  int s = 2 * Il + 1 - (AMR_N + 1) / 2;
  s = max(0, min(s, nf - AMR_N));
  lagrange_quarters(s, 8 * Il + 2, w);      // target 2 Il + 1/2
  ref = 2 * Il - s;                         // the lower child, as an index into the stencil
  return s;
}

// Prolongation stencil of the fine node i (relative to the corner of the fine region, any sign): the n nearest
// coarse nodes. Returns the first coarse node, relative to the region's corner cell.
__device__ __forceinline__ int prolong_axis(const int i, double* w, int& ref) {
  const int I = floor_half(i), p = i - 2 * I;
  const int s = (AMR_N % 2 == 0) ? I - AMR_N / 2 + p : I - (AMR_N - 1) / 2;
  lagrange_quarters(s, 4 * I - 1 + 2 * p, w);   // target I - 1/4 + p/2
  ref = I - s;                                  // the parent node, as an index into the stencil
  return s;
}

struct AmrGeom {
  int origin[3];   // coarse global cell index of the fine region's corner
  int Mc[3];       // coarse cells covered per axis = fine cells / 2
};

// Step B.1: covered coarse interior cells <- restriction of the fine active cells.
// One thread per (covered coarse cell, field).
__global__ void __launch_bounds__(128) k_restrict(Pack gf, const double* __restrict__ yf, Pack gc,
                                                  double* __restrict__ yc, AmrGeom a) {
  const long long ncov = (long long)a.Mc[0] * a.Mc[1] * a.Mc[2];
  const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (t >= ncov * NF) return;
  const int f = (int)(t / ncov);
  const long long c = t - f * ncov;
  const int C[3] = {(int)(c % a.Mc[0]), (int)((c / a.Mc[0]) % a.Mc[1]), (int)(c / ((long long)a.Mc[0] * a.Mc[1]))};
  double w[3][AMR_N];
  int s[3], fb[3], ref[3];
  const int half = gf.n / 2;
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    fb[d] = C[d] / half;                                               // fine block that owns the two children
    s[d] = restrict_axis(C[d] - fb[d] * half, gf.n, w[d], ref[d]) + NG;   // padded index of the first stencil node
  }
  const double* src = yf + f * gf.fs + (((long long)fb[2] * gf.nb[1] + fb[1]) * gf.nb[0] + fb[0]) * gf.m3 +
                      ((long long)s[2] * gf.m + s[1]) * gf.m + s[0];
  const double fr = __ldg(src + ((long long)ref[2] * gf.m + ref[1]) * gf.m + ref[0]);
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
  // destination: the coarse interior cell (origin + C)
  int cb[3], cl[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const int G = a.origin[d] + C[d];
    cb[d] = G / gc.n;
    cl[d] = G - cb[d] * gc.n + NG;
  }
  yc[f * gc.fs + (((long long)cb[2] * gc.nb[1] + cb[1]) * gc.nb[0] + cb[0]) * gc.m3 +
     ((long long)cl[2] * gc.m + cl[1]) * gc.m + cl[0]] = sz;
}

// Step B.5: every ghost cell of every fine block that lies OUTSIDE the fine region <- prolongation of
// the coarse level (its interior cells, reached by the same wrap / clamp rule as O2, so coarse ghosts need not be
// current). Ghost cells inside the region belong to the same-level exchange and are left alone.
// One thread per (field, block, ghost cell): consecutive threads take consecutive ghost cells of one field.
__global__ void __launch_bounds__(128) k_prolong(Pack gc, const double* __restrict__ yc, Pack gf,
                                                 double* __restrict__ yf, AmrGeom a) {
  const int n = gf.n, m = gf.m;
  constexpr int G2 = 2 * NG;
  const int nZ = G2 * m * m, nY = G2 * n * m, nX = G2 * n * n;
  const int per_block = nZ + nY + nX;
  const long long cells = (long long)per_block * gf.nblk;
  const long long tt = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (tt >= cells * NF) return;
  const int f = (int)(tt / cells);
  const long long t = tt - f * cells;
  const int b = (int)(t / per_block);
  int r = (int)(t - (long long)b * per_block);
  int l[3];
  if (r < nZ) {
    l[0] = r % m; l[1] = (r / m) % m; l[2] = (r / (m * m) < NG) ? r / (m * m) : n + r / (m * m);
  } else if (r < nZ + nY) {
    r -= nZ;
    const int q = (r / m) % G2;
    l[0] = r % m; l[1] = q < NG ? q : n + q; l[2] = NG + r / (G2 * m);
  } else {
    r -= nZ + nY;
    const int q = r % G2;
    l[0] = q < NG ? q : n + q; l[1] = NG + (r / G2) % n; l[2] = NG + r / (G2 * n);
  }
  int bc3[3];
  block_coords(gf, b, bc3[0], bc3[1], bc3[2]);
  int gi[3];
  bool outside = false;
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    gi[d] = bc3[d] * n + l[d] - NG;                       // fine index relative to the region's corner
    outside |= gi[d] < 0 || gi[d] >= n * gf.nb[d];
  }
  if (!outside) return;
  double w[3][AMR_N];
  long long off[3][AMR_N];   // per axis: offset contribution of every stencil node inside the coarse pack
  int ref[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const int s = a.origin[d] + prolong_axis(gi[d], w[d], ref[d]);
    const int N = gc.n * gc.nb[d];
    const long long bstride = d == 0 ? gc.m3 : (d == 1 ? (long long)gc.nb[0] * gc.m3 : (long long)gc.nb[0] * gc.nb[1] * gc.m3);
    const long long lstride = d == 0 ? 1 : (d == 1 ? gc.m : gc.m2);
#pragma unroll
    for (int q = 0; q < AMR_N; ++q) {
      int G = s + q;
      if (gc.bc == 0) { G %= N; if (G < 0) G += N; } else { G = G < 0 ? 0 : (G >= N ? N - 1 : G); }
      const int cb = G / gc.n;
      off[d][q] = cb * bstride + (long long)(G - cb * gc.n + NG) * lstride;
    }
  }
  const double* src = yc + f * gc.fs;
  double fr = 0.0;
#pragma unroll
  for (int q = 0; q < AMR_N; ++q)          // ref[] is a run-time index: select instead of indexing the register array
    if (q == ref[2])
#pragma unroll
      for (int r2 = 0; r2 < AMR_N; ++r2)
        if (r2 == ref[1])
#pragma unroll
          for (int r1 = 0; r1 < AMR_N; ++r1)
            if (r1 == ref[0]) fr = __ldg(src + off[2][q] + off[1][r2] + off[0][r1]);
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
  yf[f * gf.fs + (long long)b * gf.m3 + ((long long)l[2] * m + l[1]) * m + l[0]] = sz;
}

}  // namespace z4c
