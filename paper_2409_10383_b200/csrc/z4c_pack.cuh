// Geometry of the MeshBlockPack in HBM (D3 of SURVEY.md section 2.1) and the index maps
// every kernel uses.  State y: double[22][N_b][m][m][m] (x fastest, ghosts included);
// RK registers P, Q: double[22][N_b][n][n][n] (interior cells only).
#pragma once
#include <cstddef>
#include <cstdint>

#include "z4c_math.cuh"

namespace z4c {

struct Pack {
  int n, m;            // interior / padded cells per block edge (m = n + 2*NG)
  int nb[3];           // block lattice
  int nblk;            // N_b
  int bc;              // 0 periodic, 1 outflow-copy
  int m2;              // m*m
  int n3;              // n^3
  int m3;              // m^3
  long long fs;        // field stride of y   = N_b * m^3
  long long is;        // field stride of P,Q = N_b * n^3
  long long ncell;     // N_b * n^3
};

__host__ __device__ inline void block_coords(const Pack& g, int b, int& bx, int& by, int& bz) {
  bx = b % g.nb[0];
  by = (b / g.nb[0]) % g.nb[1];
  bz = b / (g.nb[0] * g.nb[1]);
}

// O2 (periodic PAPER.md:162): local index l in [0,m) of block coordinate bc_ along an
// axis with nbl blocks -> (source block coordinate, source local index) of the interior cell with the same
// global index after periodic wrap or outflow clamp.
__host__ __device__ inline void ghost_source(int l, int bcoord, int n, int nbl, int bc, int& sb, int& sl) {
  int G = bcoord * n + l - NG;
  const int N = n * nbl;
  if (bc == 0) {
    G %= N;
    if (G < 0) G += N;
  } else {
    G = G < 0 ? 0 : (G >= N ? N - 1 : G);
  }
  sb = G / n;
  sl = G - sb * n + NG;
}

}  // namespace z4c
