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

// NEXT-2 (the exchange itself at PAPER.md:65, 75-76): the block lattice of the whole mesh is cut
// into slabs along z, one MeshBlockPack (one process, one GPU) per slab. A cell's ghost images then live either in
// this pack or in the pack of the slab below / above; the kernels that write (or read) ghost cells address the three
// packs through this table. Entry 0 is the pack itself; entries 1 / 2 are the lower / upper neighbour, whose buffers
// are mapped into this process (peer memory over NVLink). An unpartitioned pack is the one-entry case.
struct Slab {
  double* y[3];       // state buffer of each entry (the buffer being written -- or read, for the pull kernel)
  long long fs[3];    // field stride of each entry's pack
  int bz0[3], nbz[3]; // global z-range of the blocks of each entry (nbz = 0: absent)
  int nbz_global;     // blocks along z of the whole lattice
};
// which entry owns the global block coordinate bz (after wrap / clamp in the global lattice)
__host__ __device__ inline int slab_entry(const Slab& s, int bz) {
  if (bz >= s.bz0[0] && bz < s.bz0[0] + s.nbz[0]) return 0;
  if (bz >= s.bz0[1] && bz < s.bz0[1] + s.nbz[1]) return 1;
  return 2;
}
// entry lookups by selects: a run-time index into a kernel-parameter array would send the table to local memory
__host__ __device__ inline double* slab_y(const Slab& s, int e) { return e == 0 ? s.y[0] : (e == 1 ? s.y[1] : s.y[2]); }
__host__ __device__ inline long long slab_fs(const Slab& s, int e) { return e == 0 ? s.fs[0] : (e == 1 ? s.fs[1] : s.fs[2]); }
__host__ __device__ inline int slab_bz0(const Slab& s, int e) { return e == 0 ? s.bz0[0] : (e == 1 ? s.bz0[1] : s.bz0[2]); }

}  // namespace z4c
