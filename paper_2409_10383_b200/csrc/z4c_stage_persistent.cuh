// One RK stage as ONE PERSISTENT kernel (sm_100a): S2 + S3 + S4 + S1 of SURVEY.md 8(a) for a stream of tiles.
//
// Same arithmetic as k_rhs_tiled<Cfg, STAGE> (z4c_rhs_tiled.cuh), different scheduling. The grid is at most
// 2 CTAs per SM; each CTA walks the tiles t = blockIdx.x, blockIdx.x + gridDim.x, ...  The TMA ring is never
// drained between tiles: halo-tile loads are issued in one global order m = 22*(tile ordinal) + field ordinal, the
// load for m + NSTAGE goes out as soon as every thread is done with m, so the shift tiles of the NEXT tile land
// while the current tile is still in its tensor algebra and write-out. The per-CTA prologue (first-tile latency),
// 10 % of the stall samples of the non-persistent kernel (profiles/r01_fused_stage_kernel_ncu.md), disappears
// except for the first tile of each CTA. The RK registers are read straight from global memory in the epilogue
// (22 independent coalesced loads per register, lines requested into L2 by a prefetch at the top of the tile).
//
// STATUS (round 1): correct (same parity tests as the default kernel) but SLOWER -- 0.240 ms per launch at 64^3
// against 0.185 ms for k_rhs_tiled<TileCfg<16,4,2,3,2>, STAGE> (bench.py --variant 3 vs 0). ncu: the first-tile wait
// is gone as intended (stall samples spread evenly over the instruction stream), but the tile loop's carried state
// pushes ptxas into 208-552 B of spills inside the stencil/algebra body, which costs more than the prologue saved.
// Kept as variant 3 for the next round (candidate fix: split the tile loop body so that ptxas sees the same
// live ranges as in the non-persistent kernel).
#pragma once
#include "z4c_rhs_tiled.cuh"

namespace z4c {

template <int TX_, int TY_, int TZ_, int NSTAGE_>
struct PersistCfg {
  static constexpr int TX = TX_, TY = TY_, TZ = TZ_, NSTAGE = NSTAGE_;
  static constexpr int THREADS = TX * TY * TZ;
  static constexpr int HX = TX + 2 * NG, HY = TY + 2 * NG, HZ = TZ + 2 * NG;
  static constexpr int SY = HX, SZ = HX * HY;
  static constexpr int TILE_BYTES = HX * HY * HZ * 8;
  static constexpr int STAGE_BYTES = (TILE_BYTES + 127) / 128 * 128;
  static constexpr int BAR_OFF = NSTAGE * STAGE_BYTES;
  static constexpr int A_OFF = BAR_OFF + 128;                 // advection + KO sums [22][THREADS]; later the new tile
  static constexpr int B_OFF = A_OFF + NF * THREADS * 8;      // late-use derivatives parked across geometry()
  static constexpr int LIST_OFF = B_OFF + NPARK * THREADS * 8;
  static constexpr int MAXLIST = 32;
  static constexpr int SMEM_BYTES = LIST_OFF + 9 * MAXLIST * 4 + 16;
  static constexpr bool EARLY_PARK = false;                   // (members field_from_tile looks at)
  static constexpr int S_OFF = A_OFF, E_OFF = B_OFF;
  static_assert(NSTAGE >= 3, "the three shift components are staged together");
};

// tile ordinal -> (halo origin in padded coordinates, block)
struct TileAt { int cx, cy, cz, b; };
template <class Cfg>
__device__ __forceinline__ TileAt tile_at(int t, int tiles_x, int tiles_y, int tiles_z) {
  TileAt a;
  a.cx = (t % tiles_x) * Cfg::TX; t /= tiles_x;
  a.cy = (t % tiles_y) * Cfg::TY; t /= tiles_y;
  a.cz = (t % tiles_z) * Cfg::TZ; t /= tiles_z;
  a.b = t;
  return a;
}

// Field loop of one tile. n0 = global iteration index of this tile's first field (runtime: the ring slot of field
// IT is (n0 + IT) % NSTAGE). After field IT is consumed by every thread, thread 0 issues load n0 + IT + NSTAGE,
// which belongs to this tile or to the CTA's next one.
template <class Cfg, int IT>
struct PersistLoop {
  __device__ __forceinline__ static void run(const CUtensorMap* map, unsigned char* ring, uint64_t* full,
                                             const unsigned n0, const int toff, const TileAt cur, const TileAt nxt,
                                             const bool has_next, const bool active, const double* bw,
                                             const double* aw, const FdConst& fd, const SrcParams& sp, double* u,
                                             Derivs& D, double* park) {
    constexpr int F = stream_field(IT);
    const unsigned n = n0 + IT;
    const unsigned slot = n % Cfg::NSTAGE;
    if (IT >= 3) mbar_wait(&full[slot], (n / Cfg::NSTAGE) & 1);   // the three shift tiles were waited for up front
    const double* t = reinterpret_cast<const double*>(ring + slot * Cfg::STAGE_BYTES) + toff;
    if (active) field_from_tile<Cfg, F>(t, bw, aw, fd, sp, u, D, park);
    __syncthreads();   // every thread is done reading this slot
    if (threadIdx.x == 0) {
      constexpr int ITN = IT + Cfg::NSTAGE;   // same slot, NSTAGE fields later
      if (ITN < NF) {
        mbar_expect_tx(&full[slot], Cfg::TILE_BYTES);
        tma_load_5d(ring + slot * Cfg::STAGE_BYTES, map, &full[slot], cur.cx, cur.cy, cur.cz, cur.b, stream_field(ITN));
      } else if (has_next) {
        mbar_expect_tx(&full[slot], Cfg::TILE_BYTES);
        tma_load_5d(ring + slot * Cfg::STAGE_BYTES, map, &full[slot], nxt.cx, nxt.cy, nxt.cz, nxt.b,
                    stream_field(ITN - NF));
      }
    }
    PersistLoop<Cfg, IT + 1>::run(map, ring, full, n0, toff, cur, nxt, has_next, active, bw, aw, fd, sp, u, D, park);
  }
};
template <class Cfg>
struct PersistLoop<Cfg, NF> {
  __device__ __forceinline__ static void run(const CUtensorMap*, unsigned char*, uint64_t*, unsigned, int, TileAt,
                                             TileAt, bool, bool, const double*, const double*, const FdConst&,
                                             const SrcParams&, double*, Derivs&, double*) {}
};

template <class Cfg, int STAGE>
__global__ void __launch_bounds__(Cfg::THREADS, 2)
    k_stage_persistent(const __grid_constant__ CUtensorMap map, Pack g, double* __restrict__ Preg, FdConst fd,
                       SrcParams sp, double dt, int tiles_x, int tiles_y, int tiles_z, int ntiles, StageArgs sa) {
  static_assert(STAGE >= 1 && STAGE <= 4, "RK stage");
  extern __shared__ __align__(128) unsigned char smem[];
  unsigned char* ring = smem;
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + Cfg::BAR_OFF);
  double* sA = reinterpret_cast<double*>(smem + Cfg::A_OFF);
  double* sB = reinterpret_cast<double*>(smem + Cfg::B_OFF);
  int* lists = reinterpret_cast<int*>(smem + Cfg::LIST_OFF);
  const int tid = threadIdx.x;
  const int lx = tid % Cfg::TX, ly = (tid / Cfg::TX) % Cfg::TY, lz = tid / (Cfg::TX * Cfg::TY);
  const int toff = (lz + NG) * Cfg::SZ + (ly + NG) * Cfg::SY + lx + NG;

  int tile = blockIdx.x;
  if (tile >= ntiles) return;
  const TileAt first = tile_at<Cfg>(tile, tiles_x, tiles_y, tiles_z);
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < Cfg::NSTAGE; ++s) mbar_init(&full[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < Cfg::NSTAGE; ++s) {
      mbar_expect_tx(&full[s], Cfg::TILE_BYTES);
      tma_load_5d(ring + s * Cfg::STAGE_BYTES, &map, &full[s], first.cx, first.cy, first.cz, first.b, stream_field(s));
    }
  }
  // centre values of gt_ij of the first tile, kept in the (idle) parking area so that they cost no registers
  // across the tile loop; later tiles: fetched during the previous tile's write-out
  {
    const int i = first.cx + lx, j = first.cy + ly, k = first.cz + lz;
    const bool act = i < g.n && j < g.n && k < g.n;
    const double* yc = sa.y_in + (long long)first.b * g.m3 + ((long long)(k + NG) * g.m + (j + NG)) * g.m + (i + NG);
#pragma unroll
    for (int p = 0; p < 6; ++p)
      sB[p * Cfg::THREADS + tid] = act ? __ldg(yc + (GXX + p) * g.fs) : (p == 0 || p == 3 || p == 5 ? 1.0 : 0.0);
  }

  unsigned n0 = 0;
  for (;; n0 += NF) {
    const int next_tile = tile + (int)gridDim.x;
    const bool has_next = next_tile < ntiles;
    const TileAt cur = tile_at<Cfg>(tile, tiles_x, tiles_y, tiles_z);
    const TileAt nxt = tile_at<Cfg>(has_next ? next_tile : tile, tiles_x, tiles_y, tiles_z);
    const int i = cur.cx + lx, j = cur.cy + ly, k = cur.cz + lz;
    const bool active = i < g.n && j < g.n && k < g.n;
    const long long ci = (long long)cur.b * g.n3 + ((long long)k * g.n + j) * g.n + i;

    if (tid == 0) {
      // push lists (O2) of this tile: per axis every (source cell -> destination block, padded index) pair
      int bxyz[3];
      block_coords(g, cur.b, bxyz[0], bxyz[1], bxyz[2]);
      const int c0[3] = {cur.cx, cur.cy, cur.cz}, T[3] = {Cfg::TX, Cfg::TY, Cfg::TZ};
      for (int a = 0; a < 3; ++a) {
        int* L = lists + a * 3 * Cfg::MAXLIST;
        int cnt = 0;
        for (int l = c0[a]; l < c0[a] + T[a] && l < g.n; ++l) {
          int tb[NG + 1], tl[NG + 1];
          const int nt = push_targets(l, bxyz[a], g.n, g.nb[a], g.bc, tb, tl);
          for (int q = 0; q < nt; ++q) {
            L[cnt] = l - c0[a]; L[Cfg::MAXLIST + cnt] = tb[q]; L[2 * Cfg::MAXLIST + cnt] = tl[q];
            ++cnt;
          }
        }
        lists[9 * Cfg::MAXLIST + a] = cnt;
      }
    }
    if (STAGE >= 2 && active && lx == 0) {
      // ask L2 for this tile's rows of the RK registers (one 128-byte line per row and field)
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        asm volatile("prefetch.global.L2 [%0];" ::"l"(sa.Q + ci + f * g.is));
        if (STAGE >= 3) asm volatile("prefetch.global.L2 [%0];" ::"l"(Preg + ci + f * g.is));
      }
    }

    double u[NF];
    Derivs D;
    {
      double gc[6];
#pragma unroll
      for (int p = 0; p < 6; ++p) gc[p] = sB[p * Cfg::THREADS + tid];
      derivs_begin(gc, D);
    }
    double bw[3], aw[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const unsigned n = n0 + a;
      mbar_wait(&full[n % Cfg::NSTAGE], (n / Cfg::NSTAGE) & 1);
      const double beta = reinterpret_cast<const double*>(ring + (n % Cfg::NSTAGE) * Cfg::STAGE_BYTES)[toff];
      bw[a] = beta * (0.5 * fd.inv12h);
      aw[a] = fabs(beta) * (0.5 * fd.inv12h) + fd.ko;
    }
    double* park = sA + tid;
    PersistLoop<Cfg, 0>::run(&map, ring, full, n0, toff, cur, nxt, has_next, active, bw, aw, fd, sp, u, D, park);

    double out[NF];
    if (active) {
#pragma unroll
      for (int f = 0; f < NF; ++f) out[f] = 0.0;
      Geom G;
      double* slot = sB + tid;
      park_late_derivs<true>(D, slot, Cfg::THREADS);
      asm volatile("" ::: "memory");
      geometry(u, D, G);
      asm volatile("" ::: "memory");
      park_late_derivs<false>(D, slot, Cfg::THREADS);
      z4c_sources_post(sp, u, D, G, out);
      double* pc = Preg + ci;
      double* qc = sa.Q + ci;
      // all loads of the RK registers first, as one batch of independent requests (stores to Q/P below may alias
      // them as far as the compiler knows, which would otherwise serialise load -> use -> store -> load ...)
      double Pold[NF], Qold[NF];
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        Qold[f] = STAGE >= 2 ? __ldcg(qc + f * g.is) : 0.0;
        Pold[f] = STAGE >= 3 ? __ldcg(pc + f * g.is) : 0.0;
      }
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        const double L = dt * (out[f] + park[f * Cfg::THREADS]);
        if (STAGE == 1) {
          qc[f * g.is] = L;
          u[f] = u[f] + 0.5 * L;
        } else if (STAGE == 2) {
          const double Q = Qold[f];
          pc[f * g.is] = L;
          u[f] = u[f] + 0.5 * (L - Q);
          qc[f * g.is] = Q / 6.0;
        } else if (STAGE == 3) {
          const double P = -0.5 * Pold[f] + L;
          const double Q = Qold[f];
          pc[f * g.is] = P;
          u[f] = u[f] + P;
          qc[f * g.is] = Q - P;
        } else {
          const double P = 2.0 * Pold[f] + L;
          const double Q = Qold[f];
          u[f] = u[f] + (Q + P / 6.0);
        }
      }
      bool bad = enforce_cell(u, sa.chi_floor);
      bad |= any_nonfinite(u);
      if (bad) *sa.flag = 1;
      // stage the new tile (each thread overwrites only its own slots of the advection/KO area)
#pragma unroll
      for (int f = 0; f < NF; ++f) sA[f * Cfg::THREADS + tid] = u[f];
    }
    // centre values of gt_ij for the CTA's next tile: in flight during the write-out
    double gc[6];
    if (has_next) {
      const int in = nxt.cx + lx, jn = nxt.cy + ly, kn = nxt.cz + lz;
      const bool actn = in < g.n && jn < g.n && kn < g.n;
      const double* yc = sa.y_in + (long long)nxt.b * g.m3 + ((long long)(kn + NG) * g.m + (jn + NG)) * g.m + (in + NG);
#pragma unroll
      for (int p = 0; p < 6; ++p) gc[p] = actn ? __ldg(yc + (GXX + p) * g.fs) : (p == 0 || p == 3 || p == 5 ? 1.0 : 0.0);
    }
    __syncthreads();
    {
      // cooperative write-out of the tile and all of its ghost images, x fastest: coalesced rows
      const int* Lx = lists;
      const int* Ly = lists + 3 * Cfg::MAXLIST;
      const int* Lz = lists + 6 * Cfg::MAXLIST;
      const int ncx = lists[9 * Cfg::MAXLIST], ncy = lists[9 * Cfg::MAXLIST + 1], ncz = lists[9 * Cfg::MAXLIST + 2];
      const int total = ncx * ncy * ncz;
      const float rcx = 1.0f / (float)ncx, rcy = 1.0f / (float)ncy;   // exact reciprocal decode, see z4c_rhs_tiled.cuh
      for (int q = tid; q < total; q += Cfg::THREADS) {
        const int r = (int)(((float)q + 0.5f) * rcx), qx = q - r * ncx;
        const int qz = (int)(((float)r + 0.5f) * rcy), qy = r - qz * ncy;
        const int src = (Lz[qz] * Cfg::TY + Ly[qy]) * Cfg::TX + Lx[qx];
        const long long tb =
            ((long long)Lz[Cfg::MAXLIST + qz] * g.nb[1] + Ly[Cfg::MAXLIST + qy]) * g.nb[0] + Lx[Cfg::MAXLIST + qx];
        double* d = sa.y_out + tb * g.m3 +
                    ((long long)Lz[2 * Cfg::MAXLIST + qz] * g.m + Ly[2 * Cfg::MAXLIST + qy]) * g.m + Lx[2 * Cfg::MAXLIST + qx];
#pragma unroll
        for (int f = 0; f < NF; ++f) d[f * g.fs] = sA[f * Cfg::THREADS + src];
      }
    }
    if (!has_next) break;
#pragma unroll
    for (int p = 0; p < 6; ++p) sB[p * Cfg::THREADS + tid] = gc[p];
    __syncthreads();   // lists and the staged tile are free for the next tile
    tile = next_tile;
  }
}

#if Z4C_NG == 3
using StageTile = PersistCfg<16, 4, 2, 4>;
#else
using StageTile = PersistCfg<16, 4, 2, 3>;   // (1 CTA per SM at this halo size; experimental variant)
#endif

template <class Cfg, int STAGE>
inline cudaError_t launch_stage_persistent_t(const CUtensorMap& map, const Pack& g, double* P, const FdConst& fd,
                                             const SrcParams& sp, double dt, cudaStream_t st, const StageArgs& sa,
                                             int num_sms) {
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(k_stage_persistent<Cfg, STAGE>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         Cfg::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    // two CTAs of 111 KB each must be resident per SM: ask for the largest shared-memory carve-out
    e = cudaFuncSetAttribute(k_stage_persistent<Cfg, STAGE>, cudaFuncAttributePreferredSharedMemoryCarveout,
                             cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  const int tx = (g.n + Cfg::TX - 1) / Cfg::TX, ty = (g.n + Cfg::TY - 1) / Cfg::TY, tz = (g.n + Cfg::TZ - 1) / Cfg::TZ;
  const long long ntiles = (long long)tx * ty * tz * g.nblk;
  if (ntiles > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
  const long long grid = ntiles < 2LL * num_sms ? ntiles : 2LL * num_sms;
  k_stage_persistent<Cfg, STAGE><<<(unsigned)grid, Cfg::THREADS, Cfg::SMEM_BYTES, st>>>(map, g, P, fd, sp, dt, tx, ty,
                                                                                        tz, (int)ntiles, sa);
  return cudaSuccess;
}

}  // namespace z4c
