// Kernels of the Z4c hot path (sm_100a): K1 ghost fill, K2 RHS, K3 RK4 stage update + enforcement,
// K4 constraint monitors, plus the layout kernels behind z4c_set_initial_data / z4c_get_interior.
// Citations: SURVEY.md section 8(a) S1-S5 / section 8(c) O2-O7 (restated in DESIGN.md).
#pragma once
#include <cuda_runtime.h>

#include "z4c_pack.cuh"
#include "z4c_rhs.cuh"

namespace z4c {

// ---------------------------------------------------------------------------------------------
// Layout kernels: interior array [F][Nz][Ny][Nx] (global, block-free) <-> pack.
// One thread per (field, global cell); x fastest on both sides so runs of n doubles coalesce.
// ---------------------------------------------------------------------------------------------
// dir 0: interior array -> y ; dir 1: y -> interior array ; dir 2: register (P layout) -> interior array
template <int DIR>
__global__ void __launch_bounds__(256) k_layout(Pack g, double* __restrict__ pack, double* __restrict__ glob,
                                                int nfields) {
  const long long Nx = (long long)g.n * g.nb[0], Ny = (long long)g.n * g.nb[1], Nz = (long long)g.n * g.nb[2];
  const long long ncell = Nx * Ny * Nz;
  const long long total = ncell * nfields;
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total;
       t += (long long)gridDim.x * blockDim.x) {
    const int f = (int)(t / ncell);
    const long long c = t - f * ncell;
    const int gx = (int)(c % Nx), gy = (int)((c / Nx) % Ny), gz = (int)(c / (Nx * Ny));
    const int bx = gx / g.n, by = gy / g.n, bz = gz / g.n;
    const int i = gx - bx * g.n, j = gy - by * g.n, k = gz - bz * g.n;
    const long long b = ((long long)bz * g.nb[1] + by) * g.nb[0] + bx;
    if (DIR == 2) {
      glob[t] = pack[f * g.is + b * g.n3 + ((long long)k * g.n + j) * g.n + i];
    } else {
      const long long q = f * g.fs + b * g.m3 + ((long long)(k + NG) * g.m + (j + NG)) * g.m + (i + NG);
      if (DIR == 0) pack[q] = glob[t]; else glob[t] = pack[q];
    }
  }
}

// ---------------------------------------------------------------------------------------------
// K1 same-level ghost fill (S1). One thread per (ghost cell, block); it moves all 22 fields of that
// cell (22 independent 8-byte copies in flight). Ghost cells are enumerated shell by shell so no thread
// is idle: z-slabs (2 NG m^2 cells), y-slabs (2 NG n m), x-slabs (2 NG n^2).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ int ghost_coord(int q, int n) { return q < NG ? q : n + q; }  // q in [0, 2 NG)

__global__ void __launch_bounds__(256) k_ghost_fill(Pack g, double* __restrict__ y, Slab sl) {
  const int n = g.n, m = g.m;
  constexpr int G2 = 2 * NG;
  const int nZ = G2 * m * m, nY = G2 * n * m, nX = G2 * n * n;
  const int per_block = nZ + nY + nX;
  const long long total = (long long)per_block * g.nblk;
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total;
       t += (long long)gridDim.x * blockDim.x) {
    const int b = (int)(t / per_block);
    int r = (int)(t - (long long)b * per_block);
    int i, j, k;
    if (r < nZ) {
      i = r % m; j = (r / m) % m; k = ghost_coord(r / (m * m), n);
    } else if (r < nZ + nY) {
      r -= nZ;
      i = r % m; j = ghost_coord((r / m) % G2, n); k = NG + r / (G2 * m);
    } else {
      r -= nZ + nY;
      i = ghost_coord(r % G2, n); j = NG + (r / G2) % n; k = NG + r / (G2 * n);
    }
    int bx, by, bz;
    block_coords(g, b, bx, by, bz);
    int sbx, sby, sbz, si, sj, sk;
    ghost_source(i, bx, n, g.nb[0], g.bc, sbx, si);
    ghost_source(j, by, n, g.nb[1], g.bc, sby, sj);
    ghost_source(k, sl.bz0[0] + bz, n, sl.nbz_global, g.bc, sbz, sk);   // z in the lattice of the whole mesh
    const int e = slab_entry(sl, sbz);                                   // the pack that holds the source block
    const long long sb = ((long long)(sbz - slab_bz0(sl, e)) * g.nb[1] + sby) * g.nb[0] + sbx;
    const long long src = sb * g.m3 + ((long long)sk * m + sj) * m + si;
    const long long dst = (long long)b * g.m3 + ((long long)k * m + j) * m + i;
    const double* ys = slab_y(sl, e);
    const long long sfs = slab_fs(sl, e);
    double v[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) v[f] = ys[f * sfs + src];
#pragma unroll
    for (int f = 0; f < NF; ++f) y[f * g.fs + dst] = v[f];
  }
}

// ---------------------------------------------------------------------------------------------
// S2 derivative gather straight from global memory (L1/L2 serve the stencil reuse).
// yc points at the cell in field 0. Produces the centre values, the centred derivatives, and
// out[f] = c_adv(f) * beta^k D^{+-}_k u_f + Q_KO u_f.
// ---------------------------------------------------------------------------------------------
template <bool ALL_D1, int F>
__device__ __forceinline__ void gather_fields(const double* __restrict__ yc, const long long fs, const int* st,
                                              const FdConst& fd, const SrcParams& P, const double* ab,
                                              const bool* pos, const double* u, Derivs& D, double* out) {
  if constexpr (F < NF) {
    const double* p = yc + F * fs;
    double adv = 0.0, ko = 0.0, d2[6];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      AxisRaw r;
      if (need_d2(F)) r = axis_raw<true, true>(p, st[a], u[F], pos[a]);
      else if (need_d1(F) || ALL_D1) r = axis_raw<true, false>(p, st[a], u[F], pos[a]);
      else r = axis_raw<false, false>(p, st[a], u[F], pos[a]);
      if (need_d1(F) || ALL_D1) D.d1[F][a] = r.d1 * fd.inv12h;
      if (need_d2(F)) d2[sym(a, a)] = r.d2 * fd.inv12h2;
      adv += ab[a] * r.up;
      ko += r.ko;
    }
    const double cadv = (F == ALPHA) ? P.lapse_advect : (F >= BETAX ? P.shift_advect : 1.0);
    out[F] = cadv * (adv * fd.inv12h) + ko * fd.ko;
    if (need_d2(F)) {
      d2[sym(0, 1)] = mixed_raw(p, st[0], st[1]) * fd.inv144h2;
      d2[sym(0, 2)] = mixed_raw(p, st[0], st[2]) * fd.inv144h2;
      d2[sym(1, 2)] = mixed_raw(p, st[1], st[2]) * fd.inv144h2;
      consume_d2<F>(d2, D);
    }
    gather_fields<ALL_D1, F + 1>(yc, fs, st, fd, P, ab, pos, u, D, out);
  }
}

template <bool ALL_D1>
__device__ __forceinline__ void gather_global(const double* __restrict__ yc, const long long fs, const int sy,
                                              const int sz, const FdConst& fd, const SrcParams& P, double* u,
                                              Derivs& D, double* out) {
#pragma unroll
  for (int f = 0; f < NF; ++f) u[f] = __ldg(yc + f * fs);
  double ab[3];
  bool pos[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    ab[a] = fabs(u[BETAX + a]);
    pos[a] = u[BETAX + a] >= 0.0;
  }
  const int st[3] = {1, sy, sz};
  derivs_begin(u + GXX, D);
  gather_fields<ALL_D1, 0>(yc, fs, st, fd, P, ab, pos, u, D, out);
}

// ---------------------------------------------------------------------------------------------
// K2, plain variant: one thread per interior cell, tile TX x TY x TZ per CTA.
//   P <- c*P + dt*(F(y) + Q_KO(y))       (c = 0 at stages 1-2: P is not read)
// ---------------------------------------------------------------------------------------------
constexpr int K2_TX = 16, K2_TY = 4, K2_TZ = 2;

__global__ void __launch_bounds__(K2_TX* K2_TY* K2_TZ)
    k_rhs_global(Pack g, const double* __restrict__ y, double* __restrict__ Preg, FdConst fd, SrcParams sp,
                 double c, double dt, int tiles_x, int tiles_y, int tiles_z) {
  int t = blockIdx.x;
  const int tx = t % tiles_x; t /= tiles_x;
  const int ty = t % tiles_y; t /= tiles_y;
  const int tz = t % tiles_z; t /= tiles_z;
  const int b = t;
  const int i = tx * K2_TX + threadIdx.x, j = ty * K2_TY + threadIdx.y, k = tz * K2_TZ + threadIdx.z;
  if (i >= g.n || j >= g.n || k >= g.n) return;
  const double* yc = y + (long long)b * g.m3 + ((long long)(k + NG) * g.m + (j + NG)) * g.m + (i + NG);
  double u[NF], out[NF];
  Derivs D;
  gather_global<false>(yc, g.fs, g.m, g.m2, fd, sp, u, D, out);
  z4c_sources(sp, u, D, out);
  double* pc = Preg + (long long)b * g.n3 + ((long long)k * g.n + j) * g.n + i;
  if (c != 0.0) {
#pragma unroll
    for (int f = 0; f < NF; ++f) pc[f * g.is] = c * pc[f * g.is] + dt * out[f];
  } else {
#pragma unroll
    for (int f = 0; f < NF; ++f) pc[f * g.is] = dt * out[f];
  }
}

// ---------------------------------------------------------------------------------------------
// O7 enforcement of one cell, in place (u = 22 values). det and the rescale follow a fixed sequence of
// separately rounded IEEE operations (reading R-E1) so that gt_ij is reproducible bit for bit.
// Returns true if det <= 0 or a non-finite value was seen (cell then left as is).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double det3_spec(const double* g) {
  const double a = __dsub_rn(__dmul_rn(g[3], g[5]), __dmul_rn(g[4], g[4]));
  const double b = __dsub_rn(__dmul_rn(g[1], g[5]), __dmul_rn(g[4], g[2]));
  const double c = __dsub_rn(__dmul_rn(g[1], g[4]), __dmul_rn(g[3], g[2]));
  return __dadd_rn(__dsub_rn(__dmul_rn(g[0], a), __dmul_rn(g[1], b)), __dmul_rn(g[2], c));
}

__device__ __forceinline__ bool enforce_cell(double* u, const double chi_floor) {
  double* g = u + GXX;
  double* A = u + AXX;
  const double det = det3_spec(g);
  if (!(det > 0.0) || isinf(det)) return true;
  const double s = inv_cbrt_spec(det);
#pragma unroll
  for (int p = 0; p < 6; ++p) g[p] = __dmul_rn(s, g[p]);
  double gi[6];
  inv3(g, gi);
  const double t = contract(gi, A);
  const double third = 1.0 / 3.0;
#pragma unroll
  for (int p = 0; p < 6; ++p) A[p] = A[p] - third * (g[p] * t);
  if (!isfinite(u[CHI])) return true;
  if (u[CHI] < chi_floor) u[CHI] = chi_floor;
  return false;
}

__device__ __forceinline__ bool any_nonfinite(const double* u) {
  bool bad = false;
#pragma unroll
  for (int f = 0; f < NF; ++f) bad |= !isfinite(u[f]);
  return bad;
}

// ---------------------------------------------------------------------------------------------
// The two factors 1/6 of the recurrence: a product with the correctly rounded double 1/6 (reading O6 as amended in
// round 2), product and sum rounded separately, as in the oracle.
__device__ constexpr double SIXTH = 1.0 / 6.0;

// K3: RK4 stage update in the 3-register recurrence (O6) + enforcement (O7), interior cells.
//   stage 1: Q = P;  y = E(y + P/2)
//   stage 2: y = E(y + (P - Q)/2);  Q = Q * (1/6)
//   stage 3: y = E(y + P);  Q = Q - P
//   stage 4: y = E(y + (Q + P * (1/6)))
//   stage 0: y = E(y)                               (z4c_enforce / z4c_set_initial_data)
// One thread per cell; every access is a run of n consecutive doubles per (j,k) row.
// ---------------------------------------------------------------------------------------------
// PUSH = true fuses K1 into K3 ("ghost push"): besides its own cell the thread writes every ghost image of
// that cell (same global index after wrap / clamp, O2) in the neighbouring blocks, so no separate ghost-fill
// pass has to re-read the state. Each padded cell has exactly one writer, hence no race and no atomics.
__device__ __forceinline__ int push_targets(int l, int bcoord, int n, int nbl, int bc, int* tb, int* tl) {
  int c = 0;
  tb[c] = bcoord; tl[c] = l + NG; ++c;
  if (bc == 0) {
    if (l < NG) { tb[c] = bcoord == 0 ? nbl - 1 : bcoord - 1; tl[c] = l + n + NG; ++c; }
    else if (l >= n - NG) { tb[c] = bcoord + 1 == nbl ? 0 : bcoord + 1; tl[c] = l - n + NG; ++c; }
  } else {
    if (l < NG) {
      if (bcoord > 0) { tb[c] = bcoord - 1; tl[c] = l + n + NG; ++c; }
      else if (l == 0) { for (int q = 0; q < NG; ++q) { tb[c] = bcoord; tl[c] = q; ++c; } }
    } else if (l >= n - NG) {
      if (bcoord < nbl - 1) { tb[c] = bcoord + 1; tl[c] = l - n + NG; ++c; }
      else if (l == n - 1) { for (int q = 0; q < NG; ++q) { tb[c] = bcoord; tl[c] = n + NG + q; ++c; } }
    }
  }
  return c;
}

template <int STAGE, bool PUSH>
__global__ void __launch_bounds__(128) k_stage_update(Pack g, double* __restrict__ y, const double* __restrict__ Preg,
                                                      double* __restrict__ Qreg, double chi_floor,
                                                      int* __restrict__ flag, Slab sl) {
  const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (t >= g.ncell) return;
  const int b = (int)(t / g.n3);
  const int r = (int)(t - (long long)b * g.n3);
  const int i = r % g.n, j = (r / g.n) % g.n, k = r / (g.n * g.n);
  double* yc = y + (long long)b * g.m3 + ((long long)(k + NG) * g.m + (j + NG)) * g.m + (i + NG);
  double u[NF];
#pragma unroll
  for (int f = 0; f < NF; ++f) u[f] = yc[f * g.fs];
  if (STAGE != 0) {
    const double* pc = Preg + t;
    double* qc = Qreg + t;
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const double P = pc[f * g.is];
      if (STAGE == 1) {
        qc[f * g.is] = P;
        u[f] = u[f] + 0.5 * P;
      } else if (STAGE == 2) {
        const double Q = qc[f * g.is];
        u[f] = u[f] + 0.5 * (P - Q);
        qc[f * g.is] = __dmul_rn(Q, SIXTH);
      } else if (STAGE == 3) {
        const double Q = qc[f * g.is];
        u[f] = u[f] + P;
        qc[f * g.is] = Q - P;
      } else {
        const double Q = qc[f * g.is];
        u[f] = u[f] + __dadd_rn(Q, __dmul_rn(P, SIXTH));
      }
    }
  }
  bool bad = enforce_cell(u, chi_floor);
  bad |= any_nonfinite(u);
  if (bad) *flag = 1;
#pragma unroll
  for (int f = 0; f < NF; ++f) yc[f * g.fs] = u[f];
  if (PUSH) {
    const bool edge = i < NG || i >= g.n - NG || j < NG || j >= g.n - NG || k < NG || k >= g.n - NG;
    if (edge) {
      int bx, by, bz;
      block_coords(g, b, bx, by, bz);
      int tbx[NG + 1], tlx[NG + 1], tby[NG + 1], tly[NG + 1], tbz[NG + 1], tlz[NG + 1];
      const int cx = push_targets(i, bx, g.n, g.nb[0], g.bc, tbx, tlx);
      const int cy = push_targets(j, by, g.n, g.nb[1], g.bc, tby, tly);
      const int cz = push_targets(k, sl.bz0[0] + bz, g.n, sl.nbz_global, g.bc, tbz, tlz);   // global z lattice
#pragma unroll 1
      for (int a = 0; a < cz; ++a) {
        const int e = slab_entry(sl, tbz[a]);                      // the pack that holds the target block (NEXT-2)
        double* ye = slab_y(sl, e);
        const long long efs = slab_fs(sl, e);
#pragma unroll 1
        for (int bb = 0; bb < cy; ++bb)
#pragma unroll 1
          for (int cc = 0; cc < cx; ++cc) {
            if (a + bb + cc == 0) continue;  // the cell itself, already written
            const long long tb = ((long long)(tbz[a] - slab_bz0(sl, e)) * g.nb[1] + tby[bb]) * g.nb[0] + tbx[cc];
            double* d = ye + tb * g.m3 + ((long long)tlz[a] * g.m + tly[bb]) * g.m + tlx[cc];
#pragma unroll
            for (int f = 0; f < NF; ++f) d[f * efs] = u[f];
          }
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// K4: constraint monitors (S5). Grid-stride over interior cells with a FIXED grid, per-CTA partials in
// fixed order, then a one-CTA second pass: bitwise reproducible. partial[cta][8] =
// {sum H^2, max|H|, sum |M|^2, max |M|, sum Theta^2, max|Theta|, sum |Z|^2, max |Z|}.
// ---------------------------------------------------------------------------------------------
constexpr int K4_THREADS = 128;

__device__ __forceinline__ void block_reduce8(double* v, double* smem /* [8][K4_THREADS/32] */) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
  for (int q = 0; q < 8; ++q) {
    double x = v[q];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const double other = __shfl_down_sync(0xffffffffu, x, o);
      x = (q & 1) ? fmax(x, other) : x + other;
    }
    if (lane == 0) smem[q * (K4_THREADS / 32) + w] = x;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      double x = smem[q * (K4_THREADS / 32)];
      for (int ww = 1; ww < K4_THREADS / 32; ++ww) {
        const double other = smem[q * (K4_THREADS / 32) + ww];
        x = (q & 1) ? fmax(x, other) : x + other;
      }
      v[q] = x;
    }
  }
}

__global__ void __launch_bounds__(K4_THREADS)
    k_constraints(Pack g, const double* __restrict__ y, FdConst fd, SrcParams sp, double* __restrict__ partial,
                  double* __restrict__ percell) {
  __shared__ double red[8 * (K4_THREADS / 32)];
  double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  const long long Nx = (long long)g.n * g.nb[0], Ny = (long long)g.n * g.nb[1];
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < g.ncell;
       t += (long long)gridDim.x * blockDim.x) {
    const int b = (int)(t / g.n3);
    const int r = (int)(t - (long long)b * g.n3);
    const int i = r % g.n, j = (r / g.n) % g.n, k = r / (g.n * g.n);
    const double* yc = y + (long long)b * g.m3 + ((long long)(k + NG) * g.m + (j + NG)) * g.m + (i + NG);
    double u[NF], out[NF], c[6];
    Derivs D;
    gather_global<false>(yc, g.fs, g.m, g.m2, fd, sp, u, D, out);
    const int st[3] = {1, g.m, g.m2};
    z4c_constraints_point(u, D, [&](const int a, double* q) {
#pragma unroll
      for (int p = 0; p < 6; ++p) q[p] = d1_raw(yc + (AXX + p) * g.fs, st[a]) * fd.inv12h;
    }, c);
    if (percell) {
      int bx, by, bz;
      block_coords(g, b, bx, by, bz);
      const long long cell = ((long long)(bz * g.n + k) * Ny + (by * g.n + j)) * Nx + (bx * g.n + i);
#pragma unroll
      for (int q = 0; q < 4; ++q) percell[q * g.ncell + cell] = c[q];
    }
    acc[0] += c[0] * c[0];          acc[1] = fmax(acc[1], fabs(c[0]));
    acc[2] += c[4];                 acc[3] = fmax(acc[3], sqrt(c[4]));
    acc[4] += u[THETA] * u[THETA];  acc[5] = fmax(acc[5], fabs(u[THETA]));
    acc[6] += c[5];                 acc[7] = fmax(acc[7], sqrt(c[5]));
  }
  block_reduce8(acc, red);
  if (threadIdx.x == 0) {
#pragma unroll
    for (int q = 0; q < 8; ++q) partial[(long long)blockIdx.x * 8 + q] = acc[q];
  }
}

// ---------------------------------------------------------------------------------------------
// NEXT-4: per-MeshBlock refinement indicators: min chi and max |grad chi| over the interior
// cells of each block, and the two flags (bit 0: min chi < chi_min, bit 1: max |grad chi| > dchi_max). One CTA per
// block; min/max reductions are exact in any order, so the result is deterministic.
// ---------------------------------------------------------------------------------------------
constexpr int KR_THREADS = 256;
__global__ void __launch_bounds__(KR_THREADS)
    k_refine_indicators(Pack g, const double* __restrict__ y, FdConst fd, double chi_min, double dchi_max,
                        double* __restrict__ minchi, double* __restrict__ maxdchi, int* __restrict__ flags) {
  __shared__ double smn[KR_THREADS / 32], smx[KR_THREADS / 32];
  const int b = blockIdx.x;
  const double* chi = y + (long long)CHI * g.fs + (long long)b * g.m3;
  double mn = INFINITY, mx = 0.0;
  for (int r = threadIdx.x; r < g.n3; r += KR_THREADS) {
    const int i = r % g.n, j = (r / g.n) % g.n, k = r / (g.n * g.n);
    const double* p = chi + ((long long)(k + NG) * g.m + (j + NG)) * g.m + (i + NG);
    const double dx = d1_raw(p, 1) * fd.inv12h, dy = d1_raw(p, g.m) * fd.inv12h, dz = d1_raw(p, g.m2) * fd.inv12h;
    mn = fmin(mn, __ldg(p));
    mx = fmax(mx, sqrt(dx * dx + dy * dy + dz * dz));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    mn = fmin(mn, __shfl_down_sync(0xffffffffu, mn, o));
    mx = fmax(mx, __shfl_down_sync(0xffffffffu, mx, o));
  }
  if ((threadIdx.x & 31) == 0) { smn[threadIdx.x >> 5] = mn; smx[threadIdx.x >> 5] = mx; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < KR_THREADS / 32; ++w) { mn = fmin(mn, smn[w]); mx = fmax(mx, smx[w]); }
    if (minchi) minchi[b] = mn;
    if (maxdchi) maxdchi[b] = mx;
    if (flags) flags[b] = (mn < chi_min ? 1 : 0) | (mx > dchi_max ? 2 : 0);
  }
}

// second pass: one CTA, fixed order. out[8] = {H_rms,H_max,M_rms,M_max,Theta_rms,Theta_max,Z_rms,Z_max};
// ncell < 0: the sums of squares are left as they are (a slab's share of a partitioned mesh, NEXT-2)
__global__ void __launch_bounds__(K4_THREADS)
    k_constraints_final(const double* __restrict__ partial, int nparts, double ncell, double* __restrict__ out) {
  __shared__ double red[8 * (K4_THREADS / 32)];
  double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  for (int p = threadIdx.x; p < nparts; p += K4_THREADS) {
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      const double x = partial[(long long)p * 8 + q];
      acc[q] = (q & 1) ? fmax(acc[q], x) : acc[q] + x;
    }
  }
  block_reduce8(acc, red);
  if (threadIdx.x == 0) {
#pragma unroll
    for (int q = 0; q < 8; ++q) out[q] = (q & 1) || ncell < 0.0 ? acc[q] : sqrt(acc[q] / ncell);
  }
}

}  // namespace z4c
