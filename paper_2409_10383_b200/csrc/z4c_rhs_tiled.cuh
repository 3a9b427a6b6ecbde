// K2, tuned variant: the RHS kernel with TMA-staged shared-memory tiles (sm_100a).
//
// One CTA of TX*TY*TZ threads owns a TX x TY x TZ tile of interior cells of one MeshBlock, one cell per
// thread. The 22 fields are streamed through a ring of NSTAGE shared-memory buffers, one (TX+6)(TY+6)(TZ+6)
// halo tile per field, each fetched by a single 5-D TMA box copy (cp.async.bulk.tensor, fp64 elements,
// coordinates (i, j, k, block, field) of the state pack) that completes on an mbarrier. While the threads take
// the stencils of field f out of shared memory -- centred 1st/2nd derivatives, upwinded advection and
// Kreiss-Oliger dissipation (S2 of SURVEY.md 8(a)) -- the copy engine is already fetching fields f+1..f+NSTAGE-1,
// so no thread ever waits on a global-memory load. The Z4c sources (S3) then run in registers.
//
// Upwinding without selects: with e_s = u_{+s} - u_{-s} and the Kreiss-Oliger sum ko = s3 - 6 s2 + 15 s1,
//   D^+ + D^- = (e3 - 6 e2 + 21 e1)/(12h),   D^+ - D^- = ko/(12h)
// hence beta D^{sign(beta)} u = [ beta (e3 - 6 e2 + 21 e1) + |beta| ko ] / (24h): the 7 values loaded for the
// KO operator serve the advection term too, with no per-axis branch or select (O3, reading Q9).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include "z4c_kernels.cuh"

namespace z4c {

// ---- mbarrier / TMA primitives (PTX) ------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {}
}
// one lane of a fully active warp (elect.sync): lets the tile issue sit behind a warp-uniform branch that the other
// three warps jump over, instead of 14 predicated-off instructions per field in every warp
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
  return pred != 0;
}
__device__ __forceinline__ void tma_load_5d(void* smem_dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1,
                                            int c2, int c3, int c4) {
  asm volatile(
      "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
      ::"r"(smem_u32(smem_dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
      : "memory");
}

// shared -> global box store (the reverse of tma_load_5d); elements outside the tensor's extents are not written
__device__ __forceinline__ void tma_store_5d(const CUtensorMap* map, const void* smem_src, int c0, int c1, int c2,
                                             int c3, int c4) {
  asm volatile("cp.async.bulk.tensor.5d.global.shared::cta.bulk_group [%0, {%2, %3, %4, %5, %6}], [%1];"
               ::"l"(map), "r"(smem_u32(smem_src)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
               : "memory");
}
__device__ __forceinline__ void tma_store_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
// the issuing thread: shared memory of all its committed stores has been read (it may be reused / released)
__device__ __forceinline__ void tma_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
// generic-proxy writes to shared memory made visible to the async proxy (TMA) that will read them
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---- tile geometry ---------------------------------------------------------------------------------
// PQ_TMA_: true = the CTA's P/Q register tiles are TMA-prefetched into shared memory at kernel start;
// false = they are read in the epilogue as one batch of independent global loads (lines requested into L2 by a
// prefetch at kernel start), which frees 2 x 22 x THREADS x 8 bytes of shared memory for a deeper tile ring.
template <int TX_, int TY_, int TZ_, int NSTAGE_, int MINB_ = 1, bool PQ_TMA_ = true, bool EARLY_PARK_ = !PQ_TMA_>
struct TileCfg {
  static constexpr int TX = TX_, TY = TY_, TZ = TZ_, NSTAGE = NSTAGE_, MINB = MINB_;
  static constexpr bool PQ_TMA = PQ_TMA_;
  static constexpr int THREADS = TX * TY * TZ;
  static constexpr int HX = TX + 2 * NG, HY = TY + 2 * NG, HZ = TZ + 2 * NG;
  static constexpr int SY = HX, SZ = HX * HY;          // element strides inside the halo tile
  static constexpr int TILE_ELEMS = HX * HY * HZ;
  static constexpr int TILE_BYTES = TILE_ELEMS * 8;
  static constexpr int STAGE_BYTES = (TILE_BYTES + 127) / 128 * 128;
  // With the RK-register tiles in shared memory a 4th ring slot lives at the end of the Q tile's area, which is idle
  // during the field stream (both register tiles are then asked for after the stream), and a 5th one behind the plane
  // set in the P tile's area, reaching a little into the front of the Q area.
  static constexpr int PHYS = (PQ_TMA_ && (NSTAGE_ == 4 || NSTAGE_ == 5)) ? 3 : NSTAGE_;
  static constexpr int BAR_OFF = PHYS * STAGE_BYTES;              // NSTAGE + 1 mbarriers
  static constexpr int REG_BYTES = NF * THREADS * 8;              // one RK-register tile [22][TZ][TY][TX]
  static constexpr int P_OFF = BAR_OFF + 128;                     // P tile, later the staged new state
  static constexpr int Q_OFF = P_OFF + (PQ_TMA ? REG_BYTES : 0);
  // per-thread parking of the advection + KO sums (without PQ_TMA it coincides with the staging tile at P_OFF)
  static constexpr int S_OFF = Q_OFF + (PQ_TMA ? REG_BYTES : 0);
  // without PQ_TMA the freed space holds a dedicated parking area for the late-use derivatives (written as each
  // field is done, so they stay out of registers through the whole field stream)
  static constexpr bool EARLY_PARK = EARLY_PARK_;
  static constexpr int E_OFF = S_OFF + REG_BYTES;
  // two-pass mixed derivatives: planes of D_x u and D_y u of the current field (raw, unscaled) on the tile plus the rows
  // / planes the second pass reaches, R = NG - 1 cells on either side. With PQ_TMA they live in the P/Q tile area, which
  // is idle until the field stream ends (the RK-register tiles are asked for after the last field); else in their own area.
  static constexpr int MIX_R = NG - 1;
  static constexpr int PXY = TY + 2 * MIX_R, PZ = TZ + 2 * MIX_R;
  static constexpr int PX_PLANE = PXY * TX, PX_ELEMS = PZ * PX_PLANE, PY_PLANE = TY * TX, PY_ELEMS = PZ * PY_PLANE;
  static constexpr int MIX_BYTES = ((PX_ELEMS + PY_ELEMS) * 8 + 127) / 128 * 128;
  static constexpr int SCR_OFF = PQ_TMA ? P_OFF : E_OFF + (EARLY_PARK ? NPARK * THREADS * 8 : 0);
  static_assert(!PQ_TMA || MIX_BYTES <= REG_BYTES, "the planes fit the P tile area (the Q tile arrives during the stream)");
  static constexpr int LIST_OFF = E_OFF + (EARLY_PARK ? NPARK * THREADS * 8 : 0) + (PQ_TMA ? 0 : MIX_BYTES);   // push lists
  static constexpr int MAXLIST = 32;
  __host__ __device__ static constexpr int slot_off(int s) {
    return s < PHYS ? s * STAGE_BYTES : (s == PHYS ? Q_OFF + REG_BYTES - STAGE_BYTES : P_OFF + MIX_BYTES);
  }
  static_assert(PHYS == NSTAGE_ || (STAGE_BYTES <= REG_BYTES && (REG_BYTES - STAGE_BYTES) % 128 == 0),
                "the 4th slot fits the end of the Q tile area");
  static_assert(NSTAGE_ - PHYS < 2 || P_OFF + MIX_BYTES + STAGE_BYTES <= Q_OFF + REG_BYTES - STAGE_BYTES,
                "the 5th slot ends before the 4th begins");
  static constexpr int SMEM_BYTES_RHS = LIST_OFF;                 // STAGE 0 (no lists)
  static constexpr int SMEM_BYTES = LIST_OFF + 9 * MAXLIST * 4 + 16;
  static_assert(TX + 2 * NG <= MAXLIST && TY + 2 * NG <= MAXLIST && TZ + 2 * NG <= MAXLIST, "push list size");
};

// Field streaming order: fields with second derivatives (two passes over the tile, a barrier in between) alternate with
// the others (one pass), so that the ring drains at an even rate and the single set of D_x / D_y planes is never
// rewritten before every thread has finished reading it (a whole field, with its barrier, lies in between).
__host__ __device__ constexpr int stream_field(int it) {
  constexpr int order[NF] = {BETAX, AXX,  BETAY, AXY,  BETAZ, AXZ,  CHI,  AYY,  GXX,  AYZ,  GXY,
                             AZZ,   GXZ,  KHAT,  GYY,  GAMX,  GYZ,  GAMY, GZZ,  GAMZ, ALPHA, THETA};
  return order[it];
}

// Which fields keep the difference-from-centre form of the symmetric sums (reading Q14): the ones that sit at O(1)
// with a small variation on top -- chi, gt_ij, alpha -- where u_{i+s} + u_{i-s} - 2 u_i would round at the size of the
// field instead of the size of its variation. The other 14 fields (At_ij, Khat, Gamt^i, Theta, beta^i) vanish on the
// flat background, so for them the sum-form s_k = (u_{+k} + u_{-k}) - 2 u_0 loses nothing and the centre terms of one
// axis fold into a single FMA each: 5 FP64 instructions fewer per axis (4 where d2 is wanted), ~200 per cell.
__host__ __device__ constexpr bool wants_dform(int f) { return f <= GZZ || f == ALPHA; }

// One axis of one field out of the shared-memory tile. t points at the cell, S is the compile-time stride.
template <int S, bool WANT_D1, bool WANT_D2, bool DFORM>
__device__ __forceinline__ void axis_tile(const double* t, const double c, const double bw, const double aw,
                                          const FdConst& fd, double& d1, double& d2, double& adv, double& raw1) {
#if Z4C_NG == 3
  const double lm3 = t[-3 * S], lm2 = t[-2 * S], lm1 = t[-S], lp1 = t[S], lp2 = t[2 * S], lp3 = t[3 * S];
  const double e1 = lp1 - lm1, e2 = lp2 - lm2, e3 = lp3 - lm3;
  double k;
  if (DFORM) {
    const double s1 = (lp1 - c) + (lm1 - c), s2 = (lp2 - c) + (lm2 - c), s3 = (lp3 - c) + (lm3 - c);
    if (WANT_D2) d2 = (16.0 * s1 - s2) * fd.inv12h2;
    k = s3 - 6.0 * s2 + 15.0 * s1;
  } else {
    const double t1 = lp1 + lm1, t2 = lp2 + lm2, t3 = lp3 + lm3;
    if (WANT_D2) d2 = (16.0 * t1 - t2 - 30.0 * c) * fd.inv12h2;
    k = t3 - 6.0 * t2 + 15.0 * t1 - 20.0 * c;
  }
  raw1 = 8.0 * e1 - e2;   // the centred first derivative before scaling: also the first pass of the mixed derivatives
  if (WANT_D1) d1 = raw1 * fd.inv12h;
  const double sy = e3 - 6.0 * e2 + 21.0 * e1;
#else
  // 6th order (NEXT-1). The lopsided pair obeys the same identity as at 4th order:
  //   D^+ + D^- = (104 e1 - 32 e2 + 8 e3 - e4)/(60h),   D^+ - D^- = (56 s1 - 28 s2 + 8 s3 - s4)/(60h) = KO sum/(60h)
  const double lm4 = t[-4 * S], lm3 = t[-3 * S], lm2 = t[-2 * S], lm1 = t[-S];
  const double lp1 = t[S], lp2 = t[2 * S], lp3 = t[3 * S], lp4 = t[4 * S];
  const double e1 = lp1 - lm1, e2 = lp2 - lm2, e3 = lp3 - lm3, e4 = lp4 - lm4;
  double k;
  if (DFORM) {
    const double s1 = (lp1 - c) + (lm1 - c), s2 = (lp2 - c) + (lm2 - c), s3 = (lp3 - c) + (lm3 - c),
                 s4 = (lp4 - c) + (lm4 - c);
    if (WANT_D2) d2 = (270.0 * s1 - 27.0 * s2 + 2.0 * s3) * fd.inv12h2;
    k = 56.0 * s1 - 28.0 * s2 + 8.0 * s3 - s4;
  } else {
    const double t1 = lp1 + lm1, t2 = lp2 + lm2, t3 = lp3 + lm3, t4 = lp4 + lm4;
    if (WANT_D2) d2 = (270.0 * t1 - 27.0 * t2 + 2.0 * t3 - 490.0 * c) * fd.inv12h2;
    k = 56.0 * t1 - 28.0 * t2 + 8.0 * t3 - t4 - 70.0 * c;
  }
  raw1 = 45.0 * e1 - 9.0 * e2 + e3;
  if (WANT_D1) d1 = raw1 * fd.inv12h;
  const double sy = 104.0 * e1 - 32.0 * e2 + 8.0 * e3 - e4;
#endif
  // bw = c_adv beta/(24h) [120h], aw = c_adv |beta|/(24h) + eps/(64h) [.., 256h]: advection and dissipation in two FMAs
  adv += bw * sy + aw * k;
}

// centred first derivative, raw (unscaled), along a compile-time stride: the operator that is applied twice
template <int S>
__device__ __forceinline__ double d1_tile(const double* q) {
#if Z4C_NG == 3
  return 8.0 * (q[S] - q[-S]) - (q[2 * S] - q[-2 * S]);
#else
  return 45.0 * (q[S] - q[-S]) - 9.0 * (q[2 * S] - q[-2 * S]) + (q[3 * S] - q[-3 * S]);
#endif
}

// One field out of its shared-memory tile. Fields with second derivatives take TWO passes: pass 1 (every thread, also
// the ones whose cell lies outside the block: their rows are somebody's neighbours) takes the axis stencils and stores
// D_x u and D_y u of its own cell and of the 2R rows / planes around the tile into the plane set `scr`; `release()` is
// the CTA barrier (after which nobody reads the tile any more, so it also frees the ring slot); pass 2 takes D_y and
// D_z of those planes: D_xy = D_y(D_x u), D_xz = D_z(D_x u), D_yz = D_z(D_y u) -- the same operator applied twice, in the
// same order and form as the one-pass evaluation (bit-identical), at 32 + 7 instead of 48 shared-memory accesses and
// 24 instead of 48 FP64 instructions per field (63 + 10 instead of 108, 53 instead of 141 at 6th order).
template <class Cfg, int F, class REL>
__device__ __forceinline__ void field_from_tile(const double* t, const double* bw, const double* aw,
                                                const FdConst& fd, const SrcParams& sp, double* u, Derivs& D,
                                                double* out, double* scr, const int ly, const int lz, REL release) {
  constexpr bool W1 = need_d1(F), W2 = need_d2(F);
  const double c = t[0];
  u[F] = c;
  double adv = 0.0, d1x = 0, d1y = 0, d1z = 0, d2x = 0, d2y = 0, d2z = 0;
  // bw[a] = beta^a/(24h), aw[a] = |beta^a|/(24h) + eps/(64h) (the Kreiss-Oliger weight folded in) for fields whose
  // advection is not switched by a gauge parameter; alpha and beta^i rebuild their weights with c_adv
  double w1[3], w2[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    if (F == ALPHA || F >= BETAX) {
      const double cadv = (F == ALPHA) ? sp.lapse_advect : sp.shift_advect;
      w1[a] = cadv * bw[a];
      w2[a] = cadv * (aw[a] - fd.ko) + fd.ko;
    } else {
      w1[a] = bw[a];
      w2[a] = aw[a];
    }
  }
  constexpr bool DF = wants_dform(F);
  double rx, ry, rz;
  axis_tile<1, W1, W2, DF>(t, c, w1[0], w2[0], fd, d1x, d2x, adv, rx);
  axis_tile<Cfg::SY, W1, W2, DF>(t, c, w1[1], w2[1], fd, d1y, d2y, adv, ry);
  axis_tile<Cfg::SZ, W1, W2, DF>(t, c, w1[2], w2[2], fd, d1z, d2z, adv, rz);
  if (W1) { D.d1[F][0] = d1x; D.d1[F][1] = d1y; D.d1[F][2] = d1z; }
  if (W2) {
    static_assert(Cfg::TY == 4 && Cfg::TZ == 2, "the halo-row assignment below is written for 16 x 4 x 2 tiles");
    constexpr int R = Cfg::MIX_R;
    double* px = scr + ((lz + R) * Cfg::PXY + (ly + R)) * Cfg::TX + (threadIdx.x % Cfg::TX);
    double* py = scr + Cfg::PX_ELEMS + ((lz + R) * Cfg::TY + ly) * Cfg::TX + (threadIdx.x % Cfg::TX);
    // every tile load first, every store after: the compiler cannot know that tile, planes and parking area are disjoint
#if Z4C_NG == 3
    const int dy = ly < R ? -R : R;   // rows -2, -1 (threads ly = 0, 1) and 4, 5 (ly = 2, 3) of the tile's own planes
    const double hxy = d1_tile<1>(t + dy * Cfg::SY);
    double hxz[2], hyz[2];            // planes -2, -1 (lz = 0, 1 with dz = -2) and 2, 3 (dz = +2)
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      hxz[q] = d1_tile<1>(t + (2 * q - 1) * R * Cfg::SZ);
      hyz[q] = d1_tile<Cfg::SY>(t + (2 * q - 1) * R * Cfg::SZ);
    }
    out[F * Cfg::THREADS] = adv;
    px[0] = rx;
    py[0] = ry;
    px[dy * Cfg::TX] = hxy;
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      px[(2 * q - 1) * R * Cfg::PX_PLANE] = hxz[q];
      py[(2 * q - 1) * R * Cfg::PY_PLANE] = hyz[q];
    }
#else
    double hxy[2], hxz[3], hyz[3];
#pragma unroll
    for (int q = 0; q < 2; ++q)       // rows -3..0 and 3..6 (rows 0 and 3 are rewritten with the same value)
      hxy[q] = d1_tile<1>(t + (2 * q - 1) * R * Cfg::SY);
    const int dzm = lz == 0 ? -1 : 1;  // planes -3, -2 | 3, 4 | -1 (lz = 0), 2 (lz = 1)
#pragma unroll
    for (int q = 0; q < 3; ++q) {
      const int dz = q == 0 ? -R : (q == 1 ? R : dzm);
      hxz[q] = d1_tile<1>(t + dz * Cfg::SZ);
      hyz[q] = d1_tile<Cfg::SY>(t + dz * Cfg::SZ);
    }
    out[F * Cfg::THREADS] = adv;
    px[0] = rx;
    py[0] = ry;
#pragma unroll
    for (int q = 0; q < 2; ++q) px[(2 * q - 1) * R * Cfg::TX] = hxy[q];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
      const int dz = q == 0 ? -R : (q == 1 ? R : dzm);
      px[dz * Cfg::PX_PLANE] = hxz[q];
      py[dz * Cfg::PY_PLANE] = hyz[q];
    }
#endif
    release();
    double d2[6];
    d2[sym(0, 0)] = d2x; d2[sym(1, 1)] = d2y; d2[sym(2, 2)] = d2z;
    d2[sym(0, 1)] = d1_tile<Cfg::TX>(px) * fd.inv144h2;
    d2[sym(0, 2)] = d1_tile<Cfg::PX_PLANE>(px) * fd.inv144h2;
    d2[sym(1, 2)] = d1_tile<Cfg::PY_PLANE>(py) * fd.inv144h2;
    consume_d2<F>(d2, D);
  } else {
    // parked in shared memory until the sources are assembled: 22 doubles fewer live through the tensor algebra
    out[F * Cfg::THREADS] = adv;
  }
  if (Cfg::EARLY_PARK) park_field_early<F>(D, out + (Cfg::E_OFF - Cfg::S_OFF) / 8, Cfg::THREADS);
}

// the field at whose barrier the Q tile of the RK registers is asked for (it is needed only in the epilogue; asked for at
// kernel start it queues ahead of the first ring refills)
constexpr int Q_AT = 6;
template <class Cfg, int IT>
struct FieldLoop {
  template <class EARLY>
  __device__ __forceinline__ static void run(const CUtensorMap* map, unsigned char* tiles, uint64_t* full,
                                             const int toff, const int cx, const int cy, const int cz, const int b,
                                             const bool active, double* bw, double* aw, const FdConst& fd,
                                             const SrcParams& sp, double* u, Derivs& D, double* out, double* scr,
                                             const int ly, const int lz, EARLY early) {
    constexpr int S = IT % Cfg::NSTAGE;
    constexpr int F = stream_field(IT);
    constexpr bool TWO = need_d2(F);
    // Every thread waits on the tile's barrier itself, right before it reads the tile. (Probing the barrier one field
    // ahead with mbarrier.test_wait and skipping this wait when the probe had already seen the phase complete was
    // measured: no faster, and on 256^3 runs a few cells per step read stale tile data -- DESIGN.md section 15.)
    mbar_wait(&full[S], (IT / Cfg::NSTAGE) & 1);
    const double* t = reinterpret_cast<const double*>(tiles + Cfg::slot_off(S)) + toff;
    // the barrier after which nobody reads stage S (and, for a two-pass field, everybody has written its planes)
    auto release = [&]() {
      __syncthreads();
      if (IT + Cfg::NSTAGE < NF && threadIdx.x < 32) {
        if (elect_one()) {
          mbar_expect_tx(&full[S], Cfg::TILE_BYTES);
          tma_load_5d(tiles + Cfg::slot_off(S), map, &full[S], cx, cy, cz, b, stream_field(IT + Cfg::NSTAGE));
          if (IT == Q_AT && Cfg::PHYS == Cfg::NSTAGE) early();
        }
      }
    };
    if (TWO) {
      field_from_tile<Cfg, F>(t, bw, aw, fd, sp, u, D, out, scr, ly, lz, release);
    } else {
      if (active) field_from_tile<Cfg, F>(t, bw, aw, fd, sp, u, D, out, scr, ly, lz, release);
      // needed to free the ring slot, or because the next field rewrites the planes the previous one is still reading
      constexpr bool NEXT_TWO = IT + 1 < NF && need_d2(stream_field(IT + 1 < NF ? IT + 1 : 0));
      if (IT + Cfg::NSTAGE < NF || NEXT_TWO) release();
    }
    FieldLoop<Cfg, IT + 1>::run(map, tiles, full, toff, cx, cy, cz, b, active, bw, aw, fd, sp, u, D, out, scr, ly, lz,
                                early);
  }
};
template <class Cfg>
struct FieldLoop<Cfg, NF> {
  template <class EARLY>
  __device__ __forceinline__ static void run(const CUtensorMap*, unsigned char*, uint64_t*, int, int, int, int, int,
                                             bool, double*, double*, const FdConst&, const SrcParams&, double*,
                                             Derivs&, double*, double*, int, int, EARLY) {}
};

// Arguments of the fused stage epilogue (STAGE 1..4): the RK registers, the OTHER state buffer (the stage
// reads y_in through the tensor map and writes the updated, enforced state and its ghost images to y_out, so
// no CTA ever reads a cell another CTA is writing), the chi floor and the error flag.
struct StageArgs {
  const double* y_in;   // the state buffer the tensor map describes (centre values of gt_ij are read up front)
  double* Q;
  Slab out;             // where the new state goes: this pack's other buffer and, for a partitioned mesh (NEXT-2), the
                        // other buffers of the z-neighbours' packs (peer memory)
  double chi_floor;
  int* flag;
  const int* blist = nullptr;   // blocks to run (device, nrun entries), or null: all blocks of the pack in order
  int nrun = 0;                 // (NEXT-3: the coarse blocks a fine level covers completely are not advanced)
};

// STAGE 0: P <- c*P + dt*(F(y) + Q_KO(y)) only (z4c_eval_rhs and the unfused path).
// STAGE 1..4: K2 + K3 + K1 in one pass ("one kernel per RK stage"): the same recurrence and the same
// expression forms as k_stage_update, applied to the cell while its 22 values are still in registers.
template <class Cfg, int STAGE>
__global__ void __launch_bounds__(Cfg::THREADS, Cfg::MINB)
    k_rhs_tiled(const __grid_constant__ CUtensorMap map, const __grid_constant__ CUtensorMap pmap,
                const __grid_constant__ CUtensorMap qmap, const __grid_constant__ CUtensorMap omap, Pack g,
                double* __restrict__ Preg, FdConst fd, SrcParams sp,
                double c, double dt, int tiles_y, int b0, StageArgs sa) {
  static_assert(Cfg::NSTAGE >= 3, "the three shift components are staged together");
  extern __shared__ __align__(128) unsigned char tiles[];   // NSTAGE halo tiles, then the mbarriers
  uint64_t* full = reinterpret_cast<uint64_t*>(tiles + Cfg::BAR_OFF);
  uint64_t* pqbar = full + Cfg::NSTAGE;
  // sP: staging tile of the new state (with PQ_TMA also the TMA'd P tile); sQ: the TMA'd Q tile
  double* sP = reinterpret_cast<double*>(tiles + Cfg::P_OFF);
  double* sQ = reinterpret_cast<double*>(tiles + Cfg::Q_OFF);
  int* lists = reinterpret_cast<int*>(tiles + Cfg::LIST_OFF);
  const int tid = threadIdx.x;
  const int lx = tid % Cfg::TX, ly = (tid / Cfg::TX) % Cfg::TY, lz = tid / (Cfg::TX * Cfg::TY);
  // grid = (tiles_x, tiles_y * tiles_z, blocks of this launch): one integer division per CTA instead of three
  const int tx = blockIdx.x, tz = blockIdx.y / tiles_y, ty = blockIdx.y - tz * tiles_y;
  const int b = sa.blist ? sa.blist[b0 + blockIdx.z] : b0 + blockIdx.z;
  // padded coordinates of the halo tile's origin = interior coordinates of the tile's first cell
  const int cx = tx * Cfg::TX, cy = ty * Cfg::TY, cz = tz * Cfg::TZ;
  const int i = cx + lx, j = cy + ly, k = cz + lz;
  const bool active = i < g.n && j < g.n && k < g.n;
  // gt^{ij} is needed while the very first fields stream in: the six centre values are requested before anything
  // else, so their latency overlaps the barrier set-up and the first tile copies
  // (the same for the shift, whose sign and size weight every field's advection)
  double gc[6], bc[3];
  {
    const double* yc = sa.y_in + (long long)b * g.m3 + ((long long)(k + NG) * g.m + (j + NG)) * g.m + (i + NG) + g.fs;
#pragma unroll
    for (int p = 0; p < 6; ++p, yc += g.fs)   // one running pointer: gt_xx .. gt_zz are fields 1..6
      gc[p] = active ? __ldcg(yc) : (p == 0 || p == 3 || p == 5 ? 1.0 : 0.0);
    yc += (long long)(BETAX - GZZ - 1) * g.fs;
#pragma unroll
    for (int a = 0; a < 3; ++a, yc += g.fs) bc[a] = active ? __ldcg(yc) : 0.0;
  }
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < Cfg::NSTAGE; ++s) mbar_init(&full[s], 1);
    mbar_init(pqbar, (STAGE >= 3 && Cfg::PHYS == Cfg::NSTAGE) ? 2 : 1);   // one arrival per RK-register tile asked for (Q early, P late)
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    // the first tiles are asked for by the thread that set the barriers up, before the CTA barrier (which only keeps
    // the other threads from polling a barrier that is not there yet)
#pragma unroll
    for (int s = 0; s < Cfg::NSTAGE; ++s) {
      mbar_expect_tx(&full[s], Cfg::TILE_BYTES);
      tma_load_5d(tiles + Cfg::slot_off(s), &map, &full[s], cx, cy, cz, b, stream_field(s));
    }
  }
  __syncthreads();
  // push lists (O2): per axis, every (source cell of this tile -> destination block, padded index) pair, the
  // cell's own position included; the destinations of the tile are the product of the three lists. Built by warps
  // 1..3, one axis each, one lane per source cell with a warp prefix sum for the list positions: a few dozen
  // instructions, so that no warp arrives late at the first barrier (a serial build by thread 0 cost ~1 us per CTA).
  static_assert(Cfg::THREADS == 128, "warps 1..3 build the lists of the axes x, y, z");
  if (STAGE >= 1 && tid >= 32) {
    const int lane = tid & 31;
    int bx, by, bz;
    block_coords(g, b, bx, by, bz);
    bz += sa.out.bz0[0];                                          // z in the lattice of the whole mesh (NEXT-2)
    {   // one copy of the body, run by three warps side by side (warp 0 holds the thread that issues the tile copies)
      const int a = (tid >> 5) - 1;
      const int c0 = a == 0 ? cx : (a == 1 ? cy : cz), T = a == 0 ? Cfg::TX : (a == 1 ? Cfg::TY : Cfg::TZ);
      const int nbl = a == 0 ? g.nb[0] : (a == 1 ? g.nb[1] : sa.out.nbz_global), bco = a == 0 ? bx : (a == 1 ? by : bz);
      int* L = lists + a * 3 * Cfg::MAXLIST;
      const int l = c0 + lane;
      const int na = min(T, g.n - c0);                              // source cells of the tile on this axis
      int tb[NG + 1], tl[NG + 1];
      const int nt = lane < na ? push_targets(l, bco, g.n, nbl, g.bc, tb, tl) : 0;
      if (a == 2) {   // z targets: (table entry of the pack that holds the block) << 24 | block z inside that pack
#pragma unroll
        for (int q = 0; q < NG + 1; ++q)
          if (q < nt) {
            const int e = slab_entry(sa.out, tb[q]);
            tb[q] = (e << 24) | (tb[q] - slab_bz0(sa.out, e));
          }
      }
      // list order: the cells' own positions first (entry = source cell), then the ghost images; so the tile's own
      // box is the corner [0, na)^3 of the product of the three lists and the images are the rest
      const int ni = nt > 0 ? nt - 1 : 0;
      int incl = ni;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int up = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += up;
      }
      const int pos = na + incl - ni;
#pragma unroll
      for (int q = 0; q < NG + 1; ++q)
        if (q < nt) {
          const int at = q == 0 ? lane : pos + q - 1;
          L[at] = lane; L[Cfg::MAXLIST + at] = tb[q]; L[2 * Cfg::MAXLIST + at] = tl[q];
        }
      if (lane == 31) lists[9 * Cfg::MAXLIST + a] = na + incl;
    }
  }
  const int toff = (lz + NG) * Cfg::SZ + (ly + NG) * Cfg::SY + lx + NG;
  if (STAGE >= 2 && !Cfg::PQ_TMA && active && lx == 0) {
    // ask L2 for this tile's rows of the RK registers (one 128-byte line per row and field)
    const long long c0 = (long long)b * g.n3 + ((long long)k * g.n + j) * g.n + i;
    const double* pq = sa.Q + c0;
    const double* pp = Preg + c0;
#pragma unroll 1   // a real loop: this kernel is instruction-fetch bound, straight-line code is not free
    for (int f = 0; f < NF; ++f, pq += g.is, pp += g.is) {
      asm volatile("prefetch.global.L2 [%0];" ::"l"(pq));
      if (STAGE >= 3) asm volatile("prefetch.global.L2 [%0];" ::"l"(pp));
    }
  }
  double bw[3], aw[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double beta = bc[a];
    bw[a] = beta * (0.5 * fd.inv12h);
    aw[a] = fabs(beta) * (0.5 * fd.inv12h) + fd.ko;
  }
  double u[NF];
  double* park = reinterpret_cast<double*>(tiles + Cfg::S_OFF) + tid;
  Derivs D;
  derivs_begin(gc, D);
  FieldLoop<Cfg, 0>::run(&map, tiles, full, toff, cx, cy, cz, b, active, bw, aw, fd, sp, u, D, park,
                         reinterpret_cast<double*>(tiles + Cfg::SCR_OFF), ly, lz, [&]() {
    // the Q tile of the RK registers, all 22 fields in one box (run by the one elected thread): its area is idle
    if (STAGE >= 2 && Cfg::PQ_TMA) {
      mbar_expect_tx(pqbar, Cfg::REG_BYTES);
      tma_load_5d(sQ, &qmap, pqbar, cx, cy, cz, b, 0);
    }
  });
  double out[NF];
  constexpr bool PARK = Cfg::PHYS * Cfg::STAGE_BYTES >= NPARK * Cfg::THREADS * 8;
  static_assert(PARK || !Cfg::PQ_TMA, "the barrier below also frees the planes in the P/Q tile area");
  if (PARK) __syncthreads();   // all threads (active or not) are done with the tile ring and with the planes
  if (Cfg::PHYS != Cfg::NSTAGE) {
    if (STAGE >= 2 && Cfg::PQ_TMA && tid < 32) {   // both register tiles now: the 4th ring slot used the Q area
      if (elect_one()) {
        mbar_expect_tx(pqbar, (STAGE >= 3 ? 2 : 1) * Cfg::REG_BYTES);
        tma_load_5d(sQ, &qmap, pqbar, cx, cy, cz, b, 0);
        if (STAGE >= 3) tma_load_5d(sP, &pmap, pqbar, cx, cy, cz, b, 0);
      }
    }
  } else if (STAGE >= 3 && Cfg::PQ_TMA && tid < 32) {
    // the P tile: asked for now that the planes of the two-pass derivatives no longer need its area; it lands while
    // the tensor algebra runs
    if (elect_one()) {
      mbar_expect_tx(pqbar, Cfg::REG_BYTES);
      tma_load_5d(sP, &pmap, pqbar, cx, cy, cz, b, 0);
    }
  }
  if (active) {
#pragma unroll
    for (int f = 0; f < NF; ++f) out[f] = 0.0;
    Geom G;
    if (Cfg::EARLY_PARK) {
      double* slot = reinterpret_cast<double*>(tiles + Cfg::E_OFF) + tid;
      asm volatile("" ::: "memory");
      geometry(u, D, G);
      asm volatile("" ::: "memory");
      park_late_derivs<false>(D, slot, Cfg::THREADS);
    } else if (PARK) {
      // the tile ring is idle now: park what only the final assembly reads while geometry() peaks
      // (this thread's last stencil loads are complete -- their values were consumed above -- and no TMA is
      // pending; other threads' reads of the ring are fenced by the barrier above)
      double* slot = reinterpret_cast<double*>(tiles) + tid;
      park_late_derivs<true>(D, slot, Cfg::THREADS);
      asm volatile("" ::: "memory");
      geometry(u, D, G);
      asm volatile("" ::: "memory");
      park_late_derivs<false>(D, slot, Cfg::THREADS);
    } else {
      geometry(u, D, G);
    }
    z4c_sources_post(sp, u, D, G, out);
#pragma unroll
    for (int f = 0; f < NF; ++f) out[f] += park[f * Cfg::THREADS];
  }
  const long long ci = (long long)b * g.n3 + ((long long)k * g.n + j) * g.n + i;
  double* pc = Preg + ci;
  if (STAGE == 0) {
    if (!active) return;
    if (c != 0.0) {
#pragma unroll
      for (int f = 0; f < NF; ++f) pc[f * g.is] = c * pc[f * g.is] + dt * out[f];
    } else {
#pragma unroll
      for (int f = 0; f < NF; ++f) pc[f * g.is] = dt * out[f];
    }
    return;
  }
  if (STAGE >= 2 && Cfg::PQ_TMA) mbar_wait(pqbar, 0);
  // (without PQ_TMA the two tiles could be staged in the idle ring; measured at 4 ghosts: 0.4 % slower than plain stores)
  constexpr bool PQ_BOX_STORE = STAGE <= 3 && Cfg::PQ_TMA;
  double* stP = reinterpret_cast<double*>(tiles + Cfg::S_OFF);
  double* stQ = sQ;
  if (active) {
    double* qc = sa.Q + ci;
    // without PQ_TMA: all loads of the RK registers first, as one batch of independent requests (the stores to P/Q
    // below may alias the loads as far as the compiler knows, which would otherwise serialise them)
    double Pold[NF], Qold[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      Qold[f] = (!Cfg::PQ_TMA && STAGE >= 2) ? __ldcg(qc + f * g.is) : 0.0;
      Pold[f] = (!Cfg::PQ_TMA && STAGE >= 3) ? __ldcg(pc + f * g.is) : 0.0;
    }
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      // With PQ_TMA the new register values go to shared memory -- Q over the old Q tile, P into the parking area of
      // the advection sums (read above), each thread its own slots -- and leave as two box stores after the barrier.
      double& Pnew = PQ_BOX_STORE ? stP[f * Cfg::THREADS + tid] : pc[f * g.is];
      double& Qnew = PQ_BOX_STORE ? stQ[f * Cfg::THREADS + tid] : qc[f * g.is];
      if (STAGE == 1) {
        const double P = dt * out[f];
        Qnew = P;
        u[f] = u[f] + 0.5 * P;
      } else if (STAGE == 2) {
        const double P = dt * out[f];
        const double Q = Cfg::PQ_TMA ? sQ[f * Cfg::THREADS + tid] : Qold[f];
        Pnew = P;
        u[f] = u[f] + 0.5 * (P - Q);
        Qnew = __dmul_rn(Q, SIXTH);
      } else if (STAGE == 3) {
        const double P = -0.5 * (Cfg::PQ_TMA ? sP[f * Cfg::THREADS + tid] : Pold[f]) + dt * out[f];
        const double Q = Cfg::PQ_TMA ? sQ[f * Cfg::THREADS + tid] : Qold[f];
        Pnew = P;
        u[f] = u[f] + P;
        Qnew = Q - P;
      } else {
        const double P = 2.0 * (Cfg::PQ_TMA ? sP[f * Cfg::THREADS + tid] : Pold[f]) + dt * out[f];
        const double Q = Cfg::PQ_TMA ? sQ[f * Cfg::THREADS + tid] : Qold[f];
        u[f] = u[f] + __dadd_rn(Q, __dmul_rn(P, SIXTH));
      }
    }
    bool bad = enforce_cell(u, sa.chi_floor);
    bad |= any_nonfinite(u);
    if (bad) *sa.flag = 1;
    // stage the new state of the tile (each thread overwrites only its own slots of the P tile)
#pragma unroll
    for (int f = 0; f < NF; ++f) sP[f * Cfg::THREADS + tid] = u[f];
  }
  fence_proxy_async_smem();   // the staged tile (and the new RK registers) are read by box stores
  __syncthreads();
  // A full tile's own cells leave as ONE box store of all 22 fields; a tile cut by the block's edge (n not a multiple
  // of the tile) goes through the loop below with the images, because its box would reach into ghost cells.
  // The box store needs its first element on a 16-byte boundary of global memory: true for the interior of a row at
  // 4 ghosts (offset 32 bytes), not at 3 (24 bytes: the copy engine raises an illegal-instruction fault), so the
  // 3-ghost build writes its own cells in the loop as well.
#ifdef Z4C_DBG_MISALIGNED_STORE
  constexpr bool TILE_STORE = true;
  constexpr int OX = NG + 1;
#else
  constexpr bool TILE_STORE = (NG * 8) % 16 == 0;
  constexpr int OX = NG;
#endif
  const bool full_tile = TILE_STORE && cx + Cfg::TX <= g.n && cy + Cfg::TY <= g.n && cz + Cfg::TZ <= g.n;
  if (tid == 0) {
    if (full_tile) tma_store_5d(&omap, sP, cx + OX, cy + NG, cz + NG, b, 0);
    if (PQ_BOX_STORE) {
      // the RK registers of the tile: one box store of all 22 fields each (cells beyond the block are clipped)
      tma_store_5d(&qmap, stQ, cx, cy, cz, b, 0);
      if (STAGE >= 2) tma_store_5d(&pmap, stP, cx, cy, cz, b, 0);
    }
    tma_store_commit();
  }
  // cooperative write-out of the tile's ghost images, x fastest. The destinations are the product of the three
  // per-axis lists minus the corner [0, nax) x [0, nay) x [0, naz) of own positions, enumerated as three slabs:
  //   A: qz >= naz (all qy, qx);  B: qz < naz, qy >= nay (all qx);  C: qz < naz, qy < nay, qx >= nax
  const int* Lx = lists;
  const int* Ly = lists + 3 * Cfg::MAXLIST;
  const int* Lz = lists + 6 * Cfg::MAXLIST;
  const int ncx = lists[9 * Cfg::MAXLIST], ncy = lists[9 * Cfg::MAXLIST + 1], ncz = lists[9 * Cfg::MAXLIST + 2];
  const int nax = full_tile ? Cfg::TX : 0, nay = full_tile ? Cfg::TY : 0, naz = full_tile ? Cfg::TZ : 0;
  const int wx = ncx - nax, wy = ncy - nay;
  const int nA = (ncz - naz) * ncy * ncx, nB = naz * wy * ncx, total = nA + nB + naz * nay * wx;
  // quotients by reciprocal multiplies: exact for these small ranges (q < 2^11, divisors <= 22: the quotient's
  // fractional part stays >= 0.5/22 away from an integer, float error is ~1e-4 of that); unused when a width is 0
  const float rcx = 1.0f / (float)ncx, rcy = 1.0f / (float)ncy, rwx = 1.0f / (float)wx, rwy = 1.0f / (float)wy,
              ray = 1.0f / (float)Cfg::TY;
  for (int q = tid; q < total; q += Cfg::THREADS) {
    int qx, qy, qz;
    if (q < nA) {
      const int r = (int)(((float)q + 0.5f) * rcx);
      qx = q - r * ncx;
      const int z = (int)(((float)r + 0.5f) * rcy);
      qy = r - z * ncy;
      qz = naz + z;
    } else if (q < nA + nB) {
      const int q2 = q - nA, r = (int)(((float)q2 + 0.5f) * rcx);
      qx = q2 - r * ncx;
      qz = (int)(((float)r + 0.5f) * rwy);
      qy = nay + r - qz * wy;
    } else {
      const int q2 = q - nA - nB, r = (int)(((float)q2 + 0.5f) * rwx);
      qx = nax + q2 - r * wx;
      qz = (int)(((float)r + 0.5f) * ray);
      qy = r - qz * Cfg::TY;
    }
    const int src = (Lz[qz] * Cfg::TY + Ly[qy]) * Cfg::TX + Lx[qx];
    const int zb = Lz[Cfg::MAXLIST + qz], e = zb >> 24;            // which pack, which block z inside it
    const long long tb = ((long long)(zb & 0xffffff) * g.nb[1] + Ly[Cfg::MAXLIST + qy]) * g.nb[0] + Lx[Cfg::MAXLIST + qx];
    double* d = slab_y(sa.out, e) + tb * g.m3 +
                ((long long)Lz[2 * Cfg::MAXLIST + qz] * g.m + Ly[2 * Cfg::MAXLIST + qy]) * g.m + Lx[2 * Cfg::MAXLIST + qx];
    const long long efs = slab_fs(sa.out, e);
#pragma unroll
    for (int f = 0; f < NF; ++f) d[f * efs] = sP[f * Cfg::THREADS + src];
  }
  if (tid == 0) tma_store_wait_read();   // shared memory stays put until the box stores have read it
}

// ---- host side -------------------------------------------------------------------------------------
// Default: 16x4x2 tile, 128 threads at 255 registers, 2 CTAs per SM, so one CTA's prologue (first TMA wait) and
// epilogue (write-out) overlap the other's stencil work. Measured (bench.py, one kernel per stage, B200):
//   64^3 wave: 0.202 ms per launch against 0.213 ms for the 16x4x4 tile (256 threads, 1 CTA per SM);
//   256^3 two punctures: 9.94 against 10.76 ms.  128-thread tiles capped at 168 / 128 registers (3 / 4 CTAs per
//   SM) were slower still (RHS only: 0.183 / 0.219 ms against 0.170 ms): the spills cost more than the warps hide.
//   8-wide tiles (8x4x4, 8x8x2: 20 % fewer halo bytes) are 20 % slower: 64-byte rows halve the coalescing of the
//   register / state rows and put two tile rows of a warp on the same shared-memory banks.
#if Z4C_NG == 3
// 5-deep ring: three slots of their own, the 4th at the end of the Q tile's area (+1.1 % on configs[3], +1.6 % on
// configs[1] over the 3-deep ring with the Q tile asked for during the stream), the 5th behind the plane set in the P
// tile's area (another +0.4 % / +0.9 %)
using RhsTile = TileCfg<16, 4, 2, 5, 2>;
#else
// 4 ghosts: the halo tile grows to 24 x 12 x 10 (23 KB); to keep 2 CTAs per SM the P/Q tiles are read by batched
// global loads instead of TMA (93 KB of shared memory per CTA)
using RhsTile = TileCfg<16, 4, 2, 3, 2, false, false>;
#endif
inline bool rhs_tiled_supported(const Pack& g) { return g.n % 2 == 0; }   // TMA strides must be 16-byte multiples

// Encode the 5-D tensor map (i, j, k, block, field) of the state pack with a halo-tile box. Returns false if
// the driver entry point is unavailable or rejects the geometry (the caller then keeps the plain variant).
template <class Cfg>
inline bool make_state_tensor_map(const Pack& g, const double* y, CUtensorMap* out, bool tile_box = false) {
  typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                               const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                               CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
      qres != cudaDriverEntryPointSuccess)
    return false;
  const cuuint64_t m = (cuuint64_t)g.m;
  const cuuint64_t dims[5] = {m, m, m, (cuuint64_t)g.nblk, (cuuint64_t)NF};
  const cuuint64_t strides[4] = {m * 8, m * m * 8, m * m * m * 8, (cuuint64_t)g.fs * 8};
  // halo tile of one field (loads), or the bare tile of all 22 fields (the store of a tile's new interior values)
  const cuuint32_t box[5] = {(cuuint32_t)(tile_box ? Cfg::TX : Cfg::HX), (cuuint32_t)(tile_box ? Cfg::TY : Cfg::HY),
                             (cuuint32_t)(tile_box ? Cfg::TZ : Cfg::HZ), 1, (cuuint32_t)(tile_box ? NF : 1)};
  const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
  const CUresult r = ((EncodeFn)fn)(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, (void*)y, dims, strides, box, estr,
                                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                    CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

// 5-D tensor map (i, j, k, block, field) of an RK register (interior cells only) with a whole-tile box.
template <class Cfg>
inline bool make_register_tensor_map(const Pack& g, const double* reg, CUtensorMap* out) {
  typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                               const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                               CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
      qres != cudaDriverEntryPointSuccess)
    return false;
  const cuuint64_t n = (cuuint64_t)g.n;
  const cuuint64_t dims[5] = {n, n, n, (cuuint64_t)g.nblk, (cuuint64_t)NF};
  const cuuint64_t strides[4] = {n * 8, n * n * 8, n * n * n * 8, (cuuint64_t)g.is * 8};
  const cuuint32_t box[5] = {(cuuint32_t)Cfg::TX, (cuuint32_t)Cfg::TY, (cuuint32_t)Cfg::TZ, 1, (cuuint32_t)NF};
  const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
  const CUresult r = ((EncodeFn)fn)(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, (void*)reg, dims, strides, box, estr,
                                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                    CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

struct RegMaps { CUtensorMap p, q, o[2]; };   // RK registers P, Q; the two state buffers with a bare-tile box (stores)

// Shared-memory opt-in of every stage instantiation, for the CURRENT device (function attributes are per device:
// z4c_create calls this once per context, so a process may drive several devices).
template <class Cfg, int STAGE>
inline cudaError_t configure_rhs_tiled_stage() {
  constexpr int smem = STAGE == 0 ? Cfg::SMEM_BYTES_RHS : Cfg::SMEM_BYTES;
  cudaError_t e = cudaFuncSetAttribute(k_rhs_tiled<Cfg, STAGE>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(k_rhs_tiled<Cfg, STAGE>, cudaFuncAttributePreferredSharedMemoryCarveout,
                              cudaSharedmemCarveoutMaxShared);
}
template <class Cfg>
inline cudaError_t configure_rhs_tiled() {
  cudaError_t e = configure_rhs_tiled_stage<Cfg, 0>();
  if (e == cudaSuccess) e = configure_rhs_tiled_stage<Cfg, 1>();
  if (e == cudaSuccess) e = configure_rhs_tiled_stage<Cfg, 2>();
  if (e == cudaSuccess) e = configure_rhs_tiled_stage<Cfg, 3>();
  if (e == cudaSuccess) e = configure_rhs_tiled_stage<Cfg, 4>();
  return e;
}

template <class Cfg, int STAGE>
inline cudaError_t launch_rhs_tiled_t(const CUtensorMap& map, const RegMaps& rm, const Pack& g, double* P, const FdConst& fd,
                                      const SrcParams& sp, double coef, double dt, cudaStream_t st,
                                      const StageArgs& sa, int out_buf = 0) {
  constexpr int smem = STAGE == 0 ? Cfg::SMEM_BYTES_RHS : Cfg::SMEM_BYTES;
  const int tx = (g.n + Cfg::TX - 1) / Cfg::TX, ty = (g.n + Cfg::TY - 1) / Cfg::TY, tz = (g.n + Cfg::TZ - 1) / Cfg::TZ;
  if ((long long)ty * tz > 65535) return cudaErrorInvalidConfiguration;
  const int nrun = sa.blist ? sa.nrun : g.nblk;
  for (int b0 = 0; b0 < nrun; b0 += 65535) {     // gridDim.z <= 65535: packs with more blocks take several launches
    const int nb = nrun - b0 < 65535 ? nrun - b0 : 65535;
    k_rhs_tiled<Cfg, STAGE><<<dim3(tx, ty * tz, nb), Cfg::THREADS, smem, st>>>(map, rm.p, rm.q, rm.o[out_buf], g, P, fd, sp,
                                                                                coef, dt, ty, b0, sa);
  }
  return cudaSuccess;
}

}  // namespace z4c
