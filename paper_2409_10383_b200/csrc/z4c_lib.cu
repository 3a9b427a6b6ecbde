// C ABI of the Z4c hot path (include/z4c.h): host-side context, launch sequencing of one RK4 step
// (ghost zones are refilled at every Runge-Kutta stage), CUDA-graph replay, error reporting.
// The library never allocates device memory and never touches the CPU oracle.
#include <cuda_runtime.h>

#include <cmath>
#include <mutex>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/z4c.h"
#include "z4c_amr.cuh"
#include "z4c_kernels.cuh"
#include "z4c_rhs_tiled.cuh"

using namespace z4c;

struct z4c_ctx {
  z4c_params prm;
  Pack g;
  FdConst fd;
  SrcParams sp;
  double dt;
  double* y;        // device, caller-owned
  double* P;        // device, workspace
  double* Q;        // device, workspace
  double* partial;  // device, workspace: K4 partials
  double* result;   // device, workspace: 8 doubles
  int* flag;        // device, workspace: error flag
  cudaStream_t stream;
  long long steps;
  int64_t launches;
  int variant;
  int use_graph;
  int fuse_ghosts;
  cudaGraphExec_t graph_exec;
  int graph_launches;
  double* ybuf[2];    // ybuf[0] = y (caller's state), ybuf[1] = second state buffer in the workspace
  CUtensorMap ymap[2];  // TMA descriptors of the two state buffers (tuned K2)
  int num_sms;
  RegMaps rmap;         // TMA descriptors of the RK registers P, Q
  int have_ymap;
  // NEXT-2: this pack is the slab [bz0, bz0 + nb[2]) of a lattice with nbz_global blocks along z
  int bz0, nbz_global;
  double* nbr_y[2][2];   // [lower, upper][state buffer 0, 1] of the neighbouring slabs (peer memory), or null
  int nbr_bz0[2], nbr_nbz[2];
  // NEXT-3: list of the blocks a two-level step advances on this (coarse) pack -- all but those a fine level covers
  int* blist;            // device, workspace: N_b ints
  int nactive;           // entries of blist in use; -1 = no list (every block runs)
  int blist_key[6];      // origin and extent of the fine region the list was built for
  std::string err;
};

namespace {

constexpr int K4_MAX_PARTS = 148 * 8;
constexpr size_t ALIGN = 256;
size_t align_up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

bool valid_params(const z4c_params* p) {
  if (!p) return false;
  if (p->ng != NG || p->n < 2 * NG) return false;
  if (p->nb[0] < 1 || p->nb[1] < 1 || p->nb[2] < 1) return false;
  if (p->bc != 0 && p->bc != 1) return false;
  if (!(p->dx > 0.0) || !std::isfinite(p->dx) || !(p->cfl > 0.0) || !std::isfinite(p->cfl)) return false;
  const long long nblk = (long long)p->nb[0] * p->nb[1] * p->nb[2];
  const long long m = p->n + 2 * NG;
  if (nblk > (1LL << 24) || m > 1024) return false;
  if (nblk * m * m * m > (1LL << 40)) return false;
  return true;
}

Pack make_pack(const z4c_params& p) {
  Pack g;
  g.n = p.n;
  g.m = p.n + 2 * NG;
  g.nb[0] = p.nb[0]; g.nb[1] = p.nb[1]; g.nb[2] = p.nb[2];
  g.nblk = p.nb[0] * p.nb[1] * p.nb[2];
  g.bc = p.bc;
  g.m2 = g.m * g.m;
  g.n3 = g.n * g.n * g.n;
  g.m3 = g.m * g.m * g.m;
  g.fs = (long long)g.nblk * g.m3;
  g.is = (long long)g.nblk * g.n3;
  g.ncell = g.is;
  return g;
}

bool partitioned(const z4c_ctx* c) { return c->nbz_global != c->g.nb[2]; }

// The table the ghost-writing (or -reading) kernels address: this pack's buffer `buf` and the same buffer of the two
// z-neighbours (NEXT-2). Unpartitioned: one entry.
Slab make_slab(const z4c_ctx* c, int buf) {
  Slab s;
  s.y[0] = c->ybuf[buf]; s.fs[0] = c->g.fs; s.bz0[0] = c->bz0; s.nbz[0] = c->g.nb[2];
  for (int side = 0; side < 2; ++side) {
    s.y[1 + side] = c->nbr_y[side][buf];
    s.bz0[1 + side] = c->nbr_bz0[side];
    s.nbz[1 + side] = c->nbr_y[side][buf] ? c->nbr_nbz[side] : 0;
    s.fs[1 + side] = (long long)c->g.nb[0] * c->g.nb[1] * c->nbr_nbz[side] * c->g.m3;
  }
  s.nbz_global = c->nbz_global;
  return s;
}

int fail(z4c_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg;
  return code;
}
int check_cuda(z4c_ctx* c, cudaError_t e, const char* what) {
  if (e == cudaSuccess) return Z4C_OK;
  return fail(c, Z4C_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
int check_launch(z4c_ctx* c, const char* what) {
  c->launches += 1;
  return check_cuda(c, cudaGetLastError(), what);
}

int grid_for(long long total, int threads, long long cap = (1LL << 30)) {
  long long b = (total + threads - 1) / threads;
  if (b > cap) b = cap;
  if (b < 1) b = 1;
  return (int)b;
}

// ---- launch helpers (all asynchronous on c->stream) ---------------------------------------
int launch_ghost_fill(z4c_ctx* c, int buf = 0) {
  const long long per_block = 2LL * NG * ((long long)c->g.m * c->g.m + (long long)c->g.n * c->g.m + (long long)c->g.n * c->g.n);
  k_ghost_fill<<<grid_for(per_block * c->g.nblk, 256), 256, 0, c->stream>>>(c->g, c->ybuf[buf], make_slab(c, buf));
  return check_launch(c, "k_ghost_fill");
}

int launch_rhs(z4c_ctx* c, double coef, double dt) {
  const Pack& g = c->g;
  if (c->variant != 1 && c->have_ymap) {
    cudaError_t e = launch_rhs_tiled_t<RhsTile, 0>(c->ymap[0], c->rmap, g, c->P, c->fd, c->sp, coef, dt, c->stream, StageArgs{c->y, nullptr, Slab{}, 0.0, nullptr});
    if (e != cudaSuccess) return check_cuda(c, e, "k_rhs_tiled launch");
    return check_launch(c, "k_rhs_tiled");
  }
  const int tx = (g.n + K2_TX - 1) / K2_TX, ty = (g.n + K2_TY - 1) / K2_TY, tz = (g.n + K2_TZ - 1) / K2_TZ;
  const long long nblocks = (long long)tx * ty * tz * g.nblk;
  if (nblocks > 0x7fffffffLL) return fail(c, Z4C_EINVAL, "pack too large for one K2 launch");
  k_rhs_global<<<(unsigned)nblocks, dim3(K2_TX, K2_TY, K2_TZ), 0, c->stream>>>(g, c->y, c->P, c->fd, c->sp, coef,
                                                                                  dt, tx, ty, tz);
  return check_launch(c, "k_rhs_global");
}

template <bool PUSH>
void launch_stage_update_t(z4c_ctx* c, int stage, int grid) {
  const Pack& g = c->g;
  const Slab sl = make_slab(c, 0);
  switch (stage) {
    case 0: k_stage_update<0, PUSH><<<grid, 128, 0, c->stream>>>(g, c->y, c->P, c->Q, c->prm.chi_floor, c->flag, sl); break;
    case 1: k_stage_update<1, PUSH><<<grid, 128, 0, c->stream>>>(g, c->y, c->P, c->Q, c->prm.chi_floor, c->flag, sl); break;
    case 2: k_stage_update<2, PUSH><<<grid, 128, 0, c->stream>>>(g, c->y, c->P, c->Q, c->prm.chi_floor, c->flag, sl); break;
    case 3: k_stage_update<3, PUSH><<<grid, 128, 0, c->stream>>>(g, c->y, c->P, c->Q, c->prm.chi_floor, c->flag, sl); break;
    default: k_stage_update<4, PUSH><<<grid, 128, 0, c->stream>>>(g, c->y, c->P, c->Q, c->prm.chi_floor, c->flag, sl); break;
  }
}

// K3 (+ K1 when the ghost push is fused in)
int launch_stage_update(z4c_ctx* c, int stage, bool push) {
  const int grid = grid_for(c->g.ncell, 128);
  if (push) launch_stage_update_t<true>(c, stage, grid);
  else launch_stage_update_t<false>(c, stage, grid);
  return check_launch(c, "k_stage_update");
}

// One RK stage as ONE kernel: RHS from ybuf[in] (TMA tiles), recurrence + enforcement in registers, updated
// state and its ghost images written to ybuf[1-in].
template <class Cfg>
cudaError_t launch_fused_stage_t(z4c_ctx* c, const CUtensorMap& map, const RegMaps& rm, int stage,
                                 const StageArgs& sa, int out_buf) {
  switch (stage) {
    case 1: return launch_rhs_tiled_t<Cfg, 1>(map, rm, c->g, c->P, c->fd, c->sp, 0.0, c->dt, c->stream, sa, out_buf);
    case 2: return launch_rhs_tiled_t<Cfg, 2>(map, rm, c->g, c->P, c->fd, c->sp, 0.0, c->dt, c->stream, sa, out_buf);
    case 3: return launch_rhs_tiled_t<Cfg, 3>(map, rm, c->g, c->P, c->fd, c->sp, -0.5, c->dt, c->stream, sa, out_buf);
    default: return launch_rhs_tiled_t<Cfg, 4>(map, rm, c->g, c->P, c->fd, c->sp, 2.0, c->dt, c->stream, sa, out_buf);
  }
}
int launch_fused_stage(z4c_ctx* c, int stage, int in, bool listed_blocks_only = false) {
  StageArgs sa{c->ybuf[in], c->Q, make_slab(c, 1 - in), c->prm.chi_floor, c->flag};
  if (listed_blocks_only && c->nactive >= 0) {
    if (c->nactive == 0) return Z4C_OK;   // a fine level covers the whole pack
    sa.blist = c->blist;
    sa.nrun = c->nactive;
  }
  cudaError_t e = launch_fused_stage_t<RhsTile>(c, c->ymap[in], c->rmap, stage, sa, 1 - in);
  if (e != cudaSuccess) return check_cuda(c, e, "k_rhs_tiled launch");
  return check_launch(c, "k_rhs_tiled<stage>");
}
bool fully_fused(const z4c_ctx* c) { return c->fuse_ghosts == 2 && c->variant != 1 && c->have_ymap; }

// One classical RK4 step in the 3-register recurrence: per stage
// K2 (P <- c_s P + dt L(y)) -> K3 (update + enforcement) -> K1 (ghost fill).
int enqueue_step(z4c_ctx* c) {
  static const double coef[4] = {0.0, 0.0, -0.5, 2.0};
  if (fully_fused(c)) {   // 4 launches; the state ping-pongs y -> y2 -> y -> y2 -> y
    for (int s = 1; s <= 4; ++s) {
      int rc = launch_fused_stage(c, s, (s - 1) & 1);
      if (rc) return rc;
    }
    return Z4C_OK;
  }
  for (int s = 1; s <= 4; ++s) {
    int rc = launch_rhs(c, coef[s - 1], c->dt);
    if (rc) return rc;
    rc = launch_stage_update(c, s, c->fuse_ghosts != 0);
    if (rc) return rc;
    if (!c->fuse_ghosts) {
      rc = launch_ghost_fill(c);
      if (rc) return rc;
    }
  }
  return Z4C_OK;
}

// The same launches as enqueue_step with a CUDA event between every pair of kernels, for per-kernel
// durations measured on the launching stream. ms[0..2] += time in K2, K3, K1.
int enqueue_step_timed(z4c_ctx* c, cudaEvent_t* ev, double* ms) {
  static const double coef[4] = {0.0, 0.0, -0.5, 2.0};
  int ne = 0;
  int kind[16];
  int rc = check_cuda(c, cudaEventRecord(ev[ne++], c->stream), "event record");
  if (rc) return rc;
  for (int s = 1; s <= 4 && fully_fused(c); ++s) {
    rc = launch_fused_stage(c, s, (s - 1) & 1);
    if (rc) return rc;
    kind[ne] = 0;
    cudaEventRecord(ev[ne++], c->stream);
  }
  for (int s = 1; s <= 4 && !fully_fused(c); ++s) {
    rc = launch_rhs(c, coef[s - 1], c->dt);
    if (rc) return rc;
    kind[ne] = 0;
    cudaEventRecord(ev[ne++], c->stream);
    rc = launch_stage_update(c, s, c->fuse_ghosts != 0);
    if (rc) return rc;
    kind[ne] = 1;
    cudaEventRecord(ev[ne++], c->stream);
    if (!c->fuse_ghosts) {
      rc = launch_ghost_fill(c);
      if (rc) return rc;
      kind[ne] = 2;
      cudaEventRecord(ev[ne++], c->stream);
    }
  }
  rc = check_cuda(c, cudaEventSynchronize(ev[ne - 1]), "event sync");
  if (rc) return rc;
  for (int e = 1; e < ne; ++e) {
    float t = 0.f;
    rc = check_cuda(c, cudaEventElapsedTime(&t, ev[e - 1], ev[e]), "event elapsed");
    if (rc) return rc;
    ms[kind[e]] += (double)t;
  }
  return Z4C_OK;
}

__global__ void __launch_bounds__(256) k_probe_dfma(double* out, int iters) {
  // 8 independent dependency chains of DFMA per thread: measures the FP64 pipe's issue rate
  double a0 = threadIdx.x * 1e-9, a1 = a0 + 1.0, a2 = a0 + 2.0, a3 = a0 + 3.0, a4 = a0 + 4.0, a5 = a0 + 5.0,
         a6 = a0 + 6.0, a7 = a0 + 7.0;
  const double m = 1.0000001, b = 1e-9;
  for (int i = 0; i < iters; ++i) {
    a0 = fma(a0, m, b); a1 = fma(a1, m, b); a2 = fma(a2, m, b); a3 = fma(a3, m, b);
    a4 = fma(a4, m, b); a5 = fma(a5, m, b); a6 = fma(a6, m, b); a7 = fma(a7, m, b);
  }
  const double r = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
  if (r == 123.456) out[0] = r;   // never true: keeps the loop alive
}

void drop_graph(z4c_ctx* c) {
  if (c->graph_exec) {
    cudaGraphExecDestroy(c->graph_exec);
    c->graph_exec = nullptr;
  }
}

int read_flag(z4c_ctx* c) {
  int h = 0;
  int rc = check_cuda(c, cudaMemcpyAsync(&h, c->flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream), "flag copy");
  if (rc) return rc;
  rc = check_cuda(c, cudaStreamSynchronize(c->stream), "stream sync");
  if (rc) return rc;
  if (h) return fail(c, Z4C_ESTATE, "device error flag set: non-finite value or det(gt) <= 0 in the stage update");
  return Z4C_OK;
}

}  // namespace

// ---- constraint monitors without any allocation (z4c_constraints_static, include/z4c.h) ---------------------------
// For callers that cannot allocate (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).
// The scratch of the two-pass reduction -- one row of 8 partial norms per MeshBlock -- lives in a file-scope device
// array of a fixed, modest size instead of the caller's workspace: 4096 rows x 8 doubles = 256 KiB, held by every GPU
// that loads this library until the process exits. In HOST code the array's name is only a stand-in for the symbol:
// the device address is looked up once per device with cudaGetSymbolAddress (static_scratch_ptr below) and handed to
// the kernels as an ordinary pointer. All calls on a device share the array; it keeps the last call's rows.
static __device__ __align__(256) double g_static_partial[(size_t)Z4C_STATIC_MAX_BLOCKS * 8];

namespace z4c {
// K4 with one CTA per MeshBlock: row b of `partial` <- {sum H^2, max|H|, sum |M|^2, max|M|, sum Theta^2, max|Theta|,
// sum |Z|^2, max|Z|} over the interior cells of block b (same point function and per-CTA reduction as k_constraints).
// Every row in [0, N_b) is written by its CTA on every call, so nothing in the scratch has to start at zero.
__global__ void __launch_bounds__(K4_THREADS)
    k_constraints_blocks(Pack g, const double* __restrict__ y, FdConst fd, SrcParams sp, double* __restrict__ partial) {
  __shared__ double red[8 * (K4_THREADS / 32)];
  double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  const int b = blockIdx.x;
  for (int r = threadIdx.x; r < g.n3; r += K4_THREADS) {
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
    acc[0] += c[0] * c[0];          acc[1] = fmax(acc[1], fabs(c[0]));
    acc[2] += c[4];                 acc[3] = fmax(acc[3], sqrt(c[4]));
    acc[4] += u[THETA] * u[THETA];  acc[5] = fmax(acc[5], fabs(u[THETA]));
    acc[6] += c[5];                 acc[7] = fmax(acc[7], sqrt(c[5]));
  }
  block_reduce8(acc, red);
  if (threadIdx.x == 0) {
#pragma unroll
    for (int q = 0; q < 8; ++q) partial[(long long)b * 8 + q] = acc[q];
  }
}
}  // namespace z4c

namespace {
// Device address of g_static_partial on the CURRENT device: looked up once per device, return code checked.
constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mutex;
double* g_static_ptr[STATIC_MAX_DEVICES] = {};
cudaError_t static_scratch_ptr(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_static_mutex);
  if (!g_static_ptr[dev]) {
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_static_partial);
    if (e != cudaSuccess) return e;
    g_static_ptr[dev] = p;
  }
  *out = g_static_ptr[dev];
  return cudaSuccess;
}
}  // namespace

extern "C" {

size_t z4c_state_bytes(const z4c_params* p) {
  if (!valid_params(p)) return 0;
  const Pack g = make_pack(*p);
  return (size_t)NF * (size_t)g.fs * sizeof(double);
}

size_t z4c_workspace_bytes(const z4c_params* p) {
  if (!valid_params(p)) return 0;
  const Pack g = make_pack(*p);
  const size_t reg = align_up((size_t)NF * (size_t)g.is * sizeof(double));
  return 2 * reg + align_up((size_t)K4_MAX_PARTS * 8 * sizeof(double)) + align_up(8 * sizeof(double)) + ALIGN +
         align_up((size_t)NF * (size_t)g.fs * sizeof(double)) + align_up((size_t)g.nblk * sizeof(int));
}

int z4c_create(const z4c_params* p, void* d_state, void* d_work, void* cuda_stream, z4c_ctx** out) {
  if (!out) return Z4C_EINVAL;
  *out = nullptr;
  if (!valid_params(p) || !d_state || !d_work) return Z4C_EINVAL;
  if (((uintptr_t)d_state % ALIGN) || ((uintptr_t)d_work % ALIGN)) return Z4C_EINVAL;
  z4c_ctx* c = new (std::nothrow) z4c_ctx();
  if (!c) return Z4C_EINVAL;
  c->prm = *p;
  c->g = make_pack(*p);
  const double h = p->dx;
  if (NG == 3) {   // 4th-order set (O3)
    c->fd.inv12h = 1.0 / (12.0 * h);
    c->fd.inv12h2 = 1.0 / (12.0 * h * h);
    c->fd.inv144h2 = 1.0 / (144.0 * h * h);
    c->fd.ko = p->ko_eps / (64.0 * h);
  } else {         // 6th-order set (NEXT-1)
    c->fd.inv12h = 1.0 / (60.0 * h);
    c->fd.inv12h2 = 1.0 / (180.0 * h * h);
    c->fd.inv144h2 = 1.0 / (3600.0 * h * h);
    c->fd.ko = p->ko_eps / (256.0 * h);
  }
  c->sp.kappa1 = p->kappa1; c->sp.kappa2 = p->kappa2;
  c->sp.lapse_oplog = p->lapse_oplog; c->sp.lapse_harmonic = p->lapse_harmonic; c->sp.lapse_advect = p->lapse_advect;
  c->sp.shift_gamma = p->shift_gamma; c->sp.shift_eta = p->shift_eta; c->sp.shift_advect = p->shift_advect;
  c->dt = p->cfl * p->dx;
  c->y = (double*)d_state;
  const size_t reg = align_up((size_t)NF * (size_t)c->g.is * sizeof(double));
  char* w = (char*)d_work;
  c->P = (double*)w;
  c->Q = (double*)(w + reg);
  c->partial = (double*)(w + 2 * reg);
  c->result = (double*)(w + 2 * reg + align_up((size_t)K4_MAX_PARTS * 8 * sizeof(double)));
  c->flag = (int*)((char*)c->result + align_up(8 * sizeof(double)));
  c->ybuf[0] = c->y;
  c->ybuf[1] = (double*)((char*)c->flag + ALIGN);
  c->blist = (int*)((char*)c->ybuf[1] + align_up((size_t)NF * (size_t)c->g.fs * sizeof(double)));
  c->nactive = -1;
  c->stream = (cudaStream_t)cuda_stream;
  c->steps = 0;
  c->launches = 0;
  c->variant = 0;
  c->use_graph = 0;
  c->fuse_ghosts = 2;
  c->graph_exec = nullptr;
  c->graph_launches = 0;
  c->bz0 = 0;
  c->nbz_global = c->g.nb[2];
  for (int side = 0; side < 2; ++side) {
    c->nbr_y[side][0] = c->nbr_y[side][1] = nullptr;
    c->nbr_bz0[side] = c->nbr_nbz[side] = 0;
  }
  {
    int dev = 0;
    c->num_sms = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev);
  }
  // The tuned kernels need TMA descriptors (16-byte strides: even n) and their shared-memory opt-in, which is a
  // per-device attribute: set here, for the current device, for every instantiation this context can launch.
  c->have_ymap = rhs_tiled_supported(c->g) && make_state_tensor_map<RhsTile>(c->g, c->ybuf[0], &c->ymap[0]) &&
                 make_state_tensor_map<RhsTile>(c->g, c->ybuf[1], &c->ymap[1]) &&
                 make_register_tensor_map<RhsTile>(c->g, c->P, &c->rmap.p) &&
                 make_register_tensor_map<RhsTile>(c->g, c->Q, &c->rmap.q) &&
                 make_state_tensor_map<RhsTile>(c->g, c->ybuf[0], &c->rmap.o[0], true) &&
                 make_state_tensor_map<RhsTile>(c->g, c->ybuf[1], &c->rmap.o[1], true) &&
                 configure_rhs_tiled<RhsTile>() == cudaSuccess ? 1 : 0;
  cudaError_t e = cudaMemsetAsync(d_work, 0, z4c_workspace_bytes(p), c->stream);
  if (e != cudaSuccess) {
    delete c;
    return Z4C_ECUDA;
  }
  *out = c;
  return Z4C_OK;
}

int z4c_set_initial_data(z4c_ctx* c, const double* interior, int on_device) {
  if (!c || !interior) return Z4C_EINVAL;
  const size_t bytes = (size_t)NF * (size_t)c->g.ncell * sizeof(double);
  const double* src = interior;
  int rc;
  if (!on_device) {
    // stage through the RK register area (P and Q are contiguous and together hold 2x this size)
    rc = check_cuda(c, cudaMemcpyAsync(c->P, interior, bytes, cudaMemcpyHostToDevice, c->stream), "H2D copy");
    if (rc) return rc;
    src = c->P;
  }
  // ghosts are overwritten below; clear the state first so no uninitialised value is ever read
  rc = check_cuda(c, cudaMemsetAsync(c->y, 0, (size_t)NF * (size_t)c->g.fs * sizeof(double), c->stream), "memset");
  if (rc) return rc;
  k_layout<0><<<grid_for((long long)NF * c->g.ncell, 256, 148 * 32), 256, 0, c->stream>>>(c->g, c->y,
                                                                                            (double*)src, NF);
  rc = check_launch(c, "k_layout<0>");
  if (rc) return rc;
  rc = check_cuda(c, cudaMemsetAsync(c->flag, 0, sizeof(int), c->stream), "memset flag");
  if (rc) return rc;
  rc = launch_stage_update(c, 0, false);
  if (rc) return rc;
  if (!partitioned(c)) {   // a slab's ghosts need its neighbours' data: z4c_fill_ghosts after a barrier (NEXT-2)
    rc = launch_ghost_fill(c);
    if (rc) return rc;
  }
  const size_t reg = align_up((size_t)NF * (size_t)c->g.is * sizeof(double));
  rc = check_cuda(c, cudaMemsetAsync(c->P, 0, 2 * reg, c->stream), "memset registers");
  if (rc) return rc;
  c->steps = 0;
  if (!on_device) return check_cuda(c, cudaStreamSynchronize(c->stream), "stream sync");
  return Z4C_OK;
}

int z4c_step(z4c_ctx* c, int nsteps) {
  if (!c || nsteps < 0) return Z4C_EINVAL;
  if (partitioned(c))
    return fail(c, Z4C_EINVAL, "a slab of a partitioned mesh advances stage by stage: z4c_stage + a barrier between stages");
  if (c->use_graph) {
    if (!c->graph_exec) {
      cudaGraph_t graph = nullptr;
      int rc = check_cuda(c, cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal), "begin capture");
      if (rc) return rc;
      const int64_t before = c->launches;
      rc = enqueue_step(c);
      c->graph_launches = (int)(c->launches - before);
      c->launches = before;
      cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
      if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
      rc = check_cuda(c, e, "end capture");
      if (rc) return rc;
      e = cudaGraphInstantiate(&c->graph_exec, graph, 0);
      cudaGraphDestroy(graph);
      rc = check_cuda(c, e, "graph instantiate");
      if (rc) { c->graph_exec = nullptr; return rc; }
    }
    for (int s = 0; s < nsteps; ++s) {
      int rc = check_cuda(c, cudaGraphLaunch(c->graph_exec, c->stream), "graph launch");
      if (rc) return rc;
      c->launches += c->graph_launches;
    }
  } else {
    for (int s = 0; s < nsteps; ++s) {
      int rc = enqueue_step(c);
      if (rc) return rc;
    }
  }
  c->steps += nsteps;
  return Z4C_OK;
}

int z4c_constraints(z4c_ctx* c, double* out, double* d_percell) {
  if (!c || !out) return Z4C_EINVAL;
  int nparts = grid_for(c->g.ncell, K4_THREADS, K4_MAX_PARTS);
  k_constraints<<<nparts, K4_THREADS, 0, c->stream>>>(c->g, c->y, c->fd, c->sp, c->partial, d_percell);
  int rc = check_launch(c, "k_constraints");
  if (rc) return rc;
  k_constraints_final<<<1, K4_THREADS, 0, c->stream>>>(c->partial, nparts, (double)c->g.ncell, c->result);
  rc = check_launch(c, "k_constraints_final");
  if (rc) return rc;
  rc = check_cuda(c, cudaMemcpyAsync(out, c->result, 8 * sizeof(double), cudaMemcpyDeviceToHost, c->stream),
                  "D2H copy");
  if (rc) return rc;
  return read_flag(c);
}

int z4c_refine_indicators(z4c_ctx* c, double chi_min, double dchi_max, double* d_minchi, double* d_maxdchi,
                          int32_t* d_flags) {
  if (!c || (!d_minchi && !d_maxdchi && !d_flags)) return Z4C_EINVAL;
  k_refine_indicators<<<c->g.nblk, KR_THREADS, 0, c->stream>>>(c->g, c->y, c->fd, chi_min, dchi_max, d_minchi,
                                                                d_maxdchi, (int*)d_flags);
  return check_launch(c, "k_refine_indicators");
}

int z4c_get_interior(z4c_ctx* c, double* interior, int on_device) {
  if (!c || !interior) return Z4C_EINVAL;
  const size_t bytes = (size_t)NF * (size_t)c->g.ncell * sizeof(double);
  double* dst = on_device ? interior : c->P;
  k_layout<1><<<grid_for((long long)NF * c->g.ncell, 256, 148 * 32), 256, 0, c->stream>>>(c->g, c->y, dst, NF);
  int rc = check_launch(c, "k_layout<1>");
  if (rc) return rc;
  if (!on_device) {
    rc = check_cuda(c, cudaMemcpyAsync(interior, c->P, bytes, cudaMemcpyDeviceToHost, c->stream), "D2H copy");
    if (rc) return rc;
    return check_cuda(c, cudaStreamSynchronize(c->stream), "stream sync");
  }
  return Z4C_OK;
}

int z4c_fill_ghosts(z4c_ctx* c) {
  if (!c) return Z4C_EINVAL;
  return launch_ghost_fill(c);
}

int z4c_eval_rhs(z4c_ctx* c, double* d_out) {
  if (!c || !d_out) return Z4C_EINVAL;
  int rc = launch_rhs(c, 0.0, 1.0);
  if (rc) return rc;
  k_layout<2><<<grid_for((long long)NF * c->g.ncell, 256, 148 * 32), 256, 0, c->stream>>>(c->g, c->P, d_out, NF);
  return check_launch(c, "k_layout<2>");
}

int z4c_enforce(z4c_ctx* c) {
  if (!c) return Z4C_EINVAL;
  if (c->fuse_ghosts) return launch_stage_update(c, 0, true);  // K3 with ghost push
  int rc = launch_stage_update(c, 0, false);
  if (rc) return rc;
  return launch_ghost_fill(c);
}

int z4c_step_timed(z4c_ctx* c, int nsteps, double* ms_out) {
  if (!c || nsteps < 0 || !ms_out) return Z4C_EINVAL;
  cudaEvent_t ev[16];
  for (int e = 0; e < 16; ++e)
    if (cudaEventCreate(&ev[e]) != cudaSuccess) return fail(c, Z4C_ECUDA, "event create");
  ms_out[0] = ms_out[1] = ms_out[2] = 0.0;
  int rc = Z4C_OK;
  for (int s = 0; s < nsteps && rc == Z4C_OK; ++s) rc = enqueue_step_timed(c, ev, ms_out);
  for (int e = 0; e < 16; ++e) cudaEventDestroy(ev[e]);
  if (rc == Z4C_OK) c->steps += nsteps;
  return rc;
}

int z4c_probe_fp64(void* cuda_stream, void* d_scratch, int iters, double* tflops_out) {
  if (!d_scratch || !tflops_out || iters < 1) return Z4C_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return Z4C_ECUDA;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return Z4C_ECUDA;
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return Z4C_ECUDA;
  const int grid = sms * 8, threads = 256;
  k_probe_dfma<<<grid, threads, 0, st>>>((double*)d_scratch, iters);   // warm-up
  cudaEventRecord(e0, st);
  k_probe_dfma<<<grid, threads, 0, st>>>((double*)d_scratch, iters);
  cudaEventRecord(e1, st);
  cudaError_t e = cudaEventSynchronize(e1);
  float ms = 0.f;
  if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) return Z4C_ECUDA;
  *tflops_out = 2.0 * 8.0 * (double)iters * (double)grid * threads / ((double)ms * 1e-3) * 1e-12;
  return Z4C_OK;
}

// ---- NEXT-3: two-level static refinement ------------------------------------------------
namespace {
// The fine pack must be the factor-2 refinement of a box of the coarse pack, both on one stream with one dt.
int check_levels(z4c_ctx* coarse, z4c_ctx* fine, const int32_t* origin, AmrGeom* a) {
  if (!coarse || !fine || !origin || coarse == fine) return Z4C_EINVAL;
  if (coarse->stream != fine->stream) return fail(fine, Z4C_EINVAL, "two-level calls need both contexts on one stream");
  if (partitioned(coarse) || partitioned(fine)) return fail(fine, Z4C_EINVAL, "two-level calls need unpartitioned packs");
  if (fine->g.n % 2) return fail(fine, Z4C_EINVAL, "restriction needs an even block size");
  if (std::fabs(2.0 * fine->prm.dx - coarse->prm.dx) > 1e-12 * coarse->prm.dx)
    return fail(fine, Z4C_EINVAL, "fine dx must be half the coarse dx");
  for (int d = 0; d < 3; ++d) {
    a->origin[d] = origin[d];
    a->Mc[d] = fine->g.n * fine->g.nb[d] / 2;
    if (origin[d] < 0 || origin[d] + a->Mc[d] > coarse->g.n * coarse->g.nb[d])
      return fail(fine, Z4C_EINVAL, "fine region does not lie inside the coarse mesh");
  }
  return Z4C_OK;
}
int launch_restrict(z4c_ctx* coarse, z4c_ctx* fine, const AmrGeom& a, int buf = 0) {
  const long long bricks = a.layer >= 0 ? (restrict_layer_cells(a) + RB_X * RB_Y * RB_Z - 1) / (RB_X * RB_Y * RB_Z)
                                        : (long long)((a.Mc[0] + RB_X - 1) / RB_X) * ((a.Mc[1] + RB_Y - 1) / RB_Y) *
                                              ((a.Mc[2] + RB_Z - 1) / RB_Z);
  if (bricks > 0x7fffffffLL) return fail(fine, Z4C_EINVAL, "fine region too large for one k_restrict launch");
  k_restrict<<<dim3((unsigned)bricks, NF), RB_X * RB_Y * RB_Z, 0, fine->stream>>>(
      fine->g, fine->ybuf[buf], coarse->g, coarse->ybuf[buf], a, make_amr_weights(fine->g.n));
  return check_launch(fine, "k_restrict");
}
int launch_prolong(z4c_ctx* coarse, z4c_ctx* fine, const AmrGeom& a, int buf = 0) {
  const Pack& g = fine->g;
  if (coarse->g.fs > 0x7fffffffLL) return fail(fine, Z4C_EINVAL, "coarse pack too large for k_prolong's 32-bit offsets");
  k_prolong<<<grid_for(prolong_shell_cells(g.n, g.nb), 128), 128, 0, fine->stream>>>(coarse->g, coarse->ybuf[buf], g,
                                                                               fine->ybuf[buf], a,
                                                                               make_amr_weights(g.n));
  return check_launch(fine, "k_prolong");
}
// The coarse blocks that are not completely covered by the fine region, in pack order, into the workspace's list.
int list_uncovered_blocks(z4c_ctx* coarse, const AmrGeom& a) {
  const int key[6] = {a.origin[0], a.origin[1], a.origin[2], a.Mc[0], a.Mc[1], a.Mc[2]};
  if (coarse->nactive >= 0 && std::memcmp(key, coarse->blist_key, sizeof(key)) == 0) return Z4C_OK;
  const Pack& g = coarse->g;
  std::vector<int> list;
  list.reserve(g.nblk);
  for (int b = 0; b < g.nblk; ++b) {
    const int bx = b % g.nb[0], by = (b / g.nb[0]) % g.nb[1], bz = b / (g.nb[0] * g.nb[1]);
    const int lo[3] = {bx * g.n, by * g.n, bz * g.n};
    bool covered = true;
    for (int d = 0; d < 3; ++d) covered = covered && lo[d] >= a.origin[d] && lo[d] + g.n <= a.origin[d] + a.Mc[d];
    if (!covered) list.push_back(b);
  }
  // pageable source: the copy is staged before the call returns, so the vector may go
  int rc = check_cuda(coarse, cudaMemcpyAsync(coarse->blist, list.data(), list.size() * sizeof(int), cudaMemcpyHostToDevice,
                                              coarse->stream), "block list copy");
  if (rc) return rc;
  coarse->nactive = (int)list.size();
  std::memcpy(coarse->blist_key, key, sizeof(key));
  return Z4C_OK;
}
// steps B.1, A.2/B.2 (k_restrict writes the ghost images of the covered coarse nodes itself), B.5; on state buffer `buf`
int sync_levels(z4c_ctx* coarse, z4c_ctx* fine, const AmrGeom& a, int buf = 0) {
  int rc = launch_restrict(coarse, fine, a, buf);
  if (rc) return rc;
  return launch_prolong(coarse, fine, a, buf);
}
}  // namespace

int z4c_restrict(z4c_ctx* fine, z4c_ctx* coarse, const int32_t* origin) {
  AmrGeom a;
  int rc = check_levels(coarse, fine, origin, &a);
  if (rc) return rc;
  return launch_restrict(coarse, fine, a);
}

int z4c_prolongate(z4c_ctx* coarse, z4c_ctx* fine, const int32_t* origin) {
  AmrGeom a;
  int rc = check_levels(coarse, fine, origin, &a);
  if (rc) return rc;
  return launch_prolong(coarse, fine, a);
}

int z4c_two_level_step(z4c_ctx* coarse, z4c_ctx* fine, const int32_t* origin, int nsteps) {
  static const double coef[4] = {0.0, 0.0, -0.5, 2.0};
  AmrGeom a;
  int rc = check_levels(coarse, fine, origin, &a);
  if (rc) return rc;
  if (nsteps < 0) return Z4C_EINVAL;
  if (std::fabs(coarse->dt - fine->dt) > 1e-14 * fine->dt)
    return fail(fine, Z4C_EINVAL, "both levels advance with one dt (no subcycling): set cfl so that cfl*dx agrees");
  rc = sync_levels(coarse, fine, a);
  // Both levels in mode 2: one stage kernel per level and stage (state ping-pong ybuf[in] -> ybuf[1 - in], ghost images
  // written by the kernel), then the level exchange on the buffer just written. Otherwise K2 + K3-with-push in place.
  const bool fused = fully_fused(coarse) && fully_fused(fine);
  // A region made of whole coarse blocks (the paper's refinement unit): whatever the coarse stage kernel
  // computes on those blocks is overwritten by the restriction, so they are not advanced at all, and between stages
  // only the covered cells that anyone reads are restricted: the N_g layers under the region's faces (ghost images
  // of the coarse neighbours, step A.2 / B.2; the prolongation stencils reach 2 nodes in). The last stage of the call
  // restricts every covered cell, so the caller finds the coarse level complete.
  bool whole_blocks = fused && rc == Z4C_OK;
  for (int d = 0; d < 3; ++d) whole_blocks = whole_blocks && a.origin[d] % coarse->g.n == 0 && a.Mc[d] % coarse->g.n == 0;
  if (whole_blocks) rc = list_uncovered_blocks(coarse, a);
  AmrGeom faces = a;
  faces.layer = NG;
  for (int d = 0; d < 3; ++d) if (2 * NG > a.Mc[d]) faces.layer = -1;   // a region thinner than two layers: all of it
  z4c_ctx* lv[2] = {coarse, fine};
  for (int st = 0; st < nsteps && rc == Z4C_OK; ++st)
    for (int s = 1; s <= 4 && rc == Z4C_OK; ++s) {
      const int in = (s - 1) & 1;
      if (fused) {
        rc = launch_fused_stage(coarse, s, in, whole_blocks);
        if (rc == Z4C_OK) rc = launch_fused_stage(fine, s, in);
        const bool last = st == nsteps - 1 && s == 4;
        if (rc == Z4C_OK) rc = sync_levels(coarse, fine, whole_blocks && !last ? faces : a, 1 - in);
      } else {
        for (int q = 0; q < 2 && rc == Z4C_OK; ++q) rc = launch_rhs(lv[q], coef[s - 1], lv[q]->dt);
        for (int q = 0; q < 2 && rc == Z4C_OK; ++q) rc = launch_stage_update(lv[q], s, true);
        if (rc == Z4C_OK) rc = sync_levels(coarse, fine, a);
      }
    }
  if (rc == Z4C_OK) { coarse->steps += nsteps; fine->steps += nsteps; }
  return rc;
}

// ---- NEXT-2: partitioned mesh (ghost exchange at every stage) -----------
int z4c_enable_peer(int32_t peer_device) {
  int dev = -1, count = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceCount(&count) != cudaSuccess) return Z4C_ECUDA;
  if (peer_device < 0 || peer_device >= count) return Z4C_ECUDA;
  if (peer_device == dev) return Z4C_OK;
  int can = 0;
  if (cudaDeviceCanAccessPeer(&can, dev, peer_device) != cudaSuccess || !can) return Z4C_ECUDA;
  const cudaError_t e = cudaDeviceEnablePeerAccess(peer_device, 0);
  if (e == cudaErrorPeerAccessAlreadyEnabled) {
    cudaGetLastError();   // not an error: clear it
    return Z4C_OK;
  }
  return e == cudaSuccess ? Z4C_OK : Z4C_ECUDA;
}

int z4c_set_partition(z4c_ctx* c, int32_t nbz_global, int32_t bz0) {
  if (!c) return Z4C_EINVAL;
  if (bz0 < 0 || nbz_global < 1 || bz0 + c->g.nb[2] > nbz_global || nbz_global > (1 << 24)) return Z4C_EINVAL;
  drop_graph(c);
  c->nbz_global = nbz_global;
  c->bz0 = bz0;
  if (partitioned(c) && c->fuse_ghosts == 0) c->fuse_ghosts = 1;
  return Z4C_OK;
}

int z4c_set_neighbor(z4c_ctx* c, int32_t side, void* d_state, void* d_state2, int32_t bz0, int32_t nbz) {
  if (!c || side < 0 || side > 1) return Z4C_EINVAL;
  if ((d_state || d_state2) && (!d_state || !d_state2 || nbz < 1 || bz0 < 0 || bz0 + nbz > c->nbz_global)) return Z4C_EINVAL;
  drop_graph(c);
  c->nbr_y[side][0] = (double*)d_state;
  c->nbr_y[side][1] = (double*)d_state2;
  c->nbr_bz0[side] = bz0;
  c->nbr_nbz[side] = nbz;
  return Z4C_OK;
}

void* z4c_state2(const z4c_ctx* c) { return c ? (void*)c->ybuf[1] : nullptr; }

int z4c_stage(z4c_ctx* c, int stage) {
  static const double coef[4] = {0.0, 0.0, -0.5, 2.0};
  if (!c || stage < 1 || stage > 4) return Z4C_EINVAL;
  int rc;
  if (fully_fused(c)) {
    rc = launch_fused_stage(c, stage, (stage - 1) & 1);
  } else {
    if (partitioned(c))
      return fail(c, Z4C_EINVAL, "in modes 0/1 the state is updated in place: a slab needs a barrier between the RHS "
                                 "and the update of a stage (z4c_stage_rhs, barrier, z4c_stage_update, barrier)");
    rc = launch_rhs(c, coef[stage - 1], c->dt);
    if (rc == Z4C_OK) rc = launch_stage_update(c, stage, c->fuse_ghosts != 0);
    if (rc == Z4C_OK && !c->fuse_ghosts) rc = launch_ghost_fill(c);
  }
  if (rc == Z4C_OK && stage == 4) c->steps += 1;
  return rc;
}

int z4c_stage_rhs(z4c_ctx* c, int stage) {
  static const double coef[4] = {0.0, 0.0, -0.5, 2.0};
  if (!c || stage < 1 || stage > 4) return Z4C_EINVAL;
  return launch_rhs(c, coef[stage - 1], c->dt);
}

int z4c_stage_update(z4c_ctx* c, int stage) {
  if (!c || stage < 1 || stage > 4) return Z4C_EINVAL;
  int rc = launch_stage_update(c, stage, true);
  if (rc == Z4C_OK && stage == 4) c->steps += 1;
  return rc;
}

int z4c_constraints_raw(z4c_ctx* c, double* out) {
  if (!c || !out) return Z4C_EINVAL;
  int nparts = grid_for(c->g.ncell, K4_THREADS, K4_MAX_PARTS);
  k_constraints<<<nparts, K4_THREADS, 0, c->stream>>>(c->g, c->y, c->fd, c->sp, c->partial, nullptr);
  int rc = check_launch(c, "k_constraints");
  if (rc) return rc;
  k_constraints_final<<<1, K4_THREADS, 0, c->stream>>>(c->partial, nparts, -1.0, c->result);
  rc = check_launch(c, "k_constraints_final");
  if (rc) return rc;
  rc = check_cuda(c, cudaMemcpyAsync(out, c->result, 8 * sizeof(double), cudaMemcpyDeviceToHost, c->stream),
                  "D2H copy");
  if (rc) return rc;
  return read_flag(c);
}

int z4c_constraints_static(z4c_ctx* c, double* d_out) {
  if (!c || !d_out) return Z4C_EINVAL;
  if (c->g.nblk > Z4C_STATIC_MAX_BLOCKS)
    return fail(c, Z4C_EINVAL, "z4c_constraints_static: the pack has " + std::to_string(c->g.nblk) +
                               " MeshBlocks, the static scratch holds " + std::to_string(Z4C_STATIC_MAX_BLOCKS) +
                               " rows (use z4c_constraints, whose partials live in the caller's workspace)");
  double* scratch = nullptr;
  int rc = check_cuda(c, static_scratch_ptr(&scratch), "cudaGetSymbolAddress(static scratch)");
  if (rc) return rc;
  k_constraints_blocks<<<c->g.nblk, K4_THREADS, 0, c->stream>>>(c->g, c->y, c->fd, c->sp, scratch);
  rc = check_launch(c, "k_constraints_blocks");
  if (rc) return rc;
  k_constraints_final<<<1, K4_THREADS, 0, c->stream>>>(scratch, c->g.nblk, (double)c->g.ncell, d_out);
  return check_launch(c, "k_constraints_final");
}

int z4c_sync(z4c_ctx* c) {
  if (!c) return Z4C_EINVAL;
  return read_flag(c);
}

int64_t z4c_launch_count(const z4c_ctx* c) { return c ? c->launches : 0; }

int z4c_set_variant(z4c_ctx* c, int variant) {
  if (!c || variant < 0 || variant > 1) return Z4C_EINVAL;
  if (variant != c->variant) drop_graph(c);
  c->variant = variant;
  return Z4C_OK;
}

int z4c_use_graph(z4c_ctx* c, int enable) {
  if (!c) return Z4C_EINVAL;
  c->use_graph = enable ? 1 : 0;
  if (!enable) drop_graph(c);
  return Z4C_OK;
}

int z4c_set_fused(z4c_ctx* c, int enable) {
  if (!c) return Z4C_EINVAL;
  if (enable < 0 || enable > 2) return Z4C_EINVAL;
  if (enable == 0 && partitioned(c))
    return fail(c, Z4C_EINVAL, "a slab of a partitioned mesh pushes its ghost images (modes 1, 2): mode 0 would pull mid-stage");
  if (enable != c->fuse_ghosts) drop_graph(c);
  c->fuse_ghosts = enable;
  return Z4C_OK;
}

int z4c_effective_mode(const z4c_ctx* c, int* variant, int* fused) {
  if (!c || !variant || !fused) return Z4C_EINVAL;
  const bool tuned = c->variant != 1 && c->have_ymap;
  *variant = tuned ? 0 : 1;
  *fused = fully_fused(c) ? 2 : (c->fuse_ghosts ? 1 : 0);
  return Z4C_OK;
}

double z4c_time(const z4c_ctx* c) { return c ? (double)c->steps * c->dt : 0.0; }
const char* z4c_last_error(const z4c_ctx* c) { return c ? c->err.c_str() : "null context"; }

void z4c_destroy(z4c_ctx* c) {
  if (!c) return;
  drop_graph(c);
  delete c;
}

}  // extern "C"
