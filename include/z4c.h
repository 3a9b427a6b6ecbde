/* =====================================================================================
 * z4c.h -- C ABI of the B200-native Z4c hot path (arXiv 2409.10383, "Performance-Portable
 * Numerical Relativity with AthenaK").
 *
 * What the library computes: the fp64 Z4c right-hand side + classical RK4 step over ONE pack
 * of same-level MeshBlocks on one GPU.  The paper describes the pieces at
 *   PAPER.md:49-57  (section 2: Z4c formulation, Bona-Masso lapse, Gamma-driver shift; the
 *                    equations themselves are deferred to Daszuta et al. 2021 -- the reading
 *                    used here is written out in DESIGN.md / SURVEY.md section 8(c) O3-O7),
 *   PAPER.md:63-65  (section 3: Mesh -> MeshBlock -> MeshBlockPack, ghost zones refilled at
 *                    every Runge-Kutta stage),
 *   PAPER.md:75-76, 84 (section 3.1: same-level ghost fill from the neighbour's active region),
 *   PAPER.md:122-126 (section 3.2: cell-centred finite differences, order tied to ghost count),
 *   PAPER.md:203    (section 4.3: RK4, CFL 0.25, KO dissipation 0.5, kappa1 = 0.02, kappa2 = 0).
 *
 * Conventions
 *  - All functions return 0 (Z4C_OK) or a negative error code; they never throw or abort.
 *    A message for the last failing call on a context is available from z4c_last_error().
 *  - "device pointer" = CUDA device memory on the current device of the calling thread;
 *    "host pointer" = ordinary host memory. Every pointer argument says which it is.
 *  - Ownership: the CALLER owns the state buffer and the workspace buffer (e.g. torch tensors)
 *    and must keep them alive and unaliased until z4c_destroy(). The library owns only the
 *    host-side z4c_ctx and never allocates device memory.
 *  - Stream semantics: every call enqueues its work on the CUDA stream given to z4c_create()
 *    and returns without synchronising, except where stated ("synchronises").
 *  - Stream ordering of caller-owned DEVICE buffers (on_device = 1 arguments, d_percell, d_out, d_minchi ...):
 *    the library reads and writes them on ITS stream only and inserts no event against any other stream. A
 *    caller that produces or consumes such a buffer on another stream must order the two itself: make the
 *    library's stream wait for the producer before the call, and make the consumer wait for the library's
 *    stream (or call z4c_sync) after it. The Python binding does exactly this against torch's current stream.
 *  - Determinism: results are bitwise reproducible run to run (no atomics on the state path).
 *
 * State layout (part of the contract so a caller may view the buffer as a tensor):
 *    double y[22][N_b][m][m][m],  m = n + 2*ng,  x index fastest, block id
 *    b = (bz*nb[1] + by)*nb[0] + bx;  local cell (i,j,k) of block b has global cell index
 *    (bx*n + i - ng, ...).  Field order: 0 chi; 1-6 gt_xx,xy,xz,yy,yz,zz; 7 Khat;
 *    8-13 At_xx,xy,xz,yy,yz,zz; 14-16 Gamt^x,y,z; 17 Theta; 18 alpha; 19-21 beta^x,y,z
 *    (BASELINE.json north_star (a)).
 * "Interior array" = double[22][Nz][Ny][Nx] in GLOBAL, block-free cell order (x fastest),
 *    Nx = nb[0]*n etc.; cell centres x = xmin + (i + 1/2) dx.
 * ===================================================================================== */
#ifndef Z4C_H_
#define Z4C_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define Z4C_NFIELDS 22

enum {
  Z4C_OK = 0,
  Z4C_EINVAL = -1, /* bad argument / unsupported parameter */
  Z4C_ECUDA = -2,  /* a CUDA runtime call or kernel launch failed */
  Z4C_ESTATE = -3  /* device error flag set: non-finite value or det(gt) <= 0 seen by the stage update */
};

typedef struct z4c_ctx z4c_ctx; /* opaque, host memory, owned by the library */

typedef struct {
  int32_t n;      /* interior cells per MeshBlock edge (16, 32, 64 are the tuned sizes; any n >= 6 accepted) */
  int32_t ng;     /* ghost zones per side = stencil half-width, fixed per build: 3 in libz4c.so (4th order by the rule
                     at PAPER.md:124), 4 in libz4c_ng4.so (6th order); other values: Z4C_EINVAL */
  int32_t nb[3];  /* block lattice (x,y,z); N_b = nb[0]*nb[1]*nb[2] */
  int32_t bc;     /* 0 periodic; 1 outflow-copy: ghost = nearest interior cell, all six faces */
  double xmin[3]; /* lower corner of the domain */
  double dx;      /* cell size, same on all axes */
  double cfl;     /* dt = cfl*dx */
  double kappa1, kappa2;                             /* constraint damping */
  double lapse_oplog, lapse_harmonic, lapse_advect;  /* d_t a = -(oplog*a + harmonic*a^2) Khat + advect*b^k d_k a */
  double shift_gamma, shift_eta, shift_advect;       /* d_t b^i = gamma*Gamt^i - eta*b^i + advect*b^k d_k b^i */
  double ko_eps;                                     /* Kreiss-Oliger strength (0.5) */
  double chi_floor;                                  /* chi <- max(chi, chi_floor) in the stage update */
} z4c_params;

/* Bytes of the state buffer y: 22*N_b*m^3*8. Returns 0 if the parameters are invalid. */
size_t z4c_state_bytes(const z4c_params* p);

/* Bytes of the workspace (RK registers P and Q on interior cells, reduction scratch, error flag, the
 * second state buffer of the one-kernel-per-stage mode and a list of N_b block indices: about
 * 2*22*N_b*n^3*8 + 22*N_b*m^3*8).
 * Returns 0 if the parameters are invalid. */
size_t z4c_workspace_bytes(const z4c_params* p);

/* Create a context. p: host pointer (copied). d_state, d_work: device pointers of at least
 * z4c_state_bytes / z4c_workspace_bytes bytes, 256-byte aligned. cuda_stream: a cudaStream_t
 * passed as void* (NULL = legacy default stream). out: host pointer receiving the context.
 * Zero-fills the workspace (asynchronously). Errors: Z4C_EINVAL, Z4C_ECUDA. */
int z4c_create(const z4c_params* p, void* d_state, void* d_work, void* cuda_stream, z4c_ctx** out);

/* Load initial data. interior: an interior array; host pointer (on_device = 0; pageable or
 * pinned; the call synchronises) or device pointer (on_device = 1; async). The library never
 * allocates device memory, so host input is staged through the RK register area of the
 * workspace. The data are scattered into the pack, the algebraic constraints are enforced
 * (det gt = 1, tr At = 0, chi floor), ghosts are filled, time is reset to 0
 * and the RK registers are cleared. */
int z4c_set_initial_data(z4c_ctx* ctx, const double* interior, int on_device);

/* Advance nsteps classical RK4 steps: per stage  RHS -> stage update with
 * enforcement -> ghost fill.  Asynchronous on the context's stream; no host synchronisation. */
int z4c_step(z4c_ctx* ctx, int nsteps);

/* Constraint diagnostics on the current state (ghosts must be valid, which every call above
 * guarantees). out: host pointer to 8 doubles {H_rms, H_max, M_rms, M_max, Theta_rms,
 * Theta_max, Z_rms, Z_max} over interior cells. d_percell: NULL or device pointer to
 * double[4][Nz][Ny][Nx] receiving H, M_x, M_y, M_z. Synchronises the stream.
 * Returns Z4C_ESTATE if the device error flag is set. */
int z4c_constraints(z4c_ctx* ctx, double* out, double* d_percell);

/* The same eight norms WITHOUT touching any allocator and without synchronising: for callers that cannot allocate or
 * block (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc). Inputs: the context's
 * current state (ghosts valid). Output: d_out, DEVICE pointer to 8 doubles, same order as z4c_constraints, written
 * by the second of two kernels enqueued on the context's stream (asynchronous; no device error-flag read).
 * Scratch: one row of 8 partial norms per MeshBlock in a file-scope `static __device__` array of the library,
 * Z4C_STATIC_MAX_BLOCKS = 4096 rows = 256 KiB, which every GPU that loads the library holds until the process exits.
 * Its device address is looked up with cudaGetSymbolAddress on the first call on each device (the context's device
 * must be current, as for every call): make that first call outside graph capture. The call uses no cudaMalloc,
 * cudaFree or other allocating routine, and no part of the caller's workspace.
 * Limit: packs of more than 4096 MeshBlocks are refused with Z4C_EINVAL and a message (z4c_last_error); use
 * z4c_constraints for those.
 * Sharing: ALL calls on a device, from every context and stream, use the same array. It keeps the last call's rows;
 * every row a call reads it has written first (one CTA per MeshBlock writes its row unconditionally), so nothing has to
 * be cleared between calls. Two calls that OVERLAP on the GPU (different streams, or graphs replayed concurrently)
 * race on the rows and return garbage: order them on one stream or with events.
 * Numerics: the sums of squares are taken per MeshBlock and then over MeshBlocks in a fixed order (bitwise
 * reproducible from call to call); z4c_constraints groups the same terms differently, so the rms values agree with
 * it to rounding (a few ulp), the max values exactly. */
#define Z4C_STATIC_MAX_BLOCKS 4096
int z4c_constraints_static(z4c_ctx* ctx, double* d_out);

/* AMR refinement indicators per MeshBlock (sections 3.3.1-3.3.2; no regridding here): for every
 * block b, d_minchi[b] = min of chi and d_maxdchi[b] = max of |grad chi| (Euclidean norm of the scheme's centred first
 * derivative) over the block's interior cells, d_flags[b] = (min chi < chi_min ? 1 : 0) | (max |grad chi| > dchi_max ?
 * 2 : 0), i.e. bit 0 = the chi-min criterion, bit 1 = the d-chi-max criterion. All three outputs are device pointers
 * to N_b elements, each may be NULL (not all). Ghosts must be valid. Async. */
int z4c_refine_indicators(z4c_ctx* ctx, double chi_min, double dchi_max, double* d_minchi, double* d_maxdchi,
                          int32_t* d_flags);

/* --- NEXT-3: two-level static refinement (section 3.1) ------------------------------------------
 * Two contexts on ONE stream: `coarse` covers the whole mesh, `fine` is a pack whose blocks tile a box of the coarse
 * mesh at half the spacing (fine dx = coarse dx / 2, even n); origin[3] (host pointer) = global coarse cell index of
 * the box's lower corner. The operators are Lagrange interpolation, Eq. (1)-(2) with n = N_g + 1
 * nodes per axis and the outer product of the per-axis weights; all 22 fields are
 * interpolated as they are (no re-enforcement of det gt = 1 / tr At = 0 on interpolated values).
 *
 * z4c_restrict: step 1 of MeshBlock B's protocol: every coarse interior cell covered by the fine box <-
 *   interpolation of the fine ACTIVE cells; the stencil is the n nearest fine nodes, shifted so that it never leaves
 *   the active region of the fine block that owns the cell's children. The same kernel writes every
 *   ghost image of the cells it restricts (wrap / clamp rule of O2), which hands the new values to the coarse
 *   neighbours (steps A.2 / B.2): coarse ghosts that were current before the call are current after
 *   it. Async.
 * z4c_prolongate: step 5: every ghost cell of the fine pack that lies outside the fine box (faces, edges
 *   and corners) <- interpolation of the n^3 nearest coarse nodes, read from the coarse INTERIOR cells through the
 *   coarse level's own wrap / clamp rule. Fine ghosts inside the box are the same-level exchange's. Async.
 * z4c_two_level_step: nsteps RK4 steps of both levels with one dt (no subcycling: coarse cfl*dx must equal fine
 *   cfl*dx); after every stage: stage update with same-level ghost push on both packs, z4c_restrict, z4c_prolongate
 *   (and once on entry, so the levels are consistent whatever the caller loaded). The set-up of the paper's
 *   refined-corner wave test. With both contexts in mode 2 (z4c_set_fused) every stage is the fused
 *   stage kernel on each level followed by the two exchange kernels on the buffer just written (4 launches per stage);
 *   otherwise RHS, update + push per level, then the exchange (6 launches per stage). In mode 2, when the region is
 *   made of whole coarse MeshBlocks (the paper's refinement unit), the coarse blocks under it are not
 *   advanced at all (the restriction overwrites them) and between stages only the covered cells that are read --
 *   the N_g layers under the region's faces -- are restricted; the last stage of the call restricts every covered
 *   cell, so on return the coarse level is complete and equal to what the full sequence gives. The list of blocks
 *   to advance lives in the coarse context's workspace (N_b ints, counted by z4c_workspace_bytes). Async.
 * Errors: Z4C_EINVAL (different streams, spacing not 2:1, box outside the coarse mesh, odd n, unequal dt, a
 *   partitioned pack). */
int z4c_restrict(z4c_ctx* fine, z4c_ctx* coarse, const int32_t* origin);
int z4c_prolongate(z4c_ctx* coarse, z4c_ctx* fine, const int32_t* origin);
int z4c_two_level_step(z4c_ctx* coarse, z4c_ctx* fine, const int32_t* origin, int nsteps);

/* --- NEXT-2: one mesh partitioned over several packs / GPUs (the exchange: "at each
 * stage ... the ghost zones are filled by ... the active region of neighboring MeshBlocks", 75-76 "Pack and send") ----
 * The block lattice nb[0] x nb[1] x nbz_global of the whole mesh is cut into slabs along z; a context created with
 * nb[2] = the slab's thickness owns the blocks bz0 <= bz < bz0 + nb[2] (one process and one GPU per slab). There is no
 * pack / send / receive / unpack: the kernel that updates a cell writes that cell's ghost images straight into the
 * pack that holds them, its own or a z-neighbour's (peer memory over NVLink, mapped into this process by the caller,
 * e.g. through CUDA IPC), addressing three packs through one table. What remains of the exchange is a barrier between
 * stages, which is the caller's (a stream-ordered collective of torch.distributed; see partition.py).
 *
 * z4c_set_partition: declare the slab. bc and wrap / clamp then refer to the whole lattice. Switches mode 0 to 1.
 * z4c_set_neighbor: side 0 = the slab below (towards bz = 0; the top slab if periodic), 1 = the slab above.
 *   d_state, d_state2: DEVICE pointers, valid in this process, of that slab's state buffer and second state buffer
 *   (z4c_state2 of its context); bz0, nbz: its z-range. NULL, NULL = none on that side (outflow boundary). A slab
 *   may be its own neighbour (one slab, periodic) -- then no call is needed: entry 0 of the table covers it.
 * z4c_state2: device pointer of the context's second state buffer (lives in the workspace), to hand to neighbours.
 * z4c_stage: ONE Runge-Kutta stage (1..4) in the context's fuse mode, asynchronous. Between two stages every slab
 *   must have finished the previous one (barrier): stage s+1 reads ghosts its neighbours wrote in stage s, and writes
 *   ghosts into the buffer they read in stage s. Stage 4 advances the context's time. z4c_step refuses a slab.
 *   z4c_stage needs the one-kernel-per-stage mode (2), whose two state buffers make one barrier per stage enough. Where
 *   that mode is unavailable (odd n, variant 1) the state is updated in place and a stage is two calls with a barrier
 *   after each: z4c_stage_rhs (K2 into the RK register P), z4c_stage_update (K3 with ghost push; stage 4 advances time).
 * z4c_set_initial_data on a slab loads and enforces the slab's interior only; after a barrier every slab calls
 *   z4c_fill_ghosts (which pulls across slab faces), then another barrier.
 * z4c_constraints_raw: like z4c_constraints but the four sums of squares are NOT divided and rooted:
 *   out = {sum H^2, max|H|, sum |M|^2, max|M|, sum Theta^2, max|Theta|, sum |Z|^2, max|Z|} over this slab, so that the
 *   mesh-wide norms are one 8-double all-reduce away (SUM on even, MAX on odd entries). Synchronises the stream. */
/* z4c_enable_peer: lets kernels launched on the CURRENT device store into memory that lives on `peer_device`
 *   (cudaDeviceEnablePeerAccess; already-enabled access is not an error; the current device itself is accepted and
 *   needs nothing). Call it once per neighbour on another GPU before the first z4c_stage: opening a neighbour's
 *   buffers through CUDA IPC maps them, it does not by itself let this GPU's kernels reach them.
 *   Errors: Z4C_ECUDA (no such device, or the two GPUs cannot reach each other). */
int z4c_enable_peer(int32_t peer_device);
int z4c_set_partition(z4c_ctx* ctx, int32_t nbz_global, int32_t bz0);
int z4c_set_neighbor(z4c_ctx* ctx, int32_t side, void* d_state, void* d_state2, int32_t bz0, int32_t nbz);
void* z4c_state2(const z4c_ctx* ctx);
int z4c_stage(z4c_ctx* ctx, int stage);
int z4c_stage_rhs(z4c_ctx* ctx, int stage);
int z4c_stage_update(z4c_ctx* ctx, int stage);
int z4c_constraints_raw(z4c_ctx* ctx, double* out);

/* Inverse of z4c_set_initial_data: gather the interior cells of the pack into an interior
 * array. host pointer (on_device = 0; synchronises; staged through the workspace, so the RK
 * registers must not be live, i.e. not between stages -- always true between API calls) or
 * device pointer (on_device = 1; async). */
int z4c_get_interior(z4c_ctx* ctx, double* interior, int on_device);

/* --- single stages of the hot path, exported for unit parity tests and profiling ------- */
/* K1: refill every ghost cell of every block from the interior cell with the same global index
 * after periodic wrap / outflow clamp. Async. */
int z4c_fill_ghosts(z4c_ctx* ctx);
/* K2 with c = 0, dt = 1: evaluate F(y) + Q_KO(y) on interior cells and write it as an interior
 * array to d_out (device pointer). Overwrites RK register P. Async. */
int z4c_eval_rhs(z4c_ctx* ctx, double* d_out);
/* O7 enforcement alone on the interior cells of the pack, then ghost fill. Async. */
int z4c_enforce(z4c_ctx* ctx);

/* --- measurement aids (bench.py) -------------------------------------------------------- */
/* z4c_step with a CUDA event recorded on the context's stream between every pair of kernels.
 * ms_out: host pointer to 3 doubles receiving the summed device time in milliseconds of
 * {K2 RHS, K3 stage update (+ghost push), K1 ghost fill}. Synchronises. Never uses graph replay. */
int z4c_step_timed(z4c_ctx* ctx, int nsteps, double* ms_out);
/* FP64 pipe probe: runs a dependency-free DFMA loop on every SM of the current device (8 CTAs of 256
 * threads per SM, 8 chains per thread, `iters` iterations) and returns the achieved TFLOP/s (2 flop per
 * DFMA) in *tflops_out (host pointer). d_scratch: device pointer to >= 8 bytes. Synchronises. This is the
 * measured denominator of the "alu" roofline (MEASURED_PEAKS.json has no FP64 figure). */
int z4c_probe_fp64(void* cuda_stream, void* d_scratch, int iters, double* tflops_out);

/* Block until the stream is idle and report the device error flag (Z4C_ESTATE if set). */
int z4c_sync(z4c_ctx* ctx);

/* Number of kernel launches the library has enqueued on this context so far. */
int64_t z4c_launch_count(const z4c_ctx* ctx);
/* Select the RHS kernel variant: 0 = tuned kernel with TMA-staged shared-memory tiles (default); 1 = plain
 * global-memory kernel (the first correct kernel; also what runs when the tuned one is unavailable: odd n).
 * For A/B measurements; both compute the same values. Other values: Z4C_EINVAL. */
int z4c_set_variant(z4c_ctx* ctx, int variant);
/* Enable (1) / disable (0) CUDA-graph replay of the RK4 step inside z4c_step. Default 0. */
int z4c_use_graph(z4c_ctx* ctx, int enable);

/* How much of an RK stage runs in one kernel. mode 0: three launches per stage, K2 -> K3 -> K1.
 * mode 1: K2 -> K3 with "ghost push" (the thread that updates an interior cell also writes that cell's ghost
 * images in the neighbouring blocks; same values as K1, one pass less over the state).
 * mode 2 (default): ONE launch per stage -- the tuned K2 applies the RK recurrence, the enforcement and the
 * ghost push to each cell while its values are still in registers, reading the state from one buffer and
 * writing the next one to a second buffer kept in the workspace (4 stages: the caller's buffer is current
 * again at the end of every step). Falls back to mode 1 where the tuned K2 is unavailable (odd n, variant 1). */
int z4c_set_fused(z4c_ctx* ctx, int mode);

/* What actually runs, after fallbacks: *variant = 0 (tuned TMA kernel) or 1 (plain kernel: requested, or n is odd, or
 * the driver refused a tensor map); *fused = 0, 1 or 2 as in z4c_set_fused (2 needs the tuned kernel, else 1 runs).
 * Both are host pointers. bench.py reports these, and the GPU tests assert them, so that a silent fallback cannot
 * pass for the tuned path. */
int z4c_effective_mode(const z4c_ctx* ctx, int* variant, int* fused);

double z4c_time(const z4c_ctx* ctx);             /* simulation time = steps taken * dt */
const char* z4c_last_error(const z4c_ctx* ctx);  /* host string owned by the context ("" if none) */
void z4c_destroy(z4c_ctx* ctx);                  /* frees the host context only */

#ifdef __cplusplus
}
#endif
#endif /* Z4C_H_ */
