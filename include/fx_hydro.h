/*
 * fx_hydro.h -- C ABI of libfxhydro: the batched block Euler update on one B200 (sm_100a).
 *
 * The operation: the unsplit finite-volume update of the compressible Euler equations over a batch
 * of fixed-size mesh blocks with guard cells, the block-by-block hot path of a Flash-X style run
 * [PAPER.md L69 section 2 "block-by-block update"; L71 "explicit methods ... strong shocks"; L103
 * section 2.2 Spark: "second- or third-order strong stability preserving (SSP) Runge-Kutta"; L105
 * "perfect-gas EOS"].  PAPER.md prints no formula; the discretisation is the one BASELINE.json's
 * north_star names, in the readings DESIGN.md lists (tags O1..O8, A1..A27 of SURVEY.md 8(c)).
 *
 * Conventions
 *  - All functions return int: FX_OK (0) or a negative FX_ERR_*; nothing aborts or throws across the
 *    ABI.  fx_last_error() returns a thread-local message for the last failure on this thread.
 *  - "dev" pointers are device (HBM) pointers, "host" pointers are host pointers.  Every device
 *    buffer is CALLER-OWNED (allocate it with PyTorch or cudaMalloc); the library never allocates
 *    device memory.  `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *  - Unless stated, a call only enqueues work on `stream` and returns without synchronising.
 *  - State layout [a0]: U[v][b][k][j][i], fp64, SoA with one contiguous slab per variable, i fastest:
 *        element(v,b,k,j,i) = v*S_v + b*S_b + k*S_k + j*S_j + i        (int64 arithmetic)
 *    v in (rho, m_x, m_y, m_z, E); padded extents np[d] = n[d] + 2*gd[d], gd[d] = nguard if n[d] > 1
 *    else 0 (a dimension of extent 1 is inactive: no guards, no sweep, no dt contribution [A26]);
 *    FX_OPT_GUARD_X may deepen gd[0] alone (a layout choice: wider row pitch, same results).
 *    Interior zone (i,j,k) has gd[0] <= i < gd[0]+n[0] etc.  Query strides with fx_hydro_plan_layout.
 */
#ifndef FX_HYDRO_H
#define FX_HYDRO_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FX_OK 0
#define FX_ERR_INVALID_ARG (-1)
#define FX_ERR_STATE (-2)       /* call order: topology or workspace not set */
#define FX_ERR_UNSUPPORTED (-3) /* coarse/fine neighbour relation, nvars > FX_MAX_NVARS, ... */
#define FX_MAX_NVARS 32     /* 5 hydro variables + at most 27 passive mass scalars [B11] */
#define FX_ERR_WORKSPACE (-4)   /* workspace missing, too small or not 256-byte aligned */
#define FX_ERR_CUDA (-5)        /* a CUDA runtime call or launch failed; see fx_last_error() */

enum { FX_RECON_PLM_MINMOD = 0, FX_RECON_WENO5 = 1 };
enum { FX_RIEMANN_HLLE = 0, FX_RIEMANN_HLLC = 1 };
enum { FX_BC_OUTFLOW = -1, FX_BC_NONE = -2, FX_BC_REFLECT = -3,        /* neighbour-table codes */
       FX_NEIGH_COARSER = -4, FX_NEIGH_FINER = -5 };                    /* refinement jumps, see fx_hydro_plan_set_refinement */
enum { FX_TOPO_PERIODIC = 0, FX_TOPO_OUTFLOW = 1, FX_TOPO_NONE = 2, FX_TOPO_REFLECT = 3 }; /* fx_topology_cartesian bc codes */
enum { FX_ORDER_LEX = 0, FX_ORDER_MORTON = 1 };
enum {
  FX_OPT_RHO_FLOOR = 0, /* primitive density floor, default 1e-12 [A7] */
  FX_OPT_P_FLOOR = 1,   /* primitive pressure floor, default 1e-12 [A7] */
  FX_OPT_WENO_EPS = 2,  /* WENO5-JS epsilon, default 1e-6 [A5].  Supported magnitudes: the kernels form the WENO5 weights with one
                           division (products of the smoothness indicators, ~ (difference)^9): differences of a primitive
                           between neighbouring zones must stay below ~1e33 in the units used, or the products overflow and
                           the positivity fallback takes the face (the oracle's quotient form only underflows there) */
  FX_OPT_WAVESPEED = 3, /* 0 = Einfeldt (default), 1 = Davis [A8] */
  FX_OPT_PATH = 4,      /* 0 = auto: the fused TMA stage kernel for 16 x 16 x nz blocks and for 8 x 8 x nz blocks whose topology
                           groups them completely into 2 x 2 bundles of mutual x / y neighbours (regular tilings with even
                           counts; no wall, gravity or passive scalar), else the shared-memory tile kernel
                           when the padded block fits a CTA's shared memory (8^3 blocks with WENO5, 2-D, 1-D), else
                           the generic zone kernel (also 3-D PLM blocks that would fit: it is the faster one there, measured);
                           1 = generic; 2 = tile kernel where it fits, else generic; 3 = the fused kernel's
                           two-zones-per-thread variant where it applies (PLM, no wall, no gravity; measured slower
                           than the default, kept for comparison), else as 0.
                           With refinement jumps (fx_hydro_plan_set_refinement): the generic kernel; under 0 and with 16 x 16 x nz
                           blocks the fused kernel (5): a block that HAS a jump face is marched alone, takes its halo behind
                           the jump from its own interpolated guard zones and stores the jump faces' fluxes for the correction.
                           fx_hydro_plan_path reports the choice (1 fused, 4 fused on bundles of 8 x 8 blocks, 3 the pair variant,
                           5 fused with refinement jumps, 2 tile, 0 generic). */
  FX_OPT_ZCHAIN = 5,    /* fused path: longest chain of z-neighbour blocks one CTA marches through, 1..8 (1..16 for 8 x 8 x nz
                           blocks; a larger value is clamped to what the kernel takes); 0 (default) =
                           chosen from the number of blocks and of SMs so that the launch still fills the GPU.
                           Set before fx_hydro_plan_set_topology.  Results do not depend on it (bit for bit). */
  FX_OPT_GRAVITY_X = 6, /* constant acceleration g_x (default 0): every stage adds beta dt (0, rho g, g.m) [B10] */
  FX_OPT_GRAVITY_Y = 7,
  FX_OPT_GRAVITY_Z = 8,
  FX_OPT_GUARD_X = 9,   /* guard depth of the x dimension alone, an integer in [nguard, nx] (default nguard).  CHANGES THE
                           LAYOUT (np[0], strides: query fx_hydro_plan_layout again); set it before workspace and
                           topology.  See "Layout and DRAM lines" below: 8 with nx = 16 makes the row pitch 256 bytes. */
  FX_OPT_OWNED_BLOCKS = 10 /* sharded runs [SURVEY 8(e)]: blocks [0, value) are advanced, blocks [value, nblocks) are
                           GHOST blocks -- copies of other ranks' blocks, read as halo sources and never written by a stage
                           (fx_shard_* builds the numbering).  Default nblocks.  Set before fx_hydro_plan_set_topology. */
};
enum {
  FX_STATUS_NONFINITE = 1u,
  FX_STATUS_RHO_FLOOR = 2u,
  FX_STATUS_P_FLOOR = 4u,
  FX_STATUS_WENO_FALLBACK = 8u
};

typedef struct fx_hydro_plan fx_hydro_plan;

typedef struct fx_layout {
  int32_t np[3];                 /* padded extents (x, y, z) */
  int32_t gd[3];                 /* guard depth per dimension */
  int64_t S_j, S_k, S_b, S_v;    /* element strides */
  int64_t bytes_per_state;       /* nvars * S_v * 8 */
} fx_layout;

/* Every compute call (fill, compute_dt, advance, advance_devdt, step) only enqueues kernels on `stream`: no host
 * synchronisation, no allocation, kernel arguments by value.  A loop of fx_hydro_step calls can therefore be captured
 * in a CUDA graph and replayed (tested; it removes a third of the step time of launch-bound small problems).
 * set_workspace, set_topology, status and the *_host calls synchronise. */

/* Thread-local text of the last error on the calling thread ("" if none). */
const char *fx_last_error(void);

/* Plan: a host object owned by the library, freed by fx_hydro_plan_destroy.
 * block_dims = interior zones (nx, ny, nz) per block; nvars = 5 + ns: (rho, m_x, m_y, m_z, E) [A1] followed by ns
 * passive mass scalars rho*X_s ("a perfect-gas EOS with a multispecies variant"; reading B11):
 * X_s = rho X_s / rho is reconstructed like the other primitives and gets from the Riemann solver the flux of an
 * advected quantity (for HLLC: the upwind X_s times the mass flux); no floor, no source term, not in the time step;
 * copied unchanged into guard zones (walls included).  Plans with ns > 0 run on the fused kernel followed by the scalar pass
 * (fx_hydro_plan_path = 1: the stage kernel leaves every face's mass flux and scalar coefficient, a second kernel advances the
 * scalars) where that applies -- 16 x 16 x nz blocks, PLM; physical boundaries, gravity, the ghost blocks of a sharded plan
 * and refinement jumps (then fx_hydro_plan_path = 5) included -- and on the generic path (0) otherwise;
 * recon FX_RECON_*; riemann FX_RIEMANN_*; rk_order 2 or 3 (SSP-RK).
 * FX_ERR_INVALID_ARG: a dim < 1; no active dim; nguard < 2 (PLM) or < 3 (WENO5); nguard > an active
 * block dim; gamma <= 1; nblocks < 0; unknown enum; nvars < 5.  FX_ERR_UNSUPPORTED: nvars > FX_MAX_NVARS. */
int fx_hydro_plan_create(fx_hydro_plan **out, const int block_dims[3], int nguard, int nvars, int64_t nblocks,
                         double gamma, int recon, int riemann, int rk_order);
int fx_hydro_plan_destroy(fx_hydro_plan *plan);

/* Strides and padded extents of the state array (pure).
 * Layout and DRAM lines: DRAM is read in whole 128-byte lines.  With nx = 16 and 4 guard zones an interior row is 128
 * bytes inside a 192-byte padded row, so reading the interior rows of a plane fetches the x guard columns as well
 * (1.5x the bytes).  With FX_OPT_GUARD_X = 8 the pitch is 256 bytes, and if the array is placed so that
 * U_dev + 8*gd[0] is a multiple of 128 every interior row is exactly one line (1.0x; measured).  Any 16-byte aligned
 * placement is correct; only the traffic differs.  The library places its own stage copies that way. */
int fx_hydro_plan_layout(const fx_hydro_plan *plan, fx_layout *out);

/* Options.  The physics options (floors, WENO epsilon, wave speeds, gravity) travel with every launch and may be changed
 * between calls; FX_OPT_GUARD_X before the workspace, FX_OPT_OWNED_BLOCKS, FX_OPT_ZCHAIN and FX_OPT_PATH before the topology
 * (FX_ERR_STATE afterwards).  Unknown key / bad value (a floor or the WENO epsilon <= 0 or non-finite,
 * wave speeds not 0 / 1, ...) -> FX_ERR_INVALID_ARG. */
int fx_hydro_plan_set_option(fx_hydro_plan *plan, int key, double value);

/* Workspace (device, caller-owned, 256-byte aligned): a 256-byte scratch block (dt reduction word,
 * status word and counters) + a 256-byte pad + (rk_order - 1) state copies for the RK stages + the z-segment table
 * (12 int32 per block, 19 for 8 x 8 x nz blocks; see FX_OPT_ZCHAIN); with a refinement table also the list of jump faces
 * (6 int32 per block) and the jump faces' flux buffer (6 faces x nvars x the largest face, per block); with passive scalars
 * on 16 x 16 x nz blocks and PLM also what the fused kernel hands the scalar pass (6 doubles per zone and 6 per zone of a
 * block face of 16 x max(nz, 16)).  fx_hydro_plan_workspace_bytes is the authority.  set_workspace initialises the scratch
 * block and synchronises the device once. */
size_t fx_hydro_plan_workspace_bytes(const fx_hydro_plan *plan);
int fx_hydro_plan_set_workspace(fx_hydro_plan *plan, void *workspace_dev, size_t bytes);

/* Topology: neigh_dev is int32 [nblocks][6] in the order -x,+x,-y,+y,-z,+z; an entry >= 0 is the id of
 * the same-level neighbour block (periodic boundaries are expressed by wrapped ids), FX_BC_OUTFLOW a
 * zero-gradient physical boundary, FX_BC_REFLECT a reflecting wall (guard zone -1-m images interior zone m
 * with the momentum normal to the wall negated; reading B9); entries of inactive dimensions are ignored.  The table stays
 * caller-owned and must outlive the plan's use of it.  The call copies it to the host once to validate
 * (synchronises).  FX_NEIGH_COARSER / FX_NEIGH_FINER mark a refinement jump and need fx_hydro_plan_set_refinement first
 * (FX_ERR_UNSUPPORTED without it, with passive scalars, or in a sharded plan); any other negative entry in an active
 * dimension: FX_ERR_UNSUPPORTED. */
int fx_hydro_plan_set_topology(fx_hydro_plan *plan, const int32_t *neigh_dev);

/* Fine-coarse boundaries ("fine-coarse boundary resolution related API functions of the Grid unit"; DESIGN.md
 * readings B12-B14).  Blocks of all levels have the same zone counts; a block one level finer has half the zone width (the
 * caller's dx_dev says so); face neighbours differ by at most one level.  jump_dev is int32 [nblocks][6][4], caller-owned:
 *   neigh[b][f] == FX_NEIGH_COARSER: jump[b][f][0] = the coarser block, jump[b][f][1] = which part of its face block b abuts:
 *     bit 0 = upper half along the first transverse dimension, bit 1 = along the second (transverse dimensions in
 *     ascending order; 0 for an inactive one);
 *   neigh[b][f] == FX_NEIGH_FINER: jump[b][f][q], q = that bit pattern, are the 2^(ndim-1) finer blocks behind the face.
 * What the library then does, per stage and in fx_fill_guardcells: the face guard zones behind a face with finer
 * neighbours are the RESTRICTION of their interiors (plain mean of the 2^ndim children); behind a face with a coarser
 * neighbour they are PROLONGED from the parent coarse zone C, q = q_C + sum_d sigma_d (1/4) minmod(q_C - q_{C-e_d},
 * q_{C+e_d} - q_C) on the conserved variables (children average to the parent; a neighbour of C that lies behind a coarser
 * jump gives slope 0); and the flux of a coarse face at a jump is replaced by the mean of the fine face fluxes that cover
 * it (FLUX CORRECTION: what leaves the fine blocks enters the coarse one).  Edge and corner guard zones next to a jump hold
 * a clamp (the stage reads none [A11]); fx_guardcell_index_map reports the clamp for zones behind a jump.  Plans with
 * jumps run on the generic path, or on the fused one where the block shape is its (FX_OPT_PATH).  Passive mass scalars
 * (nvars > 5) go through the jumps like the conserved variables they are -- restricted, prolonged, their fluxes corrected --
 * on either path.  Call before the workspace (which grows by the jump faces' flux buffer) and the
 * topology.  Needs even block extents and nguard <= n_d / 2 in active dimensions (FX_ERR_INVALID_ARG). */
int fx_hydro_plan_set_refinement(fx_hydro_plan *plan, const int32_t *jump_dev);

/* Host helper: neighbour table and block coordinates of a regular nb[0] x nb[1] x nb[2] tiling.
 * bc_lo/bc_hi per dimension: FX_TOPO_*; order FX_ORDER_LEX (x fastest) or FX_ORDER_MORTON.
 * neigh_out_host int32 [nblocks][6]; coords_out_host int32 [nblocks][3] (may be NULL). */
int fx_topology_cartesian(const int nb[3], const int bc_lo[3], const int bc_hi[3], int order,
                          int32_t *neigh_out_host, int32_t *coords_out_host);

/* a1 Guard-cell fill [O1, A14]: every guard zone (faces, edges, corners) of every block of U_dev, in
 * place, gets the 5 variables of the interior zone it images: hops z, then y, then x through the
 * neighbour table; outflow clamps to the nearest interior index, a reflecting wall mirrors the index and
 * negates the normal momentum.  Needs the topology (FX_ERR_STATE). */
int fx_fill_guardcells(fx_hydro_plan *plan, double *U_dev, void *stream);

/* Test hook: for blocks [block_begin, block_begin+block_count), the flat variable-0 element index each
 * padded zone is filled from (itself for interior zones): src_dev int64 [block_count][np2][np1][np0]. */
int fx_guardcell_index_map(fx_hydro_plan *plan, int64_t block_begin, int64_t block_count, int64_t *src_dev,
                           void *stream);

/* a7 CFL time step [O7, A13]: *dt_out_dev = cfl * min over blocks, interior zones and active d of
 * dx[b][d] / (|u_d| + c).  dx_dev is double [nblocks][3].  Reads interior zones only; writes +inf when
 * nblocks == 0.  A non-finite or non-positive signal speed sets FX_STATUS_NONFINITE.  Needs the
 * workspace (FX_ERR_STATE). */
int fx_hydro_compute_dt(fx_hydro_plan *plan, const double *U_dev, const double *dx_dev, double cfl,
                        double *dt_out_dev, void *stream);

/* fx_hydro_compute_dt for callers that may not allocate (code under CUDA graph capture, serving loops, harnesses that
 * forbid cudaMalloc) and so have no workspace: the same reduction [O7, A13] with its scratch -- one partial maximum per
 * owned block plus a 32-word header -- in a file-scope device array of the library, (32 + FX_STATIC_DT_MAX_BLOCKS) * 8 =
 * 524 544 bytes that every GPU loading the library holds until the process exits.  Needs only the plan (neither topology
 * nor workspace); U_dev, dx_dev, dt_out_dev as above, caller-owned; flags_out_dev (device uint32, may be NULL) receives
 * this call's FX_STATUS_* bits (they do NOT go to fx_hydro_status, whose words live in the workspace).  The result equals
 * fx_hydro_compute_dt's bit for bit (same per-zone arithmetic; a maximum has no order).  The call makes no cudaMalloc /
 * cudaFree and calls no allocating library routine; the first call on each device looks the array's address up
 * (cudaGetSymbolAddress), so make that one outside a capture.  More than FX_STATIC_DT_MAX_BLOCKS owned blocks ->
 * FX_ERR_UNSUPPORTED, nothing launched.  All calls on a device share the array, which keeps the last call's contents
 * (the header is cleared on `stream` before each launch): two calls that overlap on the GPU -- different streams with no
 * dependency between them -- RACE and both results are undefined. */
#define FX_STATIC_DT_MAX_BLOCKS 65536
int fx_hydro_compute_dt_static(fx_hydro_plan *plan, const double *U_dev, const double *dx_dev, double cfl,
                               double *dt_out_dev, uint32_t *flags_out_dev, void *stream);

/* a1..a6 One SSP-RK step [O5, O6], all stages, in place on the INTERIOR zones of U_dev:
 *   U1 = U0 - S(U0);  RK2: U = U0 + 1/2((U1-U0) - S(U1));
 *   RK3: U2 = U0 + 1/4((U1-U0) - S(U1)); U = U0 + 2/3((U2-U0) - S(U2));
 *   S(X) = sum_{d active} dt/dx[b][d] (F_{d,+} - F_{d,-}), fluxes from cons->prim (gamma law),
 *   PLM-minmod or WENO5-JS on primitives, HLLE or HLLC.
 * Guard zones of U_dev need not be valid on entry (the call fills or gathers halos of each stage input
 * itself) and are unspecified on exit [A15].  dt <= 0 or non-finite -> FX_ERR_INVALID_ARG.  Needs
 * topology and workspace (FX_ERR_STATE). */
int fx_hydro_advance(fx_hydro_plan *plan, double *U_dev, const double *dx_dev, double dt, void *stream);

/* End-to-end variant with HOST buffers: copies U_host (whole padded state) and dx_host to the device
 * staging buffers U_stage_dev / dx_stage_dev (caller-owned, bytes_per_state and nblocks*24 bytes), runs
 * `nsteps` steps of { compute_dt with `cfl`; advance } entirely on the device (dt never visits the
 * host), copies the state back into U_host and the last dt into *dt_last_host, and synchronises
 * `stream`.  Host buffers should be pinned for full PCIe speed. */
int fx_hydro_advance_host(fx_hydro_plan *plan, double *U_host, const double *dx_host, double cfl, int nsteps,
                          double *U_stage_dev, double *dx_stage_dev, double *dt_last_host, void *stream);

/* The same with the host holding INTERIOR zones only: Uint_host is double [5][nblocks][nz][ny][nx] (no guard zones:
 * they carry no information, and the padded state is 3.4x the bytes of a 16^3 block's interior).  The call copies it
 * to packed_stage_dev (same size, caller-owned), scatters it into the padded staging state U_stage_dev
 * (bytes_per_state, caller-owned; its guard zones need not be initialised), runs the steps as above, gathers the
 * interiors and copies them back into Uint_host.  PCIe carries interior bytes only, each way. */
int fx_hydro_advance_host_interior(fx_hydro_plan *plan, double *Uint_host, const double *dx_host, double cfl, int nsteps,
                                   double *U_stage_dev, double *packed_stage_dev, double *dx_stage_dev,
                                   double *dt_last_host, void *stream);

/* As fx_hydro_advance, but dt is read on the device from dt_dev (e.g. written by fx_hydro_compute_dt
 * on the same stream): no host round trip per step. */
int fx_hydro_advance_devdt(fx_hydro_plan *plan, double *U_dev, const double *dx_dev, const double *dt_dev,
                           void *stream);

/* The communication-avoiding form of the step [DESIGN.md B17; "fills guards once per step and updates a
 * shrinking guard region"]: ONE guard fill of U_dev (every guard zone, edges and corners: what fx_fill_guardcells does),
 * then stage s of n = rk_order on the interior extended by (n - s) R zones in every active dimension (R = 2 PLM, 3 WENO5),
 * stencils read in place; after every stage but the last, the extended zones behind a physical boundary (outflow, wall) are
 * re-imaged from the block's own zones (local; no neighbour is read after the fill).  The result on the interior equals
 * fx_hydro_advance's bit for bit on the generic path PROVIDED every block shares dx with its same-level neighbours (an
 * extended zone is then the neighbour's interior zone, updated with the same formula from the same numbers); guard zones
 * of U_dev hold the fill of the step's INPUT on exit.  dt: the host value, or read from dt_dev when that is not NULL.
 * What it buys is one exchange per step instead of one per stage where the fill is an exchange between devices; on one
 * GPU it costs a full fill and ((n_d + 2 (n - s) R) / n_d)^ndim times the zones in the early stages, on the generic
 * kernels (see DESIGN.md section 9 for the measured cost).  FX_ERR_UNSUPPORTED: nguard < rk_order x R (4 for RK2 + PLM,
 * 6 for RK3 + PLM or RK2 + WENO5, 9 for RK3 + WENO5), refinement jumps, passive scalars, a sharded plan.  Needs topology
 * and workspace (FX_ERR_STATE). */
int fx_hydro_advance_ca(fx_hydro_plan *plan, double *U_dev, const double *dx_dev, double dt, const double *dt_dev,
                        void *stream);

/* One step with the time step kept on the device and the next one formed on the way [O6 + O7]: advances U_dev by
 * *dt_inout_dev exactly as fx_hydro_advance_devdt does, and replaces *dt_inout_dev by cfl * min dx/(|u_d| + c) of
 * the ADVANCED state -- on the fused path the reduction rides in the last RK stage (each zone's rate is formed from
 * the values just computed, before they leave the SM), so a time loop is fx_hydro_compute_dt once, then one
 * fx_hydro_step per step with no separate reduction pass and no host round trip.  The value equals what
 * fx_hydro_compute_dt would return for the advanced state to rounding (a few ulp).  cfl <= 0 or non-finite ->
 * FX_ERR_INVALID_ARG.  Needs topology and workspace (FX_ERR_STATE). */
int fx_hydro_step(fx_hydro_plan *plan, double *U_dev, const double *dx_dev, double cfl, double *dt_inout_dev,
                  void *stream);

/* Status word and counters {non-finite, rho floor, p floor, WENO fallback} accumulated by all kernels
 * since the last reset; synchronises `stream`.  counts_host may be NULL. */
int fx_hydro_status(fx_hydro_plan *plan, uint32_t *flags_host, unsigned long long counts_host[4], void *stream);
int fx_hydro_status_reset(fx_hydro_plan *plan, void *stream);

/* Debug / per-kernel parity: face fluxes of direction dir (0,1,2) from U_dev whose guard zones are
 * already filled [A17]: F_dev[v][b][k][j][i], extents (nz, ny, nx) with n_dir + 1 along dir, i fastest;
 * face f lies between padded cells gd+f-1 and gd+f.  Not on the timed path. */
int fx_debug_compute_fluxes(fx_hydro_plan *plan, const double *U_dev, int dir, double *F_dev, void *stream);

/* ---- Sharded runs over several GPUs, one process per GPU [SURVEY.md 8(e); PAPER.md L75 (MPI between ranks), L69 (blocks
 * are independent within a stage once their boundaries are resolved)].  The library itself talks to no other process:
 * it provides the partition (host index logic), the owned/ghost split of a plan (FX_OPT_OWNED_BLOCKS), one RK stage at a
 * time, and the pack / unpack kernels of the face slabs; the caller moves the packed buffers between ranks (the Python
 * binding: torch.distributed all_to_all over NCCL) and takes the minimum of the ranks' time steps.
 *
 * Partition: rank r owns the contiguous run [N r / nranks, N (r+1) / nranks) of the global block order (Morton runs if
 * the table came from fx_topology_cartesian(..., FX_ORDER_MORTON)).  Local numbering: the owned blocks in global order,
 * then one ghost block per foreign block an owned block names, ascending global id.  neigh_global_host: the global table
 * [N][6] on the host, the same on every rank.  Items: (local block, side 0..5 = -x +x -y +y -z +z) = the slab of depth R
 * (2 PLM, 3 WENO5) of that block's INTERIOR behind that face, all variables, packed [v][k][j][i] over the slab's extents;
 * send items name owned blocks, receive items ghost blocks; both are grouped by peer rank (counts per peer) and ordered
 * by (global block id, side) inside a group, so that the two ends of an exchange agree without talking. */
typedef struct fx_shard fx_shard;
int fx_shard_create(fx_shard **out, int64_t nblocks_global, const int32_t *neigh_global_host, int nranks, int rank);
int fx_shard_destroy(fx_shard *shard);
int fx_shard_sizes(const fx_shard *shard, int64_t *owned_begin, int64_t *n_owned, int64_t *n_ghost, int64_t *n_send_items,
                   int64_t *n_recv_items);
/* neigh_local_host [n_owned + n_ghost][6] (ghost rows: FX_BC_OUTFLOW, never resolved by a stage), global_id_host [n_owned + n_ghost] */
int fx_shard_tables(const fx_shard *shard, int32_t *neigh_local_host, int64_t *global_id_host);
/* send_items_host [n_send][2], recv_items_host [n_recv][2] (either may be NULL), *_counts_host [nranks] */
int fx_shard_items(const fx_shard *shard, int32_t *send_items_host, int64_t *send_counts_host, int32_t *recv_items_host,
                   int64_t *recv_counts_host);
/* Elements (doubles) of one item on `side` for this plan: nvars x R x the two other extents (0 for an inactive dimension). */
int64_t fx_halo_item_elems(const fx_hydro_plan *plan, int side);
/* Gather the items' slabs of U into buf / scatter buf into the items' slabs of U.  items_dev int32 [n][2], offsets_dev int64
 * [n] (element offset of each item in buf); all device pointers, caller-owned; enqueue only. */
int fx_halo_pack(fx_hydro_plan *plan, const double *U, const int32_t *items_dev, const int64_t *offsets_dev, int64_t n, double *buf,
                 void *stream);
int fx_halo_unpack(fx_hydro_plan *plan, double *U, const int32_t *items_dev, const int64_t *offsets_dev, int64_t n, const double *buf,
                   void *stream);
/* One RK stage (stage = 0 .. rk_order - 1, to be called in order) of the step fx_hydro_advance takes [O6]: the caller acts
 * between stages (exchange of the ghost slabs of the stage's input).  dt_dev != NULL: dt is read on the device.  dt_next_dev
 * (last stage only, may be NULL): receives cfl_next times the CFL minimum over the OWNED blocks of the advanced state.
 * fx_hydro_stage_arrays: the array stage `stage` reads (whose ghosts must be current) and the one it writes -- U or a stage
 * copy inside the workspace. */
int fx_hydro_advance_stage(fx_hydro_plan *plan, double *U, const double *dx_dev, double dt, const double *dt_dev, int stage,
                           double cfl_next, double *dt_next_dev, void *stream);
int fx_hydro_stage_arrays(fx_hydro_plan *plan, double *U, int stage, double **stage_input, double **stage_output);
/* A stage in two parts, so that the exchange of the ghost slabs can overlap the part of the stage that does not need them
 * ("blocks are independent within a stage once halos are known"): FX_PART_INNER advances the
 * owned blocks none of whose faces (nor those of the blocks chained with them in z) has a ghost block behind it -- it reads
 * no ghost zone and may run while the slabs are under way --, FX_PART_BOUNDARY the others, once the ghosts are current.
 * Both parts of a stage, in either order or side by side on two streams, equal fx_hydro_advance_stage bit for bit; dt_next_dev is given to BOTH parts of
 * the last stage (the stage's last CTA finalises the reduction).  Only the fused kernel without passive scalars is split
 * (fx_hydro_plan_path = 1): on every other path FX_PART_INNER does nothing and FX_PART_BOUNDARY is the whole stage.
 * fx_hydro_plan_stage_parts: how many owned blocks each part advances (after the topology). */
enum { FX_PART_INNER = 1, FX_PART_BOUNDARY = 2 };
int fx_hydro_advance_stage_part(fx_hydro_plan *plan, double *U, const double *dx_dev, double dt, const double *dt_dev, int stage,
                                int part, double cfl_next, double *dt_next_dev, void *stream);
int fx_hydro_plan_stage_parts(const fx_hydro_plan *plan, int64_t *inner_blocks, int64_t *boundary_blocks);

/* Which stage kernel fx_hydro_advance will use for this plan: 0 generic (zone kernel that reads its halo cells through
 * the neighbour table; the only path for plans with passive scalars, whose face guard zones it fills first),
 * 1 fused and TMA-fed (16 x 16 x nz blocks: halos gathered from neighbour interiors inside the stage kernel,
 * every plane moved by TMA), 2 shared-memory tile kernel (one CTA per block whose padded zones fit its shared
 * memory: halos gathered through the neighbour table, each zone converted once, one Riemann solve per face),
 * 3 the fused kernel with two zones per thread (only on request, FX_OPT_PATH = 3), 4 the fused kernel marching 2 x 2
 * bundles of 8 x 8 x nz blocks as one 16 x 16 cross-section (csrc/fx_stage_bundle.cu). */
int fx_hydro_plan_path(const fx_hydro_plan *plan);

/* Measurement aid: when enabled, fx_hydro_advance brackets every stage-kernel launch (the dominant
 * kernel; excludes the guard fill of the generic path) with CUDA events on the launching stream (at most
 * 4096 launches are recorded between two reads).  get_timing synchronises the recorded events, returns
 * the summed kernel time in milliseconds and the number of launches, and clears the record. */
int fx_hydro_plan_set_timing(fx_hydro_plan *plan, int enable);
int fx_hydro_plan_get_timing(fx_hydro_plan *plan, double *stage_ms_sum_host, long long *stage_launches_host);

#ifdef __cplusplus
}
#endif
#endif /* FX_HYDRO_H */
