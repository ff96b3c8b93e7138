// fx_internal.h -- plan object and kernel parameter block of libfxhydro (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/fx_hydro.h"

// Parameter block passed by value to every kernel (a0: the block-layout manager's address map).
struct FxParams {
  int n[3];       // interior zones per block (x, y, z)
  int gd[3];      // guard depth per dimension (0 if inactive)
  int np[3];      // padded extents
  int active[3];
  int nvars;      // 5 hydro variables + passive mass scalars [B11]
  long long S_j, S_k, S_b, S_v;  // element strides of U[v][b][k][j][i]
  long long nblocks;
  long long nown;                   // blocks [0, nown) are advanced; [nown, nblocks) are ghost blocks of a shard: halo sources only
  double gamma, gm1, igm1;
  double rho_floor, p_floor, weno_eps;
  int recon, riemann, wavespeed;
  const int *neigh;                 // [nblocks][6], device
  const int *seg;                   // z-chain segments of the fused kernel: [nseg][FX_SEG_STRIDE], device (in the workspace)
  int nseg;
  int nseg_all;                     // segments of the whole stage (= nseg unless a launch covers a part of them: the fused CFL
                                    // reduction is finalised by the last CTA of the stage, whichever launch it belongs to)
  int nseg_inner;                   // sharded plans: the first nseg_inner segments touch no ghost block (fx_hydro_advance_stage_part)
  const int *bseg;                  // 8 x 8 blocks: segments of 2 x 2 BUNDLES, [nbseg][FX_BSEG_STRIDE] (same place in the workspace)
  int nbseg;
  int walls;                        // some block has a reflecting wall in an active dimension [B9]
  int grav_on;                      // any component of grav is non-zero [B10]
  double grav[3];
  double *fq;                       // scalar pass [B11]: mass flux and Aq of every zone's low x, y, z faces, [6][nblocks nz ny nx], in the workspace
  double *fqb;                      // the same for the HIGH face of a block that has no owned same-level block behind it (a physical
  int fqb_area;                     // boundary, a ghost block): [2 (F_rho, Aq)][3][nblocks][fqb_area], behind fq; the 17th face's solve
  int all_interior;                 // every active face of every owned block has a same-level neighbour (no physical boundary, no jump)
  const int *jump;                  // refinement jumps [B12]: [nblocks][6][4], device; nullptr if none was given
  int has_jumps;                    // some active face carries FX_NEIGH_COARSER / FX_NEIGH_FINER
  const int *jface;                 // the faces that carry a jump, as b * 6 + f, device (behind the segment tables in the workspace), or nullptr
  long long njface;
  int dt_defer;                     // fused AMR path, last stage: the stage kernel leaves the CFL maximum of the blocks the flux correction
                                    // does not touch in the scratch word; fx_launch_compute_dt_corrected adds the others and writes dt
  double *fjump;                    // boundary-face fluxes captured at jump faces [B14]: [nblocks][6][5][fj_area], in the workspace
  int fj_area;                      // largest face of a block, in zones
  long long njump;                  // fused AMR path (fx_hydro_plan_path = 5): how many blocks have a jump face (each a segment of its own)
  unsigned long long *scratch;      // device scratch block, see FX_SCR_*
};

// A segment = up to FX_SEG_MAX blocks that follow one another in +z (each the other's z neighbour both ways); one CTA
// of the fused stage kernel marches through a whole segment.  Row: {count, below, id_0 .. id_{count-1}, above}, where
// below / above are the z neighbours of the first / last block as the neighbour table gives them (id or FX_BC_OUTFLOW).
enum { FX_SEG_MAX = 8, FX_SEG_STRIDE = 12 };
// Bundle segments (fx_stage_bundle.cu): {count, 4 x (FX_BSEG_MAX + 2) block ids: the layer below (or each block's own boundary
// code), the count layers of 2 x 2 blocks (x half + 2 y half), the layer above}.  8-plane blocks: chains twice as long as the
// 16-plane blocks' keep the planes per pipeline fill the same.  One row per bundle at worst: 19 ints per block.
enum { FX_BSEG_MAX = 16, FX_BSEG_STRIDE = 76 };

// 64-bit words of the scratch block
enum {
  FX_SCR_DTBITS = 0,   // running max of (|u|+c)/dx as the bit pattern of a non-negative double
  FX_SCR_COUNTER = 1,  // CTAs finished in the dt reduction
  FX_SCR_FLAGS = 2,    // status bits
  FX_SCR_COUNT0 = 4,   // 4 counters: non-finite, rho floor, p floor, WENO fallback
  FX_SCR_WORDS = 32
};

struct fx_hydro_plan {
  FxParams P;
  int nguard, nvars, rk;
  int path_option;      // FX_OPT_PATH
  void *workspace;      // device
  size_t workspace_bytes;
  double *stage[2];     // RK stage copies inside the workspace
  bool topology_set;
  int zchain;           // FX_OPT_ZCHAIN: longest segment (1 .. FX_SEG_MAX)
  int32_t *jump_host;   // host copy of the refinement-jump table (new[]), or nullptr
  int *seg_host;        // segment table built by set_topology (new[]), nseg_host rows
  int *jlist_host;      // blocks with a jump face (fused AMR path), njump_host entries, or nullptr
  int *jface_host;      // faces with a jump (b * 6 + f), njface_host entries, or nullptr: the grids of fx_k_amr_fill / _flux_correct
  long long njface_host;
  long long njump_host;
  int *bseg_host;       // bundle segments (8 x 8 blocks whose topology bundles completely), nbseg_host rows, or nullptr
  int nbseg_host;
  int nseg_host;
  int nseg_inner_host;  // the leading segments none of whose blocks has a ghost block behind a face
  bool seg_uploaded;
  // optional per-launch timing of the stage kernels (fx_hydro_plan_set_timing)
  bool timing;
  cudaEvent_t *ev;  // 2 * FX_MAX_REC events, created on demand
  int nrec;
};
enum { FX_MAX_REC = 4096 };

// number of SMs of the current device (queried once per device; fx_api.cu)
int fx_sm_count();

// error plumbing (fx_api.cu)
int fx_fail(int code, const char *fmt, ...);
int fx_cuda_check(cudaError_t e, const char *what);
#define FX_CUDA(call)                                   \
  do {                                                  \
    int _rc = fx_cuda_check((call), #call);             \
    if (_rc) return _rc;                                \
  } while (0)
#define FX_LAUNCH_CHECK(name) FX_CUDA(cudaGetLastError())

// kernel launchers (one per .cu file); all enqueue on `st`
int fx_launch_fill_guardcells(const FxParams &P, double *U, cudaStream_t st);
// communication-avoiding step [B17]: a stage over the interior extended by `ext` zones (stencils in place); the re-imaging
// of the extended zones behind physical boundaries
int fx_launch_generic_stage_ca(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt,
                               const double *dt_dev, double beta, int first, int ext, cudaStream_t st);
int fx_launch_ca_refill(const FxParams &P, double *U, int ext, cudaStream_t st);
int fx_launch_fill_faces(const FxParams &P, double *U, int v0, cudaStream_t st);  // face guard zones of depth R, variables >= v0
int fx_launch_index_map(const FxParams &P, long long b0, long long nb, long long *src, cudaStream_t st);
int fx_launch_pack_interior(const FxParams &P, double *U, double *packed, int to_packed, cudaStream_t st);
int fx_launch_compute_dt(const FxParams &P, const double *U, const double *dx, double cfl, double *dt_out,
                         cudaStream_t st);
// the same over the owned blocks with a finer neighbour only (the blocks the flux correction changes), on top of the maximum
// a stage kernel launched with P.dt_defer left in the scratch word
int fx_launch_compute_dt_corrected(const FxParams &P, const double *U, const double *dx, double cfl, double *dt_out,
                                   cudaStream_t st);
int fx_launch_generic_stage(const FxParams &P, const double *X, const double *U0, double *out, const double *dx,
                            double dt, const double *dt_dev, double beta, int first, cudaStream_t st);
int fx_launch_debug_fluxes(const FxParams &P, const double *U, int dir, double *F, cudaStream_t st);
int fx_launch_amr_fill(const FxParams &P, double *U, int depth, cudaStream_t st);  // face guard zones behind refinement jumps
int fx_launch_amr_flux_correct(const FxParams &P, double *out, const double *dx, double dt, const double *dt_dev, double beta,
                               cudaStream_t st);
bool fx_stage_bundle_supported(const FxParams &P);
int fx_launch_stage_bundle(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt,
                           const double *dt_dev, double beta, int first, double cfl_next, double *dt_next, cudaStream_t st);
bool fx_scalar_pass_supported(const FxParams &P);
int fx_launch_scalar_pass(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt,
                          const double *dt_dev, double beta, int first, cudaStream_t st);
bool fx_stage_tma_supported(const FxParams &P);
bool fx_stage_pair_supported(const FxParams &P);  // the two-zones-per-thread variant: PLM, no wall, no gravity
bool fx_stage_tile_supported(const FxParams &P);
int fx_launch_stage_tile(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt,
                         const double *dt_dev, double beta, int first, cudaStream_t st);
int fx_launch_stage_pair(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt,
                         const double *dt_dev, double beta, int first, double cfl_next, double *dt_next, cudaStream_t st);
int fx_launch_stage_tma(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt,
                        const double *dt_dev, double beta, int first, double cfl_next, double *dt_next, cudaStream_t st);
