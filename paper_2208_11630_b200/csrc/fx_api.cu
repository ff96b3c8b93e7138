// fx_api.cu -- the C ABI of include/fx_hydro.h: plan / layout manager (a0), call sequencing of the RK
// stages, error plumbing.  Every entry point is extern "C"; nothing throws across the boundary.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <new>
#include <vector>

#include "fx_internal.h"

static thread_local char fx_errbuf[512] = "";

int fx_fail(int code, const char *fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(fx_errbuf, sizeof(fx_errbuf), fmt, ap);
  va_end(ap);
  return code;
}

int fx_cuda_check(cudaError_t e, const char *what) {
  if (e == cudaSuccess) return FX_OK;
  return fx_fail(FX_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

int fx_sm_count() {
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
    cudaGetLastError();
    return 148;  // no device visible (host-only use of the library): B200's count, used for sizing heuristics only
  }
  return sms;
}

extern "C" const char *fx_last_error(void) { return fx_errbuf; }

// ------------------------------------------------------------------ plan (a0)
// Padded extents and strides from the guard depths.
static int fx_relayout(fx_hydro_plan *p) {
  FxParams &P = p->P;
  for (int d = 0; d < 3; ++d) P.np[d] = P.n[d] + 2 * P.gd[d];
  P.S_j = P.np[0];
  P.S_k = (long long)P.np[0] * P.np[1];
  P.S_b = P.S_k * P.np[2];
  P.S_v = P.S_b * P.nblocks;
  return P.S_b > 2147483647LL ? -1 : 0;
}

extern "C" int fx_hydro_plan_create(fx_hydro_plan **out, const int block_dims[3], int nguard, int nvars,
                                    int64_t nblocks, double gamma, int recon, int riemann, int rk_order) {
  if (!out || !block_dims) return fx_fail(FX_ERR_INVALID_ARG, "plan_create: null argument");
  *out = nullptr;
  if (nvars < 5) return fx_fail(FX_ERR_INVALID_ARG, "plan_create: nvars must be at least 5 (rho, mx, my, mz, E), got %d", nvars);
  if (nvars > FX_MAX_NVARS)
    return fx_fail(FX_ERR_UNSUPPORTED, "plan_create: nvars = %d: at most %d passive scalars after the 5 hydro variables",
                   nvars, FX_MAX_NVARS - 5);
  if (nblocks < 0 || nblocks > 2147483647LL) return fx_fail(FX_ERR_INVALID_ARG, "plan_create: nblocks out of range");
  if (!(gamma > 1.0) || !isfinite(gamma)) return fx_fail(FX_ERR_INVALID_ARG, "plan_create: gamma must be > 1");
  if (recon != FX_RECON_PLM_MINMOD && recon != FX_RECON_WENO5) return fx_fail(FX_ERR_INVALID_ARG, "plan_create: unknown reconstruction %d", recon);
  if (riemann != FX_RIEMANN_HLLE && riemann != FX_RIEMANN_HLLC) return fx_fail(FX_ERR_INVALID_ARG, "plan_create: unknown Riemann solver %d", riemann);
  if (rk_order != 2 && rk_order != 3) return fx_fail(FX_ERR_INVALID_ARG, "plan_create: rk_order must be 2 or 3");
  const int need = recon == FX_RECON_WENO5 ? 3 : 2;
  if (nguard < need) return fx_fail(FX_ERR_INVALID_ARG, "plan_create: nguard %d < %d needed by the reconstruction", nguard, need);
  fx_hydro_plan *p = new (std::nothrow) fx_hydro_plan();
  if (!p) return fx_fail(FX_ERR_INVALID_ARG, "plan_create: out of host memory");
  memset(p, 0, sizeof(*p));
  FxParams &P = p->P;
  int nactive = 0;
  for (int d = 0; d < 3; ++d) {
    if (block_dims[d] < 1 || block_dims[d] > 4096) {
      delete p;
      return fx_fail(FX_ERR_INVALID_ARG, "plan_create: block_dims[%d] = %d out of range", d, block_dims[d]);
    }
    P.n[d] = block_dims[d];
    P.active[d] = block_dims[d] > 1;
    if (P.active[d]) {
      ++nactive;
      if (nguard > block_dims[d]) {
        delete p;
        return fx_fail(FX_ERR_INVALID_ARG, "plan_create: nguard %d exceeds block_dims[%d] = %d", nguard, d, block_dims[d]);
      }
    }
    P.gd[d] = P.active[d] ? nguard : 0;
  }
  if (nactive == 0) {
    delete p;
    return fx_fail(FX_ERR_INVALID_ARG, "plan_create: no active dimension");
  }
  P.nblocks = nblocks;
  P.nown = nblocks;
  if (fx_relayout(p)) {
    delete p;
    return fx_fail(FX_ERR_INVALID_ARG, "plan_create: padded block too large");
  }
  P.gamma = gamma;
  P.gm1 = gamma - 1.0;
  P.igm1 = 1.0 / (gamma - 1.0);
  P.rho_floor = 1e-12;
  P.p_floor = 1e-12;
  P.weno_eps = 1e-6;
  P.recon = recon;
  P.riemann = riemann;
  P.wavespeed = 0;
  p->zchain = 0;  // auto
  p->nguard = nguard;
  p->nvars = nvars;
  p->P.nvars = nvars;
  p->rk = rk_order;
  *out = p;
  return FX_OK;
}

extern "C" int fx_hydro_plan_destroy(fx_hydro_plan *plan) {
  if (plan) delete[] plan->seg_host;
  if (plan) delete[] plan->jump_host;
  if (plan) delete[] plan->bseg_host;
  if (plan) delete[] plan->jlist_host;
  if (plan) delete[] plan->jface_host;
  if (plan && plan->ev) {
    for (int i = 0; i < 2 * FX_MAX_REC; ++i) cudaEventDestroy(plan->ev[i]);
    delete[] plan->ev;
  }
  delete plan;
  return FX_OK;
}

extern "C" int fx_hydro_plan_layout(const fx_hydro_plan *plan, fx_layout *out) {
  if (!plan || !out) return fx_fail(FX_ERR_INVALID_ARG, "plan_layout: null argument");
  for (int d = 0; d < 3; ++d) {
    out->np[d] = plan->P.np[d];
    out->gd[d] = plan->P.gd[d];
  }
  out->S_j = plan->P.S_j;
  out->S_k = plan->P.S_k;
  out->S_b = plan->P.S_b;
  out->S_v = plan->P.S_v;
  out->bytes_per_state = plan->P.S_v * plan->nvars * (int64_t)sizeof(double);
  return FX_OK;
}

extern "C" int fx_hydro_plan_set_option(fx_hydro_plan *plan, int key, double value) {
  if (!plan) return fx_fail(FX_ERR_INVALID_ARG, "set_option: null plan");
  switch (key) {
  case FX_OPT_RHO_FLOOR:
  case FX_OPT_P_FLOOR:
    // a floor <= 0 or non-finite would let 1/rho or sqrt(p/rho) produce Inf/NaN where the floor is meant to prevent it
    if (!(value > 0.0) || !isfinite(value)) return fx_fail(FX_ERR_INVALID_ARG, "set_option: a floor must be positive and finite");
    if (key == FX_OPT_RHO_FLOOR) plan->P.rho_floor = value; else plan->P.p_floor = value;
    return FX_OK;
  case FX_OPT_WENO_EPS:
    if (!(value > 0.0)) return fx_fail(FX_ERR_INVALID_ARG, "set_option: WENO eps must be > 0");
    plan->P.weno_eps = value;
    return FX_OK;
  case FX_OPT_WAVESPEED:
    if (value != 0.0 && value != 1.0) return fx_fail(FX_ERR_INVALID_ARG, "set_option: wavespeed must be 0 or 1");
    plan->P.wavespeed = (int)value;
    return FX_OK;
  case FX_OPT_GRAVITY_X:
  case FX_OPT_GRAVITY_Y:
  case FX_OPT_GRAVITY_Z:
    if (!(value == value) || value > 1e300 || value < -1e300) return fx_fail(FX_ERR_INVALID_ARG, "set_option: gravity must be finite");
    plan->P.grav[key - FX_OPT_GRAVITY_X] = value;
    plan->P.grav_on = plan->P.grav[0] != 0.0 || plan->P.grav[1] != 0.0 || plan->P.grav[2] != 0.0;
    return FX_OK;
  case FX_OPT_GUARD_X: {
    if (plan->workspace || plan->topology_set)
      return fx_fail(FX_ERR_STATE, "set_option: the x guard depth changes the layout and must be set before workspace and topology");
    const int g = (int)value;
    if (!plan->P.active[0] || (double)g != value || g < plan->nguard || g > plan->P.n[0])
      return fx_fail(FX_ERR_INVALID_ARG, "set_option: x guard depth must be an integer in [nguard, nx] of an active x dimension");
    const int old = plan->P.gd[0];
    plan->P.gd[0] = g;
    if (fx_relayout(plan)) {
      plan->P.gd[0] = old;
      fx_relayout(plan);
      return fx_fail(FX_ERR_INVALID_ARG, "set_option: padded block too large");
    }
    return FX_OK;
  }
  case FX_OPT_ZCHAIN:
    if (!(value >= 0.0 && value <= (double)FX_BSEG_MAX)) return fx_fail(FX_ERR_INVALID_ARG, "set_option: zchain must be 0 (auto) or 1..%d", (int)FX_BSEG_MAX);
    if (plan->topology_set) return fx_fail(FX_ERR_STATE, "set_option: FX_OPT_ZCHAIN must be set before the topology (the chains are built there)");
    plan->zchain = (int)value;
    return FX_OK;
  case FX_OPT_OWNED_BLOCKS:
    if (!(value >= 0.0 && value <= (double)plan->P.nblocks) || value != floor(value))
      return fx_fail(FX_ERR_INVALID_ARG, "set_option: owned blocks must be an integer in [0, nblocks]");
    if (plan->topology_set) return fx_fail(FX_ERR_STATE, "set_option: FX_OPT_OWNED_BLOCKS must be set before the topology");
    plan->P.nown = (long long)value;
    return FX_OK;
  case FX_OPT_PATH:
    if (value != 0.0 && value != 1.0 && value != 2.0 && value != 3.0) return fx_fail(FX_ERR_INVALID_ARG, "set_option: path must be 0, 1, 2 or 3");
    if (plan->topology_set) return fx_fail(FX_ERR_STATE, "set_option: FX_OPT_PATH must be set before the topology (the path's tables are built there)");
    plan->path_option = (int)value;
    return FX_OK;
  default: return fx_fail(FX_ERR_INVALID_ARG, "set_option: unknown key %d", key);
  }
}

extern "C" int fx_hydro_plan_path(const fx_hydro_plan *plan) {
  if (!plan) return fx_fail(FX_ERR_INVALID_ARG, "plan_path: null plan");
  if (plan->P.has_jumps) {
    // refinement jumps [B12-B14]: the generic kernel reads the interpolated guard zones.  Where the fused kernel takes the
    // block shape (5), it advances every block: those WITH a jump face as segments of their own, their halo boxes behind a
    // jump taken from their own guard zones and the jump faces' fluxes stored for the correction
    return (plan->jlist_host && fx_stage_tma_supported(plan->P) && (plan->nvars == 5 || fx_scalar_pass_supported(plan->P))) ? 5 : 0;
  }
  // passive scalars [B11]: behind the fused kernel by the scalar pass where it applies (PLM, same-level neighbours
  // everywhere, no gravity), else on the generic path
  if (plan->nvars > 5 && !(plan->path_option == 0 && fx_stage_tma_supported(plan->P) && fx_scalar_pass_supported(plan->P))) return 0;
  if (plan->path_option == 0 && fx_stage_bundle_supported(plan->P)) return 4;  // 8 x 8 blocks in 2 x 2 bundles
  if ((plan->path_option == 0 || plan->path_option == 3) && fx_stage_tma_supported(plan->P))
    return (plan->path_option == 3 && fx_stage_pair_supported(plan->P)) ? 3 : 1;
  // 3-D blocks with PLM: the generic zone kernel, which gathers its halo cells itself, is ahead of the tile kernel
  // (8^3 blocks: 34.6 against 41.2 ms per step, measured); FX_OPT_PATH = 2 still selects the tile kernel
  const bool generic_ahead = plan->path_option == 0 && plan->P.active[0] && plan->P.active[1] && plan->P.active[2] &&
                             plan->P.recon == FX_RECON_PLM_MINMOD;
  if (plan->path_option != 1 && plan->path_option != 3 && !generic_ahead && fx_stage_tile_supported(plan->P)) return 2;
  return 0;
}

static size_t fx_state_bytes_aligned(const fx_hydro_plan *plan) {
  size_t b = (size_t)plan->P.S_v * plan->nvars * sizeof(double);
  return (b + 255) & ~(size_t)255;
}

static size_t fx_seg_ints(const fx_hydro_plan *plan) {  // room for one segment per block, or one bundle segment per four 8 x 8 blocks
  const FxParams &P = plan->P;
  size_t ints = (size_t)P.nblocks * FX_SEG_STRIDE;
  if (P.n[0] == 8 && P.n[1] == 8) {
    const size_t b = ((size_t)P.nblocks / 4 + 1) * FX_BSEG_STRIDE;
    if (b > ints) ints = b;
  }
  return ints;
}

static size_t fx_seg_bytes(const fx_hydro_plan *plan) {  // the segment tables and, with a refinement table, the list of jump faces
  const size_t ints = fx_seg_ints(plan) + (plan->P.jump ? (size_t)plan->P.nblocks * 6 : 0);
  return ((ints * sizeof(int)) + 255) & ~(size_t)255;
}

static size_t fx_fq_bytes(const fx_hydro_plan *plan) {  // scalar pass [B11]: (mass flux, Aq) x 3 low faces per interior zone
  const FxParams &P = plan->P;
  if (plan->nvars <= 5 || P.recon != FX_RECON_PLM_MINMOD || P.n[0] != 16 || P.n[1] != 16 || !P.active[2]) return 0;
  // + the high faces of the blocks at a physical boundary or a cut: (mass flux, Aq) x 3 directions x a face of 16 x max(nz, 16) zones
  const size_t area = (size_t)16 * (P.n[2] > 16 ? P.n[2] : 16);
  return (((size_t)6 * P.nblocks * (P.n[0] * P.n[1] * P.n[2] + area) * sizeof(double)) + 255) & ~(size_t)255;
}

static size_t fx_fjump_bytes(const fx_hydro_plan *plan) {  // boundary fluxes at refinement jumps [B14]
  if (!plan->P.jump) return 0;
  return (((size_t)plan->P.nblocks * 6 * (size_t)plan->nvars * (size_t)plan->P.fj_area * sizeof(double)) + 255) & ~(size_t)255;
}

// The stage copies start `fx_stage_pad` bytes into a 256-byte pad block, so that their interior rows start on a
// 128-byte boundary like the caller's array should (include/fx_hydro.h, "Layout and DRAM lines").
static size_t fx_stage_pad(const fx_hydro_plan *plan) { return (128 - ((size_t)plan->P.gd[0] * 8) % 128) % 128; }

extern "C" size_t fx_hydro_plan_workspace_bytes(const fx_hydro_plan *plan) {
  if (!plan) return 0;
  return (size_t)FX_SCR_WORDS * 8 + 256 + (size_t)(plan->rk - 1) * fx_state_bytes_aligned(plan) + fx_seg_bytes(plan) + fx_fjump_bytes(plan) + fx_fq_bytes(plan);
}

// Upload the segment table into its place behind the stage copies (needs both the workspace and the topology).
static int fx_seg_upload(fx_hydro_plan *plan) {
  if (!plan->workspace || !plan->seg_host) return FX_OK;
  int *dst = (int *)((char *)plan->workspace + FX_SCR_WORDS * 8 + 256 + (size_t)(plan->rk - 1) * fx_state_bytes_aligned(plan));
  if (plan->nseg_host > 0)
    FX_CUDA(cudaMemcpy(dst, plan->seg_host, (size_t)plan->nseg_host * FX_SEG_STRIDE * sizeof(int), cudaMemcpyHostToDevice));
  plan->P.seg = dst;
  plan->P.nseg = plan->nseg_host;
  plan->P.nseg_all = plan->nseg_host;
  plan->P.nseg_inner = plan->nseg_inner_host;
  plan->P.bseg = nullptr;
  plan->P.nbseg = 0;
  plan->P.njump = plan->jlist_host ? plan->njump_host : 0;  // (fused AMR path: the blocks with a jump face are single-block segments)
  plan->P.jface = nullptr;
  plan->P.njface = 0;
  if (plan->jface_host && plan->P.jump && plan->njface_host > 0) {
    int *jf = dst + fx_seg_ints(plan);
    FX_CUDA(cudaMemcpy(jf, plan->jface_host, (size_t)plan->njface_host * sizeof(int), cudaMemcpyHostToDevice));
    plan->P.jface = jf;
    plan->P.njface = plan->njface_host;
  }
  if (plan->bseg_host && plan->nbseg_host > 0) {  // bundle segments take the place of the (unused: blocks are not 16 wide) block segments
    FX_CUDA(cudaMemcpy(dst, plan->bseg_host, (size_t)plan->nbseg_host * FX_BSEG_STRIDE * sizeof(int), cudaMemcpyHostToDevice));
    plan->P.bseg = dst;
    plan->P.nbseg = plan->nbseg_host;
    plan->P.seg = nullptr;
    plan->P.nseg = 0;
    plan->P.nseg_all = 0;
    plan->P.nseg_inner = 0;
  }
  plan->seg_uploaded = true;
  return FX_OK;
}

extern "C" int fx_hydro_plan_set_workspace(fx_hydro_plan *plan, void *ws, size_t bytes) {
  if (!plan) return fx_fail(FX_ERR_INVALID_ARG, "set_workspace: null plan");
  if (!ws || ((uintptr_t)ws & 255) != 0) return fx_fail(FX_ERR_WORKSPACE, "set_workspace: workspace null or not 256-byte aligned");
  if (bytes < fx_hydro_plan_workspace_bytes(plan))
    return fx_fail(FX_ERR_WORKSPACE, "set_workspace: %zu bytes given, %zu needed", bytes, fx_hydro_plan_workspace_bytes(plan));
  unsigned long long init[FX_SCR_WORDS];
  memset(init, 0, sizeof(init));
  init[FX_SCR_DTBITS] = 0ull;  // running max of (|u|+c)/dx: 0
  FX_CUDA(cudaMemcpy(ws, init, sizeof(init), cudaMemcpyHostToDevice));
  FX_CUDA(cudaDeviceSynchronize());
  plan->workspace = ws;
  plan->workspace_bytes = bytes;
  plan->P.scratch = (unsigned long long *)ws;
  char *base = (char *)ws + FX_SCR_WORDS * 8 + fx_stage_pad(plan);
  plan->stage[0] = (double *)base;
  plan->stage[1] = plan->rk == 3 ? (double *)(base + fx_state_bytes_aligned(plan)) : nullptr;
  plan->P.fjump = plan->P.jump ? (double *)((char *)ws + FX_SCR_WORDS * 8 + 256 + (size_t)(plan->rk - 1) * fx_state_bytes_aligned(plan) +
                                            fx_seg_bytes(plan))
                               : nullptr;
  plan->P.fq = fx_fq_bytes(plan) ? (double *)((char *)ws + FX_SCR_WORDS * 8 + 256 + (size_t)(plan->rk - 1) * fx_state_bytes_aligned(plan) +
                                              fx_seg_bytes(plan) + fx_fjump_bytes(plan))
                                 : nullptr;
  plan->P.fqb_area = 16 * (plan->P.n[2] > 16 ? plan->P.n[2] : 16);
  plan->P.fqb = plan->P.fq ? plan->P.fq + (size_t)6 * plan->P.nblocks * plan->P.n[0] * plan->P.n[1] * plan->P.n[2] : nullptr;
  return fx_seg_upload(plan);
}

// ------------------------------------------------------------------ bundles of 2 x 2 blocks (fx_stage_bundle.cu)
// Blocks of 8 x 8 x nz zones: group them into bundles {b00, b10, b01, b11} that name each other as x / y neighbours (every
// link mutual), then chain bundles whose four blocks lie above each other's.  Succeeds only if EVERY owned block finds its
// bundle (regular tilings with even counts do, in lexicographic and Morton order: the lowest unbundled id sits at even
// coordinates); otherwise the plan keeps the tile / generic path.  h: host copy of the neighbour table.
static int fx_build_bundles(fx_hydro_plan *plan, const std::vector<int32_t> &h) {
  delete[] plan->bseg_host;
  plan->bseg_host = nullptr;
  plan->nbseg_host = 0;
  const FxParams &P = plan->P;
  const long long nown = P.nown;
  if (P.n[0] != 8 || P.n[1] != 8 || !P.active[0] || !P.active[1] || !P.active[2] || nown < 4 || nown % 4 != 0 || P.n[2] > 64) return FX_OK;
  auto nbr = [&](long long b, int f) -> long long { const long long v = h[b * 6 + f]; return (v >= 0 && v < nown) ? v : -1; };
  std::vector<int> bundle_of((size_t)nown, -1);
  std::vector<int> ids;  // 4 per bundle
  for (long long b = 0; b < nown; ++b) {
    if (bundle_of[b] >= 0) continue;
    const long long b10 = nbr(b, 1), b01 = nbr(b, 3);
    if (b10 < 0 || b01 < 0) return FX_OK;
    const long long b11 = nbr(b10, 3);
    if (b11 < 0 || nbr(b01, 1) != b11 || nbr(b10, 0) != b || nbr(b01, 2) != b || nbr(b11, 0) != b01 || nbr(b11, 2) != b10) return FX_OK;
    const long long q[4] = {b, b10, b01, b11};
    for (int x = 0; x < 4; ++x)
      for (int y = x + 1; y < 4; ++y)
        if (q[x] == q[y]) return FX_OK;  // a periodic direction one block wide
    for (int x = 0; x < 4; ++x) {
      if (bundle_of[q[x]] >= 0) return FX_OK;
      bundle_of[q[x]] = (int)(ids.size() / 4);
    }
    for (int x = 0; x < 4; ++x) ids.push_back((int)q[x]);
  }
  const int nbun = (int)(ids.size() / 4);
  // the bundle above / below: all four blocks' z links lead, mutually, to the four blocks of one bundle in the same places
  auto zlink = [&](int B, int f) -> int {
    int T = -1;
    for (int x = 0; x < 4; ++x) {
      const long long t = nbr(ids[4 * B + x], f);
      if (t < 0 || nbr(t, f ^ 1) != ids[4 * B + x]) return -1;
      const int tb = bundle_of[t];
      if (ids[4 * tb + x] != t || (T >= 0 && tb != T) || tb == B) return -1;
      T = tb;
    }
    return T;
  };
  int M = plan->zchain > FX_BSEG_MAX ? FX_BSEG_MAX : plan->zchain;
  if (M <= 0) {
    const long long slots = (long long)fx_sm_count() * (P.recon == FX_RECON_WENO5 ? 1 : 2);
    double best = 0.0;
    for (int m = 1; m <= FX_BSEG_MAX; m *= 2) {
      const long long nseg = (nbun + m - 1) / m;
      const double cost = (double)((nseg + slots - 1) / slots) * (m + 0.09);
      if (M <= 0 || cost < best) {
        best = cost;
        M = m;
      }
    }
  }
  plan->bseg_host = new (std::nothrow) int[(size_t)nbun * FX_BSEG_STRIDE];
  if (!plan->bseg_host) return fx_fail(FX_ERR_INVALID_ARG, "set_topology: out of host memory");
  std::vector<char> seen((size_t)nbun, 0);
  for (int B0 = 0; B0 < nbun; ++B0) {
    if (seen[B0]) continue;
    int start = B0;
    for (int steps = 0; steps < nbun; ++steps) {
      const int d = zlink(start, 4);
      if (d < 0 || seen[d] || d == B0) break;
      start = d;
    }
    int B = start;
    while (B >= 0 && !seen[B]) {
      int *row = plan->bseg_host + (size_t)plan->nbseg_host * FX_BSEG_STRIDE;
      for (int x = 0; x < FX_BSEG_STRIDE; ++x) row[x] = FX_BC_OUTFLOW;
      int cnt = 0, last = B;
      for (int x = 0; x < 4; ++x) row[1 + x] = h[(long long)ids[4 * B + x] * 6 + 4];  // below: each block's own -z entry
      while (B >= 0 && !seen[B] && cnt < M) {
        seen[B] = 1;
        for (int x = 0; x < 4; ++x) row[1 + 4 * (1 + cnt) + x] = ids[4 * B + x];
        ++cnt;
        last = B;
        B = zlink(B, 5);
      }
      row[0] = cnt;
      for (int x = 0; x < 4; ++x) row[1 + 4 * (1 + cnt) + x] = h[(long long)ids[4 * last + x] * 6 + 5];  // above
      ++plan->nbseg_host;
    }
  }
  return FX_OK;
}

// ------------------------------------------------------------------ topology
// Refinement-jump table [B12]: see include/fx_hydro.h.  A host copy is kept for the validation of the neighbour table.
extern "C" int fx_hydro_plan_set_refinement(fx_hydro_plan *plan, const int32_t *jump_dev) {
  if (!plan) return fx_fail(FX_ERR_INVALID_ARG, "set_refinement: null plan");
  if (plan->topology_set || plan->workspace) return fx_fail(FX_ERR_STATE, "set_refinement: call before the workspace and the topology");
  for (int d = 0; d < 3; ++d)
    if (plan->P.active[d] && (plan->P.n[d] % 2 != 0 || 2 * plan->nguard > plan->P.n[d]))
      return fx_fail(FX_ERR_INVALID_ARG, "set_refinement: needs even block extents and nguard <= n_d / 2 in every active dimension");
  delete[] plan->jump_host;
  plan->jump_host = nullptr;
  plan->P.jump = nullptr;
  if (!jump_dev) return FX_OK;
  const size_t n = (size_t)plan->P.nblocks * 24;
  plan->jump_host = new (std::nothrow) int32_t[n ? n : 1];
  if (!plan->jump_host) return fx_fail(FX_ERR_INVALID_ARG, "set_refinement: out of host memory");
  FX_CUDA(cudaMemcpy(plan->jump_host, jump_dev, n * sizeof(int32_t), cudaMemcpyDeviceToHost));
  plan->P.jump = jump_dev;
  int a = 1;
  for (int d = 0; d < 3; ++d) {
    int f = 1;
    for (int e = 0; e < 3; ++e)
      if (e != d) f *= plan->P.n[e];
    if (f > a) a = f;
  }
  plan->P.fj_area = a;
  return FX_OK;
}

extern "C" int fx_hydro_plan_set_topology(fx_hydro_plan *plan, const int32_t *neigh_dev) {
  if (!plan) return fx_fail(FX_ERR_INVALID_ARG, "set_topology: null plan");
  const long long nb = plan->P.nblocks;
  int jumps = 0, all_interior = 1;
  delete[] plan->jface_host;
  plan->jface_host = nullptr;
  plan->njface_host = 0;
  if (nb > 0) {
    if (!neigh_dev) return fx_fail(FX_ERR_INVALID_ARG, "set_topology: null table");
    std::vector<int32_t> h((size_t)nb * 6);
    FX_CUDA(cudaMemcpy(h.data(), neigh_dev, h.size() * sizeof(int32_t), cudaMemcpyDeviceToHost));
    for (long long b = 0; b < nb; ++b)
      for (int f = 0; f < 6; ++f) {
        if (!plan->P.active[f / 2]) continue;
        const int32_t v = h[b * 6 + f];
        if (v < 0 && b < plan->P.nown) all_interior = 0;
        if (v >= 0) {
          if (v >= nb) return fx_fail(FX_ERR_INVALID_ARG, "set_topology: block %lld face %d -> id %d out of range", b, f, v);
        } else if (v == FX_NEIGH_COARSER || v == FX_NEIGH_FINER) {
          if (!plan->jump_host) return fx_fail(FX_ERR_UNSUPPORTED, "set_topology: block %lld face %d is a refinement jump: call fx_hydro_plan_set_refinement first", b, f);
          if (plan->P.nown != nb) return fx_fail(FX_ERR_UNSUPPORTED, "set_topology: refinement jumps in a sharded plan are not supported");
          const int nq = v == FX_NEIGH_COARSER ? 1 : (1 << (plan->P.active[0] + plan->P.active[1] + plan->P.active[2] - 1));
          for (int q = 0; q < nq; ++q) {
            const int32_t id = plan->jump_host[(b * 6 + f) * 4 + q];
            if (id < 0 || id >= nb) return fx_fail(FX_ERR_INVALID_ARG, "set_topology: block %lld face %d: jump entry %d = %d out of range", b, f, q, id);
          }
          jumps = 1;
          if (!plan->jface_host) {
            plan->jface_host = new (std::nothrow) int[(size_t)nb * 6];
            if (!plan->jface_host) return fx_fail(FX_ERR_INVALID_ARG, "set_topology: out of host memory");
          }
          plan->jface_host[plan->njface_host++] = (int)(b * 6 + f);
        } else if (v != FX_BC_OUTFLOW && v != FX_BC_REFLECT) {
          return fx_fail(FX_ERR_UNSUPPORTED, "set_topology: block %lld face %d has unknown code %d", b, f, v);
        }
      }
  }
  plan->P.neigh = neigh_dev;
  plan->P.has_jumps = jumps;
  plan->P.all_interior = all_interior;
  plan->topology_set = true;
  plan->P.walls = 0;
  // z-chain segments: walk down (-z) from every unvisited block to the start of its chain (or once around a periodic
  // ring), then up (+z), cutting every `zchain` blocks and wherever the two blocks do not name each other
  delete[] plan->seg_host;
  plan->seg_host = nullptr;
  plan->nseg_host = 0;
  plan->nseg_inner_host = 0;
  plan->seg_uploaded = false;
  if (nb > 0) {
    std::vector<int32_t> h((size_t)nb * 6);
    FX_CUDA(cudaMemcpy(h.data(), neigh_dev, h.size() * sizeof(int32_t), cudaMemcpyDeviceToHost));
    const bool zact = plan->P.active[2] != 0;
    const long long nown = plan->P.nown;  // chains run through owned blocks only; a ghost block ends one (and is its halo)
    auto up = [&](long long b) -> long long {  // the block above b if the link is mutual, else -1
      if (!zact) return -1;
      const long long a = h[b * 6 + 5];
      return (a >= 0 && a < nown && a != b && h[a * 6 + 4] == b) ? a : -1;
    };
    auto down = [&](long long b) -> long long {
      if (!zact) return -1;
      const long long a = h[b * 6 + 4];
      return (a >= 0 && a < nown && a != b && h[a * 6 + 5] == b) ? a : -1;
    };
    for (long long b = 0; b < nb; ++b)
      for (int f = 0; f < 6; ++f)
        if (plan->P.active[f / 2] && h[b * 6 + f] == FX_BC_REFLECT) plan->P.walls = 1;
    {
      const int rcb = fx_build_bundles(plan, h);  // 8 x 8 blocks: bundles of 2 x 2 for the fused kernel's 16 x 16 cross-section
      if (rcb) return rcb;
    }
    std::vector<char> seen((size_t)nb, 0);
    // Refinement jumps on the fused path: where the block shape is the fused kernel's, the blocks WITH a jump face are taken
    // out of the chains and appended as segments of one block (the kernel reads their halo behind a jump from their own
    // interpolated guard zones and stores the jump faces' fluxes, which it can only attribute to a single-block segment);
    // every face of the others has a same-level neighbour or a physical boundary.
    delete[] plan->jlist_host;
    plan->jlist_host = nullptr;
    plan->njump_host = 0;
    {
      const int Rr = plan->P.recon == FX_RECON_WENO5 ? 3 : 2;
      const FxParams &Q = plan->P;
      const bool shape = Q.n[0] == 16 && Q.n[1] == 16 && Q.n[2] >= Rr && Q.active[2] && Q.gd[0] >= Rr && (Q.S_j % 2) == 0 && (Q.gd[0] % 2) == 0;
      // (with passive scalars: where the scalar pass can follow the fused kernel, i.e. PLM)
      if (jumps && shape && plan->path_option == 0 && (plan->nvars == 5 || Q.recon == FX_RECON_PLM_MINMOD) && Q.n[2] <= 64) {
        plan->jlist_host = new (std::nothrow) int[(size_t)nb];
        if (!plan->jlist_host) return fx_fail(FX_ERR_INVALID_ARG, "set_topology: out of host memory");
        for (long long b = 0; b < nown; ++b) {
          bool jb = false;
          for (int f = 0; f < 6; ++f) jb |= Q.active[f / 2] && h[b * 6 + f] <= FX_NEIGH_COARSER;
          if (jb) {
            plan->jlist_host[plan->njump_host++] = (int)b;
            seen[b] = 1;  // ends a chain from either side; never starts one
          }
        }
      }
    }
    plan->seg_host = new (std::nothrow) int[(size_t)nb * FX_SEG_STRIDE];
    if (!plan->seg_host) return fx_fail(FX_ERR_INVALID_ARG, "set_topology: out of host memory");
    // (blocks taller than 64 planes are not chained: the kernel's plane -> block map is exact up to 2^20 / nz planes)
    int M = plan->zchain > FX_SEG_MAX ? FX_SEG_MAX : plan->zchain;
    if (M <= 0) {
      // auto: a segment of M blocks costs about M + 0.09 block times (measured: the start-up of a CTA and the z halo of
      // a segment are 9 % of a block), and the launch takes ceil(segments / resident CTAs) rounds of them
      const int sms = fx_sm_count();
      const long long slots = (long long)sms * (plan->P.recon == FX_RECON_WENO5 ? 1 : 2);
      double best = 0.0;
      for (int m = 1; m <= FX_SEG_MAX; m *= 2) {
        const long long nseg = (nown + m - 1) / m;
        const double cost = (double)((nseg + slots - 1) / slots) * (m + 0.09);
        if (M <= 0 || cost < best) {
          best = cost;
          M = m;
        }
      }
    }
    if (plan->P.n[2] > 64) M = 1;
    // Sharded plans: a block with a ghost block behind a face is chained only with its like, so that the layers of a
    // column next to a cut do not drag the rest of it into the part of a stage that waits for the exchange
    std::vector<char> touch((size_t)nb, 0);
    if (nown < nb)
      for (long long b = 0; b < nown; ++b)
        for (int f = 0; f < 6; ++f)
          if (plan->P.active[f / 2] && h[b * 6 + f] >= nown) touch[b] = 1;
    for (long long b0 = 0; b0 < nown; ++b0) {
      if (seen[b0]) continue;
      long long start = b0;
      for (long long steps = 0; steps < nb; ++steps) {
        const long long d = down(start);
        if (d < 0 || seen[d] || d == b0) break;
        start = d;
      }
      long long b = start;
      while (b >= 0 && !seen[b]) {
        int *row = plan->seg_host + (size_t)plan->nseg_host * FX_SEG_STRIDE;
        for (int q = 0; q < FX_SEG_STRIDE; ++q) row[q] = -1;
        int cnt = 0;
        row[1] = zact ? h[b * 6 + 4] : -1;
        long long last = b;
        const char kind = touch[b];
        while (b >= 0 && !seen[b] && cnt < M && touch[b] == kind) {
          seen[b] = 1;
          row[2 + cnt++] = (int)b;
          last = b;
          b = up(b);
        }
        row[0] = cnt;
        row[2 + cnt] = zact ? h[last * 6 + 5] : -1;
        ++plan->nseg_host;
      }
    }
    // Sharded plans: the segments that touch no ghost block first, so that a stage can be launched in two parts -- those
    // while the ghost slabs are still under way, the others once they have arrived (fx_hydro_advance_stage_part)
    plan->nseg_inner_host = plan->nseg_host;
    if (nown < nb && plan->nseg_host > 0) {
      std::vector<int> rows((size_t)plan->nseg_host * FX_SEG_STRIDE);
      memcpy(rows.data(), plan->seg_host, rows.size() * sizeof(int));
      auto inner = [&](const int *row) {
        if (row[1] >= nown || row[2 + row[0]] >= nown) return false;  // the z neighbours below / above the segment
        for (int q = 0; q < row[0]; ++q)
          for (int f = 0; f < 4; ++f)
            if (plan->P.active[f / 2] && h[(long long)row[2 + q] * 6 + f] >= nown) return false;
        return true;
      };
      int w = 0;
      for (int pass = 0; pass < 2; ++pass) {
        for (int r = 0; r < plan->nseg_host; ++r) {
          const int *row = rows.data() + (size_t)r * FX_SEG_STRIDE;
          if (inner(row) == (pass == 0)) memcpy(plan->seg_host + (size_t)w++ * FX_SEG_STRIDE, row, FX_SEG_STRIDE * sizeof(int));
        }
        if (pass == 0) plan->nseg_inner_host = w;
      }
    }
    for (long long q = 0; q < plan->njump_host; ++q) {  // the blocks with a jump face: one segment each
      const long long b = plan->jlist_host[q];
      int *row = plan->seg_host + (size_t)plan->nseg_host * FX_SEG_STRIDE;
      for (int t = 0; t < FX_SEG_STRIDE; ++t) row[t] = -1;
      row[0] = 1;
      row[1] = zact ? h[b * 6 + 4] : -1;
      row[2] = (int)b;
      row[3] = zact ? h[b * 6 + 5] : -1;
      ++plan->nseg_host;
    }
  }
  return fx_seg_upload(plan);
}

static uint64_t fx_morton3(uint32_t x, uint32_t y, uint32_t z) {
  auto spread = [](uint64_t v) {
    v &= 0x1fffff;
    v = (v | v << 32) & 0x1f00000000ffffull;
    v = (v | v << 16) & 0x1f0000ff0000ffull;
    v = (v | v << 8) & 0x100f00f00f00f00full;
    v = (v | v << 4) & 0x10c30c30c30c30c3ull;
    v = (v | v << 2) & 0x1249249249249249ull;
    return v;
  };
  return spread(x) | spread(y) << 1 | spread(z) << 2;
}

extern "C" int fx_topology_cartesian(const int nb[3], const int bc_lo[3], const int bc_hi[3], int order,
                                     int32_t *neigh_out, int32_t *coords_out) {
  if (!nb || !bc_lo || !bc_hi || !neigh_out) return fx_fail(FX_ERR_INVALID_ARG, "topology_cartesian: null argument");
  if (order != FX_ORDER_LEX && order != FX_ORDER_MORTON) return fx_fail(FX_ERR_INVALID_ARG, "topology_cartesian: unknown order");
  for (int d = 0; d < 3; ++d) {
    if (nb[d] < 1) return fx_fail(FX_ERR_INVALID_ARG, "topology_cartesian: nb[%d] < 1", d);
    if (bc_lo[d] < 0 || bc_lo[d] > 3 || bc_hi[d] < 0 || bc_hi[d] > 3) return fx_fail(FX_ERR_INVALID_ARG, "topology_cartesian: bad bc code");
  }
  const long long N = (long long)nb[0] * nb[1] * nb[2];
  if (N > 2147483647LL) return fx_fail(FX_ERR_INVALID_ARG, "topology_cartesian: too many blocks");
  std::vector<int32_t> lex_of_id((size_t)N), id_of_lex((size_t)N);
  for (long long l = 0; l < N; ++l) lex_of_id[l] = (int32_t)l;
  if (order == FX_ORDER_MORTON) {
    std::vector<uint64_t> key((size_t)N);
    for (long long l = 0; l < N; ++l)
      key[l] = fx_morton3((uint32_t)(l % nb[0]), (uint32_t)((l / nb[0]) % nb[1]), (uint32_t)(l / ((long long)nb[0] * nb[1])));
    std::stable_sort(lex_of_id.begin(), lex_of_id.end(), [&](int32_t a, int32_t b) { return key[a] < key[b]; });
  }
  for (long long id = 0; id < N; ++id) id_of_lex[lex_of_id[id]] = (int32_t)id;
  for (long long id = 0; id < N; ++id) {
    const long long l = lex_of_id[id];
    const int c[3] = {(int)(l % nb[0]), (int)((l / nb[0]) % nb[1]), (int)(l / ((long long)nb[0] * nb[1]))};
    if (coords_out)
      for (int d = 0; d < 3; ++d) coords_out[id * 3 + d] = c[d];
    for (int d = 0; d < 3; ++d)
      for (int s = 0; s < 2; ++s) {
        const int bc = s ? bc_hi[d] : bc_lo[d];
        int32_t v;
        if (bc == FX_TOPO_NONE) {
          v = FX_BC_NONE;
        } else {
          int cc[3] = {c[0], c[1], c[2]};
          cc[d] += s ? 1 : -1;
          const bool outside = cc[d] < 0 || cc[d] >= nb[d];
          if (outside && (bc == FX_TOPO_OUTFLOW || bc == FX_TOPO_REFLECT)) {
            v = bc == FX_TOPO_REFLECT ? FX_BC_REFLECT : FX_BC_OUTFLOW;
          } else {
            cc[d] = (cc[d] + nb[d]) % nb[d];
            v = id_of_lex[((long long)cc[2] * nb[1] + cc[1]) * nb[0] + cc[0]];
          }
        }
        neigh_out[id * 6 + 2 * d + s] = v;
      }
  }
  return FX_OK;
}
