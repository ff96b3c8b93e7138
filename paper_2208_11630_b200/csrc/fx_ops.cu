// fx_ops.cu -- the operations of the C ABI: guard fill, index map, dt, advance (stage sequencing),
// host-buffer end-to-end variant, status, debug fluxes.
#include <math.h>
#include <string.h>

#include <new>

#include "fx_internal.h"

static int fx_need(const fx_hydro_plan *plan, bool topo, bool ws, const char *who) {
  if (!plan) return fx_fail(FX_ERR_INVALID_ARG, "%s: null plan", who);
  if (topo && !plan->topology_set) return fx_fail(FX_ERR_STATE, "%s: call fx_hydro_plan_set_topology first", who);
  if (ws && !plan->workspace) return fx_fail(FX_ERR_STATE, "%s: call fx_hydro_plan_set_workspace first", who);
  return FX_OK;
}

extern "C" int fx_fill_guardcells(fx_hydro_plan *plan, double *U, void *stream) {
  int rc = fx_need(plan, true, false, "fill_guardcells");
  if (rc) return rc;
  if (!U && plan->P.nblocks > 0) return fx_fail(FX_ERR_INVALID_ARG, "fill_guardcells: null U");
  rc = fx_launch_fill_guardcells(plan->P, U, (cudaStream_t)stream);
  if (rc) return rc;
  return fx_launch_amr_fill(plan->P, U, plan->nguard, (cudaStream_t)stream);  // second pass: the jump faces [B12, B13]
}

extern "C" int fx_guardcell_index_map(fx_hydro_plan *plan, int64_t b0, int64_t nb, int64_t *src, void *stream) {
  int rc = fx_need(plan, true, false, "guardcell_index_map");
  if (rc) return rc;
  if (b0 < 0 || nb < 0 || b0 + nb > plan->P.nblocks || (!src && nb > 0))
    return fx_fail(FX_ERR_INVALID_ARG, "guardcell_index_map: bad block range or null output");
  return fx_launch_index_map(plan->P, b0, nb, (long long *)src, (cudaStream_t)stream);
}

extern "C" int fx_hydro_compute_dt(fx_hydro_plan *plan, const double *U, const double *dx, double cfl, double *dt_out,
                                   void *stream) {
  int rc = fx_need(plan, false, true, "compute_dt");
  if (rc) return rc;
  if (!dt_out || ((!U || !dx) && plan->P.nblocks > 0)) return fx_fail(FX_ERR_INVALID_ARG, "compute_dt: null argument");
  return fx_launch_compute_dt(plan->P, U, dx, cfl, dt_out, (cudaStream_t)stream);
}

// One stage: out = U0 + beta((X - U0) - S(X)); halos of X come from a K1 fill (generic path) or are
// gathered from neighbour interiors inside the fused kernel.

// part (fx_hydro_advance_stage_part): 0 the whole stage; 1 the segments that touch no ghost block; 2 the others.  Only the
// fused kernel without passive scalars is launched in parts; every other path does nothing for part 1 and all for part 2.
static int fx_stage(fx_hydro_plan *plan, double *X, const double *U0, double *out, const double *dx, double dt,
                    const double *dt_dev, double beta, int first, cudaStream_t st, double cfl_next = 0.0,
                    double *dt_next = nullptr, int part = 0) {
  const int path = fx_hydro_plan_path(plan);  // 1 fused TMA kernel (3: its pair variant), 2 shared-memory tile kernel, 0 generic
  const bool fused = path == 1 || path == 3 || path == 4;
  int rc = FX_OK;
  if (part != 0) {
    if (path == 1 && plan->nvars == 5) {
      FxParams Q = plan->P;
      const int ni = Q.nseg_inner;
      Q.seg = part == 1 ? Q.seg : Q.seg + (size_t)ni * FX_SEG_STRIDE;
      Q.nseg = part == 1 ? ni : Q.nseg - ni;
      if (Q.nseg == 0) return FX_OK;
      const bool rec = plan->timing && plan->ev && plan->nrec < FX_MAX_REC;
      if (rec) FX_CUDA(cudaEventRecord(plan->ev[2 * plan->nrec], st));
      if ((rc = fx_launch_stage_tma(Q, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st))) return rc;
      if (rec) {
        FX_CUDA(cudaEventRecord(plan->ev[2 * plan->nrec + 1], st));
        ++plan->nrec;
      }
      return FX_OK;
    }
    if (part == 1) return FX_OK;
  }
  if (path == 5) {
    // fused AMR path: guard zones behind the jumps, then the fused kernel on every block (the blocks with a jump face read
    // their own guard zones behind it and store the jump faces' fluxes), then the flux correction; the time step of the
    // finished state, if asked for: the stage kernel's fused reduction over the blocks the correction does not touch, then
    // a pass over the corrected blocks (a first stage, which has no fused reduction: a pass over every block)
    const FxParams &P = plan->P;
    if ((rc = fx_launch_amr_fill(P, X, P.recon == FX_RECON_WENO5 ? 3 : 2, st))) return rc;
    const bool rec = plan->timing && plan->ev && plan->nrec < FX_MAX_REC;
    if (rec) FX_CUDA(cudaEventRecord(plan->ev[2 * plan->nrec], st));
    const bool fuse_dt = dt_next && !first && P.jface && P.njface > 0;
    FxParams Pd = P;
    Pd.dt_defer = fuse_dt ? 1 : 0;
    if ((rc = fx_launch_stage_tma(Pd, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, fuse_dt ? dt_next : nullptr, st))) return rc;
    if (plan->nvars > 5 && (rc = fx_launch_scalar_pass(P, X, U0, out, dx, dt, dt_dev, beta, first, st))) return rc;  // [B11]
    if (rec) {
      FX_CUDA(cudaEventRecord(plan->ev[2 * plan->nrec + 1], st));
      ++plan->nrec;
    }
    if ((rc = fx_launch_amr_flux_correct(P, out, dx, dt, dt_dev, first ? 1.0 : beta, st))) return rc;
    if (fuse_dt) return fx_launch_compute_dt_corrected(P, out, dx, cfl_next, dt_next, st);
    if (dt_next) return fx_launch_compute_dt(P, out, dx, cfl_next, dt_next, st);
    return FX_OK;
  }
  if (path == 0 && plan->nvars > 5) {
    // the generic zone kernel reads the hydro variables' halo cells through the neighbour table, like the other two
    // paths; only the passive scalars' face guard zones are filled [A15]
    rc = fx_launch_fill_faces(plan->P, X, 5, st);
    if (rc) return rc;
  }
  const bool amr = plan->P.has_jumps != 0;  // (generic path)
  if (amr) {  // the face guard zones behind refinement jumps: restriction / prolongation of the stage input [B12, B13]
    rc = fx_launch_amr_fill(plan->P, X, plan->P.recon == FX_RECON_WENO5 ? 3 : 2, st);
    if (rc) return rc;
  }
  const bool rec = plan->timing && plan->ev && plan->nrec < FX_MAX_REC;
  if (rec) FX_CUDA(cudaEventRecord(plan->ev[2 * plan->nrec], st));
  // with a scalar pass behind the fused kernel the next time step waits in a scratch word until the pass, which still
  // reads this step's dt from the device, has been enqueued
  double *dt_user = dt_next;
  const bool park_dt = fused && plan->nvars > 5 && dt_next != nullptr;
  if (park_dt) dt_next = (double *)&plan->P.scratch[FX_SCR_WORDS - 3];
  rc = fused ? (path == 3 ? fx_launch_stage_pair(plan->P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st)
                : path == 4 ? fx_launch_stage_bundle(plan->P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st)
                          : fx_launch_stage_tma(plan->P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st))
             : (path == 2 ? fx_launch_stage_tile(plan->P, X, U0, out, dx, dt, dt_dev, beta, first, st)
                          : fx_launch_generic_stage(plan->P, X, U0, out, dx, dt, dt_dev, beta, first, st));
  if (rc) return rc;
  if (fused && plan->nvars > 5) {  // passive scalars [B11] behind the fused kernel: the scalar pass (inside the timing bracket)
    rc = fx_launch_scalar_pass(plan->P, X, U0, out, dx, dt, dt_dev, beta, first, st);
    if (rc) return rc;
    if (park_dt) FX_CUDA(cudaMemcpyAsync(dt_user, dt_next, sizeof(double), cudaMemcpyDeviceToDevice, st));
  }
  if (rec) {  // the pair brackets the stage kernel alone (fx_hydro.h), not the reduction pass below
    FX_CUDA(cudaEventRecord(plan->ev[2 * plan->nrec + 1], st));
    ++plan->nrec;
  }
  if (amr) {  // coarse face fluxes at the jumps <- the mean of the fine ones [B14]
    rc = fx_launch_amr_flux_correct(plan->P, out, dx, dt, dt_dev, first ? 1.0 : beta, st);
    if (rc) return rc;
  }
  if (!fused && dt_next) {  // the generic and tile paths have no fused reduction: a7 as its own pass over the finished state
    rc = fx_launch_compute_dt(plan->P, out, dx, cfl_next, dt_next, st);
    if (rc) return rc;
  }
  return FX_OK;
}

extern "C" int fx_hydro_plan_set_timing(fx_hydro_plan *plan, int enable) {
  if (!plan) return fx_fail(FX_ERR_INVALID_ARG, "set_timing: null plan");
  if (enable && !plan->ev) {
    plan->ev = new (std::nothrow) cudaEvent_t[2 * FX_MAX_REC];
    if (!plan->ev) return fx_fail(FX_ERR_INVALID_ARG, "set_timing: out of host memory");
    for (int i = 0; i < 2 * FX_MAX_REC; ++i) FX_CUDA(cudaEventCreate(&plan->ev[i]));
  }
  plan->timing = enable != 0;
  plan->nrec = 0;
  return FX_OK;
}

extern "C" int fx_hydro_plan_get_timing(fx_hydro_plan *plan, double *ms_sum, long long *launches) {
  if (!plan || !ms_sum || !launches) return fx_fail(FX_ERR_INVALID_ARG, "get_timing: null argument");
  double sum = 0.0;
  for (int i = 0; i < plan->nrec; ++i) {
    float ms = 0.f;
    FX_CUDA(cudaEventSynchronize(plan->ev[2 * i + 1]));
    FX_CUDA(cudaEventElapsedTime(&ms, plan->ev[2 * i], plan->ev[2 * i + 1]));
    sum += ms;
  }
  *ms_sum = sum;
  *launches = plan->nrec;
  plan->nrec = 0;
  return FX_OK;
}

// Stage s of the step: input X_s, output, beta_s [O6].  The last stage may overwrite U0 in place: its halos come from
// U1 (RK2) / U2 (RK3), never from U0.
static void fx_stage_arrays(fx_hydro_plan *plan, double *U, int s, double **X, double **out, double *beta) {
  double *U1 = plan->stage[0], *U2 = plan->stage[1];
  const bool last = s == plan->rk - 1;
  *X = s == 0 ? U : (s == 1 ? U1 : U2);
  *out = last ? U : (s == 0 ? U1 : U2);
  *beta = s == 0 ? 1.0 : (plan->rk == 2 ? 0.5 : (s == 1 ? 0.25 : 2.0 / 3.0));
}

extern "C" int fx_hydro_stage_arrays(fx_hydro_plan *plan, double *U, int stage, double **stage_input, double **stage_output) {
  int rc = fx_need(plan, false, true, "stage_arrays");
  if (rc) return rc;
  if (stage < 0 || stage >= plan->rk || !stage_input || !stage_output) return fx_fail(FX_ERR_INVALID_ARG, "stage_arrays: bad stage or null output");
  double beta;
  fx_stage_arrays(plan, U, stage, stage_input, stage_output, &beta);
  return FX_OK;
}

extern "C" int fx_hydro_advance_stage(fx_hydro_plan *plan, double *U, const double *dx, double dt, const double *dt_dev, int stage,
                                      double cfl_next, double *dt_next_dev, void *stream) {
  int rc = fx_need(plan, true, true, "advance_stage");
  if (rc) return rc;
  if (stage < 0 || stage >= plan->rk) return fx_fail(FX_ERR_INVALID_ARG, "advance_stage: stage must be 0 .. rk_order - 1");
  if (!dt_dev && (!(dt > 0.0) || !isfinite(dt))) return fx_fail(FX_ERR_INVALID_ARG, "advance_stage: dt must be positive and finite");
  if ((!U || !dx) && plan->P.nblocks > 0) return fx_fail(FX_ERR_INVALID_ARG, "advance_stage: null argument");
  if (dt_next_dev && stage != plan->rk - 1) return fx_fail(FX_ERR_INVALID_ARG, "advance_stage: the next time step comes out of the last stage only");
  if (dt_next_dev && (!(cfl_next > 0.0) || !isfinite(cfl_next))) return fx_fail(FX_ERR_INVALID_ARG, "advance_stage: cfl must be positive and finite");
  if (plan->P.nown == 0) return FX_OK;
  double *X, *out, beta;
  fx_stage_arrays(plan, U, stage, &X, &out, &beta);
  return fx_stage(plan, X, U, out, dx, dt, dt_dev, beta, stage == 0, (cudaStream_t)stream, cfl_next, dt_next_dev);
}

extern "C" int fx_hydro_advance_stage_part(fx_hydro_plan *plan, double *U, const double *dx, double dt, const double *dt_dev, int stage,
                                           int part, double cfl_next, double *dt_next_dev, void *stream) {
  int rc = fx_need(plan, true, true, "advance_stage_part");
  if (rc) return rc;
  if (part != FX_PART_INNER && part != FX_PART_BOUNDARY) return fx_fail(FX_ERR_INVALID_ARG, "advance_stage_part: part must be FX_PART_INNER or FX_PART_BOUNDARY");
  if (stage < 0 || stage >= plan->rk) return fx_fail(FX_ERR_INVALID_ARG, "advance_stage_part: stage must be 0 .. rk_order - 1");
  if (!dt_dev && (!(dt > 0.0) || !isfinite(dt))) return fx_fail(FX_ERR_INVALID_ARG, "advance_stage_part: dt must be positive and finite");
  if ((!U || !dx) && plan->P.nblocks > 0) return fx_fail(FX_ERR_INVALID_ARG, "advance_stage_part: null argument");
  if (dt_next_dev && stage != plan->rk - 1) return fx_fail(FX_ERR_INVALID_ARG, "advance_stage_part: the next time step comes out of the last stage only");
  if (dt_next_dev && (!(cfl_next > 0.0) || !isfinite(cfl_next))) return fx_fail(FX_ERR_INVALID_ARG, "advance_stage_part: cfl must be positive and finite");
  if (plan->P.nown == 0) return FX_OK;
  double *X, *out, beta;
  fx_stage_arrays(plan, U, stage, &X, &out, &beta);
  return fx_stage(plan, X, U, out, dx, dt, dt_dev, beta, stage == 0, (cudaStream_t)stream, cfl_next, dt_next_dev, part);
}

extern "C" int fx_hydro_plan_stage_parts(const fx_hydro_plan *plan, int64_t *inner_blocks, int64_t *boundary_blocks) {
  if (!plan || !inner_blocks || !boundary_blocks) return fx_fail(FX_ERR_INVALID_ARG, "stage_parts: null argument");
  if (!plan->topology_set) return fx_fail(FX_ERR_STATE, "stage_parts: set the topology first");
  int64_t ni = 0;
  if (fx_hydro_plan_path(plan) == 1 && plan->nvars == 5 && plan->seg_host)
    for (int r = 0; r < plan->nseg_inner_host; ++r) ni += plan->seg_host[(size_t)r * FX_SEG_STRIDE];
  *inner_blocks = ni;
  *boundary_blocks = plan->P.nown - ni;
  return FX_OK;
}

static int fx_advance_impl(fx_hydro_plan *plan, double *U, const double *dx, double dt, const double *dt_dev,
                           cudaStream_t st, double cfl_next = 0.0, double *dt_next = nullptr) {
  if (plan->P.nown == 0) return FX_OK;
  double *U1 = plan->stage[0], *U2 = plan->stage[1];
  // The last stage may overwrite U0 in place: its halos come from U1 (RK2) / U2 (RK3), never from U0.
  int rc = fx_stage(plan, U, U, U1, dx, dt, dt_dev, 1.0, 1, st);  // U1 = U0 - S(U0)
  if (rc) return rc;
  if (plan->rk == 2) return fx_stage(plan, U1, U, U, dx, dt, dt_dev, 0.5, 0, st, cfl_next, dt_next);
  rc = fx_stage(plan, U1, U, U2, dx, dt, dt_dev, 0.25, 0, st);
  if (rc) return rc;
  return fx_stage(plan, U2, U, U, dx, dt, dt_dev, 2.0 / 3.0, 0, st, cfl_next, dt_next);
}

extern "C" int fx_hydro_advance(fx_hydro_plan *plan, double *U, const double *dx, double dt, void *stream) {
  int rc = fx_need(plan, true, true, "advance");
  if (rc) return rc;
  if (!(dt > 0.0) || !isfinite(dt)) return fx_fail(FX_ERR_INVALID_ARG, "advance: dt must be positive and finite");
  if ((!U || !dx) && plan->P.nblocks > 0) return fx_fail(FX_ERR_INVALID_ARG, "advance: null argument");
  return fx_advance_impl(plan, U, dx, dt, nullptr, (cudaStream_t)stream);
}

// The communication-avoiding step [B17; SURVEY 8(f) NEXT-4]: the step's one guard fill, then stage s of n on the interior
// extended by (n - s) R zones, each reading its stencils in place; after every stage but the last the extended zones
// behind a physical boundary are re-imaged from the block's own zones.  Each stage kernel is bracketed like fx_stage's.
extern "C" int fx_hydro_advance_ca(fx_hydro_plan *plan, double *U, const double *dx, double dt, const double *dt_dev,
                                   void *stream) {
  int rc = fx_need(plan, true, true, "advance_ca");
  if (rc) return rc;
  if (!dt_dev && (!(dt > 0.0) || !isfinite(dt))) return fx_fail(FX_ERR_INVALID_ARG, "advance_ca: dt must be positive and finite");
  if ((!U || !dx) && plan->P.nblocks > 0) return fx_fail(FX_ERR_INVALID_ARG, "advance_ca: null argument");
  const FxParams &P = plan->P;
  const int R = P.recon == FX_RECON_WENO5 ? 3 : 2;
  for (int d = 0; d < 3; ++d)
    if (P.active[d] && plan->rk * R > plan->nguard)
      return fx_fail(FX_ERR_UNSUPPORTED, "advance_ca: needs nguard >= rk_order x %d = %d (the plan has %d)", R, plan->rk * R, plan->nguard);
  if (P.has_jumps || P.jump) return fx_fail(FX_ERR_UNSUPPORTED, "advance_ca: refinement jumps are not supported");
  if (plan->nvars > 5) return fx_fail(FX_ERR_UNSUPPORTED, "advance_ca: passive scalars are not supported");
  if (P.nown != P.nblocks) return fx_fail(FX_ERR_UNSUPPORTED, "advance_ca: not for a sharded plan (its ghost blocks carry no edge neighbours)");
  if (P.nown == 0) return FX_OK;
  cudaStream_t st = (cudaStream_t)stream;
  double *U1 = plan->stage[0], *U2 = plan->stage[1];
  if ((rc = fx_launch_fill_guardcells(P, U, st))) return rc;  // the step's only O1: every guard zone, edges and corners too
  auto stage = [&](const double *X, double *out, double beta, int first, int ext) -> int {
    const bool rec = plan->timing && plan->ev && plan->nrec < FX_MAX_REC;
    if (rec) FX_CUDA(cudaEventRecord(plan->ev[2 * plan->nrec], st));
    int r2 = fx_launch_generic_stage_ca(P, X, U, out, dx, dt, dt_dev, beta, first, ext, st);
    if (r2) return r2;
    if (rec) {
      FX_CUDA(cudaEventRecord(plan->ev[2 * plan->nrec + 1], st));
      ++plan->nrec;
    }
    return fx_launch_ca_refill(P, out, ext, st);
  };
  if ((rc = stage(U, U1, 1.0, 1, (plan->rk - 1) * R))) return rc;
  if (plan->rk == 2) return stage(U1, U, 0.5, 0, 0);
  if ((rc = stage(U1, U2, 0.25, 0, R))) return rc;
  return stage(U2, U, 2.0 / 3.0, 0, 0);
}

extern "C" int fx_hydro_advance_devdt(fx_hydro_plan *plan, double *U, const double *dx, const double *dt_dev,
                                      void *stream) {
  int rc = fx_need(plan, true, true, "advance_devdt");
  if (rc) return rc;
  if (!dt_dev || ((!U || !dx) && plan->P.nblocks > 0)) return fx_fail(FX_ERR_INVALID_ARG, "advance_devdt: null argument");
  return fx_advance_impl(plan, U, dx, 0.0, dt_dev, (cudaStream_t)stream);
}

extern "C" int fx_hydro_step(fx_hydro_plan *plan, double *U, const double *dx, double cfl, double *dt_inout_dev,
                             void *stream) {
  int rc = fx_need(plan, true, true, "step");
  if (rc) return rc;
  if (!dt_inout_dev || ((!U || !dx) && plan->P.nblocks > 0)) return fx_fail(FX_ERR_INVALID_ARG, "step: null argument");
  if (!(cfl > 0.0) || !isfinite(cfl)) return fx_fail(FX_ERR_INVALID_ARG, "step: cfl must be positive and finite");
  if (plan->P.nown == 0) return FX_OK;
  // every stage reads dt from dt_inout_dev when it starts; the last CTA of the last stage to finish overwrites it
  return fx_advance_impl(plan, U, dx, 0.0, dt_inout_dev, (cudaStream_t)stream, cfl, dt_inout_dev);
}

extern "C" int fx_hydro_advance_host(fx_hydro_plan *plan, double *U_host, const double *dx_host, double cfl, int nsteps,
                                     double *U_stage, double *dx_stage, double *dt_last_host, void *stream) {
  int rc = fx_need(plan, true, true, "advance_host");
  if (rc) return rc;
  if (nsteps < 0 || !U_host || !dx_host || !U_stage || !dx_stage)
    return fx_fail(FX_ERR_INVALID_ARG, "advance_host: null argument or negative nsteps");
  cudaStream_t st = (cudaStream_t)stream;
  const size_t ub = (size_t)plan->P.S_v * plan->nvars * sizeof(double);
  const size_t db = (size_t)plan->P.nblocks * 3 * sizeof(double);
  FX_CUDA(cudaMemcpyAsync(U_stage, U_host, ub, cudaMemcpyHostToDevice, st));
  FX_CUDA(cudaMemcpyAsync(dx_stage, dx_host, db, cudaMemcpyHostToDevice, st));
  double *dt_dev = (double *)&plan->P.scratch[FX_SCR_WORDS - 1];  // last scratch word holds the step's dt
  double *dt_used = dt_dev - 1;  // the dt the last step was taken with (what the caller gets back)
  if (nsteps > 0) {
    rc = fx_launch_compute_dt(plan->P, U_stage, dx_stage, cfl, dt_dev, st);
    if (rc) return rc;
  }
  for (int s = 0; s < nsteps; ++s) {
    FX_CUDA(cudaMemcpyAsync(dt_used, dt_dev, sizeof(double), cudaMemcpyDeviceToDevice, st));
    rc = fx_advance_impl(plan, U_stage, dx_stage, 0.0, dt_dev, st, cfl, dt_dev);  // leaves the next step's dt in dt_dev
    if (rc) return rc;
  }
  FX_CUDA(cudaMemcpyAsync(U_host, U_stage, ub, cudaMemcpyDeviceToHost, st));
  if (dt_last_host && nsteps > 0) FX_CUDA(cudaMemcpyAsync(dt_last_host, dt_used, sizeof(double), cudaMemcpyDeviceToHost, st));
  FX_CUDA(cudaStreamSynchronize(st));
  return FX_OK;
}

extern "C" int fx_hydro_advance_host_interior(fx_hydro_plan *plan, double *Uint_host, const double *dx_host, double cfl,
                                              int nsteps, double *U_stage, double *packed_stage, double *dx_stage,
                                              double *dt_last_host, void *stream) {
  int rc = fx_need(plan, true, true, "advance_host_interior");
  if (rc) return rc;
  if (nsteps < 0 || !Uint_host || !dx_host || !U_stage || !packed_stage || !dx_stage)
    return fx_fail(FX_ERR_INVALID_ARG, "advance_host_interior: null argument or negative nsteps");
  cudaStream_t st = (cudaStream_t)stream;
  const FxParams &P = plan->P;
  const size_t ib = (size_t)plan->nvars * P.nblocks * P.n[0] * P.n[1] * P.n[2] * sizeof(double);
  const size_t db = (size_t)P.nblocks * 3 * sizeof(double);
  FX_CUDA(cudaMemcpyAsync(packed_stage, Uint_host, ib, cudaMemcpyHostToDevice, st));
  FX_CUDA(cudaMemcpyAsync(dx_stage, dx_host, db, cudaMemcpyHostToDevice, st));
  if ((rc = fx_launch_pack_interior(P, U_stage, packed_stage, 0, st))) return rc;
  double *dt_dev = (double *)&plan->P.scratch[FX_SCR_WORDS - 1];
  double *dt_used = dt_dev - 1;
  if (nsteps > 0 && (rc = fx_launch_compute_dt(P, U_stage, dx_stage, cfl, dt_dev, st))) return rc;
  for (int s = 0; s < nsteps; ++s) {
    FX_CUDA(cudaMemcpyAsync(dt_used, dt_dev, sizeof(double), cudaMemcpyDeviceToDevice, st));
    if ((rc = fx_advance_impl(plan, U_stage, dx_stage, 0.0, dt_dev, st, cfl, dt_dev))) return rc;
  }
  if ((rc = fx_launch_pack_interior(P, U_stage, packed_stage, 1, st))) return rc;
  FX_CUDA(cudaMemcpyAsync(Uint_host, packed_stage, ib, cudaMemcpyDeviceToHost, st));
  if (dt_last_host && nsteps > 0) FX_CUDA(cudaMemcpyAsync(dt_last_host, dt_used, sizeof(double), cudaMemcpyDeviceToHost, st));
  FX_CUDA(cudaStreamSynchronize(st));
  return FX_OK;
}

extern "C" int fx_hydro_status(fx_hydro_plan *plan, uint32_t *flags, unsigned long long counts[4], void *stream) {
  int rc = fx_need(plan, false, true, "status");
  if (rc) return rc;
  if (!flags) return fx_fail(FX_ERR_INVALID_ARG, "status: null flags");
  unsigned long long h[FX_SCR_WORDS];
  FX_CUDA(cudaMemcpyAsync(h, plan->P.scratch, sizeof(h), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
  FX_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
  *flags = (uint32_t)(h[FX_SCR_FLAGS] & 0xffffffffull);
  if (counts)
    for (int i = 0; i < 4; ++i) counts[i] = h[FX_SCR_COUNT0 + i];
  return FX_OK;
}

extern "C" int fx_hydro_status_reset(fx_hydro_plan *plan, void *stream) {
  int rc = fx_need(plan, false, true, "status_reset");
  if (rc) return rc;
  FX_CUDA(cudaMemsetAsync(&plan->P.scratch[FX_SCR_FLAGS], 0, 6 * sizeof(unsigned long long), (cudaStream_t)stream));
  return FX_OK;
}

extern "C" int fx_debug_compute_fluxes(fx_hydro_plan *plan, const double *U, int dir, double *F, void *stream) {
  int rc = fx_need(plan, false, true, "debug_compute_fluxes");
  if (rc) return rc;
  if (dir < 0 || dir > 2 || !plan->P.active[dir]) return fx_fail(FX_ERR_INVALID_ARG, "debug_compute_fluxes: inactive or bad direction %d", dir);
  if ((!U || !F) && plan->P.nblocks > 0) return fx_fail(FX_ERR_INVALID_ARG, "debug_compute_fluxes: null argument");
  return fx_launch_debug_fluxes(plan->P, U, dir, F, (cudaStream_t)stream);
}
