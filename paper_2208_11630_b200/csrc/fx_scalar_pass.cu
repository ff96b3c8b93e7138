// fx_scalar_pass.cu -- passive mass scalars [B11] behind the fused stage kernel.
//
// A scalar's flux at a face is Aq X_L + (F_rho - Aq) X_R [B11], where the mass flux F_rho and the coefficient Aq come out of
// the hydro Riemann solve of that face.  The fused kernel (fx_stage_tma.cu, SCAL) leaves both for the three low faces of
// every zone in P.fq (HLLC: F_rho alone -- there Aq = max(F_rho, 0), the flux being upwind in the sign of S*); the kernel
// here does what is left for each scalar: X = (rho X) / rho on the cells of each direction's stencil (the reciprocal
// densities are formed once and serve all scalars), PLM face values of cells -1, 0, +1, the two face fluxes per direction
// (the high face's F_rho and Aq are the next zone's low-face values, through the neighbour table at a block face -- or, where
// no owned same-level block lies behind a block's high face (a physical boundary, a ghost block of a sharded plan, a
// refinement jump), the fused kernel's own solve of that face, which it leaves in P.fqb), divergence and RK combination.
// Halo abundances behind an outflow boundary are the block's edge cell's, behind a wall its mirror cells' [B9, B11], behind
// a refinement jump the block's own interpolated guard zones' [B13].  Expressions and their order are those of the generic
// kernel's scalar loop (fx_generic.cu), which remains the path for WENO5 and for other block shapes.
// Applies to: PLM, 16 x 16 x nz blocks (fx_scalar_pass_supported).
// (The first form of this pass, one thread per zone with everything in registers -- 19.2 ms per stage pair at config 5 with
// 4 scalars, bound by the L2 -> L1 traffic of its y and z stencil rows -- was replaced by the marching form below and, once
// nothing could reach it any more, removed.)
#include "fx_physics.cuh"

namespace {

// ------------------------------------------------------------------ the marching form (16 x 16 x nz blocks)
// One CTA of 256 threads per block marches through the block's planes; thread (i, j) carries its column's z stencil in
// registers (X of cells k and k+1, the plus value of cell k, the flux through the low z face: one evaluation per z face),
// the plane's X with its two-deep x / y halo (taken from the neighbour blocks' interiors through the table, like every halo
// of the fused path) goes through shared memory, double-buffered so that one CTA barrier per plane suffices.  What a plane
// needs from HBM before that barrier -- the new cell of each window (rho, rho X_s), the halo cells' (rho, rho X_s), the
// faces' (F_rho, Aq) of the x and y directions -- is fetched one plane ahead with cp.async into a two-stage buffer (each
// thread reads back what it fetched itself, except the high faces' (F_rho, Aq), which are the next zone's low-face values:
// read from the neighbour's slot after the barrier instead of a second time from memory), and so are U0 and the z face's
// (F_rho, Aq), which only the end of the plane needs but which come from DRAM; the stage input's own zone (fetched two
// planes earlier as a window cell: an L2 hit) is a plain load issued right after the barrier and used last.  Up to NSC = 4
// scalars per launch share the densities and the (F_rho, Aq).
// Measured, config 5 with 4 scalars, whole step (fused kernel + this pass, two stages):
//   * every load at the top of the plane, 184 registers, one CTA per SM: this pass alone 10.8 ms per stage; the z carry and
//     128 registers (two CTAs): 7.4 ms; cp.async staging one plane ahead: 5.1 ms (first stage) / 7.5 ms (later ones) --
//     24.4 ms per step.  At that point ncu showed as many instructions as the hydro kernel issues (3.5 G per launch, 847
//     SASS instructions per plane and thread, 215 of them 64-bit address arithmetic), 60 % of the issue slots busy.
//   * running 64-bit offsets advanced by one plane per prefetch instead of addresses formed from k, the stencil's centre
//     from the z window, the non-finite test on the result's upper word: 758 instructions, 22.3 ms per step.
//   * two planes per loop trip (constant staging index, no register moves for the carried values): 666 instructions, but
//     22.6 ms: no longer bound by the issue rate.  ncu's stall samples: 35 % long-scoreboard, nearly all at the first uses
//     of U0 and of the z face's F_rho (plain loads issued after the barrier).
//   * those two staged through cp.async with the rest of the plane (this version): 21.6 ms per step.  Loading them one
//     plane ahead into registers instead: 24.5 ms (15 spill loads per plane at 128 registers).
//   * every cell's PLM face values formed once and shared through shared memory (three evaluations per scalar and zone
//     instead of seven; the cells beyond the block faces by one extra evaluation per warp; single-buffered arrays and two
//     barriers per plane, since double-buffering them does not fit two CTAs per SM): 640 instructions per plane, 23.3 ms
//     without and 24.8 ms with the staging above -- the second barrier costs more than the 28 % fewer instructions save;
//     a ninth warp for the outer cells: 96 registers, 37 spill instructions per plane.  Not kept.
template <int NSC>
struct ScalSmem {
  double XS[2][NSC][20][20];      // abundances of the plane with halo
  double raw[2][1 + NSC][256];    // (rho, rho X_s) of the window's new cell, per thread
  double hal[2][1 + NSC][128];    // (rho, rho X_s) of the halo cells: 64 x-halo cells, 64 y-halo cells
  double fx[2][2][16][17];        // (F_rho, Aq) of the low x faces of zones i = 0 .. 16 (16: the x+ neighbour's first zone)
  double fy[2][2][17][16];        // the same along y
  double late[2][NSC + 2][256];   // U0 of the plane's zones and the (F_rho, Aq) of their high z faces, per thread
};

__device__ __forceinline__ void cp_async8(void *dst, const void *src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// HLLC: Aq is F_rho where F_rho > 0 and 0 elsewhere (the flux is upwind in the sign of S*, which is the sign of the mass flux), so
// the fused kernel leaves F_rho alone for it and this pass reads half the face data.
__device__ __forceinline__ double fx_aq_hllc(double F) { return F > 0.0 ? F : 0.0; }

// AMRS: the plan has refinement jumps [B12-B14]: behind a jump face the halo abundances are the block's own guard zones'
// (interpolated by fx_k_amr_fill for every variable) and the scalars' fluxes through the jump faces are stored with the
// hydro variables' for the flux correction.
template <int NSC, bool FIRST, bool HLLC, bool AMRS = false>
__global__ void __launch_bounds__(256, 2) fx_k_scalar_march(const FxParams P, const double *__restrict__ X, const double *U0, double *out,
                                                            const double *__restrict__ dx, double dt, const double *__restrict__ dt_dev,
                                                            double beta, int sv0) {
  extern __shared__ __align__(16) unsigned char fx_scal_smem[];
  ScalSmem<NSC> &S = *reinterpret_cast<ScalSmem<NSC> *>(fx_scal_smem);
  const int b = blockIdx.x, tid = threadIdx.x, i = tid & 15, j = tid >> 4;
  const int nz = P.n[2];
  const int g0 = P.gd[0], g1 = P.gd[1], g2 = P.gd[2];
  int nb[6];
#pragma unroll
  for (int f = 0; f < 6; ++f) nb[f] = __ldg(&P.neigh[(long long)b * 6 + f]);
  const long long colo = (long long)(j + g1) * P.S_j + (i + g0);  // this column inside a block's plane
  const long long nzt = P.nblocks * (long long)nz * 256;
  const double *Q0 = X + (long long)sv0 * P.S_v, *U0q = U0 + (long long)sv0 * P.S_v;
  double *outq = out + (long long)sv0 * P.S_v;
  // this column's zone in plane k of the column (k in [-2, nz + 2)): the z neighbour's planes, or behind a physical
  // boundary this block's own edge plane (outflow) / mirror plane (wall: scalars and density are copied unchanged [B11])
  auto plane_off = [&](int k) -> long long {
    int blk = b, kk = k;
    if (k < 0) {
      if (nb[4] >= 0) { blk = nb[4]; kk = k + nz; }
      else if (!(AMRS && nb[4] <= FX_NEIGH_COARSER)) kk = nb[4] == FX_BC_REFLECT ? -1 - k : 0;  // (a jump: the own guard plane k)
    } else if (k >= nz) {
      if (nb[5] >= 0) { blk = nb[5]; kk = k - nz; }
      else if (!(AMRS && nb[5] <= FX_NEIGH_COARSER)) kk = nb[5] == FX_BC_REFLECT ? 2 * nz - 1 - k : nz - 1;
    }
    return (long long)blk * P.S_b + (long long)(kk + g2) * P.S_k + colo;
  };
  // the halo cell this thread also provides for each plane (threads in the two outermost columns / rows): where it comes
  // from inside the neighbour block's plane, its slot in the staging buffer, and where it goes in the shared plane
  const bool hx = i < 2 || i >= 14, hy = j < 2 || j >= 14;
  // (behind a physical boundary: the block's own edge cell, or its mirror cells at a wall)
  const int nxs = i < 2 ? nb[0] : nb[1], nys = j < 2 ? nb[2] : nb[3];
  const bool jx = AMRS && nxs <= FX_NEIGH_COARSER, jy = AMRS && nys <= FX_NEIGH_COARSER;  // a jump: the own guard zones behind the face
  const int xi = jx ? (i < 2 ? i - 2 : i + 2)
                    : (i < 2 ? (nxs >= 0 ? 14 + i : (nxs == FX_BC_REFLECT ? 1 - i : 0)) : (nxs >= 0 ? i - 14 : (nxs == FX_BC_REFLECT ? 29 - i : 15)));
  const int yj = jy ? (j < 2 ? j - 2 : j + 2)
                    : (j < 2 ? (nys >= 0 ? 14 + j : (nys == FX_BC_REFLECT ? 1 - j : 0)) : (nys >= 0 ? j - 14 : (nys == FX_BC_REFLECT ? 29 - j : 15)));
  const long long hxo = (long long)(nxs >= 0 ? nxs : b) * P.S_b + (long long)(j + g1) * P.S_j + (xi + g0);
  const long long hyo = (long long)(nys >= 0 ? nys : b) * P.S_b + (long long)(yj + g1) * P.S_j + (i + g0);
  const int hxs = j * 4 + (i < 2 ? i : i - 12), hys = 64 + (j < 2 ? j : j - 12) * 16 + i;
  const int hxc = i < 2 ? i : i + 4, hyr = j < 2 ? j : j + 4;
  const long long zb = (long long)b * nz * 256 + tid;
  // everything plane k needs before its barrier, into stage k & 1.  All addresses are running 64-bit offsets advanced by
  // one plane per call (the planes are prefetched in turn, k = 0, 1, ...): forming them from k each time cost a quarter of
  // the loop's instructions (215 of 847 integer instructions per plane were address arithmetic)
  long long e_pf = plane_off(2);              // new window cell of the plane being prefetched
  const long long top0 = plane_off(nz), top1 = plane_off(nz + 1);  // the two planes beyond the block's top
  // (the other offsets of a plane follow from its own-zone offset cpf and from kp: fewer values carried across the loop --
  // the spilled piece of one of them, reloaded from local memory behind the streaming cp.async traffic, was 10 % of the
  // stall samples)
  const long long hxr = hxo - ((long long)b * P.S_b + colo), hyr_o = hyo - ((long long)b * P.S_b + colo);
  // a zone's HIGH-face data are the next zone's low-face values; behind a block face: the neighbour block's, if that is an
  // owned same-level block -- else (physical boundary, ghost block) what the fused kernel's 17th-face solve left in P.fqb
  // Resolved once per thread: where the data of plane 0 are (x: thread i = 15 of row j; y: thread j = 15 of column i), how
  // far apart two planes' are (256 zones in the neighbour block, 16 on a stored face), and for z the block's top face.
  auto owned = [&](int h) { return h >= 0 && h < P.nown; };
  const long long fqbc = 3 * P.nblocks * (long long)P.fqb_area;  // (F_rho -> Aq in P.fqb)
  const bool ox = owned(nb[1]), oy = owned(nb[3]), oz = owned(nb[5]);
  const double *const hsx = ox ? P.fq + (long long)nb[1] * nz * 256 + j * 16 : P.fqb + (long long)b * P.fqb_area + j;
  const double *const hsy = oy ? P.fq + 2 * nzt + (long long)nb[3] * nz * 256 + i : P.fqb + (P.nblocks + b) * (long long)P.fqb_area + i;
  const double *const hsz = oz ? P.fq + 4 * nzt + (long long)nb[5] * nz * 256 + tid : P.fqb + (2 * P.nblocks + b) * (long long)P.fqb_area + tid;
  auto prefetch = [&](int kp, long long cpf) {  // called for kp = 0, 1, 2, ... in turn; cpf: this thread's zone of plane kp
    const int st = kp & 1;
    {
      const double *p = Q0 + e_pf;
      cp_async8(&S.raw[st][0][tid], X + e_pf);
#pragma unroll
      for (int s = 0; s < NSC; ++s, p += P.S_v) cp_async8(&S.raw[st][1 + s][tid], p);
    }
    if (hx) {
      const long long o = cpf + hxr;
      const double *p = Q0 + o;
      cp_async8(&S.hal[st][0][hxs], X + o);
#pragma unroll
      for (int s = 0; s < NSC; ++s, p += P.S_v) cp_async8(&S.hal[st][1 + s][hxs], p);
    }
    if (hy) {
      const long long o = cpf + hyr_o;
      const double *p = Q0 + o;
      cp_async8(&S.hal[st][0][hys], X + o);
#pragma unroll
      for (int s = 0; s < NSC; ++s, p += P.S_v) cp_async8(&S.hal[st][1 + s][hys], p);
    }
    const double *f = P.fq + zb + ((long long)kp << 8);
    cp_async8(&S.fx[st][0][j][i], f);
    if (!HLLC) cp_async8(&S.fx[st][1][j][i], f + nzt);
    cp_async8(&S.fy[st][0][j][i], f + 2 * nzt);
    if (!HLLC) cp_async8(&S.fy[st][1][j][i], f + 3 * nzt);
    if (i == 15) {
      const double *h = hsx + kp * (ox ? 256 : 16);
      cp_async8(&S.fx[st][0][j][16], h);
      if (!HLLC) cp_async8(&S.fx[st][1][j][16], h + (ox ? nzt : fqbc));
    }
    if (j == 15) {
      const double *h = hsy + kp * (oy ? 256 : 16);
      cp_async8(&S.fy[st][0][16][i], h);
      if (!HLLC) cp_async8(&S.fy[st][1][16][i], h + (oy ? nzt : fqbc));
    }
    {  // what only the end of the plane needs (it comes from DRAM: fetched a plane ahead like the rest)
      const double *pu = U0q + cpf;
#pragma unroll
      for (int s = 0; s < NSC; ++s, pu += P.S_v) cp_async8(&S.late[st][s][tid], pu);
      const bool top = kp + 1 >= nz;
      const double *fzh = top ? hsz : f + 4 * nzt + 256;
      cp_async8(&S.late[st][NSC][tid], fzh);
      if (!HLLC) cp_async8(&S.late[st][NSC + 1][tid], fzh + ((top && !oz) ? fqbc : nzt));
    }
    cp_async_commit();
    e_pf = kp + 3 == nz ? top0 : (kp + 3 == nz + 1 ? top1 : e_pf + P.S_k);  // (beyond the block's top: wherever those planes live)
  };
  prefetch(0, (long long)b * P.S_b + (long long)g2 * P.S_k + colo);
  if (dt_dev) dt = *dt_dev;
  const double rd0 = dt / __ldg(&dx[b * 3 + 0]), rd1 = dt / __ldg(&dx[b * 3 + 1]), rd2 = dt / __ldg(&dx[b * 3 + 2]);
  // abundances: (rho X_s) / max(rho, floor), the reciprocal as the hydro part forms it
  auto abund = [&](double rho, const double q[NSC], double x[NSC]) {
    if (rho < P.rho_floor) rho = P.rho_floor;
    const double ri = fx_rcp3(rho);
#pragma unroll
    for (int s = 0; s < NSC; ++s) x[s] = q[s] * ri;
  };
  auto abund_at = [&](long long e, double x[NSC]) {
    const double rho = X[e];
    double q[NSC];
#pragma unroll
    for (int s = 0; s < NSC; ++s) q[s] = Q0[s * P.S_v + e];
    abund(rho, q, x);
  };
  // z direction, carried from plane to plane: X of cells k and k+1, the plus value of cell k, and the scalar flux through
  // the low z face of cell k (the high face's of the plane before)
  double xw[2][NSC], apc[NSC], Fz[NSC];
  {
    double xm2[NSC], xm1[NSC], am, ap;
    abund_at(plane_off(-2), xm2);
    abund_at(plane_off(-1), xm1);
    abund_at(plane_off(0), xw[0]);
    abund_at(plane_off(1), xw[1]);
    const double Fl = P.fq[4 * nzt + zb], Al = HLLC ? fx_aq_hllc(Fl) : P.fq[5 * nzt + zb];
#pragma unroll
    for (int s = 0; s < NSC; ++s) {
      double apm;
      fx_plm(xm2[s], xm1[s], xw[0][s], am, apm);
      fx_plm(xm1[s], xw[0][s], xw[1][s], am, ap);
      apc[s] = ap;
      Fz[s] = Al * apm + (Fl - Al) * am;
    }
  }
  // AMRS: which of this zone column's faces are jump faces of the block (bit f: face f; z faces at the first / last plane)
  unsigned cap = 0;
  if (AMRS) {
    cap = (i == 0 && nb[0] <= FX_NEIGH_COARSER ? 1u : 0u) | (i == 15 && nb[1] <= FX_NEIGH_COARSER ? 2u : 0u) |
          (j == 0 && nb[2] <= FX_NEIGH_COARSER ? 4u : 0u) | (j == 15 && nb[3] <= FX_NEIGH_COARSER ? 8u : 0u) |
          (nb[4] <= FX_NEIGH_COARSER ? 16u : 0u) | (nb[5] <= FX_NEIGH_COARSER ? 32u : 0u);
    if (cap & 16u) {
#pragma unroll
      for (int s = 0; s < NSC; ++s) P.fjump[(((long long)b * 6 + 4) * P.nvars + sv0 + s) * P.fj_area + tid] = Fz[s];
    }
  }
  unsigned hit = 0;
  int hmax = 0;  // largest upper word (sign cleared) of the results: Inf / NaN anywhere in a flux reaches the result
  // this thread's zone of the current plane: in fq (zone of the plane above: the z face's data) and in the state arrays
  long long c = (long long)b * P.S_b + (long long)g2 * P.S_k + colo;
#pragma unroll 2  // (two planes per trip: the staging buffer's index is a constant, the carried values rotate without moves)
  for (int k = 0; k < nz; ++k, c += P.S_k) {
    const int buf = k & 1;
    cp_async_wait_all();  // this thread's part of stage k
    double xn[NSC];
    {
      double q[NSC];
#pragma unroll
      for (int s = 0; s < NSC; ++s) q[s] = S.raw[buf][1 + s][tid];
      abund(S.raw[buf][0][tid], q, xn);
    }
#pragma unroll
    for (int s = 0; s < NSC; ++s) S.XS[buf][s][j + 2][i + 2] = xw[0][s];
    if (hx) {
      double q[NSC], xh[NSC];
#pragma unroll
      for (int s = 0; s < NSC; ++s) q[s] = S.hal[buf][1 + s][hxs];
      abund(S.hal[buf][0][hxs], q, xh);
#pragma unroll
      for (int s = 0; s < NSC; ++s) S.XS[buf][s][j + 2][hxc] = xh[s];
    }
    if (hy) {
      double q[NSC], yh[NSC];
#pragma unroll
      for (int s = 0; s < NSC; ++s) q[s] = S.hal[buf][1 + s][hys];
      abund(S.hal[buf][0][hys], q, yh);
#pragma unroll
      for (int s = 0; s < NSC; ++s) S.XS[buf][s][hyr][i + 2] = yh[s];
    }
    __syncthreads();  // plane k's X and (F_rho, Aq) complete; every thread is done with plane k-1 (stage buf ^ 1)
    if (k + 1 < nz) prefetch(k + 1, c + P.S_k);
    const double Fzh = S.late[buf][NSC][tid], Azh = HLLC ? fx_aq_hllc(Fzh) : S.late[buf][NSC + 1][tid];
    double xs[NSC];
    if (!FIRST) {
      const double *px = Q0 + c;
#pragma unroll
      for (int s = 0; s < NSC; ++s, px += P.S_v) xs[s] = *px;
    }
    double *po = outq + c;
    const double F0[2] = {S.fx[buf][0][j][i], S.fx[buf][0][j][i + 1]}, F1[2] = {S.fy[buf][0][j][i], S.fy[buf][0][j + 1][i]};
    double A0[2], A1[2];
    if (HLLC) {
      A0[0] = fx_aq_hllc(F0[0]); A0[1] = fx_aq_hllc(F0[1]);
      A1[0] = fx_aq_hllc(F1[0]); A1[1] = fx_aq_hllc(F1[1]);
    } else {
      A0[0] = S.fx[buf][1][j][i]; A0[1] = S.fx[buf][1][j][i + 1];
      A1[0] = S.fy[buf][1][j][i]; A1[1] = S.fy[buf][1][j + 1][i];
    }
    // (AMRS: face f0 / f0 + 1 of the block is the zone's low / high face and a jump: the fluxes are stored [B14])
    auto flux = [&](const double x[5], double rd, const double Fd[2], const double Ad[2], int f0, int t, int sv) {
      double am[3], ap[3];
#pragma unroll
      for (int n = 0; n < 3; ++n) fx_plm(x[n], x[n + 1], x[n + 2], am[n], ap[n]);
      const double Fm = Ad[0] * ap[0] + (Fd[0] - Ad[0]) * am[1];
      const double Fp = Ad[1] * ap[1] + (Fd[1] - Ad[1]) * am[2];
      if (AMRS && ((cap >> f0) & 3u)) {
        double *dst = P.fjump + (((long long)b * 6 + f0) * P.nvars + sv) * P.fj_area + t;
        if ((cap >> f0) & 1u) dst[0] = Fm;
        if ((cap >> f0) & 2u) dst[(long long)P.nvars * P.fj_area] = Fp;
      }
      return rd * (Fp - Fm);
    };
    double Sv[NSC];
#pragma unroll
    for (int s = 0; s < NSC; ++s) {
      double x[5], Ss = 0.0;
#pragma unroll
      for (int m = 0; m < 5; ++m) x[m] = m == 2 ? xw[0][s] : S.XS[buf][s][j + 2][i + m];  // (the centre is in the z window)
      Ss += flux(x, rd0, F0, A0, 0, k * 16 + j, sv0 + s);
#pragma unroll
      for (int m = 0; m < 5; ++m) x[m] = m == 2 ? xw[0][s] : S.XS[buf][s][j + m][i + 2];
      Ss += flux(x, rd1, F1, A1, 2, k * 16 + i, sv0 + s);
      {  // z: the new face only
        double amn, apn;
        fx_plm(xw[0][s], xw[1][s], xn[s], amn, apn);
        const double Fp = Azh * apc[s] + (Fzh - Azh) * amn;
        if (AMRS && (cap & 32u) && k == nz - 1) P.fjump[(((long long)b * 6 + 5) * P.nvars + sv0 + s) * P.fj_area + tid] = Fp;
        Ss += rd2 * (Fp - Fz[s]);
        Fz[s] = Fp;
        apc[s] = apn;
        xw[0][s] = xw[1][s];
        xw[1][s] = xn[s];
      }
      Sv[s] = Ss;
    }
#pragma unroll
    for (int s = 0; s < NSC; ++s) {
      const double Ss = Sv[s];
      const double u0 = S.late[buf][s][tid];
      const double res = FIRST ? (u0 - Ss) : (u0 + beta * ((xs[s] - u0) - Ss));
      *po = res;
      po += P.S_v;
      hmax = max(hmax, __double2hiint(res) & 0x7fffffff);
    }
  }
  if (hmax >= 0x7ff00000) hit |= FX_STATUS_NONFINITE;
  if (hit) fx_note(P, hit);
}

template <int NSC, bool FIRST, bool HLLC>
static int fx_scalar_march_launch2(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt,
                                   const double *dt_dev, double beta, int sv0, cudaStream_t st) {
  const int smem = (int)sizeof(ScalSmem<NSC>);
  if (P.has_jumps) {
    FX_CUDA(cudaFuncSetAttribute(fx_k_scalar_march<NSC, FIRST, HLLC, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    fx_k_scalar_march<NSC, FIRST, HLLC, true><<<(unsigned)P.nown, 256, smem, st>>>(P, X, U0, out, dx, dt, dt_dev, beta, sv0);
    FX_LAUNCH_CHECK("scalar_march");
    return FX_OK;
  }
  FX_CUDA(cudaFuncSetAttribute(fx_k_scalar_march<NSC, FIRST, HLLC>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  fx_k_scalar_march<NSC, FIRST, HLLC><<<(unsigned)P.nown, 256, smem, st>>>(P, X, U0, out, dx, dt, dt_dev, beta, sv0);
  FX_LAUNCH_CHECK("scalar_march");
  return FX_OK;
}

template <int NSC>
static int fx_scalar_march_launch(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt,
                                  const double *dt_dev, double beta, int first, int sv0, cudaStream_t st) {
  const bool hllc = P.riemann == FX_RIEMANN_HLLC;
  if (first) return hllc ? fx_scalar_march_launch2<NSC, true, true>(P, X, U0, out, dx, dt, dt_dev, beta, sv0, st)
                         : fx_scalar_march_launch2<NSC, true, false>(P, X, U0, out, dx, dt, dt_dev, beta, sv0, st);
  return hllc ? fx_scalar_march_launch2<NSC, false, true>(P, X, U0, out, dx, dt, dt_dev, beta, sv0, st)
              : fx_scalar_march_launch2<NSC, false, false>(P, X, U0, out, dx, dt, dt_dev, beta, sv0, st);
}

}  // namespace

bool fx_scalar_pass_supported(const FxParams &P) {
  // The marching form serves 16 x 16 x nz blocks with same-level neighbours, physical boundaries (outflow, walls) and ghost
  // blocks behind their faces (the high-face data behind such a face are the fused kernel's own 17th-face solve, P.fqb);
  // gravity acts on the hydro variables only [B11]; refinement jumps (AMRS variant) on the fused AMR path.
  return P.nvars > 5 && P.recon == FX_RECON_PLM_MINMOD && (!P.has_jumps || P.fjump != nullptr) && P.fq != nullptr && P.fqb != nullptr && P.n[0] == 16 &&
         P.n[1] == 16 && P.n[2] >= 2 && P.active[0] && P.active[1] && P.active[2];
}

int fx_launch_scalar_pass(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt,
                          const double *dt_dev, double beta, int first, cudaStream_t st) {
  if (P.nown == 0 || P.nvars <= 5) return FX_OK;
  if (!fx_scalar_pass_supported(P)) return fx_fail(FX_ERR_UNSUPPORTED, "scalar pass: PLM and 16 x 16 x nz blocks only");
  for (int sv = 5; sv < P.nvars; sv += 4) {  // up to four scalars per launch
    const int n = P.nvars - sv < 4 ? P.nvars - sv : 4;
    int rc;
    if (n == 4) rc = fx_scalar_march_launch<4>(P, X, U0, out, dx, dt, dt_dev, beta, first, sv, st);
    else if (n == 3) rc = fx_scalar_march_launch<3>(P, X, U0, out, dx, dt, dt_dev, beta, first, sv, st);
    else if (n == 2) rc = fx_scalar_march_launch<2>(P, X, U0, out, dx, dt, dt_dev, beta, first, sv, st);
    else rc = fx_scalar_march_launch<1>(P, X, U0, out, dx, dt, dt_dev, beta, first, sv, st);
    if (rc) return rc;
  }
  return FX_OK;
}
