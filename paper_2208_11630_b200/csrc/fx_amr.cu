// fx_amr.cu -- fine-coarse boundaries [B12-B14; "fine-coarse boundary resolution related API functions of
// the Grid unit"]: the face guard zones behind a refinement jump (restriction of the finer blocks' interiors, conservative
// limited prolongation from the coarser block) and the flux correction of coarse face fluxes.  Written from the readings
// in DESIGN.md section 2; shares nothing with oracle/.
//
// Both fills are pure functions of INTERIOR zones (a coarse zone's neighbour behind a face is resolved by one hop: the
// same-level neighbour's interior, the boundary condition, or the restriction of finer interiors), so one launch fills
// every jump face of every level at once and needs no ordering.  The arithmetic is written with explicit _rn operations
// in the oracle's order (children summed i fastest, then j, then k; slopes added x, y, z): the filled zones are bit for
// bit the oracle's (tested).
#include "fx_internal.h"

namespace {

__device__ __forceinline__ double amr_minmod(double a, double b) {  // comparison form [A4]
  if (a > 0.0 && b > 0.0) return a < b ? a : b;
  if (a < 0.0 && b < 0.0) return a > b ? a : b;
  return 0.0;
}

// Variable v of the zone at interior coordinates c of block cb; at most one coordinate outside [0, n): one hop [B13].
// Returns false behind a coarser jump (undefined there).
__device__ bool amr_zone(const FxParams &P, const double *__restrict__ X, long long cb, const int cin[3], int v, double &val) {
  int c[3] = {cin[0], cin[1], cin[2]};
  double sign = 1.0;
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    if (c[d] >= 0 && c[d] < P.n[d]) continue;
    const int side = c[d] >= P.n[d], f = 2 * d + side;
    const int nb = __ldg(&P.neigh[cb * 6 + f]);
    if (nb >= 0) {
      cb = nb;
      c[d] += side ? -P.n[d] : P.n[d];
    } else if (nb == FX_BC_REFLECT) {
      c[d] = side ? 2 * P.n[d] - 1 - c[d] : -1 - c[d];
      if (v == 1 + d) sign = -1.0;
    } else if (nb == FX_NEIGH_FINER) {
      const int tr[2] = {d == 0 ? 1 : 0, d == 2 ? 1 : 2};
      int q = 0, fc[3], cnt[3];
#pragma unroll
      for (int t = 0; t < 2; ++t) {
        const int e = tr[t];
        if (!P.active[e]) { fc[e] = 0; cnt[e] = 1; continue; }
        const int half = c[e] >= P.n[e] / 2;
        q |= half << t;
        fc[e] = 2 * (c[e] - half * (P.n[e] / 2));
        cnt[e] = 2;
      }
      const int m = side ? c[d] - P.n[d] : -1 - c[d];
      fc[d] = side ? 2 * m : P.n[d] - 2 - 2 * m;
      cnt[d] = 2;
      const long long fb = __ldg(&P.jump[(cb * 6 + f) * 4 + q]);
      double sum = 0.0;
      for (int kk = 0; kk < cnt[2]; ++kk)
        for (int jj = 0; jj < cnt[1]; ++jj)
          for (int ii = 0; ii < cnt[0]; ++ii)
            sum = __dadd_rn(sum, X[v * P.S_v + fb * P.S_b + (long long)(fc[2] + kk + P.gd[2]) * P.S_k +
                                   (long long)(fc[1] + jj + P.gd[1]) * P.S_j + (fc[0] + ii + P.gd[0])]);
      val = __dmul_rn(sum, 1.0 / (double)(cnt[0] * cnt[1] * cnt[2]));
      return true;
    } else if (nb == FX_NEIGH_COARSER) {
      return false;
    } else {
      c[d] = side ? P.n[d] - 1 : 0;  // outflow
    }
    break;  // one hop
  }
  val = sign * X[v * P.S_v + cb * P.S_b + (long long)(c[2] + P.gd[2]) * P.S_k + (long long)(c[1] + P.gd[1]) * P.S_j + (c[0] + P.gd[0])];
  return true;
}

// One CTA per (block, face); threads over the face guard zones of depth `depth` and the variables.
__global__ void __launch_bounds__(128) fx_k_amr_fill(const FxParams P, double *U, int depth) {
  const long long b = blockIdx.x / 6;
  const int f = blockIdx.x % 6, d = f >> 1, side = f & 1;
  if (!P.active[d]) return;
  const int code = __ldg(&P.neigh[b * 6 + f]);
  if (code != FX_NEIGH_COARSER && code != FX_NEIGH_FINER) return;
  const int d1 = d == 0 ? 1 : 0, d2 = d == 2 ? 1 : 2;
  const int n1 = P.n[d1], n2 = P.n[d2];
  const int total = depth * n1 * n2 * P.nvars;
  for (int t = threadIdx.x; t < total; t += blockDim.x) {
    const int v = t / (depth * n1 * n2), r = t - v * (depth * n1 * n2);
    const int m = r / (n1 * n2), r2 = r - m * (n1 * n2), t2 = r2 / n1, t1 = r2 - t2 * n1;
    int c[3];
    c[d] = side ? P.n[d] + m : -1 - m;
    c[d1] = t1;
    c[d2] = t2;
    const long long e = v * P.S_v + b * P.S_b + (long long)(c[2] + P.gd[2]) * P.S_k + (long long)(c[1] + P.gd[1]) * P.S_j + (c[0] + P.gd[0]);
    double val = 0.0;
    if (code == FX_NEIGH_FINER) {
      amr_zone(P, U, b, c, v, val);
    } else {
      const long long cb = __ldg(&P.jump[(b * 6 + f) * 4 + 0]);
      const int qd = __ldg(&P.jump[(b * 6 + f) * 4 + 1]);
      int C[3] = {0, 0, 0};
      double sg[3] = {0.0, 0.0, 0.0};
      C[d] = side ? m / 2 : P.n[d] - 1 - m / 2;
      sg[d] = ((m % 2 == 0) == (side == 0)) ? 1.0 : -1.0;
      const int tr[2] = {d1, d2}, tc[2] = {t1, t2};
#pragma unroll
      for (int t_ = 0; t_ < 2; ++t_) {
        const int e2 = tr[t_];
        if (!P.active[e2]) continue;
        C[e2] = ((qd >> t_) & 1) * (P.n[e2] / 2) + tc[t_] / 2;
        sg[e2] = (tc[t_] % 2) ? 1.0 : -1.0;
      }
      double qC;
      amr_zone(P, U, cb, C, v, qC);
      val = qC;
#pragma unroll
      for (int e2 = 0; e2 < 3; ++e2) {
        if (!P.active[e2]) continue;
        int Cm[3] = {C[0], C[1], C[2]}, Cp[3] = {C[0], C[1], C[2]};
        Cm[e2] -= 1;
        Cp[e2] += 1;
        double qm, qp;
        if (amr_zone(P, U, cb, Cm, v, qm) && amr_zone(P, U, cb, Cp, v, qp))
          val = __dadd_rn(val, __dmul_rn(sg[e2] * 0.25, amr_minmod(__dsub_rn(qC, qm), __dsub_rn(qp, qC))));
      }
    }
    U[e] = val;
  }
}

// Flux correction [B14]: one CTA per (block, face) with finer neighbours; out -= (+-) beta dt/dx (mean of the fine fluxes
// - the block's own flux) in the zones next to the face.  fjump[((b 6 + f) 5 + v) A + t2 n1 + t1] holds the boundary
// fluxes the stage kernel captured at every jump face (both sides).
__global__ void __launch_bounds__(128) fx_k_amr_flux_correct(const FxParams P, double *out, const double *__restrict__ dx, double dt,
                                                             const double *__restrict__ dt_dev, double beta) {
  const long long b = blockIdx.x / 6;
  const int f = blockIdx.x % 6, d = f >> 1, side = f & 1;
  if (!P.active[d] || __ldg(&P.neigh[b * 6 + f]) != FX_NEIGH_FINER) return;
  if (dt_dev) dt = *dt_dev;
  const int d1 = d == 0 ? 1 : 0, d2 = d == 2 ? 1 : 2;
  const int n1 = P.n[d1], n2 = P.n[d2];
  const long long A = (long long)P.fj_area;
  const double r = beta * (dt / __ldg(&dx[b * 3 + d]));
  for (int t = threadIdx.x; t < 5 * n1 * n2; t += blockDim.x) {
    const int v = t / (n1 * n2), r2 = t - v * (n1 * n2), t2 = r2 / n1, t1 = r2 - t2 * n1;
    const int tr[2] = {d1, d2}, tc[2] = {t1, t2};
    int q = 0, ft[2] = {0, 0}, cnt[2] = {1, 1};
#pragma unroll
    for (int t_ = 0; t_ < 2; ++t_) {
      const int e = tr[t_];
      if (!P.active[e]) continue;
      const int half = tc[t_] >= P.n[e] / 2;
      q |= half << t_;
      ft[t_] = 2 * (tc[t_] - half * (P.n[e] / 2));
      cnt[t_] = 2;
    }
    const long long fb = __ldg(&P.jump[(b * 6 + f) * 4 + q]);
    const int ff = 2 * d + (1 - side);
    double sum = 0.0;
    for (int j2 = 0; j2 < cnt[1]; ++j2)
      for (int j1 = 0; j1 < cnt[0]; ++j1) sum += P.fjump[((fb * 6 + ff) * 5 + v) * A + (long long)(ft[1] + j2) * n1 + (ft[0] + j1)];
    const double fbar = sum * (1.0 / (double)(cnt[0] * cnt[1]));
    const double fown = P.fjump[((b * 6 + f) * 5 + v) * A + (long long)t2 * n1 + t1];
    int c[3];
    c[d] = side ? P.n[d] - 1 : 0;
    c[d1] = t1;
    c[d2] = t2;
    const long long e = v * P.S_v + b * P.S_b + (long long)(c[2] + P.gd[2]) * P.S_k + (long long)(c[1] + P.gd[1]) * P.S_j + (c[0] + P.gd[0]);
    // S = sum r (F+ - F-): a corrected high-face flux adds r (fbar - fown) to S, a low-face one subtracts it; out = .. - beta S
    out[e] += (side ? -r : r) * (fbar - fown);
  }
}

}  // namespace

int fx_launch_amr_fill(const FxParams &P, double *U, int depth, cudaStream_t st) {
  if (!P.jump || !P.has_jumps || P.nblocks == 0) return FX_OK;
  fx_k_amr_fill<<<(unsigned)(P.nblocks * 6), 128, 0, st>>>(P, U, depth);
  FX_LAUNCH_CHECK("amr_fill");
  return FX_OK;
}

int fx_launch_amr_flux_correct(const FxParams &P, double *out, const double *dx, double dt, const double *dt_dev, double beta,
                               cudaStream_t st) {
  if (!P.jump || !P.has_jumps || P.nown == 0) return FX_OK;
  fx_k_amr_flux_correct<<<(unsigned)(P.nown * 6), 128, 0, st>>>(P, out, dx, dt, dt_dev, beta);
  FX_LAUNCH_CHECK("amr_flux_correct");
  return FX_OK;
}
