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

// Where the zone at interior coordinates c of block cb lives; at most one coordinate outside [0, n): one hop [B13].  The
// location is the same for every variable, so it is resolved once (kind 0: the zone at element `off` of each variable, its
// `flipv` momentum negated behind a reflecting wall; kind 1: the restriction of the cnt[0] x cnt[1] x cnt[2] finer zones that
// start at `off`) and then evaluated per variable.  Returns false behind a coarser jump (undefined there).
struct AmrSrc {
  long long off;
  int kind, flipv, cnt[3];
};

__device__ __forceinline__ bool amr_locate(const FxParams &P, long long cb, const int cin[3], AmrSrc &s) {
  int c[3] = {cin[0], cin[1], cin[2]};
  s.kind = 0;
  s.flipv = -1;
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
      s.flipv = 1 + d;
    } else if (nb == FX_NEIGH_FINER) {
      const int tr[2] = {d == 0 ? 1 : 0, d == 2 ? 1 : 2};
      int q = 0, fc[3];
#pragma unroll
      for (int t = 0; t < 2; ++t) {
        const int e = tr[t];
        if (!P.active[e]) { fc[e] = 0; s.cnt[e] = 1; continue; }
        const int half = c[e] >= P.n[e] / 2;
        q |= half << t;
        fc[e] = 2 * (c[e] - half * (P.n[e] / 2));
        s.cnt[e] = 2;
      }
      const int m = side ? c[d] - P.n[d] : -1 - c[d];
      fc[d] = side ? 2 * m : P.n[d] - 2 - 2 * m;
      s.cnt[d] = 2;
      const long long fb = __ldg(&P.jump[(cb * 6 + f) * 4 + q]);
      s.kind = 1;
      s.off = fb * P.S_b + (long long)(fc[2] + P.gd[2]) * P.S_k + (long long)(fc[1] + P.gd[1]) * P.S_j + (fc[0] + P.gd[0]);
      return true;
    } else if (nb == FX_NEIGH_COARSER) {
      return false;
    } else {
      c[d] = side ? P.n[d] - 1 : 0;  // outflow
    }
    break;  // one hop
  }
  s.off = cb * P.S_b + (long long)(c[2] + P.gd[2]) * P.S_k + (long long)(c[1] + P.gd[1]) * P.S_j + (c[0] + P.gd[0]);
  return true;
}

__device__ __forceinline__ double amr_value(const FxParams &P, const double *__restrict__ X, const AmrSrc &s, int v) {
  const double *Xv = X + (long long)v * P.S_v + s.off;
  if (s.kind == 0) {
    const double x = *Xv;
    return v == s.flipv ? -x : x;
  }
  // children summed i fastest, then j, then k; all (up to eight) loads issued before the first addition -- as a loop with
  // run-time counts every addition waited for its own load, eight memory round trips per value
  double x[8];
#pragma unroll
  for (int t = 0; t < 8; ++t) {
    const bool on = (t & 1) < s.cnt[0] && ((t >> 1) & 1) < s.cnt[1] && (t >> 2) < s.cnt[2];
    x[t] = on ? Xv[(t >> 2) * P.S_k + ((t >> 1) & 1) * P.S_j + (t & 1)] : 0.0;
  }
  double sum = 0.0;
#pragma unroll
  for (int t = 0; t < 8; ++t) {
    const bool on = (t & 1) < s.cnt[0] && ((t >> 1) & 1) < s.cnt[1] && (t >> 2) < s.cnt[2];
    sum = on ? __dadd_rn(sum, x[t]) : sum;
  }
  return __dmul_rn(sum, 1.0 / (double)(s.cnt[0] * s.cnt[1] * s.cnt[2]));
}

// CTAs of 64 threads per (block, face).  Behind finer neighbours a thread per face guard zone of depth `depth` (the zones
// split over the grid's y extent): it resolves the one location its data comes from and evaluates all variables.  Behind a
// coarser neighbour a thread per parent zone (below).  (First version: a thread per zone AND variable, 128 threads per CTA,
// every value resolving its seven locations itself, the restriction a loop whose every addition waited for its own load:
// 0.43 ms per fill on the two-level workload of bench.py --amr, a fifth of the step; a thread per guard zone on both sides,
// 256 threads: 0.23 ms; a thread per parent zone in 256-thread CTAs: 188 registers, one CTA per SM with two busy warps,
// 0.29 ms; 64-thread CTAs held to 128 registers, eight per SM: 0.11 ms.)
__global__ void __launch_bounds__(64, 8) fx_k_amr_fill(const FxParams P, double *U, int depth) {
  // (the grid is the list of jump faces where the plan has one: a CTA per face of EVERY block, most of which only look
  // their face up and leave, took 0.07 ms more.  The face's dimension as a template parameter -- no dynamically indexed
  // coordinate triples -- was slower both ways: as three branches of this kernel 0.27 against 0.23 ms, as three launches
  // over a list sorted by dimension 0.17 + 0.13 + 0.12 ms (165 registers, a third of the CTAs each).)
  const long long bf = P.jface ? (long long)__ldg(&P.jface[blockIdx.x]) : (long long)blockIdx.x;
  const long long b = bf / 6;
  const int f = (int)(bf % 6), d = f >> 1, side = f & 1;
  if (!P.active[d]) return;
  const int code = __ldg(&P.neigh[b * 6 + f]);
  if (code != FX_NEIGH_COARSER && code != FX_NEIGH_FINER) return;
  const int d1 = d == 0 ? 1 : 0, d2 = d == 2 ? 1 : 2;
  const int n1 = P.n[d1], n2 = P.n[d2];
  if (code == FX_NEIGH_FINER) {
    const int total = depth * n1 * n2;
    for (int r = threadIdx.x + blockDim.x * blockIdx.y; r < total; r += blockDim.x * gridDim.y) {
      const int m = r / (n1 * n2), r2 = r - m * (n1 * n2), t2 = r2 / n1, t1 = r2 - t2 * n1;
      int c[3];
      c[d] = side ? P.n[d] + m : -1 - m;
      c[d1] = t1;
      c[d2] = t2;
      double *dst = U + b * P.S_b + (long long)(c[2] + P.gd[2]) * P.S_k + (long long)(c[1] + P.gd[1]) * P.S_j + (c[0] + P.gd[0]);
      // (every value a zone needs is loaded before its first store: the loads of all variables are then in flight together
      // instead of one DRAM round trip per variable)
      AmrSrc s;
      amr_locate(P, b, c, s);
      for (int v0 = 0; v0 < P.nvars; v0 += 5) {  // (five variables at a time: the hydro set, then the passive scalars)
        double val[5];
#pragma unroll
        for (int v = 0; v < 5; ++v)
          if (v0 + v < P.nvars) val[v] = amr_value(P, U, s, v0 + v);
#pragma unroll
        for (int v = 0; v < 5; ++v)
          if (v0 + v < P.nvars) dst[(long long)(v0 + v) * P.S_v] = val[v];
      }
    }
    return;
  }
  if (blockIdx.y) return;  // (the grid's y extent splits the restriction faces' zones only)
  // Behind a coarser neighbour: a thread per PARENT zone of the neighbour.  The (up to eight) guard zones it covers share
  // the parent's value, its two neighbours per active dimension and so the limited slopes; only the signs of the quarter
  // offsets differ.  (A thread per guard zone resolved the same seven locations and loaded the same values eight times over:
  // 2400 warp instructions per 32 zones, 0.23 ms per fill of the two-level workload.)
  const long long cb = __ldg(&P.jump[(b * 6 + f) * 4 + 0]);
  const int qd = __ldg(&P.jump[(b * 6 + f) * 4 + 1]);
  const int a1 = P.active[d1] ? 2 : 1, a2 = P.active[d2] ? 2 : 1;  // children per parent across the face
  const int p1n = n1 / a1, p2n = n2 / a2, pmn = (depth + 1) / 2;
  for (int r = threadIdx.x; r < pmn * p1n * p2n; r += blockDim.x) {
    const int mc = r / (p1n * p2n), r2 = r - mc * (p1n * p2n), p2 = r2 / p1n, p1 = r2 - p2 * p1n;
    int C[3] = {0, 0, 0};
    C[d] = side ? mc : P.n[d] - 1 - mc;
    if (P.active[d1]) C[d1] = ((qd >> 0) & 1) * (P.n[d1] / 2) + p1;
    if (P.active[d2]) C[d2] = ((qd >> 1) & 1) * (P.n[d2] / 2) + p2;
    AmrSrc sC, sm[3], sp[3];
    bool both[3] = {false, false, false};
    amr_locate(P, cb, C, sC);
#pragma unroll
    for (int e2 = 0; e2 < 3; ++e2) {
      if (!P.active[e2]) continue;
      int Cm[3] = {C[0], C[1], C[2]}, Cp[3] = {C[0], C[1], C[2]};
      Cm[e2] -= 1;
      Cp[e2] += 1;
      both[e2] = amr_locate(P, cb, Cm, sm[e2]) && amr_locate(P, cb, Cp, sp[e2]);
    }
    for (int v0 = 0; v0 < P.nvars; v0 += 5) {
      double qC[5], qm[3][5], qp[3][5];
#pragma unroll
      for (int v = 0; v < 5; ++v)
        if (v0 + v < P.nvars) qC[v] = amr_value(P, U, sC, v0 + v);
#pragma unroll
      for (int e2 = 0; e2 < 3; ++e2) {
        if (!both[e2]) continue;
#pragma unroll
        for (int v = 0; v < 5; ++v) {
          if (v0 + v >= P.nvars) continue;
          qm[e2][v] = amr_value(P, U, sm[e2], v0 + v);
          qp[e2][v] = amr_value(P, U, sp[e2], v0 + v);
        }
      }
      double sl[3][5];  // the limited slopes, per dimension and variable
#pragma unroll
      for (int e2 = 0; e2 < 3; ++e2)
#pragma unroll
        for (int v = 0; v < 5; ++v)
          sl[e2][v] = (both[e2] && v0 + v < P.nvars) ? amr_minmod(__dsub_rn(qC[v], qm[e2][v]), __dsub_rn(qp[e2][v], qC[v])) : 0.0;
      for (int ch = 0; ch < 2 * a1 * a2; ++ch) {
        const int b1 = ch % a1, b2 = (ch / a1) % a2, mm = ch / (a1 * a2), m = 2 * mc + mm;
        if (m >= depth) continue;
        int c[3];
        double sg[3] = {0.0, 0.0, 0.0};
        c[d] = side ? P.n[d] + m : -1 - m;
        c[d1] = a1 * p1 + b1;
        c[d2] = a2 * p2 + b2;
        sg[d] = ((mm == 0) == (side == 0)) ? 1.0 : -1.0;
        if (P.active[d1]) sg[d1] = b1 ? 1.0 : -1.0;
        if (P.active[d2]) sg[d2] = b2 ? 1.0 : -1.0;
        double *dst = U + b * P.S_b + (long long)(c[2] + P.gd[2]) * P.S_k + (long long)(c[1] + P.gd[1]) * P.S_j + (c[0] + P.gd[0]);
#pragma unroll
        for (int v = 0; v < 5; ++v) {
          if (v0 + v >= P.nvars) continue;
          double val = qC[v];
#pragma unroll
          for (int e2 = 0; e2 < 3; ++e2) {
            if (!both[e2]) continue;
            val = __dadd_rn(val, __dmul_rn(sg[e2] * 0.25, sl[e2][v]));
          }
          dst[(long long)(v0 + v) * P.S_v] = val;
        }
      }
    }
  }
}

// Flux correction [B14]: one CTA per (block, face) with finer neighbours; out -= (+-) beta dt/dx (mean of the fine fluxes
// - the block's own flux) in the zones next to the face.  fjump[((b 6 + f) nvars + v) A + t2 n1 + t1] holds the boundary
// fluxes the stage kernel captured at every jump face (both sides).
__global__ void __launch_bounds__(128) fx_k_amr_flux_correct(const FxParams P, double *out, const double *__restrict__ dx, double dt,
                                                             const double *__restrict__ dt_dev, double beta) {
  const long long bf = P.jface ? (long long)__ldg(&P.jface[blockIdx.x]) : (long long)blockIdx.x;
  const long long b = bf / 6;
  const int f = (int)(bf % 6), d = f >> 1, side = f & 1;
  if (b >= P.nown || !P.active[d] || __ldg(&P.neigh[b * 6 + f]) != FX_NEIGH_FINER) return;
  if (dt_dev) dt = *dt_dev;
  const int d1 = d == 0 ? 1 : 0, d2 = d == 2 ? 1 : 2;
  const int n1 = P.n[d1], n2 = P.n[d2];
  const long long A = (long long)P.fj_area;
  const double r = beta * (dt / __ldg(&dx[b * 3 + d]));
  const int nv = P.nvars;  // the passive scalars' fluxes are corrected like the others [B11]
  for (int t = threadIdx.x; t < nv * n1 * n2; t += blockDim.x) {
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
      for (int j1 = 0; j1 < cnt[0]; ++j1) sum += P.fjump[((fb * 6 + ff) * nv + v) * A + (long long)(ft[1] + j2) * n1 + (ft[0] + j1)];
    const double fbar = sum * (1.0 / (double)(cnt[0] * cnt[1]));
    const double fown = P.fjump[((b * 6 + f) * nv + v) * A + (long long)t2 * n1 + t1];
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
  fx_k_amr_fill<<<dim3((unsigned)(P.jface ? P.njface : P.nblocks * 6), 4), 64, 0, st>>>(P, U, depth);
  FX_LAUNCH_CHECK("amr_fill");
  return FX_OK;
}

int fx_launch_amr_flux_correct(const FxParams &P, double *out, const double *dx, double dt, const double *dt_dev, double beta,
                               cudaStream_t st) {
  if (!P.jump || !P.has_jumps || P.nown == 0) return FX_OK;
  fx_k_amr_flux_correct<<<(unsigned)(P.jface ? P.njface : P.nown * 6), 128, 0, st>>>(P, out, dx, dt, dt_dev, beta);
  FX_LAUNCH_CHECK("amr_flux_correct");
  return FX_OK;
}
