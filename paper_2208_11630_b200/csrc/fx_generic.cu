// fx_generic.cu -- generic (any block shape, 1/2/3-D) stage kernel and the debug flux kernel.
//
// The generic path is this zone kernel (the hydro variables' stencil cells beyond a face are read from where O1 would copy
// them from: no fill pass for them; the passive scalars' face guard zones are filled by fx_k_fill_faces first): one thread per
// interior zone computes the two face fluxes of each active direction from the padded stage input
// (each face is evaluated by both zones that share it, bit-identically, so conservation holds to
// rounding; the 2R+1 stencil cells of a direction are converted once and serve both faces), forms
// S = sum_d dt/dx_d (F+ - F-) and the SSP-RK combination; then, for plans with passive scalars [B11], the same for
// every scalar from the mass fluxes and coefficients the hydro part left in shared memory.  It is the path for block
// shapes the fused kernel (fx_stage_tma.cu) does not cover (configs 1 and 2) and the scaffold its parity is
// checked against; it is not the roofline path.
#include "fx_physics.cuh"

// Face flux of direction d at the face whose left cell is element cL of X (variable-0 index).  Aq: what the passive
// scalars need from the solve (fx_riemann); fb: which sides took the WENO5 positivity fallback (bit 0 left, bit 1 right).
template <int RECON, int RIEMANN>
__device__ __forceinline__ unsigned fx_face_flux_global(const FxParams &P, const double *__restrict__ X, long long cL,
                                                        int d, long long s, double F[5], double &Aq, unsigned &fb) {
  constexpr int R = (RECON == FX_RECON_PLM_MINMOD) ? 2 : 3;  // cells each side of the face
  double W[2 * R][5];
  unsigned hit = 0;
#pragma unroll
  for (int m = 0; m < 2 * R; ++m) {
    const long long c = cL + (m - (R - 1)) * s;
    hit |= fx_c2p(P, X[c], X[P.S_v + c], X[2 * P.S_v + c], X[3 * P.S_v + c], X[4 * P.S_v + c], W[m]);
  }
  const int in = 1 + d, it1 = 1 + (d + 1) % 3, it2 = 1 + (d + 2) % 3;
  const int map[5] = {0, in, it1, it2, 4};
  double WL[5], WR[5];
#pragma unroll
  for (int f = 0; f < 5; ++f) {
    const int v = map[f];
    if (RECON == FX_RECON_PLM_MINMOD) {
      const double a = W[0][v], b = W[1][v], c = W[2][v], e = W[3][v];
      WL[f] = b + 0.5 * fx_minmod(b - a, c - b);
      WR[f] = c - 0.5 * fx_minmod(c - b, e - c);
    } else {
      WL[f] = fx_weno5(W[0][v], W[1][v], W[2][v], W[3][v], W[4][v], P.weno_eps);
      WR[f] = fx_weno5(W[5][v], W[4][v], W[3][v], W[2][v], W[1][v], P.weno_eps);
    }
  }
  fb = 0;
  if (RECON == FX_RECON_WENO5) {  // positivity fallback per side [A6]
    if (!(WL[0] > 0.0) || !(WL[4] > 0.0)) {
#pragma unroll
      for (int f = 0; f < 5; ++f) WL[f] = W[R - 1][map[f]];
      hit |= FX_STATUS_WENO_FALLBACK;
      fb |= 1u;
    }
    if (!(WR[0] > 0.0) || !(WR[4] > 0.0)) {
#pragma unroll
      for (int f = 0; f < 5; ++f) WR[f] = W[R][map[f]];
      hit |= FX_STATUS_WENO_FALLBACK;
      fb |= 2u;
    }
  }
  double Ff[5];
  fx_riemann<RIEMANN>(P, WL, WR, Ff, Aq);
  F[0] = Ff[0];
  F[in] = Ff[1];
  F[it1] = Ff[2];
  F[it2] = Ff[3];
  F[4] = Ff[4];
  const double sum = Ff[0] + Ff[1] + Ff[2] + Ff[3] + Ff[4];
  if (!(fabs(sum) <= 1.79e308)) hit |= FX_STATUS_NONFINITE;
  return hit & (FX_STATUS_NONFINITE | FX_STATUS_WENO_FALLBACK);  // floors are counted where a zone is owned
}

template <int RECON, int RIEMANN>
__device__ __forceinline__ unsigned fx_face_flux_global(const FxParams &P, const double *__restrict__ X, long long cL,
                                                        int d, long long s, double F[5]) {
  double Aq;
  unsigned fb;
  return fx_face_flux_global<RECON, RIEMANN>(P, X, cL, d, s, F, Aq, fb);
}

// Passive scalar [B11] (debug flux kernel): left / right abundances X = (rho X) / rho at the face whose left cell is cL, reconstructed like
// every other primitive (Q = the scalar's slab, X = the density's); a side that took the positivity fallback keeps
// its cell value.
template <int RECON>
__device__ __forceinline__ void fx_scalar_face(const FxParams &P, const double *__restrict__ X,
                                               const double *__restrict__ Q, long long cL, long long s, unsigned fb,
                                               double &qL, double &qR) {
  constexpr int R = (RECON == FX_RECON_PLM_MINMOD) ? 2 : 3;
  double x[2 * R];
#pragma unroll
  for (int m = 0; m < 2 * R; ++m) {
    const long long c = cL + (m - (R - 1)) * s;
    double rho = X[c];
    if (rho < P.rho_floor) rho = P.rho_floor;
    x[m] = Q[c] * (1.0 / rho);
  }
  if (RECON == FX_RECON_PLM_MINMOD) {
    qL = x[1] + 0.5 * fx_minmod(x[1] - x[0], x[2] - x[1]);
    qR = x[2] - 0.5 * fx_minmod(x[2] - x[1], x[3] - x[2]);
  } else {
    qL = (fb & 1u) ? x[R - 1] : fx_weno5(x[0], x[1], x[2], x[3], x[4], P.weno_eps);
    qR = (fb & 2u) ? x[R] : fx_weno5(x[5], x[4], x[3], x[2], x[1], P.weno_eps);
  }
}

// Where the stencil cell o zones along direction D from zone idx (interior coordinate along D) of block b lives, as an
// offset from the zone's own element c: inside the block it is c + o s; beyond a face it is the neighbour block's
// interior zone, this block's own edge zone (outflow) or its mirror zone with the normal momentum negated (wall) --
// the single hop of O1 [A14], taken while reading: the generic path fills no guard zone.
template <int D>
__device__ __forceinline__ long long fx_stencil_cell(const FxParams &P, long long b, long long c, int idx, int o,
                                                     long long s, bool &flip) {
  flip = false;
  const int n = P.n[D], t = idx + o;
  if (t >= 0 && t < n) return c + o * s;
  const int side = t >= n;
  const int nb = __ldg(&P.neigh[b * 6 + 2 * D + side]);
  if (nb >= 0) return c + (nb - b) * P.S_b + (long long)(o + (side ? -n : n)) * s;
  if (nb <= FX_NEIGH_COARSER) return c + o * s;  // a refinement jump [B12]: this block's own guard zone, filled by fx_k_amr_fill
  if (nb == FX_BC_REFLECT) {
    flip = true;
    return c + (long long)((side ? 2 * n - 1 - t : -1 - t) - idx) * s;
  }
  return c + (long long)((side ? n - 1 : 0) - idx) * s;  // outflow: zero-gradient clamp
}

// What the scalar loop of a zone needs from its hydro part, per direction, kept in shared memory (one column per
// thread: conflict-free) so that it costs the hydro part no registers.
template <int RECON> struct FxScalarShared {
  static constexpr int RS = (RECON == FX_RECON_PLM_MINMOD) ? 2 : 3;
  double A[3][2][128], F[3][2][128];  // per direction and face (low, high): scalar coefficient Aq and mass flux [B11]
  double ri[3][2 * RS + 1][128];      // 1 / rho of the zone's stencil cells
};

// Direction D of one zone, in the lean arithmetic of the fused kernel (fx_c2p_v2, fx_recon_cell, fx_riemann_v2: one
// Newton step on the MUFU seeds instead of IEEE division and square root; same formulas, rounding differs): the 2R+1
// stencil cells are converted once, cells -1, 0, +1 are reconstructed once each, and the zone's two faces are solved.
// CA (communication-avoiding step [B17]): every stencil cell is read in place from the padded array -- the guard zones hold
// the step's one fill or the previous stage's extended result -- and idx may lie outside [0, n).
template <int RECON, int RIEMANN, int WS, int D, bool SCALARS, bool AMR = false, bool CA = false>
__device__ __forceinline__ unsigned fx_zone_direction(const FxParams &P, const double *__restrict__ X, long long b,
                                                      long long c, int idx, long long s, double rd, double S[5],
                                                      unsigned &qfb, FxScalarShared<RECON> *sh, int tflat = 0) {
  constexpr int R = (RECON == FX_RECON_PLM_MINMOD) ? 2 : 3, r = R - 1;
  constexpr int in = 1 + D, it1 = 1 + (D + 1) % 3, it2 = 1 + (D + 2) % 3;
  constexpr int map[5] = {0, in, it1, it2, 4};
  double W[2 * R + 1][5];
  unsigned hit = 0;
#pragma unroll
  for (int m = 0; m <= 2 * R; ++m) {
    bool flip = false;
    const long long e = CA ? c + (long long)(m - R) * s : fx_stencil_cell<D>(P, b, c, idx, m - R, s, flip);
    double u[5] = {X[e], X[P.S_v + e], X[2 * P.S_v + e], X[3 * P.S_v + e], X[4 * P.S_v + e]}, ri;
    if (flip) u[1 + D] = -u[1 + D];
    hit |= fx_c2p_v2(P, u[0], u[1], u[2], u[3], u[4], W[m], &ri);
    if (SCALARS) sh->ri[D][m][threadIdx.x] = ri;
  }
  hit &= FX_STATUS_NONFINITE;  // floors are counted where a zone is owned
  // face states of cells -1, 0, +1 in the face frame; fb bit 2n: minus side of cell n-1 fell back, bit 2n+1: plus side
  double qm[3][5], qp[3][5];
  unsigned fb = 0;
#pragma unroll
  for (int n = 0; n < 3; ++n) {
    double am[5], ap[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      double st[2 * r + 1];
#pragma unroll
      for (int m = 0; m <= 2 * r; ++m) st[m] = W[n + m][v];  // cell n - 1 sits at index n + r
      fx_recon_cell<RECON>(st, P.weno_eps, am[v], ap[v]);
    }
    if (RECON == FX_RECON_WENO5) {  // positivity fallback per side [A6]
      if (!(am[0] > 0.0) || !(am[4] > 0.0)) {
#pragma unroll
        for (int v = 0; v < 5; ++v) am[v] = W[n + R - 1][v];
        fb |= 1u << (2 * n);
      }
      if (!(ap[0] > 0.0) || !(ap[4] > 0.0)) {
#pragma unroll
        for (int v = 0; v < 5; ++v) ap[v] = W[n + R - 1][v];
        fb |= 2u << (2 * n);
      }
    }
#pragma unroll
    for (int f = 0; f < 5; ++f) {
      qm[n][f] = am[map[f]];
      qp[n][f] = ap[map[f]];
    }
  }
  // the faces see: low = (plus of cell -1, minus of cell 0), high = (plus of cell 0, minus of cell +1)
  const unsigned fbm = ((fb >> 1) & 1u) | (((fb >> 2) & 1u) << 1), fbp = ((fb >> 3) & 1u) | (((fb >> 4) & 1u) << 1);
  if (fbm | fbp) hit |= FX_STATUS_WENO_FALLBACK;
  double Fm[5], Fp[5], Am, Ap;
  fx_riemann_v2<RIEMANN, WS, true>(P, qp[0], qm[1], Fm, &Am);
  fx_riemann_v2<RIEMANN, WS, true>(P, qp[1], qm[2], Fp, &Ap);
  const double sum = (Fm[0] + Fm[1] + Fm[2] + Fm[3] + Fm[4]) + (Fp[0] + Fp[1] + Fp[2] + Fp[3] + Fp[4]);
  if (!(fabs(sum) <= 1.79e308)) hit |= FX_STATUS_NONFINITE;
#pragma unroll
  for (int f = 0; f < 5; ++f) S[map[f]] += rd * (Fp[f] - Fm[f]);
  if (AMR) {  // the boundary fluxes at refinement jumps, both sides, for the flux correction [B14]
    if (idx == 0 && __ldg(&P.neigh[b * 6 + 2 * D]) <= FX_NEIGH_COARSER) {
#pragma unroll
      for (int f = 0; f < 5; ++f) P.fjump[((b * 6 + 2 * D) * P.nvars + map[f]) * (long long)P.fj_area + tflat] = Fm[f];
    }
    if (idx == P.n[D] - 1 && __ldg(&P.neigh[b * 6 + 2 * D + 1]) <= FX_NEIGH_COARSER) {
#pragma unroll
      for (int f = 0; f < 5; ++f) P.fjump[((b * 6 + 2 * D + 1) * P.nvars + map[f]) * (long long)P.fj_area + tflat] = Fp[f];
    }
  }
  if (SCALARS) {
    sh->A[D][0][threadIdx.x] = Am;
    sh->A[D][1][threadIdx.x] = Ap;
    sh->F[D][0][threadIdx.x] = Fm[0];
    sh->F[D][1][threadIdx.x] = Fp[0];
    qfb |= (fbm | (fbp << 2)) << (4 * D);
  }
  return hit;
}

// One scalar, direction D: r dt/dx (F+ - F-) with flux = Aq X_L + (mass flux - Aq) X_R [B11].
// AMR: the scalar's fluxes through the block's jump faces are stored with the hydro variables' [B14]; jf = bit 0 / 1: the
// zone's low / high face along D is such a face, slot = the face's entry of variable sv in P.fjump (for the low face;
// the high face's is one face further)
template <int RECON, int D, bool AMR = false>
__device__ __forceinline__ double fx_zone_scalar_direction(const FxParams &P, const double *__restrict__ Q, long long c,
                                                           long long s, double rd, unsigned qfb,
                                                           const FxScalarShared<RECON> *sh, unsigned &hit, unsigned jf = 0,
                                                           long long slot = 0) {
  constexpr int RS = (RECON == FX_RECON_PLM_MINMOD) ? 2 : 3;
  double x[2 * RS + 1];
#pragma unroll
  // (the scalars' face guard zones were filled by fx_k_fill_faces: looking every cell of every scalar up through the
  // neighbour table as the hydro part does cost 25 % of the step with 4 scalars)
  for (int m = 0; m <= 2 * RS; ++m) x[m] = Q[c + (m - RS) * s] * sh->ri[D][m][threadIdx.x];
  double am[3], ap[3];  // minus / plus face abundances of cells -1, 0, +1
#pragma unroll
  for (int n = 0; n < 3; ++n) fx_recon_cell<RECON>(&x[n], P.weno_eps, am[n], ap[n]);
  const unsigned fbm = (qfb >> (4 * D)) & 3u, fbp = (qfb >> (4 * D + 2)) & 3u;
  const double mL = (fbm & 1u) ? x[RS - 1] : ap[0], mR = (fbm & 2u) ? x[RS] : am[1];
  const double pL = (fbp & 1u) ? x[RS] : ap[1], pR = (fbp & 2u) ? x[RS + 1] : am[2];
  const double Am = sh->A[D][0][threadIdx.x], Ap = sh->A[D][1][threadIdx.x];
  const double Fm = Am * mL + (sh->F[D][0][threadIdx.x] - Am) * mR;
  const double Fp = Ap * pL + (sh->F[D][1][threadIdx.x] - Ap) * pR;
  if (!(fabs(Fm + Fp) <= 1.79e308)) hit |= FX_STATUS_NONFINITE;
  if (AMR) {
    if (jf & 1u) P.fjump[slot] = Fm;
    if (jf & 2u) P.fjump[slot + (long long)P.nvars * P.fj_area] = Fp;
  }
  return rd * (Fp - Fm);
}

#ifndef FX_GENERIC_MINB_PLM
#define FX_GENERIC_MINB_PLM 6
#endif
#ifndef FX_GENERIC_MINB_WENO
#define FX_GENERIC_MINB_WENO 4
#endif
// Resident CTAs aimed at (measured on the generic path, ms per stage launch; the kernel is latency-bound, so up to a
// point the spills are cheaper than the lost warps).  PLM at config 5 without / with 4 scalars: 4 CTAs 15.4 / 29.9,
// 5 CTAs 13.9 / 25.9, 6 CTAs (80 registers) 13.5 / 24.7, 8 CTAs (64 registers; its spills reach DRAM: 28.6 GB written
// for 9.7 GB) 16.3 / 31.0.  WENO5 at config 4 without / with 2 scalars: 3 CTAs 5.5 / 7.8, 4 CTAs 5.5 / 7.4, 5 CTAs
// 5.6 / 7.3.  (The IEEE-arithmetic version of this kernel: PLM uncapped 38.3, 8 CTAs 30.0; WENO5 uncapped 15.2, 4 CTAs 8.2.)
// CA [B17]: the zones are those of the interior extended by `ext` zones in every active dimension (nzones counts them).
template <int RECON, int RIEMANN, int WS, bool SCALARS, bool AMR = false, bool CA = false>
__global__ void __launch_bounds__(128, RECON == FX_RECON_PLM_MINMOD ? FX_GENERIC_MINB_PLM : FX_GENERIC_MINB_WENO) fx_k_generic_stage(FxParams P, const double *__restrict__ X,
                                                          const double *U0, double *out,
                                                          const double *__restrict__ dx, double dt,
                                                          const double *__restrict__ dt_dev, double beta, int first,
                                                          long long nzones, int ext = 0) {
  extern __shared__ __align__(16) unsigned char fx_generic_smem[];
  FxScalarShared<RECON> *sh = reinterpret_cast<FxScalarShared<RECON> *>(fx_generic_smem);  // SCALARS only
  const long long z = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (z >= nzones) return;
  const int e0 = CA && P.active[0] ? ext : 0, e1 = CA && P.active[1] ? ext : 0, e2 = CA && P.active[2] ? ext : 0;
  const int nx = P.n[0] + 2 * e0, ny = P.n[1] + 2 * e1, nz = P.n[2] + 2 * e2;
  const long long per_block = (long long)nx * ny * nz;
  const long long b = z / per_block;
  const int r = (int)(z - b * per_block);
  // (a CTA of 16 x 4 x 2 zones instead of 8 rows of one plane, for L1 reuse of the y and z neighbours: measured, no gain)
  const int i = r % nx - e0, j = (r / nx) % ny - e1, k = r / (nx * ny) - e2;  // interior coordinates (CA: from -ext)
  const long long c = b * P.S_b + (k + P.gd[2]) * P.S_k + (j + P.gd[1]) * P.S_j + (i + P.gd[0]);
  if (dt_dev) dt = *dt_dev;
  double S[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
  unsigned qfb = 0;  // 4 bits per direction: fallback sides of the low and the high face
  unsigned hit = 0;
  if (!CA || (i >= 0 && i < P.n[0] && j >= 0 && j < P.n[1] && k >= 0 && k < P.n[2])) {  // floors are counted once per owned zone
    double W[5];
    hit |= fx_c2p_v2(P, X[c], X[P.S_v + c], X[2 * P.S_v + c], X[3 * P.S_v + c], X[4 * P.S_v + c], W) &
           (FX_STATUS_RHO_FLOOR | FX_STATUS_P_FLOOR | FX_STATUS_NONFINITE);
  }
  const double rd0 = P.active[0] ? dt / __ldg(&dx[b * 3 + 0]) : 0.0;
  const double rd1 = P.active[1] ? dt / __ldg(&dx[b * 3 + 1]) : 0.0;
  const double rd2 = P.active[2] ? dt / __ldg(&dx[b * 3 + 2]) : 0.0;
  // (tflat: the zone's position on the face, transverse dimensions ascending, first one fastest)
  if (P.active[0]) hit |= fx_zone_direction<RECON, RIEMANN, WS, 0, SCALARS, AMR, CA>(P, X, b, c, i, 1, rd0, S, qfb, sh, k * ny + j);
  if (P.active[1]) hit |= fx_zone_direction<RECON, RIEMANN, WS, 1, SCALARS, AMR, CA>(P, X, b, c, j, P.S_j, rd1, S, qfb, sh, k * nx + i);
  if (P.active[2]) hit |= fx_zone_direction<RECON, RIEMANN, WS, 2, SCALARS, AMR, CA>(P, X, b, c, k, P.S_k, rd2, S, qfb, sh, j * nx + i);
  if (P.grav_on) {  // constant-gravity source of the stage input's own zone [B10]
    const double rho = X[c];
    double gm = 0.0;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      S[1 + d] -= dt * (rho * P.grav[d]);
      gm += P.grav[d] * X[(1 + d) * P.S_v + c];
    }
    S[4] -= dt * gm;
  }
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    const long long g = v * P.S_v + c;
    const double u0 = U0[g];
    out[g] = first ? (u0 - S[v]) : (u0 + beta * ((X[g] - u0) - S[v]));
  }
  unsigned jfc = 0;  // AMR with scalars: two bits per direction, the zone's low / high face is a refinement jump of its block
  if (SCALARS && AMR) {
    const int id3[3] = {i, j, k};
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      if (!P.active[d]) continue;
      if (id3[d] == 0 && __ldg(&P.neigh[b * 6 + 2 * d]) <= FX_NEIGH_COARSER) jfc |= 1u << (2 * d);
      if (id3[d] == P.n[d] - 1 && __ldg(&P.neigh[b * 6 + 2 * d + 1]) <= FX_NEIGH_COARSER) jfc |= 2u << (2 * d);
    }
  }
  if (SCALARS) {
    // passive scalars [B11]: same divergence and combination, no source term
#pragma unroll 1
    for (int sv = 5; sv < P.nvars; ++sv) {
      const double *Q = X + sv * P.S_v;
      double Ss = 0.0;
      if (AMR) {
        const long long A = P.fj_area;
        if (P.active[0]) Ss += fx_zone_scalar_direction<RECON, 0, true>(P, Q, c, 1, rd0, qfb, sh, hit, jfc & 3u, ((b * 6 + 0) * P.nvars + sv) * A + (k * ny + j));
        if (P.active[1]) Ss += fx_zone_scalar_direction<RECON, 1, true>(P, Q, c, P.S_j, rd1, qfb, sh, hit, (jfc >> 2) & 3u, ((b * 6 + 2) * P.nvars + sv) * A + (k * nx + i));
        if (P.active[2]) Ss += fx_zone_scalar_direction<RECON, 2, true>(P, Q, c, P.S_k, rd2, qfb, sh, hit, (jfc >> 4) & 3u, ((b * 6 + 4) * P.nvars + sv) * A + (j * nx + i));
      } else {
        if (P.active[0]) Ss += fx_zone_scalar_direction<RECON, 0>(P, Q, c, 1, rd0, qfb, sh, hit);
        if (P.active[1]) Ss += fx_zone_scalar_direction<RECON, 1>(P, Q, c, P.S_j, rd1, qfb, sh, hit);
        if (P.active[2]) Ss += fx_zone_scalar_direction<RECON, 2>(P, Q, c, P.S_k, rd2, qfb, sh, hit);
      }
      const long long g = sv * P.S_v + c;
      const double u0 = U0[g];
      out[g] = first ? (u0 - Ss) : (u0 + beta * ((Q[c] - u0) - Ss));
    }
  }
  if (hit) fx_note(P, hit);
}

template <int RECON, int RIEMANN>
__global__ void __launch_bounds__(128) fx_k_debug_fluxes(FxParams P, const double *__restrict__ U, int dir,
                                                         double *__restrict__ F, long long nfaces, int e0, int e1,
                                                         int e2) {
  const long long z = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (z >= nfaces) return;
  const long long per_block = (long long)e0 * e1 * e2;
  const long long b = z / per_block;
  const int r = (int)(z - b * per_block);
  int cc[3] = {r % e0 + P.gd[0], (r / e0) % e1 + P.gd[1], r / (e0 * e1) + P.gd[2]};
  cc[dir] -= 1;  // left cell of face f is padded cell gd + f - 1 [A17]
  const long long stride[3] = {1, P.S_j, P.S_k};
  const long long cL = b * P.S_b + cc[2] * P.S_k + cc[1] * P.S_j + cc[0];
  double Ff[5], Aq;
  unsigned fb;
  unsigned hit = fx_face_flux_global<RECON, RIEMANN>(P, U, cL, dir, stride[dir], Ff, Aq, fb);
  const long long FS_v = per_block * P.nblocks;
#pragma unroll
  for (int v = 0; v < 5; ++v) F[v * FS_v + z] = Ff[v];
  for (int sv = 5; sv < P.nvars; ++sv) {  // passive scalars [B11]
    double qL, qR;
    fx_scalar_face<RECON>(P, U, U + sv * P.S_v, cL, stride[dir], fb, qL, qR);
    const double Fs = Aq * qL + (Ff[0] - Aq) * qR;
    if (!(fabs(Fs) <= 1.79e308)) hit |= FX_STATUS_NONFINITE;
    F[sv * FS_v + z] = Fs;
  }
  if (hit) fx_note(P, hit);
}

#define FX_DISPATCH(P, CALL)                                                                       \
  do {                                                                                             \
    if (P.recon == FX_RECON_PLM_MINMOD && P.riemann == FX_RIEMANN_HLLE) { CALL(FX_RECON_PLM_MINMOD, FX_RIEMANN_HLLE); } \
    else if (P.recon == FX_RECON_PLM_MINMOD) { CALL(FX_RECON_PLM_MINMOD, FX_RIEMANN_HLLC); }       \
    else if (P.riemann == FX_RIEMANN_HLLE) { CALL(FX_RECON_WENO5, FX_RIEMANN_HLLE); }              \
    else { CALL(FX_RECON_WENO5, FX_RIEMANN_HLLC); }                                                \
  } while (0)

int fx_launch_generic_stage(const FxParams &P, const double *X, const double *U0, double *out, const double *dx,
                            double dt, const double *dt_dev, double beta, int first, cudaStream_t st) {
  const long long nzones = P.nown * P.n[0] * P.n[1] * P.n[2];  // owned blocks come first
  if (nzones == 0) return FX_OK;
  const unsigned grid = (unsigned)((nzones + 127) / 128);
#define CALL(RC, RM)                                                                                              \
  do {                                                                                                          \
    if (P.nvars > 5 && P.has_jumps) {                                                                           \
      if (P.wavespeed == 0) fx_k_generic_stage<RC, RM, 0, true, true><<<grid, 128, sizeof(FxScalarShared<RC>), st>>>(P, X, U0, out, dx, dt, dt_dev, beta, first, nzones); \
      else fx_k_generic_stage<RC, RM, 1, true, true><<<grid, 128, sizeof(FxScalarShared<RC>), st>>>(P, X, U0, out, dx, dt, dt_dev, beta, first, nzones); \
    } else if (P.nvars > 5) {                                                                                   \
      if (P.wavespeed == 0) fx_k_generic_stage<RC, RM, 0, true><<<grid, 128, sizeof(FxScalarShared<RC>), st>>>(P, X, U0, out, dx, dt, dt_dev, beta, first, nzones); \
      else fx_k_generic_stage<RC, RM, 1, true><<<grid, 128, sizeof(FxScalarShared<RC>), st>>>(P, X, U0, out, dx, dt, dt_dev, beta, first, nzones); \
    } else if (P.has_jumps) {                                                                                   \
      if (P.wavespeed == 0) fx_k_generic_stage<RC, RM, 0, false, true><<<grid, 128, 0, st>>>(P, X, U0, out, dx, dt, dt_dev, beta, first, nzones); \
      else fx_k_generic_stage<RC, RM, 1, false, true><<<grid, 128, 0, st>>>(P, X, U0, out, dx, dt, dt_dev, beta, first, nzones); \
    } else {                                                                                                    \
      if (P.wavespeed == 0) fx_k_generic_stage<RC, RM, 0, false><<<grid, 128, 0, st>>>(P, X, U0, out, dx, dt, dt_dev, beta, first, nzones); \
      else fx_k_generic_stage<RC, RM, 1, false><<<grid, 128, 0, st>>>(P, X, U0, out, dx, dt, dt_dev, beta, first, nzones); \
    }                                                                                                           \
  } while (0)
  FX_DISPATCH(P, CALL);
#undef CALL
  FX_LAUNCH_CHECK("generic_stage");
  return FX_OK;
}

// ------------------------------------------------------------------ communication-avoiding step [B17]
// A stage over the interior extended by `ext` zones in every active dimension, stencils in place.
int fx_launch_generic_stage_ca(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt,
                               const double *dt_dev, double beta, int first, int ext, cudaStream_t st) {
  long long per = 1;
  for (int d = 0; d < 3; ++d) per *= P.n[d] + (P.active[d] ? 2 * ext : 0);
  const long long nzones = P.nown * per;
  if (nzones == 0) return FX_OK;
  const unsigned grid = (unsigned)((nzones + 127) / 128);
#define CALL(RC, RM)                                                                                                                          \
  do {                                                                                                                                        \
    if (P.wavespeed == 0) fx_k_generic_stage<RC, RM, 0, false, false, true><<<grid, 128, 0, st>>>(P, X, U0, out, dx, dt, dt_dev, beta, first, nzones, ext); \
    else fx_k_generic_stage<RC, RM, 1, false, false, true><<<grid, 128, 0, st>>>(P, X, U0, out, dx, dt, dt_dev, beta, first, nzones, ext); \
  } while (0)
  FX_DISPATCH(P, CALL);
#undef CALL
  FX_LAUNCH_CHECK("generic_stage_ca");
  return FX_OK;
}

// The zones of the extended box that lie behind a PHYSICAL boundary take that boundary's image of the block's own zone
// (clamp; at a wall the mirror zone with the normal momentum negated) -- what O1 of the stage result would put there;
// zones behind a neighbour keep the value the extended stage computed.  Sources are never destinations.
__global__ void __launch_bounds__(128) fx_k_ca_refill(FxParams P, double *U, int ext, long long nzones) {
  const long long z = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (z >= nzones) return;
  const int e0 = P.active[0] ? ext : 0, e1 = P.active[1] ? ext : 0, e2 = P.active[2] ? ext : 0;
  const int nx = P.n[0] + 2 * e0, ny = P.n[1] + 2 * e1, nz = P.n[2] + 2 * e2;
  const long long per_block = (long long)nx * ny * nz;
  const long long b = z / per_block;
  const int r = (int)(z - b * per_block);
  const int t[3] = {r % nx - e0, (r / nx) % ny - e1, r / (nx * ny) - e2};
  int c[3] = {t[0], t[1], t[2]};
  unsigned flip = 0;
  bool moved = false;
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    if (!P.active[d] || (c[d] >= 0 && c[d] < P.n[d])) continue;
    const int side = c[d] >= P.n[d];
    const int nb = __ldg(&P.neigh[b * 6 + 2 * d + side]);
    if (nb >= 0) continue;
    if (nb == FX_BC_REFLECT) {
      c[d] = side ? 2 * P.n[d] - 1 - c[d] : -1 - c[d];
      flip |= 1u << d;
    } else {
      c[d] = side ? P.n[d] - 1 : 0;
    }
    moved = true;
  }
  if (!moved) return;
  const long long dst = b * P.S_b + (t[2] + P.gd[2]) * P.S_k + (t[1] + P.gd[1]) * P.S_j + (t[0] + P.gd[0]);
  const long long src = b * P.S_b + (c[2] + P.gd[2]) * P.S_k + (c[1] + P.gd[1]) * P.S_j + (c[0] + P.gd[0]);
  for (int v = 0; v < P.nvars; ++v) {
    const double x = U[v * P.S_v + src];
    U[v * P.S_v + dst] = (v >= 1 && v <= 3 && ((flip >> (v - 1)) & 1u)) ? -x : x;
  }
}

int fx_launch_ca_refill(const FxParams &P, double *U, int ext, cudaStream_t st) {
  if (ext <= 0 || P.all_interior) return FX_OK;  // no physical boundary anywhere
  long long per = 1;
  for (int d = 0; d < 3; ++d) per *= P.n[d] + (P.active[d] ? 2 * ext : 0);
  const long long nzones = P.nown * per;
  if (nzones == 0) return FX_OK;
  fx_k_ca_refill<<<(unsigned)((nzones + 127) / 128), 128, 0, st>>>(P, U, ext, nzones);
  FX_LAUNCH_CHECK("ca_refill");
  return FX_OK;
}

int fx_launch_debug_fluxes(const FxParams &P, const double *U, int dir, double *F, cudaStream_t st) {
  int e[3] = {P.n[0], P.n[1], P.n[2]};
  e[dir] += 1;
  const long long nfaces = P.nblocks * e[0] * e[1] * e[2];
  if (nfaces == 0) return FX_OK;
  const unsigned grid = (unsigned)((nfaces + 127) / 128);
#define CALL(RC, RM) fx_k_debug_fluxes<RC, RM><<<grid, 128, 0, st>>>(P, U, dir, F, nfaces, e[0], e[1], e[2])
  FX_DISPATCH(P, CALL);
#undef CALL
  FX_LAUNCH_CHECK("debug_fluxes");
  return FX_OK;
}
