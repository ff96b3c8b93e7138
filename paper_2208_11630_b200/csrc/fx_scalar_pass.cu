// fx_scalar_pass.cu -- passive mass scalars [B11] behind the fused stage kernel.
//
// A scalar's flux at a face is Aq X_L + (F_rho - Aq) X_R [B11], where the mass flux F_rho and the coefficient Aq come out of
// the hydro Riemann solve of that face.  The fused kernel (fx_stage_tma.cu, SCAL) leaves both for the three low faces of
// every zone in P.fq; this kernel, one thread per zone, does what is left for each scalar: X = (rho X) / rho on the 2R+1
// cells of each direction's stencil (the reciprocal densities are formed once and serve all scalars), PLM face values of
// cells -1, 0, +1, the two face fluxes per direction (the high face's F_rho and Aq are the next zone's low-face values,
// through the neighbour table at a block face), divergence and RK combination.  Expressions and their order are those of
// the generic kernel's scalar loop (fx_generic.cu), which remains the path for WENO5, physical boundaries and gravity.
// Applies to: PLM, every face of every block with a same-level neighbour (periodic tilings), no gravity.
#include "fx_physics.cuh"

namespace {

// (Measured at config 5 with 4 scalars, fused kernel + this pass per stage: 19.2 ms with everything in registers (159, 12
// warps per SM) as below; 21.2 - 21.6 ms with the reciprocal densities in shared memory and 80 - 128 registers (20 - 24
// warps): the pass is bound by the L2 -> L1 traffic of its y and z stencil rows, not by latency.)
template <int D>
__device__ __forceinline__ void fx_sp_direction(const FxParams &P, const double *__restrict__ X, long long b, long long c, int idx,
                                                long long s, long long zi, long long sz, long long per_block, long long nzt,
                                                long long off[5], double ri[5], double &Flo, double &Alo, double &Fhi, double &Ahi) {
  const int n = P.n[D];
  const int nlo = __ldg(&P.neigh[b * 6 + 2 * D]), nhi = __ldg(&P.neigh[b * 6 + 2 * D + 1]);
  const long long dlo = (long long)(nlo - b) * P.S_b + (long long)n * s, dhi = (long long)(nhi - b) * P.S_b - (long long)n * s;
#pragma unroll
  for (int m = 0; m < 5; ++m) {
    const int t = idx + m - 2;
    off[m] = c + (m - 2) * s + (t < 0 ? dlo : (t >= n ? dhi : 0));
    double rho = X[off[m]];
    if (rho < P.rho_floor) rho = P.rho_floor;
    ri[m] = fx_rcp3(rho);
  }
  const double *fq = P.fq + 2 * D * nzt;
  Flo = fq[zi];
  Alo = fq[nzt + zi];
  const long long zh = idx + 1 < n ? zi + sz : zi - (long long)(n - 1) * sz + (long long)(nhi - b) * per_block;
  Fhi = fq[zh];
  Ahi = fq[nzt + zh];
}

template <bool FIRST>
__global__ void __launch_bounds__(128) fx_k_scalar_pass(const FxParams P, const double *__restrict__ X, const double *U0, double *out,
                                                        const double *__restrict__ dx, double dt, const double *__restrict__ dt_dev,
                                                        double beta, long long nzones) {
  const long long z = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (z >= nzones) return;
  const int nx = P.n[0], ny = P.n[1], nz = P.n[2];
  const long long per_block = (long long)nx * ny * nz;
  const long long b = z / per_block;
  const int r = (int)(z - b * per_block);
  const int i = r % nx, j = (r / nx) % ny, k = r / (nx * ny);
  const long long c = b * P.S_b + (k + P.gd[2]) * P.S_k + (j + P.gd[1]) * P.S_j + (i + P.gd[0]);
  const long long nzt = P.nblocks * per_block;
  if (dt_dev) dt = *dt_dev;
  const double rd0 = dt / __ldg(&dx[b * 3 + 0]), rd1 = dt / __ldg(&dx[b * 3 + 1]), rd2 = dt / __ldg(&dx[b * 3 + 2]);
  long long o0[5], o1[5], o2[5];
  double r0[5], r1[5], r2[5], F[3][2], A[3][2];
  fx_sp_direction<0>(P, X, b, c, i, 1, z, 1, per_block, nzt, o0, r0, F[0][0], A[0][0], F[0][1], A[0][1]);
  fx_sp_direction<1>(P, X, b, c, j, P.S_j, z, nx, per_block, nzt, o1, r1, F[1][0], A[1][0], F[1][1], A[1][1]);
  fx_sp_direction<2>(P, X, b, c, k, P.S_k, z, (long long)nx * ny, per_block, nzt, o2, r2, F[2][0], A[2][0], F[2][1], A[2][1]);
  unsigned hit = 0;
#pragma unroll 1
  for (int sv = 5; sv < P.nvars; ++sv) {
    const double *Q = X + sv * P.S_v;
    double Ss = 0.0;
    auto direction = [&](const long long off[5], const double ri[5], double rd, const double Fd[2], const double Ad[2]) {
      double x[5];
#pragma unroll
      for (int m = 0; m < 5; ++m) x[m] = Q[off[m]] * ri[m];
      double am[3], ap[3];
#pragma unroll
      for (int n = 0; n < 3; ++n) fx_plm(x[n], x[n + 1], x[n + 2], am[n], ap[n]);
      const double Fm = Ad[0] * ap[0] + (Fd[0] - Ad[0]) * am[1];
      const double Fp = Ad[1] * ap[1] + (Fd[1] - Ad[1]) * am[2];
      if (!(fabs(Fm + Fp) <= 1.79e308)) hit |= FX_STATUS_NONFINITE;
      return rd * (Fp - Fm);
    };
    Ss += direction(o0, r0, rd0, F[0], A[0]);
    Ss += direction(o1, r1, rd1, F[1], A[1]);
    Ss += direction(o2, r2, rd2, F[2], A[2]);
    const long long g = sv * P.S_v + c;
    const double u0 = U0[g];
    out[g] = FIRST ? (u0 - Ss) : (u0 + beta * ((Q[c] - u0) - Ss));
  }
  if (hit) fx_note(P, hit);
}

}  // namespace

bool fx_scalar_pass_supported(const FxParams &P) {
  return P.nvars > 5 && P.recon == FX_RECON_PLM_MINMOD && P.all_interior && !P.grav_on && !P.walls && P.fq != nullptr &&
         P.active[0] && P.active[1] && P.active[2];
}

int fx_launch_scalar_pass(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt,
                          const double *dt_dev, double beta, int first, cudaStream_t st) {
  const long long nzones = P.nown * P.n[0] * P.n[1] * P.n[2];
  if (nzones == 0 || P.nvars <= 5) return FX_OK;
  const unsigned grid = (unsigned)((nzones + 127) / 128);
  if (first) fx_k_scalar_pass<true><<<grid, 128, 0, st>>>(P, X, U0, out, dx, dt, dt_dev, beta, nzones);
  else fx_k_scalar_pass<false><<<grid, 128, 0, st>>>(P, X, U0, out, dx, dt, dt_dev, beta, nzones);
  FX_LAUNCH_CHECK("scalar_pass");
  return FX_OK;
}
