// fx_fused.cu -- fused per-stage kernel for 3-D blocks with a 16 x 16 (x, y) cross-section (K1+K2+K3).
//
// One CTA per block marches the 16 x 16 column of zones through z.  Thread (i,j) of the 256 "zone"
// threads owns the zones (i,j,k), k = 0..nz-1:
//   * z direction: a sliding window of primitive cells lives in registers; each new plane is loaded once
//     from HBM (coalesced 128-byte rows), converted to primitives once, and used for the z reconstruction,
//     the z Riemann problem and, R planes later, the in-plane work of the same zone;
//   * x and y directions: per plane, the threads exchange primitives, plus-side face states and face
//     fluxes through shared memory (three barriers per plane);
//   * a ninth "edge" warp supplies what a 16-wide row lacks: the halo cells of the plane (gathered straight
//     from the neighbour blocks' interiors through the neighbour table, or clamped at an outflow
//     boundary -- no guard cell in HBM is read or written), the plus-side state of cell -1 and the flux of
//     the 17th face of every row and column, so no zone thread does redundant work.
// The zone thread then forms S = sum_d dt/dx_d (F+ - F-) and the SSP-RK combination and stores its zone:
// HBM traffic is one read of the stage input (+ U0 in later stages) and one write per zone, plus halos.
#include "fx_physics.cuh"

#ifndef FX_FUSED_MINB_PLM
#define FX_FUSED_MINB_PLM 1  // resident CTAs per SM the PLM kernels are compiled for
#endif

namespace {

constexpr int NX = 16, NY = 16;
constexpr int NZONE_THREADS = NX * NY;      // 256
constexpr int NTHREADS = NZONE_THREADS + 32;  // + edge warp

template <int RECON> struct Rc {
  static constexpr int r = (RECON == FX_RECON_PLM_MINMOD) ? 1 : 2;  // stencil radius of one cell's reconstruction
  static constexpr int R = r + 1;                                    // halo depth
  static constexpr int NP = NX + 2 * R;                              // padded plane extent
};

// Shared-memory plane buffers (doubles).
template <int RECON> struct Smem {
  static constexpr int NP = Rc<RECON>::NP;
  double P[5][NP][NP];       // primitives of the plane incl. halo rows/columns (corners unused)
  double Lx[5][NY][NX + 1];  // Lx[v][j][i+1] = plus-side x state of cell (i,j), i = -1..15
  double Ly[5][NY + 1][NX];  // Ly[v][j+1][i] = plus-side y state of cell (i,j), j = -1..15
  double Gx[5][NY][NX + 1];  // Gx[v][j][i]   = x flux at face i-1/2, i = 0..16 (un-rotated variable order)
  double Gy[5][NY + 1][NX];  // Gy[v][j][i]   = y flux at face j-1/2, j = 0..16
};

__device__ __forceinline__ void cta_sync() { asm volatile("bar.sync 0, %0;" ::"n"(NTHREADS) : "memory"); }

// a3: minus/plus face states of one cell from its stencil s[0..2r] (centre s[r]).
template <int RECON>
__device__ __forceinline__ void recon_cell(const double *s, double eps, double &qm, double &qp) {
  if (RECON == FX_RECON_PLM_MINMOD) {
    const double h = 0.5 * fx_minmod_fast(s[1] - s[0], s[2] - s[1]);
    qm = s[1] - h;
    qp = s[1] + h;
  } else {
    // WENO5-JS, both faces of the cell share the smoothness indicators (beta_0 <-> beta_2 under mirroring)
    const double a = s[0], b = s[1], c = s[2], d = s[3], e = s[4];
    const double sixth = 1.0 / 6.0;
    const double t0 = a - 2.0 * b + c, u0 = a - 4.0 * b + 3.0 * c;
    const double t1 = b - 2.0 * c + d, u1 = b - d;
    const double t2 = c - 2.0 * d + e, u2 = 3.0 * c - 4.0 * d + e;
    const double b0 = (13.0 / 12.0) * (t0 * t0) + 0.25 * (u0 * u0) + eps;
    const double b1 = (13.0 / 12.0) * (t1 * t1) + 0.25 * (u1 * u1) + eps;
    const double b2 = (13.0 / 12.0) * (t2 * t2) + 0.25 * (u2 * u2) + eps;
    const double q0 = b1 * b2, q1 = b0 * b2, q2 = b0 * b1;
    const double s0 = q0 * q0, s1 = q1 * q1, s2 = q2 * q2;  // ~ 1/b0^2, 1/b1^2, 1/b2^2 up to a common factor
    {  // plus face: candidates from (a,b,c), (b,c,d), (c,d,e); weights 0.1, 0.6, 0.3
      const double p0 = (2.0 * a - 7.0 * b + 11.0 * c) * sixth, p1 = (-b + 5.0 * c + 2.0 * d) * sixth,
                   p2 = (2.0 * c + 5.0 * d - e) * sixth;
      const double a0 = 0.1 * s0, a1 = 0.6 * s1, a2 = 0.3 * s2;
      qp = (a0 * p0 + a1 * p1 + a2 * p2) / (a0 + a1 + a2);
    }
    {  // minus face: mirrored stencil (e,d,c,b,a)
      const double p0 = (2.0 * e - 7.0 * d + 11.0 * c) * sixth, p1 = (-d + 5.0 * c + 2.0 * b) * sixth,
                   p2 = (2.0 * c + 5.0 * b - a) * sixth;
      const double a0 = 0.1 * s2, a1 = 0.6 * s1, a2 = 0.3 * s0;
      qm = (a0 * p0 + a1 * p1 + a2 * p2) / (a0 + a1 + a2);
    }
  }
}

// Reconstruct all five primitives of one cell; st[m][v] is cell m of the stencil.  WENO positivity
// fallback per side [A6]: a face state with rho <= 0 or p <= 0 reverts to the cell's own values.
template <int RECON>
__device__ __forceinline__ unsigned recon_cell5(const double (*st)[5], double eps, double qm[5], double qp[5]) {
  constexpr int r = Rc<RECON>::r;
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    double s[2 * r + 1];
#pragma unroll
    for (int m = 0; m < 2 * r + 1; ++m) s[m] = st[m][v];
    recon_cell<RECON>(s, eps, qm[v], qp[v]);
  }
  unsigned hit = 0;
  if (RECON == FX_RECON_WENO5) {
    if (!(qm[0] > 0.0) || !(qm[4] > 0.0)) {
#pragma unroll
      for (int v = 0; v < 5; ++v) qm[v] = st[r][v];
      hit = FX_STATUS_WENO_FALLBACK;
    }
    if (!(qp[0] > 0.0) || !(qp[4] > 0.0)) {
#pragma unroll
      for (int v = 0; v < 5; ++v) qp[v] = st[r][v];
      hit = FX_STATUS_WENO_FALLBACK;
    }
  }
  return hit;
}

// Riemann flux for direction D (compile-time) from un-rotated primitive states; flux returned in the
// un-rotated variable order (rho, mx, my, mz, E).
template <int RIEMANN, int D>
__device__ __forceinline__ void flux_dir(const FxParams &P, const double WL[5], const double WR[5], double F[5]) {
  constexpr int in = 1 + D, it1 = 1 + (D + 1) % 3, it2 = 1 + (D + 2) % 3;
  const double wl[5] = {WL[0], WL[in], WL[it1], WL[it2], WL[4]};
  const double wr[5] = {WR[0], WR[in], WR[it1], WR[it2], WR[4]};
  double f[5];
  fx_riemann_fast<RIEMANN>(P, wl, wr, f);
  F[0] = f[0];
  F[in] = f[1];
  F[it1] = f[2];
  F[it2] = f[3];
  F[4] = f[4];
}

// Where plane k (k in [-R, nz+R)) of this block's column lives: block id and padded k index.  Outflow
// clamps to the nearest interior plane of this block [O1].
__device__ __forceinline__ void z_source(const FxParams &P, long long b, int nlo, int nhi, int k, long long &bs, int &kp) {
  const int nz = P.n[2], g = P.gd[2];
  bs = b;
  if (k < 0) {
    if (nlo >= 0) { bs = nlo; k += nz; } else k = 0;
  } else if (k >= nz) {
    if (nhi >= 0) { bs = nhi; k -= nz; } else k = nz - 1;
  }
  kp = k + g;
}

}  // namespace

namespace {

template <int RECON, int RIEMANN, int MINB>
__global__ void __launch_bounds__(NTHREADS, MINB)
fx_k_fused_stage(FxParams P, const double *__restrict__ X, const double *U0, double *out,
                 const double *__restrict__ dx, double dt, const double *__restrict__ dt_dev, double beta, int first) {
  constexpr int r = Rc<RECON>::r, R = Rc<RECON>::R, W = 2 * r + 1, NP = Rc<RECON>::NP;
  extern __shared__ __align__(16) unsigned char fx_smem_raw[];
  Smem<RECON> &S = *reinterpret_cast<Smem<RECON> *>(fx_smem_raw);
  const long long b = blockIdx.x;
  const int tid = threadIdx.x;
  const int nz = P.n[2];
  if (dt_dev) dt = __ldg(dt_dev);
  unsigned hit = 0;

  if (tid < NZONE_THREADS) {
    // ------------------------------------------------------------ zone threads
    const int i = tid & 15, j = tid >> 4;
    const int nlo = __ldg(&P.neigh[b * 6 + 4]), nhi = __ldg(&P.neigh[b * 6 + 5]);
    const long long col = (long long)(j + P.gd[1]) * P.S_j + (i + P.gd[0]);
    const double rx = dt / __ldg(&dx[b * 3 + 0]), ry = dt / __ldg(&dx[b * 3 + 1]), rz = dt / __ldg(&dx[b * 3 + 2]);
    const long long Sv = P.S_v;
    double q[W][5];          // q[m] = primitives of cell c - r + m at iteration c
    double qpz[5], Fz[5];    // plus-side z state of cell c-1; z flux of face c-1
#pragma unroll
    for (int v = 0; v < 5; ++v) qpz[v] = Fz[v] = 0.0;

    auto z_addr = [&](int k) -> long long {
      long long bs;
      int kp;
      z_source(P, b, nlo, nhi, k, bs, kp);
      return bs * P.S_b + (long long)kp * P.S_k + col;
    };
    auto load_raw = [&](int k, double u[5]) {
      const long long a = z_addr(k);
#pragma unroll
      for (int v = 0; v < 5; ++v) u[v] = X[a + v * Sv];
    };
    auto to_prim = [&](int k, const double u[5], double w[5]) {
      const unsigned h = fx_c2p_fast(P, u[0], u[1], u[2], u[3], u[4], w);
      if (k >= 0 && k < nz) hit |= h;  // a zone's floor hits are counted by its owner only
    };

    double Un[5];  // raw conserved variables of the next new cell (software prefetch, one plane ahead)
#pragma unroll
    for (int m = 0; m < 2 * r; ++m) {
      load_raw(-R + m, Un);
      to_prim(-R + m, Un, q[m]);
    }
    load_raw(-1 + r, Un);

#pragma unroll 1
    for (int c = -1; c <= nz; ++c) {
      to_prim(c + r, Un, q[2 * r]);
      if (c < nz) load_raw(c + r + 1, Un);
      const bool inplane = c >= 1;  // in-plane work for plane p = c - 1, whose primitives are q[r-1]
      const int p = c - 1;
      double qmx[5], qmy[5];
      if (inplane) {
#pragma unroll
        for (int v = 0; v < 5; ++v) S.P[v][j + R][i + R] = q[r - 1][v];
        cta_sync();  // A: plane primitives (zone threads) and halo (edge warp) visible
        {
          double st[W][5], qp[5];
#pragma unroll
          for (int m = 0; m < W; ++m)
#pragma unroll
            for (int v = 0; v < 5; ++v) st[m][v] = (m == r) ? q[r - 1][v] : S.P[v][j + R][i + R + m - r];
          hit |= recon_cell5<RECON>(st, P.weno_eps, qmx, qp);
#pragma unroll
          for (int v = 0; v < 5; ++v) S.Lx[v][j][i + 1] = qp[v];
        }
        {
          double st[W][5], qp[5];
#pragma unroll
          for (int m = 0; m < W; ++m)
#pragma unroll
            for (int v = 0; v < 5; ++v) st[m][v] = (m == r) ? q[r - 1][v] : S.P[v][j + R + m - r][i + R];
          hit |= recon_cell5<RECON>(st, P.weno_eps, qmy, qp);
#pragma unroll
          for (int v = 0; v < 5; ++v) S.Ly[v][j + 1][i] = qp[v];
        }
        cta_sync();  // B: plus-side states visible
      }
      // operands of the stage combination, requested now and consumed after the Riemann solves
      double u0[5], xs[5];
      if (inplane) {
        const long long a0 = b * P.S_b + (long long)(p + P.gd[2]) * P.S_k + col;
#pragma unroll
        for (int v = 0; v < 5; ++v) {
          u0[v] = U0[a0 + v * Sv];
          xs[v] = first ? 0.0 : X[a0 + v * Sv];
        }
      }
      // z: reconstruct cell c, flux of face c (between cells c-1 and c)
      double qmz[5], qpz_new[5], Fz_new[5];
      hit |= recon_cell5<RECON>(q, P.weno_eps, qmz, qpz_new);
      if (c >= 0) flux_dir<RIEMANN, 2>(P, qpz, qmz, Fz_new);
      if (inplane) {
        double WL[5], F[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) WL[v] = S.Lx[v][j][i];
        flux_dir<RIEMANN, 0>(P, WL, qmx, F);
#pragma unroll
        for (int v = 0; v < 5; ++v) S.Gx[v][j][i] = F[v];
#pragma unroll
        for (int v = 0; v < 5; ++v) WL[v] = S.Ly[v][j][i];
        flux_dir<RIEMANN, 1>(P, WL, qmy, F);
#pragma unroll
        for (int v = 0; v < 5; ++v) S.Gy[v][j][i] = F[v];
        cta_sync();  // C: fluxes visible
        const long long a0 = b * P.S_b + (long long)(p + P.gd[2]) * P.S_k + col;
        double chk = 0.0;
#pragma unroll
        for (int v = 0; v < 5; ++v) {
          const double dFx = S.Gx[v][j][i + 1] - S.Gx[v][j][i];
          const double dFy = S.Gy[v][j + 1][i] - S.Gy[v][j][i];
          const double dFz = Fz_new[v] - Fz[v];
          const double Sd = rx * dFx + ry * dFy + rz * dFz;
          const long long a = a0 + v * Sv;
          const double res = first ? (u0[v] - Sd) : (u0[v] + beta * ((xs[v] - u0[v]) - Sd));
          out[a] = res;
          chk += res;
        }
        if (!(fabs(chk) <= 1.79e308)) hit |= FX_STATUS_NONFINITE;
      }
#pragma unroll
      for (int v = 0; v < 5; ++v) {
        qpz[v] = qpz_new[v];
        Fz[v] = Fz_new[v];
      }
#pragma unroll
      for (int m = 0; m < 2 * r; ++m)
#pragma unroll
        for (int v = 0; v < 5; ++v) q[m][v] = q[m + 1][v];
    }
  } else {
    // ------------------------------------------------------------ edge warp
    const int lane = tid - NZONE_THREADS;
    const bool isx = lane >= 16;
    const int m = lane & 15;
    const int d = isx ? 0 : 1;
    const int nlo = __ldg(&P.neigh[b * 6 + 2 * d]), nhi = __ldg(&P.neigh[b * 6 + 2 * d + 1]);
    const long long sd = isx ? 1 : P.S_j;  // stride along the edge direction
    const long long st_ = isx ? P.S_j : 1; // stride along the row/column index m
    const int gdd = P.gd[d], gdt = isx ? P.gd[1] : P.gd[0];
    const long long Sv = P.S_v;
    double *Pf = &S.P[0][0][0];
    const int pd = isx ? 1 : NP, pt = isx ? NP : 1;  // smem strides of P along direction / transverse
    double *Lf = isx ? &S.Lx[0][0][0] : &S.Ly[0][0][0];
    double *Gf = isx ? &S.Gx[0][0][0] : &S.Gy[0][0][0];
    const int ld = isx ? 1 : NX, lt = isx ? (NX + 1) : 1;  // strides of L/G along direction / transverse
    constexpr int LV = NY * (NX + 1);                       // per-variable size of L/G arrays (272)

    // global address of halo cell t (low: cell -R+t, high: cell 16+t) of row/column m in plane p
    auto halo_addr = [&](int p, int t, bool high) -> long long {
      const long long plane = (long long)(p + P.gd[2]) * P.S_k + (long long)(m + gdt) * st_;
      long long bs = b;
      int cd;
      if (!high) {
        cd = -R + t;
        if (nlo >= 0) { bs = nlo; cd += NX; } else cd = 0;
      } else {
        cd = NX + t;
        if (nhi >= 0) { bs = nhi; cd -= NX; } else cd = NX - 1;
      }
      return bs * P.S_b + plane + (long long)(cd + gdd) * sd;
    };
    double Hn[2 * R][5];  // raw halo cells of the next plane (software prefetch)
    auto load_halo = [&](int p) {
#pragma unroll
      for (int t = 0; t < 2 * R; ++t) {
        const long long a = halo_addr(p, t % R, t >= R);
#pragma unroll
        for (int v = 0; v < 5; ++v) Hn[t][v] = X[a + v * Sv];
      }
    };
    load_halo(0);

#pragma unroll 1
    for (int p = 0; p < nz; ++p) {
#pragma unroll
      for (int t = 0; t < 2 * R; ++t) {
        double w[5];
        fx_c2p_fast(P, Hn[t][0], Hn[t][1], Hn[t][2], Hn[t][3], Hn[t][4], w);
        const int pos = (t < R) ? t : (NX + t);  // padded position along the edge direction
#pragma unroll
        for (int v = 0; v < 5; ++v) Pf[v * NP * NP + pos * pd + (m + R) * pt] = w[v];
      }
      if (p + 1 < nz) load_halo(p + 1);
      cta_sync();  // A
      double qm16[5];
      {
        double st[W][5], qm[5], qp[5];
        // cell -1: padded positions 0 .. 2r along the direction (cell -1 sits at R-1 = r)
#pragma unroll
        for (int mm = 0; mm < W; ++mm)
#pragma unroll
          for (int v = 0; v < 5; ++v) st[mm][v] = Pf[v * NP * NP + mm * pd + (m + R) * pt];
        hit |= recon_cell5<RECON>(st, P.weno_eps, qm, qp);
#pragma unroll
        for (int v = 0; v < 5; ++v) Lf[v * LV + 0 * ld + m * lt] = qp[v];
        // cell 16: padded positions 16+R-r .. 16+R+r
#pragma unroll
        for (int mm = 0; mm < W; ++mm)
#pragma unroll
          for (int v = 0; v < 5; ++v) st[mm][v] = Pf[v * NP * NP + (NX + R - r + mm) * pd + (m + R) * pt];
        hit |= recon_cell5<RECON>(st, P.weno_eps, qm16, qp);
      }
      cta_sync();  // B
      {
        double WL[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) WL[v] = Lf[v * LV + NX * ld + m * lt];
        const double wl[5] = {WL[0], isx ? WL[1] : WL[2], isx ? WL[2] : WL[3], isx ? WL[3] : WL[1], WL[4]};
        const double wr[5] = {qm16[0], isx ? qm16[1] : qm16[2], isx ? qm16[2] : qm16[3], isx ? qm16[3] : qm16[1], qm16[4]};
        double f[5];
        fx_riemann_fast<RIEMANN>(P, wl, wr, f);
        double F[5];
        F[0] = f[0];
        F[1] = isx ? f[1] : f[3];
        F[2] = isx ? f[2] : f[1];
        F[3] = isx ? f[3] : f[2];
        F[4] = f[4];
#pragma unroll
        for (int v = 0; v < 5; ++v) Gf[v * LV + NX * ld + m * lt] = F[v];
      }
      cta_sync();  // C
    }
  }
  if (hit) fx_note(P, hit);
}

template <int RECON, int RIEMANN, int MINB>
int launch(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt,
           const double *dt_dev, double beta, int first, cudaStream_t st) {
  auto kern = fx_k_fused_stage<RECON, RIEMANN, MINB>;
  const int smem = (int)sizeof(Smem<RECON>);
  static bool configured = false;  // per instantiation
  if (!configured) {
    FX_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    configured = true;
  }
  kern<<<(unsigned)P.nblocks, NTHREADS, smem, st>>>(P, X, U0, out, dx, dt, dt_dev, beta, first);
  FX_LAUNCH_CHECK("fused_stage");
  return FX_OK;
}

}  // namespace

bool fx_fused_supported(const FxParams &P) {
  const int R = P.recon == FX_RECON_WENO5 ? 3 : 2;
  return P.n[0] == NX && P.n[1] == NY && P.n[2] >= R && P.active[2] && P.gd[0] >= R;
}

int fx_launch_fused_stage(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt,
                          const double *dt_dev, double beta, int first, cudaStream_t st) {
  if (!fx_fused_supported(P)) return fx_fail(FX_ERR_UNSUPPORTED, "fused stage kernel: block shape not supported");
  if (P.nblocks == 0) return FX_OK;
  if (P.recon == FX_RECON_PLM_MINMOD) {
    if (P.riemann == FX_RIEMANN_HLLE) return launch<FX_RECON_PLM_MINMOD, FX_RIEMANN_HLLE, FX_FUSED_MINB_PLM>(P, X, U0, out, dx, dt, dt_dev, beta, first, st);
    return launch<FX_RECON_PLM_MINMOD, FX_RIEMANN_HLLC, FX_FUSED_MINB_PLM>(P, X, U0, out, dx, dt, dt_dev, beta, first, st);
  }
  if (P.riemann == FX_RIEMANN_HLLE) return launch<FX_RECON_WENO5, FX_RIEMANN_HLLE, 1>(P, X, U0, out, dx, dt, dt_dev, beta, first, st);
  return launch<FX_RECON_WENO5, FX_RIEMANN_HLLC, 1>(P, X, U0, out, dx, dt, dt_dev, beta, first, st);
}
