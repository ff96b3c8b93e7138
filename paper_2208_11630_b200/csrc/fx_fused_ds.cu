// fx_fused_ds.cu -- "direction-split" fused stage kernel for blocks with a 16 x 16 (x, y) cross-section.
//
// The fp64 pipe (64 lanes per SM) is the binding unit of this path and a Riemann solve is a long dependent
// chain, so the kernel is organised for thread-level parallelism: one 896-thread CTA per block marches the
// block's 16 x 16 column of zones through z, and every zone of the current plane is served by THREE worker
// threads, one per direction (warps 0-7: x, 8-15: y, 16-23: z).  A worker reconstructs its zone along its
// direction and solves the Riemann problem at the zone's low face; nothing else, so it needs few registers and
// 28 warps stay resident.  Primitives live in a shared-memory ring of planes (2r+1 of them: the z stencil);
// plus-side face states and face fluxes are exchanged through shared memory.  Four more warps carry the rest:
//   warp 24 (E0): the 32 pencil ends of the plane -- halo cells gathered from the neighbour blocks' interiors
//                 through the neighbour table (cp.async; or clamped at an outflow boundary), their primitives,
//                 and the plus-side state of cell -1 of every row and column;
//   warp 25 (E1): minus-side state of cell 16 and the flux of the 17th face of every row and column;
//   warps 26-27 (IO): stream the next plane (cp.async), convert it to primitives once, and stage U0 / X rows
//                 for the stage combination.
// Two CTA barriers per plane: phase A = reconstruct plane t (z: plane t+1) + combine/store plane t-1;
// phase B = Riemann solves of plane t (z: face t+1) + primitives of plane t+2+r.  Guard cells in HBM are
// neither read nor written; HBM traffic is one read of the stage input (+ U0) and one write per zone + halos.
#include "fx_physics.cuh"

namespace fxds {

constexpr int NX = 16, NY = 16, NZONE = NX * NY;
constexpr int NWARPS = 28, NTHREADS = NWARPS * 32;  // 896
constexpr int W_E0 = 24, W_E1 = 25, W_IO = 26;

template <int RECON> struct Rc {
  static constexpr int r = (RECON == FX_RECON_PLM_MINMOD) ? 1 : 2;  // stencil radius of one cell's reconstruction
  static constexpr int R = r + 1;                                    // halo depth
  static constexpr int NP = NX + 2 * R;                              // padded plane extent
  static constexpr int NR = 2 * r + 1;                               // planes in the ring
};

template <int RECON> struct Smem {
  static constexpr int NP = Rc<RECON>::NP, NR = Rc<RECON>::NR, R = Rc<RECON>::R;
  double P[NR][5][NP][NP];   // ring of primitive planes incl. x/y halo (corners unused)
  double L[2][5][NZONE];     // [x|y][v][zone]: plus-side state of the zone's cell
  double G[2][5][NZONE];     // [x|y][v][zone]: flux at the zone's low face (un-rotated variable order)
  double Gz[2][5][NZONE];    // [face parity][v][zone]: z flux at face f (between planes f-1 and f)
  double EL[2][5][16];       // [x|y][v][m]: plus-side state of cell -1 of row / column m
  double EG[2][5][16];       // [x|y][v][m]: flux at face 16 of row / column m
  double raw[2][5][NZONE];   // [plane parity][v][zone]: conserved variables of an incoming plane (cp.async)
  double sU0[5][NZONE];      // U0 rows of the plane being combined (cp.async)
  double sX[5][NZONE];       // stage-input rows of the plane being combined (cp.async; unused in stage 1)
  double H[2][2 * R][5][32]; // [plane parity][cell][v][lane]: raw halo cells of E0's pencil ends (cp.async)
};

__device__ __forceinline__ void cta_sync() { asm volatile("bar.sync 0, %0;" ::"n"(NTHREADS) : "memory"); }
__device__ __forceinline__ void cp_async8(void *s, const void *g) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(s)), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async16(void *s, const void *g) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(s)), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// a3: minus/plus face states of one cell from its stencil s[0..2r] (centre s[r]).
template <int RECON>
__device__ __forceinline__ void recon1(const double *s, double eps, double &qm, double &qp) {
  if (RECON == FX_RECON_PLM_MINMOD) {
    const double h = 0.5 * fx_minmod_fast(s[1] - s[0], s[2] - s[1]);
    qm = s[1] - h;
    qp = s[1] + h;
  } else {
    // WENO5-JS; the two faces of a cell share the smoothness indicators (beta_0 <-> beta_2 under mirroring)
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
    {
      const double p0 = (2.0 * a - 7.0 * b + 11.0 * c) * sixth, p1 = (-b + 5.0 * c + 2.0 * d) * sixth,
                   p2 = (2.0 * c + 5.0 * d - e) * sixth;
      const double a0 = 0.1 * s0, a1 = 0.6 * s1, a2 = 0.3 * s2;
      qp = (a0 * p0 + a1 * p1 + a2 * p2) / (a0 + a1 + a2);
    }
    {
      const double p0 = (2.0 * e - 7.0 * d + 11.0 * c) * sixth, p1 = (-d + 5.0 * c + 2.0 * b) * sixth,
                   p2 = (2.0 * c + 5.0 * b - a) * sixth;
      const double a0 = 0.1 * s2, a1 = 0.6 * s1, a2 = 0.3 * s0;
      qm = (a0 * p0 + a1 * p1 + a2 * p2) / (a0 + a1 + a2);
    }
  }
}

// Reconstruct the five primitives of the cell at smem address c (variable stride vs doubles) from the cells at
// c + m*step, m = -r..r.  WENO positivity fallback per side [A6].
template <int RECON>
__device__ __forceinline__ unsigned recon5(const double *c, int vs, int step, double eps, double qm[5], double qp[5]) {
  constexpr int r = Rc<RECON>::r;
  double ctr[5];
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    double s[2 * r + 1];
#pragma unroll
    for (int m = 0; m < 2 * r + 1; ++m) s[m] = c[v * vs + (m - r) * step];
    ctr[v] = s[r];
    recon1<RECON>(s, eps, qm[v], qp[v]);
  }
  unsigned hit = 0;
  if (RECON == FX_RECON_WENO5) {
    if (!(qm[0] > 0.0) || !(qm[4] > 0.0)) {
#pragma unroll
      for (int v = 0; v < 5; ++v) qm[v] = ctr[v];
      hit = FX_STATUS_WENO_FALLBACK;
    }
    if (!(qp[0] > 0.0) || !(qp[4] > 0.0)) {
#pragma unroll
      for (int v = 0; v < 5; ++v) qp[v] = ctr[v];
      hit = FX_STATUS_WENO_FALLBACK;
    }
  }
  return hit;
}

// z reconstruction: the stencil cells sit at the same (i,j) of different ring planes.
template <int RECON>
__device__ __forceinline__ unsigned recon5_z(const double *const pl[], int vs, int off, double eps, double qm[5], double qp[5]) {
  constexpr int r = Rc<RECON>::r;
  double ctr[5];
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    double s[2 * r + 1];
#pragma unroll
    for (int m = 0; m < 2 * r + 1; ++m) s[m] = pl[m][v * vs + off];
    ctr[v] = s[r];
    recon1<RECON>(s, eps, qm[v], qp[v]);
  }
  unsigned hit = 0;
  if (RECON == FX_RECON_WENO5) {
    if (!(qm[0] > 0.0) || !(qm[4] > 0.0)) {
#pragma unroll
      for (int v = 0; v < 5; ++v) qm[v] = ctr[v];
      hit = FX_STATUS_WENO_FALLBACK;
    }
    if (!(qp[0] > 0.0) || !(qp[4] > 0.0)) {
#pragma unroll
      for (int v = 0; v < 5; ++v) qp[v] = ctr[v];
      hit = FX_STATUS_WENO_FALLBACK;
    }
  }
  return hit;
}

// Riemann flux for compile-time direction D from un-rotated primitive states, returned un-rotated.
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

}  // namespace fxds
