// fx_stage_bundle.cu -- the fused TMA stage kernel (fx_stage_tma.cu) for blocks of 8 x 8 x nz zones: a CTA marches a
// BUNDLE of 2 x 2 blocks that are each other's x / y neighbours -- a 16 x 16 cross-section, the shape the kernel's 256
// zone threads, edge warp and producer warp are built for -- through a chain of such bundles in +z.  [NS]: "many 8^3 -
// 16^3 blocks"; VERDICT r1 item 7.
//
// What differs from fx_stage_tma.cu (whose comments describe the protocol: ring of stage-input planes, halo boxes taken
// from the neighbours' interiors, U0 planes, result plane, two CTA barriers per plane, z window in registers, fused CFL
// reduction): every plane moves as FOUR boxes {8,8,1,1,5}, one per block of the bundle, into quadrant-major shared
// memory [q][v][8][8] (q = x half + 2 * y half); the x / y halo strips are two boxes per side (one per half); plane -> block
// bookkeeping is per quadrant (S.blk: the four block ids of the layer below the segment, of each of its layers and of the
// layer above; a negative id is that block's own boundary code); beta dt / dx_d is kept per block.  Inside the bundle
// the faces between the four blocks are ordinary interior faces: no halo, no 17th-face solve, no second conversion --
// which is what an 8^3 block pays 9/8 for in each direction when it is advanced alone.
// Walls and gravity (EXTRAS) and passive scalars are not instantiated here: such plans keep the tile / generic path.
#include <cuda.h>
#include <string.h>

#include "fx_physics.cuh"
#include "fx_tma.cuh"

namespace fxb {

using namespace fxtma;

constexpr int NX = 16, NY = 16, NB = 8;       // cross-section of a bundle; extent of one block
constexpr int NZONE_THREADS = NX * NY;
constexpr int NTHREADS = NZONE_THREADS + 64;  // + edge warp + producer warp
constexpr int QV = NB * NB;                   // one variable of one quadrant box
constexpr int QS = 5 * QV;                    // one quadrant box
constexpr int PLANE_BYTES = 4 * QS * 8;

template <int RECON> struct Rc {
  static constexpr int r = (RECON == FX_RECON_PLM_MINMOD) ? 1 : 2;
  static constexpr int R = r + 1;
  static constexpr int NP = NX + 2 * R;
  static constexpr int BW = (R + 1) & ~1;
  static constexpr int NRING = r + 3;
  static constexpr int NREG = (RECON == FX_RECON_PLM_MINMOD) ? 96 : 168;
};

template <int RECON> struct alignas(128) Smem {
  static constexpr int R = Rc<RECON>::R, NP = Rc<RECON>::NP, BW = Rc<RECON>::BW, NRING = Rc<RECON>::NRING;
  double ring[NRING][4][5][NB][NB];  // TMA: stage-input planes, quadrant-major
  double U0[2][4][5][NB][NB];        // TMA: U0 planes (later stages)
  double Out[4][5][NB][NB];          // result plane, drained by four TMA stores
  double Hx[2][2][5][NB][BW];        // TMA: [lo|hi][y half] raw x-halo cells of the plane
  static constexpr int HYB = (5 * R * NB + 15) & ~15;  // one y-halo box, padded to a multiple of 128 bytes (TMA destination)
  double Hy[2][2][HYB];              // TMA: [lo|hi][x half] raw y-halo cells of the plane, each box [5][R][8]
  double P[5][NP][NP + 1];           // primitives of the plane incl. halo rows / columns
  double Lx[5][NY][NX + 1];
  double Ly[5][NY + 1][NX];
  double rd[4][3];                   // beta dt / dx_d of the block of each quadrant whose planes are being combined
  double idx[4][3];                  // 1 / dx_d (DTOUT)
  unsigned long long rmax;           // DTOUT: bit pattern of the CTA's maximum of (|u_d| + c) / dx_d
  unsigned long long barX[2], barH;
  // 115 584 bytes with PLM, the size of fx_stage_tma.cu's: two CTAs per SM (2 x (115 584 + 1024) <= 233 472).  The segment's
  // block ids stay in global memory (BLK below: read once per plane by one lane, once per layer by a few): with them, the
  // per-warp maxima and 4-wide rd / idx rows in here the struct was 512 bytes larger and ONE CTA fitted (ncu:
  // launch__occupancy_limit_shared_mem = 1, 15.8 G zone-updates/s at 8^3).
};
static_assert(sizeof(Smem<FX_RECON_PLM_MINMOD>) <= 115712, "PLM: two CTAs per SM need <= 115 712 bytes each");

__device__ __forceinline__ void cta_sync() { asm volatile("bar.sync 0, %0;" ::"n"(NTHREADS) : "memory"); }
// Barrier C has a hardware barrier of its own: the zone threads and the edge warp wait at it, the producer warp only ARRIVES
// (its halo primitives written, the result plane's store read out) and goes on issuing the next tick's copies; its next wait
// is barrier B, on barrier 0, which the others reach only after C -- so it is never more than one arrival ahead.
__device__ __forceinline__ void cta_sync_c() { asm volatile("bar.sync 1, %0;" ::"n"(NTHREADS) : "memory"); }
__device__ __forceinline__ void cta_arrive_c() { asm volatile("bar.arrive 1, %0;" ::"n"(NTHREADS) : "memory"); }

template <int RIEMANN, int WS, int D>
__device__ __forceinline__ void flux_dir(const FxParams &P, const double WL[5], const double WR[5], double F[5]) {
  constexpr int in = 1 + D, it1 = 1 + (D + 1) % 3, it2 = 1 + (D + 2) % 3;
  const double wl[5] = {WL[0], WL[in], WL[it1], WL[it2], WL[4]};
  const double wr[5] = {WR[0], WR[in], WR[it1], WR[it2], WR[4]};
  double f[5];
  fx_riemann_v2<RIEMANN, WS>(P, wl, wr, f);
  F[0] = f[0];
  F[in] = f[1];
  F[it1] = f[2];
  F[it2] = f[3];
  F[4] = f[4];
}

template <int RECON, int RIEMANN, int WS, bool FIRST, bool DTOUT>
__global__ void __launch_bounds__(NTHREADS) __maxnreg__(Rc<RECON>::NREG)
fx_k_stage_bundle(const __grid_constant__ CUtensorMap mXm, const __grid_constant__ CUtensorMap mXx,
                  const __grid_constant__ CUtensorMap mXy, const __grid_constant__ CUtensorMap mU0,
                  const __grid_constant__ CUtensorMap mOut, const FxParams P, const double *__restrict__ X,
                  const double *__restrict__ dx, double dt, const double *dt_dev, double beta,
                  double cfl_next, double *dt_next) {
  constexpr int r = Rc<RECON>::r, R = Rc<RECON>::R, W = 2 * r + 1, NP = Rc<RECON>::NP, BW = Rc<RECON>::BW;
  constexpr int NRING = Rc<RECON>::NRING;
  extern __shared__ __align__(1024) unsigned char fx_smem_raw[];
  Smem<RECON> &S = *reinterpret_cast<Smem<RECON> *>(fx_smem_raw);
  const int tid = threadIdx.x;
  const int nzb = P.n[2];
  const int g0 = P.gd[0], g1 = P.gd[1], g2 = P.gd[2];
  unsigned hit = 0;
  if (tid == 0) S.rmax = 0ull;
  // this CTA's segment: {count, 4 x (count + 2) block ids}; block ids of the segment: layer l (0: the layer below, or each block's own boundary code; 1 .. M: its layers; M + 1: above)
  const int *brow = P.bseg + (long long)blockIdx.x * FX_BSEG_STRIDE + 1;
#define BLK(l, q) __ldg(&brow[4 * (l) + (q)])
  __syncthreads();
  const int M = __ldg(&brow[-1]);
  const int nz = M * nzb;
  const unsigned zmagic = ((1u << 20) + (unsigned)nzb - 1u) / (unsigned)nzb;
  // where plane Z of quadrant q's column lives: block id and padded k (outflow below / above: clamp [O1])
  auto zmap = [&](int Z, int q, int &bs, int &kp) {
    int qb = Z < 0 ? -1 : (M == 1 ? (int)(Z >= nzb) : (int)(((unsigned)Z * zmagic) >> 20));
    int k = Z - qb * nzb;
    int id = BLK(1 + qb, q);
    if (id < 0) {
      if (qb < 0) { id = BLK(1, q); k = 0; } else { id = BLK(M, q); k = nzb - 1; }
    }
    bs = id;
    kp = k + g2;
  };

  // ---------------------------------------------------------------- producer set-up (producer warp, lane 0).  (Issuing a
  // tick's twenty bulk copies from several lanes side by side was measured: 4.54 against 4.23 ms per stage -- slower.)
  const bool producer = tid == NZONE_THREADS + 32;
  auto issue_X = [&](int c) {
    mbar_expect_tx(&S.barX[c & 1], PLANE_BYTES);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      int bs, kp;
      zmap(c + r, q, bs, kp);
      tma_load(&S.ring[(c + r) % NRING][q][0][0][0], &mXm, &S.barX[c & 1], g0, g1, kp, bs);
    }
  };
  // producer warp: the layer the next halo plane is in (plane hk of layer hq) and its blocks' x / y neighbours
  int hk = 0, hq = 0;
  int xlo[2], xhi[2], ylo[2], yhi[2], hbx[2][2], hby[2][2];  // [half]; hbx[side][half]: the bundle's own block on that side
  auto halo_block = [&]() {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      hbx[0][h] = BLK(1 + hq, 2 * h);      // x-lo side, y half h: quadrant (0, h)
      hbx[1][h] = BLK(1 + hq, 2 * h + 1);  // x-hi side: quadrant (1, h)
      hby[0][h] = BLK(1 + hq, h);          // y-lo side, x half h: quadrant (h, 0)
      hby[1][h] = BLK(1 + hq, 2 + h);      // y-hi side: quadrant (h, 1)
      xlo[h] = __ldg(&P.neigh[(long long)hbx[0][h] * 6 + 0]);
      xhi[h] = __ldg(&P.neigh[(long long)hbx[1][h] * 6 + 1]);
      ylo[h] = __ldg(&P.neigh[(long long)hby[0][h] * 6 + 2]);
      yhi[h] = __ldg(&P.neigh[(long long)hby[1][h] * 6 + 3]);
    }
  };
  if (tid >= NZONE_THREADS + 32) halo_block();
  auto issue_H = [&]() {
    const int kp = hk + g2;
    mbar_expect_tx(&S.barH, 2 * 5 * NY * BW * 8 + 2 * 5 * R * NX * 8);
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      tma_load(&S.Hx[0][h][0][0][0], &mXx, &S.barH, g0 + (xlo[h] >= 0 ? NB - BW : 0), g1, kp, xlo[h] >= 0 ? xlo[h] : hbx[0][h]);
      tma_load(&S.Hx[1][h][0][0][0], &mXx, &S.barH, g0 + (xhi[h] >= 0 ? 0 : NB - BW), g1, kp, xhi[h] >= 0 ? xhi[h] : hbx[1][h]);
      tma_load(&S.Hy[0][h][0], &mXy, &S.barH, g0, g1 + (ylo[h] >= 0 ? NB - R : 0), kp, ylo[h] >= 0 ? ylo[h] : hby[0][h]);
      tma_load(&S.Hy[1][h][0], &mXy, &S.barH, g0, g1 + (yhi[h] >= 0 ? 0 : NB - R), kp, yhi[h] >= 0 ? yhi[h] : hby[1][h]);
    }
  };
  auto issue_U0 = [&](int p, int layer, int k) {  // plane p of the column = plane k of the layer-th layer
    mbar_expect_tx(&S.barX[(p + 1) & 1], PLANE_BYTES);
#pragma unroll
    for (int q = 0; q < 4; ++q) tma_load(&S.U0[p & 1][q][0][0][0], &mU0, &S.barX[(p + 1) & 1], g0, g1, k + g2, BLK(1 + layer, q));
  };
  if (producer) {
    mbar_init(&S.barX[0], FIRST ? 1 : 2); mbar_init(&S.barX[1], FIRST ? 1 : 2);
    mbar_init(&S.barH, 1);
    fence_mbar_init();
    fence_async_smem();
    issue_X(1);
    issue_H();
    if (!FIRST) issue_U0(0, 0, 0);
  }
  if (dt_dev) dt = *dt_dev;
  cta_sync();

  if (tid < NZONE_THREADS) {
    // ------------------------------------------------------------ zone threads: zone (i, j) of the 16 x 16 cross-section lies
    // in quadrant zq = (i >> 3) + 2 (j >> 3) at (i & 7, j & 7)
    const int i = tid & 15, j = tid >> 4;
    const int zq = (i >> 3) + 2 * (j >> 3);
    const int zoff = zq * QS + (j & 7) * NB + (i & 7);  // + v * QV: this zone in a quadrant-major plane
    double *const ringf = &S.ring[0][0][0][0][0];
    double *const u0f = &S.U0[0][0][0][0][0];
    double *const outf = &S.Out[0][0][0][0];
    double rate = 0.0;
    double q[W][5];
    double qpz[5], Fz[5];
    {
      const long long col = (long long)((j & 7) + g1) * P.S_j + ((i & 7) + g0);
      double w[2 * R][5];
#pragma unroll
      for (int m = 0; m < 2 * R; ++m) {
        int bs, kp;
        zmap(m - R, zq, bs, kp);
        const long long a = (long long)bs * P.S_b + (long long)kp * P.S_k + col;
#pragma unroll
        for (int v = 0; v < 5; ++v) w[m][v] = X[a + v * P.S_v];
      }
#pragma unroll
      for (int m = 0; m < 2 * R; ++m) {
        double u[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) u[v] = w[m][v];
        if (m >= R) {  // planes 0 .. r do not come through the TMA ring: keep them there for the combine
#pragma unroll
          for (int v = 0; v < 5; ++v) ringf[((m - R) % NRING) * 4 * QS + v * QV + zoff] = u[v];
        }
        const unsigned h = fx_c2p_v2(P, u[0], u[1], u[2], u[3], u[4], w[m]);
        if (m >= R && m - R < nz) hit |= h;
      }
      double qm[5], qpm1[5];
      hit |= fx_recon_cell5<RECON>(&w[0], P.weno_eps, qm, qpm1);  // cell -1
      hit |= fx_recon_cell5<RECON>(&w[1], P.weno_eps, qm, qpz);   // cell 0
      flux_dir<RIEMANN, WS, 2>(P, qpm1, qm, Fz);
#pragma unroll
      for (int m = 0; m < 2 * r; ++m)
#pragma unroll
        for (int v = 0; v < 5; ++v) q[m][v] = w[m + 2][v];
    }

#pragma unroll
    for (int v = 0; v < 5; ++v) S.P[v][j + R][i + R] = q[r - 1][v];  // plane 0
    cta_sync();  // A0

#pragma unroll 1
    for (int c = 1; c <= nz; ++c) {
      const int p = c - 1;
      double qmx[5], qmy[5];
      {
        double st[W][5], qp[5];
#pragma unroll
        for (int m = 0; m < W; ++m)
#pragma unroll
          for (int v = 0; v < 5; ++v) st[m][v] = (m == r) ? q[r - 1][v] : S.P[v][j + R][i + R + m - r];
        hit |= fx_recon_cell5<RECON>(st, P.weno_eps, qmx, qp);
#pragma unroll
        for (int v = 0; v < 5; ++v) S.Lx[v][j][i + 1] = qp[v];
      }
      {
        double st[W][5], qp[5];
#pragma unroll
        for (int m = 0; m < W; ++m)
#pragma unroll
          for (int v = 0; v < 5; ++v) st[m][v] = (m == r) ? q[r - 1][v] : S.P[v][j + R + m - r][i + R];
        hit |= fx_recon_cell5<RECON>(st, P.weno_eps, qmy, qp);
#pragma unroll
        for (int v = 0; v < 5; ++v) S.Ly[v][j + 1][i] = qp[v];
      }
      cta_sync();  // B
      {
        double u[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) u[v] = ringf[((c + r) % NRING) * 4 * QS + v * QV + zoff];
        const unsigned h = fx_c2p_v2(P, u[0], u[1], u[2], u[3], u[4], q[2 * r]);
        if (c + r < nz) hit |= h;
      }
      double Fz_new[5];
      {
        double qmz[5], qpz_new[5];
        hit |= fx_recon_cell5<RECON>(q, P.weno_eps, qmz, qpz_new);
        flux_dir<RIEMANN, WS, 2>(P, qpz, qmz, Fz_new);
#pragma unroll
        for (int v = 0; v < 5; ++v) qpz[v] = qpz_new[v];
      }
      double Fx[5], Fy[5];
      {
        double WL[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) WL[v] = S.Lx[v][j][i];
        flux_dir<RIEMANN, WS, 0>(P, WL, qmx, Fx);
#pragma unroll
        for (int v = 0; v < 5; ++v) S.Lx[v][j][i] = Fx[v];
#pragma unroll
        for (int v = 0; v < 5; ++v) WL[v] = S.Ly[v][j][i];
        flux_dir<RIEMANN, WS, 1>(P, WL, qmy, Fy);
#pragma unroll
        for (int v = 0; v < 5; ++v) S.Ly[v][j][i] = Fy[v];
      }
      if (c < nz) {
#pragma unroll
        for (int v = 0; v < 5; ++v) S.P[v][j + R][i + R] = q[r][v];
      }
      cta_sync_c();  // C
      {
        const double rx = S.rd[zq][0], ry = S.rd[zq][1], rz = S.rd[zq][2];
        int hmax = 0;
        double res5[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) {
          const double dFx = S.Lx[v][j][i + 1] - Fx[v];
          const double dFy = S.Ly[v][j + 1][i] - Fy[v];
          const double dFz = Fz_new[v] - Fz[v];
          const double xs = ringf[(p % NRING) * 4 * QS + v * QV + zoff];
          const double u0 = FIRST ? xs : u0f[(p & 1) * 4 * QS + v * QV + zoff];
          const double a = FIRST ? u0 : fma(beta, xs - u0, u0);
          const double res = fma(-rz, dFz, fma(-ry, dFy, fma(-rx, dFx, a)));
          outf[v * QV + zoff] = res;
          if (!DTOUT) hmax = max(hmax, __double2hiint(res) & 0x7fffffff);
          res5[v] = res;
          Fz[v] = Fz_new[v];
        }
        if (!DTOUT && hmax >= 0x7ff00000) hit |= FX_STATUS_NONFINITE;
        if (DTOUT) {
          double w[5], ir;
          hit |= fx_c2p_v2(P, res5[0], res5[1], res5[2], res5[3], res5[4], w, &ir) & FX_STATUS_NONFINITE;
          const double cs = fx_sqrt3(P.gamma * w[4] * ir);
          const double r01 = fx_max_sel((fabs(w[1]) + cs) * S.idx[zq][0], (fabs(w[2]) + cs) * S.idx[zq][1]);
          rate = fx_max_sel(fx_max_sel((fabs(w[3]) + cs) * S.idx[zq][2], r01), rate);
        }
        fence_async_smem();
      }
#pragma unroll
      for (int m = 0; m < 2 * r; ++m)
#pragma unroll
        for (int v = 0; v < 5; ++v) q[m][v] = q[m + 1][v];
    }
    if (DTOUT) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) rate = fmax(rate, __shfl_xor_sync(0xffffffffu, rate, o));
      if ((tid & 31) == 0) atomicMax(&S.rmax, (unsigned long long)__double_as_longlong(rate));  // non-negative doubles order like their bits
    }
    cta_sync();  // D
  } else if (tid < NZONE_THREADS + 32) {
    // ------------------------------------------------------------ edge warp (cells -1 and 16 of every row and column of the
    // bundle's cross-section, their 17th face; beta dt / dx_d of each layer's four blocks)
    const int lane = tid - NZONE_THREADS;
    const bool isx = lane >= 16;
    const int m = lane & 15;
    double *Pf = &S.P[0][0][0];
    constexpr int NPS = NP + 1;
    const int pd = isx ? 1 : NPS, pt = isx ? NPS : 1;
    double *Lf = isx ? &S.Lx[0][0][0] : &S.Ly[0][0][0];
    const int ld = isx ? 1 : NX, lt = isx ? (NX + 1) : 1;
    constexpr int LV = NY * (NX + 1);
    cta_sync();  // A0
    int pk = 0, pq = 0;

#pragma unroll 1
    for (int c = 1; c <= nz; ++c) {
      double qm16[5];
      {
        double st[W][5], qm[5], qp[5];
#pragma unroll
        for (int mm = 0; mm < W; ++mm)
#pragma unroll
          for (int v = 0; v < 5; ++v) st[mm][v] = Pf[v * NP * NPS + mm * pd + (m + R) * pt];
        hit |= fx_recon_cell5<RECON>(st, P.weno_eps, qm, qp);
#pragma unroll
        for (int v = 0; v < 5; ++v) Lf[v * LV + 0 * ld + m * lt] = qp[v];
#pragma unroll
        for (int mm = 0; mm < W; ++mm)
#pragma unroll
          for (int v = 0; v < 5; ++v) st[mm][v] = Pf[v * NP * NPS + (NX + R - r + mm) * pd + (m + R) * pt];
        hit |= fx_recon_cell5<RECON>(st, P.weno_eps, qm16, qp);
      }
      cta_sync();  // B
      {
        double WL[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) WL[v] = Lf[v * LV + NX * ld + m * lt];
        const double wl[5] = {WL[0], isx ? WL[1] : WL[2], isx ? WL[2] : WL[3], isx ? WL[3] : WL[1], WL[4]};
        const double wr[5] = {qm16[0], isx ? qm16[1] : qm16[2], isx ? qm16[2] : qm16[3], isx ? qm16[3] : qm16[1], qm16[4]};
        double f[5];
        fx_riemann_v2<RIEMANN, WS>(P, wl, wr, f);
        double F[5];
        F[0] = f[0];
        F[1] = isx ? f[1] : f[3];
        F[2] = isx ? f[2] : f[1];
        F[3] = isx ? f[3] : f[2];
        F[4] = f[4];
#pragma unroll
        for (int v = 0; v < 5; ++v) Lf[v * LV + NX * ld + m * lt] = F[v];
      }
      if (pk == 0 && lane < 12) {
        // a layer's first plane: the combines of the layer below ended before barrier B, this tick's start after C
        const int qq = lane / 3, d = lane - 3 * qq;
        const double dxd = __ldg(&dx[(long long)BLK(1 + pq, qq) * 3 + d]);
        S.rd[qq][d] = (FIRST ? 1.0 : beta) * dt / dxd;
        if (DTOUT) S.idx[qq][d] = 1.0 / dxd;
      }
      if (++pk == nzb) {
        pk = 0;
        ++pq;
      }
      cta_sync_c();  // C
    }
    cta_sync();  // D
  } else {
    // ------------------------------------------------------------ producer warp: lane 0 issues the bulk copies, all lanes
    // convert the halo cells (lanes 0..15 the y edges of column m, lanes 16..31 the x edges of row m)
    const int lane = tid - NZONE_THREADS - 32;
    const bool isx = lane >= 16;
    const int m = lane & 15, half = m >> 3, mm8 = m & 7;
    double *Pf = &S.P[0][0][0];
    constexpr int NPS = NP + 1;
    const int pd = isx ? 1 : NPS, pt = isx ? NPS : 1;
    constexpr int HXV = NB * BW, HYV = R * NB;  // per-variable sizes inside one box
    int nlo = isx ? xlo[half] : ylo[half], nhi = isx ? xhi[half] : yhi[half];
    auto halo_off = [&](int t, bool high) -> int {
      int idx;  // cell index inside the box: a neighbour's cells, or this block's edge cell at an outflow boundary
      if (isx) idx = high ? (nhi >= 0 ? t : BW - 1) : (nlo >= 0 ? BW - R + t : 0);
      else idx = high ? (nhi >= 0 ? t : R - 1) : (nlo >= 0 ? t : 0);
      return isx ? ((high ? 2 * 5 * HXV : 0) + half * 5 * HXV + mm8 * BW + idx) : ((high ? 2 * Smem<RECON>::HYB : 0) + half * Smem<RECON>::HYB + idx * NB + mm8);
    };
    int hoff[2 * R];
#pragma unroll
    for (int t = 0; t < 2 * R; ++t) hoff[t] = halo_off(t % R, t >= R);
    const int hv = isx ? HXV : HYV;

    auto halo_plane = [&](int pl) {
      mbar_wait(&S.barH, pl & 1);
      const double *Hf = isx ? &S.Hx[0][0][0][0][0] : &S.Hy[0][0][0];
#pragma unroll
      for (int t = 0; t < 2 * R; ++t) {
        double u[5], w[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) u[v] = Hf[hoff[t] + v * hv];
        fx_c2p_v2(P, u[0], u[1], u[2], u[3], u[4], w);
        const int pos = (t < R) ? t : (NX + t);
#pragma unroll
        for (int v = 0; v < 5; ++v) Pf[v * NP * NPS + pos * pd + (m + R) * pt] = w[v];
      }
      __syncwarp();
    };
    auto halo_next = [&](int pl) {  // the single halo slot is free (every lane has read its cells): the next plane's boxes
      if (pl + 1 < nz) {
        if (++hk == nzb) {
          hk = 0;
          ++hq;
          halo_block();
          nlo = isx ? xlo[half] : ylo[half];
          nhi = isx ? xhi[half] : yhi[half];
#pragma unroll
          for (int t = 0; t < 2 * R; ++t) hoff[t] = halo_off(t % R, t >= R);
        }
        if (lane == 0) issue_H();
      }
    };
    halo_plane(0);
    halo_next(0);
    cta_sync();  // A0
    int pk = 0, pq = 0;
    // The block ids a tick's twelve plane copies need -- rows pq, pq + 1, pq + 2 of the segment table: the layers below, of
    // and above the plane being combined -- are kept in registers and refreshed when a new layer starts, BEFORE the wait for
    // barrier B.  Read from the table one by one between the copies (each bulk-copy statement is a memory barrier to the
    // compiler, so every id was a dependent global load in the issuing lane's path, with hardly any L1 beside two CTAs'
    // shared memory), they made the producer warp the last to arrive at barrier C: ncu showed the zone warps waiting
    // there for 13 % of their time.
    int cid[3][4];
    auto load_rows = [&]() {
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int q = 0; q < 4; ++q) cid[a][q] = BLK(pq + a, q);
    };
    auto row_id = [&](int row, int q) -> int {
      const int a = row - pq;
      return a == 0 ? cid[0][q] : (a == 1 ? cid[1][q] : cid[2][q]);
    };
    load_rows();
#pragma unroll 1
    for (int c = 1; c <= nz; ++c) {
      const int p = c - 1;
      if (pk == 0 && c > 1) load_rows();
      mbar_wait(&S.barX[c & 1], ((c - 1) >> 1) & 1);
      cta_sync();  // B
      if (lane == 0) {
        if (c + 1 <= nz) {  // issue_X(c + 1) with the cached ids
          const int Z = c + 1 + r;
          const int qb = M == 1 ? (int)(Z >= nzb) : (int)(((unsigned)Z * zmagic) >> 20);
          mbar_expect_tx(&S.barX[(c + 1) & 1], PLANE_BYTES);
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            int id = row_id(1 + qb, q), k = Z - qb * nzb;
            if (id < 0) { id = BLK(M, q); k = nzb - 1; }  // above the segment: outflow clamps to the top plane [O1]
            tma_load(&S.ring[Z % NRING][q][0][0][0], &mXm, &S.barX[(c + 1) & 1], g0, g1, k + g2, id);
          }
        }
        if (p >= 1) {
          const int layer = pk >= 1 ? pq : pq - 1, k = (pk >= 1 ? pk - 1 : nzb - 1) + g2;
#pragma unroll
          for (int q = 0; q < 4; ++q) tma_store(&mOut, &S.Out[q][0][0][0], g0, g1, k, row_id(1 + layer, q));
          tma_commit();
        }
      }
      if (c < nz) halo_plane(c);  // halo of plane p + 1: nobody reads P between barriers B and C
      if (lane == 0 && p >= 1) tma_wait_read();  // Out is free for the combine after barrier C
      cta_arrive_c();  // C: what the others wait for is done; the rest of the tick is off their path
      if (lane == 0 && !FIRST && p + 1 < nz) {  // issue_U0(p + 1, ...): its slot was last read before barrier B
        const int layer = pk + 1 < nzb ? pq : pq + 1, k = pk + 1 < nzb ? pk + 1 : 0;
        mbar_expect_tx(&S.barX[(p + 2) & 1], PLANE_BYTES);
#pragma unroll
        for (int q = 0; q < 4; ++q) tma_load(&S.U0[(p + 1) & 1][q][0][0][0], &mU0, &S.barX[(p + 2) & 1], g0, g1, k + g2, row_id(1 + layer, q));
      }
      if (c < nz) halo_next(c);
      if (++pk == nzb) {
        pk = 0;
        ++pq;
      }
    }
    cta_sync();  // D
    if (lane == 0) {
#pragma unroll
      for (int q = 0; q < 4; ++q) tma_store(&mOut, &S.Out[q][0][0][0], g0, g1, nzb - 1 + g2, BLK(M, q));
      tma_commit();
      if (DTOUT) {
        atomicMax(&P.scratch[FX_SCR_DTBITS], S.rmax);
        __threadfence();
        const unsigned long long done = atomicAdd(&P.scratch[FX_SCR_COUNTER], 1ull);
        if (done == gridDim.x - 1) {
          __threadfence();
          const unsigned long long bits = atomicExch(&P.scratch[FX_SCR_DTBITS], 0ull);
          P.scratch[FX_SCR_COUNTER] = 0ull;
          *dt_next = cfl_next / __longlong_as_double((long long)bits);
        }
      }
      tma_wait_all();
    }
  }
  if (hit) fx_note(P, hit);
}

// ------------------------------------------------------------------ launch
template <int RECON, int RIEMANN, int WS, bool FIRST, bool DTOUT>
int launch(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt, const double *dt_dev,
           double beta, double cfl_next, double *dt_next, cudaStream_t st) {
  constexpr int R = Rc<RECON>::R, BW = Rc<RECON>::BW;
  CUtensorMap mXm, mXx, mXy, mU0, mOut;
  int rc;
  if ((rc = make_map(&mXm, P, X, NB, NB))) return rc;
  if ((rc = make_map(&mXx, P, X, BW, NB))) return rc;
  if ((rc = make_map(&mXy, P, X, NB, R))) return rc;
  if ((rc = make_map(&mU0, P, U0, NB, NB))) return rc;
  if ((rc = make_map(&mOut, P, out, NB, NB))) return rc;
  auto kern = fx_k_stage_bundle<RECON, RIEMANN, WS, FIRST, DTOUT>;
  const int smem = (int)sizeof(Smem<RECON>);
  FX_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  kern<<<(unsigned)P.nbseg, NTHREADS, smem, st>>>(mXm, mXx, mXy, mU0, mOut, P, X, dx, dt, dt_dev, beta, cfl_next, dt_next);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fx_fail(FX_ERR_CUDA, "stage_bundle launch: %s (smem %d)", cudaGetErrorString(e), smem);
  return FX_OK;
}

template <int RECON, int RIEMANN, int WS>
int launch_ws(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt, const double *dt_dev,
              double beta, int first, double cfl_next, double *dt_next, cudaStream_t st) {
  if (first) return launch<RECON, RIEMANN, WS, true, false>(P, X, U0, out, dx, dt, dt_dev, beta, 0.0, nullptr, st);
  if (dt_next) return launch<RECON, RIEMANN, WS, false, true>(P, X, U0, out, dx, dt, dt_dev, beta, cfl_next, dt_next, st);
  return launch<RECON, RIEMANN, WS, false, false>(P, X, U0, out, dx, dt, dt_dev, beta, 0.0, nullptr, st);
}

template <int RECON, int RIEMANN>
int launch_rr(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt, const double *dt_dev,
              double beta, int first, double cfl_next, double *dt_next, cudaStream_t st) {
  return P.wavespeed == 0 ? launch_ws<RECON, RIEMANN, 0>(P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st)
                          : launch_ws<RECON, RIEMANN, 1>(P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st);
}

}  // namespace fxb

bool fx_stage_bundle_supported(const FxParams &P) {
  const int R = P.recon == FX_RECON_WENO5 ? 3 : 2;
  return P.n[0] == fxb::NB && P.n[1] == fxb::NB && P.n[2] >= R && P.active[2] && P.gd[0] >= R && (P.S_j % 2) == 0 && (P.gd[0] % 2) == 0 &&
         P.nblocks <= 0x7fffffffLL && P.bseg != nullptr && P.nbseg > 0 && !P.walls && !P.grav_on && P.nvars == 5 && !P.has_jumps;
}

int fx_launch_stage_bundle(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt,
                           const double *dt_dev, double beta, int first, double cfl_next, double *dt_next, cudaStream_t st) {
  if (!fx_stage_bundle_supported(P)) return fx_fail(FX_ERR_UNSUPPORTED, "bundle stage kernel: plan not supported");
  if (first && X != U0) return fx_fail(FX_ERR_INVALID_ARG, "bundle stage kernel: the first stage takes U0 from its stage input (X must be U0)");
  if (((uintptr_t)X | (uintptr_t)U0 | (uintptr_t)out) & 15)
    return fx_fail(FX_ERR_INVALID_ARG, "bundle stage kernel: state arrays must be 16-byte aligned");
  if (P.recon == FX_RECON_PLM_MINMOD) {
    if (P.riemann == FX_RIEMANN_HLLE) return fxb::launch_rr<FX_RECON_PLM_MINMOD, FX_RIEMANN_HLLE>(P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st);
    return fxb::launch_rr<FX_RECON_PLM_MINMOD, FX_RIEMANN_HLLC>(P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st);
  }
  if (P.riemann == FX_RIEMANN_HLLE) return fxb::launch_rr<FX_RECON_WENO5, FX_RIEMANN_HLLE>(P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st);
  return fxb::launch_rr<FX_RECON_WENO5, FX_RIEMANN_HLLC>(P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st);
}
