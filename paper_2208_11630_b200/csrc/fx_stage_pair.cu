// fx_stage_pair.cu -- the fused TMA stage kernel (fx_stage_tma.cu) for PLM with TWO x-adjacent zones per thread.
// FX_OPT_PATH = 3 selects it; it is NOT the default: measured at config 5 it takes 5.9 ms per stage against the
// one-zone-per-thread kernel's 5.55 ms (profiles/README.md, round 2).  It is kept, tested for parity, as the record of
// the experiment VERDICT r1 asked for ("two x-adjacent zones per thread ... 128 zone threads x 168 registers x 2 CTAs").
//
// What pairs change.  A thread owns zones (2i, 2i+1) of row j:
//   * the face between its two zones is its own -- no exchange -- and the three slopes of the pair share the middle
//     difference; the thread's two x solves (its own face, the low face of zone 2i), its two y solves and its two z
//     solves run side by side as two-wide values (fx_vec2.cuh);
//   * everything that crosses rows or planes (y neighbours, plus-side y states, y fluxes, the TMA planes, the result)
//     moves as 16-byte shared-memory accesses for both zones at once: 41 shared-memory instructions per zone, not 82;
//   * 128 zone threads + edge warp + producer warp per CTA, two CTAs per SM.  The CTA is launched with 256 threads at
//     128 registers; the second warpgroup (edge, producer, two idle warps) drops to 64 registers and the zone warps
//     rise to 192 (setmaxnreg): one spill instruction per plane instead of 24 at 168 registers (5.87 vs 6.39 ms);
//   * the flux differences are folded into a running result as each flux becomes known; every flux enters as a
//     DIFFERENCE of two face fluxes, so a uniform state is preserved bit for bit as in the other kernels.
// What was measured (each a gpurun of config 5, ms per stage): first version at 168 registers 6.5; integer-pipe minmod
// (nine integer instructions for one DSETP) 6.9; the z window rotated by a three-fold unrolled loop (63 KB of loop body:
// instruction-cache misses) 7.3-7.6; setmaxnreg 192/64: 5.87; two-wide values: 5.99; helper warps moved to warps 4 and 6
// (one per sub-partition by %warpid): 6.24.  ncu on the first version: 683 thread instructions per zone against 726 --
// the selects, compares and moves of two zones do not shrink with the shared-memory traffic --, issue slots 47 % busy with
// 3 warps per scheduler (56 % with 5), 25 % of the warp time at the two CTA barriers per plane.  Fewer, fatter warps
// lose more to the barriers than the shorter exchange phases win.
//
// Roles, planes, ring slots, halo boxes, z chains and the fused CFL reduction are those of fx_stage_tma.cu; the comments
// there describe the protocol (the wall / gravity code is written but not instantiated here).  Differences: P has an
// even row stride (16-byte accesses), Lx holds one slot per EVEN face (9 per row), and beta dt/dx_d of a block lives in
// a slot chosen by the parity of the block's position in the segment, because the running result needs it on both
// sides of the CTA barriers.
#include <cuda.h>
#include <string.h>

#include "fx_physics.cuh"
#include "fx_tma.cuh"
#include "fx_vec2.cuh"

namespace fxp {

using namespace fxtma;

constexpr int NX = 16, NY = 16;
constexpr int NZT = NX * NY / 2;       // 128 zone threads, two zones each
constexpr int NTHREADS = NZT + 64;     // + edge warp + producer warp: the threads that work and meet at the CTA barriers
constexpr int NLAUNCH = 256;           // two whole warpgroups (setmaxnreg is a warpgroup operation): warps 6 and 7 only give
                                       // their registers to the zone warps and leave
constexpr int ZONE_REGS = 192, HELPER_REGS = 64;  // 4 x 32 x (192 + 64) = the 8 x 32 x 128 registers of the launch
constexpr int PLANE_BYTES = 5 * NY * NX * 8;
constexpr int r = 1, R = 2, NP = NX + 2 * R, BW = 2, NRING = 4;
constexpr int PS = NP + 2;             // row stride of P: even (16-byte accesses); 22 puts the edge warp's column accesses
                                       // on 8 distinct bank pairs (2-way conflict, that warp only)
constexpr int LXS = 9;                 // slots per row of Lx: faces 0, 2, .., 16

struct alignas(128) Smem {
  double ring[NRING][5][NY][NX];  // TMA: stage-input planes, plane z in slot z mod NRING
  double U0[2][5][NY][NX];        // TMA: U0 planes (later stages)
  double Out[5][NY][NX];          // result plane, drained by a TMA store
  double Hx[2][5][NY][BW];        // TMA: [lo|hi] raw x-halo cells of the plane
  double Hy[2][5][R][NX];         // TMA: [lo|hi] raw y-halo cells of the plane
  double P[5][NP][PS];            // primitives of the plane incl. halo rows/columns (corners unused)
  double Lx[5][NY][LXS];          // Lx[v][j][f/2], f even: plus-side x state of cell f-1, then the x flux at face f
  double Ly[5][NY + 1][NX];       // Ly[v][f][i]: plus-side y state of cell (i, f-1), then the y flux at face f
  double rd[2][4];                // beta dt / dx_d of the block being worked on, slot = parity of its position in the segment
  double idx[2][4];               // 1 / dx_d (DTOUT)
  int chain[FX_SEG_STRIDE];
  double wmax[4];
  unsigned long long barX[2], barH;
};

__device__ __forceinline__ void cta_sync() { asm volatile("bar.sync 0, %0;" ::"n"(NTHREADS) : "memory"); }

__device__ __forceinline__ double2 lds2(const double *p) { return *reinterpret_cast<const double2 *>(p); }
__device__ __forceinline__ void sts2(double *p, double a, double b) { *reinterpret_cast<double2 *>(p) = make_double2(a, b); }

template <int RIEMANN, int WS, int D, class T>
__device__ __forceinline__ void flux_dir(const FxParams &P, const T WL[5], const T WR[5], T F[5]) {
  constexpr int in = 1 + D, it1 = 1 + (D + 1) % 3, it2 = 1 + (D + 2) % 3;
  const T wl[5] = {WL[0], WL[in], WL[it1], WL[it2], WL[4]};
  const T wr[5] = {WR[0], WR[in], WR[it1], WR[it2], WR[4]};
  T f[5];
  fx2::riemann<RIEMANN, WS>(P, wl, wr, f);
  F[0] = f[0];
  F[in] = f[1];
  F[it1] = f[2];
  F[it2] = f[3];
  F[4] = f[4];
}

template <int RIEMANN, int WS, bool FIRST, bool DTOUT, bool EXTRAS>
__global__ void __launch_bounds__(NLAUNCH, 2)
fx_k_stage_pair(const __grid_constant__ CUtensorMap mXm, const __grid_constant__ CUtensorMap mXx,
                const __grid_constant__ CUtensorMap mXy, const __grid_constant__ CUtensorMap mU0,
                const __grid_constant__ CUtensorMap mOut, const FxParams P, const double *__restrict__ X,
                const double *__restrict__ dx, double dt, const double *dt_dev, double beta,
                double cfl_next, double *dt_next) {
  extern __shared__ __align__(1024) unsigned char fx_smem_raw[];
  Smem &S = *reinterpret_cast<Smem *>(fx_smem_raw);
  const int tid = threadIdx.x;
  const int nzb = P.n[2];
  const int g0 = P.gd[0], g1 = P.gd[1], g2 = P.gd[2];
  unsigned hit = 0;
  if (tid < FX_SEG_STRIDE) S.chain[tid] = __ldg(&P.seg[(long long)blockIdx.x * FX_SEG_STRIDE + tid]);
  __syncthreads();
  const int M = S.chain[0];
  const int nz = M * nzb;
  const unsigned zmagic = ((1u << 20) + (unsigned)nzb - 1u) / (unsigned)nzb;
  auto zmap = [&](int Z, int &bs, int &kp) {  // where plane Z of the column lives: block id and padded k
    int qb = Z < 0 ? -1 : (M == 1 ? (int)(Z >= nzb) : (int)(((unsigned)Z * zmagic) >> 20));
    int k = Z - qb * nzb;
    int id = S.chain[2 + qb];
    if (id < 0) {
      const bool wall = EXTRAS && id == FX_BC_REFLECT;
      if (qb < 0) { id = S.chain[2]; k = wall ? -1 - Z : 0; } else { id = S.chain[1 + M]; k = wall ? nzb - 1 - (Z - nz) : nzb - 1; }
    }
    bs = id;
    kp = k + g2;
  };
  const bool wall_below = EXTRAS && S.chain[1] == FX_BC_REFLECT;
  const int zflip_from = (EXTRAS && S.chain[2 + M] == FX_BC_REFLECT) ? nz : 0x7fffffff;

  // ---------------------------------------------------------------- producer set-up (producer warp, lane 0)
  constexpr int PROD0 = NZT + 32;
  const bool is_prod = tid >= PROD0 && tid < PROD0 + 32;
  const bool is_edge = tid >= NZT && tid < NZT + 32;
  const bool producer = tid == PROD0;
  auto issue_X = [&](int c) {  // stage-input plane consumed at tick c: z index c + r
    int bs, kp;
    zmap(c + r, bs, kp);
    mbar_expect_tx(&S.barX[c & 1], PLANE_BYTES);
    tma_load(&S.ring[(c + r) % NRING][0][0][0], &mXm, &S.barX[c & 1], g0, g1, kp, bs);
  };
  int hk = 0, hq = 0, hb = 0, xlo = 0, xhi = 0, ylo = 0, yhi = 0;
  auto halo_block = [&]() {
    hb = S.chain[2 + hq];
    xlo = __ldg(&P.neigh[(long long)hb * 6 + 0]);
    xhi = __ldg(&P.neigh[(long long)hb * 6 + 1]);
    ylo = __ldg(&P.neigh[(long long)hb * 6 + 2]);
    yhi = __ldg(&P.neigh[(long long)hb * 6 + 3]);
  };
  if (is_prod) halo_block();
  auto issue_H = [&]() {
    const int b = hb, kp = hk + g2;
    mbar_expect_tx(&S.barH, 2 * 5 * NY * BW * 8 + 2 * 5 * R * NX * 8);
    tma_load(&S.Hx[0][0][0][0], &mXx, &S.barH, g0 + (xlo >= 0 ? NX - BW : 0), g1, kp, xlo >= 0 ? xlo : b);
    tma_load(&S.Hx[1][0][0][0], &mXx, &S.barH, g0 + (xhi >= 0 ? 0 : NX - BW), g1, kp, xhi >= 0 ? xhi : b);
    tma_load(&S.Hy[0][0][0][0], &mXy, &S.barH, g0, g1 + (ylo >= 0 ? NY - R : 0), kp, ylo >= 0 ? ylo : b);
    tma_load(&S.Hy[1][0][0][0], &mXy, &S.barH, g0, g1 + (yhi >= 0 ? 0 : NY - R), kp, yhi >= 0 ? yhi : b);
  };
  auto issue_U0 = [&](int p, int b, int k) {
    mbar_expect_tx(&S.barX[(p + 1) & 1], PLANE_BYTES);
    tma_load(&S.U0[p & 1][0][0][0], &mU0, &S.barX[(p + 1) & 1], g0, g1, k + g2, b);
  };
  if (producer) {
    mbar_init(&S.barX[0], FIRST ? 1 : 2); mbar_init(&S.barX[1], FIRST ? 1 : 2);
    mbar_init(&S.barH, 1);
    fence_mbar_init();
    fence_async_smem();
    issue_X(1);
    issue_H();
    if (!FIRST) issue_U0(0, S.chain[2], 0);
  }
  if (dt_dev) dt = *dt_dev;
  __syncthreads();  // barriers initialised before anyone waits on them (all launched threads: the idle warps too)

  // (the second warpgroup -- edge warp, producer warp, two idle warps -- gives registers back to the
  // CTA's pool and the zone warps take them: launch 8 x 32 x 128 = 4 x 32 x (ZONE_REGS + HELPER_REGS).
  // Each role changes its count at the head of its own branch: after a join ptxas assumes the smaller count.)
#define FX_REG_INC() asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(ZONE_REGS))
#define FX_REG_DEC() asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(HELPER_REGS))
  if (tid >= NTHREADS) {  // idle warps
    FX_REG_DEC();
  } else if (tid < NZT) {
    FX_REG_INC();
    // ------------------------------------------------------------ zone threads: zones (i2, j) and (i2 + 1, j), every value a
    // pair (fx_vec2.cuh): .a is zone i2, .b is zone i2 + 1
    using fx2::d2;
    using fx2::mk;
    const int ip = tid & 7, i2 = 2 * ip, j = tid >> 3;
    double rate = 0.0;
    d2 qA[5], qB[5], qC[5];  // the z window: primitives of cells c-1, c, c+1 at tick c
    d2 qpz[5], Fz[5];        // plus-side z state of cell c-1; z flux of face c-1
    {
      const long long col = (long long)(j + g1) * P.S_j + (i2 + g0);
      d2 w[2 * R][5];
#pragma unroll
      for (int m = 0; m < 2 * R; ++m) {
        int bs, kp;
        zmap(m - R, bs, kp);
        const long long a = (long long)bs * P.S_b + (long long)kp * P.S_k + col;
#pragma unroll
        for (int v = 0; v < 5; ++v) {
          const double2 t = *reinterpret_cast<const double2 *>(X + a + v * P.S_v);
          w[m][v] = mk(t.x, t.y);
        }
        if (m < R && wall_below) w[m][3] = -w[m][3];
      }
#pragma unroll
      for (int m = 0; m < 2 * R; ++m) {
        if (m >= R) {  // planes 0 .. r do not come through the TMA ring: keep them there for the combine
#pragma unroll
          for (int v = 0; v < 5; ++v) sts2(&S.ring[(m - R) % NRING][v][j][i2], w[m][v].a, w[m][v].b);
        }
        const unsigned h = fx2::c2p(P, w[m], w[m]);
        if (m >= R && m - R < nz) hit |= h;
      }
      d2 qpm1[5], qm0[5];
#pragma unroll
      for (int v = 0; v < 5; ++v) {
        const d2 mm1 = fx2::minmod(w[1][v] - w[0][v], w[2][v] - w[1][v]);  // cell -1
        const d2 m0 = fx2::minmod(w[2][v] - w[1][v], w[3][v] - w[2][v]);   // cell 0
        qpm1[v] = fx2::vfma(0.5, mm1, w[1][v]);
        qm0[v] = fx2::vfma(-0.5, m0, w[2][v]);
        qpz[v] = fx2::vfma(0.5, m0, w[2][v]);
      }
      flux_dir<RIEMANN, WS, 2>(P, qpm1, qm0, Fz);
#pragma unroll
      for (int v = 0; v < 5; ++v) { qA[v] = w[2][v]; qB[v] = w[3][v]; }
    }
#pragma unroll
    for (int v = 0; v < 5; ++v) sts2(&S.P[v][j + R][i2 + R], qA[v].a, qA[v].b);  // plane 0
    cta_sync();  // A0

    int pk = 0, par = 0;  // plane p is plane pk of its block; par = parity of the block's position in the segment
    // one tick: q0 = cell c-1 (plane p, the in-plane work), q1 = cell c, q2 receives cell c+1
    auto tick = [&](const int c, d2 (&q0)[5], d2 (&q1)[5], d2 (&q2)[5]) __attribute__((always_inline)) {
      const int p = c - 1;
      // ---------------------------------------------------------------- phase 1: in-plane reconstruction of plane p
      d2 qmx[5], qmy[5];  // minus-side x and y states of both zones
      double xap[5];      // plus-side x state of zone a: the left state of the pair's own face
#pragma unroll
      for (int v = 0; v < 5; ++v) {
        const double l = S.P[v][j + R][i2 + R - 1], rr = S.P[v][j + R][i2 + R + 2];
        const double d1 = q0[v].b - q0[v].a;  // the middle difference serves both zones
        const d2 m = fx2::minmod(mk(q0[v].a - l, d1), mk(d1, rr - q0[v].b));
        qmx[v] = fx2::vfma(-0.5, m, q0[v]);
        const d2 qp = fx2::vfma(0.5, m, q0[v]);
        xap[v] = qp.a;
        S.Lx[v][j][ip + 1] = qp.b;
      }
#pragma unroll
      for (int v = 0; v < 5; ++v) {
        const double2 dn = lds2(&S.P[v][j + R - 1][i2 + R]), up = lds2(&S.P[v][j + R + 1][i2 + R]);
        const d2 m = fx2::minmod(q0[v] - mk(dn.x, dn.y), mk(up.x, up.y) - q0[v]);
        qmy[v] = fx2::vfma(-0.5, m, q0[v]);
        const d2 qp = fx2::vfma(0.5, m, q0[v]);
        sts2(&S.Ly[v][j + 1][i2], qp.a, qp.b);
      }
      cta_sync();  // B: plus-side states visible; this tick's TMA planes have landed (the producer waited for them)
      // ---------------------------------------------------------------- phase 2: fluxes, folded into the running result.
      // Every flux enters as a DIFFERENCE of two face fluxes: a uniform state has equal fluxes at all faces and stays what it
      // was, bit for bit
      const double rx = S.rd[par][0], ry = S.rd[par][1], rz = S.rd[par][2];
      d2 acc[5];  // [U0 + beta (X - U0)] - sum_d (beta dt/dx_d) (F_d+ - F_d-), as the fluxes become known
      d2 xs5[5];
#pragma unroll
      for (int v = 0; v < 5; ++v) {
        const double2 xs = lds2(&S.ring[p % NRING][v][j][i2]);
        if (FIRST) {
          acc[v] = mk(xs.x, xs.y);
        } else {
          const double2 u0 = lds2(&S.U0[p & 1][v][j][i2]);
          acc[v] = fx2::vfma(beta, mk(xs.x, xs.y) - mk(u0.x, u0.y), mk(u0.x, u0.y));
        }
        if (EXTRAS) xs5[v] = mk(xs.x, xs.y);
      }
      if (EXTRAS && P.grav_on) {  // + beta dt (0, rho g, g . m) of the stage input's own zone [B10]
        const double bdt = (FIRST ? 1.0 : beta) * dt;
        acc[4] = fx2::vfma(bdt, fx2::vfma(P.grav[2], xs5[3], fx2::vfma(P.grav[1], xs5[2], P.grav[0] * xs5[1])), acc[4]);
#pragma unroll
        for (int d = 0; d < 3; ++d) acc[1 + d] = fx2::vfma(bdt * P.grav[d], xs5[0], acc[1 + d]);
      }
      double Fxi[5];  // flux at the pair's own x face: high face of zone a, low face of zone b
      {  // the two x solves of the thread side by side: .a = low face of zone a, .b = the pair's own face
        d2 WL[5], F[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) WL[v] = mk(S.Lx[v][j][ip], xap[v]);
        flux_dir<RIEMANN, WS, 0>(P, WL, qmx, F);
#pragma unroll
        for (int v = 0; v < 5; ++v) {
          S.Lx[v][j][ip] = F[v].a;  // in place: only this thread read the state
          acc[v].a = fma(-rx, F[v].b - F[v].a, acc[v].a);
          Fxi[v] = F[v].b;
        }
      }
      {  // new cells of the z windows
        d2 u[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) {
          const double2 t = lds2(&S.ring[(c + r) % NRING][v][j][i2]);
          u[v] = mk(t.x, t.y);
        }
        if (EXTRAS && c + r >= zflip_from) u[3] = -u[3];
        const unsigned h = fx2::c2p(P, u, q2);
        if (c + r < nz) hit |= h;
      }
      {  // z: reconstruct cell c, flux of face c (between cells c-1 and c)
        d2 mz[5], qmz[5], F[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) {
          mz[v] = fx2::minmod(q1[v] - q0[v], q2[v] - q1[v]);
          qmz[v] = fx2::vfma(-0.5, mz[v], q1[v]);
        }
        flux_dir<RIEMANN, WS, 2>(P, qpz, qmz, F);
#pragma unroll
        for (int v = 0; v < 5; ++v) {
          qpz[v] = fx2::vfma(0.5, mz[v], q1[v]);  // (after the solve that read the old one)
          acc[v] = fx2::vfma(-rz, F[v] - Fz[v], acc[v]);
          Fz[v] = F[v];
        }
      }
      d2 Fy[5];  // y fluxes at the low faces of both zones (kept for the differences after barrier C: the slot they are
                 // published in belongs to the row below from the next tick's phase 1 on)
      {
        d2 WL[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) {
          const double2 t = lds2(&S.Ly[v][j][i2]);
          WL[v] = mk(t.x, t.y);
        }
        flux_dir<RIEMANN, WS, 1>(P, WL, qmy, Fy);
#pragma unroll
        for (int v = 0; v < 5; ++v) sts2(&S.Ly[v][j][i2], Fy[v].a, Fy[v].b);
      }
      if (c < nz) {  // primitives of plane p + 1: nobody reads P between barriers B and C
#pragma unroll
        for (int v = 0; v < 5; ++v) sts2(&S.P[v][j + R][i2 + R], q1[v].a, q1[v].b);
      }
      cta_sync();  // C: fluxes and the next plane's primitives visible
      // ---------------------------------------------------------------- phase 3: the neighbours' fluxes, result
      {
        int hmax = 0;
#pragma unroll
        for (int v = 0; v < 5; ++v) {
          const double fxh = S.Lx[v][j][ip + 1];
          const double2 fyh = lds2(&S.Ly[v][j + 1][i2]);
          acc[v] = fx2::vfma(-ry, mk(fyh.x, fyh.y) - Fy[v], acc[v]);
          acc[v].b = fma(-rx, fxh - Fxi[v], acc[v].b);
          sts2(&S.Out[v][j][i2], acc[v].a, acc[v].b);
          if (!DTOUT) hmax = max(hmax, max(__double2hiint(acc[v].a) & 0x7fffffff, __double2hiint(acc[v].b) & 0x7fffffff));
        }
        if (!DTOUT && hmax >= 0x7ff00000) hit |= FX_STATUS_NONFINITE;
        if (DTOUT) {  // a7 on the finished zones: (|u_d| + c) / dx_d, folded into a running maximum [O7]
          d2 w[5], ir;
          hit |= fx2::c2p(P, acc, w, &ir) & FX_STATUS_NONFINITE;
          const d2 cs = fx2::sqrt3(P.gamma * w[4] * ir);
          const d2 r01 = fx2::max_sel((fx2::vabs(w[1]) + cs) * S.idx[par][0], (fx2::vabs(w[2]) + cs) * S.idx[par][1]);
          const d2 r2 = fx2::max_sel((fx2::vabs(w[3]) + cs) * S.idx[par][2], r01);
          rate = fx_max_sel(fx_max_sel(r2.a, r2.b), rate);
        }
        fence_async_smem();  // the TMA store reads Out through the async proxy
      }
      if (++pk == nzb) { pk = 0; par ^= 1; }
    };
#pragma unroll 1
    for (int c = 1; c <= nz; ++c) {
      tick(c, qA, qB, qC);
#pragma unroll
      for (int v = 0; v < 5; ++v) { qA[v] = qB[v]; qB[v] = qC[v]; }
    }
    if (DTOUT) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) rate = fmax(rate, __shfl_xor_sync(0xffffffffu, rate, o));
      if ((tid & 31) == 0) S.wmax[tid >> 5] = rate;
    }
    cta_sync();  // D: the last plane is in Out
  } else if (is_edge) {
    FX_REG_DEC();
    // ------------------------------------------------------------ edge warp: cell -1 and cell 16 of every row (lanes
    // 16..31) and column (lanes 0..15), their 17th face, and beta dt / dx_d of each block
    const int lane = tid - NZT;
    const bool isx = lane >= 16;
    const int m = lane & 15;
    double *Pf = &S.P[0][0][0];
    const int pd = isx ? 1 : PS, pt = isx ? PS : 1;
    double *Lf = isx ? &S.Lx[0][0][0] : &S.Ly[0][0][0];
    const int lv = isx ? NY * LXS : (NY + 1) * NX;                      // per-variable size
    const int l0 = isx ? m * LXS : m, l16 = isx ? m * LXS + 8 : NY * NX + m;  // slots of faces 0 and 16 of this row / column
    int pk = 0, pq = 0, pb = S.chain[2];
    auto block_rates = [&]() {
      if (lane < 3) {
        const double dxd = __ldg(&dx[(long long)pb * 3 + lane]);
        S.rd[pq & 1][lane] = (FIRST ? 1.0 : beta) * dt / dxd;
        if (DTOUT) S.idx[pq & 1][lane] = 1.0 / dxd;
      }
    };
    block_rates();
    cta_sync();  // A0

#pragma unroll 1
    for (int c = 1; c <= nz; ++c) {
      double qm16[5];
#pragma unroll
      for (int v = 0; v < 5; ++v) {
        const double *pv = Pf + v * NP * PS + (m + R) * pt;
        double qm, qp;
        fx_plm(pv[0], pv[pd], pv[2 * pd], qm, qp);  // cell -1 (padded position 1)
        Lf[v * lv + l0] = qp;
        fx_plm(pv[(NX + 1) * pd], pv[(NX + 2) * pd], pv[(NX + 3) * pd], qm16[v], qp);  // cell 16 (padded position 18)
      }
      // a block's first plane: its rates go to the slot of its parity (read by the zone threads from barrier B on; the
      // other slot is still in use by the combines of the block below)
      if (pk == 0 && c > 1) block_rates();
      cta_sync();  // B
      {
        double WL[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) WL[v] = Lf[v * lv + l16];
        const double wl[5] = {WL[0], isx ? WL[1] : WL[2], isx ? WL[2] : WL[3], isx ? WL[3] : WL[1], WL[4]};
        const double wr[5] = {qm16[0], isx ? qm16[1] : qm16[2], isx ? qm16[2] : qm16[3], isx ? qm16[3] : qm16[1], qm16[4]};
        double f[5];
        fx2::riemann<RIEMANN, WS>(P, wl, wr, f);
        double F[5];
        F[0] = f[0];
        F[1] = isx ? f[1] : f[3];
        F[2] = isx ? f[2] : f[1];
        F[3] = isx ? f[3] : f[2];
        F[4] = f[4];
#pragma unroll
        for (int v = 0; v < 5; ++v) Lf[v * lv + l16] = F[v];
      }
      if (++pk == nzb) {
        pk = 0;
        ++pq;
        pb = S.chain[2 + pq];
      }
      cta_sync();  // C
    }
    cta_sync();  // D
  } else {
    FX_REG_DEC();
    // ------------------------------------------------------------ producer warp: lane 0 issues the bulk copies, all
    // lanes convert the halo cells (lanes 0..15 the y edges of column m, lanes 16..31 the x edges of row m)
    const int lane = tid - PROD0;
    const bool isx = lane >= 16;
    const int m = lane & 15;
    double *Pf = &S.P[0][0][0];
    const int pd = isx ? 1 : PS, pt = isx ? PS : 1;
    constexpr int HXV = NY * BW, HYV = R * NX;
    int nlo = isx ? xlo : ylo, nhi = isx ? xhi : yhi;
    auto halo_off = [&](int t, bool high) -> int {
      int idx;
      if (isx) idx = high ? (nhi >= 0 ? t : ((EXTRAS && nhi == FX_BC_REFLECT) ? BW - 1 - t : BW - 1)) : (nlo >= 0 ? BW - R + t : ((EXTRAS && nlo == FX_BC_REFLECT) ? R - 1 - t : 0));
      else idx = high ? (nhi >= 0 ? t : ((EXTRAS && nhi == FX_BC_REFLECT) ? R - 1 - t : R - 1)) : (nlo >= 0 ? t : ((EXTRAS && nlo == FX_BC_REFLECT) ? R - 1 - t : 0));
      return isx ? ((high ? 5 * HXV : 0) + m * BW + idx) : ((high ? 5 * HYV : 0) + idx * NX + m);
    };
    int hoff[2 * R];
#pragma unroll
    for (int t = 0; t < 2 * R; ++t) hoff[t] = halo_off(t % R, t >= R);
    const int hv = isx ? HXV : HYV;

    auto halo_plane = [&](int pl) {
      mbar_wait(&S.barH, pl & 1);
      const double *Hf = isx ? &S.Hx[0][0][0][0] : &S.Hy[0][0][0][0];
#pragma unroll
      for (int t = 0; t < 2 * R; ++t) {
        double u[5], w[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) u[v] = Hf[hoff[t] + v * hv];
        if (EXTRAS && (t < R ? nlo : nhi) == FX_BC_REFLECT) {
          if (isx) u[1] = -u[1]; else u[2] = -u[2];
        }
        fx_c2p_v2(P, u[0], u[1], u[2], u[3], u[4], w);
        const int pos = (t < R) ? t : (NX + t);
#pragma unroll
        for (int v = 0; v < 5; ++v) Pf[v * NP * PS + pos * pd + (m + R) * pt] = w[v];
      }
      __syncwarp();
      if (pl + 1 < nz) {
        if (++hk == nzb) {
          hk = 0;
          ++hq;
          halo_block();
          nlo = isx ? xlo : ylo;
          nhi = isx ? xhi : yhi;
#pragma unroll
          for (int t = 0; t < 2 * R; ++t) hoff[t] = halo_off(t % R, t >= R);
        }
        if (lane == 0) issue_H();
      }
    };
    halo_plane(0);
    cta_sync();  // A0
    int pk = 0, pq = 0, pb = S.chain[2], pb_prev = pb;
#pragma unroll 1
    for (int c = 1; c <= nz; ++c) {
      const int p = c - 1;
      mbar_wait(&S.barX[c & 1], ((c - 1) >> 1) & 1);
      cta_sync();  // B
      if (lane == 0) {
        if (c + 1 <= nz) issue_X(c + 1);
        if (p >= 1) {
          tma_store(&mOut, &S.Out[0][0][0], g0, g1, (pk >= 1 ? pk - 1 : nzb - 1) + g2, pk >= 1 ? pb : pb_prev);
          tma_commit();
        }
        if (!FIRST && p + 1 < nz) {
          if (pk + 1 < nzb) issue_U0(p + 1, pb, pk + 1);
          else issue_U0(p + 1, S.chain[3 + pq], 0);
        }
      }
      if (++pk == nzb) {
        pk = 0;
        ++pq;
        pb_prev = pb;
        pb = S.chain[2 + pq];
      }
      if (c < nz) halo_plane(c);
      if (lane == 0 && p >= 1) tma_wait_read();
      cta_sync();  // C
    }
    cta_sync();  // D
    if (lane == 0) {
      tma_store(&mOut, &S.Out[0][0][0], g0, g1, nzb - 1 + g2, S.chain[1 + M]);
      tma_commit();
      if (DTOUT) {
        double mx = S.wmax[0];
#pragma unroll
        for (int w4 = 1; w4 < 4; ++w4) mx = fmax(mx, S.wmax[w4]);
        atomicMax(&P.scratch[FX_SCR_DTBITS], (unsigned long long)__double_as_longlong(mx));
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
template <int RIEMANN, int WS, bool FIRST, bool DTOUT, bool EXTRAS>
int launch(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt, const double *dt_dev,
           double beta, double cfl_next, double *dt_next, cudaStream_t st) {
  CUtensorMap mXm, mXx, mXy, mU0, mOut;
  int rc;
  if ((rc = make_map(&mXm, P, X, NX, NY))) return rc;
  if ((rc = make_map(&mXx, P, X, BW, NY))) return rc;
  if ((rc = make_map(&mXy, P, X, NX, R))) return rc;
  if ((rc = make_map(&mU0, P, U0, NX, NY))) return rc;
  if ((rc = make_map(&mOut, P, out, NX, NY))) return rc;
  auto kern = fx_k_stage_pair<RIEMANN, WS, FIRST, DTOUT, EXTRAS>;
  const int smem = (int)sizeof(Smem);
  FX_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  kern<<<(unsigned)P.nseg, NLAUNCH, smem, st>>>(mXm, mXx, mXy, mU0, mOut, P, X, dx, dt, dt_dev, beta, cfl_next, dt_next);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fx_fail(FX_ERR_CUDA, "stage_pair launch: %s (smem %d)", cudaGetErrorString(e), smem);
  return FX_OK;
}

template <int RIEMANN, int WS>
int launch_ws(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt, const double *dt_dev,
              double beta, int first, double cfl_next, double *dt_next, cudaStream_t st) {
  if (first) return launch<RIEMANN, WS, true, false, false>(P, X, U0, out, dx, dt, dt_dev, beta, 0.0, nullptr, st);
  if (dt_next) return launch<RIEMANN, WS, false, true, false>(P, X, U0, out, dx, dt, dt_dev, beta, cfl_next, dt_next, st);
  return launch<RIEMANN, WS, false, false, false>(P, X, U0, out, dx, dt, dt_dev, beta, 0.0, nullptr, st);
}

}  // namespace fxp

// PLM without walls or gravity on the shapes fx_stage_tma_supported accepts (the EXTRAS code paths are written but not
// instantiated: this kernel is the slower one, kept selectable as the record of the experiment -- FX_OPT_PATH = 3)
bool fx_stage_pair_supported(const FxParams &P) {
  return fx_stage_tma_supported(P) && P.recon == FX_RECON_PLM_MINMOD && !P.walls && !P.grav_on;
}

int fx_launch_stage_pair(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt,
                         const double *dt_dev, double beta, int first, double cfl_next, double *dt_next, cudaStream_t st) {
  if (!fx_stage_pair_supported(P)) return fx_fail(FX_ERR_UNSUPPORTED, "pair stage kernel: plan not supported");
  if (P.nblocks == 0) return FX_OK;
  if (first && X != U0) return fx_fail(FX_ERR_INVALID_ARG, "pair stage kernel: the first stage takes U0 from its stage input (X must be U0)");
  if (((uintptr_t)X | (uintptr_t)U0 | (uintptr_t)out) & 15)
    return fx_fail(FX_ERR_INVALID_ARG, "pair stage kernel: state arrays must be 16-byte aligned");
#ifdef FX_DEV_FAST
  return fxp::launch_ws<FX_RIEMANN_HLLC, 0>(P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st);
#else
  if (P.riemann == FX_RIEMANN_HLLE)
    return P.wavespeed == 0 ? fxp::launch_ws<FX_RIEMANN_HLLE, 0>(P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st)
                            : fxp::launch_ws<FX_RIEMANN_HLLE, 1>(P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st);
  return P.wavespeed == 0 ? fxp::launch_ws<FX_RIEMANN_HLLC, 0>(P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st)
                          : fxp::launch_ws<FX_RIEMANN_HLLC, 1>(P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st);
#endif
}
