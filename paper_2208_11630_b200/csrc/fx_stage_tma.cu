// fx_stage_tma.cu -- fused per-stage kernel for 3-D blocks with a 16 x 16 (x, y) cross-section (K1+K2+K3),
// fed and drained by TMA.
//
// One 320-thread CTA per SEGMENT -- up to 8 blocks that follow one another in +z (fx_hydro_plan_set_topology builds
// the table) -- marches a 16 x 16 column of zones through the segment's planes; two CTAs share an SM, so that one
// of them computes while the other waits at a barrier or for data.  Thread (i,j) of the 256 zone threads owns the
// zones (i,j,k) of every block of the segment (a block's top halo is the next block's first planes, already in the ring):
//   * every plane of the stage input arrives as ONE 5-D TMA box {16,16,1,1,5} of U[v][b][k][j][i] in a ring of r + 3
//     shared-memory slots, a tick ahead of its use, and stays there until the zones of that plane are combined
//     (the combine needs the stage input again: it is U0 in the first stage, X in the later ones -- no second
//     load); in the later stages the U0 plane arrives the same way (2 slots), and the finished plane leaves as one
//     TMA box store.  No thread computes a global address inside the z loop and nothing is prefetched through
//     registers;
//   * z direction: a sliding window of primitive cells lives in registers; each plane is converted to
//     primitives once and serves the z reconstruction, the z Riemann problem and, R planes later, the
//     in-plane work of the same zone;
//   * x and y directions: per plane the threads exchange primitives, plus-side face states and face fluxes
//     through shared memory with TWO CTA barriers per plane: (B) plus-side states published -> Riemann solves,
//     each face's flux overwriting, in place, the plus-side state it was computed from, and the primitives of the
//     NEXT plane written (nobody reads them in that phase); (C) fluxes visible -> flux divergence and RK
//     combination, which runs on into the next plane's reconstruction without a barrier;
//   * two more warps supply what a 16-wide row lacks.  The "edge" warp reconstructs cell -1 (its plus-side state) and
//     cell 16 of every row and column and solves their 17th face.  The "producer" warp issues every TMA operation
//     (lane 0) and converts the halo cells of the plane -- TMA boxes {2|4,16,1,1,5} and {16,R,1,1,5} taken straight
//     from the neighbour blocks' interiors through the neighbour table (or from this block's own edge cells at an
//     outflow boundary or, mirrored and with the normal momentum negated, at a reflecting wall; no guard cell in HBM
//     is read or written).  They are two warps because the per-plane dependent chain of one warp doing both was as
//     long as a zone warp's and delayed the CTA barriers.
// In the last stage of fx_hydro_step (DTOUT) each finished zone also contributes (|u_d| + c)/dx_d to a running
// maximum, reduced per warp, per CTA and with one atomicMax per CTA: the CFL step of the advanced state costs no pass.
// HBM traffic per zone: one read of the stage input (+ U0 in later stages), one write, plus halos.
#include <cuda.h>
#include <string.h>

#include "fx_physics.cuh"
#include "fx_tma.cuh"

namespace fxt {

constexpr int NX = 16, NY = 16;
constexpr int NZONE_THREADS = NX * NY;        // 256
constexpr int NTHREADS = NZONE_THREADS + 64;  // + edge warp + producer warp
constexpr int PLANE_BYTES = 5 * NY * NX * 8;  // one TMA box of the main kind

template <int RECON> struct Rc {
  static constexpr int r = (RECON == FX_RECON_PLM_MINMOD) ? 1 : 2;  // stencil radius of one cell's reconstruction
  static constexpr int R = r + 1;                                    // halo depth
  static constexpr int NP = NX + 2 * R;                              // padded plane extent
  static constexpr int BW = (R + 1) & ~1;                            // x-halo box width: TMA rows are multiples of 16 B
  static constexpr int NRING = r + 3;  // a stage-input plane stays in shared memory from its conversion (tick z - r) to the
                                       // combination of its zones (until barrier B of tick z + 2) while the next one loads
  static constexpr int NREG = (RECON == FX_RECON_PLM_MINMOD) ? 96 : 168;  // registers per thread for 2 / 1 CTAs per SM: the register file is 16384 per SM sub-partition, and 20 / 10 warps put 5 / 3 on one of them
};

template <int RECON> struct alignas(128) Smem {
  static constexpr int R = Rc<RECON>::R, NP = Rc<RECON>::NP, BW = Rc<RECON>::BW, NRING = Rc<RECON>::NRING;
  double ring[NRING][5][NY][NX];  // TMA: stage-input planes, plane z in slot z mod NRING; read twice: converted to
                                  // primitives for the fluxes, and again as X (or, in the first stage, U0 = X) by the combine
  double U0[2][5][NY][NX];     // TMA: U0 planes, slot = plane & 1 (later stages; in the first stage U0 is the stage input)
  double Out[5][NY][NX];       // result plane, drained by a TMA store
  double Hx[2][5][NY][BW];     // TMA: [lo|hi] raw x-halo cells of the plane (one slot: the edge warp alone reads it)
  double Hy[2][5][R][NX];      // TMA: [lo|hi] raw y-halo cells of the plane
  double P[5][NP][NP + 1];     // primitives of the plane incl. halo rows/columns (corners unused); the odd row
                               // stride keeps the edge warp's column accesses free of bank conflicts
  double Lx[5][NY][NX + 1];    // Lx[v][j][i] = plus-side x state of cell (i-1,j), then the x flux at face i-1/2
  double Ly[5][NY + 1][NX];    // Ly[v][j][i] = plus-side y state of cell (i,j-1), then the y flux at face j-1/2
  double rd[3];                // beta dt / dx_d (beta = 1 in the first stage) of the block whose planes are being combined;
                               // rewritten by the edge warp between barriers B and C of a block's first tick
  double idx[3];               // 1 / dx_d (DTOUT: the CFL rate of the finished state is formed in the last stage)
  int chain[FX_SEG_STRIDE];    // this CTA's segment: {count, below, id_0 .. id_{count-1}, above}
  double wmax[8];              // DTOUT: per-warp maximum of (|u_d| + c) / dx_d
  unsigned long long barX[2], barH;  // barX[c & 1]: stage-input plane of tick c AND (later stages) the U0 plane of plane c - 1
};

using namespace fxtma;
__device__ __forceinline__ void cta_sync() { asm volatile("bar.sync 0, %0;" ::"n"(NTHREADS) : "memory"); }

// Riemann flux for direction D (compile-time) from un-rotated primitive states; flux returned in the
// un-rotated variable order (rho, mx, my, mz, E).
template <int RIEMANN, int WS, int D, bool AQ = false>
__device__ __forceinline__ void flux_dir(const FxParams &P, const double WL[5], const double WR[5], double F[5], double *Aq = nullptr) {
  constexpr int in = 1 + D, it1 = 1 + (D + 1) % 3, it2 = 1 + (D + 2) % 3;
  const double wl[5] = {WL[0], WL[in], WL[it1], WL[it2], WL[4]};
  const double wr[5] = {WR[0], WR[in], WR[it1], WR[it2], WR[4]};
  double f[5];
  fx_riemann_v2<RIEMANN, WS, AQ>(P, wl, wr, f, Aq);
  F[0] = f[0];
  F[in] = f[1];
  F[it1] = f[2];
  F[it2] = f[3];
  F[4] = f[4];
}

// EXTRAS: some block of the launch has a reflecting wall [B9], gravity is on [B10] or some face carries a refinement jump
// [B12-B14]: the image cells' sign flips, the source term, the halo boxes taken from a block's own (interpolated) guard
// zones behind a jump and the capture of the jump faces' fluxes are compiled in only then
// SCAL: the plan carries passive scalars [B11] and they take the scalar pass (fx_scalar_pass.cu): every zone also leaves the
// mass flux and the advected-quantity coefficient Aq of its three low faces in P.fq for it
template <int RECON, int RIEMANN, int WS, bool FIRST, bool DTOUT, bool EXTRAS, bool SCAL = false>
__global__ void __launch_bounds__(NTHREADS) __maxnreg__(Rc<RECON>::NREG)
fx_k_stage_tma(const __grid_constant__ CUtensorMap mXm, const __grid_constant__ CUtensorMap mXx,
               const __grid_constant__ CUtensorMap mXy, const __grid_constant__ CUtensorMap mU0,
               const __grid_constant__ CUtensorMap mOut, const FxParams P, const double *__restrict__ X,
               const double *__restrict__ dx, double dt, const double *dt_dev, double beta,
               double cfl_next, double *dt_next) {  // dt_next may be dt_dev (fx_hydro_step): read at the start, written by the last CTA
  constexpr int r = Rc<RECON>::r, R = Rc<RECON>::R, W = 2 * r + 1, NP = Rc<RECON>::NP, BW = Rc<RECON>::BW;
  constexpr int NRING = Rc<RECON>::NRING;
  constexpr bool AQS = SCAL && RIEMANN != FX_RIEMANN_HLLC;  // the faces' Aq are needed (HLLC: Aq = max(F_rho, 0))
  extern __shared__ __align__(1024) unsigned char fx_smem_raw[];  // TMA destinations need 128-byte alignment
  Smem<RECON> &S = *reinterpret_cast<Smem<RECON> *>(fx_smem_raw);
  const int tid = threadIdx.x;
  const int nzb = P.n[2];  // planes per block
  const int g0 = P.gd[0], g1 = P.gd[1], g2 = P.gd[2];
  unsigned hit = 0;
  // This CTA marches through a SEGMENT: M blocks that follow one another in +z, as one column of nz = M nzb planes.
  // A block's top halo is then the next block's first planes, already on their way through the ring: they are
  // neither loaded nor converted twice, and the pipeline is filled once per segment instead of once per block.
  if (tid < FX_SEG_STRIDE) S.chain[tid] = __ldg(&P.seg[(long long)blockIdx.x * FX_SEG_STRIDE + tid]);
  __syncthreads();
  const int M = S.chain[0];
  const int nz = M * nzb;
  // where plane Z of the column (Z in [-R, nz + R)) lives: block id and padded k.  Outflow below / above the segment
  // clamps to the nearest interior plane [O1]; a reflecting wall [B9] mirrors the plane index (plane -1-m is plane m, its
  // z momentum negated by whoever converts it: the prologue below the segment, the z loop above it).
  // Z / nzb without a division: exact for Z < 2^20 / nzb, and the host only chains blocks of at most 64 planes
  const unsigned zmagic = ((1u << 20) + (unsigned)nzb - 1u) / (unsigned)nzb;
  auto zmap = [&](int Z, int &bs, int &kp) {
    int qb = Z < 0 ? -1 : (M == 1 ? (int)(Z >= nzb) : (int)(((unsigned)Z * zmagic) >> 20));
    int k = Z - qb * nzb;
    int id = S.chain[2 + qb];
    if (id < 0) {
      const bool wall = EXTRAS && id == FX_BC_REFLECT;
      // behind a refinement jump [B12]: the block's OWN guard planes, which fx_k_amr_fill has interpolated [B13]
      const bool own = EXTRAS && id <= FX_NEIGH_COARSER;
      if (qb < 0) { id = S.chain[2]; k = own ? Z : (wall ? -1 - Z : 0); } else { id = S.chain[1 + M]; k = own ? nzb + (Z - nz) : (wall ? nzb - 1 - (Z - nz) : nzb - 1); }
    }
    bs = id;
    kp = k + g2;
  };
  const bool wall_below = EXTRAS && S.chain[1] == FX_BC_REFLECT;
  const int zflip_from = (EXTRAS && S.chain[2 + M] == FX_BC_REFLECT) ? nz : 0x7fffffff;  // planes >= this carry a negated z momentum

  // ---------------------------------------------------------------- producer set-up (producer warp, lane 0)
  const bool producer = tid == NZONE_THREADS + 32;
  auto issue_X = [&](int c) {  // stage-input plane consumed at tick c: z index c + r
    int bs, kp;
    zmap(c + r, bs, kp);
    mbar_expect_tx(&S.barX[c & 1], PLANE_BYTES);
    tma_load(&S.ring[(c + r) % NRING][0][0][0], &mXm, &S.barX[c & 1], g0, g1, kp, bs);
  };
  // producer warp: the block the next halo plane is in (plane hk of block hq of the segment) and its x / y neighbours
  int hk = 0, hq = 0, hb = 0, xlo = 0, xhi = 0, ylo = 0, yhi = 0;
  auto halo_block = [&]() {
    hb = S.chain[2 + hq];
    xlo = __ldg(&P.neigh[(long long)hb * 6 + 0]);
    xhi = __ldg(&P.neigh[(long long)hb * 6 + 1]);
    ylo = __ldg(&P.neigh[(long long)hb * 6 + 2]);
    yhi = __ldg(&P.neigh[(long long)hb * 6 + 3]);
  };
  if (tid >= NZONE_THREADS + 32) halo_block();
  auto issue_H = [&]() {  // halo cells of interior plane hk of block hb, from the block's x and y neighbours
    const int b = hb, kp = hk + g2;
    mbar_expect_tx(&S.barH, 2 * 5 * NY * BW * 8 + 2 * 5 * R * NX * 8);
    // (a face with a refinement jump [B12]: the block's own guard zones behind it, interpolated by fx_k_amr_fill)
    const bool jxl = EXTRAS && xlo <= FX_NEIGH_COARSER, jxh = EXTRAS && xhi <= FX_NEIGH_COARSER;
    const bool jyl = EXTRAS && ylo <= FX_NEIGH_COARSER, jyh = EXTRAS && yhi <= FX_NEIGH_COARSER;
    tma_load(&S.Hx[0][0][0][0], &mXx, &S.barH, g0 + (xlo >= 0 ? NX - BW : (jxl ? -BW : 0)), g1, kp, xlo >= 0 ? xlo : b);
    tma_load(&S.Hx[1][0][0][0], &mXx, &S.barH, g0 + (xhi >= 0 ? 0 : (jxh ? NX : NX - BW)), g1, kp, xhi >= 0 ? xhi : b);
    tma_load(&S.Hy[0][0][0][0], &mXy, &S.barH, g0, g1 + (ylo >= 0 ? NY - R : (jyl ? -R : 0)), kp, ylo >= 0 ? ylo : b);
    tma_load(&S.Hy[1][0][0][0], &mXy, &S.barH, g0, g1 + (yhi >= 0 ? 0 : (jyh ? NY : NY - R)), kp, yhi >= 0 ? yhi : b);
  };
  auto issue_U0 = [&](int p, int b, int k) {  // plane p of the column = plane k of block b
    // completes on the barrier of tick p + 1, the tick that combines plane p: one wait per tick covers both loads
    mbar_expect_tx(&S.barX[(p + 1) & 1], PLANE_BYTES);
    tma_load(&S.U0[p & 1][0][0][0], &mU0, &S.barX[(p + 1) & 1], g0, g1, k + g2, b);
  };
  if (producer) {
    // arrivals per tick: issue_X(c) and, in the later stages, issue_U0(c - 1)
    mbar_init(&S.barX[0], FIRST ? 1 : 2); mbar_init(&S.barX[1], FIRST ? 1 : 2);
    mbar_init(&S.barH, 1);
    fence_mbar_init();
    fence_async_smem();
    issue_X(1);
    issue_H();
    if (!FIRST) issue_U0(0, S.chain[2], 0);
  }
  if (dt_dev) dt = *dt_dev;
  cta_sync();  // barriers initialised before anyone waits on them

  if (tid < NZONE_THREADS) {
    // ------------------------------------------------------------ zone threads
    const int i = tid & 15, j = tid >> 4;
    double rate = 0.0;     // DTOUT: running maximum of (|u_d| + c) / dx_d over this thread's finished zones
    double q[W][5];        // q[m] = primitives of cell c - r + m at tick c
    double qpz[5], Fz[5];  // plus-side z state of cell c-1; z flux of face c-1 (between cells c-2 and c-1)
    double Aqz = 0.0;      // AQS: Aq of that face
    int sq = 0, sk = 0;    // SCAL: plane p is plane sk of the sq-th block of the segment
    // Refinement jumps [B14]: the fluxes through a block's jump faces are stored for the flux correction (both sides of a
    // jump).  Such a block is a segment of its own (fx_hydro_plan_set_topology keeps it out of the chains), so the planes of
    // this CTA are the planes of block chain[2]; bit f of cap: face f carries a jump.
    unsigned cap = 0;
    if (EXTRAS && P.has_jumps && M == 1) {
#pragma unroll
      for (int f = 0; f < 6; ++f) cap |= (__ldg(&P.neigh[(long long)S.chain[2] * 6 + f]) <= FX_NEIGH_COARSER ? 1u : 0u) << f;
    }
    auto capture = [&](int f, int tflat, const double F[5]) {
      double *dst = P.fjump + ((long long)S.chain[2] * 6 + f) * P.nvars * (long long)P.fj_area + tflat;
#pragma unroll
      for (int v = 0; v < 5; ++v) dst[(long long)v * P.fj_area] = F[v];
    };
    {
      // prologue: cells -R .. r straight from global memory (all loads in flight together), the plus-side state
      // of cell 0 and the flux of face 0
      const long long col = (long long)(j + g1) * P.S_j + (i + g0);
      double w[2 * R][5];
#pragma unroll
      for (int m = 0; m < 2 * R; ++m) {
        int bs, kp;
        zmap(m - R, bs, kp);
        const long long a = (long long)bs * P.S_b + (long long)kp * P.S_k + col;
#pragma unroll
        for (int v = 0; v < 5; ++v) w[m][v] = X[a + v * P.S_v];
        if (m < R && wall_below) w[m][3] = -w[m][3];
      }
#pragma unroll
      for (int m = 0; m < 2 * R; ++m) {
        double u[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) u[v] = w[m][v];
        if (m >= R) {  // this block's planes 0 .. r do not come through the TMA ring: keep them there for the combine
#pragma unroll
          for (int v = 0; v < 5; ++v) S.ring[(m - R) % NRING][v][j][i] = u[v];
        }
        const unsigned h = fx_c2p_v2(P, u[0], u[1], u[2], u[3], u[4], w[m]);
        if (m >= R && m - R < nz) hit |= h;  // a zone's floor hits are counted by its owner only
      }
      double qm[5], qpm1[5];
      hit |= fx_recon_cell5<RECON>(&w[0], P.weno_eps, qm, qpm1);  // cell -1
      hit |= fx_recon_cell5<RECON>(&w[1], P.weno_eps, qm, qpz);   // cell 0
      flux_dir<RIEMANN, WS, 2, AQS>(P, qpm1, qm, Fz, &Aqz);
      if (EXTRAS && (cap & 16u)) capture(4, j * NX + i, Fz);
#pragma unroll
      for (int m = 0; m < 2 * r; ++m)
#pragma unroll
        for (int v = 0; v < 5; ++v) q[m][v] = w[m + 2][v];
    }

#pragma unroll
    for (int v = 0; v < 5; ++v) S.P[v][j + R][i + R] = q[r - 1][v];  // plane 0
    cta_sync();  // A0: plane 0 and its halo (edge warp) visible

#pragma unroll 1
    for (int c = 1; c <= nz; ++c) {
      const int p = c - 1;  // plane of the in-plane work; its primitives are q[r-1]
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
      cta_sync();  // B: plus-side states visible; this tick's TMA planes have landed (the producer waited for them)
      {  // new cell of the z window.  No mbarrier poll here: the producer observed the completion of this tick's loads
         // before it arrived at barrier B, and the barrier orders that observation before these reads
        double u[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) u[v] = S.ring[(c + r) % NRING][v][j][i];
        if (EXTRAS && c + r >= zflip_from) u[3] = -u[3];  // image planes above a reflecting wall
        const unsigned h = fx_c2p_v2(P, u[0], u[1], u[2], u[3], u[4], q[2 * r]);
        if (c + r < nz) hit |= h;
      }
      // z: reconstruct cell c, flux of face c (between cells c-1 and c)
      double Fz_new[5], Aqz_new = 0.0, Aqx = 0.0, Aqy = 0.0;
      {
        double qmz[5], qpz_new[5];
        hit |= fx_recon_cell5<RECON>(q, P.weno_eps, qmz, qpz_new);
        flux_dir<RIEMANN, WS, 2, AQS>(P, qpz, qmz, Fz_new, &Aqz_new);
#pragma unroll
        for (int v = 0; v < 5; ++v) qpz[v] = qpz_new[v];
      }
      double Fx[5], Fy[5];
      {
        double WL[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) WL[v] = S.Lx[v][j][i];
        flux_dir<RIEMANN, WS, 0, AQS>(P, WL, qmx, Fx, &Aqx);
#pragma unroll
        for (int v = 0; v < 5; ++v) S.Lx[v][j][i] = Fx[v];  // in place: only this thread read the state
#pragma unroll
        for (int v = 0; v < 5; ++v) WL[v] = S.Ly[v][j][i];
        flux_dir<RIEMANN, WS, 1, AQS>(P, WL, qmy, Fy, &Aqy);
#pragma unroll
        for (int v = 0; v < 5; ++v) S.Ly[v][j][i] = Fy[v];
      }
      if (c < nz) {  // primitives of plane p + 1 (cell c of the window): nobody reads P between barriers B and C
#pragma unroll
        for (int v = 0; v < 5; ++v) S.P[v][j + R][i + R] = q[r][v];
      }
      if (SCAL) {  // mass flux and Aq of the zone's low x, y and z faces, for the scalar pass: fq[6][zone], zones block by block
        const long long zone = (((long long)S.chain[2 + sq] * nzb + sk) * NY + j) * NX + i;
        const long long nzt = (long long)P.nblocks * nzb * (NY * NX);
        P.fq[zone] = Fx[0];
        P.fq[2 * nzt + zone] = Fy[0];
        P.fq[4 * nzt + zone] = Fz[0];
        if (RIEMANN != FX_RIEMANN_HLLC) {  // HLLC: Aq = max(F_rho, 0), the pass forms it itself
          P.fq[nzt + zone] = Aqx;
          P.fq[3 * nzt + zone] = Aqy;
          P.fq[5 * nzt + zone] = Aqz;
        }
        Aqz = Aqz_new;
        if (++sk == nzb) { sk = 0; ++sq; }
      }
      cta_sync();  // C: fluxes and the next plane's primitives visible
      if (EXTRAS && cap) {
        if ((cap & 1u) && i == 0) capture(0, p * NY + j, Fx);
        if ((cap & 4u) && j == 0) capture(2, p * NX + i, Fy);
        if ((cap & 32u) && c == nz) capture(5, j * NX + i, Fz_new);
      }
      {
        // out = [U0 + beta (X - U0)] - sum_d (beta dt/dx_d) (F_d+ - F_d-)
        const double rx = S.rd[0], ry = S.rd[1], rz = S.rd[2];
        int hmax = 0;
        double res5[5], xs5[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) {
          const double dFx = S.Lx[v][j][i + 1] - Fx[v];
          const double dFy = S.Ly[v][j + 1][i] - Fy[v];
          const double dFz = Fz_new[v] - Fz[v];
          const double xs = S.ring[p % NRING][v][j][i];  // the zone's stage input; in the first stage it is U0
          const double u0 = FIRST ? xs : S.U0[p & 1][v][j][i];
          const double a = FIRST ? u0 : fma(beta, xs - u0, u0);
          const double res = fma(-rz, dFz, fma(-ry, dFy, fma(-rx, dFx, a)));
          if (!EXTRAS) {  // (the plain kernel keeps its one-pass form: splitting the loop costs it 2 %)
            S.Out[v][j][i] = res;
            if (!DTOUT) hmax = max(hmax, __double2hiint(res) & 0x7fffffff);
          }
          res5[v] = res;
          if (EXTRAS) xs5[v] = xs;
          Fz[v] = Fz_new[v];
        }
        if (EXTRAS) {
          if (P.grav_on) {  // + beta dt (0, rho g, g . m) of the stage input's own zone [B10]
            const double bdt = (FIRST ? 1.0 : beta) * dt;
            res5[4] = fma(bdt, fma(P.grav[2], xs5[3], fma(P.grav[1], xs5[2], P.grav[0] * xs5[1])), res5[4]);
#pragma unroll
            for (int d = 0; d < 3; ++d) res5[1 + d] = fma(bdt * P.grav[d], xs5[0], res5[1 + d]);
          }
#pragma unroll
          for (int v = 0; v < 5; ++v) {
            S.Out[v][j][i] = res5[v];
            if (!DTOUT) hmax = max(hmax, __double2hiint(res5[v]) & 0x7fffffff);
          }
        }
        if (!DTOUT && hmax >= 0x7ff00000) hit |= FX_STATUS_NONFINITE;
        if (DTOUT) {  // a7 on the finished zone: (|u_d| + c) / dx_d, folded into a running maximum [O7]
          double w[5], ir;
          // (a non-finite result reaches the pressure or the density: the conversion's own test stands in for hmax)
          hit |= fx_c2p_v2(P, res5[0], res5[1], res5[2], res5[3], res5[4], w, &ir) & FX_STATUS_NONFINITE;
          const double cs = fx_sqrt3(P.gamma * w[4] * ir);
          // (compare-selects a > b ? a : b with the running value second: a NaN candidate loses, and the state it came
          // from is already flagged)
          const double r01 = fx_max_sel((fabs(w[1]) + cs) * S.idx[0], (fabs(w[2]) + cs) * S.idx[1]);
          rate = fx_max_sel(fx_max_sel((fabs(w[3]) + cs) * S.idx[2], r01), rate);
        }
        fence_async_smem();  // the TMA store reads Out through the async proxy
      }
#pragma unroll
      for (int m = 0; m < 2 * r; ++m)
#pragma unroll
        for (int v = 0; v < 5; ++v) q[m][v] = q[m + 1][v];
    }
    if (SCAL) {  // the segment's top face has no owned block above it: its mass flux (the last one carried) goes where the
                 // scalar pass looks for it.  (Behind the loop: inside it the few registers this needs spilled loop values.)
      const int ab = S.chain[2 + M];
      if (ab < 0 || ab >= P.nown) {
        const long long t = ((2 * P.nblocks + S.chain[1 + M]) * (long long)P.fqb_area) + j * NX + i;
        P.fqb[t] = Fz[0];
        if (AQS) P.fqb[t + 3 * P.nblocks * (long long)P.fqb_area] = Aqz;
      }
    }
    if (DTOUT) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) rate = fmax(rate, __shfl_xor_sync(0xffffffffu, rate, o));
      if ((tid & 31) == 0) S.wmax[tid >> 5] = rate;
    }
    cta_sync();  // D: the last plane is in Out
  } else if (tid < NZONE_THREADS + 32) {
    // ------------------------------------------------------------ edge warp
    const int lane = tid - NZONE_THREADS;
    const bool isx = lane >= 16;
    const int m = lane & 15;
    double *Pf = &S.P[0][0][0];
    constexpr int NPS = NP + 1;
    const int pd = isx ? 1 : NPS, pt = isx ? NPS : 1;  // smem strides of P along direction / transverse
    double *Lf = isx ? &S.Lx[0][0][0] : &S.Ly[0][0][0];
    const int ld = isx ? 1 : NX, lt = isx ? (NX + 1) : 1;  // strides of L along direction / transverse
    constexpr int LV = NY * (NX + 1);                       // per-variable size of the L arrays (272)
    cta_sync();  // A0
    int pk = 0, pq = 0, pb = S.chain[2];  // plane p is plane pk of block pb, the pq-th of the segment
    // the high x / y face of this lane's row / column carries a refinement jump: its flux is stored [B14]
    const int ef = isx ? 1 : 3;
    const bool ecap = EXTRAS && P.has_jumps && M == 1 && __ldg(&P.neigh[(long long)pb * 6 + ef]) <= FX_NEIGH_COARSER;
    // SCAL: no owned same-level block behind that face (a physical boundary, a ghost block): the scalar pass takes the face's
    // mass flux (and Aq) from P.fqb, where this warp leaves it -- nobody else computes it
    auto no_owner = [&](int blk) { const int h = __ldg(&P.neigh[(long long)blk * 6 + ef]); return h < 0 || h >= P.nown; };
    bool ebnd = SCAL && no_owner(pb);

#pragma unroll 1
    for (int c = 1; c <= nz; ++c) {
      double qm16[5];
      {
        double st[W][5], qm[5], qp[5];
        // cell -1: padded positions 0 .. 2r along the direction (cell -1 sits at R-1 = r)
#pragma unroll
        for (int mm = 0; mm < W; ++mm)
#pragma unroll
          for (int v = 0; v < 5; ++v) st[mm][v] = Pf[v * NP * NPS + mm * pd + (m + R) * pt];
        hit |= fx_recon_cell5<RECON>(st, P.weno_eps, qm, qp);
#pragma unroll
        for (int v = 0; v < 5; ++v) Lf[v * LV + 0 * ld + m * lt] = qp[v];
        // cell 16: padded positions 16+R-r .. 16+R+r
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
        double f[5], Aqe = 0.0;
        fx_riemann_v2<RIEMANN, WS, AQS>(P, wl, wr, f, &Aqe);
        if (SCAL && ebnd) {
          const long long t = (((isx ? 0 : 1) * P.nblocks + pb) * (long long)P.fqb_area) + pk * NX + m;
          P.fqb[t] = f[0];
          if (AQS) P.fqb[t + 3 * P.nblocks * (long long)P.fqb_area] = Aqe;
        }
        double F[5];
        F[0] = f[0];
        F[1] = isx ? f[1] : f[3];
        F[2] = isx ? f[2] : f[1];
        F[3] = isx ? f[3] : f[2];
        F[4] = f[4];
#pragma unroll
        for (int v = 0; v < 5; ++v) Lf[v * LV + NX * ld + m * lt] = F[v];
        if (EXTRAS && ecap) {
          double *dst = P.fjump + ((long long)pb * 6 + ef) * P.nvars * (long long)P.fj_area + (c - 1) * NX + m;
#pragma unroll
          for (int v = 0; v < 5; ++v) dst[(long long)v * P.fj_area] = F[v];
        }
      }
      if (pk == 0 && lane < 3) {
        // a block's first plane: the combines of the block below ended before barrier B, this tick's starts after C
        const double dxd = __ldg(&dx[(long long)pb * 3 + lane]);
        S.rd[lane] = (FIRST ? 1.0 : beta) * dt / dxd;
        if (DTOUT) S.idx[lane] = 1.0 / dxd;
      }
      if (++pk == nzb) {
        pk = 0;
        ++pq;
        pb = S.chain[2 + pq];
        if (SCAL && c < nz) ebnd = no_owner(pb);
      }
      cta_sync();  // C
    }
    cta_sync();  // D
  } else {
    // ------------------------------------------------------------ producer warp: lane 0 issues the bulk copies, all
    // lanes convert the halo cells (lanes 0..15 the y edges of column m, lanes 16..31 the x edges of row m)
    const int lane = tid - NZONE_THREADS - 32;
    const bool isx = lane >= 16;
    const int m = lane & 15;
    double *Pf = &S.P[0][0][0];
    constexpr int NPS = NP + 1;
    const int pd = isx ? 1 : NPS, pt = isx ? NPS : 1;  // smem strides of P along direction / transverse
    // raw halo cell t of this lane's row / column: Hx[s][side][v][m][ix], Hy[s][side][v][iy][m]
    constexpr int HXV = NY * BW, HYV = R * NX;  // per-variable sizes
    int nlo = isx ? xlo : ylo, nhi = isx ? xhi : yhi;  // this lane's pair of neighbours of the block the halo plane is in
    auto halo_off = [&](int t, bool high) -> int {
      int idx;  // cell index inside the box
      // a neighbour's cells; at a reflecting wall this block's own cells in mirrored order [B9]; at outflow its edge cell
      // (the guard zones behind a refinement jump lie in the box like a neighbour's cells)
      const bool clo = nlo >= 0 || (EXTRAS && nlo <= FX_NEIGH_COARSER), chi = nhi >= 0 || (EXTRAS && nhi <= FX_NEIGH_COARSER);
      if (isx) idx = high ? (chi ? t : ((EXTRAS && nhi == FX_BC_REFLECT) ? BW - 1 - t : BW - 1)) : (clo ? BW - R + t : ((EXTRAS && nlo == FX_BC_REFLECT) ? R - 1 - t : 0));
      else idx = high ? (chi ? t : ((EXTRAS && nhi == FX_BC_REFLECT) ? R - 1 - t : R - 1)) : (clo ? t : ((EXTRAS && nlo == FX_BC_REFLECT) ? R - 1 - t : 0));
      return isx ? ((high ? 5 * HXV : 0) + m * BW + idx) : ((high ? 5 * HYV : 0) + idx * NX + m);
    };
    int hoff[2 * R];
#pragma unroll
    for (int t = 0; t < 2 * R; ++t) hoff[t] = halo_off(t % R, t >= R);
    const int hv = isx ? HXV : HYV;

    auto halo_plane = [&](int pl) {  // primitives of the halo cells of plane pl into P (called for pl = 0, 1, 2, ... in turn)
      mbar_wait(&S.barH, pl & 1);
      const double *Hf = isx ? &S.Hx[0][0][0][0] : &S.Hy[0][0][0][0];
#pragma unroll
      for (int t = 0; t < 2 * R; ++t) {
        double u[5], w[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) u[v] = Hf[hoff[t] + v * hv];
        if (EXTRAS && (t < R ? nlo : nhi) == FX_BC_REFLECT) {  // image cells behind a wall: normal momentum negated
          if (isx) u[1] = -u[1]; else u[2] = -u[2];
        }
        fx_c2p_v2(P, u[0], u[1], u[2], u[3], u[4], w);
        const int pos = (t < R) ? t : (NX + t);  // padded position along the edge direction
#pragma unroll
        for (int v = 0; v < 5; ++v) Pf[v * NP * NPS + pos * pd + (m + R) * pt] = w[v];
      }
      __syncwarp();  // every lane has read its raw halo cells: the (single) slot can take the next plane's
      if (pl + 1 < nz) {
        if (++hk == nzb) {  // a new block: where its halo cells sit inside the boxes depends on which neighbours exist
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
    int pk = 0, pq = 0, pb = S.chain[2], pb_prev = pb;  // plane p is plane pk of block pb, the pq-th of the segment
#pragma unroll 1
    for (int c = 1; c <= nz; ++c) {
      const int p = c - 1;
      // this tick's stage-input plane (requested two ticks ago) and U0 plane (one tick ago): the zone threads read them
      // after barrier B without polling the mbarrier themselves
      mbar_wait(&S.barX[c & 1], ((c - 1) >> 1) & 1);
      cta_sync();  // B
      if (lane == 0) {
        // every slot whose last reader finished before barrier B of this tick is free again: the ring slot of plane p - 1
        // (combined in the phase that just ended) takes the plane of the next tick
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
      if (c < nz) halo_plane(c);  // halo of plane p + 1: nobody reads P between barriers B and C
      if (lane == 0 && p >= 1) tma_wait_read();  // Out is free for the combine after barrier C
      cta_sync();  // C
    }
    cta_sync();  // D
    if (lane == 0) {
      tma_store(&mOut, &S.Out[0][0][0], g0, g1, nzb - 1 + g2, S.chain[1 + M]);
      tma_commit();
      if (DTOUT) {
        // CTA maximum -> scratch word (non-negative doubles order like unsigned integers); the last CTA to finish
        // writes the next time step cfl / max and re-arms the scratch words, as fx_k_compute_dt does
        double mx = S.wmax[0];
#pragma unroll
        for (int w8 = 1; w8 < 8; ++w8) mx = fmax(mx, S.wmax[w8]);
        if (EXTRAS && P.dt_defer) {
          // fused AMR path: the flux correction still changes the blocks with a finer neighbour (each a segment of its own);
          // the others' maximum waits in the scratch word for fx_launch_compute_dt_corrected, which writes the time step
          bool corr = false;
          for (int f = 0; f < 6; ++f) corr |= __ldg(&P.neigh[(long long)S.chain[2] * 6 + f]) == FX_NEIGH_FINER;
          if (!corr) atomicMax(&P.scratch[FX_SCR_DTBITS], (unsigned long long)__double_as_longlong(mx));
        } else {
          atomicMax(&P.scratch[FX_SCR_DTBITS], (unsigned long long)__double_as_longlong(mx));
          __threadfence();
          const unsigned long long done = atomicAdd(&P.scratch[FX_SCR_COUNTER], 1ull);
          if (done == (unsigned long long)P.nseg_all - 1) {  // the stage's last CTA (the stage may be launched in two parts)
            __threadfence();
            const unsigned long long bits = atomicExch(&P.scratch[FX_SCR_DTBITS], 0ull);
            P.scratch[FX_SCR_COUNTER] = 0ull;
            *dt_next = cfl_next / __longlong_as_double((long long)bits);
          }
        }
      }
      tma_wait_all();
    }
  }
  if (hit) fx_note(P, hit);
}

// ------------------------------------------------------------------ host side: tensor maps and launch
template <int RECON, int RIEMANN, int WS, bool FIRST, bool DTOUT, bool EXTRAS, bool SCAL = false>
int launch(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt, const double *dt_dev,
           double beta, double cfl_next, double *dt_next, cudaStream_t st) {
  constexpr int R = Rc<RECON>::R, BW = Rc<RECON>::BW;
  CUtensorMap mXm, mXx, mXy, mU0, mOut;
  int rc;
  if ((rc = make_map(&mXm, P, X, NX, NY))) return rc;
  if ((rc = make_map(&mXx, P, X, BW, NY))) return rc;
  if ((rc = make_map(&mXy, P, X, NX, R))) return rc;
  if ((rc = make_map(&mU0, P, U0, NX, NY))) return rc;
  if ((rc = make_map(&mOut, P, out, NX, NY))) return rc;
  auto kern = fx_k_stage_tma<RECON, RIEMANN, WS, FIRST, DTOUT, EXTRAS, SCAL>;
  const int smem = (int)sizeof(Smem<RECON>);
  // (per device and context, and cheap: set on every launch rather than cached per process)
  FX_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  kern<<<(unsigned)P.nseg, NTHREADS, smem, st>>>(mXm, mXx, mXy, mU0, mOut, P, X, dx, dt, dt_dev, beta, cfl_next, dt_next);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    cudaFuncAttributes a;
    memset(&a, 0, sizeof(a));
    cudaFuncGetAttributes(&a, kern);
    cudaGetLastError();
    return fx_fail(FX_ERR_CUDA, "stage_tma launch: %s (regs %d, threads %d of max %d, smem dynamic %d of max %d + static %d)",
                   cudaGetErrorString(e), a.numRegs, NTHREADS, a.maxThreadsPerBlock, smem, a.maxDynamicSharedSizeBytes,
                   (int)a.sharedSizeBytes);
  }
  return FX_OK;
}

template <int RECON, int RIEMANN, int WS>
int launch_ws(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt, const double *dt_dev,
              double beta, int first, double cfl_next, double *dt_next, cudaStream_t st) {
  if constexpr (RECON == FX_RECON_PLM_MINMOD) {
    if (P.nvars > 5) {  // with passive scalars: also leave the faces' mass flux and Aq for the scalar pass
      if (P.walls || P.grav_on || P.has_jumps) {
        if (first) return launch<RECON, RIEMANN, WS, true, false, true, true>(P, X, U0, out, dx, dt, dt_dev, beta, 0.0, nullptr, st);
        if (dt_next) return launch<RECON, RIEMANN, WS, false, true, true, true>(P, X, U0, out, dx, dt, dt_dev, beta, cfl_next, dt_next, st);
        return launch<RECON, RIEMANN, WS, false, false, true, true>(P, X, U0, out, dx, dt, dt_dev, beta, 0.0, nullptr, st);
      }
      if (first) return launch<RECON, RIEMANN, WS, true, false, false, true>(P, X, U0, out, dx, dt, dt_dev, beta, 0.0, nullptr, st);
      if (dt_next) return launch<RECON, RIEMANN, WS, false, true, false, true>(P, X, U0, out, dx, dt, dt_dev, beta, cfl_next, dt_next, st);
      return launch<RECON, RIEMANN, WS, false, false, false, true>(P, X, U0, out, dx, dt, dt_dev, beta, 0.0, nullptr, st);
    }
  }
  if (P.walls || P.grav_on || P.has_jumps) {  // (the kernel variant that also knows the refinement-jump faces [B12-B14])
    if (first) return launch<RECON, RIEMANN, WS, true, false, true>(P, X, U0, out, dx, dt, dt_dev, beta, 0.0, nullptr, st);
    if (dt_next) return launch<RECON, RIEMANN, WS, false, true, true>(P, X, U0, out, dx, dt, dt_dev, beta, cfl_next, dt_next, st);
    return launch<RECON, RIEMANN, WS, false, false, true>(P, X, U0, out, dx, dt, dt_dev, beta, 0.0, nullptr, st);
  }
  if (first) return launch<RECON, RIEMANN, WS, true, false, false>(P, X, U0, out, dx, dt, dt_dev, beta, 0.0, nullptr, st);
  if (dt_next) return launch<RECON, RIEMANN, WS, false, true, false>(P, X, U0, out, dx, dt, dt_dev, beta, cfl_next, dt_next, st);
  return launch<RECON, RIEMANN, WS, false, false, false>(P, X, U0, out, dx, dt, dt_dev, beta, 0.0, nullptr, st);
}

template <int RECON, int RIEMANN>
int launch_rr(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt, const double *dt_dev,
              double beta, int first, double cfl_next, double *dt_next, cudaStream_t st) {
  return P.wavespeed == 0 ? launch_ws<RECON, RIEMANN, 0>(P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st)
                          : launch_ws<RECON, RIEMANN, 1>(P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st);
}

}  // namespace fxt

bool fx_stage_tma_supported(const FxParams &P) {
  const int R = P.recon == FX_RECON_WENO5 ? 3 : 2;
  // TMA: global strides must be multiples of 16 bytes (S_j even), every box must start on a 16-byte boundary (guard
  // depth even: measured, a box starting at an odd element faults), the arrays 16-byte aligned (checked at launch)
  return P.n[0] == fxt::NX && P.n[1] == fxt::NY && P.n[2] >= R && P.active[2] && P.gd[0] >= R && (P.S_j % 2) == 0 &&
         (P.gd[0] % 2) == 0 && P.nblocks <= 0x7fffffffLL && P.seg != nullptr && P.nseg > 0;
}

// dt_next != nullptr (a later stage only): also form cfl_next * min dx/(|u|+c) of the finished state and write it there.
int fx_launch_stage_tma(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt,
                        const double *dt_dev, double beta, int first, double cfl_next, double *dt_next, cudaStream_t st) {
  if (!fx_stage_tma_supported(P)) return fx_fail(FX_ERR_UNSUPPORTED, "TMA stage kernel: block shape not supported");
  if (P.nvars > 5 && !fx_scalar_pass_supported(P)) return fx_fail(FX_ERR_UNSUPPORTED, "TMA stage kernel: passive scalars need the scalar pass");
  if (P.nblocks == 0) return FX_OK;
  if (first && X != U0) return fx_fail(FX_ERR_INVALID_ARG, "TMA stage kernel: the first stage takes U0 from its stage input (X must be U0)");
  if (((uintptr_t)X | (uintptr_t)U0 | (uintptr_t)out) & 15)
    return fx_fail(FX_ERR_INVALID_ARG, "TMA stage kernel: state arrays must be 16-byte aligned");
  if (P.recon == FX_RECON_PLM_MINMOD) {
    if (P.riemann == FX_RIEMANN_HLLE) return fxt::launch_rr<FX_RECON_PLM_MINMOD, FX_RIEMANN_HLLE>(P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st);
    return fxt::launch_rr<FX_RECON_PLM_MINMOD, FX_RIEMANN_HLLC>(P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st);
  }
  if (P.riemann == FX_RIEMANN_HLLE) return fxt::launch_rr<FX_RECON_WENO5, FX_RIEMANN_HLLE>(P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st);
  return fxt::launch_rr<FX_RECON_WENO5, FX_RIEMANN_HLLC>(P, X, U0, out, dx, dt, dt_dev, beta, first, cfl_next, dt_next, st);
}
