// fx_tile.cu -- per-stage kernel for blocks whose padded zones fit in shared memory (8^3 blocks, 2-D and 1-D blocks):
// K1 (gather) + K2 + K3 in one launch, one CTA per block.
//
// The fused TMA kernel (fx_stage_tma.cu) covers 16 x 16 cross-sections; every other shape used to run the generic
// zone kernel, which fills the guard cells in a pass of its own and then, per zone, converts 24 cells, reconstructs 12
// face states and solves 6 Riemann problems from global memory.  Here a CTA
//   1. gathers the zones of its block and of the R-deep face slabs around it through the neighbour table (no guard cell
//      in HBM is read or written; outflow clamps, walls mirror and negate), converts each ONCE to primitives and keeps
//      them in shared memory W[5][(n + 2R)^3] (8^3 blocks with PLM: 112 KB with the flux and accumulator arrays, so
//      two CTAs share an SM);
//   2. per active direction: one thread per face reconstructs the two face states from W and solves ONE Riemann problem
//      into a shared flux array; after a barrier every interior zone adds (dt/dx_d)(F+ - F-) to its accumulator in
//      shared memory (order x, y, z as in O5);
//   3. combines: out = U0 + beta((X - U0) - S) (+ the gravity source), coalesced along x.
// Arithmetic is the lean set of fx_physics.cuh (the fused kernel's), so the two paths agree to rounding.
#include "fx_physics.cuh"

namespace fxtile {


struct Geo {
  int e[3];          // extents of the primitive tile: n_d + 2R in active dimensions (R = reach of the reconstruction)
  int ntile;         // e0 e1 e2
  int faces_max;     // largest (n_d + 1) n_d1 n_d2 over the active directions
  int nint;          // interior zones per block
  size_t smem;       // bytes: W[5][ntile] + F[5][faces_max] + Sacc[5][nint]
};

static Geo geometry(const FxParams &P) {
  Geo g;
  const int R = P.recon == FX_RECON_WENO5 ? 3 : 2;
  g.nint = P.n[0] * P.n[1] * P.n[2];
  g.faces_max = 0;
  g.ntile = 1;
  for (int d = 0; d < 3; ++d) {
    g.e[d] = P.active[d] ? P.n[d] + 2 * R : 1;
    g.ntile *= g.e[d];
    if (!P.active[d]) continue;
    const int f = (P.n[d] + 1) * P.n[(d + 1) % 3] * P.n[(d + 2) % 3];
    if (f > g.faces_max) g.faces_max = f;
  }
  g.smem = sizeof(double) * 5 * ((size_t)g.ntile + (size_t)g.faces_max + (size_t)g.nint);
  return g;
}

// x / d for 0 <= x < 2^15 and 1 <= d <= 2^10 through a float reciprocal: (x + 0.5) / d is at least 0.5/d away from an
// integer and the float error is below x 2^-22, so truncation gives the exact quotient (an integer division is ~20
// instructions, and index arithmetic was a third of this kernel's instructions)
struct Div {
  int d;
  float inv;
  __host__ __device__ Div() : d(1), inv(1.0f) {}
  __host__ __device__ explicit Div(int dd) : d(dd), inv(1.0f / (float)dd) {}
  __device__ __forceinline__ int quot(int x) const { return __float2int_rz(((float)x + 0.5f) * inv); }
  __device__ __forceinline__ void divmod(int x, int &q, int &rem) const { q = quot(x); rem = x - q * d; }
};

struct Tile {  // what the direction passes need, in registers
  double *Wp, *Ff, *Sa;
  int ntile, faces_max, nint;
  int e0, e1;        // tile extents in x and y
  int n[3];
  int off[3];        // tile coordinate of interior zone 0 in each dimension (R if active, else 0)
  Div dn0, dn1;      // divisors n0, n1 (interior decode)
};

// Direction D (compile-time): one Riemann solve per face into Ff, then S += (dt/dx_D)(F+ - F-) for every interior zone.
template <int RECON, int RIEMANN, int WS, int NT, int D>
__device__ __forceinline__ unsigned tile_direction(const FxParams &P, const Tile &T, double rd, int tid) {
  constexpr int r = (RECON == FX_RECON_PLM_MINMOD) ? 1 : 2, W5 = 2 * r + 1;
  constexpr int d1 = (D + 1) % 3, d2 = (D + 2) % 3;      // momentum rotation of the face frame (as in the fused kernel)
  constexpr int ta = D == 0 ? 1 : 0, tb = D == 2 ? 1 : 2;  // the two transverse dimensions, ascending
  unsigned hit = 0;
  const int nf = T.n[D] + 1, nta = T.n[ta], nfaces = nf * nta * T.n[tb];
  const int sd = D == 0 ? 1 : (D == 1 ? T.e0 : T.e0 * T.e1);
  // face order: x runs fastest in every direction (for D = 0 that is the face's own coordinate), so that a warp reads
  // W along rows; fs = distance between the two faces of a zone in that order
  const int fs = D == 0 ? 1 : nta;
  const Div dnf(nf), dnta(nta);
  for (int f = tid; f < nfaces; f += NT) {
    int fd, ca, cb, t;
    if (D == 0) { dnf.divmod(f, t, fd); dnta.divmod(t, cb, ca); }
    else { dnta.divmod(f, t, ca); dnf.divmod(t, cb, fd); }
    int cc[3];
    cc[D] = T.off[D] + fd;  // the cell on the plus side of the face
    cc[ta] = T.off[ta] + ca;
    cc[tb] = T.off[tb] + cb;
    const int zR = cc[0] + T.e0 * (cc[1] + T.e1 * cc[2]), zL = zR - sd;
    double stL[W5][5], stR[W5][5];
#pragma unroll
    for (int m = 0; m < W5; ++m)
#pragma unroll
      for (int v = 0; v < 5; ++v) {
        stL[m][v] = T.Wp[v * T.ntile + zL + (m - r) * sd];
        stR[m][v] = T.Wp[v * T.ntile + zR + (m - r) * sd];
      }
    double qm[5], qpL[5], qmR[5], qp[5];
    hit |= fx_recon_cell5<RECON>(stL, P.weno_eps, qm, qpL);  // plus-side state of the left cell
    hit |= fx_recon_cell5<RECON>(stR, P.weno_eps, qmR, qp);  // minus-side state of the right cell
    constexpr int in = 1 + D, it1 = 1 + d1, it2 = 1 + d2;
    const double wl[5] = {qpL[0], qpL[in], qpL[it1], qpL[it2], qpL[4]};
    const double wr[5] = {qmR[0], qmR[in], qmR[it1], qmR[it2], qmR[4]};
    double fl[5];
    fx_riemann_v2<RIEMANN, WS>(P, wl, wr, fl);
    const double sum = fl[0] + fl[1] + fl[2] + fl[3] + fl[4];
    if (fx_hi_nonfinite(__double2hiint(sum))) hit |= FX_STATUS_NONFINITE;
    T.Ff[0 * T.faces_max + f] = fl[0];
    T.Ff[in * T.faces_max + f] = fl[1];
    T.Ff[it1 * T.faces_max + f] = fl[2];
    T.Ff[it2 * T.faces_max + f] = fl[3];
    T.Ff[4 * T.faces_max + f] = fl[4];
  }
  __syncthreads();
  for (int e = tid; e < T.nint; e += NT) {
    int ci[3], t;
    T.dn0.divmod(e, t, ci[0]);
    T.dn1.divmod(t, ci[2], ci[1]);
    const int f = D == 0 ? ci[0] + nf * (ci[ta] + nta * ci[tb]) : ci[ta] + nta * (ci[D] + nf * ci[tb]);
#pragma unroll
    for (int v = 0; v < 5; ++v) T.Sa[v * T.nint + e] += rd * (T.Ff[v * T.faces_max + f + fs] - T.Ff[v * T.faces_max + f]);
  }
  __syncthreads();
  return hit;
}

// MINB: resident CTAs per SM the register allocation aims at (4 for tiles of a few hundred zones, whose shared memory
// would allow it; 1 otherwise: shared memory limits those to one or two CTAs anyway)
template <int RECON, int RIEMANN, int WS, int NT, int MINB>
__global__ void __launch_bounds__(NT, MINB) fx_k_stage_tile(const FxParams P, const double *__restrict__ X, const double *U0,
                                                      double *out, const double *__restrict__ dx, double dt,
                                                      const double *__restrict__ dt_dev, double beta, int first,
                                                      int ntile, int faces_max, int nint) {
  constexpr int R = (RECON == FX_RECON_PLM_MINMOD) ? 2 : 3;
  extern __shared__ __align__(16) unsigned char fx_tile_smem[];
  Tile T;
  T.Wp = reinterpret_cast<double *>(fx_tile_smem);  // W[v][zone of the tile]
  T.Ff = T.Wp + 5 * ntile;                           // F[v][face]
  T.Sa = T.Ff + 5 * faces_max;                       // S[v][interior zone]
  T.ntile = ntile; T.faces_max = faces_max; T.nint = nint;
  const long long b = blockIdx.x;
  const int tid = threadIdx.x;
  if (dt_dev) dt = *dt_dev;
  unsigned hit = 0;
  int e2;
  {
    T.n[0] = P.n[0]; T.n[1] = P.n[1]; T.n[2] = P.n[2];
    T.off[0] = P.active[0] ? R : 0; T.off[1] = P.active[1] ? R : 0; T.off[2] = P.active[2] ? R : 0;
    T.e0 = T.n[0] + 2 * T.off[0]; T.e1 = T.n[1] + 2 * T.off[1]; e2 = T.n[2] + 2 * T.off[2];
    T.dn0 = Div(T.n[0]); T.dn1 = Div(T.n[1]);
  }
  const Div de0(T.e0), de1(T.e1);

  // ---- 1. gather + cons -> prim, once per zone of the block and of its R-deep face slabs
  // Pass A: every zone's five conserved values travel global -> shared by cp.async (no registers: all of a thread's
  // loads, up to 60, are in flight together -- the gather is latency-bound); 5 bits per zone remember what pass B needs.
  unsigned long long tag = 0;  // per zone of this thread: bit 0-1 = coordinates outside the interior (3 = skip), 2-4 = flip
  {
    int q = 0;
    for (int z = tid; z < ntile; z += NT, ++q) {
      int t, t0, t1, t2;
      de0.divmod(z, t, t0);
      de1.divmod(t, t2, t1);
      // how many coordinates lie outside the interior box: 1-D stencils never look at edge or corner zones
      const int outside = (t0 < T.off[0] || t0 >= T.off[0] + T.n[0]) + (t1 < T.off[1] || t1 >= T.off[1] + T.n[1]) +
                          (t2 < T.off[2] || t2 >= T.off[2] + T.n[2]);
      if (outside > 1) {
        tag |= 3ull << (5 * q);
        continue;
      }
      unsigned flip;
      const long long s = fx_guard_source(P, b, t0 - T.off[0] + P.gd[0], t1 - T.off[1] + P.gd[1], t2 - T.off[2] + P.gd[2], flip);
      tag |= (unsigned long long)(outside | (flip << 2)) << (5 * q);
#pragma unroll
      for (int v = 0; v < 5; ++v) {
        const unsigned dst = (unsigned)__cvta_generic_to_shared(&T.Wp[v * ntile + z]);
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(X + v * P.S_v + s) : "memory");
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
    asm volatile("cp.async.wait_group 0;" ::: "memory");
  }
  // Pass B: each thread converts the zones it fetched, in place
  {
    int q = 0;
    for (int z = tid; z < ntile; z += NT, ++q) {
      const unsigned tg = (unsigned)(tag >> (5 * q)) & 31u;
      if ((tg & 3u) == 3u) continue;
      double u[5], w[5];
#pragma unroll
      for (int v = 0; v < 5; ++v) u[v] = T.Wp[v * ntile + z];
      if (tg & 4u) u[1] = -u[1];
      if (tg & 8u) u[2] = -u[2];
      if (tg & 16u) u[3] = -u[3];
      const unsigned h = fx_c2p_v2(P, u[0], u[1], u[2], u[3], u[4], w);
      if ((tg & 3u) == 0u) hit |= h;  // floors and non-finite states are counted where a zone is owned
#pragma unroll
      for (int v = 0; v < 5; ++v) T.Wp[v * ntile + z] = w[v];
    }
  }
  (void)e2;
  for (int e = tid; e < 5 * nint; e += NT) T.Sa[e] = 0.0;
  __syncthreads();

  // ---- 2. per direction (order x, y, z [O5]): one Riemann solve per face, then the divergence
  if (P.active[0]) hit |= tile_direction<RECON, RIEMANN, WS, NT, 0>(P, T, dt / __ldg(&dx[b * 3 + 0]), tid);
  if (P.active[1]) hit |= tile_direction<RECON, RIEMANN, WS, NT, 1>(P, T, dt / __ldg(&dx[b * 3 + 1]), tid);
  if (P.active[2]) hit |= tile_direction<RECON, RIEMANN, WS, NT, 2>(P, T, dt / __ldg(&dx[b * 3 + 2]), tid);

  // ---- 3. out = U0 + beta((X - U0) - S), minus S's gravity part [B10]
  for (int e = tid; e < nint; e += NT) {
    int c0, c1, c2, t;
    T.dn0.divmod(e, t, c0);
    T.dn1.divmod(t, c2, c1);
    const long long c = b * P.S_b + (long long)(c2 + P.gd[2]) * P.S_k + (long long)(c1 + P.gd[1]) * P.S_j + (c0 + P.gd[0]);
    double S5[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) S5[v] = T.Sa[v * nint + e];
    if (P.grav_on) {
      const double rho = X[c];
      double gm = 0.0;
#pragma unroll
      for (int dd = 0; dd < 3; ++dd) {
        S5[1 + dd] -= dt * (rho * P.grav[dd]);
        gm += P.grav[dd] * X[(1 + dd) * P.S_v + c];
      }
      S5[4] -= dt * gm;
    }
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      const long long g = v * P.S_v + c;
      const double u0 = U0[g];
      out[g] = first ? (u0 - S5[v]) : (u0 + beta * ((X[g] - u0) - S5[v]));
    }
  }
  if (hit) fx_note(P, hit);
}

template <int RECON, int RIEMANN, int WS, int NT, int MINB>
static int launch_nt(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt,
                     const double *dt_dev, double beta, int first, cudaStream_t st) {
  const Geo g = geometry(P);
  auto kern = fx_k_stage_tile<RECON, RIEMANN, WS, NT, MINB>;
  // (per device and context, and cheap: set on every launch rather than cached per process)
  FX_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
  kern<<<(unsigned)P.nown, NT, g.smem, st>>>(P, X, U0, out, dx, dt, dt_dev, beta, first, g.ntile, g.faces_max, g.nint);
  FX_LAUNCH_CHECK("stage_tile");
  return FX_OK;
}

// Threads per CTA (measured): 256 for blocks of a few hundred zones (8^3 with PLM: two CTAs per SM; 16 x 16 in 2-D),
// 512 for 1024 zones and more and for WENO5 on 512 (one CTA per SM either way: more warps hide more latency).
template <int RECON, int RIEMANN, int WS>
static int launch(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt,
                  const double *dt_dev, double beta, int first, cudaStream_t st) {
  const int nint = P.n[0] * P.n[1] * P.n[2];
  if (nint >= 1024 || (RECON == FX_RECON_WENO5 && nint >= 512))
    return launch_nt<RECON, RIEMANN, WS, 512, 1>(P, X, U0, out, dx, dt, dt_dev, beta, first, st);
  if (geometry(P).ntile >= 1024) return launch_nt<RECON, RIEMANN, WS, 256, 1>(P, X, U0, out, dx, dt, dt_dev, beta, first, st);
  return launch_nt<RECON, RIEMANN, WS, 256, 4>(P, X, U0, out, dx, dt, dt_dev, beta, first, st);
}

}  // namespace fxtile

// Blocks whose primitives (padded block), one direction's fluxes and the accumulators fit the 227 KB of a CTA.
bool fx_stage_tile_supported(const FxParams &P) {
  if (P.nblocks > 0x7fffffffLL || P.nblocks < 1) return false;
  const fxtile::Geo g = fxtile::geometry(P);
  const int nint = P.n[0] * P.n[1] * P.n[2];
  const int nt = (nint >= 1024 || (P.recon == FX_RECON_WENO5 && nint >= 512)) ? 512 : 256;
  // (the gather keeps 5 bits per zone of a thread in one 64-bit word: at most 12 zones per thread)
  return g.smem <= (size_t)227 * 1024 && g.ntile <= 12 * nt;
}

int fx_launch_stage_tile(const FxParams &P, const double *X, const double *U0, double *out, const double *dx, double dt,
                         const double *dt_dev, double beta, int first, cudaStream_t st) {
  if (!fx_stage_tile_supported(P)) return fx_fail(FX_ERR_UNSUPPORTED, "tile stage kernel: block too large for shared memory");
  using namespace fxtile;
  const int key = (P.recon == FX_RECON_WENO5 ? 4 : 0) | (P.riemann == FX_RIEMANN_HLLC ? 2 : 0) | (P.wavespeed ? 1 : 0);
  switch (key) {
  case 0: return launch<FX_RECON_PLM_MINMOD, FX_RIEMANN_HLLE, 0>(P, X, U0, out, dx, dt, dt_dev, beta, first, st);
  case 1: return launch<FX_RECON_PLM_MINMOD, FX_RIEMANN_HLLE, 1>(P, X, U0, out, dx, dt, dt_dev, beta, first, st);
  case 2: return launch<FX_RECON_PLM_MINMOD, FX_RIEMANN_HLLC, 0>(P, X, U0, out, dx, dt, dt_dev, beta, first, st);
  case 3: return launch<FX_RECON_PLM_MINMOD, FX_RIEMANN_HLLC, 1>(P, X, U0, out, dx, dt, dt_dev, beta, first, st);
  case 4: return launch<FX_RECON_WENO5, FX_RIEMANN_HLLE, 0>(P, X, U0, out, dx, dt, dt_dev, beta, first, st);
  case 5: return launch<FX_RECON_WENO5, FX_RIEMANN_HLLE, 1>(P, X, U0, out, dx, dt, dt_dev, beta, first, st);
  case 6: return launch<FX_RECON_WENO5, FX_RIEMANN_HLLC, 0>(P, X, U0, out, dx, dt, dt_dev, beta, first, st);
  default: return launch<FX_RECON_WENO5, FX_RIEMANN_HLLC, 1>(P, X, U0, out, dx, dt, dt_dev, beta, first, st);
  }
}
