// fx_guard_dt.cu -- K1 guard-cell fill + index-map export (a1) and K4 CFL min-reduction (a7).
#include "fx_physics.cuh"

// ------------------------------------------------------------------ a1 guard fill
// One thread per padded zone of one block (blockIdx.y, folded with gridDim.z for > 65535 blocks).
__global__ void __launch_bounds__(256) fx_k_fill_guardcells(FxParams P, double *__restrict__ U) {
  const long long b = blockIdx.y + (long long)blockIdx.z * gridDim.y;
  if (b >= P.nblocks) return;
  const int z = blockIdx.x * blockDim.x + threadIdx.x;
  if (z >= P.S_b) return;
  const int i = z % P.np[0], j = (z / P.np[0]) % P.np[1], k = z / (P.np[0] * P.np[1]);
  const bool interior = i >= P.gd[0] && i < P.gd[0] + P.n[0] && j >= P.gd[1] && j < P.gd[1] + P.n[1] &&
                        k >= P.gd[2] && k < P.gd[2] + P.n[2];
  if (interior) return;
  unsigned flip;
  const long long s = fx_guard_source(P, b, i, j, k, flip);
  const long long t = b * P.S_b + z;
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    const double x = U[v * P.S_v + s];
    U[v * P.S_v + t] = (v >= 1 && v <= 3 && ((flip >> (v - 1)) & 1u)) ? -x : x;
  }
  for (int v = 5; v < P.nvars; ++v) U[v * P.S_v + t] = U[v * P.S_v + s];  // passive scalars: copied, never negated [B11]
}

__global__ void __launch_bounds__(256) fx_k_index_map(FxParams P, long long b0, long long nb, long long *__restrict__ src) {
  const long long bb = blockIdx.y + (long long)blockIdx.z * gridDim.y;
  if (bb >= nb) return;
  const int z = blockIdx.x * blockDim.x + threadIdx.x;
  if (z >= P.S_b) return;
  const int i = z % P.np[0], j = (z / P.np[0]) % P.np[1], k = z / (P.np[0] * P.np[1]);
  unsigned flip;
  src[bb * P.S_b + z] = fx_guard_source(P, b0 + bb, i, j, k, flip);
}

static void fx_block_grid(long long nblocks, long long per_block_threads, dim3 &grid) {
  unsigned gx = (unsigned)((per_block_threads + 255) / 256);
  unsigned gy = (unsigned)(nblocks < 32768 ? (nblocks > 0 ? nblocks : 1) : 32768);
  unsigned gz = (unsigned)((nblocks + gy - 1) / gy);
  grid = dim3(gx, gy, gz ? gz : 1);
}

// The same with one thread per PAIR of x-adjacent padded zones (i even) and 16-byte accesses.  With nx, the x guard
// depth and the strides even a pair lies wholly in the interior or wholly in one guard region and takes the same hops,
// so its two sources are adjacent unless the x hop clamps (outflow) or mirrors (wall): those pairs go zone by zone.
__global__ void __launch_bounds__(256) fx_k_fill_guardcells_pairs(FxParams P, double *__restrict__ U) {
  const long long b = blockIdx.y + (long long)blockIdx.z * gridDim.y;
  if (b >= P.nblocks) return;
  const int zp = blockIdx.x * blockDim.x + threadIdx.x;
  if (2LL * zp >= P.S_b) return;
  const int hp = P.np[0] / 2;
  const int i = 2 * (zp % hp), j = (zp / hp) % P.np[1], k = zp / (hp * P.np[1]);
  const bool interior = i >= P.gd[0] && i < P.gd[0] + P.n[0] && j >= P.gd[1] && j < P.gd[1] + P.n[1] &&
                        k >= P.gd[2] && k < P.gd[2] + P.n[2];
  if (interior) return;
  unsigned f0, f1;
  const long long s0 = fx_guard_source(P, b, i, j, k, f0), s1 = fx_guard_source(P, b, i + 1, j, k, f1);
  const long long t = b * P.S_b + (long long)k * P.S_k + (long long)j * P.S_j + i;
  if (s1 == s0 + 1 && f0 == f1 && (s0 & 1) == 0) {
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      double2 x = *reinterpret_cast<const double2 *>(U + v * P.S_v + s0);
      if (v >= 1 && v <= 3 && ((f0 >> (v - 1)) & 1u)) { x.x = -x.x; x.y = -x.y; }
      *reinterpret_cast<double2 *>(U + v * P.S_v + t) = x;
    }
    for (int v = 5; v < P.nvars; ++v)  // passive scalars [B11]
      *reinterpret_cast<double2 *>(U + v * P.S_v + t) = *reinterpret_cast<const double2 *>(U + v * P.S_v + s0);
  } else {
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      const double x0 = U[v * P.S_v + s0], x1 = U[v * P.S_v + s1];
      const bool n0 = v >= 1 && v <= 3 && ((f0 >> (v - 1)) & 1u), n1 = v >= 1 && v <= 3 && ((f1 >> (v - 1)) & 1u);
      *reinterpret_cast<double2 *>(U + v * P.S_v + t) = make_double2(n0 ? -x0 : x0, n1 ? -x1 : x1);
    }
    for (int v = 5; v < P.nvars; ++v)
      *reinterpret_cast<double2 *>(U + v * P.S_v + t) = make_double2(U[v * P.S_v + s0], U[v * P.S_v + s1]);
  }
}

int fx_launch_fill_guardcells(const FxParams &P, double *U, cudaStream_t st) {
  if (P.nblocks == 0) return FX_OK;
  dim3 grid;
  if (P.active[0] && P.n[0] % 2 == 0 && P.gd[0] % 2 == 0 && P.S_v % 2 == 0 && ((uintptr_t)U & 15) == 0) {
    fx_block_grid(P.nblocks, P.S_b / 2, grid);
    fx_k_fill_guardcells_pairs<<<grid, 256, 0, st>>>(P, U);
    FX_LAUNCH_CHECK("fill_guardcells");
    return FX_OK;
  }
  fx_block_grid(P.nblocks, P.S_b, grid);
  fx_k_fill_guardcells<<<grid, 256, 0, st>>>(P, U);
  FX_LAUNCH_CHECK("fill_guardcells");
  return FX_OK;
}

// The generic path's per-stage fill of the passive scalars (variables v0 = 5 and up; the hydro variables' halo cells
// are read through the neighbour table by the zone kernel itself): only what its stencil reads.  The spatial operator is dimension by dimension [A11],
// so a stage reads the R zones behind each FACE of a block and no edge or corner zone; fx_hydro_advance leaves guard
// zones unspecified [A15], so nothing else has to be written (fx_fill_guardcells, the user's call, fills everything
// [A14]).  One thread per face guard zone; the layer index runs fastest on the x faces, i on the y and z faces.
__global__ void __launch_bounds__(256) fx_k_fill_faces(FxParams P, double *__restrict__ U, int R, int c0, int c1, int c2,
                                                       int v0) {
  const long long b = blockIdx.y + (long long)blockIdx.z * gridDim.y;
  if (b >= P.nblocks) return;
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= c0 + c1 + c2) return;
  const int nx = P.n[0], ny = P.n[1], nz = P.n[2];
  int i, j, k;
  if (t < c0) {  // x faces: (layer, j, k, side)
    const int l = t % R, jj = (t / R) % ny, kk = (t / (R * ny)) % nz, side = t / (R * ny * nz);
    i = side ? P.gd[0] + nx + l : P.gd[0] - 1 - l;
    j = P.gd[1] + jj;
    k = P.gd[2] + kk;
  } else if (t < c0 + c1) {  // y faces: (i, layer, k, side)
    t -= c0;
    const int ii = t % nx, l = (t / nx) % R, kk = (t / (nx * R)) % nz, side = t / (nx * R * nz);
    i = P.gd[0] + ii;
    j = side ? P.gd[1] + ny + l : P.gd[1] - 1 - l;
    k = P.gd[2] + kk;
  } else {  // z faces: (i, j, layer, side)
    t -= c0 + c1;
    const int ii = t % nx, jj = (t / nx) % ny, l = (t / (nx * ny)) % R, side = t / (nx * ny * R);
    i = P.gd[0] + ii;
    j = P.gd[1] + jj;
    k = side ? P.gd[2] + nz + l : P.gd[2] - 1 - l;
  }
  unsigned flip;
  const long long s = fx_guard_source(P, b, i, j, k, flip);
  const long long d = b * P.S_b + (long long)k * P.S_k + (long long)j * P.S_j + i;
  for (int v = v0; v < P.nvars; ++v) {  // variables v0 .. nvars-1
    const double x = U[v * P.S_v + s];
    U[v * P.S_v + d] = (v >= 1 && v <= 3 && ((flip >> (v - 1)) & 1u)) ? -x : x;
  }
}

int fx_launch_fill_faces(const FxParams &P, double *U, int v0, cudaStream_t st) {
  if (P.nblocks == 0 || v0 >= P.nvars) return FX_OK;
  const int R = (P.recon == FX_RECON_PLM_MINMOD) ? 2 : 3;
  const int c0 = P.active[0] ? 2 * R * P.n[1] * P.n[2] : 0, c1 = P.active[1] ? 2 * R * P.n[0] * P.n[2] : 0,
            c2 = P.active[2] ? 2 * R * P.n[0] * P.n[1] : 0;
  dim3 grid;
  fx_block_grid(P.nblocks, (long long)c0 + c1 + c2, grid);
  fx_k_fill_faces<<<grid, 256, 0, st>>>(P, U, R, c0, c1, c2, v0);
  FX_LAUNCH_CHECK("fill_faces");
  return FX_OK;
}

// ------------------------------------------------------------------ interior <-> padded state (host-buffer path)
// packed[v][b][k][j][i] over interior zones only  <->  U[v][b][k+g2][j+g1][i+g0].  One thread per interior zone and
// variable; rows of nx doubles are contiguous on both sides.  TO_PACKED: gather, else scatter (guard zones untouched).
template <bool TO_PACKED>
__global__ void __launch_bounds__(256) fx_k_pack_interior(FxParams P, double *__restrict__ U, double *__restrict__ packed,
                                                          long long n) {
  const int nx = P.n[0], ny = P.n[1], nz = P.n[2];
  const long long per_block = (long long)nx * ny * nz;
  for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
    const long long vb = e / per_block;  // v * nblocks + b: S_v = nblocks * S_b, so the padded offset is vb * S_b
    const int r = (int)(e - vb * per_block);
    const int i = r % nx, j = (r / nx) % ny, k = r / (nx * ny);
    const long long a = vb * P.S_b + (long long)(k + P.gd[2]) * P.S_k + (long long)(j + P.gd[1]) * P.S_j + (i + P.gd[0]);
    if (TO_PACKED) packed[e] = U[a]; else U[a] = packed[e];
  }
}

int fx_launch_pack_interior(const FxParams &P, double *U, double *packed, int to_packed, cudaStream_t st) {
  const long long n = (long long)P.nvars * P.nblocks * P.n[0] * P.n[1] * P.n[2];
  if (n == 0) return FX_OK;
  const long long want = (n + 255) / 256;
  const long long cap = (long long)fx_sm_count() * 32;
  const unsigned grid = (unsigned)(want < cap ? want : cap);
  if (to_packed) fx_k_pack_interior<true><<<grid, 256, 0, st>>>(P, U, packed, n);
  else fx_k_pack_interior<false><<<grid, 256, 0, st>>>(P, U, packed, n);
  FX_LAUNCH_CHECK("pack_interior");
  return FX_OK;
}

int fx_launch_index_map(const FxParams &P, long long b0, long long nb, long long *src, cudaStream_t st) {
  if (nb == 0) return FX_OK;
  dim3 grid;
  fx_block_grid(nb, P.S_b, grid);
  fx_k_index_map<<<grid, 256, 0, st>>>(P, b0, nb, src);
  FX_LAUNCH_CHECK("index_map");
  return FX_OK;
}

// ------------------------------------------------------------------ a7 CFL reduction
// dt = cfl * min over zones and active d of dx_d / (|u_d| + c)  =  cfl / max (|u_d| + c) (1 / dx_d).
// One CTA walks whole blocks (1/dx_d once per block, 32-bit index arithmetic inside a block); every thread keeps
// four zones' loads in flight; the per-zone work is 1/rho and sqrt by one cubic Newton step on the MUFU seeds (a few
// ulp: the tolerance on dt is 1e-14 relative) and no division.  Warp-shuffle max, one atomicMax per CTA on the bit
// pattern (non-negative doubles order like unsigned integers); the last CTA to finish writes cfl / max and re-arms
// the scratch words for the next call.  HBM-bound: one 40 B/zone read pass.
__global__ void __launch_bounds__(256) fx_k_compute_dt(FxParams P, const double *__restrict__ U,
                                                       const double *__restrict__ dx, double cfl,
                                                       double *__restrict__ dt_out, const int *__restrict__ jface,
                                                       long long njface) {
  const unsigned nx = P.n[0], ny = P.n[1];
  const unsigned per_block = nx * ny * (unsigned)P.n[2];
  double rate = 0.0;  // max of (|u_d| + c) / dx_d
  unsigned hit = 0;
  // 16-byte loads need every zone pair (i even) on a 16-byte boundary: even nx, guard depth and strides, aligned base
  const bool pairs = (nx % 2 == 0) && (P.gd[0] % 2 == 0) && (P.S_j % 2 == 0) && (P.S_v % 2 == 0) &&
                     ((reinterpret_cast<unsigned long long>(U) & 15ull) == 0);
  // (jface: only the owned blocks with a finer neighbour, each at the first such face of the jump-face list)
  const long long nit = jface ? njface : P.nown;
  for (long long it = blockIdx.x; it < nit; it += gridDim.x) {  // owned blocks only (a shard's ghosts are halo sources)
    long long b = it;
    if (jface) {
      const int bf = __ldg(&jface[it]);
      b = bf / 6;
      const int f = bf % 6;
      bool mine = b < P.nown && __ldg(&P.neigh[b * 6 + f]) == FX_NEIGH_FINER;
      for (int g = 0; g < f; ++g) mine = mine && __ldg(&P.neigh[b * 6 + g]) != FX_NEIGH_FINER;
      if (!mine) continue;
    }
    double idx[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) idx[d] = P.active[d] ? 1.0 / __ldg(&dx[b * 3 + d]) : 0.0;
    const double *Ub = U + b * P.S_b;
    auto zone_rate = [&](double u0, double u1, double u2, double u3, double u4, bool live) {
      double W[5];
      double ir;
      fx_c2p_v2(P, u0, u1, u2, u3, u4, W, &ir);
      const double cs = fx_sqrt3(P.gamma * W[4] * ir);
      double m = 0.0;
#pragma unroll
      for (int d = 0; d < 3; ++d) m = fx_max_sel((fabs(W[1 + d]) + cs) * idx[d], m);  // (a > b ? a : b: a NaN candidate loses)
      // a NaN anywhere reaches cs or a velocity; the maxima drop it, so test the sum
      const double chk = (fabs(W[1]) + fabs(W[2])) + (fabs(W[3]) + cs);
      if (live) {
        if (fx_hi_nonfinite(__double2hiint(chk)) || !(cs > 0.0)) hit |= FX_STATUS_NONFINITE;
        rate = fx_max_sel(m, rate);
      }
    };
    if (pairs) {
      // two x-adjacent zones per 16-byte load, two such pairs in flight per thread
      const unsigned hx = nx / 2, per_half = per_block / 2;
      for (unsigned r0 = threadIdx.x; r0 < per_half; r0 += 2 * 256) {
        double2 u[2][5];
        bool on[2];
#pragma unroll
        for (int q = 0; q < 2; ++q) {
          const unsigned r = r0 + q * 256;
          on[q] = r < per_half;
          const unsigned rr = on[q] ? r : r0;
          const unsigned i = 2 * (rr % hx), t = rr / hx, j = t % ny, k = t / ny;
          const long long c = (long long)(k + P.gd[2]) * P.S_k + (long long)(j + P.gd[1]) * P.S_j + (i + P.gd[0]);
#pragma unroll
          for (int v = 0; v < 5; ++v) u[q][v] = *reinterpret_cast<const double2 *>(Ub + v * P.S_v + c);
        }
#pragma unroll
        for (int q = 0; q < 2; ++q) {
          zone_rate(u[q][0].x, u[q][1].x, u[q][2].x, u[q][3].x, u[q][4].x, on[q]);
          zone_rate(u[q][0].y, u[q][1].y, u[q][2].y, u[q][3].y, u[q][4].y, on[q]);
        }
      }
    } else {
      for (unsigned r0 = threadIdx.x; r0 < per_block; r0 += 4 * 256) {
        double u[4][5];
        bool on[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const unsigned r = r0 + q * 256;
          on[q] = r < per_block;
          const unsigned rr = on[q] ? r : r0;
          const unsigned i = rr % nx, t = rr / nx, j = t % ny, k = t / ny;
          const long long c = (long long)(k + P.gd[2]) * P.S_k + (long long)(j + P.gd[1]) * P.S_j + (i + P.gd[0]);
#pragma unroll
          for (int v = 0; v < 5; ++v) u[q][v] = Ub[v * P.S_v + c];
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) zone_rate(u[q][0], u[q][1], u[q][2], u[q][3], u[q][4], on[q]);
      }
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) rate = fmax(rate, __shfl_xor_sync(0xffffffffu, rate, o));
  __shared__ double wmax[8];
  __shared__ bool last;
  if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = rate;
  if (hit) fx_note(P, hit);
  __syncthreads();
  if (threadIdx.x == 0) {
    double m = wmax[0];
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) m = fmax(m, wmax[w]);
    atomicMax(&P.scratch[FX_SCR_DTBITS], (unsigned long long)__double_as_longlong(m));
    __threadfence();
    unsigned long long done = atomicAdd(&P.scratch[FX_SCR_COUNTER], 1ull);
    last = (done == gridDim.x - 1);
  }
  __syncthreads();
  if (last && threadIdx.x == 0) {
    __threadfence();
    unsigned long long bits = atomicExch(&P.scratch[FX_SCR_DTBITS], 0ull);
    P.scratch[FX_SCR_COUNTER] = 0ull;
    *dt_out = cfl / __longlong_as_double((long long)bits);  // +inf for an empty batch
  }
}

int fx_launch_compute_dt(const FxParams &P, const double *U, const double *dx, double cfl, double *dt_out,
                         cudaStream_t st) {
  const long long want = P.nown < 1 ? 1 : P.nown;
  const long long cap = (long long)fx_sm_count() * 8;
  const int grid = (int)(want > cap ? cap : want);
  fx_k_compute_dt<<<grid, 256, 0, st>>>(P, U, dx, cfl, dt_out, nullptr, 0);
  FX_LAUNCH_CHECK("compute_dt");
  return FX_OK;
}

int fx_launch_compute_dt_corrected(const FxParams &P, const double *U, const double *dx, double cfl, double *dt_out,
                                   cudaStream_t st) {
  const long long want = P.njface < 1 ? 1 : P.njface;
  const long long cap = (long long)fx_sm_count() * 8;
  const int grid = (int)(want > cap ? cap : want);
  fx_k_compute_dt<<<grid, 256, 0, st>>>(P, U, dx, cfl, dt_out, P.jface, P.jface ? P.njface : 0);
  FX_LAUNCH_CHECK("compute_dt_corrected");
  return FX_OK;
}
