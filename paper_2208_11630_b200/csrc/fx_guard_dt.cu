// fx_guard_dt.cu -- K1 guard-cell fill + index-map export (a1) and K4 CFL min-reduction (a7).
#include "fx_physics.cuh"

// ------------------------------------------------------------------ a1 guard fill
// Source of padded zone (i,j,k) of block b: hops z, y, x through the neighbour table [O1, A14].
__device__ __forceinline__ long long fx_guard_source(const FxParams &P, long long b, int i, int j, int k) {
  int c[3] = {i, j, k};
  long long bs = b;
#pragma unroll
  for (int d = 2; d >= 0; --d) {
    if (!P.active[d]) continue;
    const int lo = P.gd[d], hi = P.gd[d] + P.n[d];
    if (c[d] < lo) {
      int nb = __ldg(&P.neigh[bs * 6 + 2 * d]);
      if (nb >= 0) { bs = nb; c[d] += P.n[d]; } else c[d] = lo;
    } else if (c[d] >= hi) {
      int nb = __ldg(&P.neigh[bs * 6 + 2 * d + 1]);
      if (nb >= 0) { bs = nb; c[d] -= P.n[d]; } else c[d] = hi - 1;
    }
  }
  return bs * P.S_b + c[2] * P.S_k + c[1] * P.S_j + c[0];
}

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
  const long long s = fx_guard_source(P, b, i, j, k);
  const long long t = b * P.S_b + z;
#pragma unroll
  for (int v = 0; v < 5; ++v) U[v * P.S_v + t] = U[v * P.S_v + s];
}

__global__ void __launch_bounds__(256) fx_k_index_map(FxParams P, long long b0, long long nb, long long *__restrict__ src) {
  const long long bb = blockIdx.y + (long long)blockIdx.z * gridDim.y;
  if (bb >= nb) return;
  const int z = blockIdx.x * blockDim.x + threadIdx.x;
  if (z >= P.S_b) return;
  const int i = z % P.np[0], j = (z / P.np[0]) % P.np[1], k = z / (P.np[0] * P.np[1]);
  src[bb * P.S_b + z] = fx_guard_source(P, b0 + bb, i, j, k);
}

static void fx_block_grid(long long nblocks, long long per_block_threads, dim3 &grid) {
  unsigned gx = (unsigned)((per_block_threads + 255) / 256);
  unsigned gy = (unsigned)(nblocks < 32768 ? (nblocks > 0 ? nblocks : 1) : 32768);
  unsigned gz = (unsigned)((nblocks + gy - 1) / gy);
  grid = dim3(gx, gy, gz ? gz : 1);
}

int fx_launch_fill_guardcells(const FxParams &P, double *U, cudaStream_t st) {
  if (P.nblocks == 0) return FX_OK;
  dim3 grid;
  fx_block_grid(P.nblocks, P.S_b, grid);
  fx_k_fill_guardcells<<<grid, 256, 0, st>>>(P, U);
  FX_LAUNCH_CHECK("fill_guardcells");
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
// Each thread folds several interior zones; warp-shuffle min; one atomicMin per CTA on the bit pattern
// (non-negative doubles order like unsigned integers); the last CTA to finish writes cfl*min and re-arms
// the scratch words for the next call.
__global__ void __launch_bounds__(256) fx_k_compute_dt(FxParams P, const double *__restrict__ U,
                                                       const double *__restrict__ dx, double cfl,
                                                       double *__restrict__ dt_out, long long nzones) {
  const int nx = P.n[0], ny = P.n[1], nz = P.n[2];
  const long long per_block = (long long)nx * ny * nz;
  double best = __longlong_as_double(0x7ff0000000000000ll);  // +inf
  unsigned hit = 0;
  for (long long z = (long long)blockIdx.x * blockDim.x + threadIdx.x; z < nzones; z += (long long)gridDim.x * blockDim.x) {
    const long long b = z / per_block;
    const int r = (int)(z - b * per_block);
    const int i = r % nx, j = (r / nx) % ny, k = r / (nx * ny);
    const long long c = b * P.S_b + (k + P.gd[2]) * P.S_k + (j + P.gd[1]) * P.S_j + (i + P.gd[0]);
    double W[5];
    fx_c2p(P, U[c], U[P.S_v + c], U[2 * P.S_v + c], U[3 * P.S_v + c], U[4 * P.S_v + c], W);
    const double cs = sqrt(P.gamma * W[4] / W[0]);
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      if (!P.active[d]) continue;
      const double s = fabs(W[1 + d]) + cs;
      if (!(s > 0.0) || !(s <= 1.79e308)) hit |= FX_STATUS_NONFINITE;
      best = fmin(best, __ldg(&dx[b * 3 + d]) / s);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) best = fmin(best, __shfl_xor_sync(0xffffffffu, best, o));
  __shared__ double wmin[8];
  __shared__ bool last;
  if ((threadIdx.x & 31) == 0) wmin[threadIdx.x >> 5] = best;
  if (hit) fx_note(P, hit);
  __syncthreads();
  if (threadIdx.x == 0) {
    double m = wmin[0];
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) m = fmin(m, wmin[w]);
    atomicMin(&P.scratch[FX_SCR_DTBITS], (unsigned long long)__double_as_longlong(m));
    __threadfence();
    unsigned long long done = atomicAdd(&P.scratch[FX_SCR_COUNTER], 1ull);
    last = (done == gridDim.x - 1);
  }
  __syncthreads();
  if (last && threadIdx.x == 0) {
    __threadfence();
    unsigned long long bits = atomicExch(&P.scratch[FX_SCR_DTBITS], 0x7ff0000000000000ull);
    P.scratch[FX_SCR_COUNTER] = 0ull;
    *dt_out = cfl * __longlong_as_double((long long)bits);
  }
}

int fx_launch_compute_dt(const FxParams &P, const double *U, const double *dx, double cfl, double *dt_out,
                         cudaStream_t st) {
  const long long nzones = P.nblocks * P.n[0] * P.n[1] * P.n[2];
  long long want = (nzones + 256 * 8 - 1) / (256 * 8);
  int grid = (int)(want < 1 ? 1 : (want > 148 * 16 ? 148 * 16 : want));
  fx_k_compute_dt<<<grid, 256, 0, st>>>(P, U, dx, cfl, dt_out, nzones);
  FX_LAUNCH_CHECK("compute_dt");
  return FX_OK;
}
