// fx_static_dt.cu -- fx_hydro_compute_dt_static: the CFL reduction a7 for callers that may not allocate (code under CUDA
// graph capture, serving loops, harnesses that forbid cudaMalloc) and therefore have no workspace to hand to the plan.
//
// fx_hydro_compute_dt keeps its two reduction words in the caller's workspace.  This variant keeps its scratch -- one
// partial maximum per block and two header words -- in a file-scope device array of fixed size, so the call needs nothing
// but the plan (a host object), the state, dx and the output word:
//
//   fx_static_scratch: 32 header words + FX_STATIC_DT_MAX_BLOCKS partials, 8 bytes each = 524 544 bytes of device memory,
//   held by every GPU that loads the library until the process exits.
//
// Rules that follow from the scratch being one array per device:
//   * a plan with more than FX_STATIC_DT_MAX_BLOCKS owned blocks is refused (FX_ERR_UNSUPPORTED), nothing is launched;
//   * the array keeps the last call's contents: the header (finished-CTA counter, status bits) is cleared on the call's
//     stream before every launch, the partials of the owned blocks are all rewritten by the launch;
//   * two calls that overlap on the GPU (different streams, no dependency between them) RACE on the array and both
//     results are undefined.  Calls on one stream, or ordered by events, are fine.
// The call itself makes no cudaMalloc / cudaFree and uses no allocating library routine; the first call on each device
// looks the array's device address up (cudaGetSymbolAddress), which is set-up and should happen outside a capture.
//
// Arithmetic per zone: that of fx_k_compute_dt (fx_guard_dt.cu), expression for expression; a maximum does not depend on
// the order it is taken in, so the two entry points return the same bits.
#include <mutex>

#include "fx_physics.cuh"

#define FX_STATIC_DT_HEADER 32  // words: [0] CTAs finished, [1] status bits of this call

namespace {

// In HOST code this name is a host-side stand-in, not a device address: only cudaGetSymbolAddress turns it into one.
static __device__ __align__(256) unsigned long long fx_static_scratch[FX_STATIC_DT_HEADER + FX_STATIC_DT_MAX_BLOCKS];

constexpr int FX_STATIC_MAX_DEVICES = 64;
unsigned long long *fx_static_addr[FX_STATIC_MAX_DEVICES] = {};  // device address of the array, per device ordinal
std::mutex fx_static_mutex;

// Once per device, with that device current.
int fx_static_scratch_ptr(unsigned long long **out) {
  int dev = -1;
  FX_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= FX_STATIC_MAX_DEVICES) return fx_fail(FX_ERR_UNSUPPORTED, "compute_dt_static: device ordinal %d out of range", dev);
  std::lock_guard<std::mutex> lock(fx_static_mutex);
  if (!fx_static_addr[dev]) {
    void *p = nullptr;
    FX_CUDA(cudaGetSymbolAddress(&p, fx_static_scratch));
    if (!p) return fx_fail(FX_ERR_CUDA, "compute_dt_static: cudaGetSymbolAddress returned a null address");
    fx_static_addr[dev] = static_cast<unsigned long long *>(p);
  }
  *out = fx_static_addr[dev];
  return FX_OK;
}

// One CTA walks whole blocks and leaves each block's maximum of (|u_d| + c) / dx_d in scr[HEADER + b]; the last CTA to
// finish takes the maximum of the partials and writes cfl / max (and the status bits, if asked for).
__global__ void __launch_bounds__(256) fx_k_compute_dt_static(FxParams P, const double *__restrict__ U, const double *__restrict__ dx,
                                                              double cfl, double *__restrict__ dt_out, unsigned *flags_out,
                                                              unsigned long long *scr) {
  const unsigned nx = P.n[0], ny = P.n[1];
  const unsigned per_block = nx * ny * (unsigned)P.n[2];
  __shared__ double wmax[8];
  __shared__ bool last;
  unsigned hit = 0;
  for (long long b = blockIdx.x; b < P.nown; b += gridDim.x) {
    double rate = 0.0;
    double idx[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) idx[d] = P.active[d] ? 1.0 / __ldg(&dx[b * 3 + d]) : 0.0;
    const double *Ub = U + b * P.S_b;
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
      for (int q = 0; q < 4; ++q) {
        double W[5], ir;
        fx_c2p_v2(P, u[q][0], u[q][1], u[q][2], u[q][3], u[q][4], W, &ir);
        const double cs = fx_sqrt3(P.gamma * W[4] * ir);
        double m = 0.0;
#pragma unroll
        for (int d = 0; d < 3; ++d) m = fx_max_sel((fabs(W[1 + d]) + cs) * idx[d], m);
        const double chk = (fabs(W[1]) + fabs(W[2])) + (fabs(W[3]) + cs);
        if (on[q]) {
          if (fx_hi_nonfinite(__double2hiint(chk)) || !(cs > 0.0)) hit |= FX_STATUS_NONFINITE;
          rate = fx_max_sel(m, rate);
        }
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) rate = fmax(rate, __shfl_xor_sync(0xffffffffu, rate, o));
    if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = rate;
    __syncthreads();
    if (threadIdx.x == 0) {
      double m = wmax[0];
      for (int w = 1; w < 8; ++w) m = fmax(m, wmax[w]);
      scr[FX_STATIC_DT_HEADER + b] = (unsigned long long)__double_as_longlong(m);
    }
    __syncthreads();  // wmax is free for the next block
  }
  if (hit) atomicOr(reinterpret_cast<unsigned *>(&scr[1]), hit);
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();  // this CTA's partials and status bits before its count
    const unsigned long long done = atomicAdd(&scr[0], 1ull);
    last = (done == gridDim.x - 1);
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  double rate = 0.0;
  for (long long b = threadIdx.x; b < P.nown; b += 256)
    rate = fmax(rate, __longlong_as_double((long long)__ldcg(&scr[FX_STATIC_DT_HEADER + b])));
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) rate = fmax(rate, __shfl_xor_sync(0xffffffffu, rate, o));
  if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = rate;
  __syncthreads();
  if (threadIdx.x == 0) {
    double m = wmax[0];
    for (int w = 1; w < 8; ++w) m = fmax(m, wmax[w]);
    *dt_out = cfl / m;  // +inf for an empty batch
    if (flags_out) *flags_out = (unsigned)__ldcg(&scr[1]);
  }
}

}  // namespace

extern "C" int fx_hydro_compute_dt_static(fx_hydro_plan *plan, const double *U, const double *dx, double cfl, double *dt_out,
                                          uint32_t *flags_out, void *stream) {
  if (!plan) return fx_fail(FX_ERR_INVALID_ARG, "compute_dt_static: null plan");
  const FxParams &P = plan->P;
  if (!dt_out || ((!U || !dx) && P.nown > 0)) return fx_fail(FX_ERR_INVALID_ARG, "compute_dt_static: null argument");
  if (P.nown > (long long)FX_STATIC_DT_MAX_BLOCKS)
    return fx_fail(FX_ERR_UNSUPPORTED, "compute_dt_static: %lld owned blocks exceed the static scratch array's %d (use fx_hydro_compute_dt with a workspace)",
                   P.nown, (int)FX_STATIC_DT_MAX_BLOCKS);
  unsigned long long *scr = nullptr;
  int rc = fx_static_scratch_ptr(&scr);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  // what must start at zero: the finished-CTA counter and the status bits (a call that failed half way may have left them set)
  FX_CUDA(cudaMemsetAsync(scr, 0, FX_STATIC_DT_HEADER * sizeof(unsigned long long), st));
  const long long want = P.nown < 1 ? 1 : P.nown;
  const long long cap = (long long)fx_sm_count() * 8;
  const int grid = (int)(want > cap ? cap : want);
  fx_k_compute_dt_static<<<grid, 256, 0, st>>>(P, U, dx, cfl, dt_out, flags_out, scr);
  FX_LAUNCH_CHECK("compute_dt_static");
  return FX_OK;
}
