// fx_tma.cuh -- the handful of PTX wrappers (mbarrier, 5-D bulk tensor copies, proxy fence) and the tensor-map
// encoder the TMA-fed stage kernels share (fx_stage_tma.cu, fx_stage_pair.cu).
#pragma once
#include <cuda.h>

#include "fx_internal.h"

namespace fxtma {

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long *bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, int bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// Wait for phase `parity` of the barrier.  A wait that lasts seconds means a lost TMA: trap (the launch then
// fails with an error) rather than hang the device.
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, int parity) {
  const unsigned a = smem_u32(bar);
  unsigned ok;
  int spins = 0;
  do {
    asm volatile(
        "{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
        : "=r"(ok)
        : "r"(a), "r"(parity)
        : "memory");
    if (!ok && ++spins > (1 << 22)) __trap();
  } while (!ok);
}
__device__ __forceinline__ void tma_load(void *dst, const CUtensorMap *map, unsigned long long *bar, int c0, int c1, int c2, int c3,
                                         int c4 = 0) {
  asm volatile(
      "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
      : "memory");
}
__device__ __forceinline__ void tma_store(const CUtensorMap *map, const void *src, int c0, int c1, int c2, int c3, int c4 = 0) {
  asm volatile("cp.async.bulk.tensor.5d.global.shared::cta.tile.bulk_group [%0, {%2, %3, %4, %5, %6}], [%1];"
               ::"l"(map), "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
               : "memory");
}
__device__ __forceinline__ void tma_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

// ------------------------------------------------------------------ host side: tensor maps
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline EncodeTiledFn lookup_encode_fn() {
  void *p = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
    return (EncodeTiledFn)p;
  return nullptr;
}

inline EncodeTiledFn encode_fn() {
  static const EncodeTiledFn fn = lookup_encode_fn();  // initialised once, thread-safely (C++11 static local)
  return fn;
}

// 5-D view of a state array, U[v][b][k][j][i] (i fastest), with a box of bx x by zones of nv variables.
inline int make_map(CUtensorMap *m, const FxParams &P, const double *base, int bx, int by, int nv = 5, int nvars_total = 5) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return fx_fail(FX_ERR_CUDA, "stage kernel: cuTensorMapEncodeTiled is not available from this driver");
  const cuuint64_t dims[5] = {(cuuint64_t)P.np[0], (cuuint64_t)P.np[1], (cuuint64_t)P.np[2], (cuuint64_t)P.nblocks, (cuuint64_t)nvars_total};
  const cuuint64_t strides[4] = {(cuuint64_t)P.S_j * 8, (cuuint64_t)P.S_k * 8, (cuuint64_t)P.S_b * 8, (cuuint64_t)P.S_v * 8};
  const cuuint32_t box[5] = {(cuuint32_t)bx, (cuuint32_t)by, 1, 1, (cuuint32_t)nv};
  const cuuint32_t es[5] = {1, 1, 1, 1, 1};
  const CUresult rc = fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, (void *)base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                         CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (rc != CUDA_SUCCESS) return fx_fail(FX_ERR_CUDA, "stage kernel: cuTensorMapEncodeTiled failed with code %d", (int)rc);
  return FX_OK;
}

}  // namespace fxtma
