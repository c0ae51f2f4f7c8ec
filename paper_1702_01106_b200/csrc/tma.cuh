// tma.cuh -- bulk tensor copies (TMA) of grid tiles into shared memory: the host side encodes a tensor map of a
// primitive array P[v][k][j][i]; the device side is a handful of PTX wrappers (mbarrier + cp.async.bulk.tensor).
// Used by the face-flux kernels (kernels_flux.cu) to stage the stencil zones of a tile of faces -- all N variables in one
// 4-D box -- without per-thread address arithmetic or staging registers, one tile ahead of the arithmetic.
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace grim {

// ---- host -------------------------------------------------------------------------------------------------
// Tensor map of the fp64 array at `base` with extents (s1, s2, s3, nvar), i fastest, variable stride zg, and a box of
// (b0, b1, b2, nvar) elements.  Out-of-range elements of a box read as zero.  Returns false when the driver entry point is
// missing or the layout does not meet the TMA constraints (row stride and box row a multiple of 16 bytes).
inline bool make_tile_map(CUtensorMap *out, const double *base, int s1, int s2, int s3, int nvar, long long zg, int b0,
                          int b1, int b2) {
  typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static encode_fn enc = nullptr;
  static bool looked = false;
  if (!looked) {
    looked = true;
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      enc = (encode_fn)p;
  }
  if (!enc) return false;
  if ((s1 % 2) || (b0 % 2) || (((uintptr_t)base) & 15) || b0 > 256 || b1 > 256 || b2 > 256 || nvar > 256) return false;
  const cuuint64_t gdim[4] = {(cuuint64_t)s1, (cuuint64_t)s2, (cuuint64_t)s3, (cuuint64_t)nvar};
  const cuuint64_t gstr[3] = {(cuuint64_t)s1 * 8, (cuuint64_t)s1 * s2 * 8, (cuuint64_t)zg * 8};
  const cuuint32_t box[4] = {(cuuint32_t)b0, (cuuint32_t)b1, (cuuint32_t)b2, (cuuint32_t)nvar};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  return enc(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, (void *)base, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

#ifdef __CUDACC__
// ---- device -----------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
// makes the initialised barriers visible to the asynchronous proxy (call once, before the block-wide sync)
__device__ __forceinline__ void mbar_init_fence() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t"
      "}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
// one 4-D box (c0, c1, c2, c3 = element coordinates of its first element) -> shared memory, completion on `bar`
__device__ __forceinline__ void tma_load_4d(void *smem_dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1, int c2,
                                            int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];" ::"r"(
          smem_u32(smem_dst)),
      "l"((uint64_t)map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}
#endif

}  // namespace grim
