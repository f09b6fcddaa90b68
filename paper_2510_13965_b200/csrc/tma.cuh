// TMA (cp.async.bulk.tensor) and mbarrier helpers shared by the stencil kernels (ccz4.cu, les.cu), plus the host-side tensor map of a slot
// seen as a 4-D tensor (x, y, z, field) of doubles. sm_100a only.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdlib.h>
#include "mhd_internal.cuh"

namespace mhd {

__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(parity) : "memory");
}
// one box of the 4-D tensor into shared memory; coordinates past the end of the array are zero-filled by the copy engine
__device__ __forceinline__ void tma_load_4d(double* smem, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2, int c3) {
  asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];\n"
               ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"((uint64_t)map), "r"((unsigned)__cvta_generic_to_shared(bar)),
                 "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}

// Tensor map of `nfields` fields at `base` (field stride `stride` elements) as a 4-D tensor (x, y, z, field) with a bx x by x bz x 1 box.
// Legal when the row pitch and the field stride are multiples of 16 bytes (MX even, stride even) and the base is 16-byte aligned; the caller
// must also keep every box origin on an even x index (a box must start on a 16-byte boundary: measured on sm_100a, an odd x origin of
// 8-byte elements raises "illegal instruction"). Returns false when the patch does not qualify or the driver entry point is missing.
inline bool make_tensor_map_4d(const Dims& d, const double* base, size_t stride, int nfields, int bx, int by, int bz, CUtensorMap* out) {
  typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                               const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static EncodeFn encode = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess) encode = (EncodeFn)fn;
    const char* v = getenv("MHD_TMA");
    if (v && atoi(v) == 0) encode = nullptr;
  }
  if (!encode || (d.mx & 1) || (stride & 1) || ((uintptr_t)base & 15) || ((bx * 8) & 15)) return false;
  const cuuint64_t dims[4] = {(cuuint64_t)d.mx, (cuuint64_t)d.my, (cuuint64_t)d.mz, (cuuint64_t)nfields};
  const cuuint64_t strides[3] = {(cuuint64_t)d.mx * 8, (cuuint64_t)d.sz * 8, (cuuint64_t)stride * 8};
  const cuuint32_t box[4] = {(cuuint32_t)bx, (cuuint32_t)by, (cuuint32_t)bz, 1};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  return encode(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, (void*)base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace mhd
