// Tensor-memory-accelerator plumbing for the panel kernels: tensor maps over the row-major state matrices of PAPER.md:39
// (host), and the mbarrier / cp.async.bulk(.tensor) PTX wrappers the producer and consumer warps use (device).
//
// Shared-memory image of one K-chunk of a panel ("stage"), identical for every source kind:
//   FP64: [v][cb16][step][16 doubles], each (v, cb16) plane written by the TMA unit with the 128-byte swizzle
//         (16-byte piece index ^= row & 7), so the (k = lane%4, column = lane/4) fragment loads of mma.m8n8k4.f64
//         are bank-conflict free without padding rows;
//   FP32: [v][step][NE floats], no swizzle (all lanes of a warp read one row).
// A state matrix [rows][5][ld] reaches that image with ONE tiled copy per chunk from a map whose dimensions are permuted
// to (element-in-16-block, row, 16-block, variable) (FP64) or (element, row, variable) (FP32); a plain matrix [K][N] of
// PAPER.md:37 eq. 1 (fr_gemm, S1, S5) with one copy per 16-column (FP64) / NE-column (FP32) block, ragged N and K
// zero-filled by the copy itself.
#pragma once
#include <cstring>
#include <cuda.h>

#include "common.cuh"

namespace frb {

typedef CUresult (*TmapEncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                 const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// cuTensorMapEncodeTiled through the runtime's driver entry point (no -lcuda).
inline TmapEncodeFn tmap_encode_fn() {
  static TmapEncodeFn fn = nullptr;
  if (!fn) {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q);
    if (e != cudaSuccess || q != cudaDriverEntryPointSuccess || !p)
      throw Error{FR_ECUDA, "cuTensorMapEncodeTiled is not available from this driver"};
    fn = (TmapEncodeFn)p;
  }
  return fn;
}

template <typename T>
inline CUtensorMapDataType tmap_dtype() {
  return sizeof(T) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
}

inline void tmap_check(CUresult r, const char *what) {
  if (r != CUDA_SUCCESS) throw Error{FR_ECUDA, std::string("cuTensorMapEncodeTiled failed for ") + what + " (" + std::to_string((int)r) + ")"};
}

// State matrix [rows][5][ld] (element fastest), chunks of `step` rows, panels of NE elements.
template <typename T>
inline CUtensorMap tmap_state(const T *p, long long rows, long long ld, int NE, int step) {
  CUtensorMap tm;
  const cuuint32_t es[4] = {1, 1, 1, 1};
  if (sizeof(T) == 8) {
    const cuuint64_t dims[4] = {16, (cuuint64_t)rows, (cuuint64_t)(ld / 16), 5};
    const cuuint64_t strides[3] = {(cuuint64_t)5 * ld * 8, 128, (cuuint64_t)ld * 8};
    const cuuint32_t box[4] = {16, (cuuint32_t)step, (cuuint32_t)(NE / 16), 5};
    tmap_check(tmap_encode_fn()(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, (void *)p, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE),
               "a state matrix (FP64)");
  } else {
    const cuuint64_t dims[3] = {(cuuint64_t)ld, (cuuint64_t)rows, 5};
    const cuuint64_t strides[2] = {(cuuint64_t)5 * ld * 4, (cuuint64_t)ld * 4};
    const cuuint32_t box[3] = {(cuuint32_t)NE, (cuuint32_t)step, 5};
    tmap_check(tmap_encode_fn()(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void *)p, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE),
               "a state matrix (FP32)");
  }
  return tm;
}

// Plain matrix [nbatch][K][ldb] with N valid columns, chunks of `step` rows, column blocks of 16 (FP64) / NE (FP32).
template <typename T>
inline CUtensorMap tmap_plain(const T *p, long long K, long long N, long long ldb, long long bstride, int nbatch, int NE, int step) {
  CUtensorMap tm;
  const cuuint32_t es[3] = {1, 1, 1};
  const cuuint64_t dims[3] = {(cuuint64_t)N, (cuuint64_t)K, (cuuint64_t)(nbatch > 0 ? nbatch : 1)};
  const cuuint64_t bs = nbatch > 1 ? (cuuint64_t)bstride : (cuuint64_t)K * ldb;
  const cuuint64_t strides[2] = {(cuuint64_t)ldb * sizeof(T), bs * sizeof(T)};
  const cuuint32_t box[3] = {(cuuint32_t)(sizeof(T) == 8 ? 16 : NE), (cuuint32_t)step, 1};
  tmap_check(tmap_encode_fn()(&tm, tmap_dtype<T>(), 3, (void *)p, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                              sizeof(T) == 8 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
                              CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE),
             "a plain matrix");
  return tm;
}

// What a fused epilogue reads per panel, for prefetching into L2 by the producer warp (cp.async.bulk.prefetch.tensor: one instruction
// for the whole box, no shared memory): an array [nplanes][rows][ld] (nplanes * rows metric terms or stage-register rows of NE
// elements each).  Boxes are limited to 256 per dimension: ok = false beyond that (the caller then skips the prefetch).
template <typename T>
inline CUtensorMap tmap_epi(const T *p, int nplanes, long long rows, long long ld, int NE, bool &ok) {
  CUtensorMap tm;
  memset(&tm, 0, sizeof tm);
  ok = rows >= 1 && rows <= 256 && nplanes >= 1 && nplanes <= 256;
  if (!ok) return tm;
  const cuuint32_t es[3] = {1, 1, 1};
  const cuuint64_t dims[3] = {(cuuint64_t)ld, (cuuint64_t)rows, (cuuint64_t)nplanes};
  const cuuint64_t strides[2] = {(cuuint64_t)ld * sizeof(T), (cuuint64_t)rows * ld * sizeof(T)};
  const cuuint32_t box[3] = {(cuuint32_t)NE, (cuuint32_t)rows, (cuuint32_t)nplanes};
  tmap_check(tmap_encode_fn()(&tm, tmap_dtype<T>(), 3, (void *)p, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE),
             "an epilogue operand");
  return tm;
}

#ifdef __CUDACC__

// the box at (c0, c1, c2) into L2; nothing to wait for
__device__ __forceinline__ void tma_prefetch_3d(const CUtensorMap *tm, int c0, int c1, int c2) {
  asm volatile("cp.async.bulk.prefetch.tensor.3d.L2.global.tile [%0, {%1, %2, %3}];" ::"l"(tm), "r"(c0), "r"(c1), "r"(c2) : "memory");
}

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
      : "=r"(ok)
      : "r"(bar), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {
  }
}

// One tiled copy global -> shared, completion counted in bytes on `bar`.
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap *tm, int c0, int c1, int c2, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(dst),
               "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap *tm, int c0, int c1, int c2, int c3, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(dst),
               "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar)
               : "memory");
}
// Contiguous bulk copy global -> shared (the operator image); bytes a multiple of 16, both addresses 16-byte aligned.
__device__ __forceinline__ void bulk_load(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src), "r"(bytes),
               "r"(bar)
               : "memory");
}
__device__ __forceinline__ void tmap_prefetch(const CUtensorMap *tm) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(tm) : "memory");
}

#endif  // __CUDACC__

}  // namespace frb
