// osbli_tma.cuh -- the plane-tile machinery shared by the kernels that march along z over 32 x 8 (x,y) tiles
// (osbli_visc.cu, osbli_central.cu): tile constants, mbarrier / TMA wrappers, the tensor map of a state.
#pragma once
#include "osbli_common.cuh"
#include "osbli_kernels.h"

#include <cuda.h>          // CUtensorMap (types only; the encoder is fetched through the runtime)

namespace osbli {

constexpr int kVX = 32, kVY = 8, kVH = 2;
constexpr int kVPX = kVX + 2 * kVH, kVPY = kVY + 2 * kVH;        // 36 x 12 plane tile
constexpr unsigned kVTileBytes = 5 * kVPY * kVPX * sizeof(double);

#ifdef __CUDACC__
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// bounded spin: a transaction count that never completes traps instead of hanging the device
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity) {
  const unsigned a = smem_u32(bar);
  for (unsigned spin = 0; spin < (1u << 28); ++spin) {
    unsigned ok;
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(ok) : "r"(a), "r"(parity) : "memory");
    if (ok) return;
  }
  __trap();
}
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *map, int c0, int c1, int c2, int c3,
                                            unsigned long long *bar) {
  asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
               ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}

#endif

// 4-D tensor map over a state: (x incl. row padding, y incl. halo, z incl. halo, variable), box = one plane
// tile of all five variables.  The encoder lives in the driver library; it is fetched through the runtime
// so that libosbli links against nothing but cudart.
inline bool encode_state_map(const Layout &L, const double *Q, CUtensorMap *map, int box_rows = kVPY) {
  typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static encode_fn fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void *ptr = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<encode_fn>(ptr);
  }
  if (!fn) return false;
  const cuuint64_t dims[4] = {(cuuint64_t)L.sy, (cuuint64_t)(L.n[1] + 2 * L.h[1]), (cuuint64_t)(L.n[2] + 2 * L.h[2]), 5};
  const cuuint64_t strides[3] = {(cuuint64_t)L.sy * 8, (cuuint64_t)L.sz * 8, (cuuint64_t)L.sv * 8};
  const cuuint32_t box[4] = {kVPX, (cuuint32_t)box_rows, 1, 5};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  return fn(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<double *>(Q), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// The tensor map depends on the state's base address only; a step cycles through three states (Q, Q2, Q3), so
// the handle keeps a small cache and the driver's encoder runs once per address instead of once per launch.
inline const CUtensorMap *state_tensor_map(const Layout &L, const double *Q, TmapCache *cache, int box_rows = kVPY) {
  static_assert(sizeof(CUtensorMap) == sizeof(cache->map[0]), "TmapCache::map must hold a CUtensorMap");
  int hit = -1;
  for (int e = 0; e < cache->count; ++e)
    if (cache->ptr[e] == Q && cache->rows[e] == box_rows) hit = e;
  if (hit < 0) {
    hit = cache->count < TmapCache::kSlots ? cache->count++ : (cache->next++ % TmapCache::kSlots);
    if (!encode_state_map(L, Q, reinterpret_cast<CUtensorMap *>(&cache->map[hit]), box_rows)) { cache->count = 0; return nullptr; }
    cache->ptr[hit] = Q;
    cache->rows[hit] = box_rows;
  }
  return reinterpret_cast<const CUtensorMap *>(&cache->map[hit]);
}

}  // namespace osbli
