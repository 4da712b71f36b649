// fs_tma.cu -- host side of the TMA (tensor memory accelerator) descriptors used by the streaming kernels.
//
// The streaming kernels march an xy tile through z with their DRAM fetches running a few planes ahead of the register
// loads as L2 prefetches of whole tile planes: ONE cp.async.bulk.prefetch.tensor instruction per field and plane,
// issued by one thread, addressed through a CUtensorMap of the field (box = the tile's extended plane).  The part of
// a box that falls outside the array (the periodic seam) is skipped by the hardware; the tile on the other side of the
// seam prefetches it.  The descriptor is encoded here with the driver's cuTensorMapEncodeTiled, looked up at run time
// through the runtime (libfs links cudart statically and has no link-time dependency on libcuda).
#include "fs_internal.cuh"

namespace fs {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) p = nullptr;
    return reinterpret_cast<EncodeTiledFn>(p);
  }();
  return fn;
}

bool tmap_encode(Tmap* out, const void* ptr, int esize, int nx, int ny, int nz, int boxx, int boxy) {
  EncodeTiledFn fn = encode_fn();
  if (!fn || !ptr || (esize != 4 && esize != 8)) return false;
  if (boxx > nx || boxy > ny || boxx > 256 || boxy > 256) return false;                 // small levels: no prefetch (they live in L2 anyway)
  if (((size_t)nx * esize) % 16 != 0 || ((size_t)boxx * esize) % 16 != 0 || (reinterpret_cast<uintptr_t>(ptr) & 15)) return false;
  const cuuint64_t dims[3] = {(cuuint64_t)nx, (cuuint64_t)ny, (cuuint64_t)nz};
  const cuuint64_t strides[2] = {(cuuint64_t)nx * esize, (cuuint64_t)nx * ny * esize};
  const cuuint32_t box[3] = {(cuuint32_t)boxx, (cuuint32_t)boxy, 1u};
  const cuuint32_t estr[3] = {1u, 1u, 1u};
  const CUresult r = fn(&out->m, esize == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<void*>(ptr),
                        dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                        CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

}  // namespace fs
