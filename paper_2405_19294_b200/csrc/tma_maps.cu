// tma_maps.cu -- tensor-map descriptors (TMA) over the [plane][site] record layout of hr_internal.h, for the bulk kernel
// (dphi_bulk_kernel.cuh).  cuTensorMapEncodeTiled is a driver entry point; it is fetched through the runtime
// (cudaGetDriverEntryPoint) so that libhr.so carries no link-time dependency on libcuda.
#include <cuda.h>

#include <cstring>
#include <mutex>

#include "hr_internal.h"

namespace hr {

typedef CUresult (*encode_tiled_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                    const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static encode_tiled_fn get_encode()
{
    static encode_tiled_fn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
            return nullptr;
        fn = (encode_tiled_fn)p;
    }
    return fn;
}

// A record field of `nplanes` 16-byte planes over vh sites ([plane][site], plane stride vh * 16 bytes), `nfields` such
// fields `field_stride` bytes apart (1 for a spinor half field; 8 for a gauge field).  Elements are 8-byte words (two per
// site and plane); a box is `box_sites` consecutive sites of all planes of one field, landing in shared memory as
// [plane][box_sites] 16-byte vectors.
// Encoding is a pure function of its arguments and costs a driver call (microseconds, which a solver on a small lattice
// would pay six times per launch): the last 64 descriptors are kept.
struct MapKey { const void *base; size_t vh, field_stride; int nplanes, nfields, box; };
static hr_status encode_uncached(void *map64, const void *base, size_t vh, int nplanes, int nfields, size_t field_stride, int box_sites);

hr_status encode_plane_map(void *map64, const void *base, size_t vh, int nplanes, int nfields, size_t field_stride, int box_sites)
{
    static std::mutex mtx;
    static MapKey keys[64];
    static CUtensorMap maps[64];   // (CUtensorMap is declared 64-byte aligned)
    static int used = 0, next = 0;
    const MapKey k = { base, vh, field_stride, nplanes, nfields, box_sites };
    std::lock_guard<std::mutex> lock(mtx);
    for (int i = 0; i < used; ++i)
        if (keys[i].base == k.base && keys[i].vh == k.vh && keys[i].field_stride == k.field_stride && keys[i].nplanes == k.nplanes &&
            keys[i].nfields == k.nfields && keys[i].box == k.box) {
            memcpy(map64, &maps[i], sizeof(CUtensorMap));
            return HR_OK;
        }
    hr_status rc = encode_uncached(map64, base, vh, nplanes, nfields, field_stride, box_sites);
    if (rc != HR_OK) return rc;
    const int slot = used < 64 ? used++ : (next = (next + 1) % 64);
    keys[slot] = k;
    memcpy(&maps[slot], map64, sizeof(CUtensorMap));
    return HR_OK;
}

static hr_status encode_uncached(void *map64, const void *base, size_t vh, int nplanes, int nfields, size_t field_stride, int box_sites)
{
    encode_tiled_fn enc = get_encode();
    if (!enc) { set_error("bulk kernel: cuTensorMapEncodeTiled is not available from this driver"); return HR_EUNSUPPORTED; }
    if (box_sites < 1 || 2 * box_sites > 256 || nplanes < 1 || nplanes > 256) { set_error("bulk kernel: box of %d sites x %d planes", box_sites, nplanes); return HR_EUNSUPPORTED; }
    const cuuint64_t dims[3] = { (cuuint64_t)(2 * vh), (cuuint64_t)nplanes, (cuuint64_t)nfields };
    const cuuint64_t strides[2] = { (cuuint64_t)(vh * 16), (cuuint64_t)field_stride };
    const cuuint32_t box[3] = { (cuuint32_t)(2 * box_sites), (cuuint32_t)nplanes, 1u };
    const cuuint32_t estr[3] = { 1u, 1u, 1u };
    const cuuint32_t rank = nfields > 1 ? 3u : 2u;
    CUresult r = enc((CUtensorMap *)map64, CU_TENSOR_MAP_DATA_TYPE_UINT64, rank, const_cast<void *>(base), dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        set_error("bulk kernel: cuTensorMapEncodeTiled failed (%d) for vh=%zu planes=%d fields=%d stride=%zu box=%d", (int)r, vh, nplanes,
                  nfields, field_stride, box_sites);
        return HR_EUNSUPPORTED;
    }
    return HR_OK;
}

} // namespace hr
