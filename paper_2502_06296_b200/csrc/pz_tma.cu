// pz_tma.cu -- host side of pz_tma.cuh: tensor-map encoding through the driver entry point.
#include "pz_tma.cuh"
#include "pz_internal.h"

#include <mutex>

namespace pz {

namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn g_encode = nullptr;
std::once_flag g_once;

void resolve()
{
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult q = cudaDriverEntryPointSymbolNotFound;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
        g_encode = reinterpret_cast<EncodeTiledFn>(fn);
    else
        cudaGetLastError();
}

} // namespace

int encode_column_tile_map(CUtensorMap *map, const double *field, size_t ncols, int nz, int tx, int box_rows, int l2promo,
                           bool swizzle128)
{
    std::call_once(g_once, resolve);
    if (!g_encode) {
        set_error("cuTensorMapEncodeTiled is not available from this driver");
        return PZ_ECUDA;
    }
    const cuuint64_t gdim[2] = {(cuuint64_t)ncols, (cuuint64_t)nz};
    const cuuint64_t gstride[1] = {(cuuint64_t)ncols * sizeof(double)};
    const cuuint32_t box[2] = {(cuuint32_t)tx, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = g_encode(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double *>(field), gdim, gstride, box,
                                estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                swizzle128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
                                l2promo == 0 ? CU_TENSOR_MAP_L2_PROMOTION_NONE : l2promo == 2 ? CU_TENSOR_MAP_L2_PROMOTION_L2_256B
                                                                               : l2promo == 3 ? CU_TENSOR_MAP_L2_PROMOTION_L2_64B
                                                                                              : CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                                CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        set_error("cuTensorMapEncodeTiled failed (%d) for %zu columns x %d rows, box %d x %d", (int)r, ncols, nz, tx,
                  box_rows);
        return PZ_ECUDA;
    }
    return PZ_OK;
}

int cached_column_map(pz_plan *pl, const CUtensorMap **out, const double *field, size_t ncols, int nz, int tx, int box_rows,
                      int l2promo, bool swizzle128)
{
    const int swz = swizzle128 ? 1 : 0;
    for (auto &e : pl->maps)
        if (e.ptr == field && e.ncols == ncols && e.nz == nz && e.tx == tx && e.box_rows == box_rows && e.l2promo == l2promo &&
            e.swz == swz) {
            *out = &e.map;
            return PZ_OK;
        }
    pz_plan::MapEntry e;
    e.ptr = field; e.ncols = ncols; e.nz = nz; e.tx = tx; e.box_rows = box_rows; e.l2promo = l2promo; e.swz = swz;
    const int rc = encode_column_tile_map(&e.map, field, ncols, nz, tx, box_rows, l2promo, swizzle128);
    if (rc != PZ_OK) return rc;
    if (pl->maps.size() < 16) {
        pl->maps.reserve(16);   // entries never move: callers keep the pointer until their launch returns
        pl->maps.push_back(e);
        *out = &pl->maps.back().map;
    } else {
        pl->maps[pl->maps_next % 16] = e;
        *out = &pl->maps[pl->maps_next % 16].map;
        ++pl->maps_next;
    }
    return PZ_OK;
}

} // namespace pz
