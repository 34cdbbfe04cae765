// Host side of tma.cuh: tensor-map encoding through the driver entry point looked up at run time.
#include "tma.cuh"

namespace {
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
        else
            cudaGetLastError();
    }
    return fn;
}
}  // namespace

cbct_status cbct_tensor_map_3d(CUtensorMap *out, const float *base, unsigned long long d0, unsigned long long d1,
                               unsigned long long d2, unsigned long long pitch1_bytes, unsigned long long pitch2_bytes,
                               unsigned b0, unsigned b1, unsigned b2)
{
    EncodeTiledFn fn = encode_fn();
    if (!fn) { cbct_set_error("cuTensorMapEncodeTiled is not available from this driver"); return CBCT_ERR_CUDA; }
    const cuuint64_t dims[3] = {d0, d1, d2};
    const cuuint64_t strides[2] = {pitch1_bytes, pitch2_bytes};
    const cuuint32_t box[3] = {b0, b1, b2};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float *>(base), dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        cbct_set_error("cuTensorMapEncodeTiled failed (%d): dims %llu x %llu x %llu, box %u x %u x %u", (int)r, d0, d1, d2, b0, b1, b2);
        return CBCT_ERR_CUDA;
    }
    return CBCT_OK;
}
