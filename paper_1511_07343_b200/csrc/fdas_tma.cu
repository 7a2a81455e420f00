// fdas_tma.cu -- host side of fdas_tma.cuh: tensor maps are encoded by the driver (cuTensorMapEncodeTiled),
// reached through cudaGetDriverEntryPoint so that libfdas.so does not link libcuda itself.
#include "fdas_tma.cuh"

typedef CUresult (*fdas_encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                   const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                   CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static fdas_encode_fn encode_entry()
{
    static fdas_encode_fn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q = cudaDriverEntryPointSymbolNotFound;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<fdas_encode_fn>(p);
        else
            cudaGetLastError();
        tried = true;
    }
    return fn;
}

bool fdas_encode_tensor_map(CUtensorMap* out, const void* base, int rank, const uint64_t* dims, const uint64_t* strides_bytes,
                            const uint32_t* box)
{
    fdas_encode_fn fn = encode_entry();
    if (!fn || rank < 2 || rank > 3) return false;
    if (reinterpret_cast<uintptr_t>(base) & 15) return false;
    cuuint64_t gd[3], gs[2];
    cuuint32_t bx[3], es[3];
    for (int i = 0; i < rank; i++) {
        if (dims[i] == 0 || box[i] == 0 || box[i] > 256) return false;
        gd[i] = dims[i];
        bx[i] = box[i];
        es[i] = 1;
    }
    for (int i = 0; i + 1 < rank; i++) {
        if (strides_bytes[i] & 15) return false;
        gs[i] = strides_bytes[i];
    }
    // 8-byte elements (one complex value each): no interleave, no swizzle, zeros outside the tensor
    return fn(out, CU_TENSOR_MAP_DATA_TYPE_UINT64, (cuuint32_t)rank, const_cast<void*>(base), gd, gs, bx, es,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
