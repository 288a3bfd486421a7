// Host side of the TMA paths: tensor maps over a batch of cubes (x, y, z, cube), box tile_x x tile_y x tile_z x 1,
// encoded through the driver entry point cuTensorMapEncodeTiled (looked up at run time, so the library does
// not link against libcuda).  Out-of-bounds elements are zero-filled; the kernels reflect at the cube faces.
#include "idg_kernels.cuh"

namespace idg {

namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

cudaMemPool_t temp_pool()
{
    static cudaMemPool_t pool[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
    if (!pool[dev]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t p = nullptr;
        if (cudaMemPoolCreate(&p, &props) != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
        unsigned long long keep = ~0ull;
        (void)cudaMemPoolSetAttribute(p, cudaMemPoolAttrReleaseThreshold, &keep);
        pool[dev] = p;
    }
    return pool[dev];
}

}  // namespace

cudaError_t temp_alloc(void **p, size_t bytes, cudaStream_t st)
{
    cudaMemPool_t pool = temp_pool();
    return pool ? cudaMallocFromPoolAsync(p, bytes, pool, st) : cudaMallocAsync(p, bytes, st);
}

cudaError_t temp_trim()
{
    cudaMemPool_t pool = temp_pool();
    return pool ? cudaMemPoolTrimTo(pool, 0) : cudaSuccess;
}

bool tmap_available() { return encode_fn() != nullptr; }

bool tmap_encode(CUtensorMap *m, const float *base, int nx, int ny, int nz, int batch, int tile_x, int tile_y,
                 int tile_z)
{
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    const cuuint64_t dims[4] = {(cuuint64_t)nx, (cuuint64_t)ny, (cuuint64_t)nz, (cuuint64_t)batch};
    const cuuint64_t strides[3] = {(cuuint64_t)nx * 4, (cuuint64_t)nx * ny * 4, (cuuint64_t)nx * ny * (cuuint64_t)nz * 4};
    const cuuint32_t box[4] = {(cuuint32_t)tile_x, (cuuint32_t)tile_y, (cuuint32_t)tile_z, 1};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (void *)base, dims, strides, box, estr,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace idg
