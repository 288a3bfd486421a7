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
        pool[dev] = p;
    }
    return pool[dev];
}

}  // namespace

cudaError_t set_max_dynamic_smem(DeviceOnce &once, const void *kernel, size_t bytes)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool tracked = dev >= 0 && dev < 256;
    unsigned long long *word = &once.done_mask[tracked ? dev >> 6 : 0];
    const unsigned long long bit = 1ull << (dev & 63);
    if (tracked && (__atomic_load_n(word, __ATOMIC_ACQUIRE) & bit)) return cudaSuccess;
    e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess && tracked) __atomic_fetch_or(word, bit, __ATOMIC_RELEASE);
    return e;
}

int device_sm_count()
{
    thread_local int cached_dev = -1, cached_sms = 148;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 148;
    if (dev != cached_dev) {
        int n = 0;
        cached_sms = (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n > 0) ? n : 148;
        cached_dev = dev;
    }
    return cached_sms;
}

// What the pool may keep between calls (its release threshold) follows the requests: at least twice the largest
// recent one; after 64 requests in a row that are all below a quarter of it, it is halved.  Repeated calls of one
// size keep their temporaries mapped (no driver map / unmap per call); once the caller has moved on to small cubes
// the memory of a large call goes back to the driver, so a co-resident allocator is not starved for ever.
cudaError_t temp_alloc(void **p, size_t bytes, cudaStream_t st)
{
    cudaMemPool_t pool = temp_pool();
    if (!pool) return cudaMallocAsync(p, bytes, st);
    static unsigned long long keep[64] = {};
    static int small_run[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < 64) {
        unsigned long long thr = keep[dev];
        if (2ull * bytes >= thr) {
            thr = 2ull * bytes;
            small_run[dev] = 0;
        } else if (8ull * bytes < thr && ++small_run[dev] >= 64) {
            thr /= 2;
            small_run[dev] = 0;
        }
        if (thr != keep[dev]) {
            keep[dev] = thr;
            unsigned long long v = thr;
            (void)cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &v);
        }
    }
    return cudaMallocFromPoolAsync(p, bytes, pool, st);
}

cudaError_t temp_trim()
{
    cudaMemPool_t pool = temp_pool();
    return pool ? cudaMemPoolTrimTo(pool, 0) : cudaSuccess;
}

bool tmap_available() { return encode_fn() != nullptr; }

// pitch: row pitch in floats (0 = nx); elements nx .. pitch-1 of a row lie outside the tensor (zero fill)
bool tmap_encode(CUtensorMap *m, const float *base, int nx, int ny, int nz, int batch, int tile_x, int tile_y,
                 int tile_z, int pitch)
{
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    const cuuint64_t ld = (cuuint64_t)(pitch ? pitch : nx);
    const cuuint64_t dims[4] = {(cuuint64_t)nx, (cuuint64_t)ny, (cuuint64_t)nz, (cuuint64_t)batch};
    const cuuint64_t strides[3] = {ld * 4, ld * ny * 4, ld * ny * (cuuint64_t)nz * 4};
    const cuuint32_t box[4] = {(cuuint32_t)tile_x, (cuuint32_t)tile_y, (cuuint32_t)tile_z, 1};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (void *)base, dims, strides, box, estr,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace idg
