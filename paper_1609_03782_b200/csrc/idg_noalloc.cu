// idg_gaussian_filter_static: the rotated Gaussian filter (Eq. 3) for callers that cannot allocate --
// code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// idg_gaussian_filter() with a rotation takes (2r+1)^3 floats of kernel weights from the library's stream-ordered
// allocator on every call; it is the one filter whose scratch the caller cannot supply.  Here the weights live in a
// file-scope device array of fixed size (kStaticMaxRadius = 9: 19^3 floats = 27 436 bytes, held by every GPU that loads
// the library until the process exits).  This entry point calls no cudaMalloc / cudaFree / cudaMallocAsync and no
// allocating library routine; kernels with a larger support are rejected with IDG_ERR_STATIC_LIMIT.
//
// In HOST code the name `g_static_weights` is a host-side stand-in for the symbol, not a device address: a kernel handed
// it would fault (or, where the GPU can reach host memory, silently use the wrong memory).  The device address is asked
// for once per device, with that device current, through cudaGetSymbolAddress, and that pointer is what the kernel gets.
//
// Every call shares the one array, which keeps the previous call's contents: a call overwrites the (2r+1)^3 entries its
// kernel reads before the kernel runs (stream order), nothing has to start at zero, the rest is never read.  Calls
// that OVERLAP on the GPU -- different streams, or different host threads without a common stream -- race on the array
// and are not supported; calls on one stream, or ordered by events, are fine.
#include <math.h>

#include <mutex>

#include "../../include/idg.h"
#include "idg_kernels.cuh"

namespace {

constexpr int kStaticMaxRadius = 9;                                     // FWHM <= 7.4 voxels: every FWHM of the paper (1 .. 7)
constexpr int kStaticMaxWeights = (2 * kStaticMaxRadius + 1) * (2 * kStaticMaxRadius + 1) * (2 * kStaticMaxRadius + 1);

static __device__ __align__(256) float g_static_weights[kStaticMaxWeights];

// Device address of g_static_weights on the CURRENT device (cached per device ordinal; asked for again every time on
// ordinals beyond the cache).
cudaError_t static_weights_ptr(float **ptr)
{
    constexpr int kMaxDev = 64;
    static float *cache[kMaxDev] = {};
    static std::mutex mu;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool cached = dev >= 0 && dev < kMaxDev;
    if (cached) {
        std::lock_guard<std::mutex> lock(mu);
        if (cache[dev]) {
            *ptr = cache[dev];
            return cudaSuccess;
        }
    }
    float *p = nullptr;
    e = cudaGetSymbolAddress((void **)&p, g_static_weights);            // the current device's copy of the array
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    if (cached) {
        std::lock_guard<std::mutex> lock(mu);
        cache[dev] = p;
    }
    *ptr = p;
    return cudaSuccess;
}

bool overlap(const void *a, size_t na, const void *b, size_t nb)
{
    const char *pa = (const char *)a, *pb = (const char *)b;
    return pa < pb + nb && pb < pa + na;
}

}  // namespace

extern "C" int idg_gaussian_filter_static(const float *cube, int nx, int ny, int nz, float fwhm_x, float fwhm_y,
                                          float fwhm_z, float theta_x, float theta_y, float theta_z, float *out,
                                          void *stream)
{
    if (!cube || !out) return IDG_ERR_NULL;
    if (nx < 1 || ny < 1 || nz < 1) return IDG_ERR_DIMS;
    const unsigned long long N = (unsigned long long)nx * (unsigned long long)ny * (unsigned long long)nz;
    if ((unsigned long long)nx * (unsigned long long)ny > (1ull << 40) || N > (1ull << 40)) return IDG_ERR_DIMS;
    if (overlap(cube, (size_t)N * sizeof(float), out, (size_t)N * sizeof(float))) return IDG_ERR_OVERLAP;
    if (theta_x == 0.0f && theta_y == 0.0f && theta_z == 0.0f) return IDG_ERR_PARAM;      // separable: idg_gaussian_filter
    int r[3];
    const int rc = idg_gaussian_radii(fwhm_x, fwhm_y, fwhm_z, theta_x, theta_y, theta_z, r);       // validates; reading F3
    if (rc != IDG_OK) return rc;
    const int rr = r[0], W = 2 * rr + 1, nw = W * W * W;
    if (rr > kStaticMaxRadius) return IDG_ERR_STATIC_LIMIT;

    // Eq. 3 as in idg_gaussian_filter (reading F4): K(p) = G(R^-1 p), R = Rz Ry Rx, right-handed, degrees,
    // sampled on |p_j| <= r and normalised to unit sum in fp64 (reading F2).  Host stack only.
    const double f[3] = {fwhm_x, fwhm_y, fwhm_z}, th[3] = {theta_x, theta_y, theta_z};
    const double d2r = acos(-1.0) / 180.0;
    const double cx = cos(th[0] * d2r), sx = sin(th[0] * d2r), cy = cos(th[1] * d2r), sy = sin(th[1] * d2r),
                 cz = cos(th[2] * d2r), sz = sin(th[2] * d2r);
    const double R[3][3] = {{cz * cy, cz * sy * sx - sz * cx, cz * sy * cx + sz * sx},
                            {sz * cy, sz * sy * sx + cz * cx, sz * sy * cx - cz * sx},
                            {-sy, cy * sx, cy * cx}};
    double i2[3];
    for (int a = 0; a < 3; ++a) {
        const double s = f[a] / (2.0 * sqrt(2.0 * log(2.0)));           // Eq. 2
        i2[a] = 1.0 / (2.0 * s * s);
    }
    double g[kStaticMaxWeights];
    float gf[kStaticMaxWeights];
    double sum = 0.0;
    int m = 0;
    for (int k = -rr; k <= rr; ++k)
        for (int j = -rr; j <= rr; ++j)
            for (int i = -rr; i <= rr; ++i) {
                double q2 = 0.0;
                for (int a = 0; a < 3; ++a) {
                    const double q = R[0][a] * i + R[1][a] * j + R[2][a] * k;      // (R^T p)_a
                    q2 += q * q * i2[a];
                }
                g[m] = exp(-q2);
                sum += g[m++];
            }
    for (int t = 0; t < nw; ++t) gf[t] = (float)(g[t] / sum);

    float *d_w = nullptr;
    cudaError_t e = static_weights_ptr(&d_w);
    if (e != cudaSuccess) return (int)e;
    cudaStream_t st = (cudaStream_t)stream;
    // pageable source: the runtime stages it before returning, so `gf` may die with this frame
    e = cudaMemcpyAsync(d_w, gf, (size_t)nw * sizeof(float), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return (int)e;
    e = idg::launch_conv3d(cube, out, nx, ny, nz, rr, d_w, st);
    return e == cudaSuccess ? IDG_OK : (int)e;
}
