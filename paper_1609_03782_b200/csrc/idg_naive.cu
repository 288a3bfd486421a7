// Naive IDG kernel: one thread per voxel, seven global loads, index clamping.
// Any shape and alignment; one iteration per launch.  It is the correctness
// baseline of the CUDA path and the route for shapes the tiled kernel rejects.
// Eq. 7; boundary reading R1.
#include "idg_kernels.cuh"

namespace idg {

__global__ void __launch_bounds__(256) idg_naive_kernel(const __grid_constant__ Launch L)
{
    const int b = blockIdx.y;
    const CubeParams p = cube_params(L, b);
    const float *src;
    float *dst;
    if (route(L, b, p, src, dst) == 0) return;

    const size_t plane = (size_t)L.nx * (size_t)L.ny;
    const size_t N = plane * (size_t)L.nz;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N;
         i += (size_t)gridDim.x * blockDim.x) {
        const int x = (int)(i % (size_t)L.nx);
        const int y = (int)((i / (size_t)L.nx) % (size_t)L.ny);
        const int z = (int)(i / plane);
        const float c = src[i];
        const float xm = x > 0 ? src[i - 1] : c;
        const float xp = x < L.nx - 1 ? src[i + 1] : c;
        const float ym = y > 0 ? src[i - L.nx] : c;
        const float yp = y < L.ny - 1 ? src[i + L.nx] : c;
        const float zm = z > 0 ? src[i - plane] : c;
        const float zp = z < L.nz - 1 ? src[i + plane] : c;
        dst[i] = L.mode == 1 ? update_pm(c, xm, xp, ym, yp, zm, zp, p.ax, p.ay, p.az, p.s, p.w)
                             : update(c, xm, xp, ym, yp, zm, zp, p.ax, p.ay, p.az, p.s, p.w);
    }
}

cudaError_t launch_naive(const Launch &L, cudaStream_t st)
{
    const size_t N = (size_t)L.nx * L.ny * L.nz;
    size_t blocks = (N + 255) / 256;
    if (blocks > (unsigned)device_sm_count() * 64u) blocks = (unsigned)device_sm_count() * 64u;      // grid-stride beyond 64 CTAs per SM
    dim3 grid((unsigned)blocks, (unsigned)L.batch);
    idg_naive_kernel<<<grid, 256, 0, st>>>(L);
    return cudaGetLastError();
}

}  // namespace idg
