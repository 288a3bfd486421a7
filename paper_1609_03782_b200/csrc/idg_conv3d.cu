// Dense 3-D convolution with replicated faces: the rotated Gaussian filter (Eq. 3),
// whose kernel K = Rz Ry Rx G is not separable along the cube axes.
//
//   out(x,y,z) = sum_{|i|,|j|,|k| <= r} K(i,j,k) I(cx(x+i), cy(y+j), cz(z+k))
//
// (K is even, so convolution and correlation coincide.)  A CTA produces a 32 x 8 x 16 block from the
// block plus halo staged in shared memory together with the (2r+1)^3 weights.  A thread owns one
// (x, y) column of 16 outputs along z: for every (i, j) it loads the 16 + 2r inputs of the shifted
// column and the 2r + 1 weights K(i, j, .) into registers once and issues 16 (2r+1) FMAs on them, so
// shared-memory traffic is ~1/4 load per FMA and the kernel is bound by the FP32 pipe, as a
// (2r+1)^3-tap filter should be.  r is a template parameter (register windows).
#include "idg_kernels.cuh"

namespace idg {

namespace {

constexpr int BX = 32, BY = 8, NT = 256;
// outputs per thread along z: 16 where the halo block still fits shared memory (shared-memory
// wavefronts per FMA 0.23, FP32-bound), 8 for the two largest radii
__host__ __device__ constexpr int bz_of(int r) { return r <= 8 ? 16 : 8; }

struct ConvArgs {
    const float *in;
    float *out;
    const float *kern;
    int nx, ny, nz;
};

template <int R>
__global__ void __launch_bounds__(NT) idg_conv3d_kernel(const __grid_constant__ ConvArgs S)
{
    constexpr int W = 2 * R + 1, BZ = bz_of(R);
    constexpr int SX = BX + 2 * R, SY = BY + 2 * R, SZ = BZ + 2 * R;
    extern __shared__ __align__(16) float smem[];
    float *tile = smem;                          // SZ x SY x SX
    float *wk = smem + SZ * SY * SX;             // W x W x W, x fastest

    const int x0 = blockIdx.x * BX, y0 = blockIdx.y * BY, z0 = blockIdx.z * BZ;
    const size_t plane = (size_t)S.nx * (size_t)S.ny;
    for (int e = threadIdx.x; e < SZ * SY * SX; e += NT) {
        const int zz = e / (SY * SX), rem = e - zz * (SY * SX), yy = rem / SX, xx = rem - yy * SX;
        const int gx = min(max(x0 - R + xx, 0), S.nx - 1);
        const int gy = min(max(y0 - R + yy, 0), S.ny - 1);
        const int gz = min(max(z0 - R + zz, 0), S.nz - 1);
        tile[e] = __ldg(S.in + (size_t)gz * plane + (size_t)gy * S.nx + gx);
    }
    for (int e = threadIdx.x; e < W * W * W; e += NT) wk[e] = __ldg(S.kern + e);
    __syncthreads();

    const int tx = threadIdx.x & (BX - 1), ty = threadIdx.x / BX;
    float acc[BZ];
#pragma unroll
    for (int o = 0; o < BZ; ++o) acc[o] = 0.f;
    for (int j = 0; j < W; ++j) {
        for (int i = 0; i < W; ++i) {
            float col[SZ], w[W];
            const float *c = tile + (ty + j) * SX + tx + i;
#pragma unroll
            for (int zz = 0; zz < SZ; ++zz) col[zz] = c[zz * SY * SX];
            const float *kw = wk + j * W + i;
#pragma unroll
            for (int k = 0; k < W; ++k) w[k] = kw[k * W * W];
#pragma unroll
            for (int k = 0; k < W; ++k)
#pragma unroll
                for (int o = 0; o < BZ; ++o) acc[o] = fmaf(w[k], col[o + k], acc[o]);
        }
    }
    const int gx = x0 + tx, gy = y0 + ty;
    if (gx < S.nx && gy < S.ny) {
#pragma unroll
        for (int o = 0; o < BZ; ++o)
            if (z0 + o < S.nz) S.out[(size_t)(z0 + o) * plane + (size_t)gy * S.nx + gx] = acc[o];
    }
}

template <int R>
cudaError_t launch_r(const ConvArgs &S, cudaStream_t st)
{
    constexpr int W = 2 * R + 1, BZ = bz_of(R);
    constexpr size_t smem = sizeof(float) * ((size_t)(BX + 2 * R) * (BY + 2 * R) * (BZ + 2 * R) + (size_t)W * W * W);
    static_assert(smem <= 227u * 1024u, "shared memory budget");
    static DeviceOnce smem_once;
    {
        const cudaError_t e = set_max_dynamic_smem(smem_once, (const void *)(idg_conv3d_kernel<R>), smem);
        if (e != cudaSuccess) return e;
    }
    const unsigned gx = (unsigned)((S.nx + BX - 1) / BX), gy = (unsigned)((S.ny + BY - 1) / BY),
                   gz = (unsigned)((S.nz + BZ - 1) / BZ);
    if (gy > 65535u || gz > 65535u) return cudaErrorInvalidValue;
    idg_conv3d_kernel<R><<<dim3(gx, gy, gz), NT, smem, st>>>(S);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_conv3d(const float *in, float *out, int nx, int ny, int nz, int r, const float *kern,
                          cudaStream_t st)
{
    ConvArgs S{in, out, kern, nx, ny, nz};
    switch (r) {
    case 0: return launch_r<0>(S, st);
    case 1: return launch_r<1>(S, st);
    case 2: return launch_r<2>(S, st);
    case 3: return launch_r<3>(S, st);
    case 4: return launch_r<4>(S, st);
    case 5: return launch_r<5>(S, st);
    case 6: return launch_r<6>(S, st);
    case 7: return launch_r<7>(S, st);
    case 8: return launch_r<8>(S, st);
    case 9: return launch_r<9>(S, st);
    case 10: return launch_r<10>(S, st);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace idg
