// Internal declarations shared by the CUDA translation units of libidg_b200.so.
// Not part of the public boundary (include/idg.h) and not used by oracle/.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace idg {

// Per-cube constants derived on the host in fp64 and rounded once (step a0):
//   ax = tau*Cx, ay = tau*Cy, az = tau*Cz   (Eq. 7 numerator)
//   s  = 1/(K*rms), 0 when K = +inf         (Eq. 6:  S = 1/(1 + (I*s)^2))
//   w  = -2*(ax + ay + az)                  (the centre weight of the expanded numerator)
struct CubeParams {
    float ax, ay, az, s;
    int n_iter;
    float w;                // -2 (ax + ay + az), from the fp64 sum, rounded once
    int pad_[2];
};
static_assert(sizeof(CubeParams) == 32, "CubeParams is uploaded as a 32-byte record");

// One launch over `batch` cubes; iterations [iter_done, iter_done + fuse) of each cube that
// still has iterations left.
struct Launch {
    const float *in;        // I_0 of cube 0 (read only by each cube's first launch)
    float *out;             // final destination of cube 0
    float *scratch;         // scratch cube 0
    const CubeParams *tab;  // device table [batch], or nullptr -> use `one`
    CubeParams one;
    int nx, ny, nz, batch;
    int iter_done;          // iterations already applied to every cube by earlier launches
    int fuse;               // iterations per launch of this plan (T)
    int in_place;           // out == in: the host staged a copy of I_0 in `scratch`
    int mode;               // 0: intensity-driven conductance (Eq. 6); 1: gradient-driven (Eq. 5, idg_filter_pm)
    int pitch;              // row pitch in floats of the three buffers; 0 = dense (nx).  > nx: the library's own
                            // pitched copies of cubes with nx % 4 != 0 (kernel 3 only)
};

// floats from one cube of a batch to the next
__host__ __device__ __forceinline__ size_t cube_stride(const Launch &L)
{
    return (size_t)(L.pitch ? L.pitch : L.nx) * (size_t)L.ny * (size_t)L.nz;
}

// Which buffers cube b reads / writes in this launch so that its LAST launch writes `out`.
// Returns the number of iterations to apply now (0 = cube already finished).
// iter_done: iterations applied before this launch (L.iter_done), or before this round of a cooperative launch.
__device__ __forceinline__ int route(const Launch &L, int iter_done, int b, const CubeParams &p,
                                     const float *&src, float *&dst)
{
    const int remaining = p.n_iter - iter_done;
    if (remaining <= 0) return 0;
    const int now = remaining < L.fuse ? remaining : L.fuse;
    const int after = (remaining - now + L.fuse - 1) / L.fuse;      // launches still to come
    const size_t off = (size_t)b * cube_stride(L);
    float *o = L.out + off, *s = L.scratch + off;
    dst = (after & 1) ? s : o;
    if (iter_done == 0)     // first launch: read I_0 (from the staged copy if it would alias dst)
        src = (L.in_place && !(after & 1)) ? s : (L.in + off);
    else
        src = (after & 1) ? o : s;
    return now;
}
__device__ __forceinline__ int route(const Launch &L, int b, const CubeParams &p, const float *&src, float *&dst)
{
    return route(L, L.iter_done, b, p, src, dst);
}

__device__ __forceinline__ CubeParams cube_params(const Launch &L, int b)
{
    return L.tab ? L.tab[b] : L.one;
}

// Conductance S = 1/(1 + u^2), u = I*s  (Eq. 6).  den >= 1, so the approximate reciprocal
// (one MUFU.RCP, <= 1 ulp) needs no range handling; rcp(1) == 1 exactly (K = +inf limit).
__device__ __forceinline__ float conductance(float c, float s)
{
    const float u = c * s;
    const float den = fmaf(u, u, 1.0f);
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(den));
    return r;
}

// One voxel update (Eq. 7).  The numerator tau (Cx Dx I + Cy Dy I + Cz Dz I) is expanded to
//   ax (xp + xm) + ay (yp + ym) + az (zp + zm) + w c,   w = -2 (ax + ay + az),
// evaluated as fma(ax, sx, fma(ay, sy, fma(az, sz, w c))): 10 FP32 operations + 1 reciprocal per voxel instead
// of 12 for the difference form.  Every kernel (scalar or packed) uses exactly this order, so they agree bit
// for bit.  A constant cube is a fixed point up to the rounding of w c (not bitwise).
__device__ __forceinline__ float update(float c, float xm, float xp, float ym, float yp,
                                        float zm, float zp, float ax, float ay, float az, float s, float w)
{
    const float lap = fmaf(ax, xp + xm, fmaf(ay, yp + ym, fmaf(az, zp + zm, w * c)));
    return fmaf(lap, conductance(c, s), c);
}

// Gradient-driven variant of update(): conductance 1/(1 + |grad I|^2 s^2) with central differences
// (Eq. 5; readings P1-P3).  Same operation order as update2_pm() of idg_stream.cu.
__device__ __forceinline__ float update_pm(float c, float xm, float xp, float ym, float yp,
                                           float zm, float zp, float ax, float ay, float az, float s, float w)
{
    const float lap = fmaf(ax, xp + xm, fmaf(ay, yp + ym, fmaf(az, zp + zm, w * c)));
    const float gx = xp - xm, gy = fmaf(-1.0f, ym, yp), gz = fmaf(-1.0f, zm, zp);
    const float G = fmaf(gz, gz, fmaf(gy, gy, gx * gx));
    const float den = fmaf(0.25f * s * s, G, 1.0f);
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(den));
    return fmaf(lap, r, c);
}

// Kernel launchers (each returns cudaGetLastError of its launch).
cudaError_t launch_naive(const Launch &L, cudaStream_t st);
cudaError_t launch_tiled(const Launch &L, int zchunk, cudaStream_t st);
bool tiled_supported(int nx, int ny, int nz, const void *in, const void *out, const void *scratch);
cudaError_t launch_tma(const Launch &L, int zchunk, int tile, cudaStream_t st);
// Cubes with nx % 4 != 0 run kernel 3 on pitched copies (row pitch = nx rounded up to 4 floats): dense -> pitched
// before the first launch, pitched -> dense after the last (cubes with n_iter = 0 take their input copy).
bool tma_pitched_supported(int nx, int ny, int nz);
cudaError_t launch_repitch(const float *src, int src_pitch, float *dst, int dst_pitch, const float *src_zero,
                           const CubeParams *tab, int nx, int ny, int nz, int batch, cudaStream_t st);
// All `rounds` launches of a plan (fuse iterations each) as ONE cooperative launch with grid barriers in between, for
// workloads whose whole grid is co-resident (small, L2-resident cubes).  bar: 8 zeroed bytes of device memory.
// cudaErrorNotSupported / cudaErrorCooperativeLaunchTooLarge: use launch_tma per round instead.
cudaError_t launch_tma_coop(const Launch &L, int zchunk, int tile, int rounds, unsigned *bar, cudaStream_t st);
bool tma_supported(int nx, int ny, int nz, const void *in, const void *out, const void *scratch);

// Resident kernel (idg_resident.cu): the cube(s) stay in shared memory for all iterations of a call; block faces are
// exchanged through mailboxes in the workspace.  resident_plan() picks the block decomposition (false: the shape does
// not fit); launch_resident() enqueues one cooperative launch per wave of cubes.
struct ResidentPlan {
    int ty, tz;             // blocks per cube along y, z
    int by, bz;             // nominal block extents
    int ls;                 // z cells per warp work item
    int cubes;              // cubes per launch (wave)
    int words;              // 64-bit mailbox words per (block, parity)
    size_t smem;            // dynamic shared memory per CTA
    bool small;             // the kernel will take its small-block path (one item per warp, <= 2 inbound entries per thread)
};
constexpr size_t kResidentMailBytes = (size_t)32 << 20;       // mailbox region reserved in the workspace
constexpr size_t kResidentMaxCubeVoxels = (size_t)4 << 20;     // larger cubes cannot be held on chip
bool resident_plan(int nx, int ny, int nz, int batch, int max_n, size_t mail_bytes, int sms, ResidentPlan *out);
cudaError_t launch_resident(const Launch &L, const ResidentPlan &P, unsigned long long *mail, cudaStream_t st,
                            int *launches);
int device_sm_count();      // SMs of the current device (148 when it cannot be queried)

// Per-device one-time work (idg_tmap.cu).  cudaFuncSetAttribute applies to the CURRENT device only, so "done" is
// remembered per device ordinal; a benign race just sets the attribute twice.
struct DeviceOnce {
    unsigned long long done_mask[4] = {0, 0, 0, 0};      // devices 0..255
};
cudaError_t set_max_dynamic_smem(DeviceOnce &once, const void *kernel, size_t bytes);

// Stream-ordered temporaries (idg_tmap.cu): cudaMallocAsync from a private memory pool that keeps what it has
// been given (release threshold = everything), so a call that needs a cube-sized temporary does not pay the
// driver's map / unmap every time; temp_trim() hands the unused part back.  Free with cudaFreeAsync.
cudaError_t temp_alloc(void **p, size_t bytes, cudaStream_t st);
cudaError_t temp_trim();

// Tensor maps for the TMA kernels (idg_tmap.cu): 4-D (x, y, z, cube), box tile_x x tile_y x 1 x 1, zero fill.
bool tmap_available();
bool tmap_encode(CUtensorMap *m, const float *base, int nx, int ny, int nz, int batch, int tile_x, int tile_y,
                 int tile_z = 1, int pitch = 0);

// Reference filters (PAPER.md sections 3.1-3.2): separable single-pass filter (box, axis-aligned
// Gaussian) and dense 3-D convolution (rotated Gaussian, Eq. 3).
constexpr int kSepMaxRadius = 16;      // per-axis radius limit of the separable kernel
constexpr int kConvMaxRadius = 10;     // radius limit of the dense kernel (cube support (2r+1)^3)
cudaError_t launch_sep3d(const float *in, float *out, int nx, int ny, int nz, int rx, int ry, int rz,
                         const float *wx, const float *wy, const float *wz, cudaStream_t st);
// TMA-fed barrier-free variant for radii <= 4, nx % 4 == 0, 16-byte aligned cubes (idg_sep3d_tma.cu)
bool sep3d_tma_supported(int nx, int ny, int nz, int rx, int ry, int rz, const void *in, const void *out);
cudaError_t launch_sep3d_tma(const float *in, float *out, int nx, int ny, int nz, int rx, int ry, int rz,
                             const float *wx, const float *wy, const float *wz, int zchunk, int variant, cudaStream_t st);
// the same for radii 5 .. 9 (idg_sep3d_big.cu): HL halo lanes per side, z window shifted in super-steps
bool sep3d_big_supported(int nx, int ny, int nz, int rx, int ry, int rz, const void *in, const void *out);
cudaError_t launch_sep3d_big(const float *in, float *out, int nx, int ny, int nz, int rx, int ry, int rz,
                             const float *wx, const float *wy, const float *wz, int zchunk, int variant, cudaStream_t st);
// kern [device]: (2r+1)^3 weights, x fastest
cudaError_t launch_conv3d(const float *in, float *out, int nx, int ny, int nz, int r, const float *kern,
                          cudaStream_t st);


// Quality diagnostics (Eq. 12-18): masked sums and cube statistics over a ROI, 8 doubles out.
cudaError_t launch_mask_sums(const float *o, const float *f, const float *m, int nx, int ny, const int roi[6],
                             float thr_o, float thr_f, double *out, cudaStream_t st);
cudaError_t launch_cube_stats(const float *cube, int nx, int ny, const int roi[6], double *out, cudaStream_t st);
cudaError_t launch_histogram(const float *cube, int nx, int ny, const int roi[6], float lo, float hi, int nbins,
                             const float *mask_thr, unsigned long long *counts, cudaStream_t st);


// Wavelet lifting (section 3.4, Eq. 8-11): in-place transform and hard thresholding.
cudaError_t launch_wavelet_transform(float *a, int nx, int ny, int nz, int wavelet, int levels, bool inverse,
                                     bool two_phase, cudaStream_t st, int *launches);
cudaError_t launch_haar_filter(const float *in, float *out, int nx, int ny, int nz, int levels, const float *thr,
                               bool warp_blocks, bool *used_warp, cudaStream_t st);
// idg_legall.cu: Le Gall 5/3 thresholding filter with the axes of a level fused (needs ~1.3 cubes of temporary;
// cudaErrorMemoryAllocation with nothing launched when there is no room).
cudaError_t launch_legall_filter(const float *in, float *out, int nx, int ny, int nz, int levels, const float *thr,
                                 cudaStream_t st, int *launches);
cudaError_t launch_wavelet_threshold(float *a, int nx, int ny, int nz, int levels, const float *thr, cudaStream_t st);

}  // namespace idg
