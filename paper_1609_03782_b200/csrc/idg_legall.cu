// Le Gall 5/3 wavelet thresholding filter with the three axes of a level fused (section 3.4,
// Eq. 8 and 10 with P = (even_i + even_{i+1}) / 2, U = (d_{i-1} + d_i) / 4; readings W1-W5).
//
// The in-place passes of idg_wavelet.cu move the cube through HBM once per (level, axis, direction).  Here a
// CTA stages a 32 x 16 x 32 tile of the level's lattice plus the 3 extra samples per axis that the two lifting
// steps reach (forward: 2 below, 1 above; inverse: 1 below, 2 above) -- ONE cp.async.bulk.tensor box of
// 40 x 19 x 35 floats starting 4 samples left of the tile (TMA wants the innermost start coordinate on a
// 16-byte boundary), zero-filled outside the lattice; plain loads when the lattice is not TMA-addressable --
// lifts along x, y and z with one thread per line holding the line in registers, and writes the tile: one read
// and one write of the lattice per level and direction.  Halo samples are recomputed by the neighbouring CTA,
// so source and destination must differ; the levels therefore work on COMPACT lattices in a stream-ordered
// temporary:
//
//   forward  level l:  C_{l-1} (compact lattice, C_0 = the cube)  ->  T_l (all coefficients of the level)
//                                                                     C_l (its approximation band, compact)
//   inverse  level l:  T_l, hard-thresholded on load (details with t_l; the approximation band with t_L at the
//                      deepest level, untouched otherwise)  ->  the all-even positions of T_{l-1}, or `out`
//
// Every sample goes through the same fp32 operations in the same order as in idg_lift_kernel (x, then y, then
// z; predict, then update), so the result is bit-identical to the in-place path (test_gpu_wavelet.py).
#include <cuda.h>

#include <cstring>

#include "idg_kernels.cuh"
#include "idg_ptx.cuh"

namespace idg {

namespace {

constexpr int FX = 32, FY = 16, FZ = 32;                    // interior tile, lattice samples (all even)
constexpr int EY = FY + 3, EZ = FZ + 3;                     // with the lifting halo (x: see PX)
constexpr int PX = 40, XO = 4;                              // staged row: samples x0 - XO .. x0 - XO + PX - 1
constexpr int PP = PX * EY;                                 // plane pitch
constexpr int FNT = 256;
constexpr uint32_t kTileBytes = (uint32_t)(EZ * PP * sizeof(float));
constexpr size_t kSmem = kTileBytes + 16;                   // + the mbarrier

struct LArgs {
    const float *src;          // forward: lattice of the level (compact);  inverse: coefficients T_l
    float *full;               // forward: T_l;  inverse: destination (dense `out`, or T_{l-1} with stride 2)
    float *coarse_out;         // forward: C_l (compact approximation band) or nullptr at the deepest level
    int mx, my, mz;            // lattice extents of the level
    int ox, oy, os;            // inverse: x, y extents of the destination and its index stride (1 or 2)
    float thr_d, thr_a;        // inverse: hard thresholds for details / approximations (0 = none)
};

// One lifting step pair on a line segment held in registers.  v[l] is sample g = a0 - 2 + l of a line of m
// samples (a0 even, so the parity of g is the parity of l); outputs are valid for l = 2 .. T+1.  EDGE = false:
// the segment lies strictly inside the line (a0 > 0 and a0 + T < m), no symmetric extension to select.
template <int T, int OFF, bool EDGE, int NV>
__device__ __forceinline__ void fwd_steps(float (&w)[NV], int a0, int m)
{
    float *v = w + OFF;                                     // static indices after unrolling: stays in registers
#pragma unroll
    for (int l = 1; l <= T + 1; l += 2) {                   // predict (Eq. 8): d = odd - (e_i + e_{i+1}) / 2
        const int g = a0 - 2 + l;
        const float e1 = (!EDGE || g + 1 < m) ? v[l + 1] : v[l - 1];
        v[l] = v[l] - 0.5f * (v[l - 1] + e1);
    }
#pragma unroll
    for (int l = 2; l <= T; l += 2) {                       // update (Eq. 10): c = even + (d_{i-1} + d_i) / 4
        const int g = a0 - 2 + l;
        const float dr = (!EDGE || g + 1 < m) ? v[l + 1] : v[l - 1];
        const float dl = (!EDGE || g > 0) ? v[l - 1] : dr;
        v[l] = v[l] + 0.25f * (dl + dr);
    }
}
template <int T, int OFF, int NV>
__device__ __forceinline__ void fwd_line(float (&w)[NV], int a0, int m)
{
    static_assert(NV >= OFF + T + 3, "segment too short");
    if (m < 2) return;
    if (a0 > 0 && a0 + T < m) fwd_steps<T, OFF, false>(w, a0, m);
    else fwd_steps<T, OFF, true>(w, a0, m);
}

// Inverse: v[l] is sample g = a0 - 1 + l (even g <-> odd l); outputs are valid for l = 1 .. T.  EDGE = false
// when a0 > 0 and a0 + T + 1 < m.
template <int T, int OFF, bool EDGE, int NV>
__device__ __forceinline__ void inv_steps(float (&w)[NV], int a0, int m)
{
    float *v = w + OFF;
#pragma unroll
    for (int l = 1; l <= T + 1; l += 2) {                   // undo the update
        const int g = a0 - 1 + l;
        const float dr = (!EDGE || g + 1 < m) ? v[l + 1] : v[l - 1];
        const float dl = (!EDGE || g > 0) ? v[l - 1] : dr;
        v[l] = v[l] - 0.25f * (dl + dr);
    }
#pragma unroll
    for (int l = 2; l <= T; l += 2) {                       // undo the predict
        const int g = a0 - 1 + l;
        const float e1 = (!EDGE || g + 1 < m) ? v[l + 1] : v[l - 1];
        v[l] = v[l] + 0.5f * (v[l - 1] + e1);
    }
}
template <int T, int OFF, int NV>
__device__ __forceinline__ void inv_line(float (&w)[NV], int a0, int m)
{
    static_assert(NV >= OFF + T + 3, "segment too short");
    if (m < 2) return;
    if (a0 > 0 && a0 + T + 1 < m) inv_steps<T, OFF, false>(w, a0, m);
    else inv_steps<T, OFF, true>(w, a0, m);
}

// Stage the box [bx, bx+40) x [by, by+19) x [bz, bz+35) of the lattice, zeros outside (bx a multiple of 4).
template <bool TMA>
__device__ __forceinline__ void stage_tile(float *sm, const LArgs &A, const CUtensorMap *map, int bx, int by, int bz)
{
    if (TMA) {
        const uint32_t bar = ptx::smem_u32(sm) + kTileBytes;
        if (threadIdx.x == 0) {
            ptx::mbar_init(bar, 1);
            ptx::mbar_fence_init();
            ptx::mbar_expect_tx(bar, kTileBytes);
            ptx::tma_load_4d(ptx::smem_u32(sm), map, bar, bx, by, bz, 0);
        }
        __syncthreads();                                    // the barrier is initialised before anyone polls it
        ptx::mbar_wait(bar, 0);
    } else {
        const long long plane = (long long)A.mx * A.my;
        for (int p = threadIdx.x; p < PX * EY; p += FNT) {  // a thread walks one (x, y) column along z
            const int lx = p % PX, ly = p / PX;
            const int gx = bx + lx, gy = by + ly;
            const bool ok = gx >= 0 && gx < A.mx && gy >= 0 && gy < A.my;
            const float *q = A.src + (ok ? (long long)gy * A.mx + gx : 0);
            float *s = sm + ly * PX + lx;
#pragma unroll 7
            for (int lz = 0; lz < EZ; ++lz) {
                const int gz = bz + lz;
                s[lz * PP] = (ok && gz >= 0 && gz < A.mz) ? q[gz * plane] : 0.f;
            }
        }
        __syncthreads();
    }
}

// A complete row of the staged tile <-> registers, as ten 16-byte accesses.  The row pitch is an even number of
// 16-byte quads, so rows R and R + 4 start in the same bank group: threads whose row has bit 2 set touch the
// quads of each pair in the opposite order (q ^ 1), which makes the eight lanes of a phase hit distinct banks.
__device__ __forceinline__ void load_row(float (&v)[PX], const float *row, bool swap)
{
#pragma unroll
    for (int q = 0; q < PX / 4; q += 2) {
        const float4 a = reinterpret_cast<const float4 *>(row)[swap ? q + 1 : q];
        const float4 b = reinterpret_cast<const float4 *>(row)[swap ? q : q + 1];
        v[4 * q + 0] = swap ? b.x : a.x; v[4 * q + 1] = swap ? b.y : a.y;
        v[4 * q + 2] = swap ? b.z : a.z; v[4 * q + 3] = swap ? b.w : a.w;
        v[4 * q + 4] = swap ? a.x : b.x; v[4 * q + 5] = swap ? a.y : b.y;
        v[4 * q + 6] = swap ? a.z : b.z; v[4 * q + 7] = swap ? a.w : b.w;
    }
}
__device__ __forceinline__ void store_row(float *row, const float (&v)[PX], bool swap)
{
#pragma unroll
    for (int q = 0; q < PX / 4; q += 2) {
        const float4 lo = make_float4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
        const float4 hi = make_float4(v[4 * q + 4], v[4 * q + 5], v[4 * q + 6], v[4 * q + 7]);
        reinterpret_cast<float4 *>(row)[swap ? q + 1 : q] = swap ? hi : lo;
        reinterpret_cast<float4 *>(row)[swap ? q : q + 1] = swap ? lo : hi;
    }
}

template <bool TMA>
__global__ void __launch_bounds__(FNT, 2) idg_legall_fwd_kernel(const __grid_constant__ LArgs A,
                                                                const __grid_constant__ CUtensorMap map)
{
    extern __shared__ __align__(128) float sm[];            // [EZ][EY][PX]
    const int x0 = blockIdx.x * FX, y0 = blockIdx.y * FY, z0 = blockIdx.z * FZ;
    stage_tile<TMA>(sm, A, &map, x0 - XO, y0 - 2, z0 - 2);
    // x lines: one thread per (y, z) row of the staged tile
    for (int r = threadIdx.x; r < EY * EZ; r += FNT) {
        float v[PX];
        const bool swap = (r & 4) != 0;
        load_row(v, sm + r * PX, swap);
        fwd_line<FX, XO - 2>(v, x0, A.mx);
        store_row(sm + r * PX, v, swap);
    }
    __syncthreads();
    // y lines: (interior x, every z)
    for (int t = threadIdx.x; t < FX * EZ; t += FNT) {
        float v[EY];
        float *col = sm + (t / FX) * PP + XO + (t % FX);
#pragma unroll
        for (int l = 0; l < EY; ++l) v[l] = col[l * PX];
        fwd_line<FY, 0>(v, y0, A.my);
#pragma unroll
        for (int l = 2; l <= FY + 1; ++l) col[l * PX] = v[l];
    }
    __syncthreads();
    // z lines: (interior x, interior y); results go straight to global memory
    const long long plane = (long long)A.mx * A.my;
    const int cmx = (A.mx + 1) / 2, cmy = (A.my + 1) / 2;
    for (int t = threadIdx.x; t < FX * FY; t += FNT) {
        const int gx = x0 + (t % FX), gy = y0 + (t / FX);
        float v[EZ];
        const float *col = sm + (2 + t / FX) * PX + XO + (t % FX);
#pragma unroll
        for (int l = 0; l < EZ; ++l) v[l] = col[l * PP];
        fwd_line<FZ, 0>(v, z0, A.mz);
        if (gx >= A.mx || gy >= A.my) continue;
        float *o = A.full + (long long)gy * A.mx + gx + (long long)z0 * plane;
        const bool to_coarse = A.coarse_out != nullptr && ((gx | gy) & 1) == 0;
        const long long cplane = (long long)cmx * cmy;
        float *oc = A.coarse_out + (long long)(gy >> 1) * cmx + (gx >> 1) + (long long)(z0 >> 1) * cplane;
        if (z0 + FZ <= A.mz) {                              // the tile ends inside the lattice: no z guards
#pragma unroll
            for (int l = 0; l < FZ; ++l) o[l * plane] = v[l + 2];
            if (to_coarse) {
#pragma unroll
                for (int l = 0; l < FZ; l += 2) oc[(l >> 1) * cplane] = v[l + 2];
            }
        } else {
#pragma unroll
            for (int l = 0; l < FZ; ++l)
                if (z0 + l < A.mz) {
                    o[l * plane] = v[l + 2];
                    if (to_coarse && (l & 1) == 0) oc[(l >> 1) * cplane] = v[l + 2];
                }
        }
    }
}

template <bool TMA>
__global__ void __launch_bounds__(FNT, 2) idg_legall_inv_kernel(const __grid_constant__ LArgs A,
                                                                const __grid_constant__ CUtensorMap map)
{
    extern __shared__ __align__(128) float sm[];            // [EZ][EY][PX]
    const int x0 = blockIdx.x * FX, y0 = blockIdx.y * FY, z0 = blockIdx.z * FZ;
    stage_tile<TMA>(sm, A, &map, x0 - XO, y0 - 1, z0 - 1);
    // z lines: hard thresholds by band as the column is read (reading W3), then the inverse lifting
    for (int p = threadIdx.x; p < PX * EY; p += FNT) {      // every staged column: a warp never straddles rows
        const int lx = p % PX, ly = p / PX;
        const bool even_xy = (((x0 - XO + lx) | (y0 - 1 + ly)) & 1) == 0;
        float *col = sm + ly * PX + lx;
        float v[EZ];
#pragma unroll
        for (int l = 0; l < EZ; ++l) {
            const float a = col[l * PP];                    // even z <-> odd l
            const float thr = (even_xy && (l & 1) == 1) ? A.thr_a : A.thr_d;
            v[l] = fabsf(a) < thr ? 0.f : a;
        }
        inv_line<FZ, 0>(v, z0, A.mz);
#pragma unroll
        for (int l = 1; l <= FZ; ++l) col[l * PP] = v[l];
    }
    __syncthreads();
    // y lines: (every x, interior z)
    // (columns 0 .. 31 of a plane by one warp, then columns 32 .. 39 of four planes: conflict-free both ways)
    for (int t = threadIdx.x; t < PX * FZ; t += FNT) {
        float v[EY];
        const int lx = t < 32 * FZ ? t % 32 : 32 + t % 8, lz = t < 32 * FZ ? t / 32 : (t - 32 * FZ) / 8;
        float *col = sm + (1 + lz) * PP + lx;
#pragma unroll
        for (int l = 0; l < EY; ++l) v[l] = col[l * PX];
        inv_line<FY, 0>(v, y0, A.my);
#pragma unroll
        for (int l = 1; l <= FY; ++l) col[l * PX] = v[l];
    }
    __syncthreads();
    // x lines: (interior y, interior z)
    for (int r = threadIdx.x; r < FY * FZ; r += FNT) {
        float v[PX];
        const int R = (1 + r / FY) * EY + 1 + r % FY;      // row index in the staged tile
        float *row = sm + R * PX;
        const bool swap = (R & 4) != 0;
        load_row(v, row, swap);
        inv_line<FX, XO - 1>(v, x0, A.mx);
        store_row(row, v, swap);
    }
    __syncthreads();
    // coalesced write of the interior: dense (16-byte stores when the rows allow), or onto the all-even
    // positions of the next finer level
    const long long oplane = (long long)A.ox * A.oy;
    if (A.os == 1 && (A.ox & 3) == 0 && ((uintptr_t)A.full & 15u) == 0) {
        const int q = threadIdx.x % (FX / 4), gx = x0 + 4 * q;            // ox % 4 == 0: a quad is inside or outside
        const int nzv = min(FZ, A.mz - z0), nyv = min(FY, A.my - y0);
        if (gx < A.mx) {
            float *o = A.full + (long long)y0 * A.ox + gx + (long long)z0 * oplane;
            const float *s = sm + PP + PX + XO + 4 * q;
#pragma unroll 4
            for (int r = threadIdx.x / (FX / 4); r < FY * FZ; r += FNT / (FX / 4)) {       // r = (lz, ly)
                const int ly = r % FY, lz = r / FY;
                if (ly < nyv && lz < nzv)
                    *reinterpret_cast<float4 *>(o + lz * oplane + (long long)ly * A.ox) =
                        *reinterpret_cast<const float4 *>(s + lz * PP + ly * PX);
            }
        }
    } else {
        const int lx = threadIdx.x % FX, gx = x0 + lx;
        if (gx < A.mx) {
            for (int ly = threadIdx.x / FX; ly < FY; ly += FNT / FX) {
                const int gy = y0 + ly;
                if (gy >= A.my) break;
                float *o = A.full + ((long long)gy * A.ox + gx + (long long)z0 * oplane) * A.os;
                const float *s = sm + PP + (1 + ly) * PX + XO + lx;
                const int nzv = min(FZ, A.mz - z0);
#pragma unroll 8
                for (int lz = 0; lz < nzv; ++lz) o[lz * A.os * oplane] = s[lz * PP];
            }
        }
    }
}

inline size_t align64(size_t n) { return (n + 63) & ~(size_t)63; }       // floats: 256-byte sub-buffers

template <bool TMA>
cudaError_t launch_level(bool inverse, const LArgs &A, const CUtensorMap &map, cudaStream_t st)
{
    auto k = inverse ? idg_legall_inv_kernel<TMA> : idg_legall_fwd_kernel<TMA>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmem);
    if (e != cudaSuccess) return e;
    const dim3 grid((unsigned)((A.mx + FX - 1) / FX), (unsigned)((A.my + FY - 1) / FY), (unsigned)((A.mz + FZ - 1) / FZ));
    k<<<grid, FNT, kSmem, st>>>(A, map);
    return cudaGetLastError();
}

cudaError_t run_level(bool inverse, const LArgs &A, cudaStream_t st)
{
    CUtensorMap map;
    const bool tma = A.mx % 4 == 0 && ((uintptr_t)A.src & 15u) == 0 && tmap_available() &&
                     tmap_encode(&map, A.src, A.mx, A.my, A.mz, 1, PX, EY, EZ);
    if (tma) return launch_level<true>(inverse, A, map, st);
    memset(&map, 0, sizeof(map));
    return launch_level<false>(inverse, A, map, st);
}

}  // namespace

// Le Gall 5/3 thresholding filter, `levels` <= 16, thr[l-1] = t_l * rms.  Allocates ~1.3 cubes of stream-ordered
// temporary; returns cudaErrorMemoryAllocation (nothing launched) when that fails so the caller can fall back
// to the in-place passes.  in == out is allowed.
cudaError_t launch_legall_filter(const float *in, float *out, int nx, int ny, int nz, int levels, const float *thr,
                                 cudaStream_t st, int *launches)
{
    if (levels < 1 || levels > 16) return cudaErrorInvalidValue;
    int mx[18], my[18], mz[18];
    size_t M[18];
    mx[0] = nx; my[0] = ny; mz[0] = nz;
    for (int l = 0; l <= levels; ++l) {
        if (l > 0) { mx[l] = (mx[l - 1] + 1) / 2; my[l] = (my[l - 1] + 1) / 2; mz[l] = (mz[l - 1] + 1) / 2; }
        M[l] = (size_t)mx[l] * my[l] * (size_t)mz[l];
    }
    if ((mz[0] + FZ - 1) / FZ > 65535 || (my[0] + FY - 1) / FY > 65535) return cudaErrorInvalidValue;
    // temporary: T_l (size M[l-1]) for l = 1 .. levels and C_l (size M[l]) for l = 1 .. levels - 1
    size_t total = 0;
    for (int l = 1; l <= levels; ++l) total += align64(M[l - 1]) + (l < levels ? align64(M[l]) : 0);
    float *tmp = nullptr;
    cudaError_t e = temp_alloc((void **)&tmp, total * sizeof(float), st);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return cudaErrorMemoryAllocation; }
    float *T[17], *C[17];
    size_t off = 0;
    for (int l = 1; l <= levels; ++l) {
        T[l] = tmp + off; off += align64(M[l - 1]);
        C[l] = nullptr;
        if (l < levels) { C[l] = tmp + off; off += align64(M[l]); }
    }
    for (int l = 1; l <= levels && e == cudaSuccess; ++l) {
        LArgs A{l == 1 ? in : C[l - 1], T[l], C[l], mx[l - 1], my[l - 1], mz[l - 1], 0, 0, 1, 0.f, 0.f};
        e = run_level(false, A, st);
        ++*launches;
    }
    for (int l = levels; l >= 1 && e == cudaSuccess; --l) {
        LArgs A{T[l], l == 1 ? out : T[l - 1], nullptr, mx[l - 1], my[l - 1], mz[l - 1],
                l == 1 ? mx[0] : mx[l - 2], l == 1 ? my[0] : my[l - 2], l == 1 ? 1 : 2,
                thr[l - 1], l == levels ? thr[l - 1] : 0.f};
        e = run_level(true, A, st);
        ++*launches;
    }
    const cudaError_t ef = cudaFreeAsync(tmp, st);
    return e != cudaSuccess ? e : ef;
}

}  // namespace idg
