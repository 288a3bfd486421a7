// Masked reductions behind the paper's smoothing-quality diagnostics (Eq. 12-16;
// PAPER.md:344-355, Eq. 17-18) and the rms estimate of a cube (readings Q1-Q4):
//
//   M_i = [I_i >= thr_i]  (fp32 compare, Eq. 14);  S_oo = sum I_o M_o;  S_of = sum I_o M_f  (Eq. 13);
//   S_mf = sum I_m M_f;  S_m = sum I_m  (Eq. 18);  N_o, N_f = mask populations  (Eq. 16)
//
// over a half-open ROI box, in ONE pass over the two (three) cubes: a warp takes ROI rows, lanes read
// coalesced float4 where the row allows it, every thread accumulates in fp64, warps combine by
// shuffles and add their totals to the eight result doubles with one atomic each.  Bound by HBM
// reads: 8 B (12 B with a model cube) per ROI voxel.
#include "idg_kernels.cuh"

namespace idg {

namespace {

constexpr int NT = 256, WARPS = NT / 32;

struct QArgs {
    const float *o, *f, *m;      // original, filtered, model (may be null)
    int nx, ny;
    int x0, x1, y0, y1, z0, z1;  // ROI, half open
    float thr_o, thr_f;
    int vec;                     // rows are float4-addressable (nx % 4 == 0, 16-byte aligned bases)
    double *out;                 // 8 doubles
};

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}

struct Acc { double s_oo, s_of, s_mf, s_m, n_o, n_f; };

template <bool MODEL>
__device__ __forceinline__ void voxel(Acc &a, float o, float f, float m, float thr_o, float thr_f)
{
    const bool mo = o >= thr_o, mf = f >= thr_f;            // Eq. 14; NaN compares false
    if (mo) { a.s_oo += (double)o; a.n_o += 1.0; }
    if (mf) { a.s_of += (double)o; a.n_f += 1.0; }
    if (MODEL) {
        a.s_m += (double)m;
        if (mf) a.s_mf += (double)m;
    }
}

template <bool MODEL>
__global__ void __launch_bounds__(NT) idg_mask_sums_kernel(const __grid_constant__ QArgs Q)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int rows_y = Q.y1 - Q.y0;
    const long long rows = (long long)rows_y * (Q.z1 - Q.z0);
    Acc a{0, 0, 0, 0, 0, 0};
    for (long long r = (long long)blockIdx.x * WARPS + warp; r < rows; r += (long long)gridDim.x * WARPS) {
        const int z = Q.z0 + (int)(r / rows_y), y = Q.y0 + (int)(r % rows_y);
        const size_t base = ((size_t)z * Q.ny + y) * (size_t)Q.nx;
        int xa = Q.x0, xb = Q.x1;                           // scalar head [x0, xa), vector body [xa, xb), scalar tail
        if (Q.vec) { xa = min((Q.x0 + 3) & ~3, Q.x1); xb = max(xa, Q.x1 & ~3); } else { xa = xb = Q.x1; }
        for (int x = Q.x0 + lane; x < xa; x += 32)
            voxel<MODEL>(a, Q.o[base + x], Q.f[base + x], MODEL ? Q.m[base + x] : 0.f, Q.thr_o, Q.thr_f);
        for (int x = xa + 4 * lane; x < xb; x += 128) {
            const float4 o = *reinterpret_cast<const float4 *>(Q.o + base + x);
            const float4 f = *reinterpret_cast<const float4 *>(Q.f + base + x);
            float4 m = make_float4(0.f, 0.f, 0.f, 0.f);
            if (MODEL) m = *reinterpret_cast<const float4 *>(Q.m + base + x);
            voxel<MODEL>(a, o.x, f.x, m.x, Q.thr_o, Q.thr_f);
            voxel<MODEL>(a, o.y, f.y, m.y, Q.thr_o, Q.thr_f);
            voxel<MODEL>(a, o.z, f.z, m.z, Q.thr_o, Q.thr_f);
            voxel<MODEL>(a, o.w, f.w, m.w, Q.thr_o, Q.thr_f);
        }
        for (int x = xb + lane; x < Q.x1; x += 32)
            if (x >= xa) voxel<MODEL>(a, Q.o[base + x], Q.f[base + x], MODEL ? Q.m[base + x] : 0.f, Q.thr_o, Q.thr_f);
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) Q.out[6] = (double)rows * (double)(Q.x1 - Q.x0);     // n_roi
    const double v[6] = {warp_sum(a.s_oo), warp_sum(a.s_of), warp_sum(a.n_o), warp_sum(a.n_f), warp_sum(a.s_mf),
                         warp_sum(a.s_m)};
    if (lane == 0) {
#pragma unroll
        for (int i = 0; i < 6; ++i)
            if (v[i] != 0.0) atomicAdd(Q.out + i, v[i]);
    }
}

__global__ void __launch_bounds__(NT) idg_cube_stats_kernel(const __grid_constant__ QArgs Q)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int rows_y = Q.y1 - Q.y0;
    const long long rows = (long long)rows_y * (Q.z1 - Q.z0);
    double s1 = 0.0, s2 = 0.0;
    for (long long r = (long long)blockIdx.x * WARPS + warp; r < rows; r += (long long)gridDim.x * WARPS) {
        const int z = Q.z0 + (int)(r / rows_y), y = Q.y0 + (int)(r % rows_y);
        const size_t base = ((size_t)z * Q.ny + y) * (size_t)Q.nx;
        int xa, xb;
        if (Q.vec) { xa = min((Q.x0 + 3) & ~3, Q.x1); xb = max(xa, Q.x1 & ~3); } else { xa = xb = Q.x1; }
        for (int x = Q.x0 + lane; x < xa; x += 32) { const double v = Q.o[base + x]; s1 += v; s2 += v * v; }
        for (int x = xa + 4 * lane; x < xb; x += 128) {
            const float4 o = *reinterpret_cast<const float4 *>(Q.o + base + x);
            const double a = o.x, b = o.y, c = o.z, d = o.w;
            s1 += (a + b) + (c + d);
            s2 += (a * a + b * b) + (c * c + d * d);
        }
        for (int x = xb + lane; x < Q.x1; x += 32)
            if (x >= xa) { const double v = Q.o[base + x]; s1 += v; s2 += v * v; }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) Q.out[0] = (double)rows * (double)(Q.x1 - Q.x0);     // n
    s1 = warp_sum(s1);
    s2 = warp_sum(s2);
    if (lane == 0) {
        atomicAdd(Q.out + 1, s1);
        atomicAdd(Q.out + 2, s2);
    }
}

// Intensity histogram of a ROI (Fig. 6; reading Q5): nbins equal bins over [lo, hi), bin
// decided in fp32 as floor((v - lo) * scale) with scale = nbins / (hi - lo) rounded to fp32 on the host (no FMA
// contraction, so that the integer decision is the oracle's), per-CTA counts in shared memory, merged with one
// 64-bit atomic per non-empty bin.
struct HistArgs {
    const float *a;
    int nx, ny;
    int x0, x1, y0, y1, z0, z1;
    float lo, hi, scale, thr;
    int use_thr, nbins;
    unsigned long long *counts;
};

__global__ void __launch_bounds__(NT) idg_histogram_kernel(const __grid_constant__ HistArgs H)
{
    extern __shared__ unsigned hist[];
    for (int b = threadIdx.x; b < H.nbins; b += NT) hist[b] = 0u;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int rows_y = H.y1 - H.y0;
    const long long rows = (long long)rows_y * (H.z1 - H.z0);
    for (long long r = (long long)blockIdx.x * WARPS + warp; r < rows; r += (long long)gridDim.x * WARPS) {
        const int z = H.z0 + (int)(r / rows_y), y = H.y0 + (int)(r % rows_y);
        const float *row = H.a + ((size_t)z * H.ny + y) * (size_t)H.nx;
        for (int x = H.x0 + lane; x < H.x1; x += 32) {
            const float v = row[x];
            if (v >= H.lo && v < H.hi && (!H.use_thr || v >= H.thr)) {
                int b = (int)floorf(__fmul_rn(__fsub_rn(v, H.lo), H.scale));
                b = b < H.nbins - 1 ? b : H.nbins - 1;
                atomicAdd(&hist[b], 1u);
            }
        }
    }
    __syncthreads();
    for (int b = threadIdx.x; b < H.nbins; b += NT)
        if (hist[b]) atomicAdd(H.counts + b, (unsigned long long)hist[b]);
}

unsigned grid_for(long long rows)
{
    long long g = (rows + WARPS - 1) / WARPS;
    const long long cap = (long long)device_sm_count() * 8;                         // 8 CTAs of 256 threads per SM
    if (g > cap) g = cap;
    return (unsigned)(g < 1 ? 1 : g);
}

}  // namespace

// roi = {x0, x1, y0, y1, z0, z1} (validated by the caller); out [device] 8 doubles, zeroed here.
cudaError_t launch_mask_sums(const float *o, const float *f, const float *m, int nx, int ny, const int roi[6],
                             float thr_o, float thr_f, double *out, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(out, 0, 8 * sizeof(double), st);
    if (e != cudaSuccess) return e;
    QArgs Q{o, f, m, nx, ny, roi[0], roi[1], roi[2], roi[3], roi[4], roi[5], thr_o, thr_f, 0, out};
    const uintptr_t al = (uintptr_t)o | (uintptr_t)f | (uintptr_t)(m ? m : o);
    Q.vec = (nx % 4 == 0 && (al & 15u) == 0) ? 1 : 0;
    const long long rows = (long long)(roi[3] - roi[2]) * (roi[5] - roi[4]);
    if (rows <= 0 || roi[1] <= roi[0]) return cudaSuccess;   // empty ROI: all sums zero
    if (m) idg_mask_sums_kernel<true><<<grid_for(rows), NT, 0, st>>>(Q);
    else idg_mask_sums_kernel<false><<<grid_for(rows), NT, 0, st>>>(Q);
    return cudaGetLastError();
}

// counts [device] nbins 64-bit counters, zeroed here.  A CTA sees fewer than 2^32 voxels (grid-stride over rows).
cudaError_t launch_histogram(const float *cube, int nx, int ny, const int roi[6], float lo, float hi, int nbins,
                             const float *mask_thr, unsigned long long *counts, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(counts, 0, (size_t)nbins * sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    HistArgs H{cube, nx, ny, roi[0], roi[1], roi[2], roi[3], roi[4], roi[5], lo, hi, (float)nbins / (hi - lo),
               mask_thr ? *mask_thr : 0.f, mask_thr ? 1 : 0, nbins, counts};
    const long long rows = (long long)(roi[3] - roi[2]) * (roi[5] - roi[4]);
    if (rows <= 0 || roi[1] <= roi[0]) return cudaSuccess;
    idg_histogram_kernel<<<grid_for(rows), NT, (size_t)nbins * sizeof(unsigned), st>>>(H);
    return cudaGetLastError();
}

cudaError_t launch_cube_stats(const float *cube, int nx, int ny, const int roi[6], double *out, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(out, 0, 8 * sizeof(double), st);
    if (e != cudaSuccess) return e;
    QArgs Q{cube, cube, nullptr, nx, ny, roi[0], roi[1], roi[2], roi[3], roi[4], roi[5], 0.f, 0.f, 0, out};
    Q.vec = (nx % 4 == 0 && ((uintptr_t)cube & 15u) == 0) ? 1 : 0;
    const long long rows = (long long)(roi[3] - roi[2]) * (roi[5] - roi[4]);
    if (rows <= 0 || roi[1] <= roi[0]) return cudaSuccess;
    idg_cube_stats_kernel<<<grid_for(rows), NT, 0, st>>>(Q);
    return cudaGetLastError();
}

}  // namespace idg
