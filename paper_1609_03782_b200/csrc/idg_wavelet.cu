// Wavelet lifting and the wavelet thresholding filter (section 3.4, Eq. 8-11), fp32,
// in place ("does not require additional memory"): after level l the approximation
// coefficients c sit on the lattice of points whose three indices are multiples of 2^l, the details d on
// the rest of the level-l lattice (readings W1-W5).
//
//   predict  d_i = odd_i - P(even)      Haar: P = even_i             Le Gall 5/3: P = (even_i + even_{i+1}) / 2
//   update   c_i = even_i + U(d)        Haar: U = d_i / 2            Le Gall 5/3: U = (d_{i-1} + d_i) / 4
//
// One kernel launch per (level, axis, phase): a thread owns one target sample (an odd one in the
// predict phase, an even one in the update phase), so a phase only reads samples the phase does not
// write.  Threads are laid out with the lattice x index fastest.  The threshold pass is one more
// elementwise kernel (band level from the trailing zero bits of the indices).  All of it is bound by
// HBM traffic; level 1 dominates (the level-l lattice holds 8^-(l-1) of the voxels).
#include <type_traits>

#include "idg_kernels.cuh"

namespace idg {

namespace {

constexpr int NT = 256;

struct WArgs {
    float *a;
    int nx, ny, nz;
    int s;              // lattice stride 2^(l-1)
    int axis;           // 0 x, 1 y, 2 z
    int mx, my, mz;     // lattice extents ceil(n / s)
};

// PHASE 0: predict (targets = odd samples), 1: update (targets = even samples); INV undoes the phase.
template <int WAVELET, int PHASE, bool INV>
__global__ void __launch_bounds__(NT) idg_lift_kernel(const __grid_constant__ WArgs W)
{
    const int m = W.axis == 0 ? W.mx : (W.axis == 1 ? W.my : W.mz);       // samples on a line
    const int no = m / 2, ne = m - no;
    const int nt = PHASE == 0 ? no : ne;                                  // targets on a line
    // thread -> (target i along the axis, lattice coordinates of the other two axes), x fastest
    const int ex = W.axis == 0 ? nt : W.mx, ey = W.axis == 1 ? nt : W.my, ez = W.axis == 2 ? nt : W.mz;
    const long long total = (long long)ex * ey * ez;
    const size_t sx = (size_t)W.s, sy = (size_t)W.s * W.nx, sz = (size_t)W.s * W.nx * (size_t)W.ny;
    const size_t st = W.axis == 0 ? sx : (W.axis == 1 ? sy : sz);         // stride between line samples
    for (long long t = (long long)blockIdx.x * NT + threadIdx.x; t < total; t += (long long)gridDim.x * NT) {
        const int cx = (int)(t % ex), cy = (int)((t / ex) % ey), cz = (int)(t / ((long long)ex * ey));
        const int i = W.axis == 0 ? cx : (W.axis == 1 ? cy : cz);
        float *line = W.a + (W.axis == 0 ? 0 : (size_t)cx * sx) + (W.axis == 1 ? 0 : (size_t)cy * sy) +
                      (W.axis == 2 ? 0 : (size_t)cz * sz);
        if (PHASE == 0) {
            const float e0 = line[(size_t)(2 * i) * st];
            float p = e0;
            if (WAVELET == 1) {
                const float e1 = (i + 1 < ne) ? line[(size_t)(2 * i + 2) * st] : e0;      // reading W4
                p = 0.5f * (e0 + e1);
            }
            float *d = line + (size_t)(2 * i + 1) * st;
            *d = INV ? *d + p : *d - p;                                   // Eq. 8
        } else {
            float u;
            if (WAVELET == 0) {
                if (i >= no) continue;                                    // unpaired last even sample (W2)
                u = 0.5f * line[(size_t)(2 * i + 1) * st];                // Eq. 11
            } else {
                const float dr = (i < no) ? line[(size_t)(2 * i + 1) * st] : line[(size_t)(2 * i - 1) * st];
                const float dl = (i > 0) ? line[(size_t)(2 * i - 1) * st] : dr;
                u = 0.25f * (dl + dr);
            }
            float *c = line + (size_t)(2 * i) * st;
            *c = INV ? *c - u : *c + u;                                   // Eq. 10
        }
    }
}

// Haar only: predict and update of one (even, odd) pair touch nothing but the pair (Eq. 8-11 with P = even_i,
// U = d_i / 2), so both phases run in one race-free in-place pass with a thread per pair; same operations in
// the same order as the two-phase kernel.
template <bool INV>
__global__ void __launch_bounds__(NT) idg_haar_pair_kernel(const __grid_constant__ WArgs W)
{
    const int m = W.axis == 0 ? W.mx : (W.axis == 1 ? W.my : W.mz);
    const int no = m / 2;
    const int ex = W.axis == 0 ? no : W.mx, ey = W.axis == 1 ? no : W.my, ez = W.axis == 2 ? no : W.mz;
    const long long total = (long long)ex * ey * ez;
    const size_t sx = (size_t)W.s, sy = (size_t)W.s * W.nx, sz = (size_t)W.s * W.nx * (size_t)W.ny;
    const size_t st = W.axis == 0 ? sx : (W.axis == 1 ? sy : sz);
    for (long long t = (long long)blockIdx.x * NT + threadIdx.x; t < total; t += (long long)gridDim.x * NT) {
        const int cx = (int)(t % ex), cy = (int)((t / ex) % ey), cz = (int)(t / ((long long)ex * ey));
        const int i = W.axis == 0 ? cx : (W.axis == 1 ? cy : cz);
        float *line = W.a + (W.axis == 0 ? 0 : (size_t)cx * sx) + (W.axis == 1 ? 0 : (size_t)cy * sy) +
                      (W.axis == 2 ? 0 : (size_t)cz * sz);
        float *pe = line + (size_t)(2 * i) * st, *po = pe + st;
        float e = *pe, o = *po;
        if (!INV) { o = o - e; e = e + 0.5f * o; }          // d = odd - even;  c = even + d/2
        else { e = e - 0.5f * o; o = o + e; }               // even = c - d/2;  odd = d + even
        *pe = e;
        *po = o;
    }
}

struct TArgs {
    float *a;
    int nx, ny, nz, levels;
    float thr[16];      // t_l * rms
};

// Hard threshold (reading W3): band level = 1 + min trailing zeros of (x, y, z), capped at `levels`.
__global__ void __launch_bounds__(NT) idg_wavelet_threshold_kernel(const __grid_constant__ TArgs T)
{
    const size_t N = (size_t)T.nx * T.ny * (size_t)T.nz;
    for (size_t i = (size_t)blockIdx.x * NT + threadIdx.x; i < N; i += (size_t)gridDim.x * NT) {
        const int x = (int)(i % (size_t)T.nx), y = (int)((i / (size_t)T.nx) % (size_t)T.ny),
                  z = (int)(i / ((size_t)T.nx * T.ny));
        const int tz = __ffs(x | y | z | (1 << 30)) - 1;                  // min of the three trailing-zero counts
        const int l = tz + 1 < T.levels ? tz + 1 : T.levels;
        const float v = T.a[i];
        if (fabsf(v) < T.thr[l - 1]) T.a[i] = 0.f;
    }
}

// ---- whole lines in shared memory: predict + update of one axis in ONE in-place pass ----------------------
// A CTA that holds complete lines can run both lifting phases without another CTA touching its samples, so the
// pass is race-free in place (what the two-phase kernels buy with a second launch).  x lines: one warp per
// line.  y / z lines: a CTA takes 32 neighbouring lattice columns (lane = column, coalesced for level 1) and
// the full line of each.  Same operations in the same order as idg_lift_kernel.
template <int WAVELET, bool INV>
__device__ __forceinline__ void lift_line_smem(float *v, int m, int stride, int first, int step, bool block_sync)
{
    // v[j * stride]: sample j of the line; this thread handles pair / even indices first, first+step, ...
    const int no = m / 2, ne = m - no;
    auto sync = [&]() { if (block_sync) __syncthreads(); else __syncwarp(); };
    auto predict = [&]() {
        for (int i = first; i < no; i += step) {
            const float e0 = v[(2 * i) * stride];
            float p = e0;
            if (WAVELET == 1) p = 0.5f * (e0 + ((i + 1 < ne) ? v[(2 * i + 2) * stride] : e0));
            float &d = v[(2 * i + 1) * stride];
            d = INV ? d + p : d - p;
        }
    };
    auto update = [&]() {
        for (int i = first; i < ne; i += step) {
            float u;
            if (WAVELET == 0) {
                if (i >= no) continue;
                u = 0.5f * v[(2 * i + 1) * stride];
            } else {
                const float dr = (i < no) ? v[(2 * i + 1) * stride] : v[(2 * i - 1) * stride];
                const float dl = (i > 0) ? v[(2 * i - 1) * stride] : dr;
                u = 0.25f * (dl + dr);
            }
            float &c = v[(2 * i) * stride];
            c = INV ? c - u : c + u;
        }
    };
    if (!INV) { predict(); sync(); update(); } else { update(); sync(); predict(); }
    sync();
}

constexpr int LW = 4;        // warps (= x lines) per CTA of the x-line kernel

template <int WAVELET, bool INV>
__global__ void __launch_bounds__(LW * 32) idg_lift_xline_kernel(const __grid_constant__ WArgs W)
{
    extern __shared__ float lsm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float *v = lsm + (size_t)warp * W.mx;
    const long long lines = (long long)W.my * W.mz;
    for (long long l = (long long)blockIdx.x * LW + warp; l < lines; l += (long long)gridDim.x * LW) {
        const int cy = (int)(l % W.my), cz = (int)(l / W.my);
        float *g = W.a + ((size_t)cz * W.s * W.ny + (size_t)cy * W.s) * (size_t)W.nx;
        for (int j = lane; j < W.mx; j += 32) v[j] = g[(size_t)j * W.s];
        __syncwarp();
        lift_line_smem<WAVELET, INV>(v, W.mx, 1, lane, 32, false);
        for (int j = lane; j < W.mx; j += 32) g[(size_t)j * W.s] = v[j];
        __syncwarp();
    }
}

// axis 1 (y) or 2 (z): strip of SW lattice-x columns, full lines; smem [m][SW]
constexpr int SW = 16;
template <int WAVELET, bool INV>
__global__ void __launch_bounds__(NT) idg_lift_strip_kernel(const __grid_constant__ WArgs W)
{
    extern __shared__ float lsm[];
    const int col = threadIdx.x % SW, row = threadIdx.x / SW;
    constexpr int ROWS = NT / SW;
    const int m = W.axis == 1 ? W.my : W.mz;                      // line length
    const int mo = W.axis == 1 ? W.mz : W.my;                     // lattice extent of the third axis
    const int strips = (W.mx + SW - 1) / SW;
    const size_t sline = W.axis == 1 ? (size_t)W.s * W.nx : (size_t)W.s * W.nx * (size_t)W.ny;     // along the line
    const size_t sother = W.axis == 1 ? (size_t)W.s * W.nx * (size_t)W.ny : (size_t)W.s * W.nx;    // third axis
    for (long long t = blockIdx.x; t < (long long)strips * mo; t += gridDim.x) {
        const int sx = (int)(t % strips), co = (int)(t / strips);
        const int cx = sx * SW + col;
        const bool on = cx < W.mx;
        float *g = W.a + (size_t)co * sother + (size_t)cx * W.s;
        if (on)
            for (int j = row; j < m; j += ROWS) lsm[j * SW + col] = g[(size_t)j * sline];
        __syncthreads();
        lift_line_smem<WAVELET, INV>(lsm + col, m, SW, row, ROWS, true);
        if (on)
            for (int j = row; j < m; j += ROWS) g[(size_t)j * sline] = lsm[j * SW + col];
        __syncthreads();
    }
}

// ---- Haar thresholding filter, up to 3 levels, in ONE pass ------------------------------------------------
// A Haar pair never leaves its 2-block, so the whole L-level transform of an 8 x 8 x 8 aligned block depends on
// that block only.  A CTA stages a 64 x 8 x 8 region in shared memory, runs forward levels 1..L (a thread per
// 2 x 2 x 2 lattice block: its four x pairs, then y pairs, then z pairs -- the same operations in the same order
// as the per-axis passes), thresholds, runs the inverse levels L..1 and writes the region back: the cube is read
// once and written once (8 B per voxel) instead of ~19 in-place passes.  Safe in place (out == cube).
struct HArgs {
    const float *in;
    float *out;
    int nx, ny, nz, levels;
    float thr[3];
};

constexpr int HX = 64, HY = 8, HZ = 8, HPAD = 65;            // region and padded row length (bank conflicts)

template <bool INV>
__device__ __forceinline__ void haar_pair(float &e, float &o)
{
    if (!INV) { o = o - e; e = e + 0.5f * o; }              // d = odd - even;  c = even + d/2   (Eq. 8-11)
    else { e = e - 0.5f * o; o = o + e; }
}

// One level (lattice stride s) of the region held in `sm`; gx0, gy0, gz0 = global origin of the region.
template <bool INV, int s>
__device__ __forceinline__ void haar_level(float *sm, int gx0, int gy0, int gz0, const HArgs &H)
{
    constexpr int bx = HX / (2 * s), by = HY / (2 * s), bz = HZ / (2 * s);
    const int mx = (H.nx + s - 1) / s, my = (H.ny + s - 1) / s, mz = (H.nz + s - 1) / s;     // lattice extents
    for (int t = threadIdx.x; t < bx * by * bz; t += NT) {
        const int ix = t % bx, iy = (t / bx) % by, iz = t / (bx * by);
        const int lx = 2 * s * ix, ly = 2 * s * iy, lz = 2 * s * iz;                       // local corner
        // does the odd partner exist on the global lattice? (reading W2: otherwise the even sample is left alone)
        const bool px = (gx0 + lx) / s + 1 < mx, py = (gy0 + ly) / s + 1 < my, pz = (gz0 + lz) / s + 1 < mz;
        // which of the 8 corners exist at all (even corners of an existing block always do)
        float v[2][2][2];
#pragma unroll
        for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int b = 0; b < 2; ++b)
#pragma unroll
                for (int a = 0; a < 2; ++a) v[c][b][a] = sm[((lz + c * s) * HY + ly + b * s) * HPAD + lx + a * s];
        auto xs = [&]() {
            if (px) {
#pragma unroll
                for (int c = 0; c < 2; ++c)
#pragma unroll
                    for (int b = 0; b < 2; ++b)
                        if ((c == 0 || pz) && (b == 0 || py)) haar_pair<INV>(v[c][b][0], v[c][b][1]);
            }
        };
        auto ys = [&]() {
            if (py) {
#pragma unroll
                for (int c = 0; c < 2; ++c)
#pragma unroll
                    for (int a = 0; a < 2; ++a)
                        if ((c == 0 || pz) && (a == 0 || px)) haar_pair<INV>(v[c][0][a], v[c][1][a]);
            }
        };
        auto zs = [&]() {
            if (pz) {
#pragma unroll
                for (int b = 0; b < 2; ++b)
#pragma unroll
                    for (int a = 0; a < 2; ++a)
                        if ((b == 0 || py) && (a == 0 || px)) haar_pair<INV>(v[0][b][a], v[1][b][a]);
            }
        };
        if (!INV) { xs(); ys(); zs(); } else { zs(); ys(); xs(); }
#pragma unroll
        for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int b = 0; b < 2; ++b)
#pragma unroll
                for (int a = 0; a < 2; ++a) sm[((lz + c * s) * HY + ly + b * s) * HPAD + lx + a * s] = v[c][b][a];
    }
}

__global__ void __launch_bounds__(NT) idg_haar_filter_kernel(const __grid_constant__ HArgs H)
{
    __shared__ float sm[HZ * HY * HPAD];
    const int gx0 = blockIdx.x * HX, gy0 = blockIdx.y * HY, gz0 = blockIdx.z * HZ;
    const size_t plane = (size_t)H.nx * H.ny;
    const bool vec = (H.nx % 4 == 0) && ((((uintptr_t)H.in | (uintptr_t)H.out) & 15u) == 0);
    if (vec) {
        for (int e = threadIdx.x; e < (HX / 4) * HY * HZ; e += NT) {
            const int x = 4 * (e % (HX / 4)), y = (e / (HX / 4)) % HY, z = e / ((HX / 4) * HY);
            const int gx = gx0 + x, gy = gy0 + y, gz = gz0 + z;
            float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
            if (gx < H.nx && gy < H.ny && gz < H.nz)
                v = *reinterpret_cast<const float4 *>(H.in + (size_t)gz * plane + (size_t)gy * H.nx + gx);
            float *p = sm + (z * HY + y) * HPAD + x;
            p[0] = v.x; p[1] = v.y; p[2] = v.z; p[3] = v.w;
        }
    } else {
        for (int e = threadIdx.x; e < HX * HY * HZ; e += NT) {
            const int x = e % HX, y = (e / HX) % HY, z = e / (HX * HY);
            const int gx = gx0 + x, gy = gy0 + y, gz = gz0 + z;
            sm[(z * HY + y) * HPAD + x] = (gx < H.nx && gy < H.ny && gz < H.nz) ? H.in[(size_t)gz * plane + (size_t)gy * H.nx + gx] : 0.f;
        }
    }
    __syncthreads();
    haar_level<false, 1>(sm, gx0, gy0, gz0, H);
    __syncthreads();
    if (H.levels >= 2) { haar_level<false, 2>(sm, gx0, gy0, gz0, H); __syncthreads(); }
    if (H.levels >= 3) { haar_level<false, 4>(sm, gx0, gy0, gz0, H); __syncthreads(); }
    for (int e = threadIdx.x; e < HX * HY * HZ; e += NT) {      // hard thresholds by band (reading W3)
        const int x = e % HX, y = (e / HX) % HY, z = e / (HX * HY);
        const int tz = __ffs((gx0 + x) | (gy0 + y) | (gz0 + z) | (1 << 30)) - 1;
        const int l = tz + 1 < H.levels ? tz + 1 : H.levels;
        float *p = sm + (z * HY + y) * HPAD + x;
        if (fabsf(*p) < H.thr[l - 1]) *p = 0.f;
    }
    __syncthreads();
    if (H.levels >= 3) { haar_level<true, 4>(sm, gx0, gy0, gz0, H); __syncthreads(); }
    if (H.levels >= 2) { haar_level<true, 2>(sm, gx0, gy0, gz0, H); __syncthreads(); }
    haar_level<true, 1>(sm, gx0, gy0, gz0, H);
    __syncthreads();
    if (vec) {
        for (int e = threadIdx.x; e < (HX / 4) * HY * HZ; e += NT) {
            const int x = 4 * (e % (HX / 4)), y = (e / (HX / 4)) % HY, z = e / ((HX / 4) * HY);
            const int gx = gx0 + x, gy = gy0 + y, gz = gz0 + z;
            const float *p = sm + (z * HY + y) * HPAD + x;
            if (gx < H.nx && gy < H.ny && gz < H.nz)
                *reinterpret_cast<float4 *>(H.out + (size_t)gz * plane + (size_t)gy * H.nx + gx) = make_float4(p[0], p[1], p[2], p[3]);
        }
    } else {
        for (int e = threadIdx.x; e < HX * HY * HZ; e += NT) {
            const int x = e % HX, y = (e / HX) % HY, z = e / (HX * HY);
            const int gx = gx0 + x, gy = gy0 + y, gz = gz0 + z;
            if (gx < H.nx && gy < H.ny && gz < H.nz) H.out[(size_t)gz * plane + (size_t)gy * H.nx + gx] = sm[(z * HY + y) * HPAD + x];
        }
    }
}

// ---- the same filter with an 8 x 8 x 8 block per WARP, in registers --------------------------------------------
// Lane (xh, yp, zp) = (bit 0, bits 1-2, bits 3-4) holds the 4 x 2 x 2 voxels x = 4 xh + a, y = 2 yp + b, z = 2 zp + c
// of the block: every level-1 pair (x, y and z) lies inside a lane, the level-2 lattice (even indices) leaves each
// lane the two values a = 0, 2 of (b, c) = (0, 0), whose y / z partners sit in lanes l ^ 2 / l ^ 8, and the level-3
// lattice (multiples of 4) one value in the lanes with even yp and zp, partners in lanes l ^ 1, l ^ 4, l ^ 16.  A
// pair across lanes is one shuffle: both lanes evaluate the pair from the same two operands with the expressions of
// haar_pair, so the result is bit-identical to the shared-memory kernel and to the per-axis passes.  No shared
// memory, no barrier; 4 LDG.128 + 4 STG.128 per lane (a warp touches whole 32-byte sectors).  Needs nx % 4 == 0
// and 16-byte aligned cubes.  Safe in place.
template <bool INV>
__device__ __forceinline__ float haar_pair_lanes(float mine, bool odd, unsigned xor_mask)
{
    const float other = __shfl_xor_sync(0xffffffffu, mine, xor_mask);
    if (!INV) {                                   // d = odd - even;  c = even + d/2
        const float e = odd ? other : mine, o = odd ? mine : other;
        const float d = o - e;
        return odd ? d : e + 0.5f * d;
    } else {                                      // even = c - d/2;  odd = d + even
        const float c = odd ? other : mine, d = odd ? mine : other;
        const float e = c - 0.5f * d;
        return odd ? d + e : e;
    }
}

__global__ void __launch_bounds__(NT) idg_haar_warp_kernel(const __grid_constant__ HArgs H)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int gx0 = (blockIdx.x * (NT / 32) + warp) * 8, gy0 = blockIdx.y * 8, gz0 = blockIdx.z * 8;
    if (gx0 >= H.nx) return;                      // warp uniform
    const int xh = lane & 1, yp = (lane >> 1) & 3, zp = (lane >> 3) & 3;
    const int gx = gx0 + 4 * xh, gy = gy0 + 2 * yp, gz = gz0 + 2 * zp;
    const size_t plane = (size_t)H.nx * H.ny;
    const bool in_x = gx < H.nx;
    // reading W2: a pair exists if its odd partner lies on the lattice; otherwise the even sample is left alone
    const bool py1 = gy + 1 < H.ny, pz1 = gz + 1 < H.nz;
    const bool py2 = gy0 + 4 * (yp >> 1) + 2 < H.ny, pz2 = gz0 + 4 * (zp >> 1) + 2 < H.nz;
    const bool px3 = gx0 + 4 < H.nx, py3 = gy0 + 4 < H.ny, pz3 = gz0 + 4 < H.nz;
    const bool on3 = !(yp & 1) && !(zp & 1);      // this lane holds a level-3 lattice point (a = b = c = 0)

    float v[2][2][4];
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            float4 t = make_float4(0.f, 0.f, 0.f, 0.f);
            if (in_x && gy + b < H.ny && gz + c < H.nz)
                t = __ldg(reinterpret_cast<const float4 *>(H.in + (size_t)(gz + c) * plane + (size_t)(gy + b) * H.nx + gx));
            v[c][b][0] = t.x; v[c][b][1] = t.y; v[c][b][2] = t.z; v[c][b][3] = t.w;
        }

    auto level1 = [&](auto inv) {
        constexpr bool INV = decltype(inv)::value;
        auto xs = [&]() {                         // lines outside the cube hold zeros and stay zero
#pragma unroll
            for (int c = 0; c < 2; ++c)
#pragma unroll
                for (int b = 0; b < 2; ++b) {
                    haar_pair<INV>(v[c][b][0], v[c][b][1]);
                    haar_pair<INV>(v[c][b][2], v[c][b][3]);
                }
        };
        auto ys = [&]() {
            if (py1) {
#pragma unroll
                for (int c = 0; c < 2; ++c)
#pragma unroll
                    for (int a = 0; a < 4; ++a) haar_pair<INV>(v[c][0][a], v[c][1][a]);
            }
        };
        auto zs = [&]() {
            if (pz1) {
#pragma unroll
                for (int b = 0; b < 2; ++b)
#pragma unroll
                    for (int a = 0; a < 4; ++a) haar_pair<INV>(v[0][b][a], v[1][b][a]);
            }
        };
        if (!INV) { xs(); ys(); zs(); } else { zs(); ys(); xs(); }
    };
    auto level2 = [&](auto inv) {
        constexpr bool INV = decltype(inv)::value;
        float &u0 = v[0][0][0], &u1 = v[0][0][2];
        auto xs = [&]() { haar_pair<INV>(u0, u1); };
        auto ys = [&]() {
            const float a0 = haar_pair_lanes<INV>(u0, yp & 1, 2), a1 = haar_pair_lanes<INV>(u1, yp & 1, 2);
            if (py2) { u0 = a0; u1 = a1; }
        };
        auto zs = [&]() {
            const float a0 = haar_pair_lanes<INV>(u0, zp & 1, 8), a1 = haar_pair_lanes<INV>(u1, zp & 1, 8);
            if (pz2) { u0 = a0; u1 = a1; }
        };
        if (!INV) { xs(); ys(); zs(); } else { zs(); ys(); xs(); }
    };
    auto level3 = [&](auto inv) {
        constexpr bool INV = decltype(inv)::value;
        float &u = v[0][0][0];
        auto xs = [&]() { const float a = haar_pair_lanes<INV>(u, xh, 1); if (on3 && px3) u = a; };
        auto ys = [&]() { const float a = haar_pair_lanes<INV>(u, (yp >> 1) & 1, 4); if (on3 && py3) u = a; };
        auto zs = [&]() { const float a = haar_pair_lanes<INV>(u, (zp >> 1) & 1, 16); if (on3 && pz3) u = a; };
        if (!INV) { xs(); ys(); zs(); } else { zs(); ys(); xs(); }
    };

    level1(std::false_type{});
    if (H.levels >= 2) level2(std::false_type{});
    if (H.levels >= 3) level3(std::false_type{});
    // hard thresholds by band (reading W3): level of a coefficient = trailing zero bits of its indices + 1, capped
    const float t1 = H.thr[0];
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int b = 0; b < 2; ++b)
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                float t = t1;
                if (c == 0 && b == 0 && (a & 1) == 0) {
                    const int tz = __ffs((4 * xh + a) | (2 * yp) | (2 * zp) | 8) - 1;
                    t = H.thr[(tz + 1 < H.levels ? tz + 1 : H.levels) - 1];
                }
                if (fabsf(v[c][b][a]) < t) v[c][b][a] = 0.f;
            }
    if (H.levels >= 3) level3(std::true_type{});
    if (H.levels >= 2) level2(std::true_type{});
    level1(std::true_type{});

#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int b = 0; b < 2; ++b)
            if (in_x && gy + b < H.ny && gz + c < H.nz)
                *reinterpret_cast<float4 *>(H.out + (size_t)(gz + c) * plane + (size_t)(gy + b) * H.nx + gx) =
                    make_float4(v[c][b][0], v[c][b][1], v[c][b][2], v[c][b][3]);
}

template <int WAVELET, int PHASE, bool INV>
cudaError_t launch_phase(const WArgs &W, cudaStream_t st)
{
    const int m = W.axis == 0 ? W.mx : (W.axis == 1 ? W.my : W.mz);
    const int nt = PHASE == 0 ? m / 2 : m - m / 2;
    const long long total = (long long)(W.axis == 0 ? nt : W.mx) * (W.axis == 1 ? nt : W.my) * (W.axis == 2 ? nt : W.mz);
    if (total <= 0 || m < 2) return cudaSuccess;
    long long grid = (total + NT - 1) / NT;
    if (grid > (long long)device_sm_count() * 32) grid = (long long)device_sm_count() * 32;
    idg_lift_kernel<WAVELET, PHASE, INV><<<(unsigned)grid, NT, 0, st>>>(W);
    return cudaGetLastError();
}

template <int WAVELET>
cudaError_t transform(float *a, int nx, int ny, int nz, int levels, bool inverse, bool two_phase, cudaStream_t st,
                      int *launches)
{
    cudaError_t e = cudaSuccess;
    for (int li = 0; li < levels && e == cudaSuccess; ++li) {
        const int l = inverse ? levels - li : li + 1;
        const int s = 1 << (l - 1);
        WArgs W{a, nx, ny, nz, s, 0, (nx + s - 1) / s, (ny + s - 1) / s, (nz + s - 1) / s};
        for (int ai = 0; ai < 3 && e == cudaSuccess; ++ai) {
            W.axis = inverse ? 2 - ai : ai;
            const int m = W.axis == 0 ? W.mx : (W.axis == 1 ? W.my : W.mz);
            if (m < 2) continue;
            if (WAVELET == 0) {
                const long long total = (long long)(W.axis == 0 ? m / 2 : W.mx) * (W.axis == 1 ? m / 2 : W.my) *
                                        (W.axis == 2 ? m / 2 : W.mz);
                long long grid = (total + NT - 1) / NT;
                if (grid > (long long)device_sm_count() * 32) grid = (long long)device_sm_count() * 32;
                if (inverse) idg_haar_pair_kernel<true><<<(unsigned)grid, NT, 0, st>>>(W);
                else idg_haar_pair_kernel<false><<<(unsigned)grid, NT, 0, st>>>(W);
                e = cudaGetLastError();
                *launches += 1;
                continue;
            }
            // whole lines in shared memory: one pass per axis (falls back to two phases for very long lines)
            const size_t line_smem = W.axis == 0 ? (size_t)LW * W.mx * sizeof(float) : (size_t)m * SW * sizeof(float);
            if (line_smem <= 200u * 1024u && !two_phase) {
                if (W.axis == 0) {
                    auto k = inverse ? idg_lift_xline_kernel<WAVELET, true> : idg_lift_xline_kernel<WAVELET, false>;
                    e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
                    long long grid = ((long long)W.my * W.mz + LW - 1) / LW;
                    if (grid > (long long)device_sm_count() * 16) grid = (long long)device_sm_count() * 16;
                    if (e == cudaSuccess) k<<<(unsigned)grid, LW * 32, line_smem, st>>>(W);
                } else {
                    auto k = inverse ? idg_lift_strip_kernel<WAVELET, true> : idg_lift_strip_kernel<WAVELET, false>;
                    e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
                    long long grid = (long long)((W.mx + SW - 1) / SW) * (W.axis == 1 ? W.mz : W.my);
                    if (grid > (long long)device_sm_count() * 16) grid = (long long)device_sm_count() * 16;
                    if (e == cudaSuccess) k<<<(unsigned)grid, NT, line_smem, st>>>(W);
                }
                if (e == cudaSuccess) e = cudaGetLastError();
                *launches += 1;
                continue;
            }
            if (!inverse) {
                e = launch_phase<WAVELET, 0, false>(W, st);
                if (e == cudaSuccess) e = launch_phase<WAVELET, 1, false>(W, st);
            } else {
                e = launch_phase<WAVELET, 1, true>(W, st);
                if (e == cudaSuccess) e = launch_phase<WAVELET, 0, true>(W, st);
            }
            *launches += 2;
        }
    }
    return e;
}

}  // namespace

// In-place forward / inverse transform of `a` to `levels` (wavelet 0 Haar, 1 Le Gall 5/3).
cudaError_t launch_wavelet_transform(float *a, int nx, int ny, int nz, int wavelet, int levels, bool inverse,
                                     bool two_phase, cudaStream_t st, int *launches)
{
    return wavelet == 0 ? transform<0>(a, nx, ny, nz, levels, inverse, two_phase, st, launches)
                        : transform<1>(a, nx, ny, nz, levels, inverse, two_phase, st, launches);
}

// Haar, 1..3 levels: the fused single-pass filter.  thr[l-1] = t_l * rms.  warp_blocks: an 8^3 block per warp in
// registers where the cube allows float4 access (*used_warp reports it), else 64 x 8 x 8 regions in shared memory.
cudaError_t launch_haar_filter(const float *in, float *out, int nx, int ny, int nz, int levels, const float *thr,
                               bool warp_blocks, bool *used_warp, cudaStream_t st)
{
    if (levels < 1 || levels > 3) return cudaErrorInvalidValue;
    HArgs H{in, out, nx, ny, nz, levels, {0.f, 0.f, 0.f}};
    for (int i = 0; i < levels; ++i) H.thr[i] = thr[i];
    const unsigned gx = (unsigned)((nx + HX - 1) / HX), gy = (unsigned)((ny + HY - 1) / HY), gz = (unsigned)((nz + HZ - 1) / HZ);
    if (gy > 65535u || gz > 65535u) return cudaErrorInvalidValue;
    const bool vec = (nx % 4 == 0) && ((((uintptr_t)in | (uintptr_t)out) & 15u) == 0);
    *used_warp = warp_blocks && vec;
    if (*used_warp) idg_haar_warp_kernel<<<dim3(gx, gy, gz), NT, 0, st>>>(H);      // 8 warps = 64 columns, as the regions
    else idg_haar_filter_kernel<<<dim3(gx, gy, gz), NT, 0, st>>>(H);
    return cudaGetLastError();
}

// thr[l-1] = t_l * rms, levels <= 16.
cudaError_t launch_wavelet_threshold(float *a, int nx, int ny, int nz, int levels, const float *thr, cudaStream_t st)
{
    TArgs T;
    T.a = a; T.nx = nx; T.ny = ny; T.nz = nz; T.levels = levels;
    for (int i = 0; i < 16; ++i) T.thr[i] = i < levels ? thr[i] : 0.f;
    const size_t N = (size_t)nx * ny * (size_t)nz;
    size_t grid = (N + NT - 1) / NT;
    if (grid > (unsigned)device_sm_count() * 32u) grid = (unsigned)device_sm_count() * 32u;
    idg_wavelet_threshold_kernel<<<(unsigned)grid, NT, 0, st>>>(T);
    return cudaGetLastError();
}

}  // namespace idg
