// Separable 3-D filter with replicated faces in ONE pass over the cube: the box filter
// and the axis-aligned Gaussian filter (Eq. 1-2; "three
// separate 1-D Gaussian convolutions").
//
//   out(x,y,z) = sum_k wz[k] sum_j wy[j] sum_i wx[i] I(cx(x+i), cy(y+j), cz(z+k)),   c. = clamp to the cube
//
// A CTA owns a 64 x 16 xy tile and streams along z.  Per input plane: the tile plus its xy halo goes
// to shared memory (coalesced rows, clamped coordinates; the next plane is prefetched into registers
// while the current one is filtered), an x pass and a y pass (each thread 4 consecutive outputs from
// a register window, radius known at compile time) give the xy-filtered plane, which enters a ring of
// 2 rz + 1 planes; the z pass combines the ring into one output plane.  Ring entries are private to
// the thread that wrote them, so a plane step needs two CTA barriers.  The cube is read once and
// written once (8 B per voxel plus halo), instead of three round trips for three 1-D passes.
#include "idg_kernels.cuh"

namespace idg {

namespace {

constexpr int TX = 64, TY = 16, NT = 256;

struct SepArgs {
    const float *in;
    float *out;
    int nx, ny, nz;
    int rx, ry, rz;
    int zchunk;
    int hx;                      // left halo rounded up to a multiple of 4 (row stride = TX + 2*hx)
    float wx[2 * kSepMaxRadius + 1], wy[2 * kSepMaxRadius + 1], wz[2 * kSepMaxRadius + 1];
};

// x pass of one work item: 4 consecutive outputs of one halo row from a window of 4 + 2R inputs.
template <int R>
__device__ __forceinline__ void xpass_item(const float *__restrict__ a, float *__restrict__ b, const float *w)
{
    float win[4 + 2 * R];
#pragma unroll
    for (int i = 0; i < 4 + 2 * R; ++i) win[i] = a[i];
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int k = 0; k <= 2 * R; ++k) {
        const float wk = w[k];
#pragma unroll
        for (int o = 0; o < 4; ++o) acc[o] = fmaf(wk, win[o + k], acc[o]);
    }
    *reinterpret_cast<float4 *>(b) = make_float4(acc[0], acc[1], acc[2], acc[3]);
}

template <int R>
__device__ __forceinline__ void xpass(const float *A, float *B, const SepArgs &S, int rows, int stride)
{
    // items: rows x (TX/4) groups of 4 outputs
    for (int it = threadIdx.x; it < rows * (TX / 4); it += NT) {
        const int row = it / (TX / 4), g = it - row * (TX / 4);
        xpass_item<R>(A + row * stride + S.hx - R + 4 * g, B + row * TX + 4 * g, S.wx);
    }
}

// y pass: thread (yg, x) produces rows 4*yg .. 4*yg+3 of column x from a window of 4 + 2R rows of B.
template <int R>
__device__ __forceinline__ void ypass(const float *B, const SepArgs &S, int yg, int x, float (&p)[4])
{
    float win[4 + 2 * R];
#pragma unroll
    for (int j = 0; j < 4 + 2 * R; ++j) win[j] = B[(4 * yg + j) * TX + x];
#pragma unroll
    for (int o = 0; o < 4; ++o) p[o] = 0.f;
#pragma unroll
    for (int k = 0; k <= 2 * R; ++k) {
        const float wk = S.wy[k];
#pragma unroll
        for (int o = 0; o < 4; ++o) p[o] = fmaf(wk, win[o + k], p[o]);
    }
}

// z pass: combine the 2R+1 ring planes, starting at ring slot `sl` (the plane zo - R), for my 4 rows.
template <int R>
__device__ __forceinline__ void zpass(const float *ring_col, int sl, const SepArgs &S, float (&acc)[4])
{
    constexpr int W = 2 * R + 1;
#pragma unroll
    for (int o = 0; o < 4; ++o) acc[o] = 0.f;
#pragma unroll
    for (int k = 0; k < W; ++k) {
        const float wk = S.wz[k];
#pragma unroll
        for (int o = 0; o < 4; ++o) acc[o] = fmaf(wk, ring_col[(sl * TY + o) * TX], acc[o]);
        sl = (sl + 1 == W) ? 0 : sl + 1;
    }
}

#define IDG_SEP_SWITCH(r, CALL)                                                                      \
    switch (r) {                                                                                     \
    case 0: { constexpr int R_ = 0; CALL; } break;   case 1: { constexpr int R_ = 1; CALL; } break;   \
    case 2: { constexpr int R_ = 2; CALL; } break;   case 3: { constexpr int R_ = 3; CALL; } break;   \
    case 4: { constexpr int R_ = 4; CALL; } break;   case 5: { constexpr int R_ = 5; CALL; } break;   \
    case 6: { constexpr int R_ = 6; CALL; } break;   case 7: { constexpr int R_ = 7; CALL; } break;   \
    case 8: { constexpr int R_ = 8; CALL; } break;   case 9: { constexpr int R_ = 9; CALL; } break;   \
    case 10: { constexpr int R_ = 10; CALL; } break; case 11: { constexpr int R_ = 11; CALL; } break; \
    case 12: { constexpr int R_ = 12; CALL; } break; case 13: { constexpr int R_ = 13; CALL; } break; \
    case 14: { constexpr int R_ = 14; CALL; } break; case 15: { constexpr int R_ = 15; CALL; } break; \
    default: { constexpr int R_ = 16; CALL; } break;                                                 \
    }

constexpr int kRowIters = (TY + 2 * kSepMaxRadius + NT / 32 - 1) / (NT / 32);   // halo rows per warp: <= 6
constexpr int kColIters = (TX + 2 * kSepMaxRadius + 31) / 32;                    // halo columns per lane: <= 3

__global__ void __launch_bounds__(NT, 3) idg_sep3d_kernel(const __grid_constant__ SepArgs S)
{
    extern __shared__ __align__(16) float smem[];
    const int stride = TX + 2 * S.hx;
    const int rows = TY + 2 * S.ry;
    float *A = smem;                                  // rows x stride   input tile with halo
    float *B = A + ((rows + 7) & ~7) * stride;        // rows x TX       after the x pass (A padded to 8 rows)
    float *ring = B + rows * TX;                      // (2rz+1) x TY x TX   xy-filtered planes
    const int W = 2 * S.rz + 1;

    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
    const int z0 = blockIdx.z * S.zchunk, z1 = min(z0 + S.zchunk, S.nz);
    const size_t plane = (size_t)S.nx * (size_t)S.ny;
    const int cols = TX + 2 * S.rx;                   // columns actually loaded per row

    const int yg = threadIdx.x / TX, xl = threadIdx.x - yg * TX;     // y/z-pass ownership: rows 4yg..4yg+3, column xl
    const bool col_ok = x0 + xl < S.nx;

    // Tile loads: warp w takes halo rows w, w+8, ...; lane l takes halo columns l, l+32, l+64 of a row.
    // The clamped global x of those columns does not change from plane to plane.
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int gxo[kColIters];
#pragma unroll
    for (int c = 0; c < kColIters; ++c) gxo[c] = min(max(x0 - S.rx + lane + 32 * c, 0), S.nx - 1);

    // rows are padded to a multiple of 8 in A (the extra rows reload clamped rows and are never read)
    const int n_it = (rows + NT / 32 - 1) / (NT / 32);
    const bool c2 = lane + 64 < cols;                 // columns lane, lane+32 always exist (cols >= 64)
    float pre[kRowIters * kColIters];
    auto fetch = [&](int q) {                         // plane clamp(q) -> registers
        const float *src = S.in + (size_t)min(max(q, 0), S.nz - 1) * plane;
#pragma unroll
        for (int i = 0; i < kRowIters; ++i) {
            if (i < n_it) {
                const float *rp = src + (size_t)min(max(y0 - S.ry + warp + (NT / 32) * i, 0), S.ny - 1) * S.nx;
                pre[i * kColIters + 0] = __ldg(rp + gxo[0]);
                pre[i * kColIters + 1] = __ldg(rp + gxo[1]);
                if (c2) pre[i * kColIters + 2] = __ldg(rp + gxo[2]);
            }
        }
    };
    float *a_thr = A + warp * stride + S.hx - S.rx + lane;
    auto stash = [&]() {                              // registers -> A
#pragma unroll
        for (int i = 0; i < kRowIters; ++i) {
            if (i < n_it) {
                float *ap = a_thr + (NT / 32) * i * stride;
                ap[0] = pre[i * kColIters + 0];
                ap[32] = pre[i * kColIters + 1];
                if (c2) ap[64] = pre[i * kColIters + 2];
            }
        }
    };

    const int q_first = z0 - S.rz, q_last = z1 - 1 + S.rz;
    fetch(q_first);
    int slot = 0;
    for (int q = q_first; q <= q_last; ++q) {
        stash();
        __syncthreads();                              // A complete; everybody is done with B of the previous plane
        if (q < q_last) fetch(q + 1);
        IDG_SEP_SWITCH(S.rx, xpass<R_>(A, B, S, rows, stride));
        __syncthreads();                              // B complete; A may be overwritten
        float p[4];
        IDG_SEP_SWITCH(S.ry, ypass<R_>(B, S, yg, xl, p));
        // my four ring entries of the slot of plane q (private to this thread)
        float *ring_col = ring + (4 * yg) * TX + xl;
#pragma unroll
        for (int o = 0; o < 4; ++o) ring_col[(slot * TY + o) * TX] = p[o];
        const int zo = q - S.rz;                      // output plane whose window [zo-rz, zo+rz] is now complete
        const int slot0 = (slot + 1 == W) ? 0 : slot + 1;     // slot of plane q - 2rz = zo - rz
        slot = slot0;                                 // = slot of plane q + 1
        if (zo >= z0) {
            float acc[4];
            IDG_SEP_SWITCH(S.rz, zpass<R_>(ring_col, slot0, S, acc));
            if (col_ok) {
                float *dst = S.out + (size_t)zo * plane + (size_t)(y0 + 4 * yg) * S.nx + x0 + xl;
#pragma unroll
                for (int o = 0; o < 4; ++o)
                    if (y0 + 4 * yg + o < S.ny) dst[(size_t)o * S.nx] = acc[o];
            }
        }
    }
}

}  // namespace

// w*: 2r+1 weights per axis (already normalised); radii <= kSepMaxRadius.
cudaError_t launch_sep3d(const float *in, float *out, int nx, int ny, int nz, int rx, int ry, int rz,
                         const float *wx, const float *wy, const float *wz, cudaStream_t st)
{
    if (rx > kSepMaxRadius || ry > kSepMaxRadius || rz > kSepMaxRadius) return cudaErrorInvalidValue;
    SepArgs S;
    S.in = in; S.out = out;
    S.nx = nx; S.ny = ny; S.nz = nz;
    S.rx = rx; S.ry = ry; S.rz = rz;
    S.hx = (rx + 3) / 4 * 4;
    for (int i = 0; i <= 2 * rx; ++i) S.wx[i] = wx[i];
    for (int i = 0; i <= 2 * ry; ++i) S.wy[i] = wy[i];
    for (int i = 0; i <= 2 * rz; ++i) S.wz[i] = wz[i];
    const int tiles_x = (nx + TX - 1) / TX, tiles_y = (ny + TY - 1) / TY;
    // z chunks: minimise waves x (planes per chunk + warm-up planes) for ~4 resident CTAs per SM
    const long tiles = (long)tiles_x * tiles_y, slots = 148L * 4;
    long best_cost = -1;
    int chunks = 1;
    for (int c = 1; c <= nz && c <= 4096; ++c) {
        const int zc = (nz + c - 1) / c;
        const long ctas = tiles * ((nz + zc - 1) / zc);
        const long cost = ((ctas + slots - 1) / slots) * (long)(zc + 2 * rz + 1);
        if (best_cost < 0 || cost < best_cost) { best_cost = cost; chunks = c; }
    }
    S.zchunk = (nz + chunks - 1) / chunks;
    chunks = (nz + S.zchunk - 1) / S.zchunk;
    if (tiles_y > 65535 || chunks > 65535) return cudaErrorInvalidValue;
    const int rows = TY + 2 * ry, stride = TX + 2 * S.hx;
    const size_t smem = sizeof(float) * ((size_t)((rows + 7) & ~7) * stride + (size_t)rows * TX + (size_t)(2 * rz + 1) * TY * TX);
    static size_t attr = 0;
    if (smem > attr) {
        cudaError_t e = cudaFuncSetAttribute(idg_sep3d_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr = smem;
    }
    dim3 grid((unsigned)tiles_x, (unsigned)tiles_y, (unsigned)chunks);
    idg_sep3d_kernel<<<grid, NT, smem, st>>>(S);
    return cudaGetLastError();
}

}  // namespace idg
