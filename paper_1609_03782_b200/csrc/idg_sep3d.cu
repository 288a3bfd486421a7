// Separable 3-D filter with replicated faces in ONE pass over the cube: the box filter
// and the axis-aligned Gaussian filter (Eq. 1-2; "three
// separate 1-D Gaussian convolutions").
//
//   out(x,y,z) = sum_k wz[k] sum_j wy[j] sum_i wx[i] I(cx(x+i), cy(y+j), cz(z+k)),   c. = clamp to the cube
//
// A CTA owns a 64 x 16 xy tile and streams along z.  Per input plane: the tile plus its xy halo goes
// to shared memory (coalesced rows, clamped coordinates; the next plane is prefetched into registers
// while the current one is filtered), an x pass (4 consecutive outputs per item from aligned float4
// loads) and a y pass (4 rows per thread from a register window) give the xy-filtered plane, which
// enters a ring of 2 rz + 1 planes; the z pass combines the ring into one output plane.  Ring entries
// are private to the thread that wrote them (a register shift array for rz <= 4, shared memory
// above), so a plane step needs two CTA barriers.  The cube is read
// once and written once (8 B per voxel plus halo), instead of three round trips for three 1-D passes.
//
// The radii are template parameters (everything unrolls, no address arithmetic is left in the plane
// loop): a filter of radii (rx, ry, rz) runs in the smallest class RXY >= max(rx, ry), RZ >= rz of
// {0, 1, 2, 4, 9, 16} with its weights zero-padded to the class width.
#include "idg_kernels.cuh"

namespace idg {

namespace {

constexpr int TX = 64, TY = 16, NT = 256;

struct SepArgs {
    const float *in;
    float *out;
    int nx, ny, nz;
    int zchunk;
    float wx[2 * kSepMaxRadius + 1], wy[2 * kSepMaxRadius + 1], wz[2 * kSepMaxRadius + 1];   // padded to the class
};

template <int RXY, int RZ>
struct Geo {
    static constexpr int HX = (RXY + 3) / 4 * 4;             // left halo rounded up to a multiple of 4
    static constexpr int STRIDE = TX + 2 * HX;               // floats per row of A
    static constexpr int ROWS = TY + 2 * RXY;
    static constexpr int ROWS_PAD = (ROWS + 7) / 8 * 8;      // rows of A (warps load 8 rows per round)
    static constexpr int COLS = TX + 2 * RXY;                // columns loaded per row
    static constexpr int OFF = HX - RXY;                     // pad columns in front of the loaded ones: 0..3
    static constexpr int NV = (OFF + 4 + 2 * RXY + 3) / 4;   // float4 loads per x-pass item
    static constexpr int W = 2 * RZ + 1;
    static constexpr int ROW_IT = ROWS_PAD / 8, COL_IT = (COLS + 31) / 32;
    static constexpr bool REG_RING = RZ <= 4;                // z ring in registers (4 W per thread) or in shared memory
    static constexpr size_t kSmem = sizeof(float) * ((size_t)ROWS_PAD * STRIDE + (size_t)ROWS * TX +
                                                     (REG_RING ? 0 : (size_t)W * TY * TX));
    // register budget: the z shift array costs 4 W registers per thread
    static constexpr int kMinBlocks = REG_RING ? (RZ <= 2 ? 3 : 2) : (kSmem * 3 <= 200 * 1024 ? 3 : (kSmem * 2 <= 220 * 1024 ? 2 : 1));
};

template <int RXY, int RZ>
__global__ void __launch_bounds__(NT, Geo<RXY, RZ>::kMinBlocks) idg_sep3d_kernel(const __grid_constant__ SepArgs S)
{
    using G = Geo<RXY, RZ>;
    extern __shared__ __align__(16) float smem[];
    float *A = smem;                                  // ROWS_PAD x STRIDE   input tile with halo
    float *B = A + G::ROWS_PAD * G::STRIDE;           // ROWS x TX           after the x pass
    float *ring = B + G::ROWS * TX;                   // W x TY x TX         xy-filtered planes

    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
    const int z0 = blockIdx.z * S.zchunk, z1 = min(z0 + S.zchunk, S.nz);
    const size_t plane = (size_t)S.nx * (size_t)S.ny;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int yg = threadIdx.x / TX, xl = threadIdx.x - yg * TX;     // y/z-pass ownership: rows 4yg..4yg+3, column xl

    // Tile loads: warp w takes halo rows w, w+8, ...; lane l takes halo columns l, l+32, (l+64) of a row.
    // Clamped global x and row offsets do not change from plane to plane.
    // 32-bit element offsets inside a plane (the launcher rejects planes of 2^32 voxels and more), so a load
    // is plane base (uniform) + offset
    unsigned off[G::ROW_IT][G::COL_IT];
#pragma unroll
    for (int i = 0; i < G::ROW_IT; ++i)
#pragma unroll
        for (int c = 0; c < G::COL_IT; ++c)
            off[i][c] = (unsigned)min(max(y0 - RXY + warp + 8 * i, 0), S.ny - 1) * (unsigned)S.nx +
                        (unsigned)min(max(x0 - RXY + lane + 32 * c, 0), S.nx - 1);

    float pre[G::ROW_IT * G::COL_IT];
    auto fetch = [&](int q) {                         // plane clamp(q) -> registers
        const float *src = S.in + (size_t)min(max(q, 0), S.nz - 1) * plane;
#pragma unroll
        for (int i = 0; i < G::ROW_IT; ++i)
#pragma unroll
            for (int c = 0; c < G::COL_IT; ++c)
                if (32 * c + 31 < G::COLS || lane + 32 * c < G::COLS) pre[i * G::COL_IT + c] = __ldg(src + off[i][c]);
    };
    float *a_thr = A + warp * G::STRIDE + G::OFF + lane;
    auto stash = [&]() {                              // registers -> A
#pragma unroll
        for (int i = 0; i < G::ROW_IT; ++i)
#pragma unroll
            for (int c = 0; c < G::COL_IT; ++c)
                if (32 * c + 31 < G::COLS || lane + 32 * c < G::COLS)
                    a_thr[8 * i * G::STRIDE + 32 * c] = pre[i * G::COL_IT + c];
    };

    const int q_first = z0 - RZ, q_last = z1 - 1 + RZ;
    fetch(q_first);
    int slot = 0;
    float *ring_col = ring + (4 * yg) * TX + xl;
    float zr[G::REG_RING ? G::W : 1][4];
#pragma unroll
    for (int k = 0; k < (G::REG_RING ? G::W : 1); ++k)
#pragma unroll
        for (int o = 0; o < 4; ++o) zr[k][o] = 0.f;
    const bool col_ok = x0 + xl < S.nx;
    for (int q = q_first; q <= q_last; ++q) {
        stash();
        __syncthreads();                              // A complete; everybody is done with B of the previous plane
        if (q < q_last) fetch(q + 1);
        // x pass: items = ROWS x 16 groups of 4 outputs; window of NV aligned float4
#pragma unroll
        for (int it0 = 0; it0 < G::ROWS * (TX / 4); it0 += NT) {
            const int it = it0 + threadIdx.x;
            if (it0 + NT <= G::ROWS * (TX / 4) || it < G::ROWS * (TX / 4)) {
                const int row = it / (TX / 4), g = it % (TX / 4);
                const float4 *a4 = reinterpret_cast<const float4 *>(A + row * G::STRIDE + 4 * g);
                float win[4 * G::NV];
#pragma unroll
                for (int v = 0; v < G::NV; ++v) {
                    const float4 t = a4[v];
                    win[4 * v] = t.x; win[4 * v + 1] = t.y; win[4 * v + 2] = t.z; win[4 * v + 3] = t.w;
                }
                float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                for (int k = 0; k <= 2 * RXY; ++k)
#pragma unroll
                    for (int o = 0; o < 4; ++o) acc[o] = fmaf(S.wx[k], win[G::OFF + o + k], acc[o]);
                *reinterpret_cast<float4 *>(B + row * TX + 4 * g) = make_float4(acc[0], acc[1], acc[2], acc[3]);
            }
        }
        __syncthreads();                              // B complete; A may be overwritten
        // y pass: rows 4yg .. 4yg+3 of column xl from a window of 4 + 2 RXY rows of B
        float p[4] = {0.f, 0.f, 0.f, 0.f};
        {
            float win[4 + 2 * RXY];
#pragma unroll
            for (int j = 0; j < 4 + 2 * RXY; ++j) win[j] = B[(4 * yg + j) * TX + xl];
#pragma unroll
            for (int k = 0; k <= 2 * RXY; ++k)
#pragma unroll
                for (int o = 0; o < 4; ++o) p[o] = fmaf(S.wy[k], win[o + k], p[o]);
        }
        const int zo = q - RZ;                        // output plane whose window [zo-rz, zo+rz] is now complete
        float acc[4] = {0.f, 0.f, 0.f, 0.f};
        if (G::REG_RING) {
            // shift register of my last W xy-filtered values: zr[k] = plane zo - RZ + k
#pragma unroll
            for (int k = 0; k + 1 < G::W; ++k)
#pragma unroll
                for (int o = 0; o < 4; ++o) zr[k][o] = zr[k + 1][o];
#pragma unroll
            for (int o = 0; o < 4; ++o) zr[G::W - 1][o] = p[o];
            if (zo >= z0) {
#pragma unroll
                for (int k = 0; k < G::W; ++k)
#pragma unroll
                    for (int o = 0; o < 4; ++o) acc[o] = fmaf(S.wz[k], zr[k][o], acc[o]);
            }
        } else {
            // my four ring entries of the slot of plane q (private to this thread)
#pragma unroll
            for (int o = 0; o < 4; ++o) ring_col[(slot * TY + o) * TX] = p[o];
            slot = (slot + 1 == G::W) ? 0 : slot + 1; // slot of plane q - 2 RZ = zo - RZ (and of plane q + 1)
            if (zo >= z0) {
                int sl = slot;
#pragma unroll
                for (int k = 0; k < G::W; ++k) {
#pragma unroll
                    for (int o = 0; o < 4; ++o) acc[o] = fmaf(S.wz[k], ring_col[(sl * TY + o) * TX], acc[o]);
                    sl = (sl + 1 == G::W) ? 0 : sl + 1;
                }
            }
        }
        if (zo >= z0) {
            if (col_ok) {
                float *dst = S.out + (size_t)zo * plane + (size_t)(y0 + 4 * yg) * S.nx + x0 + xl;
#pragma unroll
                for (int o = 0; o < 4; ++o)
                    if (y0 + 4 * yg + o < S.ny) dst[(size_t)o * S.nx] = acc[o];
            }
        }
    }
}

constexpr int kClasses[6] = {0, 1, 2, 4, 9, 16};
inline int class_of(int r)
{
    for (int c : kClasses)
        if (r <= c) return c;
    return -1;
}

template <int RXY, int RZ>
cudaError_t launch_class(const SepArgs &S, dim3 grid, cudaStream_t st)
{
    using G = Geo<RXY, RZ>;
    static DeviceOnce smem_once;
    {
        const cudaError_t e = set_max_dynamic_smem(smem_once, (const void *)(idg_sep3d_kernel<RXY, RZ>), G::kSmem);
        if (e != cudaSuccess) return e;
    }
    idg_sep3d_kernel<RXY, RZ><<<grid, NT, G::kSmem, st>>>(S);
    return cudaGetLastError();
}

template <int RXY>
cudaError_t launch_rz(int cz, const SepArgs &S, dim3 grid, cudaStream_t st)
{
    switch (cz) {
    case 0: return launch_class<RXY, 0>(S, grid, st);
    case 1: return launch_class<RXY, 1>(S, grid, st);
    case 2: return launch_class<RXY, 2>(S, grid, st);
    case 4: return launch_class<RXY, 4>(S, grid, st);
    case 9: return launch_class<RXY, 9>(S, grid, st);
    default: return launch_class<RXY, 16>(S, grid, st);
    }
}

}  // namespace

// w*: 2r+1 weights per axis (already normalised); radii <= kSepMaxRadius.
cudaError_t launch_sep3d(const float *in, float *out, int nx, int ny, int nz, int rx, int ry, int rz,
                         const float *wx, const float *wy, const float *wz, cudaStream_t st)
{
    if (rx > kSepMaxRadius || ry > kSepMaxRadius || rz > kSepMaxRadius) return cudaErrorInvalidValue;
    const int cxy = class_of(rx > ry ? rx : ry), cz = class_of(rz);
    SepArgs S;
    S.in = in; S.out = out;
    S.nx = nx; S.ny = ny; S.nz = nz;
    for (int i = 0; i < 2 * kSepMaxRadius + 1; ++i) S.wx[i] = S.wy[i] = S.wz[i] = 0.f;
    for (int i = 0; i <= 2 * rx; ++i) S.wx[i + cxy - rx] = wx[i];        // centred in the class window
    for (int i = 0; i <= 2 * ry; ++i) S.wy[i + cxy - ry] = wy[i];
    for (int i = 0; i <= 2 * rz; ++i) S.wz[i + cz - rz] = wz[i];
    const int tiles_x = (nx + TX - 1) / TX, tiles_y = (ny + TY - 1) / TY;
    // z chunks: minimise waves x (planes per chunk + warm-up planes) for ~3 resident CTAs per SM
    const long tiles = (long)tiles_x * tiles_y, slots = (long)device_sm_count() * 3;
    long best_cost = -1;
    int chunks = 1;
    for (int c = 1; c <= nz && c <= 4096; ++c) {
        const int zc = (nz + c - 1) / c;
        const long ctas = tiles * ((nz + zc - 1) / zc);
        const long cost = ((ctas + slots - 1) / slots) * (long)(zc + 2 * cz + 1);
        if (best_cost < 0 || cost < best_cost) { best_cost = cost; chunks = c; }
    }
    S.zchunk = (nz + chunks - 1) / chunks;
    chunks = (nz + S.zchunk - 1) / S.zchunk;
    if (tiles_y > 65535 || chunks > 65535 || (unsigned long long)nx * (unsigned long long)ny >= (1ull << 32))
        return cudaErrorInvalidValue;
    const dim3 grid((unsigned)tiles_x, (unsigned)tiles_y, (unsigned)chunks);
    switch (cxy) {
    case 0: return launch_rz<0>(cz, S, grid, st);
    case 1: return launch_rz<1>(cz, S, grid, st);
    case 2: return launch_rz<2>(cz, S, grid, st);
    case 4: return launch_rz<4>(cz, S, grid, st);
    case 9: return launch_rz<9>(cz, S, grid, st);
    default: return launch_rz<16>(cz, S, grid, st);
    }
}

}  // namespace idg
