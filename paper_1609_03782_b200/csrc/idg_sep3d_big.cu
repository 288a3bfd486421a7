// Separable 3-D filter for radii 5 .. 9 (Gaussian FWHM 5 and 7 of PAPER.md:283 and :222, box widths 11 .. 19) on
// 16-byte aligned cubes with nx % 4 == 0: the decomposition of idg_sep3d_tma.cu -- a CTA owns a 128 x (WARPS*R) xy tile
// and streams along z, raw planes + RXY halo rows by TMA into a ring of stages, y pass from shared memory, x pass by
// warp shuffles, z pass over xy-filtered planes in registers, no CTA barrier in the plane loop -- with two changes that
// the wider support forces:
//
//   x pass   a radius r reaches HL = ceil(r / 4) float4 to either side: tiles overlap by HL lanes per side
//            (32 - 2 HL valid lanes), and all HL lanes outside a cube face take the replicated face value;
//   z pass   a window of 2 RZ + 1 planes rotated by unrolling the plane loop over its phases (as for radii <= 4) would
//            be 13 or 19 copies of the loop body -- more than the instruction cache holds.  Instead the loop advances in
//            super-steps of ZB planes: the thread keeps the last 2 RZ xy-filtered planes of its column, filters ZB new
//            ones, forms the ZB outputs whose windows are now complete (all register indices static), and shifts the
//            ring by ZB planes (2 RZ register moves per ZB planes and float).
//
//   out(x,y,z) = sum_k wz[k] sum_i wx[i] sum_j wy[j] I(cx(x+i), cy(y+j), cz(z+k)),   c. = clamp to the cube (reading F1)
#include <cuda.h>

#include "idg_kernels.cuh"
#include "idg_ptx.cuh"
#include "idg_update.cuh"

namespace idg {

namespace {

constexpr int kTileX = 128;
constexpr int kBigMaxR = 9;

__device__ __forceinline__ float comp(const F4 &a, int i) { return i == 0 ? a.x : (i == 1 ? a.y : (i == 2 ? a.z : a.w)); }

struct SepBigArgs {
    float *out;
    int nx, ny, nz;
    int tiles_x, zchunk;
    float wx[2 * kBigMaxR + 1], wy[2 * kBigMaxR + 1], wz[2 * kBigMaxR + 1];     // zero-padded to the class width
};

template <int RXY, int R, int WARPS, int NS>
struct BigGeo {
    static constexpr int HL = (RXY + 3) / 4;             // halo lanes per side
    static constexpr int V = 32 - 2 * HL;                // valid lanes of a tile
    static constexpr int VY = WARPS * R;                 // output rows per tile
    static constexpr int ROWS = VY + 2 * RXY;            // rows loaded per plane
    static constexpr int kStageFloats = ROWS * kTileX;
    static constexpr size_t kStageBytes = (size_t)kStageFloats * sizeof(float);
    static constexpr size_t kBarOff = NS * kStageBytes;
    static constexpr size_t kBytes = kBarOff + 2 * NS * sizeof(uint64_t);
};

template <int RXY, int RZ, int R, int WARPS, int NS, int ZB, int MINB>
__global__ void __launch_bounds__(WARPS * 32, MINB)
idg_sep3d_big_kernel(const __grid_constant__ SepBigArgs S, const __grid_constant__ CUtensorMap map)
{
    using G = BigGeo<RXY, R, WARPS, NS>;
    constexpr int HL = G::HL, WIN = R + 2 * RXY, AHEAD = NS - 2, RING = 2 * RZ;
    extern __shared__ __align__(1024) unsigned char smem[];
    float *stage0 = reinterpret_cast<float *>(smem);
    const uint32_t full = ptx::smem_u32(smem + G::kBarOff), empty = full + NS * 8;

    const int lane = threadIdx.x & 31, wy = threadIdx.x >> 5;
    const int nx4 = S.nx >> 2;
    const int ti = blockIdx.x % S.tiles_x, tj = blockIdx.x / S.tiles_x;
    const int x4 = ti * G::V - HL + lane;
    const int tx0 = (ti * G::V - HL) * 4;                // cube x of tile column 0
    const int ty0 = tj * G::VY;                          // cube y of the first output row
    const int z0 = blockIdx.y * S.zchunk, z1 = min(z0 + S.zchunk, S.nz);
    const int q_first = z0 - RZ, q_last = z1 - 1 + RZ;
    const bool left_halo = x4 < 0, right_halo = x4 >= nx4;
    const bool edge_x = ti == 0 || (ti + 1) * G::V >= nx4;            // the tile touches an x face (CTA uniform)
    const int lane_first = HL - ti * G::V;                             // lane of the cube's first / last float4
    const int lane_last = min(max(nx4 - 1 - (ti * G::V - HL), 0), 31);

    // window rows of this thread: stage row s holds cube row ty0 - RXY + s; rows outside the cube read the face row
    int roff[WIN];
#pragma unroll
    for (int j = 0; j < WIN; ++j) {
        const int gy = min(max(ty0 - RXY + wy * R + j, 0), S.ny - 1);
        roff[j] = (gy - (ty0 - RXY)) * kTileX + lane * 4;
    }
    unsigned ok = 0;
#pragma unroll
    for (int r = 0; r < R; ++r)
        if (lane >= HL && lane < HL + G::V && x4 < nx4 && ty0 + wy * R + r < S.ny) ok |= 1u << r;

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            ptx::mbar_init(full + 8 * s, 1);
            ptx::mbar_init(empty + 8 * s, WARPS);
        }
        ptx::mbar_fence_init();
    }
    __syncthreads();
    auto issue = [&](int i) {       // thread 0: i-th plane of the chunk -> stage i % NS
        const int s = i % NS;
        ptx::mbar_expect_tx(full + 8 * s, (uint32_t)G::kStageBytes);
        ptx::tma_load_4d(ptx::smem_u32(stage0 + (size_t)s * G::kStageFloats), &map, full + 8 * s, tx0, ty0 - RXY,
                         min(max(q_first + i, 0), S.nz - 1), 0);
    };
    const int n_planes = q_last - q_first + 1;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < AHEAD; ++i)
            if (i < n_planes) issue(i);
    }

    // xy-filtered planes of my column: win[0 .. RING-1] the last 2 RZ, win[RING .. RING+ZB-1] this super-step's
    F4 win[RING + ZB][R];
#pragma unroll
    for (int k = 0; k < RING + ZB; ++k)
#pragma unroll
        for (int r = 0; r < R; ++r) win[k][r] = F4{0.f, 0.f, 0.f, 0.f};

    const size_t plane = (size_t)S.nx * (size_t)S.ny;
    float *po = S.out + (size_t)(ty0 + wy * R) * S.nx + (long long)x4 * 4;

    for (int base = 0; base < n_planes; base += ZB) {
#pragma unroll
        for (int j = 0; j < ZB; ++j) {
            const int it = base + j;
            if (it >= n_planes) break;                  // (uniform over the CTA)
            const int s = it % NS;
            if (threadIdx.x == 0 && it + AHEAD < n_planes) {
                const int i = it + AHEAD;   // its stage held plane it - 2: wait until every warp has read it
                if (i >= NS) ptx::mbar_wait_spin(empty + 8 * (i % NS), (uint32_t)((i / NS - 1) & 1));
                issue(i);
            }
            const float *st = stage0 + (size_t)s * G::kStageFloats;
            ptx::mbar_wait_spin(full + 8 * s, (uint32_t)((it / NS) & 1));

            // y pass, streamed over the window rows (row jj feeds output row r with weight k = jj - r)
            F4 yf[R];
#pragma unroll
            for (int jj = 0; jj < WIN; ++jj) {
                const F4 w = lds4(st + roff[jj]);
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int k = jj - r;
                    if (k == 0) {
                        yf[r] = F4{S.wy[0] * w.x, S.wy[0] * w.y, S.wy[0] * w.z, S.wy[0] * w.w};
                    } else if (k > 0 && k <= 2 * RXY) {
                        yf[r].x = fmaf(S.wy[k], w.x, yf[r].x);
                        yf[r].y = fmaf(S.wy[k], w.y, yf[r].y);
                        yf[r].z = fmaf(S.wy[k], w.z, yf[r].z);
                        yf[r].w = fmaf(S.wy[k], w.w, yf[r].w);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(empty + 8 * s);
            if (edge_x) {                   // replicated x faces: every lane outside takes the face value
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const float a = __shfl_sync(0xffffffffu, yf[r].x, lane_first & 31);
                    const float b = __shfl_sync(0xffffffffu, yf[r].w, lane_last);
                    if (left_halo) yf[r] = F4{a, a, a, a};
                    else if (right_halo) yf[r] = F4{b, b, b, b};
                }
            }
            // x pass -> win[RING + j]
#pragma unroll
            for (int r = 0; r < R; ++r) {
                float line[4 + 8 * HL];
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    line[4 * HL + i] = comp(yf[r], i);
#pragma unroll
                    for (int d = 1; d <= HL; ++d) {
                        if (4 * HL - 4 * d + i >= 4 * HL - RXY)
                            line[4 * HL - 4 * d + i] = __shfl_up_sync(0xffffffffu, comp(yf[r], i), d);
                        if (4 * HL + 4 * d + i <= 4 * HL + 3 + RXY)
                            line[4 * HL + 4 * d + i] = __shfl_down_sync(0xffffffffu, comp(yf[r], i), d);
                    }
                }
                float o[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    float a = S.wx[0] * line[4 * HL - RXY + c];
#pragma unroll
                    for (int k = 1; k <= 2 * RXY; ++k) a = fmaf(S.wx[k], line[4 * HL - RXY + c + k], a);
                    o[c] = a;
                }
                win[RING + j][r] = F4{o[0], o[1], o[2], o[3]};
            }
        }
        // z pass: output plane zo = q_first + base + j - RZ uses win[j .. j + 2 RZ]
#pragma unroll
        for (int j = 0; j < ZB; ++j) {
            const int zo = q_first + base + j - RZ;
            if (zo >= z0 && zo < z1) {
                float *p = po + (size_t)zo * plane;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const F4 &f = win[j][r];
                    F4 a = F4{S.wz[0] * f.x, S.wz[0] * f.y, S.wz[0] * f.z, S.wz[0] * f.w};
#pragma unroll
                    for (int k = 1; k <= 2 * RZ; ++k) {
                        const F4 &g = win[j + k][r];
                        a.x = fmaf(S.wz[k], g.x, a.x);
                        a.y = fmaf(S.wz[k], g.y, a.y);
                        a.z = fmaf(S.wz[k], g.z, a.z);
                        a.w = fmaf(S.wz[k], g.w, a.w);
                    }
                    if (ok & (1u << r))
                        *reinterpret_cast<float4 *>(p + (size_t)r * S.nx) = make_float4(a.x, a.y, a.z, a.w);
                }
            }
        }
        // the last 2 RZ planes move to the front
#pragma unroll
        for (int k = 0; k < RING; ++k)
#pragma unroll
            for (int r = 0; r < R; ++r) win[k][r] = win[k + ZB][r];
    }
}

int pick_zchunk_big(int nz, long tiles, int rz, long slots)
{
    long best_cost = -1;
    int best = nz;
    for (int c = 1; c <= nz && c <= 4096; ++c) {
        const int zc = (nz + c - 1) / c;
        const long ctas = tiles * ((nz + zc - 1) / zc);
        const long cost = ((ctas + slots - 1) / slots) * (long)(zc + 2 * rz + 2);
        if (best_cost < 0 || cost < best_cost) { best_cost = cost; best = zc; }
        if (zc == 1) break;
    }
    return best;
}

template <int RXY, int RZ, int R, int WARPS, int NS, int ZB, int MINB>
cudaError_t launch_big(SepBigArgs &S, const float *in, int zchunk, cudaStream_t st)
{
    using G = BigGeo<RXY, R, WARPS, NS>;
    static_assert(G::kBytes * MINB <= 227 * 1024, "shared memory budget");
    const int nx4 = S.nx / 4;
    S.tiles_x = (nx4 + G::V - 1) / G::V;
    const long tiles_y = (S.ny + G::VY - 1) / G::VY;
    const long tiles = (long)S.tiles_x * tiles_y;
    if (tiles > 0x7fffffffL) return cudaErrorInvalidValue;
    S.zchunk = zchunk > 0 ? (zchunk < S.nz ? zchunk : S.nz) : pick_zchunk_big(S.nz, tiles, RZ, (long)device_sm_count() * MINB);
    if ((S.nz + S.zchunk - 1) / S.zchunk > 65535) S.zchunk = (S.nz + 65534) / 65535;
    CUtensorMap map;
    if (!tmap_encode(&map, in, S.nx, S.ny, S.nz, 1, kTileX, G::ROWS)) return cudaErrorNotSupported;
    auto kern = idg_sep3d_big_kernel<RXY, RZ, R, WARPS, NS, ZB, MINB>;
    static DeviceOnce smem_once;
    {
        const cudaError_t e = set_max_dynamic_smem(smem_once, (const void *)(kern), G::kBytes);
        if (e != cudaSuccess) return e;
    }
    const dim3 grid((unsigned)tiles, (unsigned)((S.nz + S.zchunk - 1) / S.zchunk));
    kern<<<grid, WARPS * 32, G::kBytes, st>>>(S, map);
    return cudaGetLastError();
}

}  // namespace

bool sep3d_big_supported(int nx, int ny, int nz, int rx, int ry, int rz, const void *in, const void *out)
{
    (void)ny; (void)nz;
    if (rx > kBigMaxR || ry > kBigMaxR || rz > kBigMaxR || nx % 4 != 0) return false;
    if ((((uintptr_t)in | (uintptr_t)out) & 15u) != 0) return false;
    return tmap_available();
}

// w*: 2r+1 normalised weights per axis, radii <= 9 (used for radii the radius-4 kernel does not take).  Radius classes
// 6 and 9 per axis group (xy, z); variant 2: the other strip height of class (6, 6).
cudaError_t launch_sep3d_big(const float *in, float *out, int nx, int ny, int nz, int rx, int ry, int rz,
                             const float *wx, const float *wy, const float *wz, int zchunk, int variant, cudaStream_t st)
{
    if (!sep3d_big_supported(nx, ny, nz, rx, ry, rz, in, out)) return cudaErrorNotSupported;
    const int mxy = rx > ry ? rx : ry;
    const int cxy = mxy <= 6 ? 6 : 9, cz = rz <= 6 ? 6 : 9;
    SepBigArgs S;
    S.out = out;
    S.nx = nx; S.ny = ny; S.nz = nz;
    for (int i = 0; i < 2 * kBigMaxR + 1; ++i) S.wx[i] = S.wy[i] = S.wz[i] = 0.f;
    for (int i = 0; i <= 2 * rx; ++i) S.wx[i + cxy - rx] = wx[i];        // centred in the class window
    for (int i = 0; i <= 2 * ry; ++i) S.wy[i + cxy - ry] = wy[i];
    for (int i = 0; i <= 2 * rz; ++i) S.wz[i + cz - rz] = wz[i];
    // strips of two rows at radius class 6 (211 registers, one 8-warp CTA per SM), single rows on 12 warps beyond
    // (the 18 + ZB planes of a column and the 19 window-row offsets need ~160 registers)
    if (cxy == 6 && cz == 6)
        return variant == 2 ? launch_big<6, 6, 1, 12, 4, 4, 1>(S, in, zchunk, st) : launch_big<6, 6, 2, 8, 4, 4, 1>(S, in, zchunk, st);
    if (cxy == 6) return launch_big<6, 9, 1, 12, 4, 6, 1>(S, in, zchunk, st);
    if (cz == 6) return launch_big<9, 6, 1, 12, 4, 4, 1>(S, in, zchunk, st);
    return launch_big<9, 9, 1, 12, 4, 6, 1>(S, in, zchunk, st);
}

}  // namespace idg
