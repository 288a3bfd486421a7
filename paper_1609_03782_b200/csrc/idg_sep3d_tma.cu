// Separable 3-D filter (box; axis-aligned Gaussian, Eq. 1-2) for radii <= 4 on
// 16-byte aligned cubes with nx % 4 == 0: the TMA-fed, barrier-free variant of idg_sep3d.cu.
//
//   out(x,y,z) = sum_k wz[k] sum_i wx[i] sum_j wy[j] I(cx(x+i), cy(y+j), cz(z+k)),   c. = clamp to the cube (reading F1)
//
// Decomposition of the IDG kernel (idg_tma.cu): a CTA owns a 128 x (WARPS*R) xy tile and streams along z; a thread
// owns a float4 column of an R-row strip.  Per input plane the raw tile plus RXY halo rows above and below arrives
// by TMA (one 128 x ROWS box, zero fill outside the cube, z clamped in the plane coordinate) in a ring of NS stages:
//   y pass  from shared memory: R + 2 RXY LDS.128 per thread, row offsets clamped to the cube once per CTA, streamed
//           row by row into the R accumulators (few live registers);
//   x pass  on the y-filtered strip by warp shuffles (a radius <= 4 reaches one float4 to either side; tiles
//           overlap by one lane on both sides; the lane just outside a cube face takes the replicated face value,
//           which is exact because the y pass is linear and acts column by column);
//   z pass  over a ring of 2 RZ + 1 xy-filtered planes in registers; the plane loop is unrolled over the ring phases,
//           so the ring rotates by register renaming, not by moves.
// No thread reads what another thread computed, so the plane loop has NO CTA barrier: a stage is handed back to the
// producer thread through an `empty` mbarrier (one arrival per warp, right after the warp has read its window) and
// refilled NS-2 planes ahead.  The cube is read once and written once: 8 B per voxel.
#include <cuda.h>

#include "idg_kernels.cuh"
#include "idg_ptx.cuh"

namespace idg {

namespace {

constexpr int kValidLanes = 30;
constexpr int kTileX = 128;
constexpr int kMaxR = 4;

struct F4 { float x, y, z, w; };

__device__ __forceinline__ F4 lds4(const float *p)
{
    const float4 v = *reinterpret_cast<const float4 *>(p);
    return F4{v.x, v.y, v.z, v.w};
}
__device__ __forceinline__ float comp(const F4 &a, int i) { return i == 0 ? a.x : (i == 1 ? a.y : (i == 2 ? a.z : a.w)); }

struct SepTmaArgs {
    float *out;
    int nx, ny, nz;
    int tiles_x, zchunk;
    float wx[2 * kMaxR + 1], wy[2 * kMaxR + 1], wz[2 * kMaxR + 1];     // zero-padded to the class width
};

template <int RXY, int R, int WARPS, int NS>
struct SepGeo {
    static constexpr int VY = WARPS * R;                 // output rows per tile
    static constexpr int ROWS = VY + 2 * RXY;            // rows loaded per plane
    static constexpr int kStageFloats = ROWS * kTileX;
    static constexpr size_t kStageBytes = (size_t)kStageFloats * sizeof(float);
    static constexpr size_t kBarOff = NS * kStageBytes;
    static constexpr size_t kBytes = kBarOff + 2 * NS * sizeof(uint64_t);
};

template <int RXY, int RZ, int R, int WARPS, int NS, int MINB>
__global__ void __launch_bounds__(WARPS * 32, MINB)
idg_sep3d_tma_kernel(const __grid_constant__ SepTmaArgs S, const __grid_constant__ CUtensorMap map)
{
    using G = SepGeo<RXY, R, WARPS, NS>;
    constexpr int W = 2 * RZ + 1, WIN = R + 2 * RXY, AHEAD = NS - 2;
    extern __shared__ __align__(1024) unsigned char smem[];
    float *stage0 = reinterpret_cast<float *>(smem);
    const uint32_t full = ptx::smem_u32(smem + G::kBarOff), empty = full + NS * 8;

    const int lane = threadIdx.x & 31, wy = threadIdx.x >> 5;
    const int nx4 = S.nx >> 2;
    const int ti = blockIdx.x % S.tiles_x, tj = blockIdx.x / S.tiles_x;
    const int x4 = ti * kValidLanes - 1 + lane;
    const int tx0 = (ti * kValidLanes - 1) * 4;          // cube x of tile column 0
    const int ty0 = tj * G::VY;                          // cube y of the first output row
    const int z0 = blockIdx.y * S.zchunk, z1 = min(z0 + S.zchunk, S.nz);
    const int q_first = z0 - RZ, q_last = z1 - 1 + RZ;
    const bool left_halo = x4 < 0, right_halo = x4 >= nx4;
    const bool edge_x = ti == 0 || (ti + 1) * kValidLanes >= nx4;      // the tile touches an x face (CTA uniform)

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
        if (lane >= 1 && lane <= kValidLanes && x4 < nx4 && ty0 + wy * R + r < S.ny) ok |= 1u << r;

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

    F4 ring[W][R];
#pragma unroll
    for (int k = 0; k < W; ++k)
#pragma unroll
        for (int r = 0; r < R; ++r) ring[k][r] = F4{0.f, 0.f, 0.f, 0.f};

    const size_t plane = (size_t)S.nx * (size_t)S.ny;
    float *po = S.out + (size_t)(ty0 + wy * R) * S.nx + (long long)x4 * 4;

    int it = 0;
    bool more = n_planes > 0;
    while (more) {
#pragma unroll
        for (int P = 0; P < W; ++P) {       // P = ring phase (compile time after unrolling)
            const int s = it % NS;
            if (threadIdx.x == 0 && it + AHEAD < n_planes) {
                const int i = it + AHEAD;   // its stage held plane it - 2: wait until every warp has read it
                if (i >= NS) ptx::mbar_wait_spin(empty + 8 * (i % NS), (uint32_t)((i / NS - 1) & 1));
                issue(i);
            }
            const float *st = stage0 + (size_t)s * G::kStageFloats;
            ptx::mbar_wait_spin(full + 8 * s, (uint32_t)((it / NS) & 1));

            // y pass, streamed over the window rows (row j feeds output row r with weight k = j - r): few live registers
            F4 yf[R];
#pragma unroll
            for (int j = 0; j < WIN; ++j) {
                const F4 w = lds4(st + roff[j]);
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int k = j - r;
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
            if (edge_x) {                   // replicated x faces: the lane just outside takes the face value
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const float a = __shfl_down_sync(0xffffffffu, yf[r].x, 1);
                    const float b = __shfl_up_sync(0xffffffffu, yf[r].w, 1);
                    if (left_halo) yf[r] = F4{a, a, a, a};
                    else if (right_halo) yf[r] = F4{b, b, b, b};
                }
            }
            // x pass -> newest ring plane
#pragma unroll
            for (int r = 0; r < R; ++r) {
                float line[12];
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    line[4 + i] = comp(yf[r], i);
                    if (i >= 4 - RXY) line[i] = __shfl_up_sync(0xffffffffu, comp(yf[r], i), 1);
                    if (i < RXY) line[8 + i] = __shfl_down_sync(0xffffffffu, comp(yf[r], i), 1);
                }
                float o[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    float a = S.wx[0] * line[4 - RXY + c];
#pragma unroll
                    for (int k = 1; k <= 2 * RXY; ++k) a = fmaf(S.wx[k], line[4 - RXY + c + k], a);
                    o[c] = a;
                }
                ring[P][r] = F4{o[0], o[1], o[2], o[3]};
            }
            // z pass: window plane k = ring[(P + 1 + k) % W], k = W - 1 is the newest
            const int zo = q_first + it - RZ;
            if (zo >= z0) {
                float *p = po + (size_t)zo * plane;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const F4 &f = ring[(P + 1) % W][r];
                    F4 a = F4{S.wz[0] * f.x, S.wz[0] * f.y, S.wz[0] * f.z, S.wz[0] * f.w};
#pragma unroll
                    for (int k = 1; k < W; ++k) {
                        const F4 &g = ring[(P + 1 + k) % W][r];
                        a.x = fmaf(S.wz[k], g.x, a.x);
                        a.y = fmaf(S.wz[k], g.y, a.y);
                        a.z = fmaf(S.wz[k], g.z, a.z);
                        a.w = fmaf(S.wz[k], g.w, a.w);
                    }
                    if (ok & (1u << r))
                        *reinterpret_cast<float4 *>(p + (size_t)r * S.nx) = make_float4(a.x, a.y, a.z, a.w);
                }
            }
            ++it;
            if (it >= n_planes) { more = false; break; }
        }
    }
}

int pick_zchunk(int nz, long tiles, int rz, long slots)
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

template <int RXY, int RZ, int R, int WARPS, int NS, int MINB>
cudaError_t launch_cfg(SepTmaArgs &S, const float *in, int zchunk, cudaStream_t st)
{
    using G = SepGeo<RXY, R, WARPS, NS>;
    static_assert(G::kBytes * MINB <= 227 * 1024, "shared memory budget");
    const int nx4 = S.nx / 4;
    S.tiles_x = (nx4 + kValidLanes - 1) / kValidLanes;
    const long tiles_y = (S.ny + G::VY - 1) / G::VY;
    const long tiles = (long)S.tiles_x * tiles_y;
    if (tiles > 0x7fffffffL) return cudaErrorInvalidValue;
    S.zchunk = zchunk > 0 ? (zchunk < S.nz ? zchunk : S.nz) : pick_zchunk(S.nz, tiles, RZ, (long)device_sm_count() * MINB);
    if ((S.nz + S.zchunk - 1) / S.zchunk > 65535) S.zchunk = (S.nz + 65534) / 65535;
    CUtensorMap map;
    if (!tmap_encode(&map, in, S.nx, S.ny, S.nz, 1, kTileX, G::ROWS)) return cudaErrorNotSupported;
    auto kern = idg_sep3d_tma_kernel<RXY, RZ, R, WARPS, NS, MINB>;
    static DeviceOnce smem_once;
    {
        const cudaError_t e = set_max_dynamic_smem(smem_once, (const void *)(kern), G::kBytes);
        if (e != cudaSuccess) return e;
    }
    const dim3 grid((unsigned)tiles, (unsigned)((S.nz + S.zchunk - 1) / S.zchunk));
    kern<<<grid, WARPS * 32, G::kBytes, st>>>(S, map);
    return cudaGetLastError();
}

// Register budget: the z ring costs 4 R (2 RZ + 1) registers, the y window 4 (R + 2 RXY).  variant 0, 1 (default;
// measured faster everywhere, profiles/r1i_notes.md): strips of 2 rows (RZ = 1: three 8-warp CTAs per SM, two for
// RXY = 4; RZ = 2: two; RZ = 4: one 12-warp CTA); variant 2: strips of 4 rows on eight warps (RZ = 1, RXY <= 2: two
// CTAs per SM; else one).
template <int RXY, int RZ>
cudaError_t launch_class(SepTmaArgs &S, const float *in, int zchunk, int variant, cudaStream_t st)
{
    if constexpr (RZ == 1 && RXY <= 2) {
        return variant != 2 ? launch_cfg<RXY, RZ, 2, 8, 4, 3>(S, in, zchunk, st) : launch_cfg<RXY, RZ, 4, 8, 4, 2>(S, in, zchunk, st);
    } else if constexpr (RZ <= 2) {
        return variant != 2 ? launch_cfg<RXY, RZ, 2, 8, 4, 2>(S, in, zchunk, st) : launch_cfg<RXY, RZ, 4, 8, 4, 1>(S, in, zchunk, st);
    } else {
        return variant != 2 ? launch_cfg<RXY, RZ, 2, 12, 4, 1>(S, in, zchunk, st) : launch_cfg<RXY, RZ, 4, 8, 4, 1>(S, in, zchunk, st);
    }
}

template <int RXY>
cudaError_t launch_rz(int cz, SepTmaArgs &S, const float *in, int zchunk, int variant, cudaStream_t st)
{
    switch (cz) {
    case 1: return launch_class<RXY, 1>(S, in, zchunk, variant, st);
    case 2: return launch_class<RXY, 2>(S, in, zchunk, variant, st);
    default: return launch_class<RXY, 4>(S, in, zchunk, variant, st);
    }
}

inline int class_of(int r) { return r <= 1 ? 1 : (r <= 2 ? 2 : 4); }

}  // namespace

bool sep3d_tma_supported(int nx, int ny, int nz, int rx, int ry, int rz, const void *in, const void *out)
{
    (void)ny; (void)nz;
    if (rx > kMaxR || ry > kMaxR || rz > kMaxR || nx % 4 != 0) return false;
    if ((((uintptr_t)in | (uintptr_t)out) & 15u) != 0) return false;
    return tmap_available();
}

// w*: 2r+1 normalised weights per axis, radii <= 4.  variant: 0, 1 strips of 2 rows (default) | 2 strips of 4 rows.
cudaError_t launch_sep3d_tma(const float *in, float *out, int nx, int ny, int nz, int rx, int ry, int rz,
                             const float *wx, const float *wy, const float *wz, int zchunk, int variant, cudaStream_t st)
{
    if (!sep3d_tma_supported(nx, ny, nz, rx, ry, rz, in, out)) return cudaErrorNotSupported;
    const int cxy = class_of(rx > ry ? rx : ry), cz = class_of(rz);
    SepTmaArgs S;
    S.out = out;
    S.nx = nx; S.ny = ny; S.nz = nz;
    for (int i = 0; i < 2 * kMaxR + 1; ++i) S.wx[i] = S.wy[i] = S.wz[i] = 0.f;
    for (int i = 0; i <= 2 * rx; ++i) S.wx[i + cxy - rx] = wx[i];        // centred in the class window
    for (int i = 0; i <= 2 * ry; ++i) S.wy[i + cxy - ry] = wy[i];
    for (int i = 0; i <= 2 * rz; ++i) S.wz[i + cz - rz] = wz[i];
    switch (cxy) {
    case 1: return launch_rz<1>(cz, S, in, zchunk, variant, st);
    case 2: return launch_rz<2>(cz, S, in, zchunk, variant, st);
    default: return launch_rz<4>(cz, S, in, zchunk, variant, st);
    }
}

}  // namespace idg
