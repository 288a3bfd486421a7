// Tiled z-streaming IDG kernel with temporal fusion (steps a1-a6 of DESIGN.md section 7).
//
// One CTA owns an xy tile of 128 x (WARPS*R) voxels and marches along z (the slowest
// axis) through its z-chunk.  A thread owns one float4 column (4 voxels along x) of an
// R-row strip, and for each of the T fused time levels keeps the previous and current
// z-plane of that strip in registers.  Neighbours:
//   z +-1   registers (the per-level z ring)
//   y +-1   registers inside the strip; the strips' edge rows go through shared memory
//   x +-1   warp shuffles (a warp spans the tile's 128 voxels along x)
// T iterations of Eq. 7 are applied per launch: while level-0 plane q is
// loaded, level t+1 is produced for plane q-t-1, so the cube is read and written once
// per T iterations instead of once per iteration.
//
// Boundary (reading R1): the cube is extended by even reflection (I(-1) = I(0),
// I(-2) = I(1), ...) when level-0 planes are loaded.  The update is symmetric under that
// reflection, so every fused level keeps I_t(-1) == I_t(0) bit for bit, which IS the
// zero-flux replicate condition -- the inner loop needs no boundary predicates at all.
//
// Tile halo: T voxels in y and one float4 (4 voxels) in x on each side are recomputed by
// neighbouring CTAs; 2T planes at each end of a z-chunk likewise.
#include "idg_kernels.cuh"

namespace idg {

namespace {

constexpr int kLanes = 32;            // float4 columns per tile row (one warp)
constexpr int kValidLanes = 30;       // lanes 1..30 produce output; 0 and 31 are x halo

__device__ __forceinline__ int mirror(int i, int n)
{
    const int p = 2 * n;
    int m = i % p;
    if (m < 0) m += p;
    return m < n ? m : p - 1 - m;
}

struct F4 { float x, y, z, w; };

__device__ __forceinline__ F4 ld4(const float *p)
{
    const float4 v = __ldg(reinterpret_cast<const float4 *>(p));
    return F4{v.x, v.y, v.z, v.w};
}

// Four voxel updates (Eq. 7) of one float4 column: c with its six neighbour vectors.
__device__ __forceinline__ F4 update4(const F4 &c, float left, float right, const F4 &ym, const F4 &yp,
                                      const F4 &zm, const F4 &zp, const CubeParams &p)
{
    F4 o;
    o.x = update(c.x, left, c.y, ym.x, yp.x, zm.x, zp.x, p.ax, p.ay, p.az, p.s, p.w);
    o.y = update(c.y, c.x, c.z, ym.y, yp.y, zm.y, zp.y, p.ax, p.ay, p.az, p.s, p.w);
    o.z = update(c.z, c.y, c.w, ym.z, yp.z, zm.z, zp.z, p.ax, p.ay, p.az, p.s, p.w);
    o.w = update(c.w, c.z, right, ym.w, yp.w, zm.w, zp.w, p.ax, p.ay, p.az, p.s, p.w);
    return o;
}

struct TileArgs {
    int tiles_x, tiles_y;   // tiles per plane
    int zchunk;             // output planes per CTA
    int halo;               // y halo rows of this launch's tiling (= L.fuse)
};

// TL = time levels applied by this CTA (<= halo), R = rows per thread, WARPS = strips per tile.
template <int TL, int R, int WARPS>
__device__ __forceinline__ void tile_body(const float *__restrict__ src, float *__restrict__ dst,
                                          const Launch &L, const TileArgs &A, const CubeParams &prm,
                                          float4 *edge /* [TL][2][WARPS][2][32] */)
{
    constexpr int TILE_Y = WARPS * R;
    const int lane = threadIdx.x & 31;
    const int wy = threadIdx.x >> 5;
    const int nx4 = L.nx >> 2;
    const int vy = TILE_Y - 2 * A.halo;                 // valid rows per tile

    const int tile = blockIdx.x;
    const int ti = tile % A.tiles_x, tj = tile / A.tiles_x;
    const int x4 = ti * kValidLanes - 1 + lane;          // float4 column of this lane (may be outside)
    const int row0 = wy * R;                             // first tile row of this strip
    const int gy0 = tj * vy - A.halo + row0;             // cube row of strip row 0 (may be outside)
    const int z0 = blockIdx.y * A.zchunk;
    const int z1 = min(z0 + A.zchunk, L.nz);

    // level-0 source addresses (even reflection about the cube faces)
    int xs = x4 % (2 * nx4);
    if (xs < 0) xs += 2 * nx4;
    const bool rev = xs >= nx4;                          // reflected column: components reversed
    if (rev) xs = 2 * nx4 - 1 - xs;
    size_t roff[R];
    unsigned ok = 0;                                     // bit r: this thread stores row r
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int gy = gy0 + r;
        roff[r] = (size_t)mirror(gy, L.ny) * (size_t)L.nx + (size_t)xs * 4;
        const int row = row0 + r;
        if (lane >= 1 && lane <= kValidLanes && x4 < nx4 && row >= A.halo && row < TILE_Y - A.halo &&
            gy < L.ny)
            ok |= 1u << r;
    }
    const size_t plane = (size_t)L.nx * (size_t)L.ny;
    const long long ooff = (long long)gy0 * L.nx + (long long)x4 * 4;   // dereferenced only where ok

    F4 zm[TL][R], cc[TL][R];
#pragma unroll
    for (int t = 0; t < TL; ++t)
#pragma unroll
        for (int r = 0; r < R; ++r) {
            zm[t][r] = F4{0.f, 0.f, 0.f, 0.f};
            cc[t][r] = F4{0.f, 0.f, 0.f, 0.f};
        }

    auto load_plane = [&](int q, F4 (&v)[R]) {
        const float *pz = src + (size_t)mirror(q, L.nz) * plane;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            F4 a = ld4(pz + roff[r]);
            if (rev) a = F4{a.w, a.z, a.y, a.x};
            v[r] = a;
        }
    };

    const int q_first = z0 - TL, q_last = z1 - 1 + TL;
    F4 nxt[R];
    load_plane(q_first, nxt);
    int par = 0;
    for (int q = q_first; q <= q_last; ++q) {
        F4 zp[R];
#pragma unroll
        for (int r = 0; r < R; ++r) zp[r] = nxt[r];
        if (q < q_last) load_plane(q + 1, nxt);          // in flight while this step computes

#pragma unroll
        for (int t = 0; t < TL; ++t) {
            // zp = level-t plane (q - t); cc[t] = plane (q - t - 1); zm[t] = plane (q - t - 2)
            float4 *e_rd = edge + ((t * 2 + par) * WARPS) * 2 * kLanes;
            float4 *e_wr = edge + ((t * 2 + (par ^ 1)) * WARPS) * 2 * kLanes;
            e_wr[(wy * 2 + 0) * kLanes + lane] = make_float4(zp[0].x, zp[0].y, zp[0].z, zp[0].w);
            e_wr[(wy * 2 + 1) * kLanes + lane] =
                make_float4(zp[R - 1].x, zp[R - 1].y, zp[R - 1].z, zp[R - 1].w);
            F4 up = cc[t][0], dn = cc[t][R - 1];          // tile-edge strips: halo rows, any finite value
            if (wy > 0) {
                const float4 v = e_rd[((wy - 1) * 2 + 1) * kLanes + lane];
                up = F4{v.x, v.y, v.z, v.w};
            }
            if (wy < WARPS - 1) {
                const float4 v = e_rd[((wy + 1) * 2 + 0) * kLanes + lane];
                dn = F4{v.x, v.y, v.z, v.w};
            }
            F4 out[R];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const F4 &c = cc[t][r];
                const float left = __shfl_up_sync(0xffffffffu, c.w, 1);
                const float right = __shfl_down_sync(0xffffffffu, c.x, 1);
                const F4 &ym = (r == 0) ? up : cc[t][r - 1];
                const F4 &yp = (r == R - 1) ? dn : cc[t][r + 1];
                out[r] = update4(c, left, right, ym, yp, zm[t][r], zp[r], prm);
            }
#pragma unroll
            for (int r = 0; r < R; ++r) {
                zm[t][r] = cc[t][r];
                cc[t][r] = zp[r];
                zp[r] = out[r];                           // level t+1, plane (q - t - 1)
            }
        }
        // zp = level-TL plane (q - TL)
        const int zo = q - TL;
        if (zo >= z0 && zo < z1) {
            float *po = dst + (long long)((size_t)zo * plane) + ooff;
#pragma unroll
            for (int r = 0; r < R; ++r)
                if (ok & (1u << r))
                    *reinterpret_cast<float4 *>(po + (long long)r * L.nx) =
                        make_float4(zp[r].x, zp[r].y, zp[r].z, zp[r].w);
        }
        par ^= 1;
        __syncthreads();
    }
}

template <int T, int R, int WARPS>
__global__ void __launch_bounds__(WARPS * 32, 1)
idg_tiled_kernel(const __grid_constant__ Launch L, const __grid_constant__ TileArgs A)
{
    extern __shared__ float4 edge[];
    const int b = blockIdx.z;
    const CubeParams prm = cube_params(L, b);
    const float *src;
    float *dst;
    const int now = route(L, b, prm, src, dst);
    if (now == 0) return;
    // `now` is uniform over the CTA; fewer levels than T only on a cube's last launch
    if (now == T) tile_body<T, R, WARPS>(src, dst, L, A, prm, edge);
    else if (T > 1 && now == 1) tile_body<1, R, WARPS>(src, dst, L, A, prm, edge);
    else if (T > 2 && now == 2) tile_body<(T > 2 ? 2 : 1), R, WARPS>(src, dst, L, A, prm, edge);
    else if (T > 3 && now == 3) tile_body<(T > 3 ? 3 : 1), R, WARPS>(src, dst, L, A, prm, edge);
}

// z-chunk length minimising waves * (planes per CTA) with one CTA per SM of the current device.
int pick_zchunk(int nz, int tiles, int T)
{
    const long sms = device_sm_count();
    long best_cost = -1;
    int best = nz;
    for (int nchunks = 1; nchunks <= nz; ++nchunks) {
        const int zc = (nz + nchunks - 1) / nchunks;
        const int real_chunks = (nz + zc - 1) / zc;
        const long ctas = (long)tiles * real_chunks;
        const long waves = (ctas + sms - 1) / sms;
        const long cost = waves * (zc + 2 * T + 2);      // +2: per-CTA prologue, in plane-steps
        if (best_cost < 0 || cost < best_cost) {
            best_cost = cost;
            best = zc;
        }
        if (zc == 1) break;
    }
    return best;
}

template <int T, int R, int WARPS>
cudaError_t launch_cfg(const Launch &L, int zchunk, cudaStream_t st)
{
    constexpr int TILE_Y = WARPS * R;
    static_assert(TILE_Y > 2 * T, "tile must be taller than its halo");
    TileArgs A;
    A.halo = T;
    const int nx4 = L.nx / 4;
    A.tiles_x = (nx4 + kValidLanes - 1) / kValidLanes;
    A.tiles_y = (L.ny + (TILE_Y - 2 * T) - 1) / (TILE_Y - 2 * T);
    const int tiles = A.tiles_x * A.tiles_y;
    A.zchunk = zchunk > 0 ? (zchunk < L.nz ? zchunk : L.nz) : pick_zchunk(L.nz, tiles * L.batch, T);
    const int chunks = (L.nz + A.zchunk - 1) / A.zchunk;
    if (chunks > 65535) A.zchunk = (L.nz + 65534) / 65535;
    const size_t smem = (size_t)T * 2 * WARPS * 2 * kLanes * sizeof(float4);
    auto kern = idg_tiled_kernel<T, R, WARPS>;
    static DeviceOnce smem_once;
    {
        const cudaError_t e = set_max_dynamic_smem(smem_once, (const void *)(kern), smem);
        if (e != cudaSuccess) return e;
    }
    dim3 grid((unsigned)tiles, (unsigned)((L.nz + A.zchunk - 1) / A.zchunk), (unsigned)L.batch);
    kern<<<grid, WARPS * 32, smem, st>>>(L, A);
    return cudaGetLastError();
}

}  // namespace

bool tiled_supported(int nx, int ny, int nz, const void *in, const void *out, const void *scratch)
{
    (void)ny; (void)nz;
    if (nx % 4 != 0) return false;
    const uintptr_t m = (uintptr_t)in | (uintptr_t)out | (uintptr_t)scratch;
    return (m & 15u) == 0;
}

cudaError_t launch_tiled(const Launch &L, int zchunk, cudaStream_t st)
{
    switch (L.fuse) {
    case 1: return launch_cfg<1, 4, 16>(L, zchunk, st);
    case 2: return launch_cfg<2, 4, 16>(L, zchunk, st);
    case 3: return launch_cfg<3, 4, 8>(L, zchunk, st);
    case 4: return launch_cfg<4, 4, 8>(L, zchunk, st);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace idg
