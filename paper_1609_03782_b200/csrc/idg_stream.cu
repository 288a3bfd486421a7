// Persistent, warp-decoupled, TMA-fed, temporally fused IDG kernel (steps a1-a6 of SURVEY.md 8(a)).
//
// Decomposition.  The (cube, xy-tile, z) space of a launch is flattened into "tile-planes"
// g = tile_id * nz + z and split evenly over a persistent grid (one range [g0, g1) per CTA; a
// range is cut into segments at tile borders).  A CTA streams its segments plane by plane: a
// warp owns R rows x 128 columns of the 128 x (WARPS*R) tile, a thread a float4 column of that
// strip.  x neighbours come by warp shuffle, y neighbours are registers inside the strip and
// shared memory between strips, z neighbours are three-deep register rings per fused level, so
// TL Jacobi iterations (Eq. 7) are applied per pass over the data.
//
// Pipeline.  Level-0 planes are loaded by TMA (cp.async.bulk.tensor, box 128 x TILE_Y x 1 x 1)
// into a ring of NS shared-memory stages.  There is no CTA-wide barrier in the plane loop:
//   * a stage is handed back by a shared counter; the last warp to release it issues the next
//     load into it (any warp can be the producer, nobody waits for the slowest warp);
//   * strips exchange their edge rows through double-buffered shared slots guarded by one
//     mbarrier per warp and step parity, so a warp only ever waits for its two neighbours.
//
// Boundary (reading R1, zero flux by replication).  TMA zero-fills outside the cube;
// a thread whose cell lies within one reflection outside a face reads the even-reflected cell
// instead (x: mirrored lane with reversed components, y: mirrored row, z: mirrored TMA plane
// coordinate).  Eq. 7 is symmetric under the reflection, hence every fused level satisfies the
// replicate condition bit for bit with no predicate in the arithmetic.
#include <type_traits>

#include "idg_kernels.cuh"
#include "idg_ptx.cuh"

namespace idg {

namespace {

using namespace ptx;

constexpr int kLanes = 32;
constexpr int kValidLanes = 30;
constexpr int kTileX = 128;
constexpr uint32_t kRowBytes = kTileX * 4;

struct F4 { float x, y, z, w; };

__device__ __forceinline__ F4 ld4(uint32_t a)
{
    const float4 v = lds128(a);
    return F4{v.x, v.y, v.z, v.w};
}
__device__ __forceinline__ F4 reversed(const F4 &a) { return F4{a.w, a.z, a.y, a.x}; }

// Four voxel updates of one float4 column with packed fp32x2 arithmetic.  Each component rounds
// exactly like the scalar update() of idg_kernels.cuh (same operations in the same order).
struct Consts { float2 m2, ax, ay, az, s, one; };
__device__ __forceinline__ Consts make_consts(const CubeParams &p)
{
    Consts k;
    k.m2 = make_float2(-2.0f, -2.0f);
    k.ax = make_float2(p.ax, p.ax);
    k.ay = make_float2(p.ay, p.ay);
    k.az = make_float2(p.az, p.az);
    k.s = make_float2(p.s, p.s);
    k.one = make_float2(1.0f, 1.0f);
    return k;
}
__device__ __forceinline__ float2 update2(float2 c, float2 sx, float2 ym, float2 yp, float2 zm, float2 zp,
                                          const Consts &k)
{
    const float2 dx = __ffma2_rn(k.m2, c, sx);
    const float2 dy = __ffma2_rn(k.m2, c, __fadd2_rn(yp, ym));
    const float2 dz = __ffma2_rn(k.m2, c, __fadd2_rn(zp, zm));
    const float2 lap = __ffma2_rn(k.az, dz, __ffma2_rn(k.ay, dy, __fmul2_rn(k.ax, dx)));
    const float2 u = __fmul2_rn(c, k.s);
    const float2 den = __ffma2_rn(u, u, k.one);
    const float2 r = make_float2(rcp_approx(den.x), rcp_approx(den.y));
    return __ffma2_rn(lap, r, c);
}
__device__ __forceinline__ F4 update4(const F4 &c, float left, float right, const F4 &ym, const F4 &yp,
                                      const F4 &zm, const F4 &zp, const Consts &k)
{
    const float2 sx01 = make_float2(c.y + left, c.z + c.x);
    const float2 sx23 = make_float2(c.w + c.y, right + c.z);
    const float2 o01 = update2(make_float2(c.x, c.y), sx01, make_float2(ym.x, ym.y), make_float2(yp.x, yp.y),
                               make_float2(zm.x, zm.y), make_float2(zp.x, zp.y), k);
    const float2 o23 = update2(make_float2(c.z, c.w), sx23, make_float2(ym.z, ym.w), make_float2(yp.z, yp.w),
                               make_float2(zm.z, zm.w), make_float2(zp.z, zp.w), k);
    return F4{o01.x, o01.y, o23.x, o23.y};
}

__device__ __forceinline__ int mirror(int i, int n)
{
    const int p = 2 * n;
    int m = i % p;
    if (m < 0) m += p;
    return m < n ? m : p - 1 - m;
}

struct StreamArgs {
    int tiles_x, tiles_y;         // xy tiles per cube
    int vy;                       // valid rows per tile = TILE_Y - 2*halo
    int halo;                     // = fuse (T) of the plan
    unsigned long long planes;    // tile-planes of the launch = batch * tiles_x * tiles_y * nz
};

struct Maps {
    CUtensorMap in, out, scratch; // the three cubes (batch as 4th dimension) a launch may read
};

template <int T, int R, int WARPS, int NS>
struct Lay {
    static constexpr int TILE_Y = WARPS * R;
    static constexpr uint32_t kStage = (uint32_t)TILE_Y * kRowBytes;
    static constexpr uint32_t kEdgeLevel = 2u * WARPS * 2u * kLanes * 16u;      // both parities of one level
    static constexpr uint32_t kEdge = (uint32_t)(T > 1 ? T - 1 : 0) * kEdgeLevel;
    static constexpr uint32_t oEdge = NS * kStage;
    static constexpr uint32_t oFull = oEdge + kEdge;                            // NS mbarriers
    static constexpr uint32_t oNb = oFull + NS * 8u;                            // 2 * WARPS mbarriers
    static constexpr uint32_t oCnt = oNb + 2u * WARPS * 8u;                     // NS release counters
    static constexpr uint32_t kBytes = oCnt + NS * 4u;
};

// A position in the CTA's stream of plane jobs: level-0 plane q of xy tile `tile` (global tile
// index over the batch).  A segment produces output planes [z0, z1) from level-0 planes
// [z0-TL, z1-1+TL]; qs = z0+TL is the first job of the segment that stores a plane.
struct Cursor {
    unsigned long long g_end;     // end of the run (tile-planes)
    unsigned tile;
    int q, q_last, qs;
    bool live;
};

template <int TL>
__device__ __forceinline__ void cursor_open(Cursor &c, unsigned long long g, unsigned long long g_end, int nz)
{
    c.g_end = g_end;
    c.live = g < g_end;
    c.tile = (unsigned)(g / (unsigned)nz);
    const int z0 = (int)(g - (unsigned long long)c.tile * (unsigned)nz);
    const unsigned long long room = g_end - g;
    const int z1 = (room < (unsigned long long)(nz - z0)) ? z0 + (int)room : nz;
    c.q = z0 - TL;
    c.qs = z0 + TL;
    c.q_last = z1 - 1 + TL;
}
// Advance by one plane job; returns true when a new segment (tile) starts.
template <int TL>
__device__ __forceinline__ bool cursor_next(Cursor &c, int nz)
{
    if (c.q < c.q_last) { ++c.q; return false; }
    cursor_open<TL>(c, (unsigned long long)(c.tile + 1) * (unsigned)nz, c.g_end, nz);
    return true;
}

struct TileXY { int tx0, ty0, b; };
__device__ __forceinline__ TileXY tile_xy(unsigned tile, const StreamArgs &A)
{
    const unsigned per = (unsigned)(A.tiles_x * A.tiles_y);
    const unsigned b = tile / per, t = tile - b * per;
    const int tj = (int)(t / (unsigned)A.tiles_x), ti = (int)(t - (unsigned)tj * A.tiles_x);
    return TileXY{(ti * kValidLanes - 1) * 4, tj * A.vy - A.halo, (int)b};
}

// Persistent per-thread pipeline state (survives across runs of different TL).
struct Pipe {
    unsigned it;                  // plane jobs consumed so far by this CTA
};

// One thread: load the level-0 plane that lies `ahead` jobs after cursor `c` (job number `job`).
template <int TL, int NS, class Y>
__device__ __noinline__ void issue_ahead(const Launch &L, const StreamArgs &A, const Maps &M, Cursor c, int ahead,
                                         unsigned job, uint32_t sbase)
{
    for (int i = 0; i < ahead && c.live; ++i) cursor_next<TL>(c, L.nz);
    if (!c.live) return;
    const TileXY xy = tile_xy(c.tile, A);
    const CubeParams p = cube_params(L, xy.b);
    const float *src;
    float *dst;
    route(L, xy.b, p, src, dst);
    const size_t off = (size_t)xy.b * (size_t)L.nx * (size_t)L.ny * (size_t)L.nz;
    const CUtensorMap *map = (src == L.scratch + off) ? &M.scratch : (src == L.out + off) ? &M.out : &M.in;
    const unsigned s = job % NS;
    const uint32_t bar = sbase + Y::oFull + s * 8u;
    fence_proxy_async();
    mbar_expect_tx(bar, Y::kStage);
    tma_load_4d(sbase + s * Y::kStage, map, bar, xy.tx0, xy.ty0, mirror(c.q, L.nz), xy.b);
}

// One run: consecutive plane jobs [g, g_end) whose cubes all take TL iterations in this launch.
template <int TL, int R, int WARPS, int NS, int TMAX>
__device__ __forceinline__ void run(const Launch &L, const StreamArgs &A, const Maps &M, unsigned long long g,
                                    unsigned long long g_end, Pipe &P, uint32_t sbase)
{
    using Y = Lay<TMAX, R, WARPS, NS>;
    constexpr int TILE_Y = WARPS * R;
    const int lane = threadIdx.x & 31;
    const int wy = threadIdx.x >> 5;
    const int row0 = wy * R;
    const size_t plane = (size_t)L.nx * (size_t)L.ny;

    Cursor cur;
    cursor_open<TL>(cur, g, g_end, L.nz);
    // prologue: jobs it .. it+NS-2 (their stages were released by everybody before the last drain)
    if (threadIdx.x == 0) {
        for (int i = 0; i < NS - 1; ++i) issue_ahead<TL, NS, Y>(L, A, M, cur, i, P.it + i, sbase);
    }

    // per-segment thread state
    uint32_t own = 0;                         // byte offset of my (possibly x-mirrored) row-0 cell in a stage
    bool rev = false, ymir = false;
    unsigned ok = 0;
    int ty0 = 0;
    float *po = nullptr;
    Consts kc;
    auto mrow = [&](int row) -> uint32_t {   // tile row to read for tile row `row` (mirrored outside the cube)
        int gy = ty0 + row;
        if (gy < 0) gy = -1 - gy;
        else if (gy >= L.ny) gy = 2 * L.ny - 1 - gy;
        int srow = gy - ty0;
        if (srow < 0 || srow >= TILE_Y) srow = row;
        return (uint32_t)srow * kRowBytes;
    };
    auto segment_setup = [&]() {
        const TileXY xy = tile_xy(cur.tile, A);
        ty0 = xy.ty0;
        const CubeParams prm = cube_params(L, xy.b);
        const float *src;
        float *dst;
        route(L, xy.b, prm, src, dst);
        kc = make_consts(prm);
        const int nx4 = L.nx >> 2;
        const int x4 = (xy.tx0 >> 2) + lane;
        int slane = lane;
        rev = false;
        if (x4 < 0) { slane = lane + (-1 - x4) - x4; rev = true; }
        else if (x4 >= nx4) { slane = lane + (2 * nx4 - 1 - x4) - x4; rev = true; }
        if (slane < 0 || slane >= kLanes) { slane = lane; rev = false; }
        own = (uint32_t)row0 * kRowBytes + (uint32_t)slane * 16u;
        ymir = (ty0 + row0 - 1 < 0) || (ty0 + row0 + R >= L.ny);     // a row of rows row0-1 .. row0+R is outside
        ok = 0;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int row = row0 + r, gy = ty0 + row;
            if (lane >= 1 && lane <= kValidLanes && x4 < nx4 && row >= A.halo && row < TILE_Y - A.halo && gy < L.ny)
                ok |= 1u << r;
        }
        po = dst + (long long)(ty0 + row0) * L.nx + (long long)x4 * 4 + (long long)(cur.q - TL - 1) * (long long)plane;
    };
    if (cur.live) segment_setup();

    F4 ring[3][TL][R];
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int t = 0; t < TL; ++t)
#pragma unroll
            for (int r = 0; r < R; ++r) ring[a][t][r] = F4{0.f, 0.f, 0.f, 0.f};

    constexpr uint32_t kNbPar = (uint32_t)WARPS * 8u;
    constexpr uint32_t kParStride = (uint32_t)WARPS * 2u * kLanes * 16u;
    const uint32_t nb_self = sbase + Y::oNb + (uint32_t)wy * 8u;
    const uint32_t e_self = sbase + Y::oEdge + (uint32_t)(wy * 2 * kLanes + lane) * 16u;
    const uint32_t up_d = wy > 0 ? 1u : 0u, dn_d = wy < WARPS - 1 ? 1u : 0u;     // neighbour strips exist
    const uint32_t e_up = e_self - up_d * (kLanes * 16u);                        // bottom row of strip wy-1
    const uint32_t e_dn = e_self + dn_d * (2u * kLanes * 16u);                   // top row of strip wy+1

    // One plane job; PH = rotation phase of the register rings (compile time).
    auto step = [&](auto Pc) {
        constexpr int PH = decltype(Pc)::value;
        F4(&zm)[TL][R] = ring[PH % 3];
        F4(&cc)[TL][R] = ring[(PH + 1) % 3];
        F4(&nw)[TL][R] = ring[(PH + 2) % 3];

        const unsigned it = P.it;
        const unsigned s = it % NS, sp = (it + NS - 1) % NS;
        const uint32_t par = it & 1u;
        // neighbours finished step it-1: their edge rows are published and they no longer read what I overwrite
        if (it > 0) {
            const uint32_t pb = (par ^ 1u) * kNbPar, pp = ((it - 1) >> 1) & 1u;
            if (up_d) mbar_wait(nb_self - 8u + pb, pp);
            if (dn_d) mbar_wait(nb_self + 8u + pb, pp);
        }
        mbar_wait(sbase + Y::oFull + s * 8u, (it / NS) & 1u);
        const uint32_t st = sbase + s * Y::kStage, stp = sbase + sp * Y::kStage;

        // level-0 plane q (own rows) and the strip-edge rows of plane q-1
        F4 up0, dn0;
        if (!ymir) {
#pragma unroll
            for (int r = 0; r < R; ++r) nw[0][r] = ld4(st + own + (uint32_t)r * kRowBytes);
            up0 = ld4(stp + own - up_d * kRowBytes);
            dn0 = ld4(stp + own + (uint32_t)(R - 1) * kRowBytes + dn_d * kRowBytes);
        } else {
            const uint32_t xo = own - (uint32_t)row0 * kRowBytes;
#pragma unroll
            for (int r = 0; r < R; ++r) nw[0][r] = ld4(st + xo + mrow(row0 + r));
            up0 = ld4(stp + xo + mrow(row0 - (int)up_d));
            dn0 = ld4(stp + xo + mrow(row0 + R - 1 + (int)dn_d));
        }
        if (__any_sync(0xffffffffu, rev)) {
            if (rev) {
#pragma unroll
                for (int r = 0; r < R; ++r) nw[0][r] = reversed(nw[0][r]);
                up0 = reversed(up0);
                dn0 = reversed(dn0);
            }
        }
        F4 out[R];
#pragma unroll
        for (int t = 0; t < TL; ++t) {
            F4 up, dn;
            if (t == 0) {
                up = up0;
                dn = dn0;
            } else {
                const uint32_t lvl = (uint32_t)(t - 1) * Y::kEdgeLevel;
                const uint32_t wr = lvl + (par ^ 1u) * kParStride, rd = lvl + par * kParStride;
                sts128(e_self + wr, nw[t][0].x, nw[t][0].y, nw[t][0].z, nw[t][0].w);
                sts128(e_self + wr + kLanes * 16u, nw[t][R - 1].x, nw[t][R - 1].y, nw[t][R - 1].z, nw[t][R - 1].w);
                up = ld4(e_up + rd);
                dn = ld4(e_dn + rd);
            }
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const F4 &c = cc[t][r];
                const float left = __shfl_up_sync(0xffffffffu, c.w, 1);
                const float right = __shfl_down_sync(0xffffffffu, c.x, 1);
                const F4 &ym = (r == 0) ? up : cc[t][r - 1];
                const F4 &yp = (r == R - 1) ? dn : cc[t][r + 1];
                const F4 o = update4(c, left, right, ym, yp, zm[t][r], nw[t][r], kc);
                if (t + 1 < TL) nw[t + 1][r] = o;
                else out[r] = o;
            }
        }
        // out = level-TL plane q - TL
        po += plane;
        if (cur.q >= cur.qs) {
#pragma unroll
            for (int r = 0; r < R; ++r)
                if (ok & (1u << r)) stg128(po + (long long)r * L.nx, out[r].x, out[r].y, out[r].z, out[r].w);
        }
        // publish my edge rows, hand back the stage of plane q-1; the last warp to do so refills it
        __syncwarp();
        if (lane == 0) {
            mbar_arrive(nb_self + par * kNbPar);
            const uint32_t cnt = sbase + Y::oCnt + sp * 4u;
            if (atom_add_acq_rel(cnt, 1u) == (uint32_t)(WARPS - 1)) {
                sts32(cnt, 0u);
                issue_ahead<TL, NS, Y>(L, A, M, cur, NS - 1, it + NS - 1, sbase);
            }
        }
        P.it = it + 1;
        if (cursor_next<TL>(cur, L.nz) && cur.live) segment_setup();
    };

    while (cur.live) {
        step(std::integral_constant<int, 0>{});
        if (!cur.live) break;
        step(std::integral_constant<int, 1>{});
        if (!cur.live) break;
        step(std::integral_constant<int, 2>{});
    }
}

// Iterations cube b takes in this launch (0 = already finished).
__device__ __forceinline__ int now_of(const Launch &L, int b)
{
    const int remaining = cube_params(L, b).n_iter - L.iter_done;
    return remaining <= 0 ? 0 : (remaining < L.fuse ? remaining : L.fuse);
}

template <int T, int R, int WARPS, int NS, int MINB>
__global__ void __launch_bounds__(WARPS * 32, MINB)
idg_stream_kernel(const __grid_constant__ Launch L, const __grid_constant__ StreamArgs A,
                  const __grid_constant__ Maps M)
{
    using Y = Lay<T, R, WARPS, NS>;
    extern __shared__ __align__(1024) unsigned char smem[];
    const uint32_t sbase = smem_u32(smem);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            mbar_init(sbase + Y::oFull + s * 8u, 1);
            sts32(sbase + Y::oCnt + s * 4u, 0u);
        }
        for (int i = 0; i < 2 * WARPS; ++i) mbar_init(sbase + Y::oNb + i * 8u, 1);
        mbar_fence_init();
    }
    __syncthreads();

    // this CTA's share of the tile-planes
    const unsigned long long per_cta = A.planes / gridDim.x, extra = A.planes % gridDim.x;
    const unsigned long long c = blockIdx.x;
    unsigned long long g = c * per_cta + (c < extra ? c : extra);
    const unsigned long long g1 = g + per_cta + (c < extra ? 1 : 0);
    const unsigned long long per_cube = (unsigned long long)(A.tiles_x * A.tiles_y) * (unsigned)L.nz;

    Pipe P{0u};
    while (g < g1) {
        int b = (int)(g / per_cube);
        const int now = now_of(L, b);
        unsigned long long ge = (unsigned long long)(b + 1) * per_cube;
        while (ge < g1 && now_of(L, b + 1) == now) {       // extend the run over cubes taking the same TL
            ++b;
            ge += per_cube;
        }
        if (ge > g1) ge = g1;
        if (now == T) run<T, R, WARPS, NS, T>(L, A, M, g, ge, P, sbase);
        else if (T > 1 && now == 1) run<1, R, WARPS, NS, T>(L, A, M, g, ge, P, sbase);
        else if (T > 2 && now == 2) run<(T > 2 ? 2 : 1), R, WARPS, NS, T>(L, A, M, g, ge, P, sbase);
        else if (T > 3 && now == 3) run<(T > 3 ? 3 : 1), R, WARPS, NS, T>(L, A, M, g, ge, P, sbase);
        __syncthreads();          // drain: every stage is free again before the next run's prologue
        g = ge;
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

bool encode_map(CUtensorMap *m, const float *base, const Launch &L, int tile_y)
{
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    const cuuint64_t dims[4] = {(cuuint64_t)L.nx, (cuuint64_t)L.ny, (cuuint64_t)L.nz, (cuuint64_t)L.batch};
    const cuuint64_t strides[3] = {(cuuint64_t)L.nx * 4, (cuuint64_t)L.nx * L.ny * 4,
                                   (cuuint64_t)L.nx * L.ny * (cuuint64_t)L.nz * 4};
    const cuuint32_t box[4] = {(cuuint32_t)kTileX, (cuuint32_t)tile_y, 1, 1};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (void *)base, dims, strides, box, estr,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

int sm_count()
{
    static int n = 0;
    if (n == 0) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0)
            n = 148;
    }
    return n;
}

template <int T, int R, int WARPS, int NS, int MINB>
cudaError_t launch_cfg(const Launch &L, int nctas, cudaStream_t st)
{
    using Y = Lay<T, R, WARPS, NS>;
    constexpr int TILE_Y = WARPS * R;
    static_assert(TILE_Y > 2 * T, "tile must be taller than its halo");
    static_assert((size_t)Y::kBytes * MINB <= 227u * 1024u, "shared memory budget");
    StreamArgs A;
    A.halo = T;
    A.vy = TILE_Y - 2 * T;
    A.tiles_x = (L.nx / 4 + kValidLanes - 1) / kValidLanes;
    A.tiles_y = (L.ny + A.vy - 1) / A.vy;
    const unsigned long long tiles = (unsigned long long)A.tiles_x * A.tiles_y * (unsigned)L.batch;
    if (tiles > 0x7fffffffull) return cudaErrorInvalidValue;
    A.planes = tiles * (unsigned)L.nz;
    unsigned long long grid = nctas > 0 ? (unsigned long long)nctas : (unsigned long long)sm_count() * MINB;
    if (grid > A.planes) grid = A.planes;
    Maps M;
    if (!encode_map(&M.in, L.in, L, TILE_Y) || !encode_map(&M.out, L.out, L, TILE_Y) ||
        !encode_map(&M.scratch, L.scratch, L, TILE_Y))
        return cudaErrorNotSupported;
    auto kern = idg_stream_kernel<T, R, WARPS, NS, MINB>;
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Y::kBytes);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    kern<<<(unsigned)grid, WARPS * 32, Y::kBytes, st>>>(L, A, M);
    return cudaGetLastError();
}

}  // namespace

bool stream_supported(int nx, int ny, int nz, const void *in, const void *out, const void *scratch)
{
    (void)nz;
    if (nx % 4 != 0 || ny < 4) return false;
    const uintptr_t m = (uintptr_t)in | (uintptr_t)out | (uintptr_t)scratch;
    if ((m & 15u) != 0) return false;
    return encode_fn() != nullptr;
}

// tile: 0 auto | 1 = 128x64 tile, 512 threads, one CTA per SM | 2 = 128x32 tile, 256 threads, two CTAs per SM
cudaError_t launch_stream(const Launch &L, int nctas, int tile, cudaStream_t st)
{
    const bool small = (tile == 2);
    switch (L.fuse) {
    case 1: return small ? launch_cfg<1, 4, 8, 4, 2>(L, nctas, st) : launch_cfg<1, 4, 16, 4, 1>(L, nctas, st);
    case 2: return small ? launch_cfg<2, 4, 8, 4, 2>(L, nctas, st) : launch_cfg<2, 4, 16, 4, 1>(L, nctas, st);
    case 3: return launch_cfg<3, 4, 12, 4, 1>(L, nctas, st);
    case 4: return launch_cfg<4, 4, 8, 4, 1>(L, nctas, st);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace idg
