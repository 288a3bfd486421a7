// Persistent, warp-decoupled, TMA-fed, temporally fused IDG kernel (steps a1-a6 of SURVEY.md 8(a)).
//
// Decomposition.  The persistent grid is organised in teams of tiles_x CTAs; member ti of a team
// owns tile column ti.  The (cube, tile row, z) space of a launch is flattened into "row-planes"
// g = (b * tiles_y + tj) * nz + z and split evenly over the teams (one range per team, cut into
// segments at tile-row borders).  The members of a team walk the same range at the same pace, so
// the x-adjacent tiles of one plane are read together.  A CTA streams its segments plane by
// plane: a warp owns R rows x 128 columns of the 128 x (WARPS*R) tile, a thread a float4 column
// of that strip.
//
// Where the seven operands of Eq. 7 come from:
//   level 0 (the input of this launch)  -- the three planes q-2, q-1, q sit in a ring of NS
//            shared-memory stages filled by TMA (cp.async.bulk.tensor, box 128 x TILE_Y x 1 x 1);
//            centre, y and z neighbours are plain shared-memory loads, so level 0 costs no
//            registers between plane steps;
//   levels 1..TL-1 (intermediate iterates of the TL fused Jacobi steps) -- three-deep register
//            rings per level for z, neighbouring registers for y inside a strip, double-buffered
//            shared-memory slots for the strip-edge rows of neighbouring warps;
//   x neighbours at every level -- warp shuffles of the float4 end components.
//
// Pipeline.  There is no CTA-wide barrier in the plane loop:
//   * a stage is handed back through a shared counter; the last warp to release it issues the
//     next TMA load into it (any warp can be the producer, nobody waits for the slowest warp);
//   * the edge slots are guarded by one mbarrier per warp and step parity, so a warp only ever
//     waits for its two neighbours.
//
// Boundary (reading R1, zero flux by replication).  TMA zero-fills outside the cube.
// y: every strip reads its level-0 rows through a per-warp table of row offsets in which rows
// outside the cube are replaced by their even reflection; z: the TMA plane coordinate is
// reflected; x: the thread holding the first (last) float4 of a cube row replaces the shuffled
// left (right) neighbour by its own end component.  Eq. 7 is symmetric under the reflection, so
// the redundantly computed outside rows keep satisfying the replicate condition bit for bit at
// every fused level.
#include <type_traits>

#include "idg_kernels.cuh"
#include "idg_ptx.cuh"
#include "idg_update.cuh"

namespace idg {

namespace {

using namespace ptx;

constexpr int kLanes = 32;
constexpr int kStepLanes = 30;     // lanes an x tile advances by (lanes 0 and 31 are halo between tiles)
constexpr int kTileX = 128;
constexpr uint32_t kRowBytes = kTileX * 4;

__device__ __forceinline__ F4 ld4(uint32_t a)
{
    const float4 v = lds128(a);
    return F4{v.x, v.y, v.z, v.w};
}

struct StreamArgs {
    int tiles_x, tiles_y;         // xy tiles per cube
    int vy;                       // valid rows per tile = TILE_Y - 2*halo
    int halo;                     // = fuse (T) of the plan
    unsigned planes;              // row-planes of the launch = batch * tiles_y * nz
};

struct Maps {
    CUtensorMap m[3];             // in, out, scratch (batch as 4th dimension): the cubes a launch may read
};
enum { kMapIn = 0, kMapOut = 1, kMapScratch = 2 };

// What the thread that refills a stage needs to know about a segment (kept in shared memory, two
// slots indexed by segment parity; every warp writes the same values when it enters the segment).
struct SegInfo { int tx0, ty0, b, map; };

template <int T, int R, int WARPS, int NS>
struct Lay {
    static constexpr int TILE_Y = WARPS * R;
    static constexpr uint32_t kStage = (uint32_t)TILE_Y * kRowBytes;
    static constexpr uint32_t kEdgeLevel = 2u * WARPS * 2u * kLanes * 16u;      // both parities of one level
    static constexpr uint32_t kEdge = (uint32_t)(T > 1 ? T - 1 : 0) * kEdgeLevel;
    static constexpr uint32_t oEdge = NS * kStage;
    static constexpr uint32_t oRow = oEdge + kEdge;                             // WARPS x 8 row offsets
    static constexpr uint32_t oSeg = oRow + (uint32_t)WARPS * 32u;              // 4 SegInfo slots (16-byte aligned)
    static constexpr uint32_t oFull = oSeg + 4u * 16u;                          // NS mbarriers
    static constexpr uint32_t oNb = oFull + NS * 8u;                            // 2 * WARPS mbarriers
    static constexpr uint32_t oCnt = oNb + 2u * WARPS * 8u;                     // NS release counters
    static constexpr uint32_t kBytes = oCnt + NS * 4u;
};

// A position in the CTA's stream of plane jobs: level-0 plane q of tile row `tile` (global tile-row
// index b * tiles_y + tj over the batch; the tile column is fixed per CTA).  A segment produces
// output planes [z0, z1) of one tile from level-0 planes [z0-TL, z1-1+TL]; qs = z0+TL is the first
// job of the segment that stores a plane; `rem` row-planes of the run follow the segment.
struct Cursor {
    unsigned tile, rem;
    int q, q_last, qs;
};
__device__ __forceinline__ bool live(const Cursor &c) { return c.q <= c.q_last; }

template <int TL>
__device__ __forceinline__ void cursor_open(Cursor &c, unsigned tile, int z0, unsigned count, int nz)
{
    const unsigned room = (unsigned)(nz - z0);
    const unsigned take = count < room ? count : room;
    c.tile = tile;
    c.rem = count - take;
    c.q = z0 - TL;
    c.qs = z0 + TL;
    c.q_last = take ? z0 + (int)take - 1 + TL : c.q - 1;       // empty run: dead on arrival
}
// Advance by one plane job (walks into the next segment when the current one is exhausted).
template <int TL>
__device__ __forceinline__ void cursor_next(Cursor &c, int nz)
{
    if (c.q < c.q_last || c.rem == 0) ++c.q;
    else cursor_open<TL>(c, c.tile + 1, 0, c.rem, nz);
}

__device__ __forceinline__ SegInfo seg_info(const Launch &L, const StreamArgs &A, unsigned tile, float *&dst,
                                            CubeParams &prm)
{
    const unsigned b = tile / (unsigned)A.tiles_y;
    const int tj = (int)(tile - b * (unsigned)A.tiles_y), ti = (int)(blockIdx.x % (unsigned)A.tiles_x);
    prm = cube_params(L, (int)b);
    const float *src;
    route(L, (int)b, prm, src, dst);
    const size_t off = (size_t)b * (size_t)L.nx * (size_t)L.ny * (size_t)L.nz;
    const int map = (src == L.scratch + off) ? kMapScratch : (src == L.out + off) ? kMapOut : kMapIn;
    return SegInfo{ti * kStepLanes * 4, tj * A.vy - A.halo, (int)b, map};
}

// One thread: load the level-0 plane `ahead` jobs after cursor `c` into stage `s` (slow path: walks
// the cursor; used by the prologue and when the target lies in the next segment).
template <int TL, class Y>
__device__ __noinline__ void issue_ahead(const Launch &L, const StreamArgs &A, const Maps &M, Cursor c, int ahead,
                                         unsigned s, uint32_t sbase)
{
    for (int i = 0; i < ahead && live(c); ++i) cursor_next<TL>(c, L.nz);
    if (!live(c)) return;
    float *dst;
    CubeParams prm;
    const SegInfo si = seg_info(L, A, c.tile, dst, prm);
    const uint32_t bar = sbase + Y::oFull + s * 8u;
    mbar_expect_tx(bar, Y::kStage);
    tma_load_4d(sbase + s * Y::kStage, &M.m[si.map], bar, si.tx0, si.ty0, mirror(c.q, L.nz), si.b);
}

// Per-thread state of one segment.
struct Seg {
    uint32_t xo;        // byte offset of my (possibly x-mirrored) lane inside a stage row
    unsigned ok;        // bits 0..R-1: row r is stored; bit 28: first float4 of the cube row; bit 29: last
    float *po;          // where my row-0 float4 of the plane before the first output goes
    float ax, ay, az, sc, w;
};

// Entered by every warp at the start of a segment (rare): thread state, the warp's row-offset
// table (rows row0-1 .. row0+R, reflected at the cube faces) and the segment's SegInfo slot.
template <int TL, int R, int WARPS, class Y>
__device__ __noinline__ void segment_setup(const Launch &L, const StreamArgs &A, const Cursor &cur, unsigned seg,
                                           uint32_t sbase, Seg &S)
{
    constexpr int TILE_Y = WARPS * R;
    const int lane = threadIdx.x & 31, wy = threadIdx.x >> 5, row0 = wy * R;
    float *dst;
    CubeParams prm;
    const SegInfo si = seg_info(L, A, cur.tile, dst, prm);
    S.ax = prm.ax; S.ay = prm.ay; S.az = prm.az; S.sc = prm.s; S.w = prm.w;
    if (lane == 0) {
        const uint32_t a = sbase + Y::oSeg + (seg & 3u) * 16u;
        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(si.tx0), "r"(si.ty0), "r"(si.b),
                     "r"(si.map) : "memory");
    }
    if (lane < R + 2) {         // table entry `lane` <-> tile row row0 - 1 + lane
        int row = row0 - 1 + lane;
        row = row < 0 ? 0 : (row > TILE_Y - 1 ? TILE_Y - 1 : row);      // rows beyond the tile: unused halo
        int gy = si.ty0 + row;
        if (gy < 0) gy = -1 - gy;
        else if (gy >= L.ny) gy = 2 * L.ny - 1 - gy;
        int srow = gy - si.ty0;
        if (srow < 0 || srow >= TILE_Y) srow = row;
        sts32(sbase + Y::oRow + (uint32_t)(wy * 8 + lane) * 4u, (uint32_t)srow * kRowBytes);
    }
    // lane <-> float4 column x4; lanes 1..30 are valid everywhere, lane 0 / 31 only where they are the
    // first / last float4 of the cube row (their outer neighbour is then their own end component)
    const int nx4 = L.nx >> 2;
    const int x4 = (si.tx0 >> 2) + lane;
    unsigned ok = 0;
    if (x4 == 0) ok |= 1u << 28;
    if (x4 == nx4 - 1) ok |= 1u << 29;
    S.xo = (uint32_t)lane * 16u;
    const bool lane_ok = x4 < nx4 && ((lane >= 1 && lane <= kLanes - 2) || x4 == 0 || x4 == nx4 - 1);
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int row = row0 + r, gy = si.ty0 + row;
        if (lane_ok && row >= A.halo && row < TILE_Y - A.halo && gy < L.ny) ok |= 1u << r;
    }
    S.ok = ok;
    const size_t plane = (size_t)L.nx * (size_t)L.ny;
    S.po = dst + (long long)(si.ty0 + row0) * L.nx + (long long)x4 * 4 + (long long)(cur.q - TL - 1) * (long long)plane;
    __syncwarp();
}

// Pipeline position of the CTA (survives across runs of different TL).
struct Pipe {
    unsigned it;        // plane jobs consumed so far
    unsigned s;         // stage of job `it`   (= it % NS)
    unsigned fph;       // phase parity of that stage's full barrier (= (it / NS) & 1)
};

// One run: `count` consecutive row-planes starting at plane z0 of tile row `tile`, whose cubes all
// take TL iterations in this launch.
template <int TL, int R, int WARPS, int NS, int TMAX, bool PM>
__device__ __forceinline__ void run(const Launch &L, const StreamArgs &A, const Maps &M, unsigned tile, int z0,
                                    unsigned count, Pipe &P, uint32_t sbase)
{
    using Y = Lay<TMAX, R, WARPS, NS>;
    static_assert(R + 2 <= 8, "row-offset table holds 8 entries per warp");
    constexpr int TR = TL > 1 ? TL - 1 : 1;               // register-ring levels (levels 1..TL-1)
    const int lane = threadIdx.x & 31;
    const int wy = threadIdx.x >> 5;
    const size_t plane = (size_t)L.nx * (size_t)L.ny;

    Cursor cur;
    cursor_open<TL>(cur, tile, z0, count, L.nz);
    // prologue: jobs it .. it+NS-3 (their stages were released by everybody before the last drain)
    if (threadIdx.x == 0) {
        for (int i = 0; i < NS - 2; ++i) issue_ahead<TL, Y>(L, A, M, cur, i, (P.s + i) % NS, sbase);
    }

    Seg S = {};      // filled by segment_setup before the first plane job
    unsigned seg = 0;
    F4 ring[3][TR][R];
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int t = 0; t < TR; ++t)
#pragma unroll
            for (int r = 0; r < R; ++r) ring[a][t][r] = F4{0.f, 0.f, 0.f, 0.f};

    constexpr uint32_t kNbPar = (uint32_t)WARPS * 8u;
    constexpr uint32_t kParStride = (uint32_t)WARPS * 2u * kLanes * 16u;
    const uint32_t up_d = wy > 0 ? 1u : 0u, dn_d = wy < WARPS - 1 ? 1u : 0u;     // neighbour strips exist
    const uint32_t nb_self = sbase + Y::oNb + (uint32_t)wy * 8u;
    const uint32_t row_tab = sbase + Y::oRow + (uint32_t)wy * 32u;

    // One plane job; PH = rotation phase of the register rings (compile time).
    auto step = [&](auto Pc) {
        constexpr int PH = decltype(Pc)::value;
        F4(&zm)[TR][R] = ring[PH % 3];
        F4(&cc)[TR][R] = ring[(PH + 1) % 3];
        F4(&nw)[TR][R] = ring[(PH + 2) % 3];

        const unsigned it = P.it, s0 = P.s;
        const unsigned s1 = s0 ? s0 - 1 : NS - 1, s2 = s1 ? s1 - 1 : NS - 1;     // stages of planes q-1, q-2
        const uint32_t par = it & 1u;
        if (TL > 1 && it > 0) {
            // neighbours finished step it-1: their edge rows are published, mine of step it-2 were read
            const uint32_t pb = (par ^ 1u) * kNbPar, pp = ((it - 1) >> 1) & 1u;
            if (up_d) mbar_wait(nb_self - 8u + pb, pp);
            if (dn_d) mbar_wait(nb_self + 8u + pb, pp);
        }
        mbar_wait(sbase + Y::oFull + s0 * 8u, P.fph);

        // level 0: rows row0-1 .. row0+R of plane q-1, rows row0 .. row0+R-1 of planes q-2 and q
        uint32_t ro[8];
        {
            uint32_t a, b, c, d;
            asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(a), "=r"(b), "=r"(c), "=r"(d) : "r"(row_tab));
            ro[0] = a; ro[1] = b; ro[2] = c; ro[3] = d;
            asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(a), "=r"(b), "=r"(c), "=r"(d) : "r"(row_tab + 16u));
            ro[4] = a; ro[5] = b; ro[6] = c; ro[7] = d;
        }
        const uint32_t a0 = sbase + s0 * Y::kStage + S.xo, a1 = sbase + s1 * Y::kStage + S.xo,
                       a2 = sbase + s2 * Y::kStage + S.xo;
        const bool first = (S.ok >> 28) & 1u, last = (S.ok >> 29) & 1u;
        const Consts kc = make_consts(S.ax, S.ay, S.az, PM ? 0.25f * S.sc * S.sc : S.sc, S.w);
        const bool st_on = cur.q >= cur.qs;
        S.po += plane;

        F4 pm[R + 2];
#pragma unroll
        for (int i = 0; i < R + 2; ++i) pm[i] = ld4(a1 + ro[i]);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const F4 zmv = ld4(a2 + ro[r + 1]), nwv = ld4(a0 + ro[r + 1]);
            const F4 &c = pm[r + 1];
            float left = __shfl_up_sync(0xffffffffu, c.w, 1);
            float right = __shfl_down_sync(0xffffffffu, c.x, 1);
            left = first ? c.x : left;
            right = last ? c.w : right;
            const F4 o = update4<PM>(c, left, right, pm[r], pm[r + 2], zmv, nwv, kc);
            if (TL > 1) nw[0][r] = o;                       // level-1 plane q-1
            else if (st_on && (S.ok & (1u << r))) stg128(S.po + (long long)r * L.nx, o.x, o.y, o.z, o.w);
        }
        // all level-0 loads are done: hand back the stage of plane q-2; the last warp to do so refills it
        __syncwarp();
        if (lane == 0) {
            const uint32_t cnt = sbase + Y::oCnt + s2 * 4u;
            if (atom_add_relaxed(cnt, 1u) == (uint32_t)(WARPS - 1)) {
                sts32(cnt, 0u);
                const int iq = cur.q + (NS - 2);
                if (iq <= cur.q_last) {          // same segment: only the plane coordinate moves
                    int tx0, ty0, b, map;
                    asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];"
                                 : "=r"(tx0), "=r"(ty0), "=r"(b), "=r"(map)
                                 : "r"(sbase + Y::oSeg + (seg & 3u) * 16u));
                    const int z = ((unsigned)iq < (unsigned)L.nz) ? iq : mirror(iq, L.nz);
                    const uint32_t bar = sbase + Y::oFull + s2 * 8u;
                    mbar_expect_tx(bar, Y::kStage);
                    tma_load_4d(sbase + s2 * Y::kStage, &M.m[map], bar, tx0, ty0, z, b);
                } else {
                    issue_ahead<TL, Y>(L, A, M, cur, NS - 2, s2, sbase);
                }
            }
            if (TL == 1) mbar_arrive(nb_self + par * kNbPar);     // keeps the phases in step with `it`
        }
#pragma unroll
        for (int t = 1; t < TL; ++t) {                      // level t -> t+1 from ring level t-1
            const uint32_t e_self = sbase + Y::oEdge + (uint32_t)(t - 1) * Y::kEdgeLevel +
                                    (uint32_t)(wy * 2 * kLanes + lane) * 16u;
            const uint32_t wr = e_self + (par ^ 1u) * kParStride, rd = e_self + par * kParStride;
            const F4 &e0 = nw[t - 1][0], &e1 = nw[t - 1][R - 1];
            sts128(wr, e0.x, e0.y, e0.z, e0.w);
            sts128(wr + kLanes * 16u, e1.x, e1.y, e1.z, e1.w);
            const F4 up = ld4(rd - up_d * (kLanes * 16u));               // bottom row of strip wy-1
            const F4 dn = ld4(rd + dn_d * (2u * kLanes * 16u));          // top row of strip wy+1
            if (t == TL - 1) {      // last exchange of the step: my edge rows are published, the neighbours' read
                __syncwarp();
                if (lane == 0) mbar_arrive(nb_self + par * kNbPar);
            }
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const F4 &c = cc[t - 1][r];
                float left = __shfl_up_sync(0xffffffffu, c.w, 1);
                float right = __shfl_down_sync(0xffffffffu, c.x, 1);
                left = first ? c.x : left;
                right = last ? c.w : right;
                const F4 &ym = (r == 0) ? up : cc[t - 1][r - 1];
                const F4 &yp = (r == R - 1) ? dn : cc[t - 1][r + 1];
                const F4 o = update4<PM>(c, left, right, ym, yp, zm[t - 1][r], nw[t - 1][r], kc);
                if (t + 1 < TL) nw[t][r] = o;
                else if (st_on && (S.ok & (1u << r))) stg128(S.po + (long long)r * L.nx, o.x, o.y, o.z, o.w);
            }
        }
        P.it = it + 1;
        if (s0 == NS - 1) { P.s = 0; P.fph ^= 1u; }
        else P.s = s0 + 1;
    };

    while (live(cur)) {
        segment_setup<TL, R, WARPS, Y>(L, A, cur, seg, sbase, S);
        int jobs = cur.q_last - cur.q + 1;
        while (true) {
            step(std::integral_constant<int, 0>{});
            ++cur.q;
            if (--jobs == 0) break;
            step(std::integral_constant<int, 1>{});
            ++cur.q;
            if (--jobs == 0) break;
            step(std::integral_constant<int, 2>{});
            ++cur.q;
            if (--jobs == 0) break;
        }
        // cur.q == q_last + 1: open the next segment of the run, if any
        if (cur.rem == 0) break;
        cursor_open<TL>(cur, cur.tile + 1, 0, cur.rem, L.nz);
        ++seg;
    }
}

// Iterations cube b takes in this launch (0 = already finished).
__device__ __forceinline__ int now_of(const Launch &L, int b)
{
    const int remaining = cube_params(L, b).n_iter - L.iter_done;
    return remaining <= 0 ? 0 : (remaining < L.fuse ? remaining : L.fuse);
}

template <int T, int R, int WARPS, int NS, int MINB, bool PM>
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

    // this team's share of the row-planes
    const unsigned teams = gridDim.x / (unsigned)A.tiles_x;
    const unsigned per_team = A.planes / teams, extra = A.planes % teams;
    const unsigned c = blockIdx.x / (unsigned)A.tiles_x;
    unsigned g = c * per_team + (c < extra ? c : extra);
    const unsigned g1 = g + per_team + (c < extra ? 1u : 0u);
    const unsigned per_cube = (unsigned)A.tiles_y * (unsigned)L.nz;

    Pipe P{0u, 0u, 0u};
    while (g < g1) {
        int b = (int)(g / per_cube);
        const int now = now_of(L, b);
        unsigned ge = (unsigned)(b + 1) * per_cube;
        while (ge < g1 && now_of(L, b + 1) == now) {       // extend the run over cubes taking the same TL
            ++b;
            ge += per_cube;
        }
        if (ge > g1) ge = g1;
        const unsigned tile = g / (unsigned)L.nz;
        const int z0 = (int)(g - tile * (unsigned)L.nz);
        if (now == T) run<T, R, WARPS, NS, T, PM>(L, A, M, tile, z0, ge - g, P, sbase);
        else if (T > 1 && now == 1) run<1, R, WARPS, NS, T, PM>(L, A, M, tile, z0, ge - g, P, sbase);
        else if (T > 2 && now == 2) run<(T > 2 ? 2 : 1), R, WARPS, NS, T, PM>(L, A, M, tile, z0, ge - g, P, sbase);
        else if (T > 3 && now == 3) run<(T > 3 ? 3 : 1), R, WARPS, NS, T, PM>(L, A, M, tile, z0, ge - g, P, sbase);
        __syncthreads();          // drain: every stage is free again before the next run's prologue
        g = ge;
    }
}

bool encode_map(CUtensorMap *m, const float *base, const Launch &L, int tile_y)
{
    return tmap_encode(m, base, L.nx, L.ny, L.nz, L.batch, kTileX, tile_y);
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

template <int T, int R, int WARPS, int NS, int MINB, bool PM = false>
cudaError_t launch_cfg(const Launch &L, int nctas, cudaStream_t st)
{
    using Y = Lay<T, R, WARPS, NS>;
    constexpr int TILE_Y = WARPS * R;
    static_assert(TILE_Y > 2 * T, "tile must be taller than its halo");
    static_assert(NS >= 4, "three planes in use plus at least one in flight");
    static_assert((size_t)Y::kBytes * MINB <= 227u * 1024u, "shared memory budget");
    StreamArgs A;
    A.halo = T;
    A.vy = TILE_Y - 2 * T;
    const int nx4 = L.nx / 4;
    A.tiles_x = nx4 <= 2 ? 1 : (nx4 - 2 + kStepLanes - 1) / kStepLanes;
    A.tiles_y = (L.ny + A.vy - 1) / A.vy;
    const unsigned long long rows = (unsigned long long)A.tiles_y * (unsigned)L.batch;
    if (rows * (unsigned)L.nz > 0x7fffffffull || A.tiles_x > 0x3fffff) return cudaErrorInvalidValue;
    A.planes = (unsigned)(rows * (unsigned)L.nz);
    // teams of tiles_x CTAs; as many teams as fit the resident slots (at least one)
    const unsigned long long slots = nctas > 0 ? (unsigned long long)nctas : (unsigned long long)sm_count() * MINB;
    unsigned long long teams = slots / (unsigned)A.tiles_x;
    if (teams < 1) teams = 1;
    if (teams > A.planes) teams = A.planes;
    const unsigned long long grid = teams * (unsigned)A.tiles_x;
    Maps M;
    if (!encode_map(&M.m[kMapIn], L.in, L, TILE_Y) || !encode_map(&M.m[kMapOut], L.out, L, TILE_Y) ||
        !encode_map(&M.m[kMapScratch], L.scratch, L, TILE_Y))
        return cudaErrorNotSupported;
    auto kern = idg_stream_kernel<T, R, WARPS, NS, MINB, PM>;
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
    return tmap_available();
}

// tile: 0 auto | 1 = 128x64 tile, 512 threads, one CTA per SM | 2 = 128x32 tile, 256 threads, two CTAs per SM
//       | 3 = 128x40 tile, 320 threads, two CTAs per SM | 4 = 128x80 tile, 640 threads, one CTA per SM
cudaError_t launch_stream(const Launch &L, int nctas, int tile, cudaStream_t st)
{
    if (L.mode == 1) {          // gradient-driven variant: the two standard tilings, T <= 2
        switch (L.fuse * 10 + tile) {
        case 10: case 11: return launch_cfg<1, 4, 16, 5, 1, true>(L, nctas, st);
        case 12: return launch_cfg<1, 4, 8, 5, 2, true>(L, nctas, st);
        case 20: case 21: return launch_cfg<2, 4, 16, 5, 1, true>(L, nctas, st);
        case 22: return launch_cfg<2, 4, 8, 5, 2, true>(L, nctas, st);
        default: return cudaErrorInvalidValue;
        }
    }
    switch (L.fuse * 10 + tile) {
    case 10: case 11: return launch_cfg<1, 4, 16, 5, 1>(L, nctas, st);
    case 12: return launch_cfg<1, 4, 8, 5, 2>(L, nctas, st);
    case 13: return launch_cfg<1, 4, 20, 5, 1>(L, nctas, st);
    case 14: return launch_cfg<1, 4, 10, 5, 2>(L, nctas, st);
    case 20: case 21: return launch_cfg<2, 4, 16, 5, 1>(L, nctas, st);
    case 22: return launch_cfg<2, 4, 8, 5, 2>(L, nctas, st);
    case 23: return launch_cfg<2, 3, 20, 5, 1>(L, nctas, st);
    case 24: return launch_cfg<2, 3, 16, 5, 1>(L, nctas, st);
    case 30: case 31: return launch_cfg<3, 4, 16, 5, 1>(L, nctas, st);
    case 32: return launch_cfg<3, 4, 8, 5, 2>(L, nctas, st);
    case 33: return launch_cfg<3, 4, 12, 5, 1>(L, nctas, st);
    case 34: return launch_cfg<3, 3, 16, 5, 1>(L, nctas, st);
    case 40: case 41: return launch_cfg<4, 4, 12, 5, 1>(L, nctas, st);
    case 42: return launch_cfg<4, 4, 8, 5, 1>(L, nctas, st);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace idg
