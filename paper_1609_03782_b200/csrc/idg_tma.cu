// TMA-pipelined, temporally fused IDG kernel (the fast path; steps a1-a6 of DESIGN.md section 7).
//
// Same decomposition as idg_tiled.cu -- a CTA owns a 128 x (WARPS*R) xy tile and streams along
// z; a thread owns a float4 column of an R-row strip; x neighbours by warp shuffle, y
// neighbours in registers with strip edges through shared memory, z neighbours in registers --
// but level-0 planes are brought in by the Tensor Memory Accelerator: one elected thread issues
// cp.async.bulk.tensor (3-D/4-D box 128 x TILE_Y x 1) into a ring of NS shared-memory stages,
// NS-2 planes ahead of the plane being consumed, completion signalled on mbarriers.  The
// per-level z rings are rotated by unrolling the plane loop three times (register renaming
// instead of moves).
//
// Boundary (reading R1): TMA zero-fills outside the cube, so each thread whose cell lies just
// outside a cube face reads the even-reflected cell instead (and writes it back to its own
// cell for its neighbours); z reflection is done by the TMA plane coordinate.  The update is
// symmetric under the reflection, so all fused levels satisfy the zero-flux replicate condition
// bit for bit without any predicate in the arithmetic (see idg_tiled.cu).
#include <cuda.h>

#include <type_traits>

#include "idg_kernels.cuh"
#include "idg_ptx.cuh"
#include "idg_update.cuh"

namespace idg {

namespace {

constexpr int kLanes = 32;
constexpr int kValidLanes = 30;
constexpr int kTileX = 128;

// pointer-taking wrappers over the address-taking helpers of idg_ptx.cuh
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) { ptx::mbar_init(ptx::smem_u32(bar), count); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) { ptx::mbar_expect_tx(ptx::smem_u32(bar), bytes); }
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) { ptx::mbar_wait_spin(ptx::smem_u32(bar), parity); }
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *map, uint64_t *bar, int x, int y, int z, int b)
{
    ptx::tma_load_4d(ptx::smem_u32(dst), map, ptx::smem_u32(bar), x, y, z, b);
}

struct TmaArgs {
    int tiles_x, tiles_y;
    int zchunk;
    int halo;
    int rounds;            // cooperative launch: launches folded into this one (else 1)
    unsigned *bar;         // cooperative launch: arrival counter of the grid barrier (zeroed by the host)
};

struct Maps {
    CUtensorMap in, out, scratch;      // the three cubes (batch as 4th dimension) a launch may read
};

// CL: two CTAs of a cluster share a tile of 2 TILE_Y rows (see tma_body): a stage holds one more row above and below
// the CTA's rows, and the strip-edge buffer one more slot pair for the rows the partner sends.
template <int T, int R, int WARPS, int NS, bool CL = false>
struct Smem {
    static constexpr int TILE_Y = WARPS * R;
    static constexpr int kRows = TILE_Y + (CL ? 2 : 0);
    static constexpr int kSlots = WARPS + (CL ? 1 : 0);
    static constexpr int kStageFloats = kRows * kTileX;
    static constexpr size_t kStageBytes = (size_t)kStageFloats * sizeof(float);
    static constexpr size_t kEdgeBytes = (size_t)(T > 1 ? T - 1 : 0) * 2 * kSlots * 2 * kLanes * sizeof(float4);
    static constexpr size_t kBarOff = NS * kStageBytes + kEdgeBytes;
    static constexpr int kXBars = CL ? 2 : 0;           // CL: one per plane parity for the partner's rows of all levels
    static constexpr size_t kBytes = kBarOff + (NS + kXBars) * sizeof(uint64_t);
};

// ONE: the cube has at most 128 columns, so a single tile column covers a row with all 32 lanes valid and no halo
// lanes; the x faces are replicated by patching the shuffled neighbour of the first / last float4 of the row.
// UNAL: nx % 4 != 0 -- the buffers are pitched copies (row pitch L.pitch), the x face at nx - 1 lies INSIDE a float4:
// cells beyond it take the even reflection element by element (cell x <- cell 2 nx - 1 - x) from the level-0 stage.
// CL: the CTA is one of a cluster pair stacked along y.  The pair covers 2 TILE_Y rows with the T halo rows at its two
// OUTER edges only (useful rows 2 TILE_Y - 2 T of 2 TILE_Y, against TILE_Y - 2 T of TILE_Y alone); across the seam the
// two CTAs exchange the strip-edge rows of every fused level through distributed shared memory: the warp at the seam
// sends its row with st.async into the partner's edge buffer, completion counted on an mbarrier of the partner, and
// waits on its own mbarrier for the partner's row -- no cluster-wide barrier in the plane loop (a release at cluster
// scope would also wait for the global stores of the plane).  A CTA reads the partner's row of the previous plane
// BEFORE it sends its own of this plane, so the partner, which needs that row to go on, cannot overwrite a slot that
// is still to be read; the two CTAs stay within one plane of each other.
template <int TL, int R, int WARPS, int NS, int TMAX, bool ONE, bool PM = false, bool UNAL = false, bool CL = false>
__device__ __forceinline__ void tma_body(const CUtensorMap *map, float *__restrict__ dst, const Launch &L,
                                         const TmaArgs &A, const CubeParams &prm, int b,
                                         unsigned char *smem, bool reinit = false)
{
    using S = Smem<TMAX, R, WARPS, NS, CL>;
    constexpr int TILE_Y = WARPS * R;
    constexpr int RB = CL ? 1 : 0;                       // stage row of the CTA's row 0
    float *stage0 = reinterpret_cast<float *>(smem);
    float4 *edge = reinterpret_cast<float4 *>(smem + NS * S::kStageBytes);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + S::kBarOff);

    const int lane = threadIdx.x & 31;
    const int wy = threadIdx.x >> 5;
    const int nx4 = UNAL ? (L.nx + 3) >> 2 : L.nx >> 2;       // float4 columns that hold cube voxels
    const int ld = UNAL ? L.pitch : L.nx;                      // row pitch of the buffers
    const int rank = CL ? (int)(blockIdx.x & 1u) : 0;     // position in the cluster pair (0: upper rows)
    const int tile = CL ? (int)(blockIdx.x >> 1) : (int)blockIdx.x;
    const int vy = (CL ? 2 : 1) * TILE_Y - 2 * A.halo;
    const int ti = tile % A.tiles_x, tj = tile / A.tiles_x;
    const int tx0 = ONE ? 0 : (ti * kValidLanes - 1) * 4;   // cube x of tile column 0
    const int ty0 = tj * vy - A.halo + rank * TILE_Y;    // cube y of the CTA's row 0
    const int x4 = ONE ? lane : ti * kValidLanes - 1 + lane;
    const bool x_first = ONE && lane == 0, x_last = ONE && lane == nx4 - 1;
    const int row0 = wy * R;
    const int z0 = blockIdx.y * A.zchunk;
    const int z1 = min(z0 + A.zchunk, L.nz);
    const int q_first = z0 - TL, q_last = z1 - 1 + TL;

    // own cells, reflected source cells for positions just outside a cube face, store mask
    int cell[R], scell[R];
    unsigned ok = 0, fix = 0;
    bool rev = false;
    int slane = lane;
    // UNAL: tile column of the first cell beyond the x face, and the sum of a cell's and its mirror image's columns
    const int xw = UNAL ? L.nx - tx0 : 0, xc = 2 * xw - 1;
    const bool xfix = UNAL && lane * 4 + 3 >= xw;              // some component of my float4 lies beyond the face
    if (!ONE) {
        if (x4 < 0) { slane = lane + (-1 - x4) - x4; rev = true; }             // x4' = -1 - x4
        else if (!UNAL && x4 >= nx4) { slane = lane + (2 * nx4 - 1 - x4) - x4; rev = true; }
        if (slane < 0 || slane >= kLanes) { slane = lane; rev = false; }        // beyond one reflection: unused cell
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int row = row0 + r, gy = ty0 + row;
        cell[r] = (row + RB) * kTileX + lane * 4;
        int srow = row;
        if (gy < 0) srow = (-1 - gy) - ty0;
        else if (gy >= L.ny) srow = (2 * L.ny - 1 - gy) - ty0;
        if (srow < -RB || srow >= TILE_Y + RB) srow = row;
        scell[r] = (srow + RB) * kTileX + slane * 4;
        if (scell[r] != cell[r] || xfix) fix |= 1u << r;
        if ((ONE || (lane >= 1 && lane <= kValidLanes)) && x4 < nx4 && (row >= A.halo || (CL && rank == 1)) &&
            (row < TILE_Y - A.halo || (CL && rank == 0)) && gy < L.ny)
            ok |= 1u << r;
    }
    // level-0 strip-edge rows (plane q-1 of the stage).  CL: the stage has the rows -1 and TILE_Y too; a neighbour row
    // beyond the cube's last row is its mirror image, the strip's own last row (the seam may lie on the face)
    int up_row = CL ? row0 - 1 : max(row0 - 1, 0), dn_row = CL ? row0 + R : min(row0 + R, TILE_Y - 1);
    if (CL && ty0 + dn_row >= L.ny && ty0 + dn_row - 1 >= 0) dn_row = min(max(2 * L.ny - 1 - (ty0 + dn_row) - ty0, -1), TILE_Y);
    if (CL && ty0 + up_row < 0) up_row = min(max(-1 - (ty0 + up_row) - ty0, -1), TILE_Y);
    // (CL: rows -1 and TILE_Y of a stage have no owner that would write the x-reflected cells back: read the source lane)
    const int up_cell = (up_row + RB) * kTileX + (CL ? slane : lane) * 4;
    const int dn_cell = (dn_row + RB) * kTileX + (CL ? slane : lane) * 4;
    // slots of the strip-edge buffer my up / down neighbour rows come from; CL: slot WARPS holds what the partner sent
    const int wy_up = (CL && rank == 1 && wy == 0) ? WARPS : max(wy - 1, 0);
    const int wy_dn = (CL && rank == 0 && wy == WARPS - 1) ? WARPS : min(wy + 1, WARPS - 1);
    // CL: the warp at the seam also writes its seam row into the partner's slot WARPS (the row the partner lacks)
    const bool seam = CL && ((rank == 0 && wy == WARPS - 1) || (rank == 1 && wy == 0));
    uint32_t peer_edge = 0, peer_xbar = 0;
    const uint32_t xbar = ptx::smem_u32(smem + S::kBarOff + NS * sizeof(uint64_t));
    if (CL) {
        const uint32_t mine = ptx::smem_u32(smem + NS * S::kStageBytes);
        asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(peer_edge) : "r"(mine), "r"(rank ^ 1));
        asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(peer_xbar) : "r"(xbar), "r"(rank ^ 1));
    }
    const uint32_t send_base = peer_edge + (uint32_t)((WARPS * 2 + (rank == 0 ? 1 : 0)) * kLanes + lane) * 16u;

    const size_t plane = (size_t)ld * (size_t)L.ny;
    float *po = dst + (long long)(ty0 + row0) * ld + (long long)x4 * 4 + (long long)(q_first - TL - 1) * (long long)plane;

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            if (reinit) ptx::mbar_inval(ptx::smem_u32(&full[s]));      // a later round of a cooperative launch
            mbar_init(&full[s], 1);
        }
        if (CL) {
#pragma unroll
            for (int i = 0; i < S::kXBars; ++i) ptx::mbar_init(xbar + 8 * i, 1);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (CL) {                   // the partner runs: its shared memory may be written from here on
        ptx::cluster_arrive();
        ptx::cluster_wait();
    } else {
        __syncthreads();
    }
    auto issue = [&](int q) {       // thread 0: plane q -> stage (q - q_first) % NS
        const int s = (q - q_first) % NS;
        mbar_expect_tx(&full[s], (uint32_t)S::kStageBytes);
        tma_load_4d(stage0 + (size_t)s * S::kStageFloats, map, &full[s], tx0, ty0 - RB, mirror(q, L.nz), b);
    };
    if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < NS - 2; ++i)
            if (q_first + i <= q_last) issue(q_first + i);
    }

    const Consts kc = make_consts<PM>(prm);
    F4 ring[3][TL][R];
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int t = 0; t < TL; ++t)
#pragma unroll
            for (int r = 0; r < R; ++r) ring[a][t][r] = F4{0.f, 0.f, 0.f, 0.f};

    int q = q_first;
    int par = 0;

    // One plane step; P = rotation phase of the register rings (compile time).
    auto step = [&](auto Pc) {
        constexpr int P = decltype(Pc)::value;
        F4(&zm)[TL][R] = ring[P % 3];
        F4(&cc)[TL][R] = ring[(P + 1) % 3];
        F4(&nw)[TL][R] = ring[(P + 2) % 3];

        const unsigned it = (unsigned)(q - q_first);
        const unsigned s = it % NS;
        if (threadIdx.x == 0 && q + NS - 2 <= q_last) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            issue(q + NS - 2);                              // its stage held plane q-2: free since last barrier
        }
        // CL: the partner's seam rows of the previous plane (every level) are normally in by now: ask early, so that
        // the answer is there when level 1 needs the rows
        bool xready = true;
        if (CL && TL > 1 && seam && it > 0) {
            const uint32_t mb = xbar + 8u * (uint32_t)par;
            if (lane == 0) ptx::mbar_expect_tx(mb, (uint32_t)(TL - 1) * kLanes * 16u);
            xready = ptx::mbar_test(mb, ((it - 1u) >> 1) & 1u);
        }
        const float *st = stage0 + (size_t)s * S::kStageFloats;                      // plane q
        const float *stp = stage0 + (size_t)((it + NS - 1) % NS) * S::kStageFloats;  // plane q-1
        mbar_wait(&full[s], (uint32_t)((it / NS) & 1));

        // level-0 plane q: own cells (reflected source just outside a cube face)
#pragma unroll
        for (int r = 0; r < R; ++r) nw[0][r] = lds4(st + scell[r]);
        if (fix) {
#pragma unroll
            for (int r = 0; r < R; ++r)
                if (fix & (1u << r)) {
                    if (rev) nw[0][r] = F4{nw[0][r].w, nw[0][r].z, nw[0][r].y, nw[0][r].x};
                    if (UNAL && xfix) {      // beyond the x face: the mirror image, component by component
                        const float *row = st + (scell[r] - slane * 4);
                        const int c0 = lane * 4;
                        if (c0 >= xw) nw[0][r].x = row[min(max(xc - c0, 0), kTileX - 1)];
                        if (c0 + 1 >= xw) nw[0][r].y = row[min(max(xc - c0 - 1, 0), kTileX - 1)];
                        if (c0 + 2 >= xw) nw[0][r].z = row[min(max(xc - c0 - 2, 0), kTileX - 1)];
                        if (c0 + 3 >= xw) nw[0][r].w = row[min(max(xc - c0 - 3, 0), kTileX - 1)];
                    }
                    sts4(const_cast<float *>(st) + cell[r], nw[0][r]);
                }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // the stage is refilled by TMA later on
        }
        F4 out[R];
#pragma unroll
        for (int t = 0; t < TL; ++t) {
            F4 up, dn;
            if (t == 0) {
                up = lds4(stp + up_cell);
                dn = lds4(stp + dn_cell);
                if (CL && rev) {
                    up = F4{up.w, up.z, up.y, up.x};
                    dn = F4{dn.w, dn.z, dn.y, dn.x};
                }
            } else {
                float4 *e_rd = edge + (((t - 1) * 2 + par) * S::kSlots) * 2 * kLanes;
                float4 *e_wr = edge + (((t - 1) * 2 + (par ^ 1)) * S::kSlots) * 2 * kLanes;
                e_wr[(wy * 2 + 0) * kLanes + lane] = make_float4(nw[t][0].x, nw[t][0].y, nw[t][0].z, nw[t][0].w);
                e_wr[(wy * 2 + 1) * kLanes + lane] =
                    make_float4(nw[t][R - 1].x, nw[t][R - 1].y, nw[t][R - 1].z, nw[t][R - 1].w);
                if (CL && t == 1 && !xready) ptx::mbar_wait_spin(xbar + 8u * (uint32_t)par, ((it - 1u) >> 1) & 1u);
                const float4 u = e_rd[(wy_up * 2 + 1) * kLanes + lane];
                const float4 d = e_rd[(wy_dn * 2 + 0) * kLanes + lane];
                up = F4{u.x, u.y, u.z, u.w};
                dn = F4{d.x, d.y, d.z, d.w};
                if (CL && seam) {               // only now my seam row of this plane -> the partner's slot WARPS
                    // (the loaded neighbour row is an operand: the send cannot be scheduled ahead of that load)
                    const F4 &v = rank == 0 ? nw[t][R - 1] : nw[t][0];
                    const uint32_t a = send_base + (uint32_t)((t - 1) * 2 + (par ^ 1)) * (uint32_t)(S::kSlots * 2 * kLanes * 16);
                    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.f32 [%0], {%1, %2, %3, %4}, [%5];"
                                 ::"r"(a), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "r"(peer_xbar + 8u * (uint32_t)(par ^ 1)),
                                   "f"(rank == 0 ? d.x : u.x));
                }
            }
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const F4 &c = cc[t][r];
                float left = __shfl_up_sync(0xffffffffu, c.w, 1);
                float right = __shfl_down_sync(0xffffffffu, c.x, 1);
                if (ONE) {
                    left = x_first ? c.x : left;                  // zero-flux faces (reading R1)
                    right = x_last ? c.w : right;
                }
                const F4 &ym = (r == 0) ? up : cc[t][r - 1];
                const F4 &yp = (r == R - 1) ? dn : cc[t][r + 1];
                const F4 o = update4<PM>(c, left, right, ym, yp, zm[t][r], nw[t][r], kc);
                if (t + 1 < TL) nw[t + 1][r] = o;
                else out[r] = o;
            }
        }
        // out = level-TL plane (q - TL)
        po += plane;
        const int zo = q - TL;
        if (zo >= z0 && zo < z1) {
#pragma unroll
            for (int r = 0; r < R; ++r)
                if (ok & (1u << r))
                    *reinterpret_cast<float4 *>(po + (long long)r * ld) =
                        make_float4(out[r].x, out[r].y, out[r].z, out[r].w);
        }
        par ^= 1;
        ++q;
        __syncthreads();
    };

    while (true) {
        step(std::integral_constant<int, 0>{});
        if (q > q_last) break;
        step(std::integral_constant<int, 1>{});
        if (q > q_last) break;
        step(std::integral_constant<int, 2>{});
        if (q > q_last) break;
    }
    if (CL) {                           // neither CTA leaves while the other may still send into its shared memory
        ptx::cluster_arrive();
        ptx::cluster_wait();
    }
}

template <int T, int R, int WARPS, int NS, int MINB, bool ONE, bool PM = false, bool UNAL = false, bool CL = false>
__global__ void __launch_bounds__(WARPS * 32, MINB)
idg_tma_kernel(const __grid_constant__ Launch L, const __grid_constant__ TmaArgs A,
               const __grid_constant__ Maps M)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    const int b = blockIdx.z;
    const CubeParams prm = cube_params(L, b);
    const float *src;
    float *dst;
    const int now = route(L, b, prm, src, dst);
    if (now == 0) return;               // (both CTAs of a cluster pair: same cube)
    const size_t off = (size_t)b * cube_stride(L);
    const CUtensorMap *map = (src == L.scratch + off) ? &M.scratch : (src == L.out + off) ? &M.out : &M.in;
    if (now == T) tma_body<T, R, WARPS, NS, T, ONE, PM, UNAL, CL>(map, dst, L, A, prm, b, smem);
    else if (T > 1 && now == 1) tma_body<1, R, WARPS, NS, T, ONE, PM, UNAL, CL>(map, dst, L, A, prm, b, smem);
    else if (T > 2 && now == 2) tma_body<(T > 2 ? 2 : 1), R, WARPS, NS, T, ONE, PM, UNAL, CL>(map, dst, L, A, prm, b, smem);
    else if (T > 3 && now == 3) tma_body<(T > 3 ? 3 : 1), R, WARPS, NS, T, ONE, PM, UNAL, CL>(map, dst, L, A, prm, b, smem);
}

// Cooperative variant: all `A.rounds` launches of a plan in one, a grid barrier between rounds (the whole grid is
// co-resident); for small, L2-resident cubes, whose launches are bound by launch latency and the prologue.
template <int T, int R, int WARPS, int NS, int MINB, bool ONE>
__global__ void __launch_bounds__(WARPS * 32, MINB)
idg_tma_coop_kernel(const __grid_constant__ Launch L, const __grid_constant__ TmaArgs A,
               const __grid_constant__ Maps M)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    const int b = blockIdx.z;
    const CubeParams prm = cube_params(L, b);
    const size_t off = (size_t)b * cube_stride(L);
    constexpr bool COOP = true;
    const int rounds = A.rounds;
    const unsigned ctas = gridDim.x * gridDim.y * gridDim.z;
    for (int round = 0; round < rounds; ++round) {
        const float *src;
        float *dst;
        const int now = route(L, L.iter_done + round * L.fuse, b, prm, src, dst);
        if (now > 0) {
            const CUtensorMap *map = (src == L.scratch + off) ? &M.scratch : (src == L.out + off) ? &M.out : &M.in;
            const bool re = COOP && round > 0;
            if (now == T) tma_body<T, R, WARPS, NS, T, ONE>(map, dst, L, A, prm, b, smem, re);
            else if (T > 1 && now == 1) tma_body<1, R, WARPS, NS, T, ONE>(map, dst, L, A, prm, b, smem, re);
            else if (T > 2 && now == 2) tma_body<(T > 2 ? 2 : 1), R, WARPS, NS, T, ONE>(map, dst, L, A, prm, b, smem, re);
            else if (T > 3 && now == 3) tma_body<(T > 3 ? 3 : 1), R, WARPS, NS, T, ONE>(map, dst, L, A, prm, b, smem, re);
        } else if (!COOP) {
            return;
        }
        if (COOP && round + 1 < rounds) ptx::grid_barrier(A.bar, ctas * (unsigned)(round + 1));
    }
}

bool encode_map(CUtensorMap *m, const float *base, const Launch &L, int tile_y)
{
    return tmap_encode(m, base, L.nx, L.ny, L.nz, L.batch, kTileX, tile_y, 1, L.pitch);
}

// max_ctas > 0: only chunkings whose whole grid is at most max_ctas CTAs (cooperative launch); 0 if none is.
int pick_zchunk(int nz, long tiles, int T, int slots, long max_ctas = 0)
{
    long best_cost = -1;
    int best = max_ctas > 0 ? 0 : nz;
    for (int nchunks = 1; nchunks <= nz; ++nchunks) {
        const int zc = (nz + nchunks - 1) / nchunks;
        const long ctas = tiles * ((nz + zc - 1) / zc);
        if (max_ctas > 0 && ctas > max_ctas) break;
        const long waves = (ctas + slots - 1) / slots;
        const long cost = waves * (zc + 2 * T + 3);      // +3: prologue and pipeline fill, in plane-steps
        if (best_cost < 0 || cost < best_cost) {
            best_cost = cost;
            best = zc;
        }
        if (zc == 1) break;
    }
    return best;
}

// The cluster-pair tiling is valid unless the cube's last row lies within a few rows of a seam between the two CTAs of a
// pair: rows beyond a face take their mirror images from the CTA's own stage, and those would be the partner's rows.
bool pair_tiling_ok(int ny, int tile_y, int T)
{
    const int vy = 2 * tile_y - 2 * T;
    const int last = (ny + vy - 1) / vy - 1;
    const int f = ny - (last * vy - T + tile_y);         // rows of the last pair's lower CTA that lie inside the cube
    return f < -(T - 1) || f > T - 2;
}

// rounds > 1: cooperative launch of all rounds (COOP instantiation); the grid must be co-resident.
// pair: two CTAs of a cluster share a tile of 2 TILE_Y rows (T >= 2, plain launches, aligned rows only).
template <int T, int R, int WARPS, int NS, int MINB, bool COOP = false, bool PM = false, bool PAIR = false>
cudaError_t launch_cfg(const Launch &L, int zchunk, cudaStream_t st, int rounds = 1, unsigned *bar = nullptr)
{
    using S = Smem<T, R, WARPS, NS, PAIR>;
    constexpr int TILE_Y = WARPS * R;
    static_assert(TILE_Y > 2 * T, "tile must be taller than its halo");
    static_assert(S::kBytes * MINB <= 227 * 1024, "shared memory budget");
    static_assert(!(PAIR && (COOP || PM)), "the cluster-pair tiling exists for the plain intensity-driven kernel");
    constexpr bool coop = COOP;
    TmaArgs A;
    A.halo = T;
    A.rounds = rounds;
    A.bar = bar;
    const bool unal = L.pitch > 0;                       // nx % 4 != 0: pitched buffers, the face inside a float4
    const bool one = L.nx <= kTileX && !unal;            // a single tile column: no halo lanes
    if (PAIR && (unal || one)) return cudaErrorNotSupported;
    A.tiles_x = one ? 1 : ((L.nx + 3) / 4 + kValidLanes - 1) / kValidLanes;
    const int vy = (PAIR ? 2 : 1) * TILE_Y - 2 * T;
    A.tiles_y = (L.ny + vy - 1) / vy;
    const long tiles = (long)A.tiles_x * A.tiles_y * (PAIR ? 2 : 1);        // CTAs per cube and z chunk
    if (tiles > 0x7fffffffL) return cudaErrorInvalidValue;
    void (*kern)(Launch, TmaArgs, Maps);
    if constexpr (COOP) kern = one ? idg_tma_coop_kernel<T, R, WARPS, NS, MINB, true> : idg_tma_coop_kernel<T, R, WARPS, NS, MINB, false>;
    else if constexpr (PAIR) kern = idg_tma_kernel<T, R, WARPS, NS, MINB, false, false, false, true>;
    else if (unal && !PM) kern = idg_tma_kernel<T, R, WARPS, NS, MINB, false, false, !PM>;      // (!PM: no pm instantiation)
    else kern = one ? idg_tma_kernel<T, R, WARPS, NS, MINB, true, PM> : idg_tma_kernel<T, R, WARPS, NS, MINB, false, PM>;
    if (unal && (COOP || PM)) return cudaErrorNotSupported;
    static DeviceOnce smem_once[4];
    {
        const cudaError_t e = set_max_dynamic_smem(smem_once[PAIR ? 3 : unal ? 2 : one], (const void *)kern, S::kBytes);
        if (e != cudaSuccess) return e;
    }
    const int sms = device_sm_count();
    long slots = (long)sms * MINB;
    if (coop) {
        int per_sm = 0;                      // of the current device (the cooperative path is rare: asked every time)
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, WARPS * 32, S::kBytes) != cudaSuccess) per_sm = 0;
        slots = (long)per_sm * sms;
        if (slots <= 0 || tiles * L.batch > slots) return cudaErrorCooperativeLaunchTooLarge;
        A.zchunk = pick_zchunk(L.nz, tiles * L.batch, T, (int)slots, slots);
        if (zchunk > 0 && tiles * L.batch * ((L.nz + zchunk - 1) / zchunk) <= slots) A.zchunk = zchunk < L.nz ? zchunk : L.nz;
        if (A.zchunk <= 0) return cudaErrorCooperativeLaunchTooLarge;
    } else {
        A.zchunk = zchunk > 0 ? (zchunk < L.nz ? zchunk : L.nz) : pick_zchunk(L.nz, tiles * L.batch, T, sms * MINB);
    }
    if ((L.nz + A.zchunk - 1) / A.zchunk > 65535) A.zchunk = (L.nz + 65534) / 65535;
    Maps M;
    if (!encode_map(&M.in, L.in, L, S::kRows) || !encode_map(&M.out, L.out, L, S::kRows) ||
        !encode_map(&M.scratch, L.scratch, L, S::kRows))
        return cudaErrorNotSupported;
    dim3 grid((unsigned)tiles, (unsigned)((L.nz + A.zchunk - 1) / A.zchunk), (unsigned)L.batch);
    if (coop) {
        if ((long)grid.x * grid.y * grid.z > slots) return cudaErrorCooperativeLaunchTooLarge;
        void *args[3] = {(void *)&L, (void *)&A, (void *)&M};
        return cudaLaunchCooperativeKernel((const void *)kern, grid, dim3(WARPS * 32), args, S::kBytes, st);
    }
    if constexpr (PAIR) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = grid;
        cfg.blockDim = dim3(WARPS * 32);
        cfg.dynamicSmemBytes = S::kBytes;
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 2;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        return cudaLaunchKernelEx(&cfg, kern, L, A, M);
    }
    kern<<<grid, WARPS * 32, S::kBytes, st>>>(L, A, M);
    return cudaGetLastError();
}

}  // namespace

// The reflected source of a halo cell must lie inside the same tile: needs ny >= 4 (max halo)
// and a usable driver entry point for tensor-map encoding.
bool tma_supported(int nx, int ny, int nz, const void *in, const void *out, const void *scratch)
{
    (void)nz;
    if (nx % 4 != 0 || ny < 4) return false;
    const uintptr_t m = (uintptr_t)in | (uintptr_t)out | (uintptr_t)scratch;
    if ((m & 15u) != 0) return false;
    return tmap_available();
}

bool tma_pitched_supported(int nx, int ny, int nz)
{
    (void)nz;
    return nx % 4 != 0 && nx >= 5 && ny >= 4 && tmap_available();
}

namespace {
// Copy between a dense cube (row pitch nx, rows not 16-byte aligned) and its pitched copy (row pitch a multiple of 4
// floats): a thread moves one float4 of the pitched side and the 1..4 voxels of it that exist, the dense side by scalar
// accesses (coalesced across the warp).  TO_PITCHED: dense -> pitched, else pitched -> dense; cubes whose n_iter is 0
// take src_zero (their untouched input copy) instead of src.
template <bool TO_PITCHED>
__global__ void idg_repitch_kernel(const float *__restrict__ src, float *__restrict__ dst, int pitch,
                                   const float *__restrict__ src_zero, const CubeParams *__restrict__ tab, int nx,
                                   size_t rows_per_cube, size_t rows)
{
    const int p4 = pitch >> 2;
    const size_t total = rows * (size_t)p4;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const size_t row = i / (size_t)p4;
        const int x = (int)(i - row * (size_t)p4) * 4;
        if (TO_PITCHED) {
            const float *sr = src + row * (size_t)nx + x;
            float4 v;
            v.x = sr[0];
            v.y = x + 1 < nx ? sr[1] : 0.f;
            v.z = x + 2 < nx ? sr[2] : 0.f;
            v.w = x + 3 < nx ? sr[3] : 0.f;
            *reinterpret_cast<float4 *>(dst + row * (size_t)pitch + x) = v;
        } else {
            const float *s = src;
            if (src_zero && tab && tab[row / rows_per_cube].n_iter == 0) s = src_zero;
            const float4 v = *reinterpret_cast<const float4 *>(s + row * (size_t)pitch + x);
            float *dr = dst + row * (size_t)nx + x;
            dr[0] = v.x;
            if (x + 1 < nx) dr[1] = v.y;
            if (x + 2 < nx) dr[2] = v.z;
            if (x + 3 < nx) dr[3] = v.w;
        }
    }
}
}  // namespace

cudaError_t launch_repitch(const float *src, int src_pitch, float *dst, int dst_pitch, const float *src_zero,
                           const CubeParams *tab, int nx, int ny, int nz, int batch, cudaStream_t st)
{
    const size_t rows_per_cube = (size_t)ny * (size_t)nz, rows = rows_per_cube * (size_t)batch;
    const bool to_pitched = dst_pitch > src_pitch;
    const int pitch = to_pitched ? dst_pitch : src_pitch;
    const size_t total = rows * (size_t)(pitch / 4);
    size_t blocks = (total + 255) / 256;
    const size_t cap = (size_t)device_sm_count() * 16;
    if (blocks > cap) blocks = cap;
    if (to_pitched) idg_repitch_kernel<true><<<(unsigned)blocks, 256, 0, st>>>(src, dst, pitch, nullptr, nullptr, nx, rows_per_cube, rows);
    else idg_repitch_kernel<false><<<(unsigned)blocks, 256, 0, st>>>(src, dst, pitch, src_zero, tab, nx, rows_per_cube, rows);
    return cudaGetLastError();
}

// tile (T = fused iterations): T <= 2: 0, 1 = 128x64 tile, 512 threads, one CTA per SM | 2 = 128x32 tile, 256
// threads, two CTAs per SM.  T >= 3 needs the registers of a lone CTA: 0, 1 = 128x32 tile, 256 threads | 3 =
// 128x48 / 128x36 tile, 384 threads (T = 3: strips of 4 rows; T = 4: strips of 3).
cudaError_t launch_tma(const Launch &L, int zchunk, int tile, cudaStream_t st)
{
    if (L.mode == 1) {          // gradient-driven variant (Eq. 5): the default tilings
        switch (L.fuse) {
        case 1: return launch_cfg<1, 4, 8, 4, 2, false, true>(L, zchunk, st);
        case 2: return launch_cfg<2, 4, 8, 4, 2, false, true>(L, zchunk, st);
        case 3: return launch_cfg<3, 4, 8, 4, 1, false, true>(L, zchunk, st);
        case 4: return launch_cfg<4, 4, 8, 4, 1, false, true>(L, zchunk, st);
        default: return cudaErrorInvalidValue;
        }
    }
    const bool small = (tile == 2);
    switch (L.fuse) {
    case 1: return small ? launch_cfg<1, 4, 8, 4, 2>(L, zchunk, st) : launch_cfg<1, 4, 16, 4, 1>(L, zchunk, st);
    case 2: return small ? launch_cfg<2, 4, 8, 4, 2>(L, zchunk, st) : launch_cfg<2, 4, 16, 4, 1>(L, zchunk, st);
    case 3:
        switch (tile) {
        case 3: return launch_cfg<3, 4, 12, 4, 1>(L, zchunk, st);
        case 4:
            if (L.nx > kTileX && L.pitch == 0 && pair_tiling_ok(L.ny, 32, 3))
                return launch_cfg<3, 4, 8, 4, 1, false, false, true>(L, zchunk, st);
            return launch_cfg<3, 4, 8, 4, 1>(L, zchunk, st);
        default: return launch_cfg<3, 4, 8, 4, 1>(L, zchunk, st);
        }
    case 4:
        switch (tile) {
        case 3: return launch_cfg<4, 3, 12, 4, 1>(L, zchunk, st);
        case 4:
            if (L.nx > kTileX && L.pitch == 0 && pair_tiling_ok(L.ny, 32, 4))
                return launch_cfg<4, 4, 8, 4, 1, false, false, true>(L, zchunk, st);
            return launch_cfg<4, 4, 8, 4, 1>(L, zchunk, st);
        default: return launch_cfg<4, 4, 8, 4, 1>(L, zchunk, st);
        }
    default: return cudaErrorInvalidValue;
    }
}

// The default tilings only: T = 2 on two CTAs per SM, T = 3 / T = 4 on one 8-warp CTA per SM.
cudaError_t launch_tma_coop(const Launch &L, int zchunk, int tile, int rounds, unsigned *bar, cudaStream_t st)
{
    (void)tile;
    if (rounds < 2 || !bar) return cudaErrorNotSupported;
    switch (L.fuse) {
    case 2: return launch_cfg<2, 4, 8, 4, 2, true>(L, zchunk, st, rounds, bar);
    case 3: return launch_cfg<3, 4, 8, 4, 1, true>(L, zchunk, st, rounds, bar);
    case 4: return launch_cfg<4, 4, 8, 4, 1, true>(L, zchunk, st, rounds, bar);
    default: return cudaErrorNotSupported;
    }
}

}  // namespace idg
