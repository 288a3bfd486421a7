// Resident IDG kernel for small, L2-sized cubes and interactive batches (steps a1-a7 of DESIGN.md section 7; the
// regime of PAPER.md:21, :424, :507: "for small N it is not possible to fully load the GPU").
//
// One cooperative launch runs ALL n iterations.  A cube is cut into ty x tz blocks of full x rows; a CTA (one per
// SM) loads its block once, keeps it in shared memory for the whole call -- two copies, the Jacobi ping-pong of
// PAPER.md:430-432 on chip -- and writes it back once.  Per iteration only the four block faces travel, through
// mailboxes in the workspace (L2-resident), with the flag packed into the data: every voxel is one 64-bit word
// (iteration tag, fp32 bits) written and polled with relaxed gpu-scope accesses, so a face costs one L2 write and
// one L2 read latency and needs no fence and no grid barrier (a CTA waits for its <= 4 neighbours only).  Mailboxes
// are double buffered by iteration parity: a neighbour can be at most one iteration ahead.  They are cleared by
// their owner at the start of the call, before the launch's single grid-wide barrier.
//
// Each block is stored with a one-cell frame in y and z.  A frame cell on a true cube face holds a copy of the
// face voxel (reading R1: zero flux by replication, written by the thread that computes the face voxel); one on an
// interior face holds the neighbour's voxel of the same iterate.  x faces: the first / last float4 of a row uses its
// own end component.  A thread owns a float4 column of a block and walks a segment of it along z with the z
// neighbours in registers; the arithmetic is update4() of idg_update.cuh, so results are bit-identical to every
// other kernel.
#include <cooperative_groups.h>

#include <type_traits>

#include "idg_kernels.cuh"
#include "idg_ptx.cuh"
#include "idg_update.cuh"

namespace cg = cooperative_groups;

namespace idg {

namespace {

constexpr int kThreads = 512;
constexpr size_t kSmemBudget = 220 * 1024;
constexpr int kMaxChunk = kThreads > 512 ? 2 : 4;      // independent z cells a thread computes at a time (registers)

struct ResArgs {
    const float *in;                // cube 0 of this launch
    float *out;
    const CubeParams *tab;          // device table (first cube of this launch), or nullptr -> `one`
    CubeParams one;
    unsigned long long *mail;       // mailboxes: [block][parity][words]
    int nx, ny, nz;
    int ty, tz;                     // blocks per cube along y, z
    int by, bz;                     // nominal block extents (the last block of an axis may be smaller)
    int ls;                         // z cells per work item
    int words;                      // 64-bit words per (block, parity): 8 nx4 (by + bz) of faces + 8 (4 flags)
    unsigned m_nx4;                 // ceil(2^32 / nx4), nx4 = ceil(nx / 4): division by multiplication
    int tail;                       // nx % 4: voxels in the last float4 of a row (0: all four)
    int unal;                       // rows of the cubes are not 16-byte aligned (tail != 0 or odd base pointers): scalar global access
};

__device__ __forceinline__ void st_relaxed_v2(unsigned long long *p, unsigned long long a, unsigned long long b)
{
    asm volatile("st.relaxed.gpu.global.v2.b64 [%0], {%1, %2};" ::"l"(p), "l"(a), "l"(b));
}
__device__ __forceinline__ void ld_relaxed_v2(const unsigned long long *p, unsigned long long &a, unsigned long long &b)
{
    asm volatile("ld.relaxed.gpu.global.v2.b64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "l"(p));
}
__device__ __forceinline__ unsigned long long pack(float v, unsigned tag)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(__float_as_uint(v)), "r"(tag));
    return r;
}
// One float4 of a face -> the neighbour's mailbox: four (tag, value) words.  A face of E float4 entries is stored as
// E (x, y) pairs followed by E (z, w) pairs, so that both accesses of a warp are contiguous (full 32-byte sectors).
__device__ __forceinline__ void push(unsigned long long *lo, int hi, const F4 &o, unsigned tag)
{
    st_relaxed_v2(lo, pack(o.x, tag), pack(o.y, tag));
    st_relaxed_v2(lo + hi, pack(o.z, tag), pack(o.w, tag));
}
// Wait for one float4 of a face of iterate `tag`.
__device__ __forceinline__ F4 pull(const unsigned long long *lo, int hi, unsigned tag)
{
    unsigned long long a, b, c, d;
    do {
        ld_relaxed_v2(lo, a, b);
        ld_relaxed_v2(lo + hi, c, d);
    } while ((unsigned)(a >> 32) != tag || (unsigned)(b >> 32) != tag || (unsigned)(c >> 32) != tag ||
             (unsigned)(d >> 32) != tag);
    return F4{__uint_as_float((unsigned)a), __uint_as_float((unsigned)b), __uint_as_float((unsigned)c),
              __uint_as_float((unsigned)d)};
}

// x / d for x < 2^32 / d with m = ceil(2^32 / d) from the host
__device__ __forceinline__ int fdiv(int x, unsigned m) { return (int)__umulhi((unsigned)x, m); }

// One warp work item: 32 consecutive float4 columns (x fastest, then y) of the block over the planes [zs, ze).
struct Item {
    int off;                // shared-memory offset (floats) of the thread's cell in plane zs
    int x4, y, zs, ze;
    bool valid;             // the lane has a column (the last item of a segment may be ragged)
};

// CH cells of one column, planes z .. z+CH-1: every load first, then CH independent updates (Eq. 7), then the stores.
// pm / p0: the column's cells in planes z-1 and z; on return those of planes z+CH-1 and z+CH.
template <int CH, bool PM>
__device__ __forceinline__ void chunk(const float *cur, float *nxt, int off, int PP, int RP, F4 &pm, F4 &p0, bool first,
                                      bool last, bool lds_l, bool lds_r, bool valid, const Consts &kc, F4 (&o)[CH],
                                      int tail)
{
    F4 pl[CH + 2], ym[CH], yp[CH];
    float l[CH], r[CH];
    pl[0] = pm;
    pl[1] = p0;
#pragma unroll
    for (int k = 0; k < CH; ++k) {
        pl[k + 2] = lds4(cur + off + (k + 1) * PP);
        ym[k] = lds4(cur + off + k * PP - RP);
        yp[k] = lds4(cur + off + k * PP + RP);
    }
#pragma unroll
    for (int k = 0; k < CH; ++k) {
        l[k] = __shfl_up_sync(0xffffffffu, pl[k + 1].w, 1);
        r[k] = __shfl_down_sync(0xffffffffu, pl[k + 1].x, 1);
        if (lds_l) l[k] = cur[off + k * PP - 1];          // lane 0 of a warp that starts inside a row
        if (lds_r) r[k] = cur[off + k * PP + 4];
    }
#pragma unroll
    for (int k = 0; k < CH; ++k)
        o[k] = update4<PM>(pl[k + 1], first ? pl[k + 1].x : l[k], last ? pl[k + 1].w : r[k], ym[k], yp[k], pl[k],
                           pl[k + 2], kc);
    if (tail && last) {             // nx % 4 != 0: the pad components of a row's last float4 repeat the last voxel --
#pragma unroll                      // the replicated x face (reading R1) of the next iteration
        for (int k = 0; k < CH; ++k) {
            if (tail == 1) o[k].y = o[k].z = o[k].w = o[k].x;
            else if (tail == 2) o[k].z = o[k].w = o[k].y;
            else o[k].w = o[k].z;
        }
    }
    if (valid) {
#pragma unroll
        for (int k = 0; k < CH; ++k) sts4(nxt + off + k * PP, o[k]);
    }
    pm = pl[CH];
    p0 = pl[CH + 1];
}

// UNAL: rows of the cubes are not 16-byte aligned (nx % 4 != 0 or odd base pointers): scalar global access, and the pad
// components of a row's last float4 are kept equal to the last voxel.  The aligned instantiation has none of that.
template <bool PM, bool UNAL>
__global__ void __launch_bounds__(kThreads, 1) idg_resident_kernel(const __grid_constant__ ResArgs A)
{
    const int tail = UNAL ? A.tail : 0;
    extern __shared__ __align__(16) float smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int s = blockIdx.x;
    const int iy = s % A.ty, iz = (s / A.ty) % A.tz, cube = s / (A.ty * A.tz);
    const CubeParams prm = A.tab ? A.tab[cube] : A.one;
    const int nx = A.nx, nx4 = (nx + 3) >> 2;              // float4 columns of a (padded) row
    const unsigned mx4 = A.m_nx4;
    const int y0 = iy * A.by, h = min(A.by, A.ny - y0);
    const int z0 = iz * A.bz, d = min(A.bz, A.nz - z0);
    const int RP = 4 * nx4, PP = (A.by + 2) * RP;                  // row / plane pitch in floats (rows padded to float4)
    const int buf = (A.bz + 2) * PP + 8;                             // one copy (+ slack for the x reads at the ends)
    float *cur = smem + 4, *nxt = smem + 4 + buf;
    // neighbours: the block holding my y-1 / y+h rows and my z-1 / z+d planes (-1: a true cube face)
    const int nb_ym = iy > 0 ? s - 1 : -1, nb_yp = iy + 1 < A.ty ? s + 1 : -1;
    const int nb_zm = iz > 0 ? s - A.ty : -1, nb_zp = iz + 1 < A.tz ? s + A.ty : -1;
    // mailbox layout per (block, parity): faces YM | YP (nx4 x bz float4 each) | ZM | ZP (nx4 x by each), 4 words per float4
    const int f_yp = 4 * nx4 * A.bz, f_zm = 2 * f_yp, f_zp = f_zm + 4 * nx4 * A.by;
    const size_t plane_g = (size_t)nx * (size_t)A.ny;
    const size_t cube_off = (size_t)cube * plane_g * (size_t)A.nz;

    // clear my mailboxes (both parities): tag 0 is never expected
    {
        ulonglong2 *m = reinterpret_cast<ulonglong2 *>(A.mail + (size_t)s * 2 * A.words);
        for (int i = tid; i < A.words; i += kThreads) m[i] = make_ulonglong2(0ull, 0ull);      // 2 parities x words / 2
    }
    // load the block with its frame: outside the cube the nearest voxel (R1), else the neighbour's voxel
    {
        const float *src = A.in + cube_off;
        const int cells = (d + 2) * (h + 2) * nx4;
        for (int i = tid; i < cells; i += kThreads) {
            const int r = fdiv(i, mx4), x4 = i - r * nx4, zz = r / (h + 2), y = r - zz * (h + 2) - 1, z = zz - 1;
            const int gy = min(max(y0 + y, 0), A.ny - 1), gz = min(max(z0 + z, 0), A.nz - 1);
            const float *row = src + (size_t)gz * plane_g + (size_t)gy * nx;
            float4 v;
            if (!UNAL) {
                v = __ldg(reinterpret_cast<const float4 *>(row) + x4);
            } else {                    // scalar loads; components beyond the row repeat its last voxel
                const int x = 4 * x4;
                v.x = __ldg(row + x);
                v.y = __ldg(row + min(x + 1, nx - 1));
                v.z = __ldg(row + min(x + 2, nx - 1));
                v.w = __ldg(row + min(x + 3, nx - 1));
            }
            *reinterpret_cast<float4 *>(cur + (z + 1) * PP + (y + 1) * RP + 4 * x4) = v;
        }
    }
    __threadfence();
    cg::this_grid().sync();          // every mailbox is clear and every block loaded (in-place calls: before any store)

    const Consts kc = make_consts<PM>(prm);
    const int n = prm.n_iter;
    const int ncols = nx4 * h, cw = (ncols + 31) / 32, nseg = (d + A.ls - 1) / A.ls, nwitems = cw * nseg;
    const int ney = nx4 * d, nez = nx4 * h;
    unsigned long long *const inbox = A.mail + (size_t)s * 2 * A.words;
    // where my faces go: the neighbour's inbox face that borders on me (parity 0; + words for parity 1)
    unsigned long long *const o_ym = nb_ym >= 0 ? A.mail + (size_t)nb_ym * 2 * A.words + f_yp : nullptr;
    unsigned long long *const o_yp = nb_yp >= 0 ? A.mail + (size_t)nb_yp * 2 * A.words : nullptr;
    unsigned long long *const o_zm = nb_zm >= 0 ? A.mail + (size_t)nb_zm * 2 * A.words + f_zp : nullptr;
    unsigned long long *const o_zp = nb_zp >= 0 ? A.mail + (size_t)nb_zp * 2 * A.words + f_zm : nullptr;

    auto decode = [&](int wi) {
        Item I;
        const int seg = wi / cw, col_raw = (wi - seg * cw) * 32 + lane;
        I.valid = col_raw < ncols;
        const int col = I.valid ? col_raw : ncols - 1;
        I.y = fdiv(col, mx4);
        I.x4 = col - I.y * nx4;
        I.zs = seg * A.ls;
        I.ze = min(d, I.zs + A.ls);
        I.off = (I.zs + 1) * PP + (I.y + 1) * RP + 4 * I.x4;
        return I;
    };
    // One face cell of the new iterate: a true cube face is replicated into the frame, an interior face is sent.
    auto face = [&](int off, int delta, unsigned long long *lo, int hi, bool xchg, unsigned tag) {
        const F4 v = lds4(nxt + off);
        if (!lo) sts4(nxt + off + delta, v);
        else if (xchg) push(lo, hi, v, tag);
    };
    const int hi_y = 2 * nx4 * A.bz, hi_z = 2 * nx4 * A.by;          // words from the (x, y) to the (z, w) pair of an entry
    auto run_item = [&](const Item &I, bool xchg, unsigned tag, int pw) {
        const bool first = I.x4 == 0, last = I.x4 == nx4 - 1;
        const bool lds_l = lane == 0 && !first, lds_r = lane == 31 && !last;
        int off = I.off;
        F4 pm = lds4(cur + off - PP), p0 = lds4(cur + off);
        int z = I.zs;
        F4 oM[kMaxChunk], o1[1];
        for (; z + kMaxChunk <= I.ze; z += kMaxChunk, off += kMaxChunk * PP)
            chunk<kMaxChunk, PM>(cur, nxt, off, PP, RP, pm, p0, first, last, lds_l, lds_r, I.valid, kc, oM, tail);
        for (; z < I.ze; ++z, off += PP) chunk<1, PM>(cur, nxt, off, PP, RP, pm, p0, first, last, lds_l, lds_r, I.valid, kc, o1, tail);
        if (!I.valid) return;
        // my own face cells (read back from `nxt`: this thread wrote them)
        if (I.y == 0 || I.y == h - 1) {
            for (int zz = I.zs; zz < I.ze; ++zz) {
                const int o = I.off + (zz - I.zs) * PP, e = 2 * (zz * nx4 + I.x4);
                if (I.y == 0) face(o, -RP, o_ym ? o_ym + pw + e : nullptr, hi_y, xchg, tag);
                if (I.y == h - 1) face(o, RP, o_yp ? o_yp + pw + e : nullptr, hi_y, xchg, tag);
            }
        }
        const int e = 2 * (I.y * nx4 + I.x4);
        if (I.zs == 0) face(I.off, -PP, o_zm ? o_zm + pw + e : nullptr, hi_z, xchg, tag);
        if (I.ze == d) face(I.off + (d - 1 - I.zs) * PP, PP, o_zp ? o_zp + pw + e : nullptr, hi_z, xchg, tag);
    };
    // An inbound face entry e of this block: where it arrives (parity 0) and where it goes in the frame.
    struct Inbound { const unsigned long long *lo; int hi, dst; };
    const int n_in = 2 * ney + 2 * nez;
    auto inbound = [&](int e) {
        Inbound r{nullptr, 0, 0};
        if (e >= n_in) return r;
        int idx = e, nb = nb_ym, fo = 0;
        if (e >= 2 * ney + nez) { idx = e - 2 * ney - nez; nb = nb_zp; fo = f_zp; }
        else if (e >= 2 * ney) { idx = e - 2 * ney; nb = nb_zm; fo = f_zm; }
        else if (e >= ney) { idx = e - ney; nb = nb_yp; fo = f_yp; }
        if (nb < 0) return r;
        const int k = fdiv(idx, mx4), x4 = idx - k * nx4;            // k: z (y faces) or y (z faces)
        r.lo = inbox + fo + 2 * idx;
        r.hi = e < 2 * ney ? hi_y : hi_z;
        r.dst = e < ney ? (k + 1) * PP + 4 * x4
              : e < 2 * ney ? (k + 1) * PP + (h + 1) * RP + 4 * x4
              : e < 2 * ney + nez ? (k + 1) * RP + 4 * x4
                                  : (d + 1) * PP + (k + 1) * RP + 4 * x4;
        return r;
    };

    // Small blocks (the single-cube interactive case): at most one item per warp and two inbound
    // entries per thread.  Everything that does not change from one iteration to the next is worked out once, and a
    // warp runs the loop built for its number of cells.
    // The choice must be the SAME for every CTA of the grid (the two paths hand faces over differently: only the
    // large-block path raises and waits for the per-face flags), so it is taken on the NOMINAL block extents, not on
    // this CTA's -- a ragged last block is smaller and would otherwise pick the other path than its neighbours.
    const int nom_items = ((nx4 * A.by + 31) / 32) * ((A.bz + A.ls - 1) / A.ls);
    const int nom_in = 2 * nx4 * (A.by + A.bz);
    const bool small = nom_items <= kThreads / 32 && nom_in <= 2 * kThreads && A.ls <= kMaxChunk;
    if (small) {
        const Item I = decode(warp < nwitems ? warp : 0);
        const int cnt = warp < nwitems ? I.ze - I.zs : 0;
        const Inbound in0 = inbound(tid), in1 = inbound(tid + kThreads);
        auto loop = [&](auto CHc) {
            constexpr int CH = decltype(CHc)::value;
            const bool first = I.x4 == 0, last = I.x4 == nx4 - 1;
            const bool lds_l = lane == 0 && !first, lds_r = lane == 31 && !last;
            const bool yf0 = I.y == 0, yf1 = I.y == h - 1, zf0 = I.zs == 0, zf1 = I.ze == d;
            unsigned long long *const s_ym = o_ym ? o_ym + 2 * (I.zs * nx4 + I.x4) : nullptr;
            unsigned long long *const s_yp = o_yp ? o_yp + 2 * (I.zs * nx4 + I.x4) : nullptr;
            unsigned long long *const s_zm = o_zm ? o_zm + 2 * (I.y * nx4 + I.x4) : nullptr;
            unsigned long long *const s_zp = o_zp ? o_zp + 2 * (I.y * nx4 + I.x4) : nullptr;
            for (int it = 1; it <= n; ++it) {
                const bool xchg = it < n;
                const unsigned tag = (unsigned)it;
                const int pw = (it & 1) * A.words;
                if (CH > 0) {
                    F4 o[CH > 0 ? CH : 1];
                    F4 pm = lds4(cur + I.off - PP), p0 = lds4(cur + I.off);
                    chunk<(CH > 0 ? CH : 1), PM>(cur, nxt, I.off, PP, RP, pm, p0, first, last, lds_l, lds_r, I.valid, kc, o, tail);
                    if (I.valid) {
#pragma unroll
                        for (int k = 0; k < CH; ++k) {
                            const int ok = I.off + k * PP;
                            if (yf0) {
                                if (!s_ym) sts4(nxt + ok - RP, o[k]);
                                else if (xchg) push(s_ym + pw + 2 * k * nx4, hi_y, o[k], tag);
                            }
                            if (yf1) {
                                if (!s_yp) sts4(nxt + ok + RP, o[k]);
                                else if (xchg) push(s_yp + pw + 2 * k * nx4, hi_y, o[k], tag);
                            }
                        }
                        if (zf0) {
                            if (!s_zm) sts4(nxt + I.off - PP, o[0]);
                            else if (xchg) push(s_zm + pw, hi_z, o[0], tag);
                        }
                        if (zf1) {
                            if (!s_zp) sts4(nxt + I.off + CH * PP, o[CH > 0 ? CH - 1 : 0]);
                            else if (xchg) push(s_zp + pw, hi_z, o[CH > 0 ? CH - 1 : 0], tag);
                        }
                    }
                }
                if (xchg) {
                    // both entries of the thread are requested before either is examined (one L2 round trip)
                    bool w0 = in0.lo != nullptr, w1 = in1.lo != nullptr;
                    while (w0 || w1) {
                        unsigned long long a0, b0, c0, d0, a1, b1, c1, d1;
                        if (w0) { ld_relaxed_v2(in0.lo + pw, a0, b0); ld_relaxed_v2(in0.lo + pw + in0.hi, c0, d0); }
                        if (w1) { ld_relaxed_v2(in1.lo + pw, a1, b1); ld_relaxed_v2(in1.lo + pw + in1.hi, c1, d1); }
                        if (w0 && (unsigned)(a0 >> 32) == tag && (unsigned)(b0 >> 32) == tag && (unsigned)(c0 >> 32) == tag &&
                            (unsigned)(d0 >> 32) == tag) {
                            sts4(nxt + in0.dst, F4{__uint_as_float((unsigned)a0), __uint_as_float((unsigned)b0),
                                                   __uint_as_float((unsigned)c0), __uint_as_float((unsigned)d0)});
                            w0 = false;
                        }
                        if (w1 && (unsigned)(a1 >> 32) == tag && (unsigned)(b1 >> 32) == tag && (unsigned)(c1 >> 32) == tag &&
                            (unsigned)(d1 >> 32) == tag) {
                            sts4(nxt + in1.dst, F4{__uint_as_float((unsigned)a1), __uint_as_float((unsigned)b1),
                                                   __uint_as_float((unsigned)c1), __uint_as_float((unsigned)d1)});
                            w1 = false;
                        }
                    }
                }
                __syncthreads();
                float *t = cur;
                cur = nxt;
                nxt = t;
            }
        };
        if (kMaxChunk > 2 && cnt == 4) loop(std::integral_constant<int, (kMaxChunk > 2 ? 4 : 0)>{});
        else if (kMaxChunk > 2 && cnt == 3) loop(std::integral_constant<int, (kMaxChunk > 2 ? 3 : 0)>{});
        else if (cnt == 2) loop(std::integral_constant<int, 2>{});
        else if (cnt == 1) loop(std::integral_constant<int, 1>{});
        else loop(std::integral_constant<int, 0>{});
    } else {
        for (int it = 1; it <= n; ++it) {
            const bool xchg = it < n;                    // the last iterate is not sent on
            const unsigned tag = (unsigned)it;
            const int pw = (it & 1) * A.words;
            for (int wi = warp; wi < nwitems; wi += kThreads / 32) run_item(decode(wi), xchg, tag, pw);
            if (xchg) {
                // Large blocks: polling every face entry from the moment the block is computed floods the L2 with
                // requests (12 rounds per entry were measured) that delay the very stores they wait for.  So a CTA
                // raises one flag per face AFTER all its warps have issued their face stores, the receiver waits on
                // its four flags with four threads, and only then reads the faces -- once, as a rule; every entry
                // still carries its tag and is re-read until it matches (flag and data are not ordered).
                __syncthreads();
                const int fl = A.words - 8;
                if (tid < 4) {
                    const int nb = tid == 0 ? nb_ym : tid == 1 ? nb_yp : tid == 2 ? nb_zm : nb_zp;
                    if (nb >= 0) {
                        unsigned long long *f = A.mail + (size_t)nb * 2 * A.words + pw + fl + (tid ^ 1);
                        asm volatile("st.relaxed.gpu.global.b64 [%0], %1;" ::"l"(f), "l"((unsigned long long)tag));
                        const unsigned long long *mine = inbox + pw + fl + tid;
                        unsigned long long v;
                        do {
                            asm volatile("ld.relaxed.gpu.global.b64 %0, [%1];" : "=l"(v) : "l"(mine));
                        } while (v != (unsigned long long)tag);
                    }
                }
                __syncthreads();
                for (int e = tid; e < n_in; e += kThreads) {     // my neighbours' faces of this iterate -> the frame of `nxt`
                    const Inbound in = inbound(e);
                    if (in.lo) sts4(nxt + in.dst, pull(in.lo + pw, in.hi, tag));
                }
            }
            __syncthreads();
            float *t = cur;
            cur = nxt;
            nxt = t;
        }
    }

    // I_n -> out
    {
        float *dst = A.out + cube_off;
        const int cells = d * h * nx4;
        for (int i = tid; i < cells; i += kThreads) {
            const int r = fdiv(i, mx4), x4 = i - r * nx4, z = r / h, y = r - z * h;
            const float4 v = *reinterpret_cast<const float4 *>(cur + (z + 1) * PP + (y + 1) * RP + 4 * x4);
            float *row = dst + (size_t)(z0 + z) * plane_g + (size_t)(y0 + y) * nx;
            if (!UNAL) {
                reinterpret_cast<float4 *>(row)[x4] = v;
            } else {
                const int x = 4 * x4;
                row[x] = v.x;
                if (x + 1 < nx) row[x + 1] = v.y;
                if (x + 2 < nx) row[x + 2] = v.z;
                if (x + 3 < nx) row[x + 3] = v.w;
            }
        }
    }
}

struct DevInfo { int sms = 0, coop = 0; };
DevInfo dev_info()
{
    DevInfo d;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return d;
    cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&d.coop, cudaDevAttrCooperativeLaunch, dev);
    return d;
}

}  // namespace

// Cost model (SM cycles per wave, calibrated on B200: profiles/r2a_notes.md): a cell costs ~18 clk of shared-memory
// bandwidth per warp, a face entry ~24, an iteration ~700 of exchange latency and barrier; load + store + launch.
namespace {
// The search below costs tens of microseconds: remember the last few answers per thread.
struct PlanKey { int nx, ny, nz, batch, max_n, sms; size_t mail; };
struct PlanSlot { PlanKey key; ResidentPlan plan; bool ok, used; };
thread_local PlanSlot t_plans[8];
thread_local int t_next_slot = 0;
bool same_key(const PlanKey &a, const PlanKey &b)
{
    return a.nx == b.nx && a.ny == b.ny && a.nz == b.nz && a.batch == b.batch && a.max_n == b.max_n && a.sms == b.sms &&
           a.mail == b.mail;
}
bool search_plan(int nx, int ny, int nz, int batch, int max_n, size_t mail_bytes, int sms, ResidentPlan *out);
}  // namespace

bool resident_plan(int nx, int ny, int nz, int batch, int max_n, size_t mail_bytes, int sms, ResidentPlan *out)
{
    const PlanKey key{nx, ny, nz, batch, max_n, sms, mail_bytes};
    for (PlanSlot &p : t_plans)
        if (p.used && same_key(p.key, key)) {
            *out = p.plan;
            return p.ok;
        }
    PlanSlot &slot = t_plans[t_next_slot];
    t_next_slot = (t_next_slot + 1) % 8;
    slot.key = key;
    slot.used = true;
    slot.ok = search_plan(nx, ny, nz, batch, max_n, mail_bytes, sms, &slot.plan);
    *out = slot.plan;
    return slot.ok;
}

namespace {
bool search_plan(int nx, int ny, int nz, int batch, int max_n, size_t mail_bytes, int sms, ResidentPlan *out)
{
    if (nx < 8 || sms < 1 || max_n < 1) return false;      // (the division by multiplication needs nx4 > 1)
    const int nx4 = (nx + 3) / 4, nxp = 4 * nx4;           // rows are padded to whole float4 in shared memory
    double best = -1.0;
    ResidentPlan bp{};
    for (int ty = 1; ty <= ny && ty <= sms; ++ty) {
        const int by = (ny + ty - 1) / ty;
        if ((ty - 1) * by >= ny) continue;                          // an empty last block
        for (int tz = 1; tz <= nz && ty * tz <= sms; ++tz) {
            const int bz = (nz + tz - 1) / tz;
            if ((tz - 1) * bz >= nz) continue;
            const size_t smem = 2 * ((size_t)(bz + 2) * (by + 2) * nxp + 8) * sizeof(float);
            if (smem > kSmemBudget) continue;
            const int per_wave = sms / (ty * tz);                   // cubes per launch
            const int cubes = per_wave < batch ? per_wave : batch;
            const size_t words = (size_t)2 * nxp * (by + bz) + 8;     // faces + one arrival flag per face
            if ((size_t)cubes * ty * tz * 2 * words * 8 > mail_bytes) continue;
            const int waves = (batch + per_wave - 1) / per_wave;
            // a warp item = 32 columns x ls cells; pick the segment length that balances the 16 warps best
            const int cw = (nx4 * by + 31) / 32;
            int ls_best = bz;
            double t_best = -1.0;
            for (int ls = 1; ls <= bz; ++ls) {
                if (ls > kMaxChunk && ls % kMaxChunk != 0) continue;          // whole chunks
                const int items = cw * ((bz + ls - 1) / ls);
                const double t = (double)((items + kThreads / 32 - 1) / (kThreads / 32)) * (ls * 18.0 + 16.0);
                if (t_best < 0 || t < t_best) { t_best = t; ls_best = ls; }
            }
            const double faces = 2.0 * nx4 * (by + bz);
            const double iter = t_best * (kThreads / 32) + faces / 32.0 * 24.0 + 700.0;     // shared-memory bound: warps serialise
            const double io = (double)(bz + 2) * (by + 2) * nx4 / 32.0 * 12.0 + 6000.0;
            const double cost = waves * (max_n * iter + io);
            if (best < 0 || cost < best) {
                best = cost;
                // the kernel's own predicate (nominal block extents; idg_resident_kernel: `small`)
                const int nom_items = ((nx4 * by + 31) / 32) * ((bz + ls_best - 1) / ls_best);
                const bool small = nom_items <= kThreads / 32 && 2 * nx4 * (by + bz) <= 2 * kThreads && ls_best <= kMaxChunk;
                bp = ResidentPlan{ty, tz, by, bz, ls_best, cubes, (int)words, smem, small};
            }
        }
    }
    if (best < 0) return false;
    *out = bp;
    return true;
}
}  // namespace

cudaError_t launch_resident(const Launch &L, const ResidentPlan &P, unsigned long long *mail, cudaStream_t st,
                            int *launches)
{
    const bool unal = (L.nx & 3) != 0 || (((uintptr_t)L.in | (uintptr_t)L.out) & 15u) != 0;
    void (*kern)(ResArgs) = L.mode == 1 ? (unal ? idg_resident_kernel<true, true> : idg_resident_kernel<true, false>)
                                        : (unal ? idg_resident_kernel<false, true> : idg_resident_kernel<false, false>);
    // function attribute and co-residency check once per (thread, device, variant, shared-memory size)
    struct Checked { int dev, mode; size_t smem; long slots; };
    thread_local Checked chk{-1, 0, 0, 0};
    const int variant = L.mode * 2 + (unal ? 1 : 0);
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (chk.dev != dev || chk.mode != variant || chk.smem != P.smem) {
        const DevInfo di = dev_info();
        if (!di.coop) return cudaErrorNotSupported;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P.smem);
        if (e != cudaSuccess) return e;
        int per_sm = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kThreads, P.smem);
        if (e != cudaSuccess) return e;
        chk = Checked{dev, variant, P.smem, (long)per_sm * di.sms};
    }
    if ((long)P.ty * P.tz * P.cubes > chk.slots) return cudaErrorCooperativeLaunchTooLarge;
    const size_t N = (size_t)L.nx * (size_t)L.ny * (size_t)L.nz;
    *launches = 0;
    for (int b0 = 0; b0 < L.batch; b0 += P.cubes) {
        const int nc = L.batch - b0 < P.cubes ? L.batch - b0 : P.cubes;
        ResArgs A;
        A.in = L.in + (size_t)b0 * N;
        A.out = L.out + (size_t)b0 * N;
        A.tab = L.tab ? L.tab + b0 : nullptr;
        A.one = L.one;
        A.mail = mail;
        A.nx = L.nx; A.ny = L.ny; A.nz = L.nz;
        A.ty = P.ty; A.tz = P.tz; A.by = P.by; A.bz = P.bz; A.ls = P.ls;
        A.words = P.words;
        const unsigned nx4 = (unsigned)((L.nx + 3) / 4);
        A.m_nx4 = (unsigned)((0x100000000ull + nx4 - 1) / nx4);
        A.tail = L.nx & 3;
        A.unal = unal ? 1 : 0;
        void *args[1] = {(void *)&A};
        e = cudaLaunchCooperativeKernel((const void *)kern, dim3((unsigned)(P.ty * P.tz * nc)), dim3(kThreads), args,
                                        P.smem, st);
        if (e != cudaSuccess) return e;
        ++*launches;
    }
    return cudaSuccess;
}

}  // namespace idg
