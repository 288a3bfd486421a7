// C-ABI entry points of libidg_b200.so (declared in include/idg.h): argument
// validation, parameter preparation (step a0), launch planning.  Every voxel
// update runs in the kernels of idg_naive.cu / idg_tiled.cu.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <vector>

#include "../../include/idg.h"
#include "idg_kernels.cuh"

namespace {

thread_local int g_opt[IDG_OPT_COUNT_] = {0, 0, 0, 0, 0, 0, 0};      // tuning knobs of the calling host thread
thread_local int t_launches = 0;
thread_local char t_plan[96] = "none";

constexpr size_t kAlign = 256;
constexpr double kCoopMaxVoxels = 1.5e6;      // auto plan: cooperative single launch up to this many voxels per call
inline size_t align_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

bool voxel_count(int nx, int ny, int nz, int batch, size_t *n_one)
{
    if (nx < 1 || ny < 1 || nz < 1 || batch < 1 || batch > 65535) return false;
    const unsigned long long n = (unsigned long long)nx * (unsigned long long)ny;
    if (n > (1ull << 40)) return false;
    const unsigned long long N = n * (unsigned long long)nz;
    if (N > (1ull << 40) || N * (unsigned long long)batch > (1ull << 42)) return false;
    *n_one = (size_t)N;
    return true;
}

// Shapes the resident kernel can take (a cube small enough to sit in the SMs' shared memory; any nx >= 8, rows are
// padded to float4 on chip): the workspace then carries the mailbox region.
bool resident_shape(int nx, size_t N) { return nx >= 8 && N <= idg::kResidentMaxCubeVoxels; }

// Bytes of one pitched copy of a batch (row pitch = nx rounded up to a multiple of 4 floats = 16 bytes).
size_t pitched_bytes(int nx, int ny, int nz, int batch)
{
    return (size_t)((nx + 3) / 4 * 4) * (size_t)ny * (size_t)nz * (size_t)batch * sizeof(float);
}

bool params_valid(const idg_params &p)
{
    if (!(p.K > 0.0f)) return false;                         // rejects NaN, 0, negatives; +inf passes
    if (!(p.tau >= 0.0f) || !isfinite(p.tau)) return false;
    if (!(p.cx >= 0.0f) || !(p.cy >= 0.0f) || !(p.cz >= 0.0f)) return false;
    if (!isfinite(p.cx) || !isfinite(p.cy) || !isfinite(p.cz)) return false;
    if (!(p.rms > 0.0f) || !isfinite(p.rms)) return false;
    return true;
}

// Step a0: constants in fp64, rounded once to fp32 (Eq. 6-7).
idg::CubeParams prepare(const idg_params &p, int n_iter)
{
    idg::CubeParams c;
    memset(&c, 0, sizeof(c));
    c.ax = (float)((double)p.tau * (double)p.cx);
    c.ay = (float)((double)p.tau * (double)p.cy);
    c.az = (float)((double)p.tau * (double)p.cz);
    c.s = isinf(p.K) ? 0.0f : (float)(1.0 / ((double)p.K * (double)p.rms));
    c.w = (float)(-2.0 * (double)p.tau * ((double)p.cx + (double)p.cy + (double)p.cz));
    c.n_iter = n_iter;
    return c;
}

bool ranges_overlap(const void *a, size_t na, const void *b, size_t nb)
{
    const char *pa = (const char *)a, *pb = (const char *)b;
    return pa < pb + nb && pb < pa + na;
}

int run(const float *cubes, int nx, int ny, int nz, int batch, const int *n_iter, int n_iter_all,
        const idg_params *params, float *out, void *workspace, size_t workspace_bytes,
        cudaStream_t st, int mode = 0)
{
    t_launches = 0;
    if (!cubes || !out || !params) return IDG_ERR_NULL;
    size_t N;
    if (!voxel_count(nx, ny, nz, batch, &N)) return IDG_ERR_DIMS;
    int max_n = 0;
    for (int b = 0; b < batch; ++b) {
        const int n = n_iter ? n_iter[b] : n_iter_all;
        if (n < 0) return IDG_ERR_NITER;
        if (n > max_n) max_n = n;
        if (!params_valid(params[b])) return IDG_ERR_PARAM;
    }
    const size_t need = idg_workspace_bytes(nx, ny, nz, batch);
    if (!workspace || workspace_bytes < need || ((uintptr_t)workspace % kAlign) != 0)
        return IDG_ERR_WORKSPACE;
    const size_t bytes = N * (size_t)batch * sizeof(float);
    const bool in_place = (const float *)out == cubes;
    if (!in_place && ranges_overlap(cubes, bytes, out, bytes)) return IDG_ERR_OVERLAP;
    if (ranges_overlap(workspace, need, out, bytes) || ranges_overlap(workspace, need, cubes, bytes))
        return IDG_ERR_OVERLAP;

    float *scratch = (float *)workspace;
    const size_t pbytes = pitched_bytes(nx, ny, nz, batch);
    idg::CubeParams *tab = (idg::CubeParams *)((char *)workspace + align_up(nx % 4 ? 3 * pbytes : bytes));
    unsigned *coop_bar = (unsigned *)((char *)tab + align_up(sizeof(idg::CubeParams) * (size_t)batch));
    unsigned long long *mail = (unsigned long long *)((char *)coop_bar + kAlign);
    const size_t mail_bytes = resident_shape(nx, N) ? idg::kResidentMailBytes : 0;

    // Plan: kernel variant and iterations fused per launch.
    const bool can_tile = idg::tiled_supported(nx, ny, nz, cubes, out, scratch);
    const bool can_tma = idg::tma_supported(nx, ny, nz, cubes, out, scratch);
    int kernel = g_opt[IDG_OPT_KERNEL];
    int fuse = g_opt[IDG_OPT_FUSE];
    int tile = g_opt[IDG_OPT_TILE];
    // nx % 4 != 0: kernel 3 on the library's pitched copies in the workspace (intensity-driven filter only)
    const bool pitched_ok = mode == 0 && idg::tma_pitched_supported(nx, ny, nz);
    bool pitched = false;
    // Small cubes and interactive batches: everything on chip for the whole call (profiles/r2a_notes.md).
    idg::ResidentPlan rplan;
    const bool can_resident = mail_bytes > 0 && max_n > 0 && (kernel == 0 || kernel == 5) &&
                              idg::resident_plan(nx, ny, nz, batch, max_n, mail_bytes, idg::device_sm_count(), &rplan);
    if (kernel == 5 && !can_resident) kernel = 0;
    // Measured (profiles/r2a_notes.md): faster than kernel 3 when the whole call fits on chip at once (one wave) AND the
    // blocks are small enough for the kernel's small-block path (up to ~1.3 Mvoxel: 30 against 40 us on 100 x 100 x 67,
    // 37 against 43 on 128 x 128 x 64); with larger blocks kernel 3 at T = 4 wins by 6-25 % (160 x 160 x 64 .. 256 x 256 x 40).
    if (kernel == 0 && can_resident && fuse == 0 && rplan.cubes >= batch && rplan.small) kernel = 5;
    if (kernel == 0) {
        // Measured on B200 (profiles/r1g_notes.md, r1h_notes.md): the z-chunked TMA kernel everywhere it applies.
        // Four fused iterations per launch (one 8-warp CTA per SM) move a quarter of the DRAM bytes of an un-fused
        // sweep and need the fewest launches; only when the GPU is full AND the cubes are thin in z do the 2 T
        // warm-up planes per z chunk and the taller halo cost more than that saves: then two iterations on two
        // CTAs per SM.  The tail of n_iter mod T iterations runs as one launch of the kernel built for that depth.
        // Cubes of at most 128 columns (the interactive batches) use the single-tile-column variant.
        const double work = (double)N * (double)batch;
        if (can_tma) {
            kernel = 3;
            // Small cubes: a round costs ~10 us (T = 3) to ~14 us (T = 4) whatever the cube, so three iterations per
            // round, all rounds in one cooperative launch, beat four per launch from five iterations on
            // (profiles/r1k_notes.md).
            if (!fuse && work <= kCoopMaxVoxels && g_opt[IDG_OPT_COOP] != 1 && max_n >= 5) fuse = 3;
            if (!fuse) fuse = (nz < 100 && work >= 4.0e6) ? 2 : 4;
        } else if (pitched_ok && (double)N * (double)batch >= 1.0e5) {
            kernel = 3;                        // on pitched copies (profiles/r2c_notes.md)
            pitched = true;
            if (!fuse) fuse = (nz < 100 && work >= 4.0e6) ? 2 : 4;
        } else {
            kernel = can_tile ? 2 : 1;
        }
    }
    if (g_opt[IDG_OPT_KERNEL] == 3 && !can_tma && pitched_ok) pitched = true;
    if (mode == 1 && kernel != 5) {          // gradient-driven variant: kernel 3 (any T) or the naive kernel
        const int ko = g_opt[IDG_OPT_KERNEL];
        fuse = g_opt[IDG_OPT_FUSE];
        if ((ko == 0 || ko == 3 || ko == 4) && can_tma) {
            kernel = 3;
            if (!fuse) fuse = (nz < 100 && (double)N * (double)batch >= 4.0e6) ? 2 : 4;
        } else {
            kernel = 1;
        }
    }
    if (kernel == 4) kernel = can_tma ? 3 : 2;      // kernel 4 (persistent warp-decoupled variant) was retired in 1.1
    if (kernel == 3 && !can_tma && !pitched) kernel = 2;
    if (kernel != 3) pitched = false;
    if (kernel == 2 && !can_tile) kernel = 1;
    if (kernel == 5) {
        fuse = max_n;
    } else if (kernel >= 2) {
        if (!fuse) fuse = 2;
        if (fuse > max_n && max_n > 0) fuse = max_n;
    } else {
        fuse = 1;
    }
    {
        static const char *const names[6] = {"", "idg_naive_kernel", "idg_tiled_kernel", "idg_tma_kernel",
                                             "", "idg_resident_kernel"};
        snprintf(t_plan, sizeof(t_plan), "%s%s%s fuse=%d tile=%d", names[kernel], mode == 1 ? " pm" : "",
                 pitched ? " pitched" : "", fuse, tile);
    }

    std::vector<idg::CubeParams> host_tab((size_t)batch);
    bool any_zero = false, all_zero = true;
    for (int b = 0; b < batch; ++b) {
        const int n = n_iter ? n_iter[b] : n_iter_all;
        host_tab[(size_t)b] = prepare(params[b], n);
        any_zero |= (n == 0);
        all_zero &= (n == 0);
    }
    cudaError_t e;
    if (any_zero && !in_place) {     // n = 0: I_n = I_0
        if (all_zero) {
            e = cudaMemcpyAsync(out, cubes, bytes, cudaMemcpyDeviceToDevice, st);
            if (e != cudaSuccess) return (int)e;
        } else {
            for (int b = 0; b < batch; ++b)
                if (host_tab[(size_t)b].n_iter == 0) {
                    e = cudaMemcpyAsync(out + (size_t)b * N, cubes + (size_t)b * N, N * sizeof(float),
                                        cudaMemcpyDeviceToDevice, st);
                    if (e != cudaSuccess) return (int)e;
                }
        }
    }
    if (max_n == 0) return IDG_OK;

    idg::Launch L;
    memset(&L, 0, sizeof(L));
    L.in = cubes;
    L.out = out;
    L.scratch = scratch;
    L.nx = nx; L.ny = ny; L.nz = nz; L.batch = batch;
    L.fuse = fuse;
    L.in_place = in_place ? 1 : 0;
    L.mode = mode;
    if (batch == 1) {
        L.tab = nullptr;
        L.one = host_tab[0];
    } else {
        // pageable source: the runtime stages it before returning, so host_tab may die after the call
        e = cudaMemcpyAsync(tab, host_tab.data(), sizeof(idg::CubeParams) * (size_t)batch,
                            cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return (int)e;
        L.tab = tab;
    }
    if (kernel == 5) {  // one cooperative launch per wave of cubes; reads `cubes` once, writes `out` once (in place is safe)
        int launches = 0;
        e = idg::launch_resident(L, rplan, mail, st, &launches);
        if (e == cudaSuccess) {
            t_launches = launches;
            snprintf(t_plan, sizeof(t_plan), "idg_resident_kernel%s blocks=%dx%d of %dx%dx%d waves=%d", mode == 1 ? " pm" : "",
                     rplan.ty, rplan.tz, nx, rplan.by, rplan.bz, launches);
            return IDG_OK;
        }
        return (int)e;
    }
    if (pitched) {      // dense -> pitched input copy; the launches ping-pong between the other two pitched buffers
        const int pitch = (nx + 3) / 4 * 4;
        float *p0 = scratch, *p1 = (float *)((char *)scratch + pbytes), *p2 = (float *)((char *)scratch + 2 * pbytes);
        e = idg::launch_repitch(cubes, nx, p0, pitch, nullptr, nullptr, nx, ny, nz, batch, st);
        if (e != cudaSuccess) return (int)e;
        ++t_launches;
        L.in = p0;
        L.out = p1;
        L.scratch = p2;
        L.pitch = pitch;
        L.in_place = 0;
    } else if (in_place) {     // stage I_0 so a cube whose first launch targets `out` does not read what it writes
        e = cudaMemcpyAsync(scratch, cubes, bytes, cudaMemcpyDeviceToDevice, st);
        if (e != cudaSuccess) return (int)e;
    }
    // Small cubes (launch latency and prologue dominate a launch): all rounds in ONE cooperative launch if the whole
    // grid is co-resident.  Measured on B200 (profiles/r1k_notes.md).
    const int rounds = (max_n + fuse - 1) / fuse;
    const int coop = g_opt[IDG_OPT_COOP];
    if (kernel == 3 && mode == 0 && !pitched && rounds >= 2 && coop != 1 &&
        (coop == 2 || (double)N * (double)batch <= kCoopMaxVoxels)) {
        e = cudaMemsetAsync(coop_bar, 0, 8, st);
        if (e != cudaSuccess) return (int)e;
        L.iter_done = 0;
        e = idg::launch_tma_coop(L, g_opt[IDG_OPT_ZCHUNK], tile, rounds, coop_bar, st);
        if (e == cudaSuccess) {
            t_launches = 1;
            snprintf(t_plan, sizeof(t_plan), "idg_tma_coop_kernel fuse=%d rounds=%d", fuse, rounds);
            return IDG_OK;
        }
        if (e != cudaErrorNotSupported && e != cudaErrorCooperativeLaunchTooLarge) return (int)e;
        (void)cudaGetLastError();           // does not fit: one launch per round
    }
    for (int done = 0; done < max_n; done += fuse) {
        L.iter_done = done;
        int tile_now = tile;
        if (kernel == 3) {
            // the last launch applies the remaining r < fuse iterations: give it the kernel built for depth r
            // (route() sees remaining <= r for every cube, so it is that cube's last launch either way)
            const int rem = max_n - done;
            L.fuse = rem < fuse ? rem : fuse;
            if (tile_now == 0) tile_now = L.fuse <= 2 ? 2 : (L.fuse == 3 ? 3 : 1);
            else if (L.fuse <= 2 && tile_now > 2) tile_now = 0;
        }
        e = (kernel == 3)   ? idg::launch_tma(L, g_opt[IDG_OPT_ZCHUNK], tile_now, st)
            : (kernel == 2) ? idg::launch_tiled(L, g_opt[IDG_OPT_ZCHUNK], st)
                            : idg::launch_naive(L, st);
        if (e != cudaSuccess) return (int)e;
        ++t_launches;
    }
    if (pitched) {      // pitched result -> the caller's dense cubes (cubes with n_iter = 0: their input copy)
        e = idg::launch_repitch(L.out, L.pitch, out, nx, L.in, L.tab, nx, ny, nz, batch, st);
        if (e != cudaSuccess) return (int)e;
        ++t_launches;
    }
    return IDG_OK;
}

}  // namespace

extern "C" {

int idg_version(void) { return IDG_VERSION; }

const char *idg_status_string(int status)
{
    switch (status) {
    case IDG_OK: return "ok";
    case IDG_ERR_NULL: return "a required pointer is NULL";
    case IDG_ERR_DIMS: return "invalid cube dimensions or batch";
    case IDG_ERR_NITER: return "negative iteration count";
    case IDG_ERR_PARAM: return "invalid filter parameters";
    case IDG_ERR_WORKSPACE: return "workspace missing, too small or misaligned";
    case IDG_ERR_OVERLAP: return "buffers overlap";
    case IDG_ERR_OPTION: return "unknown option or value out of range";
    case IDG_ERR_STATIC_LIMIT: return "kernel larger than the static scratch array of idg_gaussian_filter_static (radius > 9)";
    default: return status > 0 ? cudaGetErrorString((cudaError_t)status) : "unknown status";
    }
}

unsigned idg_params_check(const idg_params *p)
{
    if (!p || !params_valid(*p)) return 4u;
    unsigned m = 0;
    if (p->tau < 0.0025f || p->tau > 0.0625f) m |= 1u;
    if (p->cx > 10.0f || p->cy > 10.0f || p->cz > 10.0f) m |= 1u;
    if (p->K < 0.5f || p->K > 10.0f) m |= 1u;
    if ((double)p->tau * ((double)p->cx + (double)p->cy + (double)p->cz) > 0.5) m |= 2u;
    return m;
}

size_t idg_workspace_bytes(int nx, int ny, int nz, int batch)
{
    size_t N;
    if (!voxel_count(nx, ny, nz, batch, &N)) return 0;
    // nx % 4 != 0: three pitched copies of the batch (input, and the two ping-pong buffers) instead of one scratch
    const size_t cubes = nx % 4 ? 3 * pitched_bytes(nx, ny, nz, batch) : N * (size_t)batch * sizeof(float);
    return align_up(cubes) + align_up(sizeof(idg::CubeParams) * (size_t)batch) +
           kAlign +     // scratch cubes | per-cube constants | arrival counter of the cooperative launch
           (resident_shape(nx, N) ? idg::kResidentMailBytes : 0);      // | mailboxes of the resident kernel
}

int idg_filter_ws(const float *cube, int nx, int ny, int nz, int n_iter, const idg_params *params,
                  float *out, void *workspace, size_t workspace_bytes, void *stream)
{
    return run(cube, nx, ny, nz, 1, nullptr, n_iter, params, out, workspace, workspace_bytes,
               (cudaStream_t)stream);
}

int idg_filter_pm(const float *cube, int nx, int ny, int nz, int n_iter, const idg_params *params,
                  float *out, void *workspace, size_t workspace_bytes, void *stream)
{
    return run(cube, nx, ny, nz, 1, nullptr, n_iter, params, out, workspace, workspace_bytes,
               (cudaStream_t)stream, 1);
}

int idg_filter_batched(const float *cubes, int nx, int ny, int nz, int batch, const int *n_iter,
                       int n_iter_all, const idg_params *params, float *out, void *workspace,
                       size_t workspace_bytes, void *stream)
{
    return run(cubes, nx, ny, nz, batch, n_iter, n_iter_all, params, out, workspace, workspace_bytes,
               (cudaStream_t)stream);
}

int idg_filter_pm_batched(const float *cubes, int nx, int ny, int nz, int batch, const int *n_iter,
                          int n_iter_all, const idg_params *params, float *out, void *workspace,
                          size_t workspace_bytes, void *stream)
{
    return run(cubes, nx, ny, nz, batch, n_iter, n_iter_all, params, out, workspace, workspace_bytes,
               (cudaStream_t)stream, 1);
}

int idg_filter(const float *cube, int nx, int ny, int nz, int n_iter, const idg_params *params,
               float *out, void *stream)
{
    const size_t need = idg_workspace_bytes(nx, ny, nz, 1);
    if (need == 0) return IDG_ERR_DIMS;
    if (!cube || !out || !params) return IDG_ERR_NULL;
    if (n_iter < 0) return IDG_ERR_NITER;
    if (!params_valid(*params)) return IDG_ERR_PARAM;
    cudaStream_t st = (cudaStream_t)stream;
    void *ws = nullptr;
    cudaError_t e = idg::temp_alloc(&ws, need, st);
    if (e != cudaSuccess) return (int)e;
    const int rc = run(cube, nx, ny, nz, 1, nullptr, n_iter, params, out, ws, need, st);
    e = cudaFreeAsync(ws, st);
    if (rc != IDG_OK) return rc;
    return e == cudaSuccess ? IDG_OK : (int)e;
}

constexpr int kMaxSlabs = 16;      // z slabs of the idg_filter_host pipeline

// Streams and events of one idg_filter_host call (destroyed when the call returns; the destructor runs after the
// call has synchronised both copy streams).
struct SlabSync {
    cudaStream_t h2d = nullptr, d2h = nullptr;
    cudaEvent_t ev_h[kMaxSlabs] = {}, ev_c[kMaxSlabs] = {}, ev_d[kMaxSlabs] = {}, begin = nullptr;
    cudaError_t create(int slabs)
    {
        cudaError_t e = cudaStreamCreateWithFlags(&h2d, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&d2h, cudaStreamNonBlocking);
        for (int i = 0; i < slabs && i < kMaxSlabs && e == cudaSuccess; ++i) {
            e = cudaEventCreateWithFlags(&ev_h[i], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ev_c[i], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ev_d[i], cudaEventDisableTiming);
        }
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&begin, cudaEventDisableTiming);
        return e;
    }
    ~SlabSync()
    {
        for (int i = 0; i < kMaxSlabs; ++i) {
            if (ev_h[i]) cudaEventDestroy(ev_h[i]);
            if (ev_c[i]) cudaEventDestroy(ev_c[i]);
            if (ev_d[i]) cudaEventDestroy(ev_d[i]);
        }
        if (begin) cudaEventDestroy(begin);
        if (h2d) cudaStreamDestroy(h2d);
        if (d2h) cudaStreamDestroy(d2h);
    }
};

int idg_filter_host(const float *cube_host, int nx, int ny, int nz, int n_iter,
                    const idg_params *params, float *out_host, void *dev_buffers,
                    size_t dev_buffers_bytes, void *stream)
{
    const size_t ws_bytes = idg_workspace_bytes(nx, ny, nz, 1);
    if (ws_bytes == 0) return IDG_ERR_DIMS;
    if (!cube_host || !out_host || !params) return IDG_ERR_NULL;
    if (n_iter < 0) return IDG_ERR_NITER;
    if (!params_valid(*params)) return IDG_ERR_PARAM;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = (size_t)nx * ny * nz * sizeof(float);
    const size_t cube_al = align_up(bytes);
    const size_t need = 2 * cube_al + ws_bytes;
    char *base = (char *)dev_buffers;
    bool own = false;
    cudaError_t e;
    if (base) {
        if (dev_buffers_bytes < need || ((uintptr_t)base % kAlign) != 0) return IDG_ERR_WORKSPACE;
    } else {
        e = idg::temp_alloc((void **)&base, need, st);
        if (e != cudaSuccess) return (int)e;
        own = true;
    }
    float *d_in = (float *)base, *d_out = (float *)(base + cube_al);
    void *ws = base + 2 * cube_al;
    int rc = IDG_OK;
    e = cudaSuccess;

    // Slab pipeline: the paper's T_p includes the transfers, and on a PCIe link they
    // dominate.  The cube is cut into z slabs; slab s is filtered on planes [z0-n, z1+n) (an error made
    // at an artificial slab face travels one plane per iteration, so after n iterations planes [z0, z1)
    // are exact: domain of dependence, pinned by P8) while slab s+1 is still arriving and slab s-1 is
    // leaving, on two internal copy streams.  Results are bit-identical to the one-piece path.
    int slabs = g_opt[IDG_OPT_HOST_SLABS];
    if (slabs == 0) {
        slabs = 1;
        if (bytes >= (64u << 20) && n_iter > 0) {
            // thin slabs shorten the pipeline's tail (the last slab's filtering and download); their 2 n halo planes
            // are recomputed, which the GPU has time for: it idles on the PCIe link
            const int thick = 3 * n_iter / 2 > 16 ? 3 * n_iter / 2 : 16;
            slabs = nz / thick;
            if (slabs > kMaxSlabs) slabs = kMaxSlabs;
            if (slabs < 1) slabs = 1;
        }
    }
    if (slabs > kMaxSlabs) slabs = kMaxSlabs;
    if (slabs > nz) slabs = nz;
    const size_t plane_b = (size_t)nx * ny * sizeof(float);
    // Slab boundaries.  Nothing can be downloaded before the first slab and its halo have been uploaded and filtered, and
    // that lag adds to the total download time: the first slab is a quarter as thick as the others (from 4 slabs on;
    // measured 0.91 of the copy-only floor against 0.89-0.90 with equal slabs; a thin last slab as well gave nothing).
    int zb[kMaxSlabs + 1];
    {
        const int zs_u = (nz + slabs - 1) / slabs;
        const int first = slabs >= 4 ? (zs_u / 4 > 1 ? zs_u / 4 : 1) : zs_u;
        zb[0] = 0;
        for (int i = 1; i <= slabs; ++i) {
            long long z = slabs >= 4 ? first + ((long long)(nz - first) * (i - 1) + (slabs - 2)) / (slabs - 1)
                                     : (long long)i * zs_u;
            zb[i] = z < nz ? (int)z : nz;
        }
        zb[slabs] = nz;
    }
    int zs = 1;
    for (int i = 0; i < slabs; ++i)
        if (zb[i + 1] - zb[i] > zs) zs = zb[i + 1] - zb[i];                  // the thickest slab
    const int max_planes = zs + 2 * n_iter < nz ? zs + 2 * n_iter : nz;
    const size_t slab_al = align_up((size_t)max_planes * plane_b);
    const size_t slab_ws = idg_workspace_bytes(nx, ny, max_planes, 1);
    if (slabs > 1 && n_iter > 0 && 2 * slab_al + slab_ws <= need - cube_al) {
        // two copy streams and the per-slab events of THIS call on the CURRENT device (nothing shared between
        // callers, host threads or devices); created per call: a call that gets here moves >= 64 MB each way
        SlabSync sync;
        e = sync.create(slabs);
        cudaStream_t s_h2d = sync.h2d, s_d2h = sync.d2h;
        cudaEvent_t *ev_h = sync.ev_h, *ev_c = sync.ev_c, *ev_d = sync.ev_d, ev_begin = sync.begin;
        char *region = base + cube_al;
        float *d_slab[2] = {(float *)region, (float *)(region + slab_al)};
        void *ws_slab = region + 2 * slab_al;
        int launches = 0, copied = 0;                                   // planes of I_0 already requested
        if (e == cudaSuccess) e = cudaEventRecord(ev_begin, st);         // earlier work on `st` may own the buffers
        if (e == cudaSuccess) e = cudaStreamWaitEvent(s_h2d, ev_begin, 0);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(s_d2h, ev_begin, 0);
        for (int sl = 0; sl < slabs && e == cudaSuccess && rc == IDG_OK; ++sl) {
            const int z0 = zb[sl], z1 = zb[sl + 1];
            if (z0 >= z1) continue;
            const int lo = z0 - n_iter > 0 ? z0 - n_iter : 0, hi = z1 + n_iter < nz ? z1 + n_iter : nz;
            if (hi > copied) {
                e = cudaMemcpyAsync((char *)d_in + (size_t)copied * plane_b, (const char *)cube_host + (size_t)copied * plane_b,
                                    (size_t)(hi - copied) * plane_b, cudaMemcpyHostToDevice, s_h2d);
                copied = hi;
            }
            if (e == cudaSuccess) e = cudaEventRecord(ev_h[sl], s_h2d);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(st, ev_h[sl], 0);
            if (e == cudaSuccess && sl >= 2) e = cudaStreamWaitEvent(st, ev_d[sl - 2], 0);     // its output buffer is free
            if (e != cudaSuccess) break;
            float *d_o = d_slab[sl & 1];
            rc = run(d_in + (size_t)lo * nx * ny, nx, ny, hi - lo, 1, nullptr, n_iter, params, d_o, ws_slab, slab_ws, st);
            launches += t_launches;
            if (rc != IDG_OK) break;
            e = cudaEventRecord(ev_c[sl], st);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(s_d2h, ev_c[sl], 0);
            if (e == cudaSuccess)
                e = cudaMemcpyAsync((char *)out_host + (size_t)z0 * plane_b, (const char *)d_o + (size_t)(z0 - lo) * plane_b,
                                    (size_t)(z1 - z0) * plane_b, cudaMemcpyDeviceToHost, s_d2h);
            if (e == cudaSuccess) e = cudaEventRecord(ev_d[sl], s_d2h);
            if (e == cudaSuccess && sl == slabs - 1) e = cudaStreamWaitEvent(st, ev_d[sl], 0);  // `st` ends after the last copy
        }
        t_launches = launches;
        cudaStreamSynchronize(s_h2d);          // on an error path the copies must not outlive the buffers
        cudaStreamSynchronize(s_d2h);
    } else {
        e = cudaMemcpyAsync(d_in, cube_host, bytes, cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) {
            rc = run(d_in, nx, ny, nz, 1, nullptr, n_iter, params, d_out, ws, ws_bytes, st);
            if (rc == IDG_OK) e = cudaMemcpyAsync(out_host, d_out, bytes, cudaMemcpyDeviceToHost, st);
        }
    }
    if (own) {
        cudaError_t e2 = cudaFreeAsync(base, st);
        if (e == cudaSuccess) e = e2;
    }
    cudaError_t e3 = cudaStreamSynchronize(st);
    if (rc != IDG_OK) return rc;
    if (e != cudaSuccess) return (int)e;
    return e3 == cudaSuccess ? IDG_OK : (int)e3;
}

// ---- reference filters (PAPER.md sections 3.1-3.2) -------------------------------------------

static int ref_args(const float *cube, int nx, int ny, int nz, const float *out, size_t *N)
{
    if (!cube || !out) return IDG_ERR_NULL;
    if (!voxel_count(nx, ny, nz, 1, N)) return IDG_ERR_DIMS;
    if (ranges_overlap(cube, *N * sizeof(float), out, *N * sizeof(float))) return IDG_ERR_OVERLAP;
    return IDG_OK;
}

// Separable filter: the TMA-fed kernel where it applies (radii <= 4, nx % 4 == 0, 16-byte aligned; option kernel = 1
// forces the general kernel), else idg_sep3d_kernel.  Returns the kernel name through `name`.
static cudaError_t run_sep3d(const float *cube, float *out, int nx, int ny, int nz, const int r[3], const float *wx,
                             const float *wy, const float *wz, cudaStream_t st, const char **name)
{
    *name = "idg_sep3d_kernel";
    if (g_opt[IDG_OPT_KERNEL] != 1 && idg::sep3d_tma_supported(nx, ny, nz, r[0], r[1], r[2], cube, out)) {
        const cudaError_t e = idg::launch_sep3d_tma(cube, out, nx, ny, nz, r[0], r[1], r[2], wx, wy, wz,
                                                    g_opt[IDG_OPT_ZCHUNK], g_opt[IDG_OPT_TILE], st);
        if (e != cudaErrorNotSupported) {
            *name = "idg_sep3d_tma_kernel";
            return e;
        }
    }
    if (g_opt[IDG_OPT_KERNEL] != 1 && idg::sep3d_big_supported(nx, ny, nz, r[0], r[1], r[2], cube, out)) {
        const cudaError_t e = idg::launch_sep3d_big(cube, out, nx, ny, nz, r[0], r[1], r[2], wx, wy, wz,
                                                    g_opt[IDG_OPT_ZCHUNK], g_opt[IDG_OPT_TILE], st);
        if (e != cudaErrorNotSupported) {
            *name = "idg_sep3d_big_kernel";
            return e;
        }
    }
    return idg::launch_sep3d(cube, out, nx, ny, nz, r[0], r[1], r[2], wx, wy, wz, st);
}

int idg_box_filter(const float *cube, int nx, int ny, int nz, int wx, int wy, int wz, float *out, void *stream)
{
    t_launches = 0;
    size_t N;
    const int rc = ref_args(cube, nx, ny, nz, out, &N);
    if (rc != IDG_OK) return rc;
    const int w[3] = {wx, wy, wz};
    float wt[3][2 * idg::kSepMaxRadius + 1];
    for (int a = 0; a < 3; ++a) {
        if (w[a] < 1 || !(w[a] & 1) || w[a] > 2 * idg::kSepMaxRadius + 1) return IDG_ERR_PARAM;
        for (int i = 0; i < w[a]; ++i) wt[a][i] = (float)(1.0 / (double)w[a]);     // PAPER.md:123, the mean
    }
    const int r[3] = {wx / 2, wy / 2, wz / 2};
    const char *name;
    const cudaError_t e = run_sep3d(cube, out, nx, ny, nz, r, wt[0], wt[1], wt[2], (cudaStream_t)stream, &name);
    if (e != cudaSuccess) return (int)e;
    t_launches = 1;
    snprintf(t_plan, sizeof(t_plan), "%s box %dx%dx%d", name, wx, wy, wz);
    return IDG_OK;
}

// Eq. 2 and reading F3: sigma and support radius of one axis.
static double sigma_of(double fwhm) { return fwhm / (2.0 * sqrt(2.0 * log(2.0))); }
static int radius_of(double sigma) { return (int)floor(3.0 * sigma + 0.5); }

int idg_gaussian_radii(float fwhm_x, float fwhm_y, float fwhm_z, float theta_x, float theta_y, float theta_z,
                       int radii[3])
{
    if (!radii) return IDG_ERR_NULL;
    const double f[3] = {fwhm_x, fwhm_y, fwhm_z}, th[3] = {theta_x, theta_y, theta_z};
    for (int a = 0; a < 3; ++a)
        if (!(f[a] >= 0.0) || !isfinite(f[a]) || !isfinite(th[a])) return IDG_ERR_PARAM;
    const bool rotated = th[0] != 0.0 || th[1] != 0.0 || th[2] != 0.0;
    if (rotated) {
        double smax = 0.0;
        for (int a = 0; a < 3; ++a) {
            if (!(f[a] > 0.0)) return IDG_ERR_PARAM;                         // reading F5
            smax = fmax(smax, sigma_of(f[a]));
        }
        radii[0] = radii[1] = radii[2] = radius_of(smax);
        if (radii[0] > idg::kConvMaxRadius) return IDG_ERR_PARAM;
    } else {
        for (int a = 0; a < 3; ++a) {
            radii[a] = radius_of(sigma_of(f[a]));
            if (radii[a] > idg::kSepMaxRadius) return IDG_ERR_PARAM;
        }
    }
    return IDG_OK;
}

int idg_gaussian_filter(const float *cube, int nx, int ny, int nz, float fwhm_x, float fwhm_y, float fwhm_z,
                        float theta_x, float theta_y, float theta_z, float *out, void *stream)
{
    t_launches = 0;
    size_t N;
    int rc = ref_args(cube, nx, ny, nz, out, &N);
    if (rc != IDG_OK) return rc;
    int r[3];
    rc = idg_gaussian_radii(fwhm_x, fwhm_y, fwhm_z, theta_x, theta_y, theta_z, r);
    if (rc != IDG_OK) return rc;
    const double f[3] = {fwhm_x, fwhm_y, fwhm_z}, th[3] = {theta_x, theta_y, theta_z};
    cudaStream_t st = (cudaStream_t)stream;
    const bool rotated = th[0] != 0.0 || th[1] != 0.0 || th[2] != 0.0;
    if (!rotated) {
        // Eq. 1 factorises along the axes: three 1-D kernels, each normalised to unit sum (reading F2)
        float wt[3][2 * idg::kSepMaxRadius + 1];
        for (int a = 0; a < 3; ++a) {
            const double s = sigma_of(f[a]);
            double g[2 * idg::kSepMaxRadius + 1], sum = 0.0;
            for (int i = -r[a]; i <= r[a]; ++i) {
                g[i + r[a]] = s > 0.0 ? exp(-(double)(i * i) / (2.0 * s * s)) : 1.0;
                sum += g[i + r[a]];
            }
            for (int i = 0; i <= 2 * r[a]; ++i) wt[a][i] = (float)(g[i] / sum);
        }
        const char *name;
        const cudaError_t e = run_sep3d(cube, out, nx, ny, nz, r, wt[0], wt[1], wt[2], st, &name);
        if (e != cudaSuccess) return (int)e;
        t_launches = 1;
        snprintf(t_plan, sizeof(t_plan), "%s gauss r=%d,%d,%d", name, r[0], r[1], r[2]);
        return IDG_OK;
    }
    // Eq. 3: K(p) = G(R^-1 p), R = Rz Ry Rx (right-handed, degrees), sampled on the cube |p_j| <= r
    const double d2r = acos(-1.0) / 180.0;
    const double cx = cos(th[0] * d2r), sx = sin(th[0] * d2r), cy = cos(th[1] * d2r), sy = sin(th[1] * d2r),
                 cz = cos(th[2] * d2r), sz = sin(th[2] * d2r);
    const double R[3][3] = {{cz * cy, cz * sy * sx - sz * cx, cz * sy * cx + sz * sx},
                            {sz * cy, sz * sy * sx + cz * cx, sz * sy * cx - cz * sx},
                            {-sy, cy * sx, cy * cx}};
    double i2[3];
    for (int a = 0; a < 3; ++a) i2[a] = 1.0 / (2.0 * sigma_of(f[a]) * sigma_of(f[a]));
    const int rr = r[0], W = 2 * rr + 1;
    std::vector<double> g((size_t)W * W * W);
    double sum = 0.0;
    size_t m = 0;
    for (int k = -rr; k <= rr; ++k)
        for (int j = -rr; j <= rr; ++j)
            for (int i = -rr; i <= rr; ++i) {
                double q2 = 0.0;
                for (int a = 0; a < 3; ++a) {
                    const double q = R[0][a] * i + R[1][a] * j + R[2][a] * k;      // (R^T p)_a
                    q2 += q * q * i2[a];
                }
                g[m] = exp(-q2);
                sum += g[m++];
            }
    std::vector<float> gf(g.size());
    for (size_t t = 0; t < g.size(); ++t) gf[t] = (float)(g[t] / sum);
    float *d_k = nullptr;
    cudaError_t e = idg::temp_alloc((void **)&d_k, gf.size() * sizeof(float), st);
    if (e != cudaSuccess) return (int)e;
    e = cudaMemcpyAsync(d_k, gf.data(), gf.size() * sizeof(float), cudaMemcpyHostToDevice, st);   // pageable: staged before return
    if (e == cudaSuccess) e = idg::launch_conv3d(cube, out, nx, ny, nz, rr, d_k, st);
    const cudaError_t e2 = cudaFreeAsync(d_k, st);
    if (e != cudaSuccess) return (int)e;
    if (e2 != cudaSuccess) return (int)e2;
    t_launches = 1;
    snprintf(t_plan, sizeof(t_plan), "idg_conv3d_kernel<r=%d>", rr);
    return IDG_OK;
}

// ---- quality diagnostics (section 4-5, Eq. 12-18) ------------------------------------

static int roi_box(const idg_roi *roi, int nx, int ny, int nz, int r[6])
{
    if (!roi) { r[0] = 0; r[1] = nx; r[2] = 0; r[3] = ny; r[4] = 0; r[5] = nz; return IDG_OK; }
    r[0] = roi->x0; r[1] = roi->x1; r[2] = roi->y0; r[3] = roi->y1; r[4] = roi->z0; r[5] = roi->z1;
    if (r[0] < 0 || r[0] > r[1] || r[1] > nx || r[2] < 0 || r[2] > r[3] || r[3] > ny || r[4] < 0 || r[4] > r[5] ||
        r[5] > nz)
        return IDG_ERR_DIMS;
    return IDG_OK;
}

int idg_mask_sums(const float *orig, const float *filt, const float *model, int nx, int ny, int nz,
                  const idg_roi *roi, float thr_o, float thr_f, double *sums, void *stream)
{
    t_launches = 0;
    if (!orig || !filt || !sums) return IDG_ERR_NULL;
    size_t N;
    if (!voxel_count(nx, ny, nz, 1, &N)) return IDG_ERR_DIMS;
    if (isnan(thr_o) || isnan(thr_f)) return IDG_ERR_PARAM;
    if (((uintptr_t)sums & 7u) != 0) return IDG_ERR_WORKSPACE;
    int r[6];
    const int rc = roi_box(roi, nx, ny, nz, r);
    if (rc != IDG_OK) return rc;
    const cudaError_t e = idg::launch_mask_sums(orig, filt, model, nx, ny, r, thr_o, thr_f, sums, (cudaStream_t)stream);
    if (e != cudaSuccess) return (int)e;
    t_launches = 1;
    snprintf(t_plan, sizeof(t_plan), "idg_mask_sums_kernel<model=%d>", model ? 1 : 0);
    return IDG_OK;
}

int idg_cube_stats(const float *cube, int nx, int ny, int nz, const idg_roi *roi, double *stats, void *stream)
{
    t_launches = 0;
    if (!cube || !stats) return IDG_ERR_NULL;
    size_t N;
    if (!voxel_count(nx, ny, nz, 1, &N)) return IDG_ERR_DIMS;
    if (((uintptr_t)stats & 7u) != 0) return IDG_ERR_WORKSPACE;
    int r[6];
    const int rc = roi_box(roi, nx, ny, nz, r);
    if (rc != IDG_OK) return rc;
    const cudaError_t e = idg::launch_cube_stats(cube, nx, ny, r, stats, (cudaStream_t)stream);
    if (e != cudaSuccess) return (int)e;
    t_launches = 1;
    snprintf(t_plan, sizeof(t_plan), "idg_cube_stats_kernel");
    return IDG_OK;
}

int idg_stats_rms(const double *stats, double *mean, double *rms)
{
    if (!stats) return IDG_ERR_NULL;
    const double n = stats[0], m = n > 0.0 ? stats[1] / n : NAN;
    if (mean) *mean = m;
    if (rms) *rms = n > 0.0 ? sqrt(fmax(stats[2] / n - m * m, 0.0)) : NAN;
    return IDG_OK;
}

int idg_histogram(const float *cube, int nx, int ny, int nz, const idg_roi *roi, float lo, float hi, int nbins,
                  const float *mask_thr, unsigned long long *counts, void *stream)
{
    t_launches = 0;
    if (!(hi > lo) || !isfinite(lo) || !isfinite(hi) || nbins < 1 || nbins > 8192 || (mask_thr && isnan(*mask_thr)))
        return IDG_ERR_PARAM;
    if (!cube || !counts) return IDG_ERR_NULL;
    size_t N;
    if (!voxel_count(nx, ny, nz, 1, &N)) return IDG_ERR_DIMS;
    if (((uintptr_t)counts & 7u) != 0) return IDG_ERR_WORKSPACE;
    int r[6];
    const int rc = roi_box(roi, nx, ny, nz, r);
    if (rc != IDG_OK) return rc;
    const cudaError_t e = idg::launch_histogram(cube, nx, ny, r, lo, hi, nbins, mask_thr, counts, (cudaStream_t)stream);
    if (e != cudaSuccess) return (int)e;
    t_launches = 1;
    snprintf(t_plan, sizeof(t_plan), "idg_histogram_kernel nbins=%d", nbins);
    return IDG_OK;
}

int idg_quality(const double *sums, double rms_o, double rms_f, double voxels_per_beam, double *F, double *sigma_F,
                double *F_M)
{
    if (!sums) return IDG_ERR_NULL;
    if (!(rms_o > 0.0) || !(rms_f > 0.0) || !(voxels_per_beam >= 1.0)) return IDG_ERR_PARAM;
    const double S_oo = sums[0], S_of = sums[1], N_o = sums[2], N_f = sums[3], S_mf = sums[4], S_m = sums[5];
    const double nan = NAN;
    if (F) *F = S_oo != 0.0 ? fabs(S_of) / fabs(S_oo) : nan;                                     // Eq. 12
    if (sigma_F) {
        const double sig_of = sqrt(N_f / voxels_per_beam) * rms_f, sig_oo = sqrt(N_o / voxels_per_beam) * rms_o;   // Eq. 16
        *sigma_F = S_oo != 0.0 ? sqrt(sig_of * sig_of / (S_oo * S_oo) +
                                      S_of * S_of * sig_oo * sig_oo / (S_oo * S_oo * S_oo * S_oo)) : nan;          // Eq. 15
    }
    if (F_M) *F_M = S_m != 0.0 ? fabs(S_mf) / fabs(S_m) : nan;                                   // Eq. 17
    return IDG_OK;
}

// ---- wavelet lifting (section 3.4, Eq. 8-11) ------------------------------------------

static int wavelet_args(const float *cube, int nx, int ny, int nz, int wavelet, int levels, const float *out, size_t *N)
{
    if (!cube || !out) return IDG_ERR_NULL;
    if (!voxel_count(nx, ny, nz, 1, N)) return IDG_ERR_DIMS;
    if ((wavelet != IDG_WAVELET_HAAR && wavelet != IDG_WAVELET_LEGALL53) || levels < 0 || levels > 16) return IDG_ERR_PARAM;
    if ((const float *)out != cube && ranges_overlap(cube, *N * sizeof(float), out, *N * sizeof(float)))
        return IDG_ERR_OVERLAP;
    return IDG_OK;
}

int idg_wavelet_transform(const float *cube, int nx, int ny, int nz, int wavelet, int levels, int inverse, float *out,
                          void *stream)
{
    t_launches = 0;
    size_t N;
    const int rc = wavelet_args(cube, nx, ny, nz, wavelet, levels, out, &N);
    if (rc != IDG_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = cudaSuccess;
    if ((const float *)out != cube) e = cudaMemcpyAsync(out, cube, N * sizeof(float), cudaMemcpyDeviceToDevice, st);
    int launches = 0;
    if (e == cudaSuccess) e = idg::launch_wavelet_transform(out, nx, ny, nz, wavelet, levels, inverse != 0, g_opt[IDG_OPT_KERNEL] == 1, st, &launches);
    if (e != cudaSuccess) return (int)e;
    t_launches = launches;
    snprintf(t_plan, sizeof(t_plan), "idg_lift_kernel %s levels=%d %s", wavelet == 0 ? "haar" : "legall53", levels,
             inverse ? "inverse" : "forward");
    return IDG_OK;
}

int idg_wavelet_filter(const float *cube, int nx, int ny, int nz, int wavelet, int levels, const float *thresholds,
                       float rms, float *out, void *stream)
{
    t_launches = 0;
    size_t N;
    const int rc = wavelet_args(cube, nx, ny, nz, wavelet, levels, out, &N);
    if (rc != IDG_OK) return rc;
    if (!thresholds) return IDG_ERR_NULL;
    if (levels < 1 || !(rms > 0.0f) || !isfinite(rms)) return IDG_ERR_PARAM;
    float thr[16];
    for (int l = 0; l < levels; ++l) {
        if (!(thresholds[l] >= 0.0f)) return IDG_ERR_PARAM;                 // also rejects NaN
        thr[l] = (float)((double)thresholds[l] * (double)rms);              // t_l in units of rms
    }
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = cudaSuccess;
    if (wavelet == IDG_WAVELET_HAAR && levels <= 3 && ny <= 65535 * 8 && nz <= 65535 * 8 &&
        g_opt[IDG_OPT_KERNEL] != 1) {          // Haar blocks are independent: one fused pass (option kernel = 1: per-axis
        bool warp = false;                     // passes, 2: the shared-memory regions also where a warp could hold a block)
        e = idg::launch_haar_filter(cube, out, nx, ny, nz, levels, thr, g_opt[IDG_OPT_KERNEL] != 2, &warp, st);
        if (e != cudaSuccess) return (int)e;
        t_launches = 1;
        snprintf(t_plan, sizeof(t_plan), "%s levels=%d", warp ? "idg_haar_warp_kernel" : "idg_haar_filter_kernel", levels);
        return IDG_OK;
    }
    int launches = 0;
    if (wavelet == IDG_WAVELET_LEGALL53 && g_opt[IDG_OPT_KERNEL] == 0) {
        // three axes of a level fused, out of place in a stream-ordered temporary (option kernel = 2: in-place
        // passes with whole lines in shared memory, 1: two-phase in-place passes)
        e = idg::launch_legall_filter(cube, out, nx, ny, nz, levels, thr, st, &launches);
        if (e == cudaSuccess) {
            t_launches = launches;
            snprintf(t_plan, sizeof(t_plan), "idg_legall_fwd_kernel/idg_legall_inv_kernel levels=%d", levels);
            return IDG_OK;
        }
        if (e != cudaErrorMemoryAllocation) return (int)e;
        e = cudaSuccess;                       // no room for the temporary: the in-place path needs none
        launches = 0;
    }
    if ((const float *)out != cube) e = cudaMemcpyAsync(out, cube, N * sizeof(float), cudaMemcpyDeviceToDevice, st);
    if (e == cudaSuccess) e = idg::launch_wavelet_transform(out, nx, ny, nz, wavelet, levels, false, g_opt[IDG_OPT_KERNEL] == 1, st, &launches);
    if (e == cudaSuccess) { e = idg::launch_wavelet_threshold(out, nx, ny, nz, levels, thr, st); ++launches; }
    if (e == cudaSuccess) e = idg::launch_wavelet_transform(out, nx, ny, nz, wavelet, levels, true, g_opt[IDG_OPT_KERNEL] == 1, st, &launches);
    if (e != cudaSuccess) return (int)e;
    t_launches = launches;
    snprintf(t_plan, sizeof(t_plan), "idg_lift_kernel %s levels=%d filter", wavelet == 0 ? "haar" : "legall53", levels);
    return IDG_OK;
}

int idg_set_option(int key, int value)
{
    if (key < 0 || key >= IDG_OPT_COUNT_) return IDG_ERR_OPTION;
    if (key == IDG_OPT_KERNEL && (value < 0 || value > 5)) return IDG_ERR_OPTION;
    if (key == IDG_OPT_FUSE && (value < 0 || value > 4)) return IDG_ERR_OPTION;
    if (key == IDG_OPT_ZCHUNK && value < 0) return IDG_ERR_OPTION;
    if (key == IDG_OPT_TILE && (value < 0 || value > 4)) return IDG_ERR_OPTION;
    if (key == IDG_OPT_CTAS && value < 0) return IDG_ERR_OPTION;
    if (key == IDG_OPT_HOST_SLABS && (value < 0 || value > kMaxSlabs)) return IDG_ERR_OPTION;
    if (key == IDG_OPT_COOP && (value < 0 || value > 2)) return IDG_ERR_OPTION;
    g_opt[key] = value;
    return IDG_OK;
}

int idg_get_option(int key)
{
    if (key < 0 || key >= IDG_OPT_COUNT_) return IDG_ERR_OPTION;
    return g_opt[key];
}

int idg_release_temporaries(void) { return (int)idg::temp_trim(); }

int idg_last_launch_count(void) { return t_launches; }

const char *idg_last_plan(void) { return t_plan; }

}  // extern "C"
