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

int g_opt[IDG_OPT_COUNT_] = {0, 0, 0, 0, 0};
thread_local int t_launches = 0;
thread_local char t_plan[96] = "none";

constexpr size_t kAlign = 256;
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
        cudaStream_t st)
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
    idg::CubeParams *tab = (idg::CubeParams *)((char *)workspace + align_up(bytes));

    // Plan: kernel variant and iterations fused per launch.
    const bool can_tile = idg::tiled_supported(nx, ny, nz, cubes, out, scratch);
    const bool can_tma = idg::tma_supported(nx, ny, nz, cubes, out, scratch);
    const bool can_stream = idg::stream_supported(nx, ny, nz, cubes, out, scratch);
    int kernel = g_opt[IDG_OPT_KERNEL];
    int fuse = g_opt[IDG_OPT_FUSE];
    int tile = g_opt[IDG_OPT_TILE];
    if (kernel == 0) {
        // Measured on B200 (profiles/): batches and cubes of at most 128 columns run best on the persistent
        // kernel (one tile column, no idle tail between cubes); large single cubes on the z-chunked TMA
        // kernel with two CTAs per SM; cubes too small to fill the GPU want few, deeply fused launches.
        const double work = (double)N * (double)batch;
        if (can_stream && (batch > 1 || nx <= 128) && work >= 4.0e6) {
            kernel = 4;
            if (!fuse) fuse = 2;
            if (!tile) tile = 2;
        } else if (can_tma) {
            kernel = 3;
            if (work >= 1.6e7) {
                if (!fuse) fuse = 2;
                if (!tile) tile = 2;
            } else if (!fuse) {
                fuse = 3;
            }
        } else {
            kernel = can_tile ? 2 : 1;
        }
    }
    if (kernel == 4 && !can_stream) kernel = 2;
    if (kernel == 3 && !can_tma) kernel = 2;
    if (kernel == 2 && !can_tile) kernel = 1;
    if (kernel >= 2) {
        if (!fuse) fuse = 2;
        if (fuse > max_n && max_n > 0) fuse = max_n;
    } else {
        fuse = 1;
    }
    if (kernel == 3 && tile > 2) tile = 0;
    if (kernel == 3 && fuse > 2 && tile == 2) tile = 1;
    {
        static const char *const names[5] = {"", "idg_naive_kernel", "idg_tiled_kernel", "idg_tma_kernel",
                                             "idg_stream_kernel"};
        snprintf(t_plan, sizeof(t_plan), "%s fuse=%d tile=%d", names[kernel], fuse, tile);
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
    if (in_place) {     // stage I_0 so a cube whose first launch targets `out` does not read what it writes
        e = cudaMemcpyAsync(scratch, cubes, bytes, cudaMemcpyDeviceToDevice, st);
        if (e != cudaSuccess) return (int)e;
    }
    for (int done = 0; done < max_n; done += fuse) {
        L.iter_done = done;
        e = (kernel == 4)   ? idg::launch_stream(L, g_opt[IDG_OPT_CTAS], tile, st)
            : (kernel == 3) ? idg::launch_tma(L, g_opt[IDG_OPT_ZCHUNK], tile, st)
            : (kernel == 2) ? idg::launch_tiled(L, g_opt[IDG_OPT_ZCHUNK], st)
                            : idg::launch_naive(L, st);
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
    return align_up(N * (size_t)batch * sizeof(float)) + align_up(sizeof(idg::CubeParams) * (size_t)batch);
}

int idg_filter_ws(const float *cube, int nx, int ny, int nz, int n_iter, const idg_params *params,
                  float *out, void *workspace, size_t workspace_bytes, void *stream)
{
    return run(cube, nx, ny, nz, 1, nullptr, n_iter, params, out, workspace, workspace_bytes,
               (cudaStream_t)stream);
}

int idg_filter_batched(const float *cubes, int nx, int ny, int nz, int batch, const int *n_iter,
                       int n_iter_all, const idg_params *params, float *out, void *workspace,
                       size_t workspace_bytes, void *stream)
{
    return run(cubes, nx, ny, nz, batch, n_iter, n_iter_all, params, out, workspace, workspace_bytes,
               (cudaStream_t)stream);
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
    cudaError_t e = cudaMallocAsync(&ws, need, st);
    if (e != cudaSuccess) return (int)e;
    const int rc = run(cube, nx, ny, nz, 1, nullptr, n_iter, params, out, ws, need, st);
    e = cudaFreeAsync(ws, st);
    if (rc != IDG_OK) return rc;
    return e == cudaSuccess ? IDG_OK : (int)e;
}

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
        e = cudaMallocAsync((void **)&base, need, st);
        if (e != cudaSuccess) return (int)e;
        own = true;
    }
    float *d_in = (float *)base, *d_out = (float *)(base + cube_al);
    void *ws = base + 2 * cube_al;
    int rc = IDG_OK;
    e = cudaMemcpyAsync(d_in, cube_host, bytes, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) {
        rc = run(d_in, nx, ny, nz, 1, nullptr, n_iter, params, d_out, ws, ws_bytes, st);
        if (rc == IDG_OK) e = cudaMemcpyAsync(out_host, d_out, bytes, cudaMemcpyDeviceToHost, st);
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

int idg_set_option(int key, int value)
{
    if (key < 0 || key >= IDG_OPT_COUNT_) return IDG_ERR_OPTION;
    if (key == IDG_OPT_KERNEL && (value < 0 || value > 4)) return IDG_ERR_OPTION;
    if (key == IDG_OPT_FUSE && (value < 0 || value > 4)) return IDG_ERR_OPTION;
    if (key == IDG_OPT_ZCHUNK && value < 0) return IDG_ERR_OPTION;
    if (key == IDG_OPT_TILE && (value < 0 || value > 4)) return IDG_ERR_OPTION;
    if (key == IDG_OPT_CTAS && value < 0) return IDG_ERR_OPTION;
    g_opt[key] = value;
    return IDG_OK;
}

int idg_get_option(int key)
{
    if (key < 0 || key >= IDG_OPT_COUNT_) return IDG_ERR_OPTION;
    return g_opt[key];
}

int idg_last_launch_count(void) { return t_launches; }

const char *idg_last_plan(void) { return t_plan; }

}  // extern "C"
