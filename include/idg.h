/*
 * idg.h -- C ABI of the B200-native intensity-driven gradient (IDG) filter.
 *
 * The operation is the adaptive filter of Punzo, van der Hulst & Roerdink,
 * arXiv:1609.03782, section 3.3: n explicit steps of
 *
 *   I_{i+1} = I_i + tau (Cx Dx I_i + Cy Dy I_i + Cz Dz I_i) / (1 + I_i^2/(K^2 rms^2))   (Eq. 7)
 *   Dx I    = [I(x+1,y,z) - I(x,y,z)] + [I(x-1,y,z) - I(x,y,z)]
 *
 * over a dense fp32 cube (RA x Dec x velocity).  The conductance (Eq. 6,
 * PAPER.md:178) is evaluated at the centre voxel of the current iterate; the
 * update is Jacobi (two buffers); an out-of-cube neighbour
 * equals the centre voxel (zero-flux boundary, reading R1); rms is a
 * caller-supplied constant.  All arithmetic runs in hand-written sm_100a CUDA
 * kernels; there is no CPU fallback.  The library also holds the paper's two reference filters
 * (box, Gaussian; sections 3.1-3.2), declared after the IDG entry points.
 *
 * Conventions for every entry point
 *   layout    dense, idx = x + nx*(y + ny*z); x = RA (fastest), y = Dec,
 *             z = velocity (slowest); batched cubes are contiguous, stride nx*ny*nz.
 *   pointers  marked [device] or [host].  All buffers are caller-owned; the
 *             library never frees or keeps them.  `cube` is read-only unless
 *             out == cube (in place is allowed); otherwise cube/out/workspace
 *             must not overlap.
 *   stream    a cudaStream_t passed as void* (NULL = legacy default stream).
 *             All device work is enqueued on it; calls do not synchronise the
 *             host except where stated (idg_filter_host).
 *   return    0 = IDG_OK; negative = argument error found on the host before
 *             any launch (nothing was enqueued); positive = a cudaError_t.
 *   NaN       voxels propagate by IEEE rules (FITS blanks are not treated).
 */
#ifndef IDG_H_
#define IDG_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define IDG_VERSION 10100           /* major*10000 + minor*100 + patch */

enum {
    IDG_OK = 0,
    IDG_ERR_NULL = -1,             /* a required pointer is NULL */
    IDG_ERR_DIMS = -2,             /* nx, ny, nz or batch < 1, or voxel count overflows */
    IDG_ERR_NITER = -3,            /* n_iter < 0 */
    IDG_ERR_PARAM = -4,            /* K <= 0 or NaN; tau, Cj < 0; rms <= 0; non-finite (K = +inf is allowed) */
    IDG_ERR_WORKSPACE = -5,        /* workspace NULL, too small or not 256-byte aligned */
    IDG_ERR_OVERLAP = -6,          /* cube/out/workspace partially overlap */
    IDG_ERR_OPTION = -7,           /* unknown option key or value out of range */
    IDG_ERR_STATIC_LIMIT = -8      /* idg_gaussian_filter_static: the kernel does not fit the static scratch array */
};

/*
 * Filter parameters.  Paper GUI ranges: tau in [0.0025, 0.0625],
 * Cj in [0, 10], K in [0.5, 10]; defaults K = 1.5, tau = 0.0325, Cj = 5, n = 20.
 * Values outside the ranges are accepted (idg_params_check reports them).
 */
typedef struct idg_params {
    float K;            /* conductance scale in units of rms; > 0; +INFINITY = constant conductance */
    float tau;          /* time step; >= 0 */
    float cx, cy, cz;   /* axis weights Cx (RA), Cy (Dec), Cz (velocity); >= 0 */
    float rms;          /* noise level of the ORIGINAL cube, in cube units; > 0; constant over iterations */
} idg_params;

/* Library version (IDG_VERSION of the build). */
int idg_version(void);

/* Static, NUL-terminated description of a status returned by any entry point. */
const char *idg_status_string(int status);

/*
 * Host-only check of one parameter set.  Returns a bit mask:
 *   bit 0  some value lies outside the paper's GUI range
 *   bit 1  tau*(Cx+Cy+Cz) > 1/2: the explicit scheme is linearly unstable where
 *          the conductance is ~1 (reading R9)
 *   bit 2  the set is invalid (the filter entry points would return IDG_ERR_PARAM)
 */
unsigned idg_params_check(const idg_params *params /*[host]*/);

/*
 * Bytes of device workspace idg_filter_ws / idg_filter_batched need for `batch`
 * cubes of nx*ny*nz voxels: one scratch cube per cube (the "temporary eta" of
 * PAPER.md:430; for nx % 4 != 0 instead three copies of the batch with the row
 * pitch rounded up to 16 bytes, on which the TMA-fed kernel runs) plus a small
 * parameter table, the 256-byte block holding the
 * arrival counter of the cooperative single-launch path and, for cubes the resident
 * kernel can take (nx >= 8, at most 4 Mi voxels), 32 MB of mailboxes for the
 * block faces.  0 on invalid dimensions.  A batch of more than ~2000 cubes uploads
 * its parameter table from pageable memory, which may synchronise the host.
 */
size_t idg_workspace_bytes(int nx, int ny, int nz, int batch);

/*
 * n_iter IDG updates (Eq. 7) of one cube.  north_star signature: the scratch
 * cube is a stream-ordered temporary (see idg_release_temporaries) taken on
 * `stream` and returned before the call returns.
 *   cube   [device] nx*ny*nz fp32, input I_0
 *   params [host]   one idg_params, copied during the call
 *   out    [device] nx*ny*nz fp32, receives I_n (n_iter = 0 copies cube)
 */
int idg_filter(const float *cube, int nx, int ny, int nz, int n_iter,
               const idg_params *params, float *out, void *stream);

/*
 * As idg_filter, never allocating: `workspace` [device] must hold
 * idg_workspace_bytes(nx, ny, nz, 1) bytes, 256-byte aligned.
 */
int idg_filter_ws(const float *cube, int nx, int ny, int nz, int n_iter,
                  const idg_params *params, float *out,
                  void *workspace, size_t workspace_bytes, void *stream);

/*
 * Gradient-driven variant: as idg_filter_ws, but the conductance of Eq. 7 is the classic Perona-Malik
 * one (Eq. 5), S = 1 / (1 + |grad I_i|^2 / (K^2 rms^2)), with |grad I|^2 the sum over
 * the axes of the squared central difference [I(+1) - I(-1)] / 2 of the same six neighbours
 * (replicated faces; K in units of rms per voxel: DESIGN.md readings P1-P3).  K = +INFINITY gives the
 * same linear diffusion as idg_filter.
 */
int idg_filter_pm(const float *cube, int nx, int ny, int nz, int n_iter, const idg_params *params,
                  float *out, void *workspace, size_t workspace_bytes, void *stream);

/*
 * The gradient-driven variant for `batch` cubes in one call: arguments, layout and errors as idg_filter_batched,
 * arithmetic as idg_filter_pm.
 */
int idg_filter_pm_batched(const float *cubes, int nx, int ny, int nz, int batch,
                          const int *n_iter, int n_iter_all, const idg_params *params,
                          float *out, void *workspace, size_t workspace_bytes, void *stream);

/*
 * `batch` independent cubes of equal shape in one call (interactive parameter
 * exploration), each with its own parameters and
 * iteration count.
 *   cubes  [device] batch*nx*ny*nz fp32
 *   n_iter [host]   batch ints (each >= 0), or NULL to use n_iter_all for all
 *   params [host]   batch idg_params
 *   out    [device] batch*nx*ny*nz fp32 (may equal cubes)
 *   workspace [device] idg_workspace_bytes(nx, ny, nz, batch) bytes, 256-byte aligned
 */
int idg_filter_batched(const float *cubes, int nx, int ny, int nz, int batch,
                       const int *n_iter, int n_iter_all, const idg_params *params,
                       float *out, void *workspace, size_t workspace_bytes, void *stream);

/*
 * End-to-end convenience for HOST buffers (the paper's T_p includes the
 * transfers): copies cube_host to the device, filters, copies
 * I_n to out_host and synchronises `stream` before returning.  Cubes of 64 MB
 * and more are cut into up to 16 z slabs (each filtered with n_iter halo planes
 * per side, bit-identical results) so that upload, filtering and download
 * overlap on two copy streams created (and destroyed) by the call on the current
 * device; pinned host memory is needed for that.  Safe to call from several host
 * threads and on several devices at once: no state is shared between calls.
 *   cube_host, out_host [host] nx*ny*nz fp32 (pinned memory gives full PCIe rate)
 *   dev_buffers [device] 2*nx*ny*nz*4 + idg_workspace_bytes(nx,ny,nz,1) bytes,
 *               256-byte aligned, or NULL to use the stream-ordered allocator.
 */
int idg_filter_host(const float *cube_host, int nx, int ny, int nz, int n_iter,
                    const idg_params *params, float *out_host,
                    void *dev_buffers, size_t dev_buffers_bytes, void *stream);

/*
 * Box filter (section 3.1): every voxel becomes the mean of its wx x wy x wz
 * neighbourhood, itself included (the paper's N_x, N_y, N_z).  Out-of-cube
 * neighbours are the nearest in-cube voxel (reading F1).  One fused separable pass.
 *   cube [device] nx*ny*nz fp32;  out [device] nx*ny*nz fp32, must not overlap cube
 *   wx, wy, wz   odd, 1 .. 33 (wx along x = RA); anything else returns IDG_ERR_PARAM
 */
int idg_box_filter(const float *cube, int nx, int ny, int nz, int wx, int wy, int wz, float *out, void *stream);

/*
 * Gaussian filter (section 3.2): 3-D convolution with
 *   G = A exp(-(x^2/2sx^2 + y^2/2sy^2 + z^2/2sz^2))  (Eq. 1),  FWHM_j = 2 sqrt(2 ln 2) s_j  (Eq. 2),
 *   K = Rz(theta_z) Ry(theta_y) Rx(theta_x) G        (Eq. 3).
 * Readings (F1-F5): replicated faces; the sampled kernel is normalised to unit sum;
 * support |p_j| <= floor(3 s_j + 1/2), for a rotated kernel the cube of the largest such radius;
 * (R G)(p) = G(R^-1 p) with right-handed matrices, angles in degrees; FWHM_j = 0 switches axis j off
 * (not allowed together with a rotation).  All angles zero: one fused separable pass (radius <= 16
 * per axis, FWHM <= 12.9); otherwise a dense (2r+1)^3 convolution (r <= 10, FWHM <= 8.2).  Parameters
 * outside these limits, negative or non-finite return IDG_ERR_PARAM.
 *   cube [device] nx*ny*nz fp32;  out [device] nx*ny*nz fp32, must not overlap cube
 *   fwhm_* in voxels, theta_* in degrees.  The rotated path takes (2r+1)^3 floats from the
 *   stream-ordered allocator for the kernel weights and returns them before the call returns.
 */
int idg_gaussian_filter(const float *cube, int nx, int ny, int nz, float fwhm_x, float fwhm_y, float fwhm_z,
                        float theta_x, float theta_y, float theta_z, float *out, void *stream);

/*
 * No-allocation variant of the ROTATED Gaussian filter (Eq. 3), for callers that cannot call cudaMalloc: code under CUDA
 * graph capture, tight serving loops, harnesses that forbid allocation.  As idg_gaussian_filter with a rotation (same
 * readings, same kernel, same result), but the (2r+1)^3 kernel weights live in a static device array inside the library
 * instead of a stream-ordered temporary: the call runs no cudaMalloc, cudaFree or other allocating routine.
 *   limit     support radius r <= 9, i.e. 19^3 floats = 27 436 bytes, held by every GPU that loads the library until the
 *             process exits (FWHM <= 7.4 voxels: every FWHM of the paper).  A larger kernel (which idg_gaussian_filter
 *             takes up to r = 10) returns IDG_ERR_STATIC_LIMIT; nothing is enqueued.
 *   angles    at least one must be non-zero; all zero returns IDG_ERR_PARAM (the separable path of idg_gaussian_filter
 *             has no scratch and allocates nothing as it is).
 *   sharing   every call on a device uses the ONE array and overwrites what the previous call left there, in stream
 *             order.  Calls that overlap on the GPU (different streams not ordered by events, several host threads)
 *             race on it and are not supported.  Nothing in it has to start at zero.
 *   cube [device] nx*ny*nz fp32;  out [device] nx*ny*nz fp32, must not overlap cube.  Other errors as idg_gaussian_filter.
 *   idg_last_launch_count / idg_last_plan are not updated by this call.
 */
int idg_gaussian_filter_static(const float *cube, int nx, int ny, int nz, float fwhm_x, float fwhm_y, float fwhm_z,
                               float theta_x, float theta_y, float theta_z, float *out, void *stream);

/*
 * Host-only: support radii (rx, ry, rz) idg_gaussian_filter would use, or IDG_ERR_PARAM.
 *   radii [host] 3 ints
 */
int idg_gaussian_radii(float fwhm_x, float fwhm_y, float fwhm_z, float theta_x, float theta_y, float theta_z,
                       int radii[3]);

/*
 * Smoothing-quality diagnostics (Eq. 12-16; Eq. 17-18).
 * A region of interest is the half-open index box [x0,x1) x [y0,y1) x [z0,z1) (NULL = whole cube).
 */
typedef struct idg_roi { int x0, x1, y0, y1, z0, z1; } idg_roi;

/*
 * One pass over the original, the filtered and (optionally) the noiseless model cube:
 *   M_o = [I_o >= thr_o], M_f = [I_f >= thr_f]   (Eq. 14 with thr_i = 3 rms_i; fp32 compare, NaN never passes)
 *   sums[0] = S_oo = sum I_o M_o     sums[1] = S_of = sum I_o M_f      (Eq. 13)
 *   sums[2] = N_o  = sum M_o         sums[3] = N_f  = sum M_f          (Eq. 16)
 *   sums[4] = S_mf = sum I_m M_f     sums[5] = S_m  = sum I_m          (Eq. 18; 0 when model is NULL)
 *   sums[6] = voxels in the ROI      sums[7] = 0
 * over the ROI, accumulated in fp64 (counts are exact).
 *   orig, filt, model [device] nx*ny*nz fp32 (model may be NULL);  roi [host] or NULL
 *   sums [device] 8 doubles, 8-byte aligned; overwritten.  Errors: IDG_ERR_DIMS for a ROI outside the
 *   cube, IDG_ERR_PARAM for a NaN threshold, IDG_ERR_WORKSPACE for a misaligned `sums`.
 */
int idg_mask_sums(const float *orig, const float *filt, const float *model, int nx, int ny, int nz,
                  const idg_roi *roi, float thr_o, float thr_f, double *sums, void *stream);

/*
 * stats[0] = n, stats[1] = sum, stats[2] = sum of squares of the voxels of the ROI (fp64); the noise
 * level of a signal-free ROI is sqrt(stats[2]/n - (stats[1]/n)^2) (reading Q4).
 *   cube [device];  stats [device] 8 doubles, 8-byte aligned; overwritten
 */
int idg_cube_stats(const float *cube, int nx, int ny, int nz, const idg_roi *roi, double *stats, void *stream);

/*
 * Host-only: mean and noise level rms = sqrt(<x^2> - <x>^2) (reading Q4) from a HOST copy of the
 * idg_cube_stats output.  Either output pointer may be NULL; n = 0 gives NaN.  IDG_ERR_NULL for stats == NULL.
 */
int idg_stats_rms(const double *stats, double *mean, double *rms);

/*
 * Histogram of the voxel intensities of the ROI (Fig. 6): `nbins` (1..8192) equal bins over
 * [lo, hi); a voxel v with lo <= v < hi (and v >= *mask_thr when mask_thr is given) counts in bin
 * floor((v - lo) * (nbins / (hi - lo))), every operation in fp32 (reading Q5); NaN never counts.
 *   cube [device];  mask_thr [host] one float or NULL;  counts [device] nbins 64-bit counters, overwritten
 */
int idg_histogram(const float *cube, int nx, int ny, int nz, const idg_roi *roi, float lo, float hi, int nbins,
                  const float *mask_thr, unsigned long long *counts, void *stream);

/*
 * Host-only: F = |S_of|/|S_oo| (Eq. 12), its error (Eq. 15-16, with N_i = population / voxels_per_beam,
 * voxels_per_beam >= 1) and F_M = |S_mf|/|S_m| (Eq. 17) from a HOST copy of the sums.  Any of the three
 * output pointers may be NULL; a ratio with a zero denominator is NaN.
 */
int idg_quality(const double *sums, double rms_o, double rms_f, double voxels_per_beam, double *F, double *sigma_F,
                double *F_M);

/*
 * Wavelet lifting (section 3.4).  One level along a line: split into even and odd
 * samples, predict d_i = odd_i - P(even) (Eq. 8), update c_i = even_i + U(d) (Eq. 10), with
 *   Haar          P = even_i (Eq. 9),               U = d_i / 2 (Eq. 11)
 *   Le Gall 5/3   P = (even_i + even_{i+1}) / 2,    U = (d_{i-1} + d_i) / 4   (symmetric extension at the ends)
 * Coefficients stay interleaved in place: after level l the approximation band lives on
 * the voxels whose three indices are multiples of 2^l.  Per level the lines along x, then y, then z of
 * the current lattice are transformed (readings W1-W5).
 */
enum { IDG_WAVELET_HAAR = 0, IDG_WAVELET_LEGALL53 = 1 };

/*
 * Forward (inverse = 0) or inverse (inverse != 0) transform to `levels` (0..16) of a cube.
 *   cube [device] nx*ny*nz fp32;  out [device] nx*ny*nz fp32, may equal cube (in place), else disjoint
 */
int idg_wavelet_transform(const float *cube, int nx, int ny, int nz, int wavelet, int levels, int inverse, float *out,
                          void *stream);

/*
 * Wavelet thresholding filter: transform to `levels` (1..16; the paper stops at 3), set to
 * zero every coefficient with |v| < t_l * rms -- detail coefficients created at level l with t_l, the
 * approximation band with t_levels ("it is necessary to threshold both the detail and approximation
 * bands") -- and transform back.  Pre-smoothing is a separate idg_gaussian_filter call.
 *   thresholds [host] `levels` floats >= 0, in units of rms;  rms > 0: noise level of the original cube
 *   cube, out as for idg_wavelet_transform.  Invalid wavelet, levels, thresholds or rms: IDG_ERR_PARAM.
 * Le Gall 5/3: the default path fuses the three axes of a level and works out of place on compact lattices in a
 * stream-ordered temporary of ~1.3 cubes (see idg_release_temporaries); when that cannot be allocated, or with
 * IDG_OPT_KERNEL = 2 (1: two-phase passes), it runs the in-place passes, which need no memory ("does not require
 * additional memory").  Haar, levels <= 3: one fused pass (an 8 x 8 x 8 block per warp in registers when
 * nx % 4 == 0 and the cubes are 16-byte aligned, else -- or with IDG_OPT_KERNEL = 2 -- 64 x 8 x 8 regions in shared
 * memory; IDG_OPT_KERNEL = 1: the in-place passes).  All paths give bit-identical results.
 */
int idg_wavelet_filter(const float *cube, int nx, int ny, int nz, int wavelet, int levels, const float *thresholds,
                       float rms, float *out, void *stream);

/*
 * Tuning knobs of the CALLING HOST THREAD (tests and benchmarks; defaults give the fastest plan): an option set by
 * one thread affects the calls that thread makes afterwards and no other thread's.
 *   IDG_OPT_KERNEL   0 auto (the resident kernel 5 when the whole call fits in the SMs' shared memory at once in small
 *                    blocks -- cubes of up to ~1.3 Mvoxel --, else kernel 3: directly where nx % 4 == 0 and the buffers
 *                    are 16-byte aligned, on pitched copies in the workspace otherwise) | 1 naive (one thread per
 *                    voxel) | 2 tiled z-streaming kernel (global loads) | 3 tiled z-streaming kernel fed by TMA (the
 *                    fast path for large cubes) | 4 (retired: runs kernel 3) | 5 resident kernel: blocks of
 *                    the cube(s) stay in shared memory for all iterations of the call, block faces are exchanged
 *                    through mailboxes in the workspace, one cooperative launch per wave of cubes (cubes of up to
 *                    4 Mi voxels with nx >= 8, any alignment: rows are padded to float4 on chip; otherwise the auto
 *                    plan).  Reference filters: 1 = the
 *                    general separable kernel also where the TMA-fed one applies.  Wavelets: see idg_wavelet_filter
 *   IDG_OPT_FUSE     0 auto (4, or 2 for full-GPU workloads of cubes thinner than 100 planes) | 1..4 = diffusion
 *                    iterations fused per launch (kernels 2-4)
 *   IDG_OPT_ZCHUNK   0 auto | >0  = planes per CTA along z (kernels 2, 3)
 *   IDG_OPT_TILE     0 auto | kernel 3: 1 = one CTA per SM (T <= 2: 128x64 tile, 512 threads; T >= 3: 128x32
 *                    tile, 256 threads), 2 = 128x32 tile, two 256-thread CTAs per SM (T <= 2), 3 = 384-thread CTA
 *                    (T >= 3), 4 = cluster pairs (T >= 3): two 256-thread CTAs stacked along y share a 128x64 tile and
 *                    exchange their seam rows through distributed shared memory (measured slower than 1 at T = 4,
 *                    faster at T = 3: profiles/r2b_notes.md) | separable reference filters: 2 = strips of 4
 *                    rows per thread instead of 2 in idg_sep3d_tma_kernel
 *   IDG_OPT_CTAS     reserved (was the grid size of the retired kernel 4); ignored
 *   IDG_OPT_HOST_SLABS  0 auto | 1..16 = z slabs of the idg_filter_host transfer/compute pipeline (1 = one piece)
 *   IDG_OPT_COOP     0 auto (small cubes whose whole grid is co-resident: all launches of kernel 3 folded into ONE
 *                    cooperative launch with grid barriers between the fused rounds) | 1 never | 2 whenever the grid fits
 * idg_get_option returns the current value, or IDG_ERR_OPTION.
 */
enum { IDG_OPT_KERNEL = 0, IDG_OPT_FUSE = 1, IDG_OPT_ZCHUNK = 2, IDG_OPT_TILE = 3, IDG_OPT_CTAS = 4,
       IDG_OPT_HOST_SLABS = 5, IDG_OPT_COOP = 6, IDG_OPT_COUNT_ = 7 };
int idg_set_option(int key, int value);
int idg_get_option(int key);

/*
 * Stream-ordered temporaries (the scratch cube of idg_filter, the device buffers of idg_filter_host when none
 * are passed, the kernel weights of a rotated Gaussian, the lattices of the Le Gall filter) come from a memory
 * pool private to the library, one per device, which keeps memory between calls so that a call does not pay the
 * driver's map / unmap again -- at most twice the size of the largest recent request, halved after every 64
 * requests in a row below a quarter of it (so a 2 GB temporary is not held for ever once the caller moves on to
 * small cubes).
 * idg_release_temporaries() returns everything that is not in use on the current device to the driver at once
 * (synchronise the streams that used the library first).
 * Returns IDG_OK or a cudaError_t.
 */
int idg_release_temporaries(void);

/*
 * Number of kernel launches the last filter call on this thread enqueued
 * (for bench.py's "gpu_launches" claim).
 */
int idg_last_launch_count(void);

/*
 * Plan of the last filter call on this thread: "<kernel name> fuse=<T> tile=<variant>" (static
 * thread-local storage; for bench.py's roofline record).
 */
const char *idg_last_plan(void);

#ifdef __cplusplus
}
#endif
#endif /* IDG_H_ */
