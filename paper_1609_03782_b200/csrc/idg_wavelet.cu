// Wavelet lifting and the wavelet thresholding filter (section 3.4, Eq. 8-11), fp32,
// in place ("does not require additional memory"): after level l the approximation
// coefficients c sit on the lattice of points whose three indices are multiples of 2^l, the details d on
// the rest of the level-l lattice (readings W1-W5).
//
//   predict  d_i = odd_i - P(even)      Haar: P = even_i             Le Gall 5/3: P = (even_i + even_{i+1}) / 2
//   update   c_i = even_i + U(d)        Haar: U = d_i / 2            Le Gall 5/3: U = (d_{i-1} + d_i) / 4
//
// One kernel launch per (level, axis, phase): a thread owns one target sample (an odd one in the
// predict phase, an even one in the update phase), so a phase only reads samples the phase does not
// write.  Threads are laid out with the lattice x index fastest.  The threshold pass is one more
// elementwise kernel (band level from the trailing zero bits of the indices).  All of it is bound by
// HBM traffic; level 1 dominates (the level-l lattice holds 8^-(l-1) of the voxels).
#include "idg_kernels.cuh"

namespace idg {

namespace {

constexpr int NT = 256;

struct WArgs {
    float *a;
    int nx, ny, nz;
    int s;              // lattice stride 2^(l-1)
    int axis;           // 0 x, 1 y, 2 z
    int mx, my, mz;     // lattice extents ceil(n / s)
};

// PHASE 0: predict (targets = odd samples), 1: update (targets = even samples); INV undoes the phase.
template <int WAVELET, int PHASE, bool INV>
__global__ void __launch_bounds__(NT) idg_lift_kernel(const __grid_constant__ WArgs W)
{
    const int m = W.axis == 0 ? W.mx : (W.axis == 1 ? W.my : W.mz);       // samples on a line
    const int no = m / 2, ne = m - no;
    const int nt = PHASE == 0 ? no : ne;                                  // targets on a line
    // thread -> (target i along the axis, lattice coordinates of the other two axes), x fastest
    const int ex = W.axis == 0 ? nt : W.mx, ey = W.axis == 1 ? nt : W.my, ez = W.axis == 2 ? nt : W.mz;
    const long long total = (long long)ex * ey * ez;
    const size_t sx = (size_t)W.s, sy = (size_t)W.s * W.nx, sz = (size_t)W.s * W.nx * (size_t)W.ny;
    const size_t st = W.axis == 0 ? sx : (W.axis == 1 ? sy : sz);         // stride between line samples
    for (long long t = (long long)blockIdx.x * NT + threadIdx.x; t < total; t += (long long)gridDim.x * NT) {
        const int cx = (int)(t % ex), cy = (int)((t / ex) % ey), cz = (int)(t / ((long long)ex * ey));
        const int i = W.axis == 0 ? cx : (W.axis == 1 ? cy : cz);
        float *line = W.a + (W.axis == 0 ? 0 : (size_t)cx * sx) + (W.axis == 1 ? 0 : (size_t)cy * sy) +
                      (W.axis == 2 ? 0 : (size_t)cz * sz);
        if (PHASE == 0) {
            const float e0 = line[(size_t)(2 * i) * st];
            float p = e0;
            if (WAVELET == 1) {
                const float e1 = (i + 1 < ne) ? line[(size_t)(2 * i + 2) * st] : e0;      // reading W4
                p = 0.5f * (e0 + e1);
            }
            float *d = line + (size_t)(2 * i + 1) * st;
            *d = INV ? *d + p : *d - p;                                   // Eq. 8
        } else {
            float u;
            if (WAVELET == 0) {
                if (i >= no) continue;                                    // unpaired last even sample (W2)
                u = 0.5f * line[(size_t)(2 * i + 1) * st];                // Eq. 11
            } else {
                const float dr = (i < no) ? line[(size_t)(2 * i + 1) * st] : line[(size_t)(2 * i - 1) * st];
                const float dl = (i > 0) ? line[(size_t)(2 * i - 1) * st] : dr;
                u = 0.25f * (dl + dr);
            }
            float *c = line + (size_t)(2 * i) * st;
            *c = INV ? *c - u : *c + u;                                   // Eq. 10
        }
    }
}

// Haar only: predict and update of one (even, odd) pair touch nothing but the pair (Eq. 8-11 with P = even_i,
// U = d_i / 2), so both phases run in one race-free in-place pass with a thread per pair; same operations in
// the same order as the two-phase kernel.
template <bool INV>
__global__ void __launch_bounds__(NT) idg_haar_pair_kernel(const __grid_constant__ WArgs W)
{
    const int m = W.axis == 0 ? W.mx : (W.axis == 1 ? W.my : W.mz);
    const int no = m / 2;
    const int ex = W.axis == 0 ? no : W.mx, ey = W.axis == 1 ? no : W.my, ez = W.axis == 2 ? no : W.mz;
    const long long total = (long long)ex * ey * ez;
    const size_t sx = (size_t)W.s, sy = (size_t)W.s * W.nx, sz = (size_t)W.s * W.nx * (size_t)W.ny;
    const size_t st = W.axis == 0 ? sx : (W.axis == 1 ? sy : sz);
    for (long long t = (long long)blockIdx.x * NT + threadIdx.x; t < total; t += (long long)gridDim.x * NT) {
        const int cx = (int)(t % ex), cy = (int)((t / ex) % ey), cz = (int)(t / ((long long)ex * ey));
        const int i = W.axis == 0 ? cx : (W.axis == 1 ? cy : cz);
        float *line = W.a + (W.axis == 0 ? 0 : (size_t)cx * sx) + (W.axis == 1 ? 0 : (size_t)cy * sy) +
                      (W.axis == 2 ? 0 : (size_t)cz * sz);
        float *pe = line + (size_t)(2 * i) * st, *po = pe + st;
        float e = *pe, o = *po;
        if (!INV) { o = o - e; e = e + 0.5f * o; }          // d = odd - even;  c = even + d/2
        else { e = e - 0.5f * o; o = o + e; }               // even = c - d/2;  odd = d + even
        *pe = e;
        *po = o;
    }
}

struct TArgs {
    float *a;
    int nx, ny, nz, levels;
    float thr[16];      // t_l * rms
};

// Hard threshold (reading W3): band level = 1 + min trailing zeros of (x, y, z), capped at `levels`.
__global__ void __launch_bounds__(NT) idg_wavelet_threshold_kernel(const __grid_constant__ TArgs T)
{
    const size_t N = (size_t)T.nx * T.ny * (size_t)T.nz;
    for (size_t i = (size_t)blockIdx.x * NT + threadIdx.x; i < N; i += (size_t)gridDim.x * NT) {
        const int x = (int)(i % (size_t)T.nx), y = (int)((i / (size_t)T.nx) % (size_t)T.ny),
                  z = (int)(i / ((size_t)T.nx * T.ny));
        const int tz = __ffs(x | y | z | (1 << 30)) - 1;                  // min of the three trailing-zero counts
        const int l = tz + 1 < T.levels ? tz + 1 : T.levels;
        const float v = T.a[i];
        if (fabsf(v) < T.thr[l - 1]) T.a[i] = 0.f;
    }
}

template <int WAVELET, int PHASE, bool INV>
cudaError_t launch_phase(const WArgs &W, cudaStream_t st)
{
    const int m = W.axis == 0 ? W.mx : (W.axis == 1 ? W.my : W.mz);
    const int nt = PHASE == 0 ? m / 2 : m - m / 2;
    const long long total = (long long)(W.axis == 0 ? nt : W.mx) * (W.axis == 1 ? nt : W.my) * (W.axis == 2 ? nt : W.mz);
    if (total <= 0 || m < 2) return cudaSuccess;
    long long grid = (total + NT - 1) / NT;
    if (grid > 148LL * 32) grid = 148LL * 32;
    idg_lift_kernel<WAVELET, PHASE, INV><<<(unsigned)grid, NT, 0, st>>>(W);
    return cudaGetLastError();
}

template <int WAVELET>
cudaError_t transform(float *a, int nx, int ny, int nz, int levels, bool inverse, cudaStream_t st, int *launches)
{
    cudaError_t e = cudaSuccess;
    for (int li = 0; li < levels && e == cudaSuccess; ++li) {
        const int l = inverse ? levels - li : li + 1;
        const int s = 1 << (l - 1);
        WArgs W{a, nx, ny, nz, s, 0, (nx + s - 1) / s, (ny + s - 1) / s, (nz + s - 1) / s};
        for (int ai = 0; ai < 3 && e == cudaSuccess; ++ai) {
            W.axis = inverse ? 2 - ai : ai;
            const int m = W.axis == 0 ? W.mx : (W.axis == 1 ? W.my : W.mz);
            if (m < 2) continue;
            if (WAVELET == 0) {
                const long long total = (long long)(W.axis == 0 ? m / 2 : W.mx) * (W.axis == 1 ? m / 2 : W.my) *
                                        (W.axis == 2 ? m / 2 : W.mz);
                long long grid = (total + NT - 1) / NT;
                if (grid > 148LL * 32) grid = 148LL * 32;
                if (inverse) idg_haar_pair_kernel<true><<<(unsigned)grid, NT, 0, st>>>(W);
                else idg_haar_pair_kernel<false><<<(unsigned)grid, NT, 0, st>>>(W);
                e = cudaGetLastError();
                *launches += 1;
                continue;
            }
            if (!inverse) {
                e = launch_phase<WAVELET, 0, false>(W, st);
                if (e == cudaSuccess) e = launch_phase<WAVELET, 1, false>(W, st);
            } else {
                e = launch_phase<WAVELET, 1, true>(W, st);
                if (e == cudaSuccess) e = launch_phase<WAVELET, 0, true>(W, st);
            }
            *launches += 2;
        }
    }
    return e;
}

}  // namespace

// In-place forward / inverse transform of `a` to `levels` (wavelet 0 Haar, 1 Le Gall 5/3).
cudaError_t launch_wavelet_transform(float *a, int nx, int ny, int nz, int wavelet, int levels, bool inverse,
                                     cudaStream_t st, int *launches)
{
    return wavelet == 0 ? transform<0>(a, nx, ny, nz, levels, inverse, st, launches)
                        : transform<1>(a, nx, ny, nz, levels, inverse, st, launches);
}

// thr[l-1] = t_l * rms, levels <= 16.
cudaError_t launch_wavelet_threshold(float *a, int nx, int ny, int nz, int levels, const float *thr, cudaStream_t st)
{
    TArgs T;
    T.a = a; T.nx = nx; T.ny = ny; T.nz = nz; T.levels = levels;
    for (int i = 0; i < 16; ++i) T.thr[i] = i < levels ? thr[i] : 0.f;
    const size_t N = (size_t)nx * ny * (size_t)nz;
    size_t grid = (N + NT - 1) / NT;
    if (grid > 148u * 32u) grid = 148u * 32u;
    idg_wavelet_threshold_kernel<<<(unsigned)grid, NT, 0, st>>>(T);
    return cudaGetLastError();
}

}  // namespace idg
