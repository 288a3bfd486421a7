/*
 * oracle/wavelet_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of the wavelet-lifting thresholding filter of Punzo, van der Hulst &
 * Roerdink (arXiv:1609.03782), PAPER.md:191-241 (section 3.4, Eq. 8-11).  Shares no code with the
 * CUDA path; same access rules as idg_oracle.c.
 *
 * Lifting, one level, along one line a[0..m):
 *   split    even_i = a[2i], odd_i = a[2i+1]                                   ("lazy wavelet")
 *   predict  d_i = odd_i - P(even)                                             (Eq. 8)
 *   update   c_i = even_i + U(d)                                               (Eq. 10)
 *   Haar:       P = even_i                     (Eq. 9),   U = d_i / 2                      (Eq. 11)
 *   Le Gall 5/3: P = (even_i + even_{i+1}) / 2,           U = (d_{i-1} + d_i) / 4          (reading W4)
 * "does not require additional memory": coefficients stay interleaved in place, c at the
 * even and d at the odd positions of the line; level l+1 works on the c of level l, i.e. on the
 * samples at stride 2^l.  The filter decomposes to level L (<= 3 in the paper), thresholds the
 * detail AND the approximation bands and transforms back.
 *
 * Readings where the paper is silent (W1-W5):
 *   W1  3-D: per level the 1-D transform runs along x, then y, then z over the current lattice
 *       (all points whose three indices are multiples of 2^(l-1)); the inverse undoes z, y, x from
 *       level L down to 1.
 *   W2  odd length: a last even sample without an odd partner gets no Haar update (c = even).
 *   W3  thresholding is hard: a coefficient with |v| < t_l * rms becomes 0; a detail coefficient
 *       created at level l uses t_l, the approximation band left after level L uses t_L; thresholds
 *       are in units of the rms of the original cube.
 *   W4  Le Gall 5/3 is the Cohen-Daubechies-Feauveau 5/3 lifting pair (the paper names the wavelet,
 *       PAPER.md:193, and prints only the Haar operators) with whole-sample symmetric extension at
 *       the line ends: a missing even_{i+1} is even_i, a missing d_{i-1} is d_i and a missing d_i is d_{i-1}.
 *   W5  pre-smoothing is a separate Gaussian-filter call, not part of this routine.
 *
 * Layout: idx = x + nx*(y + ny*z).
 */
#include <math.h>
#include <stddef.h>
#include <string.h>

/* one level along one line: m samples at stride `st` (in elements) starting at a */
static void lift_forward(double *a, int m, size_t st, int wavelet)
{
    const int no = m / 2, ne = m - no;
    if (no == 0) return;
    for (int i = 0; i < no; ++i) {                                  /* predict (Eq. 8) */
        const double e0 = a[(size_t)(2 * i) * st];
        const double e1 = (i + 1 < ne) ? a[(size_t)(2 * i + 2) * st] : e0;          /* W4 */
        a[(size_t)(2 * i + 1) * st] -= wavelet == 0 ? e0 : 0.5 * (e0 + e1);
    }
    for (int i = 0; i < ne; ++i) {                                  /* update (Eq. 10) */
        if (wavelet == 0) {
            if (i < no) a[(size_t)(2 * i) * st] += 0.5 * a[(size_t)(2 * i + 1) * st];   /* Eq. 11; W2 */
        } else {
            const double dr = (i < no) ? a[(size_t)(2 * i + 1) * st] : a[(size_t)(2 * i - 1) * st];
            const double dl = (i > 0) ? a[(size_t)(2 * i - 1) * st] : dr;
            a[(size_t)(2 * i) * st] += 0.25 * (dl + dr);
        }
    }
}

static void lift_inverse(double *a, int m, size_t st, int wavelet)
{
    const int no = m / 2, ne = m - no;
    if (no == 0) return;
    for (int i = 0; i < ne; ++i) {                                  /* undo update */
        if (wavelet == 0) {
            if (i < no) a[(size_t)(2 * i) * st] -= 0.5 * a[(size_t)(2 * i + 1) * st];
        } else {
            const double dr = (i < no) ? a[(size_t)(2 * i + 1) * st] : a[(size_t)(2 * i - 1) * st];
            const double dl = (i > 0) ? a[(size_t)(2 * i - 1) * st] : dr;
            a[(size_t)(2 * i) * st] -= 0.25 * (dl + dr);
        }
    }
    for (int i = 0; i < no; ++i) {                                  /* undo predict */
        const double e0 = a[(size_t)(2 * i) * st];
        const double e1 = (i + 1 < ne) ? a[(size_t)(2 * i + 2) * st] : e0;
        a[(size_t)(2 * i + 1) * st] += wavelet == 0 ? e0 : 0.5 * (e0 + e1);
    }
}

/* all lines of the level-`s` lattice (stride s) along axis 0 (x), 1 (y) or 2 (z)  (reading W1) */
static void lift_axis(double *a, int nx, int ny, int nz, int s, int axis, int wavelet, int inverse)
{
    const size_t sx = 1, sy = (size_t)nx, sz = (size_t)nx * (size_t)ny;
    const int n[3] = {nx, ny, nz};
    const size_t str[3] = {sx, sy, sz};
    const int u = (axis + 1) % 3, v = (axis + 2) % 3;
    const int m = (n[axis] + s - 1) / s;
    for (int q = 0; q < n[v]; q += s)
        for (int p = 0; p < n[u]; p += s) {
            double *line = a + (size_t)p * str[u] + (size_t)q * str[v];
            if (inverse) lift_inverse(line, m, (size_t)s * str[axis], wavelet);
            else lift_forward(line, m, (size_t)s * str[axis], wavelet);
        }
}

static int trailing(int p)      /* number of trailing zero bits, "infinite" for 0 */
{
    if (p == 0) return 31;
    int t = 0;
    while (!(p & 1)) { p >>= 1; ++t; }
    return t;
}

/*
 * Forward transform to `levels`, in place (fp64).  wavelet: 0 Haar, 1 Le Gall 5/3.
 */
int wavelet_forward_oracle(double *a, int nx, int ny, int nz, int wavelet, int levels)
{
    if (!a || nx < 1 || ny < 1 || nz < 1 || levels < 0 || levels > 16 || (wavelet != 0 && wavelet != 1)) return -1;
    for (int l = 1; l <= levels; ++l)
        for (int axis = 0; axis < 3; ++axis) lift_axis(a, nx, ny, nz, 1 << (l - 1), axis, wavelet, 0);
    return 0;
}

int wavelet_inverse_oracle(double *a, int nx, int ny, int nz, int wavelet, int levels)
{
    if (!a || nx < 1 || ny < 1 || nz < 1 || levels < 0 || levels > 16 || (wavelet != 0 && wavelet != 1)) return -1;
    for (int l = levels; l >= 1; --l)
        for (int axis = 2; axis >= 0; --axis) lift_axis(a, nx, ny, nz, 1 << (l - 1), axis, wavelet, 1);
    return 0;
}

/* hard thresholds t[l-1] (already multiplied by rms) on the interleaved coefficients (reading W3) */
int wavelet_threshold_oracle(double *a, int nx, int ny, int nz, int levels, const double *thr)
{
    if (!a || !thr || levels < 1) return -1;
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                int t = trailing(x);
                if (trailing(y) < t) t = trailing(y);
                if (trailing(z) < t) t = trailing(z);
                const int l = t + 1 < levels ? t + 1 : levels;      /* detail of level t+1, else approximation */
                double *v = a + (size_t)x + (size_t)nx * ((size_t)y + (size_t)ny * (size_t)z);
                if (fabs(*v) < thr[l - 1]) *v = 0.0;
            }
    return 0;
}

/* the filter: forward to `levels`, threshold with t_l * rms, inverse */
int wavelet_filter_oracle(const double *in, int nx, int ny, int nz, int wavelet, int levels, const double *t,
                          double rms, double *out)
{
    if (!in || !out || !t || levels < 1 || levels > 16 || !(rms > 0.0)) return -1;
    double thr[16];
    for (int l = 0; l < levels; ++l) {
        if (!(t[l] >= 0.0)) return -1;
        thr[l] = t[l] * rms;
    }
    if (in != out) memcpy(out, in, sizeof(double) * (size_t)nx * (size_t)ny * (size_t)nz);
    if (wavelet_forward_oracle(out, nx, ny, nz, wavelet, levels) != 0) return -1;
    wavelet_threshold_oracle(out, nx, ny, nz, levels, thr);
    return wavelet_inverse_oracle(out, nx, ny, nz, wavelet, levels);
}
