/*
 * oracle/ref_filters_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statements of the two reference filters of Punzo,
 * van der Hulst & Roerdink (arXiv:1609.03782): the box filter (PAPER.md:121-136,
 * section 3.1) and the Gaussian filter (section 3.2,
 * Eq. 1-3).  Both are written as the definition: one direct 3-D sum per output
 * voxel, no separable passes, no running sums.  Shares no code with the CUDA
 * path; same access rules as idg_oracle.c.
 *
 * Box filter: each voxel is replaced by the mean of its
 * Nx x Ny x Nz neighbourhood, itself included (N_j odd: 1, 3, 5, 7, 9 in
 * PAPER.md:282, :402-403).
 *
 * Gaussian filter: 3-D convolution with
 *   G(x,y,z) = A exp(-(x^2/2sx^2 + y^2/2sy^2 + z^2/2sz^2))          (Eq. 1)
 *   FWHM_i   = 2 sqrt(2 ln 2) s_i                                    (Eq. 2)
 *   K        = Rz(theta_z) Ry(theta_y) Rx(theta_x) G                 (Eq. 3)
 *
 * Readings where the paper is silent (F1-F5):
 *   F1  boundary: an out-of-cube neighbour is the nearest in-cube voxel
 *       (replication, the same zero-flux policy as reading R1 of the IDG filter).
 *   F2  A: the sampled kernel is normalised to unit sum over its support.
 *   F3  support: offsets |p_j| <= r_j with r_j = floor(3 s_j + 1/2) (three sigma,
 *       rounded to the nearest voxel); for a rotated kernel the support is the
 *       cube |p_j| <= floor(3 max(s) + 1/2) on every axis.
 *   F4  rotation: (R G)(p) = G(R^-1 p) with R = Rz Ry Rx, right-handed rotation
 *       matrices, angles in degrees; x = RA (fastest axis), y = Dec, z = velocity.
 *   F5  FWHM_j = 0 means no smoothing along axis j (r_j = 0); not allowed together
 *       with a rotation.
 *
 * Layout: idx = x + nx*(y + ny*z).
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>

static int clampi(int v, int n) { return v < 0 ? 0 : (v >= n ? n - 1 : v); }

/* mean over the Nx x Ny x Nz neighbourhood; reading F1 at the faces. */
int box_oracle_f64(const double *in, int nx, int ny, int nz, int wx, int wy, int wz, double *out)
{
    if (!in || !out || in == out || nx < 1 || ny < 1 || nz < 1) return -1;
    if (wx < 1 || wy < 1 || wz < 1 || !(wx & 1) || !(wy & 1) || !(wz & 1)) return -1;
    const int hx = wx / 2, hy = wy / 2, hz = wz / 2;
    const double count = (double)wx * (double)wy * (double)wz;
    const size_t sy = (size_t)nx, sz = (size_t)nx * (size_t)ny;
    long z;
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                double s = 0.0;
                for (int k = -hz; k <= hz; ++k)
                    for (int j = -hy; j <= hy; ++j)
                        for (int i = -hx; i <= hx; ++i)
                            s += in[(size_t)clampi(x + i, nx) + sy * (size_t)clampi(y + j, ny) +
                                    sz * (size_t)clampi((int)z + k, nz)];
                out[(size_t)x + sy * (size_t)y + sz * (size_t)z] = s / count;
            }
    return 0;
}

/* Eq. 2: sigma from FWHM. */
static double sigma_of(double fwhm) { return fwhm / (2.0 * sqrt(2.0 * log(2.0))); }

/* Reading F3: support radius of one axis. */
static int radius_of(double sigma) { return (int)floor(3.0 * sigma + 0.5); }

/*
 * Support radii of the kernel for the given FWHM (voxels) and Euler angles (degrees):
 * r[0..2] = (rx, ry, rz).  Returns 0, or -1 on invalid parameters.
 */
int gaussian_radii_oracle(const double fwhm[3], const double theta_deg[3], int r[3])
{
    for (int j = 0; j < 3; ++j)
        if (!(fwhm[j] >= 0.0) || !isfinite(fwhm[j]) || !isfinite(theta_deg[j])) return -1;
    const int rotated = theta_deg[0] != 0.0 || theta_deg[1] != 0.0 || theta_deg[2] != 0.0;
    if (rotated) {
        double smax = 0.0;
        for (int j = 0; j < 3; ++j) {
            if (!(fwhm[j] > 0.0)) return -1;                  /* F5 */
            if (sigma_of(fwhm[j]) > smax) smax = sigma_of(fwhm[j]);
        }
        r[0] = r[1] = r[2] = radius_of(smax);
    } else {
        for (int j = 0; j < 3; ++j) r[j] = radius_of(sigma_of(fwhm[j]));
    }
    return 0;
}

/*
 * The sampled, normalised kernel K[(k+rz)][(j+ry)][(i+rx)] for offsets (i, j, k) = (x, y, z)
 * (Eq. 1-3, readings F2-F5).  `kern` holds (2rx+1)(2ry+1)(2rz+1) doubles, x fastest.
 */
int gaussian_kernel_oracle(const double fwhm[3], const double theta_deg[3], const int r[3], double *kern)
{
    int rr[3];
    if (!kern || gaussian_radii_oracle(fwhm, theta_deg, rr) != 0) return -1;
    if (rr[0] != r[0] || rr[1] != r[1] || rr[2] != r[2]) return -1;
    const double d2r = acos(-1.0) / 180.0;
    const double cx = cos(theta_deg[0] * d2r), sx = sin(theta_deg[0] * d2r);
    const double cy = cos(theta_deg[1] * d2r), sy = sin(theta_deg[1] * d2r);
    const double cz = cos(theta_deg[2] * d2r), sz = sin(theta_deg[2] * d2r);
    /* right-handed rotation matrices */
    const double Rx[3][3] = {{1, 0, 0}, {0, cx, -sx}, {0, sx, cx}};
    const double Ry[3][3] = {{cy, 0, sy}, {0, 1, 0}, {-sy, 0, cy}};
    const double Rz[3][3] = {{cz, -sz, 0}, {sz, cz, 0}, {0, 0, 1}};
    double T[3][3], R[3][3];
    for (int a = 0; a < 3; ++a)                               /* T = Ry Rx */
        for (int b = 0; b < 3; ++b) {
            T[a][b] = 0.0;
            for (int c = 0; c < 3; ++c) T[a][b] += Ry[a][c] * Rx[c][b];
        }
    for (int a = 0; a < 3; ++a)                               /* R = Rz Ry Rx  (Eq. 3) */
        for (int b = 0; b < 3; ++b) {
            R[a][b] = 0.0;
            for (int c = 0; c < 3; ++c) R[a][b] += Rz[a][c] * T[c][b];
        }
    double inv2s2[3];
    for (int j = 0; j < 3; ++j) {
        const double s = sigma_of(fwhm[j]);
        inv2s2[j] = s > 0.0 ? 1.0 / (2.0 * s * s) : 0.0;      /* F5: axis with r_j = 0 has the single offset 0 */
    }
    double sum = 0.0;
    size_t n = 0;
    for (int k = -r[2]; k <= r[2]; ++k)
        for (int j = -r[1]; j <= r[1]; ++j)
            for (int i = -r[0]; i <= r[0]; ++i) {
                const double p[3] = {(double)i, (double)j, (double)k};
                double q[3];                                  /* q = R^-1 p = R^T p  (reading F4) */
                for (int a = 0; a < 3; ++a) q[a] = R[0][a] * p[0] + R[1][a] * p[1] + R[2][a] * p[2];
                const double g = exp(-(q[0] * q[0] * inv2s2[0] + q[1] * q[1] * inv2s2[1] + q[2] * q[2] * inv2s2[2]));
                kern[n++] = g;                                /* Eq. 1 with A = 1 */
                sum += g;
            }
    for (size_t m = 0; m < n; ++m) kern[m] /= sum;            /* reading F2 */
    return 0;
}

/* Direct 3-D convolution of the cube with the kernel above; reading F1 at the faces. */
int gaussian_oracle_f64(const double *in, int nx, int ny, int nz, const double fwhm[3],
                        const double theta_deg[3], double *out)
{
    if (!in || !out || in == out || nx < 1 || ny < 1 || nz < 1) return -1;
    int r[3];
    if (gaussian_radii_oracle(fwhm, theta_deg, r) != 0) return -1;
    const int wx = 2 * r[0] + 1, wy = 2 * r[1] + 1, wz = 2 * r[2] + 1;
    double *kern = (double *)malloc(sizeof(double) * (size_t)wx * (size_t)wy * (size_t)wz);
    if (!kern) return -2;
    if (gaussian_kernel_oracle(fwhm, theta_deg, r, kern) != 0) { free(kern); return -1; }
    const size_t sy = (size_t)nx, sz = (size_t)nx * (size_t)ny;
    long z;
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                double s = 0.0;
                size_t m = 0;
                /* the kernel is even (G(-p) = G(p)), so convolution and correlation coincide */
                for (int k = -r[2]; k <= r[2]; ++k)
                    for (int j = -r[1]; j <= r[1]; ++j)
                        for (int i = -r[0]; i <= r[0]; ++i)
                            s += kern[m++] * in[(size_t)clampi(x - i, nx) + sy * (size_t)clampi(y - j, ny) +
                                                sz * (size_t)clampi((int)z - k, nz)];
                out[(size_t)x + sy * (size_t)y + sz * (size_t)z] = s;
            }
    free(kern);
    return 0;
}
