/*
 * oracle/idg_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of the intensity-driven gradient (IDG)
 * filter of Punzo, van der Hulst & Roerdink (arXiv:1609.03782), written from
 * PAPER.md section 3.3 only.  It shares no code with the CUDA path under
 * paper_1609_03782_b200/csrc/ and neither includes the other.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call it.
 *
 * What it computes (Eq. 7), for every voxel, n times:
 *
 *     I_{i+1} = I_i + tau * (Cx*Dx I_i + Cy*Dy I_i + Cz*Dz I_i)
 *                           / (1 + I_i^2 / (K^2 rms^2))
 *
 * with the nearest-neighbour differences of PAPER.md:185-187
 *
 *     Dx I = [I(x+1,y,z) - I(x,y,z)] + [I(x-1,y,z) - I(x,y,z)]   (same for y, z)
 *
 * and the conductance of PAPER.md:178 (Eq. 6) evaluated at the centre voxel of
 * the current iterate.  "n times" is read as exactly n updates.
 *
 * Readings where the paper is silent:
 *   R1  boundary: an out-of-cube neighbour is replaced by the centre voxel, so
 *       that difference is zero (zero-flux by replication).
 *   R2  update order: Jacobi -- every read of iteration i comes from I_i; two
 *       buffers, as in the paper's memory scheme.
 *   R3  rms is a caller-supplied constant, never re-estimated.
 *   R4  K = +infinity means conductance 1 (linear diffusion limit).
 *
 * Layout: idx = x + nx*(y + ny*z); x = RA (fastest), y = Dec, z = velocity.
 *
 * The one `omp parallel for` over z only distributes independent voxels of
 * one Jacobi sweep; it does not change any arithmetic or its order per voxel.
 */
#include <math.h>
#include <stddef.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* One Jacobi sweep A -> B (Eq. 7). */
static void idg_sweep(const double *A, double *B, int nx, int ny, int nz,
                      double K, double tau, double Cx, double Cy, double Cz,
                      double rms)
{
    const size_t sy = (size_t)nx, sz = (size_t)nx * (size_t)ny;
    long z;
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (z = 0; z < nz; ++z) {
        for (int y = 0; y < ny; ++y) {
            for (int x = 0; x < nx; ++x) {
                const size_t i = (size_t)x + sy * (size_t)y + sz * (size_t)z;
                const double c = A[i];
                /* R1: out-of-cube neighbour := centre voxel */
                const double xm = (x > 0)      ? A[i - 1]  : c;
                const double xp = (x < nx - 1) ? A[i + 1]  : c;
                const double ym = (y > 0)      ? A[i - sy] : c;
                const double yp = (y < ny - 1) ? A[i + sy] : c;
                const double zm = (z > 0)      ? A[i - sz] : c;
                const double zp = (z < nz - 1) ? A[i + sz] : c;
                /* PAPER.md:187 nearest-neighbour differences */
                const double Dx = (xp - c) + (xm - c);
                const double Dy = (yp - c) + (ym - c);
                const double Dz = (zp - c) + (zm - c);
                /* PAPER.md:178 Eq. 6, centre voxel, current iterate; R4 */
                const double S = isinf(K) ? 1.0
                               : 1.0 / (1.0 + (c * c) / (K * K * rms * rms));
                /* PAPER.md:183 Eq. 7 */
                B[i] = c + tau * (Cx * Dx + Cy * Dy + Cz * Dz) * S;
            }
        }
    }
}

/*
 * n Jacobi sweeps starting from `in` (fp64).  `out` receives I_n.  `scratch`
 * is a second cube of the same size.  in may equal out.  n = 0 copies.
 * Returns 0, or -1 on a bad argument.
 */
int idg_oracle_f64(const double *in, int nx, int ny, int nz, int n,
                   double K, double tau, double Cx, double Cy, double Cz,
                   double rms, double *out, double *scratch)
{
    if (!in || !out || !scratch || nx < 1 || ny < 1 || nz < 1 || n < 0)
        return -1;
    const size_t N = (size_t)nx * (size_t)ny * (size_t)nz;
    if (in != out)
        memcpy(out, in, N * sizeof(double));
    double *A = out, *B = scratch;
    for (int i = 0; i < n; ++i) {
        idg_sweep(A, B, nx, ny, nz, K, tau, Cx, Cy, Cz, rms);
        double *t = A; A = B; B = t;
    }
    if (A != out)
        memcpy(out, A, N * sizeof(double));
    return 0;
}

/*
 * Gradient-driven variant: the classic Perona-Malik conductance of PAPER.md:172-174 (Eq. 5) in the
 * discretisation of Eq. 7:
 *
 *     I_{i+1} = I_i + tau * (Cx*Dx I_i + Cy*Dy I_i + Cz*Dz I_i) / (1 + |grad I_i|^2 / (K^2 rms^2))
 *
 * Readings (P1-P3): |grad I|^2 is the sum over the three axes of the squared
 * central difference [I(+1) - I(-1)] / 2 of the same six neighbours, evaluated at the voxel, with the
 * replicated faces of R1; K is in units of rms per voxel, so that Eq. 5's K^2 reads K^2 rms^2 and the
 * parameter has the meaning it has in Eq. 6; everything else (tau, C_j, Jacobi, n updates) as Eq. 7.
 */
static void pm_sweep(const double *A, double *B, int nx, int ny, int nz,
                     double K, double tau, double Cx, double Cy, double Cz, double rms)
{
    const size_t sy = (size_t)nx, sz = (size_t)nx * (size_t)ny;
    long z;
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (z = 0; z < nz; ++z) {
        for (int y = 0; y < ny; ++y) {
            for (int x = 0; x < nx; ++x) {
                const size_t i = (size_t)x + sy * (size_t)y + sz * (size_t)z;
                const double c = A[i];
                const double xm = (x > 0)      ? A[i - 1]  : c;
                const double xp = (x < nx - 1) ? A[i + 1]  : c;
                const double ym = (y > 0)      ? A[i - sy] : c;
                const double yp = (y < ny - 1) ? A[i + sy] : c;
                const double zm = (z > 0)      ? A[i - sz] : c;
                const double zp = (z < nz - 1) ? A[i + sz] : c;
                const double Dx = (xp - c) + (xm - c);
                const double Dy = (yp - c) + (ym - c);
                const double Dz = (zp - c) + (zm - c);
                const double gx = 0.5 * (xp - xm), gy = 0.5 * (yp - ym), gz = 0.5 * (zp - zm);
                const double g2 = gx * gx + gy * gy + gz * gz;             /* |grad I|^2 */
                const double S = isinf(K) ? 1.0 : 1.0 / (1.0 + g2 / (K * K * rms * rms));   /* Eq. 5 */
                B[i] = c + tau * (Cx * Dx + Cy * Dy + Cz * Dz) * S;
            }
        }
    }
}

int pm_oracle_f64(const double *in, int nx, int ny, int nz, int n,
                  double K, double tau, double Cx, double Cy, double Cz,
                  double rms, double *out, double *scratch)
{
    if (!in || !out || !scratch || nx < 1 || ny < 1 || nz < 1 || n < 0)
        return -1;
    const size_t N = (size_t)nx * (size_t)ny * (size_t)nz;
    if (in != out)
        memcpy(out, in, N * sizeof(double));
    double *A = out, *B = scratch;
    for (int i = 0; i < n; ++i) {
        pm_sweep(A, B, nx, ny, nz, K, tau, Cx, Cy, Cz, rms);
        double *t = A; A = B; B = t;
    }
    if (A != out)
        memcpy(out, A, N * sizeof(double));
    return 0;
}

/* Thread control for the timed CPU baseline (no effect on results). */
int idg_oracle_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
    return omp_get_max_threads();
#else
    (void)n;
    return 1;
#endif
}
