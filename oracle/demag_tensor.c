/*
 * oracle/demag_tensor.c  --  TEST INFRASTRUCTURE, not product code.
 *
 * Cell-averaged demagnetisation tensor N_ij(R) between two equal cuboid cells,
 * i.e. Eq. (2) of the paper (section 2.1.1) integrated over a source
 * cell and averaged over an observation cell:
 *
 *     H_ms(r_i) = - sum_j  N(r_i - r_j) . M_j
 *
 * The paper prints no closed form (reading A1); the closed form used is
 * the classical one for uniformly magnetised cuboids, written as a second
 * difference (weights 1,-2,1 along each axis = 27 points) of two auxiliary
 * functions f (diagonal) and g (off-diagonal).  Everything here is evaluated in
 * __float128 because the 27-point sum cancels catastrophically at long range
 * (terms ~R^3, result ~R^-3); fp64 is only the type of the returned values.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may load
 * this file.  It shares no code, header or table with the CUDA library.
 *
 * Pins (tests/test_oracle_tensor.py): cube self terms = 1/3, trace(0) = 1,
 * trace(R != 0) = 0, parity of each component, far field -> point dipole,
 * coarse-graining identity (a 2x1x1 block cell = average over fine-cell pairs),
 * an independent numerical quadrature of the defining 6-fold integral reduced
 * to surface-charge form.
 */
#include <quadmath.h>
#include <stdlib.h>
#include <string.h>

typedef __float128 real;

static real sq(real x) { return x * x; }

/* f(x,y,z): generator of the diagonal component N_xx.  Even in x, y, z.
 * Every term whose prefactor vanishes is taken as 0 (also at R = 0). */
static real newell_f(real x, real y, real z)
{
    x = fabsq(x); y = fabsq(y); z = fabsq(z);
    real x2 = x * x, y2 = y * y, z2 = z * z;
    real R = sqrtq(x2 + y2 + z2);
    real r = 0;
    if (y != 0 && (x2 + z2) != 0 && (z2 - x2) != 0)
        r += (y / 2) * (z2 - x2) * asinhq(y / sqrtq(x2 + z2));
    if (z != 0 && (x2 + y2) != 0 && (y2 - x2) != 0)
        r += (z / 2) * (y2 - x2) * asinhq(z / sqrtq(x2 + y2));
    if (x != 0 && y != 0 && z != 0)
        r -= x * y * z * atanq(y * z / (x * R));
    r += (2 * x2 - y2 - z2) * R / 6;
    return r;
}

/* g(x,y,z): generator of the off-diagonal component N_xy.  Odd in x, odd in y,
 * even in z. */
static real newell_g(real x, real y, real z)
{
    real sgn = 1;
    if (x < 0) { x = -x; sgn = -sgn; }
    if (y < 0) { y = -y; sgn = -sgn; }
    z = fabsq(z);
    real x2 = x * x, y2 = y * y, z2 = z * z;
    real R = sqrtq(x2 + y2 + z2);
    real r = 0;
    if (x == 0 || y == 0) return 0;              /* odd in x and in y */
    if (z != 0)
        r += x * y * z * asinhq(z / sqrtq(x2 + y2));
    if ((3 * z2 - y2) != 0)
        r += (y / 6) * (3 * z2 - y2) * asinhq(x / sqrtq(y2 + z2));
    if ((3 * z2 - x2) != 0)
        r += (x / 6) * (3 * z2 - x2) * asinhq(y / sqrtq(x2 + z2));
    if (z != 0) {
        r -= (z * z2 / 6) * atanq(x * y / (z * R));
        r -= (z * y2 / 2) * atanq(x * z / (y * R));
        r -= (z * x2 / 2) * atanq(y * z / (x * R));
    }
    r -= x * y * R / 3;
    return sgn * r;
}

/* 27-point second difference  sum_{i,j,k in {-1,0,1}} w_i w_j w_k F(X+i dx, Y+j dy, Z+k dz),
 * w_0 = -2, w_{+-1} = 1, divided by -(4 pi dx dy dz). */
static const real W3[3] = { 1, -2, 1 };

static real stencil27(real (*F)(real, real, real), int perm,
                      real X, real Y, real Z, real dx, real dy, real dz)
{
    real s = 0;
    for (int i = -1; i <= 1; ++i)
        for (int j = -1; j <= 1; ++j)
            for (int k = -1; k <= 1; ++k) {
                real x = X + i * dx, y = Y + j * dy, z = Z + k * dz, v;
                switch (perm) {              /* argument order for each component */
                case 0: v = F(x, y, z); break;   /* xx: f(x,y,z)   xy: g(x,y,z) */
                case 1: v = F(y, x, z); break;   /* yy: f(y,x,z)                */
                case 2: v = F(z, y, x); break;   /* zz: f(z,y,x)                */
                case 3: v = F(x, z, y); break;   /* xz: g(x,z,y)                */
                default: v = F(y, z, x); break;  /* yz: g(y,z,x)                */
                }
                s += W3[i + 1] * W3[j + 1] * W3[k + 1] * v;
            }
    return -s / (4 * M_PIq * dx * dy * dz);
}

/* N at one offset; out = (xx, yy, zz, xy, xz, yz). */
static void tensor_at(real X, real Y, real Z, real dx, real dy, real dz, real out[6])
{
    out[0] = stencil27(newell_f, 0, X, Y, Z, dx, dy, dz);
    out[1] = stencil27(newell_f, 1, X, Y, Z, dx, dy, dz);
    out[2] = stencil27(newell_f, 2, X, Y, Z, dx, dy, dz);
    out[3] = stencil27(newell_g, 0, X, Y, Z, dx, dy, dz);
    out[4] = stencil27(newell_g, 3, X, Y, Z, dx, dy, dz);
    out[5] = stencil27(newell_g, 4, X, Y, Z, dx, dy, dz);
}

/* ---- exported (ctypes) -------------------------------------------------- */

/* N at n integer cell offsets (off[3*i..]) for cell size (dx,dy,dz); out[6*i..].
 * If nimg[a] > 0 the periodic images -nimg[a]..nimg[a] along axis a, spaced by
 * period[a] cells, are summed (reading A8). */
void oracle_tensor_at(long n, const long *off, const double *cell,
                      const int *nimg, const long *period, double *out)
{
    real dx = cell[0], dy = cell[1], dz = cell[2];
#pragma omp parallel for schedule(dynamic, 16)
    for (long i = 0; i < n; ++i) {
        real acc[6] = { 0, 0, 0, 0, 0, 0 };
        for (long a = -nimg[0]; a <= nimg[0]; ++a)
            for (long b = -nimg[1]; b <= nimg[1]; ++b)
                for (long c = -nimg[2]; c <= nimg[2]; ++c) {
                    real t[6];
                    tensor_at((off[3 * i + 0] + a * period[0]) * dx,
                              (off[3 * i + 1] + b * period[1]) * dy,
                              (off[3 * i + 2] + c * period[2]) * dz, dx, dy, dz, t);
                    for (int q = 0; q < 6; ++q) acc[q] += t[q];
                }
        for (int q = 0; q < 6; ++q) out[6 * i + q] = (double)acc[q];
    }
}

/* N on the whole non-negative octant lattice 0<=i<nx, 0<=j<ny, 0<=k<nz of cell
 * offsets: out[q][k][j][i], q = xx,yy,zz,xy,xz,yz.  Same definition as above;
 * the only difference is that each generator is evaluated once per lattice
 * point (-1..n) and the 27-point difference is then taken from that table, so
 * that large grids are affordable in __float128.  tests pin it to
 * oracle_tensor_at. */
void oracle_tensor_octant(long nx, long ny, long nz, const double *cell, double *out)
{
    real dx = cell[0], dy = cell[1], dz = cell[2];
    long lx = nx + 2, ly = ny + 2, lz = nz + 2;
    size_t npts = (size_t)lx * ly * lz;
    real *tab = (real *)malloc(npts * sizeof(real));
    for (int q = 0; q < 6; ++q) {
#pragma omp parallel for schedule(static)
        for (long k = 0; k < lz; ++k)
            for (long j = 0; j < ly; ++j)
                for (long i = 0; i < lx; ++i) {
                    real x = (i - 1) * dx, y = (j - 1) * dy, z = (k - 1) * dz, v;
                    switch (q) {
                    case 0: v = newell_f(x, y, z); break;
                    case 1: v = newell_f(y, x, z); break;
                    case 2: v = newell_f(z, y, x); break;
                    case 3: v = newell_g(x, y, z); break;
                    case 4: v = newell_g(x, z, y); break;
                    default: v = newell_g(y, z, x); break;
                    }
                    tab[((size_t)k * ly + j) * lx + i] = v;
                }
#pragma omp parallel for schedule(static)
        for (long k = 0; k < nz; ++k)
            for (long j = 0; j < ny; ++j)
                for (long i = 0; i < nx; ++i) {
                    real s = 0;
                    for (int c = 0; c < 3; ++c)
                        for (int b = 0; b < 3; ++b)
                            for (int a = 0; a < 3; ++a)
                                s += W3[a] * W3[b] * W3[c] *
                                     tab[((size_t)(k + c) * ly + (j + b)) * lx + (i + a)];
                    out[(((size_t)q * nz + k) * ny + j) * nx + i] =
                        (double)(-s / (4 * M_PIq * dx * dy * dz));
                }
    }
    free(tab);
}
