/*
 * CPU ORACLE for the two steps adjacent to the Poisson solve in the space-charge step of arXiv:1509.07685:
 * the charge deposit that produces rho before the solve and the field E = -grad(phi) (and its interpolation
 * back to the particles) after it.
 *
 * THIS IS TEST INFRASTRUCTURE (same rules as poisson_oracle.c): only tests/, __graft_entry__.smoke() and bench.py's
 * CPU legs may build, load or call it; it shares no code with the CUDA path.
 *
 * What the paper says: OPAL is built on IPPL, which provides "particles with the respective interpolation operators"
 * (section 3); the solver works on a mesh that is fitted to the bunch every time step; the
 * host <-> device transfer of rho and phi costs "up to 55 %" of the total time, which is what moving
 * these two steps onto the device removes.  The paper gives NO formula for either step, so both are readings
 * (F1-F4), written out here step by step:
 *
 *   F1  Positions are physical coordinates; node (i, j, k) sits at origin + (i hx, j hy, k hz); the mesh index of a
 *       particle is u = (X - ox) / hx (one IEEE division), likewise v, w.
 *   F2  Cloud-in-cell (trilinear) deposit: with i = floor(u), f = u - i, the charge q goes to the 8 nodes
 *       (i + di, j + dj, k + dk), di, dj, dk in {0, 1}, with weight prod (di ? f : 1 - f); rho = charge / (hx hy hz).
 *       A particle is DROPPED unless 0 <= u < nx - 1, 0 <= v < ny - 1, 0 <= w < nz - 1 (the rule of the input
 *       generator).
 *   F3  E = -grad(phi) by second-order differences: central in the interior, -(phi[i+1] - phi[i-1]) / (2 hx); one-sided
 *       second order at the two ends, -(-3 phi[0] + 4 phi[1] - phi[2]) / (2 hx) and -(3 phi[n-1] - 4 phi[n-2] + phi[n-3]) / (2 hx).
 *   F4  The field at a particle is the trilinear interpolation of the node values with the weights of F2 (the
 *       adjoint of the deposit); dropped particles get 0.
 *
 * Accumulation is sequential, in REAL (long double in the -DORACLE_LD build), in particle order.
 *
 * Pins (tests/test_field_ops_pins.py, -m "not gpu"): total charge and first moment (dipole) conserved by the deposit;
 * a particle on a node / at a cell centre; the drop rule; superposition; integer translation; agreement with the numpy
 * bincount deposit of the input generator (an independent implementation); gradient exact on linear and quadratic
 * fields including the boundary nodes, second-order convergence on a point-charge potential, sign (E points away from a
 * positive charge); gather exact on constant and trilinear fields; deposit and gather adjoint to each other.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stddef.h>

#ifdef ORACLE_LD
typedef long double REAL;
#define R_FLOOR floorl
#define FN(name) oracle_ld_##name
#else
typedef double REAL;
#define R_FLOOR floor
#define FN(name) oracle_d_##name
#endif

/* F1 + the drop rule of F2: mesh coordinates of a particle; returns 0 if the particle is dropped. */
static int locate(double X, double Y, double Z, double ox, double oy, double oz, double hx, double hy, double hz,
                  int nx, int ny, int nz, long long *i, long long *j, long long *k, REAL *fx, REAL *fy, REAL *fz)
{
    /* the division is done in double on both builds: it is part of the method's input handling (F1) */
    double u = (X - ox) / hx, v = (Y - oy) / hy, w = (Z - oz) / hz;
    if (!(u >= 0.0 && u < (double)(nx - 1) && v >= 0.0 && v < (double)(ny - 1) && w >= 0.0 && w < (double)(nz - 1))) return 0;
    *i = (long long)floor(u); *j = (long long)floor(v); *k = (long long)floor(w);
    *fx = (REAL)u - (REAL)*i; *fy = (REAL)v - (REAL)*j; *fz = (REAL)w - (REAL)*k;
    return 1;
}

/* F2.  x, y, z, q: np doubles each.  rho: [nz][ny][nx] doubles, overwritten.  Returns the number of deposited particles. */
long long FN(cic_deposit)(int nx, int ny, int nz, double hx, double hy, double hz, double ox, double oy, double oz,
                          const double *x, const double *y, const double *z, const double *q, long long np, double *rho)
{
    size_t N = (size_t)nx * ny * nz;
    REAL *acc = (REAL *)calloc(N, sizeof(REAL));
    long long kept = 0;
    for (long long n = 0; n < np; ++n) {
        long long i, j, k; REAL fx, fy, fz;
        if (!locate(x[n], y[n], z[n], ox, oy, oz, hx, hy, hz, nx, ny, nz, &i, &j, &k, &fx, &fy, &fz)) continue;
        ++kept;
        for (int dk = 0; dk < 2; ++dk) for (int dj = 0; dj < 2; ++dj) for (int di = 0; di < 2; ++di) {
            REAL w = (di ? fx : 1 - fx) * (dj ? fy : 1 - fy) * (dk ? fz : 1 - fz);
            acc[((size_t)(k + dk) * ny + (size_t)(j + dj)) * nx + (size_t)(i + di)] += (REAL)q[n] * w;
        }
    }
    REAL vol = (REAL)hx * (REAL)hy * (REAL)hz;
    for (size_t m = 0; m < N; ++m) rho[m] = (double)(acc[m] / vol);
    free(acc);
    return kept;
}

/* F3.  phi, ex, ey, ez: [nz][ny][nx] doubles.  Every extent >= 3. */
static REAL diff2(const double *f, long long i, long long n, size_t stride, REAL h)
{
    if (i == 0) return (-3 * (REAL)f[0] + 4 * (REAL)f[stride] - (REAL)f[2 * stride]) / (2 * h);
    if (i == n - 1) return (3 * (REAL)f[0] - 4 * (REAL)*(f - stride) + (REAL)*(f - 2 * stride)) / (2 * h);
    return ((REAL)f[stride] - (REAL)*(f - stride)) / (2 * h);
}

void FN(gradient)(int nx, int ny, int nz, double hx, double hy, double hz, const double *phi,
                  double *ex, double *ey, double *ez)
{
    for (long long k = 0; k < nz; ++k) for (long long j = 0; j < ny; ++j) for (long long i = 0; i < nx; ++i) {
        size_t m = ((size_t)k * ny + (size_t)j) * nx + (size_t)i;
        ex[m] = (double)(-diff2(phi + m, i, nx, 1, (REAL)hx));
        ey[m] = (double)(-diff2(phi + m, j, ny, (size_t)nx, (REAL)hy));
        ez[m] = (double)(-diff2(phi + m, k, nz, (size_t)nx * ny, (REAL)hz));
    }
}

/* F4.  field: [nz][ny][nx] doubles; out: np doubles (0 for dropped particles). */
void FN(cic_gather)(int nx, int ny, int nz, double hx, double hy, double hz, double ox, double oy, double oz,
                    const double *field, const double *x, const double *y, const double *z, long long np, double *out)
{
    for (long long n = 0; n < np; ++n) {
        long long i, j, k; REAL fx, fy, fz;
        out[n] = 0.0;
        if (!locate(x[n], y[n], z[n], ox, oy, oz, hx, hy, hz, nx, ny, nz, &i, &j, &k, &fx, &fy, &fz)) continue;
        REAL s = 0;
        for (int dk = 0; dk < 2; ++dk) for (int dj = 0; dj < 2; ++dj) for (int di = 0; di < 2; ++di) {
            REAL w = (di ? fx : 1 - fx) * (dj ? fy : 1 - fy) * (dk ? fz : 1 - fz);
            s += w * (REAL)field[((size_t)(k + dk) * ny + (size_t)(j + dj)) * nx + (size_t)(i + di)];
        }
        out[n] = (double)s;
    }
}
