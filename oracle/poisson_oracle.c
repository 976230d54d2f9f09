/*
 * CPU ORACLE for the open-boundary FFT Poisson solve of arXiv:1509.07685 (DKS, part 1).
 *
 * THIS IS TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it.  It shares no code,
 * header, table or constant with the CUDA path under paper_1509_07685_b200/csrc and is
 * written to be checked against the paper by eye: plain, slow, textbook.
 *
 * What it computes (section 3.1.1, Eq. (2)):
 *     phi[i,j,k] = hx*hy*hz * sum_{i',j',k'} rho[i',j',k'] * G((i-i')hx, (j-j')hy, (k-k')hz)
 * by the route the paper states (section 3.1.1, unnumbered equation after Eq. (2)):
 *     phi = hx*hy*hz * FT^-1{ FT{rho} (x) FT{G} }            ((x) = Hadamard product)
 * on Hockney's doubled grid 2Mx x 2My x 2Mz (section 3.1).
 *
 * Readings of the paper:
 *   A1  G(u,v,w) = 1/(4*pi*eps0*sqrt(u^2+v^2+w^2)); PAPER.md:117 prints 1/sqrt(...) only, but
 *       the PDE is laplace(phi) = -rho/eps0.  eps0 = 8.8541878128e-12 F/m.
 *   A2  G(0,0,0) = g0 is an argument (callers use 1/(4 pi eps0 r0), r0 = min(h)/2).
 *   A4  doubled-grid Green's function: periodic mirror i' = min(i, 2n-i) per axis.
 *   A5  forward transform e^{-i theta} unnormalised, inverse e^{+i theta} with 1/(8 nx ny nz).
 *
 * Algorithm, deliberately un-optimised (full doubled grid, complex-to-complex, no pruning,
 * no symmetry, no folded constants):
 *   1. R[2nz][2ny][2nx] = 0; copy rho into the low corner.
 *   2. Gt[k][j][i] = G(i'hx, j'hy, k'hz) with the mirror rule; Gt[0][0][0] = g0.
 *   3. 3-D forward DFT of R and Gt: 1-D transforms along x, then y, then z, each a plain
 *      recursive radix-2 FFT whose twiddles come from cos/sin(2 pi k / L) evaluated per entry.
 *   4. R <- R (x) Gt (complex multiply).
 *   5. 3-D inverse DFT of R, divide by 8 nx ny nz.
 *   6. phi = hx*hy*hz * Re R on the low corner; max|Im R| is reported (must be ~0).
 *
 * Built twice from this file: -DORACLE_LD (REAL = long double, x87 80-bit: the parity
 * reference values) and without (REAL = double: the timed CPU baseline).  OpenMP runs
 * independent 1-D lines in parallel; nothing else is parallel.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): direct summation of Eq. (2) on tiny meshes
 * and at sampled nodes of every config, single point charge = q*G(r) (incl. no wrap-around),
 * linearity, mirror / axis-permutation symmetry, translation, independence from the Gt values
 * on the planes i=nx/j=ny/k=nz, Im ~ 0, Ghat real and even, positivity, continuum sphere,
 * 1-D FFT vs O(L^2) DFT, numpy.fft as a third opinion.  Parity is therefore pinned.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifdef ORACLE_LD
typedef long double REAL;
#define R_COS cosl
#define R_SIN sinl
#define R_SQRT sqrtl
#define R_FABS fabsl
#define FN(name) oracle_ld_##name
#else
typedef double REAL;
#define R_COS cos
#define R_SIN sin
#define R_SQRT sqrt
#define R_FABS fabs
#define FN(name) oracle_d_##name
#endif

typedef struct { REAL re, im; } cplx;

/* pi and eps0 as long double literals; eps0 is CODATA 2018 (reading A1). */
#define ORACLE_PI   3.14159265358979323846264338327950288L
#define ORACLE_EPS0 8.8541878128e-12L

/* ------------------------------------------------------------------------------------------
 * 1-D transforms
 * ---------------------------------------------------------------------------------------- */

/* Twiddle table for length L: tw[k] = exp(sign * 2 pi i k / L), k = 0..L/2-1, each entry from
 * cos/sin directly (no recurrence). */
static cplx *make_twiddles(int L, int sign)
{
    int half = L / 2 > 0 ? L / 2 : 1;
    cplx *tw = (cplx *)malloc(sizeof(cplx) * (size_t)half);
    for (int k = 0; k < half; ++k) {
        REAL th = (REAL)(2.0L * ORACLE_PI * (long double)k / (long double)L);
        tw[k].re = R_COS(th);
        tw[k].im = (REAL)sign * R_SIN(th);
    }
    return tw;
}

/* Textbook recursive radix-2 decimation-in-time FFT.
 * in: L samples at stride `stride`; out: L contiguous results; tw: table for the TOP length,
 * tstep = (top length)/L so that tw[k*tstep] = exp(sign 2 pi i k / L).  L must be a power of two. */
static void fft_rec(const cplx *in, cplx *out, int L, int stride, const cplx *tw, int tstep)
{
    if (L == 1) { out[0] = in[0]; return; }
    int half = L / 2;
    fft_rec(in, out, half, 2 * stride, tw, 2 * tstep);                 /* even samples */
    fft_rec(in + stride, out + half, half, 2 * stride, tw, 2 * tstep); /* odd samples  */
    for (int k = 0; k < half; ++k) {
        cplx w = tw[k * tstep];
        cplx o = out[k + half];
        cplx e = out[k];
        cplx t;
        t.re = w.re * o.re - w.im * o.im;
        t.im = w.re * o.im + w.im * o.re;
        out[k].re = e.re + t.re;        out[k].im = e.im + t.im;
        out[k + half].re = e.re - t.re; out[k + half].im = e.im - t.im;
    }
}

/* exported for pin P11: FFT of one line (double in/out, REAL inside); sign = -1 forward, +1 inverse
 * (unnormalised either way). */
void FN(fft1d)(const double *in_re, const double *in_im, double *out_re, double *out_im, int L, int sign)
{
    cplx *a = (cplx *)malloc(sizeof(cplx) * (size_t)L), *b = (cplx *)malloc(sizeof(cplx) * (size_t)L);
    cplx *tw = make_twiddles(L, sign);
    for (int i = 0; i < L; ++i) { a[i].re = (REAL)in_re[i]; a[i].im = (REAL)in_im[i]; }
    fft_rec(a, b, L, 1, tw, 1);
    for (int i = 0; i < L; ++i) { out_re[i] = (double)b[i].re; out_im[i] = (double)b[i].im; }
    free(a); free(b); free(tw);
}

/* exported for pin P11: the O(L^2) definition X[k] = sum_j x[j] exp(sign 2 pi i j k / L), any L. */
void FN(dft1d)(const double *in_re, const double *in_im, double *out_re, double *out_im, int L, int sign)
{
    for (int k = 0; k < L; ++k) {
        REAL sr = 0, si = 0;
        for (int j = 0; j < L; ++j) {
            long long jk = ((long long)j * (long long)k) % L;
            REAL th = (REAL)(2.0L * ORACLE_PI * (long double)jk / (long double)L);
            REAL c = R_COS(th), s = (REAL)sign * R_SIN(th);
            sr += (REAL)in_re[j] * c - (REAL)in_im[j] * s;
            si += (REAL)in_re[j] * s + (REAL)in_im[j] * c;
        }
        out_re[k] = (double)sr; out_im[k] = (double)si;
    }
}

/* ------------------------------------------------------------------------------------------
 * 3-D transform on an array a[d2][d1][d0] (d0 fastest): 1-D transforms along axis 0, 1, 2.
 * ---------------------------------------------------------------------------------------- */
static void fft_axis(cplx *a, size_t d0, size_t d1, size_t d2, int axis, int sign)
{
    size_t dims[3] = { d0, d1, d2 };
    size_t strides[3] = { 1, d0, d0 * d1 };
    int L = (int)dims[axis];
    size_t s = strides[axis];
    int ax1 = (axis + 1) % 3, ax2 = (axis + 2) % 3;
    size_t n1 = dims[ax1], n2 = dims[ax2], s1 = strides[ax1], s2 = strides[ax2];
    cplx *tw = make_twiddles(L, sign);
    long long nlines = (long long)(n1 * n2);
#pragma omp parallel
    {
        cplx *line = (cplx *)malloc(sizeof(cplx) * (size_t)L);
        cplx *res = (cplx *)malloc(sizeof(cplx) * (size_t)L);
#pragma omp for schedule(static)
        for (long long l = 0; l < nlines; ++l) {
            size_t i1 = (size_t)l % n1, i2 = (size_t)l / n1;
            cplx *base = a + i1 * s1 + i2 * s2;
            for (int i = 0; i < L; ++i) line[i] = base[(size_t)i * s];
            fft_rec(line, res, L, 1, tw, 1);
            for (int i = 0; i < L; ++i) base[(size_t)i * s] = res[i];
        }
        free(line); free(res);
    }
    free(tw);
}

static void fft3d(cplx *a, size_t d0, size_t d1, size_t d2, int sign)
{
    fft_axis(a, d0, d1, d2, 0, sign);   /* x */
    fft_axis(a, d0, d1, d2, 1, sign);   /* y */
    fft_axis(a, d0, d1, d2, 2, sign);   /* z */
}

/* ------------------------------------------------------------------------------------------
 * Green's function, PAPER.md:117 with reading A1
 * ---------------------------------------------------------------------------------------- */
static REAL green(REAL u, REAL v, REAL w)
{
    REAL r = R_SQRT(u * u + v * v + w * w);
    return (REAL)(1.0L / (4.0L * ORACLE_PI * ORACLE_EPS0)) / r;
}

/* exported: G at (u,v,w) != 0, for the point-charge and sphere pins */
double FN(green)(double u, double v, double w) { return (double)green((REAL)u, (REAL)v, (REAL)w); }

/* Step 2.  Gt[2nz][2ny][2nx], mirror rule A4.  plane_value: if it is not NaN, the entries with
 * i == nx or j == ny or k == nz (never addressed by an (output, source) pair) are set to it instead
 * of the mirror value: pin P7. */
static void build_greens(cplx *Gt, int nx, int ny, int nz, REAL hx, REAL hy, REAL hz, REAL g0, double plane_value)
{
    size_t X = 2 * (size_t)nx, Y = 2 * (size_t)ny, Z = 2 * (size_t)nz;
    int use_plane = !(plane_value != plane_value);
#pragma omp parallel for schedule(static)
    for (long long k = 0; k < (long long)Z; ++k) {
        int kp = (int)(k <= nz ? k : (long long)Z - k);
        for (size_t j = 0; j < Y; ++j) {
            int jp = (int)(j <= (size_t)ny ? j : Y - j);
            for (size_t i = 0; i < X; ++i) {
                int ip = (int)(i <= (size_t)nx ? i : X - i);
                cplx *g = &Gt[((size_t)k * Y + j) * X + i];
                g->im = 0;
                if (ip == 0 && jp == 0 && kp == 0) g->re = g0;
                else if (use_plane && ((int)i == nx || (int)j == ny || (int)k == nz)) g->re = (REAL)plane_value;
                else g->re = green((REAL)ip * hx, (REAL)jp * hy, (REAL)kp * hz);
            }
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * Opaque handle holding FT{Gt} so that a solve with the transform precomputed can be timed
 * (what dks_poisson_solve covers; reading A11).
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    int nx, ny, nz;
    REAL hx, hy, hz;
    cplx *Ghat;   /* FT{Gt}, [2nz][2ny][2nx] */
    cplx *R;      /* work array, same shape   */
} oracle_plan;

void *FN(plan_create)(int nx, int ny, int nz, double hx, double hy, double hz, double g0, double plane_value)
{
    oracle_plan *p = (oracle_plan *)calloc(1, sizeof(oracle_plan));
    size_t N = 8 * (size_t)nx * (size_t)ny * (size_t)nz;
    p->nx = nx; p->ny = ny; p->nz = nz; p->hx = (REAL)hx; p->hy = (REAL)hy; p->hz = (REAL)hz;
    p->Ghat = (cplx *)malloc(sizeof(cplx) * N);
    p->R = (cplx *)malloc(sizeof(cplx) * N);
    if (!p->Ghat || !p->R) { free(p->Ghat); free(p->R); free(p); return NULL; }
    build_greens(p->Ghat, nx, ny, nz, p->hx, p->hy, p->hz, (REAL)g0, plane_value);   /* step 2 */
    fft3d(p->Ghat, 2 * (size_t)nx, 2 * (size_t)ny, 2 * (size_t)nz, -1);                /* step 3 (G) */
    return p;
}

void FN(plan_destroy)(void *vp)
{
    oracle_plan *p = (oracle_plan *)vp;
    if (!p) return;
    free(p->Ghat); free(p->R); free(p);
}

/* Pin P8: max |Im Ghat|, max |Ghat|, and the largest defect of evenness |Ghat[k] - Ghat[-k]| per axis. */
void FN(plan_ghat_stats)(void *vp, double *max_im, double *max_abs, double *max_even_defect)
{
    oracle_plan *p = (oracle_plan *)vp;
    size_t X = 2 * (size_t)p->nx, Y = 2 * (size_t)p->ny, Z = 2 * (size_t)p->nz;
    REAL mi = 0, ma = 0, me = 0;
    for (size_t k = 0; k < Z; ++k) for (size_t j = 0; j < Y; ++j) for (size_t i = 0; i < X; ++i) {
        cplx g = p->Ghat[(k * Y + j) * X + i];
        REAL a = R_SQRT(g.re * g.re + g.im * g.im);
        if (R_FABS(g.im) > mi) mi = R_FABS(g.im);
        if (a > ma) ma = a;
        cplx gx = p->Ghat[(k * Y + j) * X + (X - i) % X];
        cplx gy = p->Ghat[(k * Y + (Y - j) % Y) * X + i];
        cplx gz = p->Ghat[(((Z - k) % Z) * Y + j) * X + i];
        REAL d = R_FABS(g.re - gx.re); if (d > me) me = d;
        d = R_FABS(g.re - gy.re); if (d > me) me = d;
        d = R_FABS(g.re - gz.re); if (d > me) me = d;
    }
    *max_im = (double)mi; *max_abs = (double)ma; *max_even_defect = (double)me;
}

/* Accessor (no arithmetic): Re FT{Gt}[k][j][i] on the octant k <= nz, j <= ny, i <= nx of the doubled grid, as
 * [nz+1][ny+1][nx+1] doubles.  FT{Gt} is real and even (pin P8), so the octant carries the whole transform; tests
 * compare the CUDA path's Green's octant (step a0) with this directly. */
void FN(plan_ghat_octant)(void *vp, double *out)
{
    oracle_plan *p = (oracle_plan *)vp;
    size_t X = 2 * (size_t)p->nx, Y = 2 * (size_t)p->ny;
    for (int k = 0; k <= p->nz; ++k) for (int j = 0; j <= p->ny; ++j) for (int i = 0; i <= p->nx; ++i)
        out[((size_t)k * (p->ny + 1) + j) * (p->nx + 1) + i] = (double)p->Ghat[((size_t)k * Y + j) * X + i].re;
}

/* Steps 1, 3 (rho), 4, 5, 6.  rho, phi: [nz][ny][nx] doubles, x fastest.  Returns max |Im R| over the
 * low corner after step 5, relative to max |Re R| there (0 if phi == 0). */
double FN(plan_solve)(void *vp, const double *rho, double *phi)
{
    oracle_plan *p = (oracle_plan *)vp;
    int nx = p->nx, ny = p->ny, nz = p->nz;
    size_t X = 2 * (size_t)nx, Y = 2 * (size_t)ny, Z = 2 * (size_t)nz, N = X * Y * Z;
    cplx *R = p->R;
    /* step 1 */
    memset(R, 0, sizeof(cplx) * N);
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i)
        R[((size_t)k * Y + (size_t)j) * X + (size_t)i].re = (REAL)rho[((size_t)k * ny + j) * nx + i];
    /* step 3 */
    fft3d(R, X, Y, Z, -1);
    /* step 4 */
#pragma omp parallel for schedule(static)
    for (long long q = 0; q < (long long)N; ++q) {
        cplx a = R[q], g = p->Ghat[q], r;
        r.re = a.re * g.re - a.im * g.im;
        r.im = a.re * g.im + a.im * g.re;
        R[q] = r;
    }
    /* step 5 */
    fft3d(R, X, Y, Z, +1);
    REAL inv = (REAL)1 / (REAL)N;       /* N = 8 nx ny nz */
    /* step 6 */
    REAL hv = p->hx * p->hy * p->hz, mre = 0, mim = 0;
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
        cplx r = R[((size_t)k * Y + (size_t)j) * X + (size_t)i];
        REAL re = r.re * inv, im = r.im * inv;
        phi[((size_t)k * ny + j) * nx + i] = (double)(hv * re);
        if (R_FABS(re) > mre) mre = R_FABS(re);
        if (R_FABS(im) > mim) mim = R_FABS(im);
    }
    return mre > 0 ? (double)(mim / mre) : 0.0;
}

/* One-shot: steps 1-6. */
double FN(solve)(int nx, int ny, int nz, double hx, double hy, double hz, double g0, double plane_value,
                 const double *rho, double *phi)
{
    void *p = FN(plan_create)(nx, ny, nz, hx, hy, hz, g0, plane_value);
    if (!p) return -1.0;
    double r = FN(plan_solve)(p, rho, phi);
    FN(plan_destroy)(p);
    return r;
}

/* ------------------------------------------------------------------------------------------
 * Direct summation of Eq. (2): the definition itself, no FFT.  Used to pin the
 * oracle.  nodes: count rows of (i, j, k); out[count].  Accumulates in REAL.
 * ---------------------------------------------------------------------------------------- */
void FN(direct_sum_nodes)(int nx, int ny, int nz, double hx, double hy, double hz, double g0,
                          const double *rho, const long long *nodes, int count, double *out)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int q = 0; q < count; ++q) {
        int i = (int)nodes[3 * q], j = (int)nodes[3 * q + 1], k = (int)nodes[3 * q + 2];
        REAL acc = 0;
        for (int kp = 0; kp < nz; ++kp) for (int jp = 0; jp < ny; ++jp) for (int ip = 0; ip < nx; ++ip) {
            REAL r = (REAL)rho[((size_t)kp * ny + jp) * nx + ip];
            if (r == 0) continue;
            REAL g = (i == ip && j == jp && k == kp) ? (REAL)g0
                     : green((REAL)(i - ip) * (REAL)hx, (REAL)(j - jp) * (REAL)hy, (REAL)(k - kp) * (REAL)hz);
            acc += r * g;
        }
        out[q] = (double)((REAL)hx * (REAL)hy * (REAL)hz * acc);
    }
}

int FN(num_threads)(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
