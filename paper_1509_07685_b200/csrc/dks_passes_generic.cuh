// Generic (any power-of-two mesh) kernels for the five passes of the solve and for the Green's
// function setup.  One CTA = one tile of W lines staged in shared memory (dks_fft_generic.cuh).
//
// Axis order: z first (real-to-complex), then y, then x in the middle,
// so that the heaviest pass (forward x, multiply, inverse x) runs on contiguous lines, and the odd
// (nz+1) extent produced by the real-to-complex step is the slowest dimension of every buffer.
//
//   rho [nz][ny][nx] real --P1--> A [nz+1][ny][nx] cplx --P2--> B [nz+1][2ny][nx] cplx
//       --P3 (in place)--> B --P4--> A --P5--> phi [nz][ny][nx] real
//
// Zero padding is never materialised: each forward pass loads only the n non-zero
// entries of its 2n line; each inverse pass stores only the n entries that survive the crop.
#pragma once
#include "dks_fft_generic.cuh"

namespace dks {

struct MeshDims {
    int nx, ny, nz;        // mesh (paper's Mx, My, Mz)
    int lx, ly, lz;        // log2 of the doubled line lengths 2nx, 2ny, 2nz
    int gpitch;            // row pitch (doubles) of the Green's octant
};

// ---------------------------------------------------------------------------------------------
// P1: forward z, real -> complex, two real columns (x, x+1) packed into one complex line.
// grid (nx / (2W), ny); smem 2nz * W complex.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
p1_z_r2c_generic(const double *__restrict__ rho, cplx *__restrict__ A, MeshDims d, int W,
                 const cplx *__restrict__ tw)
{
    extern __shared__ cplx s[];
    const int nx = d.nx, ny = d.ny, nz = d.nz, L = 2 * nz, logL = d.lz;
    const int x0 = blockIdx.x * 2 * W, y = blockIdx.y;
    const int tid = threadIdx.x, nt = blockDim.x;
    rho += (size_t)blockIdx.z * nz * ny * nx;             // blockIdx.z: mesh of the batch
    A += (size_t)blockIdx.z * (nz + 1) * ny * nx;
    for (int idx = tid; idx < nz * W; idx += nt) {
        int r = idx / W, w = idx % W;
        s[r * W + w] = *reinterpret_cast<const cplx *>(&rho[((size_t)r * ny + y) * nx + x0 + 2 * w]);
        s[(r + nz) * W + w] = cmake(0.0, 0.0);
    }
    __syncthreads();
    tile_fft_dif<-1>(s, L, logL, W, W, tw);
    // split the packed transform: C = FT{a + i b}  ->  FT{a}[k] = (C[k] + conj C[-k]) / 2,
    //                                                 FT{b}[k] = (C[k] - conj C[-k]) / (2 i)
    for (int idx = tid; idx < (nz + 1) * W; idx += nt) {
        int k = idx / W, w = idx % W;
        cplx ck = s[brev(k, logL) * W + w];
        cplx cm = s[brev((L - k) & (L - 1), logL) * W + w];
        cplx fa = cmake(0.5 * (ck.x + cm.x), 0.5 * (ck.y - cm.y));
        cplx fb = cmake(0.5 * (ck.y + cm.y), -0.5 * (ck.x - cm.x));
        cplx *out = &A[((size_t)k * ny + y) * nx + x0 + 2 * w];
        out[0] = fa;
        out[1] = fb;
    }
}

// ---------------------------------------------------------------------------------------------
// P5: inverse z, complex -> real (Hermitian extension of two spectra packed into one line), crop.
// grid (nx / (2W), ny)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
p5_z_c2r_generic(const cplx *__restrict__ A, double *__restrict__ phi, MeshDims d, int W,
                 const cplx *__restrict__ tw)
{
    extern __shared__ cplx s[];
    const int nx = d.nx, ny = d.ny, nz = d.nz, L = 2 * nz, logL = d.lz;
    const int x0 = blockIdx.x * 2 * W, y = blockIdx.y;
    const int tid = threadIdx.x, nt = blockDim.x;
    A += (size_t)blockIdx.z * (nz + 1) * ny * nx;         // blockIdx.z: mesh of the batch
    phi += (size_t)blockIdx.z * nz * ny * nx;
    for (int idx = tid; idx < (nz + 1) * W; idx += nt) {
        int k = idx / W, w = idx % W;
        const cplx *in = &A[((size_t)k * ny + y) * nx + x0 + 2 * w];
        cplx fa = in[0], fb = in[1];
        s[brev(k, logL) * W + w] = cmake(fa.x - fb.y, fa.y + fb.x);             // fa + i fb
        if (k > 0 && k < nz)
            s[brev(L - k, logL) * W + w] = cmake(fa.x + fb.y, fb.x - fa.y);     // conj(fa) + i conj(fb)
    }
    __syncthreads();
    tile_fft_dit<+1>(s, L, logL, W, W, tw);
    for (int idx = tid; idx < nz * W; idx += nt) {
        int r = idx / W, w = idx % W;
        *reinterpret_cast<cplx *>(&phi[((size_t)r * ny + y) * nx + x0 + 2 * w]) = s[r * W + w];
    }
}

// ---------------------------------------------------------------------------------------------
// P2: forward y.  grid (nx / W, nz + 1)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
p2_y_fwd_generic(const cplx *__restrict__ A, cplx *__restrict__ B, MeshDims d, int kz0, int W,
                 const cplx *__restrict__ tw)
{
    extern __shared__ cplx s[];
    const int nx = d.nx, ny = d.ny, L = 2 * ny, logL = d.ly;
    const int x0 = blockIdx.x * W, kz = blockIdx.y;
    const int tid = threadIdx.x, nt = blockDim.x;
    for (int idx = tid; idx < ny * W; idx += nt) {
        int r = idx / W, w = idx % W;
        s[r * W + w] = A[((size_t)(kz0 + kz) * ny + r) * nx + x0 + w];
        s[(r + ny) * W + w] = cmake(0.0, 0.0);
    }
    __syncthreads();
    tile_fft_dif<-1>(s, L, logL, W, W, tw);
    for (int idx = tid; idx < L * W; idx += nt) {
        int ky = idx / W, w = idx % W;
        B[((size_t)kz * L + ky) * nx + x0 + w] = s[brev(ky, logL) * W + w];
    }
}

// ---------------------------------------------------------------------------------------------
// P4: inverse y, crop to ny.  grid (nx / W, nz + 1)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
p4_y_inv_generic(const cplx *__restrict__ B, cplx *__restrict__ A, MeshDims d, int kz0, int W,
                 const cplx *__restrict__ tw)
{
    extern __shared__ cplx s[];
    const int nx = d.nx, ny = d.ny, L = 2 * ny, logL = d.ly;
    const int x0 = blockIdx.x * W, kz = blockIdx.y;
    const int tid = threadIdx.x, nt = blockDim.x;
    for (int idx = tid; idx < L * W; idx += nt) {
        int ky = idx / W, w = idx % W;
        s[brev(ky, logL) * W + w] = B[((size_t)kz * L + ky) * nx + x0 + w];
    }
    __syncthreads();
    tile_fft_dit<+1>(s, L, logL, W, W, tw);
    for (int idx = tid; idx < ny * W; idx += nt) {
        int r = idx / W, w = idx % W;
        A[((size_t)(kz0 + kz) * ny + r) * nx + x0 + w] = s[r * W + w];
    }
}

// ---------------------------------------------------------------------------------------------
// P3: forward x, multiply by the Green's transform, inverse x, crop to nx; in place on B.
// One CTA = W consecutive lines (same kz).  grid ((nz+1) * 2ny / W).  smem 2nx * (W+1) complex.
// Ghat is the real octant [(nz+1)][(ny+1)][gpitch] with hx hy hz / (8 nx ny nz) folded in; the full
// spectrum follows from evenness: Ghat(kx, ky, kz) = Ghat(min(kx, 2nx-kx), min(ky, 2ny-ky), kz).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
p3_x_conv_generic(cplx *__restrict__ B, const double *__restrict__ Ghat, MeshDims d, int kz0, int W,
                  const cplx *__restrict__ tw)
{
    extern __shared__ cplx s[];
    const int nx = d.nx, ny = d.ny, L = 2 * nx, logL = d.lx, WP = W + 1;
    const int line0 = blockIdx.x * W;
    const int kz = (kz0 + line0 / (2 * ny)) % (d.nz + 1), ky0 = line0 % (2 * ny);    // line0 counts within the slab; a batch repeats kz
    const int tid = threadIdx.x, nt = blockDim.x;
    cplx *base = B + (size_t)line0 * nx;
    for (int idx = tid; idx < nx * W; idx += nt) {
        int w = idx / nx, p = idx % nx;
        s[p * WP + w] = base[(size_t)w * nx + p];
        s[(p + nx) * WP + w] = cmake(0.0, 0.0);
    }
    __syncthreads();
    tile_fft_dif<-1>(s, L, logL, W, WP, tw);
    for (int idx = tid; idx < L * W; idx += nt) {
        int p = idx / W, w = idx % W;
        int kx = brev(p, logL), ky = ky0 + w;
        int kxp = min(kx, L - kx), kyp = min(ky, 2 * ny - ky);
        double g = __ldg(&Ghat[((size_t)kz * (ny + 1) + kyp) * d.gpitch + kxp]);
        cplx v = s[p * WP + w];
        s[p * WP + w] = cmake(v.x * g, v.y * g);
    }
    __syncthreads();
    tile_fft_dit<+1>(s, L, logL, W, WP, tw);
    for (int idx = tid; idx < nx * W; idx += nt) {
        int w = idx / nx, p = idx % nx;
        base[(size_t)w * nx + p] = s[p * WP + w];
    }
}

// ---------------------------------------------------------------------------------------------
// Green's function setup (step a0).
// ---------------------------------------------------------------------------------------------
// G on the octant of the doubled grid: Goct[k][j][i] = coef / sqrt((i hx)^2 + (j hy)^2 + (k hz)^2),
// coef = 1/(4 pi eps0) (PAPER.md:117 with the constant the PDE at PAPER.md:104 implies); Goct[0][0][0] = g0.
__global__ void greens_fill_kernel(double *__restrict__ G, MeshDims d, double hx, double hy, double hz,
                                   double coef, double g0)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    if (i >= d.gpitch) return;
    double x = i * hx, y = j * hy, z = k * hz;
    double v = (i == 0 && j == 0 && k == 0) ? g0 : coef / sqrt(x * x + y * y + z * z);
    G[((size_t)k * (d.ny + 1) + j) * d.gpitch + i] = i <= d.nx ? v : 0.0;      // pad entries stay zero (dks_greens_r16.cuh)
}

// One axis of the transform of the even extension (i' = min(i, 2n-i), PAPER.md:98 / reading A4):
// out[k] = sum_{p<2n} g[min(p, 2n-p)] e^{-2 pi i p k / 2n}, k = 0..n, which is real.  In place.
// Lines are enumerated as l = b * na + a with base offset a*sa + b*sb; elements at stride es.
// Two lines share one complex transform: the transform of a real EVEN sequence is real, so for
// c = g1 + i g2 simply FT{g1} = Re FT{c} and FT{g2} = Im FT{c}; slot w of a CTA carries lines 2(l0+w), +1.
__global__ void __launch_bounds__(256)
greens_axis_kernel(double *__restrict__ G, int n, int logL, int W, long long es, int na, long long sa,
                   int nb, long long sb, double scale, const cplx *__restrict__ tw)
{
    extern __shared__ cplx s[];
    const int L = 2 * n, WP = W + 1;
    const int tid = threadIdx.x, nt = blockDim.x;
    const long long l0 = 2 * (long long)blockIdx.x * W, nlines = (long long)na * nb;
    for (int idx = tid; idx < L * W; idx += nt) {
        int p = idx / W, w = idx % W;
        long long l1 = l0 + 2 * w, l2 = l1 + 1;
        const long long e = (long long)min(p, L - p) * es;
        double v1 = 0.0, v2 = 0.0;
        if (l1 < nlines) v1 = G[(l1 % na) * sa + (l1 / na) * sb + e];
        if (l2 < nlines) v2 = G[(l2 % na) * sa + (l2 / na) * sb + e];
        s[p * WP + w] = cmake(v1, v2);
    }
    __syncthreads();
    tile_fft_dif<-1>(s, L, logL, W, WP, tw);
    for (int idx = tid; idx < (n + 1) * W; idx += nt) {
        int k = idx / W, w = idx % W;
        long long l1 = l0 + 2 * w, l2 = l1 + 1;
        const cplx c = s[brev(k, logL) * WP + w];
        if (l1 < nlines) G[(l1 % na) * sa + (l1 / na) * sb + (long long)k * es] = c.x * scale;
        if (l2 < nlines) G[(l2 % na) * sa + (l2 / na) * sb + (long long)k * es] = c.y * scale;
    }
}

}  // namespace dks
