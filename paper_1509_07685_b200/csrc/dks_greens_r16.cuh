// Step a0 with the register-resident transforms: the Green's function build and its transform for mesh
// extents n = 16 A (32..256).  PAPER.md:117 (G), :98 (doubled grid, reading A4: even extension), :132
// ("separate kernel to calculate the Greens function", rebuilt every time step because h changes).
//
// Along one axis the even extension x[m] = g[min(m, 2n - m)], m < L = 2n, has the real transform
//   X[2K + p] = sum_{m<n} ( g[m] + (-1)^p g[n - m] ) w_L^(p m) w_n^(m K),      k = 2K + p = 0..n,
// i.e. the usual two parity sub-transforms of length n, fed with u_p[m] = g[m] +- g[n - m].  Two real lines
// share one complex transform: for c = g1 + i g2 simply X1 = Re C, X2 = Im C, because both transforms are
// real.  Only k <= n is kept (the octant), so only registers r <= 8 of a thread are stored.
//
//   greens_x_r16<A>    : x axis, fused with the evaluation of G (no input at all): one warp per group of 16 / A
//                        pairs of octant rows (ky, ky + 1), the structure of p3_x_conv_r16's forward half.
//   greens_axis_r16<A> : y or z axis, in place on the octant: the structure of p2_y_fwd_r16; a CTA takes 16
//                        adjacent x entries (8 packed pairs) of all n + 1 rows along the axis.
// The pad entries nx < kx < gpitch of every octant row are written as zero by the x pass: they are the imaginary
// partners of valid columns in the packed y / z passes and must stay finite (entry nx + 1, the partner of column nx,
// picks up that column's rounding leakage, ~1e-16 of it; P3 never reads a pad entry).
#pragma once
#include "dks_passes_r16.cuh"

namespace dks {

constexpr int kGxWarps = 12;
constexpr int kGxSmemPerWarp = kP3ExBytes + 128;
constexpr int kGxSmem = kGxWarps * kGxSmemPerWarp;

template <int A>
__global__ void __launch_bounds__(kGxWarps * 32, 1)
greens_x_r16(double *__restrict__ G, MeshDims d, double hx, double hy, double hz, double coef, double g0,
             const cplx *__restrict__ tw1)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int N = 16 * A, J = 16 / A, GG = 16 / A;
    constexpr int REG = 16 * A + (A < 8 ? A : 0);
    constexpr int SWZ = A >= 8 ? 7 : A - 1;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int a = lane & (A - 1), p = (lane / A) & 1, j = lane / (2 * A);
    cplx *ex = reinterpret_cast<cplx *>(smem_raw + warp * kGxSmemPerWarp) + (j * 2 + p) * REG;
    const int ny = d.ny, pp = (ny + 2) / 2;                  // row pairs per plane
    const unsigned total = (unsigned)(d.nz + 1) * pp, ngroups = (total + J - 1) / J, stride = gridDim.x * kGxWarps;
    cplx tb[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) tb[k] = __ldg(&tw1[p * N + k * A + a]);

    for (unsigned grp = blockIdx.x * kGxWarps + warp; grp < ngroups; grp += stride) {
        const unsigned q = grp * J + j;
        const bool valid = q < total;
        const int kz = (int)(min(q, total - 1) / pp), ky0 = 2 * (int)(min(q, total - 1) % pp);
        const double z = kz * hz, y1 = ky0 * hy, y2 = (ky0 + 1) * hy;
        const double s1 = y1 * y1 + z * z, s2 = y2 * y2 + z * z;
        cplx v[16];
#pragma unroll
        for (int b = 0; b < 16; ++b) {
            const int m = a + A * b, i = p ? N - m : m;      // parity 0 evaluates g[m], parity 1 g[n - m]
            const double x = i * hx;
            // coef * rsqrt(r^2) instead of coef / sqrt(r^2): one Newton-refined reciprocal square root (<= 1 ulp) in place of an
            // IEEE square root and an IEEE division, which were four fifths of this kernel's instructions (ncu r3: 176 us of
            // a0's 349 at 256^3 with 6 % DRAM throughput).  The product is within 1.5 ulp of the quotient; the octant test
            // holds 1e-12 of the maximum against the oracle.  r = 0 gives inf as before and is replaced by g0 below.
            cplx mine = cmake(coef * rsqrt(x * x + s1), coef * rsqrt(x * x + s2));
            if (i == 0 && kz == 0 && ky0 == 0) mine.x = g0;
            const cplx other = shfl_xor_c(mine, A);
            v[b] = p ? csub(other, mine) : cadd(mine, other);
        }
        if (p) parity_consts<-1>(v);
        fft16<-1>(v);
#pragma unroll
        for (int k = 0; k < 16; ++k) v[k] = cmul(v[k], tb[k]);
#pragma unroll
        for (int k = 0; k < 16; ++k) ex[k * A + (a ^ (k & SWZ))] = v[k];
        __syncwarp();
#pragma unroll
        for (int g = 0; g < GG; ++g)
#pragma unroll
            for (int ap = 0; ap < A; ++ap) v[g * A + ap] = ex[(a + A * g) * A + (ap ^ (a & SWZ))];
        fft_second<A, -1>(v);                                // v[r] = X1[k] + i X2[k], k = 2 (a + A r) + p
        __syncwarp();
        if (valid) {
            double *row = G + ((size_t)kz * (ny + 1) + ky0) * d.gpitch;
            const bool two = ky0 + 1 <= ny;
#pragma unroll
            for (int r = 0; r < 9; ++r) {
                const int k = 2 * (a + A * r) + p;
                if (k <= N) {
                    row[k] = v[r].x;
                    if (two) row[d.gpitch + k] = v[r].y;
                }
            }
            for (int t = N + 1 + a + A * p; t < d.gpitch; t += 2 * A) {      // pad entries stay zero
                row[t] = 0.0;
                if (two) row[d.gpitch + t] = 0.0;
            }
        }
    }
}

// y or z axis, in place.  grid (ceil(gpitch / 16), count); element (row m, outer o) of the line set lives at
// G[o * os + m * rs + x]; 16 A threads; dynamic shared memory R16Geom<A>::SMEM.
template <int A>
__global__ void __launch_bounds__(R16Geom<A>::THREADS, DKS_R16_MINB(A))
greens_axis_r16(double *__restrict__ G, int gpitch, long long rs, long long os, double scale, const cplx *__restrict__ tw1)
{
    extern __shared__ cplx ex[];
    constexpr int N = R16Geom<A>::N;
    const int tid = threadIdx.x, c = tid & 7, p = (tid >> 3) & 1, a = tid >> 4;
    const int x = blockIdx.x * 2 * kCols + 2 * c;
    const bool valid = x < gpitch;                           // gpitch is a multiple of 8: x + 1 is valid too
    double *base = G + (size_t)blockIdx.y * os + x;
    cplx v[16];
#pragma unroll
    for (int b = 0; b < 16; ++b) {
        const int m = a + A * b;
        cplx gm = cmake(0.0, 0.0), gn = gm;
        if (valid) {
            gm = *reinterpret_cast<const cplx *>(base + (size_t)m * rs);
            gn = *reinterpret_cast<const cplx *>(base + (size_t)(N - m) * rs);
        }
        v[b] = p ? csub(gm, gn) : cadd(gm, gn);
    }
    strided_forward<A>(v, ex, c, p, a, tw1, nullptr);        // its barrier also orders every load before every store
    if (valid) {
#pragma unroll
        for (int r = 0; r < 9; ++r) {
            const int k = 2 * (a + A * r) + p;
            if (k <= N) *reinterpret_cast<cplx *>(base + (size_t)k * rs) = cscale(v[r], scale);
        }
    }
}

}  // namespace dks
