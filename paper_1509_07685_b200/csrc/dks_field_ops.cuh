// The two steps adjacent to the solve, on the device: cloud-in-cell charge deposit before,
// E = -grad(phi) and its interpolation to the particles after.  PAPER.md:86 only names IPPL's "particles with the
// respective interpolation operators"; PAPER.md:160 names the host <-> device transfer of rho and phi ("up to 55 %" of
// the run) as the limiter, which is what keeping these steps next to the solve removes.  Readings F1-F4:
//   F1  node (i, j, k) sits at origin + (i hx, j hy, k hz); mesh coordinate u = (X - ox) / hx (IEEE division).
//   F2  trilinear weights on the 8 surrounding nodes, rho = charge / (hx hy hz); a particle is dropped unless
//       0 <= u < nx - 1 (and likewise in y, z).
//   F3  second-order differences: central inside, one-sided second order at the two ends of every axis.
//   F4  the field at a particle = the same trilinear weights applied to the node values; 0 for dropped particles.
// All three are bandwidth / atomic-throughput bound streaming kernels: SoA particle arrays read with coalesced 64-bit
// loads, fp64 reductions into rho with red.global.add.f64 (the summation order is free, so results agree with a
// sequential sum to a few ulp of the node's total, not bit for bit).
#pragma once
#include "dks_passes_generic.cuh"   // MeshDims

namespace dks {

struct ParticleFrame {
    double ox, oy, oz;      // origin: position of node (0, 0, 0)
    double hx, hy, hz;
};

// F1 + drop rule.  Returns false for a dropped particle.
__device__ __forceinline__ bool cic_locate(double X, double Y, double Z, const ParticleFrame &f, const MeshDims &d,
                                           int &i, int &j, int &k, double &fx, double &fy, double &fz)
{
    const double u = (X - f.ox) / f.hx, v = (Y - f.oy) / f.hy, w = (Z - f.oz) / f.hz;
    if (!(u >= 0.0 && u < (double)(d.nx - 1) && v >= 0.0 && v < (double)(d.ny - 1) && w >= 0.0 && w < (double)(d.nz - 1))) return false;
    const double fu = floor(u), fv = floor(v), fw = floor(w);
    i = (int)fu; j = (int)fv; k = (int)fw;
    fx = u - fu; fy = v - fv; fz = w - fw;
    return true;
}

__device__ __forceinline__ void red_add(double *p, double v)
{
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory");
}

// rho must be zero on entry.  grid-stride over the particles.
__global__ void __launch_bounds__(256)
cic_deposit_kernel(const double *__restrict__ x, const double *__restrict__ y, const double *__restrict__ z,
                   const double *__restrict__ q, long long np, ParticleFrame f, MeshDims d, double inv_vol, double *__restrict__ rho)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x; n < np; n += stride) {
        int i, j, k;
        double fx, fy, fz;
        if (!cic_locate(x[n], y[n], z[n], f, d, i, j, k, fx, fy, fz)) continue;
        const double c = q[n] * inv_vol;
        double *base = rho + ((size_t)k * d.ny + j) * d.nx + i;
        const size_t sy = d.nx, sz = (size_t)d.nx * d.ny;
        const double wx0 = 1.0 - fx, wy0 = 1.0 - fy, wz0 = (1.0 - fz) * c, wz1 = fz * c;
        red_add(base, wx0 * wy0 * wz0);
        red_add(base + 1, fx * wy0 * wz0);
        red_add(base + sy, wx0 * fy * wz0);
        red_add(base + sy + 1, fx * fy * wz0);
        red_add(base + sz, wx0 * wy0 * wz1);
        red_add(base + sz + 1, fx * wy0 * wz1);
        red_add(base + sz + sy, wx0 * fy * wz1);
        red_add(base + sz + sy + 1, fx * fy * wz1);
    }
}

// F3 along one axis: f points at the node, stride in elements
__device__ __forceinline__ double diff2(const double *__restrict__ f, int i, int n, size_t stride, double inv2h)
{
    if (i == 0) return (-3.0 * f[0] + 4.0 * f[stride] - f[2 * stride]) * inv2h;
    if (i == n - 1) return (3.0 * f[0] - 4.0 * *(f - stride) + *(f - 2 * stride)) * inv2h;
    return (f[stride] - *(f - stride)) * inv2h;
}

// one thread per node, x fastest; grid (ceil(nx / 128), ny, nz)
__global__ void __launch_bounds__(128)
gradient_kernel(const double *__restrict__ phi, double *__restrict__ ex, double *__restrict__ ey, double *__restrict__ ez,
                MeshDims d, double ihx, double ihy, double ihz)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    if (i >= d.nx) return;
    const size_t m = ((size_t)k * d.ny + j) * d.nx + i;
    ex[m] = -diff2(phi + m, i, d.nx, 1, ihx);
    ey[m] = -diff2(phi + m, j, d.ny, (size_t)d.nx, ihy);
    ez[m] = -diff2(phi + m, k, d.nz, (size_t)d.nx * d.ny, ihz);
}

// F4 for the three field components at once
__global__ void __launch_bounds__(256)
gather_field_kernel(const double *__restrict__ ex, const double *__restrict__ ey, const double *__restrict__ ez,
                    const double *__restrict__ x, const double *__restrict__ y, const double *__restrict__ z, long long np,
                    ParticleFrame f, MeshDims d, double *__restrict__ epx, double *__restrict__ epy, double *__restrict__ epz)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x; n < np; n += stride) {
        int i, j, k;
        double fx, fy, fz;
        double sx = 0.0, sy_ = 0.0, sz_ = 0.0;
        if (cic_locate(x[n], y[n], z[n], f, d, i, j, k, fx, fy, fz)) {
            const size_t m0 = ((size_t)k * d.ny + j) * d.nx + i, sy = d.nx, sz = (size_t)d.nx * d.ny;
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                const int di = c & 1, dj = (c >> 1) & 1, dk = c >> 2;
                const double w = (di ? fx : 1.0 - fx) * (dj ? fy : 1.0 - fy) * (dk ? fz : 1.0 - fz);
                const size_t m = m0 + di + dj * sy + dk * sz;
                sx = fma(w, __ldg(ex + m), sx);
                sy_ = fma(w, __ldg(ey + m), sy_);
                sz_ = fma(w, __ldg(ez + m), sz_);
            }
        }
        epx[n] = sx; epy[n] = sy_; epz[n] = sz_;
    }
}

// ---- F3 + F4 in one call (dks_field_at_particles): the field goes through an interleaved scratch, one 32-byte record
// (ex, ey, ez, 0) per node, so that the gather costs one 256-bit load per node -- 8 sectors per particle instead of the 12
// that three separate arrays cost (x-neighbours share a sector there), and no 64-byte DRAM burst is half wasted.
__global__ void __launch_bounds__(128)
gradient_aos_kernel(const double *__restrict__ phi, double4 *__restrict__ e, MeshDims d, double ihx, double ihy, double ihz)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    if (i >= d.nx) return;
    const size_t m = ((size_t)k * d.ny + j) * d.nx + i;
    const double gx = -diff2(phi + m, i, d.nx, 1, ihx), gy = -diff2(phi + m, j, d.ny, (size_t)d.nx, ihy),
                 gz = -diff2(phi + m, k, d.nz, (size_t)d.nx * d.ny, ihz);
    asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(e + m), "d"(gx), "d"(gy), "d"(gz), "d"(0.0) : "memory");
}

__global__ void __launch_bounds__(256)
gather_aos_kernel(const double4 *__restrict__ e, const double *__restrict__ x, const double *__restrict__ y,
                  const double *__restrict__ z, long long np, ParticleFrame f, MeshDims d, double *__restrict__ epx,
                  double *__restrict__ epy, double *__restrict__ epz)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x; n < np; n += stride) {
        int i, j, k;
        double fx, fy, fz;
        double sx = 0.0, sy_ = 0.0, sz_ = 0.0;
        if (cic_locate(x[n], y[n], z[n], f, d, i, j, k, fx, fy, fz)) {
            const size_t m0 = ((size_t)k * d.ny + j) * d.nx + i, sy = d.nx, sz = (size_t)d.nx * d.ny;
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                const int di = c & 1, dj = (c >> 1) & 1, dk = c >> 2;
                const double w = (di ? fx : 1.0 - fx) * (dj ? fy : 1.0 - fy) * (dk ? fz : 1.0 - fz);
                double gx, gy, gz, pad;
                asm volatile("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(gx), "=d"(gy), "=d"(gz), "=d"(pad)
                             : "l"(e + m0 + di + dj * sy + dk * sz));
                sx = fma(w, gx, sx);
                sy_ = fma(w, gy, sy_);
                sz_ = fma(w, gz, sz_);
            }
        }
        epx[n] = sx; epy[n] = sy_; epz[n] = sz_;
    }
}

}  // namespace dks
