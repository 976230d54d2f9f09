// Specialised passes for mesh extents n = 16 A, A in {2,4,8,16} (n = 32..256) on the pass's own axis.
// Same buffers and layouts as the generic passes (dks_passes_generic.cuh), so any pass may use
// either variant:
//
//   rho [nz][ny][nx] real --P1--> A [nz+1][ny][nx] cplx --P2--> B [nz+1][2ny][nx] cplx
//       --P3 (in place)--> B --P4--> A --P5--> phi [nz][ny][nx] real
//
// Every padded line = two length-n sub-transforms (parity p = 0,1; dks_fft_r16.cuh), each a four-step
// FFT over A threads x 16 registers with ONE shared-memory exchange.  Global loads go straight to
// registers (16 independent 128-bit loads per thread); the two parities of one line sit in the same
// warp and load the same addresses, which the coalescer merges.
//
// Strided lines (P1, P2, P4, P5): CTA = 8 adjacent columns x 2 parities x A threads (16 A threads);
//   tid -> c = tid & 7 (column, 128 B contiguous per quarter warp), p = (tid >> 3) & 1, a = tid >> 4.
//   Exchange buffer ex[p][k][a][c]: every quarter-warp access is 8 x 16 B contiguous: conflict free.
// Contiguous lines (P3): one warp = one line, lane -> a = lane & 15, p = lane >> 4; exchange buffer
//   per warp ex[p][k][17] (row padded by one element: conflict free both ways); __syncwarp only.
#pragma once
#include "dks_fft_r16.cuh"
#include "dks_passes_generic.cuh"   // MeshDims

namespace dks {

constexpr int kCols = 8;   // columns per CTA of the strided passes

template <int A>
struct R16Geom {
    static constexpr int N = 16 * A;          // mesh extent on this axis
    static constexpr int L = 32 * A;          // padded line length
    static constexpr int THREADS = 16 * A;    // kCols * 2 * A
    static constexpr int SMEM = 2 * 16 * A * kCols * (int)sizeof(cplx);   // exchange buffer = [L][kCols] tile
};

// ---- the two halves of a strided-line transform, around the shared-memory exchange -------------
// forward: v[b] = x[a + A b] on entry; v[r] = X[2 (a + A r) + p] on exit
template <int A>
__device__ __forceinline__ void strided_forward(cplx (&v)[16], cplx *ex, int c, int p, int a,
                                                const cplx *__restrict__ tw1, const cplx *__restrict__ tw2)
{
    if (p) twiddle_parity<A, -1>(v, tw2, a);
    fft16<-1>(v);
    twiddle_between<A, -1>(v, tw1, a);
#pragma unroll
    for (int k = 0; k < 16; ++k) ex[((p * 16 + k) * A + a) * kCols + c] = v[k];
    __syncthreads();
    constexpr int G = 16 / A;
#pragma unroll
    for (int g = 0; g < G; ++g)
#pragma unroll
        for (int ap = 0; ap < A; ++ap) v[g * A + ap] = ex[((p * 16 + a + A * g) * A + ap) * kCols + c];
    fft_second<A, -1>(v);
}

// inverse: v[b] = X[2 (a + A b) + p] on entry; on exit v[r] = IFFT_n(X_p)[a + A r] (* w_L^-(a + A r) if p)
template <int A>
__device__ __forceinline__ void strided_inverse(cplx (&v)[16], cplx *ex, int c, int p, int a,
                                                const cplx *__restrict__ tw1, const cplx *__restrict__ tw2)
{
    fft16<+1>(v);
    twiddle_between<A, +1>(v, tw1, a);
#pragma unroll
    for (int k = 0; k < 16; ++k) ex[((p * 16 + k) * A + a) * kCols + c] = v[k];
    __syncthreads();
    constexpr int G = 16 / A;
#pragma unroll
    for (int g = 0; g < G; ++g)
#pragma unroll
        for (int ap = 0; ap < A; ++ap) v[g * A + ap] = ex[((p * 16 + a + A * g) * A + ap) * kCols + c];
    fft_second<A, +1>(v);
    if (p) twiddle_parity<A, +1>(v, tw2, a);
}

// ---------------------------------------------------------------------------------------------
// P2: forward y.  grid (nx / 8, nz + 1), 16 A threads.
// ---------------------------------------------------------------------------------------------
template <int A>
__global__ void __launch_bounds__(R16Geom<A>::THREADS, 512 / R16Geom<A>::THREADS)
p2_y_fwd_r16(const cplx *__restrict__ Ain, cplx *__restrict__ B, MeshDims d,
             const cplx *__restrict__ tw1, const cplx *__restrict__ tw2)
{
    extern __shared__ cplx ex[];
    const int tid = threadIdx.x, c = tid & 7, p = (tid >> 3) & 1, a = tid >> 4;
    const int nx = d.nx, ny = d.ny, kz = blockIdx.y;
    const size_t x = (size_t)blockIdx.x * kCols + c;
    cplx v[16];
#pragma unroll
    for (int b = 0; b < 16; ++b) v[b] = ldg_stream(&Ain[((size_t)kz * ny + a + A * b) * nx + x]);
    strided_forward<A>(v, ex, c, p, a, tw1, tw2);
#pragma unroll
    for (int r = 0; r < 16; ++r)
        stg_stream(&B[((size_t)kz * 2 * ny + 2 * (a + A * r) + p) * nx + x], v[r]);
}

// ---------------------------------------------------------------------------------------------
// P4: inverse y, crop to ny.  grid (nx / 8, nz + 1)
// ---------------------------------------------------------------------------------------------
template <int A>
__global__ void __launch_bounds__(R16Geom<A>::THREADS, 512 / R16Geom<A>::THREADS)
p4_y_inv_r16(const cplx *__restrict__ B, cplx *__restrict__ Aout, MeshDims d,
             const cplx *__restrict__ tw1, const cplx *__restrict__ tw2)
{
    extern __shared__ cplx ex[];
    const int tid = threadIdx.x, c = tid & 7, p = (tid >> 3) & 1, a = tid >> 4;
    const int nx = d.nx, ny = d.ny, kz = blockIdx.y;
    const size_t x = (size_t)blockIdx.x * kCols + c;
    cplx v[16];
#pragma unroll
    for (int b = 0; b < 16; ++b)
        v[b] = ldg_stream(&B[((size_t)kz * 2 * ny + 2 * (a + A * b) + p) * nx + x]);
    strided_inverse<A>(v, ex, c, p, a, tw1, tw2);
    cplx out[8];
    combine_parities<8>(v, p, out);
#pragma unroll
    for (int i = 0; i < 8; ++i)
        stg_stream(&Aout[((size_t)kz * ny + a + A * (i + 8 * p)) * nx + x], out[i]);
}

// ---------------------------------------------------------------------------------------------
// P1: forward z, real -> complex; the real columns (x, x+1) are packed into one complex line and
// the packed spectrum C is split with FT{a}[k] = (C[k] + conj C[L-k]) / 2, FT{b}[k] = (C[k] - conj C[L-k]) / (2i).
// grid (nx / 16, ny)
// ---------------------------------------------------------------------------------------------
template <int A>
__global__ void __launch_bounds__(R16Geom<A>::THREADS, 512 / R16Geom<A>::THREADS)
p1_z_r2c_r16(const double *__restrict__ rho, cplx *__restrict__ Aout, MeshDims d,
             const cplx *__restrict__ tw1, const cplx *__restrict__ tw2)
{
    extern __shared__ cplx ex[];
    constexpr int N = R16Geom<A>::N, L = R16Geom<A>::L, THREADS = R16Geom<A>::THREADS;
    const int tid = threadIdx.x, c = tid & 7, p = (tid >> 3) & 1, a = tid >> 4;
    const int nx = d.nx, ny = d.ny, y = blockIdx.y;
    const size_t x0 = (size_t)blockIdx.x * 2 * kCols;
    cplx v[16];
#pragma unroll
    for (int b = 0; b < 16; ++b)
        v[b] = ldg_stream(reinterpret_cast<const cplx *>(&rho[((size_t)(a + A * b) * ny + y) * nx + x0 + 2 * c]));
    strided_forward<A>(v, ex, c, p, a, tw1, tw2);
    __syncthreads();                                  // exchange reads done: reuse ex as C[K][c]
#pragma unroll
    for (int r = 0; r < 16; ++r) ex[(2 * (a + A * r) + p) * kCols + c] = v[r];
    __syncthreads();
    for (int idx = tid; idx < (N + 1) * kCols; idx += THREADS) {
        const int k = idx >> 3, cc = idx & 7;
        const cplx ck = ex[k * kCols + cc], cm = ex[((L - k) & (L - 1)) * kCols + cc];
        cplx *out = &Aout[((size_t)k * ny + y) * nx + x0 + 2 * cc];
        stg_stream(out, cmake(0.5 * (ck.x + cm.x), 0.5 * (ck.y - cm.y)));
        stg_stream(out + 1, cmake(0.5 * (ck.y + cm.y), -0.5 * (ck.x - cm.x)));
    }
}

// ---------------------------------------------------------------------------------------------
// P5: inverse z, complex -> real, crop to nz.  Rebuilds the packed spectrum C[k] = Fa[k] + i Fb[k],
// C[L-k] = conj Fa[k] + i conj Fb[k] in shared memory first.  grid (nx / 16, ny)
// ---------------------------------------------------------------------------------------------
template <int A>
__global__ void __launch_bounds__(R16Geom<A>::THREADS, 512 / R16Geom<A>::THREADS)
p5_z_c2r_r16(const cplx *__restrict__ Ain, double *__restrict__ phi, MeshDims d,
             const cplx *__restrict__ tw1, const cplx *__restrict__ tw2)
{
    extern __shared__ cplx ex[];
    constexpr int N = R16Geom<A>::N, L = R16Geom<A>::L, THREADS = R16Geom<A>::THREADS;
    const int tid = threadIdx.x, c = tid & 7, p = (tid >> 3) & 1, a = tid >> 4;
    const int nx = d.nx, ny = d.ny, y = blockIdx.y;
    const size_t x0 = (size_t)blockIdx.x * 2 * kCols;
    // all loads of the tile in flight at once (the last round is ragged: row k = N only)
    constexpr int ITEMS = (N + 1) * kCols, ROUNDS = (ITEMS + THREADS - 1) / THREADS;
    cplx fa[ROUNDS], fb[ROUNDS];
#pragma unroll
    for (int i = 0; i < ROUNDS; ++i) {
        const int idx = tid + i * THREADS, k = idx >> 3, cc = idx & 7;
        if (idx < ITEMS) {
            const cplx *in = &Ain[((size_t)k * ny + y) * nx + x0 + 2 * cc];
            fa[i] = ldg_stream(in);
            fb[i] = ldg_stream(in + 1);
        }
    }
#pragma unroll
    for (int i = 0; i < ROUNDS; ++i) {
        const int idx = tid + i * THREADS, k = idx >> 3, cc = idx & 7;
        if (idx < ITEMS) {
            ex[k * kCols + cc] = cmake(fa[i].x - fb[i].y, fa[i].y + fb[i].x);
            if (k > 0 && k < N) ex[(L - k) * kCols + cc] = cmake(fa[i].x + fb[i].y, fb[i].x - fa[i].y);
        }
    }
    __syncthreads();
    cplx v[16];
#pragma unroll
    for (int b = 0; b < 16; ++b) v[b] = ex[(2 * (a + A * b) + p) * kCols + c];
    __syncthreads();                                  // C consumed: ex becomes the exchange buffer
    strided_inverse<A>(v, ex, c, p, a, tw1, tw2);
    cplx out[8];
    combine_parities<8>(v, p, out);
#pragma unroll
    for (int i = 0; i < 8; ++i)
        stg_stream(reinterpret_cast<cplx *>(&phi[((size_t)(a + A * (i + 8 * p)) * ny + y) * nx + x0 + 2 * c]), out[i]);
}

// ---------------------------------------------------------------------------------------------
// P3 for nx = 256: forward x, multiply by the Green's transform, inverse x, crop; in place on B.
// One warp = one line; block = 8 warps; grid ((nz+1) * 2ny / 8).  Ghat as in the generic pass.
// ---------------------------------------------------------------------------------------------
constexpr int kP3Warps = 8;
constexpr int kP3RowPad = 17;
constexpr int kP3GhatDoubles = 264;               // gpitch for nx = 256: one Ghat row, staged per warp
constexpr int kP3SmemPerWarp = 2 * 16 * kP3RowPad * (int)sizeof(cplx) + kP3GhatDoubles * (int)sizeof(double);

__global__ void __launch_bounds__(kP3Warps * 32, 2)
p3_x_conv_r16(cplx *__restrict__ B, const double *__restrict__ Ghat, MeshDims d,
              const cplx *__restrict__ tw1, const cplx *__restrict__ tw2)
{
    extern __shared__ cplx smem[];
    constexpr int A = 16, N = 256, L = 512;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, a = lane & 15, p = lane >> 4;
    char *wbase = reinterpret_cast<char *>(smem) + warp * kP3SmemPerWarp;
    cplx *ex = reinterpret_cast<cplx *>(wbase) + p * 16 * kP3RowPad;
    double *gs = reinterpret_cast<double *>(wbase + 2 * 16 * kP3RowPad * sizeof(cplx));
    const int ny = d.ny;
    const unsigned line = blockIdx.x * kP3Warps + warp;
    const int kz = (int)(line / (unsigned)(2 * ny)), ky = (int)(line % (unsigned)(2 * ny));
    const int kyp = min(ky, 2 * ny - ky);
    const double *__restrict__ grow = Ghat + ((size_t)kz * (ny + 1) + kyp) * d.gpitch;
    // the Ghat row (nx + 1 reals, pitch 264) goes to shared memory asynchronously: it is needed only
    // after the forward transform, and waiting for it there would expose a second DRAM latency
    for (int i = lane; i < kP3GhatDoubles / 2; i += 32) cp_async16(gs + 2 * i, grow + 2 * i);
    cp_async_commit();
    cplx *base = B + (size_t)line * N;
    cplx v[16];
#pragma unroll
    for (int b = 0; b < 16; ++b) v[b] = ldg_stream(&base[a + A * b]);
    // forward
    if (p) twiddle_parity<A, -1>(v, tw2, a);
    fft16<-1>(v);
    twiddle_between<A, -1>(v, tw1, a);
#pragma unroll
    for (int k = 0; k < 16; ++k) ex[k * kP3RowPad + a] = v[k];
    __syncwarp();
#pragma unroll
    for (int ap = 0; ap < 16; ++ap) v[ap] = ex[a * kP3RowPad + ap];
    fft16<-1>(v);
    // multiply: v[r] = X[K], K = 2 (a + 16 r) + p
    cp_async_wait_all();
    __syncwarp();
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const int K = 2 * (a + A * r) + p;
        v[r] = cscale(v[r], gs[min(K, L - K)]);
    }
    // inverse
    fft16<+1>(v);
    twiddle_between<A, +1>(v, tw1, a);
    __syncwarp();                                     // forward exchange reads done in every lane
#pragma unroll
    for (int k = 0; k < 16; ++k) ex[k * kP3RowPad + a] = v[k];
    __syncwarp();
#pragma unroll
    for (int ap = 0; ap < 16; ++ap) v[ap] = ex[a * kP3RowPad + ap];
    fft16<+1>(v);
    if (p) twiddle_parity<A, +1>(v, tw2, a);
    cplx out[8];
    combine_parities<16>(v, p, out);
#pragma unroll
    for (int i = 0; i < 8; ++i) stg_stream(&base[a + A * (i + 8 * p)], out[i]);
}

}  // namespace dks
