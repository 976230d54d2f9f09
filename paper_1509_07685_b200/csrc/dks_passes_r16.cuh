// Specialised passes for mesh extents n = 16 A, A in {1,2,4,8,16} (n = 16..256) on the pass's own axis (A = 1: the whole
// sub-transform is one thread's radix-16, the exchange degenerates to the identity).
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

// Sharded solve: rho / phi are split into y slabs over the ranks, the
// half-spectrum planes kz into kz slabs.  P1 (z lines, y-slab local) stores every output row straight into the buffer of
// the rank that owns its kz plane, and P4 (y lines, kz-slab local) stores every output row into the buffer of the rank that
// owns its y row: base[] holds device pointers that are peer-mapped over NVLink (or local, when ranks are emulated on one
// device), so the exchange is part of the producing kernel's epilogue instead of a separate all-to-all.
constexpr int kMaxRanks = 8;
struct PeerTable {
    cplx *base[kMaxRanks];   // the receive buffer of every rank
    int nranks;              // 1: not sharded
    int lsplit;              // log2 of the slab thickness (planes per rank for P1, y rows per rank for P4)
    int first;               // P1: first global y row of this rank's slab;  P4: first global kz plane of this rank's slab
    int pitch;               // P1: global ny (rows per plane in the receiver);  P4: y rows per rank (rows per plane in the receiver)
};
// The between-step twiddle of an inverse strided pass is applied after the exchange in P5 and before it in P4 (measured:
// P4, which runs at its memory bound, loses 2 % with the 16 table loads in flight across the barrier; P5 gains 1 %).
constexpr bool kP4TwPost = false, kP5TwPost = true;
// Programmatic dependent launch (PDL variants of the kernels): the trigger sits right before a kernel's stores, not at its start.
// An early trigger lets the next kernel's CTAs take SM resources and spin in griddepcontrol.wait while this kernel still has CTAs
// to run (measured: 64^3 31.2 -> 24.6 us per solve, 128^3 96.8 -> 92.7 us with the late trigger).
#ifndef DKS_R16_OCC
#define DKS_R16_OCC 512
#endif
#define DKS_R16_MINB(A) (DKS_R16_OCC / R16Geom<A>::THREADS)

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
    if (p) parity_consts<-1>(v);
    fft16<-1>(v);
#pragma unroll
    for (int k = 0; k < 16; ++k) ex[((p * 16 + k) * A + a) * kCols + c] = v[k];
    cplx t[16];
    load_tw_post<A>(t, tw1 + p * 16 * A, a);             // in flight across the barrier (dks_fft_r16.cuh)
    __syncthreads();
    constexpr int G = 16 / A;
#pragma unroll
    for (int g = 0; g < G; ++g)
#pragma unroll
        for (int ap = 0; ap < A; ++ap) v[g * A + ap] = ex[((p * 16 + a + A * g) * A + ap) * kCols + c];
    fft_second_tw<A, -1, true>(v, t);                    // regions 0 and 1 have T = 1 at a' = 0
}

// inverse: v[b] = X[2 (a + A b) + p] on entry; on exit v[r] = IFFT_n(X_p)[a + A r] (* w_L^-(a + A r) if p)
template <int A, bool POST>
__device__ __forceinline__ void strided_inverse(cplx (&v)[16], cplx *ex, int c, int p, int a,
                                                const cplx *__restrict__ tw1, const cplx *__restrict__ tw2)
{
    fft16<+1>(v);
    constexpr int G = 16 / A;
    cplx t[16];
    if (!POST) twiddle_between<A, +1>(v, tw1 + p * 32 * A, a);
#pragma unroll
    for (int k = 0; k < 16; ++k) ex[((p * 16 + k) * A + a) * kCols + c] = v[k];
    if (POST) load_tw_post<A>(t, tw1 + p * 32 * A, a);   // in flight across the barrier
    __syncthreads();
#pragma unroll
    for (int g = 0; g < G; ++g)
#pragma unroll
        for (int ap = 0; ap < A; ++ap) v[g * A + ap] = ex[((p * 16 + a + A * g) * A + ap) * kCols + c];
    if (POST) fft_second_tw<A, +1, false>(v, t);         // region 2 carries the thread constant w_L^(k mod A): no unit entry
    else fft_second<A, +1>(v);
    if (p) parity_consts<+1>(v);
}

// ---------------------------------------------------------------------------------------------
// P2: forward y.  grid (nx / 8, nz + 1), 16 A threads.
// ---------------------------------------------------------------------------------------------
template <int A, bool PDL>
__global__ void __launch_bounds__(R16Geom<A>::THREADS, DKS_R16_MINB(A))
p2_y_fwd_r16(const cplx *__restrict__ Ain, cplx *__restrict__ B, MeshDims d, int kz0,
             const cplx *__restrict__ tw1, const cplx *__restrict__ tw2)
{
    extern __shared__ cplx ex[];
    const int tid = threadIdx.x, c = tid & 7, p = (tid >> 3) & 1, a = tid >> 4;
    const int nx = d.nx, ny = d.ny, kz = blockIdx.y;          // kz: plane within the slab
    const size_t x = (size_t)blockIdx.x * kCols + c;
    if (PDL) {
        pdl_wait();
    }
    cplx v[16];
#pragma unroll
    for (int b = 0; b < 16; ++b) v[b] = ldg_stream(&Ain[((size_t)(kz0 + kz) * ny + a + A * b) * nx + x]);
    strided_forward<A>(v, ex, c, p, a, tw1, tw2);
    if (PDL) pdl_trigger();
#pragma unroll
    for (int r = 0; r < 16; ++r)
        stg_stream(&B[((size_t)kz * 2 * ny + 2 * (a + A * r) + p) * nx + x], v[r]);
}

// ---------------------------------------------------------------------------------------------
// P2 with the two parities of a tile in two CTAs of 8 A threads each (blockIdx.x = 2 * tile + parity): the forward pass never
// combines parities, so nothing is exchanged between them.  Parity-uniform CTAs issue the parity constants only where they are
// used, and four CTAs of 128 threads per SM (instead of two of 256) overlap their load / transform / store phases more finely.
// Both CTAs of a tile read the same rows: they are neighbours in launch order, so the second read is an L2 hit.
// grid (2 nx / 8, planes)
// ---------------------------------------------------------------------------------------------
constexpr int kSplitMinA = 8;   // P1 and P2 run one CTA per parity for n >= 16 * kSplitMinA

template <int A, bool PDL>
__global__ void __launch_bounds__(8 * A, (DKS_R16_OCC / (8 * A) > 16 ? 16 : DKS_R16_OCC / (8 * A)))
p2_y_fwd_r16p(const cplx *__restrict__ Ain, cplx *__restrict__ B, MeshDims d, int kz0,
              const cplx *__restrict__ tw1, const cplx *__restrict__ tw2)
{
    extern __shared__ cplx ex[];                          // [16][A][8]
    const int tid = threadIdx.x, c = tid & 7, a = tid >> 3, p = blockIdx.x & 1;
    const int nx = d.nx, ny = d.ny, kz = blockIdx.y;
    const size_t x = (size_t)(blockIdx.x >> 1) * kCols + c;
    if (PDL) {
        pdl_wait();
    }
    cplx v[16];
#pragma unroll
    for (int b = 0; b < 16; ++b) v[b] = ldg_stream(&Ain[((size_t)(kz0 + kz) * ny + a + A * b) * nx + x]);
    if (p) parity_consts<-1>(v);
    fft16<-1>(v);
#pragma unroll
    for (int k = 0; k < 16; ++k) ex[(k * A + a) * kCols + c] = v[k];
    cplx t[16];
    load_tw_post<A>(t, tw1 + p * 16 * A, a);
    __syncthreads();
    constexpr int G = 16 / A;
#pragma unroll
    for (int g = 0; g < G; ++g)
#pragma unroll
        for (int ap = 0; ap < A; ++ap) v[g * A + ap] = ex[((a + A * g) * A + ap) * kCols + c];
    fft_second_tw<A, -1, true>(v, t);
    if (PDL) pdl_trigger();
#pragma unroll
    for (int r = 0; r < 16; ++r)
        stg_stream(&B[((size_t)kz * 2 * ny + 2 * (a + A * r) + p) * nx + x], v[r]);
}

// ---------------------------------------------------------------------------------------------
// P4: inverse y, crop to ny.  grid (nx / 8, nz + 1)
// ---------------------------------------------------------------------------------------------
template <int A, bool PDL, bool SHARD = false>
__global__ void __launch_bounds__(R16Geom<A>::THREADS, DKS_R16_MINB(A))
p4_y_inv_r16(const cplx *__restrict__ B, cplx *__restrict__ Aout, MeshDims d, int kz0,
             const cplx *__restrict__ tw1, const cplx *__restrict__ tw2, PeerTable T)
{
    extern __shared__ cplx ex[];
    const int tid = threadIdx.x, c = tid & 7, p = (tid >> 3) & 1, a = tid >> 4;
    const int nx = d.nx, ny = d.ny, kz = blockIdx.y;
    const size_t x = (size_t)blockIdx.x * kCols + c;
    if (PDL) {
        pdl_wait();
    }
    cplx v[16];
#pragma unroll
    for (int b = 0; b < 16; ++b)
        v[b] = ldg_stream(&B[((size_t)kz * 2 * ny + 2 * (a + A * b) + p) * nx + x]);
    strided_inverse<A, kP4TwPost>(v, ex, c, p, a, tw1, tw2);
    cplx out[8];
    combine_parities<8>(v, p, out);
    if (PDL) pdl_trigger();
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int yrow = a + A * (i + 8 * p);
        if (SHARD) {                                      // row y goes to the rank that owns it: [nz+1][ny / nranks][nx] there
            const int o = yrow >> T.lsplit;
            stg_stream(&T.base[o][((size_t)(T.first + kz) * T.pitch + (yrow - (o << T.lsplit))) * nx + x], out[i]);
        } else
            stg_stream(&Aout[((size_t)(kz0 + kz) * ny + yrow) * nx + x], out[i]);
    }
}

// ---------------------------------------------------------------------------------------------
// P1: forward z, real -> complex; the real columns (x, x+1) are packed into one complex line and
// the packed spectrum C is split with FT{a}[k] = (C[k] + conj C[L-k]) / 2, FT{b}[k] = (C[k] - conj C[L-k]) / (2i).
// Persistent: CTA t, t + grid, ... over the (nx / 16) * ny tiles of 16 real columns.  The next tile's
// rho rows (N rows x 128 B) arrive in the shared-memory stage through cp.async while this tile is
// transformed, so the DRAM latency is never exposed.
// The split needs C[k] and C[L-k] in one thread.  After the transform, thread (a, p) holds C[2 (a + A r) + p] in
// register r, and its mirror C[L-k] sits in register 15 - r of thread (A - a, 0) resp. (A - 1 - a, 1).  The a -> warp
// map below puts every such pair of threads into one warp, 16 lanes apart (the self-paired a = 0 and a = A/2 of
// parity 0 share warp 0), so the split is 8 register shuffles per value pair: no second pass through shared memory,
// no further block barrier.  Each thread stores its 8 (9) rows k <= n as (FT{a}[k], FT{b}[k]) with one 256-bit
// store (STG.256), 8 lanes = one 256-byte row.
// ---------------------------------------------------------------------------------------------
template <int A>
struct P1Geom {
    static constexpr int STAGE = 16 * A * kCols * (int)sizeof(cplx);     // N rows x 8 packed pairs
    static constexpr int SMEM = R16Geom<A>::SMEM + STAGE + 16;             // + two mbarriers
};

// thread -> sub-transform index a such that mirror partners are lane ^ 16 (or the lane itself)
template <int A>
__device__ __forceinline__ int p1_a_of(int p, int s, int w)
{
    if (p) return s ? A - 1 - w : w;
    if (w == 0) return s ? A / 2 : 0;
    return s ? A - w : w;
}

template <int A, bool PDL, bool SHARD = false>
__global__ void __launch_bounds__(R16Geom<A>::THREADS, DKS_R16_MINB(A))
p1_z_r2c_r16(const double *__restrict__ rho, cplx *__restrict__ Aall, MeshDims d, int nb,
             const cplx *__restrict__ tw1, const cplx *__restrict__ tw2, PeerTable T)
{
    extern __shared__ __align__(128) cplx ex[];
    constexpr int N = R16Geom<A>::N, L = R16Geom<A>::L, THREADS = R16Geom<A>::THREADS;
    cplx *stage = ex + L * kCols;
    const int tid = threadIdx.x, lane = tid & 31, c = tid & 7, p = (tid >> 3) & 1;
    const int a = p1_a_of<A>(p, (tid >> 4) & 1, tid >> 5);
    const bool a0 = a == 0 && p == 0;                     // holds k = 0 and k = n, mirrors inside its own registers
    const int partner = (A == 1 || (p == 0 && tid < 32)) ? lane : lane ^ 16;
    const int nx = d.nx, ny = d.ny, xtiles = nx / (2 * kCols), tiles = xtiles * ny * nb;   // nb meshes back to back
    uint64_t *bar = reinterpret_cast<uint64_t *>(stage + N * kCols);      // [0] stage filled, [1] exchange buffer read
    if (tid == 0) {
        mbar_init(&bar[0], THREADS);
        mbar_init(&bar[1], THREADS);
        mbar_init_fence();
    }
    __syncthreads();
    auto prefetch = [&](int t) {
        const int yy = t / xtiles, y = yy % ny;
        const double *src = rho + (size_t)(yy / ny) * N * ny * nx + (size_t)y * nx + (size_t)(t % xtiles) * 2 * kCols;
#pragma unroll
        for (int i = 0; i < N * kCols / THREADS; ++i) {
            const int idx = tid + i * THREADS;
            cp_async16(&stage[idx], &src[(size_t)(idx >> 3) * ny * nx + 2 * (idx & 7)]);
        }
        cp_async_mbar_arrive(&bar[0]);
    };
    unsigned phase = 0;
    int t = blockIdx.x;
    if (PDL) {
        pdl_wait();                                       // A is still being read by the previous solve's P5
    }
    if (t < tiles) prefetch(t);
    for (; t < tiles; t += gridDim.x, phase ^= 1) {
        const int yy = t / xtiles, y = yy % ny;
        const size_t xoff = (size_t)(t % xtiles) * 2 * kCols + 2 * c;
        cplx *Aout = Aall + (size_t)(yy / ny) * (N + 1) * ny * nx + (size_t)y * nx + xoff;
        // sharded: row k goes to the rank that owns plane k (the last rank also owns plane n): [planes][ny global][nx] there
        auto row = [&](int k) -> cplx * {
            if (!SHARD) return Aout + (size_t)k * ny * nx;
            const int o = min(k >> T.lsplit, T.nranks - 1);
            return T.base[o] + ((size_t)(k - (o << T.lsplit)) * T.pitch + T.first + y) * nx + xoff;
        };
        mbar_wait(&bar[0], phase);                        // stage complete
        cplx v[16];
#pragma unroll
        for (int b = 0; b < 16; ++b) v[b] = stage[(a + A * b) * kCols + c];
        // ---- strided_forward, with the prefetch of the next tile issued once the stage is consumed
        if (p) parity_consts<-1>(v);
        fft16<-1>(v);
        if (t != (int)blockIdx.x) mbar_wait(&bar[1], phase ^ 1);          // the last tile's exchange reads are done
#pragma unroll
        for (int k = 0; k < 16; ++k) ex[((p * 16 + k) * A + a) * kCols + c] = v[k];
        cplx twp[16];
        load_tw_post<A>(twp, tw1 + p * 16 * A, a);
        __syncthreads();
        if (t + (int)gridDim.x < tiles) prefetch(t + gridDim.x);
        constexpr int G = 16 / A;
#pragma unroll
        for (int g = 0; g < G; ++g)
#pragma unroll
            for (int ap = 0; ap < A; ++ap) v[g * A + ap] = ex[((p * 16 + a + A * g) * A + ap) * kCols + c];
        mbar_arrive(&bar[1]);
        fft_second_tw<A, -1, true>(v, twp);               // v[r] = C[2 (a + A r) + p]
        // ---- split: rows k = 2 (a + A r) + p, r < 8, and k = n (thread a0, r = 8)
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            cplx cm = cmake(__shfl_sync(0xffffffffu, v[15 - r].x, partner), __shfl_sync(0xffffffffu, v[15 - r].y, partner));
            if (a0) cm = r == 0 ? v[0] : v[16 - r];
            const cplx ck = v[r];
            stg_stream2(row(2 * (a + A * r) + p), cmake(0.5 * (ck.x + cm.x), 0.5 * (ck.y - cm.y)),
                        cmake(0.5 * (ck.y + cm.y), -0.5 * (ck.x - cm.x)));
        }
        if (a0) stg_stream2(row(N), cmake(v[8].x, 0.0), cmake(v[8].y, 0.0));
    }
    if (PDL) pdl_trigger();
}

// ---------------------------------------------------------------------------------------------
// P1 with one CTA of 8 A threads per parity (blockIdx.x = 2 * tile + parity), loads straight to registers, not persistent.
// The packed-spectrum split pairs C[k] with C[L-k], which have the same parity, so a parity's CTA splits and stores its own
// rows; mirror partners sit 8 lanes apart (p1_a_of).  grid (2 nx / 16, ny, batch)
// ---------------------------------------------------------------------------------------------
template <int A, bool PDL>
__global__ void __launch_bounds__(8 * A, (DKS_R16_OCC / (8 * A) > 16 ? 16 : DKS_R16_OCC / (8 * A)))
p1_z_r2c_r16p(const double *__restrict__ rho, cplx *__restrict__ Aall, MeshDims d,
              const cplx *__restrict__ tw1, const cplx *__restrict__ tw2)
{
    extern __shared__ cplx ex[];                          // [16][A][8]
    constexpr int N = 16 * A;
    const int tid = threadIdx.x, lane = tid & 31, c = tid & 7, p = blockIdx.x & 1;
    const int a = p1_a_of<A>(p, (tid >> 3) & 1, tid >> 4);
    const bool a0 = a == 0 && p == 0;
    const int partner = (p == 0 && tid < 16) ? lane : lane ^ 8;
    const int nx = d.nx, ny = d.ny, y = blockIdx.y;
    const size_t xoff = (size_t)(blockIdx.x >> 1) * 2 * kCols + 2 * c;
    rho += (size_t)blockIdx.z * N * ny * nx + (size_t)y * nx + xoff;
    cplx *Aout = Aall + (size_t)blockIdx.z * (N + 1) * ny * nx + (size_t)y * nx + xoff;
    if (PDL) {
        pdl_wait();
    }
    cplx v[16];
#pragma unroll
    for (int b = 0; b < 16; ++b) v[b] = ldg_stream(reinterpret_cast<const cplx *>(&rho[(size_t)(a + A * b) * ny * nx]));
    if (p) parity_consts<-1>(v);
    fft16<-1>(v);
#pragma unroll
    for (int k = 0; k < 16; ++k) ex[(k * A + a) * kCols + c] = v[k];
    cplx t[16];
    load_tw_post<A>(t, tw1 + p * 16 * A, a);
    __syncthreads();
    constexpr int G = 16 / A;
#pragma unroll
    for (int g = 0; g < G; ++g)
#pragma unroll
        for (int ap = 0; ap < A; ++ap) v[g * A + ap] = ex[((a + A * g) * A + ap) * kCols + c];
    fft_second_tw<A, -1, true>(v, t);                     // v[r] = C[2 (a + A r) + p]
    if (PDL) pdl_trigger();
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        cplx cm = cmake(__shfl_sync(0xffffffffu, v[15 - r].x, partner), __shfl_sync(0xffffffffu, v[15 - r].y, partner));
        if (a0) cm = r == 0 ? v[0] : v[16 - r];
        const cplx ck = v[r];
        stg_stream2(Aout + (size_t)(2 * (a + A * r) + p) * ny * nx, cmake(0.5 * (ck.x + cm.x), 0.5 * (ck.y - cm.y)),
                    cmake(0.5 * (ck.y + cm.y), -0.5 * (ck.x - cm.x)));
    }
    if (a0) stg_stream2(Aout + (size_t)N * ny * nx, cmake(v[8].x, 0.0), cmake(v[8].y, 0.0));
}

// ---------------------------------------------------------------------------------------------
// P5: inverse z, complex -> real, crop to nz.  The inverse of P1's split: the packed spectrum C[k] = Fa[k] + i Fb[k],
// C[L-k] = conj Fa[k] + i conj Fb[k] is formed in registers from the rows each thread loads itself.  grid (nx / 16, ny, batch)
// ---------------------------------------------------------------------------------------------
template <int A, bool PDL>
__global__ void __launch_bounds__(R16Geom<A>::THREADS, DKS_R16_MINB(A))
p5_z_c2r_r16(const cplx *__restrict__ Ain, double *__restrict__ phi, MeshDims d,
             const cplx *__restrict__ tw1, const cplx *__restrict__ tw2)
{
    extern __shared__ cplx ex[];
    constexpr int N = R16Geom<A>::N, L = R16Geom<A>::L;
    const int tid = threadIdx.x, c = tid & 7, p = (tid >> 3) & 1, a = tid >> 4;
    const int nx = d.nx, ny = d.ny, y = blockIdx.y;
    const size_t x0 = (size_t)blockIdx.x * 2 * kCols;
    Ain += (size_t)blockIdx.z * (N + 1) * ny * nx;        // blockIdx.z: mesh of the batch
    phi += (size_t)blockIdx.z * N * ny * nx;
    if (PDL) {
        pdl_wait();
    }
    // Every thread loads the 16 rows it needs itself, (FT{a}[r], FT{b}[r]) with one 256-bit load each, and forms its inputs
    // C[K] in registers: C[K] = Fa[K] + i Fb[K] for K <= n, C[K] = conj Fa[L-K] + i conj Fb[L-K] above.  Row r serves K = r and
    // K = L - r, i.e. two threads of the CTA: the second read is an L1 / L2 hit.  No pass through shared memory, no barrier.
    cplx v[16];
    {
        const cplx *in0 = &Ain[(size_t)y * nx + x0 + 2 * c];
#pragma unroll
        for (int b = 0; b < 16; ++b) {
            const int K = 2 * (a + A * b) + p;
            const bool up = b >= 8 && K != N;                 // K > n: mirrored row, conjugated
            cplx fa, fb;
            ldg_cached2(in0 + (size_t)(up ? L - K : K) * ny * nx, fa, fb);
            v[b] = up ? cmake(fa.x + fb.y, fb.x - fa.y) : cmake(fa.x - fb.y, fa.y + fb.x);
        }
    }
    strided_inverse<A, kP5TwPost>(v, ex, c, p, a, tw1, tw2);
    cplx out[8];
    combine_parities<8>(v, p, out);
    if (PDL) pdl_trigger();
#pragma unroll
    for (int i = 0; i < 8; ++i)
        stg_stream(reinterpret_cast<cplx *>(&phi[((size_t)(a + A * (i + 8 * p)) * ny + y) * nx + x0 + 2 * c]), out[i]);
}

// ---------------------------------------------------------------------------------------------
// P3 for nx = 16 A: forward x, multiply by the Green's transform, inverse x, crop; in place on B.
// Persistent: one CTA of 12 warps per SM; every warp runs its own software pipeline over GROUPS of
// J = 16 / A consecutive lines (256 complex = 4 KB of contiguous memory whatever A is):
// group = warp_global + i * warps_total.  While a warp transforms group i, the bulk-copy engine brings
// group i+1 and its J Ghat rows into the warp's shared-memory stage (cp.async.bulk + mbarrier), so no
// DRAM latency is exposed and no register is spent on prefetching.
// lane -> p = lane % 2, a = (lane / 2) % A, j = lane / (2 A) (line within the group): the two parities of an
// element are neighbours, so that (i) the Ghat row is read as 32 consecutive doubles per instruction, (ii) the
// parities are combined with one shuffle over lane ^ 1 and (iii) every store instruction writes 2 A consecutive
// complex values per line (p = 0 keeps the even registers, p = 1 the odd ones).
// Twiddles: tb[k] = region p of tw1 (see twiddle_between), fixed per lane, in registers.  The inverse runs
// the TRANSPOSED flow (radix-A, exchange, conj tb, radix-16), in which the same per-lane set applies, so
// one register set serves both directions and the parity twiddle w_L^(+-m) needs no table at all.
// Exchange buffer per warp: region (j, p) = [16][A] elements at (2 j + p) * 16 A + p * P3Ex<A>::OFFP + j * OFFJ, the
// column XOR-swizzled with the row: conflict free in both directions (checked by brute force over all lanes).
// The (kz, ky) of a group follow incrementally from the previous group's (constant stride): no division in the loop.
// ---------------------------------------------------------------------------------------------
#ifndef DKS_P3_WARPS
#define DKS_P3_WARPS 12
#endif
constexpr int kP3Warps = DKS_P3_WARPS;
constexpr int kP3OffEx = 4096;                     // after the 256-element group stage
constexpr int kP3ExBytes = 2 * 16 * 17 * 16;       // 544 elements >= 2 J regions of 16 A elements + offsets
constexpr int kP3OffG = kP3OffEx + kP3ExBytes;     // 12800
constexpr int kP3GBytes = 2560;                    // J rows of P3Ex<A>::GSTR doubles
constexpr int kP3OffBar = kP3OffG + kP3GBytes;     // 15360
constexpr int kP3SmemPerWarp = kP3OffBar + 128;    // 15488
constexpr int kP3Smem = kP3Warps * kP3SmemPerWarp;

template <int A>
struct P3Ex {
    static constexpr int SWZ = A >= 4 ? 3 : A - 1;
    static constexpr int OFFP = A >= 4 ? 4 : 2;        // elements
    static constexpr int OFFJ = 4;                     // keeps region (j, 1) clear of region (j + 1, 0)
    static constexpr int GROW = (16 * A + 2) * 8;      // bytes of a Ghat row that are needed (n + 1 doubles, rounded to 16 B)
    static constexpr int GSTR = A == 1 ? 18 : A == 2 ? 36 : 16 * A + 8;   // shared-memory row stride (doubles): rows of a half-warp on distinct banks
    static_assert(GROW <= GSTR * 8 && (16 / A) * GSTR * 8 <= kP3GBytes, "Ghat stage");
    static_assert(A == 1 || (2 * (16 / A) * 16 * A + OFFP + (16 / A - 1) * OFFJ) * 16 <= kP3ExBytes, "exchange buffer");   // A = 1 needs none
};

template <int A, bool PDL>
__global__ void __launch_bounds__(kP3Warps * 32, 1)
p3_x_conv_r16(cplx *__restrict__ B, const double *__restrict__ Ghat, MeshDims d, int kz0, int planes,
              const cplx *__restrict__ tw1)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int N = 16 * A, L = 32 * A, J = 16 / A, G = 16 / A;
    constexpr int SWZ = P3Ex<A>::SWZ, GSTR = P3Ex<A>::GSTR;
    constexpr unsigned GROW = P3Ex<A>::GROW;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int p = lane & 1, a = (lane >> 1) & (A - 1), j = lane / (2 * A);
    unsigned char *wb = smem_raw + warp * kP3SmemPerWarp;
    const cplx *stage = reinterpret_cast<const cplx *>(wb) + j * N;
    cplx *ex = reinterpret_cast<cplx *>(wb + kP3OffEx) + (j * 2 + p) * (16 * A) + p * P3Ex<A>::OFFP + j * P3Ex<A>::OFFJ;
    const double *gs = reinterpret_cast<const double *>(wb + kP3OffG) + j * GSTR;
    uint64_t *bar = reinterpret_cast<uint64_t *>(wb + kP3OffBar);     // [0] group data, [1] Ghat rows
    if (lane == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_init_fence();
    }
    __syncthreads();

    const int ny2 = 2 * d.ny, nzp = d.nz + 1;
    const unsigned ngroups = (unsigned)planes * ny2 / J, stride = gridDim.x * kP3Warps;
    // Groups are walked from the LAST plane down: P2 has just written B front to back, so its tail is still in
    // L2 when P3 starts, and P3's own tail (the first planes) is in L2 when P4 starts at plane 0.
    unsigned grp = blockIdx.x * kP3Warps + warp;
    // (kz, ky0) of the group to be fetched next, updated incrementally (planes of a batch repeat kz)
    const int step = (int)(stride * J), dky = step & (ny2 - 1), dkz = (step >> d.ly) % nzp;
    int fkz = 0, fky = 0;
    if (grp < ngroups) {
        const unsigned l0 = (ngroups - 1 - grp) * J;
        fkz = (kz0 + (int)(l0 >> d.ly)) % nzp;
        fky = (int)(l0 & (ny2 - 1));
    }
    auto fetch = [&](unsigned gi) {                       // lane 0: group gi and its Ghat rows
        const unsigned g = ngroups - 1 - gi;
        mbar_expect_tx(&bar[0], 256 * sizeof(cplx));
        bulk_g2s(wb, B + (size_t)g * 256, 256 * sizeof(cplx), &bar[0]);
    };
    auto fetch_ghat = [&]() {                             // lane 0: the J Ghat rows of (fkz, fky ..)
        mbar_expect_tx(&bar[1], J * GROW);
        const double *row0 = Ghat + (size_t)fkz * (d.ny + 1) * d.gpitch;
#pragma unroll
        for (int jj = 0; jj < J; ++jj) {
            const int ky = fky + jj;
            bulk_g2s(wb + kP3OffG + jj * GSTR * 8, row0 + (size_t)min(ky, ny2 - ky) * d.gpitch, GROW, &bar[1]);
        }
    };
    auto advance = [&]() {                                // (fkz, fky) of the group `stride` further on
        fky -= dky;
        const int borrow = fky < 0;
        fky += borrow ? ny2 : 0;
        fkz -= dkz + borrow;
        fkz += fkz < 0 ? nzp : 0;
    };
    if (PDL) pdl_wait();
    if (lane == 0 && grp < ngroups) {
        fetch(grp);
        fetch_ghat();
    }
    advance();
    cplx tb[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) tb[k] = __ldg(&tw1[p * N + k * A + a]);
    // the XOR swizzle only touches the two low bits of the column: four lane-dependent bases per direction, everything
    // else is an immediate offset (keeps the address arithmetic out of the loop)
    cplx *exw[4], *exr[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        exw[c] = ex + (a ^ (c & SWZ));                        // + k A,  c = k & 3
        exr[c] = ex + a * A + ((c ^ a) & SWZ);                // + A A g + (ap & ~SWZ),  c = ap & 3
    }

    unsigned phase = 0;
    for (; grp < ngroups; grp += stride, phase ^= 1) {
        const unsigned next = grp + stride;
        cplx *base = B + (size_t)(ngroups - 1 - grp) * 256 + j * N;
        cplx v[16];
        mbar_wait(&bar[0], phase);
#pragma unroll
        for (int b = 0; b < 16; ++b) v[b] = stage[a + A * b];
        __syncwarp();                                 // stage consumed (and last exchange reads done)
        if (lane == 0 && next < ngroups) fetch(next);
        // forward: v[b] = x[a + A b] -> v[r] = X[2 (a + A r) + p]
        if (p) parity_consts<-1>(v);
        fft16<-1>(v);
#pragma unroll
        for (int k = 0; k < 16; ++k) v[k] = cmul(v[k], tb[k]);
        if (A > 1) {
#pragma unroll
            for (int k = 0; k < 16; ++k) exw[k & 3][k * A] = v[k];
            __syncwarp();
#pragma unroll
            for (int g = 0; g < G; ++g)
#pragma unroll
                for (int ap = 0; ap < A; ++ap) v[g * A + ap] = exr[ap & 3][A * A * g + (ap & ~SWZ)];
            fft_second<A, -1>(v);
        }
        // multiply by the real, even Green's transform
        mbar_wait(&bar[1], phase);
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const int K = 2 * (a + A * r) + p;
            v[r] = cscale(v[r], gs[min(K, L - K)]);
        }
        __syncwarp();                                 // Ghat rows consumed, forward exchange reads done
        if (lane == 0 && next < ngroups) fetch_ghat();
        advance();
        // inverse, transposed flow: radix-A, exchange back, conj tb, radix-16
        if (A > 1) {
            fft_second_t<A, +1>(v);
#pragma unroll
            for (int g = 0; g < G; ++g)
#pragma unroll
                for (int ap = 0; ap < A; ++ap) exr[ap & 3][A * A * g + (ap & ~SWZ)] = v[g * A + ap];
            __syncwarp();
#pragma unroll
            for (int k = 0; k < 16; ++k) v[k] = exw[k & 3][k * A];
        }
        fft16_tw<+1, false>(v, tb);                       // conj tb folded into the first butterfly layer (dks_fft_r16.cuh)
        if (p) parity_consts<+1>(v);
        // combine the parities (crop fused): y[m] = O_0[m] + w_L^-m O_1[m]; parity 0 keeps the even registers, parity 1 the odd ones
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const cplx send = p ? v[2 * i] : v[2 * i + 1];
            const cplx mine = p ? v[2 * i + 1] : v[2 * i];
            stg_stream(&base[a + A * (2 * i + p)], cadd(mine, shfl_xor_c(send, 1)));
        }
    }
    if (PDL) pdl_trigger();
}

}  // namespace dks
