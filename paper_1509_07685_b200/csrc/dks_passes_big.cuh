// The five passes for long lines: mesh extent n = 512 or 1024 on the pass's own axis (padded L = 1024, 2048), e.g. the z axis
// of BASELINE.json config 5 (64 x 64 x 512) and the x, y axes of the paper's largest mesh (512 x 512 x 256).
// Same buffers, layouts and fusions as the other variants (dks_passes_generic.cuh), so any pass may use any variant; the
// transform is the three-stage register radix-16 tile FFT of dks_fft_big.cuh.  One CTA = BigGeom<L>::THREADS threads = one
// tile of W lines.  Stage 1 of a forward pass is fed straight from global memory and the last stage stores straight to
// global memory wherever the pass's data flow allows it (P2, P4; the load of P1; the store of P5), so those tiles cross
// shared memory twice, not four times.
#pragma once
#include "dks_fft_big.cuh"
#include "dks_passes_generic.cuh"

namespace dks {

// ---- P2: forward y.  grid (nx / W, planes * batch) ---------------------------------------------------------------------
template <int L, bool PDL = false>
__global__ void __launch_bounds__(BigGeom<L>::THREADS, BigGeom<L>::MINB)
p2_y_fwd_big(const cplx *__restrict__ A, cplx *__restrict__ B, MeshDims d, int kz0, const cplx *__restrict__ tw)
{
    extern __shared__ cplx s[];
    typedef BigGeom<L> G;
    typedef BigStage<L, G::W> St;
    constexpr int N = L / 2;
    const int nx = d.nx, tid = threadIdx.x, w = tid % G::W, u = tid / G::W;
    const size_t x = (size_t)blockIdx.x * G::W + w;
    const cplx *in = A + ((size_t)(kz0 + blockIdx.y) * N) * nx + x;
    cplx *out = B + ((size_t)blockIdx.y * L) * nx + x;
    cplx v[16];
    if (PDL) pdl_wait();
#pragma unroll
    for (int m = 0; m < 16; ++m) v[m] = m < 8 ? ldg_stream(&in[(size_t)(u + G::S1 * m) * nx]) : cmake(0.0, 0.0);
    St::fwd1(v, tw, u);
    St::put1(s, v, u, w);
    __syncthreads();
    St::template stage2<-1>(s, tw, u, w);
    __syncthreads();
    St::get3(s, v, u, w);
    St::template bfly3<-1>(v);
    if (PDL) pdl_trigger();
#pragma unroll
    for (int i = 0; i < 16; ++i) stg_stream(&out[(size_t)big_freq_of<L>(16 * u + i) * nx], v[i]);
}

// ---- P4: inverse y, crop -----------------------------------------------------------------------------------------------
template <int L, bool PDL = false>
__global__ void __launch_bounds__(BigGeom<L>::THREADS, BigGeom<L>::MINB)
p4_y_inv_big(const cplx *__restrict__ B, cplx *__restrict__ A, MeshDims d, int kz0, const cplx *__restrict__ tw)
{
    extern __shared__ cplx s[];
    typedef BigGeom<L> G;
    typedef BigStage<L, G::W> St;
    constexpr int N = L / 2;
    const int nx = d.nx, tid = threadIdx.x, w = tid % G::W, u = tid / G::W;
    const size_t x = (size_t)blockIdx.x * G::W + w;
    const cplx *in = B + ((size_t)blockIdx.y * L) * nx + x;
    cplx *out = A + ((size_t)(kz0 + blockIdx.y) * N) * nx + x;
    cplx v[16];
    if (PDL) pdl_wait();
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = ldg_stream(&in[(size_t)big_freq_of<L>(16 * u + i) * nx]);
    St::template bfly3<+1>(v);
    St::put3(s, v, u, w);
    __syncthreads();
    St::template stage2<+1>(s, tw, u, w);
    __syncthreads();
    St::get1(s, v, u, w);
    St::inv1(v, tw, u);
    if (PDL) pdl_trigger();
#pragma unroll
    for (int q = 0; q < 8; ++q) stg_stream(&out[(size_t)(u + G::S1 * q) * nx], v[q]);
}

// ---- P1: forward z, real -> complex (two real columns packed into one complex line, split afterwards) -----------------
template <int L, bool PDL = false>
__global__ void __launch_bounds__(BigGeom<L>::THREADS, BigGeom<L>::MINB)
p1_z_r2c_big(const double *__restrict__ rho, cplx *__restrict__ A, MeshDims d, const cplx *__restrict__ tw)
{
    extern __shared__ cplx s[];
    typedef BigGeom<L> G;
    typedef BigStage<L, G::W> St;
    constexpr int W = G::W, NT = G::THREADS, N = L / 2;
    const int nx = d.nx, ny = d.ny, x0 = blockIdx.x * 2 * W, y = blockIdx.y, tid = threadIdx.x, w = tid % W, u = tid / W;
    rho += (size_t)blockIdx.z * N * ny * nx;              // blockIdx.z: mesh of the batch
    A += (size_t)blockIdx.z * (N + 1) * ny * nx;
    cplx v[16];
    if (PDL) pdl_wait();                                  // A is still being read by the previous solve's P5
#pragma unroll
    for (int m = 0; m < 16; ++m)
        v[m] = m < 8 ? ldg_stream(reinterpret_cast<const cplx *>(&rho[((size_t)(u + G::S1 * m) * ny + y) * nx + x0 + 2 * w])) : cmake(0.0, 0.0);
    St::fwd1(v, tw, u);
    St::put1(s, v, u, w);
    __syncthreads();
    St::template stage2<-1>(s, tw, u, w);
    __syncthreads();
    St::get3(s, v, u, w);
    St::template bfly3<-1>(v);
    St::put3(s, v, u, w);
    __syncthreads();
    if (PDL) pdl_trigger();
    for (int idx = tid; idx < (N + 1) * W; idx += NT) {
        const int k = idx / W, ww = idx % W;
        const cplx ck = s[big_pos_of<L>(k) * W + ww], cm = s[big_pos_of<L>((L - k) & (L - 1)) * W + ww];
        stg_stream2(&A[((size_t)k * ny + y) * nx + x0 + 2 * ww], cmake(0.5 * (ck.x + cm.x), 0.5 * (ck.y - cm.y)),
                    cmake(0.5 * (ck.y + cm.y), -0.5 * (ck.x - cm.x)));
    }
}

// ---- P5: inverse z, complex -> real, crop ------------------------------------------------------------------------------
template <int L, bool PDL = false>
__global__ void __launch_bounds__(BigGeom<L>::THREADS, BigGeom<L>::MINB)
p5_z_c2r_big(const cplx *__restrict__ A, double *__restrict__ phi, MeshDims d, const cplx *__restrict__ tw)
{
    extern __shared__ cplx s[];
    typedef BigGeom<L> G;
    typedef BigStage<L, G::W> St;
    constexpr int W = G::W, NT = G::THREADS, N = L / 2;
    const int nx = d.nx, ny = d.ny, x0 = blockIdx.x * 2 * W, y = blockIdx.y, tid = threadIdx.x, w = tid % W, u = tid / W;
    A += (size_t)blockIdx.z * (N + 1) * ny * nx;
    phi += (size_t)blockIdx.z * N * ny * nx;
    if (PDL) pdl_wait();
#pragma unroll 2
    for (int idx = tid; idx < (N + 1) * W; idx += NT) {
        const int k = idx / W, ww = idx % W;
        cplx fa, fb;
        ldg_stream2(&A[((size_t)k * ny + y) * nx + x0 + 2 * ww], fa, fb);
        s[big_pos_of<L>(k) * W + ww] = cmake(fa.x - fb.y, fa.y + fb.x);                    // fa + i fb
        if (k > 0 && k < N) s[big_pos_of<L>(L - k) * W + ww] = cmake(fa.x + fb.y, fb.x - fa.y);   // conj(fa) + i conj(fb)
    }
    __syncthreads();
    cplx v[16];
    St::get3(s, v, u, w);
    __syncthreads();                                      // every position read before stage 3 writes back
    St::template bfly3<+1>(v);
    St::put3(s, v, u, w);
    __syncthreads();
    St::template stage2<+1>(s, tw, u, w);
    __syncthreads();
    St::get1(s, v, u, w);
    St::inv1(v, tw, u);
    if (PDL) pdl_trigger();
#pragma unroll
    for (int q = 0; q < 8; ++q)
        stg_stream(reinterpret_cast<cplx *>(&phi[((size_t)(u + G::S1 * q) * ny + y) * nx + x0 + 2 * w]), v[q]);
}

// ---- P3: forward x, multiply by the Green's transform, inverse x, crop; in place; W consecutive lines per CTA -----------
// The forward's stage 3, the multiplication and the inverse's stage 3 work on the same 16 registers.  The W Green's rows
// are staged in shared memory behind the tile (coalesced row reads instead of scattered 8-byte gathers from L2).
// Staged Green's rows: a warp reads them with lanes = (4 or 8 sets u) x (W lines w), and the frequencies of neighbouring sets
// differ by multiples of 64 (L = 1024) or 32 (L = 2048) -- with plain rows of L/2 + 8 doubles all 32 lanes met in two banks
// (ncu, 512 x 512 x 256: 1.2e8 conflicts per launch).  Entry k of a row therefore sits at k + (k >> SH) (injective up to
// the Nyquist entry k = L/2, which lands at L/2 + 8 or + 32), and the row stride is 4 (W = 8) or 8 (W = 4) doubles past a
// multiple of 16, which spreads (u, w) over all sixteen 8-byte banks.
// W lines per CTA and one CTA per SM, as in the strided passes (tried in round 3: W = 4 with two CTAs per SM needs an unpadded
// tile to keep the quarter-warp stage accesses conflict free and was slower, 3.83 against 3.56 ms at 512 x 512 x 256).
template <int L>
struct P3BigGeom {
    static constexpr int W = BigGeom<L>::W, WP = BigGeom<L>::WPX;
    static constexpr int THREADS = BigGeom<L>::THREADS, MINB = 1;
    static constexpr int SH = L == 1024 ? 6 : 5;
    static constexpr int GROW = L == 1024 ? 532 : 1064;       // doubles per staged Green's row (> gpos(L/2))
    static constexpr int SMEM = L * WP * (int)sizeof(cplx) + W * GROW * (int)sizeof(double);
    static __device__ __forceinline__ int gpos(int k) { return k + (k >> SH); }
    static_assert(GROW > L / 2 + ((L / 2) >> SH) && GROW % 16 == 32 / W, "Green's row stride");
    static_assert(MINB * (SMEM + 1024) <= 227 * 1024, "shared memory per SM");
    static_assert((L / 2) % THREADS == 0 && (L / 2 * W) % THREADS == 0 && W <= THREADS, "fill loops");
};

template <int L, bool PDL = false>
__global__ void __launch_bounds__(P3BigGeom<L>::THREADS, P3BigGeom<L>::MINB)
p3_x_conv_big(cplx *__restrict__ B, const double *__restrict__ Ghat, MeshDims d, int kz0, const cplx *__restrict__ tw)
{
    extern __shared__ cplx s[];
    typedef BigGeom<L> G;
    constexpr int W = P3BigGeom<L>::W, WP = P3BigGeom<L>::WP, NT = P3BigGeom<L>::THREADS, N = L / 2, GROW = P3BigGeom<L>::GROW;
    typedef BigStage<L, WP> St;
    double *gs = reinterpret_cast<double *>(s + L * WP);
    const int ny = d.ny, tid = threadIdx.x, w = tid % W, u = tid / W;
    const int line0 = blockIdx.x * W;
    const int kz = (kz0 + line0 / (2 * ny)) % (d.nz + 1), ky0 = line0 % (2 * ny);    // a batch repeats kz
    cplx *base = B + (size_t)line0 * N;
    if (PDL) pdl_wait();
    // Every global load of the CTA is issued before the first shared-memory store: the tile (N W / NT = 8 x 16 bytes per
    // thread) and the W Green's rows (row ww: entries tid + j NT, the Nyquist entry by thread ww).  Written as load-store
    // loops the compiler kept one load in flight per thread, and with one CTA per SM the nine round trips to L2 / HBM of
    // the Green's rows alone took 6 of the 16 us a tile spent on the SM (ncu r3: the STS behind the load held the samples).
    {
        constexpr int TIT = N * W / NT, KPR = N / NT;
        const double *grow0 = Ghat + (size_t)kz * (ny + 1) * d.gpitch;
        cplx t[TIT];
        double g[W][KPR], gn = 0.0;
#pragma unroll
        for (int it = 0; it < TIT; ++it) t[it] = ldg_stream(&base[tid + it * NT]);
#pragma unroll
        for (int ww = 0; ww < W; ++ww) {
            const int ky = ky0 + ww;
            const double *row = grow0 + (size_t)min(ky, 2 * ny - ky) * d.gpitch;
#pragma unroll
            for (int j = 0; j < KPR; ++j) g[ww][j] = __ldg(&row[tid + j * NT]);
        }
        if (tid < W) {
            const int ky = ky0 + tid;
            gn = __ldg(&grow0[(size_t)min(ky, 2 * ny - ky) * d.gpitch + N]);
        }
#pragma unroll
        for (int it = 0; it < TIT; ++it) {
            const int idx = tid + it * NT, ww = idx / N, pp = idx % N;
            s[pp * WP + ww] = t[it];
        }
#pragma unroll
        for (int ww = 0; ww < W; ++ww)
#pragma unroll
            for (int j = 0; j < KPR; ++j) gs[ww * GROW + P3BigGeom<L>::gpos(tid + j * NT)] = g[ww][j];
        if (tid < W) gs[tid * GROW + P3BigGeom<L>::gpos(N)] = gn;
    }
    __syncthreads();
    cplx v[16];
#pragma unroll
    for (int m = 0; m < 16; ++m) v[m] = m < 8 ? s[(u + G::S1 * m) * WP + w] : cmake(0.0, 0.0);
    __syncthreads();                                      // stage 1 reads 8 positions per set but writes 16
    St::fwd1(v, tw, u);
    St::put1(s, v, u, w);
    __syncthreads();
    St::template stage2<-1>(s, tw, u, w);
    __syncthreads();
    St::get3(s, v, u, w);
    St::template bfly3<-1>(v);
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int kx = big_freq_of<L>(16 * u + i);
        v[i] = cscale(v[i], gs[w * GROW + P3BigGeom<L>::gpos(min(kx, L - kx))]);
    }
    St::template bfly3<+1>(v);
    St::put3(s, v, u, w);
    __syncthreads();
    // The inverse stages read the same twiddle-table entries as the forward ones (tw[u q], tw[16 j q]).  Seen through the
    // same `u`, the compiler keeps all 2 x 15 of them in registers from the forward half on (read-only loads are merged) and
    // spills 270 bytes per thread to make room: at 512 x 512 x 256 that was 9 GB of local-memory traffic through L2 per
    // launch and a 4.2 ms kernel.  An opaque copy of u makes the inverse half reload them.
    int ui = u;
    asm volatile("" : "+r"(ui));
    St::template stage2<+1>(s, tw, ui, w);
    __syncthreads();
    St::get1(s, v, ui, w);
    St::inv1(v, tw, ui);
    __syncthreads();                                      // all stage-1 reads done before the cropped result is written
    St::put1(s, v, ui, w, 8);
    __syncthreads();
    if (PDL) pdl_trigger();
#pragma unroll 4
    for (int idx = tid; idx < N * W; idx += NT) {
        const int ww = idx / N, pp = idx % N;
        stg_stream(&base[(size_t)ww * N + pp], s[pp * WP + ww]);
    }
}

// ---- a0: one axis of the Green's transform (even extension, two real lines per complex transform), in place ------------
// lines are enumerated as l = b * na + a with base offset a * sa + b * sb, elements at stride es (see greens_axis_kernel)
template <int L>
__global__ void __launch_bounds__(BigGeom<L>::THREADS, 1)
greens_axis_big(double *__restrict__ G, long long es, int na, long long sa, int nb, long long sb, double scale,
                const cplx *__restrict__ tw)
{
    extern __shared__ cplx s[];
    typedef BigGeom<L> Gm;
    constexpr int W = Gm::W, WP = Gm::WPX, NT = Gm::THREADS, N = L / 2;
    typedef BigStage<L, WP> St;
    const int tid = threadIdx.x, w = tid % W, u = tid / W;
    const long long l0 = 2 * (long long)blockIdx.x * W, nlines = (long long)na * nb;
    for (int idx = tid; idx < L * W; idx += NT) {
        const int p = idx / W, ww = idx % W;
        const long long l1 = l0 + 2 * ww, l2 = l1 + 1, e = (long long)min(p, L - p) * es;
        double v1 = 0.0, v2 = 0.0;
        if (l1 < nlines) v1 = G[(l1 % na) * sa + (l1 / na) * sb + e];
        if (l2 < nlines) v2 = G[(l2 % na) * sa + (l2 / na) * sb + e];
        s[p * WP + ww] = cmake(v1, v2);
    }
    __syncthreads();
    cplx v[16];
    St::get1(s, v, u, w);
    St::fwd1(v, tw, u);
    St::put1(s, v, u, w);
    __syncthreads();
    St::template stage2<-1>(s, tw, u, w);
    __syncthreads();
    St::get3(s, v, u, w);
    St::template bfly3<-1>(v);
    St::put3(s, v, u, w);
    __syncthreads();
    for (int idx = tid; idx < (N + 1) * W; idx += NT) {
        const int k = idx / W, ww = idx % W;
        const long long l1 = l0 + 2 * ww, l2 = l1 + 1;
        const cplx c = s[big_pos_of<L>(k) * WP + ww];
        if (l1 < nlines) G[(l1 % na) * sa + (l1 / na) * sb + (long long)k * es] = c.x * scale;
        if (l2 < nlines) G[(l2 % na) * sa + (l2 / na) * sb + (long long)k * es] = c.y * scale;
    }
}

}  // namespace dks
