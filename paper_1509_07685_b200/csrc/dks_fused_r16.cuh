// P2 + P3 + P4 in ONE persistent kernel for nx = 256, ny = 16 A (A in {2,4,8,16}).
//
// Why: P2, P3 and P4 act on independent kz planes of the half-spectrum and exchange the largest
// intermediate, B = [nz+1][2ny][nx] complex (539 MB at 256^3), twice through HBM.  Here a thread-block
// CLUSTER of CL CTAs takes one plane at a time through all three passes; the plane's B
// ([2ny][nx] complex, 2 MB at 256^3) is a per-cluster scratch in global memory that is rewritten for
// every plane and therefore stays in the 126 MB L2 (measured: profiles/).  HBM
// sees only the A plane in, its Ghat rows, and the A plane out (in place).
//
//   per plane kz (cluster c takes kz = c, c + #clusters, ...):
//     S1  column tiles (8 columns each, over the cluster's CTAs and the CTA's teams):  A[kz] --y fwd--> Bs
//         cluster barrier
//     S2  lines ky (over CTAs and warps): Bs[ky] <- x inv( Ghat(kz, ky', .) * x fwd(Bs[ky]) ), crop
//         cluster barrier
//     S3  column tiles:  Bs --y inv, crop--> A[kz]
//         cluster barrier   (Bs is reused by the next plane)
//
// The arithmetic of every stage is that of the separate kernels (dks_passes_r16.cuh): the two
// pruned length-n sub-transforms per padded line.  CTA = 512 threads = 512 / (16 A) column-tile teams
// (in lockstep behind __syncthreads) in S1/S3 and 16 line warps in S2; all twiddle tables live in shared
// memory (the L1 left beside 185 KB of shared memory is too small to hold them).  Scratch reads use
// ld.global.cg: another SM wrote the data, so L1 must be bypassed.
// Opt-in (dks_poisson_set_fused): measured slower than the separate passes so far, DESIGN.md section 5.
#pragma once
#include "dks_passes_r16.cuh"

namespace dks {

constexpr int kFusedThreads = 512;
constexpr int kFusedWarps = kFusedThreads / 32;
constexpr int kFusedNx = 256;                      // the line stage is written for nx = 256 (A_x = 16)

// shared-memory layout (bytes)
constexpr int kFusedOffTw1x = 0;                                   // regions 0, 1 of the x table (twiddle_between): 2 x 256
constexpr int kFusedOffTw1y = kFusedOffTw1x + 512 * 16;            // regions 0, 1, 2 of the y table: 3 x n, n <= 256
constexpr int kFusedOffWork = kFusedOffTw1y + 768 * 16;            // union: team exchange buffers / per-warp line buffers
constexpr int kFusedLineEx = 8192;                                 // per warp: exchange [2][16][16] cplx
constexpr int kFusedLineG = 2112;                                  // per warp: Ghat row, 264 doubles
constexpr int kFusedLineBytes = kFusedLineEx + kFusedLineG;        // 10304
constexpr int kFusedWorkBytes = kFusedWarps * kFusedLineBytes;     // 164864 >= 2 teams x 64 KB
constexpr int kFusedSmem = kFusedOffWork + kFusedWorkBytes;        // 181248

// Scratch accesses: another SM wrote the data, so L1 must not serve it (ld.global.cg; nothing ever allocates
// these lines in L1); the A plane and the Ghat rows stream through with L1::no_allocate.  (L2 eviction
// policies through createpolicy / L2::cache_hint -- evict_last for the scratch, evict_first for the streams --
// cut the scratch write-back traffic by a third but are left out: see DESIGN.md section 5.)
__device__ __forceinline__ cplx ldg_scr(const cplx *p, uint64_t)
{
    cplx r;
    asm volatile("ld.global.cg.v2.f64 {%0, %1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ void stg_scr(cplx *p, cplx v, uint64_t)
{
    asm volatile("st.global.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ cplx ldg_once(const cplx *p, uint64_t) { return ldg_stream(p); }
__device__ __forceinline__ void stg_once(cplx *p, cplx v, uint64_t) { stg_stream(p, v); }
__device__ __forceinline__ void cp_async16_hint(void *smem_dst, const void *gmem_src, uint64_t) { cp_async16(smem_dst, gmem_src); }
__device__ __forceinline__ uint64_t l2_policy_evict_last() { return 0; }
__device__ __forceinline__ uint64_t l2_policy_evict_first() { return 0; }
// The column-tile teams of a CTA run in lockstep behind __syncthreads(): every team has the same number of
// tiles (the host only selects a cluster size with (nx / 8) % (CL * teams) == 0).  Named barriers per team
// (bar.sync id, count) were tried first and produced sporadic cudaErrorIllegalInstruction on some
// instantiations, depending on unrelated code changes; barrier 0 has never shown it.
__device__ __forceinline__ void team_sync(int, int) { __syncthreads(); }
__device__ __forceinline__ void cluster_sync_all()
{
    __cluster_barrier_arrive();        // release
    __cluster_barrier_wait();          // acquire
}
__device__ __forceinline__ unsigned cluster_ctarank()
{
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ unsigned cluster_id_x()
{
    unsigned r;
    asm volatile("mov.u32 %0, %%clusterid.x;" : "=r"(r));
    return r;
}
__device__ __forceinline__ unsigned nclusters_x()
{
    unsigned r;
    asm volatile("mov.u32 %0, %%nclusterid.x;" : "=r"(r));
    return r;
}

__device__ __forceinline__ void cp_async_wait_all_fused() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// Every stage is software pipelined without spending registers: while a tile (line) is transformed, the
// next one travels global -> shared memory through cp.async (LDGSTS).  The landing zone is the exchange
// buffer itself, which is idle between the exchange read of one tile and the exchange write of the next.

// ---- S1: this team's column tiles t0, t0 + tstep, ... < xtiles, forward y (arithmetic of p2_y_fwd_r16) --
template <int A>
__device__ __forceinline__ void fused_tiles_fwd(const cplx *__restrict__ Aplane, cplx *__restrict__ Bs, int nx, int t0, int tstep,
                                                int xtiles, int tt, cplx *ex, const cplx *tw1s, int bar_id,
                                                uint64_t keep, uint64_t once)
{
    constexpr int T = 16 * A, G = 16 / A, N = 16 * A;
    const int c = tt & 7, p = (tt >> 3) & 1, a = tt >> 4;
    auto prefetch = [&](int t) {                       // N rows x 128 B -> ex[row][8]
#pragma unroll
        for (int i = 0; i < N * kCols / T; ++i) {
            const int idx = tt + i * T, r = idx >> 3, cc = idx & 7;
            cp_async16_hint(&ex[idx], &Aplane[(size_t)r * nx + (size_t)t * kCols + cc], once);
        }
        cp_async_commit();
    };
    if (t0 < xtiles) prefetch(t0);
    for (int t = t0; t < xtiles; t += tstep) {
        const size_t x = (size_t)t * kCols + c;
        cplx v[16];
        cp_async_wait_all_fused();
        team_sync(bar_id, T);                          // tile landed
#pragma unroll
        for (int b = 0; b < 16; ++b) v[b] = ex[(a + A * b) * kCols + c];
        team_sync(bar_id, T);                          // tile consumed: ex becomes the exchange buffer
        if (p) parity_consts<-1>(v);
        fft16<-1>(v);
        twiddle_between_s<A, -1>(v, tw1s + p * N, a);
#pragma unroll
        for (int k = 0; k < 16; ++k) ex[((p * 16 + k) * A + a) * kCols + c] = v[k];
        team_sync(bar_id, T);
#pragma unroll
        for (int g = 0; g < G; ++g)
#pragma unroll
            for (int ap = 0; ap < A; ++ap) v[g * A + ap] = ex[((p * 16 + a + A * g) * A + ap) * kCols + c];
        team_sync(bar_id, T);                          // exchange read by all: ex free for the next tile
        if (t + tstep < xtiles) prefetch(t + tstep);
        fft_second<A, -1>(v);
#pragma unroll
        for (int r = 0; r < 16; ++r) stg_scr(&Bs[(size_t)(2 * (a + A * r) + p) * nx + x], v[r], keep);
    }
}

// ---- S3: this team's column tiles, inverse y + crop (arithmetic of p4_y_inv_r16) ----------------------
template <int A>
__device__ __forceinline__ void fused_tiles_inv(const cplx *__restrict__ Bs, cplx *__restrict__ Aplane, int nx, int t0, int tstep,
                                                int xtiles, int tt, cplx *ex, const cplx *tw1s, int bar_id,
                                                uint64_t keep, uint64_t once)
{
    constexpr int T = 16 * A, G = 16 / A, N = 16 * A;
    const int c = tt & 7, p = (tt >> 3) & 1, a = tt >> 4;
    auto prefetch = [&](int t) {                       // 2N rows x 128 B -> ex[row][8]
#pragma unroll
        for (int i = 0; i < 2 * N * kCols / T; ++i) {
            const int idx = tt + i * T, r = idx >> 3, cc = idx & 7;
            cp_async16_hint(&ex[idx], &Bs[(size_t)r * nx + (size_t)t * kCols + cc], keep);
        }
        cp_async_commit();
    };
    if (t0 < xtiles) prefetch(t0);
    for (int t = t0; t < xtiles; t += tstep) {
        const size_t x = (size_t)t * kCols + c;
        cplx v[16];
        cp_async_wait_all_fused();
        team_sync(bar_id, T);
#pragma unroll
        for (int b = 0; b < 16; ++b) v[b] = ex[(2 * (a + A * b) + p) * kCols + c];
        team_sync(bar_id, T);
        fft16<+1>(v);
        twiddle_between_s<A, +1>(v, tw1s + p * 2 * N, a);
#pragma unroll
        for (int k = 0; k < 16; ++k) ex[((p * 16 + k) * A + a) * kCols + c] = v[k];
        team_sync(bar_id, T);
#pragma unroll
        for (int g = 0; g < G; ++g)
#pragma unroll
            for (int ap = 0; ap < A; ++ap) v[g * A + ap] = ex[((p * 16 + a + A * g) * A + ap) * kCols + c];
        team_sync(bar_id, T);
        if (t + tstep < xtiles) prefetch(t + tstep);
        fft_second<A, +1>(v);
        if (p) parity_consts<+1>(v);
        cplx out[8];
        combine_parities<8>(v, p, out);
#pragma unroll
        for (int i = 0; i < 8; ++i) stg_once(&Aplane[(size_t)(a + A * (i + 8 * p)) * nx + x], out[i], once);
    }
}

// ---- S2: this warp's lines ky0, ky0 + kstep, ... < 2ny: forward x, times Ghat, inverse x, crop; in place
// (arithmetic of p3_x_conv_r16).  lane -> a = lane & 15, p = lane >> 4.  exw: the warp's exchange buffer
// [2][16][16] (its first 4 KB double as the landing zone of the next line); gs: the warp's Ghat row.
__device__ __forceinline__ void fused_lines(cplx *__restrict__ Bs, const double *__restrict__ Gplane, int gpitch, int nx, int ny2,
                                            int ky0, int kstep, int lane, cplx *exw, double *gs, const cplx *tw1s,
                                            uint64_t keep, uint64_t once)
{
    constexpr int A = 16, L = 512, N = 256;
    const int a = lane & 15, p = lane >> 4;
    cplx *ex = exw + p * 256;
    auto prefetch_line = [&](int ky) {
        const cplx *src = Bs + (size_t)ky * nx;
#pragma unroll
        for (int i = 0; i < N / 32; ++i) cp_async16_hint(&exw[lane + 32 * i], &src[lane + 32 * i], keep);
        cp_async_commit();
    };
    auto prefetch_ghat = [&](int ky) {                 // row of gpitch = 264 doubles = 132 16-byte chunks
        const double *grow = Gplane + (size_t)min(ky, ny2 - ky) * gpitch;
#pragma unroll
        for (int i = 0; i < 5; ++i) {
            const int ch = lane + 32 * i;
            if (ch < kFusedLineG / 16) cp_async16_hint(gs + 2 * ch, grow + 2 * ch, once);
        }
        cp_async_commit();
    };
    if (ky0 < ny2) {
        prefetch_line(ky0);
        prefetch_ghat(ky0);
    }
    for (int ky = ky0; ky < ny2; ky += kstep) {
        cplx *line = Bs + (size_t)ky * nx;
        const bool more = ky + kstep < ny2;
        cplx v[16];
        cp_async_wait_all_fused();
        __syncwarp();                                  // line and Ghat row landed
#pragma unroll
        for (int b = 0; b < 16; ++b) v[b] = exw[a + A * b];
        __syncwarp();                                  // line consumed: exw becomes the exchange buffer
        if (p) parity_consts<-1>(v);
        fft16<-1>(v);
        twiddle_between_s<A, -1>(v, tw1s + p * N, a);
#pragma unroll
        for (int k = 0; k < 16; ++k) ex[k * 16 + (a ^ (k & 7))] = v[k];
        __syncwarp();
#pragma unroll
        for (int ap = 0; ap < 16; ++ap) v[ap] = ex[a * 16 + (ap ^ (a & 7))];
        fft16<-1>(v);
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const int K = 2 * (a + A * r) + p;
            v[r] = cscale(v[r], gs[min(K, L - K)]);
        }
        __syncwarp();                                  // Ghat row consumed; forward exchange reads done
        if (more) prefetch_ghat(ky + kstep);
        fft16<+1>(v);                                  // transposed inverse flow (see p3_x_conv_r16)
#pragma unroll
        for (int k = 0; k < 16; ++k) ex[k * 16 + (a ^ (k & 7))] = v[k];
        __syncwarp();
#pragma unroll
        for (int ap = 0; ap < 16; ++ap) v[ap] = ex[a * 16 + (ap ^ (a & 7))];
        __syncwarp();                                  // exchange read by all lanes: exw free for the next line
        if (more) prefetch_line(ky + kstep);
        twiddle_between_s<A, +1>(v, tw1s + p * N, a);
        fft16<+1>(v);
        if (p) parity_consts<+1>(v);
        cplx out[8];
        combine_parities<16>(v, p, out);
#pragma unroll
        for (int i = 0; i < 8; ++i) stg_scr(&line[a + A * (i + 8 * p)], out[i], keep);
    }
}

// ---------------------------------------------------------------------------------------------
// The kernel.  grid = CL * (#clusters), cluster dimension (CL, 1, 1), 512 threads,
// kFusedSmem bytes of dynamic shared memory.  Bscr: #clusters scratch planes of [2ny][nx] complex.
// ---------------------------------------------------------------------------------------------
template <int A, int CL>
__global__ void __launch_bounds__(kFusedThreads, 1)
p234_fused_r16(cplx *__restrict__ Abuf, cplx *__restrict__ Bscr, const double *__restrict__ Ghat, MeshDims d,
               const cplx *__restrict__ tw1x, const cplx *__restrict__ tw1y)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int T = 16 * A, TEAMS = kFusedThreads / T, N = 16 * A;
    cplx *tw1xs = reinterpret_cast<cplx *>(smem_raw + kFusedOffTw1x);
    cplx *tw1ys = reinterpret_cast<cplx *>(smem_raw + kFusedOffTw1y);
    unsigned char *work = smem_raw + kFusedOffWork;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int i = tid; i < 768; i += kFusedThreads) {
        if (i < 512) tw1xs[i] = __ldg(&tw1x[i]);
        if (i < 3 * N) tw1ys[i] = __ldg(&tw1y[i]);
    }
    __syncthreads();

    const int nx = d.nx, ny = d.ny, ny2 = 2 * ny;
    const uint64_t keep = l2_policy_evict_last(), once = l2_policy_evict_first();
    const int rank = (int)cluster_ctarank(), cid = (int)cluster_id_x(), ncl = (int)nclusters_x();
    cplx *Bs = Bscr + (size_t)cid * ny2 * nx;
    // S1 / S3 roles
    const int team = tid / T, tt = tid % T;
    cplx *ex_team = reinterpret_cast<cplx *>(work) + (size_t)team * 2 * 16 * A * kCols;
    const int xtiles = nx / kCols;
    // S2 role
    cplx *ex_warp = reinterpret_cast<cplx *>(work + warp * kFusedLineBytes);
    double *gs_warp = reinterpret_cast<double *>(work + warp * kFusedLineBytes + kFusedLineEx);

    for (int kz = cid; kz <= d.nz; kz += ncl) {
        cplx *Aplane = Abuf + (size_t)kz * ny * nx;
        fused_tiles_fwd<A>(Aplane, Bs, nx, rank * TEAMS + team, CL * TEAMS, xtiles, tt, ex_team, tw1ys, 1 + team, keep, once);
        __syncthreads();
        cluster_sync_all();
        fused_lines(Bs, Ghat + (size_t)kz * (ny + 1) * d.gpitch, d.gpitch, nx, ny2, rank * kFusedWarps + warp, CL * kFusedWarps,
                    lane, ex_warp, gs_warp, tw1xs, keep, once);
        __syncthreads();
        cluster_sync_all();
        fused_tiles_inv<A>(Bs, Aplane, nx, rank * TEAMS + team, CL * TEAMS, xtiles, tt, ex_team, tw1ys, 1 + team, keep, once);
        __syncthreads();
        cluster_sync_all();
    }
}

}  // namespace dks
