// Shared-memory tile FFT with register radix-16 stages for the long lines, L = 1024 and 2048 (mesh extents n = 512, 1024).
//
// Tile layout as in dks_fft_generic.cuh: element at position P of line w lives at s[P * WP + w].  L = 16 x 16 x R3, R3 = 4 or
// 8, so a transform is three stages of register butterflies with compile-time strides instead of five or six radix-4 passes;
// every thread owns one set of 16 elements per stage:
//   stage 1 (sub-problem length L):      set u holds positions u + (L/16) m, m < 16
//   stage 2 (length L/16):               set u holds q1 (L/16) + j + (L/256) m with q1 = u / (L/256), j = u % (L/256)
//   stage 3 (length R3):                 set u holds the 16 contiguous positions 16 u + i (16 / R3 sub-problems)
// Forward (decimation in frequency): butterfly, then twiddle w_S^(j q); natural order in, and after stage 3 position
// P = q1 (L/16) + q2 (L/256) + q3 holds X[q1 + 16 q2 + 256 q3] (big_freq_of / big_pos_of).  Inverse (decimation in time): the
// stages in reverse order, conjugate twiddle first, then the butterfly; permuted order in, natural order out.
// The stages are exposed one by one so that a pass can feed stage 1 straight from global memory and store straight from the
// last stage's registers: the tile then crosses shared memory twice per transform, like a register-resident four-step FFT.
// Pruning (the upper half of a padded line is zero; the upper half of an inverse is cropped) falls out of the
// register code: stage 1 of a forward transform is fed constant zeros for m >= 8, stage 1 of an inverse stores q < 8 only.
// Threads: tid -> line w = tid % W (fastest: W lanes = W * 16 contiguous bytes), set u = tid / W; THREADS = (L / 16) * W.
#pragma once
#include "dks_fft_r16.cuh"

namespace dks {

#ifndef DKS_BIG_W1024
#define DKS_BIG_W1024 8
#endif
#ifndef DKS_BIG_W2048
#define DKS_BIG_W2048 4
#endif

template <int L>
struct BigGeom {
    static_assert(L == 1024 || L == 2048, "L = 1024 or 2048");
    static constexpr int W = L == 1024 ? DKS_BIG_W1024 : DKS_BIG_W2048;   // lines per tile
    static constexpr int WPX = W + 1;                         // padded row for tiles that are filled line by line (x lines)
    static constexpr int R3 = L / 256;                        // radix of the last stage: 4 or 8
    static constexpr int S1 = L / 16, S2 = L / 256;           // element strides of stages 1 and 2
    static constexpr int THREADS = (L / 16) * W;
    static constexpr int MINB = 512 / THREADS > 0 ? 512 / THREADS : 1;
    static constexpr int SMEM = L * W * (int)sizeof(cplx);
    static constexpr int SMEMX = L * WPX * (int)sizeof(cplx);
};

// position in the tile of frequency k after the forward transform (and expected by the inverse), and its inverse map
template <int L>
__device__ __forceinline__ int big_pos_of(int k) { return (k & 15) * (L / 16) + ((k >> 4) & 15) * (L / 256) + (k >> 8); }
template <int L>
__device__ __forceinline__ int big_freq_of(int P) { return P / (L / 16) + 16 * ((P / (L / 256)) & 15) + 256 * (P % (L / 256)); }

template <int R, int SIGN>
__device__ __forceinline__ void bfly_r(cplx *v)
{
    if (R == 4) bfly4<SIGN>(v[0], v[1], v[2], v[3]);
    if (R == 8) bfly8<SIGN, 1>(v);
}

// v[q] *= exp(SIGN 2 pi i (step q) / L) for q = 1..15; tw[k] = exp(-2 pi i k / L)
template <int SIGN>
__device__ __forceinline__ void big_twiddle(cplx (&v)[16], const cplx *__restrict__ tw, int step)
{
#pragma unroll
    for (int q = 1; q < 16; ++q) {
        const cplx t = __ldg(&tw[step * q]);
        v[q] = SIGN < 0 ? cmul(v[q], t) : cmulc(v[q], t);
    }
}

template <int L, int WP>
struct BigStage {
    typedef BigGeom<L> G;
    // stage 1, registers <-> tile
    static __device__ __forceinline__ void put1(cplx *s, const cplx (&v)[16], int u, int w, int count = 16)
    {
#pragma unroll
        for (int q = 0; q < 16; ++q) if (q < count) s[(u + G::S1 * q) * WP + w] = v[q];
    }
    static __device__ __forceinline__ void get1(const cplx *s, cplx (&v)[16], int u, int w)
    {
#pragma unroll
        for (int m = 0; m < 16; ++m) v[m] = s[(u + G::S1 * m) * WP + w];
    }
    // stage 3, registers <-> tile (positions 16 u + i)
    static __device__ __forceinline__ void put3(cplx *s, const cplx (&v)[16], int u, int w)
    {
#pragma unroll
        for (int i = 0; i < 16; ++i) s[(16 * u + i) * WP + w] = v[i];
    }
    static __device__ __forceinline__ void get3(const cplx *s, cplx (&v)[16], int u, int w)
    {
#pragma unroll
        for (int i = 0; i < 16; ++i) v[i] = s[(16 * u + i) * WP + w];
    }
    // the butterflies
    static __device__ __forceinline__ void fwd1(cplx (&v)[16], const cplx *__restrict__ tw, int u)
    {
        fft16<-1>(v);
        big_twiddle<-1>(v, tw, u);
    }
    static __device__ __forceinline__ void inv1(cplx (&v)[16], const cplx *__restrict__ tw, int u)
    {
        big_twiddle<+1>(v, tw, u);
        fft16<+1>(v);
    }
    template <int SIGN>
    static __device__ __forceinline__ void stage2(cplx *s, const cplx *__restrict__ tw, int u, int w)   // in place on the tile
    {
        const int j = u % G::S2;
        cplx *base = s + ((u / G::S2) * G::S1 + j) * WP + w;
        cplx v[16];
#pragma unroll
        for (int m = 0; m < 16; ++m) v[m] = base[G::S2 * m * WP];
        if (SIGN < 0) {
            fft16<-1>(v);
            big_twiddle<-1>(v, tw, 16 * j);
        } else {
            big_twiddle<+1>(v, tw, 16 * j);
            fft16<+1>(v);
        }
#pragma unroll
        for (int q = 0; q < 16; ++q) base[G::S2 * q * WP] = v[q];
    }
    template <int SIGN>
    static __device__ __forceinline__ void bfly3(cplx (&v)[16])
    {
#pragma unroll
        for (int g = 0; g < 16 / G::R3; ++g) bfly_r<G::R3, SIGN>(&v[g * G::R3]);
    }
};

}  // namespace dks
