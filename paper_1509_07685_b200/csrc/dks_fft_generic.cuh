// Generic shared-memory FFT on a tile of lines, any power-of-two length 4..2048 (runtime L).
//
// Tile layout: element p of line w lives at s[p * WP + w] (w fastest), so that every butterfly
// touches W consecutive 16-byte elements: conflict-free shared-memory access for W >= 8.
//
// Two in-place transforms, both unnormalised, SIGN = -1 (forward, e^{-i theta}) or +1 (inverse):
//   tile_fft_dif : natural-order input  -> bit-reversed output   (decimation in frequency)
//   tile_fft_dit : bit-reversed input   -> natural-order output  (decimation in time)
// Used back to back (DIF forward, pointwise multiply, DIT inverse) they need no reordering at all.
// A radix-4 stage here is exactly two fused radix-2 stages, so the permutation is plain bit reversal
// also when log2(L) is odd (one radix-2 stage at span L: first for DIF, last for DIT).
//
// tw[k] = exp(-2 pi i k / L), k = 0..L-1 (host-computed in long double), read through L1.
//
// These are the fallback passes: every mesh size works through them; the headline sizes have
// specialised register-resident kernels (dks_passes_r16.cuh).
#pragma once
#include "dks_common.cuh"

namespace dks {

template <int SIGN>
__device__ __forceinline__ cplx twiddle(const cplx *__restrict__ tw, int k)
{
    cplx t = __ldg(&tw[k]);
    if (SIGN > 0) t.y = -t.y;
    return t;
}

// multiply by W_4 = exp(SIGN * 2 pi i / 4) = SIGN * i
template <int SIGN>
__device__ __forceinline__ cplx mul_w4(cplx a) { return SIGN < 0 ? cmul_mi(a) : cmul_pi(a); }

template <int SIGN>
__device__ void tile_fft_dif(cplx *s, int L, int logL, int W, int WP, const cplx *__restrict__ tw)
{
    const int tid = threadIdx.x, nt = blockDim.x;
    int span = L;
    if (logL & 1) {
        const int half = L >> 1;
        for (int idx = tid; idx < half * W; idx += nt) {
            int w = idx % W, i = idx / W;
            cplx a = s[i * WP + w], b = s[(i + half) * WP + w];
            s[i * WP + w] = cadd(a, b);
            s[(i + half) * WP + w] = cmul(csub(a, b), twiddle<SIGN>(tw, i));
        }
        __syncthreads();
        span = half;
    }
    while (span >= 4) {
        const int m = span >> 2, tstep = L / span;
        for (int idx = tid; idx < (L >> 2) * W; idx += nt) {
            int w = idx % W, q = idx / W;
            int j = q % m, base = (q / m) * span + j;
            cplx *p0 = &s[base * WP + w];
            cplx a = p0[0], b = p0[m * WP], c = p0[2 * m * WP], d = p0[3 * m * WP];
            cplx apc = cadd(a, c), amc = csub(a, c), bpd = cadd(b, d), bmd = mul_w4<SIGN>(csub(b, d));
            p0[0] = cadd(apc, bpd);
            p0[m * WP] = cmul(csub(apc, bpd), twiddle<SIGN>(tw, 2 * j * tstep));
            p0[2 * m * WP] = cmul(cadd(amc, bmd), twiddle<SIGN>(tw, j * tstep));
            p0[3 * m * WP] = cmul(csub(amc, bmd), twiddle<SIGN>(tw, 3 * j * tstep));
        }
        __syncthreads();
        span = m;
    }
}

template <int SIGN>
__device__ void tile_fft_dit(cplx *s, int L, int logL, int W, int WP, const cplx *__restrict__ tw)
{
    const int tid = threadIdx.x, nt = blockDim.x;
    const int top = (logL & 1) ? (L >> 1) : L;     // largest radix-4 span
    for (int span = 4; span <= top; span <<= 2) {
        const int m = span >> 2, tstep = L / span;
        for (int idx = tid; idx < (L >> 2) * W; idx += nt) {
            int w = idx % W, q = idx / W;
            int j = q % m, base = (q / m) * span + j;
            cplx *p0 = &s[base * WP + w];
            cplx a = p0[0];
            cplx b = cmul(p0[m * WP], twiddle<SIGN>(tw, 2 * j * tstep));
            cplx c = cmul(p0[2 * m * WP], twiddle<SIGN>(tw, j * tstep));
            cplx d = cmul(p0[3 * m * WP], twiddle<SIGN>(tw, 3 * j * tstep));
            cplx apb = cadd(a, b), amb = csub(a, b), cpd = cadd(c, d), cmd = mul_w4<SIGN>(csub(c, d));
            p0[0] = cadd(apb, cpd);
            p0[2 * m * WP] = csub(apb, cpd);
            p0[m * WP] = cadd(amb, cmd);
            p0[3 * m * WP] = csub(amb, cmd);
        }
        __syncthreads();
    }
    if (logL & 1) {
        const int half = L >> 1;
        for (int idx = tid; idx < half * W; idx += nt) {
            int w = idx % W, i = idx / W;
            cplx a = s[i * WP + w], b = cmul(s[(i + half) * WP + w], twiddle<SIGN>(tw, i));
            s[i * WP + w] = cadd(a, b);
            s[(i + half) * WP + w] = csub(a, b);
        }
        __syncthreads();
    }
}

}  // namespace dks
