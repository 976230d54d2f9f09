// Register-resident FFT building blocks for the specialised passes (dks_passes_r16.cuh).
//
// A padded line of length L = 2n (n = mesh extent = 16 A, A in {2,4,8,16}) is never transformed as a
// whole.  PAPER.md:98 zero-pads rho to the doubled domain; a radix-2 decimation-in-frequency step on
// a line whose upper half is zero is free:
//     X[2K + p] = FFT_n( x[m] * w_L^(p m) )[K],   p = 0,1  (w_L = exp(-2 pi i / L)),
// and the crop after the inverse transform makes the last decimation-in-time step half as long:
//     y[m] = IFFT_n(X[2K])[m] + w_L^(-m) IFFT_n(X[2K+1])[m],   m < n.
// So every padded line is two length-n sub-transforms ("parities" p = 0,1) run by 2A threads.
//
// One sub-transform of length n = 16 A is a four-step FFT over A threads x 16 registers:
//   element m = a + A b lives in thread a, register b (the same mapping on input and on output);
//   radix-16 over b in registers -> twiddle w_n^(a k_b) -> transpose through shared memory
//   -> radix-A over a in registers (16/A independent butterflies per thread).
// The exchange itself (addressing, barrier) belongs to the pass kernels: lanes are laid out
// differently for contiguous and for strided lines.
#pragma once
#include "dks_common.cuh"

namespace dks {

// multiply by SIGN * i
template <int SIGN>
__device__ __forceinline__ cplx mul_si(cplx a) { return SIGN < 0 ? cmake(a.y, -a.x) : cmake(-a.y, a.x); }

// cos, sin of 2 pi m / 16
__device__ __forceinline__ constexpr double cos16(int m)
{
    return m == 0 ? 1.0 : m == 1 ? 0.92387953251128675613 : m == 2 ? 0.70710678118654752440
         : m == 3 ? 0.38268343236508977173 : m == 4 ? 0.0 : m == 5 ? -0.38268343236508977173
         : m == 6 ? -0.70710678118654752440 : m == 7 ? -0.92387953251128675613 : m == 8 ? -1.0
         : -cos16(m - 8);
}
__device__ __forceinline__ constexpr double sin16(int m)
{
    return m == 0 ? 0.0 : m == 1 ? 0.38268343236508977173 : m == 2 ? 0.70710678118654752440
         : m == 3 ? 0.92387953251128675613 : m == 4 ? 1.0 : m == 5 ? 0.92387953251128675613
         : m == 6 ? 0.70710678118654752440 : m == 7 ? 0.38268343236508977173 : m == 8 ? 0.0
         : -sin16(m - 8);
}

// a * exp(SIGN 2 pi i M / 16), M a compile-time constant
template <int SIGN, int M>
__device__ __forceinline__ cplx mul_w16(cplx a)
{
    constexpr int m = M & 15;
    if (m == 0) return a;
    if (m == 4) return mul_si<SIGN>(a);
    if (m == 8) return cmake(-a.x, -a.y);
    if (m == 12) return mul_si<-SIGN>(a);
    constexpr double c = cos16(m), s = SIGN * sin16(m);
    return cmake(fma(a.x, c, -(a.y * s)), fma(a.x, s, a.y * c));
}

template <int SIGN>
__device__ __forceinline__ void bfly2(cplx &x0, cplx &x1)
{
    cplx t = x0;
    x0 = cadd(t, x1);
    x1 = csub(t, x1);
}

// 4-point DFT, natural order in and out: x_k <- sum_n x_n exp(SIGN 2 pi i n k / 4)
template <int SIGN>
__device__ __forceinline__ void bfly4(cplx &x0, cplx &x1, cplx &x2, cplx &x3)
{
    cplx apc = cadd(x0, x2), amc = csub(x0, x2), bpd = cadd(x1, x3), bmd = mul_si<SIGN>(csub(x1, x3));
    x0 = cadd(apc, bpd);
    x1 = cadd(amc, bmd);
    x2 = csub(apc, bpd);
    x3 = csub(amc, bmd);
}

// 8-point DFT on v[0], v[S], ..., v[7S], natural order in and out
template <int SIGN, int S>
__device__ __forceinline__ void bfly8(cplx *v)
{
    bfly4<SIGN>(v[0], v[2 * S], v[4 * S], v[6 * S]);      // y0[k0] in slots 0,2,4,6
    bfly4<SIGN>(v[1 * S], v[3 * S], v[5 * S], v[7 * S]);  // y1[k0] in slots 1,3,5,7
    v[3 * S] = mul_w16<SIGN, 2>(v[3 * S]);
    v[5 * S] = mul_w16<SIGN, 4>(v[5 * S]);
    v[7 * S] = mul_w16<SIGN, 6>(v[7 * S]);
    cplx o[8];
#pragma unroll
    for (int k0 = 0; k0 < 4; ++k0) {
        o[k0] = cadd(v[2 * k0 * S], v[(2 * k0 + 1) * S]);
        o[k0 + 4] = csub(v[2 * k0 * S], v[(2 * k0 + 1) * S]);
    }
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k * S] = o[k];
}

// x * (1 + S i) and x * (-1 + S i) without the 1/sqrt(2): the 8th roots w16^2 = c (1 + S i), w16^6 = c (-1 + S i),
// c = 1/sqrt(2), S = SIGN; the factor c is folded into the FMAs of the butterfly that consumes the product.
template <int SIGN>
__device__ __forceinline__ cplx rot_p(cplx a) { return SIGN < 0 ? cmake(a.x + a.y, a.y - a.x) : cmake(a.x - a.y, a.y + a.x); }
template <int SIGN>
__device__ __forceinline__ cplx rot_m(cplx a) { return SIGN < 0 ? cmake(a.y - a.x, -a.y - a.x) : cmake(-a.x - a.y, a.x - a.y); }
__device__ __forceinline__ cplx cfma(double s, cplx t, cplx u) { return cmake(fma(s, t.x, u.x), fma(s, t.y, u.y)); }

// 4-point DFT as bfly4, with x2 given as c * t2 (t2 unscaled): the scale rides on the FMAs
template <int SIGN>
__device__ __forceinline__ void bfly4_x2scaled(cplx &x0, cplx &x1, cplx &x2, cplx &x3, cplx t2)
{
    constexpr double c = 0.70710678118654752440;
    cplx apc = cfma(c, t2, x0), amc = cfma(-c, t2, x0), bpd = cadd(x1, x3), bmd = mul_si<SIGN>(csub(x1, x3));
    x0 = cadd(apc, bpd);
    x1 = cadd(amc, bmd);
    x2 = csub(apc, bpd);
    x3 = csub(amc, bmd);
}

// 16-point DFT in registers, natural order in and out (4 x 4 decomposition, 152 fp64 instructions: the four
// 8th-root twiddles of the middle layer cost two additions each, their 1/sqrt(2) is folded into FMAs)
template <int SIGN>
__device__ __forceinline__ void fft16_tail(cplx (&v)[16]);

template <int SIGN>
__device__ __forceinline__ void fft16(cplx (&v)[16])
{
#pragma unroll
    for (int n0 = 0; n0 < 4; ++n0) bfly4<SIGN>(v[n0], v[n0 + 4], v[n0 + 8], v[n0 + 12]);   // slot n0 + 4 k0
    fft16_tail<SIGN>(v);
}

// everything after the first layer of 4-point transforms
template <int SIGN>
__device__ __forceinline__ void fft16_tail(cplx (&v)[16])
{
    constexpr double c = 0.70710678118654752440;
    // k0 = 0: no twiddles
    bfly4<SIGN>(v[0], v[1], v[2], v[3]);
    // k0 = 1: twiddles w^1, w^2, w^3 on slots 5, 6, 7
    v[5] = mul_w16<SIGN, 1>(v[5]);
    v[7] = mul_w16<SIGN, 3>(v[7]);
    bfly4_x2scaled<SIGN>(v[4], v[5], v[6], v[7], rot_p<SIGN>(v[6]));
    // k0 = 2: twiddles w^2, w^4, w^6 on slots 9, 10, 11
    {
        const cplx x2 = mul_si<SIGN>(v[10]);                       // w^4 = S i
        const cplx t1 = rot_p<SIGN>(v[9]), t3 = rot_m<SIGN>(v[11]);
        const cplx apc = cadd(v[8], x2), amc = csub(v[8], x2);
        const cplx P = cadd(t1, t3), M = mul_si<SIGN>(csub(t1, t3));
        v[8] = cfma(c, P, apc);
        v[9] = cfma(c, M, amc);
        v[10] = cfma(-c, P, apc);
        v[11] = cfma(-c, M, amc);
    }
    // k0 = 3: twiddles w^3, w^6, w^9 on slots 13, 14, 15
    v[13] = mul_w16<SIGN, 3>(v[13]);
    v[15] = mul_w16<SIGN, 9>(v[15]);
    bfly4_x2scaled<SIGN>(v[12], v[13], v[14], v[15], rot_m<SIGN>(v[14]));
    // slot 4 k0 + k1 holds X[k0 + 4 k1]: transpose the 4 x 4 register tile
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = i + 1; j < 4; ++j) {
            cplx t = v[4 * i + j];
            v[4 * i + j] = v[4 * j + i];
            v[4 * j + i] = t;
        }
}

// Second step of the four-step transform: v[g A + a'] (g < 16/A) -> radix-A over a' for every g;
// the result for k_a goes to register r = g + (16/A) k_a, i.e. sub-index tau + A r.
template <int A, int SIGN>
__device__ __forceinline__ void fft_second(cplx (&v)[16])
{
    if (A == 16) {
        fft16<SIGN>(v);
        return;
    }
    constexpr int G = 16 / A;
#pragma unroll
    for (int g = 0; g < G; ++g) {
        if (A == 8) bfly8<SIGN, 1>(&v[g * 8]);
        if (A == 4) bfly4<SIGN>(v[g * 4], v[g * 4 + 1], v[g * 4 + 2], v[g * 4 + 3]);
        if (A == 2) bfly2<SIGN>(v[g * 2], v[g * 2 + 1]);
    }
    cplx o[16];
#pragma unroll
    for (int g = 0; g < G; ++g)
#pragma unroll
        for (int ka = 0; ka < A; ++ka) o[g + G * ka] = v[g * A + ka];
#pragma unroll
    for (int r = 0; r < 16; ++r) v[r] = o[r];
}

// Transpose of fft_second (the DFT matrix is symmetric, so only the register permutation is mirrored):
// v[g + (16/A) k_a] -> radix-A over k_a -> v[g A + a'].  First step of the transposed inverse flow.
template <int A, int SIGN>
__device__ __forceinline__ void fft_second_t(cplx (&v)[16])
{
    if (A == 16) {
        fft16<SIGN>(v);
        return;
    }
    constexpr int G = 16 / A;
    cplx o[16];
#pragma unroll
    for (int g = 0; g < G; ++g)
#pragma unroll
        for (int ka = 0; ka < A; ++ka) o[g * A + ka] = v[g + G * ka];
#pragma unroll
    for (int r = 0; r < 16; ++r) v[r] = o[r];
#pragma unroll
    for (int g = 0; g < G; ++g) {
        if (A == 8) bfly8<SIGN, 1>(&v[g * 8]);
        if (A == 4) bfly4<SIGN>(v[g * 4], v[g * 4 + 1], v[g * 4 + 2], v[g * 4 + 3]);
        if (A == 2) bfly2<SIGN>(v[g * 2], v[g * 2 + 1]);
    }
}

// Twiddle between the two steps: v[k] *= T[k A + a] (SIGN < 0) or conj(T[k A + a]) (SIGN > 0), k = 0..15.
// T is one of the three n-entry regions of the per-axis table tw1 (host: build_tw1 in dks_poisson.cu):
//   [0, n)    parity 0, both directions:  w_n^(a k)
//   [n, 2n)   parity 1, forward:          w_n^(a k) w_L^a          (L = 2n)
//   [2n, 3n)  parity 1, inverse:          w_n^(a k) w_L^(k mod A)
// The parity-1 regions carry the thread-constant part of the parity twiddle w_L^(+-m), m = a + A b =
// thread part + A * register part; the register part w_32^b is a compile-time constant (parity_consts).
// So the parity twiddle costs no table access at all.  (Region 0 has T = 1 at k = 0.)
template <int A, int SIGN>
__device__ __forceinline__ void twiddle_between(cplx (&v)[16], const cplx *__restrict__ T, int a)
{
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        cplx t = __ldg(&T[k * A + a]);
        v[k] = SIGN < 0 ? cmul(v[k], t) : cmulc(v[k], t);
    }
}
// ---- twiddle AFTER the exchange ----------------------------------------------------------------
// The between-step twiddle commutes with the exchange: the thread that holds sub-transform index k = a + A g after the
// exchange multiplies its value from pre-exchange thread a' by T[k A + a'], i.e. by A consecutive table entries per g.
// The strided passes issue these loads right before the exchange barrier, when v[] is dead, so their latency hides
// behind the barrier, and for A = 16 the multiplication is folded into the first butterfly layer of the second
// radix-16 (fft16_tw): x0 + t x2 is 4 FMAs, x0 - t x2 = 2 x0 - (x0 + t x2) two more, which saves 4 of the 32 (28)
// instructions of a 4-point butterfly with 4 (3) twiddled inputs.
template <int A>
__device__ __forceinline__ void load_tw_post(cplx (&t)[16], const cplx *__restrict__ T, int a)
{
    constexpr int G = 16 / A;
    if constexpr (A > 1) {                                // A = 1: every table entry is 1 (fft_second_tw skips the product)
#pragma unroll
        for (int g = 0; g < G; ++g)
#pragma unroll
            for (int ap = 0; ap < A; ++ap) t[g * A + ap] = __ldg(&T[(a + A * g) * A + ap]);
    }
}

// u + t x  (SIGN < 0) or u + conj(t) x  (SIGN > 0)
template <int SIGN>
__device__ __forceinline__ cplx cfma_tw(cplx t, cplx x, cplx u)
{
    const double ty = SIGN < 0 ? t.y : -t.y;
    return cmake(fma(-ty, x.y, fma(t.x, x.x, u.x)), fma(ty, x.x, fma(t.x, x.y, u.y)));
}
template <int SIGN>
__device__ __forceinline__ cplx cmul_tw(cplx x, cplx t) { return SIGN < 0 ? cmul(x, t) : cmulc(x, t); }
// 2 a - b
__device__ __forceinline__ cplx ctwice_minus(cplx a, cplx b) { return cmake(fma(2.0, a.x, -b.x), fma(2.0, a.y, -b.y)); }

// bfly4 on (t0 x0, t1 x1, t2 x2, t3 x3) (conjugated twiddles for SIGN > 0); UNIT0: t0 = 1
template <int SIGN, bool UNIT0>
__device__ __forceinline__ void bfly4_tw(cplx &x0, cplx &x1, cplx &x2, cplx &x3, cplx t0, cplx t1, cplx t2, cplx t3)
{
    const cplx y0 = UNIT0 ? x0 : cmul_tw<SIGN>(x0, t0);
    const cplx apc = cfma_tw<SIGN>(t2, x2, y0), amc = ctwice_minus(y0, apc);
    const cplx y1 = cmul_tw<SIGN>(x1, t1);
    const cplx bpd = cfma_tw<SIGN>(t3, x3, y1), bmd = mul_si<SIGN>(ctwice_minus(y1, bpd));
    x0 = cadd(apc, bpd);
    x1 = cadd(amc, bmd);
    x2 = csub(apc, bpd);
    x3 = csub(amc, bmd);
}

// fft16 of (t[i] v[i]); UNIT0: t[0] = 1
template <int SIGN, bool UNIT0>
__device__ __forceinline__ void fft16_tw(cplx (&v)[16], const cplx (&t)[16])
{
    bfly4_tw<SIGN, UNIT0>(v[0], v[4], v[8], v[12], t[0], t[4], t[8], t[12]);
#pragma unroll
    for (int n0 = 1; n0 < 4; ++n0) bfly4_tw<SIGN, false>(v[n0], v[n0 + 4], v[n0 + 8], v[n0 + 12], t[n0], t[n0 + 4], t[n0 + 8], t[n0 + 12]);
    fft16_tail<SIGN>(v);
}

// second step of the four-step transform with the twiddles t[] (load_tw_post) applied to its inputs
template <int A, int SIGN, bool UNIT0>
__device__ __forceinline__ void fft_second_tw(cplx (&v)[16], const cplx (&t)[16])
{
    if (A == 16) {
        fft16_tw<SIGN, UNIT0>(v, t);
        return;
    }
    if (A > 1) {                                          // A = 1: every table entry is 1
#pragma unroll
        for (int i = 0; i < 16; ++i) v[i] = cmul_tw<SIGN>(v[i], t[i]);
    }
    fft_second<A, SIGN>(v);
}

// cos, sin of 2 pi m / 32, m = 0..15
__device__ __forceinline__ constexpr double cos32(int m)
{
    return m == 0 ? 1.0 : m == 1 ? 0.98078528040323044913 : m == 2 ? 0.92387953251128675613
         : m == 3 ? 0.83146961230254523708 : m == 4 ? 0.70710678118654752440 : m == 5 ? 0.55557023301960222474
         : m == 6 ? 0.38268343236508977173 : m == 7 ? 0.19509032201612826785 : m == 8 ? 0.0
         : -cos32(16 - m);
}
__device__ __forceinline__ constexpr double sin32(int m) { return m <= 8 ? cos32(8 - m) : cos32(m - 8); }

// a * exp(SIGN 2 pi i M / 32), M = 0..15 a compile-time constant
template <int SIGN, int M>
__device__ __forceinline__ cplx mul_w32(cplx a)
{
    if (M == 0) return a;
    if (M == 8) return mul_si<SIGN>(a);
    constexpr double c = cos32(M), s = SIGN * sin32(M);
    return cmake(fma(a.x, c, -(a.y * s)), fma(a.x, s, a.y * c));
}

// register part of the parity twiddle: v[b] *= exp(SIGN 2 pi i b / 32) = w_L^(-SIGN A b)
template <int SIGN>
__device__ __forceinline__ void parity_consts(cplx (&v)[16])
{
    v[1] = mul_w32<SIGN, 1>(v[1]);   v[2] = mul_w32<SIGN, 2>(v[2]);   v[3] = mul_w32<SIGN, 3>(v[3]);
    v[4] = mul_w32<SIGN, 4>(v[4]);   v[5] = mul_w32<SIGN, 5>(v[5]);   v[6] = mul_w32<SIGN, 6>(v[6]);
    v[7] = mul_w32<SIGN, 7>(v[7]);   v[8] = mul_w32<SIGN, 8>(v[8]);   v[9] = mul_w32<SIGN, 9>(v[9]);
    v[10] = mul_w32<SIGN, 10>(v[10]); v[11] = mul_w32<SIGN, 11>(v[11]); v[12] = mul_w32<SIGN, 12>(v[12]);
    v[13] = mul_w32<SIGN, 13>(v[13]); v[14] = mul_w32<SIGN, 14>(v[14]); v[15] = mul_w32<SIGN, 15>(v[15]);
}

__device__ __forceinline__ cplx shfl_xor_c(cplx v, int mask)
{
    return cmake(__shfl_xor_sync(0xffffffffu, v.x, mask), __shfl_xor_sync(0xffffffffu, v.y, mask));
}

// Combine of the two parities after the inverse sub-transforms (crop fused): the parity-1 thread
// holds w_L^(-m) O[m] already.  Parity 0 keeps registers r < 8, parity 1 keeps r >= 8; each sends the
// other half to its partner lane (lane ^ MASK).  out[i] belongs to register r = i + 8 p.
template <int MASK>
__device__ __forceinline__ void combine_parities(const cplx (&v)[16], int p, cplx (&out)[8])
{
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        cplx send = p ? v[i] : v[i + 8];
        cplx mine = p ? v[i + 8] : v[i];
        out[i] = cadd(mine, shfl_xor_c(send, MASK));
    }
}

}  // namespace dks
