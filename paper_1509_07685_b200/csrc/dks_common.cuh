// Shared device helpers for the dks_poisson kernels (sm_100a).  fp64 complex arithmetic on double2.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dks {

typedef double2 cplx;   // .x = re, .y = im

__device__ __forceinline__ cplx cmake(double re, double im) { return make_double2(re, im); }
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cscale(cplx a, double s) { return make_double2(a.x * s, a.y * s); }
// a * b
__device__ __forceinline__ cplx cmul(cplx a, cplx b)
{
    return make_double2(fma(a.x, b.x, -(a.y * b.y)), fma(a.x, b.y, a.y * b.x));
}
// a * conj(b)
__device__ __forceinline__ cplx cmulc(cplx a, cplx b)
{
    return make_double2(fma(a.x, b.x, a.y * b.y), fma(a.y, b.x, -(a.x * b.y)));
}
// a * (-i)  and  a * (+i)
__device__ __forceinline__ cplx cmul_mi(cplx a) { return make_double2(a.y, -a.x); }
__device__ __forceinline__ cplx cmul_pi(cplx a) { return make_double2(-a.y, a.x); }

// bit reversal of the low `bits` bits
__device__ __forceinline__ int brev(int v, int bits) { return (int)(__brev((unsigned)v) >> (32 - bits)); }

// 128-bit global access with streaming hints: every byte of the intermediate buffers is touched once
// per pass, so do not allocate in L1.
__device__ __forceinline__ cplx ldg_stream(const cplx *p)
{
    cplx r;
    asm volatile("ld.global.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p));
    return r;
}
__device__ __forceinline__ void stg_stream(cplx *p, cplx v)
{
    asm volatile("st.global.L1::no_allocate.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}

// two neighbouring complex values with one 256-bit access (sm_100: LDG.256 / STG.256); p is 32-byte aligned
__device__ __forceinline__ void stg_stream2(cplx *p, cplx v0, cplx v1)
{
    asm volatile("st.global.L1::no_allocate.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(v0.x), "d"(v0.y), "d"(v1.x), "d"(v1.y)
                 : "memory");
}
__device__ __forceinline__ void ldg_stream2(const cplx *p, cplx &v0, cplx &v1)
{
    asm volatile("ld.global.L1::no_allocate.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(v0.x), "=d"(v0.y), "=d"(v1.x), "=d"(v1.y) : "l"(p));
}

// the same through L1 (a second thread of the CTA reads the same 32 bytes shortly afterwards)
__device__ __forceinline__ void ldg_cached2(const cplx *p, cplx &v0, cplx &v1)
{
    asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(v0.x), "=d"(v0.y), "=d"(v1.x), "=d"(v1.y) : "l"(p));
}

// Programmatic dependent launch (sm_90+).  A PDL kernel calls pdl_trigger() right before its stores: once every CTA of the grid
// has triggered or exited, the next kernel in the stream may be scheduled into the SMs the tail frees and run its prologue
// (index arithmetic, twiddle loads, barrier initialisation); its pdl_wait() then blocks until the previous grid has completed
// and its memory is visible.  Nothing the previous kernel wrote is read, and nothing it read is overwritten, before pdl_wait().
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// Ampere-style asynchronous 16-byte copy global -> shared (SASS LDGSTS), bypassing L1 and registers.
__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gmem_src)
{
    unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem_src) : "memory");
}

// ---- bulk asynchronous copy global -> shared (SASS UBLKCP) completing on an mbarrier -----------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_init_fence() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// the mbarrier receives one (pre-counted) arrival once all cp.async copies this thread has issued so far have landed
__device__ __forceinline__ void cp_async_mbar_arrive(uint64_t *bar)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// bytes: multiple of 16; both addresses 16-byte aligned
__device__ __forceinline__ void bulk_g2s(void *smem_dst, const void *gmem_src, unsigned bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(smem_dst)),
                 "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

}  // namespace dks
