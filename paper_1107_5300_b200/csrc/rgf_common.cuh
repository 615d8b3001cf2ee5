// rgf_common.cuh -- device helpers shared by the kernels of the RGF library (sm_100a only).
// Complex numbers are double2 (x = re, y = im), interleaved, row-major everywhere in HBM.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace rgf {

typedef double2 cplx;

__host__ __device__ __forceinline__ cplx cmake(double re, double im) { cplx r; r.x = re; r.y = im; return r; }
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return cmake(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return cmake(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cmul(cplx a, cplx b)
{
    return cmake(fma(a.x, b.x, -(a.y * b.y)), fma(a.x, b.y, a.y * b.x));
}
// c -= a*b
__device__ __forceinline__ void cfnma(cplx &c, cplx a, cplx b)
{
    c.x = fma(-a.x, b.x, c.x); c.x = fma(a.y, b.y, c.x);
    c.y = fma(-a.x, b.y, c.y); c.y = fma(-a.y, b.x, c.y);
}
__device__ __forceinline__ double cabs2(cplx a) { return fma(a.x, a.x, a.y * a.y); }
// 1/a, scaled (Smith) so that |a|^2 cannot under/overflow for the magnitudes met here
__device__ __forceinline__ cplx crecip(cplx a)
{
    if (fabs(a.x) >= fabs(a.y)) {
        double r = a.y / a.x, d = fma(a.y, r, a.x);
        double inv = 1.0 / d;
        return cmake(inv, -r * inv);
    } else {
        double r = a.x / a.y, d = fma(a.x, r, a.y);
        double inv = 1.0 / d;
        return cmake(r * inv, -inv);
    }
}

// ---- FP64 tensor core: mma.sync m8n8k4 (SASS: DMMA.8x8x4, the only native FP64 MMA shape on sm_100a)
// Fragment ownership, lane = 4*g + t (g = lane>>2, t = lane&3):
//   A (8x4, row): a  = A[g][t]        B (4x8, col): b = B[t][g]
//   C (8x8):      c0 = C[g][2t], c1 = C[g][2t+1]
__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// complex 8x8 += (8x4)*(4x8): 4 real DMMAs; nai = -a.im precomputed by the caller
__device__ __forceinline__ void zmma884(double (&cre)[2], double (&cim)[2], double ar, double ai, double nai,
                                        double br, double bi)
{
    dmma884(cre[0], cre[1], ar, br);
    dmma884(cim[0], cim[1], ar, bi);
    dmma884(cre[0], cre[1], nai, bi);
    dmma884(cim[0], cim[1], ai, br);
}

// ---- cp.async (LDGSTS), 16 bytes = one complex128 element; src_bytes = 0 zero-fills
__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gmem_src, int src_bytes)
{
    unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(gmem_src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// ---- TMA bulk copies (cp.async.bulk, SASS: UBLKCP) completing on an mbarrier (SASS: SYNCS) ---------------------------
// One elected thread arms the barrier with the byte count of the whole stage (tma_expect), any thread issues row copies
// (16-byte aligned source, destination and size), every consumer waits on the phase parity (tma_wait).  The copy engine
// moves the rows; no thread spends registers or address arithmetic per 16 bytes as with cp.async.
__device__ __forceinline__ void tma_bar_init(unsigned long long *bar, int arrivals)
{
    const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(a), "r"(arrivals) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void tma_expect(unsigned long long *bar, unsigned bytes)
{
    const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(a), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_row(void *smem_dst, const void *gmem_src, unsigned bytes, unsigned long long *bar)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst), a = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(d), "l"(gmem_src), "r"(bytes), "r"(a) : "memory");
}
__device__ __forceinline__ void tma_wait(unsigned long long *bar, unsigned parity)
{
    const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "TMA_WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@!p bra TMA_WAIT_%=;\n\t}"
        ::"r"(a), "r"(parity) : "memory");
}
// generic-proxy writes (st.shared) of a buffer must be ordered before the async proxy overwrites it
__device__ __forceinline__ void tma_fence_proxy() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// m_i[j] = 1 iff (i + j) even; bit test so that negative (lead) slice indices work
__host__ __device__ __forceinline__ int mask_bit(int i, int j) { return (((i + j) & 1) == 0) ? 1 : 0; }

// ---- helpers shared by the fused sweep kernel and the panel kernels of the stepwise paths ----------------------------
__device__ __forceinline__ cplx ldcg(const cplx *p)
{
    double2 v = __ldcg(reinterpret_cast<const double2 *>(p));
    return v;
}

// 32-byte (two complex128) L2 load / store: LDG.E.256 / STG.E.256 on sm_100a; p must be 32-byte aligned
__device__ __forceinline__ void ld256cg(const cplx *p, double &a, double &b, double &c, double &d)
{
    asm volatile("ld.global.cg.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}
__device__ __forceinline__ void st256(cplx *p, double a, double b, double c, double d)
{
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}

// 1 / v for v = |x|^2 > 0 on the critical path of every pivot: MUFU.RCP64H seed (20 bits) + two Newton steps
// (4 dependent DFMAs, ~60 cycles) instead of the IEEE division (~130 cycles on sm_100a).  Relative error
// ~2e-16, irrelevant for a pivot reciprocal.  v outside the normal range (|x| < 1e-154 or > 1e154) gives 0 / inf /
// NaN, which the caller reports as a singular pivot through the key check and the propagated non-finite values.
__device__ __forceinline__ double hs_rcp(double v)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(v));
    double e = fma(-v, r, 1.0);
    r = fma(r, e, r);
    e = fma(-v, r, 1.0);
    r = fma(r, e, r);
    return r;
}

}  // namespace rgf
