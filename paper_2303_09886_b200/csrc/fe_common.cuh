// fe_common.cuh -- shared device helpers for the F-engine kernels (sm_100a only).
//
// Packed FP32 arithmetic: Blackwell's FFMA2 / FADD2 / FMUL2 (PTX fma.rn.f32x2 etc.) process two
// floats per issue slot.  The FP32 pipe does 128 FMA lanes/clk/SM either way (measured), so the
// packed forms do not add flops; they halve the issue slots the arithmetic needs and leave room
// for the integer unpack, loads/stores and shared-memory traffic.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#if defined(__CUDA_ARCH__) && (__CUDA_ARCH__ < 1000)
#error "fengine kernels are written for sm_100a (B200) only"
#endif

namespace fe {

struct f2 {
    float2 v;
    __device__ __forceinline__ f2() {}
    __device__ __forceinline__ f2(float2 x) : v(x) {}
    __device__ __forceinline__ f2(float a, float b) : v(make_float2(a, b)) {}
    __device__ __forceinline__ explicit f2(float a) : v(make_float2(a, a)) {}
};
__device__ __forceinline__ f2 operator+(f2 a, f2 b) { return f2(__fadd2_rn(a.v, b.v)); }
__device__ __forceinline__ f2 operator-(f2 a, f2 b) { return f2(__fadd2_rn(a.v, make_float2(-b.v.x, -b.v.y))); }
__device__ __forceinline__ f2 operator*(f2 a, f2 b) { return f2(__fmul2_rn(a.v, b.v)); }
__device__ __forceinline__ f2 operator-(f2 a) { return f2(make_float2(-a.v.x, -a.v.y)); }
// a*b + c and -a*b + c
__device__ __forceinline__ f2 fma_(f2 a, f2 b, f2 c) { return f2(__ffma2_rn(a.v, b.v, c.v)); }
__device__ __forceinline__ f2 fnma_(f2 a, f2 b, f2 c) { return f2(__ffma2_rn(make_float2(-a.v.x, -a.v.y), b.v, c.v)); }
__device__ __forceinline__ f2 scale_(f2 a, float s) { return f2(__fmul2_rn(a.v, make_float2(s, s))); }

// packed value times a scalar (broadcast to both lanes)
__device__ __forceinline__ f2 operator*(f2 a, float s) { return f2(__fmul2_rn(a.v, make_float2(s, s))); }
__device__ __forceinline__ f2 fma_(f2 a, float s, f2 c) { return f2(__ffma2_rn(a.v, make_float2(s, s), c.v)); }
__device__ __forceinline__ f2 fnma_(f2 a, float s, f2 c) { return f2(__ffma2_rn(make_float2(-a.v.x, -a.v.y), make_float2(s, s), c.v)); }

__device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ float fnma_(float a, float b, float c) { return fmaf(-a, b, c); }
__device__ __forceinline__ float scale_(float a, float s) { return a * s; }

// Complex value over V = float (one point) or f2 (two points in the two packed lanes).
template <typename V>
struct cx {
    V re, im;
};

template <typename V>
__device__ __forceinline__ cx<V> cadd(cx<V> a, cx<V> b) { return {a.re + b.re, a.im + b.im}; }
template <typename V>
__device__ __forceinline__ cx<V> csub(cx<V> a, cx<V> b) { return {a.re - b.re, a.im - b.im}; }
// a * (wr + i wi)
template <typename V, typename W>
__device__ __forceinline__ cx<V> cmul(cx<V> a, W wr, W wi)
{
    cx<V> r;
    r.re = fnma_(a.im, wi, a.re * wr);
    r.im = fma_(a.im, wr, a.re * wi);
    return r;
}
// multiply by -i:  (re + i im)(-i) = im - i re
template <typename V>
__device__ __forceinline__ cx<V> mul_neg_i(cx<V> a) { return {a.im, -a.re}; }

// streaming global accesses that should not displace the L1-resident tables.  The scratch rows are read at L2
// (ld.global.cg): they were written by another CTA (of an earlier kernel, or of the same fused kernel after a
// release / acquire handshake) and a ring slot's addresses are reused, so the L1 must never serve them.
__device__ __forceinline__ float4 ldg_stream_f4(const float4 *p)
{
    float4 v;
    asm volatile("ld.global.cg.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}
// table words that every CTA of an SM re-reads (gain x rotation): keep them in the L1 ahead of everything else
__device__ __forceinline__ float4 ldg_keep_f4(const float4 *p)
{
    float4 v;
    asm volatile("ld.global.nc.L1::evict_last.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ void stg_stream_f4(float4 *p, float4 v)
{
    asm volatile("st.global.cg.v4.f32 [%0], {%1,%2,%3,%4};"
                 :: "l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ void stg_stream_u4(uint4 *p, uint4 v)
{
    asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};"
                 :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// release / acquire handshake on a device-scope counter (fused kernel: FIR tasks -> FFT tasks -> ring slot reuse)
__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int *p)
{
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_add_u32(unsigned int *p, unsigned int v)
{
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// ---- shared-memory, mbarrier and bulk-copy (TMA) helpers of the pipelined kernel (fe_pipe.cuh) -------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ float4 lds_f4(uint32_t saddr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(saddr));
    return v;
}
// named barrier over `count` threads (a multiple of 32): the FFT team of a CTA synchronises without the other roles
__device__ __forceinline__ void bar_sync(int id, int count) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    while (!mbar_try_wait(bar, parity)) {}
}
// bulk copy global -> shared (TMA, 1-D): completes `bytes` of transactions on the mbarrier; bytes % 16 == 0
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// order generic-proxy accesses (st.global by the FIR warps) against async-proxy ones (the bulk copies)
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }

// floor division / modulus by a positive power of two given as log2
__device__ __host__ __forceinline__ int64_t floor_div_pow2(int64_t x, int lg) { return x >> lg; }
__device__ __host__ __forceinline__ int64_t floor_mod_pow2(int64_t x, int lg) { return x & ((int64_t(1) << lg) - 1); }

}  // namespace fe
