// async_copy.cuh -- PTX helpers of the tile kernels: mbarrier, bulk asynchronous copy (TMA, 1-D), named barriers,
// fast FP64 reciprocals.
#pragma once
#include <cstdint>

namespace rad {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity)
        : "memory");
}
// global -> shared bulk copy (TMA, 1-D); bytes a multiple of 16, both addresses 16-byte aligned; completion is
// signalled on the mbarrier as transaction bytes
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src), "r"(bytes),
                 "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
// Orders the calling thread's earlier ordinary (generic-proxy) shared-memory accesses before later asynchronous-proxy accesses
// (bulk copies) to the same bytes.  To be executed by every thread that WROTE the bytes, before the barrier that hands them to the
// thread issuing the copy: a barrier alone orders the generic proxy only.
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// barrier among the `nthreads` threads that use the same id (1..15; 0 is __syncthreads)
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory"); }

// ---- shared-memory access through 32-bit addresses (bytes); `volatile` keeps the program order against barriers
__device__ __forceinline__ double lds(uint32_t addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}
// v = skip ? fallback : shared[addr]; lanes with `skip` take no part in the load (fewer bank conflicts for gathers)
__device__ __forceinline__ double lds_unless(uint32_t addr, bool skip, double fallback) {
    double v = fallback;
    asm volatile("{\n.reg .pred p;\nsetp.ne.u32 p, %2, 0;\n@!p ld.shared.f64 %0, [%1];\n}" : "+d"(v) : "r"(addr), "r"((unsigned)skip));
    return v;
}
__device__ __forceinline__ double2 lds2(uint32_t addr) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts(uint32_t addr, double v) { asm volatile("st.shared.f64 [%0], %1;" ::"r"(addr), "d"(v) : "memory"); }
__device__ __forceinline__ void sts2(uint32_t addr, double x, double y) {
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(addr), "d"(x), "d"(y) : "memory");
}

__device__ __forceinline__ int hi32(double x) { return __double2hiint(x); }

__device__ __forceinline__ double rcp_seed(double d) {  // MUFU.RCP64H: ~2^-20 relative
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
    return r;
}
// 1/d for normal finite d, relative error ~ (seed error)^3 <= 2^-58: seed + one cubic step (3 DFMA)
__device__ __forceinline__ double rcp3(double d) {
    const double r = rcp_seed(d);
    const double e = fma(-d, r, 1.0);
    const double t = fma(e, e, e);
    return fma(r, t, r);
}
// a / d to the same accuracy, 4 FP64 operations in all
__device__ __forceinline__ double div3(double a, double d) {
    const double r = rcp_seed(d);
    const double e = fma(-d, r, 1.0);
    const double t = fma(e, e, e);
    const double p = a * r;
    return fma(p, t, p);
}

// sqrt(x) for finite x >= 1 (no special cases): hardware rsqrt seed (~2^-20), two coupled Newton steps and a final
// residual correction; within 1 ulp
__device__ __forceinline__ double sqrt_ge1(double x) {
    double r;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    double g = x * r, h = 0.5 * r;
    double e = fma(-h, g, 0.5);
    g = fma(g, e, g); h = fma(h, e, h);
    e = fma(-h, g, 0.5);
    g = fma(g, e, g); h = fma(h, e, h);
    const double d = fma(-g, g, x);
    return fma(d, h, g);
}

}  // namespace rad
