// pty_port.cuh -- the handful of device primitives the kernel bodies need (barriers, reductions
// into global memory, streaming loads/stores, fast math), sm_100a only.
#pragma once
#define PTY_PORT_INCLUDED
#include <cuda.h>           // CUtensorMap (type only: the driver entry point is fetched at run time)
#include <cuda_runtime.h>
#include <cooperative_groups.h>

#define PTY_DEV __device__ __forceinline__

namespace pty {
PTY_DEV void pty_cta_sync() { __syncthreads(); }
PTY_DEV void pty_cluster_sync() { cooperative_groups::this_cluster().sync(); }

// reductions into global memory, no return value (RED.E.ADD in SASS)
PTY_DEV void red_add(float* p, float v) { atomicAdd(p, v); }
PTY_DEV void red_add(double* p, double v) { atomicAdd(p, v); }
PTY_DEV void red_add2(float2* p, float2 v) {      // 8-byte vector reduction (sm_90+)
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(v.x), "f"(v.y) : "memory");
}
PTY_DEV void red_add_shared(float* p, float v) { atomicAdd(p, v); }
PTY_DEV void flag_or(int* p, int v) { atomicOr(p, v); }

PTY_DEV float2 ldg2(const float2* p) { return __ldg(p); }
PTY_DEV float ldg1(const float* p) { return __ldg(p); }
// streaming (evict-first) accesses for the saved waves: written once, read once
PTY_DEV float2 ld_stream2(const float2* p) { return __ldcs(p); }
PTY_DEV void st_stream2(float2* p, float2 v) { __stcs(p, v); }

PTY_DEV float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
PTY_DEV bool warp_leader() { return (threadIdx.x & 31) == 0; }
// ---- tensor memory (TMEM) as a per-thread staging buffer (tcgen05.st / tcgen05.ld, 32x32b shape):
// a warp owns the 32 TMEM lanes of its sub-partition (warp id % 4); lane i of the warp reads and writes
// TMEM lane 32 (warp % 4) + i, N consecutive 32-bit columns per instruction.  Used to park data that was
// fetched from global memory early (no registers, no shared memory, not the LSU pipe).
PTY_DEV void tmem_alloc512(unsigned* smem_slot) {     // one full warp
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;"
                 ::"r"((unsigned)__cvta_generic_to_shared(smem_slot)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
PTY_DEV void tmem_dealloc512(unsigned base) {         // the same warp
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(base) : "memory");
}
PTY_DEV void tmem_fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
PTY_DEV void tmem_fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
PTY_DEV void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
PTY_DEV void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
PTY_DEV void tmem_st4(unsigned ta, const float2 (&v)[4]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                 ::"r"(ta), "f"(v[0].x), "f"(v[0].y), "f"(v[1].x), "f"(v[1].y), "f"(v[2].x), "f"(v[2].y),
                   "f"(v[3].x), "f"(v[3].y) : "memory");
}
PTY_DEV void tmem_ld4(unsigned ta, float2 (&v)[4]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(v[0].x), "=f"(v[0].y), "=f"(v[1].x), "=f"(v[1].y), "=f"(v[2].x), "=f"(v[2].y),
                   "=f"(v[3].x), "=f"(v[3].y) : "r"(ta) : "memory");
}
// 8 complex values v[off .. off + 7] <-> 16 columns
PTY_DEV void tmem_st8(unsigned ta, const float2 (&v)[32], int o) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
                 ::"r"(ta), "f"(v[o].x), "f"(v[o].y), "f"(v[o + 1].x), "f"(v[o + 1].y), "f"(v[o + 2].x), "f"(v[o + 2].y),
                   "f"(v[o + 3].x), "f"(v[o + 3].y), "f"(v[o + 4].x), "f"(v[o + 4].y), "f"(v[o + 5].x), "f"(v[o + 5].y),
                   "f"(v[o + 6].x), "f"(v[o + 6].y), "f"(v[o + 7].x), "f"(v[o + 7].y) : "memory");
}
PTY_DEV void tmem_ld8(unsigned ta, float2 (&v)[32], int o) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=f"(v[o].x), "=f"(v[o].y), "=f"(v[o + 1].x), "=f"(v[o + 1].y), "=f"(v[o + 2].x), "=f"(v[o + 2].y),
                   "=f"(v[o + 3].x), "=f"(v[o + 3].y), "=f"(v[o + 4].x), "=f"(v[o + 4].y), "=f"(v[o + 5].x), "=f"(v[o + 5].y),
                   "=f"(v[o + 6].x), "=f"(v[o + 6].y), "=f"(v[o + 7].x), "=f"(v[o + 7].y)
                 : "r"(ta) : "memory");
}
PTY_DEV void tmem_st8r(unsigned ta, const float2 (&v)[8]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
                 ::"r"(ta), "f"(v[0].x), "f"(v[0].y), "f"(v[1].x), "f"(v[1].y), "f"(v[2].x), "f"(v[2].y),
                   "f"(v[3].x), "f"(v[3].y), "f"(v[4].x), "f"(v[4].y), "f"(v[5].x), "f"(v[5].y),
                   "f"(v[6].x), "f"(v[6].y), "f"(v[7].x), "f"(v[7].y) : "memory");
}
PTY_DEV void tmem_ld8r(unsigned ta, float2 (&v)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=f"(v[0].x), "=f"(v[0].y), "=f"(v[1].x), "=f"(v[1].y), "=f"(v[2].x), "=f"(v[2].y),
                   "=f"(v[3].x), "=f"(v[3].y), "=f"(v[4].x), "=f"(v[4].y), "=f"(v[5].x), "=f"(v[5].y),
                   "=f"(v[6].x), "=f"(v[6].y), "=f"(v[7].x), "=f"(v[7].y)
                 : "r"(ta) : "memory");
}
// global load that the compiler must leave where it is written (prefetch ticks)
PTY_DEV float2 ldg2_pinned(const float2* p) {
    float2 v;
    asm volatile("ld.global.nc.v2.f32 {%0,%1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}
PTY_DEV float2 ld_stream2_pinned(const float2* p) {
    float2 v;
    asm volatile("ld.global.cs.v2.f32 {%0,%1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}

// 16-byte streaming accesses (two complex values): the saved waves of the N = 128 register path
PTY_DEV float4 ld_stream4_pinned(const float4* p) {
    float4 v;
    asm volatile("ld.global.cs.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}
PTY_DEV void st_stream4(float4* p, float2 a, float2 b) { __stcs(p, make_float4(a.x, a.y, b.x, b.y)); }

// cache warming without a destination register
PTY_DEV void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }
PTY_DEV void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// bulk prefetch of a contiguous range into L2 (one thread, no registers, no L1): bytes % 16 == 0, 16-byte aligned
PTY_DEV void prefetch_l2_bulk(const void* p, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// ---- mbarrier + TMA (cp.async.bulk.tensor): tiles of a global tensor land in shared memory without passing through
// registers or L1; one elected thread issues, the consumers wait on the slot's "full" barrier and hand the slot back
// through its "empty" barrier (one arrival per consumer warp).
PTY_DEV unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
PTY_DEV void mbar_init(unsigned long long* b, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
PTY_DEV void mbar_init_fence() {      // make the initialised barriers visible to the async proxy
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
PTY_DEV void mbar_expect_tx(unsigned long long* b, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
PTY_DEV void mbar_arrive(unsigned long long* b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
PTY_DEV void mbar_wait(unsigned long long* b, unsigned parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "PTY_MBAR_WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra PTY_MBAR_DONE_%=;\n\t"
        "bra PTY_MBAR_WAIT_%=;\n\t"
        "PTY_MBAR_DONE_%=:\n\t}" ::"r"(smem_u32(b)), "r"(parity) : "memory");
}
// box of a 3-D tensor map -> shared memory (dst 128-byte aligned); completion counted in bytes on `bar`
PTY_DEV void tma_load_3d(void* dst, const CUtensorMap* tm, int c0, int c1, int c2, unsigned long long* bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(smem_u32(dst)), "l"(reinterpret_cast<unsigned long long>(tm)), "r"(c0), "r"(c1), "r"(c2),
                   "r"(smem_u32(bar)) : "memory");
}
PTY_DEV void tma_prefetch_desc(const CUtensorMap* tm) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<unsigned long long>(tm)) : "memory");
}

PTY_DEV void sincospi_f(float x, float* s, float* c) { sincospif(x, s, c); }
PTY_DEV float rsqrt_f(float x) { return rsqrtf(x); }
}  // namespace pty
