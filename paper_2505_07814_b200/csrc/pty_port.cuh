// pty_port.cuh -- the handful of device primitives the kernel bodies need (barriers, reductions
// into global memory, streaming loads/stores, fast math), sm_100a only.
#pragma once
#define PTY_PORT_INCLUDED
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
PTY_DEV void sincospi_f(float x, float* s, float* c) { sincospif(x, s, c); }
PTY_DEV float rsqrt_f(float x) { return rsqrtf(x); }
}  // namespace pty
