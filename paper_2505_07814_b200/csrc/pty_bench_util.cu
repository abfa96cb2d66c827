// pty_bench_util.cu -- bench-side helper, NOT part of libpty.so / include/pty.h: an FP32-pipe microbenchmark
// that bench.py reports beside the nominal FP32 peak ("measure an FMA microbenchmark peak and
// the clock actually held").  Built into libpty_benchutil.so by paper_2505_07814_b200/build.py.
#include <cuda_runtime.h>
#include <cstdint>

// 16 independent chains per thread (8 float2), 8 CTAs of 512 threads per SM
template <int PACKED> __global__ void __launch_bounds__(512) fma_peak_kernel(float* out, float a, float b, int iters) {
    float2 x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = make_float2(threadIdx.x * 1e-3f + i, i * 0.5f);
    const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            if (PACKED) x[i] = __ffma2_rn(x[i], a2, b2);
            else { x[i].x = fmaf(x[i].x, a, b); x[i].y = fmaf(x[i].y, a, b); }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i].x + x[i].y;
    if (s == 12345.678f) out[0] = s;
}

// Achieved TFLOP/s (2 flops per FMA lane-operation) of scalar FFMA (packed = 0) or packed FFMA2 (packed = 1)
// chains on every SM of `device`; about 20 ms per repetition, best of the last two of three.  Returns 0 on
// success, -4 on a CUDA error.  Allocates and frees 4 bytes; synchronises the device.
extern "C" int pty_bench_fma_peak(int32_t device, int32_t packed, double* tflops) {
    if (!tflops) return -1;
    int prev = -1;
    cudaGetDevice(&prev);
    cudaDeviceProp prop;
    if (cudaSetDevice(device) != cudaSuccess || cudaGetDeviceProperties(&prop, device) != cudaSuccess) return -4;
    float* d = nullptr;
    if (cudaMalloc(&d, 4) != cudaSuccess) return -4;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int grid = prop.multiProcessorCount * 8, iters = 1 << 16;
    float best = 1e30f;
    int rc = 0;
    for (int r = 0; r < 3 && rc == 0; ++r) {
        cudaEventRecord(e0);
        if (packed) fma_peak_kernel<1><<<grid, 512>>>(d, 1.0001f, 0.5f, iters);
        else fma_peak_kernel<0><<<grid, 512>>>(d, 1.0001f, 0.5f, iters);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) { rc = -4; break; }
        float ms; cudaEventElapsedTime(&ms, e0, e1);
        if (r && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
    if (prev >= 0 && prev != device) cudaSetDevice(prev);
    if (rc == 0) *tflops = 2.0 * 16.0 * (double)iters * 512.0 * grid / (best * 1e-3) / 1e12;
    return rc;
}
