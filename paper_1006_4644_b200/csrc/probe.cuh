// probe.cuh -- FP32 pipe probe behind cbmf_debug_fp32_peak (include/cbmf.h): the measured cross-check of the
// roofline denominator that bench.py reports.  A diagnostic of the library: nothing on the filter
// path calls it and it shares no code with the filter kernels.
//
// Eight independent FMA chains per thread, 1024 threads per block, one block per SM.  Scalar FFMA
// (2 flop per lane and instruction) and packed FFMA2 (fma.rn.f32x2, 4 flop).  Both should read close to
// SMs x 128 lanes x 2 flop x SM clock.
#pragma once
#include <cuda_runtime.h>

namespace cbmf_probe {

typedef unsigned long long pk2;

__device__ __forceinline__ pk2 pack2(float x, float y)
{
    pk2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(x), "f"(y));
    return r;
}
__device__ __forceinline__ pk2 fma2x(pk2 a, pk2 b, pk2 c)
{
    pk2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}

template <bool PACKED>
__global__ void __launch_bounds__(1024, 1) fp32_probe_kernel(float* __restrict__ out, const int iters, const float s)
{
    float a[8];
    pk2 p[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { a[i] = (float)threadIdx.x * 1e-3f + (float)i; p[i] = pack2(a[i], a[i] + 1.f); }
    const pk2 ps = pack2(s, s * 0.5f), pc = pack2(0.25f, 0.125f);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if constexpr (PACKED) p[i] = fma2x(p[i], ps, pc);
                else a[i] = fmaf(a[i], s, 0.25f);
            }
    }
    float acc = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        float x, y;
        asm("mov.b64 {%0, %1}, %2;" : "=f"(x), "=f"(y) : "l"(p[i]));
        acc += a[i] + x + y;
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

// Times on the legacy default stream of `device`; restores the caller's current device.
inline cudaError_t fp32_peak(int device, double* tflops_ffma, double* tflops_ffma2)
{
    int prev = -1;
    cudaGetDevice(&prev);
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return e;
    int n_sm = 0;
    float* buf = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if ((e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, device)) == cudaSuccess)
        e = cudaMalloc(&buf, sizeof(float) * 1024 * (size_t)n_sm);
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    const int iters = 4000;
    double res[2] = {0, 0};
    for (int packed = 0; packed < 2 && e == cudaSuccess; ++packed) {
        for (int rep = 0; rep < 2; ++rep) {           // the first launch warms up
            cudaEventRecord(e0, 0);
            if (packed) fp32_probe_kernel<true><<<n_sm, 1024>>>(buf, iters, 1.0001f);
            else fp32_probe_kernel<false><<<n_sm, 1024>>>(buf, iters, 1.0001f);
            cudaEventRecord(e1, 0);
            e = cudaEventSynchronize(e1);
            if (e != cudaSuccess) break;
        }
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        const double flops = 2.0 * (packed ? 2.0 : 1.0) * 8.0 * 4.0 * (double)iters * 1024.0 * (double)n_sm;
        if (e == cudaSuccess && ms > 0.f) res[packed] = flops / ((double)ms * 1e-3) / 1e12;
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(buf);
    if (prev >= 0) cudaSetDevice(prev);
    *tflops_ffma = res[0];
    *tflops_ffma2 = res[1];
    return e;
}

}  // namespace cbmf_probe
