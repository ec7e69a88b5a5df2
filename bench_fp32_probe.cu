// bench_fp32_probe.cu -- stand-alone FP32 pipe probe used by bench.py as a cross-check of the roofline
// denominator.  NOT part of the product library: it shares no code with
// paper_1006_4644_b200/csrc and nothing on the filter path calls it.
//
// Eight independent FMA chains per thread, 1024 threads per block, one block per SM.  Scalar FFMA
// (2 flop per lane and instruction) and packed FFMA2 (fma.rn.f32x2, 4 flop).  Both should read close to
// SMs x 128 lanes x 2 flop x SM clock.
//
// Build (bench.py does it on demand; __graft_entry__.build() too):
//   nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo -O3 -Xcompiler -fPIC -shared \
//        -o bench_fp32_probe.so bench_fp32_probe.cu
#include <cuda_runtime.h>

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

// Returns 0 on success, the cudaError_t otherwise.  Times on the legacy default stream of `device`.
extern "C" int fp32_probe(int device, double* tflops_ffma, double* tflops_ffma2)
{
    if (!tflops_ffma || !tflops_ffma2) return (int)cudaErrorInvalidValue;
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return (int)e;
    int n_sm = 0;
    if ((e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, device)) != cudaSuccess) return (int)e;
    float* buf = nullptr;
    if ((e = cudaMalloc(&buf, sizeof(float) * 1024 * (size_t)n_sm)) != cudaSuccess) return (int)e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
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
        res[packed] = flops / ((double)ms * 1e-3) / 1e12;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(buf);
    *tflops_ffma = res[0];
    *tflops_ffma2 = res[1];
    return (int)e;
}
