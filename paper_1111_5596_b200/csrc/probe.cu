// probe.cu -- bench-only peak probes (own shared library libqdp_probe.so; not part of the product ABI of
// include/qdp_b200.h).  bench.py times them in the same run as the kernels so that the "alu" roofline of an
// fp64-bound kernel has a measured denominator (the 37.2 TFLOP/s figure was units x clocks).
//
// qdp_probe_dfma: every thread runs 8 independent chains of dependent DFMAs (8.5-cycle latency, one warp
// instruction per ~2.3 cycles per SM sub-partition), 12 warps per SM, one block per SM: the plain (non-tensor)
// fp64 pipe at saturation.  Returns thread-level DFMA per second.
#include <cuda_runtime.h>

namespace {

constexpr int kChains = 8, kInner = 16, kThreads = 384;

__global__ void __launch_bounds__(kThreads, 1) dfma_kernel(double* out, int iters, double a, double b) {
    double v[kChains];
#pragma unroll
    for (int i = 0; i < kChains; i++) v[i] = threadIdx.x * 1e-9 + i;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int r = 0; r < kInner; r++)
#pragma unroll
            for (int i = 0; i < kChains; i++) v[i] = fma(v[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < kChains; i++) s += v[i];
    if (s == 123.456) out[0] = s;   // never true: keeps the chains alive
}

}  // namespace

// device: CUDA device index; stream: cudaStream_t or NULL.  On success *dfma_per_s = DFMA (thread-level) per second,
// median of `reps` launches timed with CUDA events on `stream`.  Returns 0, or the cudaError_t that occurred.
extern "C" int qdp_probe_dfma(int device, void* stream, int reps, double* dfma_per_s) {
    if (!dfma_per_s || reps < 1 || reps > 64) return (int)cudaErrorInvalidValue;
    cudaError_t e;
    int prev = 0, sms = 0;
    if ((e = cudaGetDevice(&prev)) != cudaSuccess) return (int)e;
    if ((e = cudaSetDevice(device)) != cudaSuccess) return (int)e;
    cudaStream_t st = (cudaStream_t)stream;
    double* out = nullptr;
    cudaEvent_t a = nullptr, b = nullptr;
    float ms[64];
    const int iters = 2000;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device)) != cudaSuccess) goto done;
    if ((e = cudaMalloc(&out, 64)) != cudaSuccess) goto done;
    if ((e = cudaEventCreate(&a)) != cudaSuccess || (e = cudaEventCreate(&b)) != cudaSuccess) goto done;
    for (int r = 0; r < reps + 2; r++) {   // two warm-up launches
        cudaEventRecord(a, st);
        dfma_kernel<<<sms, kThreads, 0, st>>>(out, iters, 1.0000001, 1e-9);
        cudaEventRecord(b, st);
        if ((e = cudaEventSynchronize(b)) != cudaSuccess) goto done;
        if (r >= 2) cudaEventElapsedTime(&ms[r - 2], a, b);
    }
    for (int i = 1; i < reps; i++)   // insertion sort, reps is small
        for (int j = i; j > 0 && ms[j] < ms[j - 1]; j--) { float t = ms[j]; ms[j] = ms[j - 1]; ms[j - 1] = t; }
    *dfma_per_s = (double)sms * kThreads * iters * kInner * kChains / (ms[reps / 2] * 1e-3);
done:
    if (a) cudaEventDestroy(a);
    if (b) cudaEventDestroy(b);
    if (out) cudaFree(out);
    cudaSetDevice(prev);
    return (int)e;
}
