// probe.cu -- bench-only peak probes (own shared library libqdp_probe.so; not part of the product ABI of
// include/qdp_b200.h).  bench.py times them in the same run as the kernels so that the "alu" roofline of an
// fp64-bound kernel has a measured denominator (the 37.2 TFLOP/s figure was units x clocks).
//
// qdp_probe_dfma: every thread runs 8 independent chains of dependent DFMAs (8.5-cycle latency, one warp
// instruction per ~2.3 cycles per SM sub-partition), 12 warps per SM, one block per SM: the plain (non-tensor)
// fp64 pipe at saturation.  Returns thread-level DFMA per second.
#include <cstdint>
#include <cuda_runtime.h>

#include "tma.cuh"

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

// ---- how far shared-memory reads, the fp64 pipe and bulk copies into shared memory overlap ---------------------
// One persistent block per SM shaped like the staged plaquette kernel (plaquette_tma.cu): 12 consumer warps, each
// doing per "step" NL LDS.128 (36 = the four 3x3 operands of one plaquette plane) and 234 DFMA, plus a producer warp
// that bulk-copies 92,160 bytes per step from an L2-resident buffer into a shared-memory ring and waits for it.
// MODE bit 0: the LDS, bit 1: the DFMA, bit 2: the bulk copies.  (profiles/r2_microbench.md)
template <int MODE, int NL>
__global__ void __launch_bounds__(416, 1) mix_kernel(double* out, const double2* __restrict__ src, int steps, double a, double b) {
    extern __shared__ __align__(128) unsigned char smem_probe[];
    double2* tile = reinterpret_cast<double2*>(smem_probe);                 // 96 KB of operands
    double2* ring = reinterpret_cast<double2*>(smem_probe + 98304);         // 96 KB target of the bulk copies
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_probe + 196608);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < 6144; i += blockDim.x) tile[i] = make_double2(i * 1e-6, 1.0 - i * 1e-6);
    if (threadIdx.x == 0) { qdp::mbar_init(&bar[0], 1); qdp::mbar_fence_init(); }
    __syncthreads();
    if (warp == 12) {
        if ((MODE & 4) && lane == 0)
            for (int s = 0; s < steps; s++) {
                qdp::mbar_arrive_expect_tx(&bar[0], 92160);
                for (int c = 0; c < 5; c++)
                    qdp::bulk_g2s(ring + c * 1152, src + ((size_t)blockIdx.x * 5 + c) * 1152, 18432, &bar[0]);
                qdp::mbar_wait(&bar[0], s & 1);
            }
        return;
    }
    double acc[18];
#pragma unroll
    for (int i = 0; i < 18; i++) acc[i] = lane * 1e-9 + i;
    double2 sink = make_double2(0, 0);
    for (int s = 0; s < steps; s++) {
        double2 m[36];
#pragma unroll
        for (int c = 0; c < 36; c++)
            m[c] = ((MODE & 1) && c < NL) ? tile[((warp * 36 + c + s) % 192) * 32 + lane] : make_double2(a + c, b - c);
        if (MODE & 2) {
#pragma unroll
            for (int r = 0; r < 13; r++)
#pragma unroll
                for (int i = 0; i < 18; i++) acc[i] = fma(acc[i], (r & 1) ? m[(i + r) % 36].x : m[(i + r + 18) % 36].y, b);
        } else {
#pragma unroll
            for (int c = 0; c < 36; c++) { sink.x += m[c].x; sink.y += m[c].y; }
        }
    }
    double t = sink.x + sink.y;
#pragma unroll
    for (int i = 0; i < 18; i++) t += acc[i];
    if (t == 123.456) out[0] = t;
}

// ---- do operand loads and DFMAs of the SAME warp overlap? -------------------------------------------------------
// The register kernels (plaquette.cu, ape.cu, hop.cu) run 2 warps per sub-partition at 255 registers; their measured
// times are close to (L1 data-pipe time) + (fp64 pipe time).  This probe isolates the cause: NW warps per SM, per step
// and warp NL 128-bit loads (SRC 0: LDS from shared memory, SRC 1: LDG that hits L1) and 234 DFMAs on the loaded values;
// PIPE 0: the loads of a step are issued at its start (a warp alternates between a load phase and an arithmetic phase,
// only other warps can fill the gaps), PIPE 1: the loads of step s+1 are issued before the arithmetic of step s
// (register double buffer), so one warp has both pipes busy at once.  MODE bit 0: loads, bit 1: DFMAs.
template <int MODE, int NL, int SRC, int PIPE, int NW>
__global__ void __launch_bounds__(NW * 32, 1) overlap_kernel(double* out, const double2* __restrict__ gsrc, int steps, double a, double b) {
    extern __shared__ __align__(128) unsigned char smem_probe[];
    double2* tile = reinterpret_cast<double2*>(smem_probe);                 // 96 KB = 192 planes of 32 double2
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const double2* src = SRC ? gsrc + (size_t)blockIdx.x * 6144 : tile;
    if (!SRC) for (int i = threadIdx.x; i < 6144; i += blockDim.x) tile[i] = make_double2(i * 1e-6, 1.0 - i * 1e-6);
    __syncthreads();
    double acc[18];
#pragma unroll
    for (int i = 0; i < 18; i++) acc[i] = lane * 1e-9 + i;
    double2 sink = make_double2(0, 0);
    auto load = [&](double2 (&m)[NL], int s) {
#pragma unroll
        for (int c = 0; c < NL; c++) {
            const double2* q = src + ((warp * NL + c + s) % 192) * 32 + lane;
            m[c] = (MODE & 1) ? (SRC ? __ldg(q) : *q) : make_double2(a + c, b - c);
        }
    };
    auto math = [&](const double2 (&m)[NL]) {
        if (MODE & 2) {
#pragma unroll
            for (int r = 0; r < 13; r++)
#pragma unroll
                for (int i = 0; i < 18; i++) acc[i] = fma(acc[i], (r & 1) ? m[(i + r) % NL].x : m[(i + r + NL / 2) % NL].y, b);
        } else {
#pragma unroll
            for (int c = 0; c < NL; c++) { sink.x += m[c].x; sink.y += m[c].y; }
        }
    };
    if (PIPE) {
        double2 m0[NL], m1[NL];
        load(m0, 0);
        for (int s = 0; s < steps; s += 2) {
            load(m1, s + 1);
            math(m0);
            load(m0, s + 2);
            math(m1);
        }
    } else {
        for (int s = 0; s < steps; s++) {
            double2 m[NL];
            load(m, s);
            math(m);
        }
    }
    double t = sink.x + sink.y;
#pragma unroll
    for (int i = 0; i < 18; i++) t += acc[i];
    if (t == 123.456) out[0] = t;
}

// ---- bulk copies from L2 into shared memory: per-SM ingest rate against the number of active SMs ------------------
// One lane per block keeps two 92,160-byte slots filled with `ncopies` cp.async.bulk copies per step from an L2-resident
// buffer, issuing step s+1 before it waits for step s.  With few blocks the rate is what one SM can ingest; with one
// block on every SM it is what the L2 can deliver to all of them (profiles/r2_microbench.md).
__global__ void __launch_bounds__(32, 1) bulk_rate_kernel(const double2* __restrict__ src, int steps, int ncopies, int bytes_each) {
    extern __shared__ __align__(128) unsigned char smem_probe[];
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_probe + 200704);
    if (threadIdx.x == 0) { qdp::mbar_init(&bar[0], 1); qdp::mbar_init(&bar[1], 1); qdp::mbar_fence_init(); }
    __syncthreads();
    if (threadIdx.x != 0) return;
    const char* base = reinterpret_cast<const char*>(src) + (size_t)blockIdx.x * ncopies * bytes_each;
    for (int s = 0; s < steps + 1; s++) {
        if (s < steps) {
            qdp::mbar_arrive_expect_tx(&bar[s & 1], ncopies * bytes_each);
            for (int c = 0; c < ncopies; c++)
                qdp::bulk_g2s(smem_probe + (s & 1) * 100352 + c * bytes_each, base + (size_t)c * bytes_each, bytes_each, &bar[s & 1]);
        }
        if (s >= 1) qdp::mbar_wait(&bar[(s - 1) & 1], ((s - 1) >> 1) & 1);
    }
}

template <int CHAINS>
__global__ void dfma_chain_kernel(double* out, int iters, double a, double b) {
    double v[CHAINS];
#pragma unroll
    for (int i = 0; i < CHAINS; i++) v[i] = threadIdx.x * 1e-9 + i;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int r = 0; r < 16; r++)
#pragma unroll
            for (int i = 0; i < CHAINS; i++) v[i] = fma(v[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < CHAINS; i++) s += v[i];
    if (s == 123.456) out[0] = s;
}

template <class F> cudaError_t time_launches(cudaStream_t st, int reps, float* med_ms, F launch) {
    cudaEvent_t a = nullptr, b = nullptr;
    cudaError_t e;
    float ms[16];
    if (reps > 16) reps = 16;
    if ((e = cudaEventCreate(&a)) != cudaSuccess) return e;
    if ((e = cudaEventCreate(&b)) != cudaSuccess) { cudaEventDestroy(a); return e; }
    for (int r = 0; r < reps + 2; r++) {
        cudaEventRecord(a, st);
        launch();
        cudaEventRecord(b, st);
        if ((e = cudaEventSynchronize(b)) != cudaSuccess) break;
        if (r >= 2) cudaEventElapsedTime(&ms[r - 2], a, b);
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    for (int i = 1; i < reps; i++)
        for (int j = i; j > 0 && ms[j] < ms[j - 1]; j--) { float t = ms[j]; ms[j] = ms[j - 1]; ms[j - 1] = t; }
    *med_ms = ms[reps / 2];
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    return e;
}

template <int MODE, int NL>
cudaError_t run_mix(cudaStream_t st, int sms, double* out, const double2* src, int steps, float* ms) {
    const int smem = 196608 + 64;
    cudaError_t e = cudaFuncSetAttribute(mix_kernel<MODE, NL>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    return time_launches(st, 7, ms, [&] { mix_kernel<MODE, NL><<<sms, 416, smem, st>>>(out, src, steps, 1.0000001, 1e-9); });
}

}  // namespace

// mode: bit 0 LDS, bit 1 DFMA, bit 2 bulk copies; nlds: 36, 28, 24 or 18 LDS.128 per warp and step.  *ms_per_step =
// median launch time / steps (221 steps, the number the staged plaquette kernel runs per SM on 32^3 x 64).
extern "C" int qdp_probe_mix(int device, void* stream, int mode, int nlds, double* ms_per_step) {
    if (!ms_per_step || mode < 1 || mode > 7) return (int)cudaErrorInvalidValue;
    cudaError_t e;
    int prev = 0, sms = 0;
    if ((e = cudaGetDevice(&prev)) != cudaSuccess) return (int)e;
    if ((e = cudaSetDevice(device)) != cudaSuccess) return (int)e;
    cudaStream_t st = (cudaStream_t)stream;
    double* out = nullptr;
    double2* src = nullptr;
    const int steps = 221;
    float ms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    if (e == cudaSuccess) e = cudaMalloc(&out, 64);
    if (e == cudaSuccess) e = cudaMalloc(&src, (size_t)sms * 5 * 1152 * sizeof(double2));
    if (e == cudaSuccess) e = cudaMemset(src, 0, (size_t)sms * 5 * 1152 * sizeof(double2));
    if (e == cudaSuccess) {
#define QDP_MIX(M) (nlds == 36 ? run_mix<M, 36>(st, sms, out, src, steps, &ms) : nlds == 28 ? run_mix<M, 28>(st, sms, out, src, steps, &ms) \
                  : nlds == 24 ? run_mix<M, 24>(st, sms, out, src, steps, &ms) : nlds == 18 ? run_mix<M, 18>(st, sms, out, src, steps, &ms) : cudaErrorInvalidValue)
        switch (mode) {
            case 1: e = QDP_MIX(1); break;
            case 2: e = QDP_MIX(2); break;
            case 3: e = QDP_MIX(3); break;
            case 4: e = QDP_MIX(4); break;
            case 5: e = QDP_MIX(5); break;
            case 6: e = QDP_MIX(6); break;
            default: e = QDP_MIX(7); break;
        }
#undef QDP_MIX
    }
    if (e == cudaSuccess) *ms_per_step = (double)ms / steps;
    if (out) cudaFree(out);
    if (src) cudaFree(src);
    cudaSetDevice(prev);
    return (int)e;
}

template <int MODE, int SRC, int PIPE, int NW>
cudaError_t run_overlap(cudaStream_t st, int sms, double* out, const double2* src, int steps, float* ms) {
    const int smem = 98304;
    cudaError_t e = cudaFuncSetAttribute(overlap_kernel<MODE, 24, SRC, PIPE, NW>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    return time_launches(st, 7, ms, [&] { overlap_kernel<MODE, 24, SRC, PIPE, NW><<<sms, NW * 32, smem, st>>>(out, src, steps, 1.0000001, 1e-9); });
}

// mode: bit 0 loads (24 x 128 bit per warp and step), bit 1 DFMAs (234 per warp and step); src: 0 shared memory, 1 global
// memory resident in L1; pipe: 0 load phase then arithmetic phase, 1 loads of the next step issued before the arithmetic
// of this one; warps: 8 (2 per sub-partition, what the 255-register kernels run).  *ms_per_step = median time / steps.
extern "C" int qdp_probe_overlap(int device, void* stream, int mode, int src_kind, int pipe, double* ms_per_step) {
    if (!ms_per_step || mode < 1 || mode > 3 || src_kind < 0 || src_kind > 1 || pipe < 0 || pipe > 1) return (int)cudaErrorInvalidValue;
    cudaError_t e;
    int prev = 0, sms = 0;
    if ((e = cudaGetDevice(&prev)) != cudaSuccess) return (int)e;
    if ((e = cudaSetDevice(device)) != cudaSuccess) return (int)e;
    cudaStream_t st = (cudaStream_t)stream;
    double* out = nullptr;
    double2* src = nullptr;
    const int steps = 400;
    float ms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    if (e == cudaSuccess) e = cudaMalloc(&out, 64);
    if (e == cudaSuccess) e = cudaMalloc(&src, ((size_t)sms * 6144 + 64) * sizeof(double2));
    if (e == cudaSuccess) e = cudaMemset(src, 0, ((size_t)sms * 6144 + 64) * sizeof(double2));
    if (e == cudaSuccess) {
#define QDP_OV(M) (src_kind == 0 ? (pipe ? run_overlap<M, 0, 1, 8>(st, sms, out, src, steps, &ms) : run_overlap<M, 0, 0, 8>(st, sms, out, src, steps, &ms)) \
                                 : (pipe ? run_overlap<M, 1, 1, 8>(st, sms, out, src, steps, &ms) : run_overlap<M, 1, 0, 8>(st, sms, out, src, steps, &ms)))
        e = mode == 1 ? QDP_OV(1) : mode == 2 ? QDP_OV(2) : QDP_OV(3);
#undef QDP_OV
    }
    if (e == cudaSuccess) *ms_per_step = (double)ms / steps;
    if (out) cudaFree(out);
    if (src) cudaFree(src);
    cudaSetDevice(prev);
    return (int)e;
}

// blocks: active SMs (1 .. SM count); ncopies: copies per 92,160-byte step (5 -> 18,432 B each, 20 -> 4,608 B each).
// *bytes_per_s = bytes copied per second by all blocks together.
extern "C" int qdp_probe_bulk_rate(int device, void* stream, int blocks, int ncopies, double* bytes_per_s) {
    if (!bytes_per_s || blocks < 1 || (ncopies != 5 && ncopies != 20)) return (int)cudaErrorInvalidValue;
    cudaError_t e;
    int prev = 0, sms = 0;
    if ((e = cudaGetDevice(&prev)) != cudaSuccess) return (int)e;
    if ((e = cudaSetDevice(device)) != cudaSuccess) return (int)e;
    cudaStream_t st = (cudaStream_t)stream;
    double2* src = nullptr;
    const int steps = 400, smem = 200704 + 64;
    float ms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    if (e == cudaSuccess && blocks > sms) e = cudaErrorInvalidValue;
    if (e == cudaSuccess) e = cudaMalloc(&src, (size_t)sms * 92160 + 1024);
    if (e == cudaSuccess) e = cudaMemset(src, 0, (size_t)sms * 92160);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(bulk_rate_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e == cudaSuccess)
        e = time_launches(st, 7, &ms, [&] { bulk_rate_kernel<<<blocks, 32, smem, st>>>(src, steps, ncopies, 92160 / ncopies); });
    if (e == cudaSuccess) *bytes_per_s = (double)blocks * steps * 92160 / (ms * 1e-3);
    if (src) cudaFree(src);
    cudaSetDevice(prev);
    return (int)e;
}

// Dependent-issue behaviour of the fp64 pipe: one warp per SM (warps = 1) or one per sub-partition (warps = 4) running
// `chains` (1, 2, 4 or 8) independent chains of dependent DFMAs.  *ns_per_dfma = time per DFMA of one warp.
extern "C" int qdp_probe_dfma_chain(int device, void* stream, int warps, int chains, double* ns_per_dfma) {
    if (!ns_per_dfma || (warps != 1 && warps != 4)) return (int)cudaErrorInvalidValue;
    cudaError_t e;
    int prev = 0, sms = 0;
    if ((e = cudaGetDevice(&prev)) != cudaSuccess) return (int)e;
    if ((e = cudaSetDevice(device)) != cudaSuccess) return (int)e;
    cudaStream_t st = (cudaStream_t)stream;
    double* out = nullptr;
    const int iters = 2000;
    float ms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    if (e == cudaSuccess) e = cudaMalloc(&out, 64);
    if (e == cudaSuccess) {
        const int th = 32 * warps;
        switch (chains) {
            case 1: e = time_launches(st, 7, &ms, [&] { dfma_chain_kernel<1><<<sms, th, 0, st>>>(out, iters, 1.0000001, 1e-9); }); break;
            case 2: e = time_launches(st, 7, &ms, [&] { dfma_chain_kernel<2><<<sms, th, 0, st>>>(out, iters, 1.0000001, 1e-9); }); break;
            case 4: e = time_launches(st, 7, &ms, [&] { dfma_chain_kernel<4><<<sms, th, 0, st>>>(out, iters, 1.0000001, 1e-9); }); break;
            case 8: e = time_launches(st, 7, &ms, [&] { dfma_chain_kernel<8><<<sms, th, 0, st>>>(out, iters, 1.0000001, 1e-9); }); break;
            default: e = cudaErrorInvalidValue;
        }
    }
    if (e == cudaSuccess) *ns_per_dfma = (double)ms * 1e6 / ((double)iters * 16 * chains);
    if (out) cudaFree(out);
    cudaSetDevice(prev);
    return (int)e;
}

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
