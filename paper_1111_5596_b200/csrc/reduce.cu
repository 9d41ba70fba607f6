// reduce.cu -- norm2, innerProduct, sum over a subset (def. 6).
// HBM-bound streaming reads: 16 B (fp64) per complex component, accumulated in
// fp64.  The subset's sites are a contiguous range of every component plane
// (checkerboard order), so the reads are fully coalesced for even/odd too.
#include "internal.h"
#include "su3.cuh"

namespace qdp {

constexpr int kUnroll = 4;

// grid = (blocks per plane, ncomp): blockIdx.y is the component plane, so no
// per-element division is needed to find the plane.
static dim3 reduce_grid(int n, int ncomp) {
    int per_block = kReduceThreads * kUnroll;
    int bx = (n + per_block - 1) / per_block;
    int cap = kMaxPartialBlocks / ncomp;
    if (bx > cap) bx = cap;
    if (bx < 1) bx = 1;
    return dim3(bx, ncomp);
}

template <class T2>
__global__ void __launch_bounds__(kReduceThreads) norm2_kernel(Geom g, const T2* __restrict__ f, int subset,
                                                              ReduceBuf rb) {
    const int n = subset_count(g, subset);
    const T2* plane = f + (size_t)blockIdx.y * g.V + subset_index(g, subset, 0);
    const int stride = gridDim.x * kReduceThreads;
    double acc[1] = {0.0};
    int i = blockIdx.x * kReduceThreads + threadIdx.x;
    for (; i + (kUnroll - 1) * stride < n; i += kUnroll * stride) {
        T2 v[kUnroll];
#pragma unroll
        for (int k = 0; k < kUnroll; k++) v[k] = __ldg(plane + i + k * stride);
#pragma unroll
        for (int k = 0; k < kUnroll; k++)
            acc[0] += (double)v[k].x * (double)v[k].x + (double)v[k].y * (double)v[k].y;
    }
    for (; i < n; i += stride) {
        T2 v = __ldg(plane + i);
        acc[0] += (double)v.x * (double)v.x + (double)v.y * (double)v.y;
    }
    grid_reduce<1>(acc, rb, nullptr);
}

template <class T2>
__global__ void __launch_bounds__(kReduceThreads) inner_kernel(Geom g, const T2* __restrict__ a,
                                                              const T2* __restrict__ b, int subset, ReduceBuf rb) {
    const int n = subset_count(g, subset);
    const size_t off = (size_t)blockIdx.y * g.V + subset_index(g, subset, 0);
    const T2 *pa = a + off, *pb = b + off;
    const int stride = gridDim.x * kReduceThreads;
    double acc[2] = {0.0, 0.0};
    int i = blockIdx.x * kReduceThreads + threadIdx.x;
    for (; i + (kUnroll - 1) * stride < n; i += kUnroll * stride) {
        T2 va[kUnroll], vb[kUnroll];
#pragma unroll
        for (int k = 0; k < kUnroll; k++) {
            va[k] = __ldg(pa + i + k * stride);
            vb[k] = __ldg(pb + i + k * stride);
        }
#pragma unroll
        for (int k = 0; k < kUnroll; k++) {   // conj(a) * b
            acc[0] += (double)va[k].x * (double)vb[k].x + (double)va[k].y * (double)vb[k].y;
            acc[1] += (double)va[k].x * (double)vb[k].y - (double)va[k].y * (double)vb[k].x;
        }
    }
    for (; i < n; i += stride) {
        T2 va = __ldg(pa + i), vb = __ldg(pb + i);
        acc[0] += (double)va.x * (double)vb.x + (double)va.y * (double)vb.y;
        acc[1] += (double)va.x * (double)vb.y - (double)va.y * (double)vb.x;
    }
    grid_reduce<2>(acc, rb, nullptr);
}

// sum: blockIdx.y = component plane; two kernels (partials, then a fixed-order finish)
constexpr int kSumBlocks = 64;
template <class T2>
__global__ void __launch_bounds__(kReduceThreads) sum_partial_kernel(Geom g, const T2* __restrict__ f, int subset,
                                                                    double* __restrict__ partials) {
    __shared__ double sm[2][kReduceThreads / 32];
    const int n = subset_count(g, subset);
    const T2* plane = f + (size_t)blockIdx.y * g.V + subset_index(g, subset, 0);
    double acc[2] = {0.0, 0.0};
    for (int i = blockIdx.x * kReduceThreads + threadIdx.x; i < n; i += gridDim.x * kReduceThreads) {
        T2 v = __ldg(plane + i);
        acc[0] += (double)v.x;
        acc[1] += (double)v.y;
    }
    block_tree<2, kReduceThreads>(acc, sm);
    if (threadIdx.x == 0) {
        partials[((size_t)blockIdx.y * gridDim.x + blockIdx.x) * 2 + 0] = acc[0];
        partials[((size_t)blockIdx.y * gridDim.x + blockIdx.x) * 2 + 1] = acc[1];
    }
}
__global__ void sum_finish_kernel(int nblk, const double* __restrict__ partials, double* __restrict__ out) {
    int c = blockIdx.x, k = threadIdx.x;   // 2 threads: re, im
    double t = 0.0;
    for (int b = 0; b < nblk; b++) t += partials[((size_t)c * nblk + b) * 2 + k];
    out[c * 2 + k] = t;
}

cudaError_t launch_norm2(int prec, const Geom& g, int ncomp, const void* f, int subset,
                         const ReduceBuf& rb, cudaStream_t st) {
    dim3 grid = reduce_grid(subset == 0 ? g.V : g.Vh, ncomp);
    if (prec) norm2_kernel<double2><<<grid, kReduceThreads, 0, st>>>(g, (const double2*)f, subset, rb);
    else      norm2_kernel<float2><<<grid, kReduceThreads, 0, st>>>(g, (const float2*)f, subset, rb);
    g_launch_count++;
    return cudaGetLastError();
}
cudaError_t launch_inner(int prec, const Geom& g, int ncomp, const void* a, const void* b, int subset,
                         const ReduceBuf& rb, cudaStream_t st) {
    dim3 grid = reduce_grid(subset == 0 ? g.V : g.Vh, ncomp);
    if (prec) inner_kernel<double2><<<grid, kReduceThreads, 0, st>>>(g, (const double2*)a, (const double2*)b, subset, rb);
    else      inner_kernel<float2><<<grid, kReduceThreads, 0, st>>>(g, (const float2*)a, (const float2*)b, subset, rb);
    g_launch_count++;
    return cudaGetLastError();
}
cudaError_t launch_sum(int prec, const Geom& g, int ncomp, const void* f, int subset,
                       double* partials, double* out_dev, cudaStream_t st) {
    dim3 grid(kSumBlocks, ncomp);
    if (prec) sum_partial_kernel<double2><<<grid, kReduceThreads, 0, st>>>(g, (const double2*)f, subset, partials);
    else      sum_partial_kernel<float2><<<grid, kReduceThreads, 0, st>>>(g, (const float2*)f, subset, partials);
    sum_finish_kernel<<<ncomp, 2, 0, st>>>(kSumBlocks, partials, out_dev);
    g_launch_count += 2;
    return cudaGetLastError();
}

}  // namespace qdp
