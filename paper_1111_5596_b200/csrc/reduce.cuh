// reduce.cuh -- deterministic global sums (hard part H4).
//
// Every reducing kernel ends in grid_reduce<K>(): warp shuffles, then a fixed
// shared-memory tree over the warps of the block, then one partial per block in
// a device buffer.  The last block to finish (ticket from an atomic counter)
// sums the partials in block-index order with the same fixed tree and writes the
// K results.  No floating-point atomics: the value depends only on the launch
// shape, so repeated runs are bit-identical.  All accumulation is fp64.
#pragma once
#ifndef __CUDACC_RTC__
#include <cuda_runtime.h>
#endif

namespace qdp {

constexpr int kReduceThreads = 256;   // default block size of the reducing kernels
constexpr int kMaxPartialBlocks = 2368;   // capacity of the partials buffer (blocks of a streaming reduction)

struct ReduceBuf {
    double* partials;        // [K][number of blocks or warps], then [K][number of groups]; K <= 4
    unsigned int* counter;   // [1 + number of groups], zero between launches
    double* result;          // [K] (device-visible)
    // Completion signal for the host: after the results are stored the final thread writes `seq` to *flag (mapped pinned
    // host memory; __threadfence_system between the two), so the host can poll instead of synchronising the stream.
    unsigned long long* flag;   // nullptr: no signal
    unsigned long long seq;
};
__device__ __forceinline__ void signal_results(const ReduceBuf& rb) {
    if (rb.flag) {
        __threadfence_system();
        *reinterpret_cast<volatile unsigned long long*>(rb.flag) = rb.seq;
    }
}
constexpr int kWarpGroup = 64;   // warps per group in warp_grid_reduce

// NT = threads per block (multiple of 32, <= 1024)
template <int K, int NT>
__device__ __forceinline__ void block_tree(double (&v)[K], double (*sm)[NT / 32]) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < K; k++) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_down_sync(0xffffffffu, v[k], o);
        if (lane == 0) sm[k][warp] = v[k];
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int k = 0; k < K; k++) {
            double t = lane < NT / 32 ? sm[k][lane] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
            v[k] = t;   // valid in thread 0
        }
    }
    __syncthreads();
}

// scale[k] multiplies result k (normalisation), applied once by the last block.
template <int K, int NT = kReduceThreads>
__device__ __forceinline__ void grid_reduce(double (&v)[K], const ReduceBuf& rb, const double* scale) {
    __shared__ double sm[K][NT / 32];
    __shared__ bool is_last;
    const unsigned int nblk = gridDim.x * gridDim.y, bid = blockIdx.y * gridDim.x + blockIdx.x;
    block_tree<K, NT>(v, sm);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < K; k++) rb.partials[k * nblk + bid] = v[k];
        __threadfence();
        unsigned int ticket = atomicAdd(rb.counter, 1u);
        is_last = ticket == nblk - 1;
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    // Thread t sums partials t, t + NT, ... in that order; eight loads are kept in flight
    // (a fused kernel has one partial per 128 sites, so a thread of the last block walks
    // ~100 of them and would otherwise pay one L2 round trip per partial).
    double t[K];
#pragma unroll
    for (int k = 0; k < K; k++) {
        const double* pk = rb.partials + (size_t)k * nblk;
        double acc = 0.0;
        unsigned int b = threadIdx.x;
        for (; b + 7u * NT < nblk; b += 8u * NT) {
            double v[8];
#pragma unroll
            for (int j = 0; j < 8; j++) v[j] = __ldcg(pk + b + j * NT);
#pragma unroll
            for (int j = 0; j < 8; j++) acc += v[j];
        }
        for (; b < nblk; b += NT) acc += __ldcg(pk + b);
        t[k] = acc;
    }
    block_tree<K, NT>(t, sm);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < K; k++) rb.result[k] = scale ? t[k] * scale[k] : t[k];
        *rb.counter = 0u;
        signal_results(rb);
    }
}

// Warp-granular variant for the fused kernels (hop + norm2, plaquette): no block barrier,
// so a warp that has finished its sites never waits for the slower warps of its block
// (ncu: the barrier of the block-level version cost hop_kernel<AXPY, NORM> 1.3 stalled warps
// per issue).  Two fixed levels keep the sum deterministic and the tail short: every warp
// stores one partial; the last warp to arrive in its group of kWarpGroup consecutive warps
// sums the group in warp order; the last group to finish sums the group partials in group
// order.  Every warp of the grid must call it (with zeros if it had no sites).
template <int K>
__device__ __forceinline__ void warp_grid_reduce(double (&v)[K], const ReduceBuf& rb, const double* scale) {
    const unsigned int lane = threadIdx.x & 31;
    const unsigned int wpb = blockDim.x >> 5;
    const unsigned int nw = gridDim.x * wpb, gw = blockIdx.x * wpb + (threadIdx.x >> 5);
    const unsigned int ng = (nw + kWarpGroup - 1) / kWarpGroup, grp = gw / kWarpGroup;
    const unsigned int g0 = grp * kWarpGroup, gsize = min((unsigned int)kWarpGroup, nw - g0);
    double* gpart = rb.partials + (size_t)K * nw;
#pragma unroll
    for (int k = 0; k < K; k++)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_down_sync(0xffffffffu, v[k], o);
    unsigned int ticket = 0;
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < K; k++) rb.partials[(size_t)k * nw + gw] = v[k];
        __threadfence();
        ticket = atomicAdd(&rb.counter[1 + grp], 1u);
    }
    ticket = __shfl_sync(0xffffffffu, ticket, 0);
    if (ticket != gsize - 1) return;
    __threadfence();
    // ---- last warp of the group: partials g0 .. g0 + gsize - 1 in warp order ----
    double t[K];
#pragma unroll
    for (int k = 0; k < K; k++) {
        const double* pk = rb.partials + (size_t)k * nw + g0;
        double a = lane < gsize ? __ldcg(pk + lane) : 0.0;
        double b = lane + 32 < gsize ? __ldcg(pk + lane + 32) : 0.0;
        t[k] = a + b;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t[k] += __shfl_down_sync(0xffffffffu, t[k], o);
    }
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < K; k++) gpart[(size_t)k * ng + grp] = t[k];
        rb.counter[1 + grp] = 0u;
        __threadfence();
        ticket = atomicAdd(&rb.counter[0], 1u);
    }
    ticket = __shfl_sync(0xffffffffu, ticket, 0);
    if (ticket != ng - 1) return;
    __threadfence();
    // ---- last group: group partials in group order, eight loads in flight per lane ----
#pragma unroll
    for (int k = 0; k < K; k++) {
        const double* pk = gpart + (size_t)k * ng;
        double acc = 0.0;
        unsigned int b = lane;
        for (; b + 7u * 32u < ng; b += 8u * 32u) {
            double w[8];
#pragma unroll
            for (int j = 0; j < 8; j++) w[j] = __ldcg(pk + b + j * 32);
#pragma unroll
            for (int j = 0; j < 8; j++) acc += w[j];
        }
        for (; b < ng; b += 32u) acc += __ldcg(pk + b);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
        t[k] = acc;
    }
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < K; k++) rb.result[k] = scale ? t[k] * scale[k] : t[k];
        rb.counter[0] = 0u;
        signal_results(rb);
    }
}

}  // namespace qdp
