// reduce.cu -- norm2, innerProduct, sum over a subset (def. 6).
// HBM-bound streaming reads: 16 B (fp64) per complex component, accumulated in fp64.
// In the blocked layout (geom.cuh) a parity half of a field is one contiguous range of
// memory, so norm2 and inner are plain 128-bit streaming loops over [begin, begin + n)
// for all three subsets.  Only lattices whose half volume is not a multiple of 32 have
// padding lanes; those use the RAGGED instantiation, which masks them.
#include "internal.h"
#include "su3.cuh"

namespace qdp {

#ifndef RED_UNROLL
#define RED_UNROLL 4
#endif
#ifndef RED_BLOCKS_PER_SM
#define RED_BLOCKS_PER_SM 16
#endif
constexpr int kUnroll = RED_UNROLL;

static int stream_grid(size_t n) {
    size_t per_block = (size_t)kReduceThreads * kUnroll;
    size_t b = (n + per_block - 1) / per_block;
    size_t cap = (size_t)device_sm_count() * RED_BLOCKS_PER_SM;
    if (cap > (size_t)kMaxPartialBlocks) cap = kMaxPartialBlocks;   // size of the partials buffer
    if (b > cap) b = cap;
    if (b < 1) b = 1;
    return (int)b;
}

// element e of the field (e counted from the start of the buffer) belongs to a real site?
template <int NCOMP>
__device__ __forceinline__ bool real_lane(const Geom& g, unsigned e) {
    const unsigned half = (unsigned)g.Vhp * NCOMP;
    const unsigned eh = e >= half ? e - half : e;
    const unsigned hs = (eh / (NCOMP * 32u)) * 32u + (eh & 31u);
    return hs < (unsigned)g.Vh;
}

template <class T2, int NCOMP, bool RAGGED>
__global__ void __launch_bounds__(kReduceThreads) norm2_kernel(Geom g, const T2* __restrict__ f, int subset,
                                                              ReduceBuf rb) {
    const unsigned half = (unsigned)g.Vhp * NCOMP;
    const unsigned begin = subset == 2 ? half : 0u, n = subset == 0 ? 2u * half : half;
    const T2* p = f + begin;
    const unsigned stride = gridDim.x * kReduceThreads;
    double acc[1] = {0.0};
    unsigned e = blockIdx.x * kReduceThreads + threadIdx.x;
    for (; e + (kUnroll - 1) * stride < n; e += kUnroll * stride) {
        T2 v[kUnroll];
#pragma unroll
        for (int k = 0; k < kUnroll; k++) v[k] = __ldg(p + e + k * stride);
#pragma unroll
        for (int k = 0; k < kUnroll; k++)
            if (!RAGGED || real_lane<NCOMP>(g, begin + e + k * stride))
                acc[0] += (double)v[k].x * (double)v[k].x + (double)v[k].y * (double)v[k].y;
    }
    for (; e < n; e += stride) {
        T2 v = __ldg(p + e);
        if (!RAGGED || real_lane<NCOMP>(g, begin + e))
            acc[0] += (double)v.x * (double)v.x + (double)v.y * (double)v.y;
    }
    grid_reduce<1>(acc, rb, nullptr);
}

template <class T2, int NCOMP, bool RAGGED>
__global__ void __launch_bounds__(kReduceThreads) inner_kernel(Geom g, const T2* __restrict__ a,
                                                              const T2* __restrict__ b, int subset, ReduceBuf rb) {
    const unsigned half = (unsigned)g.Vhp * NCOMP;
    const unsigned begin = subset == 2 ? half : 0u, n = subset == 0 ? 2u * half : half;
    const T2 *pa = a + begin, *pb = b + begin;
    const unsigned stride = gridDim.x * kReduceThreads;
    double acc[2] = {0.0, 0.0};
    unsigned e = blockIdx.x * kReduceThreads + threadIdx.x;
    for (; e + (kUnroll - 1) * stride < n; e += kUnroll * stride) {
        T2 va[kUnroll], vb[kUnroll];
#pragma unroll
        for (int k = 0; k < kUnroll; k++) {
            va[k] = __ldg(pa + e + k * stride);
            vb[k] = __ldg(pb + e + k * stride);
        }
#pragma unroll
        for (int k = 0; k < kUnroll; k++)   // conj(a) * b
            if (!RAGGED || real_lane<NCOMP>(g, begin + e + k * stride)) {
                acc[0] += (double)va[k].x * (double)vb[k].x + (double)va[k].y * (double)vb[k].y;
                acc[1] += (double)va[k].x * (double)vb[k].y - (double)va[k].y * (double)vb[k].x;
            }
    }
    for (; e < n; e += stride) {
        T2 va = __ldg(pa + e), vb = __ldg(pb + e);
        if (!RAGGED || real_lane<NCOMP>(g, begin + e)) {
            acc[0] += (double)va.x * (double)vb.x + (double)va.y * (double)vb.y;
            acc[1] += (double)va.x * (double)vb.y - (double)va.y * (double)vb.x;
        }
    }
    grid_reduce<2>(acc, rb, nullptr);
}

// fp32 fields without padding lanes: two complex numbers per 128-bit load (a float2 stream would
// issue twice the load instructions for the same bytes: measured 0.056 ms vs the 0.031 ms floor
// for norm2 of a C4 spinor).
__global__ void __launch_bounds__(kReduceThreads) norm2_f32x2_kernel(const float4* __restrict__ p, unsigned n,
                                                                    ReduceBuf rb) {
    const unsigned stride = gridDim.x * kReduceThreads;
    double acc[1] = {0.0};
    unsigned e = blockIdx.x * kReduceThreads + threadIdx.x;
    for (; e + (kUnroll - 1) * stride < n; e += kUnroll * stride) {
        float4 v[kUnroll];
#pragma unroll
        for (int k = 0; k < kUnroll; k++) v[k] = __ldg(p + e + k * stride);
#pragma unroll
        for (int k = 0; k < kUnroll; k++)
            acc[0] += ((double)v[k].x * (double)v[k].x + (double)v[k].y * (double)v[k].y) +
                      ((double)v[k].z * (double)v[k].z + (double)v[k].w * (double)v[k].w);
    }
    for (; e < n; e += stride) {
        float4 v = __ldg(p + e);
        acc[0] += ((double)v.x * (double)v.x + (double)v.y * (double)v.y) +
                  ((double)v.z * (double)v.z + (double)v.w * (double)v.w);
    }
    grid_reduce<1>(acc, rb, nullptr);
}
__global__ void __launch_bounds__(kReduceThreads) inner_f32x2_kernel(const float4* __restrict__ pa,
                                                                    const float4* __restrict__ pb, unsigned n,
                                                                    ReduceBuf rb) {
    const unsigned stride = gridDim.x * kReduceThreads;
    double acc[2] = {0.0, 0.0};
    unsigned e = blockIdx.x * kReduceThreads + threadIdx.x;
    auto add = [&](const float4& a, const float4& b) {   // conj(a) * b for both complex numbers
        acc[0] += ((double)a.x * (double)b.x + (double)a.y * (double)b.y) + ((double)a.z * (double)b.z + (double)a.w * (double)b.w);
        acc[1] += ((double)a.x * (double)b.y - (double)a.y * (double)b.x) + ((double)a.z * (double)b.w - (double)a.w * (double)b.z);
    };
    for (; e + (kUnroll - 1) * stride < n; e += kUnroll * stride) {
        float4 va[kUnroll], vb[kUnroll];
#pragma unroll
        for (int k = 0; k < kUnroll; k++) {
            va[k] = __ldg(pa + e + k * stride);
            vb[k] = __ldg(pb + e + k * stride);
        }
#pragma unroll
        for (int k = 0; k < kUnroll; k++) add(va[k], vb[k]);
    }
    for (; e < n; e += stride) add(__ldg(pa + e), __ldg(pb + e));
    grid_reduce<2>(acc, rb, nullptr);
}

// sum: blockIdx.y = component; two kernels (partials, then a fixed-order finish)
constexpr int kSumBlocks = 64;
template <class T2>
__global__ void __launch_bounds__(kReduceThreads) sum_partial_kernel(Geom g, int ncomp, const T2* __restrict__ f,
                                                                    int subset, double* __restrict__ partials) {
    __shared__ double sm[2][kReduceThreads / 32];
    const int n = subset_count(g, subset);
    double acc[2] = {0.0, 0.0};
    for (int i = blockIdx.x * kReduceThreads + threadIdx.x; i < n; i += gridDim.x * kReduceThreads) {
        T2 v = __ldg(f + field_elem(ncomp, blockIdx.y, subset_index(g, subset, i)));
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

// ---- dst = a x + b y (+ fused norm2 of dst) -------------------------------------------------
// The residual / solution-reconstruction expressions of PAPER.md:96.  Element-wise on the
// contiguous range of the subset; dst may be x or y.  Padding lanes of a ragged lattice are
// written too (nothing reads them as sites) but masked out of the norm.
// a*x + b*y with the three roundings of the definition (no contraction into an fma), so that fp64
// results equal the oracle's bit for bit
__device__ __forceinline__ double axpby1(double a, double x, double b, double y) { return __dadd_rn(__dmul_rn(a, x), __dmul_rn(b, y)); }
__device__ __forceinline__ float axpby1(float a, float x, float b, float y) { return __fadd_rn(__fmul_rn(a, x), __fmul_rn(b, y)); }

template <class T2, bool NORM>
__global__ void __launch_bounds__(kReduceThreads) axpby_kernel(Geom g, int ncomp, T2* dst, const T2* x, const T2* y,
                                                              double a, double b, int subset, ReduceBuf rb) {
    using R = decltype(T2::x);
    const unsigned half = (unsigned)g.Vhp * ncomp;
    const unsigned begin = subset == 2 ? half : 0u, n = subset == 0 ? 2u * half : half;
    const bool ragged = g.Vh != g.Vhp;
    const R ra = (R)a, rb_ = (R)b;
    const unsigned stride = gridDim.x * kReduceThreads;
    double acc[1] = {0.0};
#pragma unroll 4
    for (unsigned e = blockIdx.x * kReduceThreads + threadIdx.x; e < n; e += stride) {
        const T2 vx = x[begin + e], vy = y[begin + e];
        T2 r;
        r.x = axpby1(ra, vx.x, rb_, vy.x);
        r.y = axpby1(ra, vx.y, rb_, vy.y);
        dst[begin + e] = r;
        if (NORM) {
            bool real = true;
            if (ragged) {
                const unsigned eh = begin + e >= half ? begin + e - half : begin + e;
                real = (eh / (ncomp * 32u)) * 32u + (eh & 31u) < (unsigned)g.Vh;
            }
            if (real) acc[0] += (double)r.x * (double)r.x + (double)r.y * (double)r.y;
        }
    }
    if (NORM) grid_reduce<1>(acc, rb, nullptr);
}

cudaError_t launch_axpby(int prec, const Geom& g, int ncomp, void* dst, const void* x, const void* y, double a,
                         double b, int subset, bool want_norm2, const ReduceBuf& rb, cudaStream_t st) {
    const size_t n = (size_t)g.Vhp * ncomp * (subset == 0 ? 2 : 1);
    const int grid = stream_grid(n);
    if (prec) {
        if (want_norm2) axpby_kernel<double2, true><<<grid, kReduceThreads, 0, st>>>(g, ncomp, (double2*)dst, (const double2*)x, (const double2*)y, a, b, subset, rb);
        else            axpby_kernel<double2, false><<<grid, kReduceThreads, 0, st>>>(g, ncomp, (double2*)dst, (const double2*)x, (const double2*)y, a, b, subset, rb);
    } else {
        if (want_norm2) axpby_kernel<float2, true><<<grid, kReduceThreads, 0, st>>>(g, ncomp, (float2*)dst, (const float2*)x, (const float2*)y, a, b, subset, rb);
        else            axpby_kernel<float2, false><<<grid, kReduceThreads, 0, st>>>(g, ncomp, (float2*)dst, (const float2*)x, (const float2*)y, a, b, subset, rb);
    }
    g_launch_count++;
    return cudaGetLastError();
}

// element e of (Gamma b) for a fermion field in the blocked layout (component = (e / 32) % 12 = 3 spin + colour)
template <class T2>
__device__ __forceinline__ T2 spin_apply(const SpinMatrix& gm, const T2* __restrict__ b, unsigned e) {
    const int sp = (int)((e >> 5) % 12u) / 3;
    const T2 v = __ldg(b + (long long)e + 96 * (gm.perm[sp] - sp));
    T2 r;
    switch (gm.ph[sp]) {                       // multiply by i^ph
        case 0: r.x = v.x; r.y = v.y; break;
        case 1: r.x = -v.y; r.y = v.x; break;
        case 2: r.x = -v.x; r.y = -v.y; break;
        default: r.x = v.y; r.y = -v.x; break;
    }
    return r;
}

// ---- time-slice inner products -----------------------------------
// out[t] = sum over the sites with x3 = t of conj(a) . b.  In the blocked layout the half-indices of
// a time-slice are one run [t*s3, (t+1)*s3) per parity half, so when s3 is a multiple of 32 a slice
// is two contiguous element ranges and the kernel streams them (blockIdx.y = t, kTsBlocks blocks
// per slice); otherwise (tiny or ragged lattices) every block scans its half and keeps the
// elements whose site has x3 = t.  One partial per block, summed in block order by the finish
// kernel: deterministic, fp64.
constexpr int kTsBlocks = 16;
// GAMMA: a is paired with (Gamma b), Gamma a phased permutation of the spin index (fermions only):
// (Gamma b)_{s c} = i^ph[s] b_{perm[s] c}, which in the blocked layout is the element 96 * (perm[s] - s)
// places further on.
template <class T2, bool FAST, bool GAMMA>
__global__ void __launch_bounds__(kReduceThreads) inner_ts_kernel(Geom g, int ncomp, const T2* __restrict__ a,
                                                                 const T2* __restrict__ b, int subset,
                                                                 double* __restrict__ partials, SpinMatrix gm) {
    __shared__ double sm[2][kReduceThreads / 32];
    const int t = blockIdx.y;
    const unsigned stride = gridDim.x * kReduceThreads;
    double acc[2] = {0.0, 0.0};
    for (int p = (subset == 2 ? 1 : 0); p <= (subset == 1 ? 0 : 1); p++) {
        if (FAST) {
            const size_t begin = ((size_t)p * g.Vhp + (size_t)t * g.s3) * ncomp;
            const unsigned n = (unsigned)g.s3 * ncomp;
            const T2 *pa = a + begin, *pb = b + begin;
#pragma unroll 4
            for (unsigned e = blockIdx.x * kReduceThreads + threadIdx.x; e < n; e += stride) {
                const T2 va = __ldg(pa + e);
                T2 vb;
                if (GAMMA) vb = spin_apply(gm, pb, e); else vb = __ldg(pb + e);
                acc[0] += (double)va.x * (double)vb.x + (double)va.y * (double)vb.y;
                acc[1] += (double)va.x * (double)vb.y - (double)va.y * (double)vb.x;
            }
        } else {
            const size_t begin = (size_t)p * g.Vhp * ncomp;
            const unsigned n = (unsigned)g.Vhp * ncomp;
            for (unsigned e = blockIdx.x * kReduceThreads + threadIdx.x; e < n; e += stride) {
                const int h = (int)(e / (ncomp * 32u)) * 32 + (int)(e & 31u);
                if (h >= g.Vh || h / g.s3 != t) continue;
                const T2 va = __ldg(a + begin + e);
                T2 vb;
                if (GAMMA) vb = spin_apply(gm, b + begin, e); else vb = __ldg(b + begin + e);
                acc[0] += (double)va.x * (double)vb.x + (double)va.y * (double)vb.y;
                acc[1] += (double)va.x * (double)vb.y - (double)va.y * (double)vb.x;
            }
        }
    }
    block_tree<2, kReduceThreads>(acc, sm);
    if (threadIdx.x == 0) {
        partials[((size_t)t * gridDim.x + blockIdx.x) * 2 + 0] = acc[0];
        partials[((size_t)t * gridDim.x + blockIdx.x) * 2 + 1] = acc[1];
    }
}
__global__ void inner_ts_finish_kernel(int nblk, const double* __restrict__ partials, double* __restrict__ out) {
    const int t = blockIdx.x, k = threadIdx.x;   // 2 threads: re, im
    double s = 0.0;
    for (int b = 0; b < nblk; b++) s += partials[((size_t)t * nblk + b) * 2 + k];
    out[t * 2 + k] = s;
}

cudaError_t launch_inner_timeslices(int prec, const Geom& g, int ncomp, const void* a, const void* b, int subset,
                                    double* partials, double* out_dev, cudaStream_t st, const SpinMatrix* gamma) {
    dim3 grid(kTsBlocks, g.L3);
    const bool fast = (g.s3 & 31) == 0;
    SpinMatrix gm = gamma ? *gamma : SpinMatrix{{0, 1, 2, 3}, {0, 0, 0, 0}};
#define QDP_TS(T2, F, G) inner_ts_kernel<T2, F, G><<<grid, kReduceThreads, 0, st>>>(g, ncomp, (const T2*)a, (const T2*)b, subset, partials, gm)
    if (prec) {
        if (gamma) { if (fast) QDP_TS(double2, true, true); else QDP_TS(double2, false, true); }
        else       { if (fast) QDP_TS(double2, true, false); else QDP_TS(double2, false, false); }
    } else {
        if (gamma) { if (fast) QDP_TS(float2, true, true); else QDP_TS(float2, false, true); }
        else       { if (fast) QDP_TS(float2, true, false); else QDP_TS(float2, false, false); }
    }
#undef QDP_TS
    inner_ts_finish_kernel<<<g.L3, 2, 0, st>>>(kTsBlocks, partials, out_dev);
    g_launch_count += 2;
    return cudaGetLastError();
}

template <class T2, int NCOMP>
static void norm2_dispatch(const Geom& g, const void* f, int subset, const ReduceBuf& rb, cudaStream_t st) {
    size_t n = (size_t)g.Vhp * NCOMP * (subset == 0 ? 2 : 1);
    int grid = stream_grid(n);
    if (sizeof(T2) == 8 && g.Vh == g.Vhp) {
        const float4* p = (const float4*)((const float2*)f + (subset == 2 ? (size_t)g.Vhp * NCOMP : 0));
        norm2_f32x2_kernel<<<stream_grid(n / 2), kReduceThreads, 0, st>>>(p, (unsigned)(n / 2), rb);
        return;
    }
    if (g.Vh == g.Vhp) norm2_kernel<T2, NCOMP, false><<<grid, kReduceThreads, 0, st>>>(g, (const T2*)f, subset, rb);
    else               norm2_kernel<T2, NCOMP, true><<<grid, kReduceThreads, 0, st>>>(g, (const T2*)f, subset, rb);
}
template <class T2, int NCOMP>
static void inner_dispatch(const Geom& g, const void* a, const void* b, int subset, const ReduceBuf& rb,
                           cudaStream_t st) {
    size_t n = (size_t)g.Vhp * NCOMP * (subset == 0 ? 2 : 1);
    int grid = stream_grid(n);
    if (sizeof(T2) == 8 && g.Vh == g.Vhp) {
        const size_t off = subset == 2 ? (size_t)g.Vhp * NCOMP : 0;
        inner_f32x2_kernel<<<stream_grid(n / 2), kReduceThreads, 0, st>>>(
            (const float4*)((const float2*)a + off), (const float4*)((const float2*)b + off), (unsigned)(n / 2), rb);
        return;
    }
    if (g.Vh == g.Vhp)
        inner_kernel<T2, NCOMP, false><<<grid, kReduceThreads, 0, st>>>(g, (const T2*)a, (const T2*)b, subset, rb);
    else
        inner_kernel<T2, NCOMP, true><<<grid, kReduceThreads, 0, st>>>(g, (const T2*)a, (const T2*)b, subset, rb);
}

cudaError_t launch_norm2(int prec, const Geom& g, int ncomp, const void* f, int subset,
                         const ReduceBuf& rb, cudaStream_t st) {
    if (prec) {
        if (ncomp == 9) norm2_dispatch<double2, 9>(g, f, subset, rb, st);
        else if (ncomp == 12) norm2_dispatch<double2, 12>(g, f, subset, rb, st);
        else norm2_dispatch<double2, 36>(g, f, subset, rb, st);
    } else {
        if (ncomp == 9) norm2_dispatch<float2, 9>(g, f, subset, rb, st);
        else if (ncomp == 12) norm2_dispatch<float2, 12>(g, f, subset, rb, st);
        else norm2_dispatch<float2, 36>(g, f, subset, rb, st);
    }
    g_launch_count++;
    return cudaGetLastError();
}
cudaError_t launch_inner(int prec, const Geom& g, int ncomp, const void* a, const void* b, int subset,
                         const ReduceBuf& rb, cudaStream_t st) {
    if (prec) {
        if (ncomp == 9) inner_dispatch<double2, 9>(g, a, b, subset, rb, st);
        else if (ncomp == 12) inner_dispatch<double2, 12>(g, a, b, subset, rb, st);
        else inner_dispatch<double2, 36>(g, a, b, subset, rb, st);
    } else {
        if (ncomp == 9) inner_dispatch<float2, 9>(g, a, b, subset, rb, st);
        else if (ncomp == 12) inner_dispatch<float2, 12>(g, a, b, subset, rb, st);
        else inner_dispatch<float2, 36>(g, a, b, subset, rb, st);
    }
    g_launch_count++;
    return cudaGetLastError();
}
cudaError_t launch_sum(int prec, const Geom& g, int ncomp, const void* f, int subset,
                       double* partials, double* out_dev, cudaStream_t st) {
    dim3 grid(kSumBlocks, ncomp);
    if (prec) sum_partial_kernel<double2><<<grid, kReduceThreads, 0, st>>>(g, ncomp, (const double2*)f, subset, partials);
    else      sum_partial_kernel<float2><<<grid, kReduceThreads, 0, st>>>(g, ncomp, (const float2*)f, subset, partials);
    sum_finish_kernel<<<ncomp, 2, 0, st>>>(kSumBlocks, partials, out_dev);
    g_launch_count += 2;
    return cudaGetLastError();
}

}  // namespace qdp
