// shift.cu -- dst(x) = src(x + sign*mu_hat) on a subset (def. 1).
// Pure data movement: 2 x 16 B (fp64) per complex component, one read + one write.
// A thread moves kPlanes component planes of one site, so kPlanes independent
// 128-bit loads are in flight per thread; blockIdx.y selects the plane group.
#include "internal.h"
#include "su3.cuh"

namespace qdp {

constexpr int kPlanes = 3;   // 9, 36 and 12 components are all multiples of 3

template <class T2>
__global__ void __launch_bounds__(256) shift_kernel(Geom g, int ncomp, T2* __restrict__ dst,
                                                   const T2* __restrict__ src, int mu, int sign, int subset) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= subset_count(g, subset)) return;
    Site x = subset_site(g, subset, i);
    const int s = x.index(g);
    const int n = site_step_rt(g, x, mu, sign).index(g);
    const int c0 = blockIdx.y * kPlanes;
    const T2* from = site_ptr(src, ncomp, c0, n);
    T2* to = site_ptr(dst, ncomp, c0, s);
    T2 v[kPlanes];
#pragma unroll
    for (int k = 0; k < kPlanes; k++) v[k] = __ldg(from + k * kLane);
#pragma unroll
    for (int k = 0; k < kPlanes; k++) to[k * kLane] = v[k];
}

cudaError_t launch_shift(int prec, const Geom& g, int ncomp, void* dst, const void* src, int mu,
                         int sign, int subset, cudaStream_t st) {
    int n = subset == 0 ? g.V : g.Vh;
    dim3 grid((n + 255) / 256, ncomp / kPlanes);
    if (prec) shift_kernel<double2><<<grid, 256, 0, st>>>(g, ncomp, (double2*)dst, (const double2*)src, mu, sign, subset);
    else      shift_kernel<float2><<<grid, 256, 0, st>>>(g, ncomp, (float2*)dst, (const float2*)src, mu, sign, subset);
    g_launch_count++;
    return cudaGetLastError();
}

}  // namespace qdp
