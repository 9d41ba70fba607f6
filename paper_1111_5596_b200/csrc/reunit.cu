// reunit.cu -- every 3x3 matrix of a field projected back to SU(3) (SURVEY.md 8(f) row f2:
// alternative projections).  method 0: Proj(V) = polar factor times exp(-i arg(det V)/3), the
// projection of the APE step made robust for general matrices (su3.cuh: proj_su3_general); method 1: Gram-Schmidt on rows 0, 1 and
// row 2 = conj(row 0 x row 1).  Site-local, so it may run in place.  One thread per (site, matrix):
// 144 B in, 144 B out (fp64), HBM-bound for Gram-Schmidt (~90 fp64 instructions per matrix).
// Arithmetic in fp64 for both field precisions.
#include "internal.h"
#include "su3.cuh"

namespace qdp {

__device__ __forceinline__ Mat3<double> gram_schmidt_su3(const Mat3<double>& V) {
    Mat3<double> R;
    double n0 = 0;
#pragma unroll
    for (int j = 0; j < 3; j++) n0 = fma(V.e[j].re, V.e[j].re, fma(V.e[j].im, V.e[j].im, n0));
    const double i0 = 1.0 / sqrt(n0);
#pragma unroll
    for (int j = 0; j < 3; j++) R.e[j] = cx<double>(V.e[j].re * i0, V.e[j].im * i0);
    Cx<double> dot = cx<double>(0, 0);                       // (row0 . v1) = sum conj(row0_j) v1_j
#pragma unroll
    for (int j = 0; j < 3; j++) cmad_conj_a(dot, R.e[j], V.e[3 + j]);
    double n1 = 0;
#pragma unroll
    for (int j = 0; j < 3; j++) {
        const Cx<double> t = dot * R.e[j];
        R.e[3 + j] = V.e[3 + j] - t;
        n1 = fma(R.e[3 + j].re, R.e[3 + j].re, fma(R.e[3 + j].im, R.e[3 + j].im, n1));
    }
    const double i1 = 1.0 / sqrt(n1);
#pragma unroll
    for (int j = 0; j < 3; j++) R.e[3 + j] = cx<double>(R.e[3 + j].re * i1, R.e[3 + j].im * i1);
#pragma unroll
    for (int j = 0; j < 3; j++) {
        const int a = (j + 1) % 3, b = (j + 2) % 3;
        R.e[6 + j] = conj(R.e[a] * R.e[3 + b] - R.e[b] * R.e[3 + a]);
    }
    return R;
}

template <class T, int METHOD>
__global__ void __launch_bounds__(256) reunit_kernel(Geom g, int ncomp, typename Vec2<T>::type* out,
                                                    const typename Vec2<T>::type* in, int subset) {
    using T2 = typename Vec2<T>::type;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= subset_count(g, subset)) return;
    const int s = subset_index(g, subset, i);
    const T2* p = site_ptr(in, ncomp, blockIdx.y * 9, s);
    Mat3<double> V;
#pragma unroll
    for (int c = 0; c < 9; c++) {
        const T2 v = p[c * kLane];
        V.e[c] = cx<double>((double)v.x, (double)v.y);
    }
    Mat3<double> W;
    if (METHOD == 0) {
        W = proj_su3_general(V);
    } else {
        W = gram_schmidt_su3(V);
    }
    T2* o = site_ptr(out, ncomp, blockIdx.y * 9, s);
#pragma unroll
    for (int c = 0; c < 9; c++) {
        T2 v;
        v.x = (T)W.e[c].re; v.y = (T)W.e[c].im;
        o[c * kLane] = v;
    }
}

cudaError_t launch_reunit(int prec, const Geom& g, int ncomp, void* out, const void* in, int method, int subset,
                          cudaStream_t st) {
    const int n = subset == 0 ? g.V : g.Vh;
    dim3 grid((n + 255) / 256, ncomp / 9);
    if (prec) {
        if (method == 0) reunit_kernel<double, 0><<<grid, 256, 0, st>>>(g, ncomp, (double2*)out, (const double2*)in, subset);
        else             reunit_kernel<double, 1><<<grid, 256, 0, st>>>(g, ncomp, (double2*)out, (const double2*)in, subset);
    } else {
        if (method == 0) reunit_kernel<float, 0><<<grid, 256, 0, st>>>(g, ncomp, (float2*)out, (const float2*)in, subset);
        else             reunit_kernel<float, 1><<<grid, 256, 0, st>>>(g, ncomp, (float2*)out, (const float2*)in, subset);
    }
    g_launch_count++;
    return cudaGetLastError();
}

}  // namespace qdp
