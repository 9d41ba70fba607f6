// reunit.cu -- every 3x3 matrix of a field projected back to SU(3) (SURVEY.md 8(f) row f2:
// alternative projections).  method 0: Proj(V) = polar factor times exp(-i arg(det V)/3), the
// projection of the APE step made robust for general matrices (su3.cuh: proj_su3_general); method 1: Gram-Schmidt on rows 0, 1 and
// row 2 = conj(row 0 x row 1); method 2: iterative max-Re-tr (Cabibbo-Marinari) sweeps from the Gram-Schmidt start.  Site-local, so it may run in place.  One thread per (site, matrix):
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

// One Cabibbo-Marinari update for the SU(2) subgroup acting on rows (I, J): maximises Re tr(X V^dag) over it exactly.
// Only the 2x2 block of M = X V^dag in rows/columns (I, J) is needed (12 complex multiply-adds).  Same formulas and
// order as the definition in include/qdp_b200.h (qdp_project_max_retr).
template <int I, int J>
__device__ __forceinline__ void max_retr_update(Mat3<double>& X, const Mat3<double>& V) {
    Cx<double> m00 = cx<double>(0, 0), m01 = m00, m10 = m00, m11 = m00;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        cmad_conj_b(m00, X.e[I * 3 + c], V.e[I * 3 + c]);
        cmad_conj_b(m01, X.e[I * 3 + c], V.e[J * 3 + c]);
        cmad_conj_b(m10, X.e[J * 3 + c], V.e[I * 3 + c]);
        cmad_conj_b(m11, X.e[J * 3 + c], V.e[J * 3 + c]);
    }
    double r0 = m00.re + m11.re, r1 = -(m01.im + m10.im), r2 = -(m01.re - m10.re), r3 = -(m00.im - m11.im);
    const double n2 = r0 * r0 + r1 * r1 + r2 * r2 + r3 * r3;
    const double inv = n2 > 0.0 ? 1.0 / sqrt(n2) : 0.0;
    if (n2 > 0.0) { r0 *= inv; r1 *= inv; r2 *= inv; r3 *= inv; } else { r0 = 1.0; r1 = r2 = r3 = 0.0; }
    const Cx<double> a00 = cx<double>(r0, r3), a01 = cx<double>(r2, r1), a10 = cx<double>(-r2, r1), a11 = cx<double>(r0, -r3);
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const Cx<double> xi = X.e[I * 3 + c], xj = X.e[J * 3 + c];
        X.e[I * 3 + c] = a00 * xi + a01 * xj;
        X.e[J * 3 + c] = a10 * xi + a11 * xj;
    }
}

template <class T, int METHOD>
__global__ void __launch_bounds__(256) reunit_kernel(Geom g, int ncomp, typename Vec2<T>::type* out,
                                                    const typename Vec2<T>::type* in, int subset, int iters) {
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
        if (METHOD == 2)      // iterative max-Re-tr projection: X_0 = Gram-Schmidt(V), then sweeps over (0,1), (1,2), (0,2)
            for (int it = 0; it < iters; it++) {
                max_retr_update<0, 1>(W, V);
                max_retr_update<1, 2>(W, V);
                max_retr_update<0, 2>(W, V);
            }
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
                          cudaStream_t st, int iters) {
    const int n = subset == 0 ? g.V : g.Vh;
    dim3 grid((n + 255) / 256, ncomp / 9);
    if (prec) {
        if (method == 0)      reunit_kernel<double, 0><<<grid, 256, 0, st>>>(g, ncomp, (double2*)out, (const double2*)in, subset, 0);
        else if (method == 1) reunit_kernel<double, 1><<<grid, 256, 0, st>>>(g, ncomp, (double2*)out, (const double2*)in, subset, 0);
        else                  reunit_kernel<double, 2><<<grid, 256, 0, st>>>(g, ncomp, (double2*)out, (const double2*)in, subset, iters);
    } else {
        if (method == 0)      reunit_kernel<float, 0><<<grid, 256, 0, st>>>(g, ncomp, (float2*)out, (const float2*)in, subset, 0);
        else if (method == 1) reunit_kernel<float, 1><<<grid, 256, 0, st>>>(g, ncomp, (float2*)out, (const float2*)in, subset, 0);
        else                  reunit_kernel<float, 2><<<grid, 256, 0, st>>>(g, ncomp, (float2*)out, (const float2*)in, subset, iters);
    }
    g_launch_count++;
    return cudaGetLastError();
}

}  // namespace qdp
