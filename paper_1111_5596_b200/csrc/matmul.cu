// matmul.cu -- one fused binary colour-matrix expression (first step):
//     dst(x) = opA(A(x)) * opB(B(x + sign*mu)),   op = identity or adjoint,   x in subset,
// the building block of QDP++ expressions like  m = u[mu] * shift(adj(u[nu]), FORWARD, mu)
// ("expressions that look like their mathematical counterparts"; here shift,
// adjoint and product are one kernel with no temporary, the paper's point).  An operand is one
// 3x3 matrix slot of a field: slot 0 of a colour matrix, slot mu of a gauge field.
// One thread per site: 2 x 144 B in, 144 B out (fp64), 108 FMA: HBM-bound.
#include "internal.h"
#include "su3.cuh"

namespace qdp {

template <class T, bool ADJ_A, bool ADJ_B>
__global__ void __launch_bounds__(256) matmul_kernel(Geom g, typename Vec2<T>::type* dst, int nd, int id,
                                                    const typename Vec2<T>::type* a, int na, int ia,
                                                    const typename Vec2<T>::type* b, int nb, int ib,
                                                    int mu, int sign, int subset) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= subset_count(g, subset)) return;
    const Site x = subset_site(g, subset, i);
    const int s = x.index(g);
    const int sn = mu < 0 ? s : site_step_rt(g, x, mu, sign).index(g);
    // plain loads: dst may be one of the operands' fields (another slot, or the same slot when unshifted)
    Mat3<T> A, B;
    const typename Vec2<T>::type* pa = site_ptr(a, na, ia * 9, s);
    const typename Vec2<T>::type* pb = site_ptr(b, nb, ib * 9, sn);
#pragma unroll
    for (int c = 0; c < 9; c++) {
        const typename Vec2<T>::type va = pa[c * kLane], vb = pb[c * kLane];
        A.e[c] = cx<T>(va.x, va.y);
        B.e[c] = cx<T>(vb.x, vb.y);
    }
    Mat3<T> R;
#pragma unroll
    for (int r = 0; r < 3; r++)
#pragma unroll
        for (int cc = 0; cc < 3; cc++) {
            Cx<T> acc = cx<T>(0, 0);
#pragma unroll
            for (int k = 0; k < 3; k++) {
                const Cx<T> ea = ADJ_A ? conj(A.e[k * 3 + r]) : A.e[r * 3 + k];
                const Cx<T> eb = ADJ_B ? conj(B.e[cc * 3 + k]) : B.e[k * 3 + cc];
                cmad(acc, ea, eb);
            }
            R.e[r * 3 + cc] = acc;
        }
    st_mat_at<T>(site_ptr(dst, nd, id * 9, s), R);
}

// chi(x) = opA(A(x)) psi(x + sign*mu): the colour matrix acts on the colour index of each of the four
// spin components.  chi must not be psi when mu >= 0 (checked by the caller).
template <class T, bool ADJ_A>
__global__ void __launch_bounds__(256) matvec_kernel(Geom g, typename Vec2<T>::type* chi,
                                                    const typename Vec2<T>::type* a, int na, int ia,
                                                    const typename Vec2<T>::type* psi, int mu, int sign, int subset) {
    using T2 = typename Vec2<T>::type;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= subset_count(g, subset)) return;
    const Site x = subset_site(g, subset, i);
    const int s = x.index(g);
    const int sn = mu < 0 ? s : site_step_rt(g, x, mu, sign).index(g);
    const T2* pa = site_ptr(a, na, ia * 9, s);
    const T2* pp = site_ptr(psi, 12, 0, sn);
    Mat3<T> A;
    Spinor<T> p, r;
#pragma unroll
    for (int c = 0; c < 9; c++) { const T2 v = pa[c * kLane]; A.e[c] = cx<T>(v.x, v.y); }
#pragma unroll
    for (int c = 0; c < 12; c++) { const T2 v = pp[c * kLane]; p.e[c] = cx<T>(v.x, v.y); }
#pragma unroll
    for (int sp = 0; sp < 4; sp++)
#pragma unroll
        for (int r_ = 0; r_ < 3; r_++) {
            Cx<T> acc = cx<T>(0, 0);
#pragma unroll
            for (int k = 0; k < 3; k++) cmad(acc, ADJ_A ? conj(A.e[k * 3 + r_]) : A.e[r_ * 3 + k], p.e[sp * 3 + k]);
            r.e[sp * 3 + r_] = acc;
        }
    T2* o = site_ptr(chi, 12, 0, s);
#pragma unroll
    for (int c = 0; c < 12; c++) { T2 v; v.x = r.e[c].re; v.y = r.e[c].im; o[c * kLane] = v; }
}

cudaError_t launch_matvec(int prec, const Geom& g, void* chi, const void* a, int na, int ia, bool adj_a, const void* psi,
                          int mu, int sign, int subset, cudaStream_t st) {
    const int n = subset == 0 ? g.V : g.Vh;
    const int grid = (n + 255) / 256;
    if (prec) {
        if (adj_a) matvec_kernel<double, true><<<grid, 256, 0, st>>>(g, (double2*)chi, (const double2*)a, na, ia, (const double2*)psi, mu, sign, subset);
        else       matvec_kernel<double, false><<<grid, 256, 0, st>>>(g, (double2*)chi, (const double2*)a, na, ia, (const double2*)psi, mu, sign, subset);
    } else {
        if (adj_a) matvec_kernel<float, true><<<grid, 256, 0, st>>>(g, (float2*)chi, (const float2*)a, na, ia, (const float2*)psi, mu, sign, subset);
        else       matvec_kernel<float, false><<<grid, 256, 0, st>>>(g, (float2*)chi, (const float2*)a, na, ia, (const float2*)psi, mu, sign, subset);
    }
    g_launch_count++;
    return cudaGetLastError();
}

template <class T>
static void matmul_dispatch(const Geom& g, void* dst, int nd, int id, const void* a, int na, int ia, bool adj_a,
                            const void* b, int nb, int ib, bool adj_b, int mu, int sign, int subset, cudaStream_t st) {
    using T2 = typename Vec2<T>::type;
    const int n = subset == 0 ? g.V : g.Vh;
    const int grid = (n + 255) / 256;
#define QDP_MM(AA, BB) matmul_kernel<T, AA, BB><<<grid, 256, 0, st>>>(g, (T2*)dst, nd, id, (const T2*)a, na, ia, \
                                                                      (const T2*)b, nb, ib, mu, sign, subset)
    if (adj_a) { if (adj_b) QDP_MM(true, true); else QDP_MM(true, false); }
    else       { if (adj_b) QDP_MM(false, true); else QDP_MM(false, false); }
#undef QDP_MM
}

cudaError_t launch_matmul(int prec, const Geom& g, void* dst, int nd, int id, const void* a, int na, int ia, bool adj_a,
                          const void* b, int nb, int ib, bool adj_b, int mu, int sign, int subset, cudaStream_t st) {
    if (prec) matmul_dispatch<double>(g, dst, nd, id, a, na, ia, adj_a, b, nb, ib, adj_b, mu, sign, subset, st);
    else      matmul_dispatch<float>(g, dst, nd, id, a, na, ia, adj_a, b, nb, ib, adj_b, mu, sign, subset, st);
    g_launch_count++;
    return cudaGetLastError();
}

}  // namespace qdp
