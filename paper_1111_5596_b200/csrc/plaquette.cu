// plaquette.cu -- sum_x sum_{mu<nu} Re tr[U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag]
// fused with its global sum (def. 2).
//
// Per plane the thread forms A = U_mu(x) U_nu(x+mu) and B = U_nu(x) U_mu(x+nu) and
// takes Re tr(A B^dag) = sum_ij Re(A_ij conj(B_ij)): two 3x3 products and an
// 18-term dot product instead of three products and a trace (1404 FMA per site).
#include "internal.h"
#include "su3.cuh"

namespace qdp {

constexpr int kPlaqThreads = 128;

template <class T, int MU, int NU>
__device__ __forceinline__ T plaq_plane(const Geom& g, const Site& x, int s,
                                        const typename Vec2<T>::type* __restrict__ u, const Mat3<T>& Umu) {
    const size_t V = (size_t)g.V;
    const int s_pmu = site_step<MU, +1>(g, x).index(g);
    const int s_pnu = site_step<NU, +1>(g, x).index(g);
    Mat3<T> A = mul(Umu, ld_mat<T>(u, V, NU, s_pmu));
    Mat3<T> B = mul(ld_mat<T>(u, V, NU, s), ld_mat<T>(u, V, MU, s_pnu));
    return re_tr_mul_adj(A, B);
}

struct PlaqScale { double s[3]; };

template <class T>
__global__ void __launch_bounds__(kPlaqThreads) plaquette_kernel(Geom g, const typename Vec2<T>::type* __restrict__ u,
                                                                int subset, ReduceBuf rb, PlaqScale sc) {
    const int i = blockIdx.x * kPlaqThreads + threadIdx.x;
    double acc[3] = {0.0, 0.0, 0.0};   // all, spatial, temporal
    if (i < subset_count(g, subset)) {
        const int s = subset_index(g, subset, i);
        const Site x = site_from_index(g, s);
        const size_t V = (size_t)g.V;
        T sp = 0, tp = 0;
        {
            Mat3<T> U0 = ld_mat<T>(u, V, 0, s);
            sp += plaq_plane<T, 0, 1>(g, x, s, u, U0);
            sp += plaq_plane<T, 0, 2>(g, x, s, u, U0);
            tp += plaq_plane<T, 0, 3>(g, x, s, u, U0);
        }
        {
            Mat3<T> U1 = ld_mat<T>(u, V, 1, s);
            sp += plaq_plane<T, 1, 2>(g, x, s, u, U1);
            tp += plaq_plane<T, 1, 3>(g, x, s, u, U1);
        }
        {
            Mat3<T> U2 = ld_mat<T>(u, V, 2, s);
            tp += plaq_plane<T, 2, 3>(g, x, s, u, U2);
        }
        acc[1] = (double)sp;
        acc[2] = (double)tp;
        acc[0] = acc[1] + acc[2];
    }
    grid_reduce<3, kPlaqThreads>(acc, rb, sc.s);
}

cudaError_t launch_plaquette(int prec, const Geom& g, const void* u, int subset, const ReduceBuf& rb,
                             cudaStream_t st) {
    int n = subset == 0 ? g.V : g.Vh;
    int grid = (n + kPlaqThreads - 1) / kPlaqThreads;
    PlaqScale sc;
    sc.s[0] = 1.0 / (18.0 * (double)n);
    sc.s[1] = sc.s[2] = 1.0 / (9.0 * (double)n);
    if (prec) plaquette_kernel<double><<<grid, kPlaqThreads, 0, st>>>(g, (const double2*)u, subset, rb, sc);
    else      plaquette_kernel<float><<<grid, kPlaqThreads, 0, st>>>(g, (const float2*)u, subset, rb, sc);
    g_launch_count++;
    return cudaGetLastError();
}

}  // namespace qdp
