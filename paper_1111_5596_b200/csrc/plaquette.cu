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

// Re tr P_{mu nu}(x); mu, nu run-time so that one copy of the matrix code serves all
// six planes (small kernel, modest register count).
template <class T>
__device__ __forceinline__ T plaq_plane(const Geom& g, const Site& x, int s, int mu, int nu,
                                        const typename Vec2<T>::type* __restrict__ u) {
    const size_t V = (size_t)g.V;
    const int s_pmu = site_step_rt(g, x, mu, +1).index(g);
    const int s_pnu = site_step_rt(g, x, nu, +1).index(g);
    Mat3<T> A = mul(ld_mat<T>(u, V, mu, s), ld_mat<T>(u, V, nu, s_pmu));
    Mat3<T> B = mul(ld_mat<T>(u, V, nu, s), ld_mat<T>(u, V, mu, s_pnu));
    return re_tr_mul_adj(A, B);
}

struct PlaqScale { double s[3]; };

#ifndef PLAQ_MIN_BLOCKS
#define PLAQ_MIN_BLOCKS 3
#endif
#ifndef PLAQ_UNROLL
#define PLAQ_UNROLL 1
#endif
constexpr int kPlaqUnroll = PLAQ_UNROLL;
template <class T>
__global__ void __launch_bounds__(kPlaqThreads, PLAQ_MIN_BLOCKS) plaquette_kernel(Geom g, const typename Vec2<T>::type* __restrict__ u,
                                                                int subset, ReduceBuf rb, PlaqScale sc) {
    const int i = blockIdx.x * kPlaqThreads + threadIdx.x;
    double acc[3] = {0.0, 0.0, 0.0};   // all, spatial, temporal
    int p, h;
    if (i < work_items(g, subset) && work_site(g, subset, i, p, h)) {
        const Site x = site_decode(g, p, h);
        const int s = x.index(g);
        T sp = 0, tp = 0;
#pragma unroll kPlaqUnroll
        for (int pl = 0; pl < 6; pl++) {
            // planes (0,1) (0,2) (1,2) (0,3) (1,3) (2,3): the first three are spatial
            const int mu = pl < 3 ? (pl == 2) : pl - 3;
            const int nu = pl < 3 ? (pl == 0 ? 1 : 2) : 3;
            const T v = plaq_plane<T>(g, x, s, mu, nu, u);
            if (pl < 3) sp += v; else tp += v;
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
    int items = subset == 0 ? 2 * ((g.Vh + 31) & ~31) : g.Vh;
    int grid = (items + kPlaqThreads - 1) / kPlaqThreads;
    PlaqScale sc;
    sc.s[0] = 1.0 / (18.0 * (double)n);
    sc.s[1] = sc.s[2] = 1.0 / (9.0 * (double)n);
    if (prec) plaquette_kernel<double><<<grid, kPlaqThreads, 0, st>>>(g, (const double2*)u, subset, rb, sc);
    else      plaquette_kernel<float><<<grid, kPlaqThreads, 0, st>>>(g, (const float2*)u, subset, rb, sc);
    g_launch_count++;
    return cudaGetLastError();
}

}  // namespace qdp
