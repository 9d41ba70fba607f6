// plaquette.cu -- sum_x sum_{mu<nu} Re tr[U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag]
// fused with its global sum (def. 2).
//
// Per plane the thread forms P = U_mu(x) U_nu(x+mu) and Q = U_nu(x) U_mu(x+nu) and
// takes Re tr(P Q^dag) = sum_ij Re(P_ij conj(Q_ij)): two 3x3 products and an
// 18-term dot product instead of three products and a trace (1404 FMA per site); Q is
// never materialised, each entry goes straight into the dot product.
//
// One thread per site, the six planes fully unrolled (a rolled loop makes ptxas rotate the
// prefetched matrices through MOVs that wait for the loads: measured 0.58 -> 0.42 ms on C4)
// with an explicit software pipeline: the operands of Q are requested before P is computed
// and the operands of the next plane's P before Q is computed, so one 3x3 product (108
// DFMA) of work covers each request.  Neighbour indices are four precomputed half-index
// offsets.  Warps are persistent (see the kernel) so the block reduction runs once.
#include "internal.h"
#include "su3.cuh"

namespace qdp {

#ifndef PLAQ_THREADS
#define PLAQ_THREADS 128
#endif
#ifndef PLAQ_MIN_BLOCKS
#define PLAQ_MIN_BLOCKS 2
#endif
#ifndef PLAQ_MIN_BLOCKS_F32
#define PLAQ_MIN_BLOCKS_F32 4
#endif
// resident blocks per SM = persistent blocks per SM: fp64 2 x 128 threads at 254 registers, fp32 half the registers
template <class T> struct PlaqCfg { static constexpr int kBlocks = sizeof(T) == 8 ? PLAQ_MIN_BLOCKS : PLAQ_MIN_BLOCKS_F32; };
constexpr int kPlaqThreads = PLAQ_THREADS;
#ifndef PLAQ_UNROLL
#define PLAQ_UNROLL 6
#endif
constexpr int kPlaqUnroll = PLAQ_UNROLL;

struct PlaqScale { double s[3]; };

// sum_ij Re(P_ij conj((A B)_ij))
template <class T>
__device__ __forceinline__ T re_tr_p_adj_ab(const Mat3<T>& P, const Mat3<T>& a, const Mat3<T>& b) {
    T s0 = 0, s1 = 0, s2 = 0;   // three chains (one per row) keep the fp64 pipe's latency covered
#pragma unroll
    for (int i = 0; i < 3; i++) {
        T acc = 0;
#pragma unroll
        for (int j = 0; j < 3; j++) {
            Cx<T> q = a.e[i * 3] * b.e[j];
            cmad(q, a.e[i * 3 + 1], b.e[3 + j]);
            cmad(q, a.e[i * 3 + 2], b.e[6 + j]);
            acc = fma(P.e[i * 3 + j].re, q.re, acc);
            acc = fma(P.e[i * 3 + j].im, q.im, acc);
        }
        if (i == 0) s0 = acc; else if (i == 1) s1 = acc; else s2 = acc;
    }
    return s0 + s1 + s2;
}

template <class T>
__global__ void __launch_bounds__(kPlaqThreads, PlaqCfg<T>::kBlocks)
plaquette_kernel(Geom g, const typename Vec2<T>::type* __restrict__ u, int subset, ReduceBuf rb, PlaqScale sc) {
    using T2 = typename Vec2<T>::type;
    // Persistent warps: warp w of the grid takes the 32-site work items w, w + W, w + 2W, ...
    // (W = warps in the grid), so at any time the resident warps sweep one contiguous window
    // of the lattice and the block-level reduction runs once per block, not once per 128 sites.
    const int lane = threadIdx.x & 31;
    const int nwarps = gridDim.x * (kPlaqThreads / 32);
    const int nitems = (work_items(g, subset) + 31) >> 5;   // 32-site items (the last one may be ragged)
    double acc[3] = {0.0, 0.0, 0.0};   // all, spatial, temporal
    for (int wi = blockIdx.x * (kPlaqThreads / 32) + (threadIdx.x >> 5); wi < nitems; wi += nwarps) {
        const int i = wi * 32 + lane;
        int p, h;
        const bool live = i < work_items(g, subset) && work_site(g, subset, i, p, h);
        if (!live) continue;
        const Site x = site_decode(g, p, h);
        const int sb = p * g.Vhp + h;            // this site
        const int ob = (1 - p) * g.Vhp + h;      // same half-index in the other parity
        int dp[4];                               // half-index offsets of x+mu
        dp[0] = site_step<0, +1>(g, x).h - h;
        dp[1] = site_step<1, +1>(g, x).h - h;
        dp[2] = site_step<2, +1>(g, x).h - h;
        dp[3] = site_step<3, +1>(g, x).h - h;
        auto sel = [&](int d) { return d == 0 ? dp[0] : (d == 1 ? dp[1] : (d == 2 ? dp[2] : dp[3])); };
        // planes (0,1) (0,2) (1,2) (0,3) (1,3) (2,3): the first three are spatial
        auto plane_mu = [](int pl) { return pl < 3 ? (pl == 2) : pl - 3; };
        auto plane_nu = [](int pl) { return pl < 3 ? (pl == 0 ? 1 : 2) : 3; };
        const T2* here = site_ptr(u, 36, 0, sb);
        T sp = 0, tp = 0;
        Mat3<T> A = ld_mat_at<T>(here + plane_mu(0) * 9 * kLane);
        Mat3<T> B = ld_mat_at<T>(site_ptr(u, 36, plane_nu(0) * 9, ob + sel(plane_mu(0))));
#pragma unroll kPlaqUnroll
        for (int pl = 0; pl < 6; pl++) {
            const int mu = plane_mu(pl), nu = plane_nu(pl);
            Mat3<T> A2 = ld_mat_at<T>(here + nu * 9 * kLane);                        // U_nu(x)
            Mat3<T> B2 = ld_mat_at<T>(site_ptr(u, 36, mu * 9, ob + sel(nu)));        // U_mu(x+nu)
            Mat3<T> P = mul(A, B);                                                   // U_mu(x) U_nu(x+mu)
            if (pl + 1 < 6) {
                const int mu1 = plane_mu(pl + 1), nu1 = plane_nu(pl + 1);
                A = ld_mat_at<T>(here + mu1 * 9 * kLane);
                B = ld_mat_at<T>(site_ptr(u, 36, nu1 * 9, ob + sel(mu1)));
            }
            const T v = re_tr_p_adj_ab(P, A2, B2);
            if (pl < 3) sp += v; else tp += v;
            // A never-taken branch ptxas cannot predicate away ends the basic block between the
            // spatial and the temporal planes: measured 0.347 -> 0.332 ms (one block of 1900
            // instructions schedules worse than two; boundaries elsewhere gain nothing).
            if (pl == 2 && g.V < 0) __trap();
        }
        acc[1] += (double)sp;
        acc[2] += (double)tp;
    }
    acc[0] = acc[1] + acc[2];
    warp_grid_reduce<3>(acc, rb, sc.s);
}


cudaError_t launch_plaquette(int prec, const Geom& g, const void* u, int subset, const ReduceBuf& rb,
                             cudaStream_t st) {
    int n = subset == 0 ? g.V : g.Vh;
    int items = subset == 0 ? 2 * g.Vhp : g.Vh;
    int grid = (items + kPlaqThreads - 1) / kPlaqThreads;
    const int sms = device_sm_count();
#ifndef QDP_NO_TMA_PLAQUETTE
    if (plaquette_tma_applicable(g, subset)) return launch_plaquette_tma(prec, g, u, rb, sms, st);
#endif
    const int per_sm = prec ? PlaqCfg<double>::kBlocks : PlaqCfg<float>::kBlocks;
    if (grid > sms * per_sm) grid = sms * per_sm;
    PlaqScale sc;
    sc.s[0] = 1.0 / (18.0 * (double)n);
    sc.s[1] = sc.s[2] = 1.0 / (9.0 * (double)n);
    if (prec) plaquette_kernel<double><<<grid, kPlaqThreads, 0, st>>>(g, (const double2*)u, subset, rb, sc);
    else      plaquette_kernel<float><<<grid, kPlaqThreads, 0, st>>>(g, (const float2*)u, subset, rb, sc);
    g_launch_count++;
    return cudaGetLastError();
}

}  // namespace qdp
