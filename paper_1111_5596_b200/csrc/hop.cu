// hop.cu -- chi(x) = sum_mu [ U_mu(x) psi(x+mu) + U_mu(x-mu)^dag psi(x-mu) ]   (def. 5)
// and the fused chi = a psi + b hop(psi) with optional fused norm2 (def. 6); with NDIR = 3 the
// time direction is left out: one step of Wuppertal / Gaussian quark smearing (qdp_smear_hop).
// (SURVEY.md 8(a) rows a7, a8.)  One kernel per expression, no lattice-sized
// temporaries -- the point of the paper's expression fusion.
//
// One thread per updated site.  Per direction a thread issues 2 x (9 + 12)
// independent 128-bit loads (fp64), all coalesced along the site index; the 8-fold
// reuse of each psi(y) and 2-fold reuse of each link is left to L1/L2.
#include "internal.h"
#include "su3.cuh"

namespace qdp {

constexpr int kHopThreads = 128;
#ifndef HOP_MIN_BLOCKS_F32
#define HOP_MIN_BLOCKS_F32 6
#endif
template <class T> struct HopCfg { static constexpr int kBlocks = sizeof(T) == 8 ? 3 : HOP_MIN_BLOCKS_F32; };

template <class T, int MU>
__device__ __forceinline__ void hop_dir(const Geom& g, const Site& x, int s,
                                        const typename Vec2<T>::type* __restrict__ u,
                                        const typename Vec2<T>::type* __restrict__ psi, Spinor<T>& acc) {
    {   // forward: U_mu(x) psi(x+mu)
        const int sf = site_step<MU, +1>(g, x).index(g);
        Mat3<T> U = ld_mat_at<T>(site_ptr(u, 36, MU * 9, s));
        Spinor<T> p = ld_spinor_at<T>(site_ptr(psi, 12, 0, sf));
#pragma unroll
        for (int sp = 0; sp < 4; sp++)
#pragma unroll
            for (int a = 0; a < 3; a++)
#pragma unroll
                for (int b = 0; b < 3; b++) cmad(acc.e[sp * 3 + a], U.e[a * 3 + b], p.e[sp * 3 + b]);
    }
    {   // backward: U_mu(x-mu)^dag psi(x-mu)
        const int sb = site_step<MU, -1>(g, x).index(g);
        Mat3<T> U = ld_mat_at<T>(site_ptr(u, 36, MU * 9, sb));
        Spinor<T> p = ld_spinor_at<T>(site_ptr(psi, 12, 0, sb));
#pragma unroll
        for (int sp = 0; sp < 4; sp++)
#pragma unroll
            for (int a = 0; a < 3; a++)
#pragma unroll
                for (int b = 0; b < 3; b++) cmad_conj_a(acc.e[sp * 3 + a], U.e[b * 3 + a], p.e[sp * 3 + b]);
    }
}

template <class T, bool AXPY, bool NORM, int NDIR>
__global__ void __launch_bounds__(kHopThreads, HopCfg<T>::kBlocks) hop_kernel(Geom g, typename Vec2<T>::type* __restrict__ chi,
                                                         const typename Vec2<T>::type* __restrict__ u,
                                                         const typename Vec2<T>::type* __restrict__ psi,
                                                         int subset, T a, T b, ReduceBuf rb) {
    const int i = blockIdx.x * kHopThreads + threadIdx.x;
    int p, h;
    const bool active = i < work_items(g, subset) && work_site(g, subset, i, p, h);
    double n2[1] = {0.0};
    if (active) {
        const Site x = site_decode(g, p, h);
        const int s = x.index(g);
        Spinor<T> acc;
#pragma unroll
        for (int c = 0; c < 12; c++) acc.e[c] = cx<T>(0, 0);
        hop_dir<T, 0>(g, x, s, u, psi, acc);
        hop_dir<T, 1>(g, x, s, u, psi, acc);
        hop_dir<T, 2>(g, x, s, u, psi, acc);
        if (NDIR == 4) hop_dir<T, 3>(g, x, s, u, psi, acc);
        if (AXPY) {
            Spinor<T> p = ld_spinor_at<T>(site_ptr(psi, 12, 0, s));
#pragma unroll
            for (int c = 0; c < 12; c++) {
                // a*psi + b*hop: two roundings per part, like the definition
                acc.e[c].re = a * p.e[c].re + b * acc.e[c].re;
                acc.e[c].im = a * p.e[c].im + b * acc.e[c].im;
            }
        }
        typename Vec2<T>::type* o = site_ptr(chi, 12, 0, s);
#pragma unroll
        for (int c = 0; c < 12; c++) {
            typename Vec2<T>::type v;
            v.x = acc.e[c].re; v.y = acc.e[c].im;
            o[c * kLane] = v;
            if (NORM) n2[0] += (double)acc.e[c].re * (double)acc.e[c].re + (double)acc.e[c].im * (double)acc.e[c].im;
        }
    }
    if (NORM) warp_grid_reduce<1>(n2, rb, nullptr);
}

template <class T>
static cudaError_t launch_hop_t(const Geom& g, void* chi, const void* u, const void* psi, int subset,
                                bool axpy, double a, double b, bool want_norm2, const ReduceBuf& rb,
                                cudaStream_t st, int ndir) {
    using T2 = typename Vec2<T>::type;
    int n = subset == 0 ? 2 * g.Vhp : g.Vh;
    int grid = (n + kHopThreads - 1) / kHopThreads;
    T2* c = (T2*)chi; const T2* uu = (const T2*)u; const T2* p = (const T2*)psi;
    if (ndir == 3) {   // the smearing step is always the axpy form
        if (!want_norm2) hop_kernel<T, true, false, 3><<<grid, kHopThreads, 0, st>>>(g, c, uu, p, subset, (T)a, (T)b, rb);
        else             hop_kernel<T, true, true, 3><<<grid, kHopThreads, 0, st>>>(g, c, uu, p, subset, (T)a, (T)b, rb);
    }
    else if (!axpy)       hop_kernel<T, false, false, 4><<<grid, kHopThreads, 0, st>>>(g, c, uu, p, subset, (T)a, (T)b, rb);
    else if (!want_norm2) hop_kernel<T, true, false, 4><<<grid, kHopThreads, 0, st>>>(g, c, uu, p, subset, (T)a, (T)b, rb);
    else                  hop_kernel<T, true, true, 4><<<grid, kHopThreads, 0, st>>>(g, c, uu, p, subset, (T)a, (T)b, rb);
    g_launch_count++;
    return cudaGetLastError();
}

cudaError_t launch_hop(int prec, const Geom& g, void* chi, const void* u, const void* psi, int subset,
                       bool axpy, double a, double b, bool want_norm2, const ReduceBuf& rb, cudaStream_t st,
                       int ndir) {
    return prec ? launch_hop_t<double>(g, chi, u, psi, subset, axpy, a, b, want_norm2, rb, st, ndir)
                : launch_hop_t<float>(g, chi, u, psi, subset, axpy, a, b, want_norm2, rb, st, ndir);
}

}  // namespace qdp
