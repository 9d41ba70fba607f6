// ape.cu -- one APE smearing step: staple sum, blend, SU(3) reprojection, fused in
// one kernel (def. 3-4).  "Smearing" is the paper's
// first example of a non-kernel routine that dominates once the solver is on the
// GPU.
//
// One thread per (site, mu); blockIdx.y = mu.  With t_dir = 3 the y = 3 slice copies
// U_3 through unchanged (bit-exact).
#include "internal.h"
#include "su3.cuh"

namespace qdp {

constexpr int kApeThreads = 128;

// S += U_nu(x) U_mu(x+nu) U_nu(x+mu)^dag + U_nu(x-nu)^dag U_mu(x-nu) U_nu(x-nu+mu)
template <class T, int MU, int NU>
__device__ __forceinline__ void add_staples(const Geom& g, const Site& x, int s,
                                            const typename Vec2<T>::type* __restrict__ u, Mat3<T>& S) {
    const size_t V = (size_t)g.V;
    {
        const int s_pnu = site_step<NU, +1>(g, x).index(g);
        const int s_pmu = site_step<MU, +1>(g, x).index(g);
        Mat3<T> t = mul(ld_mat<T>(u, V, NU, s), ld_mat<T>(u, V, MU, s_pnu));
        mad_mul_adj(S, t, ld_mat<T>(u, V, NU, s_pmu));
    }
    {
        const Site xm = site_step<NU, -1>(g, x);
        const int s_mnu = xm.index(g);
        const int s_mnu_pmu = site_step<MU, +1>(g, xm).index(g);
        Mat3<T> t = adj_mul(ld_mat<T>(u, V, NU, s_mnu), ld_mat<T>(u, V, MU, s_mnu));
        mad_mul(S, t, ld_mat<T>(u, V, NU, s_mnu_pmu));
    }
}

template <class T, int MU, bool FOURD>
__device__ __forceinline__ void ape_link(const Geom& g, const Site& x, int s,
                                         typename Vec2<T>::type* __restrict__ out,
                                         const typename Vec2<T>::type* __restrict__ u, T alpha) {
    const size_t V = (size_t)g.V;
    Mat3<T> S = mat_zero<T>();
    if (MU != 0) add_staples<T, MU, 0>(g, x, s, u, S);
    if (MU != 1) add_staples<T, MU, 1>(g, x, s, u, S);
    if (MU != 2) add_staples<T, MU, 2>(g, x, s, u, S);
    if (FOURD && MU != 3) add_staples<T, MU, 3>(g, x, s, u, S);
    const T w_staple = alpha / T(FOURD ? 6 : 4), w_link = T(1) - alpha;
    Mat3<T> U = ld_mat<T>(u, V, MU, s);
#pragma unroll
    for (int i = 0; i < 9; i++) {
        // (1-alpha) U + (alpha/n) S
        U.e[i].re = w_link * U.e[i].re + w_staple * S.e[i].re;
        U.e[i].im = w_link * U.e[i].im + w_staple * S.e[i].im;
    }
    // The projection always runs in fp64: for fp32 fields the closed-form eigenvalues
    // of an ill-conditioned V^dag V (hot links: cond ~ 100) would lose ~2e-5 in fp32,
    // the whole fp32 error budget; fp64 is half the fp32 rate on B200, so this is cheap.
    Mat3<double> Vd;
#pragma unroll
    for (int i = 0; i < 9; i++) Vd.e[i] = cx<double>((double)U.e[i].re, (double)U.e[i].im);
    Mat3<double> Pd = proj_su3<double>(Vd);
#pragma unroll
    for (int i = 0; i < 9; i++) U.e[i] = cx<T>((T)Pd.e[i].re, (T)Pd.e[i].im);
    st_mat<T>(out, V, MU, s, U);
}

template <class T, bool FOURD>
__global__ void __launch_bounds__(kApeThreads) ape_kernel(Geom g, typename Vec2<T>::type* __restrict__ out,
                                                         const typename Vec2<T>::type* __restrict__ u,
                                                         T alpha, int subset) {
    const int i = blockIdx.x * kApeThreads + threadIdx.x;
    if (i >= subset_count(g, subset)) return;
    const int s = subset_index(g, subset, i);
    const Site x = site_from_index(g, s);
    switch (blockIdx.y) {
        case 0: ape_link<T, 0, FOURD>(g, x, s, out, u, alpha); break;
        case 1: ape_link<T, 1, FOURD>(g, x, s, out, u, alpha); break;
        case 2: ape_link<T, 2, FOURD>(g, x, s, out, u, alpha); break;
        default:
            if (FOURD) {
                ape_link<T, 3, FOURD>(g, x, s, out, u, alpha);
            } else {   // time links pass through unchanged
                const size_t V = (size_t)g.V;
#pragma unroll
                for (int c = 27; c < 36; c++) out[(size_t)c * V + s] = __ldg(u + (size_t)c * V + s);
            }
    }
}

template <class T>
static cudaError_t launch_ape_t(const Geom& g, void* out, const void* in, double alpha, int t_dir, int subset,
                                cudaStream_t st) {
    using T2 = typename Vec2<T>::type;
    int n = subset == 0 ? g.V : g.Vh;
    dim3 grid((n + kApeThreads - 1) / kApeThreads, 4);
    if (t_dir == 3) ape_kernel<T, false><<<grid, kApeThreads, 0, st>>>(g, (T2*)out, (const T2*)in, (T)alpha, subset);
    else            ape_kernel<T, true><<<grid, kApeThreads, 0, st>>>(g, (T2*)out, (const T2*)in, (T)alpha, subset);
    g_launch_count++;
    return cudaGetLastError();
}

cudaError_t launch_ape(int prec, const Geom& g, void* u_out, const void* u_in, double alpha, int t_dir,
                       int subset, cudaStream_t st) {
    return prec ? launch_ape_t<double>(g, u_out, u_in, alpha, t_dir, subset, st)
                : launch_ape_t<float>(g, u_out, u_in, alpha, t_dir, subset, st);
}

}  // namespace qdp
