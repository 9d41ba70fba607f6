// ape.cu -- one APE smearing step: staple sum, blend, SU(3) reprojection, fused in
// one kernel (def. 3-4).  "Smearing" is the paper's
// first example of a non-kernel routine that dominates once the solver is on the
// GPU.
//
// One thread per (site, mu).  A 128-thread block is 4 warps = the 4 directions of one
// group of 32 consecutive half-indices; consecutive blocks alternate parity over the
// same run (full lattice), so all the links a neighbourhood needs are touched by
// neighbouring blocks at one time and come from DRAM once.  With t_dir = 3 the mu = 3 warps
// copy U_3 through unchanged (bit-exact).
#include "internal.h"
#include "su3.cuh"

namespace qdp {

constexpr int kApeThreads = 128;

// S += U_nu(x) U_mu(x+nu) U_nu(x+mu)^dag + U_nu(x-nu)^dag U_mu(x-nu) U_nu(x-nu+mu)
// mu, nu are run-time values: one copy of the matrix code serves every (mu, nu) pair,
// which keeps the kernel small enough to stay in the instruction cache while the four
// mu-warps of a block run different directions.
template <class T>
__device__ __forceinline__ void add_staples(const Geom& g, const Site& x, int s, int mu, int nu,
                                            const typename Vec2<T>::type* __restrict__ u, Mat3<T>& S) {
    const size_t V = (size_t)g.V;
    {
        const int s_pnu = site_step_rt(g, x, nu, +1).index(g);
        const int s_pmu = site_step_rt(g, x, mu, +1).index(g);
        Mat3<T> t = mul(ld_mat<T>(u, V, nu, s), ld_mat<T>(u, V, mu, s_pnu));
        mad_mul_adj(S, t, ld_mat<T>(u, V, nu, s_pmu));
    }
    {
        const Site xm = site_step_rt(g, x, nu, -1);
        const int s_mnu = xm.index(g);
        const int s_mnu_pmu = site_step_rt(g, xm, mu, +1).index(g);
        Mat3<T> t = adj_mul(ld_mat<T>(u, V, nu, s_mnu), ld_mat<T>(u, V, mu, s_mnu));
        mad_mul(S, t, ld_mat<T>(u, V, nu, s_mnu_pmu));
    }
}

#ifndef APE_MIN_BLOCKS
#define APE_MIN_BLOCKS 4
#endif
template <class T, bool FOURD>
__global__ void __launch_bounds__(kApeThreads, APE_MIN_BLOCKS) ape_kernel(Geom g, typename Vec2<T>::type* __restrict__ out,
                                                         const typename Vec2<T>::type* __restrict__ u,
                                                         T alpha, int subset) {
    const int mu = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int i = blockIdx.x * 32 + lane;    // site work item
    int p, h;
    if (i >= work_items(g, subset) || !work_site(g, subset, i, p, h)) return;
    const Site x = site_decode(g, p, h);
    const int s = x.index(g);
    const size_t V = (size_t)g.V;
    if (!FOURD && mu == 3) {   // time links pass through unchanged
#pragma unroll
        for (int c = 27; c < 36; c++) out[(size_t)c * V + s] = __ldg(u + (size_t)c * V + s);
        return;
    }
    Mat3<T> S = mat_zero<T>();
    const int ndir = FOURD ? 4 : 3;
#pragma unroll 1
    for (int nu = 0; nu < ndir; nu++) {
        if (nu == mu) continue;
        add_staples<T>(g, x, s, mu, nu, u, S);
    }
    const T w_staple = alpha / T(FOURD ? 6 : 4), w_link = T(1) - alpha;
    Mat3<T> U = ld_mat<T>(u, V, mu, s);
#pragma unroll
    for (int i2 = 0; i2 < 9; i2++) {
        // (1-alpha) U + (alpha/n) S
        U.e[i2].re = w_link * U.e[i2].re + w_staple * S.e[i2].re;
        U.e[i2].im = w_link * U.e[i2].im + w_staple * S.e[i2].im;
    }
    // The projection always runs in fp64: for fp32 fields the closed-form eigenvalues
    // of an ill-conditioned V^dag V (hot links: cond ~ 100) would lose ~2e-5 in fp32,
    // the whole fp32 error budget; fp64 is half the fp32 rate on B200, so this is cheap.
    Mat3<double> Vd;
#pragma unroll
    for (int i2 = 0; i2 < 9; i2++) Vd.e[i2] = cx<double>((double)U.e[i2].re, (double)U.e[i2].im);
    Mat3<double> Pd = proj_su3<double>(Vd);
#pragma unroll
    for (int i2 = 0; i2 < 9; i2++) U.e[i2] = cx<T>((T)Pd.e[i2].re, (T)Pd.e[i2].im);
    st_mat<T>(out, V, mu, s, U);
}

template <class T>
static cudaError_t launch_ape_t(const Geom& g, void* out, const void* in, double alpha, int t_dir, int subset,
                                cudaStream_t st) {
    using T2 = typename Vec2<T>::type;
    int items = subset == 0 ? 2 * ((g.Vh + 31) & ~31) : g.Vh;
    dim3 grid((items + 31) / 32);
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
