// ape.cu -- one APE smearing step: staple sum, blend, SU(3) reprojection, fused in
// one kernel (def. 3-4).  "Smearing" is the paper's
// first example of a non-kernel routine that dominates once the solver is on the
// GPU.
//
// One thread per site; the thread walks the smeared directions mu one after the other.  The
// mu loop is unrolled: rolled, ptxas rotates the prefetched matrices of the next direction
// through MOVs that wait for their loads (measured on C4 fp64: 0.83 ms rolled at 168
// registers, 0.78 ms unrolled at 255; a variant that shares K = U_mu(x+nu) U_nu(x+mu)^dag
// between the two upper staples of a plane needs 8 % fewer DFMA but two live staple sums,
// spills, and measured 0.82 ms; persistent warps measured 0.99 ms -- DESIGN.md section 5).
// Per mu the 2(|S|-1) staples are straight-line code with an explicit software pipeline:
// the third matrix of a staple is requested before its first product starts, and the
// first two matrices of the next staple (or, at the end, of the next mu) before its
// second product starts, so about one 3x3 product (108 DFMA) of work hides each
// request.  In fp64 the kernel is bound by the fp64 pipe, so the
// point of the pipeline is to keep that pipe fed from 8-12 resident warps per SM.
//
// Neighbour indices: the half-index offset of a step +-mu depends only on x_mu (and on
// x0's parity for mu = 0), so the offsets of x-nu+mu are the sum of the two one-step
// offsets (geom.cuh); eight ints per thread replace all coordinate arithmetic in the loop.
#include "internal.h"
#include "su3.cuh"

namespace qdp {

#ifndef APE_THREADS
#define APE_THREADS 128
#endif
constexpr int kApeThreads = APE_THREADS;

// A never-taken branch ptxas cannot predicate away: it ends the basic block.  The unrolled
// directions would otherwise merge into one block of ~5000 instructions in which ptxas hoists
// the loads of all directions to the top and spills 2-4 KB per thread (measured: 1.96 ms).
#define BLOCK_BOUNDARY(g) do { if ((g).V < 0) __trap(); } while (0)
#ifndef APE_MIN_BLOCKS_F32
#define APE_MIN_BLOCKS_F32 3
#endif
// fp64: 2 blocks of 128 threads per SM (255 registers, the software pipeline needs them);
// fp32: 3 blocks (168 registers; 4 blocks x 128 registers measured the same, 5 x 96 slower)
template <class T> struct ApeCfg { static constexpr int kMinBlocks = sizeof(T) == 8 ? 2 : APE_MIN_BLOCKS_F32; };

__device__ __forceinline__ int sel4(const int (&a)[4], int i) {
    return i == 0 ? a[0] : (i == 1 ? a[1] : (i == 2 ? a[2] : a[3]));
}

template <class T, bool FOURD>
__global__ void __launch_bounds__(kApeThreads, ApeCfg<T>::kMinBlocks)
ape_kernel(Geom g, typename Vec2<T>::type* __restrict__ out, const typename Vec2<T>::type* __restrict__ u,
           T alpha, int subset) {
    using T2 = typename Vec2<T>::type;
    constexpr int ND = FOURD ? 4 : 3;        // smeared directions
    constexpr int NS = 2 * (ND - 1);         // staples per link
    // fp32, 4-D: the products run on (re, im) register pairs (su3.cuh: *_pk; 0.85 -> 0.76 ms on 32^3 x 64)
    constexpr bool kPk = sizeof(T) == 4 && FOURD;
    const int i = blockIdx.x * kApeThreads + threadIdx.x;
    int p, h;
    if (i >= work_items(g, subset) || !work_site(g, subset, i, p, h)) return;
    const Site x = site_decode(g, p, h);
    const int sb = p * g.Vhp + h;            // this site
    const int ob = (1 - p) * g.Vhp + h;      // same half-index in the other parity
    int dp[4], dm[4];                        // half-index offsets of x+mu, x-mu
    dp[0] = site_step<0, +1>(g, x).h - h; dm[0] = site_step<0, -1>(g, x).h - h;
    dp[1] = site_step<1, +1>(g, x).h - h; dm[1] = site_step<1, -1>(g, x).h - h;
    dp[2] = site_step<2, +1>(g, x).h - h; dm[2] = site_step<2, -1>(g, x).h - h;
    dp[3] = site_step<3, +1>(g, x).h - h; dm[3] = site_step<3, -1>(g, x).h - h;

    if (!FOURD) {   // time links pass through unchanged (bit-exact)
        const T2* src = site_ptr(u, 36, 27, sb);
        T2* dst = site_ptr(out, 36, 27, sb);
        T2 t[9];
#pragma unroll
        for (int c = 0; c < 9; c++) t[c] = __ldg(src + c * kLane);
#pragma unroll
        for (int c = 0; c < 9; c++) dst[c * kLane] = t[c];
    }
    const T w_staple = alpha / T(NS), w_link = T(1) - alpha;

    // operands of staple k of direction mu (nu = mu+1+k/2 mod ND):
    //   upper (k even): A = U_nu(x),    B = U_mu(x+nu), C = U_nu(x+mu):    S += (A B) C^dag
    //   lower (k odd):  A = U_nu(x-nu), B = U_mu(x-nu), C = U_nu(x-nu+mu): S += (A^dag B) C
    auto ptrA = [&](int mu, int k) -> const T2* {
        int nu = mu + 1 + (k >> 1); if (nu >= ND) nu -= ND;
        return site_ptr(u, 36, nu * 9, (k & 1) ? ob + sel4(dm, nu) : sb);
    };
    auto ptrB = [&](int mu, int k) -> const T2* {
        int nu = mu + 1 + (k >> 1); if (nu >= ND) nu -= ND;
        return site_ptr(u, 36, mu * 9, ob + ((k & 1) ? sel4(dm, nu) : sel4(dp, nu)));
    };
    auto ptrC = [&](int mu, int k) -> const T2* {
        int nu = mu + 1 + (k >> 1); if (nu >= ND) nu -= ND;
        return site_ptr(u, 36, nu * 9, (k & 1) ? sb + sel4(dm, nu) + sel4(dp, mu) : ob + sel4(dp, mu));
    };

    Mat3<T> A = ld_mat_at<T>(ptrA(0, 0)), B = ld_mat_at<T>(ptrB(0, 0));
    // 4-D: the direction loop stays rolled.  Unrolled, the 24 staples and 4 projections are ~160 KB of straight-line
    // code, more than the instruction cache holds (32^3 x 64: fp64 2.56 ms unrolled, 1.43 ms unrolled by two,
    // 1.38 ms rolled; fp32 0.83 -> 0.76 ms).  The spatial step is faster unrolled (fp64 0.73 ms against 0.81 ms rolled).
    constexpr int kUnrollMu = FOURD ? 1 : ND;
#pragma unroll kUnrollMu
    for (int mu = 0; mu < ND; mu++) {
        Mat3<T> S = mat_zero<T>();
        Mat3<T> U;
#pragma unroll
        for (int k = 0; k < NS; k++) {
            Mat3<T> C = ld_mat_at<T>(ptrC(mu, k));
            Mat3<T> Tm;
            if constexpr (kPk) Tm = (k & 1) ? adj_mul_pk(A, B) : mul_pk(A, B);
            else               Tm = (k & 1) ? adj_mul(A, B) : mul(A, B);
            if (k + 1 < NS) {
                A = ld_mat_at<T>(ptrA(mu, k + 1));
                B = ld_mat_at<T>(ptrB(mu, k + 1));
            } else {
                U = ld_mat_at<T>(site_ptr(u, 36, mu * 9, sb));
            }
            if constexpr (kPk) { if (k & 1) mad_mul_pk(S, Tm, C); else mad_mul_adj_pk(S, Tm, C); }
            else               { if (k & 1) mad_mul(S, Tm, C); else mad_mul_adj(S, Tm, C); }
        }
        if (mu + 1 < ND) {   // first operands of the next direction, in flight during the projection
            A = ld_mat_at<T>(ptrA(mu + 1, 0));
            B = ld_mat_at<T>(ptrB(mu + 1, 0));
        }
        // (1-alpha) U + (alpha/n) S, then the projection: fp64 fields in fp64 (su3.cuh: staged closed
        // form), fp32 fields entirely in fp32 (closed form + one Newton-Schulz step, su3.cuh:
        // proj_su3_f32), so the fp32 kernel never touches the fp64 pipe.
        T2* o = site_ptr(out, 36, mu * 9, sb);
        Mat3<T> W;
        if constexpr (sizeof(T) == 8) {
            Mat3<double> Vd;
#pragma unroll
            for (int c = 0; c < 9; c++)
                Vd.e[c] = cx<double>(w_link * U.e[c].re + w_staple * S.e[c].re, w_link * U.e[c].im + w_staple * S.e[c].im);
            ProjScalars ps[1];
            proj_stage_a(Vd, ps[0]);
            // The block ends here, after the seeds: the scalar Newton chains and the final product of
            // this link then share a basic block with the staples of the next direction, and ptxas
            // fills the chains' dependency stalls with independent matrix work (0.757 -> 0.732 ms;
            // a boundary after the store instead keeps them apart).
            BLOCK_BOUNDARY(g);
            proj_stage_b<1>(ps);
            W = proj_stage_c(Vd, ps[0]);
        } else {
            Mat3<float> Vf;
#pragma unroll
            for (int c = 0; c < 9; c++)
                Vf.e[c] = cx<float>(w_link * U.e[c].re + w_staple * S.e[c].re, w_link * U.e[c].im + w_staple * S.e[c].im);
            W = proj_su3_f32(Vf);
            BLOCK_BOUNDARY(g);
        }
#pragma unroll
        for (int c = 0; c < 9; c++) {
            T2 v;
            v.x = W.e[c].re; v.y = W.e[c].im;
            o[c * kLane] = v;
        }
    }
}

template <class T>
static cudaError_t launch_ape_t(const Geom& g, void* out, const void* in, double alpha, int t_dir, int subset,
                                cudaStream_t st) {
    using T2 = typename Vec2<T>::type;
    int items = subset == 0 ? 2 * ((g.Vh + 31) & ~31) : g.Vh;
    dim3 grid((items + kApeThreads - 1) / kApeThreads);
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
