// baryon.cu -- the baryon building block of the hadron-spectrum stage (PAPER.md:106, 110:
// "hadron spectrum (mesonic and baryonic)"): three quark fields contracted to a colour singlet with eps_{abc}, a
// diquark spin matrix Gamma(n) between the first two, eps_{a'b'c'} over the source colours, summed per time-slice:
//   out[t][g] = sum_{x3 = t} sum_{(a'b'c')} eps_{a'b'c'} sum_{abc} eps_{abc} [q1[a']^T_a Gamma q2[b']_b](x) q3[c']_{g c}(x).
// One thread per site of a time-slice (the half-indices of a slice are one run [t s3, (t+1) s3) per parity for every
// lattice), gridDim.y = L3 slices x kBtBlocks blocks; per source permutation the thread forms the 3x3 diquark
// M_ab = sum_al q1_{al a} (Gamma q2)_{al b}, antisymmetrises it (v_c = eps_{abc} M_ab) and accumulates v_c q3_{g c}.
// Gamma is a phased permutation of the spin index, applied while q2 is loaded.  All nine fields are read in one
// pass (fused: six separate single-triple calls would stream each field twice): 108 complex per site, HBM-bound.
// fp64 accumulation, one partial per block, summed in block order by the finish kernel (deterministic).
#include "internal.h"
#include "su3.cuh"

namespace qdp {

constexpr int kBtBlocks = 16, kBtThreads = 256;

struct BaryonArgs { const void* q[3][3]; };   // [quark][source colour]

template <class T>
__device__ __forceinline__ Cx<T> mul_i_pow(Cx<T> v, int k) {     // i^k v
    switch (k & 3) {
        case 0: return v;
        case 1: return cx<T>(-v.im, v.re);
        case 2: return cx<T>(-v.re, -v.im);
        default: return cx<T>(v.im, -v.re);
    }
}

template <class T, int NSRC>
__global__ void __launch_bounds__(kBtThreads) baryon_ts_kernel(Geom g, BaryonArgs args, SpinMatrix gm, int subset,
                                                              double* __restrict__ partials) {
    using T2 = typename Vec2<T>::type;
    __shared__ double sm[8][kBtThreads / 32];
    const int t = blockIdx.y;
    double acc[8];
#pragma unroll
    for (int i = 0; i < 8; i++) acc[i] = 0.0;
    constexpr int NPERM = NSRC == 3 ? 6 : 1;
    for (int p = (subset == 2 ? 1 : 0); p <= (subset == 1 ? 0 : 1); p++)
        for (int k = blockIdx.x * kBtThreads + threadIdx.x; k < g.s3; k += kBtBlocks * kBtThreads) {
            const int s = p * g.Vhp + t * g.s3 + k;
            Cx<T> o[4];
#pragma unroll
            for (int i = 0; i < 4; i++) o[i] = cx<T>(0, 0);
            // not unrolled: unrolled, ptxas hoists the loads of all six permutations and spills ~1.8 KB per thread
#pragma unroll 1
            for (int ps = 0; ps < NPERM; ps++) {
                // source colours (a', b', c'): the even permutations first, as in the definition
                const int sa = NSRC == 3 ? (ps < 3 ? ps : (ps == 3 ? 0 : (ps == 4 ? 2 : 1))) : 0;
                const int sb = NSRC == 3 ? (ps < 3 ? (ps + 1) % 3 : (ps == 3 ? 2 : (ps == 4 ? 1 : 0))) : 0;
                const int sc = NSRC == 3 ? 3 - sa - sb : 0;
                const T sgn = ps < 3 ? T(1) : T(-1);
                auto pick = [&](int quark, int col) {      // select chain: a run-time index into the parameter struct would copy it to local memory
                    return static_cast<const T2*>(col == 0 ? args.q[quark][0] : (col == 1 ? args.q[quark][1] : args.q[quark][2]));
                };
                const T2* pa = site_ptr(pick(0, sa), 12, 0, s);
                const T2* pb = site_ptr(pick(1, sb), 12, 0, s);
                const T2* pc = site_ptr(pick(2, sc), 12, 0, s);
                Cx<T> M[9];
#pragma unroll
                for (int i = 0; i < 9; i++) M[i] = cx<T>(0, 0);
#pragma unroll
                for (int al = 0; al < 4; al++) {
                    Cx<T> A[3], B[3];
#pragma unroll
                    for (int c = 0; c < 3; c++) {
                        const T2 va = __ldg(pa + (al * 3 + c) * kLane);
                        const T2 vb = __ldg(pb + (gm.perm[al] * 3 + c) * kLane);     // (Gamma q2)_{al c} = i^ph q2_{perm[al] c}
                        A[c] = cx<T>(va.x, va.y);
                        B[c] = mul_i_pow(cx<T>(vb.x, vb.y), gm.ph[al]);
                    }
#pragma unroll
                    for (int a = 0; a < 3; a++)
#pragma unroll
                        for (int b = 0; b < 3; b++) cmad(M[a * 3 + b], A[a], B[b]);
                }
                Cx<T> v[3];
                v[0] = M[1 * 3 + 2] - M[2 * 3 + 1];
                v[1] = M[2 * 3 + 0] - M[0 * 3 + 2];
                v[2] = M[0 * 3 + 1] - M[1 * 3 + 0];
#pragma unroll
                for (int c = 0; c < 3; c++) v[c] = cx<T>(sgn * v[c].re, sgn * v[c].im);
#pragma unroll
                for (int gsp = 0; gsp < 4; gsp++)
#pragma unroll
                    for (int c = 0; c < 3; c++) {
                        const T2 vc = __ldg(pc + (gsp * 3 + c) * kLane);
                        cmad(o[gsp], v[c], cx<T>(vc.x, vc.y));
                    }
            }
#pragma unroll
            for (int i = 0; i < 4; i++) { acc[2 * i] += (double)o[i].re; acc[2 * i + 1] += (double)o[i].im; }
        }
    block_tree<8, kBtThreads>(acc, sm);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < 8; i++) partials[((size_t)t * kBtBlocks + blockIdx.x) * 8 + i] = acc[i];
    }
}
__global__ void baryon_ts_finish_kernel(const double* __restrict__ partials, double* __restrict__ out) {
    const int t = blockIdx.x, k = threadIdx.x;   // 8 threads
    double s = 0.0;
    for (int b = 0; b < kBtBlocks; b++) s += partials[((size_t)t * kBtBlocks + b) * 8 + k];
    out[t * 8 + k] = s;
}

// q: [3 quarks][nsrc source colours] device pointers; partials: 8 * kBtBlocks * L3 doubles; out_dev: 8 * L3 doubles
cudaError_t launch_baryon_timeslices(int prec, const Geom& g, const void* const q[3][3], int nsrc, const SpinMatrix& gm,
                                     int subset, double* partials, double* out_dev, cudaStream_t st) {
    BaryonArgs args;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) args.q[i][j] = q[i][j < nsrc ? j : 0];
    dim3 grid(kBtBlocks, g.L3);
    if (prec) {
        if (nsrc == 3) baryon_ts_kernel<double, 3><<<grid, kBtThreads, 0, st>>>(g, args, gm, subset, partials);
        else           baryon_ts_kernel<double, 1><<<grid, kBtThreads, 0, st>>>(g, args, gm, subset, partials);
    } else {
        if (nsrc == 3) baryon_ts_kernel<float, 3><<<grid, kBtThreads, 0, st>>>(g, args, gm, subset, partials);
        else           baryon_ts_kernel<float, 1><<<grid, kBtThreads, 0, st>>>(g, args, gm, subset, partials);
    }
    baryon_ts_finish_kernel<<<g.L3, 8, 0, st>>>(partials, out_dev);
    g_launch_count += 2;
    return cudaGetLastError();
}

}  // namespace qdp
