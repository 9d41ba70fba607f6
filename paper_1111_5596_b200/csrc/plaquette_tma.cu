// plaquette_tma.cu -- the plaquette (def. 2) as a warp-specialised, shared-memory-staged
// kernel: BJ:north_star "shared-memory halo staging of a lattice tile (TMA where the tile is rectangular)".
//
// In the blocked layout (geom.cuh) one 32-site block of a gauge field is 36 x 512 B = 18,432 contiguous bytes
// (fp64), and for lattices whose x0 rows divide a block (Lh0 = L0/2 a power of two <= 32, e.g. 32^3 x 64) a block
// pair (both parities, same half-indices) is a rectangle of the lattice: 32/Lh0 complete x0 rows.  A persistent CTA
// (one per SM) marches through the block pairs j = 0 .. P-1 of one (x0, x1) plane after the other.  One producer
// lane keeps two rings of shared memory filled with `cp.async.bulk` copies that complete on mbarriers:
//     OWN ring,  3 slots: the two gauge blocks of pair j (all four links)            2 x 18,432 B per item
//     HALO ring, 2 slots: pair j of the plane at x2+1 (links 0, 1, 3) and of the
//                         plane at x3+1 (links 0, 1, 2)                              4 x 13,824 B per item
// Step j needs OWN items j and j+1 (the x1 neighbours of a block pair are in itself or in the next pair of the
// plane; the x0 neighbours are in itself) and HALO item j.  Twelve consumer warps = 2 parities x 6 planes (mu, nu)
// read the four operands of their plane with LDS.128 and accumulate Re tr[(U_mu(x) U_nu(x+mu)) (U_nu(x) U_mu(x+nu))^dag].
// The loads in flight no longer occupy registers (the thread-per-site kernel of plaquette.cu holds five matrices
// per thread at 255 registers and 8 warps per SM and is latency-bound, profiles/r1d_ncu_full.md), DRAM latency is
// hidden by a whole step of lookahead (~92 KB per SM), and every operand reaches the SM once per CTA step instead
// of once per thread that uses it.
#include "internal.h"
#include "su3.cuh"
#include "tma.cuh"

namespace qdp {

constexpr int kPtConsumers = 12;                     // 2 parities x 6 planes
constexpr int kPtThreads = (kPtConsumers + 1) * 32;  // + the producer warp
// ring depths: fp64 3 + 2 slots = one step of lookahead in 221 KB; fp32 slots are half as large, so 6 + 4 slots give three
// steps of lookahead in the same shared memory (a step is consumed in ~0.5 us in fp32, less than the latency of its copies)
#ifndef PT_OWN_F32
#define PT_OWN_F32 6
#endif
#ifndef PT_HALO_F32
#define PT_HALO_F32 4
#endif

struct PlaqTmaGeo {
    int P;          // block pairs per (x0, x1) plane = Lh0 * L1 / 32
    int lg, Lh0;    // Lh0 = 1 << lg
    int L2, L3, nplanes;
    int nblk_half;  // blocks per parity half = Vhp / 32
};

template <class T> struct PlaqTmaSmem {
    using T2 = typename Vec2<T>::type;
    static constexpr int kLink = 9 * 32;             // T2 elements of one link of one block
    static constexpr int kGauge = 4 * kLink;
    static constexpr uint32_t kLinkBytes = kLink * sizeof(T2);
    static constexpr uint32_t kGaugeBytes = 4 * kLinkBytes;
    static constexpr int kPtOwnSlots = sizeof(T) == 8 ? 3 : PT_OWN_F32, kPtHaloSlots = sizeof(T) == 8 ? 2 : PT_HALO_F32;
    T2 own[kPtOwnSlots][2][kGauge];                  // [slot][parity]
    T2 halo2[kPtHaloSlots][2][3 * kLink];            // links 0, 1, 3 of the plane at x2+1
    T2 halo3[kPtHaloSlots][2][3 * kLink];            // links 0, 1, 2 of the plane at x3+1
    uint64_t own_full[kPtOwnSlots], own_empty[kPtOwnSlots], halo_full[kPtHaloSlots], halo_empty[kPtHaloSlots];
};

template <class T>
__device__ __forceinline__ Mat3<T> lds_mat(const typename Vec2<T>::type* p) {
    Mat3<T> r;
#pragma unroll
    for (int c = 0; c < 9; c++) {
        const typename Vec2<T>::type v = p[c * kLane];
        r.e[c] = cx<T>(v.x, v.y);
    }
    return r;
}

// sum_ij Re(P_ij conj((A B)_ij)), as in plaquette.cu
template <class T>
__device__ __forceinline__ T re_tr_p_adj_ab_s(const Mat3<T>& P, const Mat3<T>& a, const Mat3<T>& b) {
    T s[3];
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
        s[i] = acc;
    }
    return s[0] + s[1] + s[2];
}

// The consumer loop of one warp for plane (mu, nu), mu < nu.  The plane is a run-time (warp-uniform) value that
// only enters the four operand addresses: the six planes share one copy of the ~1500-instruction body.  (With one
// template instance per plane the twelve warps of an SM ran six different 24 KB code paths and the kernel stalled on
// instruction fetch: ncu stall_no_instruction 4.4 per issue, 0.45 ms on 32^3 x 64 fp64.)
template <class T>
__device__ __forceinline__ double plaq_tma_consume(PlaqTmaSmem<T>& sm, const PlaqTmaGeo& pg, int p, int mu, int nu, int lane) {
    using T2 = typename Vec2<T>::type;
    using S = PlaqTmaSmem<T>;
    double acc = 0.0;
    int own_base = 0, halo_item = 0;
    for (int q = blockIdx.x; q < pg.nplanes; q += gridDim.x) {
        const int x2 = q % pg.L2, x3 = q / pg.L2;
        for (int j = 0; j < pg.P; j++) {
            const int it0 = own_base + j, it1 = it0 + 1;
            const int s0 = it0 % S::kPtOwnSlots, s1 = it1 % S::kPtOwnSlots, hs = halo_item % S::kPtHaloSlots;
            // geometry of site (p, 32 j + lane) of this plane
            const int o = 32 * j + lane;
            const int x1 = o >> pg.lg, hx = o & (pg.Lh0 - 1);
            const int odd0 = (p + x1 + x2 + x3) & 1;
            const T2* here = &sm.own[s0][p][lane];
            // operand U_lam(x + d), d = mu or nu
            auto nb = [&](int d, int lam) -> const T2* {
                if (d == 0) {
                    const int l0 = lane + (odd0 ? (hx == pg.Lh0 - 1 ? -(pg.Lh0 - 1) : 1) : 0);
                    return &sm.own[s0][1 - p][l0 + lam * S::kLink];
                } else if (d == 1) {
                    const int l1 = lane + pg.Lh0;
                    return (l1 < 32 ? &sm.own[s0][1 - p][l1] : &sm.own[s1][1 - p][l1 - 32]) + lam * S::kLink;
                } else if (d == 2) {
                    return &sm.halo2[hs][1 - p][lane + (lam == 3 ? 2 : lam) * S::kLink];
                } else {
                    return &sm.halo3[hs][1 - p][lane + lam * S::kLink];
                }
            };
            const T2* pA = here + mu * S::kLink;     // U_mu(x)
            const T2* pB = nb(mu, nu);               // U_nu(x+mu)
            const T2* pA2 = here + nu * S::kLink;    // U_nu(x)
            const T2* pB2 = nb(nu, mu);              // U_mu(x+nu)
            mbar_wait(&sm.own_full[s0], (it0 / S::kPtOwnSlots) & 1);
            mbar_wait(&sm.own_full[s1], (it1 / S::kPtOwnSlots) & 1);
            mbar_wait(&sm.halo_full[hs], (halo_item / S::kPtHaloSlots) & 1);
            const Mat3<T> A = lds_mat<T>(pA);
            const Mat3<T> B = lds_mat<T>(pB);
            const Mat3<T> Pm = mul(A, B);
            const Mat3<T> A2 = lds_mat<T>(pA2);
            const Mat3<T> B2 = lds_mat<T>(pB2);
            acc += (double)re_tr_p_adj_ab_s(Pm, A2, B2);
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&sm.own_empty[s0]);
                if (j == pg.P - 1) mbar_arrive(&sm.own_empty[s1]);
                mbar_arrive(&sm.halo_empty[hs]);
            }
            halo_item++;
        }
        own_base += pg.P + 1;
    }
    return acc;
}

template <class T>
__global__ void __launch_bounds__(kPtThreads, 1)
plaquette_tma_kernel(PlaqTmaGeo pg, const typename Vec2<T>::type* __restrict__ u, ReduceBuf rb, double s_all, double s_part) {
    using T2 = typename Vec2<T>::type;
    using S = PlaqTmaSmem<T>;
    extern __shared__ __align__(128) unsigned char smem_pt[];
    S& sm = *reinterpret_cast<S*>(smem_pt);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int i = 0; i < S::kPtOwnSlots; i++) { mbar_init(&sm.own_full[i], 1); mbar_init(&sm.own_empty[i], kPtConsumers); }
        for (int i = 0; i < S::kPtHaloSlots; i++) { mbar_init(&sm.halo_full[i], 1); mbar_init(&sm.halo_empty[i], kPtConsumers); }
        mbar_fence_init();
    }
    __syncthreads();
    double acc[3] = {0.0, 0.0, 0.0};   // all, spatial, temporal
    if (warp == kPtConsumers) {
        if (lane == 0) {
            // ---- producer: own(0); then per step j: own(j+1), halo(j) ----
            int own_item = 0, halo_item = 0;
            for (int q = blockIdx.x; q < pg.nplanes; q += gridDim.x) {
                const int x2 = q % pg.L2, x3 = q / pg.L2;
                const int q2 = (x2 + 1 == pg.L2 ? 0 : x2 + 1) + pg.L2 * x3;
                const int q3 = x2 + pg.L2 * (x3 + 1 == pg.L3 ? 0 : x3 + 1);
                for (int j = 0; j <= pg.P; j++) {
                    {
                        const int s = own_item % S::kPtOwnSlots;
                        mbar_wait(&sm.own_empty[s], ((own_item / S::kPtOwnSlots) & 1) ^ 1);
                        mbar_arrive_expect_tx(&sm.own_full[s], 2 * S::kGaugeBytes);
                        const int jb = j == pg.P ? 0 : j;   // the x1 wrap: the plane's first pair again
#ifdef QDP_BOUNDS_CHECK
                        if (q * pg.P + jb >= pg.nblk_half || q2 * pg.P + pg.P > pg.nblk_half || q3 * pg.P + pg.P > pg.nblk_half)
                            printf("QDP_BOUNDS plaquette_tma: plane %d/%d/%d block %d of %d\n", q, q2, q3, jb, pg.nblk_half);
#endif
                        for (int p = 0; p < 2; p++)
                            bulk_g2s(sm.own[s][p], u + (size_t)(p * pg.nblk_half + q * pg.P + jb) * S::kGauge, S::kGaugeBytes,
                                     &sm.own_full[s]);
                        own_item++;
                    }
                    if (j >= 1) {
                        const int s = halo_item % S::kPtHaloSlots;
                        mbar_wait(&sm.halo_empty[s], ((halo_item / S::kPtHaloSlots) & 1) ^ 1);
                        mbar_arrive_expect_tx(&sm.halo_full[s], 12 * S::kLinkBytes);
                        for (int p = 0; p < 2; p++) {
                            const T2* b2 = u + (size_t)(p * pg.nblk_half + q2 * pg.P + (j - 1)) * S::kGauge;
                            const T2* b3 = u + (size_t)(p * pg.nblk_half + q3 * pg.P + (j - 1)) * S::kGauge;
                            bulk_g2s(sm.halo2[s][p], b2, 2 * S::kLinkBytes, &sm.halo_full[s]);                               // links 0, 1
                            bulk_g2s(sm.halo2[s][p] + 2 * S::kLink, b2 + 3 * S::kLink, S::kLinkBytes, &sm.halo_full[s]);      // link 3
                            bulk_g2s(sm.halo3[s][p], b3, 3 * S::kLinkBytes, &sm.halo_full[s]);                               // links 0, 1, 2
                        }
                        halo_item++;
                    }
                }
            }
        }
    } else {
        const int p = warp / 6, pl = warp % 6;
        // planes (0,1) (0,2) (1,2) (0,3) (1,3) (2,3): the first three are spatial
        const int mu = pl < 3 ? (pl == 2) : pl - 3, nu = pl < 3 ? (pl == 0 ? 1 : 2) : 3;
        const double v = plaq_tma_consume<T>(sm, pg, p, mu, nu, lane);
        if (pl < 3) acc[1] = v; else acc[2] = v;
    }
    __syncwarp();
    acc[0] = acc[1] + acc[2];
    const double sc[3] = {s_all, s_part, s_part};
    warp_grid_reduce<3>(acc, rb, sc);
}

bool plaquette_tma_applicable(const Geom& g, int subset) {
    if (subset != 0 || !g.staged) return false;
    if (g.Lh0 > 32 || (g.Lh0 & (g.Lh0 - 1)) != 0) return false;   // x0 rows must tile a 32-site block
    if ((g.s2 & 31) != 0) return false;                           // an (x0, x1) plane is a whole number of blocks
    return true;
}

template <class T>
static cudaError_t launch_plaquette_tma_t(const Geom& g, const void* u, const ReduceBuf& rb, int sms, cudaStream_t st) {
    using T2 = typename Vec2<T>::type;
    PlaqTmaGeo pg;
    pg.P = g.s2 >> 5;
    pg.Lh0 = g.Lh0;
    pg.lg = 0;
    while ((1 << pg.lg) < g.Lh0) pg.lg++;
    pg.L2 = g.L2; pg.L3 = g.L3;
    pg.nplanes = g.L2 * g.L3;
    pg.nblk_half = g.Vhp >> 5;
    const int smem = (int)sizeof(PlaqTmaSmem<T>);
    // the opt-in is a per-device property of the function: set it on whichever device is current (cheap, and safe
    // from several host threads, unlike a process-wide flag)
    {
        cudaError_t e = cudaFuncSetAttribute(plaquette_tma_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
    }
    const int grid = pg.nplanes < sms ? pg.nplanes : sms;
    const double n = (double)g.V;
    plaquette_tma_kernel<T><<<grid, kPtThreads, smem, st>>>(pg, (const T2*)u, rb, 1.0 / (18.0 * n), 1.0 / (9.0 * n));
    g_launch_count++;
    return cudaGetLastError();
}

cudaError_t launch_plaquette_tma(int prec, const Geom& g, const void* u, const ReduceBuf& rb, int sms, cudaStream_t st) {
    return prec ? launch_plaquette_tma_t<double>(g, u, rb, sms, st) : launch_plaquette_tma_t<float>(g, u, rb, sms, st);
}

}  // namespace qdp
