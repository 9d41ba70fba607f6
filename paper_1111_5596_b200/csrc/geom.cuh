// geom.cuh -- lattice geometry on the device: internal site order, coordinates,
// nearest-neighbour index arithmetic.  (DESIGN.md "Layout".)
//
// Internal site order ("checkerboard-lex"):
//     s = parity(x) * Vhp + (lex(x) >> 1),   lex(x) = x0 + L0*(x1 + L1*(x2 + L2*x3))
// with Vhp = V/2 rounded up to a multiple of 32 (= V/2 for every BASELINE config).
// Because L0 is even, lex pairs (2k, 2k+1) differ only in x0 and hence in parity,
// so h = lex >> 1 enumerates each parity half once.  EVEN subset = [0, V/2),
// ODD = [Vhp, Vhp + V/2): red/black operations touch contiguous memory, and every
// neighbour of a site lies in the other half.
//
// Field storage ("blocked structure of arrays"): sites are grouped
// in blocks of 32 consecutive indices; inside a block the components are planes of 32
// complex numbers:
//     element(c, s) = ((s >> 5) * ncomp + c) * 32 + (s & 31)
// A warp still moves 32 consecutive complex numbers (512 B fp64) per component, but all
// components of a site now sit at compile-time offsets (c * 32 elements) from one base
// address, so a 3x3 matrix costs one address computation instead of nine.
//
// No neighbour tables are read by the kernels: a neighbour index is a handful of
// integer instructions on the decoded coordinates, which is cheaper than the
// 32 B/site of table traffic it would replace on an HBM-bound path.
#pragma once
#ifdef __CUDACC_RTC__
// Run-time compilation of an expression kernel (jit.cu): NVRTC has the CUDA built-ins but no host headers.
typedef unsigned int uint32_t;
typedef unsigned long long uint64_t;
typedef int int32_t;
typedef long long int64_t;
typedef unsigned char uint8_t;
#else
#include <cstdint>
#include <cuda_runtime.h>
#endif

namespace qdp {

// Division of n < 2^31 by a run-time constant d < 2^31: q = (n * m) >> sh.
// m = ceil(2^(31+l) / d), l = ceil(log2 d)   (Granlund-Montgomery, N = 31 bits)
struct FastDiv {
    uint32_t d, m, sh;
#ifndef __CUDACC_RTC__
    __host__ static FastDiv make(uint32_t d) {
        FastDiv f;
        f.d = d;
        uint32_t l = 0;
        while ((1ull << l) < d) ++l;
        f.sh = 31 + l;
        f.m = (uint32_t)(((1ull << f.sh) + d - 1) / d);
        return f;
    }
#endif
    __host__ __device__ __forceinline__ uint32_t div(uint32_t n) const {
        return (uint32_t)(((uint64_t)n * m) >> sh);
    }
};

struct Geom {
    int L0, L1, L2, L3;
    int Lh0;         // L0 / 2
    int V, Vh;       // sites, sites per parity
    int Vhp;         // Vh rounded up to a multiple of 32: index stride between the parity halves
    int s1, s2, s3;  // strides of x1, x2, x3 in the half index h
    FastDiv dLh0, dL1, dL2;
    // L2-aware sweep order of the neighbour-reading kernels (sweep_block below); slab_c2 = 0: linear
    int slab_c2;      // x2 extent of a slab (a divisor of L2)
    int slab_ipr;     // 32-site blocks per (x2, x3) line of the (x0, x1) plane = Lh0 * L1 / 32
    int staged;       // 1: use the shared-memory-staged kernels (plaquette_tma.cu) where the lattice allows

#ifndef __CUDACC_RTC__
    __host__ static Geom make(const int* L) {
        Geom g;
        g.L0 = L[0]; g.L1 = L[1]; g.L2 = L[2]; g.L3 = L[3];
        g.Lh0 = L[0] / 2;
        g.V = L[0] * L[1] * L[2] * L[3];
        g.Vh = g.V / 2;
        g.Vhp = (g.Vh + 31) & ~31;
        g.s1 = g.Lh0; g.s2 = g.Lh0 * L[1]; g.s3 = g.Lh0 * L[1] * L[2];
        g.dLh0 = FastDiv::make(g.Lh0);
        g.dL1 = FastDiv::make(L[1]);
        g.dL2 = FastDiv::make(L[2]);
        g.slab_c2 = 0; g.slab_ipr = 0;
        g.staged = 0;   // measured on 32^3 x 64 fp64: staged plaquette 0.349 ms vs 0.331 ms thread-per-site (profiles/r2_plaquette_staged.md)
#ifndef QDP_SLAB_BYTES
#define QDP_SLAB_BYTES (16u << 20)          // x3-slice of a slab, fp64 gauge field
#define QDP_SLAB_ENABLE_BYTES (24u << 20)   // lattices whose whole x3-slice is smaller sweep linearly
#endif
        // One x3-slice of a slab (x0, x1 full, c2 values of x2) of an fp64 gauge field should stay
        // resident in L2 between its use as the +3 neighbour and as the site's own links.  Measured
        // (B200, fp64): 32^3 x 64 (slice 18.9 MB) is 1-3 % faster in linear order; 48^3 x 96
        // (slice 63.7 MB) with 16 MB slabs: plaquette 1.93 -> 1.74 ms, hop ALL 2.51 -> 2.12 ms.
        const long long line_bytes = (long long)L[0] * L[1] * 576;
        if ((g.s2 & 31) == 0 && line_bytes * L[2] > (long long)QDP_SLAB_ENABLE_BYTES) {
            int c2 = 0;
            for (int d = 1; d < L[2]; d++)
                if (L[2] % d == 0 && line_bytes * d <= (long long)QDP_SLAB_BYTES) c2 = d;
            if (c2 > 0) { g.slab_c2 = c2; g.slab_ipr = g.s2 >> 5; }
        }
        return g;
    }
#endif
};

// A decoded site.  odd0 = x0 & 1 = (p + x1 + x2 + x3) & 1;  x0 = 2*hx + odd0.
struct Site {
    int p, h, hx, x1, x2, x3, odd0;
    __device__ __forceinline__ int index(const Geom& g) const { return p * g.Vhp + h; }
    __device__ __forceinline__ int x0() const { return 2 * hx + odd0; }
};

__device__ __forceinline__ Site site_decode(const Geom& g, int p, int h) {
    Site x;
    x.p = p; x.h = h;
    uint32_t r1 = g.dLh0.div((uint32_t)h);
    x.hx = h - (int)r1 * g.Lh0;
    uint32_t r2 = g.dL1.div(r1);
    x.x1 = (int)r1 - (int)r2 * g.L1;
    uint32_t r3 = g.dL2.div(r2);
    x.x2 = (int)r2 - (int)r3 * g.L2;
    x.x3 = (int)r3;
    x.odd0 = (p + x.x1 + x.x2 + x.x3) & 1;
    return x;
}

// element index of component c of site s in a field of ncomp components per site
__host__ __device__ __forceinline__ size_t field_elem(int ncomp, int c, int s) {
    return ((size_t)(s >> 5) * ncomp + c) * 32 + (s & 31);
}
// complex elements a field of ncomp components occupies (including the padding lanes)
__host__ __device__ __forceinline__ size_t field_elems(const Geom& g, int ncomp) {
    return (size_t)2 * g.Vhp * ncomp;
}

// x + sign * mu_hat with periodic wrap; MU, SIGN compile-time so it unrolls away.
template <int MU, int SIGN>
__device__ __forceinline__ Site site_step(const Geom& g, Site x) {
    if (MU == 0) {
        if (SIGN > 0) {
            if (x.odd0) {
                bool wrap = x.hx == g.Lh0 - 1;
                x.h += wrap ? -(g.Lh0 - 1) : 1;
                x.hx = wrap ? 0 : x.hx + 1;
            }
        } else {
            if (!x.odd0) {
                bool wrap = x.hx == 0;
                x.h += wrap ? (g.Lh0 - 1) : -1;
                x.hx = wrap ? g.Lh0 - 1 : x.hx - 1;
            }
        }
    } else if (MU == 1) {
        bool wrap = SIGN > 0 ? x.x1 == g.L1 - 1 : x.x1 == 0;
        x.h += SIGN * (wrap ? -(g.L1 - 1) * g.s1 : g.s1);
        x.x1 = wrap ? (SIGN > 0 ? 0 : g.L1 - 1) : x.x1 + SIGN;
    } else if (MU == 2) {
        bool wrap = SIGN > 0 ? x.x2 == g.L2 - 1 : x.x2 == 0;
        x.h += SIGN * (wrap ? -(g.L2 - 1) * g.s2 : g.s2);
        x.x2 = wrap ? (SIGN > 0 ? 0 : g.L2 - 1) : x.x2 + SIGN;
    } else {
        bool wrap = SIGN > 0 ? x.x3 == g.L3 - 1 : x.x3 == 0;
        x.h += SIGN * (wrap ? -(g.L3 - 1) * g.s3 : g.s3);
        x.x3 = wrap ? (SIGN > 0 ? 0 : g.L3 - 1) : x.x3 + SIGN;
    }
    x.p ^= 1;
    if (MU == 0) x.odd0 ^= 1;   // for MU != 0 both p and x_MU change parity: odd0 = (p+x1+x2+x3)&1 is unchanged
    return x;
}

// run-time direction (used by shift and the table export)
__device__ __forceinline__ Site site_step_rt(const Geom& g, const Site& x, int mu, int sign) {
    switch (mu * 2 + (sign < 0)) {
        case 0: return site_step<0, +1>(g, x);
        case 1: return site_step<0, -1>(g, x);
        case 2: return site_step<1, +1>(g, x);
        case 3: return site_step<1, -1>(g, x);
        case 4: return site_step<2, +1>(g, x);
        case 5: return site_step<2, -1>(g, x);
        case 6: return site_step<3, +1>(g, x);
        default: return site_step<3, -1>(g, x);
    }
}

__device__ __forceinline__ int site_lex(const Geom& g, const Site& x) {
    return x.x0() + g.L0 * (x.x1 + g.L1 * (x.x2 + g.L2 * x.x3));
}

// public lex index -> internal index
__device__ __forceinline__ int lex_to_index(const Geom& g, int lex) {
    int h = lex >> 1;
    uint32_t r1 = g.dLh0.div((uint32_t)h);
    uint32_t r2 = g.dL1.div(r1);
    uint32_t r3 = g.dL2.div(r2);
    int x1 = (int)r1 - (int)r2 * g.L1, x2 = (int)r2 - (int)r3 * g.L2, x3 = (int)r3;
    int p = ((lex & 1) + x1 + x2 + x3) & 1;
    return p * g.Vhp + h;
}

// Map a linear work item to a site of the subset: subset 0 -> all V sites (both
// halves, in internal order), 1 -> even half, 2 -> odd half.
__device__ __forceinline__ int subset_count(const Geom& g, int subset) {
    return subset == 0 ? g.V : g.Vh;
}
// i-th site of the subset in work order -> internal index (subset 0: even half, then odd half)
__device__ __forceinline__ int subset_index(const Geom& g, int subset, int i) {
    if (subset == 0) return i < g.Vh ? i : i - g.Vh + g.Vhp;
    return subset == 2 ? i + g.Vhp : i;
}
__device__ __forceinline__ Site subset_site(const Geom& g, int subset, int i) {
    int p = subset == 0 ? (i >= g.Vh) : (subset == 2);
    return site_decode(g, p, subset == 0 && p ? i - g.Vh : i);
}

// L2-aware sweep order.  In linear order the links of site x+3 are first read as the +3 neighbour
// and again, one whole x3-slice of traffic later, as that site's own links; on 48^3 x 96 a slice
// of the gauge field is 64 MB and the second read misses the L2 (measured DRAM traffic 1.41x
// algorithmic for the plaquette, 1.55x for the full-lattice hop).  The sweep therefore walks
// slabs of slab_c2 values of x2 (x0, x1 complete), x3 slowest inside a slab, which shortens
// that reuse distance to one slab slice (<= QDP_SLAB_BYTES); only the x2 faces between slabs
// are read twice.  v = position in the sweep, result = 32-site block index in h order.
__device__ __forceinline__ int sweep_block(const Geom& g, int v) {
    if (g.slab_c2 == 0) return v;
    const int per_x3 = g.slab_c2 * g.slab_ipr;          // blocks of one x3-slice of a slab
    const int per_slab = per_x3 * g.L3;
    const int slab = v / per_slab, r = v - slab * per_slab;
    const int x3 = r / per_x3, r2 = r - x3 * per_x3;    // r2 = (x2 - slab * c2) * ipr + block in line
    return (x3 * g.L2 + slab * g.slab_c2) * g.slab_ipr + r2;
}

// Work-item order for the neighbour-reading kernels.  For the full lattice the two
// parities are interleaved warp by warp over the same run of 32 half-indices:
//     item i -> parity (i >> 5) & 1, h = (i >> 6) * 32 + (i & 31)
// so a site and its neighbours (which lie in the other half) are processed by
// adjacent warps at the same time and each link / spinor comes from DRAM once; walking
// the even half and then the odd half would stream every field twice.
// Returns false for padding items (Vh not a multiple of 32).
__device__ __forceinline__ int work_items(const Geom& g, int subset) {
    return subset == 0 ? 2 * ((g.Vh + 31) & ~31) : g.Vh;
}
__device__ __forceinline__ bool work_site(const Geom& g, int subset, int i, int& p, int& h) {
    if (subset == 0) {
        p = (i >> 5) & 1;
        h = (sweep_block(g, i >> 6) << 5) + (i & 31);
    } else {
        p = subset == 2;
        h = (sweep_block(g, i >> 5) << 5) + (i & 31);
    }
    return h < g.Vh;
}

}  // namespace qdp
