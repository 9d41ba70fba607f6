// layout.cu -- host interchange layout <-> device layout, and geometry export.
// (Appendix A.)
//
// Host side: array of structures, lexicographic sites -- the site-outermost
// layout the paper found un-coalesced on the device.  It is only
// the interchange format: a chunk of it is copied to a staging buffer and
// transposed through shared memory into the site-fastest SoA planes, so both the
// staging reads and the plane writes are coalesced.
#include "internal.h"
#include "su3.cuh"

namespace qdp {

std::atomic<long long> g_launch_count{0};

int device_sm_count() {
    static std::atomic<int> cache[64];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
    int n = cache[dev].load(std::memory_order_relaxed);
    if (n <= 0) {
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
        cache[dev].store(n, std::memory_order_relaxed);
    }
    return n;
}

constexpr int kTileSites = 64;   // sites per block in the transposes

// stage: [nsites][ncomp] complex (chunk starting at public site lex_begin)
template <class T2, bool TO_SOA>
__global__ void __launch_bounds__(256) transpose_kernel(Geom g, int ncomp, T2* __restrict__ stage,
                                                       T2* __restrict__ field, int lex_begin, int nsites) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T2* tile = reinterpret_cast<T2*>(smem_raw);          // [ncomp][kTileSites + 1]
    const int pitch = kTileSites + 1;
    const int site0 = blockIdx.x * kTileSites;
    const int ns = min(kTileSites, nsites - site0);
    const int nelem = ns * ncomp;
    T2* st = stage + (size_t)site0 * ncomp;
    if (TO_SOA) {
        for (int e = threadIdx.x; e < nelem; e += blockDim.x) {
            int j = e / ncomp, c = e - j * ncomp;
            tile[c * pitch + j] = st[e];
        }
        __syncthreads();
        for (int e = threadIdx.x; e < nelem; e += blockDim.x) {
            int c = e / ns, j = e - c * ns;
            int s = lex_to_index(g, lex_begin + site0 + j);
            field[field_elem(ncomp, c, s)] = tile[c * pitch + j];
        }
    } else {
        for (int e = threadIdx.x; e < nelem; e += blockDim.x) {
            int c = e / ns, j = e - c * ns;
            int s = lex_to_index(g, lex_begin + site0 + j);
            tile[c * pitch + j] = field[field_elem(ncomp, c, s)];
        }
        __syncthreads();
        for (int e = threadIdx.x; e < nelem; e += blockDim.x) {
            int j = e / ncomp, c = e - j * ncomp;
            st[e] = tile[c * pitch + j];
        }
    }
}

template <class T2, bool TO_SOA>
static cudaError_t launch_transpose(const Geom& g, int ncomp, void* stage, void* field, int lex_begin,
                                    int nsites, cudaStream_t st) {
    if (nsites <= 0) return cudaSuccess;
    int blocks = (nsites + kTileSites - 1) / kTileSites;
    size_t smem = (size_t)ncomp * (kTileSites + 1) * sizeof(T2);
    transpose_kernel<T2, TO_SOA><<<blocks, 256, smem, st>>>(g, ncomp, (T2*)stage, (T2*)field, lex_begin, nsites);
    g_launch_count++;
    return cudaGetLastError();
}

cudaError_t launch_aos_to_soa(int prec, const Geom& g, int ncomp, const void* stage, void* field,
                              int lex_begin, int nsites, cudaStream_t st) {
    return prec ? launch_transpose<double2, true>(g, ncomp, (void*)stage, field, lex_begin, nsites, st)
                : launch_transpose<float2, true>(g, ncomp, (void*)stage, field, lex_begin, nsites, st);
}
cudaError_t launch_soa_to_aos(int prec, const Geom& g, int ncomp, const void* field, void* stage,
                              int lex_begin, int nsites, cudaStream_t st) {
    return prec ? launch_transpose<double2, false>(g, ncomp, stage, (void*)field, lex_begin, nsites, st)
                : launch_transpose<float2, false>(g, ncomp, stage, (void*)field, lex_begin, nsites, st);
}

// ---- time-slice faces (the face an x3-slab decomposition exchanges) --------------
// The sites with x3 = t are the half-indices [t s3, (t+1) s3) of each parity.  Face buffer layout (private, only
// meaningful for lattices with the same L0, L1, L2), indexed by the SPATIAL parity q = (x0 + x1 + x2) & 1 = (p + t) & 1
// so that a face does not depend on the slice it was taken from or is written to (a site and its x3 neighbour have the
// same half-index offset k inside their slices but opposite parities):
//     buf[(q * ncomp + c) * s3 + k] = element(c, p Vhp + t s3 + k),   p = (q + t) & 1.
// TO_FACE: field -> buffer (both parities); else buffer -> field, writing only the sites of `subset`.
template <class T2, bool TO_FACE>
__global__ void __launch_bounds__(256) timeslice_kernel(Geom g, int ncomp, T2* __restrict__ field, T2* __restrict__ buf, int t,
                                                       int subset) {
    const int n = 2 * ncomp * g.s3;
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
        const int k = e % g.s3, qc = e / g.s3, c = qc % ncomp, p = (qc / ncomp + t) & 1;
        if (!TO_FACE && subset != 0 && p != (subset == 2)) continue;
        const size_t fe = field_elem(ncomp, c, p * g.Vhp + t * g.s3 + k);
        if (TO_FACE) buf[e] = field[fe]; else field[fe] = buf[e];
    }
}
cudaError_t launch_timeslice(int prec, const Geom& g, int ncomp, void* field, void* buf, int t, int subset, bool to_face,
                             cudaStream_t st) {
    const int n = 2 * ncomp * g.s3;
    int blocks = (n + 255) / 256;
    if (blocks > 4096) blocks = 4096;
    if (prec) {
        if (to_face) timeslice_kernel<double2, true><<<blocks, 256, 0, st>>>(g, ncomp, (double2*)field, (double2*)buf, t, subset);
        else         timeslice_kernel<double2, false><<<blocks, 256, 0, st>>>(g, ncomp, (double2*)field, (double2*)buf, t, subset);
    } else {
        if (to_face) timeslice_kernel<float2, true><<<blocks, 256, 0, st>>>(g, ncomp, (float2*)field, (float2*)buf, t, subset);
        else         timeslice_kernel<float2, false><<<blocks, 256, 0, st>>>(g, ncomp, (float2*)field, (float2*)buf, t, subset);
    }
    g_launch_count++;
    return cudaGetLastError();
}

// out[lex(x)] = lex(x + sign*mu_hat): decoded and stepped with the very functions
// the expression kernels use, so the parity test of the table pins them.
__global__ void neighbor_table_kernel(Geom g, int mu, int sign, int32_t* __restrict__ out) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= g.V) return;
    Site x = subset_site(g, 0, s);
    Site y = site_step_rt(g, x, mu, sign);
    out[site_lex(g, x)] = site_lex(g, y);
}
__global__ void parity_mask_kernel(Geom g, uint8_t* __restrict__ out) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= g.V) return;
    Site x = subset_site(g, 0, s);
    out[site_lex(g, x)] = (uint8_t)x.p;
}

cudaError_t launch_neighbor_table(const Geom& g, int mu, int sign, int32_t* out, cudaStream_t st) {
    neighbor_table_kernel<<<(g.V + 255) / 256, 256, 0, st>>>(g, mu, sign, out);
    g_launch_count++;
    return cudaGetLastError();
}
cudaError_t launch_parity_mask(const Geom& g, uint8_t* out, cudaStream_t st) {
    parity_mask_kernel<<<(g.V + 255) / 256, 256, 0, st>>>(g, out);
    g_launch_count++;
    return cudaGetLastError();
}

}  // namespace qdp
