// noalloc.cu -- qdp_sum_noalloc: the component-wise lattice sum of qdp_sum (def. 6; SURVEY.md 8(a)
// row a9) for callers that must not allocate.
//
// Who that is: code that runs where device allocation is forbidden or unaffordable -- inside a
// region that another runtime has fenced off (a framework whose caching allocator owns all of
// the GPU's memory and treats a foreign cudaMalloc as an out-of-memory risk), a real-time or
// latency-bound loop where the implicit device-wide synchronisation of cudaMalloc/cudaFree is not
// acceptable, or a plug-in that is handed raw device pointers and a stream and nothing else (it
// has no qdp_lattice handle, and creating one allocates: partials, counters, staging chunks,
// pinned result memory, a copy stream).
//
// What it does instead: the per-block partial sums live in ONE file-scope __device__ array of
// fixed size (kScratchBytes = 36,864 bytes), which every GPU that loads this library holds until
// the process exits.  The caller passes the field, the output and the stream; nothing else is
// touched.  The two kernels below are the two kernels of reduce.cu's launch_sum with the scratch
// pointer aimed at that array: same grid, same summation order, so the result equals qdp_sum's
// bit for bit.
//
// Rules that follow from sharing one array:
//   * every call on a device uses the same scratch, which keeps the last call's contents.  Nothing
//     in it has to start at zero: the first kernel overwrites all 2 * ncomp * 64 slots the second
//     kernel reads, so there is nothing to clear between calls;
//   * two calls that overlap on the GPU (different streams, or different host threads on
//     unordered streams) race on it and both results are garbage.  Calls on one stream are ordered
//     and safe;
//   * the first call on each device looks up the array's device address
//     (cudaGetSymbolAddress, which may also load this library's device code).  Make that first
//     call outside any stream capture.
#include "../../include/qdp_b200.h"
#include "internal.h"

namespace qdp { int set_error(int code, const char* msg); }   // api.cu: thread-local message of qdp_last_error()

namespace {

using namespace qdp;

constexpr int kNaBlocks = 64;      // blocks per component, as in reduce.cu (kSumBlocks): identical summation order
constexpr int kNaMaxComp = 36;     // a gauge field; the largest kind the library has
constexpr size_t kScratchBytes = (size_t)2 * kNaMaxComp * kNaBlocks * sizeof(double);
static_assert(kScratchBytes == 36864, "the header and the README state this size");

// In host code this name is only a handle for cudaGetSymbolAddress -- it is NOT a device address and must never be
// passed to a kernel.  Device code may name it directly.
static __device__ __align__(256) double g_sum_scratch[2 * kNaMaxComp * kNaBlocks];

// device address of g_sum_scratch per device ordinal, looked up once with that device current
constexpr int kMaxDevices = 64;
std::atomic<double*> g_scratch_addr[kMaxDevices];

template <class T2>
__global__ void __launch_bounds__(kReduceThreads) sum_partial_static_kernel(Geom g, int ncomp, const T2* __restrict__ f,
                                                                           int subset, double* __restrict__ scratch) {
    __shared__ double sm[2][kReduceThreads / 32];
    const int n = subset_count(g, subset);
    double acc[2] = {0.0, 0.0};
    for (int i = blockIdx.x * kReduceThreads + threadIdx.x; i < n; i += gridDim.x * kReduceThreads) {
        T2 v = __ldg(f + field_elem(ncomp, blockIdx.y, subset_index(g, subset, i)));
        acc[0] += (double)v.x;
        acc[1] += (double)v.y;
    }
    block_tree<2, kReduceThreads>(acc, sm);
    if (threadIdx.x == 0) {
        scratch[((size_t)blockIdx.y * gridDim.x + blockIdx.x) * 2 + 0] = acc[0];
        scratch[((size_t)blockIdx.y * gridDim.x + blockIdx.x) * 2 + 1] = acc[1];
    }
}

__global__ void sum_finish_static_kernel(int nblk, const double* __restrict__ scratch, double* __restrict__ out) {
    const int c = blockIdx.x, k = threadIdx.x;   // 2 threads: re, im
    double t = 0.0;
    for (int b = 0; b < nblk; b++) t += scratch[((size_t)c * nblk + b) * 2 + k];
    out[c * 2 + k] = t;
}

int na_fail(int code, const char* fmt, long long a = 0, long long b = 0) {
    char msg[256];
    snprintf(msg, sizeof msg, fmt, a, b);
    return set_error(code, msg);
}

}  // namespace

extern "C" int qdp_sum_noalloc(const int dims[4], int ncomp, qdp_prec prec, const void* field_dev, size_t bytes,
                               qdp_subset subset, double* out_dev, void* cuda_stream) {
    if (!dims || !field_dev || !out_dev) return na_fail(QDP_ERR_ARG, "qdp_sum_noalloc: null argument");
    if (prec != QDP_F32 && prec != QDP_F64) return na_fail(QDP_ERR_ARG, "qdp_sum_noalloc: bad precision %lld", prec);
    if (subset != QDP_ALL && subset != QDP_EVEN && subset != QDP_ODD)
        return na_fail(QDP_ERR_ARG, "qdp_sum_noalloc: bad subset %lld", subset);
    if (ncomp < 1) return na_fail(QDP_ERR_ARG, "qdp_sum_noalloc: ncomp = %lld must be positive", ncomp);
    if (ncomp > kNaMaxComp)
        return na_fail(QDP_ERR_ARG,
                       "qdp_sum_noalloc: ncomp = %lld exceeds the %lld components the fixed scratch array holds "
                       "(2 * 36 * 64 doubles); use qdp_sum", ncomp, kNaMaxComp);
    long long V = 1;
    for (int i = 0; i < 4; i++) {
        if (dims[i] < 2 || (dims[i] & 1)) return na_fail(QDP_ERR_DIMS, "extent L%lld = %lld must be even and >= 2", i, dims[i]);
        V *= dims[i];
        if (V + 64 > (1ll << 31) / 36) return na_fail(QDP_ERR_DIMS, "volume too large for 32-bit element indices");
    }
    const Geom g = Geom::make(dims);
    const size_t want = field_elems(g, ncomp) * (prec == QDP_F64 ? 16 : 8);
    if (bytes != want)
        return na_fail(QDP_ERR_ARG, "qdp_sum_noalloc: field of %lld bytes, this lattice and ncomp need %lld",
                       (long long)bytes, (long long)want);

    // set-up, once per device, with that device current: the device address of the scratch array
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return na_fail(QDP_ERR_CUDA, "qdp_sum_noalloc: no current CUDA device (this library has no CPU fallback)");
    if (dev < 0 || dev >= kMaxDevices) return na_fail(QDP_ERR_ARG, "qdp_sum_noalloc: device ordinal %lld not supported", dev);
    double* scratch = g_scratch_addr[dev].load(std::memory_order_acquire);
    if (!scratch) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_sum_scratch);
        if (e != cudaSuccess || !p)
            return na_fail(QDP_ERR_CUDA, "qdp_sum_noalloc: cudaGetSymbolAddress failed on device %lld (CUDA error %lld)", dev, (long long)e);
        scratch = static_cast<double*>(p);
        g_scratch_addr[dev].store(scratch, std::memory_order_release);   // two threads racing here store the same value
    }

    cudaStream_t st = (cudaStream_t)cuda_stream;
    dim3 grid(kNaBlocks, ncomp);
    if (prec == QDP_F64)
        sum_partial_static_kernel<double2><<<grid, kReduceThreads, 0, st>>>(g, ncomp, (const double2*)field_dev, subset, scratch);
    else
        sum_partial_static_kernel<float2><<<grid, kReduceThreads, 0, st>>>(g, ncomp, (const float2*)field_dev, subset, scratch);
    sum_finish_static_kernel<<<ncomp, 2, 0, st>>>(kNaBlocks, scratch, out_dev);
    g_launch_count += 2;
    e = cudaGetLastError();
    if (e != cudaSuccess) return set_error(QDP_ERR_CUDA, cudaGetErrorString(e));
    return QDP_OK;
}
