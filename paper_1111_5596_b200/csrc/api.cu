// api.cu -- the C ABI of include/qdp_b200.h: handles, argument validation, memory,
// host<->device transfers and kernel dispatch.  No arithmetic of the method lives
// here; every step of the path runs in the kernels of the other translation units.
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

#include "../../include/qdp_b200.h"
#include "internal.h"
#include "expr.cuh"
#include "su3.cuh"

using namespace qdp;

// ---- error reporting ---------------------------------------------------------
static thread_local char t_err[512] = "";

static int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof t_err, fmt, ap);
    va_end(ap);
    return code;
}
namespace qdp { int set_error(int code, const char* msg) { return fail(code, "%s", msg); } }   // for pool.cu
#define CUDA_TRY(expr)                                                                     \
    do {                                                                                   \
        cudaError_t e_ = (expr);                                                           \
        if (e_ != cudaSuccess)                                                             \
            return fail(e_ == cudaErrorMemoryAllocation ? QDP_ERR_OOM : QDP_ERR_CUDA,      \
                        "%s: %s (%s:%d)", #expr, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

// ---- allocator hook ----------------------------------------------------------
static void* (*g_alloc)(size_t, void*) = nullptr;
static void (*g_free)(void*, void*) = nullptr;
static void* g_alloc_ctx = nullptr;

static int dev_alloc(size_t bytes, void** out) {
    if (g_alloc) {
        *out = g_alloc(bytes, g_alloc_ctx);
        if (!*out) return fail(QDP_ERR_OOM, "allocator hook returned NULL for %zu bytes", bytes);
        return QDP_OK;
    }
    CUDA_TRY(cudaMalloc(out, bytes));
    return QDP_OK;
}
static void dev_free(void* p, bool from_hook) {
    if (!p) return;
    if (from_hook && g_free) g_free(p, g_alloc_ctx);
    else cudaFree(p);
}

// ---- handles -------------------------------------------------------------------
static const uint32_t kLatMagic = 0x51445031u, kFieldMagic = 0x51445032u;
static const int kStageSites = 1 << 15;   // sites per upload/download chunk

struct qdp_lattice {
    uint32_t magic;
    int device;
    int dims[4];
    Geom geom;
    cudaStream_t stream;
    // scratch, all allocated at create time
    double* partials;        // device: 4 * kMaxPartialBlocks, also 2*36*64 for sum
    unsigned int* counter;   // device
    double* result_host;     // pinned, mapped: 72 doubles + the completion flag; the reducing kernels write their results here
    double* result_dev;      // the device address of result_host
    unsigned long long seq;  // number of the last reducing launch; the kernel stores it behind the results when they are complete
    void* stage[2];          // device staging chunks for upload/download
    size_t stage_bytes;
    cudaStream_t copy_stream;
    cudaEvent_t ev_copied[2], ev_done[2];
    bool scratch_from_hook;
    int live_fields;
};

struct qdp_field {
    uint32_t magic;
    qdp_lattice* lat;
    int kind, prec, ncomp;
    void* data;
    size_t bytes;
    bool owned, from_hook;
};

static int kind_ncomp(int kind) {
    switch (kind) {
        case QDP_COLOR_MATRIX: return 9;
        case QDP_GAUGE: return 36;
        case QDP_FERMION: return 12;
        case QDP_COMPLEX: return 1;
        default: return 0;
    }
}
static size_t elem_bytes(int prec) { return prec == QDP_F64 ? 16 : 8; }

static bool ok_lat(const qdp_lattice* l) { return l && l->magic == kLatMagic; }
static bool ok_field(const qdp_field* f) { return f && f->magic == kFieldMagic && ok_lat(f->lat); }
static bool ok_subset(int s) { return s == QDP_ALL || s == QDP_EVEN || s == QDP_ODD; }

static const int kResultSlots = 72;   // doubles of results; the completion flag follows them
static ReduceBuf reduce_buf(qdp_lattice* l) {
    ReduceBuf rb;
    rb.partials = l->partials;
    rb.counter = l->counter;
    rb.result = l->result_dev;
    rb.flag = reinterpret_cast<unsigned long long*>(l->result_dev + kResultSlots);
    rb.seq = ++l->seq;
    return rb;
}
// The last block of a reducing kernel stores the n results straight into mapped pinned host memory (no separate
// device-to-host copy to launch) and then the launch's sequence number behind them.  The host polls that number
// (a few microseconds less than cudaStreamSynchronize per scalar-returning call: DESIGN.md section 4) and checks the
// stream from time to time so that a failed kernel surfaces as an error instead of a hang.
static int fetch_result(qdp_lattice* l, int n, double* out) {
    volatile unsigned long long* flag = reinterpret_cast<volatile unsigned long long*>(l->result_host + kResultSlots);
    for (unsigned spin = 1; *flag != l->seq; spin++) {
        if ((spin & 0x3fff) == 0) {
            cudaError_t q = cudaStreamQuery(l->stream);
            if (q == cudaSuccess) {
                if (*flag == l->seq) break;
                return fail(QDP_ERR_CUDA, "reduction kernel finished without signalling its result");
            }
            if (q != cudaErrorNotReady) return fail(QDP_ERR_CUDA, "CUDA error: %s", cudaGetErrorString(q));
        }
    }
    std::atomic_thread_fence(std::memory_order_acquire);
    memcpy(out, l->result_host, n * sizeof(double));
    return QDP_OK;
}
// for results that a kernel without the completion signal wrote (qdp_sum)
static int fetch_result_sync(qdp_lattice* l, int n, double* out) {
    CUDA_TRY(cudaStreamSynchronize(l->stream));
    memcpy(out, l->result_host, n * sizeof(double));
    return QDP_OK;
}

struct DeviceGuard {
    int prev;
    bool ok;
    explicit DeviceGuard(int dev) : prev(-1), ok(false) {
        if (cudaGetDevice(&prev) != cudaSuccess) return;
        ok = prev == dev || cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard() { if (ok && prev >= 0) cudaSetDevice(prev); }
};
#define ENTER(lat)                                                        \
    DeviceGuard guard_((lat)->device);                                    \
    if (!guard_.ok) return fail(QDP_ERR_CUDA, "cannot select CUDA device %d", (lat)->device)

// ---- lattice -------------------------------------------------------------------
// frees whatever a (possibly half-constructed) lattice owns, then the handle itself
static void release_lattice(qdp_lattice* l) {
    dev_free(l->partials, l->scratch_from_hook);
    dev_free(l->counter, l->scratch_from_hook);
    if (l->result_host) cudaFreeHost(l->result_host);
    for (int i = 0; i < 2; i++) {
        dev_free(l->stage[i], l->scratch_from_hook);
        if (l->ev_copied[i]) cudaEventDestroy(l->ev_copied[i]);
        if (l->ev_done[i]) cudaEventDestroy(l->ev_done[i]);
    }
    if (l->copy_stream) cudaStreamDestroy(l->copy_stream);
    l->magic = 0;
    delete l;
}

extern "C" int qdp_lattice_create(const int dims[4], int device, qdp_lattice** out) {
    if (!dims || !out) return fail(QDP_ERR_ARG, "qdp_lattice_create: null argument");
    long long V = 1;
    for (int i = 0; i < 4; i++) {
        if (dims[i] < 2 || (dims[i] & 1)) return fail(QDP_ERR_DIMS, "extent L%d = %d must be even and >= 2", i, dims[i]);
        V *= dims[i];
        if (V + 64 > (1ll << 31) / 36) return fail(QDP_ERR_DIMS, "volume too large for 32-bit element indices");
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
        return fail(QDP_ERR_CUDA, "no CUDA device: this library has no CPU fallback");
    if (device < 0 || device >= ndev) return fail(QDP_ERR_ARG, "device %d out of range (%d devices)", device, ndev);
    qdp_lattice* l = new (std::nothrow) qdp_lattice();
    if (!l) return fail(QDP_ERR_OOM, "host allocation failed");
    memset(l, 0, sizeof *l);
    l->magic = kLatMagic;
    l->device = device;
    memcpy(l->dims, dims, sizeof l->dims);
    l->geom = Geom::make(dims);
    DeviceGuard guard_(device);
    if (!guard_.ok) { delete l; return fail(QDP_ERR_CUDA, "cannot select CUDA device %d", device); }
    l->scratch_from_hook = g_alloc != nullptr;
    // partials: K <= 4 values per block (streaming reductions: at most kMaxPartialBlocks) or per
    // warp of 32 sites plus per group of kWarpGroup warps (fused kernels, reduce.cuh); qdp_sum
    // 2*36*64 values.  counters: one per group plus one.
    const size_t nwarp_max = (size_t)l->geom.V / 32 + 64 + 8192 /* persistent staged kernels: warps of one CTA per SM */, ngroup_max = nwarp_max / kWarpGroup + 2;
    size_t npart = (size_t)4 * kMaxPartialBlocks;
    if (npart < 4 * (nwarp_max + ngroup_max)) npart = 4 * (nwarp_max + ngroup_max);
    if (npart < (size_t)2 * 36 * 64) npart = (size_t)2 * 36 * 64;
    if (npart < (size_t)136 * dims[3]) npart = (size_t)136 * dims[3];   // qdp_baryon_timeslices: 8*16*L3 partials + 8*L3 results (qdp_inner_timeslices: 2*16*L3 + 2*L3)
    const size_t counter_bytes = (ngroup_max + 1) * sizeof(unsigned int);
    // everything below is released by release_lattice() on any failure
    auto attempt = [&]() -> int {
        int rc;
        void* p = nullptr;
        if ((rc = dev_alloc(npart * sizeof(double), &p)) != QDP_OK) return rc;
        l->partials = (double*)p;
        if ((rc = dev_alloc(counter_bytes, &p)) != QDP_OK) return rc;
        l->counter = (unsigned int*)p;
        CUDA_TRY(cudaMemset(l->counter, 0, counter_bytes));
        CUDA_TRY(cudaHostAlloc((void**)&l->result_host, (kResultSlots + 1) * sizeof(double), cudaHostAllocMapped));
        memset(l->result_host, 0, (kResultSlots + 1) * sizeof(double));
        CUDA_TRY(cudaHostGetDevicePointer((void**)&l->result_dev, l->result_host, 0));
        l->stage_bytes = (size_t)kStageSites * 36 * 16;
        for (int i = 0; i < 2; i++) {
            if ((rc = dev_alloc(l->stage_bytes, &l->stage[i])) != QDP_OK) return rc;
            CUDA_TRY(cudaEventCreateWithFlags(&l->ev_copied[i], cudaEventDisableTiming));
            CUDA_TRY(cudaEventCreateWithFlags(&l->ev_done[i], cudaEventDisableTiming));
        }
        CUDA_TRY(cudaStreamCreateWithFlags(&l->copy_stream, cudaStreamNonBlocking));
        return QDP_OK;
    };
    const int rc = attempt();
    if (rc != QDP_OK) { release_lattice(l); return rc; }
    *out = l;
    return QDP_OK;
}

extern "C" int qdp_lattice_destroy(qdp_lattice* l) {
    if (!ok_lat(l)) return fail(QDP_ERR_ARG, "qdp_lattice_destroy: not a lattice");
    if (l->live_fields) return fail(QDP_ERR_ARG, "qdp_lattice_destroy: %d fields still alive", l->live_fields);
    ENTER(l);
    cudaStreamSynchronize(l->stream);
    if (l->copy_stream) cudaStreamSynchronize(l->copy_stream);
    release_lattice(l);
    return QDP_OK;
}

extern "C" int qdp_lattice_set_stream(qdp_lattice* l, void* cuda_stream) {
    if (!ok_lat(l)) return fail(QDP_ERR_ARG, "qdp_lattice_set_stream: not a lattice");
    l->stream = (cudaStream_t)cuda_stream;
    return QDP_OK;
}

extern "C" int qdp_lattice_set_sweep_slab(qdp_lattice* l, int c2) {
    if (!ok_lat(l)) return fail(QDP_ERR_ARG, "qdp_lattice_set_sweep_slab: not a lattice");
    Geom& g = l->geom;
    if (c2 == 0) { g.slab_c2 = 0; g.slab_ipr = 0; return QDP_OK; }
    if (c2 < 0 || g.L2 % c2 != 0 || (g.s2 & 31) != 0)
        return fail(QDP_ERR_ARG, "qdp_lattice_set_sweep_slab: extent %d must divide L2 = %d and L0/2*L1 = %d be a multiple of 32",
                    c2, g.L2, g.s2);
    g.slab_c2 = c2; g.slab_ipr = g.s2 >> 5;
    return QDP_OK;
}

extern "C" int qdp_lattice_set_staged(qdp_lattice* l, int on) {
    if (!ok_lat(l)) return fail(QDP_ERR_ARG, "qdp_lattice_set_staged: not a lattice");
    l->geom.staged = on ? 1 : 0;
    return QDP_OK;
}

extern "C" int qdp_set_allocator(void* (*alloc)(size_t, void*), void (*free_)(void*, void*), void* ctx) {
    if ((alloc == nullptr) != (free_ == nullptr)) return fail(QDP_ERR_ARG, "qdp_set_allocator: need both alloc and free");
    g_alloc = alloc; g_free = free_; g_alloc_ctx = ctx;
    return QDP_OK;
}

extern "C" int qdp_lattice_volume(const qdp_lattice* l, int64_t* out) {
    if (!ok_lat(l) || !out) return fail(QDP_ERR_ARG, "qdp_lattice_volume: bad argument");
    *out = l->geom.V;
    return QDP_OK;
}

extern "C" int qdp_lattice_neighbor_table(qdp_lattice* l, int mu, int sign, int32_t* host_out) {
    if (!ok_lat(l) || !host_out) return fail(QDP_ERR_ARG, "qdp_lattice_neighbor_table: bad argument");
    if (mu < 0 || mu > 3 || (sign != 1 && sign != -1)) return fail(QDP_ERR_ARG, "mu must be 0..3 and sign +-1");
    ENTER(l);
    void* tmp = nullptr;
    CUDA_TRY(cudaMalloc(&tmp, (size_t)l->geom.V * sizeof(int32_t)));
    cudaError_t e = launch_neighbor_table(l->geom, mu, sign, (int32_t*)tmp, l->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(host_out, tmp, (size_t)l->geom.V * sizeof(int32_t), cudaMemcpyDeviceToHost, l->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(l->stream);
    cudaFree(tmp);
    CUDA_TRY(e);
    return QDP_OK;
}

extern "C" int qdp_lattice_parity_mask(qdp_lattice* l, uint8_t* host_out) {
    if (!ok_lat(l) || !host_out) return fail(QDP_ERR_ARG, "qdp_lattice_parity_mask: bad argument");
    ENTER(l);
    void* tmp = nullptr;
    CUDA_TRY(cudaMalloc(&tmp, (size_t)l->geom.V));
    cudaError_t e = launch_parity_mask(l->geom, (uint8_t*)tmp, l->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(host_out, tmp, (size_t)l->geom.V, cudaMemcpyDeviceToHost, l->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(l->stream);
    cudaFree(tmp);
    CUDA_TRY(e);
    return QDP_OK;
}

extern "C" int qdp_lattice_sync(qdp_lattice* l) {
    if (!ok_lat(l)) return fail(QDP_ERR_ARG, "qdp_lattice_sync: not a lattice");
    ENTER(l);
    CUDA_TRY(cudaStreamSynchronize(l->stream));
    return QDP_OK;
}

// ---- fields --------------------------------------------------------------------
extern "C" int qdp_field_bytes(const qdp_lattice* l, qdp_kind kind, qdp_prec prec, size_t* out) {
    if (!ok_lat(l) || !out) return fail(QDP_ERR_ARG, "qdp_field_bytes: bad argument");
    int nc = kind_ncomp(kind);
    if (!nc) return fail(QDP_ERR_KIND, "unknown field kind %d", (int)kind);
    if (prec != QDP_F32 && prec != QDP_F64) return fail(QDP_ERR_PREC, "unknown precision %d", (int)prec);
    *out = field_elems(l->geom, nc) * elem_bytes(prec);   // includes the padding lanes of the blocked layout
    return QDP_OK;
}

static int make_field(qdp_lattice* l, int kind, int prec, void* ptr, bool owned, qdp_field** out) {
    qdp_field* f = new (std::nothrow) qdp_field();
    if (!f) return fail(QDP_ERR_OOM, "host allocation failed");
    f->magic = kFieldMagic;
    f->lat = l; f->kind = kind; f->prec = prec; f->ncomp = kind_ncomp(kind);
    f->bytes = field_elems(l->geom, f->ncomp) * elem_bytes(prec);
    f->data = ptr; f->owned = owned; f->from_hook = owned && g_alloc != nullptr;
    l->live_fields++;
    *out = f;
    return QDP_OK;
}

extern "C" int qdp_field_alloc(qdp_lattice* l, qdp_kind kind, qdp_prec prec, qdp_field** out) {
    size_t bytes;
    int rc = qdp_field_bytes(l, kind, prec, &bytes);
    if (rc != QDP_OK) return rc;
    if (!out) return fail(QDP_ERR_ARG, "qdp_field_alloc: null out");
    ENTER(l);
    void* p = nullptr;
    if ((rc = dev_alloc(bytes, &p)) != QDP_OK) return rc;
    return make_field(l, kind, prec, p, true, out);
}

extern "C" int qdp_field_wrap(qdp_lattice* l, qdp_kind kind, qdp_prec prec, void* dev_ptr, size_t bytes,
                              qdp_field** out) {
    size_t need;
    int rc = qdp_field_bytes(l, kind, prec, &need);
    if (rc != QDP_OK) return rc;
    if (!out || !dev_ptr) return fail(QDP_ERR_ARG, "qdp_field_wrap: null argument");
    if (bytes < need) return fail(QDP_ERR_ARG, "qdp_field_wrap: %zu bytes given, %zu needed", bytes, need);
    if ((uintptr_t)dev_ptr % 256) return fail(QDP_ERR_ARG, "qdp_field_wrap: pointer not 256-byte aligned");
    return make_field(l, kind, prec, dev_ptr, false, out);
}

extern "C" int qdp_field_free(qdp_field* f) {
    if (!ok_field(f)) return fail(QDP_ERR_ARG, "qdp_field_free: not a field");
    ENTER(f->lat);
    // Kernels enqueued on the lattice's stream may still use the memory: wait for them before the
    // owner (this library, or the caller of qdp_field_wrap) can release or reuse it.
    cudaStreamSynchronize(f->lat->stream);
    if (f->owned) dev_free(f->data, f->from_hook);
    f->lat->live_fields--;
    f->magic = 0;
    delete f;
    return QDP_OK;
}

// Upload: chunks of kStageSites sites; the H2D copy of chunk k+1 (copy stream)
// overlaps the transpose of chunk k (lattice stream); two staging buffers.
extern "C" int qdp_field_upload(qdp_field* f, const void* host) {
    if (!ok_field(f) || !host) return fail(QDP_ERR_ARG, "qdp_field_upload: bad argument");
    qdp_lattice* l = f->lat;
    ENTER(l);
    const size_t site_bytes = (size_t)f->ncomp * elem_bytes(f->prec);
    const int V = l->geom.V;
    int k = 0;
    for (int begin = 0; begin < V; begin += kStageSites, k ^= 1) {
        int n = V - begin < kStageSites ? V - begin : kStageSites;
        // staging buffer k is free once the transpose that last read it is done
        CUDA_TRY(cudaStreamWaitEvent(l->copy_stream, l->ev_done[k], 0));
        CUDA_TRY(cudaMemcpyAsync(l->stage[k], (const char*)host + (size_t)begin * site_bytes, (size_t)n * site_bytes,
                                 cudaMemcpyHostToDevice, l->copy_stream));
        CUDA_TRY(cudaEventRecord(l->ev_copied[k], l->copy_stream));
        CUDA_TRY(cudaStreamWaitEvent(l->stream, l->ev_copied[k], 0));
        CUDA_TRY(launch_aos_to_soa(f->prec, l->geom, f->ncomp, l->stage[k], f->data, begin, n, l->stream));
        CUDA_TRY(cudaEventRecord(l->ev_done[k], l->stream));
    }
    CUDA_TRY(cudaStreamSynchronize(l->stream));
    return QDP_OK;
}

extern "C" int qdp_field_download(const qdp_field* f, void* host) {
    if (!ok_field(f) || !host) return fail(QDP_ERR_ARG, "qdp_field_download: bad argument");
    qdp_lattice* l = f->lat;
    ENTER(l);
    const size_t site_bytes = (size_t)f->ncomp * elem_bytes(f->prec);
    const int V = l->geom.V;
    int k = 0;
    for (int begin = 0; begin < V; begin += kStageSites, k ^= 1) {
        int n = V - begin < kStageSites ? V - begin : kStageSites;
        // staging buffer k is free once the D2H copy that last read it is done
        CUDA_TRY(cudaStreamWaitEvent(l->stream, l->ev_copied[k], 0));
        CUDA_TRY(launch_soa_to_aos(f->prec, l->geom, f->ncomp, f->data, l->stage[k], begin, n, l->stream));
        CUDA_TRY(cudaEventRecord(l->ev_done[k], l->stream));
        CUDA_TRY(cudaStreamWaitEvent(l->copy_stream, l->ev_done[k], 0));
        CUDA_TRY(cudaMemcpyAsync((char*)host + (size_t)begin * site_bytes, l->stage[k], (size_t)n * site_bytes,
                                 cudaMemcpyDeviceToHost, l->copy_stream));
        CUDA_TRY(cudaEventRecord(l->ev_copied[k], l->copy_stream));
    }
    CUDA_TRY(cudaStreamSynchronize(l->copy_stream));
    CUDA_TRY(cudaStreamSynchronize(l->stream));
    return QDP_OK;
}

static int check_pair(const char* who, const qdp_field* a, const qdp_field* b) {
    if (a->lat != b->lat) return fail(QDP_ERR_LATTICE, "%s: fields belong to different lattices", who);
    if (a->prec != b->prec) return fail(QDP_ERR_PREC, "%s: fields differ in precision", who);
    return QDP_OK;
}
static bool overlaps(const qdp_field* a, const qdp_field* b) {
    const char *pa = (const char*)a->data, *pb = (const char*)b->data;
    return pa < pb + b->bytes && pb < pa + a->bytes;
}

extern "C" int qdp_field_copy(qdp_field* dst, const qdp_field* src) {
    if (!ok_field(dst) || !ok_field(src)) return fail(QDP_ERR_ARG, "qdp_field_copy: not a field");
    int rc = check_pair("qdp_field_copy", dst, src);
    if (rc != QDP_OK) return rc;
    if (dst->kind != src->kind) return fail(QDP_ERR_KIND, "qdp_field_copy: kinds differ");
    ENTER(dst->lat);
    if (dst->data != src->data)
        CUDA_TRY(cudaMemcpyAsync(dst->data, src->data, src->bytes, cudaMemcpyDeviceToDevice, dst->lat->stream));
    return QDP_OK;
}

// ---- time-slice faces for an x3-slab decomposition (row f4 / SURVEY.md 8(e)) ---------------------
static int timeslice_common(const char* who, qdp_field* f, int t, void* dev_buf, size_t bytes, int subset, bool to_face) {
    if (!ok_field(f) || !dev_buf || !ok_subset(subset)) return fail(QDP_ERR_ARG, "%s: bad argument", who);
    qdp_lattice* l = f->lat;
    if (t < 0 || t >= l->geom.L3) return fail(QDP_ERR_ARG, "%s: t = %d outside 0..%d", who, t, l->geom.L3 - 1);
    const size_t need = (size_t)2 * f->ncomp * l->geom.s3 * elem_bytes(f->prec);
    if (bytes < need) return fail(QDP_ERR_ARG, "%s: buffer of %zu bytes, %zu needed", who, bytes, need);
    ENTER(l);
    CUDA_TRY(launch_timeslice(f->prec, l->geom, f->ncomp, f->data, dev_buf, t, subset, to_face, l->stream));
    return QDP_OK;
}
extern "C" int qdp_field_get_timeslice(const qdp_field* f, int t, void* dev_buf, size_t bytes) {
    return timeslice_common("qdp_field_get_timeslice", const_cast<qdp_field*>(f), t, dev_buf, bytes, QDP_ALL, true);
}
extern "C" int qdp_field_set_timeslice(qdp_field* f, int t, const void* dev_buf, size_t bytes, qdp_subset subset) {
    return timeslice_common("qdp_field_set_timeslice", f, t, const_cast<void*>(dev_buf), bytes, subset, false);
}
extern "C" int qdp_field_timeslice_bytes(const qdp_field* f, size_t* out) {
    if (!ok_field(f) || !out) return fail(QDP_ERR_ARG, "qdp_field_timeslice_bytes: bad argument");
    *out = (size_t)2 * f->ncomp * f->lat->geom.s3 * elem_bytes(f->prec);
    return QDP_OK;
}

// ---- expressions ---------------------------------------------------------------
extern "C" int qdp_shift(qdp_field* dst, const qdp_field* src, int mu, int sign, qdp_subset subset) {
    if (!ok_field(dst) || !ok_field(src)) return fail(QDP_ERR_ARG, "qdp_shift: not a field");
    if (mu < 0 || mu > 3 || (sign != 1 && sign != -1) || !ok_subset(subset))
        return fail(QDP_ERR_ARG, "qdp_shift: mu must be 0..3, sign +-1, subset 0..2");
    int rc = check_pair("qdp_shift", dst, src);
    if (rc != QDP_OK) return rc;
    if (dst->kind != src->kind) return fail(QDP_ERR_KIND, "qdp_shift: kinds differ");
    if (dst->kind == QDP_COMPLEX) return fail(QDP_ERR_KIND, "qdp_shift: not available for QDP_COMPLEX fields");
    if (overlaps(dst, src)) return fail(QDP_ERR_ALIAS, "qdp_shift: dst aliases src");
    ENTER(dst->lat);
    CUDA_TRY(launch_shift(dst->prec, dst->lat->geom, dst->ncomp, dst->data, src->data, mu, sign, subset, dst->lat->stream));
    return QDP_OK;
}

extern "C" int qdp_plaquette(const qdp_field* u, qdp_subset subset, double out[3]) {
    if (!ok_field(u) || !out || !ok_subset(subset)) return fail(QDP_ERR_ARG, "qdp_plaquette: bad argument");
    if (u->kind != QDP_GAUGE) return fail(QDP_ERR_KIND, "qdp_plaquette: u must be a gauge field");
    qdp_lattice* l = u->lat;
    ENTER(l);
    CUDA_TRY(launch_plaquette(u->prec, l->geom, u->data, subset, reduce_buf(l), l->stream));
    return fetch_result(l, 3, out);
}

extern "C" int qdp_ape_smear_step(qdp_field* u_out, const qdp_field* u_in, double alpha, int t_dir,
                                  qdp_subset subset) {
    if (!ok_field(u_out) || !ok_field(u_in) || !ok_subset(subset)) return fail(QDP_ERR_ARG, "qdp_ape_smear_step: bad argument");
    if (t_dir != 3 && t_dir != -1) return fail(QDP_ERR_ARG, "qdp_ape_smear_step: t_dir must be 3 or -1");
    if (u_out->kind != QDP_GAUGE || u_in->kind != QDP_GAUGE) return fail(QDP_ERR_KIND, "qdp_ape_smear_step: gauge fields needed");
    int rc = check_pair("qdp_ape_smear_step", u_out, u_in);
    if (rc != QDP_OK) return rc;
    if (overlaps(u_out, u_in)) return fail(QDP_ERR_ALIAS, "qdp_ape_smear_step: u_out aliases u_in");
    qdp_lattice* l = u_out->lat;
    ENTER(l);
    CUDA_TRY(launch_ape(u_out->prec, l->geom, u_out->data, u_in->data, alpha, t_dir, subset, l->stream));
    return QDP_OK;
}

extern "C" int qdp_matmul(qdp_field* dst, int slot_d, const qdp_field* a, int slot_a, int adj_a,
                          const qdp_field* b, int slot_b, int adj_b, int mu, int sign, qdp_subset subset) {
    if (!ok_field(dst) || !ok_field(a) || !ok_field(b) || !ok_subset(subset)) return fail(QDP_ERR_ARG, "qdp_matmul: bad argument");
    if (dst->kind == QDP_FERMION || a->kind == QDP_FERMION || b->kind == QDP_FERMION)
        return fail(QDP_ERR_KIND, "qdp_matmul: operands are colour matrices or links of gauge fields");
    auto slots = [](const qdp_field* f) { return f->ncomp / 9; };
    if (slot_d < 0 || slot_d >= slots(dst) || slot_a < 0 || slot_a >= slots(a) || slot_b < 0 || slot_b >= slots(b))
        return fail(QDP_ERR_ARG, "qdp_matmul: slot out of range");
    if (mu < -1 || mu > 3 || (mu >= 0 && sign != 1 && sign != -1)) return fail(QDP_ERR_ARG, "qdp_matmul: bad mu / sign");
    int rc = check_pair("qdp_matmul", dst, a);
    if (rc == QDP_OK) rc = check_pair("qdp_matmul", dst, b);
    if (rc != QDP_OK) return rc;
    if (mu >= 0 && overlaps(dst, b) && (dst->data != b->data || slot_d == slot_b))
        return fail(QDP_ERR_ALIAS, "qdp_matmul: dst slot aliases the shifted operand");
    if ((overlaps(dst, a) && dst->data != a->data) || (overlaps(dst, b) && dst->data != b->data))
        return fail(QDP_ERR_ALIAS, "qdp_matmul: dst partially overlaps an operand");
    qdp_lattice* l = dst->lat;
    ENTER(l);
    CUDA_TRY(launch_matmul(dst->prec, l->geom, dst->data, dst->ncomp, slot_d, a->data, a->ncomp, slot_a, adj_a != 0,
                           b->data, b->ncomp, slot_b, adj_b != 0, mu, sign, subset, l->stream));
    return QDP_OK;
}

extern "C" int qdp_matvec(qdp_field* chi, const qdp_field* a, int slot_a, int adj_a, const qdp_field* psi,
                          int mu, int sign, qdp_subset subset) {
    if (!ok_field(chi) || !ok_field(a) || !ok_field(psi) || !ok_subset(subset)) return fail(QDP_ERR_ARG, "qdp_matvec: bad argument");
    if (chi->kind != QDP_FERMION || psi->kind != QDP_FERMION || a->kind == QDP_FERMION)
        return fail(QDP_ERR_KIND, "qdp_matvec: need (fermion, colour matrix or gauge, fermion)");
    if (slot_a < 0 || slot_a >= a->ncomp / 9) return fail(QDP_ERR_ARG, "qdp_matvec: slot out of range");
    if (mu < -1 || mu > 3 || (mu >= 0 && sign != 1 && sign != -1)) return fail(QDP_ERR_ARG, "qdp_matvec: bad mu / sign");
    int rc = check_pair("qdp_matvec", chi, psi);
    if (rc == QDP_OK) rc = check_pair("qdp_matvec", chi, a);
    if (rc != QDP_OK) return rc;
    if (overlaps(chi, psi) && (mu >= 0 || chi->data != psi->data))
        return fail(QDP_ERR_ALIAS, "qdp_matvec: chi aliases the shifted psi");
    qdp_lattice* l = chi->lat;
    ENTER(l);
    CUDA_TRY(launch_matvec(chi->prec, l->geom, chi->data, a->data, a->ncomp, slot_a, adj_a != 0, psi->data, mu, sign,
                           subset, l->stream));
    return QDP_OK;
}

static int reunit_common(const char* who, qdp_field* u_out, const qdp_field* u_in, int method, int iters, qdp_subset subset) {
    if (!ok_field(u_out) || !ok_field(u_in) || !ok_subset(subset)) return fail(QDP_ERR_ARG, "%s: bad argument", who);
    if ((u_in->kind != QDP_GAUGE && u_in->kind != QDP_COLOR_MATRIX) || u_out->kind != u_in->kind)
        return fail(QDP_ERR_KIND, "%s: need two gauge fields or two colour matrices", who);
    int rc = check_pair(who, u_out, u_in);
    if (rc != QDP_OK) return rc;
    if (u_out != u_in && u_out->data != u_in->data && overlaps(u_out, u_in))
        return fail(QDP_ERR_ALIAS, "%s: u_out partially overlaps u_in", who);
    qdp_lattice* l = u_out->lat;
    ENTER(l);
    CUDA_TRY(launch_reunit(u_out->prec, l->geom, u_out->ncomp, u_out->data, u_in->data, method, subset, l->stream, iters));
    return QDP_OK;
}
extern "C" int qdp_reunitarize(qdp_field* u_out, const qdp_field* u_in, int method, qdp_subset subset) {
    if (method != QDP_REUNIT_POLAR && method != QDP_REUNIT_GRAM_SCHMIDT)
        return fail(QDP_ERR_ARG, "qdp_reunitarize: unknown method %d", method);
    return reunit_common("qdp_reunitarize", u_out, u_in, method, 0, subset);
}
extern "C" int qdp_project_max_retr(qdp_field* u_out, const qdp_field* u_in, int iterations, qdp_subset subset) {
    if (iterations < 0 || iterations > 1000) return fail(QDP_ERR_ARG, "qdp_project_max_retr: iterations must be 0..1000");
    return reunit_common("qdp_project_max_retr", u_out, u_in, 2, iterations, subset);
}

static int hop_common(const char* who, qdp_field* chi, const qdp_field* u, const qdp_field* psi, qdp_subset subset,
                      bool axpy, double a, double b, double* norm2_out, int ndir = 4) {
    if (!ok_field(chi) || !ok_field(u) || !ok_field(psi) || !ok_subset(subset)) return fail(QDP_ERR_ARG, "%s: bad argument", who);
    if (chi->kind != QDP_FERMION || psi->kind != QDP_FERMION || u->kind != QDP_GAUGE)
        return fail(QDP_ERR_KIND, "%s: need (fermion, gauge, fermion)", who);
    int rc = check_pair(who, chi, psi);
    if (rc == QDP_OK) rc = check_pair(who, chi, u);
    if (rc != QDP_OK) return rc;
    if (overlaps(chi, psi)) return fail(QDP_ERR_ALIAS, "%s: chi aliases psi", who);
    qdp_lattice* l = chi->lat;
    ENTER(l);
    CUDA_TRY(launch_hop(chi->prec, l->geom, chi->data, u->data, psi->data, subset, axpy, a, b, norm2_out != nullptr,
                        reduce_buf(l), l->stream, ndir));
    if (norm2_out) return fetch_result(l, 1, norm2_out);
    return QDP_OK;
}

extern "C" int qdp_hop(qdp_field* chi, const qdp_field* u, const qdp_field* psi, qdp_subset subset) {
    return hop_common("qdp_hop", chi, u, psi, subset, false, 0.0, 1.0, nullptr);
}
extern "C" int qdp_axpy_hop(qdp_field* chi, double a, double b, const qdp_field* u, const qdp_field* psi,
                            qdp_subset subset, double* norm2_out) {
    return hop_common("qdp_axpy_hop", chi, u, psi, subset, true, a, b, norm2_out);
}
extern "C" int qdp_smear_hop(qdp_field* chi, double a, double b, const qdp_field* u, const qdp_field* psi,
                             int t_dir, qdp_subset subset, double* norm2_out) {
    if (t_dir != 3 && t_dir != -1) return fail(QDP_ERR_ARG, "qdp_smear_hop: t_dir must be 3 or -1");
    return hop_common("qdp_smear_hop", chi, u, psi, subset, true, a, b, norm2_out, t_dir == 3 ? 3 : 4);
}

extern "C" int qdp_norm2(const qdp_field* f, qdp_subset subset, double* out) {
    if (!ok_field(f) || !out || !ok_subset(subset)) return fail(QDP_ERR_ARG, "qdp_norm2: bad argument");
    if (f->kind == QDP_COMPLEX) return fail(QDP_ERR_KIND, "qdp_norm2: not available for QDP_COMPLEX fields (use qdp_sum)");
    qdp_lattice* l = f->lat;
    ENTER(l);
    CUDA_TRY(launch_norm2(f->prec, l->geom, f->ncomp, f->data, subset, reduce_buf(l), l->stream));
    return fetch_result(l, 1, out);
}

extern "C" int qdp_inner(const qdp_field* a, const qdp_field* b, qdp_subset subset, double out[2]) {
    if (!ok_field(a) || !ok_field(b) || !out || !ok_subset(subset)) return fail(QDP_ERR_ARG, "qdp_inner: bad argument");
    int rc = check_pair("qdp_inner", a, b);
    if (rc != QDP_OK) return rc;
    if (a->kind != b->kind) return fail(QDP_ERR_KIND, "qdp_inner: kinds differ");
    if (a->kind == QDP_COMPLEX) return fail(QDP_ERR_KIND, "qdp_inner: not available for QDP_COMPLEX fields");
    qdp_lattice* l = a->lat;
    ENTER(l);
    CUDA_TRY(launch_inner(a->prec, l->geom, a->ncomp, a->data, b->data, subset, reduce_buf(l), l->stream));
    return fetch_result(l, 2, out);
}

extern "C" int qdp_axpby(qdp_field* dst, double a, const qdp_field* x, double b, const qdp_field* y,
                         qdp_subset subset, double* norm2_out) {
    if (!ok_field(dst) || !ok_field(x) || !ok_field(y) || !ok_subset(subset)) return fail(QDP_ERR_ARG, "qdp_axpby: bad argument");
    int rc = check_pair("qdp_axpby", dst, x);
    if (rc == QDP_OK) rc = check_pair("qdp_axpby", dst, y);
    if (rc != QDP_OK) return rc;
    if (dst->kind != x->kind || dst->kind != y->kind) return fail(QDP_ERR_KIND, "qdp_axpby: kinds differ");
    if (dst->kind == QDP_COMPLEX) return fail(QDP_ERR_KIND, "qdp_axpby: not available for QDP_COMPLEX fields");
    if ((overlaps(dst, x) && dst->data != x->data) || (overlaps(dst, y) && dst->data != y->data))
        return fail(QDP_ERR_ALIAS, "qdp_axpby: dst partially overlaps an operand");
    qdp_lattice* l = dst->lat;
    ENTER(l);
    CUDA_TRY(launch_axpby(dst->prec, l->geom, dst->ncomp, dst->data, x->data, y->data, a, b, subset,
                          norm2_out != nullptr, reduce_buf(l), l->stream));
    if (norm2_out) return fetch_result(l, 1, norm2_out);
    return QDP_OK;
}

// Gamma(n) as a phased permutation, built from the four base matrices of the header:
// (A B) has perm[r] = pB[pA[r]] and phase phA[r] + phB[pA[r]] (phases count powers of i).
static SpinMatrix spin_matrix(int n) {
    static const int bperm[4][4] = { {3, 2, 1, 0}, {3, 2, 1, 0}, {2, 3, 0, 1}, {2, 3, 0, 1} };
    static const int bph[4][4] = { {1, 1, 3, 3}, {2, 0, 0, 2}, {1, 3, 3, 1}, {0, 0, 0, 0} };
    SpinMatrix m = {{0, 1, 2, 3}, {0, 0, 0, 0}};
    for (int mu = 0; mu < 4; mu++) {
        if (!((n >> mu) & 1)) continue;
        SpinMatrix r;
        for (int row = 0; row < 4; row++) {
            r.perm[row] = bperm[mu][m.perm[row]];
            r.ph[row] = (m.ph[row] + bph[mu][m.perm[row]]) & 3;
        }
        m = r;
    }
    return m;
}

static int inner_timeslices_common(const char* who, const qdp_field* a, const qdp_field* b, qdp_subset subset, double* out,
                                   const SpinMatrix* gamma);

extern "C" int qdp_inner_timeslices(const qdp_field* a, const qdp_field* b, qdp_subset subset, double* out) {
    return inner_timeslices_common("qdp_inner_timeslices", a, b, subset, out, nullptr);
}
extern "C" int qdp_inner_timeslices_gamma(const qdp_field* a, const qdp_field* b, int n, qdp_subset subset, double* out) {
    if (n < 0 || n > 15) return fail(QDP_ERR_ARG, "qdp_inner_timeslices_gamma: n must be 0..15");
    if (ok_field(a) && ok_field(b) && (a->kind != QDP_FERMION || b->kind != QDP_FERMION))
        return fail(QDP_ERR_KIND, "qdp_inner_timeslices_gamma: fermion fields needed");
    const SpinMatrix m = spin_matrix(n);
    return inner_timeslices_common("qdp_inner_timeslices_gamma", a, b, subset, out, &m);
}

static int inner_timeslices_common(const char* who, const qdp_field* a, const qdp_field* b, qdp_subset subset, double* out,
                                   const SpinMatrix* gamma) {
    if (!ok_field(a) || !ok_field(b) || !out || !ok_subset(subset))
        return fail(QDP_ERR_ARG, "%s: bad argument", who);
    int rc = check_pair(who, a, b);
    if (rc != QDP_OK) return rc;
    if (a->kind != b->kind) return fail(QDP_ERR_KIND, "%s: kinds differ", who);
    if (a->kind == QDP_COMPLEX) return fail(QDP_ERR_KIND, "%s: not available for QDP_COMPLEX fields", who);
    qdp_lattice* l = a->lat;
    ENTER(l);
    const int L3 = l->geom.L3;
    double* out_dev = l->partials + (size_t)2 * 16 * L3;   // behind the per-block partials
    CUDA_TRY(launch_inner_timeslices(a->prec, l->geom, a->ncomp, a->data, b->data, subset, l->partials, out_dev,
                                     l->stream, gamma));
    CUDA_TRY(cudaMemcpyAsync(out, out_dev, (size_t)2 * L3 * sizeof(double), cudaMemcpyDeviceToHost, l->stream));
    CUDA_TRY(cudaStreamSynchronize(l->stream));
    return QDP_OK;
}

extern "C" int qdp_baryon_timeslices(const qdp_field* const* q1, const qdp_field* const* q2, const qdp_field* const* q3,
                                     int nsrc, int n, qdp_subset subset, double* out) {
    if (!q1 || !q2 || !q3 || !out || !ok_subset(subset)) return fail(QDP_ERR_ARG, "qdp_baryon_timeslices: bad argument");
    if (nsrc != 1 && nsrc != 3) return fail(QDP_ERR_ARG, "qdp_baryon_timeslices: nsrc must be 1 or 3");
    if (n < 0 || n > 15) return fail(QDP_ERR_ARG, "qdp_baryon_timeslices: n must be 0..15");
    const qdp_field* const* qs[3] = {q1, q2, q3};
    const void* ptr[3][3] = {};
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < nsrc; j++) {
            const qdp_field* f = qs[i][j];
            if (!ok_field(f)) return fail(QDP_ERR_ARG, "qdp_baryon_timeslices: not a field");
            if (f->kind != QDP_FERMION) return fail(QDP_ERR_KIND, "qdp_baryon_timeslices: fermion fields needed");
            int rc = check_pair("qdp_baryon_timeslices", qs[0][0], f);
            if (rc != QDP_OK) return rc;
            ptr[i][j] = f->data;
        }
    qdp_lattice* l = q1[0]->lat;
    ENTER(l);
    const SpinMatrix m = spin_matrix(n);
    const int L3 = l->geom.L3;
    double* out_dev = l->partials + (size_t)8 * 16 * L3;   // behind the per-block partials
    CUDA_TRY(launch_baryon_timeslices(q1[0]->prec, l->geom, ptr, nsrc, m, subset, l->partials, out_dev, l->stream));
    CUDA_TRY(cudaMemcpyAsync(out, out_dev, (size_t)8 * L3 * sizeof(double), cudaMemcpyDeviceToHost, l->stream));
    CUDA_TRY(cudaStreamSynchronize(l->stream));
    return QDP_OK;
}

extern "C" int qdp_sum(const qdp_field* f, qdp_subset subset, double* out) {
    if (!ok_field(f) || !out || !ok_subset(subset)) return fail(QDP_ERR_ARG, "qdp_sum: bad argument");
    qdp_lattice* l = f->lat;
    ENTER(l);
    CUDA_TRY(launch_sum(f->prec, l->geom, f->ncomp, f->data, subset, l->partials, l->result_dev, l->stream));
    return fetch_result_sync(l, 2 * f->ncomp, out);
}

// ---- the expression layer (csrc/expr.cuh, expr.cu): named instantiations --------------------------
extern "C" int qdp_expr_plaquette(const qdp_field* u, qdp_subset subset, double out[3]) {
    if (!ok_field(u) || !out || !ok_subset(subset)) return fail(QDP_ERR_ARG, "qdp_expr_plaquette: bad argument");
    if (u->kind != QDP_GAUGE) return fail(QDP_ERR_KIND, "qdp_expr_plaquette: u must be a gauge field");
    qdp_lattice* l = u->lat;
    ENTER(l);
    CUDA_TRY(launch_expr_plaquette(u->prec, l->geom, u->data, subset, reduce_buf(l), l->stream));
    double r[2];
    int rc = fetch_result(l, 2, r);
    if (rc != QDP_OK) return rc;
    out[0] = 0.5 * (r[0] + r[1]); out[1] = r[0]; out[2] = r[1];
    return QDP_OK;
}

static int expr_staple_common(const char* who, qdp_field* dst, const qdp_field* u, int mu, int t_dir, bool blend, double alpha,
                              qdp_subset subset) {
    if (!ok_field(dst) || !ok_field(u) || !ok_subset(subset)) return fail(QDP_ERR_ARG, "%s: bad argument", who);
    if (t_dir != 3 && t_dir != -1) return fail(QDP_ERR_ARG, "%s: t_dir must be 3 or -1", who);
    if (mu < 0 || mu > 3 || mu == t_dir) return fail(QDP_ERR_ARG, "%s: mu must be a smeared direction", who);
    int rc = check_pair(who, dst, u);
    if (rc != QDP_OK) return rc;
    if (dst->kind != QDP_COLOR_MATRIX || u->kind != QDP_GAUGE) return fail(QDP_ERR_KIND, "%s: dst colour matrix, u gauge field", who);
    qdp_lattice* l = u->lat;
    ENTER(l);
    CUDA_TRY(launch_expr_staple(u->prec, l->geom, dst->data, u->data, mu, t_dir, blend, alpha, subset, l->stream));
    return QDP_OK;
}
extern "C" int qdp_expr_staple(qdp_field* dst, const qdp_field* u, int mu, int t_dir, qdp_subset subset) {
    return expr_staple_common("qdp_expr_staple", dst, u, mu, t_dir, false, 0.0, subset);
}
extern "C" int qdp_expr_ape_blend(qdp_field* dst, const qdp_field* u, int mu, double alpha, int t_dir, qdp_subset subset) {
    return expr_staple_common("qdp_expr_ape_blend", dst, u, mu, t_dir, true, alpha, subset);
}

static int expr_trace_mul_common(const char* who, qdp_field* dst, const qdp_field* a, int slot_a, int adj_a, const qdp_field* b,
                                 int slot_b, int adj_b, int mu, int sign, qdp_subset subset, double* out) {
    if (!ok_field(a) || !ok_field(b) || !ok_subset(subset) || (dst && !ok_field(dst)) || (!dst && !out))
        return fail(QDP_ERR_ARG, "%s: bad argument", who);
    if (mu > 3 || (mu >= 0 && sign != 1 && sign != -1)) return fail(QDP_ERR_ARG, "%s: mu must be -1..3, sign +-1", who);
    int rc = check_pair(who, a, b);
    if (rc == QDP_OK && dst) rc = check_pair(who, dst, a);
    if (rc != QDP_OK) return rc;
    auto matrix_kind = [](const qdp_field* f) { return f->kind == QDP_COLOR_MATRIX || f->kind == QDP_GAUGE; };
    if (!matrix_kind(a) || !matrix_kind(b) || (dst && dst->kind != QDP_COMPLEX))
        return fail(QDP_ERR_KIND, "%s: a, b colour matrices or gauge fields, dst QDP_COMPLEX", who);
    if (slot_a < 0 || slot_a >= a->ncomp / 9 || slot_b < 0 || slot_b >= b->ncomp / 9) return fail(QDP_ERR_ARG, "%s: slot out of range", who);
    qdp_lattice* l = a->lat;
    ENTER(l);
    CUDA_TRY(launch_expr_trace_mul(a->prec, l->geom, dst ? dst->data : nullptr, a->data, a->ncomp, slot_a, adj_a != 0, b->data,
                                   b->ncomp, slot_b, adj_b != 0, mu, sign, subset, reduce_buf(l), l->stream));
    return dst ? QDP_OK : fetch_result(l, 2, out);
}
extern "C" int qdp_expr_trace_mul(qdp_field* dst, const qdp_field* a, int slot_a, int adj_a, const qdp_field* b, int slot_b,
                                  int adj_b, int mu, int sign, qdp_subset subset) {
    if (!dst) return fail(QDP_ERR_ARG, "qdp_expr_trace_mul: bad argument");
    return expr_trace_mul_common("qdp_expr_trace_mul", dst, a, slot_a, adj_a, b, slot_b, adj_b, mu, sign, subset, nullptr);
}
extern "C" int qdp_expr_sum_trace_mul(const qdp_field* a, int slot_a, int adj_a, const qdp_field* b, int slot_b, int adj_b,
                                      int mu, int sign, qdp_subset subset, double out[2]) {
    return expr_trace_mul_common("qdp_expr_sum_trace_mul", nullptr, a, slot_a, adj_a, b, slot_b, adj_b, mu, sign, subset, out);
}

// ---- run-time expressions (row f1, second step; jit.cu) -------------------------------------------------------
static int jit_ncomp_of_kind(int kind) { return kind == QDP_COLOR_MATRIX ? 9 : (kind == QDP_GAUGE ? 36 : (kind == QDP_FERMION ? 12 : 0)); }

extern "C" int qdp_expr_jit_kind(const char* expr, const int* field_kinds, int nfields, int nscalars, int* kind_out) {
    if (!expr || !kind_out || nfields < 0 || nfields > 4 || (nfields && !field_kinds)) return fail(QDP_ERR_ARG, "qdp_expr_jit_kind: bad argument");
    int ncomp[4] = {0, 0, 0, 0};
    for (int k = 0; k < nfields; k++)
        if (!(ncomp[k] = jit_ncomp_of_kind(field_kinds[k]))) return fail(QDP_ERR_KIND, "qdp_expr_jit_kind: field arguments must be colour matrices, gauge fields or fermions");
    JitExpr e;
    std::string err;
    if (jit_parse(expr, ncomp, nfields, nscalars, &e, &err) != 0) return fail(QDP_ERR_ARG, "qdp_expr_jit_kind: %s", err.c_str());
    *kind_out = e.kind;
    return QDP_OK;
}

extern "C" int qdp_expr_jit_compile(const char* expr, const int* field_kinds, int nfields, int nscalars, qdp_prec prec, int sum,
                                    size_t* cubin_bytes) {
    if (!expr || nfields < 0 || nfields > 4 || (nfields && !field_kinds) || (prec != QDP_F32 && prec != QDP_F64))
        return fail(QDP_ERR_ARG, "qdp_expr_jit_compile: bad argument");
    int ncomp[4] = {0, 0, 0, 0};
    for (int k = 0; k < nfields; k++)
        if (!(ncomp[k] = jit_ncomp_of_kind(field_kinds[k]))) return fail(QDP_ERR_KIND, "qdp_expr_jit_compile: field arguments must be colour matrices, gauge fields or fermions");
    JitExpr e;
    std::string err;
    if (jit_parse(expr, ncomp, nfields, nscalars, &e, &err) != 0) return fail(QDP_ERR_ARG, "qdp_expr_jit_compile: %s", err.c_str());
    if (sum && (e.kind == JIT_MAT || e.kind == JIT_SPINOR)) return fail(QDP_ERR_ARG, "qdp_expr_jit_compile: a sum needs a real or complex expression");
    if (!sum && e.kind == JIT_REAL) return fail(QDP_ERR_ARG, "qdp_expr_jit_compile: an assignment needs a matrix or complex expression");
    if (jit_compile_only(e, prec == QDP_F64, sum != 0, cubin_bytes, &err) != 0) return fail(QDP_ERR_CUDA, "qdp_expr_jit_compile: %s", err.c_str());
    return QDP_OK;
}

extern "C" int64_t qdp_expr_jit_compilations(void) { return jit_compilations(); }

static int jit_common(const char* who, qdp_field* dst, int slot_d, const char* expr, const qdp_field* const* fields, int nfields,
                      const double* scalars, int nscalars, qdp_subset subset, double* out) {
    if (!expr || nfields < 1 || nfields > 4 || !fields || nscalars < 0 || nscalars > 4 || (nscalars && !scalars) || !ok_subset(subset) ||
        (dst && !ok_field(dst)) || (!dst && !out))
        return fail(QDP_ERR_ARG, "%s: bad argument", who);
    int ncomp[4] = {0, 0, 0, 0};
    ex::Args a = {};
    for (int k = 0; k < nfields; k++) {
        if (!ok_field(fields[k])) return fail(QDP_ERR_ARG, "%s: field argument %d is not a field", who, k);
        const int rc = check_pair(who, fields[0], fields[k]);
        if (rc != QDP_OK) return rc;
        if (!(ncomp[k] = jit_ncomp_of_kind(fields[k]->kind))) return fail(QDP_ERR_KIND, "%s: field arguments must be colour matrices, gauge fields or fermions", who);
        a.f[k] = fields[k]->data;
        a.ncomp[k] = ncomp[k];
    }
    for (int k = 0; k < nscalars; k++) a.sc[k] = scalars[k];
    a.mu = -1;
    JitExpr e;
    std::string err;
    if (jit_parse(expr, ncomp, nfields, nscalars, &e, &err) != 0) return fail(QDP_ERR_ARG, "%s: %s", who, err.c_str());
    qdp_lattice* l = fields[0]->lat;
    int nd = 0, cd = 0;
    if (dst) {
        const int rc = check_pair(who, dst, fields[0]);
        if (rc != QDP_OK) return rc;
        if (e.kind == JIT_MAT) {
            if (dst->kind != QDP_COLOR_MATRIX && dst->kind != QDP_GAUGE) return fail(QDP_ERR_KIND, "%s: a matrix expression needs a colour-matrix or gauge destination", who);
            if (slot_d < 0 || slot_d >= dst->ncomp / 9) return fail(QDP_ERR_ARG, "%s: destination slot out of range", who);
            cd = slot_d * 9;
        } else if (e.kind == JIT_CPLX) {
            if (dst->kind != QDP_COMPLEX) return fail(QDP_ERR_KIND, "%s: a complex expression needs a QDP_COMPLEX destination", who);
        } else if (e.kind == JIT_SPINOR) {
            if (dst->kind != QDP_FERMION) return fail(QDP_ERR_KIND, "%s: a spinor expression needs a QDP_FERMION destination", who);
        } else return fail(QDP_ERR_ARG, "%s: a real expression cannot be assigned (wrap it in a sum)", who);
        nd = dst->ncomp;
        if (e.has_shift)
            for (int k = 0; k < nfields; k++)
                if ((e.fields_used >> k & 1) && overlaps(dst, fields[k]))
                    return fail(QDP_ERR_ALIAS, "%s: the destination is an operand of an expression that reads neighbour sites", who);
    } else if (e.kind == JIT_MAT || e.kind == JIT_SPINOR) return fail(QDP_ERR_ARG, "%s: a sum needs a real or complex expression", who);
    ENTER(l);
    cudaError_t ce = dst ? jit_launch_assign(e, fields[0]->prec == QDP_F64, l->geom, a, dst->data, nd, cd, subset, l->stream, &err)
                         : jit_launch_sum(e, fields[0]->prec == QDP_F64, l->geom, a, subset, reduce_buf(l), l->stream, &err);
    if (ce != cudaSuccess) return fail(QDP_ERR_CUDA, "%s: %s", who, err.empty() ? cudaGetErrorString(ce) : err.c_str());
    return dst ? QDP_OK : fetch_result(l, 2, out);
}
extern "C" int qdp_expr_jit_assign(qdp_field* dst, int slot_d, const char* expr, const qdp_field* const* fields, int nfields,
                                   const double* scalars, int nscalars, qdp_subset subset) {
    if (!dst) return fail(QDP_ERR_ARG, "qdp_expr_jit_assign: bad argument");
    return jit_common("qdp_expr_jit_assign", dst, slot_d, expr, fields, nfields, scalars, nscalars, subset, nullptr);
}
extern "C" int qdp_expr_jit_sum(const char* expr, const qdp_field* const* fields, int nfields, const double* scalars, int nscalars,
                                qdp_subset subset, double out[2]) {
    return jit_common("qdp_expr_jit_sum", nullptr, 0, expr, fields, nfields, scalars, nscalars, subset, out);
}

#ifdef QDP_BOUNDS_CHECK
// Only in the bounds-checked build (not declared in the header): three deliberately wrong site addresses
// (past the end, a padding lane of a ragged lattice or the last real site + 1, a component outside the
// site) so that tests/test_gpu_bounds.py can see the checker fire.
namespace qdp {
__global__ void bounds_selftest_kernel(Geom g, double2* f) {
    volatile double2* a = site_ptr(f, 12, 0, 2 * g.Vhp);
    volatile double2* b = site_ptr(f, 12, 0, g.Vhp + g.Vh);
    volatile double2* c = site_ptr(f, 12, 12, 0);
    (void)a; (void)b; (void)c;
}
}  // namespace qdp
extern "C" int qdp_bc_selftest(qdp_field* f) {
    if (!ok_field(f) || f->kind != QDP_FERMION || f->prec != QDP_F64) return QDP_ERR_ARG;
    ENTER(f->lat);
    qdp::bounds_selftest_kernel<<<1, 1, 0, f->lat->stream>>>(f->lat->geom, (double2*)f->data);
    CUDA_TRY(cudaStreamSynchronize(f->lat->stream));
    return QDP_OK;
}
#endif

extern "C" int64_t qdp_kernel_launch_count(void) { return g_launch_count.load(); }

extern "C" const char* qdp_last_error(void) { return t_err; }
