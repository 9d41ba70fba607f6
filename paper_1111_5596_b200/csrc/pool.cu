// pool.cu -- device memory pool and LRU residency manager ("the pool manager
// grabs a large chunk of GPU memory at start-up", "the cache ... spills least-recently-used objects").  Host-side C++;
// the only device work is the raw copy of an object's bytes when it is paged in or spilled.
//
// On a 180 GB B200 the BASELINE workloads stay resident for their lifetime, so nothing on the hot path uses this; it is
// the paper's mechanism for working sets larger than device memory, rebuilt as a library component:
//   pool:  one up-front cudaMalloc, sub-allocated first-fit (lowest offset) in units of 256 bytes, free blocks coalesced;
//          qdp_pool_hook_alloc/free have the signature of qdp_set_allocator, so fields and the library's scratch can
//          live in the pool (the paper redirects QUDA's allocations into its pool the same way).
//   cache: an object = `bytes` of device-layout data with a caller-owned host buffer (pinned for speed).
//          qdp_cache_acquire pages it in (allocating from the pool; when nothing fits, the least recently acquired
//          unlocked resident objects are spilled one at a time -- copied back to their host buffers if they were
//          acquired for writing -- until a block fits), locks it and makes it the most recently used.
// device = -1 creates an address-range-only pool (no memory is allocated or touched): the allocator and the eviction
// policy are pure host logic and are tested without a GPU against oracle/pool_model.py.
#include <algorithm>
#include <cstdint>
#include <cstring>
#include <list>
#include <map>
#include <new>
#include <vector>

#include "../../include/qdp_b200.h"
#include "internal.h"

namespace qdp { int set_error(int code, const char* msg); }

static const uint32_t kPoolMagic = 0x51445033u, kCachedMagic = 0x51445034u;
static const size_t kGran = 256, kNone = ~(size_t)0;

struct qdp_cached {
    uint32_t magic;
    qdp_pool* pool;
    void* host;
    size_t bytes;
    size_t off;          // kNone: not resident
    int locks;
    bool dirty;
    int64_t id;
};
struct FreeBlock { size_t off, size; };
struct qdp_pool {
    uint32_t magic;
    int device;
    char* base;
    size_t cap;
    std::vector<FreeBlock> free_;        // sorted by offset, neighbours coalesced
    std::map<size_t, size_t> used_;      // offset -> size
    std::list<qdp_cached*> lru_;         // front = most recently acquired; every registered object is in it
    std::vector<int64_t> evlog;          // ids of spilled objects, in order
    int64_t next_id;
};

static bool ok_pool(const qdp_pool* p) { return p && p->magic == kPoolMagic; }
static bool ok_cached(const qdp_cached* c) { return c && c->magic == kCachedMagic && ok_pool(c->pool); }
static size_t round_up(size_t b) { return (std::max<size_t>(b, 1) + kGran - 1) / kGran * kGran; }

static size_t first_fit(qdp_pool* p, size_t need) {
    for (size_t i = 0; i < p->free_.size(); i++)
        if (p->free_[i].size >= need) {
            const size_t off = p->free_[i].off;
            if (p->free_[i].size == need) p->free_.erase(p->free_.begin() + i);
            else { p->free_[i].off += need; p->free_[i].size -= need; }
            p->used_[off] = need;
            return off;
        }
    return kNone;
}
static void give_back(qdp_pool* p, size_t off) {
    auto it = p->used_.find(off);
    FreeBlock b{off, it->second};
    p->used_.erase(it);
    auto pos = std::lower_bound(p->free_.begin(), p->free_.end(), b, [](const FreeBlock& x, const FreeBlock& y) { return x.off < y.off; });
    pos = p->free_.insert(pos, b);
    if (pos + 1 != p->free_.end() && pos->off + pos->size == (pos + 1)->off) { pos->size += (pos + 1)->size; p->free_.erase(pos + 1); }
    if (pos != p->free_.begin() && (pos - 1)->off + (pos - 1)->size == pos->off) { (pos - 1)->size += pos->size; p->free_.erase(pos); }
}
static int copy_bytes(qdp_pool* p, void* dst, const void* src, size_t n, cudaMemcpyKind kind) {
    if (p->device < 0) return QDP_OK;     // address-range-only pool: policy tests
    int prev = 0;
    cudaGetDevice(&prev);
    cudaError_t e = cudaSetDevice(p->device);
    if (e == cudaSuccess) e = cudaMemcpy(dst, src, n, kind);
    cudaSetDevice(prev);
    return e == cudaSuccess ? QDP_OK : qdp::set_error(QDP_ERR_CUDA, cudaGetErrorString(e));
}
// spill the least recently acquired unlocked resident object; false if there is none
static int spill_one(qdp_pool* p, bool* spilled) {
    *spilled = false;
    for (auto it = p->lru_.rbegin(); it != p->lru_.rend(); ++it) {
        qdp_cached* c = *it;
        if (c->off == kNone || c->locks > 0) continue;
        if (c->dirty) {
            int rc = copy_bytes(p, c->host, p->base + c->off, c->bytes, cudaMemcpyDeviceToHost);
            if (rc != QDP_OK) return rc;
            c->dirty = false;
        }
        give_back(p, c->off);
        c->off = kNone;
        p->evlog.push_back(c->id);
        *spilled = true;
        return QDP_OK;
    }
    return QDP_OK;
}
static int pool_alloc_off(qdp_pool* p, size_t bytes, size_t* off) {
    const size_t need = round_up(bytes);
    for (;;) {
        *off = first_fit(p, need);
        if (*off != kNone) return QDP_OK;
        bool spilled = false;
        int rc = spill_one(p, &spilled);
        if (rc != QDP_OK) return rc;
        if (!spilled) return qdp::set_error(QDP_ERR_OOM, "pool exhausted: no free block fits and every resident cached object is locked");
    }
}

extern "C" int qdp_pool_create(int device, size_t bytes, qdp_pool** out) {
    if (!out || bytes < kGran) return qdp::set_error(QDP_ERR_ARG, "qdp_pool_create: bad argument");
    qdp_pool* p = new (std::nothrow) qdp_pool();
    if (!p) return qdp::set_error(QDP_ERR_OOM, "host allocation failed");
    p->magic = kPoolMagic; p->device = device; p->cap = bytes / kGran * kGran; p->next_id = 0;
    if (device >= 0) {
        int prev = 0;
        cudaGetDevice(&prev);
        cudaError_t e = cudaSetDevice(device);
        void* b = nullptr;
        if (e == cudaSuccess) e = cudaMalloc(&b, p->cap);
        cudaSetDevice(prev);
        if (e != cudaSuccess) { delete p; return qdp::set_error(e == cudaErrorMemoryAllocation ? QDP_ERR_OOM : QDP_ERR_CUDA, cudaGetErrorString(e)); }
        p->base = static_cast<char*>(b);
    } else {
        p->base = reinterpret_cast<char*>((uintptr_t)1 << 32);   // a fake, 256-aligned, never dereferenced base address
    }
    p->free_.push_back(FreeBlock{0, p->cap});
    *out = p;
    return QDP_OK;
}
extern "C" int qdp_pool_destroy(qdp_pool* p) {
    if (!ok_pool(p)) return qdp::set_error(QDP_ERR_ARG, "qdp_pool_destroy: not a pool");
    if (!p->lru_.empty()) return qdp::set_error(QDP_ERR_ARG, "qdp_pool_destroy: cached objects still registered");
    // blocks handed out by qdp_pool_alloc / qdp_pool_hook_alloc (fields, a lattice's scratch) would dangle after the cudaFree below
    if (!p->used_.empty()) return qdp::set_error(QDP_ERR_ARG, "qdp_pool_destroy: blocks of this pool are still allocated (free the fields and lattices that live in it first)");
    if (p->device >= 0) {
        int prev = 0;
        cudaGetDevice(&prev);
        cudaSetDevice(p->device);
        cudaDeviceSynchronize();
        cudaFree(p->base);
        cudaSetDevice(prev);
    }
    p->magic = 0;
    delete p;
    return QDP_OK;
}
extern "C" int qdp_pool_alloc(qdp_pool* p, size_t bytes, void** out) {
    if (!ok_pool(p) || !out) return qdp::set_error(QDP_ERR_ARG, "qdp_pool_alloc: bad argument");
    size_t off;
    int rc = pool_alloc_off(p, bytes, &off);
    if (rc != QDP_OK) return rc;
    *out = p->base + off;
    return QDP_OK;
}
extern "C" int qdp_pool_free(qdp_pool* p, void* ptr) {
    if (!ok_pool(p) || !ptr) return qdp::set_error(QDP_ERR_ARG, "qdp_pool_free: bad argument");
    const size_t off = (size_t)(static_cast<char*>(ptr) - p->base);
    if (p->used_.find(off) == p->used_.end()) return qdp::set_error(QDP_ERR_ARG, "qdp_pool_free: not an allocation of this pool");
    give_back(p, off);
    return QDP_OK;
}
extern "C" int qdp_pool_stats(const qdp_pool* p, size_t out[4]) {
    if (!ok_pool(p) || !out) return qdp::set_error(QDP_ERR_ARG, "qdp_pool_stats: bad argument");
    size_t used = 0, largest = 0;
    for (const auto& kv : p->used_) used += kv.second;
    for (const auto& b : p->free_) largest = std::max(largest, b.size);
    out[0] = p->cap; out[1] = used; out[2] = largest; out[3] = p->free_.size();
    return QDP_OK;
}
// qdp_set_allocator-compatible hooks: ctx = the pool
extern "C" void* qdp_pool_hook_alloc(size_t bytes, void* ctx) {
    void* out = nullptr;
    return qdp_pool_alloc(static_cast<qdp_pool*>(ctx), bytes, &out) == QDP_OK ? out : nullptr;
}
extern "C" void qdp_pool_hook_free(void* ptr, void* ctx) { qdp_pool_free(static_cast<qdp_pool*>(ctx), ptr); }

extern "C" int qdp_cache_register(qdp_pool* p, void* host_buf, size_t bytes, qdp_cached** out) {
    if (!ok_pool(p) || !out || bytes == 0 || (p->device >= 0 && !host_buf)) return qdp::set_error(QDP_ERR_ARG, "qdp_cache_register: bad argument");
    if (round_up(bytes) > p->cap) return qdp::set_error(QDP_ERR_OOM, "qdp_cache_register: object larger than the pool");
    qdp_cached* c = new (std::nothrow) qdp_cached();
    if (!c) return qdp::set_error(QDP_ERR_OOM, "host allocation failed");
    c->magic = kCachedMagic; c->pool = p; c->host = host_buf; c->bytes = bytes; c->off = kNone; c->locks = 0; c->dirty = false;
    c->id = p->next_id++;
    p->lru_.push_back(c);       // never acquired: least recently used
    *out = c;
    return QDP_OK;
}
extern "C" int qdp_cache_acquire(qdp_cached* c, int for_write, void** dev_ptr) {
    if (!ok_cached(c) || !dev_ptr) return qdp::set_error(QDP_ERR_ARG, "qdp_cache_acquire: bad argument");
    qdp_pool* p = c->pool;
    if (c->off == kNone) {
        size_t off;
        int rc = pool_alloc_off(p, c->bytes, &off);
        if (rc != QDP_OK) return rc;
        rc = copy_bytes(p, p->base + off, c->host, c->bytes, cudaMemcpyHostToDevice);
        if (rc != QDP_OK) { give_back(p, off); return rc; }
        c->off = off;
        c->dirty = false;
    }
    c->locks++;
    if (for_write) c->dirty = true;
    p->lru_.remove(c);
    p->lru_.push_front(c);
    *dev_ptr = p->base + c->off;
    return QDP_OK;
}
extern "C" int qdp_cache_release(qdp_cached* c) {
    if (!ok_cached(c) || c->locks <= 0) return qdp::set_error(QDP_ERR_ARG, "qdp_cache_release: not acquired");
    c->locks--;
    return QDP_OK;
}
extern "C" int qdp_cache_is_resident(const qdp_cached* c) { return ok_cached(c) && c->off != kNone ? 1 : 0; }
extern "C" int64_t qdp_cache_id(const qdp_cached* c) { return ok_cached(c) ? c->id : -1; }
extern "C" int qdp_cache_unregister(qdp_cached* c) {
    if (!ok_cached(c)) return qdp::set_error(QDP_ERR_ARG, "qdp_cache_unregister: not a cached object");
    if (c->locks > 0) return qdp::set_error(QDP_ERR_ARG, "qdp_cache_unregister: still acquired");
    qdp_pool* p = c->pool;
    if (c->off != kNone) {
        if (c->dirty) {
            int rc = copy_bytes(p, c->host, p->base + c->off, c->bytes, cudaMemcpyDeviceToHost);
            if (rc != QDP_OK) return rc;
        }
        give_back(p, c->off);
    }
    p->lru_.remove(c);
    c->magic = 0;
    delete c;
    return QDP_OK;
}
// ids of the objects spilled so far, oldest first; *n = how many there are (may exceed max)
extern "C" int qdp_pool_eviction_log(const qdp_pool* p, int64_t* ids, int max, int* n) {
    if (!ok_pool(p) || !n || (max > 0 && !ids)) return qdp::set_error(QDP_ERR_ARG, "qdp_pool_eviction_log: bad argument");
    *n = (int)p->evlog.size();
    for (int i = 0; i < max && i < *n; i++) ids[i] = p->evlog[i];
    return QDP_OK;
}
