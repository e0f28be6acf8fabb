// C ABI of libfstc (include/fstc.h): argument checks, error translation, the device memory pool.
#include <cstdio>
#include <cstdlib>
#include <map>
#include <mutex>
#include <unordered_map>
#include <vector>

#include "internal.h"

namespace fstc {

namespace {
thread_local std::string g_last_error;
std::mutex g_pool_mu;
cudaMemPool_t g_pools[64] = {};
}  // namespace

cudaMemPool_t device_pool() {
    int dev = 0;
    FSTC_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) fail(FSTC_ERR_ARG, "device index %d not supported", dev);
    std::lock_guard<std::mutex> lk(g_pool_mu);
    if (!g_pools[dev]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool;
        FSTC_CUDA(cudaMemPoolCreate(&pool, &props));
        uint64_t keep = UINT64_MAX;   // never hand cached blocks back on synchronisation
        FSTC_CUDA(cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep));
        g_pools[dev] = pool;
    }
    return g_pools[dev];
}

// ---- workspace arena.  cudaMallocFromPoolAsync of a multi-GB block takes 1-5 ms per GB on the host whenever the
// pool cannot hand back a block it already holds in one piece (measured: 9.7 ms for 8.5 GB, far more under memory
// pressure), and a composition allocates dozens of big temporaries per level.  Temporaries are therefore carved out
// of a few large chunks that the library keeps (first fit, free neighbours coalesce); only the arrays that leave the
// library (results, packed operands) are separate pool allocations.  One arena per host thread: a thread's calls run
// one after the other and each ends with a synchronisation of its stream, so a freed range is idle before any later
// call reuses it; inside a call everything is ordered on one stream.  fstc_trim_pool releases the chunks.
namespace {
struct ArenaChunk {
    char *base = nullptr;
    size_t size = 0;
    int dev = 0;
    std::map<size_t, size_t> free_ranges;                  // offset -> length
};
struct Arena {
    std::vector<ArenaChunk> chunks;
    std::unordered_map<void *, std::pair<int, size_t>> live;   // pointer -> (chunk, length)
    ~Arena() {                                              // the thread ends: its calls are complete, give the chunks back
        for (auto &ch : chunks)
            if (ch.base) (void)cudaFreeAsync(ch.base, nullptr);
        (void)cudaGetLastError();                           // (at process exit the context may already be gone)
    }
};
thread_local Arena g_arena;
constexpr size_t ARENA_ALIGN = 512;
constexpr size_t ARENA_MIN_CHUNK = size_t(1) << 30;

// carves `bytes` out of the free range at `off` of chunk ci
void *arena_carve(int ci, size_t off, size_t bytes) {
    ArenaChunk &ch = g_arena.chunks[ci];
    auto it = ch.free_ranges.find(off);
    const size_t len = it->second;
    ch.free_ranges.erase(it);
    if (len > bytes) ch.free_ranges[off + bytes] = len - bytes;
    void *p = ch.base + off;
    g_arena.live[p] = {ci, bytes};
    return p;
}
}  // namespace

void arena_release_all() {
    for (auto &ch : g_arena.chunks)
        if (ch.base) (void)cudaFreeAsync(ch.base, nullptr);
    g_arena.chunks.clear();
    g_arena.live.clear();
}

void *arena_alloc(size_t bytes, cudaStream_t stream) {
    bytes = (bytes + ARENA_ALIGN - 1) / ARENA_ALIGN * ARENA_ALIGN;
    int dev = 0;
    (void)cudaGetDevice(&dev);
    // best fit over all chunks: small requests fill small holes and leave the large ranges whole, so a caller that
    // repeats the same sequence of requests finds the same layout again
    int best_ci = -1;
    size_t best_off = 0, best_len = ~size_t(0);
    for (size_t ci = 0; ci < g_arena.chunks.size(); ++ci) {
        if (g_arena.chunks[ci].dev != dev) continue;
        for (auto &r : g_arena.chunks[ci].free_ranges)
            if (r.second >= bytes && r.second < best_len) { best_ci = static_cast<int>(ci); best_off = r.first; best_len = r.second; }
    }
    if (best_ci >= 0) return arena_carve(best_ci, best_off, bytes);
    static const bool trace = getenv("FSTC_ALLOC_TRACE") != nullptr;
    if (trace) fprintf(stderr, "[fstc arena] new chunk for %.1f MB (chunks so far %zu)\n", bytes / 1048576.0, g_arena.chunks.size());
    ArenaChunk ch;
    ch.size = bytes > ARENA_MIN_CHUNK ? bytes : ARENA_MIN_CHUNK;
    ch.dev = dev;
    void *base = nullptr;
    cudaError_t e = cudaMallocFromPoolAsync(&base, ch.size, device_pool(), stream);
    if (e != cudaSuccess && ch.size > bytes) {             // no room for a whole chunk: just what is asked for
        (void)cudaGetLastError();
        ch.size = bytes;
        e = cudaMallocFromPoolAsync(&base, ch.size, device_pool(), stream);
    }
    if (e != cudaSuccess) {                                // still none: drop the chunks nobody uses, once
        (void)cudaGetLastError();
        bool dropped = false;
        for (auto &c2 : g_arena.chunks)
            if (c2.base && c2.free_ranges.size() == 1 && c2.free_ranges.begin()->second == c2.size) {
                (void)cudaFreeAsync(c2.base, stream);
                c2.base = nullptr; c2.size = 0; c2.free_ranges.clear();
                dropped = true;
            }
        if (dropped) e = cudaMallocFromPoolAsync(&base, ch.size, device_pool(), stream);
        if (e != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
    }
    ch.base = static_cast<char *>(base);
    ch.free_ranges[0] = ch.size;
    g_arena.chunks.push_back(std::move(ch));
    return arena_carve(static_cast<int>(g_arena.chunks.size()) - 1, 0, bytes);
}

bool arena_free(void *p) {
    auto it = g_arena.live.find(p);
    if (it == g_arena.live.end()) return false;
    ArenaChunk &ch = g_arena.chunks[it->second.first];
    size_t off = static_cast<char *>(p) - ch.base, len = it->second.second;
    g_arena.live.erase(it);
    auto nxt = ch.free_ranges.lower_bound(off);
    if (nxt != ch.free_ranges.end() && off + len == nxt->first) {   // merge with the free range behind
        len += nxt->second;
        nxt = ch.free_ranges.erase(nxt);
    }
    if (nxt != ch.free_ranges.begin()) {                            // and with the one in front
        auto prv = std::prev(nxt);
        if (prv->first + prv->second == off) { prv->second += len; return true; }
    }
    ch.free_ranges[off] = len;
    return true;
}

// ---- arrays that leave the library (results, packed operands, and the growing output arrays on the way there).
// They are pool allocations of their own; when one is released it is parked, with an event that marks the point of
// release, and the next request of (nearly) the same size takes it over after waiting on that event.  A caller that
// composes in a loop thus gets the same blocks back instead of paying the pool's multi-millisecond path every time.
namespace {
struct ParkedBlock { void *p; size_t bytes; int dev; cudaEvent_t ev; };
std::mutex g_park_mu;
std::vector<ParkedBlock> g_parked;
std::unordered_map<void *, size_t> g_persist_size;
size_t g_parked_bytes = 0;
constexpr size_t PARK_MIN_BYTES = size_t(32) << 20;
constexpr size_t PARK_MAX_TOTAL = size_t(64) << 30;
}  // namespace

void *persist_alloc(size_t bytes, cudaStream_t stream) {
    int dev = 0;
    (void)cudaGetDevice(&dev);
    void *p = nullptr;
    {
        std::lock_guard<std::mutex> lk(g_park_mu);
        int best = -1;
        for (size_t i = 0; i < g_parked.size(); ++i) {
            const ParkedBlock &b = g_parked[i];
            if (b.dev == dev && b.bytes >= bytes && b.bytes <= bytes + bytes / 8 && (best < 0 || b.bytes < g_parked[best].bytes))
                best = static_cast<int>(i);
        }
        if (best >= 0) {
            ParkedBlock b = g_parked[best];
            g_parked.erase(g_parked.begin() + best);
            g_parked_bytes -= b.bytes;
            (void)cudaStreamWaitEvent(stream, b.ev, 0);
            (void)cudaEventDestroy(b.ev);
            g_persist_size[b.p] = b.bytes;
            return b.p;
        }
    }
    static const bool trace = getenv("FSTC_ALLOC_TRACE") != nullptr;
    if (trace && bytes >= PARK_MIN_BYTES) fprintf(stderr, "[fstc persist] pool allocation of %.1f MB (parked %zu blocks, %.1f GB)\n",
                                                  bytes / 1048576.0, g_parked.size(), g_parked_bytes / 1e9);
    cudaError_t e = cudaMallocFromPoolAsync(&p, bytes, device_pool(), stream);
    if (e != cudaSuccess) {                                // out of memory: hand the parked blocks back, once
        (void)cudaGetLastError();
        persist_release_all();
        e = cudaMallocFromPoolAsync(&p, bytes, device_pool(), stream);
        if (e != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
    }
    if (bytes >= PARK_MIN_BYTES) {
        std::lock_guard<std::mutex> lk(g_park_mu);
        g_persist_size[p] = bytes;
    }
    return p;
}

void persist_free(void *p, cudaStream_t stream) {
    if (!p) return;
    int dev = 0;
    (void)cudaGetDevice(&dev);
    {
        std::lock_guard<std::mutex> lk(g_park_mu);
        auto it = g_persist_size.find(p);
        if (it != g_persist_size.end()) {
            const size_t bytes = it->second;
            g_persist_size.erase(it);
            cudaEvent_t ev;
            if (g_parked_bytes + bytes <= PARK_MAX_TOTAL &&
                cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) == cudaSuccess) {
                (void)cudaEventRecord(ev, stream);         // the legacy stream (null) orders after all blocking streams
                g_parked.push_back(ParkedBlock{p, bytes, dev, ev});
                g_parked_bytes += bytes;
                return;
            }
        }
    }
    static const bool trace = getenv("FSTC_ALLOC_TRACE") != nullptr;
    if (trace) fprintf(stderr, "[fstc persist] block goes back to the pool (not parked)\n");
    (void)cudaFreeAsync(p, stream);
}

void persist_release_all() {
    std::lock_guard<std::mutex> lk(g_park_mu);
    for (auto &b : g_parked) {
        (void)cudaFreeAsync(b.p, nullptr);
        (void)cudaEventDestroy(b.ev);
    }
    g_parked.clear();
    g_parked_bytes = 0;
}

// Out of memory: the workspace arena, the parked blocks and the pool's free list each hold memory the failing request
// could use (and so could another allocator on the device, e.g. PyTorch's): everything idle goes back to the driver.
void release_caches(cudaStream_t stream) {
    (void)cudaStreamSynchronize(stream);
    for (auto &ch : g_arena.chunks)                          // chunks of this thread that nobody uses
        if (ch.base && ch.free_ranges.size() == 1 && ch.free_ranges.begin()->second == ch.size) {
            (void)cudaFreeAsync(ch.base, stream);
            ch.base = nullptr; ch.size = 0; ch.free_ranges.clear();
        }
    persist_release_all();
    (void)cudaStreamSynchronize(stream);
    (void)cudaStreamSynchronize(nullptr);
    try { (void)cudaMemPoolTrimTo(device_pool(), 0); } catch (const Error &) {}
    (void)cudaGetLastError();
}

namespace {

Ctx make_ctx(void *stream, const fstc_opts_t *opts = nullptr) {
    Ctx c;
    c.stream = static_cast<cudaStream_t>(stream);
    if (opts) {
        if ((opts->alloc == nullptr) != (opts->dealloc == nullptr)) fail(FSTC_ERR_ARG, "alloc and dealloc must both be set or both be NULL");
        c.hooks.alloc = opts->alloc; c.hooks.dealloc = opts->dealloc; c.hooks.ctx = opts->alloc_ctx;
    }
    int dev = 0;
    FSTC_CUDA(cudaGetDevice(&dev));
    FSTC_CUDA(cudaDeviceGetAttribute(&c.n_sm, cudaDevAttrMultiProcessorCount, dev));
    return c;
}

// On an error the DBuf destructors have already handed their arena ranges back while kernels of the failed call may still
// run: the stream is drained before the call returns, so that the next call cannot reuse a range that is still in use.
template <typename F>
int guarded(F &&body, void *stream = nullptr, bool has_stream = false) {
    try {
        body();
        g_last_error.clear();
        return FSTC_OK;
    } catch (const Error &e) {
        if (has_stream) { (void)cudaStreamSynchronize(static_cast<cudaStream_t>(stream)); (void)cudaGetLastError(); }
        g_last_error = e.msg;
        return e.code;
    } catch (const std::bad_alloc &) {
        g_last_error = "host allocation failed";
        return FSTC_ERR_OOM;
    } catch (const std::exception &e) {
        g_last_error = e.what();
        return FSTC_ERR_CUDA;
    }
}

template <typename T>
void d2h(Ctx &c, T *dst, const T *src, int64_t n) {
    if (dst && src && n > 0)
        FSTC_CUDA(cudaMemcpyAsync(dst, src, sizeof(T) * static_cast<size_t>(n), cudaMemcpyDeviceToHost, c.stream));
}

}  // namespace
}  // namespace fstc

using namespace fstc;

extern "C" {

int fstc_version(void) { return FSTC_VERSION; }

const char *fstc_strerror(int code) {
    switch (code) {
        case FSTC_OK: return "ok";
        case FSTC_ERR_ARG: return "invalid argument";
        case FSTC_ERR_INPUT: return "state or symbol id out of range";
        case FSTC_ERR_OOM: return "out of memory";
        case FSTC_ERR_CAPACITY: return "internal capacity limit exceeded";
        case FSTC_ERR_CUDA: return "CUDA error";
        case FSTC_ERR_INTERNAL: return "internal consistency check failed";
        case FSTC_ERR_CALLBACK: return "the resolve callback failed";
        default: return "unknown error";
    }
}

const char *fstc_last_error(void) { return g_last_error.c_str(); }

int fstc_pack(const fstc_fst_t *m, int side, const fstc_opts_t *opts, void *cuda_stream, fstc_packed_t **out) {
    if (out) *out = nullptr;
    return guarded([&] {
        if (!m || !out) fail(FSTC_ERR_ARG, "null argument");
        Ctx c = make_ctx(cuda_stream, opts);
        *out = pack_fst(c, *m, side);
    }, cuda_stream, true);
}

void fstc_packed_free(fstc_packed_t *p) { free_packed(p); }

int fstc_packed_info(const fstc_packed_t *p, int64_t *info) {
    return guarded([&] {
        if (!p || !info) fail(FSTC_ERR_ARG, "null argument");
        info[0] = p->n_states; info[1] = p->n_arcs; info[2] = p->n_segs;
        info[3] = p->n_inner; info[4] = p->n_outer; info[5] = p->side; info[6] = p->n_launch;
    });
}

int fstc_packed_to_host(const fstc_packed_t *p, void *cuda_stream, uint32_t *arcs4, uint32_t *segs2, uint32_t *seg_ptr,
                        uint8_t *flags, uint32_t *accept_bits) {
    return guarded([&] {
        if (!p) fail(FSTC_ERR_ARG, "null argument");
        Ctx c = make_ctx(cuda_stream);
        d2h(c, arcs4, reinterpret_cast<const uint32_t *>(p->arcs), 4 * p->n_arcs);
        d2h(c, segs2, reinterpret_cast<const uint32_t *>(p->segs), 2 * (p->n_segs + 1));
        d2h(c, seg_ptr, p->seg_ptr, static_cast<int64_t>(p->n_states) + 1);
        d2h(c, flags, p->flags, p->n_states);
        d2h(c, accept_bits, p->accept_bits, (p->n_states + 31) / 32);
        c.sync();
    });
}

int fstc_compose_packed(const fstc_packed_t *m1, const fstc_packed_t *m2, const fstc_opts_t *opts, void *cuda_stream,
                        fstc_result_t **out, fstc_stats_t *stats) {
    if (out) *out = nullptr;
    return guarded([&] {
        if (!m1 || !m2 || !out) fail(FSTC_ERR_ARG, "null argument");
        fstc_opts_t o = {};
        if (opts) o = *opts;
        Ctx c = make_ctx(cuda_stream, &o);
        *out = compose_packed(c, *m1, *m2, o, stats);
    }, cuda_stream, true);
}

int fstc_compose_batch(const fstc_packed_t *const *m1, int32_t n, const fstc_packed_t *m2, const fstc_opts_t *opts,
                       void *cuda_stream, fstc_result_t **out, fstc_stats_t *stats) {
    if (out) for (int32_t k = 0; k < n; ++k) out[k] = nullptr;
    int rc = guarded([&] {
        if (!m1 || !m2 || !out || n < 0) fail(FSTC_ERR_ARG, "null argument");
        fstc_opts_t o = {};
        if (opts) o = *opts;
        if (o.small_path < 0 || o.small_path > 2) fail(FSTC_ERR_ARG, "bad options");
        Ctx c = make_ctx(cuda_stream, &o);
        std::vector<char> ok(static_cast<size_t>(n), 0);
        if (small_path_applies(o)) compose_small_batch(c, m1, n, *m2, o, out, stats, ok);
        else if (o.small_path == FSTC_SMALL_ONLY) fail(FSTC_ERR_ARG, "the small path does not take these options");
        fstc_opts_t big = o;
        big.small_path = FSTC_SMALL_OFF;
        for (int32_t k = 0; k < n; ++k) {                       // what did not fit a block: the level-synchronous path
            if (ok[k]) continue;
            if (!m1[k]) fail(FSTC_ERR_ARG, "null operand %d", k);
            if (o.small_path == FSTC_SMALL_ONLY) fail(FSTC_ERR_CAPACITY, "problem %d does not fit the small path", k);
            out[k] = compose_packed(c, *m1[k], *m2, big, stats ? stats + k : nullptr);
        }
    }, cuda_stream, true);
    if (rc != FSTC_OK && out)
        for (int32_t k = 0; k < n; ++k) { free_result(out[k]); out[k] = nullptr; }
    return rc;
}

int fstc_compose_static(const fstc_packed_t *m1, const fstc_packed_t *m2, const fstc_opts_t *opts, void *cuda_stream,
                        const fstc_static_out_t *out) {
    return guarded([&] {
        if (!m1 || !m2 || !out) fail(FSTC_ERR_ARG, "null argument");
        fstc_opts_t o = {};
        if (opts) o = *opts;
        Ctx c;                                   // (no allocator of any kind is reachable from here)
        c.stream = static_cast<cudaStream_t>(cuda_stream);
        compose_small_static(c, *m1, *m2, o, *out);
    }, cuda_stream, true);
}

int fstc_compose(const fstc_fst_t *m1, const fstc_fst_t *m2, const fstc_opts_t *opts, void *cuda_stream,
                 fstc_result_t **out, fstc_stats_t *stats) {
    if (out) *out = nullptr;
    fstc_packed_t *p1 = nullptr, *p2 = nullptr;
    int rc = guarded([&] {
        if (!m1 || !m2 || !out) fail(FSTC_ERR_ARG, "null argument");
        if (m1->n_osyms != m2->n_isyms)
            fail(FSTC_ERR_ARG, "inner alphabets differ: M1 has %d output symbols, M2 %d input symbols (PAPER.md:45)",
                 m1->n_osyms, m2->n_isyms);
        fstc_opts_t o = {};
        if (opts) o = *opts;
        Ctx c = make_ctx(cuda_stream, &o);
        p1 = pack_fst(c, *m1, 1);
        p2 = pack_fst(c, *m2, 2);
        *out = compose_packed(c, *p1, *p2, o, stats);
    }, cuda_stream, true);
    free_packed(p1);
    free_packed(p2);
    return rc;
}

int fstc_result_to_host(const fstc_result_t *r, void *cuda_stream, const fstc_host_result_t *dst) {
    return guarded([&] {
        if (!r || !dst) fail(FSTC_ERR_ARG, "null argument");
        Ctx c = make_ctx(cuda_stream);
        d2h(c, dst->pair, r->pair, 2 * r->n_states);
        d2h(c, dst->src, r->src, r->n_arcs);
        d2h(c, dst->ilabel, r->ilabel, r->n_arcs);
        d2h(c, dst->olabel, r->olabel, r->n_arcs);
        d2h(c, dst->tgt, r->tgt, r->n_arcs);
        d2h(c, dst->weight, r->weight, r->n_arcs);
        d2h(c, dst->accept, r->accept, r->n_accept);
        d2h(c, dst->expanded, r->expanded, r->n_states);
        c.sync();
    });
}

void fstc_result_free(fstc_result_t *r) { free_result(r); }

int fstc_trim_pool(void) {
    return guarded([&] {
        FSTC_CUDA(cudaDeviceSynchronize());
        arena_release_all();
        persist_release_all();
        FSTC_CUDA(cudaDeviceSynchronize());
        FSTC_CUDA(cudaMemPoolTrimTo(device_pool(), 0));
    });
}

}  // extern "C"
