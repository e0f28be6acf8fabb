// C ABI of libfstc (include/fstc.h): argument checks, error translation, the device memory pool.
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

// ---- cache of big device blocks.  cudaMallocFromPoolAsync of several GB takes 1-2 ms per GB on the host whenever
// the pool cannot hand back a block it already has in one piece (measured: 9.7 ms for 8.5 GB), and a composition
// allocates the same big temporaries level after level, call after call.  Blocks >= 64 MB are therefore parked here
// when released and handed out again to a request they fit closely ON THE SAME STREAM, so reuse is stream-ordered
// like the pool's own.
namespace {
struct BigBlock { void *p; size_t bytes; int dev; cudaStream_t stream; };
std::mutex g_cache_mu;
std::vector<BigBlock> g_parked;
std::unordered_map<void *, size_t> g_big_live;           // size of every live block that came through big_alloc
constexpr size_t BIG_BYTES = size_t(64) << 20;
}  // namespace

void *big_alloc(size_t bytes, cudaStream_t stream) {
    if (bytes < BIG_BYTES) return nullptr;
    int dev = 0;
    (void)cudaGetDevice(&dev);
    std::lock_guard<std::mutex> lk(g_cache_mu);
    int best = -1;
    for (size_t i = 0; i < g_parked.size(); ++i) {
        const BigBlock &b = g_parked[i];
        if (b.dev == dev && b.stream == stream && b.bytes >= bytes && b.bytes <= bytes + bytes / 8 + (size_t(1) << 20) &&
            (best < 0 || b.bytes < g_parked[best].bytes))
            best = static_cast<int>(i);
    }
    void *p = nullptr;
    size_t got = bytes;
    if (best >= 0) {
        p = g_parked[best].p;
        got = g_parked[best].bytes;
        g_parked.erase(g_parked.begin() + best);
    } else {
        cudaError_t e = cudaMallocFromPoolAsync(&p, bytes, device_pool(), stream);
        if (e != cudaSuccess) {                            // out of memory: give the parked blocks back and try again
            (void)cudaGetLastError();
            for (auto &b : g_parked) (void)cudaFreeAsync(b.p, stream);
            g_parked.clear();
            e = cudaMallocFromPoolAsync(&p, bytes, device_pool(), stream);
            if (e != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
        }
    }
    g_big_live[p] = got;
    return p;
}

bool big_free(void *p, cudaStream_t stream) {
    int dev = 0;
    (void)cudaGetDevice(&dev);
    std::lock_guard<std::mutex> lk(g_cache_mu);
    auto it = g_big_live.find(p);
    if (it == g_big_live.end()) return false;
    g_parked.push_back(BigBlock{p, it->second, dev, stream});
    g_big_live.erase(it);
    return true;
}

void big_forget(void *p) {                                 // the block leaves the library's hands (a result array)
    std::lock_guard<std::mutex> lk(g_cache_mu);
    g_big_live.erase(p);
}

void big_release_all() {
    std::lock_guard<std::mutex> lk(g_cache_mu);
    for (auto &b : g_parked) (void)cudaFreeAsync(b.p, nullptr);
    g_parked.clear();
}

namespace {

Ctx make_ctx(void *stream) {
    Ctx c;
    c.stream = static_cast<cudaStream_t>(stream);
    int dev = 0;
    FSTC_CUDA(cudaGetDevice(&dev));
    FSTC_CUDA(cudaDeviceGetAttribute(&c.n_sm, cudaDevAttrMultiProcessorCount, dev));
    return c;
}

template <typename F>
int guarded(F &&body) {
    try {
        body();
        g_last_error.clear();
        return FSTC_OK;
    } catch (const Error &e) {
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
    if (dst && n > 0)
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
        default: return "unknown error";
    }
}

const char *fstc_last_error(void) { return g_last_error.c_str(); }

int fstc_pack(const fstc_fst_t *m, int side, void *cuda_stream, fstc_packed_t **out) {
    if (out) *out = nullptr;
    return guarded([&] {
        if (!m || !out) fail(FSTC_ERR_ARG, "null argument");
        Ctx c = make_ctx(cuda_stream);
        *out = pack_fst(c, *m, side);
    });
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
        Ctx c = make_ctx(cuda_stream);
        *out = compose_packed(c, *m1, *m2, o, stats);
    });
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
        Ctx c = make_ctx(cuda_stream);
        p1 = pack_fst(c, *m1, 1);
        p2 = pack_fst(c, *m2, 2);
        *out = compose_packed(c, *p1, *p2, o, stats);
    });
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
        big_release_all();
        FSTC_CUDA(cudaDeviceSynchronize());
        FSTC_CUDA(cudaMemPoolTrimTo(device_pool(), 0));
    });
}

}  // extern "C"
