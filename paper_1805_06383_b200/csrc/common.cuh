// Internal utilities of libfstc: error type, stream-ordered device memory, launch helpers.
// Not part of the C ABI (include/fstc.h).  Shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <ctime>
#include <string>
#include <utility>

#include "../../include/fstc.h"

namespace fstc {

struct Error {
    int code;
    std::string msg;
};

[[noreturn]] inline void fail(int code, const char *fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    throw Error{code, buf};
}

#define FSTC_CUDA(expr)                                                                                   \
    do {                                                                                                  \
        cudaError_t e__ = (expr);                                                                         \
        if (e__ != cudaSuccess) {                                                                         \
            int c__ = (e__ == cudaErrorMemoryAllocation) ? FSTC_ERR_OOM : FSTC_ERR_CUDA;                  \
            (void)cudaGetLastError();                                                                     \
            ::fstc::fail(c__, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
        }                                                                                                 \
    } while (0)

#define FSTC_LAUNCH_CHECK() FSTC_CUDA(cudaGetLastError())

// One library-owned memory pool per device: freed blocks stay cached (release threshold = max),
// so repeated compositions do not go back to the driver for memory.
cudaMemPool_t device_pool();
// workspace arena of the calling thread (api.cu): temporaries are carved out of a few large chunks the library keeps
void *arena_alloc(size_t bytes, cudaStream_t stream);   // null when device memory is out
bool arena_free(void *p);                               // false if p is not an arena block
void arena_release_all();
// blocks that outlive a call (api.cu): pool allocations, parked on release and handed out again to a like-sized request
void *persist_alloc(size_t bytes, cudaStream_t stream);   // null when device memory is out
void persist_free(void *p, cudaStream_t stream);
void persist_release_all();
void release_caches(cudaStream_t stream);                 // out of memory: everything the library caches goes back to the driver

struct AllocHooks {           // fstc_opts_t's allocator hooks (both set or both null)
    void *(*alloc)(size_t, void *, void *) = nullptr;
    void (*dealloc)(void *, void *, void *) = nullptr;
    void *ctx = nullptr;
};

struct Ctx {
    cudaStream_t stream = nullptr;
    int n_sm = 148;
    int64_t n_launch = 0;
    AllocHooks hooks;         // set: all device memory of the call comes from the caller

    // persistent: the block outlives the call (a result or packed array): a pool allocation of its own
    void *alloc_bytes(size_t bytes, bool persistent = false) {
        if (bytes == 0) bytes = 16;
        void *p = nullptr;
        static const bool trace = getenv("FSTC_ALLOC_TRACE") != nullptr;       // debug knob: host time of big allocations
        timespec t0, t1;
        if (trace) clock_gettime(CLOCK_MONOTONIC, &t0);
        cudaError_t e = cudaSuccess;
        if (hooks.alloc) p = hooks.alloc(bytes, stream, hooks.ctx);
        else {
            p = persistent ? persist_alloc(bytes, stream) : arena_alloc(bytes, stream);
            if (!p) {             // the arena, the parked blocks and the pool each cache memory the other could use: all back, once
                release_caches(stream);
                p = persistent ? persist_alloc(bytes, stream) : arena_alloc(bytes, stream);
            }
        }
        if (!p) e = cudaErrorMemoryAllocation;
        if (trace && bytes >= (64u << 20)) {
            clock_gettime(CLOCK_MONOTONIC, &t1);
            fprintf(stderr, "[fstc alloc] %8.1f MB  %8.3f ms\n", bytes / 1048576.0,
                    (t1.tv_sec - t0.tv_sec) * 1e3 + (t1.tv_nsec - t0.tv_nsec) * 1e-6);
        }
        if (e != cudaSuccess) {
            (void)cudaGetLastError();
            fail(e == cudaErrorMemoryAllocation ? FSTC_ERR_OOM : FSTC_ERR_CUDA,
                 "device allocation of %zu bytes failed: %s", bytes, cudaGetErrorString(e));
        }
        return p;
    }
    void free_bytes(void *p) {
        if (!p) return;
        static const bool trace = getenv("FSTC_ALLOC_TRACE") != nullptr;
        timespec t0, t1;
        if (trace) clock_gettime(CLOCK_MONOTONIC, &t0);
        if (hooks.dealloc) hooks.dealloc(p, stream, hooks.ctx);
        else if (!arena_free(p)) persist_free(p, stream);
        if (trace) {
            clock_gettime(CLOCK_MONOTONIC, &t1);
            const double ms = (t1.tv_sec - t0.tv_sec) * 1e3 + (t1.tv_nsec - t0.tv_nsec) * 1e-6;
            if (ms > 0.2) fprintf(stderr, "[fstc free]  %8.3f ms\n", ms);
        }
    }
    void sync() { FSTC_CUDA(cudaStreamSynchronize(stream)); }
};

// Move-only device array tied to a Ctx (freed stream-ordered on destruction).
template <typename T>
struct DBuf {
    T *p = nullptr;
    int64_t n = 0;
    Ctx *ctx = nullptr;
    DBuf() = default;
    DBuf(Ctx &c, int64_t count, bool persistent = false) { alloc(c, count, persistent); }
    DBuf(const DBuf &) = delete;
    DBuf &operator=(const DBuf &) = delete;
    DBuf(DBuf &&o) noexcept : p(o.p), n(o.n), ctx(o.ctx) { o.p = nullptr; o.n = 0; }
    DBuf &operator=(DBuf &&o) noexcept {
        if (this != &o) {
            release();
            p = o.p; n = o.n; ctx = o.ctx;
            o.p = nullptr; o.n = 0;
        }
        return *this;
    }
    ~DBuf() { release(); }
    void alloc(Ctx &c, int64_t count, bool persistent = false) {
        release();
        ctx = &c;
        n = count;
        p = static_cast<T *>(c.alloc_bytes(static_cast<size_t>(count > 0 ? count : 0) * sizeof(T), persistent));
    }
    void release() {
        if (p && ctx) ctx->free_bytes(p);
        p = nullptr;
        n = 0;
    }
    T *take() { T *q = p; p = nullptr; n = 0; return q; }   // only for blocks allocated `persistent`
    operator T *() const { return p; }
};

inline int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }

inline int bits_for(uint64_t max_value) {   // number of bits needed to represent values 0..max_value
    int b = 0;
    while (max_value) { ++b; max_value >>= 1; }
    return b;
}

template <typename T>
inline T read_scalar(Ctx &c, const T *dev) {
    T h;
    FSTC_CUDA(cudaMemcpyAsync(&h, dev, sizeof(T), cudaMemcpyDeviceToHost, c.stream));
    c.sync();
    return h;
}

}  // namespace fstc
