// Internal utilities of libfstc: error type, stream-ordered device memory, launch helpers.
// Not part of the C ABI (include/fstc.h).  Shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdint>
#include <cstdio>
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

struct Ctx {
    cudaStream_t stream = nullptr;
    int n_sm = 148;
    int64_t n_launch = 0;

    void *alloc_bytes(size_t bytes) {
        if (bytes == 0) bytes = 16;
        void *p = nullptr;
        cudaError_t e = cudaMallocFromPoolAsync(&p, bytes, device_pool(), stream);
        if (e != cudaSuccess) {
            (void)cudaGetLastError();
            fail(e == cudaErrorMemoryAllocation ? FSTC_ERR_OOM : FSTC_ERR_CUDA,
                 "device allocation of %zu bytes failed: %s", bytes, cudaGetErrorString(e));
        }
        return p;
    }
    void free_bytes(void *p) {
        if (p) (void)cudaFreeAsync(p, stream);
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
    DBuf(Ctx &c, int64_t count) { alloc(c, count); }
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
    void alloc(Ctx &c, int64_t count) {
        release();
        ctx = &c;
        n = count;
        p = static_cast<T *>(c.alloc_bytes(static_cast<size_t>(count > 0 ? count : 0) * sizeof(T)));
    }
    void release() {
        if (p && ctx) ctx->free_bytes(p);
        p = nullptr;
        n = 0;
    }
    T *take() { T *q = p; p = nullptr; n = 0; return q; }
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
