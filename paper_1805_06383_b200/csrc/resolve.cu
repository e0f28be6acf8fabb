// Partitioned target resolution: the visited-set step of a BIG level (PAPER.md:237-239 adapted).
//
// The paper tests and sets one entry of a dense |Q1||Q2| table per composed arc (atomicOr, :237).  On a B200 a
// random 32-byte DRAM sector costs ~21 ps to read and ~45 ps to dirty (measured, profiles/), so at 10^9 arcs per
// level the per-arc probe of any table that does not fit the 126 MB L2 bounds the whole path.  Big levels are
// therefore resolved like a radix hash join, with streaming passes only:
//
//   1. every composed arc leaves a record (target key, output position) — written by the emit kernel in rank order;
//      every existing state leaves a record (key, id);
//   2. both record streams are partitioned by the top bits of a hash of the key (one or two staged scatter
//      passes: a block sorts a tile of 4096 records by bin in shared memory and appends whole runs), until a bin
//      holds ~10^3 distinct keys;
//   3. one block per bin builds the bin's key->id map in SHARED memory (old states first), finds or creates the id
//      of every arc record, allocates new ids (one global atomicAdd per 1024 records) and writes pair[id];
//   4. the (position, id) records are partitioned by position window and scattered into the target column; a window
//      is a few MB, so the scattered 4-byte stores combine in L2 and reach DRAM as full sectors.
//
// Nothing persists between levels except pair[] (id -> (q1,q2)): the key->id map is rebuilt per level from it.
#include <cstdlib>
#include <vector>

#include "internal.h"
#include "scan.cuh"

namespace fstc {

namespace {

constexpr unsigned long long RS_EMPTY = ~0ull;

__device__ __forceinline__ uint64_t rmix64(uint64_t k) {
    k ^= k >> 33; k *= 0xff51afd7ed558ccdULL;
    k ^= k >> 33; k *= 0xc4ceb9fe1a85ec53ULL;
    k ^= k >> 33;
    return k;
}

// ------------------------------------------------------------------------------------------ segment bookkeeping
// A record stream is a set of segments inside one buffer: segment s = data[start[s] .. start[s] + cnt[s]).
struct SegView {
    const unsigned long long *data;
    const int64_t *start;      // [n_seg + 1]
    const uint32_t *cnt;       // [n_seg]
    int n_seg;
};

constexpr int SC_TILE = 4096;
constexpr int SC_THREADS = 512;
constexpr int SC_IPT = SC_TILE / SC_THREADS;
constexpr int SC_MAX_BINS = 1024;

// tile_first[s] = number of SC_TILE tiles of the segments before s; tile_first[n_seg] = total.  n_seg <= 1024.
__global__ void __launch_bounds__(1024) rs_seg_tiles(SegView in, int tile, int64_t *__restrict__ tile_first) {
    __shared__ int64_t s_w[32];
    const int s = threadIdx.x, lane = s & 31, warp = s >> 5;
    int64_t t = (s < in.n_seg) ? (static_cast<int64_t>(in.cnt[s]) + tile - 1) / tile : 0;
    int64_t incl = t;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int64_t v = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += v;
    }
    if (lane == 31) s_w[warp] = incl;
    __syncthreads();
    int64_t base = 0;
    for (int w = 0; w < warp; ++w) base += s_w[w];
    if (s < in.n_seg) tile_first[s] = base + incl - t;
    if (s == in.n_seg - 1) tile_first[in.n_seg] = base + incl;
}

// capacity of every output bin of segment s: exact = 0: cnt[s] / nbins * (1 + 1/slack_div) + slack_add (uniform
// hashing); exact = 1: the count a previous overflowing attempt left in the cursor.
__global__ void rs_bin_caps(SegView in, int nbins, int slack_div, uint32_t slack_add, uint32_t fixed_cap,
                            const uint32_t *__restrict__ cursor, int cur_stride, int exact, uint32_t *__restrict__ cap) {
    const int64_t g = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (g >= static_cast<int64_t>(in.n_seg) * nbins) return;
    if (exact) { cap[g] = cursor[static_cast<size_t>(g) * cur_stride]; return; }
    const uint32_t n = in.cnt[g / nbins];
    if (fixed_cap) { cap[g] = fixed_cap < n ? fixed_cap : n; return; }
    const uint64_t mean = (static_cast<uint64_t>(n) + nbins - 1) / nbins;
    uint64_t c = mean + mean / slack_div + slack_add;
    if (c > n) c = n;                                           // a bin never holds more than its whole segment
    cap[g] = static_cast<uint32_t>(c);
}

__global__ void rs_check_overflow(const uint32_t *__restrict__ cursor, int cur_stride, const uint32_t *__restrict__ cap,
                                  int64_t nb, unsigned *__restrict__ flag) {
    const int64_t g = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    const bool over = g < nb && cursor[static_cast<size_t>(g) * cur_stride] > cap[g];
    if (__any_sync(0xffffffffu, over) && (threadIdx.x & 31) == 0) atomicOr(flag, 1u);
}

// ------------------------------------------------------------------------------------------ staged scatter
// FN 0: bin = bits [hshift, hshift + log2 nbins) of mix64(record >> shift)   (hash partition on the key)
// FN 1: bin = (record >> 32) >> hshift                                        (position window of a (pos,id) record)
template <int FN>
__device__ __forceinline__ uint32_t rs_bin(unsigned long long r, int shift, int hshift, uint32_t mask) {
    if (FN == 0) return static_cast<uint32_t>(rmix64(r >> shift) >> hshift) & mask;
    return static_cast<uint32_t>(r >> 32) >> hshift;
}

struct ScatterArgs {
    SegView in;
    const int64_t *tile_first;      // [n_seg + 1]
    unsigned long long *out;
    const int64_t *out_start;       // [n_seg * nbins + 1]
    uint32_t *cursor;               // [n_seg * nbins * cur_stride]
    int cur_stride;
    int shift, hshift, nbins;
};

#ifndef FSTC_SC_MINB
#define FSTC_SC_MINB 2
#endif
template <int FN>
__global__ void __launch_bounds__(SC_THREADS, FSTC_SC_MINB) rs_scatter(ScatterArgs a) {
    extern __shared__ unsigned long long sorted[];             // [SC_TILE], dynamic: the kernel needs > 48 KB in total
    __shared__ uint32_t cnt[SC_MAX_BINS];                       // count, then first slot of the bin in sorted[]
    __shared__ long long gdelta[SC_MAX_BINS];                   // global index of the bin's run minus its first slot
    __shared__ long long glimit[SC_MAX_BINS];                   // end of the bin's global range
    __shared__ uint32_t s_warp[SC_THREADS / 32];
    __shared__ int s_seg;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t mask = static_cast<uint32_t>(a.nbins - 1);

    if (tid == 0) {                                             // segment of this tile
        int lo = 0, hi = a.in.n_seg;                            // last s with tile_first[s] <= blockIdx.x
        while (hi - lo > 1) {
            int mid = (lo + hi) >> 1;
            if (a.tile_first[mid] <= static_cast<int64_t>(blockIdx.x)) lo = mid; else hi = mid;
        }
        s_seg = lo;
    }
    for (int p = tid; p < a.nbins; p += SC_THREADS) cnt[p] = 0;
    __syncthreads();
    const int seg = s_seg;
    const int64_t tile = static_cast<int64_t>(blockIdx.x) - a.tile_first[seg];
    const int64_t seg_n = a.in.cnt[seg];
    const int64_t lo = tile * SC_TILE;
    const int n = static_cast<int>(seg_n - lo < SC_TILE ? seg_n - lo : SC_TILE);
    const unsigned long long *src = a.in.data + a.in.start[seg] + lo;

    unsigned long long rec[SC_IPT];
    uint32_t rk[SC_IPT];
#pragma unroll
    for (int u = 0; u < SC_IPT; ++u) {
        const int i = u * SC_THREADS + tid;
        if (i < n) {
            rec[u] = __ldcs(src + i);
            rk[u] = atomicAdd(&cnt[rs_bin<FN>(rec[u], a.shift, a.hshift, mask)], 1u);
        }
    }
    __syncthreads();
    // exclusive scan over the bins (two per thread), one global reservation per non-empty bin
    const int p0 = 2 * tid;
    const uint32_t c0 = p0 < a.nbins ? cnt[p0] : 0u, c1 = p0 + 1 < a.nbins ? cnt[p0 + 1] : 0u;
    uint32_t incl = c0 + c1;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        uint32_t v = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += v;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    uint32_t ex = incl - (c0 + c1);
    for (int w = 0; w < warp; ++w) ex += s_warp[w];
    const int64_t gbin0 = static_cast<int64_t>(seg) * a.nbins;
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        const int p = p0 + k;
        const uint32_t c = k ? c1 : c0;
        if (p < a.nbins) {
            cnt[p] = ex;
            if (c) {
                const uint32_t g = atomicAdd(&a.cursor[static_cast<size_t>(gbin0 + p) * a.cur_stride], c);
                gdelta[p] = a.out_start[gbin0 + p] + static_cast<long long>(g) - static_cast<long long>(ex);
                glimit[p] = a.out_start[gbin0 + p + 1];
            }
            ex += c;
        }
    }
    __syncthreads();
#pragma unroll
    for (int u = 0; u < SC_IPT; ++u) {
        const int i = u * SC_THREADS + tid;
        if (i < n) sorted[cnt[rs_bin<FN>(rec[u], a.shift, a.hshift, mask)] + rk[u]] = rec[u];
    }
    __syncthreads();
    for (int i = tid; i < n; i += SC_THREADS) {
        const unsigned long long r = sorted[i];
        const uint32_t p = rs_bin<FN>(r, a.shift, a.hshift, mask);
        const long long dst = gdelta[p] + i;
        if (dst < glimit[p]) a.out[dst] = r;                    // a full bin drops the record; the host retries
    }
}

// ------------------------------------------------------------------------------------------ per-bin dedupe
// One block per bin.  keys[]/ids[] in shared memory map the bin's keys to state ids: the existing states of the bin
// are entered first, then every arc record finds its key or creates it.  New ids are handed out per round of
// DD_TILE records with one global atomicAdd; the winner of a key writes pair[id].  Output: (pos << 32 | id), dense,
// at out[out_off[bin] + i].
constexpr int DD_THREADS = 256;
constexpr int DD_IPT = 4;
constexpr int DD_TILE = DD_THREADS * DD_IPT;
#ifndef FSTC_DD_SLOTS
#define FSTC_DD_SLOTS 4096
#endif
#ifndef FSTC_DD_TARGET
#define FSTC_DD_TARGET 1400
#endif
constexpr int DD_SLOTS = FSTC_DD_SLOTS;        // keys 8 B + ids 4 B per slot, in shared memory
constexpr int DD_TARGET = FSTC_DD_TARGET;      // aimed maximum of the mean number of distinct keys per bin

struct DedupeArgs {
    SegView st;                // state records  key << ib | id
    SegView arcs;              // arc records    key << pb | pos
    int ib, pb;
    const int64_t *out_off;    // [n_bins + 1]
    unsigned long long *out;
    uint64_t nq2;
    unsigned long long *n_states;
    int2 *pair;
    unsigned *err;             // set when a bin holds more distinct keys than the shared-memory map
};

__device__ __forceinline__ int dd_find_or_claim(unsigned long long *keys, unsigned long long key, bool *won) {
    uint32_t s = static_cast<uint32_t>(rmix64(key)) & (DD_SLOTS - 1);   // low hash bits: the bins use the top ones
    for (int probes = 0; probes < DD_SLOTS; ++probes) {
        const unsigned long long old = atomicCAS(&keys[s], RS_EMPTY, key);
        if (old == RS_EMPTY) { *won = true; return static_cast<int>(s); }
        if (old == key) { *won = false; return static_cast<int>(s); }
        s = (s + 1) & (DD_SLOTS - 1);
    }
    return -1;
}

__global__ void __launch_bounds__(DD_THREADS) rs_dedupe(DedupeArgs a) {
    extern __shared__ unsigned long long keys[];               // [DD_SLOTS]
    uint32_t *ids = reinterpret_cast<uint32_t *>(keys + DD_SLOTS);
    __shared__ uint32_t s_warp[DD_THREADS / 32];
    __shared__ unsigned long long s_base;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t bin = blockIdx.x;
    const int64_t sc = a.st.cnt[bin];
    const int64_t ac = a.arcs.cnt[bin];
    if (ac == 0) return;                                       // nothing to resolve in this bin
    for (int i = tid; i < DD_SLOTS; i += DD_THREADS) keys[i] = RS_EMPTY;
    __syncthreads();
    const unsigned long long *sp = a.st.data + a.st.start[bin];
    const unsigned long long idmask = (1ull << a.ib) - 1;
    for (int64_t i = tid; i < sc; i += DD_THREADS) {
        const unsigned long long r = sp[i];
        bool won;
        const int s = dd_find_or_claim(keys, r >> a.ib, &won);
        if (s < 0) atomicOr(a.err, 1u); else ids[s] = static_cast<uint32_t>(r & idmask);
    }
    __syncthreads();
    const unsigned long long *ap = a.arcs.data + a.arcs.start[bin];
    unsigned long long *op = a.out + a.out_off[bin];
    const unsigned long long posmask = (1ull << a.pb) - 1;
    for (int64_t base = 0; base < ac; base += DD_TILE) {
        unsigned long long key[DD_IPT];
        uint32_t pos[DD_IPT];
        int slot[DD_IPT];
        uint32_t wonmask = 0;
#pragma unroll
        for (int u = 0; u < DD_IPT; ++u) {
            const int64_t i = base + u * DD_THREADS + tid;
            slot[u] = -2;
            if (i < ac) {
                const unsigned long long r = __ldcs(ap + i);
                key[u] = r >> a.pb;
                pos[u] = static_cast<uint32_t>(r & posmask);
                bool won;
                slot[u] = dd_find_or_claim(keys, key[u], &won);
                if (slot[u] < 0) atomicOr(a.err, 1u);
                else if (won) wonmask |= 1u << u;
            }
        }
        const uint32_t n_won = __popc(wonmask);
        uint32_t incl = n_won;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            uint32_t v = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += v;
        }
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        if (tid == 0) {
            uint32_t tot = 0;
#pragma unroll
            for (int w = 0; w < DD_THREADS / 32; ++w) { uint32_t c = s_warp[w]; s_warp[w] = tot; tot += c; }
            s_base = tot ? atomicAdd(a.n_states, static_cast<unsigned long long>(tot)) : 0ull;
        }
        __syncthreads();
        uint32_t next_id = static_cast<uint32_t>(s_base) + s_warp[warp] + (incl - n_won);
#pragma unroll
        for (int u = 0; u < DD_IPT; ++u) {
            if (wonmask >> u & 1u) {
                const uint32_t id = next_id++;
                ids[slot[u]] = id;
                const unsigned long long q1 = key[u] / a.nq2;
                a.pair[id] = make_int2(static_cast<int>(q1), static_cast<int>(key[u] - q1 * a.nq2));
            }
        }
        __syncthreads();
#pragma unroll
        for (int u = 0; u < DD_IPT; ++u) {
            const int64_t i = base + u * DD_THREADS + tid;
            if (i < ac) {
                const uint32_t id = slot[u] >= 0 ? ids[slot[u]] : 0u;
                __stcs(op + i, (static_cast<unsigned long long>(pos[u]) << 32) | id);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------ id scatter
// (pos << 32 | id) records of one position window -> the target column.  MODE 0: o_tgt[pos] = id;
// MODE 1: the id goes into the target field of a sort record (key bits shift_t and up).
constexpr int SI_THREADS = 256;
constexpr int SI_IPT = 8;
constexpr int SI_TILE = SI_THREADS * SI_IPT;

template <int MODE>
__global__ void __launch_bounds__(SI_THREADS) rs_scatter_ids(SegView in, const int64_t *__restrict__ tile_first,
                                                             int32_t *__restrict__ o_tgt, uint4 *__restrict__ sortrec,
                                                             int shift_t) {
    __shared__ int s_seg;
    if (threadIdx.x == 0) {
        int lo = 0, hi = in.n_seg;
        while (hi - lo > 1) {
            int mid = (lo + hi) >> 1;
            if (tile_first[mid] <= static_cast<int64_t>(blockIdx.x)) lo = mid; else hi = mid;
        }
        s_seg = lo;
    }
    __syncthreads();
    const int seg = s_seg;
    const int64_t lo = (static_cast<int64_t>(blockIdx.x) - tile_first[seg]) * SI_TILE;
    const int64_t seg_n = in.cnt[seg];
    const unsigned long long *src = in.data + in.start[seg] + lo;
    unsigned long long r[SI_IPT];
#pragma unroll
    for (int u = 0; u < SI_IPT; ++u) {
        const int64_t i = lo + u * SI_THREADS + threadIdx.x;
        r[u] = i < seg_n ? __ldcs(src + u * SI_THREADS + threadIdx.x) : RS_EMPTY;
    }
#pragma unroll
    for (int u = 0; u < SI_IPT; ++u) {
        if (r[u] != RS_EMPTY) {
            const uint32_t pos = static_cast<uint32_t>(r[u] >> 32), id = static_cast<uint32_t>(r[u]);
            if (MODE == 0) o_tgt[pos] = static_cast<int32_t>(id);
            else {
                const unsigned long long k = static_cast<unsigned long long>(id) << shift_t;
                uint32_t *w = reinterpret_cast<uint32_t *>(sortrec + pos);
                w[0] |= static_cast<uint32_t>(k);              // the emit kernel left the target bits zero
                w[1] |= static_cast<uint32_t>(k >> 32);
            }
        }
    }
}

// state records key << ib | id, in id order
__global__ void rs_state_records(const int2 *__restrict__ pair, int64_t n, uint64_t nq2, int ib,
                                 unsigned long long *__restrict__ out) {
    const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int2 p = pair[i];
    const unsigned long long key = static_cast<uint64_t>(static_cast<uint32_t>(p.x)) * nq2 + static_cast<uint32_t>(p.y);
    out[i] = (key << ib) | static_cast<unsigned long long>(i);
}

__global__ void rs_set_u32(uint32_t *p, uint32_t v) { *p = v; }
__global__ void rs_window_starts(int64_t *start, int n_win, int cshift) {
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w <= n_win) start[w] = static_cast<int64_t>(w) << cshift;
}

__global__ void rs_compact_counts(const uint32_t *__restrict__ cursor, int cur_stride, int64_t nb, uint32_t *__restrict__ cnt) {
    const int64_t g = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (g < nb) cnt[g] = cursor[static_cast<size_t>(g) * cur_stride];
}

// ------------------------------------------------------------------------------------------ host side
inline unsigned rs_blocks(int64_t n, int threads = 256) { return static_cast<unsigned>(ceil_div(n > 0 ? n : 1, threads)); }

// FSTC_RS_TRACE=1 prints the device time of every resolve kernel to stderr (debug knob, off by default)
struct RsTrace {
    struct Span { const char *name; int64_t n; cudaEvent_t a, b; };
    std::vector<Span> spans;
    bool on = getenv("FSTC_RS_TRACE") != nullptr;
    int begin(Ctx &c, const char *name, int64_t n) {
        if (!on) return -1;
        Span s{name, n, nullptr, nullptr};
        cudaEventCreate(&s.a); cudaEventCreate(&s.b);
        cudaEventRecord(s.a, c.stream);
        spans.push_back(s);
        return static_cast<int>(spans.size()) - 1;
    }
    void end(Ctx &c, int h) { if (h >= 0) cudaEventRecord(spans[h].b, c.stream); }
    void report() {
        for (auto &s : spans) {
            float ms = 0.f;
            cudaEventSynchronize(s.b);
            cudaEventElapsedTime(&ms, s.a, s.b);
            fprintf(stderr, "[fstc resolve] %-22s n=%-11lld %8.3f ms\n", s.name, static_cast<long long>(s.n), ms);
            cudaEventDestroy(s.a); cudaEventDestroy(s.b);
        }
        spans.clear();
    }
};
thread_local RsTrace g_trace;

struct SegSet {                       // device arrays of a segmented record stream
    DBuf<unsigned long long> own;     // storage, unless the stream borrows the caller's buffer
    const unsigned long long *data = nullptr;
    DBuf<int64_t> start;              // [n_seg + 1]
    DBuf<uint32_t> cnt;               // [n_seg]
    int64_t n_seg = 0;
    SegView view() const { return SegView{data, start.p, cnt.p, static_cast<int>(n_seg)}; }
};

SegSet single_segment(Ctx &c, const unsigned long long *data, int64_t n) {
    SegSet s;
    s.data = data;
    s.n_seg = 1;
    s.start.alloc(c, 2);
    s.cnt.alloc(c, 1);
    const int64_t st[2] = {0, n};
    const uint32_t cn = static_cast<uint32_t>(n);
    FSTC_CUDA(cudaMemcpyAsync(s.start.p, st, sizeof st, cudaMemcpyHostToDevice, c.stream));
    FSTC_CUDA(cudaMemcpyAsync(s.cnt.p, &cn, sizeof cn, cudaMemcpyHostToDevice, c.stream));
    return s;
}

// One staged scatter pass: every segment of `in` is split into `nbins` bins.  Bin capacities are a guess from
// uniform hashing (or `fixed_cap`); if a bin overflows, the cursors of the failed attempt hold the exact counts
// and the pass runs once more with those.
template <int FN>
SegSet scatter_pass(Ctx &c, const SegSet &in, int shift, int hshift, int nbins, uint32_t fixed_cap) {
    if (in.n_seg > 1024 || nbins > SC_MAX_BINS) fail(FSTC_ERR_CAPACITY, "resolve: too many segments (%lld x %d)",
                                                    static_cast<long long>(in.n_seg), nbins);
    const int64_t nb = in.n_seg * nbins;
    const int cur_stride = nb <= 4096 ? 32 : 8;                  // hot counters sit in sectors of their own
    DBuf<int64_t> tile_first(c, in.n_seg + 1);
    rs_seg_tiles<<<1, 1024, 0, c.stream>>>(in.view(), SC_TILE, tile_first.p);
    FSTC_LAUNCH_CHECK();
    DBuf<uint32_t> cap(c, nb), cursor(c, nb * cur_stride);
    DBuf<unsigned> flag(c, 1);
    SegSet out;
    out.n_seg = nb;
    out.start.alloc(c, nb + 1);
    static bool attr_set = false;
    if (!attr_set) {
        FSTC_CUDA(cudaFuncSetAttribute(rs_scatter<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, SC_TILE * 8));
        FSTC_CUDA(cudaFuncSetAttribute(rs_scatter<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, SC_TILE * 8));
        attr_set = true;
    }
    for (int attempt = 0;; ++attempt) {
        rs_bin_caps<<<rs_blocks(nb), 256, 0, c.stream>>>(in.view(), nbins, 16, 192u, fixed_cap, cursor.p, cur_stride,
                                                         attempt, cap.p);
        FSTC_LAUNCH_CHECK();
        exclusive_scan<uint32_t>(c, cap.p, nb, out.start.p);
        int64_t totals[2];
        FSTC_CUDA(cudaMemcpyAsync(&totals[0], tile_first.p + in.n_seg, sizeof(int64_t), cudaMemcpyDeviceToHost, c.stream));
        FSTC_CUDA(cudaMemcpyAsync(&totals[1], out.start.p + nb, sizeof(int64_t), cudaMemcpyDeviceToHost, c.stream));
        c.sync();
        out.own.alloc(c, totals[1]);
        out.data = out.own.p;
        FSTC_CUDA(cudaMemsetAsync(cursor.p, 0, sizeof(uint32_t) * nb * cur_stride, c.stream));
        FSTC_CUDA(cudaMemsetAsync(flag.p, 0, sizeof(unsigned), c.stream));
        if (totals[0] > 0) {
            ScatterArgs a{in.view(), tile_first.p, out.own.p, out.start.p, cursor.p, cur_stride, shift, hshift, nbins};
            const int h = g_trace.begin(c, FN == 0 ? "scatter(key)" : "scatter(pos)", totals[0] * SC_TILE);
            rs_scatter<FN><<<static_cast<unsigned>(totals[0]), SC_THREADS, SC_TILE * 8, c.stream>>>(a);
            FSTC_LAUNCH_CHECK();
            g_trace.end(c, h);
        }
        rs_check_overflow<<<rs_blocks(nb), 256, 0, c.stream>>>(cursor.p, cur_stride, cap.p, nb, flag.p);
        FSTC_LAUNCH_CHECK();
        c.n_launch += 4;
        if (!read_scalar(c, flag.p)) break;
        if (attempt == 1) fail(FSTC_ERR_CUDA, "internal: resolve scatter overflowed with exact capacities");
    }
    out.cnt.alloc(c, nb);
    rs_compact_counts<<<rs_blocks(nb), 256, 0, c.stream>>>(cursor.p, cur_stride, nb, out.cnt.p);
    FSTC_LAUNCH_CHECK();
    c.n_launch += 1;
    return out;
}

// hash partition of a record stream into 2^(b1+b2) bins (b1 = the top hash bits, then b2)
SegSet partition_by_key(Ctx &c, const unsigned long long *recs, int64_t n, int shift, int b1, int b2) {
    SegSet cur = single_segment(c, recs, n);
    if (b1 > 0) cur = scatter_pass<0>(c, cur, shift, 64 - b1, 1 << b1, 0);
    if (b2 > 0) cur = scatter_pass<0>(c, cur, shift, 64 - b1 - b2, 1 << b2, 0);
    return cur;
}

}  // namespace

int resolve_bits_needed(int64_t n_records_and_states) {
    int b = 0;
    while (b < 20 && (n_records_and_states >> b) > DD_TARGET) ++b;
    return b;
}

void resolve_partitioned(Ctx &c, const ResolveJob &j) {
    static bool attr_set = false;
    if (!attr_set) {
        FSTC_CUDA(cudaFuncSetAttribute(rs_dedupe, cudaFuncAttributeMaxDynamicSharedMemorySize, DD_SLOTS * 12));
        attr_set = true;
    }
    const int ib = bits_for(static_cast<uint64_t>(j.n_states_before > 1 ? j.n_states_before - 1 : 1));
    if (j.key_bits + ib > 64 || j.key_bits + j.pos_bits > 64 || j.pos_bits > 32)
        fail(FSTC_ERR_CAPACITY, "resolve: key (%d bits) + id/position (%d/%d bits) exceed 64 bits", j.key_bits, ib, j.pos_bits);
    int bits = j.force_bits >= 0 ? j.force_bits : resolve_bits_needed(j.n_states_before + j.n_records);
    for (;; ++bits) {
        if (bits > 20) fail(FSTC_ERR_CAPACITY, "resolve: more than 2^20 bins needed");
        const int b1 = bits < 10 ? bits : 10, b2 = bits - b1;
        // 1-2. records of the existing states and of the arcs, partitioned the same way
        DBuf<unsigned long long> st_recs(c, j.n_states_before);
        rs_state_records<<<rs_blocks(j.n_states_before), 256, 0, c.stream>>>(j.pair, j.n_states_before, j.nq2, ib, st_recs.p);
        FSTC_LAUNCH_CHECK();
        c.n_launch += 1;
        SegSet st = partition_by_key(c, st_recs.p, j.n_states_before, ib, b1, b2);
        if (bits > 0) st_recs.release();
        SegSet arcs = partition_by_key(c, j.keypos, j.n_records, j.pos_bits, b1, b2);
        // 3. per-bin dedupe
        const int64_t nb = int64_t(1) << bits;
        DBuf<int64_t> out_off(c, nb + 1);
        exclusive_scan<uint32_t>(c, arcs.cnt.p, nb, out_off.p);
        DBuf<unsigned long long> posid(c, j.n_records);
        DBuf<unsigned> err(c, 1);
        FSTC_CUDA(cudaMemsetAsync(err.p, 0, sizeof(unsigned), c.stream));
        const unsigned long long n_before = static_cast<unsigned long long>(j.n_states_before);
        FSTC_CUDA(cudaMemcpyAsync(j.n_states, &n_before, sizeof n_before, cudaMemcpyHostToDevice, c.stream));
        DedupeArgs d{st.view(), arcs.view(), ib, j.pos_bits, out_off.p, posid.p, j.nq2, j.n_states, j.pair, err.p};
        const int hd = g_trace.begin(c, "dedupe", nb);
        rs_dedupe<<<static_cast<unsigned>(nb), DD_THREADS, DD_SLOTS * 12, c.stream>>>(d);
        FSTC_LAUNCH_CHECK();
        g_trace.end(c, hd);
        c.n_launch += 1;
        if (read_scalar(c, err.p)) continue;                     // a bin outgrew shared memory: halve the bins, again
        st = SegSet();
        arcs = SegSet();
        // 4. ids back to the target column, one position window at a time
        const int pbits = bits_for(static_cast<uint64_t>(j.n_positions > 1 ? j.n_positions - 1 : 1));
        const int cshift = pbits - 10 > 22 ? pbits - 10 : 22;
        const int n_win = static_cast<int>(((j.n_positions > 0 ? j.n_positions : 1) + (int64_t(1) << cshift) - 1) >> cshift);
        SegSet win = single_segment(c, posid.p, j.n_records);
        if (n_win > 1) {
            win = scatter_pass<1>(c, win, 0, cshift, n_win, static_cast<uint32_t>(1u << cshift));
            posid.release();
        }
        DBuf<int64_t> tile_first(c, win.n_seg + 1);
        rs_seg_tiles<<<1, 1024, 0, c.stream>>>(win.view(), SI_TILE, tile_first.p);
        FSTC_LAUNCH_CHECK();
        const int64_t tiles = read_scalar(c, tile_first.p + win.n_seg);
        const int hs = g_trace.begin(c, "scatter_ids", tiles * SI_TILE);
        if (tiles > 0) {
            if (j.sortrec)
                rs_scatter_ids<1><<<static_cast<unsigned>(tiles), SI_THREADS, 0, c.stream>>>(win.view(), tile_first.p, nullptr,
                                                                                          j.sortrec, j.shift_t);
            else
                rs_scatter_ids<0><<<static_cast<unsigned>(tiles), SI_THREADS, 0, c.stream>>>(win.view(), tile_first.p, j.o_tgt,
                                                                                          nullptr, 0);
            FSTC_LAUNCH_CHECK();
        }
        g_trace.end(c, hs);
        c.n_launch += 2;
        c.sync();                                                // temporaries are released below
        if (g_trace.on) g_trace.report();
        return;
    }
}

}  // namespace fstc
