// Partitioned target resolution: the visited-set step of a BIG level (PAPER.md:237-239 adapted).
//
// The paper tests and sets one entry of a dense |Q1||Q2| table per composed arc (atomicOr, :237).  On a B200 a
// random 32-byte DRAM sector costs ~21 ps to read and ~45 ps to dirty (measured), so at
// 10^9 arcs per level the per-arc probe of any table that does not fit the 126 MB L2 bounds the whole path.  Big
// levels are therefore resolved like a radix hash join, with streaming passes only:
//
//   1. the emit kernel leaves the target key of every composed arc, in rank order; every existing state leaves a
//      record (key, id);
//   2. both streams are partitioned by the top bits of a hash of the key (one or two staged scatter passes: a block
//      sorts a tile of 8192 / 4096 records by bin in shared memory and appends whole runs), until a bin holds at most
//      ~2000 distinct keys.  On the arc stream a pass also records where every record went and came from;
//   3. one block per bin builds the bin's key->id map in SHARED memory (old states first), finds or creates the id
//      of every arc key, allocates new ids (one global atomicAdd per round) and writes pair[id];
//   4. the ids travel back through the recorded permutations, tile by tile: a block reads the ids of its tile's records
//      in SORTED order (runs of neighbours, not 32 far-apart words per warp), un-permutes them in shared memory and
//      writes them out in input order; the last pass writes the target column, coalesced, in rank order.
//
// Nothing persists between levels except pair[] (id -> (q1,q2)): the key->id map is rebuilt per level from it.
#include <cstdlib>
#include <ctime>
#include <vector>

#include "internal.h"
#include "scan.cuh"

namespace fstc {

namespace {

constexpr unsigned long long RS_EMPTY = ~0ull;

// 64-bit mixer (two multiply / xor-shift rounds).  The bins use its top bits, the shared-memory map its low ones.
__device__ __forceinline__ uint64_t rmix64(uint64_t k) {
    k *= 0x9E3779B97F4A7C15ULL;
    k ^= k >> 32;
    k *= 0xD6E8FEB86659FD93ULL;
    k ^= k >> 32;
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

// Tile of a scatter pass (template parameter): 8192 for the first pass — its runs are twice as long, which makes the
// last gather, the one that writes the target column, read whole sectors — and 4096 for the second.
constexpr int SC_TILE_BIG = 8192, SC_TILE_SMALL = 4096;
constexpr int SC_THREADS = 512;
constexpr int SC_MAX_BINS = 1024;

// tile_first[s] = number of tiles of the segments before s; tile_first[n_seg] = total.  n_seg <= 1024.
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
__global__ void rs_bin_caps(SegView in, int nbins, int slack_div, uint32_t slack_add, const uint32_t *__restrict__ cursor,
                            int cur_stride, int exact, uint32_t *__restrict__ cap) {
    const int64_t g = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (g >= static_cast<int64_t>(in.n_seg) * nbins) return;
    // capacities are multiples of 8 records: every bin then starts 16-byte aligned in the record, dest and perm arrays (bulk copies)
    if (exact) { cap[g] = (cursor[static_cast<size_t>(g) * cur_stride] + 7u) & ~7u; return; }
    const uint32_t n = in.cnt[g / nbins];
    const uint64_t mean = (static_cast<uint64_t>(n) + nbins - 1) / nbins;
    uint64_t c = mean + mean / slack_div + slack_add;
    if (c > n) c = n;                                           // a bin never holds more than its whole segment
    cap[g] = (static_cast<uint32_t>(c) + 7u) & ~7u;
}

__global__ void rs_check_overflow(const uint32_t *__restrict__ cursor, int cur_stride, const uint32_t *__restrict__ cap,
                                  int64_t nb, unsigned *__restrict__ flag) {
    const int64_t g = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    const bool over = g < nb && cursor[static_cast<size_t>(g) * cur_stride] > cap[g];
    if (__any_sync(0xffffffffu, over) && (threadIdx.x & 31) == 0) atomicOr(flag, 1u);
}

__global__ void rs_compact_counts(const uint32_t *__restrict__ cursor, int cur_stride, int64_t nb, uint32_t *__restrict__ cnt) {
    const int64_t g = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (g < nb) cnt[g] = cursor[static_cast<size_t>(g) * cur_stride];
}

// first tile of segment `seg` <= blockIdx.x < first tile of seg + 1
__device__ __forceinline__ int rs_find_segment(const int64_t *tile_first, int n_seg) {
    int lo = 0, hi = n_seg;
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (tile_first[mid] <= static_cast<int64_t>(blockIdx.x)) lo = mid; else hi = mid;
    }
    return lo;
}

// ------------------------------------------------------------------------------------------ staged scatter
// bin of a record = bits [hshift, hshift + log2 nbins) of mix64(record >> shift).  A tile of SC_TILE records is sorted
// by bin in shared memory; every non-empty bin reserves room for its run with one global atomicAdd and the runs go out
// with consecutive threads writing consecutive addresses.  DEST: the pass also records, per tile and in sorted order,
// where every record went (dest) and where it came from (perm), so that ids can travel back with the same locality.
struct ScatterArgs {
    SegView in;
    const int64_t *tile_first;      // [n_seg + 1]
    unsigned long long *out;
    const int64_t *out_start;       // [n_seg * nbins + 1]
    uint32_t *cursor;               // [n_seg * nbins * cur_stride]
    uint32_t *dest;                 // DEST: [input buffer length] output index of the record in SORTED slot i of its tile
    uint16_t *perm;                 // DEST: [input buffer length] tile-local input index of that record
    int cur_stride;
    int shift, hshift, nbins;
};

#ifndef FSTC_SC_MINB
#define FSTC_SC_MINB 3
#endif
// FSTC_SC_TMA=1 (default): a whole, 16-byte aligned tile is brought into shared memory with ONE 1-D bulk copy (cp.async.bulk +
// mbarrier, SASS UBLKCP) instead of 8-16 global loads per thread: rs_scatter 16.7 -> 15.1 ms on `large` (the LSU is what this
// kernel is short of: its shared-memory atomics go through it too).
#ifndef FSTC_SC_TMA
#define FSTC_SC_TMA 1
#endif
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, unsigned long long *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src),
                 "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, uint32_t parity) {
    asm volatile("{\n.reg .pred P1;\nLAB_WAIT:\nmbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n@P1 bra DONE;\nbra LAB_WAIT;\nDONE:\n}" ::"r"(smem_u32(bar)),
                 "r"(parity)
                 : "memory");
}
template <bool DEST, int SC_TILE>
__global__ void __launch_bounds__(SC_THREADS, SC_TILE == SC_TILE_BIG ? 2 : FSTC_SC_MINB) rs_scatter(ScatterArgs a) {
    constexpr int SC_IPT = SC_TILE / SC_THREADS;
    extern __shared__ unsigned long long sorted[];             // [SC_TILE] records, then uint32 smeta[SC_TILE]
    uint32_t *smeta = reinterpret_cast<uint32_t *>(sorted + SC_TILE);   // tile-local input index << 16 | bin
    __shared__ uint32_t cnt[SC_MAX_BINS];                       // count, then first slot of the bin in sorted[]
    __shared__ long long gdelta[SC_MAX_BINS];                   // global index of the bin's run minus its first slot
    __shared__ uint32_t room[SC_MAX_BINS];                      // records of the run that still fit the bin
    __shared__ uint32_t s_warp[SC_THREADS / 32];
    __shared__ int s_seg;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t mask = static_cast<uint32_t>(a.nbins - 1);

    if (tid == 0) s_seg = rs_find_segment(a.tile_first, a.in.n_seg);
    for (int p = tid; p < a.nbins; p += SC_THREADS) cnt[p] = 0;
    __syncthreads();
    const int seg = s_seg;
    const int64_t tile = static_cast<int64_t>(blockIdx.x) - a.tile_first[seg];
    const int64_t seg_n = a.in.cnt[seg];
    const int64_t lo = tile * SC_TILE;
    const int n = static_cast<int>(seg_n - lo < SC_TILE ? seg_n - lo : SC_TILE);
    const int64_t in_base = a.in.start[seg] + lo;
    const unsigned long long *src = a.in.data + in_base;

    unsigned long long rec[SC_IPT];
    uint32_t br[SC_IPT];                                        // bin << 16 | rank inside the bin (tile-local)
#if FSTC_SC_TMA
    __shared__ unsigned long long s_bar;
    const bool bulk = n == SC_TILE && (in_base & 1) == 0;       // whole tile, 16-byte aligned: one bulk copy into `sorted`
    if (bulk) {
        if (tid == 0) mbar_init(&s_bar, 1);
        __syncthreads();
        if (tid == 0) { mbar_expect_tx(&s_bar, SC_TILE * 8u); bulk_g2s(sorted, src, SC_TILE * 8u, &s_bar); }
        mbar_wait(&s_bar, 0);
#pragma unroll
        for (int u = 0; u < SC_IPT; ++u) rec[u] = sorted[u * SC_THREADS + tid];
    } else
#endif
#pragma unroll
    for (int u = 0; u < SC_IPT; ++u) {
        const int i = u * SC_THREADS + tid;
        if (i < n) rec[u] = __ldcs(src + i);
    }
#pragma unroll
    for (int u = 0; u < SC_IPT; ++u) {
        const int i = u * SC_THREADS + tid;
        if (i < n) {
            const uint32_t b = static_cast<uint32_t>(rmix64(rec[u] >> a.shift) >> a.hshift) & mask;
            br[u] = (b << 16) | atomicAdd(&cnt[b], 1u);
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
                const int64_t b0 = a.out_start[gbin0 + p], b1 = a.out_start[gbin0 + p + 1];
                const uint32_t g = atomicAdd(&a.cursor[static_cast<size_t>(gbin0 + p) * a.cur_stride], c);
                gdelta[p] = b0 + static_cast<long long>(g) - static_cast<long long>(ex);
                const int64_t left = (b1 - b0) - static_cast<int64_t>(g);
                room[p] = left <= 0 ? 0u : (left < c ? static_cast<uint32_t>(left) : c);
            }
            ex += c;
        }
    }
    __syncthreads();
#pragma unroll
    for (int u = 0; u < SC_IPT; ++u) {
        const int i = u * SC_THREADS + tid;
        if (i < n) {
            const uint32_t b = br[u] >> 16, rk = br[u] & 0xFFFFu;
            const uint32_t slot = cnt[b] + rk;
            sorted[slot] = rec[u];
            smeta[slot] = (static_cast<uint32_t>(i) << 16) | b;
        }
    }
    __syncthreads();
    for (int i = tid; i < n; i += SC_THREADS) {
        const uint32_t m = smeta[i], p = m & 0xFFFFu;
        const bool fits = static_cast<uint32_t>(i) - cnt[p] < room[p];
        const long long dst = gdelta[p] + i;
        if (fits) a.out[dst] = sorted[i];                       // a full bin drops the record; the host retries
        if (DEST) {                                             // the way back: sorted slot -> output index, input index
            a.dest[in_base + i] = fits ? static_cast<uint32_t>(dst) : 0xFFFFFFFFu;   // (a bulk store of the tile's dest[] from shared
            a.perm[in_base + i] = static_cast<uint16_t>(m >> 16);                    //  memory was tried: 15.0 -> 15.7 ms)
        }
    }
}

// ------------------------------------------------------------------------------------------ per-bin dedupe
// One block per bin.  keys[]/ids[] in shared memory map the bin's keys to state ids: the existing states of the bin
// are entered first, then every arc key finds its entry or creates it.  New ids are handed out per round of DD_TILE
// records with one global atomicAdd; the winner of a key writes pair[id].  The id of arc record i of the bin goes to
// ids_out[start[bin] + i], the index the last scatter pass recorded in dest[].
#ifndef FSTC_DD_THREADS
#define FSTC_DD_THREADS 512
#endif
#ifndef FSTC_DD_MINB
#define FSTC_DD_MINB 3
#endif
constexpr int DD_THREADS = FSTC_DD_THREADS;
constexpr int DD_IPT = 4;
constexpr int DD_TILE = DD_THREADS * DD_IPT;
#ifndef FSTC_DD_SLOTS
#define FSTC_DD_SLOTS 4096
#endif
#ifndef FSTC_DD_TARGET
#define FSTC_DD_TARGET 2000
#endif
constexpr int DD_SLOTS = FSTC_DD_SLOTS;        // keys 8 B + ids 4 B per slot, in shared memory (a power of two)
constexpr int DD_SLOT_BITS = DD_SLOTS == 2048 ? 11 : (DD_SLOTS == 4096 ? 12 : (DD_SLOTS == 8192 ? 13 : -1));
static_assert(DD_SLOT_BITS > 0, "DD_SLOTS must be 2048, 4096 or 8192");
constexpr int DD_TARGET = FSTC_DD_TARGET;      // aimed maximum of the mean number of distinct keys per bin
constexpr int DD_SMEM = DD_SLOTS * 12;         // (a bulk copy of a round's keys was tried: 9.2 -> 10.0 ms, a bin is one short round)

struct DedupeArgs {
    SegView st;                // state records  key << ib | id
    SegView arcs;              // arc records    key
    int ib;
    uint32_t *ids_out;         // [length of the arc buffer]
    int q2_bits;               // a key is (q1 << q2_bits) | q2
    unsigned long long *n_states;
    int2 *pair;
    unsigned *err;             // set when a bin holds more distinct keys than the shared-memory map
};

__device__ __forceinline__ int dd_find_or_claim(unsigned long long *keys, unsigned long long key, bool *won) {
    // the bins took the top bits of mix64(key); inside a bin a multiplicative hash of the folded key is independent enough
    uint32_t s = ((static_cast<uint32_t>(key) ^ (static_cast<uint32_t>(key >> 32) * 0x85EBCA6Bu)) * 0x9E3779B1u) >> (32 - DD_SLOT_BITS);
    for (int probes = 0; probes < DD_SLOTS; ++probes) {
        const unsigned long long old = atomicCAS(&keys[s], RS_EMPTY, key);
        if (old == RS_EMPTY) { *won = true; return static_cast<int>(s); }
        if (old == key) { *won = false; return static_cast<int>(s); }
        s = (s + static_cast<uint32_t>(probes) + 1) & (DD_SLOTS - 1);   // triangular steps: no primary clustering, every slot is visited
    }
    return -1;
}

__global__ void __launch_bounds__(DD_THREADS, FSTC_DD_MINB) rs_dedupe(DedupeArgs a) {
    extern __shared__ unsigned long long keys[];               // [DD_SLOTS], then uint32 ids[DD_SLOTS]
    uint32_t *ids = reinterpret_cast<uint32_t *>(keys + DD_SLOTS);
    __shared__ uint32_t s_warp[DD_THREADS / 32];
    __shared__ unsigned long long s_base;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t bin = blockIdx.x;
    const int64_t ac = a.arcs.cnt[bin];
    if (ac == 0) return;                                       // nothing to resolve in this bin
    const int64_t sc = a.st.cnt[bin];
    const int64_t a0 = a.arcs.start[bin], s0 = a.st.start[bin];
    for (int i = tid; i < DD_SLOTS; i += DD_THREADS) keys[i] = RS_EMPTY;
    __syncthreads();
    const unsigned long long idmask = (1ull << a.ib) - 1;
    for (int64_t i = tid; i < sc; i += DD_THREADS) {
        const unsigned long long r = a.st.data[s0 + i];
        bool won;
        const int s = dd_find_or_claim(keys, r >> a.ib, &won);
        if (s < 0) atomicOr(a.err, 1u); else ids[s] = static_cast<uint32_t>(r & idmask);
    }
    __syncthreads();
    const unsigned long long *ap = a.arcs.data + a0;
    uint32_t *op = a.ids_out + a0;
    for (int64_t base = 0; base < ac; base += DD_TILE) {
        unsigned long long key[DD_IPT];
        int slot[DD_IPT];
        uint32_t wonmask = 0;
#pragma unroll
        for (int u = 0; u < DD_IPT; ++u) {
            const int64_t i = base + u * DD_THREADS + tid;
            key[u] = i < ac ? __ldcs(ap + i) : RS_EMPTY;
        }
#pragma unroll
        for (int u = 0; u < DD_IPT; ++u) {
            slot[u] = -2;
            if (key[u] != RS_EMPTY) {
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
                a.pair[id] = make_int2(static_cast<int>(key[u] >> a.q2_bits), static_cast<int>(key[u] & ((1ull << a.q2_bits) - 1)));
            }
        }
        __syncthreads();
#pragma unroll
        for (int u = 0; u < DD_IPT; ++u) {
            const int64_t i = base + u * DD_THREADS + tid;
            if (i < ac) __stcs(op + i, slot[u] >= 0 ? ids[slot[u]] : 0u);
        }
    }
}

// ------------------------------------------------------------------------------------------ ids back through the passes
// A scatter pass undone, tile by tile (the tiles of the pass): thread i reads the id of the record in sorted slot i —
// slots of a bin are neighbours in the output, so a warp reads a few short runs instead of 32 far-apart words — and
// drops it at the record's input index in shared memory; the tile is then written out in input order.
// MODE 0: out[input index] = id (ids of the previous pass's buffer, or the target column when in rank order)
// MODE 1: o_tgt[pos[rank]] = id;  MODE 2: id into the target field (key bits shift_t and up) of sort record `rank`.
#ifndef FSTC_GA_THREADS
#define FSTC_GA_THREADS 512
#endif
constexpr int GA_THREADS = FSTC_GA_THREADS;

struct GatherArgs {
    SegView seg;                    // the INPUT segments of the pass that is undone
    const int64_t *tile_first;
    const uint32_t *dest;           // null: identity (no pass), ids are read at the input index
    const uint16_t *perm;
    const uint32_t *in;
    uint32_t *out;                  // MODE 0
    const uint32_t *pos;            // MODE 1
    int32_t *o_tgt;                 // MODE 1
    uint4 *sortrec;                 // MODE 2
    int shift_t;
};

template <int MODE, int SC_TILE>
__global__ void __launch_bounds__(GA_THREADS) rs_gather_ids(GatherArgs a) {
    constexpr int GA_IPT = SC_TILE / GA_THREADS;
    extern __shared__ __align__(16) unsigned char ga_raw[];
    uint32_t *s_id = reinterpret_cast<uint32_t *>(ga_raw);                    // [SC_TILE] ids in input order (first: the tile of dest)
    uint16_t *s_perm = reinterpret_cast<uint16_t *>(ga_raw + 4 * SC_TILE);    // [SC_TILE] the tile of perm (bulk copy)
    __shared__ int s_seg;
    __shared__ unsigned long long s_bar;
    const int tid = threadIdx.x;
    if (tid == 0) s_seg = rs_find_segment(a.tile_first, a.seg.n_seg);
    __syncthreads();
    const int s = s_seg;
    const int64_t lo = (static_cast<int64_t>(blockIdx.x) - a.tile_first[s]) * SC_TILE;
    const int64_t seg_n = a.seg.cnt[s];
    const int n = static_cast<int>(seg_n - lo < SC_TILE ? seg_n - lo : SC_TILE);
    const int64_t base = a.seg.start[s] + lo;
    if (a.dest) {
        uint32_t d[GA_IPT], li[GA_IPT];
        // a whole, 16-byte aligned tile: dest and perm come in with two bulk copies (segments start at multiples of 8 records)
        const bool bulk = FSTC_SC_TMA && n == SC_TILE && (base & 7) == 0;
        if (bulk) {
            if (tid == 0) mbar_init(&s_bar, 1);
            __syncthreads();
            if (tid == 0) {
                mbar_expect_tx(&s_bar, SC_TILE * 6u);
                bulk_g2s(s_id, a.dest + base, SC_TILE * 4u, &s_bar);
                bulk_g2s(s_perm, a.perm + base, SC_TILE * 2u, &s_bar);
            }
            mbar_wait(&s_bar, 0);
#pragma unroll
            for (int u = 0; u < GA_IPT; ++u) { d[u] = s_id[u * GA_THREADS + tid]; li[u] = s_perm[u * GA_THREADS + tid]; }
            __syncthreads();                                   // every thread holds its part of dest before s_id is overwritten
        } else {
#pragma unroll
            for (int u = 0; u < GA_IPT; ++u) {
                const int i = u * GA_THREADS + tid;
                d[u] = i < n ? __ldcs(a.dest + base + i) : 0xFFFFFFFFu;
                li[u] = i < n ? __ldcs(a.perm + base + i) : 0u;
            }
        }
        uint32_t v[GA_IPT];
#pragma unroll
        for (int u = 0; u < GA_IPT; ++u) v[u] = d[u] != 0xFFFFFFFFu ? __ldg(a.in + d[u]) : 0u;
#pragma unroll
        for (int u = 0; u < GA_IPT; ++u)
            if (u * GA_THREADS + tid < n) s_id[li[u]] = v[u];
        __syncthreads();
    }
#pragma unroll
    for (int u = 0; u < GA_IPT; ++u) {
        const int i = u * GA_THREADS + tid;
        if (i >= n) continue;
        const uint32_t id = a.dest ? s_id[i] : __ldcs(a.in + base + i);
        if (MODE == 0) __stcs(a.out + base + i, id);
        else if (MODE == 1) a.o_tgt[a.pos[base + i]] = static_cast<int32_t>(id);
        else {
            const unsigned long long k = static_cast<unsigned long long>(id) << a.shift_t;
            uint32_t *w = reinterpret_cast<uint32_t *>(a.sortrec + base + i);
            w[0] |= static_cast<uint32_t>(k);                  // the emit kernel left the target bits zero
            w[1] |= static_cast<uint32_t>(k >> 32);
        }
    }
}

// state records key << ib | id, in id order
__global__ void rs_state_records(const int2 *__restrict__ pair, int64_t n, int q2_bits, int ib,
                                 unsigned long long *__restrict__ out) {
    const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int2 p = pair[i];
    const unsigned long long key = (static_cast<unsigned long long>(static_cast<uint32_t>(p.x)) << q2_bits) | static_cast<uint32_t>(p.y);
    out[i] = (key << ib) | static_cast<unsigned long long>(i);
}

// ------------------------------------------------------------------------------------------ host side
inline unsigned rs_blocks(int64_t n, int threads = 256) { return static_cast<unsigned>(ceil_div(n > 0 ? n : 1, threads)); }

// FSTC_RS_TRACE=1 prints the device time of every resolve kernel to stderr (debug knob, off by default)
struct RsTrace {
    struct Span { const char *name; int64_t n; cudaEvent_t a, b; double host_us; unsigned long long reserved; int kind; };
    std::vector<Span> spans;
    bool print = getenv("FSTC_RS_TRACE") != nullptr;
    bool on = print;                                            // also switched on by opts.profile (stage times)
    int begin(Ctx &c, const char *name, int64_t n, int kind = -1) {
        if (!on) return -1;
        Span s{name, n, nullptr, nullptr, 0.0, 0ull, kind};
        timespec ts; clock_gettime(CLOCK_MONOTONIC, &ts);
        s.host_us = ts.tv_sec * 1e6 + ts.tv_nsec * 1e-3;
        (void)cudaMemPoolGetAttribute(device_pool(), cudaMemPoolAttrReservedMemCurrent, &s.reserved);
        cudaEventCreate(&s.a); cudaEventCreate(&s.b);
        cudaEventRecord(s.a, c.stream);
        spans.push_back(s);
        return static_cast<int>(spans.size()) - 1;
    }
    void end(Ctx &c, int h) { if (h >= 0) cudaEventRecord(spans[h].b, c.stream); }
    void report(double *stage_ms) {
        for (auto &s : spans) {
            float ms = 0.f, at = 0.f;
            cudaEventSynchronize(s.b);
            cudaEventElapsedTime(&ms, s.a, s.b);
            cudaEventElapsedTime(&at, spans[0].a, s.a);
            if (stage_ms && s.kind >= 0) stage_ms[s.kind] += ms;
            if (print) fprintf(stderr, "[fstc resolve] %-18s n=%-11lld at %8.3f  %8.3f ms   host at %9.3f ms  pool %.2f GB\n", s.name,
                    static_cast<long long>(s.n), at, ms, (s.host_us - spans[0].host_us) * 1e-3, s.reserved / 1e9);
        }
        for (auto &s : spans) { cudaEventDestroy(s.a); cudaEventDestroy(s.b); }
        spans.clear();
    }
};
thread_local RsTrace g_trace;

struct SegSet {                       // device arrays of a segmented record stream
    DBuf<unsigned long long> own;     // storage, unless the stream borrows the caller's buffer
    const unsigned long long *data = nullptr;
    int64_t length = 0;               // records the buffer spans (segments + gaps)
    DBuf<int64_t> start;              // [n_seg + 1]
    DBuf<uint32_t> cnt;               // [n_seg]
    int64_t n_seg = 0;
    SegView view() const { return SegView{data, start.p, cnt.p, static_cast<int>(n_seg)}; }
};

SegSet single_segment(Ctx &c, const unsigned long long *data, int64_t n) {
    SegSet s;
    s.data = data;
    s.length = n;
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
// uniform hashing; if a bin overflows, the cursors of the failed attempt hold the exact counts and the pass runs
// once more with those.  dest (optional): [in.length], where every input record went.
SegSet scatter_pass(Ctx &c, const SegSet &in, int shift, int hshift, int nbins, bool big_tile, DBuf<uint32_t> *dest,
                    DBuf<uint16_t> *perm) {
    const int SC_TILE = big_tile ? SC_TILE_BIG : SC_TILE_SMALL;
    if (in.n_seg > 1024 || nbins > SC_MAX_BINS) fail(FSTC_ERR_CAPACITY, "resolve: too many segments (%lld x %d)",
                                                    static_cast<long long>(in.n_seg), nbins);
    const int64_t nb = in.n_seg * nbins;
    const int cur_stride = nb <= 4096 ? 32 : 8;                  // hot counters sit in sectors of their own
    const size_t smem = SC_TILE * (sizeof(unsigned long long) + sizeof(uint32_t));
    DBuf<int64_t> tile_first(c, in.n_seg + 1);
    rs_seg_tiles<<<1, 1024, 0, c.stream>>>(in.view(), SC_TILE, tile_first.p);
    FSTC_LAUNCH_CHECK();
    DBuf<uint32_t> cap(c, nb), cursor(c, nb * cur_stride);
    DBuf<unsigned> flag(c, 1);
    SegSet out;
    out.n_seg = nb;
    out.start.alloc(c, nb + 1);
    if (dest) { dest->alloc(c, in.length); perm->alloc(c, in.length); }
    {   // per device and cheap: set on every pass rather than remembered per process
        const int s_big = SC_TILE_BIG * 12, s_small = SC_TILE_SMALL * 12;
        FSTC_CUDA(cudaFuncSetAttribute(rs_scatter<false, SC_TILE_BIG>, cudaFuncAttributeMaxDynamicSharedMemorySize, s_big));
        FSTC_CUDA(cudaFuncSetAttribute(rs_scatter<true, SC_TILE_BIG>, cudaFuncAttributeMaxDynamicSharedMemorySize, s_big));
        FSTC_CUDA(cudaFuncSetAttribute(rs_scatter<false, SC_TILE_SMALL>, cudaFuncAttributeMaxDynamicSharedMemorySize, s_small));
        FSTC_CUDA(cudaFuncSetAttribute(rs_scatter<true, SC_TILE_SMALL>, cudaFuncAttributeMaxDynamicSharedMemorySize, s_small));
    }
    for (int attempt = 0;; ++attempt) {
        rs_bin_caps<<<rs_blocks(nb), 256, 0, c.stream>>>(in.view(), nbins, 16, 192u, cursor.p, cur_stride, attempt, cap.p);
        FSTC_LAUNCH_CHECK();
        exclusive_scan<uint32_t>(c, cap.p, nb, out.start.p);
        int64_t totals[2];
        FSTC_CUDA(cudaMemcpyAsync(&totals[0], tile_first.p + in.n_seg, sizeof(int64_t), cudaMemcpyDeviceToHost, c.stream));
        FSTC_CUDA(cudaMemcpyAsync(&totals[1], out.start.p + nb, sizeof(int64_t), cudaMemcpyDeviceToHost, c.stream));
        c.sync();
        if (totals[1] >= 0xFFFFFFFFll) fail(FSTC_ERR_CAPACITY, "resolve: more than 2^32 records in a pass");
        out.own.alloc(c, totals[1]);
        out.data = out.own.p;
        out.length = totals[1];
        FSTC_CUDA(cudaMemsetAsync(cursor.p, 0, sizeof(uint32_t) * nb * cur_stride, c.stream));
        FSTC_CUDA(cudaMemsetAsync(flag.p, 0, sizeof(unsigned), c.stream));
        if (totals[0] > 0) {
            ScatterArgs a{in.view(), tile_first.p, out.own.p, out.start.p, cursor.p, dest ? dest->p : nullptr, dest ? perm->p : nullptr,
                          cur_stride, shift, hshift, nbins};
            const int h = g_trace.begin(c, dest ? "scatter+dest" : "scatter", totals[0] * SC_TILE, FSTC_T_RS_SCATTER);
            const unsigned grid = static_cast<unsigned>(totals[0]);
            if (dest && big_tile) rs_scatter<true, SC_TILE_BIG><<<grid, SC_THREADS, smem, c.stream>>>(a);
            else if (dest) rs_scatter<true, SC_TILE_SMALL><<<grid, SC_THREADS, smem, c.stream>>>(a);
            else if (big_tile) rs_scatter<false, SC_TILE_BIG><<<grid, SC_THREADS, smem, c.stream>>>(a);
            else rs_scatter<false, SC_TILE_SMALL><<<grid, SC_THREADS, smem, c.stream>>>(a);
            FSTC_LAUNCH_CHECK();
            g_trace.end(c, h);
        }
        rs_check_overflow<<<rs_blocks(nb), 256, 0, c.stream>>>(cursor.p, cur_stride, cap.p, nb, flag.p);
        FSTC_LAUNCH_CHECK();
        c.n_launch += 4;
        if (!read_scalar(c, flag.p)) break;
        if (attempt == 1) fail(FSTC_ERR_INTERNAL, "resolve scatter overflowed with exact capacities");
    }
    out.cnt.alloc(c, nb);
    rs_compact_counts<<<rs_blocks(nb), 256, 0, c.stream>>>(cursor.p, cur_stride, nb, out.cnt.p);
    FSTC_LAUNCH_CHECK();
    c.n_launch += 1;
    return out;
}

template <int MODE, int TILE>
void launch_gather(Ctx &c, unsigned grid, const GatherArgs &a) {
    constexpr int smem = 6 * TILE;
    FSTC_CUDA(cudaFuncSetAttribute(rs_gather_ids<MODE, TILE>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    rs_gather_ids<MODE, TILE><<<grid, GA_THREADS, smem, c.stream>>>(a);
}

// undoes one scatter pass (or, with dest = null, just delivers the ids): see rs_gather_ids
void gather_pass(Ctx &c, const SegSet &seg, int mode, bool big_tile, GatherArgs a) {
    const int SC_TILE = big_tile ? SC_TILE_BIG : SC_TILE_SMALL;
    DBuf<int64_t> tile_first(c, seg.n_seg + 1);
    rs_seg_tiles<<<1, 1024, 0, c.stream>>>(seg.view(), SC_TILE, tile_first.p);
    FSTC_LAUNCH_CHECK();
    const int64_t tiles = read_scalar(c, tile_first.p + seg.n_seg);
    a.seg = seg.view();
    a.tile_first = tile_first.p;
    if (tiles > 0) {
        const int h = g_trace.begin(c, mode == 0 && a.dest ? "gather" : "apply", tiles * SC_TILE, FSTC_T_RS_GATHER);
        const unsigned grid = static_cast<unsigned>(tiles);
        if (big_tile) {
            if (mode == 0) launch_gather<0, SC_TILE_BIG>(c, grid, a);
            else if (mode == 1) launch_gather<1, SC_TILE_BIG>(c, grid, a);
            else launch_gather<2, SC_TILE_BIG>(c, grid, a);
        } else {
            if (mode == 0) launch_gather<0, SC_TILE_SMALL>(c, grid, a);
            else if (mode == 1) launch_gather<1, SC_TILE_SMALL>(c, grid, a);
            else launch_gather<2, SC_TILE_SMALL>(c, grid, a);
        }
        FSTC_LAUNCH_CHECK();
        g_trace.end(c, h);
    }
    c.n_launch += 2;
}

}  // namespace

int resolve_bits_needed(int64_t n_records_and_states) {
    int b = 0;
    while (b < 20 && (n_records_and_states >> b) > DD_TARGET) ++b;
    return b;
}

// the ids of the job's keys are known (ids[r], in rank order): deliver them the way the job asks for (target column,
// indirect positions, or into the sort records)
void resolve_apply_ids(Ctx &c, const ResolveJob &j, const uint32_t *ids) {
    if (j.n_records <= 0) return;
    SegSet lvl0 = single_segment(c, j.keys, j.n_records);
    GatherArgs g{};
    g.dest = nullptr; g.perm = nullptr; g.in = ids;
    g.out = reinterpret_cast<uint32_t *>(j.o_tgt); g.pos = j.pos; g.o_tgt = j.o_tgt; g.sortrec = j.sortrec; g.shift_t = j.shift_t;
    gather_pass(c, lvl0, j.mode, true, g);
    c.sync();
}

bool resolve_can_take(int64_t n_records, int64_t n_states) {
    // a scatter pass holds up to 17/16 n + 192 per bin records, indexed by u32; 2^20 bins of DD_TARGET keys at most
    return n_records < 0xE0000000ll && ((n_records + n_states) >> 20) <= DD_TARGET;
}

namespace { void resolve_partitioned_impl(Ctx &c, const ResolveJob &j); }

void resolve_partitioned(Ctx &c, const ResolveJob &j) {
    try {
        resolve_partitioned_impl(c, j);
    } catch (...) {                                              // a failed call leaves no stage spans behind for the next one
        for (auto &s : g_trace.spans) { cudaEventDestroy(s.a); cudaEventDestroy(s.b); }
        g_trace.spans.clear();
        g_trace.on = g_trace.print;
        throw;
    }
}

namespace {
void resolve_partitioned_impl(Ctx &c, const ResolveJob &j) {
    FSTC_CUDA(cudaFuncSetAttribute(rs_dedupe, cudaFuncAttributeMaxDynamicSharedMemorySize, DD_SMEM));   // per device
    const int ib = bits_for(static_cast<uint64_t>(j.n_states_before > 1 ? j.n_states_before - 1 : 1));
    if (j.key_bits + ib > 64) fail(FSTC_ERR_CAPACITY, "resolve: key (%d bits) + state id (%d bits) exceed 64 bits", j.key_bits, ib);
    if (j.n_records >= 0xFFFFFFFFll) fail(FSTC_ERR_CAPACITY, "resolve: more than 2^32 records");
    int bits = j.force_bits >= 0 ? j.force_bits : resolve_bits_needed(j.n_states_before + j.n_records);
    g_trace.on = g_trace.print || j.profile;
    const int h_all = g_trace.begin(c, "RESOLVE TOTAL", j.n_records);
    for (;; ++bits) {
        if (bits > 20) fail(FSTC_ERR_CAPACITY, "resolve: more than 2^20 bins needed");
        const int b1 = bits < 10 ? bits : 10, b2 = bits - b1;
        // 1-2. records of the existing states and keys of the arcs, partitioned the same way
        DBuf<unsigned long long> st_recs(c, j.n_states_before);
        rs_state_records<<<rs_blocks(j.n_states_before), 256, 0, c.stream>>>(j.pair, j.n_states_before, j.q2_bits, ib, st_recs.p);
        FSTC_LAUNCH_CHECK();
        c.n_launch += 1;
        SegSet st = single_segment(c, st_recs.p, j.n_states_before);
        if (b1 > 0) st = scatter_pass(c, st, ib, 64 - b1, 1 << b1, true, nullptr, nullptr);
        if (b2 > 0) st = scatter_pass(c, st, ib, 64 - b1 - b2, 1 << b2, false, nullptr, nullptr);
        if (bits > 0) st_recs.release();
        const int h_st = g_trace.begin(c, "(states done)", 0); g_trace.end(c, h_st);
        SegSet lvl0 = single_segment(c, j.keys, j.n_records), lvl1, lvl2;
        DBuf<uint32_t> dest1, dest2;
        DBuf<uint16_t> perm1, perm2;
        if (b1 > 0) lvl1 = scatter_pass(c, lvl0, 0, 64 - b1, 1 << b1, true, &dest1, &perm1);
        if (b2 > 0) {
            lvl2 = scatter_pass(c, lvl1, 0, 64 - b1 - b2, 1 << b2, false, &dest2, &perm2);
            lvl1.own.release();                                  // only the segment table of level 1 is needed from here on
        }
        const SegSet &arcs = b2 > 0 ? lvl2 : (b1 > 0 ? lvl1 : lvl0);
        // 3. per-bin dedupe
        const int h_ar = g_trace.begin(c, "(arcs partitioned)", 0); g_trace.end(c, h_ar);
        const int64_t nb = int64_t(1) << bits;
        DBuf<uint32_t> ids_last(c, arcs.length);
        DBuf<unsigned> err(c, 1);
        FSTC_CUDA(cudaMemsetAsync(err.p, 0, sizeof(unsigned), c.stream));
        const unsigned long long n_before = static_cast<unsigned long long>(j.n_states_before);
        FSTC_CUDA(cudaMemcpyAsync(j.n_states, &n_before, sizeof n_before, cudaMemcpyHostToDevice, c.stream));
        DedupeArgs d{st.view(), arcs.view(), ib, ids_last.p, j.q2_bits, j.n_states, j.pair, err.p};
        const int hd = g_trace.begin(c, "dedupe", nb, FSTC_T_RS_DEDUPE);
        rs_dedupe<<<static_cast<unsigned>(nb), DD_THREADS, DD_SMEM, c.stream>>>(d);
        FSTC_LAUNCH_CHECK();
        g_trace.end(c, hd);
        c.n_launch += 1;
        if (read_scalar(c, err.p)) continue;                     // a bin outgrew shared memory: twice the bins, again
        if (j.stats) {
            const int passes = (b1 > 0) + (b2 > 0);
            j.stats->rs_scatter_recs += passes * j.n_states_before;
            j.stats->rs_scatter_dest_recs += passes * j.n_records;
            j.stats->rs_scatter_launches += 2 * passes;
            j.stats->rs_dedupe_arcs += j.n_records;
            j.stats->rs_dedupe_states += j.n_states_before;
            j.stats->rs_dedupe_launches += 1;
            j.stats->rs_gather_recs += (passes > 0 ? passes : 1) * j.n_records;
            j.stats->rs_gather_launches += passes > 0 ? passes : 1;
        }
        st = SegSet();
        // 4. ids back through the passes
        const uint32_t *ids = ids_last.p;
        DBuf<uint32_t> ids_mid;
        if (b2 > 0) {
            lvl2 = SegSet();
            ids_mid.alloc(c, lvl1.length);
            GatherArgs g{};
            g.dest = dest2.p; g.perm = perm2.p; g.in = ids_last.p; g.out = ids_mid.p;
            gather_pass(c, lvl1, 0, false, g);
            ids = ids_mid.p;
        }
        GatherArgs g{};
        g.dest = b1 > 0 ? dest1.p : nullptr; g.perm = perm1.p; g.in = ids;
        g.out = reinterpret_cast<uint32_t *>(j.o_tgt); g.pos = j.pos; g.o_tgt = j.o_tgt; g.sortrec = j.sortrec; g.shift_t = j.shift_t;
        gather_pass(c, lvl0, j.mode, true, g);
        g_trace.end(c, h_all);
        c.sync();                                                // temporaries are released below
        if (g_trace.on) g_trace.report(j.stats ? j.stats->ms : nullptr);
        g_trace.on = g_trace.print;
        return;
    }
}
}  // namespace

}  // namespace fstc
