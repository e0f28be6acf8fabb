// Device-resident composition of SMALL problems, one thread block per problem.
//
// The paper's own use case is many small translation lattices against one language model and it
// notes that small inputs are dominated by launch, synchronisation and copy overhead.  The level
// loop of compose.cu costs ~150 us of host round trips per BFS level whatever the level's size: 51 levels of `nlp`
// (749 arcs) took 7.6 ms.  Here the WHOLE search of one problem runs inside one block — count, scan, budget cut, match
// list, rank-parallel emit with find-or-insert in a per-problem hash table, merge, placement, next frontier, accept
// list — with block barriers between the steps and no host involvement; a batch of problems is one launch, one block
// each, all sharing the packed right operand.  The steps are those of compose.cu (same work-list, same rank -> match ->
// (i,j) emission, same N10 merge test), restated for a block:
//   * a WARP intersects the two symbol lists of a pair (q2's list staged in shared memory, lanes binary-search it):
//     latency per pair matters here, not throughput;
//   * the merge needs no sort: inside a source that can hold duplicates (N10) an arc is a HEAD if no earlier arc of the
//     source has its (tgt, a, b); a head sums the weights of the later equal arcs in rank order, and the heads are
//     compacted in rank order (sources stay ascending).  O(n^2) per source, in parallel over its arcs, n <= SP_CAP_PAIR.
// A problem that outgrows a capacity (frontier, level, states, arcs) stops with status TOO_BIG and is composed again by
// the level-synchronous path of compose.cu.  FSTC_MERGE_SORT_ALL always takes that path.
#include <cstddef>
#include <algorithm>
#include <cstring>
#include <mutex>
#include <vector>

#include "internal.h"

// Scratch of fstc_compose_static (the end of this file): one array per device that loads the library, held until the
// process exits, shared by every call on that device.  In HOST code this name is only a stand-in for the symbol, not
// a device address: the host reaches the array through cudaGetSymbolAddress (static_scratch below) and nowhere else.
static __device__ __align__(256) unsigned char g_fstc_static_scratch[FSTC_STATIC_SCRATCH_BYTES];

namespace fstc {

namespace {

constexpr int SP_THREADS = 512;       // the widest block (the narrower ones: k_small_compose<T>)
constexpr int SP_CAP_F = 4096;        // frontier pairs of a level
constexpr int SP_CAP_M = 32768;       // matches of a level
constexpr int SP_CAP_L = 65536;       // raw arcs of a level
constexpr int SP_CAP_PAIR = 8192;     // raw arcs of one duplicate-prone source (the merge is quadratic in it)
constexpr int SP_STAGE = 128;         // entries of q2's symbol list a warp stages at a time
constexpr unsigned long long SP_EMPTY = ~0ull;

enum { SP_OK = 0, SP_TOO_BIG = 1 };

struct SmallOut {                     // what a block reports (device -> host, one copy per batch)
    int64_t n_states, n_arcs, n_raw, n_accept, n_expanded, n_seg_visited, n_match_arcs, n_matches;
    int32_t n_levels, truncated, status, pad;
    int64_t level_frontier[FSTC_MAX_LEVEL_STATS], level_raw[FSTC_MAX_LEVEL_STATS], level_new[FSTC_MAX_LEVEL_STATS];
};

struct SmallProb {                    // one problem of the batch: device pointers into the batch's blocks
    MachineView A;
    const uint32_t *acc1;
    int32_t start1, n_states1;
    uint8_t any1;
    int32_t cap_s, cap_a;             // states / arcs this problem may create
    uint32_t cap_t;                   // table slots (power of two)
    // result
    int2 *pair; int32_t *src, *il, *ol, *tgt; float *w; int32_t *accept; uint8_t *expanded;
    // scratch
    ulonglong2 *table;                // {key, id}
    unsigned long long *keyv;         // [SP_CAP_F]
    uint32_t *raw, *nm, *roff, *moff; // [SP_CAP_F (+1)]
    uint8_t *cls, *selv;              // [SP_CAP_F]
    uint32_t *cum, *mpl; uint4 *rec;  // [SP_CAP_M (+1)]
    uint32_t *t_a, *t_b, *t_tgt, *t_pl, *t_slot, *hidx;   // [SP_CAP_L (+1)]
    float *t_w, *t_ws;
    SmallOut *out;
};

struct SmallArgs {
    const SmallProb *prob;
    MachineView B;
    const uint32_t *acc2;
    int32_t start2;
    uint8_t any2;
    uint64_t nq2;
    int merge_mode, max_levels;
    int64_t max_raw_arcs;
};

__device__ __forceinline__ uint64_t sp_mix64(uint64_t k) {
    k ^= k >> 33; k *= 0xff51afd7ed558ccdULL;
    k ^= k >> 33; k *= 0xc4ceb9fe1a85ec53ULL;
    k ^= k >> 33;
    return k;
}

// Intersection of the sorted inner-symbol lists of q1 and q2 by one WARP: q2's list is staged in shared memory (coalesced,
// SP_STAGE entries at a time), the lanes take 32 consecutive entries of q1's list per round and binary-search the staged
// chunk.  on_round(found, first arc of q1's segment, n1, first arc of q2's segment, n2) is called by all lanes in lockstep,
// rounds in symbol order, matches of a round in lane (= symbol) order.
template <typename F>
__device__ __forceinline__ void warp_intersect(const MachineView &A, const MachineView &B, int q1, int q2, uint2 *sB, F &&on_round) {
    const int lane = threadIdx.x & 31;
    uint32_t ka = A.seg_ptr[q1], cb = B.seg_ptr[q2];
    const uint32_t e1 = A.seg_ptr[q1 + 1], e2 = B.seg_ptr[q2 + 1];
    if (ka == e1 || cb == e2) return;
    bool need_load = true;
    int nB = 0;
    while (true) {
        if (need_load) {
            nB = static_cast<int>(e2 - cb < SP_STAGE ? e2 - cb : SP_STAGE);
            __syncwarp();
            for (int j = lane; j <= nB; j += 32) sB[j] = B.segs[cb + j];     // one entry more: the end of the last segment
            need_load = false;
            __syncwarp();
        }
        bool found = false;
        uint32_t o1 = 0, n1 = 0, o2 = 0, n2 = 0, sym = 0;
        const uint32_t e = ka + lane;
        if (e < e1) {
            const uint2 a = A.segs[e], an = A.segs[e + 1];
            sym = a.x;
            int lo = 0, hi = nB;                                              // first staged entry with symbol >= sym
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (sB[mid].x < sym) lo = mid + 1; else hi = mid;
            }
            if (lo < nB) {
                const uint2 b = sB[lo];
                if (b.x == sym) { found = true; o1 = a.y; n1 = an.y - a.y; o2 = b.y; n2 = sB[lo + 1].y - b.y; }
            }
        }
        on_round(found, o1, n1, o2, n2);
        const int nv = static_cast<int>(e1 - ka < 32 ? e1 - ka : 32);
        const uint32_t ahi = __shfl_sync(0xffffffffu, sym, nv - 1);           // largest symbol of the round
        const uint32_t bhi = sB[nB - 1].x;
        if (cb + nB < e2) {
            if (ahi > bhi) { cb += nB; need_load = true; }                    // same round against the next chunk of q2's list
            else { ka += 32; if (ka >= e1) break; }
        } else {
            ka += 32;
            if (ka >= e1 || ahi >= bhi) break;                                // q2's list is exhausted: nothing above bhi matches
        }
    }
}

// out[i] = sum of in[j], j < i (i = 0..n; out[n] = total), n <= 65536, by the whole block; returns the total.  in == out is fine.
template <int T>
__device__ uint32_t block_scan(const uint32_t *in, uint32_t *out, int n, uint32_t *s_w /* [(T / 32) + 1] */) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint32_t carry = 0;
    for (int base = 0; base < n; base += T) {
        const int i = base + tid;
        const uint32_t v = i < n ? in[i] : 0u;
        uint32_t incl = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += t;
        }
        if (lane == 31) s_w[warp] = incl;
        __syncthreads();
        uint32_t before = 0, total = 0;
#pragma unroll
        for (int w = 0; w < (T / 32); ++w) { const uint32_t c = s_w[w]; if (w < warp) before += c; total += c; }
        if (i < n) out[i] = carry + before + incl - v;
        carry += total;
        __syncthreads();
    }
    if (tid == 0) out[n] = carry;
    __syncthreads();
    return carry;
}

// The search of one problem by one block of T threads (inlined into the kernels below, which only differ in where P comes
// from and in T).
template <int T>
__device__ __forceinline__ void small_compose_block(const SmallArgs &g, const SmallProb &P) {
    __shared__ uint2 s_stage[(T / 32)][SP_STAGE + 1];
    __shared__ uint32_t s_w[(T / 32) + 1];
    __shared__ unsigned int s_nstates, s_flag, s_nsel;
    __shared__ unsigned long long s_cut, s_segs, s_marcs;
    const MachineView &A = P.A, &B = g.B;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint64_t nq2 = g.nq2;
    const bool can_merge = g.merge_mode == FSTC_MERGE_AUTO &&
                           (((P.any1 & FLAG_D) && (g.any2 & FLAG_D)) || (P.any1 & FLAG_X) || (g.any2 & FLAG_X));

    // ---- init (Alg. 2 lines 1-3): empty table, state 0 = (s1, s2)
    for (uint32_t s = tid; s < P.cap_t; s += T) P.table[s] = make_ulonglong2(SP_EMPTY, 0ull);
    if (tid == 0) {
        s_nstates = 1; s_flag = 0; s_segs = 0; s_marcs = 0;
        P.pair[0] = make_int2(P.start1, g.start2);
    }
    __syncthreads();
    if (tid == 0) {
        const unsigned long long k0 = static_cast<uint64_t>(static_cast<uint32_t>(P.start1)) * nq2 + static_cast<uint32_t>(g.start2);
        P.table[sp_mix64(k0) & (P.cap_t - 1)] = make_ulonglong2(k0, 0ull);
    }
    __syncthreads();

    int64_t n_arcs = 0, cum_raw = 0, n_expanded = 0, n_matches = 0;
    int f_lo = 0, f_hi = 1, lvl = 0;
    int last_lo = 0, last_hi = 1, last_mode = 1;      // how the last frontier was treated: 0 not expanded, 1 all, 2 cut
    int truncated = 0, status = SP_OK;
    unsigned long long cut_key = 0;

    for (;; ++lvl) {
        const int nf = f_hi - f_lo;
        if (nf == 0) break;
        last_lo = f_lo; last_hi = f_hi;
        if (g.max_levels > 0 && lvl == g.max_levels) { truncated = 1; last_mode = 0; break; }
        last_mode = 1;
        if (nf > SP_CAP_F) { status = SP_TOO_BIG; break; }

        // ---- count: a warp per pair
        for (int i = warp; i < nf; i += (T / 32)) {
            const int2 p = P.pair[f_lo + i];
            unsigned long long raw = 0;
            uint32_t nm = 0;
            warp_intersect(A, B, p.x, p.y, s_stage[warp], [&](bool found, uint32_t, uint32_t n1, uint32_t, uint32_t n2) {
                if (found) { raw += static_cast<unsigned long long>(n1) * n2; nm += 1; }
            });
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                raw += __shfl_xor_sync(0xffffffffu, raw, d);
                nm += __shfl_xor_sync(0xffffffffu, nm, d);
            }
            if (lane == 0) {
                bool f = false;
                if (can_merge) {
                    const uint8_t fa = A.flags[p.x], fb = B.flags[p.y];
                    f = ((fa & FLAG_D) && (fb & FLAG_D)) || (fa & FLAG_X) || (fb & FLAG_X);
                }
                if (raw > SP_CAP_L || (f && raw > SP_CAP_PAIR)) { atomicOr(&s_flag, 1u); raw = 0; nm = 0; }
                P.raw[i] = static_cast<uint32_t>(raw);
                P.nm[i] = nm;
                P.cls[i] = f;
                P.keyv[i] = static_cast<uint64_t>(static_cast<uint32_t>(p.x)) * nq2 + static_cast<uint32_t>(p.y);
            }
        }
        __syncthreads();
        if (s_flag) { status = SP_TOO_BIG; break; }

        // ---- scan + budget (rule T)
        unsigned long long R64 = 0;
        for (int i = tid; i < nf; i += T) R64 += P.raw[i];
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) R64 += __shfl_xor_sync(0xffffffffu, R64, d);
        if (tid == 0) s_cut = 0;
        __syncthreads();
        if (lane == 0) atomicAdd(&s_cut, R64);
        __syncthreads();
        R64 = s_cut;
        __syncthreads();
        bool stop_after = false;
        int n_sel = nf;
        if (g.max_raw_arcs > 0 && cum_raw + static_cast<int64_t>(R64) > g.max_raw_arcs) {
            // the pairs in ascending key order: pair i is expanded iff the raw arcs of all pairs up to and including it fit
            const unsigned long long remaining = static_cast<unsigned long long>(g.max_raw_arcs - cum_raw);
            if (tid == 0) { s_cut = ~0ull; s_nsel = 0; }
            __syncthreads();
            for (int i = tid; i < nf; i += T) {
                const unsigned long long ki = P.keyv[i];
                unsigned long long pre = 0;
                for (int j = 0; j < nf; ++j) if (P.keyv[j] <= ki) pre += P.raw[j];
                const bool sel = pre <= remaining;
                P.selv[i] = sel;
                if (sel) atomicAdd(&s_nsel, 1u); else atomicMin(&s_cut, ki);
            }
            __syncthreads();
            for (int i = tid; i < nf; i += T) if (!P.selv[i]) { P.raw[i] = 0; P.nm[i] = 0; }
            cut_key = s_cut;
            n_sel = static_cast<int>(s_nsel);
            truncated = 1; stop_after = true; last_mode = 2;
            __syncthreads();
        } else if (R64 > SP_CAP_L) { status = SP_TOO_BIG; break; }
        const uint32_t R = block_scan<T>(P.raw, P.roff, nf, s_w);
        const uint32_t M = block_scan<T>(P.nm, P.moff, nf, s_w);
        if (M > SP_CAP_M || R > SP_CAP_L || n_arcs + R > P.cap_a) { status = SP_TOO_BIG; break; }

        // ---- match work-list: second walk, records in (pair, symbol) order with the running arc rank
        for (int i = warp; i < nf; i += (T / 32)) {
            if (P.nm[i] == 0) continue;
            const int2 p = P.pair[f_lo + i];
            uint32_t m = P.moff[i], run = P.roff[i];
            unsigned long long marcs = 0;
            warp_intersect(A, B, p.x, p.y, s_stage[warp], [&](bool found, uint32_t o1, uint32_t n1, uint32_t o2, uint32_t n2) {
                const uint32_t fb = __ballot_sync(0xffffffffu, found);
                const uint32_t c = found ? n1 * n2 : 0u;
                uint32_t incl = c;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
                    if (lane >= d) incl += t;
                }
                if (found) {
                    const uint32_t slot = m + __popc(fb & ((1u << lane) - 1u));
                    P.cum[slot] = run + incl - c;
                    P.rec[slot] = make_uint4(o1, o2, n1, n2);
                    P.mpl[slot] = static_cast<uint32_t>(i);
                    marcs += n1 + n2;
                }
                m += __popc(fb);
                run += __shfl_sync(0xffffffffu, incl, 31);
            });
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) marcs += __shfl_xor_sync(0xffffffffu, marcs, d);
            if (lane == 0) {
                atomicAdd(&s_marcs, marcs);
                atomicAdd(&s_segs, static_cast<unsigned long long>((A.seg_ptr[p.x + 1] - A.seg_ptr[p.x]) + (B.seg_ptr[p.y + 1] - B.seg_ptr[p.y])));
            }
        }
        if (tid == 0) P.cum[M] = R;
        __syncthreads();

        // ---- emit: a thread per output rank (rank -> match -> (i,j)), find-or-insert of the target pair
        const uint32_t ns_before = s_nstates;
        for (uint32_t r = tid; r < R; r += T) {
            if (*reinterpret_cast<volatile unsigned int *>(&s_flag)) break;   // out of state ids: no more inserts (the table keeps free slots)
            uint32_t lo = 0, hi = M;                                          // last match whose first rank <= r
            while (hi - lo > 1) {
                const uint32_t mid = (lo + hi) >> 1;
                if (P.cum[mid] <= r) lo = mid; else hi = mid;
            }
            const uint4 rec = P.rec[lo];
            const uint32_t rr = r - P.cum[lo];
            const uint32_t i1 = rr / rec.w, i2 = rr - i1 * rec.w;
            const uint4 e1 = __ldg(A.arcs + rec.x + i1), e2 = __ldg(B.arcs + rec.y + i2);   // {tgt, outer, weight, inner}
            const unsigned long long key = static_cast<uint64_t>(e1.x) * nq2 + e2.x;
            uint32_t s = static_cast<uint32_t>(sp_mix64(key)) & (P.cap_t - 1);
            while (true) {
                unsigned long long *kp = reinterpret_cast<unsigned long long *>(P.table + s);
                unsigned long long k = *reinterpret_cast<volatile unsigned long long *>(kp);
                if (k == SP_EMPTY) k = atomicCAS(kp, SP_EMPTY, key);
                if (k == SP_EMPTY) {                                          // this thread created the state
                    const uint32_t id = atomicAdd(&s_nstates, 1u);
                    if (id < static_cast<uint32_t>(P.cap_s)) {
                        P.pair[id] = make_int2(static_cast<int>(e1.x), static_cast<int>(e2.x));
                        kp[1] = id;
                    } else atomicOr(&s_flag, 1u);
                    break;
                }
                if (k == key) break;
                s = (s + 1) & (P.cap_t - 1);
            }
            P.t_slot[r] = s;
            P.t_a[r] = e1.y; P.t_b[r] = e2.y; P.t_pl[r] = P.mpl[lo];
            P.t_w[r] = __uint_as_float(e1.z) * __uint_as_float(e2.z);
        }
        __syncthreads();
        if (s_flag) { status = SP_TOO_BIG; break; }
        for (uint32_t r = tid; r < R; r += T) P.t_tgt[r] = static_cast<uint32_t>(P.table[P.t_slot[r]].y);   // ids are all published now
        __syncthreads();

        // ---- merge: heads of equal (tgt, a, b) inside a source that can hold duplicates
        for (uint32_t r = tid; r < R; r += T) {
            const uint32_t i = P.t_pl[r];
            uint32_t head = 1;
            float w = P.t_w[r], comp = 0.f;                            // compensated (Kahan) sum: a few ulp whatever the run length
            if (P.cls[i]) {
                const uint32_t lo = P.roff[i], hi = lo + P.raw[i];
                const uint32_t t = P.t_tgt[r], a = P.t_a[r], b = P.t_b[r];
                for (uint32_t q = lo; q < r; ++q)
                    if (P.t_tgt[q] == t && P.t_a[q] == a && P.t_b[q] == b) { head = 0; break; }
                if (head)
                    for (uint32_t q = r + 1; q < hi; ++q)
                        if (P.t_tgt[q] == t && P.t_a[q] == a && P.t_b[q] == b) {
                            const float y = P.t_w[q] - comp, s2 = w + y;
                            comp = (s2 - w) - y;
                            w = s2;
                        }
            }
            P.hidx[r] = head;
            P.t_ws[r] = w;
        }
        __syncthreads();
        for (uint32_t r = tid; r < R; r += T) P.t_slot[r] = P.hidx[r];      // keep the flags: the scan overwrites them
        __syncthreads();
        const uint32_t Mg = block_scan<T>(P.hidx, P.hidx, static_cast<int>(R), s_w);
        for (uint32_t r = tid; r < R; r += T) {
            if (!P.t_slot[r]) continue;
            const int64_t q = n_arcs + P.hidx[r];
            P.src[q] = f_lo + static_cast<int>(P.t_pl[r]);
            P.il[q] = static_cast<int>(P.t_a[r]); P.ol[q] = static_cast<int>(P.t_b[r]);
            P.tgt[q] = static_cast<int>(P.t_tgt[r]); P.w[q] = P.t_ws[r];
        }
        __syncthreads();

        const int ns_after = static_cast<int>(s_nstates);
        if (tid == 0 && lvl < FSTC_MAX_LEVEL_STATS) {
            P.out->level_frontier[lvl] = nf; P.out->level_raw[lvl] = R; P.out->level_new[lvl] = ns_after - static_cast<int>(ns_before);
        }
        n_arcs += Mg; cum_raw += R; n_expanded += n_sel; n_matches += M;
        f_lo = f_hi; f_hi = ns_after;
        if (stop_after) { ++lvl; break; }
    }
    __syncthreads();

    // ---- assemble: expanded flags, accept list (ascending ids with q1 in F1 and q2 in F2)
    const int n_states = static_cast<int>(s_nstates);
    uint32_t n_accept = 0;
    if (status == SP_OK) {
        for (int base = 0; base < n_states; base += T) {
            const int i = base + tid;
            uint32_t acc = 0;
            if (i < n_states) {
                const int2 p = P.pair[i];
                acc = ((P.acc1[p.x >> 5] >> (p.x & 31)) & 1u) & ((g.acc2[p.y >> 5] >> (p.y & 31)) & 1u);
                uint8_t e = 1;
                if (i >= last_hi) e = 0;
                else if (i >= last_lo) {
                    if (last_mode == 0) e = 0;
                    else if (last_mode == 2) e = (static_cast<uint64_t>(static_cast<uint32_t>(p.x)) * nq2 + static_cast<uint32_t>(p.y)) < cut_key;
                }
                P.expanded[i] = e;
            }
            const uint32_t bal = __ballot_sync(0xffffffffu, acc);
            if (lane == 0) s_w[warp] = __popc(bal);
            __syncthreads();
            uint32_t before = 0, total = 0;
#pragma unroll
            for (int w = 0; w < (T / 32); ++w) { const uint32_t c = s_w[w]; if (w < warp) before += c; total += c; }
            if (acc) P.accept[n_accept + before + __popc(bal & ((1u << lane) - 1u))] = i;
            n_accept += total;
            __syncthreads();
        }
    }
    if (tid == 0) {
        SmallOut *o = P.out;
        o->n_states = n_states; o->n_arcs = n_arcs; o->n_raw = cum_raw; o->n_accept = n_accept; o->n_expanded = n_expanded;
        o->n_seg_visited = static_cast<int64_t>(s_segs); o->n_match_arcs = static_cast<int64_t>(s_marcs); o->n_matches = n_matches;
        o->n_levels = lvl; o->truncated = truncated; o->status = status;
    }
}

// a batch: block k takes problem k, whose descriptor (result and scratch pointers from the library pool) is in device memory
// T = 512 for a few problems (latency: every step of a level spreads over 16 warps); big batches take narrower blocks, 256 or
// 128 threads, so that 2 or 4 problems are resident per SM (108 registers per thread: a block of 512 fills an SM's file)
template <int T>
__global__ void __launch_bounds__(T) k_small_compose(SmallArgs g) {
    const SmallProb P = g.prob[blockIdx.x];
    small_compose_block<T>(g, P);
}

// one problem, its descriptor passed by value: the result arrays are the caller's, the scratch is g_small_scratch (below)
__global__ void __launch_bounds__(SP_THREADS) k_small_compose_static(SmallArgs g, SmallProb P) {
    small_compose_block<SP_THREADS>(g, P);
}

struct Carver {                       // consecutive 256-byte aligned pieces of one block
    char *base;
    size_t off = 0;
    explicit Carver(void *b) : base(static_cast<char *>(b)) {}
    template <typename T> T *take(size_t n) {
        T *p = reinterpret_cast<T *>(base + off);
        off += (n * sizeof(T) + 255) & ~size_t(255);
        return p;
    }
};
std::mutex g_shared_mu;

}  // namespace

void free_result(fstc_result_t *r) {
    if (!r) return;
    ResultImpl *impl = static_cast<ResultImpl *>(r->impl);
    if (impl) {
        if (impl->shared) {                                    // a result of a batch: the block goes when its last result goes
            bool last;
            { std::lock_guard<std::mutex> lk(g_shared_mu); last = --impl->shared->refs == 0; }
            if (last) { release_block(impl->shared->base, impl->shared->hooks); delete impl->shared; }
        } else {
            for (void *p : impl->bufs) release_block(p, impl->hooks);
        }
        delete impl;
    }
    delete r;
}

bool small_path_applies(const fstc_opts_t &o) {
    return o.small_path != FSTC_SMALL_OFF && o.merge_mode != FSTC_MERGE_SORT_ALL && !o.spill && !o.deterministic && o.resolve_mode != FSTC_RESOLVE_EXTERNAL &&
           o.state_capacity_hint <= (1 << 20) && o.arc_capacity_hint <= (1 << 22);
}

// Composes m1[k] with m2 for k = 0..n-1, one block each.  results[k] is set for the problems that fitted (ok[k] = 1); the
// others (ok[k] = 0) are left to the caller.  stats (nullable) is [n].
void compose_small_batch(Ctx &c, const fstc_packed_t *const *m1, int n, const fstc_packed_t &m2, const fstc_opts_t &o,
                         fstc_result_t **results, fstc_stats_t *stats, std::vector<char> &ok) {
    ok.assign(n, 0);
    if (n <= 0) return;
    if (m2.side != 2) fail(FSTC_ERR_ARG, "operands must be packed with side 1 (left) and side 2 (right)");
    for (int k = 0; k < n; ++k) {
        if (!m1[k] || m1[k]->side != 1) fail(FSTC_ERR_ARG, "operands must be packed with side 1 (left) and side 2 (right)");
        if (m1[k]->n_inner != m2.n_inner)
            fail(FSTC_ERR_ARG, "inner alphabets differ: |Γ| = %d vs %d (PAPER.md:45)", m1[k]->n_inner, m2.n_inner);
        if (m1[k]->device != m2.device) fail(FSTC_ERR_ARG, "operands were packed on different devices");
    }
    if (o.merge_mode < 0 || o.merge_mode > 2 || o.max_levels < 0 || o.max_raw_arcs < 0) fail(FSTC_ERR_ARG, "bad options");
    const int64_t cap_s = std::max<int64_t>(o.state_capacity_hint > 0 ? o.state_capacity_hint + 1 : 8192, 64);
    const int64_t cap_a = std::max<int64_t>(o.arc_capacity_hint > 0 ? o.arc_capacity_hint + 1 : 65536, 64);
    uint32_t cap_t = 1024;
    while (cap_t < 2 * cap_s + 2 * SP_THREADS) cap_t <<= 1;
    auto persist_bytes = [&](Carver &cv, SmallProb &p) {
        p.pair = cv.take<int2>(cap_s); p.src = cv.take<int32_t>(cap_a); p.il = cv.take<int32_t>(cap_a); p.ol = cv.take<int32_t>(cap_a);
        p.tgt = cv.take<int32_t>(cap_a); p.w = cv.take<float>(cap_a); p.accept = cv.take<int32_t>(cap_s); p.expanded = cv.take<uint8_t>(cap_s);
    };
    auto scratch_bytes = [&](Carver &cv, SmallProb &p) {
        p.table = cv.take<ulonglong2>(cap_t); p.keyv = cv.take<unsigned long long>(SP_CAP_F);
        p.raw = cv.take<uint32_t>(SP_CAP_F + 1); p.nm = cv.take<uint32_t>(SP_CAP_F + 1);
        p.roff = cv.take<uint32_t>(SP_CAP_F + 1); p.moff = cv.take<uint32_t>(SP_CAP_F + 1);
        p.cls = cv.take<uint8_t>(SP_CAP_F); p.selv = cv.take<uint8_t>(SP_CAP_F);
        p.cum = cv.take<uint32_t>(SP_CAP_M + 1); p.mpl = cv.take<uint32_t>(SP_CAP_M + 1); p.rec = cv.take<uint4>(SP_CAP_M);
        p.t_a = cv.take<uint32_t>(SP_CAP_L + 1); p.t_b = cv.take<uint32_t>(SP_CAP_L + 1); p.t_tgt = cv.take<uint32_t>(SP_CAP_L + 1);
        p.t_pl = cv.take<uint32_t>(SP_CAP_L + 1); p.t_slot = cv.take<uint32_t>(SP_CAP_L + 1); p.hidx = cv.take<uint32_t>(SP_CAP_L + 1);
        p.t_w = cv.take<float>(SP_CAP_L + 1); p.t_ws = cv.take<float>(SP_CAP_L + 1);
    };
    size_t per_persist, per_scratch;
    { Carver cv(nullptr); SmallProb d; persist_bytes(cv, d); per_persist = cv.off; }
    { Carver cv(nullptr); SmallProb d; scratch_bytes(cv, d); per_scratch = cv.off; }

    cudaEvent_t ev0, ev1;
    FSTC_CUDA(cudaEventCreate(&ev0));
    FSTC_CUDA(cudaEventCreate(&ev1));
    struct EvGuard { cudaEvent_t a, b; ~EvGuard() { cudaEventDestroy(a); cudaEventDestroy(b); } } evg{ev0, ev1};
    FSTC_CUDA(cudaEventRecord(ev0, c.stream));
    DBuf<uint8_t> block(c, static_cast<int64_t>(per_persist) * n, true);
    DBuf<uint8_t> scratch(c, static_cast<int64_t>(per_scratch) * n);
    DBuf<SmallOut> outs(c, n);
    DBuf<SmallProb> d_prob(c, n);
    std::vector<SmallProb> prob(n);
    for (int k = 0; k < n; ++k) {
        SmallProb &p = prob[k];
        p.A = view_of(*m1[k]); p.acc1 = m1[k]->accept_bits; p.start1 = m1[k]->start; p.n_states1 = m1[k]->n_states;
        p.any1 = m1[k]->any_flags;
        p.cap_s = static_cast<int32_t>(cap_s); p.cap_a = static_cast<int32_t>(cap_a); p.cap_t = cap_t;
        Carver cp(block.p + per_persist * k), cs(scratch.p + per_scratch * k);
        persist_bytes(cp, p);
        scratch_bytes(cs, p);
        p.out = outs.p + k;
    }
    FSTC_CUDA(cudaMemcpyAsync(d_prob.p, prob.data(), sizeof(SmallProb) * n, cudaMemcpyHostToDevice, c.stream));
    SmallArgs g;
    g.prob = d_prob.p; g.B = view_of(m2); g.acc2 = m2.accept_bits; g.start2 = m2.start; g.any2 = m2.any_flags;
    g.nq2 = static_cast<uint64_t>(m2.n_states); g.merge_mode = o.merge_mode; g.max_levels = o.max_levels; g.max_raw_arcs = o.max_raw_arcs;
    if (n >= 4 * c.n_sm) k_small_compose<128><<<static_cast<unsigned>(n), 128, 0, c.stream>>>(g);
    else if (n >= 2 * c.n_sm) k_small_compose<256><<<static_cast<unsigned>(n), 256, 0, c.stream>>>(g);
    else k_small_compose<SP_THREADS><<<static_cast<unsigned>(n), SP_THREADS, 0, c.stream>>>(g);
    FSTC_LAUNCH_CHECK();
    c.n_launch += 1;
    std::vector<SmallOut> h(n);
    FSTC_CUDA(cudaMemcpyAsync(h.data(), outs.p, sizeof(SmallOut) * n, cudaMemcpyDeviceToHost, c.stream));
    FSTC_CUDA(cudaEventRecord(ev1, c.stream));
    c.sync();
    float ms = 0.f;
    cudaEventElapsedTime(&ms, ev0, ev1);

    SharedBlock *shared = nullptr;
    for (int k = 0; k < n; ++k) {
        const SmallOut &so = h[k];
        if (so.status != SP_OK) continue;
        if (!shared) shared = new SharedBlock{block.take(), 0, c.hooks};
        const SmallProb &p = prob[k];
        fstc_result_t *r = new fstc_result_t();
        ResultImpl *impl = new ResultImpl();
        impl->shared = shared;
        shared->refs += 1;
        r->n_states = so.n_states; r->n_arcs = so.n_arcs; r->n_raw_arcs = so.n_raw; r->n_accept = so.n_accept;
        r->n_expanded = so.n_expanded; r->n_levels = so.n_levels; r->truncated = so.truncated;
        r->pair = reinterpret_cast<int32_t *>(p.pair); r->src = p.src; r->ilabel = p.il; r->olabel = p.ol; r->tgt = p.tgt;
        r->weight = p.w; r->accept = p.accept; r->expanded = p.expanded;
        r->impl = impl;
        results[k] = r;
        ok[k] = 1;
        if (stats) {
            fstc_stats_t &st = stats[k];
            std::memset(&st, 0, sizeof st);
            st.n_states = so.n_states; st.n_arcs = so.n_arcs; st.n_raw_arcs = so.n_raw; st.n_expanded = so.n_expanded;
            st.n_levels = so.n_levels; st.truncated = so.truncated;
            st.n_seg_visited = so.n_seg_visited; st.n_matches = so.n_matches; st.n_match_arcs = so.n_match_arcs;
            st.table_capacity = cap_t; st.n_kernel_launches = 1; st.small_path = 1; st.ms_total = ms;
            const int nl = std::min<int>(so.n_levels, FSTC_MAX_LEVEL_STATS);
            for (int l = 0; l < nl; ++l) {
                st.level_frontier[l] = so.level_frontier[l]; st.level_raw[l] = so.level_raw[l]; st.level_new_states[l] = so.level_new[l];
            }
        }
    }
}

// ------------------------------------------------------------------------------------------ fstc_compose_static
// The same search for ONE problem with no allocation at all (include/fstc.h): result arrays from the caller, scratch in
// g_fstc_static_scratch.  Host code never uses that name as a pointer: the device address comes from
// cudaGetSymbolAddress, asked once per device with that device current, and is what the kernel's descriptor is built on.
namespace {

static_assert(sizeof(fstc_static_header_t) == 80 && offsetof(SmallOut, level_frontier) == 80, "the header is SmallOut's first 80 bytes");
static_assert(offsetof(fstc_static_header_t, n_raw_arcs) == offsetof(SmallOut, n_raw) &&
              offsetof(fstc_static_header_t, n_matches) == offsetof(SmallOut, n_matches) &&
              offsetof(fstc_static_header_t, n_levels) == offsetof(SmallOut, n_levels) &&
              offsetof(fstc_static_header_t, status) == offsetof(SmallOut, status), "header layout");

constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mu;
unsigned char *g_static_ptr[STATIC_MAX_DEVICES] = {};       // device address of g_fstc_static_scratch, per device

unsigned char *static_scratch(int dev) {
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) fail(FSTC_ERR_ARG, "device index %d not supported", dev);
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_ptr[dev]) {
        void *p = nullptr;
        FSTC_CUDA(cudaGetSymbolAddress(&p, g_fstc_static_scratch));     // the current device's copy of the array
        if (!p) fail(FSTC_ERR_CUDA, "cudaGetSymbolAddress gave no address for the static scratch array");
        g_static_ptr[dev] = static_cast<unsigned char *>(p);
    }
    return g_static_ptr[dev];
}

uint32_t small_table_slots(int64_t cap_s) {                  // as compose_small_batch: never more than half full
    uint32_t cap_t = 1024;
    while (cap_t < 2 * cap_s + 2 * SP_THREADS) cap_t <<= 1;
    return cap_t;
}

// the scratch arrays of one problem, in compose_small_batch's order, behind the block's report
void carve_static_scratch(Carver &cv, SmallProb &p, uint32_t cap_t) {
    p.out = cv.take<SmallOut>(1);
    p.table = cv.take<ulonglong2>(cap_t); p.keyv = cv.take<unsigned long long>(SP_CAP_F);
    p.raw = cv.take<uint32_t>(SP_CAP_F + 1); p.nm = cv.take<uint32_t>(SP_CAP_F + 1);
    p.roff = cv.take<uint32_t>(SP_CAP_F + 1); p.moff = cv.take<uint32_t>(SP_CAP_F + 1);
    p.cls = cv.take<uint8_t>(SP_CAP_F); p.selv = cv.take<uint8_t>(SP_CAP_F);
    p.cum = cv.take<uint32_t>(SP_CAP_M + 1); p.mpl = cv.take<uint32_t>(SP_CAP_M + 1); p.rec = cv.take<uint4>(SP_CAP_M);
    p.t_a = cv.take<uint32_t>(SP_CAP_L + 1); p.t_b = cv.take<uint32_t>(SP_CAP_L + 1); p.t_tgt = cv.take<uint32_t>(SP_CAP_L + 1);
    p.t_pl = cv.take<uint32_t>(SP_CAP_L + 1); p.t_slot = cv.take<uint32_t>(SP_CAP_L + 1); p.hidx = cv.take<uint32_t>(SP_CAP_L + 1);
    p.t_w = cv.take<float>(SP_CAP_L + 1); p.t_ws = cv.take<float>(SP_CAP_L + 1);
}

}  // namespace

void compose_small_static(Ctx &c, const fstc_packed_t &m1, const fstc_packed_t &m2, const fstc_opts_t &o,
                          const fstc_static_out_t &out) {
    if (m1.side != 1 || m2.side != 2) fail(FSTC_ERR_ARG, "operands must be packed with side 1 (left) and side 2 (right)");
    if (m1.n_inner != m2.n_inner) fail(FSTC_ERR_ARG, "inner alphabets differ: |Γ| = %d vs %d (PAPER.md:45)", m1.n_inner, m2.n_inner);
    if (m1.device != m2.device) fail(FSTC_ERR_ARG, "operands were packed on different devices");
    int dev = 0;
    FSTC_CUDA(cudaGetDevice(&dev));
    if (dev != m2.device) fail(FSTC_ERR_ARG, "the operands live on device %d but device %d is current", m2.device, dev);
    if (o.merge_mode != FSTC_MERGE_AUTO && o.merge_mode != FSTC_MERGE_OFF)
        fail(FSTC_ERR_ARG, "fstc_compose_static merges with FSTC_MERGE_AUTO or not at all (FSTC_MERGE_OFF)");
    if (o.max_levels < 0 || o.max_raw_arcs < 0) fail(FSTC_ERR_ARG, "bad options");
    if (o.spill || o.deterministic || o.resolve_mode == FSTC_RESOLVE_EXTERNAL || o.alloc || o.dealloc)
        fail(FSTC_ERR_ARG, "fstc_compose_static reads merge_mode, max_levels and max_raw_arcs only");
    if (!out.pair || !out.src || !out.ilabel || !out.olabel || !out.tgt || !out.weight || !out.accept || !out.expanded || !out.header)
        fail(FSTC_ERR_ARG, "null output buffer");
    if (reinterpret_cast<uintptr_t>(out.pair) % 8 != 0) fail(FSTC_ERR_ARG, "pair must be 8-byte aligned");
    if (out.state_capacity < 1 || out.arc_capacity < 1) fail(FSTC_ERR_ARG, "capacities must be at least 1");
    if (out.state_capacity > FSTC_STATIC_MAX_STATES)
        fail(FSTC_ERR_CAPACITY, "state_capacity %lld is beyond FSTC_STATIC_MAX_STATES = %d: the visited table would not fit the "
             "static scratch array (%u bytes); use fstc_compose_packed", static_cast<long long>(out.state_capacity),
             FSTC_STATIC_MAX_STATES, static_cast<unsigned>(FSTC_STATIC_SCRATCH_BYTES));
    if (out.arc_capacity > 0x7FFFFFFFll)
        fail(FSTC_ERR_CAPACITY, "arc_capacity %lld is beyond 2^31 - 1", static_cast<long long>(out.arc_capacity));

    SmallProb p;
    p.A = view_of(m1); p.acc1 = m1.accept_bits; p.start1 = m1.start; p.n_states1 = m1.n_states; p.any1 = m1.any_flags;
    p.cap_s = static_cast<int32_t>(out.state_capacity); p.cap_a = static_cast<int32_t>(out.arc_capacity);
    p.cap_t = small_table_slots(out.state_capacity);
    p.pair = reinterpret_cast<int2 *>(out.pair); p.src = out.src; p.il = out.ilabel; p.ol = out.olabel; p.tgt = out.tgt;
    p.w = out.weight; p.accept = out.accept; p.expanded = out.expanded;
    Carver cv(static_scratch(dev));
    carve_static_scratch(cv, p, p.cap_t);
    if (cv.off > FSTC_STATIC_SCRATCH_BYTES)                      // (cannot happen below FSTC_STATIC_MAX_STATES: 7.2 MB there)
        fail(FSTC_ERR_CAPACITY, "the scratch of %lld states (%zu bytes) does not fit the static array (%u bytes)",
             static_cast<long long>(out.state_capacity), cv.off, static_cast<unsigned>(FSTC_STATIC_SCRATCH_BYTES));

    SmallArgs g;
    g.prob = nullptr; g.B = view_of(m2); g.acc2 = m2.accept_bits; g.start2 = m2.start; g.any2 = m2.any_flags;
    g.nq2 = static_cast<uint64_t>(m2.n_states); g.merge_mode = o.merge_mode; g.max_levels = o.max_levels; g.max_raw_arcs = o.max_raw_arcs;
    // the array keeps the last call's contents: the report starts from zero (status, counters, level statistics); the
    // kernel empties the visited table itself, and every work list is written before it is read
    FSTC_CUDA(cudaMemsetAsync(p.out, 0, sizeof(SmallOut), c.stream));
    k_small_compose_static<<<1, SP_THREADS, 0, c.stream>>>(g, p);
    FSTC_LAUNCH_CHECK();
    c.n_launch += 1;
    FSTC_CUDA(cudaMemcpyAsync(out.header, p.out, sizeof(fstc_static_header_t), cudaMemcpyDefault, c.stream));
}

}  // namespace fstc
