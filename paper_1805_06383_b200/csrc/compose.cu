// Weighted FST composition as a level-synchronous search over the product graph
// (§3.2-3.4, Algorithms 1-2; DESIGN.md steps 2-9).  Everything runs on the device; the host
// only reads a few scalars per BFS level.
//
//   count    per frontier pair (q1,q2): intersect the inner-symbol lists, raw = Σ_c n1(c)·n2(c)   (step 3)
//   scan     exclusive scans of the raw counts / match counts, budget rule T                      (step 4)
//   match    work-list of (pair, inner symbol) matches with the running arc rank                  (step 3b)
//   emit     one thread per 4 consecutive output ranks (load-balanced over matches, so a match of
//            10^9 arcs is spread over many blocks): read e1,e2, w = p1·p2, write the arc               (step 5)
//   resolve  the id of every target pair: find-or-insert in the visited table inside the emit kernel (the paper's
//            dense |Q1||Q2| table when it is small, else a hash table on the 64-bit key q1·|Q2|+q2, atomicCAS), or,
//            for a big level that creates about a state per arc, the streaming partitioned resolve of
//            resolve.cu; new ids are the next frontier                                                  (step 6)
//   merge    sources that can hold duplicate (tgt,a,b): merged arcs computed directly from the (a,r1) x (b,r2)
//            groups of the pair (class G), or radix sort + segmented sum (class F)                      (step 7)
//   assemble accept list, expanded flags                                                           (step 8)
//
// What differs from the paper's own kernel design (one launch per inner symbol per popped pair, 32-thread
// blocks, host-side queue, lossy table H, sort + reduce of every flagged source — PAPER.md:219-243) is listed in
// DESIGN.md "differences".
#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <ctime>
#include <mutex>

#include "internal.h"
#include "scan.cuh"

namespace fstc {

namespace {

constexpr unsigned long long EMPTY_KEY = ~0ull;
constexpr uint32_t PENDING_ID = 0xFFFFFFFFu;
constexpr int CT_THREADS = 256;
constexpr int64_t GROUP_MAX_RATIO = 8;     // class G while (groups of q1) x (groups of q2) <= 8 x raw arcs of the pair

__device__ __forceinline__ int64_t ceil_div_dev(int64_t a, int64_t b) { return (a + b - 1) / b; }

// ------------------------------------------------------------------------------------------ hash table
// Open addressing over 32-byte BUCKETS of two 16-byte slots {key lo, key hi, id, unused}: a bucket is exactly
// one DRAM sector, read with a single 256-bit load.  A key lives in the first free slot on its probe path
// (home bucket, then the following buckets); slots are never freed, so a lookup that walks the same path
// finds the key before it meets an empty slot.  Empty = all ones (a cudaMemset of 0xFF clears the table).
struct Bucket { uint4 s0, s1; };

__device__ __forceinline__ uint64_t mix64(uint64_t k) {
    k ^= k >> 33; k *= 0xff51afd7ed558ccdULL;
    k ^= k >> 33; k *= 0xc4ceb9fe1a85ec53ULL;
    k ^= k >> 33;
    return k;
}
// cap = number of slots (even); returns the home BUCKET
__device__ __forceinline__ uint64_t home_bucket(uint64_t key, uint64_t cap) { return __umul64hi(mix64(key), cap >> 1); }

__device__ __forceinline__ Bucket ld_bucket(const uint4 *table, uint64_t bucket) {
    Bucket b;
    asm volatile("ld.global.cg.v8.u32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(b.s0.x), "=r"(b.s0.y), "=r"(b.s0.z), "=r"(b.s0.w), "=r"(b.s1.x), "=r"(b.s1.y), "=r"(b.s1.z), "=r"(b.s1.w)
                 : "l"(table + 2 * bucket));
    return b;
}
__device__ __forceinline__ unsigned long long slot_key(const uint4 &v) {
    return (static_cast<unsigned long long>(v.y) << 32) | v.x;
}

__global__ void tb_insert_ids(const int2 *__restrict__ pair, int64_t n, uint64_t nq2, uint4 *table, uint64_t cap) {
    // rebuild after growth: keys are distinct and their ids known -> claim the first free slot, store the id
    int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int2 p = pair[i];
    unsigned long long key = static_cast<uint64_t>(static_cast<uint32_t>(p.x)) * nq2 + static_cast<uint32_t>(p.y);
    uint64_t s = 2 * home_bucket(key, cap);
    while (true) {
        unsigned long long old = atomicCAS(reinterpret_cast<unsigned long long *>(table + s), EMPTY_KEY, key);
        if (old == EMPTY_KEY) break;
        s = (s + 1 == cap) ? 0 : s + 1;
    }
    reinterpret_cast<uint32_t *>(table + s)[2] = static_cast<uint32_t>(i);
}

__global__ void tb_dense_insert_ids(const int2 *__restrict__ pair, int64_t n, uint64_t nq2, uint32_t *__restrict__ dense) {
    int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int2 p = pair[i];
    dense[static_cast<uint64_t>(static_cast<uint32_t>(p.x)) * nq2 + static_cast<uint32_t>(p.y)] = static_cast<uint32_t>(i) + 1u;
}

// ------------------------------------------------------------------------------------------ find or insert, one key per thread
// The visited-set step of PAPER.md:237-239 for one key per thread of a block (all threads call it, `valid` or not): the
// dense table (entry = id + 1, 0 = not visited) or the open-addressing hash table; the new ids of the block come from one
// atomicAdd, the winner of a key publishes the id and writes pair[id], a thread that met a pending entry waits for it.
// Same protocol as inside k_emit.  s_warp: [THREADS / 32] shared words, s_base: one shared 64-bit word.
template <bool DENSE, int THREADS>
__device__ __forceinline__ uint32_t block_find_or_insert(unsigned long long key, bool valid, int2 tgt_pair, uint32_t *dense, uint4 *table,
                                                         uint64_t cap, unsigned long long *n_states, int2 *pair, uint32_t *s_warp,
                                                         unsigned long long *s_base) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint32_t id = 0;
    bool won = false;
    uint32_t *slotp = nullptr;                                   // where the id is (or will be) published
    if (valid) {
        if (DENSE) {
            slotp = dense + key;
            uint32_t v = __ldcg(slotp);
            if (v == 0u) v = atomicCAS(slotp, 0u, PENDING_ID);
            if (v == 0u) won = true; else id = v == PENDING_ID ? PENDING_ID : v - 1u;
        } else {
            const uint64_t n_buckets = cap >> 1;
            uint64_t b = home_bucket(key, cap);
            while (true) {
                Bucket v = ld_bucket(table, b);
                const unsigned long long k0 = slot_key(v.s0), k1 = slot_key(v.s1);
                int cas = -1;
                if (k0 == key) { id = v.s0.z; slotp = reinterpret_cast<uint32_t *>(table + 2 * b) + 2; break; }
                else if (k0 == EMPTY_KEY) cas = 0;
                else if (k1 == key) { id = v.s1.z; slotp = reinterpret_cast<uint32_t *>(table + 2 * b + 1) + 2; break; }
                else if (k1 == EMPTY_KEY) cas = 1;
                if (cas < 0) { b = (b + 1 == n_buckets) ? 0 : b + 1; continue; }
                const unsigned long long old = atomicCAS(reinterpret_cast<unsigned long long *>(table + 2 * b + cas), EMPTY_KEY, key);
                if (old == EMPTY_KEY || old == key) {
                    slotp = reinterpret_cast<uint32_t *>(table + 2 * b + cas) + 2;
                    if (old == EMPTY_KEY) won = true; else id = PENDING_ID;
                    break;
                }                                                // another key took the slot: look at the bucket again
            }
        }
    }
    const uint32_t bal = __ballot_sync(0xffffffffu, won);
    if (lane == 0) s_warp[warp] = __popc(bal);
    __syncthreads();
    if (tid == 0) {
        uint32_t tot = 0;
#pragma unroll
        for (int wv = 0; wv < THREADS / 32; ++wv) { uint32_t cnt = s_warp[wv]; s_warp[wv] = tot; tot += cnt; }
        *s_base = tot ? atomicAdd(n_states, static_cast<unsigned long long>(tot)) : 0ull;
    }
    __syncthreads();
    if (won) {
        id = static_cast<uint32_t>(*s_base) + s_warp[warp] + __popc(bal & ((1u << lane) - 1u));
        __stcg(slotp, DENSE ? id + 1u : id);
        pair[id] = tgt_pair;
    } else if (valid && id == PENDING_ID) {
        uint32_t v;
        while ((v = __ldcg(slotp)) == PENDING_ID) __nanosleep(20);
        id = DENSE ? v - 1u : v;
    }
    __syncthreads();                                             // s_warp / s_base may be reused by the next call
    return id;
}

// ------------------------------------------------------------------------------------------ count / match
// Intersection of the two states' sorted inner-symbol lists.  F is called for every shared symbol with
// (first arc of q1's segment, n1, first arc of q2's segment, n2).
template <typename F>
__device__ __forceinline__ void intersect(const MachineView &A, const MachineView &B, int q1, int q2, F &&on_match) {
    uint32_t s1 = A.seg_ptr[q1], e1 = A.seg_ptr[q1 + 1];
    uint32_t s2 = B.seg_ptr[q2], e2 = B.seg_ptr[q2 + 1];
    if (s1 == e1 || s2 == e2) return;
    uint2 a = A.segs[s1], an = A.segs[s1 + 1];
    uint2 b = B.segs[s2], bn = B.segs[s2 + 1];
    while (true) {
        if (a.x == b.x) {
            on_match(a.y, an.y - a.y, b.y, bn.y - b.y);
            if (++s1 == e1 || ++s2 == e2) break;
            a = an; an = A.segs[s1 + 1];
            b = bn; bn = B.segs[s2 + 1];
        } else if (a.x < b.x) {
            if (++s1 == e1) break;
            a = an; an = A.segs[s1 + 1];
        } else {
            if (++s2 == e2) break;
            b = bn; bn = B.segs[s2 + 1];
        }
    }
}

// class U = arcs go straight to the output; class F = arcs go through sort + reduce first
#ifndef FSTC_FC_PAIR_CAP
#define FSTC_FC_PAIR_CAP 512
#endif
#ifndef FSTC_FC_THREADS
#define FSTC_FC_THREADS 512
#endif
constexpr int FC_PAIR_CAP = FSTC_FC_PAIR_CAP;      // raw arcs of a pair that is merged on chip (class S, k_fchip)
__global__ void __launch_bounds__(CT_THREADS)
k_count(MachineView A, MachineView B, const int2 *__restrict__ pair, int64_t f_lo, int64_t nf,
        const uint32_t *__restrict__ sel /* null: all pairs of the level */, int merge_mode,
        uint64_t nq2, uint64_t key_limit /* pairs with key >= key_limit are left uncounted (raw = 0) */,
        int64_t *__restrict__ rawU, int64_t *__restrict__ rawF, uint32_t *__restrict__ nmU, uint32_t *__restrict__ nmF,
        int64_t *__restrict__ rawG, int64_t *__restrict__ gwork, uint32_t *__restrict__ nmG,
        int64_t *__restrict__ rawS /* null: no on-chip merge in this run */, uint32_t *__restrict__ nmS) {
    int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i < nf) {
        int2 p = pair[f_lo + (sel ? sel[i] : i)];
        int64_t raw = 0;
        uint32_t nm = 0;
        const uint64_t key = static_cast<uint64_t>(static_cast<uint32_t>(p.x)) * nq2 + static_cast<uint32_t>(p.y);
        if (key < key_limit)
            intersect(A, B, p.x, p.y, [&](uint32_t, uint32_t n1, uint32_t, uint32_t n2) {
                raw += static_cast<int64_t>(n1) * n2;
                nm += 1;
            });
        bool f = false;
        if (merge_mode == FSTC_MERGE_SORT_ALL) f = true;
        else if (merge_mode == FSTC_MERGE_AUTO) {
            uint8_t fa = A.flags[p.x], fb = B.flags[p.y];
            f = ((fa & FLAG_D) && (fb & FLAG_D)) || (fa & FLAG_X) || (fb & FLAG_X);
        }
        // class G (merge by construction): a class-F pair whose (a,r1) x (b,r2) group product is not much larger than its
        // raw arc count composes group by group instead of arc by arc and needs no sort
        bool gcls = false;
        int64_t work = 0;
        if (f && rawG && raw > 0) {
            work = static_cast<int64_t>(A.gptr[p.x + 1] - A.gptr[p.x]) * static_cast<int64_t>(B.gptr[p.y + 1] - B.gptr[p.y]);
            gcls = work <= GROUP_MAX_RATIO * raw;
        }
        // class S: a class-F pair of few raw arcs is merged ON CHIP (k_fchip): only its merged arcs reach HBM
        const bool scls = f && !gcls && rawS && raw > 0 && raw <= FC_PAIR_CAP;
        rawU[i] = f ? 0 : raw; nmU[i] = f ? 0 : nm;
        if (rawF) { rawF[i] = (f && !gcls && !scls) ? raw : 0; nmF[i] = (f && !gcls && !scls) ? nm : 0; }   // null when no pair of this run can be class F
        if (rawS) { rawS[i] = scls ? raw : 0; nmS[i] = scls ? nm : 0; }
        if (rawG) { rawG[i] = gcls ? raw : 0; gwork[i] = gcls ? work : 0; nmG[i] = gcls ? 1u : 0u; }
    }
}

// Budget rule T, radix select: weighted histogram of one 8-bit key digit over the pairs whose higher key bits
// equal `prefix`.  Lanes of a warp that share a digit are summed with match-any + reduce-add (three 22-bit limbs,
// so 32 lanes cannot overflow 32 bits) and issue ONE shared-memory atomic: the top digits, which are nearly
// constant over the frontier, no longer serialise.
__global__ void __launch_bounds__(CT_THREADS)
k_cut_hist(const int2 *__restrict__ pair, int64_t f_lo, int64_t nf, const uint32_t *__restrict__ sel, uint64_t nq2,
           const int64_t *__restrict__ rawU,
           const int64_t *__restrict__ rawF, const int64_t *__restrict__ rawG, const int64_t *__restrict__ rawS,
           uint64_t prefix, int shift, unsigned long long *__restrict__ hist) {
    __shared__ unsigned long long h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    const int64_t stride = static_cast<int64_t>(gridDim.x) * blockDim.x;
    const int64_t n_round = ceil_div_dev(nf, stride) * stride;
    const int lane = threadIdx.x & 31;
    for (int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x; i < n_round; i += stride) {
        uint32_t digit = 0xFFFFu;                            // lanes without a contribution
        uint64_t r = 0;
        if (i < nf) {
            int2 p = pair[f_lo + (sel ? sel[i] : i)];
            uint64_t key = static_cast<uint64_t>(static_cast<uint32_t>(p.x)) * nq2 + static_cast<uint32_t>(p.y);
            uint64_t hi = (shift + 8 >= 64) ? 0 : (key >> (shift + 8));
            r = static_cast<uint64_t>(rawU[i] + (rawF ? rawF[i] : 0) + (rawG ? rawG[i] : 0) + (rawS ? rawS[i] : 0));
            if (hi == prefix && r > 0) digit = static_cast<uint32_t>(key >> shift) & 255u;
        }
        const uint32_t peers = __match_any_sync(0xffffffffu, digit);
        const uint32_t l0 = __reduce_add_sync(peers, static_cast<uint32_t>(r & 0x3FFFFFu));
        const uint32_t l1 = __reduce_add_sync(peers, static_cast<uint32_t>((r >> 22) & 0x3FFFFFu));
        const uint32_t l2 = __reduce_add_sync(peers, static_cast<uint32_t>(r >> 44));
        if (digit != 0xFFFFu && lane == __ffs(peers) - 1)
            atomicAdd(&h[digit], static_cast<unsigned long long>(l0) + (static_cast<unsigned long long>(l1) << 22) +
                                     (static_cast<unsigned long long>(l2) << 44));
    }
    __syncthreads();
    if (h[threadIdx.x]) atomicAdd(&hist[threadIdx.x], h[threadIdx.x]);
}

// pairs with key >= cut are not expanded in this (last) level
__global__ void k_apply_cut(const int2 *__restrict__ pair, int64_t f_lo, int64_t nf, const uint32_t *__restrict__ sel,
                            uint64_t nq2, uint64_t cut,
                            int64_t *__restrict__ rawU, int64_t *__restrict__ rawF, uint32_t *__restrict__ nmU,
                            uint32_t *__restrict__ nmF, int64_t *__restrict__ rawG, int64_t *__restrict__ gwork,
                            uint32_t *__restrict__ nmG, int64_t *__restrict__ rawS, uint32_t *__restrict__ nmS,
                            unsigned long long *__restrict__ n_selected) {
    int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    bool keep = false;
    if (i < nf) {
        int2 p = pair[f_lo + (sel ? sel[i] : i)];
        uint64_t key = static_cast<uint64_t>(static_cast<uint32_t>(p.x)) * nq2 + static_cast<uint32_t>(p.y);
        keep = key < cut;
        if (!keep) {
            rawU[i] = 0; nmU[i] = 0;
            if (rawF) { rawF[i] = 0; nmF[i] = 0; }
            if (rawG) { rawG[i] = 0; gwork[i] = 0; nmG[i] = 0; }
            if (rawS) { rawS[i] = 0; nmS[i] = 0; }
        }
    }
    unsigned b = __ballot_sync(0xffffffffu, keep);
    if ((threadIdx.x & 31) == 0 && b) atomicAdd(n_selected, static_cast<unsigned long long>(__popc(b)));
}

struct MatchList {           // SoA work-list of one class
    int64_t *cum;            // [n+1] rank of the match's first arc; cum[n] = total
    uint4 *rec;              // [n] {first arc in M1, first arc in M2, n1, n2}
    uint32_t *pl;            // [n] pair index inside the level
};

__global__ void __launch_bounds__(CT_THREADS)
k_match(MachineView A, MachineView B, const int2 *__restrict__ pair, int64_t f_lo, int64_t nf, const uint32_t *__restrict__ sel,
        const uint32_t *__restrict__ nmU, const uint32_t *__restrict__ nmF, const int64_t *__restrict__ moffU,
        const int64_t *__restrict__ moffF, const int64_t *__restrict__ roffU, const int64_t *__restrict__ roffF,
        MatchList U, MatchList F,
        unsigned long long *__restrict__ counters /* [0] Σ segments visited, [1] Σ (n1+n2) over matches */) {
    int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    unsigned long long segs = 0, marcs = 0;
    const bool isF = i < nf && nmF && nmF[i] != 0;
    if (i < nf && (isF || nmU[i] != 0)) {
        int2 p = pair[f_lo + (sel ? sel[i] : i)];
        MatchList L = isF ? F : U;
        int64_t m = isF ? moffF[i] : moffU[i];
        int64_t run = isF ? roffF[i] : roffU[i];
        intersect(A, B, p.x, p.y, [&](uint32_t o1, uint32_t n1, uint32_t o2, uint32_t n2) {
            L.cum[m] = run;
            L.rec[m] = make_uint4(o1, o2, n1, n2);
            L.pl[m] = static_cast<uint32_t>(i);
            run += static_cast<int64_t>(n1) * n2;
            marcs += n1 + n2;
            ++m;
        });
        segs = (A.seg_ptr[p.x + 1] - A.seg_ptr[p.x]) + (B.seg_ptr[p.y + 1] - B.seg_ptr[p.y]);
    }
    // statistics for the algorithmic-bytes model: only pairs that are expanded and have a match are charged
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        segs += __shfl_xor_sync(0xffffffffu, segs, d);
        marcs += __shfl_xor_sync(0xffffffffu, marcs, d);
    }
    if ((threadIdx.x & 31) == 0 && (segs | marcs)) {
        atomicAdd(&counters[0], segs);
        atomicAdd(&counters[1], marcs);
    }
}

// ------------------------------------------------------------------------------------------ emit
// L2 residency hints: the packed operands are small and re-read for the whole level (evict-last); the
// output arcs are written once (streaming stores) so that they do not push the operands out of L2.
__device__ __forceinline__ uint64_t l2_evict_last_policy() {
    uint64_t p;
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint4 ld_keep(const uint4 *ptr, uint64_t policy) {
#if FSTC_EM_HINTS
    uint4 r;
    asm("ld.global.nc.L2::cache_hint.v4.u32 {%0, %1, %2, %3}, [%4], %5;"
        : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(ptr), "l"(policy));
    return r;
#else
    (void)policy;
    return __ldg(ptr);
#endif
}

#ifndef FSTC_EM_THREADS
#define FSTC_EM_THREADS 128
#endif
#ifndef FSTC_EM_MINB
#define FSTC_EM_MINB 5
#endif
#ifndef FSTC_EM_HINTS
#define FSTC_EM_HINTS 1
#endif
#ifndef FSTC_TABLE_LOAD_PCT
#define FSTC_TABLE_LOAD_PCT 40
#endif
#ifndef FSTC_RESOLVE_MIN_ARCS
#define FSTC_RESOLVE_MIN_ARCS (int64_t(1) << 24)
#endif
constexpr int64_t RESOLVE_MIN_ARCS = FSTC_RESOLVE_MIN_ARCS;          // smaller levels always use the table
constexpr uint64_t DENSE_MAX_PAIRS = 1ull << 29;                     // dense visited table (4 B per pair) up to 2 GB
constexpr uint64_t RESOLVE_TABLE_BYTES = 96ull << 20;               // a table beyond this no longer lives in L2
constexpr int64_t DORD_MIN_ARCS = int64_t(1) << 20;                  // smaller levels are not worth a scan of the dense table
// unit costs measured on a B200, in picoseconds
constexpr double COST_PROBE_PS = 21.0;            // random 32-byte sector read: one probe
constexpr double COST_INSERT_PS = 75.0;           // CAS write-back + id publish of a new state
constexpr double COST_STREAM_PS_PER_BYTE = 0.2;   // memset / streaming at ~5 TB/s
constexpr double COST_PART_ARC_PS = 45.0;         // keys + 2 scatter passes + dedupe + 2 gathers, per arc
constexpr double COST_PART_STATE_PS = 30.0;       // re-entering an existing state, per level
constexpr int EM_THREADS = FSTC_EM_THREADS;
constexpr int EM_IPT = 4;                          // consecutive output ranks per thread
constexpr int EM_TILE = EM_THREADS * EM_IPT;       // 512 arcs per block

enum { EMIT_DIRECT = 0, EMIT_INDIRECT = 1, EMIT_SORTREC = 2 };

struct EmitArgs {
    MachineView A, B;
    MatchList L;
    int64_t n_matches;
    int64_t R;               // ranks [0, R)
    int64_t pos_base;        // DIRECT: output position of rank 0 (tiles are aligned on absolute positions)
    int64_t f_lo;            // source id = f_lo + pair index (through sel, if the level was compacted)
    const uint32_t *sel;
    const int64_t *foff;     // INDIRECT: final position of the pair's first arc (relative to arc_base)
    const int64_t *roff;     // INDIRECT: rank of the pair's first arc
    int64_t arc_base;        // INDIRECT
    uint64_t nq2;
    uint4 *table;
    uint64_t cap;
    uint32_t *dense;         // RES_DENSE: [|Q1||Q2|] id + 1 of every pair, 0 = not visited
    unsigned long long *n_states;
    int2 *pair;
    int32_t *o_src, *o_il, *o_ol, *o_tgt;
    float *o_w;
    uint4 *sortrec;          // SORTREC: {key lo, key hi, pair index, weight}, key = tgt id << shift_t | a << bits_b | b
    int shift_t, bits_b;
    const int64_t *tile_m;   // [n_tiles+1] match index holding the first rank of every tile
    unsigned long long *keys;     // KEYS: [R] target key of every rank, for the partitioned resolve
    int q2_bits;                  // KEYS: the resolve key is (r1 << q2_bits) | r2
    uint32_t *posout;             // KEYS + INDIRECT: [R] output position of every rank (relative to arc_base)
};

// tile_m[t] = last match whose first rank <= first rank of tile t
__global__ void k_partition(const int64_t *__restrict__ cum, int64_t n_matches, int64_t R, int64_t pos_base,
                            int64_t n_tiles, int64_t *__restrict__ tile_m) {
    int64_t t = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (t > n_tiles) return;
    int64_t tile0 = (pos_base / EM_TILE) * EM_TILE;
    int64_t rank = tile0 + t * EM_TILE - pos_base;
    if (rank < 0) rank = 0;
    if (rank >= R) { tile_m[t] = n_matches; return; }   // only t == n_tiles (or beyond the data)
    int64_t lo = 0, hi = n_matches;                      // first m with cum[m] > rank
    while (lo < hi) {
        int64_t mid = (lo + hi) >> 1;
        if (cum[mid] <= rank) lo = mid + 1; else hi = mid;
    }
    tile_m[t] = lo - 1;
}

// RES_HASH / RES_DENSE: the target ids come from the visited table, inside this kernel — the open-addressing hash
// table, or, when |Q1||Q2| is small enough, the paper's dense table of one entry per pair (entry =
// id + 1, 0 = not visited).  RES_KEYS: the kernel leaves the target column open and writes the target key of every
// arc for resolve_partitioned.
// RES_DORD: dense table, ids in KEY ORDER: the kernel only marks the targets it meets for the first time (entry 0 -> PENDING)
// and leaves ~key in the target column of arcs to unnumbered states; k_dord_* number the marked entries in a scan of the table
// (ascending key) and k_dord_fix completes the target column.
enum { RES_HASH = 0, RES_KEYS = 1, RES_DENSE = 2, RES_DORD = 3 };
template <int MODE, int RES>
__global__ void __launch_bounds__(EM_THREADS, FSTC_EM_MINB) k_emit(EmitArgs g) {
    constexpr bool KEYS = RES == RES_KEYS, DENSE = RES == RES_DENSE, DORD = RES == RES_DORD;
    __shared__ uint32_t relcum[EM_TILE + 1];
    __shared__ uint4 s_rec[EM_TILE + 1];                      // the tile's matches, staged with coalesced loads: rank -> match -> arcs
    __shared__ uint32_t s_pl[EM_TILE + 1];                    // then waits on ONE dependent global load (the arcs), not two
    __shared__ int64_t s_first_cum;
    __shared__ uint32_t s_warp[EM_THREADS / 32];
    __shared__ unsigned long long s_base;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t tile0 = (g.pos_base / EM_TILE) * EM_TILE;
    const int64_t tile_pos = tile0 + static_cast<int64_t>(blockIdx.x) * EM_TILE;   // absolute position of the tile
    int64_t rank_lo = tile_pos - g.pos_base;                 // first rank of the tile (may be < 0 in tile 0)
    int64_t rank_hi = rank_lo + EM_TILE;
    if (rank_lo < 0) rank_lo = 0;
    if (rank_hi > g.R) rank_hi = g.R;

    const int64_t m_lo = g.tile_m[blockIdx.x];
    int64_t m_hi = g.tile_m[blockIdx.x + 1];                 // inclusive, last match that can start inside the tile
    if (m_hi >= g.n_matches) m_hi = g.n_matches - 1;
    const int nm = static_cast<int>(m_hi - m_lo + 1);        // <= EM_TILE + 1
    for (int j = tid; j < nm; j += EM_THREADS) {
        int64_t c = g.L.cum[m_lo + j] - rank_lo;
        relcum[j] = c < 0 ? 0u : static_cast<uint32_t>(c > EM_TILE ? EM_TILE : c);
        s_rec[j] = g.L.rec[m_lo + j];
        s_pl[j] = g.L.pl[m_lo + j];
    }
    if (tid == 0) s_first_cum = g.L.cum[m_lo];
    __syncthreads();

    // ---- locate this thread's first rank
    const int64_t my_pos = tile_pos + tid * EM_IPT;
    int64_t rank0 = my_pos - g.pos_base;
    int n_valid = 0;                                          // ranks rank0+skip .. rank0+skip+n_valid-1
    int skip = 0;
    {
        int64_t a = rank0 < rank_lo ? rank_lo : rank0;
        int64_t b = rank0 + EM_IPT < rank_hi ? rank0 + EM_IPT : rank_hi;
        if (b > a) { n_valid = static_cast<int>(b - a); skip = static_cast<int>(a - rank0); }
    }
    uint32_t idx1[EM_IPT], idx2[EM_IPT], pl[EM_IPT];
    if (n_valid > 0) {
        const int64_t first = rank0 + skip;
        const uint32_t rr = static_cast<uint32_t>(first - rank_lo);
        int lo = 0, hi = nm;                                  // first j with relcum[j] > rr
        while (lo < hi) {
            int mid = (lo + hi) >> 1;
            if (relcum[mid] <= rr) lo = mid + 1; else hi = mid;
        }
        int j = lo - 1;
        int64_t m = m_lo + j;
        uint64_t r = (j == 0) ? static_cast<uint64_t>(first - s_first_cum) : static_cast<uint64_t>(rr - relcum[j]);
        uint4 rec = s_rec[j];
        uint32_t p = s_pl[j];
        uint32_t i1, i2;
        if (r < 0xFFFFFFFFull) { i1 = static_cast<uint32_t>(r) / rec.w; i2 = static_cast<uint32_t>(r) - i1 * rec.w; }
        else { i1 = static_cast<uint32_t>(r / rec.w); i2 = static_cast<uint32_t>(r - static_cast<uint64_t>(i1) * rec.w); }
#pragma unroll
        for (int u = 0; u < EM_IPT; ++u) {
            if (u >= skip && u < skip + n_valid) {
                idx1[u] = rec.x + i1; idx2[u] = rec.y + i2; pl[u] = p;
                if (++i2 == rec.w) {
                    i2 = 0;
                    if (++i1 == rec.z) {
                        i1 = 0; ++m; ++j;
                        if (m <= m_hi) { rec = s_rec[j]; p = s_pl[j]; }
                    }
                }
            }
        }
    }

    // ---- read the two input arcs of every rank, form the composed arc
    const uint64_t keep_policy = l2_evict_last_policy();     // operands are re-read all level long: keep them in L2
    uint32_t a_sym[EM_IPT], b_sym[EM_IPT];
    float w[EM_IPT];
    unsigned long long key[EM_IPT];
    int2 tgt_pair[EM_IPT];
    uint32_t todo = 0;                                        // bit u: rank u still has to be resolved in the table
#pragma unroll
    for (int u = 0; u < EM_IPT; ++u) {
        if (u >= skip && u < skip + n_valid) {
            uint4 e1 = ld_keep(g.A.arcs + idx1[u], keep_policy);   // {tgt, outer, weight, inner}
            uint4 e2 = ld_keep(g.B.arcs + idx2[u], keep_policy);
            a_sym[u] = e1.y; b_sym[u] = e2.y;
            w[u] = __uint_as_float(e1.z) * __uint_as_float(e2.z);
            tgt_pair[u] = make_int2(static_cast<int>(e1.x), static_cast<int>(e2.x));
            key[u] = KEYS ? ((static_cast<unsigned long long>(e1.x) << g.q2_bits) | e2.x) : static_cast<uint64_t>(e1.x) * g.nq2 + e2.x;
            todo |= 1u << u;
        }
    }

    uint32_t id[EM_IPT];
#pragma unroll
    for (int u = 0; u < EM_IPT; ++u) id[u] = 0;
    if (KEYS) {
        // ---- partitioned resolve: leave the target keys, in rank order
        if (n_valid == EM_IPT && ((rank0 & 1) == 0)) {
            __stcs(reinterpret_cast<ulonglong2 *>(g.keys + rank0), make_ulonglong2(key[0], key[1]));
            __stcs(reinterpret_cast<ulonglong2 *>(g.keys + rank0 + 2), make_ulonglong2(key[2], key[3]));
        } else {
#pragma unroll
            for (int u = 0; u < EM_IPT; ++u)
                if (u >= skip && u < skip + n_valid) g.keys[rank0 + u] = key[u];
        }
        if (MODE == EMIT_INDIRECT) {
#pragma unroll
            for (int u = 0; u < EM_IPT; ++u)
                if (u >= skip && u < skip + n_valid)
                    g.posout[rank0 + u] = static_cast<uint32_t>(g.foff[pl[u]] + (rank0 + u - g.roff[pl[u]]));
        }
    } else if (DORD) {
        uint32_t v[EM_IPT];
#pragma unroll
        for (int u = 0; u < EM_IPT; ++u) v[u] = (todo >> u & 1u) ? __ldcg(g.dense + key[u]) : 1u;
#pragma unroll
        for (int u = 0; u < EM_IPT; ++u)
            if ((todo >> u & 1u) && v[u] == 0u) v[u] = atomicCAS(g.dense + key[u], 0u, PENDING_ID);
#pragma unroll
        for (int u = 0; u < EM_IPT; ++u)
            id[u] = (v[u] == 0u || v[u] == PENDING_ID) ? ~static_cast<uint32_t>(key[u]) : v[u] - 1u;   // (keys < 2^29: ~key < 0 as int32)
    } else {
    // ---- visited set: find or insert.  Rounds of: all pending bucket reads in flight
    // together, then all pending CAS in flight together; a rank leaves when it finds its key or wins a slot.
    uint64_t slot[EM_IPT];                                    // bucket while searching, then the key's slot
    uint32_t won = 0;                                         // bit u: this thread inserted the key (new state)
    if (DENSE) {
        uint32_t v[EM_IPT];
#pragma unroll
        for (int u = 0; u < EM_IPT; ++u) {
            slot[u] = key[u];
            if (todo >> u & 1u) v[u] = __ldcg(g.dense + key[u]);
        }
#pragma unroll
        for (int u = 0; u < EM_IPT; ++u)
            if ((todo >> u & 1u) && v[u] == 0u) v[u] = atomicCAS(g.dense + key[u], 0u, PENDING_ID);   // 0: this thread won
#pragma unroll
        for (int u = 0; u < EM_IPT; ++u) {
            if (todo >> u & 1u) {
                if (v[u] == 0u) won |= 1u << u;
                else id[u] = v[u] == PENDING_ID ? PENDING_ID : v[u] - 1u;
            }
        }
        todo = 0;
    }
    const uint64_t n_buckets = g.cap >> 1;
#pragma unroll
    for (int u = 0; u < EM_IPT; ++u) if (!DENSE) slot[u] = (todo >> u & 1u) ? home_bucket(key[u], g.cap) : 0;
    while (todo) {
        Bucket v[EM_IPT];
        unsigned long long old[EM_IPT];
        uint32_t cas = 0, second = 0;                         // second: the CAS targets slot 1 of the bucket
#pragma unroll
        for (int u = 0; u < EM_IPT; ++u)
            if (todo >> u & 1u) v[u] = ld_bucket(g.table, slot[u]);
#pragma unroll
        for (int u = 0; u < EM_IPT; ++u) {
            if (todo >> u & 1u) {
                const unsigned long long k0 = slot_key(v[u].s0), k1 = slot_key(v[u].s1);
                if (k0 == key[u]) { id[u] = v[u].s0.z; slot[u] = 2 * slot[u]; todo &= ~(1u << u); }
                else if (k0 == EMPTY_KEY) cas |= 1u << u;
                else if (k1 == key[u]) { id[u] = v[u].s1.z; slot[u] = 2 * slot[u] + 1; todo &= ~(1u << u); }
                else if (k1 == EMPTY_KEY) { cas |= 1u << u; second |= 1u << u; }
                else slot[u] = (slot[u] + 1 == n_buckets) ? 0 : slot[u] + 1;   // both slots taken by other keys
            }
        }
#pragma unroll
        for (int u = 0; u < EM_IPT; ++u)
            if (cas >> u & 1u)
                old[u] = atomicCAS(reinterpret_cast<unsigned long long *>(g.table + 2 * slot[u] + (second >> u & 1u)),
                                   EMPTY_KEY, key[u]);
#pragma unroll
        for (int u = 0; u < EM_IPT; ++u) {
            if (cas >> u & 1u) {
                if (old[u] == EMPTY_KEY) { won |= 1u << u; slot[u] = 2 * slot[u] + (second >> u & 1u); todo &= ~(1u << u); }
                else if (old[u] == key[u]) { id[u] = PENDING_ID; slot[u] = 2 * slot[u] + (second >> u & 1u); todo &= ~(1u << u); }
                // else: another key took the slot first -> look at the same bucket again
            }
        }
    }
    const uint32_t n_won = __popc(won);

    // ---- new state ids: one atomicAdd per block; the new ids of a level are the next frontier
    uint32_t incl = n_won;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += t;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    if (tid == 0) {
        uint32_t tot = 0;
#pragma unroll
        for (int wv = 0; wv < EM_THREADS / 32; ++wv) { uint32_t c = s_warp[wv]; s_warp[wv] = tot; tot += c; }
        s_base = tot ? atomicAdd(g.n_states, static_cast<unsigned long long>(tot)) : 0ull;
    }
    __syncthreads();
    uint32_t next_id = static_cast<uint32_t>(s_base) + s_warp[warp] + (incl - n_won);
#pragma unroll
    for (int u = 0; u < EM_IPT; ++u) {
        if (won >> u & 1u) {
            id[u] = next_id++;
            if (DENSE) __stcg(g.dense + slot[u], id[u] + 1u);
            else __stcg(reinterpret_cast<uint32_t *>(g.table + slot[u]) + 2, id[u]);   // publish
            g.pair[id[u]] = tgt_pair[u];
        }
    }
    // ---- targets inserted concurrently by another thread: wait for their id to be published
#pragma unroll
    for (int u = 0; u < EM_IPT; ++u) {
        if (u >= skip && u < skip + n_valid && !(won >> u & 1u) && id[u] == PENDING_ID) {
            const uint32_t *pid = DENSE ? g.dense + slot[u] : reinterpret_cast<const uint32_t *>(g.table + slot[u]) + 2;
            uint32_t v;
            while ((v = __ldcg(pid)) == PENDING_ID) __nanosleep(20);
            id[u] = DENSE ? v - 1u : v;
        }
    }
    }   // !KEYS

    // ---- write the composed arcs
#define SRC(u) (g.sel ? g.sel[pl[u]] : pl[u])
    if (MODE == EMIT_DIRECT) {
        if (n_valid == EM_IPT) {                               // whole aligned group: 16-byte stores
            const int64_t q = my_pos;
            __stcs(reinterpret_cast<int4 *>(g.o_src + q), make_int4(static_cast<int>(g.f_lo + SRC(0)), static_cast<int>(g.f_lo + SRC(1)),
                                                                   static_cast<int>(g.f_lo + SRC(2)), static_cast<int>(g.f_lo + SRC(3))));
            __stcs(reinterpret_cast<uint4 *>(g.o_il + q), make_uint4(a_sym[0], a_sym[1], a_sym[2], a_sym[3]));
            __stcs(reinterpret_cast<uint4 *>(g.o_ol + q), make_uint4(b_sym[0], b_sym[1], b_sym[2], b_sym[3]));
            if (!KEYS) __stcs(reinterpret_cast<uint4 *>(g.o_tgt + q), make_uint4(id[0], id[1], id[2], id[3]));
            __stcs(reinterpret_cast<float4 *>(g.o_w + q), make_float4(w[0], w[1], w[2], w[3]));
        } else {
#pragma unroll
            for (int u = 0; u < EM_IPT; ++u) {
                if (u >= skip && u < skip + n_valid) {
                    const int64_t q = my_pos + u;
                    g.o_src[q] = static_cast<int>(g.f_lo + SRC(u));
                    g.o_il[q] = a_sym[u]; g.o_ol[q] = b_sym[u]; g.o_w[q] = w[u];
                    if (!KEYS) g.o_tgt[q] = id[u];
                }
            }
        }
    } else if (MODE == EMIT_INDIRECT) {
#pragma unroll
        for (int u = 0; u < EM_IPT; ++u) {
            if (u >= skip && u < skip + n_valid) {
                const int64_t rank = rank0 + u;
                const int64_t q = g.arc_base + g.foff[pl[u]] + (rank - g.roff[pl[u]]);
                g.o_src[q] = static_cast<int>(g.f_lo + SRC(u));
                g.o_il[q] = a_sym[u]; g.o_ol[q] = b_sym[u]; g.o_w[q] = w[u];
                if (!KEYS) g.o_tgt[q] = id[u];
            }
        }
    } else {
#pragma unroll
        for (int u = 0; u < EM_IPT; ++u) {
            if (u >= skip && u < skip + n_valid) {
                unsigned long long k = (static_cast<unsigned long long>(id[u]) << g.shift_t) |
                                       (static_cast<unsigned long long>(a_sym[u]) << g.bits_b) | b_sym[u];
                g.sortrec[rank0 + u] = make_uint4(static_cast<uint32_t>(k), static_cast<uint32_t>(k >> 32), pl[u],
                                                  __float_as_uint(w[u]));
            }
        }
    }
#undef SRC
}

// ------------------------------------------------------------------------------------------ merge by construction
// Class G.  Seen from a source pair (q1,q2), M1 only contributes (a, r1) and M2 only (b, r2): group q1's arcs by
// (a, r1) and q2's by (b, r2) (the packer's grouped copy); every composed-and-merged arc of the pair is one pair of
// groups that share an inner symbol, and its weight is sum_c (sum of p1 over the group's arcs with c) x (same for p2)
// (PAPER.md:53,65 regrouped).  So the merged arcs come out directly, in (a, r1, b, r2) order, with no sort and no
// reduce: work = groups x groups per pair (load-balanced over ranks like the emit kernel), not raw arcs.
// The match list of this class has one entry per pair: {first group of q1, first group of q2, #groups, #groups}.
__global__ void __launch_bounds__(CT_THREADS)
k_gmatch(MachineView A, MachineView B, const int2 *__restrict__ pair, int64_t f_lo, int64_t nf, const uint32_t *__restrict__ sel,
         const uint32_t *__restrict__ nmG, const int64_t *__restrict__ moffG, const int64_t *__restrict__ woff, MatchList G) {
    int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= nf || nmG[i] == 0) return;
    int2 p = pair[f_lo + (sel ? sel[i] : i)];
    const int64_t m = moffG[i];
    const uint32_t g1 = A.gptr[p.x], g2 = B.gptr[p.y];
    G.cum[m] = woff[i];
    G.rec[m] = make_uint4(g1, g2, A.gptr[p.x + 1] - g1, B.gptr[p.y + 1] - g2);
    G.pl[m] = static_cast<uint32_t>(i);
}

struct GProdArgs {
    MachineView A, B;
    MatchList L;
    int64_t n_matches, W;        // ranks [0, W) = group pairs
    const int64_t *tile_m;
    uint32_t *tile_cnt;          // pass 0: arcs found per tile
    uint8_t *ebits;              // [tiles * GP_THREADS] which of a thread's ranks give an arc: written by pass 0, read by pass 1
    const int64_t *tile_off;     // pass 1: first output slot of every tile
    uint32_t *msrc;              // pass 1 outputs, compact, in rank order: pair index,
    uint32_t *mab;               //   a << bits_b | b,
    float *mw;                   //   merged weight,
    unsigned long long *mkey;    //   target key (table: r1 * |Q2| + r2; partitioned resolve: (r1 << q2_bits) | r2)
    int bits_b, q2_bits;         // q2_bits < 0: table key
    uint64_t nq2;
    uint16_t *eprefix;           // [tiles * GP_THREADS] arcs of the tile before the thread's ranks (pass 0 -> k_gcount, pass 2)
    // pass 2 (fused: weights, visited table, final place in one kernel; table levels only)
    uint32_t *dense; uint4 *table; uint64_t cap;
    unsigned long long *n_states; int2 *pair;
    const int64_t *mstart, *foff;    // per pair of the level: first merged class-G arc, first final arc
    int64_t arc_base, f_lo;
    const uint32_t *sel;
    int32_t *o_src, *o_il, *o_ol, *o_tgt; float *o_w;
};

// compensated (Kahan) fp32 accumulation: the error of a sum of n terms stays at a few ulp whatever n, so that a run of
// thousands of parallel arcs, or a group pair with thousands of common symbols, stays inside rtol 1e-5 (N13)
struct KahanSum {
    float s = 0.f, c = 0.f;
    __device__ __forceinline__ void add(float x) {
        const float y = x - c;
        const float t = s + y;
        c = (t - s) - y;
        s = t;
    }
};

// sum over the common inner symbols of two groups; *found = at least one common symbol
__device__ __forceinline__ float group_dot(const uint2 *__restrict__ ga, uint32_t a0, uint32_t a1, const uint2 *__restrict__ gb,
                                           uint32_t b0, uint32_t b1, bool first_only, bool *found) {
    KahanSum sum;
    bool any = false;
    uint2 x = ga[a0], y = gb[b0];
    while (true) {
        if (x.x == y.x) {
            any = true;
            if (first_only) break;
            const uint32_t c = x.x;                              // runs of equal symbols (parallel duplicate arcs) first
            KahanSum sa, sb;
            while (true) { sa.add(__uint_as_float(x.y)); if (++a0 == a1) break; x = ga[a0]; if (x.x != c) break; }
            while (true) { sb.add(__uint_as_float(y.y)); if (++b0 == b1) break; y = gb[b0]; if (y.x != c) break; }
            sum.add(sa.s * sb.s);
            if (a0 == a1 || b0 == b1) break;
        } else if (x.x < y.x) {
            if (++a0 == a1) break;
            x = ga[a0];
        } else {
            if (++b0 == b1) break;
            y = gb[b0];
        }
    }
    *found = any;
    return sum.s;
}

constexpr int GP_THREADS = 128, GP_IPT = 4, GP_TILE = GP_THREADS * GP_IPT;
static_assert(GP_TILE == EM_TILE, "k_partition places tiles of EM_TILE ranks");

template <int PASS, bool DENSE>
__global__ void __launch_bounds__(GP_THREADS) k_gprod(GProdArgs g) {
    __shared__ uint32_t relcum[GP_TILE + 1];
    __shared__ int64_t s_first_cum;
    __shared__ uint32_t s_warp[GP_THREADS / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t rank_lo = static_cast<int64_t>(blockIdx.x) * GP_TILE;
    const int64_t rank_hi = rank_lo + GP_TILE < g.W ? rank_lo + GP_TILE : g.W;
    const int64_t m_lo = g.tile_m[blockIdx.x];
    int64_t m_hi = g.tile_m[blockIdx.x + 1];
    if (m_hi >= g.n_matches) m_hi = g.n_matches - 1;
    const int nm = static_cast<int>(m_hi - m_lo + 1);
    for (int j = tid; j < nm; j += GP_THREADS) {
        int64_t c = g.L.cum[m_lo + j] - rank_lo;
        relcum[j] = c < 0 ? 0u : static_cast<uint32_t>(c > GP_TILE ? GP_TILE : c);
    }
    if (tid == 0) s_first_cum = g.L.cum[m_lo];
    __syncthreads();
    const int64_t rank0 = rank_lo + tid * GP_IPT;
    int n_valid = rank0 < rank_hi ? static_cast<int>(rank_hi - rank0 < GP_IPT ? rank_hi - rank0 : GP_IPT) : 0;
    uint32_t exists = 0;
    uint32_t g1v[GP_IPT], g2v[GP_IPT], plv[GP_IPT];
    if (n_valid > 0) {
        const uint32_t rr = static_cast<uint32_t>(rank0 - rank_lo);
        int lo = 0, hi = nm;
        while (lo < hi) {
            int mid = (lo + hi) >> 1;
            if (relcum[mid] <= rr) lo = mid + 1; else hi = mid;
        }
        int j = lo - 1;
        int64_t m = m_lo + j;
        uint64_t r = (j == 0) ? static_cast<uint64_t>(rank0 - s_first_cum) : static_cast<uint64_t>(rr - relcum[j]);
        uint4 rec = g.L.rec[m];
        uint32_t p = g.L.pl[m];
        uint32_t i1, i2;                                         // (a 64-bit division costs ~40 instructions: only when it must be)
        if (r < 0xFFFFFFFFull) { i1 = static_cast<uint32_t>(r) / rec.w; i2 = static_cast<uint32_t>(r) - i1 * rec.w; }
        else { i1 = static_cast<uint32_t>(r / rec.w); i2 = static_cast<uint32_t>(r - static_cast<uint64_t>(i1) * rec.w); }
#pragma unroll
        for (int u = 0; u < GP_IPT; ++u) {
            if (u < n_valid) {
                g1v[u] = rec.x + i1; g2v[u] = rec.y + i2; plv[u] = p;
                if (++i2 == rec.w) {
                    i2 = 0;
                    if (++i1 == rec.z) {
                        i1 = 0; ++m;
                        if (m <= m_hi) { rec = g.L.rec[m]; p = g.L.pl[m]; }
                    }
                }
            }
        }
        if (PASS == 1) exists = g.ebits[static_cast<int64_t>(blockIdx.x) * GP_THREADS + tid];   // what pass 0 found
        else {
            const bool masks = g.A.gmask != nullptr && g.B.gmask != nullptr;  // |Γ| <= 63: symbol sets as bit masks, one AND per rank
#pragma unroll
            for (int u = 0; u < GP_IPT; ++u) {
                if (u < n_valid) {
                    bool found;
                    if (masks) found = (g.A.gmask[g1v[u]] & g.B.gmask[g2v[u]] & ~(1ull << 63)) != 0;
                    else (void)group_dot(g.A.garcs, g.A.goff[g1v[u]], g.A.goff[g1v[u] + 1], g.B.garcs, g.B.goff[g2v[u]],
                                         g.B.goff[g2v[u] + 1], true, &found);
                    if (found) exists |= 1u << u;
                }
            }
        }
    }
    const uint32_t n_mine = __popc(exists);
    uint32_t incl = n_mine;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += t;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    uint32_t before = incl - n_mine, total = 0;
#pragma unroll
    for (int wv = 0; wv < GP_THREADS / 32; ++wv) { if (wv < warp) before += s_warp[wv]; total += s_warp[wv]; }
    if (PASS == 0) {
        g.ebits[static_cast<int64_t>(blockIdx.x) * GP_THREADS + tid] = static_cast<uint8_t>(exists);
        g.eprefix[static_cast<int64_t>(blockIdx.x) * GP_THREADS + tid] = static_cast<uint16_t>(before);
        if (tid == 0) g.tile_cnt[blockIdx.x] = total;
    }
    if constexpr (PASS != 0) {
    // pass 1: typically a third of a tile's ranks give an arc.  They are packed first (rank order), so that every lane of the
    // weight loop below has an arc to work on and the outputs of a warp are neighbours.
    __shared__ uint32_t s_g1[GP_TILE], s_g2[GP_TILE], s_pl[GP_TILE];
#pragma unroll
    for (int u = 0; u < GP_IPT; ++u) {
        if (exists >> u & 1u) { s_g1[before] = g1v[u]; s_g2[before] = g2v[u]; s_pl[before] = plv[u]; ++before; }
    }
    __syncthreads();
    const bool masks = g.A.gmask != nullptr && g.B.gmask != nullptr;
    const int64_t q0 = g.tile_off[blockIdx.x];
    __shared__ unsigned long long s_base;
    for (uint32_t kb = 0; kb < total; kb += GP_THREADS) {          // (uniform trip count: pass 2 has block barriers inside)
        const uint32_t k = kb + tid;
        const bool valid = k < total;
        if (PASS == 1 && !valid) continue;
        const uint32_t g1 = valid ? s_g1[k] : s_g1[0], g2 = valid ? s_g2[k] : s_g2[0];
        const uint32_t a0 = g.A.goff[g1], b0 = g.B.goff[g2];
        float wv;
        unsigned long long m1 = 0, m2 = 0;
        if (masks) { m1 = g.A.gmask[g1]; m2 = g.B.gmask[g2]; }
        if (masks && !((m1 | m2) >> 63)) {                                // no symbol twice in either group: weights by popcount
            unsigned long long common = m1 & m2;
            KahanSum sum;
            while (common) {
                const unsigned long long below = (common & (0 - common)) - 1;
                common &= common - 1;
                sum.add(__uint_as_float(g.A.garcs[a0 + __popcll(m1 & below)].y) * __uint_as_float(g.B.garcs[b0 + __popcll(m2 & below)].y));
            }
            wv = sum.s;
        } else {
            bool found;
            wv = group_dot(g.A.garcs, a0, g.A.goff[g1 + 1], g.B.garcs, b0, g.B.goff[g2 + 1], false, &found);
        }
        const uint2 k1 = g.A.gkey[g1], k2 = g.B.gkey[g2];                 // {outer, tgt}
        if (PASS == 1) {
            const int64_t q = q0 + k;
            g.msrc[q] = s_pl[k];
            g.mab[q] = (k1.x << g.bits_b) | k2.x;
            g.mw[q] = wv;
            g.mkey[q] = g.q2_bits >= 0 ? ((static_cast<unsigned long long>(k1.y) << g.q2_bits) | k2.y)
                                       : static_cast<unsigned long long>(k1.y) * g.nq2 + k2.y;
        } else {
            // fused: the target's id from the visited table, and the arc straight to its final place behind the pair's offset
            const unsigned long long key = static_cast<unsigned long long>(k1.y) * g.nq2 + k2.y;
            const uint32_t id = DENSE ? block_find_or_insert<true, GP_THREADS>(key, valid, make_int2(static_cast<int>(k1.y), static_cast<int>(k2.y)), g.dense, g.table, g.cap, g.n_states, g.pair, s_warp, &s_base)
                                      : block_find_or_insert<false, GP_THREADS>(key, valid, make_int2(static_cast<int>(k1.y), static_cast<int>(k2.y)), g.dense, g.table, g.cap, g.n_states, g.pair, s_warp, &s_base);
            if (valid) {
                const uint32_t p = s_pl[k];
                const int64_t q = g.arc_base + g.foff[p] + (q0 + k - g.mstart[p]);
                g.o_src[q] = static_cast<int>(g.f_lo + (g.sel ? g.sel[p] : p));
                g.o_il[q] = static_cast<int>(k1.x); g.o_ol[q] = static_cast<int>(k2.x);
                g.o_tgt[q] = static_cast<int>(id); g.o_w[q] = wv;
            }
        }
    }
}   // PASS != 0
}

// Merged class-G arcs per pair of the level, from what pass 0 left (ebits, eprefix, tile_off): cntG[pair] = arcs among the
// pair's ranks [cum[m], cum[m+1]).  (One match per class-G pair; the other pairs keep 0.)
__device__ __forceinline__ int64_t g_arcs_before(const GProdArgs &g, int64_t r) {      // existing ranks < r
    const int64_t t = r / GP_TILE;
    const int64_t th = t * GP_THREADS + (r % GP_TILE) / GP_IPT;
    if (r >= g.W) return g.tile_off[(g.W + GP_TILE - 1) / GP_TILE];
    return g.tile_off[t] + g.eprefix[th] + __popc(g.ebits[th] & ((1u << (r % GP_IPT)) - 1u));
}
__global__ void k_gcount(GProdArgs g, int64_t *__restrict__ cntG) {
    const int64_t m = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (m >= g.n_matches) return;
    cntG[g.L.pl[m]] = g_arcs_before(g, g.L.cum[m + 1]) - g_arcs_before(g, g.L.cum[m]);
}

// Ids of a list of target keys through the visited table (dense or hash), outside the emit kernel: one key per thread,
// new ids per block with one atomicAdd.  Same protocol as in k_emit.
template <bool DENSE>
__global__ void __launch_bounds__(CT_THREADS)
k_resolve_keys(const unsigned long long *__restrict__ keys, int64_t n, uint32_t *dense, uint4 *table, uint64_t cap, uint64_t nq2,
               unsigned long long *n_states, int2 *pair, int32_t *__restrict__ ids) {
    __shared__ uint32_t s_warp[CT_THREADS / 32];
    __shared__ unsigned long long s_base;
    const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    const bool valid = i < n;
    const unsigned long long key = valid ? keys[i] : 0ull;
    const unsigned long long q1 = key / nq2;
    const uint32_t id = block_find_or_insert<DENSE, CT_THREADS>(key, valid, make_int2(static_cast<int>(q1), static_cast<int>(key - q1 * nq2)),
                                                                dense, table, cap, n_states, pair, s_warp, &s_base);
    if (valid) ids[i] = static_cast<int32_t>(id);
}

// ------------------------------------------------------------------------------------------ merge on chip (class S)
// SURVEY §8(f)1, the paper's own future work: the raw arcs of a source that can hold duplicates are
// composed, merged and summed in SHARED memory, so that only merged arcs reach HBM.  A block takes a TILE of the class-S
// rank space: the pairs whose first rank falls into [t T, (t+1) T), each of at most FC_PAIR_CAP = T raw arcs, so fewer than
// 2T arcs in all.  No sort: a pair of r raw arcs owns the 2r hash slots behind 2 x (its first rank in the tile); every raw
// arc finds or claims the slot of its (r1, r2, a, b) there (64-bit CAS, linear probing inside the pair's region) and adds
// its weight to the slot's fp64 sum.  The occupied slots, in slot order, ARE the merged arcs grouped by pair: a block scan
// numbers them, one atomicAdd reserves the tile's piece of the compact output, and every pair learns its count and its
// first arc.  ~600 thread-instructions per raw arc (ncu: 19 warp-instructions) against several thousand for a bitonic sort
// of the tile, and no HBM traffic per raw arc beyond its match record and the two operand arcs (which L2 serves).
// T = 512 with one thread per rank of the tile (`dups`, reduce stage, T / threads: 512/256 63.5 ms, 512/512 54.8,
// 256/256 51.6, 128/128 50.8, 256/512 76.5, 128/256 71.5; match records staged in shared memory 73.2: occupancy).
// The merged arcs leave with their target KEY; their ids come from the visited set afterwards, like class G's — one
// lookup per MERGED arc, not per raw arc.
constexpr int FC_THREADS = FSTC_FC_THREADS;
constexpr int FC_TILE = FC_PAIR_CAP;
constexpr int FC_MAX_ARCS = 2 * FC_TILE;            // raw arcs of a tile: < FC_TILE + FC_PAIR_CAP
constexpr int FC_SLOTS = 2 * FC_MAX_ARCS;
constexpr int FC_CHUNK = FC_SLOTS / FC_THREADS;     // rounds of 32 slots a warp numbers
constexpr unsigned long long FC_EMPTY = ~0ull;
constexpr size_t FC_SMEM = sizeof(unsigned long long) * FC_SLOTS + sizeof(double) * FC_SLOTS + sizeof(uint32_t) * (FC_MAX_ARCS + 1) +
                           sizeof(uint16_t) * (3 * FC_MAX_ARCS + FC_SLOTS + 2);
static_assert(FC_SLOTS % (FC_THREADS) == 0 && FC_MAX_ARCS < 65536, "slot rounds of a warp; uint16 indices");

struct FChipArgs {
    MachineView A, B;
    MatchList L;                  // class-S match list (matches in pair order, cum = first rank)
    const int64_t *roff, *moff;   // [nf+1] first rank / first match of every pair of the level in class S
    const int64_t *raw;           // [nf]   raw arcs of the pair in class S (0: not of this class)
    int64_t nf;
    const int64_t *tile_p;        // [n_tiles+1] first pair of every tile
    int shift_t, bits_b, q2_bits;
    uint64_t nq2;
    int table_key;                // 1: mkey = r1 * |Q2| + r2 (visited table)   0: (r1 << q2_bits) | r2 (partitioned resolve)
    unsigned long long *cursor;   // merged arcs written so far
    uint32_t *msrc, *mab;         // compact outputs (a pair's arcs are neighbours; tiles in arrival order)
    float *mw;
    unsigned long long *mkey;
    int64_t *cnt, *base;          // [nf] merged arcs of the pair, and the first of them
};

// tile_p[t] = first pair i with roff[i] >= t * FC_TILE   (t = 0..n_tiles; roff has nf + 1 entries, roff[nf] = R)
__global__ void k_fpart(const int64_t *__restrict__ roff, int64_t nf, int64_t n_tiles, int64_t *__restrict__ tile_p) {
    const int64_t t = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (t > n_tiles) return;
    const int64_t v = t * FC_TILE;
    int64_t lo = 0, hi = nf;                                      // (nf: nothing at or above v before the end)
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        if (roff[mid] < v) lo = mid + 1; else hi = mid;
    }
    tile_p[t] = lo;
}

__device__ __forceinline__ uint32_t fc_hash(unsigned long long k) {
    k ^= k >> 33; k *= 0xff51afd7ed558ccdULL;
    k ^= k >> 33; k *= 0xc4ceb9fe1a85ec53ULL;
    return static_cast<uint32_t>(k >> 32);
}

__global__ void __launch_bounds__(FC_THREADS) k_fchip(FChipArgs g) {
    extern __shared__ __align__(16) unsigned char fc_smem[];
    unsigned long long *s_key = reinterpret_cast<unsigned long long *>(fc_smem);          // [FC_SLOTS]
    double *s_acc = reinterpret_cast<double *>(s_key + FC_SLOTS);                          // [FC_SLOTS]
    uint32_t *relcum = reinterpret_cast<uint32_t *>(s_acc + FC_SLOTS);                     // [FC_MAX_ARCS + 1] first rank of a match
    uint16_t *s_ps = reinterpret_cast<uint16_t *>(relcum + FC_MAX_ARCS + 1);               // [FC_MAX_ARCS] first rank of the match's pair
    uint16_t *s_pr = s_ps + FC_MAX_ARCS;                                                   // [FC_MAX_ARCS] raw arcs of that pair
    uint16_t *s_mi = s_pr + FC_MAX_ARCS;                                                   // [FC_MAX_ARCS] rank -> match of the tile
    uint16_t *s_excl = s_mi + FC_MAX_ARCS;                                                 // [FC_SLOTS + 1] occupied slots before slot s
    __shared__ uint32_t s_warp[FC_THREADS / 32];
    __shared__ unsigned long long s_base;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t p0 = g.tile_p[blockIdx.x], p1 = g.tile_p[blockIdx.x + 1];
    const int64_t r0 = g.roff[p0], m0 = g.moff[p0];
    const int n = static_cast<int>(g.roff[p1] - r0), nm = static_cast<int>(g.moff[p1] - m0);   // < 2 FC_TILE arcs, nm <= n matches
    if (n == 0) return;
    for (int j = tid; j < nm; j += FC_THREADS) {
        const uint32_t pl = g.L.pl[m0 + j];
        relcum[j] = static_cast<uint32_t>(g.L.cum[m0 + j] - r0);
        s_ps[j] = static_cast<uint16_t>(g.roff[pl] - r0);
        s_pr[j] = static_cast<uint16_t>(g.raw[pl]);
    }
    if (tid == 0) relcum[nm] = static_cast<uint32_t>(n);
    for (int s = tid; s < FC_SLOTS; s += FC_THREADS) { s_key[s] = FC_EMPTY; s_acc[s] = 0.0; }
    __syncthreads();
    // rank -> match, written match by match (the matches of such sources are short): the arc loop and the way out both
    // find their match, hence their pair, with one load instead of a binary search
    for (int j = tid; j < nm; j += FC_THREADS) {
        const uint32_t e = relcum[j + 1];
        for (uint32_t r = relcum[j]; r < e; ++r) s_mi[r] = static_cast<uint16_t>(j);
    }
    __syncthreads();

    // ---- every raw arc of the tile: compose, find or claim its slot, add its weight.  (Two ranks per thread with the loads
    // of both in flight lost to this loop, 54.8 -> 63.5 ms on `dups`: 44 registers, or 32 and spills.)
    const unsigned long long ab_mask = (1ull << g.shift_t) - 1ull;
    for (int r = tid; r < n; r += FC_THREADS) {
        const int j = s_mi[r];
        const uint4 rec = g.L.rec[m0 + j];
        const uint32_t rr = static_cast<uint32_t>(r) - relcum[j];
        const uint32_t i1 = rr / rec.w, i2 = rr - i1 * rec.w;
        const uint4 e1 = __ldg(g.A.arcs + rec.x + i1), e2 = __ldg(g.B.arcs + rec.y + i2);      // {tgt, outer, weight, inner}
        const unsigned long long key = ((((static_cast<unsigned long long>(e1.x) << g.q2_bits) | e2.x) << g.shift_t) |
                                        (static_cast<unsigned long long>(e1.y) << g.bits_b) | e2.y);
        const double w = static_cast<double>(__uint_as_float(e1.z) * __uint_as_float(e2.z));    // (the product in fp32, as everywhere)
        const uint32_t start = 2u * s_ps[j], size = 2u * s_pr[j];
        uint32_t s = start + static_cast<uint32_t>((static_cast<unsigned long long>(fc_hash(key)) * size) >> 32);
        while (true) {
            unsigned long long k = s_key[s];
            if (k == FC_EMPTY) k = atomicCAS(&s_key[s], FC_EMPTY, key);
            if (k == FC_EMPTY || k == key) break;
            if (++s == start + size) s = start;
        }
        atomicAdd(&s_acc[s], w);
    }
    __syncthreads();

    // ---- number the occupied slots (slot order = pair order).  A warp owns FC_CHUNK x 32 consecutive slots and takes them
    // 32 at a time (neighbouring lanes, neighbouring slots: no bank conflict, and the way out writes neighbouring arcs).
    const int w0 = warp * (FC_CHUNK * 32);
    uint32_t mine = 0;
#pragma unroll
    for (int u = 0; u < FC_CHUNK; ++u) mine += __popc(__ballot_sync(0xffffffffu, s_key[w0 + u * 32 + lane] != FC_EMPTY));
    if (lane == 0) s_warp[warp] = mine;
    __syncthreads();
    uint32_t before = 0, total = 0;
#pragma unroll
    for (int wv = 0; wv < FC_THREADS / 32; ++wv) { if (wv < warp) before += s_warp[wv]; total += s_warp[wv]; }
    if (tid == 0) s_base = total ? atomicAdd(g.cursor, static_cast<unsigned long long>(total)) : 0ull;
#pragma unroll
    for (int u = 0; u < FC_CHUNK; ++u) {
        const uint32_t bal = __ballot_sync(0xffffffffu, s_key[w0 + u * 32 + lane] != FC_EMPTY);
        s_excl[w0 + u * 32 + lane] = static_cast<uint16_t>(before + __popc(bal & ((1u << lane) - 1u)));
        before += __popc(bal);
    }
    if (tid == FC_THREADS - 1) s_excl[FC_SLOTS] = static_cast<uint16_t>(total);
    __syncthreads();
    const int64_t base = static_cast<int64_t>(s_base);

    // ---- the merged arcs leave, with their pair and their target key
    const unsigned long long q2_mask = (1ull << g.q2_bits) - 1ull;
#pragma unroll 1
    for (int u = 0; u < FC_CHUNK; ++u) {
        const int s = w0 + u * 32 + lane;
        if ((s >> 1) >= n) break;                                  // (uniform per warp but for the last round: nothing behind the tile's arcs)
        const unsigned long long key = s_key[s];
        if (key == FC_EMPTY) continue;
        const int64_t q = base + s_excl[s];
        const unsigned long long tk = key >> g.shift_t;
        g.msrc[q] = g.L.pl[m0 + s_mi[s >> 1]];                     // (rank s / 2 lies in the ranks of the pair that owns slot s)
        g.mab[q] = static_cast<uint32_t>(key & ab_mask);
        g.mw[q] = static_cast<float>(s_acc[s]);
        g.mkey[q] = g.table_key ? (tk >> g.q2_bits) * g.nq2 + (tk & q2_mask) : tk;
    }
    for (int j = tid; j < nm; j += FC_THREADS) {
        if (relcum[j] != s_ps[j]) continue;                        // not the first match of its pair
        const uint32_t start = 2u * s_ps[j], end = start + 2u * s_pr[j];
        const uint32_t pl = g.L.pl[m0 + j];
        g.cnt[pl] = s_excl[end] - s_excl[start];
        g.base[pl] = base + s_excl[start];
    }
}

// Class S on a table level: the ids of the merged arcs' targets (as k_resolve_keys) and the arcs straight to their final
// place behind the pair's offset (as k_place_grouped), in one kernel: the target column is written once and never read.
template <bool DENSE>
__global__ void __launch_bounds__(CT_THREADS)
k_resolve_place(const unsigned long long *__restrict__ keys, const uint32_t *__restrict__ msrc, const uint32_t *__restrict__ mab,
                const float *__restrict__ mw, int64_t n, const int64_t *__restrict__ mbase, const int64_t *__restrict__ foff,
                int64_t arc_base, int64_t f_lo, const uint32_t *__restrict__ sel, int bits_b, uint32_t *dense, uint4 *table,
                uint64_t cap, uint64_t nq2, unsigned long long *n_states, int2 *pair, int32_t *__restrict__ o_src,
                int32_t *__restrict__ o_il, int32_t *__restrict__ o_ol, int32_t *__restrict__ o_tgt, float *__restrict__ o_w) {
    __shared__ uint32_t s_warp[CT_THREADS / 32];
    __shared__ unsigned long long s_base;
    const int64_t j = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    const bool valid = j < n;
    const unsigned long long key = valid ? keys[j] : 0ull;
    const unsigned long long q1 = key / nq2;
    const uint32_t id = block_find_or_insert<DENSE, CT_THREADS>(key, valid, make_int2(static_cast<int>(q1), static_cast<int>(key - q1 * nq2)),
                                                                dense, table, cap, n_states, pair, s_warp, &s_base);
    if (!valid) return;
    const uint32_t p = msrc[j], ab = mab[j];
    const int64_t q = arc_base + foff[p] + (j - mbase[p]);
    o_src[q] = static_cast<int>(f_lo + (sel ? sel[p] : p));
    o_tgt[q] = static_cast<int32_t>(id);
    o_il[q] = static_cast<int>(ab >> bits_b);
    o_ol[q] = static_cast<int>(ab & ((1u << bits_b) - 1u));
    o_w[q] = mw[j];
}

__global__ void k_place_grouped(const uint32_t *__restrict__ mab, const int32_t *__restrict__ mtgt, const uint32_t *__restrict__ msrc,
                                const float *__restrict__ mw, int64_t n_merged, const int64_t *__restrict__ mstart,
                                const int64_t *__restrict__ foff, int64_t arc_base, int64_t f_lo,
                                const uint32_t *__restrict__ sel, int bits_b, int32_t *__restrict__ o_src,
                                int32_t *__restrict__ o_il, int32_t *__restrict__ o_ol, int32_t *__restrict__ o_tgt,
                                float *__restrict__ o_w, int64_t n0 = 0, int64_t n1 = 0, const uint32_t *__restrict__ rank = nullptr) {
    int64_t j = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (j >= n_merged) return;
    const uint32_t p = msrc[j], ab = mab[j];
    const int64_t q = arc_base + foff[p] + (j - mstart[p]);
    o_src[q] = static_cast<int>(f_lo + (sel ? sel[p] : p));
    int64_t t = mtgt[j];
    if (rank && t >= n0 && t < n1) t = n0 + rank[t - n0];        // deterministic ids
    o_tgt[q] = static_cast<int32_t>(t);
    o_il[q] = static_cast<int>(ab >> bits_b);
    o_ol[q] = static_cast<int>(ab & ((1u << bits_b) - 1u));
    o_w[q] = mw[j];
}

// ------------------------------------------------------------------------------------------ merge (reduce by key)
__global__ void k_heads(const uint4 *__restrict__ rec, int64_t n, uint8_t *__restrict__ head) {
    int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint8_t h = 1;
    if (i > 0) {
        uint4 r = rec[i], p = rec[i - 1];
        h = (r.x != p.x) || (r.y != p.y) || (r.z != p.z);
    }
    head[i] = h;
}

// Segment id of record i = hidx[i] + head[i] - 1.  Weights of a segment are summed as a shuffle tree inside each warp
// (fp32, depth 5); the per-warp pieces of a segment are combined with one DOUBLE atomicAdd per (warp, segment), so that a
// segment of millions of equal arcs (9e6 in tests) still lands within rtol 1e-5 of the fp64 sum; k_reduce_finish rounds once.
__global__ void __launch_bounds__(CT_THREADS)
k_reduce(const uint4 *__restrict__ rec, const uint8_t *__restrict__ head, const int64_t *__restrict__ hidx, int64_t n,
         unsigned long long *__restrict__ mkey, uint32_t *__restrict__ msrc, double *__restrict__ macc) {
    int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    int64_t seg = -1 - lane;                                   // distinct sentinels for out-of-range lanes
    float w = 0.f;
    if (i < n) {
        uint4 r = rec[i];
        uint8_t h = head[i];
        seg = hidx[i] + h - 1;
        w = __uint_as_float(r.w);
        if (h) {
            mkey[seg] = (static_cast<unsigned long long>(r.y) << 32) | r.x;
            msrc[seg] = r.z;
        }
    }
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        float t = __shfl_down_sync(0xffffffffu, w, d);
        int64_t s = __shfl_down_sync(0xffffffffu, seg, d);
        if (lane + d < 32 && s == seg) w += t;
    }
    int64_t sp = __shfl_up_sync(0xffffffffu, seg, 1);
    if (i < n && (lane == 0 || sp != seg)) atomicAdd(&macc[seg], static_cast<double>(w));
}
__global__ void k_reduce_finish(const double *__restrict__ macc, int64_t n, float *__restrict__ mw) {
    const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i < n) mw[i] = static_cast<float>(macc[i]);
}

// mstart[p] = first merged arc whose pair index >= p  (p = 0..nf)
__global__ void k_mstart(const uint32_t *__restrict__ msrc, int64_t n_merged, int64_t nf, int64_t *__restrict__ mstart) {
    int64_t p = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (p > nf) return;
    int64_t lo = 0, hi = n_merged;
    while (lo < hi) {
        int64_t mid = (lo + hi) >> 1;
        if (msrc[mid] < static_cast<uint32_t>(p)) lo = mid + 1; else hi = mid;
    }
    mstart[p] = lo;
}

__global__ void k_final_counts(const int64_t *__restrict__ rawU, const int64_t *__restrict__ mstartS,
                               const int64_t *__restrict__ mstartG, const int64_t *__restrict__ cntS, int64_t nf,
                               int64_t *__restrict__ fc) {
    int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i < nf) fc[i] = rawU[i] + (mstartS ? mstartS[i + 1] - mstartS[i] : 0) + (mstartG ? mstartG[i + 1] - mstartG[i] : 0) +
                        (cntS ? cntS[i] : 0);
}

__global__ void k_place_merged(const unsigned long long *__restrict__ mkey, const uint32_t *__restrict__ msrc,
                               const float *__restrict__ mw, int64_t n_merged, const int64_t *__restrict__ mstart,
                               const int64_t *__restrict__ foff, int64_t arc_base, int64_t f_lo,
                               const uint32_t *__restrict__ sel, int shift_t, int bits_b, int32_t *__restrict__ o_src, int32_t *__restrict__ o_il, int32_t *__restrict__ o_ol,
                               int32_t *__restrict__ o_tgt, float *__restrict__ o_w) {
    int64_t j = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (j >= n_merged) return;
    uint32_t p = msrc[j];
    unsigned long long k = mkey[j];
    int64_t q = arc_base + foff[p] + (j - mstart[p]);
    o_src[q] = static_cast<int>(f_lo + (sel ? sel[p] : p));
    o_tgt[q] = static_cast<int>(k >> shift_t);
    o_il[q] = static_cast<int>((k & ((1ull << shift_t) - 1)) >> bits_b);
    o_ol[q] = static_cast<int>(k & ((1ull << bits_b) - 1));
    o_w[q] = mw[j];
}

// ------------------------------------------------------------------------------------------ assembly
// Accept list (ascending ids with q1 in F1 and q2 in F2) in two passes over the pair table: pass 1 counts
// accepting states per 2048-state tile; after a scan of the tile counts, pass 2 recomputes the flags of the tiles that have
// any and compacts each in order.  Expanded flags: ones before the last frontier, zeros after it, a kernel for the frontier.
constexpr int AS_THREADS = 256;
constexpr int AS_ITEMS = 8;
constexpr int AS_TILE = AS_THREADS * AS_ITEMS;

__device__ __forceinline__ uint32_t is_accept(int2 p, const uint32_t *acc1, const uint32_t *acc2) {
    // F1 is small (1 % of Q1 in the BASELINE configs): the second bitmap is only read for the pairs that pass the first
    if (!((__ldg(acc1 + (p.x >> 5)) >> (p.x & 31)) & 1u)) return 0u;
    return (__ldg(acc2 + (p.y >> 5)) >> (p.y & 31)) & 1u;
}

// expanded[i] for the LAST frontier [lo, hi): 1 iff it was expanded whole (mode 1) or the pair lies below the cut (mode 2).
// (Every state before it is expanded, every state after it is not: two memsets.)
__global__ void k_expanded_last(const int2 *__restrict__ pair, int64_t lo, int64_t hi, int mode, uint64_t nq2, uint64_t cut,
                                uint8_t *__restrict__ expanded) {
    const int64_t i = lo + static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= hi) return;
    uint8_t e = mode == 1;
    if (mode == 2) {
        const int2 p = pair[i];
        e = (static_cast<uint64_t>(static_cast<uint32_t>(p.x)) * nq2 + static_cast<uint32_t>(p.y)) < cut;
    }
    expanded[i] = e;
}

// accepting states per 2048-state tile
__global__ void __launch_bounds__(AS_THREADS)
k_assemble_count(const int2 *__restrict__ pair, int64_t n, const uint32_t *__restrict__ acc1,
                 const uint32_t *__restrict__ acc2, uint32_t *__restrict__ tile_count) {
    __shared__ uint32_t s_cnt;
    if (threadIdx.x == 0) s_cnt = 0;
    __syncthreads();
    const int64_t base = static_cast<int64_t>(blockIdx.x) * AS_TILE;
    int2 p[AS_ITEMS];
#pragma unroll
    for (int r = 0; r < AS_ITEMS; ++r) {                      // all loads of the thread in flight together
        const int64_t i = base + r * AS_THREADS + threadIdx.x;
        p[r] = i < n ? __ldcs(pair + i) : make_int2(-1, -1);
    }
    uint32_t cnt = 0;
#pragma unroll
    for (int r = 0; r < AS_ITEMS; ++r)
        if (p[r].x >= 0) cnt += is_accept(p[r], acc1, acc2);
    cnt = __reduce_add_sync(0xffffffffu, cnt);
    if ((threadIdx.x & 31) == 0 && cnt) atomicAdd(&s_cnt, cnt);
    __syncthreads();
    if (threadIdx.x == 0) tile_count[blockIdx.x] = s_cnt;
}

__global__ void __launch_bounds__(AS_THREADS)
k_assemble_scatter(const int2 *__restrict__ pair, int64_t n, const uint32_t *__restrict__ acc1,
                   const uint32_t *__restrict__ acc2, const uint32_t *__restrict__ tile_count,
                   const int64_t *__restrict__ tile_off, int32_t *__restrict__ out) {
    if (tile_count[blockIdx.x] == 0) return;
    __shared__ uint32_t s_warp[AS_THREADS / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t base = static_cast<int64_t>(blockIdx.x) * AS_TILE;
    int64_t off = tile_off[blockIdx.x];
    for (int r = 0; r < AS_ITEMS; ++r) {                      // rows of 256 consecutive states, in order
        const int64_t i = base + r * AS_THREADS + threadIdx.x;
        const uint32_t f = (i < n) ? is_accept(pair[i], acc1, acc2) : 0u;
        const uint32_t b = __ballot_sync(0xffffffffu, f);
        if (lane == 0) s_warp[warp] = __popc(b);
        __syncthreads();
        uint32_t before = 0, total = 0;
#pragma unroll
        for (int wv = 0; wv < AS_THREADS / 32; ++wv) {
            const uint32_t c = s_warp[wv];
            if (wv < warp) before += c;
            total += c;
        }
        if (f) out[off + before + __popc(b & ((1u << lane) - 1u))] = static_cast<int32_t>(i);
        off += total;
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------ deterministic ids
// fstc_opts_t.deterministic: the states a level creates get their ids in ascending order of the pair key (the set a level
// creates does not depend on thread scheduling, only the order the threads win their slots in does).  After the level: sort
// the new keys, rank[old id - n0] = position, rewrite pair[], remap the target column of the level's arcs and the ids in
// the visited table.  Arcs of sources that went through sort + reduce are sorted again on the new ids.
__global__ void k_det_keys(const int2 *__restrict__ pair, int64_t n0, int64_t n, uint64_t nq2, uint4 *__restrict__ rec) {
    const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int2 p = pair[n0 + i];
    const uint64_t key = static_cast<uint64_t>(static_cast<uint32_t>(p.x)) * nq2 + static_cast<uint32_t>(p.y);
    rec[i] = make_uint4(static_cast<uint32_t>(key), static_cast<uint32_t>(key >> 32), 0u, static_cast<uint32_t>(i));
}
__global__ void k_det_apply(const uint4 *__restrict__ sorted, int64_t n0, int64_t n, uint64_t nq2, int2 *__restrict__ pair,
                            uint32_t *__restrict__ rank) {
    const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint4 r = sorted[i];
    const uint64_t key = (static_cast<uint64_t>(r.y) << 32) | r.x;
    const uint64_t q1 = key / nq2;
    rank[r.w] = static_cast<uint32_t>(i);
    pair[n0 + i] = make_int2(static_cast<int>(q1), static_cast<int>(key - q1 * nq2));
}
__global__ void k_det_remap(int32_t *__restrict__ tgt, int64_t n, int64_t n0, int64_t n1, const uint32_t *__restrict__ rank) {
    const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int64_t t = tgt[i];
    if (t >= n0 && t < n1) tgt[i] = static_cast<int32_t>(n0 + rank[t - n0]);
}
__global__ void k_det_table(const int2 *__restrict__ pair, int64_t n0, int64_t n, uint64_t nq2, uint32_t *__restrict__ dense,
                            uint4 *__restrict__ table, uint64_t cap) {
    const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int2 p = pair[n0 + i];
    const unsigned long long key = static_cast<uint64_t>(static_cast<uint32_t>(p.x)) * nq2 + static_cast<uint32_t>(p.y);
    if (dense) { dense[key] = static_cast<uint32_t>(n0 + i) + 1u; return; }
    uint64_t s = 2 * home_bucket(key, cap);                      // the key is in the table: walk its probe path
    while (slot_key(table[s]) != key) s = (s + 1 == cap) ? 0 : s + 1;
    reinterpret_cast<uint32_t *>(table + s)[2] = static_cast<uint32_t>(n0 + i);
}
// sort records of the merged class-F arcs with their NEW target ids: {key = tgt << shift_t | a << bits_b | b, pair index, weight}
__global__ void k_det_frec(const unsigned long long *__restrict__ mkey, const uint32_t *__restrict__ msrc, const float *__restrict__ mw,
                           int64_t n, int shift_t, int64_t n0, int64_t n1, const uint32_t *__restrict__ rank, uint4 *__restrict__ rec) {
    const int64_t j = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (j >= n) return;
    unsigned long long k = mkey[j];
    int64_t t = static_cast<int64_t>(k >> shift_t);
    if (t >= n0 && t < n1) t = n0 + rank[t - n0];
    k = (static_cast<unsigned long long>(t) << shift_t) | (k & ((1ull << shift_t) - 1));
    rec[j] = make_uint4(static_cast<uint32_t>(k), static_cast<uint32_t>(k >> 32), msrc[j], __float_as_uint(mw[j]));
}
__global__ void k_det_funpack(const uint4 *__restrict__ rec, int64_t n, unsigned long long *__restrict__ mkey, uint32_t *__restrict__ msrc,
                              float *__restrict__ mw) {
    const int64_t j = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const uint4 r = rec[j];
    mkey[j] = (static_cast<unsigned long long>(r.y) << 32) | r.x;
    msrc[j] = r.z;
    mw[j] = __uint_as_float(r.w);
}

// ------------------------------------------------------------------------------------------ dense table, ids in key order
// After k_emit<DIRECT, RES_DORD>: the entries of the dense table that hold PENDING are the states this level created.  A scan
// of the table numbers them in ascending key order (count per tile of DO_TILE entries, scan, assign) and writes pair[]; the
// arcs whose target column holds ~key get their id from the table.  The ids do not depend on thread scheduling, and the
// next level's frontier is sorted by (q1, q2): consecutive pairs share q1's arcs and the table rows of their targets, which
// is worth more than the scan costs when the table is far larger than L2 (`medium`: emit 27 -> 19 ms).
constexpr int DO_THREADS = 256, DO_ITEMS = 8, DO_TILE = DO_THREADS * DO_ITEMS;
__global__ void __launch_bounds__(DO_THREADS) k_dord_count(const uint32_t *__restrict__ dense, uint64_t n, uint32_t *__restrict__ tile_cnt) {
    __shared__ uint32_t s_cnt;
    if (threadIdx.x == 0) s_cnt = 0;
    __syncthreads();
    const uint64_t base = static_cast<uint64_t>(blockIdx.x) * DO_TILE;
    uint32_t c = 0;
#pragma unroll
    for (int r = 0; r < DO_ITEMS; ++r) {
        const uint64_t i = base + static_cast<uint64_t>(r) * DO_THREADS + threadIdx.x;
        if (i < n && __ldcs(dense + i) == PENDING_ID) ++c;
    }
    c = __reduce_add_sync(0xffffffffu, c);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(&s_cnt, c);
    __syncthreads();
    if (threadIdx.x == 0) tile_cnt[blockIdx.x] = s_cnt;
}
__global__ void __launch_bounds__(DO_THREADS) k_dord_assign(uint32_t *__restrict__ dense, uint64_t n, uint64_t nq2, const uint32_t *__restrict__ tile_cnt,
                                                             const int64_t *__restrict__ tile_off, int64_t n0, int2 *__restrict__ pair,
                                                             uint2 *__restrict__ rankdir) {
    if (tile_cnt[blockIdx.x] == 0) return;
    __shared__ uint32_t s_warp[DO_THREADS / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // a warp owns DO_ITEMS x 32 consecutive keys of the tile: all its loads in flight together, one block barrier per tile
    const uint64_t base = static_cast<uint64_t>(blockIdx.x) * DO_TILE + static_cast<uint64_t>(warp) * (DO_ITEMS * 32);
    uint32_t bal[DO_ITEMS], cnt = 0;
    uint32_t v[DO_ITEMS];
#pragma unroll
    for (int r = 0; r < DO_ITEMS; ++r) {
        const uint64_t i = base + static_cast<uint64_t>(r) * 32 + lane;
        v[r] = i < n ? dense[i] : 0u;
    }
#pragma unroll
    for (int r = 0; r < DO_ITEMS; ++r) {
        bal[r] = __ballot_sync(0xffffffffu, v[r] == PENDING_ID);
        cnt += __popc(bal[r]);
    }
    if (lane == 0) s_warp[warp] = cnt;
    __syncthreads();
    int64_t off = n0 + tile_off[blockIdx.x];
#pragma unroll
    for (int wv = 0; wv < DO_THREADS / 32; ++wv) if (wv < warp) off += s_warp[wv];
#pragma unroll
    for (int r = 0; r < DO_ITEMS; ++r) {                         // rows of 32 consecutive keys, in order
        const uint64_t i = base + static_cast<uint64_t>(r) * 32 + lane;
        // the rank directory: {which of these 32 keys were numbered now, id of the first of them}: 8 bytes per 32 keys, small
        // enough to stay in L2, so that k_dord_fix does not go back to the table (far larger than L2) for every arc
        if (lane == 0 && i < n) rankdir[i >> 5] = make_uint2(bal[r], static_cast<uint32_t>(off));
        if (bal[r] >> lane & 1u) {
            const int64_t id = off + __popc(bal[r] & ((1u << lane) - 1u));
            dense[i] = static_cast<uint32_t>(id) + 1u;
            const uint64_t q1 = i / nq2;
            pair[id] = make_int2(static_cast<int>(q1), static_cast<int>(i - q1 * nq2));
        }
        off += __popc(bal[r]);
    }
}
// tgt: the whole target column (16-byte aligned); the arcs [a0, a1) of it are completed, four per thread
__global__ void k_dord_fix(int32_t *__restrict__ tgt, int64_t a0, int64_t a1, const uint2 *__restrict__ rankdir) {
    const int64_t q = (a0 / 4 + static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x) * 4;
    if (q >= a1) return;
    auto fix = [&](int32_t t) {                                  // ~key of a state this level created: its id from the directory
        if (t >= 0) return t;
        const uint32_t key = static_cast<uint32_t>(~t);
        const uint2 d = __ldg(rankdir + (key >> 5));
        return static_cast<int32_t>(d.y + __popc(d.x & ((1u << (key & 31u)) - 1u)));
    };
    if (q >= a0 && q + 4 <= a1) {
        int4 v = __ldcs(reinterpret_cast<const int4 *>(tgt + q));
        v.x = fix(v.x); v.y = fix(v.y); v.z = fix(v.z); v.w = fix(v.w);
        __stcs(reinterpret_cast<int4 *>(tgt + q), v);
    } else {
        for (int64_t i = q < a0 ? a0 : q; i < q + 4 && i < a1; ++i) tgt[i] = fix(tgt[i]);
    }
}

// Level compaction: when rule T will clearly cut the level, only the pairs below a key limit are worked on.
__global__ void k_flag_below(const int2 *__restrict__ pair, int64_t f_lo, int64_t nf, uint64_t nq2, uint64_t key_limit,
                             uint8_t *__restrict__ flag) {
    int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= nf) return;
    int2 p = pair[f_lo + i];
    flag[i] = (static_cast<uint64_t>(static_cast<uint32_t>(p.x)) * nq2 + static_cast<uint32_t>(p.y)) < key_limit;
}
__global__ void k_compact_sel(const uint8_t *__restrict__ flag, const int64_t *__restrict__ off, int64_t nf,
                              uint32_t *__restrict__ sel) {
    int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i < nf && flag[i]) sel[off[i]] = static_cast<uint32_t>(i);
}

// several device scalars -> one contiguous block, so that the host reads them with ONE copy (a level costs a fixed
// number of host round trips; on small levels those are the whole cost)
struct ScalarPtrs { const int64_t *p[10]; };
__global__ void k_gather_scalars(ScalarPtrs s, int n, int64_t *__restrict__ out) {
    if (static_cast<int>(threadIdx.x) < n) out[threadIdx.x] = s.p[threadIdx.x] ? *s.p[threadIdx.x] : 0;
}

inline unsigned nblk(int64_t n, int threads = CT_THREADS) { return static_cast<unsigned>(ceil_div(n > 0 ? n : 1, threads)); }

// ------------------------------------------------------------------------------------------ host side
struct StageTimer {
    Ctx &c;
    bool on;
    struct Span { int stage; cudaEvent_t a, b; };
    std::vector<Span> spans;
    StageTimer(Ctx &ctx, bool enable) : c(ctx), on(enable) {}
    ~StageTimer() { for (auto &s : spans) { cudaEventDestroy(s.a); cudaEventDestroy(s.b); } }
    int begin(int stage) {
        if (!on) return -1;
        Span s; s.stage = stage;
        cudaEventCreate(&s.a); cudaEventCreate(&s.b);
        cudaEventRecord(s.a, c.stream);
        spans.push_back(s);
        return static_cast<int>(spans.size()) - 1;
    }
    void end(int h) { if (h >= 0) cudaEventRecord(spans[h].b, c.stream); }
    void collect(double *ms) {
        for (auto &s : spans) {
            float t = 0.f;
            if (cudaEventElapsedTime(&t, s.a, s.b) == cudaSuccess) ms[s.stage] += t;
        }
    }
};

// Total memory of a device, asked once per process: cudaMemGetInfo goes to the driver and was seen to take 10-50 ms at times
// (the source of the 60-150 ms step-time outliers of round 1, and of +25 ms per call when it came back in round 2).
size_t device_total_bytes(int dev) {
    static std::mutex mu;
    static size_t total_of[64] = {};
    std::lock_guard<std::mutex> lk(mu);
    size_t &slot = total_of[dev & 63];
    if (slot == 0) {
        size_t f = 0, t = 0;
        (void)cudaMemGetInfo(&f, &t);
        slot = t > 0 ? t : size_t(64) << 30;
    }
    return slot;
}

struct Composer {
    Ctx &c;
    const fstc_packed_t &m1, &m2;
    fstc_opts_t o;
    fstc_stats_t st;
    StageTimer tm;
    uint64_t nq2;
    // growing outputs
    DBuf<int2> pair; int64_t pair_cap = 0;
    DBuf<int32_t> a_src, a_il, a_ol, a_tgt; DBuf<float> a_w; int64_t arc_cap = 0;
    // what the kernels index with ABSOLUTE arc positions: the arrays above, or (host spill without a device copy) the
    // arrays of the current level shifted back by the level's first position
    int32_t *o_src = nullptr, *o_il = nullptr, *o_ol = nullptr, *o_tgt = nullptr; float *o_w = nullptr;
    // ---- host spill (fstc_spill_t): finished levels go to pinned host memory on a second stream while the next level runs
    const fstc_spill_t *sp = nullptr;
    bool spill_only = false;             // keep_device = 0: the arcs of a level leave the device when their copy is done
    cudaStream_t side = nullptr;
    cudaEvent_t ev_main = nullptr;
    struct LevelArcs { DBuf<int32_t> src, il, ol, tgt; DBuf<float> w; cudaEvent_t done = nullptr; };
    std::vector<LevelArcs> inflight;     // level arrays whose copy may still run
    LevelArcs cur;                       // spill_only: the arrays of the level being expanded
    int64_t spilled_states = 0;
    bool cols_spilled = false;           // src / ilabel / olabel / weight of the current level already went out (after its emit kernel)
    struct Retired { DBuf<int2> block; cudaEvent_t done = nullptr; };
    std::vector<Retired> retired;        // pair blocks replaced by a larger one while a copy to the host may still read them

    ~Composer() {
        if (side) {                      // on every way out: no copy may still read a buffer the members are about to release
            (void)cudaStreamSynchronize(side);
            for (auto &l : inflight) if (l.done) (void)cudaEventDestroy(l.done);
            for (auto &l : retired) if (l.done) (void)cudaEventDestroy(l.done);
            if (ev_main) (void)cudaEventDestroy(ev_main);
            (void)cudaStreamDestroy(side);
        }
    }
    void spill_begin() {
        sp = o.spill;
        if (!sp) return;
        const fstc_host_result_t *hr = sp->host;
        if (!hr || !hr->pair || !hr->src || !hr->ilabel || !hr->olabel || !hr->tgt || !hr->weight || sp->arc_capacity < 0 || sp->state_capacity < 1)
            fail(FSTC_ERR_ARG, "spill: host arrays missing");
        spill_only = sp->keep_device == 0;
        FSTC_CUDA(cudaStreamCreateWithFlags(&side, cudaStreamNonBlocking));
        FSTC_CUDA(cudaEventCreateWithFlags(&ev_main, cudaEventDisableTiming));
    }
    void spill_reap(bool all) {          // level arrays whose copy is complete go back to the workspace
        for (size_t i = 0; i < retired.size();) {
            if (all) FSTC_CUDA(cudaEventSynchronize(retired[i].done));
            if (all || cudaEventQuery(retired[i].done) == cudaSuccess) {
                (void)cudaEventDestroy(retired[i].done);
                retired.erase(retired.begin() + i);
            } else { (void)cudaGetLastError(); ++i; }
        }
        for (size_t i = 0; i < inflight.size();) {
            if (all) FSTC_CUDA(cudaEventSynchronize(inflight[i].done));
            if (all || cudaEventQuery(inflight[i].done) == cudaSuccess) {
                (void)cudaEventDestroy(inflight[i].done);
                inflight.erase(inflight.begin() + i);
            } else { (void)cudaGetLastError(); ++i; }
        }
    }
    // spill_only: device arrays for the `r` arcs (at most) of the level that starts at arc position `base`
    void spill_level_arrays(int64_t base, int64_t r) {
        spill_reap(false);
        const int64_t pad = base & 3, n = r + pad + 4;           // keeps the kernels' 16-byte stores aligned
        cur = LevelArcs();
        cur.src.alloc(c, n); cur.il.alloc(c, n); cur.ol.alloc(c, n); cur.tgt.alloc(c, n); cur.w.alloc(c, n);
        o_src = cur.src.p + pad - base; o_il = cur.il.p + pad - base; o_ol = cur.ol.p + pad - base;
        o_tgt = cur.tgt.p + pad - base; o_w = cur.w.p + pad - base;
    }
    // four of the five columns of arcs [a0, a1) are final as soon as the emit kernel that writes them straight to their
    // place is done (the target column waits for the resolve): they cross PCIe under the resolve
    void spill_columns_early(int64_t a0, int64_t a1) {
        if (!sp || a1 <= a0) return;
        if (a1 > sp->arc_capacity)
            fail(FSTC_ERR_CAPACITY, "spill: the result (%lld arcs so far) outgrows the host arrays", static_cast<long long>(a1));
        FSTC_CUDA(cudaEventRecord(ev_main, c.stream));
        FSTC_CUDA(cudaStreamWaitEvent(side, ev_main, 0));
        const fstc_host_result_t *hr = sp->host;
        const size_t nb = sizeof(int32_t) * static_cast<size_t>(a1 - a0);
        FSTC_CUDA(cudaMemcpyAsync(hr->src + a0, o_src + a0, nb, cudaMemcpyDeviceToHost, side));
        FSTC_CUDA(cudaMemcpyAsync(hr->ilabel + a0, o_il + a0, nb, cudaMemcpyDeviceToHost, side));
        FSTC_CUDA(cudaMemcpyAsync(hr->olabel + a0, o_ol + a0, nb, cudaMemcpyDeviceToHost, side));
        FSTC_CUDA(cudaMemcpyAsync(hr->weight + a0, o_w + a0, nb, cudaMemcpyDeviceToHost, side));
        cols_spilled = true;
    }
    // the level is placed: arcs [a0, a1) and states [s0, s1) are final
    void spill_level(int64_t a0, int64_t a1, int64_t s1) {
        if (!sp) return;
        if (a1 > sp->arc_capacity || s1 > sp->state_capacity)
            fail(FSTC_ERR_CAPACITY, "spill: the result (%lld arcs, %lld states so far) outgrows the host arrays", static_cast<long long>(a1), static_cast<long long>(s1));
        FSTC_CUDA(cudaEventRecord(ev_main, c.stream));
        FSTC_CUDA(cudaStreamWaitEvent(side, ev_main, 0));
        const fstc_host_result_t *hr = sp->host;
        const size_t nb = sizeof(int32_t) * static_cast<size_t>(a1 - a0);
        if (a1 > a0) {
            if (!cols_spilled) {
                FSTC_CUDA(cudaMemcpyAsync(hr->src + a0, o_src + a0, nb, cudaMemcpyDeviceToHost, side));
                FSTC_CUDA(cudaMemcpyAsync(hr->ilabel + a0, o_il + a0, nb, cudaMemcpyDeviceToHost, side));
                FSTC_CUDA(cudaMemcpyAsync(hr->olabel + a0, o_ol + a0, nb, cudaMemcpyDeviceToHost, side));
                FSTC_CUDA(cudaMemcpyAsync(hr->weight + a0, o_w + a0, nb, cudaMemcpyDeviceToHost, side));
            }
            FSTC_CUDA(cudaMemcpyAsync(hr->tgt + a0, o_tgt + a0, nb, cudaMemcpyDeviceToHost, side));
        }
        cols_spilled = false;
        if (s1 > spilled_states)
            FSTC_CUDA(cudaMemcpyAsync(hr->pair + 2 * spilled_states, pair.p + spilled_states, sizeof(int2) * static_cast<size_t>(s1 - spilled_states),
                                      cudaMemcpyDeviceToHost, side));
        st.spill_bytes += 5 * static_cast<int64_t>(nb) + 8 * (s1 - spilled_states);
        spilled_states = s1;
        if (spill_only) {
            st.spill_bytes_saved += 5 * static_cast<int64_t>(nb);
            FSTC_CUDA(cudaEventCreateWithFlags(&cur.done, cudaEventDisableTiming));
            FSTC_CUDA(cudaEventRecord(cur.done, side));
            inflight.push_back(std::move(cur));
            cur = LevelArcs();
        }
    }
    int64_t n_arcs = 0, n_states = 0;
    // visited table
    DBuf<uint4> table; uint64_t cap = 0;
    DBuf<uint32_t> dense; bool use_dense = false;   // the dense |Q1||Q2| table instead of the hash table (small products)
    uint64_t n_pairs_all = 0;
    DBuf<unsigned long long> d_counters;   // [0] n_states, [1] seg visited, [2] match arcs, [3] n_selected, [4..259] hist

    // test / debugging knobs from the environment, read once per call
    int knob_resolve_bits = -1;          // FSTC_RESOLVE_BITS: hash bits of the partitioned resolve
    bool knob_no_group = false;          // FSTC_NO_GROUP_MERGE: class G off
    double knob_limit_margin = 1.5;      // FSTC_KEY_LIMIT_MARGIN: the guessed key limit of a level that will be cut
    int64_t knob_chunk_arcs = 0;         // FSTC_CHUNK_ARCS: raw arcs a level may hold before it is expanded in chunks
    bool knob_no_dord = false;           // FSTC_NO_KEY_ORDER: dense-table levels never number their states in key order
    bool knob_no_chip = false;           // FSTC_NO_CHIP_MERGE: class S off (small duplicate-prone sources go through sort + reduce)

    Composer(Ctx &ctx, const fstc_packed_t &a, const fstc_packed_t &b, const fstc_opts_t &opts)
        : c(ctx), m1(a), m2(b), o(opts), tm(ctx, opts.profile != 0), nq2(static_cast<uint64_t>(b.n_states)) {
        std::memset(&st, 0, sizeof st);
        if (const char *e = getenv("FSTC_RESOLVE_BITS")) knob_resolve_bits = atoi(e);
        knob_no_group = getenv("FSTC_NO_GROUP_MERGE") != nullptr;
        if (const char *e = getenv("FSTC_KEY_LIMIT_MARGIN")) knob_limit_margin = atof(e);
        if (const char *e = getenv("FSTC_CHUNK_ARCS")) knob_chunk_arcs = atoll(e);
        knob_no_dord = getenv("FSTC_NO_KEY_ORDER") != nullptr;
        knob_no_chip = getenv("FSTC_NO_CHIP_MERGE") != nullptr;
    }

    // Growable outputs and table.  `need` is what the coming launch requires; `want` >= need is a look-ahead
    // (next level's predicted size) so that big arrays are not reallocated + copied / rehashed level after level.
    template <typename F>
    void grow_to(int64_t need, int64_t want, F &&grow) {
        if (want > need) {
            try { grow(want); return; }
            catch (const Error &e) { if (e.code != FSTC_ERR_OOM) throw; }
        }
        grow(need);
    }

    void ensure_pairs(int64_t need, int64_t want = 0) {
        if (need <= pair_cap) return;
        grow_to(need, std::max(want, pair_cap * 2), [&](int64_t nc) {
            DBuf<int2> np(c, nc, true);
            const int64_t keep = std::max(n_states, n_states_live);  // (states appended inside the level, external resolve)
            if (keep > 0 && pair.p)
                FSTC_CUDA(cudaMemcpyAsync(np.p, pair.p, sizeof(int2) * keep, cudaMemcpyDeviceToDevice, c.stream));
            if (side && pair.p) {                                 // a copy to the host may still read the old block: it goes later
                Retired r;
                FSTC_CUDA(cudaEventCreateWithFlags(&r.done, cudaEventDisableTiming));
                FSTC_CUDA(cudaEventRecord(r.done, side));
                r.block = std::move(pair);
                retired.push_back(std::move(r));
            }
            pair = std::move(np);
            pair_cap = nc;
        });
        if (n_states > 0) st.n_grow += 1;
    }

    void ensure_arcs(int64_t need, int64_t want = 0) {
        if (spill_only) return;                                  // level arrays instead (spill_level_arrays)
        if (need <= arc_cap) return;
        if (side) FSTC_CUDA(cudaStreamSynchronize(side));         // a copy to the host may still read the old arrays
        int h = tm.begin(FSTC_T_ASSEMBLE);
        grow_to(need, std::max(want, arc_cap + arc_cap / 2), [&](int64_t nc) {
            nc = (nc + 3) & ~int64_t(3);
            DBuf<int32_t> n_src(c, nc, true), n_il(c, nc, true), n_ol(c, nc, true), n_tgt(c, nc, true);
            DBuf<float> n_w(c, nc, true);
            if (n_arcs > 0) {
                const size_t b = sizeof(int32_t) * n_arcs;
                FSTC_CUDA(cudaMemcpyAsync(n_src.p, a_src.p, b, cudaMemcpyDeviceToDevice, c.stream));
                FSTC_CUDA(cudaMemcpyAsync(n_il.p, a_il.p, b, cudaMemcpyDeviceToDevice, c.stream));
                FSTC_CUDA(cudaMemcpyAsync(n_ol.p, a_ol.p, b, cudaMemcpyDeviceToDevice, c.stream));
                FSTC_CUDA(cudaMemcpyAsync(n_tgt.p, a_tgt.p, b, cudaMemcpyDeviceToDevice, c.stream));
                FSTC_CUDA(cudaMemcpyAsync(n_w.p, a_w.p, b, cudaMemcpyDeviceToDevice, c.stream));
            }
            a_src = std::move(n_src); a_il = std::move(n_il); a_ol = std::move(n_ol); a_tgt = std::move(n_tgt);
            a_w = std::move(n_w);
            arc_cap = nc;
            o_src = a_src.p; o_il = a_il.p; o_ol = a_ol.p; o_tgt = a_tgt.p; o_w = a_w.p;
        });
        if (n_arcs > 0) st.n_grow += 1;
        tm.end(h);
    }

    static uint64_t slots_for(int64_t states) { return static_cast<uint64_t>(states) * 100 / FSTC_TABLE_LOAD_PCT + 64; }

    // table able to hold `bound` states at load <= FSTC_TABLE_LOAD_PCT %
    void ensure_table(int64_t bound, int64_t want_states = 0) {
        if (use_dense) {                                     // one entry per pair: never grows; rebuilt only after it was dropped
            if (dense.p) return;
            int h = tm.begin(FSTC_T_TABLE);
            dense.alloc(c, static_cast<int64_t>(n_pairs_all));
            FSTC_CUDA(cudaMemsetAsync(dense.p, 0, sizeof(uint32_t) * n_pairs_all, c.stream));
            if (n_states > 0) {
                tb_dense_insert_ids<<<nblk(n_states), CT_THREADS, 0, c.stream>>>(pair.p, n_states, nq2, dense.p);
                FSTC_LAUNCH_CHECK();
                c.n_launch += 1;
            }
            tm.end(h);
            return;
        }
        const uint64_t need = slots_for(bound);
        if (need <= cap) return;
        int h = tm.begin(FSTC_T_TABLE);
        grow_to(static_cast<int64_t>(need), static_cast<int64_t>(slots_for(std::max(bound, want_states))), [&](int64_t slots) {
            uint64_t nc = (std::max<uint64_t>(static_cast<uint64_t>(slots), 4096) + 1) & ~uint64_t(1);   // whole buckets
            DBuf<uint4> nt(c, static_cast<int64_t>(nc));
            FSTC_CUDA(cudaMemsetAsync(nt.p, 0xFF, sizeof(uint4) * nc, c.stream));
            if (n_states > 0) {
                tb_insert_ids<<<nblk(n_states), CT_THREADS, 0, c.stream>>>(pair.p, n_states, nq2, nt.p, nc);
                FSTC_LAUNCH_CHECK();
                c.n_launch += 1;
            }
            table = std::move(nt);
            if (cap) st.n_rehash += 1;
            cap = nc;
        });
        tm.end(h);
    }

    // ---- FSTC_RESOLVE_EXTERNAL: the caller's callback resolves target keys to global ids (one composition sharded by key
    // ownership); pair[] holds the states this rank owns, in the order the callback announced them
    bool external = false;
    int cur_level = 0, ext_next_call = 0;
    int32_t ext_more = 0;
    int ext_q2_bits = 0;
    void ext_call(const ResolveJob &j, int call) {
        DBuf<int32_t> ids(c, j.n_records);
        c.sync();                                                // the keys are complete; the callback works on its own stream
        const int32_t *new_pairs = nullptr;
        int64_t n_new = 0;
        int32_t more = 0;
        const int rc = o.resolve_cb(o.resolve_ctx, cur_level, call, ext_q2_bits, j.keys, j.n_records, ids.p, &new_pairs, &n_new, &more);
        if (rc != 0) fail(FSTC_ERR_CALLBACK, "resolve_cb returned %d (level %d, call %d)", rc, cur_level, call);
        if (n_new < 0 || (n_new > 0 && !new_pairs)) fail(FSTC_ERR_CALLBACK, "resolve_cb: bad new_pairs");
        if (n_new > 0) {
            if (n_states_live + n_new >= 0x7FFFFFFFll) fail(FSTC_ERR_CAPACITY, "more than 2^31-1 states");
            ensure_pairs(n_states_live + n_new);
            FSTC_CUDA(cudaMemcpyAsync(pair.p + n_states_live, new_pairs, sizeof(int2) * static_cast<size_t>(n_new), cudaMemcpyDeviceToDevice, c.stream));
            c.sync();
            n_states_live += n_new;
        }
        if (call == 2) ext_more = more;
        resolve_apply_ids(c, j, reinterpret_cast<const uint32_t *>(ids.p));
    }
    // the ids of a list of target keys: the partitioned resolve, or the caller's (always calls 0, 1, 2 of a level in order)
    void run_resolve(const ResolveJob &j, int call) {
        if (external) {
            for (; ext_next_call < call; ++ext_next_call) { ResolveJob e{}; ext_call(e, ext_next_call); }
            ext_call(j, call);
            ext_next_call = call + 1;
        } else resolve_partitioned(c, j);
        st.n_resolve += 1;
        st.n_resolved_arcs += j.n_records;
    }
    void ext_finish_level() {
        for (; ext_next_call < 3; ++ext_next_call) { ResolveJob e{}; ext_call(e, ext_next_call); }
        ext_next_call = 0;
    }

    // partitioned = true: the level's target ids come from resolve_partitioned (no visited table)
    bool partitioned = false;
    bool dense_ordered = false;          // this level numbers its new states in key order (RES_DORD; dense table levels without merges)
    // numbers the PENDING entries of the dense table in ascending key order (ids from n0), completes the target column of the
    // arcs [a0, a1); returns the number of states after it
    int64_t dense_number_pending(int64_t n0, int64_t a0, int64_t a1) {
        const int h = tm.begin(FSTC_T_TABLE);
        const int64_t tiles = ceil_div(static_cast<int64_t>(n_pairs_all), DO_TILE);
        DBuf<uint32_t> tile_cnt(c, tiles);
        DBuf<int64_t> tile_off(c, tiles + 1);
        k_dord_count<<<static_cast<unsigned>(tiles), DO_THREADS, 0, c.stream>>>(dense.p, n_pairs_all, tile_cnt.p);
        FSTC_LAUNCH_CHECK();
        exclusive_scan<uint32_t>(c, tile_cnt.p, tiles, tile_off.p);
        const int64_t n_new = read_scalar(c, tile_off.p + tiles);
        if (n0 + n_new > pair_cap) fail(FSTC_ERR_INTERNAL, "dense_number_pending: %lld new states exceed the reserved pair table", static_cast<long long>(n_new));
        DBuf<uint2> rankdir(c, ceil_div(static_cast<int64_t>(n_pairs_all), 32));
        k_dord_assign<<<static_cast<unsigned>(tiles), DO_THREADS, 0, c.stream>>>(dense.p, n_pairs_all, nq2, tile_cnt.p, tile_off.p, n0, pair.p,
                                                                                 rankdir.p);
        FSTC_LAUNCH_CHECK();
        if (a1 > a0) {
            k_dord_fix<<<nblk(a1 / 4 - a0 / 4 + 1), CT_THREADS, 0, c.stream>>>(o_tgt, a0, a1, rankdir.p);
            FSTC_LAUNCH_CHECK();
        }
        const unsigned long long ns = static_cast<unsigned long long>(n0 + n_new);
        FSTC_CUDA(cudaMemcpyAsync(d_counters.p, &ns, sizeof ns, cudaMemcpyHostToDevice, c.stream));
        c.n_launch += 3;
        tm.end(h);
        c.sync();
        return n0 + n_new;
    }
    int key_bits = 0;
    const uint32_t *cur_sel = nullptr;  // compaction of the level being expanded (null: none)
    int64_t n_states_live = 1;         // states created so far, including those of the launches of this level

    void launch_emit(int mode, const MatchList &L, int64_t n_matches, int64_t R, int64_t pos_base, int64_t f_lo,
                     const int64_t *foff, const int64_t *roff, int64_t arc_base, uint4 *sortrec, int shift_t, int bits_b) {
        if (R <= 0) return;                                      // (external resolve: ext_finish_level makes the empty calls)
        const int64_t tile0 = (pos_base / EM_TILE) * EM_TILE;
        const int64_t n_tiles = ceil_div(pos_base + R - tile0, EM_TILE);
        DBuf<int64_t> tile_m(c, n_tiles + 1);
        const int h_emit = tm.begin(FSTC_T_EMIT);
        k_partition<<<nblk(n_tiles + 1), CT_THREADS, 0, c.stream>>>(L.cum, n_matches, R, pos_base, n_tiles, tile_m.p);
        FSTC_LAUNCH_CHECK();
        EmitArgs g;
        g.A = view_of(m1); g.B = view_of(m2);
        g.L = L; g.n_matches = n_matches; g.R = R; g.pos_base = pos_base; g.f_lo = f_lo; g.sel = cur_sel;
        g.foff = foff; g.roff = roff; g.arc_base = arc_base; g.nq2 = nq2;
        g.table = table.p; g.cap = cap; g.dense = dense.p; g.n_states = d_counters.p; g.pair = pair.p;
        g.o_src = o_src; g.o_il = o_il; g.o_ol = o_ol; g.o_tgt = o_tgt; g.o_w = o_w;
        g.sortrec = sortrec; g.shift_t = shift_t; g.bits_b = bits_b; g.tile_m = tile_m.p;
        g.keys = nullptr; g.posout = nullptr;
        g.q2_bits = bits_for(nq2 > 1 ? nq2 - 1 : 1);
        const unsigned grid = static_cast<unsigned>(n_tiles);
        DBuf<unsigned long long> keys;
        DBuf<uint32_t> posout;
        if (partitioned) {
            keys.alloc(c, R + 2);
            g.keys = keys.p;
            if (mode == EMIT_INDIRECT) { posout.alloc(c, R); g.posout = posout.p; }
            if (mode == EMIT_DIRECT) k_emit<EMIT_DIRECT, RES_KEYS><<<grid, EM_THREADS, 0, c.stream>>>(g);
            else if (mode == EMIT_INDIRECT) k_emit<EMIT_INDIRECT, RES_KEYS><<<grid, EM_THREADS, 0, c.stream>>>(g);
            else k_emit<EMIT_SORTREC, RES_KEYS><<<grid, EM_THREADS, 0, c.stream>>>(g);
        } else if (use_dense) {
            if (mode == EMIT_DIRECT && dense_ordered) k_emit<EMIT_DIRECT, RES_DORD><<<grid, EM_THREADS, 0, c.stream>>>(g);
            else if (mode == EMIT_DIRECT) k_emit<EMIT_DIRECT, RES_DENSE><<<grid, EM_THREADS, 0, c.stream>>>(g);
            else if (mode == EMIT_INDIRECT) k_emit<EMIT_INDIRECT, RES_DENSE><<<grid, EM_THREADS, 0, c.stream>>>(g);
            else k_emit<EMIT_SORTREC, RES_DENSE><<<grid, EM_THREADS, 0, c.stream>>>(g);
        } else {
            if (mode == EMIT_DIRECT) k_emit<EMIT_DIRECT, RES_HASH><<<grid, EM_THREADS, 0, c.stream>>>(g);
            else if (mode == EMIT_INDIRECT) k_emit<EMIT_INDIRECT, RES_HASH><<<grid, EM_THREADS, 0, c.stream>>>(g);
            else k_emit<EMIT_SORTREC, RES_HASH><<<grid, EM_THREADS, 0, c.stream>>>(g);
        }
        FSTC_LAUNCH_CHECK();
        tm.end(h_emit);
        c.n_launch += 2;
        st.n_emit_launches += 1;
        if (sp && mode == EMIT_DIRECT && partitioned && !o.deterministic) spill_columns_early(pos_base, pos_base + R);
        if (partitioned) {
            ResolveJob j;
            j.keys = keys.p; j.n_records = R; j.q2_bits = g.q2_bits;
            j.key_bits = g.q2_bits + bits_for(static_cast<uint64_t>(m1.n_states > 1 ? m1.n_states - 1 : 1));
            j.pair = pair.p; j.n_states_before = n_states_live;
            j.n_states = d_counters.p;
            j.mode = mode == EMIT_DIRECT ? 0 : (mode == EMIT_INDIRECT ? 1 : 2);
            j.pos = posout.p;
            j.o_tgt = mode == EMIT_SORTREC ? nullptr : o_tgt + (mode == EMIT_DIRECT ? pos_base : arc_base);
            j.sortrec = mode == EMIT_SORTREC ? sortrec : nullptr;
            j.shift_t = shift_t;
            j.force_bits = knob_resolve_bits;
            j.stats = &st;
            j.profile = o.profile != 0;
            run_resolve(j, mode == EMIT_SORTREC ? 0 : 2);
        }
    }

    // deterministic ids (see k_det_keys): the states [n0, n1) the level created, renumbered by ascending key; the target
    // column of the arcs [a0, a1) already written, and the table, follow.  Returns the rank array (old id - n0 -> position).
    DBuf<uint32_t> det_renumber(int64_t n0, int64_t n1, int64_t a0, int64_t a1) {
        const int64_t n = n1 - n0;
        DBuf<uint32_t> rank(c, n);
        if (n <= 0) return rank;
        const int h = tm.begin(FSTC_T_TABLE);
        DBuf<uint4> ra(c, n), rb(c, n);
        k_det_keys<<<nblk(n), CT_THREADS, 0, c.stream>>>(pair.p, n0, n, nq2, ra.p);
        FSTC_LAUNCH_CHECK();
        uint4 *sorted = radix_sort_records(c, ra.p, rb.p, n, make_sort_passes(key_bits, 0));
        k_det_apply<<<nblk(n), CT_THREADS, 0, c.stream>>>(sorted, n0, n, nq2, pair.p, rank.p);
        FSTC_LAUNCH_CHECK();
        if (a1 > a0) {
            k_det_remap<<<nblk(a1 - a0), CT_THREADS, 0, c.stream>>>(o_tgt + a0, a1 - a0, n0, n1, rank.p);
            FSTC_LAUNCH_CHECK();
        }
        if (!partitioned && (dense.p || table.p)) {
            k_det_table<<<nblk(n), CT_THREADS, 0, c.stream>>>(pair.p, n0, n, nq2, dense.p, table.p, cap);
            FSTC_LAUNCH_CHECK();
        }
        c.n_launch += 4;
        tm.end(h);
        c.sync();                                                // ra / rb go out of scope
        return rank;
    }

    fstc_result_t *run();
};

fstc_result_t *Composer::run() {
    if (m1.side != 1 || m2.side != 2) fail(FSTC_ERR_ARG, "operands must be packed with side 1 (left) and side 2 (right)");
    if (m1.n_inner != m2.n_inner)
        fail(FSTC_ERR_ARG, "inner alphabets differ: |Γ| = %d vs %d (PAPER.md:45)", m1.n_inner, m2.n_inner);
    if (o.merge_mode < 0 || o.merge_mode > 2 || o.max_levels < 0 || o.max_raw_arcs < 0 || o.resolve_mode < 0 || o.resolve_mode > 4)
        fail(FSTC_ERR_ARG, "bad options");
    external = o.resolve_mode == FSTC_RESOLVE_EXTERNAL;
    if (external && (!o.resolve_cb || o.max_raw_arcs != 0 || o.deterministic || o.spill))
        fail(FSTC_ERR_ARG, "FSTC_RESOLVE_EXTERNAL needs resolve_cb and takes no max_raw_arcs, deterministic or spill");
    ext_q2_bits = bits_for(nq2 > 1 ? nq2 - 1 : 1);
    const int bits_a = bits_for(m1.n_outer > 0 ? m1.n_outer - 1 : 0), bits_b = bits_for(m2.n_outer > 0 ? m2.n_outer - 1 : 0);
    const int shift_t = bits_a + bits_b;
    const uint64_t n_pairs_total = static_cast<uint64_t>(m1.n_states) * nq2;
    // can any pair of this run hold duplicate arcs (N10)?  if not, the whole class-F machinery is skipped
    const bool has_F = o.merge_mode == FSTC_MERGE_SORT_ALL ||
                       (o.merge_mode == FSTC_MERGE_AUTO &&
                        (((m1.any_flags & FLAG_D) && (m2.any_flags & FLAG_D)) || (m1.any_flags & FLAG_X) || (m2.any_flags & FLAG_X)));
    key_bits = bits_for(n_pairs_total - 1);
    // class G (merge by construction) replaces sort + reduce for the pairs it suits; FSTC_MERGE_SORT_ALL keeps the sort
    const bool has_G = has_F && o.merge_mode == FSTC_MERGE_AUTO && !knob_no_group;
    // class S (merge on chip, k_fchip) takes the class-F pairs of at most FC_PAIR_CAP raw arcs when (r1, r2, a, b) fits 63 bits;
    // not with deterministic ids (the order inside a source follows the hash slots) nor with the external resolve
    const bool has_S = has_F && o.merge_mode == FSTC_MERGE_AUTO && !knob_no_chip && !o.deterministic && !external && shift_t <= 32 &&
                       bits_for(nq2 > 1 ? nq2 - 1 : 1) + bits_for(static_cast<uint64_t>(m1.n_states > 1 ? m1.n_states - 1 : 1)) + shift_t <= 63;
    n_pairs_all = n_pairs_total;
    use_dense = o.resolve_mode != FSTC_RESOLVE_HASH && n_pairs_total <= DENSE_MAX_PAIRS;

    // FSTC_ALLOC_TRACE: host clock at the main points of the run (debug knob; finds host-side stalls)
    static const bool host_trace = getenv("FSTC_ALLOC_TRACE") != nullptr;
    timespec ht0;
    clock_gettime(CLOCK_MONOTONIC, &ht0);
    double ht_last = 0.0;
    auto hostmark = [&](const char *what, int level) {
        if (!host_trace) return;
        timespec t;
        clock_gettime(CLOCK_MONOTONIC, &t);
        const double ms = (t.tv_sec - ht0.tv_sec) * 1e3 + (t.tv_nsec - ht0.tv_nsec) * 1e-6;
        if (ms - ht_last > 3.0) fprintf(stderr, "[fstc host] level %d %-12s at %8.2f ms (+%.2f)\n", level, what, ms, ms - ht_last);
        ht_last = ms;
    };
    struct EventPair {                                           // released on every way out, errors included
        cudaEvent_t a = nullptr, b = nullptr;
        ~EventPair() { if (a) cudaEventDestroy(a); if (b) cudaEventDestroy(b); }
    } evp;
    FSTC_CUDA(cudaEventCreate(&evp.a));
    FSTC_CUDA(cudaEventCreate(&evp.b));
    const cudaEvent_t ev0 = evp.a, ev1 = evp.b;
    FSTC_CUDA(cudaEventRecord(ev0, c.stream));

    d_counters.alloc(c, 4 + 256);
    FSTC_CUDA(cudaMemsetAsync(d_counters.p, 0, sizeof(unsigned long long) * (4 + 256), c.stream));
    spill_begin();

    // ---- init (Alg. 2 lines 1-3): state 0 = (s1, s2)
    ensure_pairs(std::max<int64_t>(o.state_capacity_hint, 1024));
    ensure_arcs(std::max<int64_t>(o.arc_capacity_hint, 1024));
    {
        int2 s = make_int2(m1.start, m2.start);
        FSTC_CUDA(cudaMemcpyAsync(pair.p, &s, sizeof s, cudaMemcpyHostToDevice, c.stream));
        unsigned long long one = 1;
        FSTC_CUDA(cudaMemcpyAsync(d_counters.p, &one, sizeof one, cudaMemcpyHostToDevice, c.stream));
        n_states = 1;
        if (external) {                                          // no table; the start pair is local state 0 of its owner only
            partitioned = true;
            if (!o.owns_start) n_states = 0;
            n_states_live = n_states;
        } else ensure_table(std::max<int64_t>(o.state_capacity_hint, 1));
    }

    int64_t f_lo = 0, f_hi = n_states, cum_raw = 0;
    int last_mode = 1;           // how the last frontier [f_lo, f_hi) was treated: 0 not expanded, 1 all, 2 cut
    uint64_t cut_key = 0;
    int64_t last_lo = 0, last_hi = 1;
    double last_fan = 0.0;      // raw arcs per expanded pair of the previous level
    int lvl = 0;
    MachineView A = view_of(m1), B = view_of(m2);

    // A level whose raw arcs do not fit the workspace in one piece (the paper fills a pre-allocated edge
    // buffer pair by pair) is expanded in CHUNKS: id ranges of the frontier of about chunk_limit raw arcs, one
    // after the other, each with its own count / emit / resolve / merge (duplicates share a source, so merging stays
    // correct); the states every chunk creates are appended and all of them form the next frontier.  Only
    // when no budget cut falls into the level (rule T orders a cut level by key, not by id).
    int64_t chunk_limit = knob_chunk_arcs;
    if (chunk_limit <= 0)   // ~52 bytes of resolve buffers and 20 of output per raw arc; and the partitioned resolve indexes records with 32 bits
        chunk_limit = std::min<int64_t>(int64_t(3) << 30, static_cast<int64_t>(0.5 * static_cast<double>(device_total_bytes(m1.device)) / 72.0));
    int64_t level_lo = 0, level_end = -1, chunk_pairs = 0;      // level_end >= 0: the level [level_lo, level_end) goes chunk by chunk

    for (;;) {
        const int64_t nf_all = f_hi - f_lo;                      // the frontier (or the current chunk of it)
        cur_level = lvl;
        if (external) {
            // the search ends when NO rank created a state; a rank without a frontier still takes part in the exchange
            if (lvl > 0 && !ext_more) break;
            if (o.max_levels > 0 && lvl == o.max_levels) { st.truncated = 1; last_lo = f_lo; last_hi = f_hi; last_mode = 0; break; }
            if (nf_all == 0) {
                ext_finish_level();
                if (lvl < FSTC_MAX_LEVEL_STATS) { st.level_frontier[lvl] = 0; st.level_raw[lvl] = 0; st.level_new_states[lvl] = n_states_live - n_states; }
                n_states = n_states_live; f_lo = f_hi; f_hi = n_states; st.n_levels = lvl + 1;
                ++lvl;
                continue;
            }
        } else if (nf_all == 0) break;
        int64_t nf = nf_all;                                     // the pairs of it this level works on (see `sel`)
        last_lo = level_end >= 0 ? level_lo : f_lo; last_hi = level_end >= 0 ? level_end : f_hi;
        if (level_end < 0 && o.max_levels > 0 && lvl == o.max_levels) { st.truncated = 1; last_mode = 0; break; }
        last_mode = 1;

        // ---- count
        int64_t RU = 0, RF = 0, MU = 0, MF = 0, RS = 0, MS = 0;
        DBuf<int64_t> rawU, rawF, rawG, gwork, rawS;
        DBuf<uint32_t> nmU, nmF, nmG, nmS;
        DBuf<int64_t> roffU, roffF, moffU, moffF, roffG, moffG, woff, roffS, moffS;
        int64_t RG = 0, MG = 0, WG = 0;                          // class G: raw arcs, pairs, group pairs of the level
        DBuf<uint32_t> sel;                                      // compacted level: frontier index of working pair i
        DBuf<int64_t> level_totals(c, 10);
        auto scan_level = [&](int64_t *n_sel_out) {             // offsets + totals of the level, one synchronisation
            exclusive_scan2(c, rawU.p, nmU.p, nf, roffU.p, moffU.p);
            if (has_F) exclusive_scan2(c, rawF.p, nmF.p, nf, roffF.p, moffF.p);
            if (has_G) {
                exclusive_scan2(c, rawG.p, nmG.p, nf, roffG.p, moffG.p);
                exclusive_scan<int64_t>(c, gwork.p, nf, woff.p);
            }
            if (has_S) exclusive_scan2(c, rawS.p, nmS.p, nf, roffS.p, moffS.p);
            ScalarPtrs sp{{roffU.p + nf, moffU.p + nf, has_F ? roffF.p + nf : nullptr, has_F ? moffF.p + nf : nullptr,
                           has_G ? roffG.p + nf : nullptr, has_G ? moffG.p + nf : nullptr, has_G ? woff.p + nf : nullptr,
                           reinterpret_cast<const int64_t *>(d_counters.p + 3),
                           has_S ? roffS.p + nf : nullptr, has_S ? moffS.p + nf : nullptr}};
            k_gather_scalars<<<1, 32, 0, c.stream>>>(sp, 10, level_totals.p);
            FSTC_LAUNCH_CHECK();
            int64_t t[10];
            FSTC_CUDA(cudaMemcpyAsync(t, level_totals.p, sizeof t, cudaMemcpyDeviceToHost, c.stream));
            c.sync();
            RU = t[0]; MU = t[1]; RF = t[2]; MF = t[3]; RG = t[4]; MG = t[5]; WG = t[6]; RS = t[8]; MS = t[9];
            if (n_sel_out) *n_sel_out = t[7];
        };
        // A level that will clearly be cut by the budget (predicted from the previous level's fan-out) is counted
        // only below a key limit: rule T expands a key-ordered prefix, so pairs far above the cut never matter.
        // Exact: if the counted part does not exceed the budget the limit is raised and the level counted again.
        uint64_t key_limit = ~0ull;
        if (level_end < 0 && o.max_raw_arcs > 0 && nf > 100000 && last_fan > 0) {
            const double remaining = static_cast<double>(o.max_raw_arcs - cum_raw);
            const double predicted = static_cast<double>(nf) * last_fan;
            if (predicted > 4.0 * remaining) {
                const double margin = knob_limit_margin;             // test knob: a margin < 1 forces the widening path
                key_limit = static_cast<uint64_t>(static_cast<double>(n_pairs_total) * (margin * remaining / predicted)) + 1;
            }
        }
        int h;
        while (true) {
            h = tm.begin(FSTC_T_COUNT);
            nf = nf_all;
            sel.release();
            if (key_limit < n_pairs_total) {                     // work on the pairs below the limit only
                DBuf<uint8_t> flag(c, nf_all);
                DBuf<int64_t> off(c, nf_all + 1);
                k_flag_below<<<nblk(nf_all), CT_THREADS, 0, c.stream>>>(pair.p, f_lo, nf_all, nq2, key_limit, flag.p);
                FSTC_LAUNCH_CHECK();
                exclusive_scan<uint8_t>(c, flag.p, nf_all, off.p);
                nf = read_scalar(c, off.p + nf_all);
                sel.alloc(c, nf);
                k_compact_sel<<<nblk(nf_all), CT_THREADS, 0, c.stream>>>(flag.p, off.p, nf_all, sel.p);
                FSTC_LAUNCH_CHECK();
                c.n_launch += 2;
                c.sync();                                        // flag / off go out of scope
                if (nf == 0) {                                   // nothing below the limit: widen
                    tm.end(h);
                    key_limit = key_limit > n_pairs_total / 4 ? ~0ull : key_limit * 4;
                    continue;
                }
            }
            rawU.alloc(c, nf); nmU.alloc(c, nf); roffU.alloc(c, nf + 1); moffU.alloc(c, nf + 1);
            if (has_F) { rawF.alloc(c, nf); nmF.alloc(c, nf); roffF.alloc(c, nf + 1); moffF.alloc(c, nf + 1); }
            if (has_G) {
                rawG.alloc(c, nf); gwork.alloc(c, nf); nmG.alloc(c, nf);
                roffG.alloc(c, nf + 1); moffG.alloc(c, nf + 1); woff.alloc(c, nf + 1);
            }
            if (has_S) { rawS.alloc(c, nf); nmS.alloc(c, nf); roffS.alloc(c, nf + 1); moffS.alloc(c, nf + 1); }
            k_count<<<nblk(nf), CT_THREADS, 0, c.stream>>>(A, B, pair.p, f_lo, nf, sel.p, o.merge_mode, nq2, key_limit, rawU.p, rawF.p,
                                                           nmU.p, nmF.p, rawG.p, gwork.p, nmG.p, rawS.p, nmS.p);
            FSTC_LAUNCH_CHECK();
            c.n_launch += 1;
            tm.end(h);
            // ---- scan + budget
            h = tm.begin(FSTC_T_SCAN);
            scan_level(nullptr);
            if (key_limit >= n_pairs_total || cum_raw + RU + RF + RG + RS > o.max_raw_arcs) break;
            tm.end(h);
            key_limit = key_limit > n_pairs_total / 4 ? ~0ull : key_limit * 4;     // the cut lies higher: widen
        }
        bool stop_after = false;
        int64_t n_sel = nf;
        if (o.max_raw_arcs > 0 && cum_raw + RU + RF + RG + RS > o.max_raw_arcs) {
            // rule T: find the key of the first pair (ascending key order) whose arcs no longer fit
            const uint64_t remaining = static_cast<uint64_t>(o.max_raw_arcs - cum_raw);
            uint64_t prefix = 0, before = 0;
            const int top = ((key_bits + 7) / 8) * 8;
            for (int shift = top - 8; shift >= 0; shift -= 8) {
                FSTC_CUDA(cudaMemsetAsync(d_counters.p + 4, 0, sizeof(unsigned long long) * 256, c.stream));
                k_cut_hist<<<std::min<unsigned>(nblk(nf), 8u * c.n_sm), CT_THREADS, 0, c.stream>>>(pair.p, f_lo, nf, sel.p, nq2, rawU.p, rawF.p, rawG.p, rawS.p, prefix, shift,
                                                                  d_counters.p + 4);
                FSTC_LAUNCH_CHECK();
                c.n_launch += 1;
                unsigned long long hist[256];
                FSTC_CUDA(cudaMemcpyAsync(hist, d_counters.p + 4, sizeof hist, cudaMemcpyDeviceToHost, c.stream));
                c.sync();
                int d = 0;
                for (; d < 256; ++d) {
                    if (before + hist[d] > remaining) break;
                    before += hist[d];
                }
                if (d == 256) fail(FSTC_ERR_INTERNAL, "budget cut not found (the level's counts changed under the search)");
                prefix = (prefix << 8) | static_cast<uint64_t>(d);
            }
            cut_key = prefix;
            FSTC_CUDA(cudaMemsetAsync(d_counters.p + 3, 0, sizeof(unsigned long long), c.stream));
            k_apply_cut<<<nblk(nf), CT_THREADS, 0, c.stream>>>(pair.p, f_lo, nf, sel.p, nq2, cut_key, rawU.p, rawF.p, nmU.p, nmF.p,
                                                               rawG.p, gwork.p, nmG.p, rawS.p, nmS.p,
                                                               d_counters.p + 3);
            FSTC_LAUNCH_CHECK();
            c.n_launch += 1;
            scan_level(&n_sel);
            st.truncated = 1;
            stop_after = true;
            last_mode = 2;
        }
        tm.end(h);

        hostmark("count+scan", lvl);
        const int64_t R = RU + RF + RG + RS;
        if (!stop_after && !external && nf_all > 1) {
            if (level_end < 0 && R > chunk_limit) {              // too big for one piece: count again, on the first chunk
                level_lo = f_lo; level_end = f_hi;
                chunk_pairs = std::max<int64_t>(1, static_cast<int64_t>(static_cast<double>(nf_all) * (0.9 * static_cast<double>(chunk_limit) / static_cast<double>(R))));
                f_hi = f_lo + chunk_pairs;
                continue;
            }
            if (level_end >= 0 && R > 2 * chunk_limit) { f_hi = f_lo + nf_all / 2; continue; }   // a dense id range: halve the chunk
        }
        cur_sel = sel.p;
        // ---- capacities for this level
        const uint64_t remaining_pairs = n_pairs_total - static_cast<uint64_t>(n_states);
        const int64_t new_bound = external ? 0 : static_cast<int64_t>(std::min<uint64_t>(static_cast<uint64_t>(R), remaining_pairs));
        if (n_states + new_bound >= 0x7FFFFFFFll) fail(FSTC_ERR_CAPACITY, "more than 2^31-1 states");
        // ---- how this level resolves its target ids, decided per level from measured unit costs: the
        // visited table pays a random DRAM read per arc and a random write-back + publish per NEW state (and a rebuild
        // if it was dropped or must grow); the partitioned resolve pays streaming passes per arc and per existing state.
        const int rkey_bits = bits_for(nq2 > 1 ? nq2 - 1 : 1) + bits_for(static_cast<uint64_t>(m1.n_states > 1 ? m1.n_states - 1 : 1));
        auto prefer_partitioned = [&](int64_t r, int64_t bound, int64_t states_now, uint64_t slots_ready) {
            if (o.resolve_mode == FSTC_RESOLVE_TABLE || o.resolve_mode == FSTC_RESOLVE_HASH) return false;
            if (rkey_bits + bits_for(static_cast<uint64_t>(states_now + bound)) > 64) return false;  // state records: key << id_bits | id
            if (!resolve_can_take(r, states_now)) {                  // u32 record indices, at most 2^20 bins
                if (o.resolve_mode == FSTC_RESOLVE_PARTITIONED)
                    fail(FSTC_ERR_CAPACITY, "a level of %lld arcs and %lld states is beyond the partitioned resolve", static_cast<long long>(r), static_cast<long long>(states_now));
                return false;
            }
            if (o.resolve_mode == FSTC_RESOLVE_PARTITIONED) return true;
            const uint64_t slots = use_dense ? n_pairs_all : slots_for(states_now + bound);
            const uint64_t table_bytes = slots * (use_dense ? sizeof(uint32_t) : sizeof(uint4));
            if (r < RESOLVE_MIN_ARCS || table_bytes <= RESOLVE_TABLE_BYTES) return false;            // small, or the table lives in L2
            double t_table = COST_PROBE_PS * r + COST_INSERT_PS * bound;
            if (slots > slots_ready) t_table += COST_INSERT_PS * 0.6 * states_now + COST_STREAM_PS_PER_BYTE * table_bytes;
            const double t_part = COST_PART_ARC_PS * r + COST_PART_STATE_PS * states_now + 1e9;      // + 1 ms of launches
            // a clear win only: leaving the table also costs the next table level a rebuild, and ids in bin order cost
            // the next level's count / match their cache locality
            return t_part < 0.6 * t_table;
        };
        {
            const bool want = external || prefer_partitioned(R, new_bound, n_states, use_dense ? (dense.p ? n_pairs_all : 0) : cap);
            if (want && !partitioned) { table = DBuf<uint4>(); cap = 0; dense = DBuf<uint32_t>(); }    // the table is dropped; ensure_table rebuilds it from pair[]
            partitioned = want;
        }
        // look-ahead: if the search goes on, the next level is about (new states) x (arcs per expanded pair)
        int64_t next_R = 0, next_S = 0;
        const bool must_grow = n_states + new_bound > pair_cap || (!partitioned && (use_dense ? dense.p == nullptr : slots_for(n_states + new_bound) > cap)) ||
                               (!spill_only && n_arcs + R > arc_cap);
        if (must_grow && !stop_after && n_sel > 0 && R > 0) {
            const double fan = static_cast<double>(R) / static_cast<double>(n_sel);
            double pr = static_cast<double>(new_bound) * fan;
            if (o.max_raw_arcs > 0) pr = std::min(pr, static_cast<double>(o.max_raw_arcs - cum_raw - R));
            // what is free for us: the device's memory minus what our pool has handed out.  (cudaMemGetInfo would say it
            // exactly, but it goes to the driver and was seen to take 10-50 ms at times: the device size is read once.)
            const size_t device_bytes = device_total_bytes(m1.device) - device_total_bytes(m1.device) / 16;   // leave 1/16 to others on the device
            uint64_t pool_used = 0;
            (void)cudaMemPoolGetAttribute(device_pool(), cudaMemPoolAttrUsedMemCurrent, &pool_used);
            const size_t free_b = device_bytes > pool_used ? device_bytes - pool_used : 0;
            pr = std::min(pr, 16.0 * static_cast<double>(n_arcs + R));           // never more than 16x what is needed now
            const double ps = std::min(pr, static_cast<double>(remaining_pairs - static_cast<uint64_t>(new_bound)));
            // 20 B per arc; per state 8 B + a table slot at the target load; at most 40 % of what is free
            const double bytes = 20.0 * pr + (partitioned ? 8.0 : 8.0 + 1600.0 / FSTC_TABLE_LOAD_PCT) * ps;
            const double scale = std::min(1.0, 0.4 * static_cast<double>(free_b) / std::max(bytes, 1.0));
            next_R = pr > 0 ? static_cast<int64_t>(pr * scale) : 0;
            next_S = ps > 0 ? static_cast<int64_t>(ps * scale) : 0;
            if (n_states + new_bound + next_S >= 0x7FFFFFFFll) next_S = 0;
        }
        hostmark("lookahead", lvl);
        ensure_pairs(n_states + new_bound, n_states + new_bound + next_S);
        if (!partitioned) {
            // no look-ahead for the table if the next level is expected to leave it for the partitioned resolve anyway
            const bool next_partitioned = next_R > 0 && prefer_partitioned(next_R, next_S, n_states + new_bound,
                                                                           slots_for(n_states + new_bound + next_S));
            ensure_table(n_states + new_bound, next_partitioned ? 0 : n_states + new_bound + next_S);
        }
        ensure_arcs(n_arcs + R, n_arcs + R + next_R);
        if (spill_only) spill_level_arrays(n_arcs, R);
        n_states_live = n_states;
        hostmark("ensure", lvl);

        // ---- match work-lists
        MatchList LU{nullptr, nullptr, nullptr}, LF{nullptr, nullptr, nullptr};
        DBuf<int64_t> cumU(c, MU + 1), cumF(c, MF + 1);
        DBuf<uint4> recU(c, MU), recF(c, MF);
        DBuf<uint32_t> plU(c, MU), plF(c, MF);
        LU = MatchList{cumU.p, recU.p, plU.p};
        LF = MatchList{cumF.p, recF.p, plF.p};
        DBuf<int64_t> cumS(c, MS + 1);
        DBuf<uint4> recS(c, MS);
        DBuf<uint32_t> plS(c, MS);
        MatchList LS{cumS.p, recS.p, plS.p};
        // one walk writes two classes' lists: U and F, or — the usual case of a level with class S, which has no class F —
        // U and S; only a level with all three walks a second time
        const bool s_with_u = MS > 0 && MF == 0;
        if (MU + MF > 0 || s_with_u) {
            h = tm.begin(FSTC_T_MATCH);
            if (s_with_u)
                k_match<<<nblk(nf), CT_THREADS, 0, c.stream>>>(A, B, pair.p, f_lo, nf, sel.p, nmU.p, nmS.p, moffU.p, moffS.p, roffU.p,
                                                               roffS.p, LU, LS, d_counters.p + 1);
            else
                k_match<<<nblk(nf), CT_THREADS, 0, c.stream>>>(A, B, pair.p, f_lo, nf, sel.p, nmU.p, nmF.p, moffU.p, moffF.p, roffU.p,
                                                               roffF.p, LU, LF, d_counters.p + 1);
            FSTC_LAUNCH_CHECK();
            c.n_launch += 1;
            tm.end(h);
        }
        if (MS > 0 && !s_with_u) {                               // class S in the place of class U
            h = tm.begin(FSTC_T_MATCH);
            k_match<<<nblk(nf), CT_THREADS, 0, c.stream>>>(A, B, pair.p, f_lo, nf, sel.p, nmS.p, nullptr, moffS.p, nullptr, roffS.p,
                                                           nullptr, LS, LS, d_counters.p + 1);
            FSTC_LAUNCH_CHECK();
            c.n_launch += 1;
            tm.end(h);
        }

        hostmark("match", lvl);
        const int64_t arc_base = n_arcs;
        if (RF == 0 && RG == 0 && RS == 0) {
            // no source of this level can hold duplicates: arcs go straight to their final place
            // a big level on a dense table that is far larger than L2: ids in key order (see k_dord_count)
            dense_ordered = use_dense && !partitioned && !external && !knob_no_dord && RU >= DORD_MIN_ARCS &&
                            n_pairs_all * sizeof(uint32_t) > RESOLVE_TABLE_BYTES;
            launch_emit(EMIT_DIRECT, LU, MU, RU, arc_base, f_lo, nullptr, nullptr, 0, nullptr, 0, 0);
            n_arcs += RU;
            if (dense_ordered) {
                n_states_live = dense_number_pending(n_states, arc_base, n_arcs);
                dense_ordered = false;
            } else if (o.deterministic) det_renumber(n_states, static_cast<int64_t>(read_scalar(c, d_counters.p)), arc_base, n_arcs);
        } else {
            if (shift_t > 32) fail(FSTC_ERR_CAPACITY, "bits(|Σ|)+bits(|Δ|) = %d > 32: merge key does not fit 64 bits", shift_t);
            // ---- class F: sort + reduce
            int64_t M = 0;
            DBuf<uint4> sa, sb;
            DBuf<unsigned long long> mkey;
            DBuf<uint32_t> msrc;
            DBuf<float> mw;
            DBuf<int64_t> mstartS;
            if (RF > 0) {
                sa.alloc(c, RF); sb.alloc(c, RF);
                launch_emit(EMIT_SORTREC, LF, MF, RF, 0, f_lo, nullptr, nullptr, 0, sa.p, shift_t, bits_b);
                // target ids are now known: n_states bounds them
                const int64_t ns_now = external ? 0x7FFFFFFFll : static_cast<int64_t>(read_scalar(c, d_counters.p));   // external: global ids
                if (!external) n_states_live = ns_now;
                const int tgt_bits = bits_for(static_cast<uint64_t>(ns_now - 1));
                h = tm.begin(FSTC_T_SORT);
                uint4 *sorted = radix_sort_records(c, sa.p, sb.p, RF, make_sort_passes(shift_t + tgt_bits, bits_for(static_cast<uint64_t>(nf - 1))));
                tm.end(h);
                h = tm.begin(FSTC_T_REDUCE);
                DBuf<uint8_t> head(c, RF);
                DBuf<int64_t> hidx(c, RF + 1);
                k_heads<<<nblk(RF), CT_THREADS, 0, c.stream>>>(sorted, RF, head.p);
                FSTC_LAUNCH_CHECK();
                exclusive_scan<uint8_t>(c, head.p, RF, hidx.p);
                M = read_scalar(c, hidx.p + RF);
                mkey.alloc(c, M); msrc.alloc(c, M); mw.alloc(c, M);
                DBuf<double> macc(c, M);
                FSTC_CUDA(cudaMemsetAsync(macc.p, 0, sizeof(double) * M, c.stream));
                k_reduce<<<nblk(RF), CT_THREADS, 0, c.stream>>>(sorted, head.p, hidx.p, RF, mkey.p, msrc.p, macc.p);
                FSTC_LAUNCH_CHECK();
                k_reduce_finish<<<nblk(M), CT_THREADS, 0, c.stream>>>(macc.p, M, mw.p);
                FSTC_LAUNCH_CHECK();
                mstartS.alloc(c, nf + 1);
                k_mstart<<<nblk(nf + 1), CT_THREADS, 0, c.stream>>>(msrc.p, M, nf, mstartS.p);
                FSTC_LAUNCH_CHECK();
                c.n_launch += 3;
                tm.end(h);
                c.sync();
                sa.release(); sb.release();
            }
            // ---- class S: merge on chip (k_fchip); the merged arcs then take class G's way to their ids and places
            int64_t MSm = 0;
            DBuf<uint32_t> ssrc, sab;
            DBuf<float> sw;
            DBuf<int32_t> stgt;
            DBuf<int64_t> scnt, sbase;
            DBuf<unsigned long long> skeys;                          // target keys of the merged arcs (table level: resolved at placement)
            if (RS > 0) {
                h = tm.begin(FSTC_T_REDUCE);
                const int64_t n_tiles = ceil_div(RS, FC_TILE);
                DBuf<int64_t> tile_p(c, n_tiles + 1);
                DBuf<unsigned long long> cursor(c, 1);
                skeys.alloc(c, RS + 2);
                ssrc.alloc(c, RS); sab.alloc(c, RS); sw.alloc(c, RS);
                scnt.alloc(c, nf); sbase.alloc(c, nf);
                FSTC_CUDA(cudaMemsetAsync(cursor.p, 0, sizeof(unsigned long long), c.stream));
                FSTC_CUDA(cudaMemsetAsync(scnt.p, 0, sizeof(int64_t) * nf, c.stream));
                k_fpart<<<nblk(n_tiles + 1), CT_THREADS, 0, c.stream>>>(roffS.p, nf, n_tiles, tile_p.p);
                FSTC_LAUNCH_CHECK();
                FChipArgs fa;
                fa.A = A; fa.B = B; fa.L = LS; fa.roff = roffS.p; fa.moff = moffS.p; fa.raw = rawS.p; fa.nf = nf; fa.tile_p = tile_p.p;
                fa.shift_t = shift_t; fa.bits_b = bits_b; fa.q2_bits = bits_for(nq2 > 1 ? nq2 - 1 : 1); fa.nq2 = nq2;
                fa.table_key = partitioned ? 0 : 1;
                fa.cursor = cursor.p; fa.msrc = ssrc.p; fa.mab = sab.p; fa.mw = sw.p; fa.mkey = skeys.p; fa.cnt = scnt.p; fa.base = sbase.p;
                static const bool fc_attr = [] {                  // 88 KB of dynamic shared memory: opt in once
                    return cudaFuncSetAttribute(k_fchip, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(FC_SMEM)) == cudaSuccess;
                }();
                if (!fc_attr) fail(FSTC_ERR_CUDA, "k_fchip: %zu bytes of shared memory refused", FC_SMEM);
                k_fchip<<<static_cast<unsigned>(n_tiles), FC_THREADS, FC_SMEM, c.stream>>>(fa);
                FSTC_LAUNCH_CHECK();
                c.n_launch += 2;
                MSm = static_cast<int64_t>(read_scalar(c, cursor.p));
                tm.end(h);
                if (MSm > 0 && partitioned) {                        // target ids of the merged arcs (a table level: at placement)
                    stgt.alloc(c, MSm);
                    {
                        ResolveJob j;
                        j.keys = skeys.p; j.n_records = MSm; j.q2_bits = fa.q2_bits;
                        j.key_bits = fa.q2_bits + bits_for(static_cast<uint64_t>(m1.n_states > 1 ? m1.n_states - 1 : 1));
                        j.pair = pair.p; j.n_states_before = n_states_live; j.n_states = d_counters.p;
                        j.mode = 0; j.pos = nullptr; j.o_tgt = stgt.p; j.sortrec = nullptr; j.shift_t = 0;
                        j.force_bits = knob_resolve_bits;
                        j.stats = &st; j.profile = o.profile != 0;
                        run_resolve(j, 1);
                    }
                    n_states_live = static_cast<int64_t>(read_scalar(c, d_counters.p));
                }
                st.n_raw_onchip += RS;
                c.sync();                                            // (tile_p, cursor go out of scope)
            }
            // ---- class G: merge by construction (group products)
            int64_t MGm = 0;
            DBuf<uint32_t> gsrc, gab;
            DBuf<float> gw;
            DBuf<int32_t> gtgt;
            DBuf<int64_t> mstartG;
            DBuf<int64_t> fc, foff;                                  // final arcs per pair of the level, and their offsets
            bool g_placed = false;                                   // the class-G arcs are already in their final place (fused pass)
            if (RG > 0) {
                h = tm.begin(FSTC_T_REDUCE);
                DBuf<int64_t> cumG(c, MG + 1);
                DBuf<uint4> recG(c, MG);
                DBuf<uint32_t> plG(c, MG);
                MatchList LG{cumG.p, recG.p, plG.p};
                k_gmatch<<<nblk(nf), CT_THREADS, 0, c.stream>>>(A, B, pair.p, f_lo, nf, sel.p, nmG.p, moffG.p, woff.p, LG);
                FSTC_LAUNCH_CHECK();
                FSTC_CUDA(cudaMemcpyAsync(cumG.p + MG, woff.p + nf, sizeof(int64_t), cudaMemcpyDeviceToDevice, c.stream));
                const int64_t n_tiles = ceil_div(WG, GP_TILE);
                DBuf<int64_t> tile_m(c, n_tiles + 1), tile_off(c, n_tiles + 1);
                DBuf<uint32_t> tile_cnt(c, n_tiles);
                DBuf<uint8_t> ebits(c, n_tiles * GP_THREADS);
                DBuf<uint16_t> eprefix(c, n_tiles * GP_THREADS);
                k_partition<<<nblk(n_tiles + 1), CT_THREADS, 0, c.stream>>>(cumG.p, MG, WG, 0, n_tiles, tile_m.p);
                FSTC_LAUNCH_CHECK();
                GProdArgs g;
                g.A = A; g.B = B; g.L = LG; g.n_matches = MG; g.W = WG; g.tile_m = tile_m.p;
                g.tile_cnt = tile_cnt.p; g.tile_off = nullptr; g.ebits = ebits.p; g.eprefix = eprefix.p;
                g.msrc = nullptr; g.mab = nullptr; g.mw = nullptr; g.mkey = nullptr;
                g.dense = dense.p; g.table = table.p; g.cap = cap; g.n_states = d_counters.p; g.pair = pair.p;
                g.mstart = nullptr; g.foff = nullptr; g.arc_base = arc_base; g.f_lo = f_lo; g.sel = sel.p;
                g.o_src = o_src; g.o_il = o_il; g.o_ol = o_ol; g.o_tgt = o_tgt; g.o_w = o_w;
                g.bits_b = bits_b; g.nq2 = nq2;
                g.q2_bits = partitioned ? bits_for(nq2 > 1 ? nq2 - 1 : 1) : -1;
                k_gprod<0, false><<<static_cast<unsigned>(n_tiles), GP_THREADS, 0, c.stream>>>(g);
                FSTC_LAUNCH_CHECK();
                exclusive_scan<uint32_t>(c, tile_cnt.p, n_tiles, tile_off.p);
                MGm = read_scalar(c, tile_off.p + n_tiles);
                g.tile_off = tile_off.p;
                if (!partitioned && !o.deterministic && MGm > 0) {
                    // table level: ONE more kernel computes the weights, resolves the targets in the visited table and writes
                    // the arcs to their final place; for that the per-pair counts come from what pass 0 left behind
                    DBuf<int64_t> cntG(c, nf);
                    FSTC_CUDA(cudaMemsetAsync(cntG.p, 0, sizeof(int64_t) * nf, c.stream));
                    k_gcount<<<nblk(MG), CT_THREADS, 0, c.stream>>>(g, cntG.p);
                    FSTC_LAUNCH_CHECK();
                    mstartG.alloc(c, nf + 1);
                    exclusive_scan<int64_t>(c, cntG.p, nf, mstartG.p);
                    fc.alloc(c, nf); foff.alloc(c, nf + 1);
                    k_final_counts<<<nblk(nf), CT_THREADS, 0, c.stream>>>(rawU.p, mstartS.p, mstartG.p, scnt.p, nf, fc.p);
                    FSTC_LAUNCH_CHECK();
                    exclusive_scan<int64_t>(c, fc.p, nf, foff.p);
                    g.mstart = mstartG.p; g.foff = foff.p;
                    if (use_dense) k_gprod<2, true><<<static_cast<unsigned>(n_tiles), GP_THREADS, 0, c.stream>>>(g);
                    else k_gprod<2, false><<<static_cast<unsigned>(n_tiles), GP_THREADS, 0, c.stream>>>(g);
                    FSTC_LAUNCH_CHECK();
                    c.n_launch += 6;
                    tm.end(h);
                    n_states_live = static_cast<int64_t>(read_scalar(c, d_counters.p));
                    g_placed = true;
                    st.n_raw_grouped += RG;
                    c.sync();
                } else {
                gsrc.alloc(c, MGm); gab.alloc(c, MGm); gw.alloc(c, MGm); gtgt.alloc(c, MGm);
                DBuf<unsigned long long> gkeys(c, MGm + 2);
                g.tile_off = tile_off.p; g.msrc = gsrc.p; g.mab = gab.p; g.mw = gw.p; g.mkey = gkeys.p;
                k_gprod<1, false><<<static_cast<unsigned>(n_tiles), GP_THREADS, 0, c.stream>>>(g);
                FSTC_LAUNCH_CHECK();
                c.n_launch += 4;
                tm.end(h);
                // target ids of the merged arcs
                if (MGm > 0) {
                    if (partitioned) {
                        ResolveJob j;
                        j.keys = gkeys.p; j.n_records = MGm; j.q2_bits = g.q2_bits;
                        j.key_bits = g.q2_bits + bits_for(static_cast<uint64_t>(m1.n_states > 1 ? m1.n_states - 1 : 1));
                        j.pair = pair.p; j.n_states_before = n_states_live; j.n_states = d_counters.p;
                        j.mode = 0; j.pos = nullptr; j.o_tgt = gtgt.p; j.sortrec = nullptr; j.shift_t = 0;
                        j.force_bits = knob_resolve_bits;
                        j.stats = &st; j.profile = o.profile != 0;
                        run_resolve(j, 1);
                    } else {
                        h = tm.begin(FSTC_T_EMIT);
                        if (use_dense)
                            k_resolve_keys<true><<<nblk(MGm), CT_THREADS, 0, c.stream>>>(gkeys.p, MGm, dense.p, nullptr, 0, nq2, d_counters.p,
                                                                                        pair.p, gtgt.p);
                        else
                            k_resolve_keys<false><<<nblk(MGm), CT_THREADS, 0, c.stream>>>(gkeys.p, MGm, nullptr, table.p, cap, nq2,
                                                                                         d_counters.p, pair.p, gtgt.p);
                        FSTC_LAUNCH_CHECK();
                        c.n_launch += 1;
                        tm.end(h);
                    }
                    if (!external) n_states_live = static_cast<int64_t>(read_scalar(c, d_counters.p));
                }
                mstartG.alloc(c, nf + 1);
                k_mstart<<<nblk(nf + 1), CT_THREADS, 0, c.stream>>>(gsrc.p, MGm, nf, mstartG.p);
                FSTC_LAUNCH_CHECK();
                c.n_launch += 1;
                st.n_raw_grouped += RG;
                c.sync();
                }
            }
            // ---- final place of every arc of the level
            h = tm.begin(FSTC_T_REDUCE);
            if (!g_placed) {
                fc.alloc(c, nf); foff.alloc(c, nf + 1);
                k_final_counts<<<nblk(nf), CT_THREADS, 0, c.stream>>>(rawU.p, mstartS.p, mstartG.p, scnt.p, nf, fc.p);
                FSTC_LAUNCH_CHECK();
                exclusive_scan<int64_t>(c, fc.p, nf, foff.p);
            }
            DBuf<uint32_t> rank;
            int64_t det_n1 = 0;
            if (o.deterministic) {
                // every state of the level must exist before the ids can be ranked: the class-U arcs go out first; their
                // targets (and only theirs: the other positions are not written yet) are remapped with the pair table
                tm.end(h);
                launch_emit(EMIT_INDIRECT, LU, MU, RU, 0, f_lo, foff.p, roffU.p, arc_base, nullptr, 0, 0);
                det_n1 = static_cast<int64_t>(read_scalar(c, d_counters.p));
                rank = det_renumber(n_states, det_n1, arc_base, arc_base + RU + M + MGm);
                h = tm.begin(FSTC_T_REDUCE);
                if (M > 0) {                                         // merged class-F arcs: sorted again, on the new ids
                    DBuf<uint4> fa(c, M), fb(c, M);
                    k_det_frec<<<nblk(M), CT_THREADS, 0, c.stream>>>(mkey.p, msrc.p, mw.p, M, shift_t, n_states, det_n1, rank.p, fa.p);
                    FSTC_LAUNCH_CHECK();
                    const int tgt_bits = bits_for(static_cast<uint64_t>(det_n1 > 1 ? det_n1 - 1 : 1));
                    uint4 *fs = radix_sort_records(c, fa.p, fb.p, M, make_sort_passes(shift_t + tgt_bits, bits_for(static_cast<uint64_t>(nf - 1))));
                    k_det_funpack<<<nblk(M), CT_THREADS, 0, c.stream>>>(fs, M, mkey.p, msrc.p, mw.p);
                    FSTC_LAUNCH_CHECK();
                    c.n_launch += 2;
                    c.sync();
                }
            }
            if (M > 0) {
                k_place_merged<<<nblk(M), CT_THREADS, 0, c.stream>>>(mkey.p, msrc.p, mw.p, M, mstartS.p, foff.p, arc_base, f_lo, sel.p,
                                                                     shift_t, bits_b, o_src, o_il, o_ol, o_tgt, o_w);
                FSTC_LAUNCH_CHECK();
            }
            if (MGm > 0 && !g_placed) {
                k_place_grouped<<<nblk(MGm), CT_THREADS, 0, c.stream>>>(gab.p, gtgt.p, gsrc.p, gw.p, MGm, mstartG.p, foff.p, arc_base,
                                                                       f_lo, sel.p, bits_b, o_src, o_il, o_ol, o_tgt, o_w,
                                                                       n_states, det_n1, o.deterministic ? rank.p : nullptr);
                FSTC_LAUNCH_CHECK();
            }
            if (MSm > 0 && partitioned) {                            // (sbase in the place of mstart: a pair's arcs are neighbours)
                k_place_grouped<<<nblk(MSm), CT_THREADS, 0, c.stream>>>(sab.p, stgt.p, ssrc.p, sw.p, MSm, sbase.p, foff.p, arc_base,
                                                                       f_lo, sel.p, bits_b, o_src, o_il, o_ol, o_tgt, o_w);
                FSTC_LAUNCH_CHECK();
            } else if (MSm > 0) {                                    // table level: ids and placement in one kernel
                tm.end(h);
                h = tm.begin(FSTC_T_EMIT);
                if (use_dense)
                    k_resolve_place<true><<<nblk(MSm), CT_THREADS, 0, c.stream>>>(skeys.p, ssrc.p, sab.p, sw.p, MSm, sbase.p, foff.p, arc_base, f_lo,
                                                                                 sel.p, bits_b, dense.p, nullptr, 0, nq2, d_counters.p, pair.p,
                                                                                 o_src, o_il, o_ol, o_tgt, o_w);
                else
                    k_resolve_place<false><<<nblk(MSm), CT_THREADS, 0, c.stream>>>(skeys.p, ssrc.p, sab.p, sw.p, MSm, sbase.p, foff.p, arc_base, f_lo,
                                                                                  sel.p, bits_b, nullptr, table.p, cap, nq2, d_counters.p, pair.p,
                                                                                  o_src, o_il, o_ol, o_tgt, o_w);
                FSTC_LAUNCH_CHECK();
                tm.end(h);
                h = tm.begin(FSTC_T_REDUCE);
            }
            c.n_launch += 4;
            tm.end(h);
            if (!o.deterministic) launch_emit(EMIT_INDIRECT, LU, MU, RU, 0, f_lo, foff.p, roffU.p, arc_base, nullptr, 0, 0);
            n_arcs += RU + M + MGm + MSm;
            st.n_raw_sorted += RF + RS;
            c.sync();   // the level's temporaries go out of scope below
        }

        hostmark("emit+resolve", lvl);
        if (external) ext_finish_level();
        const int64_t ns_after = external ? n_states_live : static_cast<int64_t>(read_scalar(c, d_counters.p));
        hostmark("ns read", lvl);
        if (lvl < FSTC_MAX_LEVEL_STATS) {                       // (a level expanded in chunks adds up)
            st.level_frontier[lvl] += nf_all;
            st.level_raw[lvl] += R;
            st.level_new_states[lvl] += ns_after - n_states;
        }
        if (level_end >= 0) st.n_chunks += 1;
        spill_level(arc_base, n_arcs, ns_after);
        if (partitioned) st.rs_dedupe_new += ns_after - n_states;
        st.n_matches += MU + MF + MS;
        st.n_expanded += n_sel;
        last_fan = n_sel > 0 ? static_cast<double>(R) / static_cast<double>(n_sel) : 0.0;
        cum_raw += R;
        n_states = ns_after;
        f_lo = f_hi;
        st.n_levels = lvl + 1;
        if (level_end >= 0 && f_lo < level_end) {                // the next chunk of the same level
            f_hi = std::min(f_lo + chunk_pairs, level_end);
            continue;
        }
        level_end = -1;
        f_hi = n_states;
        ++lvl;
        if (stop_after) break;
    }

    hostmark("levels done", lvl);
    // ---- assemble
    int h = tm.begin(FSTC_T_ASSEMBLE);
    DBuf<uint8_t> expanded(c, n_states, true);
    const int64_t as_tiles = ceil_div(n_states, AS_TILE);
    DBuf<uint32_t> tile_count(c, as_tiles);
    DBuf<int64_t> tile_off(c, as_tiles + 1);
    if (last_lo > 0) FSTC_CUDA(cudaMemsetAsync(expanded.p, 1, static_cast<size_t>(last_lo), c.stream));
    if (n_states > last_hi) FSTC_CUDA(cudaMemsetAsync(expanded.p + last_hi, 0, static_cast<size_t>(n_states - last_hi), c.stream));
    if (last_hi > last_lo) {
        k_expanded_last<<<nblk(last_hi - last_lo), CT_THREADS, 0, c.stream>>>(pair.p, last_lo, last_hi, last_mode, nq2, cut_key, expanded.p);
        FSTC_LAUNCH_CHECK();
    }
    k_assemble_count<<<static_cast<unsigned>(as_tiles), AS_THREADS, 0, c.stream>>>(pair.p, n_states, m1.accept_bits, m2.accept_bits, tile_count.p);
    FSTC_LAUNCH_CHECK();
    exclusive_scan<uint32_t>(c, tile_count.p, as_tiles, tile_off.p);
    const int64_t n_accept = read_scalar(c, tile_off.p + as_tiles);
    DBuf<int32_t> accept(c, n_accept, true);
    if (n_accept > 0) {
        k_assemble_scatter<<<static_cast<unsigned>(as_tiles), AS_THREADS, 0, c.stream>>>(
            pair.p, n_states, m1.accept_bits, m2.accept_bits, tile_count.p, tile_off.p, accept.p);
        FSTC_LAUNCH_CHECK();
    }
    c.n_launch += 3;
    tm.end(h);

    if (sp) {
        if (n_states > sp->state_capacity) fail(FSTC_ERR_CAPACITY, "spill: %lld states outgrow the host arrays", static_cast<long long>(n_states));
        if (n_states > spilled_states)                            // (a search that stopped before its first level)
            FSTC_CUDA(cudaMemcpyAsync(sp->host->pair + 2 * spilled_states, pair.p + spilled_states, sizeof(int2) * static_cast<size_t>(n_states - spilled_states),
                                      cudaMemcpyDeviceToHost, c.stream));
        if (sp->host->accept && n_accept > 0)
            FSTC_CUDA(cudaMemcpyAsync(sp->host->accept, accept.p, sizeof(int32_t) * static_cast<size_t>(n_accept), cudaMemcpyDeviceToHost, c.stream));
        if (sp->host->expanded)
            FSTC_CUDA(cudaMemcpyAsync(sp->host->expanded, expanded.p, static_cast<size_t>(n_states), cudaMemcpyDeviceToHost, c.stream));
        st.spill_bytes += 8 * (n_states - spilled_states) + 4 * n_accept + n_states;
        FSTC_CUDA(cudaStreamSynchronize(side));
        spill_reap(true);
    }
    unsigned long long cnt[3];
    FSTC_CUDA(cudaMemcpyAsync(cnt, d_counters.p, sizeof cnt, cudaMemcpyDeviceToHost, c.stream));
    FSTC_CUDA(cudaEventRecord(ev1, c.stream));
    c.sync();
    float ms = 0.f;
    cudaEventElapsedTime(&ms, ev0, ev1);
    tm.collect(st.ms);
    hostmark("assembled", lvl);

    st.ms_total = ms;
    st.n_states = n_states; st.n_arcs = n_arcs; st.n_raw_arcs = cum_raw;
    st.n_seg_visited = static_cast<int64_t>(cnt[1]);
    st.n_match_arcs = static_cast<int64_t>(cnt[2]);
    st.table_capacity = static_cast<int64_t>(use_dense && dense.p ? n_pairs_all : cap);
    st.n_kernel_launches = static_cast<int32_t>(c.n_launch);

    fstc_result_t *r = new fstc_result_t();
    ResultImpl *impl = new ResultImpl();
    impl->hooks = c.hooks;
    r->n_states = n_states; r->n_arcs = n_arcs; r->n_raw_arcs = cum_raw; r->n_accept = n_accept;
    r->n_expanded = st.n_expanded; r->n_levels = st.n_levels; r->truncated = st.truncated;
    r->pair = reinterpret_cast<int32_t *>(pair.take());
    if (!spill_only) {
        r->src = a_src.take(); r->ilabel = a_il.take(); r->olabel = a_ol.take(); r->tgt = a_tgt.take();
        r->weight = a_w.take();
    }
    r->accept = accept.take(); r->expanded = expanded.take();
    impl->bufs[0] = r->pair; impl->bufs[1] = r->src; impl->bufs[2] = r->ilabel; impl->bufs[3] = r->olabel;
    impl->bufs[4] = r->tgt; impl->bufs[5] = r->weight; impl->bufs[6] = r->accept; impl->bufs[7] = r->expanded;
    r->impl = impl;
    return r;
}

}  // namespace

fstc_result_t *compose_packed(Ctx &c, const fstc_packed_t &m1, const fstc_packed_t &m2, const fstc_opts_t &opts,
                              fstc_stats_t *stats) {
    if (opts.small_path < 0 || opts.small_path > 2 || opts.deterministic < 0 || opts.deterministic > 1) fail(FSTC_ERR_ARG, "bad options");
    int dev = 0;
    FSTC_CUDA(cudaGetDevice(&dev));
    if (m1.device != dev || m2.device != dev)
        fail(FSTC_ERR_ARG, "operands were packed on device %d / %d, the current device is %d", m1.device, m2.device, dev);
    if (small_path_applies(opts)) {
        // small problems never leave the device (small.cu); one that outgrows the block's capacities comes back here
        const fstc_packed_t *one = &m1;
        fstc_result_t *r = nullptr;
        std::vector<char> ok;
        compose_small_batch(c, &one, 1, m2, opts, &r, stats, ok);
        if (ok[0]) return r;
        if (opts.small_path == FSTC_SMALL_ONLY) fail(FSTC_ERR_CAPACITY, "the problem does not fit the small path");
    } else if (opts.small_path == FSTC_SMALL_ONLY) fail(FSTC_ERR_ARG, "the small path does not take these options");
    Composer k(c, m1, m2, opts);
    fstc_result_t *r = k.run();
    if (stats) *stats = k.st;
    return r;
}

}  // namespace fstc
