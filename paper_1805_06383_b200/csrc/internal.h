// Internal interfaces between the translation units of libfstc.  Not part of the C ABI.
#pragma once

#include <vector>

#include "common.cuh"

namespace fstc {

// ---------------------------------------------------------------- radix sort (radix_sort.cu)
// Records are 16 bytes: {x,y} = 64-bit key (x low word), z = 32-bit high key ("src"), w = payload.
// The sort order is (z, key64) ascending, restricted to the bits the passes name; it is a stable
// least-significant-digit radix sort with digits of up to 8 bits that may straddle key and z.
struct SortPass {
    int word;   // number of key bits: a record sorts as the number (z << key_bits) | key64
    int shift;  // bit offset of the digit inside that number (a digit may straddle key and z)
    int bits;   // 1..8
};
// LSD pass list over bits [from_bit, key_bits + z_bits) of (z << key_bits) | key, 8 bits at a time.
std::vector<SortPass> make_sort_passes(int key_bits, int z_bits, int from_bit = 0);
// Sorts n records.  `a` holds the input; `b` is scratch of the same size.  Returns the buffer
// (a or b) that holds the sorted records.
uint4 *radix_sort_records(Ctx &c, uint4 *a, uint4 *b, int64_t n, const std::vector<SortPass> &passes);

// ---------------------------------------------------------------- packed transducer (pack.cu)
enum : uint8_t { FLAG_D = 1, FLAG_X = 2 };

}  // namespace fstc

// The opaque type of include/fstc.h.  All arrays are device memory from the library pool.
struct fstc_packed_t {
    int side = 0;                 // 1: inner = olabel (left operand), 2: inner = ilabel (right operand)
    int32_t n_states = 0, n_inner = 0, n_outer = 0, start = 0;
    int64_t n_arcs = 0, n_segs = 0;
    uint4 *arcs = nullptr;        // [n_arcs]   {tgt, outer, weight bits, inner}, sorted by (src, inner, outer, tgt)
    uint2 *segs = nullptr;        // [n_segs+1] {inner symbol, first arc}; sentinel {0xFFFFFFFF, n_arcs}
    uint32_t *seg_ptr = nullptr;  // [n_states+1] first segment of each state
    uint8_t *flags = nullptr;     // [n_states] FLAG_D | FLAG_X
    uint32_t *accept_bits = nullptr;  // [(n_states+31)/32]
    int device = 0;
    int64_t n_launch = 0;         // kernel launches fstc_pack took
    uint8_t any_flags = 0;        // OR of flags[] over all states
    // The same arcs grouped by (source, outer symbol, target): a group is what a composed arc sees of this operand
    // (its a or b, and its r1 or r2); inside a group the arcs are sorted by inner symbol.  Used by the merge by
    // construction (compose.cu, class G).
    int64_t n_groups = 0;
    uint2 *garcs = nullptr;       // [n_arcs]     {inner symbol, weight bits}, sorted by (src, outer, tgt, inner)
    uint32_t *goff = nullptr;     // [n_groups+1] first arc of each group; goff[n_groups] = n_arcs
    uint2 *gkey = nullptr;        // [n_groups]   {outer symbol, target}
    uint32_t *gptr = nullptr;     // [n_states+1] first group of each state
    unsigned long long *gmask = nullptr;   // [n_groups] inner symbols of the group as a bit mask, bit 63 = a symbol twice; only when n_inner <= 63
    fstc::AllocHooks hooks;       // who owns the arrays (set: the caller's allocator)
};

namespace fstc {

// what the kernels read of a packed operand
struct MachineView {
    const uint4 *arcs;
    const uint2 *segs;
    const uint32_t *seg_ptr;
    const uint8_t *flags;
    const uint2 *garcs;          // grouped copy (internal.h): {inner, weight} sorted by (src, outer, tgt, inner)
    const uint32_t *goff;
    const uint2 *gkey;
    const uint32_t *gptr;
    const unsigned long long *gmask;   // null when the inner alphabet has more than 63 symbols
};

inline MachineView view_of(const fstc_packed_t &p) {
    return MachineView{p.arcs, p.segs, p.seg_ptr, p.flags, p.garcs, p.goff, p.gkey, p.gptr, p.gmask};
}

fstc_packed_t *pack_fst(Ctx &c, const fstc_fst_t &m, int side);
void free_packed(fstc_packed_t *p);

// ---------------------------------------------------------------- composition (compose.cu)
fstc_result_t *compose_packed(Ctx &c, const fstc_packed_t &m1, const fstc_packed_t &m2, const fstc_opts_t &opts,
                              fstc_stats_t *stats);
void free_result(fstc_result_t *r);            // small.cu

struct SharedBlock {          // one device block that the results of a batch share
    void *base;
    int refs;
    AllocHooks hooks;
};
struct ResultImpl {           // owns the device arrays of a result
    void *bufs[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    SharedBlock *shared = nullptr;   // set: the arrays are parts of a batch's block
    AllocHooks hooks;                // who owns the arrays (set: the caller's allocator)
};
inline void release_block(void *p, const AllocHooks &h) {      // an array that left the library comes back
    if (!p) return;
    if (h.dealloc) h.dealloc(p, nullptr, h.ctx); else persist_free(p, nullptr);
}

// ---------------------------------------------------------------- small problems, one block each (small.cu)
bool small_path_applies(const fstc_opts_t &o);
void compose_small_batch(Ctx &c, const fstc_packed_t *const *m1, int n, const fstc_packed_t &m2, const fstc_opts_t &o,
                         fstc_result_t **results, fstc_stats_t *stats, std::vector<char> &ok);
// one problem, no allocation: result arrays from the caller, scratch in a static device array (fstc_compose_static)
void compose_small_static(Ctx &c, const fstc_packed_t &m1, const fstc_packed_t &m2, const fstc_opts_t &o,
                          const fstc_static_out_t &out);

// ---------------------------------------------------------------- partitioned target resolution (resolve.cu)
// Finds or creates the state id of every composed arc of a big level without touching a table in DRAM at random:
// the target keys are hash-partitioned with streaming passes, deduplicated per bin in shared memory against the
// existing states, and the ids gathered back through the recorded permutations.
struct ResolveJob {
    const unsigned long long *keys;     // [n_records] target (q1 << q2_bits) | q2 of every composed arc, in rank order
    int64_t n_records;
    int key_bits;                       // bits of such a key
    int q2_bits;
    int2 *pair;                         // [>= n_states_before + new states] id -> (q1, q2); new entries are written
    int64_t n_states_before;
    unsigned long long *n_states;       // device counter: set to n_states_before, advanced by the new states
    int mode;                           // 0: o_tgt[r] = id   1: o_tgt[pos[r]] = id   2: id into sortrec[r]
    const uint32_t *pos;                // mode 1
    int32_t *o_tgt;                     // modes 0, 1
    uint4 *sortrec;                     // mode 2: id OR-ed into key bits [shift_t, ...)
    int shift_t;
    int force_bits;                     // >= 0: number of hash bits to partition on (tests); -1: from the sizes
    fstc_stats_t *stats;                // nullable: work counters and (profile) stage times are added here
    bool profile;
};
int resolve_bits_needed(int64_t n_records_and_states);
bool resolve_can_take(int64_t n_records, int64_t n_states);   // within the u32 record indices and the 2^20 bins of resolve.cu
void resolve_partitioned(Ctx &c, const ResolveJob &j);
void resolve_apply_ids(Ctx &c, const ResolveJob &j, const uint32_t *ids);   // ids known (external resolve): deliver them

}  // namespace fstc
