/* fstc — weighted FST composition M1∘M2 on one NVIDIA B200 (sm_100a).  C ABI.
 *
 * The operation is the one "Composing Finite State Transducers on GPUs" (arXiv 1805.06383;
 * citations below are /root/reference/PAPER.md line numbers) states:
 *
 *   M1 = (Q1, Σ, Γ, s1, F1, δ1),  M2 = (Q2, Γ, Δ, s2, F2, δ2)                          (:39-45)
 *   M1∘M2 = (Q1×Q2, Σ, Δ, s1s2, F1×F2, δ),
 *   δ(q1q2, a, b, r1r2) = Σ_{c∈Γ} δ1(q1,a,c,r1)·δ2(q2,c,b,r2)                           (:47-53)
 *   "Transitions with the same source, target, input, and output symbols are merged,
 *    adding their weights."                                                             (:65)
 *
 * restricted to the state pairs accessible from s1s2, found by a breadth-first search over
 * the product graph (:77, :100, Algorithms 1-2 :106-131/:157-215).  No epsilon transitions
 * (:37); real weights, sum-of-products semiring; weights are fp32, products and sums fp32.
 *
 * Every step (packing, expansion, visited-set, merging, assembly) runs in CUDA kernels of this
 * library; there is no CPU fallback.  Nothing here depends on PyTorch.
 *
 * Memory spaces.  Every array pointer inside fstc_fst_t lives in the space named by its
 * `mem` field: FSTC_MEM_DEVICE (CUDA device memory of the current device) or FSTC_MEM_HOST
 * (ordinary or pinned host memory; the library stages it to the device itself).  All arrays of
 * fstc_result_t are DEVICE memory owned by the library (allocated through fstc_opts_t.alloc when the
 * caller set allocator hooks; the arc arrays are NULL when the result was spilled to the host without
 * a device copy, fstc_spill_t).  Struct pointers themselves
 * (fstc_fst_t*, fstc_opts_t*, fstc_stats_t*, fstc_host_result_t*) are host pointers.
 *
 * Threading / streams.  All work of a call is enqueued on `cuda_stream` (a cudaStream_t; NULL =
 * the legacy default stream).  Calls synchronise that stream internally where a size has to be
 * known on the host (a few times per BFS level; not at all inside the one-block path for small
 * problems) and before returning.  Inputs are never modified and may be released as soon as the
 * call returns.
 *
 * Errors.  Every int-returning call returns FSTC_OK (0) or a negative FSTC_ERR_* code; on error
 * the output pointer is set to NULL, nothing is leaked, and fstc_last_error() (thread-local)
 * holds a one-line description.
 */
#ifndef FSTC_H_
#define FSTC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FSTC_VERSION 3      /* 2: fstc_pack takes options; fstc_compose_batch; hooks, spill, deterministic, external resolve; 3: fstc_compose_static, fstc_stats_t.n_raw_onchip */

#if defined(__GNUC__)
#define FSTC_API __attribute__((visibility("default")))
#else
#define FSTC_API
#endif

enum {
  FSTC_OK = 0,
  FSTC_ERR_ARG = -1,      /* null pointer, negative size, start out of range, inner alphabets differ (:45) */
  FSTC_ERR_INPUT = -2,    /* a state or symbol id out of range (found by a device validation pass)        */
  FSTC_ERR_OOM = -3,      /* device (or pinned host) allocation failed                                     */
  FSTC_ERR_CAPACITY = -4, /* an internal limit was exceeded (see fstc_opts_t and DESIGN.md "limits")       */
  FSTC_ERR_CUDA = -5,     /* any other CUDA runtime error                                                  */
  FSTC_ERR_INTERNAL = -6, /* a consistency check of the library failed (a bug: please report the message)  */
  FSTC_ERR_CALLBACK = -7  /* fstc_opts_t.resolve_cb returned non-zero                                        */
};

enum { FSTC_MEM_DEVICE = 0, FSTC_MEM_HOST = 1 };

/* A weighted FST (:25-35).  Borrowed; never modified; must stay valid until the call returns.
 * States are 0..n_states-1 and symbols 0..n-1; symbol 0 is an ordinary symbol (there is no
 * epsilon, :37).  Arcs may come in any order; parallel duplicates (same src,ilabel,olabel,tgt)
 * are allowed and each contributes to the sum.  Every stored arc exists, whatever its weight. */
typedef struct fstc_fst_t {
  int32_t n_states;         /* |Q| >= 1                                                          */
  int32_t n_isyms;          /* input alphabet size  (M1: |Σ|, M2: |Γ|)                           */
  int32_t n_osyms;          /* output alphabet size (M1: |Γ|, M2: |Δ|)                           */
  int32_t start;            /* s, 0 <= start < n_states                                          */
  int64_t n_arcs;           /* 0 <= n_arcs < 2^31                                                */
  const int32_t *src;       /* [n_arcs] source state                                             */
  const int32_t *ilabel;    /* [n_arcs] input symbol                                             */
  const int32_t *olabel;    /* [n_arcs] output symbol                                            */
  const int32_t *tgt;       /* [n_arcs] target state                                             */
  const float *weight;      /* [n_arcs] fp32 weight                                              */
  int32_t n_accept;         /* |F|                                                               */
  const int32_t *accept;    /* [n_accept] accept state ids (duplicates tolerated)                */
  int32_t mem;              /* FSTC_MEM_DEVICE or FSTC_MEM_HOST: where the seven arrays live     */
} fstc_fst_t;

enum {
  FSTC_MERGE_AUTO = 0,      /* default: identical (src,tgt,a,b) arcs are summed (:65).  Only the sources
                               that CAN hold duplicates (exact test, N10, replacing the lossy
                               table H of :243) are merged: by construction from the (a,r1) x (b,r2) groups of the
                               pair when that is cheaper (arcs in (a,r1,b,r2) order), else in shared memory when
                               the source has at most 512 raw arcs (arcs in no particular order), else by sort +
                               reduce (arcs sorted by (tgt,a,b)); the other sources' arcs come in generation order
                               (inner symbol, e1, e2).  Arcs are always sorted by source id.            */
  FSTC_MERGE_OFF = 1,       /* "without performing any reductions" (:289): one arc per (e1,e2) match */
  FSTC_MERGE_SORT_ALL = 2   /* every source goes through sort + reduce: arcs sorted by (src,tgt,a,b) */
};

enum {
  FSTC_RESOLVE_AUTO = 0,        /* per level: the table while it fits the L2 cache, else the partitioned resolve */
  FSTC_RESOLVE_TABLE = 1,       /* always a visited table (atomicCAS per arc, :237): the paper's dense table of one
                                   entry per pair when |Q1||Q2| <= 2^29, else the open-addressing hash table   */
  FSTC_RESOLVE_PARTITIONED = 2, /* always the streaming hash-partitioned resolve         */
  FSTC_RESOLVE_HASH = 3,        /* always the open-addressing hash table, whatever |Q1||Q2|                    */
  FSTC_RESOLVE_EXTERNAL = 4     /* the caller resolves target keys to state ids (fstc_opts_t.resolve_cb): one
                                   composition sharded over several GPUs by ownership of the pair keys          */
};

/* FSTC_RESOLVE_EXTERNAL: every rank holds both operands and expands only the state pairs it OWNS; the target
 * keys of its arcs go to resolve_cb, which exchanges them with the other ranks (one all-to-all per call), lets the owners
 * find or create the states, and returns a GLOBAL state id per key.  Three calls per BFS level on every rank, whether or
 * not the rank has arcs of that class: call 0 (arcs that go through sort + reduce), 1 (arcs merged by construction),
 * 2 (all other arcs; sets *more = 1 if any rank created a state in this level, else the search ends everywhere).
 * keys: device, [n_keys], (r1 << q2_bits) | r2.  ids_out: device, [n_keys].  *new_pairs: device [2 * *n_new], the pairs
 * (q1, q2) this rank now owns in addition (local ids continue in that order); valid until the next call.  The callback
 * must have finished its device work when it returns; a non-zero return aborts the composition (FSTC_ERR_CALLBACK).
 * The result of a rank holds ITS states (pair, accept, expanded, local ids 0..n-1 in creation order) and their outgoing
 * arcs: src is a local id, tgt a global id.  Not with max_raw_arcs, deterministic, spill or the small path. */
typedef int (*fstc_resolve_fn)(void *ctx, int32_t level, int32_t call, int32_t q2_bits, const unsigned long long *keys,
                               int64_t n_keys, int32_t *ids_out, const int32_t **new_pairs, int64_t *n_new, int32_t *more);

/* Host spill (the paper streams its edge buffer to pinned host memory while the search goes on, :153-155,217,233).
 * Caller-allocated PINNED host arrays that receive the result WHILE it is built: the arcs and state pairs of a BFS level are
 * final once the level is placed, so their device->host copies run on a second stream under the next level's kernels;
 * the call returns when the host copy is complete (accept list and expanded flags included).  keep_device = 0: the arcs
 * then live on the host only — a level's device arrays are released as soon as its copy is done, the result's src /
 * ilabel / olabel / tgt / weight are NULL and n_arcs tells how many the host arrays hold: 20 bytes of HBM per arc are
 * never held beyond one level (stats.spill_bytes_saved).  keep_device = 1: the result keeps its device arrays as usual.
 * A result that outgrows arc_capacity / state_capacity -> FSTC_ERR_CAPACITY. */
struct fstc_host_result_t;
typedef struct fstc_spill_t {
  const struct fstc_host_result_t *host;  /* every array but `accept` / `expanded` may not be NULL              */
  int64_t arc_capacity;     /* length of src, ilabel, olabel, tgt, weight                                     */
  int64_t state_capacity;   /* length of pair / 2, accept, expanded                                           */
  int32_t keep_device;
  int32_t reserved_;
} fstc_spill_t;

enum {
  FSTC_SMALL_AUTO = 0,      /* default: the whole search first runs inside ONE thread block, with no host round trip
                               per BFS level (small inputs are overhead-bound, :291-293); a problem that outgrows the
                               block's capacities (4096 pairs or 65536 raw arcs in a level, 8192 states, 65536 arcs
                               unless the capacity hints say more) is composed again by the level-synchronous path  */
  FSTC_SMALL_OFF = 1,       /* never                                                                              */
  FSTC_SMALL_ONLY = 2       /* FSTC_ERR_CAPACITY instead of the level-synchronous path (tests)                     */
};

/* Options; NULL or all-zero = defaults. */
typedef struct fstc_opts_t {
  int32_t merge_mode;       /* FSTC_MERGE_*                                                           */
  int32_t max_levels;       /* stop before expanding BFS level max_levels (0 = unlimited)             */
  int64_t max_raw_arcs;     /* output budget in RAW composed arcs, rule T below (0 = unlimited)       */
  int64_t arc_capacity_hint;   /* expected number of output arcs (0 = none): avoids regrowing        */
  int64_t state_capacity_hint; /* expected number of output states (0 = none)                        */
  int32_t profile;          /* 1: time every stage with CUDA events on the stream (fills stats ms)    */
  int32_t resolve_mode;     /* FSTC_RESOLVE_*: how composed arcs find the ids of their target states          */
  int32_t small_path;       /* FSTC_SMALL_*: the device-resident path for small problems                      */
  int32_t deterministic;    /* 1: state ids and arc order are identical from run to run (see below)           */
  /* Allocator hooks: when `alloc` is set, EVERY device allocation of the call (temporaries and the arrays of the
   * result / packed operand) goes through it instead of the library's own pool, so that e.g. PyTorch's caching allocator
   * owns the memory.  alloc(bytes, stream, ctx) returns device memory usable by work queued on `stream` (NULL = out of
   * memory -> FSTC_ERR_OOM); dealloc(ptr, stream, ctx) is called once per block: during the call for temporaries (on the
   * call's stream, after the last kernel that uses them was queued), from fstc_result_free / fstc_packed_free for the
   * arrays that left the library (stream = NULL).  Both must be set or both NULL. */
  void *(*alloc)(size_t bytes, void *cuda_stream, void *ctx);
  void (*dealloc)(void *ptr, void *cuda_stream, void *ctx);
  void *alloc_ctx;
  const fstc_spill_t *spill;/* NULL: the result stays on the device                                           */
  fstc_resolve_fn resolve_cb;   /* FSTC_RESOLVE_EXTERNAL only                                                 */
  void *resolve_ctx;
  int32_t owns_start;       /* FSTC_RESOLVE_EXTERNAL: 1 on the rank that owns the start pair (its local state 0) */
  int32_t reserved_;
} fstc_opts_t;

/* deterministic = 1.  State ids are implementation-defined (:239 numbers states in discovery order, which is a race on
 * a GPU).  With this flag the states a BFS level creates are numbered in ascending order of their pair key q1*|Q2|+q2
 * (one sort of the new keys per level), and the arcs of a source come out in an order that only depends on the inputs
 * (generation order, group order, or (tgt,a,b) order on the final ids): two runs give bit-identical pair, src, ilabel,
 * olabel, tgt, accept and expanded arrays.  Weights of arcs merged by sort + reduce are summed with atomics and may differ
 * in the last bit.  The small path is not used.  (Big levels on the dense table number their states in key order in any
 * case: DESIGN.md §6h.) */

/* Rule T (the paper only notes that the result may not fit the device, :153).  BFS levels are
 * expanded whole while the running total of raw composed arcs stays <= max_raw_arcs.  The first
 * level that would exceed it is ordered by ascending pair key k = q1*|Q2|+q2 and its longest
 * prefix that still fits is expanded; then the search stops with truncated = 1.  States created
 * but not expanded stay in the result with expanded[i] = 0 and no outgoing arcs.  The rule only
 * depends on the frontier SET, so the result does not depend on thread scheduling. */

#define FSTC_MAX_LEVEL_STATS 64
enum {                      /* indices into fstc_stats_t.ms[] (filled when opts.profile = 1)         */
  FSTC_T_COUNT = 0,         /* per-pair inner-symbol intersection + raw counts                       */
  FSTC_T_SCAN = 1,          /* exclusive scans and the budget cut                                    */
  FSTC_T_MATCH = 2,         /* match work-list construction                                          */
  FSTC_T_EMIT = 3,          /* the emit kernel: load-balanced product arcs (+ visited-table find-or-insert when the level uses the table) */
  FSTC_T_SORT = 4,          /* radix sort of the arcs that may merge                                 */
  FSTC_T_REDUCE = 5,        /* segmented reduction + placement of merged arcs                        */
  FSTC_T_TABLE = 6,         /* visited table clear / grow + rehash                                   */
  FSTC_T_ASSEMBLE = 7,      /* accept list, expanded flags, output growth copies                     */
  FSTC_T_RS_SCATTER = 8,    /* partitioned resolve: staged scatter passes (states and arc keys)                */
  FSTC_T_RS_DEDUPE = 9,     /* partitioned resolve: per-bin dedupe in shared memory, new ids, pair table        */
  FSTC_T_RS_GATHER = 10,    /* partitioned resolve: ids back through the recorded permutations                  */
  FSTC_T_NSTAGES = 11
};

typedef struct fstc_stats_t {
  int64_t n_states, n_arcs, n_raw_arcs, n_expanded;
  int32_t n_levels, truncated;
  /* terms of the algorithmic-bytes model */
  int64_t n_seg_visited;    /* Σ over expanded pairs of (distinct inner symbols of q1 + of q2)        */
  int64_t n_matches;        /* number of (pair, inner symbol) matches                                 */
  int64_t n_match_arcs;     /* Σ over matches of (n1 + n2) input arcs read                            */
  int64_t n_raw_sorted;     /* raw arcs that went through sort + reduce                               */
  int64_t n_raw_grouped;    /* raw arcs merged by construction (class G: never materialised)          */
  int64_t n_raw_onchip;     /* of n_raw_sorted: raw arcs merged in shared memory (class S: never in HBM) */
  int64_t table_capacity;   /* final number of visited-table slots                                    */
  int32_t n_rehash, n_grow; /* table rebuilds, output regrow copies                                   */
  int32_t n_emit_launches, n_kernel_launches;
  int32_t n_resolve;        /* emit launches whose target ids came from the partitioned resolve                */
  int32_t small_path;       /* 1: composed by the small path (one thread block, one launch)                    */
  int64_t n_resolved_arcs;  /* raw arcs of those launches                                                     */
  /* work of the partitioned resolve, for its roofline: records through the scatter passes without / with
   * the recorded permutation, arc keys and state records through the dedupe, ids through the gathers; launches    */
  int64_t rs_scatter_recs, rs_scatter_dest_recs, rs_dedupe_arcs, rs_dedupe_states, rs_dedupe_new, rs_gather_recs;
  int32_t rs_scatter_launches, rs_dedupe_launches, rs_gather_launches;
  int32_t n_chunks;         /* pieces of the levels that were too big for the workspace and went chunk by chunk */
  int64_t spill_bytes, spill_bytes_saved;  /* bytes copied to the host while the search ran; device bytes never held (keep_device = 0) */
  double ms[FSTC_T_NSTAGES];/* device time per stage (CUDA events), only when opts.profile = 1       */
  double ms_total;          /* device time of the whole call (CUDA events), always                    */
  int64_t level_frontier[FSTC_MAX_LEVEL_STATS];  /* |F_l|                                             */
  int64_t level_raw[FSTC_MAX_LEVEL_STATS];       /* raw arcs composed in level l                      */
  int64_t level_new_states[FSTC_MAX_LEVEL_STATS];
} fstc_stats_t;

/* The composed transducer.  Owned by the library; release with fstc_result_free.
 * State i is the pair (pair[2i], pair[2i+1]) = (q1, q2); state 0 is the start pair s1s2 (:49).
 * Other state numbers are implementation-defined (:239 numbers them in discovery order, which is
 * racy on a GPU); compare results in pair coordinates. */
typedef struct fstc_result_t {
  int64_t n_states, n_arcs, n_raw_arcs, n_accept, n_expanded;
  int32_t n_levels;         /* BFS levels at least partly expanded                                    */
  int32_t truncated;        /* 1 iff max_raw_arcs / max_levels stopped the search                     */
  int32_t *pair;            /* device [2*n_states]  interleaved (q1, q2)                              */
  int32_t *src;             /* device [n_arcs] source state id, ASCENDING                             */
  int32_t *ilabel;          /* device [n_arcs] a ∈ Σ                                                  */
  int32_t *olabel;          /* device [n_arcs] b ∈ Δ                                                  */
  int32_t *tgt;             /* device [n_arcs] target state id                                        */
  float *weight;            /* device [n_arcs]                                                        */
  int32_t *accept;          /* device [n_accept] ascending ids with q1 ∈ F1 and q2 ∈ F2 (:49,:131)    */
  uint8_t *expanded;        /* device [n_states] 1 iff the state's outgoing arcs are present          */
  void *impl;               /* private                                                                */
} fstc_result_t;

/* Caller-allocated HOST arrays that receive a copy of a result (sizes from fstc_result_t). */
typedef struct fstc_host_result_t {
  int32_t *pair, *src, *ilabel, *olabel, *tgt;
  float *weight;
  int32_t *accept;
  uint8_t *expanded;        /* any pointer may be NULL = skip that array                              */
} fstc_host_result_t;

/* A transducer in the layout the kernels read (§3.3 :141-149, adapted): arcs sorted by
 * (source, inner symbol, outer symbol, target), a per-state index of its distinct inner symbols,
 * an accept bitmap and the per-state duplicate flags of DESIGN.md N10.  Opaque, device-resident,
 * reusable across any number of compositions; release with fstc_packed_free. */
typedef struct fstc_packed_t fstc_packed_t;

/* side 1: the inner alphabet is the OUTPUT side (left operand M1); side 2: the INPUT side (M2). */
/* opts (nullable): only the allocator hooks are read. */
FSTC_API int fstc_pack(const fstc_fst_t *m, int side, const fstc_opts_t *opts, void *cuda_stream, fstc_packed_t **out);
FSTC_API void fstc_packed_free(fstc_packed_t *p);
/* info[0..6] = n_states, n_arcs, n_segments (distinct (state, inner symbol)), n_inner, n_outer, side,
 *               kernel launches the pack took */
FSTC_API int fstc_packed_info(const fstc_packed_t *p, int64_t *info);
/* Debug/test access: copies the packed arrays to HOST buffers (any may be NULL).
 * arcs4: [4*n_arcs] uint32 (tgt, outer, weight bits, inner); segs2: [2*(n_segments+1)] (symbol, arc offset);
 * seg_ptr: [n_states+1]; flags: [n_states] bit0 = D (two arcs share (outer,tgt)), bit1 = X (two arcs share
 * (inner,outer,tgt)); accept_bits: [(n_states+31)/32]. */
FSTC_API int fstc_packed_to_host(const fstc_packed_t *p, void *cuda_stream, uint32_t *arcs4, uint32_t *segs2,
                        uint32_t *seg_ptr, uint8_t *flags, uint32_t *accept_bits);

/* M1∘M2 from packed operands (m1 packed with side 1, m2 with side 2; inner alphabets must agree, :45). */
FSTC_API int fstc_compose_packed(const fstc_packed_t *m1, const fstc_packed_t *m2, const fstc_opts_t *opts,
                        void *cuda_stream, fstc_result_t **out, fstc_stats_t *stats /* nullable */);

/* M1[k]∘M2 for k = 0..n-1 against ONE packed right operand, in one call: the paper's use case of many small lattices
 * against one language model (:251-259).  Problems that fit a thread block are composed by one launch, a block each,
 * with no host round trip (FSTC_SMALL_*); the others go through fstc_compose_packed's level-synchronous path one after
 * the other.  m1: host array of n packed left operands (side 1); out: host array of n results (each released with
 * fstc_result_free; results of one call may share a device block, which is released with the last of them);
 * stats: NULL or a host array of n.  On error every out[k] is NULL and nothing is leaked. */
FSTC_API int fstc_compose_batch(const fstc_packed_t *const *m1, int32_t n, const fstc_packed_t *m2, const fstc_opts_t *opts,
                       void *cuda_stream, fstc_result_t **out, fstc_stats_t *stats /* nullable, [n] */);

/* ---- A composition that ALLOCATES NOTHING, for callers that cannot call cudaMalloc (stream capture, tight serving
 * loops, harnesses that forbid it).  fstc_compose_static is fstc_compose_batch's one-block-per-problem search (the
 * paper's small lattice against a language model, :251-259, :291-293) for ONE problem: the result arrays are the
 * CALLER's device buffers, the kernel's scratch (visited table, work lists of a level) is a static device array
 * inside the library, and the call only enqueues on cuda_stream: one clear of the report area, ONE kernel, one
 * 80-byte copy of the header.  No cudaMalloc / cudaFree / pool call, no synchronisation, no other library routine.
 *
 *   * Limits: state_capacity <= FSTC_STATIC_MAX_STATES (the visited table must fit the static array of
 *     FSTC_STATIC_SCRATCH_BYTES; every GPU that loads the library holds that array until the process exits);
 *     arc_capacity < 2^31; beyond them FSTC_ERR_CAPACITY.  The search itself has fstc_compose_batch's small-path
 *     caps per level (4096 frontier pairs, 32768 matches, 65536 raw arcs; 8192 raw arcs for one source that can
 *     hold duplicates).  A problem that outgrows a cap or a capacity ends with header.status = 1: the arrays then
 *     hold garbage and the caller composes it with fstc_compose_packed.
 *   * opts (nullable): merge_mode (AUTO or OFF), max_levels and max_raw_arcs are read; SORT_ALL, spill,
 *     deterministic, the external resolve and allocator hooks are refused (FSTC_ERR_ARG).
 *   * The operands' device must be the current device.  The first call on a device resolves the address of the
 *     static array (cudaGetSymbolAddress; it may load the module): make one call before capturing a stream.
 *   * EVERY call on a device shares the one scratch array, which keeps the last call's contents: the call clears
 *     the report area and the kernel clears the visited table before use, everything else is written before it is
 *     read.  Two calls that overlap on the GPU (different streams, or two host threads) RACE on it: order them on
 *     one stream or with events.
 *   * The result is the one fstc_compose_batch gives (same order of arcs: sources ascending, generation order
 *     inside a source, duplicates folded into their first occurrence; state numbers implementation-defined,
 *     state 0 = the start pair).  It is complete when the work on cuda_stream is: read `header` after that. */
#define FSTC_STATIC_MAX_STATES 65536
#define FSTC_STATIC_SCRATCH_BYTES (8u << 20)

typedef struct fstc_static_header_t {   /* 80 bytes, written on the stream after the kernel                   */
  int64_t n_states, n_arcs, n_raw_arcs, n_accept, n_expanded;
  int64_t n_seg_visited, n_match_arcs, n_matches;   /* as in fstc_stats_t                                     */
  int32_t n_levels, truncated;
  int32_t status;           /* 0: the arrays hold M1∘M2; 1: the problem did not fit (see above)               */
  int32_t reserved_;
} fstc_static_header_t;

typedef struct fstc_static_out_t {      /* the caller's buffers; the library keeps no pointer after the call  */
  int64_t state_capacity;   /* states the arrays can hold, 1 .. FSTC_STATIC_MAX_STATES                        */
  int64_t arc_capacity;     /* arcs the arrays can hold, >= 1                                                 */
  int32_t *pair;            /* device [2*state_capacity], 8-byte aligned                                      */
  int32_t *src, *ilabel, *olabel, *tgt;   /* device [arc_capacity]                                            */
  float *weight;            /* device [arc_capacity]                                                          */
  int32_t *accept;          /* device [state_capacity]                                                        */
  uint8_t *expanded;        /* device [state_capacity]                                                        */
  fstc_static_header_t *header;   /* device or pinned host memory (pageable host memory makes the copy block) */
} fstc_static_out_t;

FSTC_API int fstc_compose_static(const fstc_packed_t *m1, const fstc_packed_t *m2, const fstc_opts_t *opts,
                        void *cuda_stream, const fstc_static_out_t *out);

/* fst_compose(M1, M2) -> M1∘M2: packs both operands, composes, frees the packed forms. */
FSTC_API int fstc_compose(const fstc_fst_t *m1, const fstc_fst_t *m2, const fstc_opts_t *opts, void *cuda_stream,
                 fstc_result_t **out, fstc_stats_t *stats /* nullable */);

/* Copies the result arrays to caller-allocated host memory (pinned memory makes it asynchronous
 * until the final stream synchronisation, which this call performs). */
FSTC_API int fstc_result_to_host(const fstc_result_t *r, void *cuda_stream, const fstc_host_result_t *dst);
/* The caller must have finished every use of the result's device arrays (or ordered it before the legacy default
 * stream) when it frees the result: the blocks are handed to the next composition that asks for their size. */
FSTC_API void fstc_result_free(fstc_result_t *r);

/* Releases the cached device memory back to the driver: the calling thread's workspace arena, the parked result /
 * packed blocks and the pool's free blocks.  (Device memory the library caches is otherwise kept for reuse.) */
FSTC_API int fstc_trim_pool(void);

FSTC_API const char *fstc_strerror(int code);
FSTC_API const char *fstc_last_error(void);
FSTC_API int fstc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* FSTC_H_ */
