// Input packer (DESIGN.md step 1; §3.3 adapted).
//
// The paper keeps, per transducer, arrays T (targets), O (outer symbols), P (weights) sorted by inner
// symbol and a DENSE offset array R of |Q|·m+1 entries (:144), sorted on the CPU (:149,153).  Here the
// sort runs on the device and R is replaced by a sparse index: one (symbol, first-arc) entry per
// distinct (state, inner symbol) — |Q|·m would be 3.6 GB for the bigram machine of config 3.
//
// Output: arcs as one 16-byte record {tgt, outer, weight, inner} sorted by (src, inner, outer, tgt);
// segs/seg_ptr (CSR of segments over states); an accept bitmap; and per state the two flags that decide
// exactly when composed arcs can collide (N10, replacing the lossy table H of PAPER.md:243):
//   D(q): two distinct arcs of q share (outer, tgt);   X(q): two distinct arcs share (inner, outer, tgt).
#include "internal.h"
#include "scan.cuh"

namespace fstc {

namespace {

constexpr int PK_THREADS = 256;

struct RawFst {                  // device views of the caller's arrays
    const int32_t *src, *il, *ol, *tgt;
    const float *w;
    const int32_t *accept;
};

__global__ void pk_validate(RawFst f, int64_t n_arcs, int32_t n_accept, int32_t n_states, int32_t n_isyms,
                            int32_t n_osyms, int *__restrict__ bad) {
    int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    bool ok = true;
    if (i < n_arcs) {
        ok = static_cast<uint32_t>(f.src[i]) < static_cast<uint32_t>(n_states) &&
             static_cast<uint32_t>(f.tgt[i]) < static_cast<uint32_t>(n_states) &&
             static_cast<uint32_t>(f.il[i]) < static_cast<uint32_t>(n_isyms) &&
             static_cast<uint32_t>(f.ol[i]) < static_cast<uint32_t>(n_osyms);
    }
    if (i < n_accept) ok = ok && static_cast<uint32_t>(f.accept[i]) < static_cast<uint32_t>(n_states);
    if (!ok) atomicOr(bad, 1);
}

// record for sort #1: order (src, outer, tgt, inner)
__global__ void pk_make_records(RawFst f, int64_t n_arcs, int side, int bits_inner, int bits_tgt,
                                uint4 *__restrict__ rec) {
    int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= n_arcs) return;
    uint32_t inner = side == 1 ? f.ol[i] : f.il[i];
    uint32_t outer = side == 1 ? f.il[i] : f.ol[i];
    uint64_t key = (static_cast<uint64_t>(outer) << (bits_tgt + bits_inner)) |
                   (static_cast<uint64_t>(static_cast<uint32_t>(f.tgt[i])) << bits_inner) | inner;
    rec[i] = make_uint4(static_cast<uint32_t>(key), static_cast<uint32_t>(key >> 32),
                        static_cast<uint32_t>(f.src[i]), __float_as_uint(f.w[i]));
}

// On the (src, outer, tgt, inner) order: neighbours with equal (src, outer, tgt) set D, equal full key set X.
// Also rewrites the key to (inner, outer, tgt) for sort #2 (stable on (src, inner)).
__global__ void pk_flags_rekey(uint4 *__restrict__ rec, int64_t n_arcs, int bits_inner, int bits_tgt, int bits_outer,
                               uint32_t *__restrict__ flags32, uint4 *__restrict__ out) {
    int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= n_arcs) return;
    uint4 r = rec[i];
    uint64_t key = (static_cast<uint64_t>(r.y) << 32) | r.x;
    if (i > 0) {
        uint4 p = rec[i - 1];
        uint64_t pkey = (static_cast<uint64_t>(p.y) << 32) | p.x;
        if (p.z == r.z && (pkey >> bits_inner) == (key >> bits_inner)) {
            uint32_t f = FLAG_D | (pkey == key ? FLAG_X : 0);
            atomicOr(&flags32[r.z], f);
        }
    }
    uint64_t inner = key & ((uint64_t(1) << bits_inner) - 1);
    uint64_t tgt = (key >> bits_inner) & ((uint64_t(1) << bits_tgt) - 1);
    uint64_t outer = key >> (bits_inner + bits_tgt);
    uint64_t k2 = (inner << (bits_outer + bits_tgt)) | (outer << bits_tgt) | tgt;
    out[i] = make_uint4(static_cast<uint32_t>(k2), static_cast<uint32_t>(k2 >> 32), r.z, r.w);
}

// On the (src, outer, tgt, inner) order of sort #1: the grouped copy of the arcs.  A group = equal (src, outer, tgt).
__global__ void pk_group_heads(const uint4 *__restrict__ rec, int64_t n_arcs, int bits_inner, uint2 *__restrict__ garcs,
                               uint32_t *__restrict__ head) {
    int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= n_arcs) return;
    uint4 r = rec[i];
    uint64_t key = (static_cast<uint64_t>(r.y) << 32) | r.x;
    garcs[i] = make_uint2(static_cast<uint32_t>(key & ((uint64_t(1) << bits_inner) - 1)), r.w);
    uint32_t h = 1;
    if (i > 0) {
        uint4 p = rec[i - 1];
        uint64_t pkey = (static_cast<uint64_t>(p.y) << 32) | p.x;
        h = (p.z != r.z) || ((pkey >> bits_inner) != (key >> bits_inner));
    }
    head[i] = h;
}
__global__ void pk_fill_groups(const uint4 *__restrict__ rec, const uint32_t *__restrict__ head, const int64_t *__restrict__ gidx,
                               int64_t n_arcs, int bits_inner, int bits_tgt, uint32_t *__restrict__ goff,
                               uint2 *__restrict__ gkey, uint32_t *__restrict__ gsrc) {
    int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i == 0) goff[gidx[n_arcs]] = static_cast<uint32_t>(n_arcs);
    if (i >= n_arcs || !head[i]) return;
    const int64_t g = gidx[i];
    uint4 r = rec[i];
    uint64_t key = ((static_cast<uint64_t>(r.y) << 32) | r.x) >> bits_inner;        // (outer, tgt)
    goff[g] = static_cast<uint32_t>(i);
    gkey[g] = make_uint2(static_cast<uint32_t>(key >> bits_tgt), static_cast<uint32_t>(key & ((uint64_t(1) << bits_tgt) - 1)));
    gsrc[g] = r.z;
}

// On the final (src, inner, outer, tgt) order: unpack the arc record and mark segment heads.
__global__ void pk_unpack(const uint4 *__restrict__ rec, int64_t n_arcs, int bits_tgt, int bits_outer,
                          uint4 *__restrict__ arcs, uint32_t *__restrict__ head) {
    int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= n_arcs) return;
    uint4 r = rec[i];
    uint64_t key = (static_cast<uint64_t>(r.y) << 32) | r.x;
    uint32_t tgt = static_cast<uint32_t>(key & ((uint64_t(1) << bits_tgt) - 1));
    uint32_t outer = static_cast<uint32_t>((key >> bits_tgt) & ((uint64_t(1) << bits_outer) - 1));
    uint32_t inner = static_cast<uint32_t>(key >> (bits_tgt + bits_outer));
    arcs[i] = make_uint4(tgt, outer, r.w, inner);
    uint32_t h = 1;
    if (i > 0) {
        uint4 p = rec[i - 1];
        uint64_t pkey = (static_cast<uint64_t>(p.y) << 32) | p.x;
        h = (p.z != r.z) || ((pkey >> (bits_tgt + bits_outer)) != inner);
    }
    head[i] = h;
}

__global__ void pk_fill_segs(const uint4 *__restrict__ rec, const uint4 *__restrict__ arcs,
                             const uint32_t *__restrict__ head, const int64_t *__restrict__ seg_idx, int64_t n_arcs,
                             uint2 *__restrict__ segs, uint32_t *__restrict__ seg_src) {
    int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i == 0) {   // sentinel after the last segment
        int64_t ns = seg_idx[n_arcs];
        segs[ns] = make_uint2(0xFFFFFFFFu, static_cast<uint32_t>(n_arcs));
    }
    if (i >= n_arcs || !head[i]) return;
    int64_t s = seg_idx[i];
    segs[s] = make_uint2(arcs[i].w, static_cast<uint32_t>(i));
    seg_src[s] = rec[i].z;
}

// seg_ptr[q] = index of the first segment whose state is >= q (q = 0..n_states).
__global__ void pk_seg_ptr(const uint32_t *__restrict__ seg_src, int64_t n_segs, int32_t n_states,
                           uint32_t *__restrict__ seg_ptr) {
    int64_t q = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (q > n_states) return;
    int64_t lo = 0, hi = n_segs;
    while (lo < hi) {
        int64_t mid = (lo + hi) >> 1;
        if (seg_src[mid] < static_cast<uint32_t>(q)) lo = mid + 1; else hi = mid;
    }
    seg_ptr[q] = static_cast<uint32_t>(lo);
}

__global__ void pk_accept_bits(const int32_t *__restrict__ accept, int32_t n_accept, uint32_t *__restrict__ bits) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_accept) atomicOr(&bits[accept[i] >> 5], 1u << (accept[i] & 31));
}

__global__ void pk_narrow_flags(const uint32_t *__restrict__ f32, int32_t n, uint8_t *__restrict__ f8, int *__restrict__ any) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t f = (i < n) ? f32[i] : 0u;
    if (i < n) f8[i] = static_cast<uint8_t>(f);
    f = __reduce_or_sync(0xffffffffu, f);
    if ((threadIdx.x & 31) == 0 && f) atomicOr(any, static_cast<int>(f));
}

inline unsigned blocks_for(int64_t n) { return static_cast<unsigned>(ceil_div(n > 0 ? n : 1, PK_THREADS)); }

template <typename T>
const T *stage(Ctx &c, const T *p, int64_t n, int mem, DBuf<T> &hold) {
    if (mem == FSTC_MEM_DEVICE || n == 0) return p;
    hold.alloc(c, n);
    FSTC_CUDA(cudaMemcpyAsync(hold.p, p, static_cast<size_t>(n) * sizeof(T), cudaMemcpyHostToDevice, c.stream));
    return hold.p;
}

}  // namespace

// Small inner alphabets (|Γ| <= 63): the set of inner symbols of a group as a bit mask; bit 63 = the group holds the same
// symbol twice (parallel duplicate arcs).  With the masks the merge by construction sees whether two groups share a symbol
// with one AND, and finds the shared symbols' weights by popcount instead of walking both lists (compose.cu, k_gprod).
constexpr unsigned long long GMASK_DUP = 1ull << 63;
__global__ void pk_group_masks(const uint2 *__restrict__ garcs, const uint32_t *__restrict__ goff, int64_t n_groups,
                               unsigned long long *__restrict__ gmask) {
    const int64_t g = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (g >= n_groups) return;
    unsigned long long m = 0;
    for (uint32_t i = goff[g]; i < goff[g + 1]; ++i) {
        const unsigned long long b = 1ull << garcs[i].x;
        if (m & b) m |= GMASK_DUP;
        m |= b;
    }
    gmask[g] = m;
}

void free_packed(fstc_packed_t *p) {
    if (!p) return;
    // freed stream-ordered on the legacy stream: safe after any stream of ours has been synchronised
    release_block(p->arcs, p->hooks);
    release_block(p->segs, p->hooks);
    release_block(p->seg_ptr, p->hooks);
    release_block(p->flags, p->hooks);
    release_block(p->accept_bits, p->hooks);
    release_block(p->garcs, p->hooks);
    release_block(p->goff, p->hooks);
    release_block(p->gkey, p->hooks);
    release_block(p->gptr, p->hooks);
    release_block(p->gmask, p->hooks);
    delete p;
}

fstc_packed_t *pack_fst(Ctx &c, const fstc_fst_t &m, int side) {
    const int64_t launch0 = c.n_launch;
    if (side != 1 && side != 2) fail(FSTC_ERR_ARG, "side must be 1 or 2");
    if (m.n_states < 1 || m.n_isyms < 0 || m.n_osyms < 0 || m.n_arcs < 0 || m.n_accept < 0)
        fail(FSTC_ERR_ARG, "negative size or no states");
    if (m.n_arcs >= (int64_t(1) << 31)) fail(FSTC_ERR_CAPACITY, "n_arcs must be < 2^31");
    if (m.start < 0 || m.start >= m.n_states) fail(FSTC_ERR_ARG, "start state %d out of range", m.start);
    if (m.mem != FSTC_MEM_DEVICE && m.mem != FSTC_MEM_HOST) fail(FSTC_ERR_ARG, "bad mem space %d", m.mem);
    if (m.n_arcs > 0 && (!m.src || !m.ilabel || !m.olabel || !m.tgt || !m.weight))
        fail(FSTC_ERR_ARG, "null arc array");
    if (m.n_accept > 0 && !m.accept) fail(FSTC_ERR_ARG, "null accept array");

    const int64_t n = m.n_arcs;
    const int32_t n_inner = side == 1 ? m.n_osyms : m.n_isyms;
    const int32_t n_outer = side == 1 ? m.n_isyms : m.n_osyms;
    const int bi = bits_for(n_inner > 0 ? n_inner - 1 : 0), bo = bits_for(n_outer > 0 ? n_outer - 1 : 0);
    const int bt = bits_for(m.n_states - 1), bs = bt;
    if (bi + bo + bt > 64) fail(FSTC_ERR_CAPACITY, "bits(inner)+bits(outer)+bits(states) = %d > 64", bi + bo + bt);

    DBuf<int32_t> h_src, h_il, h_ol, h_tgt, h_acc;
    DBuf<float> h_w;
    RawFst f;
    f.src = stage(c, m.src, n, m.mem, h_src);
    f.il = stage(c, m.ilabel, n, m.mem, h_il);
    f.ol = stage(c, m.olabel, n, m.mem, h_ol);
    f.tgt = stage(c, m.tgt, n, m.mem, h_tgt);
    f.w = stage(c, m.weight, n, m.mem, h_w);
    f.accept = stage(c, m.accept, m.n_accept, m.mem, h_acc);

    DBuf<int> bad(c, 1);
    FSTC_CUDA(cudaMemsetAsync(bad.p, 0, sizeof(int), c.stream));
    const int64_t nv = n > m.n_accept ? n : m.n_accept;
    if (nv > 0) {
        pk_validate<<<blocks_for(nv), PK_THREADS, 0, c.stream>>>(f, n, m.n_accept, m.n_states, m.n_isyms, m.n_osyms,
                                                                 bad.p);
        FSTC_LAUNCH_CHECK();
        c.n_launch += 1;
    }
    if (read_scalar(c, bad.p)) fail(FSTC_ERR_INPUT, "a state or symbol id is out of range");

    DBuf<uint4> arcs(c, n, true);                             // the five arrays of the packed form outlive the call
    DBuf<uint2> segs;
    DBuf<uint32_t> seg_ptr(c, static_cast<int64_t>(m.n_states) + 1, true);
    DBuf<uint8_t> flags(c, m.n_states, true);
    DBuf<uint32_t> accept_bits(c, (m.n_states + 31) / 32, true);
    DBuf<uint32_t> flags32(c, m.n_states);
    FSTC_CUDA(cudaMemsetAsync(flags32.p, 0, sizeof(uint32_t) * m.n_states, c.stream));
    FSTC_CUDA(cudaMemsetAsync(accept_bits.p, 0, sizeof(uint32_t) * ((m.n_states + 31) / 32), c.stream));
    int64_t n_segs = 0, n_groups = 0;
    DBuf<uint2> garcs(c, n, true), gkey;
    DBuf<uint32_t> goff, gptr(c, static_cast<int64_t>(m.n_states) + 1, true);
    DBuf<unsigned long long> gmask;

    if (n > 0) {
        DBuf<uint4> ra(c, n), rb(c, n);
        pk_make_records<<<blocks_for(n), PK_THREADS, 0, c.stream>>>(f, n, side, bi, bt, ra.p);
        FSTC_LAUNCH_CHECK();
        uint4 *s1 = radix_sort_records(c, ra.p, rb.p, n, make_sort_passes(bi + bt + bo, bs));
        uint4 *o1 = (s1 == ra.p) ? rb.p : ra.p;
        {   // grouped copy, on this (src, outer, tgt, inner) order
            DBuf<uint32_t> ghead(c, n);
            DBuf<int64_t> gidx(c, n + 1);
            pk_group_heads<<<blocks_for(n), PK_THREADS, 0, c.stream>>>(s1, n, bi, garcs.p, ghead.p);
            FSTC_LAUNCH_CHECK();
            exclusive_scan<uint32_t>(c, ghead.p, n, gidx.p);
            n_groups = read_scalar(c, gidx.p + n);
            goff.alloc(c, n_groups + 1, true);
            gkey.alloc(c, n_groups, true);
            DBuf<uint32_t> gsrc(c, n_groups);
            pk_fill_groups<<<blocks_for(n), PK_THREADS, 0, c.stream>>>(s1, ghead.p, gidx.p, n, bi, bt, goff.p, gkey.p, gsrc.p);
            FSTC_LAUNCH_CHECK();
            pk_seg_ptr<<<blocks_for(static_cast<int64_t>(m.n_states) + 1), PK_THREADS, 0, c.stream>>>(gsrc.p, n_groups, m.n_states,
                                                                                                     gptr.p);
            FSTC_LAUNCH_CHECK();
            c.n_launch += 3;
            if (n_inner <= 63 && n_groups > 0) {
                gmask.alloc(c, n_groups, true);
                pk_group_masks<<<blocks_for(n_groups), PK_THREADS, 0, c.stream>>>(garcs.p, goff.p, n_groups, gmask.p);
                FSTC_LAUNCH_CHECK();
                c.n_launch += 1;
            }
            c.sync();
        }
        pk_flags_rekey<<<blocks_for(n), PK_THREADS, 0, c.stream>>>(s1, n, bi, bt, bo, flags32.p, o1);
        FSTC_LAUNCH_CHECK();
        // stable sort on (src, inner) only: (outer, tgt) order inside a segment is inherited from sort #1
        // only the (inner, src) bits: the key is (inner, outer, tgt) with inner on top, directly below z = src
        std::vector<SortPass> p2 = make_sort_passes(bi + bo + bt, bs, bo + bt);
        uint4 *s2 = radix_sort_records(c, o1, s1, n, p2);
        DBuf<uint32_t> head(c, n);
        DBuf<int64_t> seg_idx(c, n + 1);
        pk_unpack<<<blocks_for(n), PK_THREADS, 0, c.stream>>>(s2, n, bt, bo, arcs.p, head.p);
        FSTC_LAUNCH_CHECK();
        exclusive_scan<uint32_t>(c, head.p, n, seg_idx.p);
        n_segs = read_scalar(c, seg_idx.p + n);
        segs.alloc(c, n_segs + 1, true);
        DBuf<uint32_t> seg_src(c, n_segs);
        pk_fill_segs<<<blocks_for(n), PK_THREADS, 0, c.stream>>>(s2, arcs.p, head.p, seg_idx.p, n, segs.p, seg_src.p);
        FSTC_LAUNCH_CHECK();
        pk_seg_ptr<<<blocks_for(static_cast<int64_t>(m.n_states) + 1), PK_THREADS, 0, c.stream>>>(seg_src.p, n_segs,
                                                                                                 m.n_states, seg_ptr.p);
        FSTC_LAUNCH_CHECK();
        c.n_launch += 5;
        c.sync();   // temporaries (ra, rb, head, ...) are released below; keep the stream ordered and simple
    } else {
        segs.alloc(c, 1, true);
        goff.alloc(c, 1, true);
        gkey.alloc(c, 1, true);
        FSTC_CUDA(cudaMemsetAsync(goff.p, 0, sizeof(uint32_t), c.stream));
        FSTC_CUDA(cudaMemsetAsync(gptr.p, 0, sizeof(uint32_t) * (static_cast<size_t>(m.n_states) + 1), c.stream));
        uint2 sentinel = make_uint2(0xFFFFFFFFu, 0u);
        FSTC_CUDA(cudaMemcpyAsync(segs.p, &sentinel, sizeof sentinel, cudaMemcpyHostToDevice, c.stream));
        FSTC_CUDA(cudaMemsetAsync(seg_ptr.p, 0, sizeof(uint32_t) * (static_cast<size_t>(m.n_states) + 1), c.stream));
        c.sync();
    }
    pk_narrow_flags<<<blocks_for(m.n_states), PK_THREADS, 0, c.stream>>>(flags32.p, m.n_states, flags.p, bad.p);
    FSTC_LAUNCH_CHECK();
    if (m.n_accept > 0) {
        pk_accept_bits<<<blocks_for(m.n_accept), PK_THREADS, 0, c.stream>>>(f.accept, m.n_accept, accept_bits.p);
        FSTC_LAUNCH_CHECK();
    }
    c.n_launch += 2;
    const int any_flags = read_scalar(c, bad.p);      // `bad` was zero after validation; reused as the OR of all flags

    fstc_packed_t *p = new fstc_packed_t();
    p->any_flags = static_cast<uint8_t>(any_flags);
    p->side = side;
    p->n_states = m.n_states; p->n_inner = n_inner; p->n_outer = n_outer; p->start = m.start;
    p->n_arcs = n; p->n_segs = n_segs;
    p->hooks = c.hooks;
    p->arcs = arcs.take(); p->segs = segs.take(); p->seg_ptr = seg_ptr.take();
    p->flags = flags.take(); p->accept_bits = accept_bits.take();
    p->n_groups = n_groups;
    p->garcs = garcs.take(); p->goff = goff.take(); p->gkey = gkey.take(); p->gptr = gptr.take();
    p->gmask = gmask.p ? gmask.take() : nullptr;
    FSTC_CUDA(cudaGetDevice(&p->device));
    p->n_launch = c.n_launch - launch0;
    return p;
}

}  // namespace fstc
