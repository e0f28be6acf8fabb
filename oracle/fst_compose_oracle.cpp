// ORACLE — TEST INFRASTRUCTURE ONLY.
//
// A plain, slow, serial CPU implementation of weighted FST composition, written
// from the paper (arXiv 1805.06383, /root/reference/PAPER.md).  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// build, load or call it.  It shares no code with the CUDA path
// (paper_1805_06383_b200/csrc) and neither includes the other.
//
// What it computes (citations are PAPER.md line numbers):
//   * Definition, PAPER.md:47-65 (§2):  M1∘M2 = (Q1×Q2, Σ, Δ, s1s2, F1×F2, δ) with
//       δ(q1q2, a, b, r1r2) = Σ_{c∈Γ} δ1(q1,a,c,r1)·δ2(q2,c,b,r2)
//     (the printed sum index "b∈Γ" at :53 is a typo for the inner symbol, N1);
//     "Transitions with the same source, target, input, and output symbols are
//     merged, adding their weights" (:65).
//   * Algorithm 1, PAPER.md:106-131 (§3.2): breadth-first search from s1s2 with a
//     frontier queue A and a visited set Q, so that only accessible state pairs are
//     created (:77, :100).  Line 8: δ(q1q2,a,c,r1r2) += p1·p2; lines 9-11: push unseen
//     targets.  No co-accessibility trim (N4).
//   * §3.3: arcs of a state are kept sorted by their inner symbol;
//     the arcs of (q, c) are found by binary search in that sorted list (instead of
//     the paper's dense offset array R[q·m+c], which is a pure indexing device).
//   * The visited set doubles as the pair -> state-number map (:239).  It is the
//     paper's dense lookup table of length |Q1||Q2| (:237) when that is small, else a
//     std::unordered_map; tests force both and compare.
//   * Output budget, rule T (the paper only notes that the output may not
//     fit, :153): levels are expanded whole while the cumulative number of RAW
//     composed arcs stays within max_raw_arcs; the first level that would overflow is
//     sorted by ascending pair key k = q1·|Q2|+q2 and its maximal prefix that still
//     fits is expanded; then the search stops with truncated = 1.
//
// Arithmetic: every product p1·p2 is formed in fp64 from the fp32 inputs (exact:
// 24+24 significant bits) and sums are fp64, in generation order.
//
// Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): brute force over the full
// Q1×Q2 product + trim (oracle/brute_force.py), the closed form
// Σ_out w = Σ_c W1(q1,c)·W2(q2,c), one-state machines == matrix product, identity
// transducer, linear chains, HMM forward recursion on a lattice∘bigram pair, the
// structure of the printed Fig. 1/2 example.  Nothing is unpinned
// except the WEIGHTS of that printed example (its figures are missing).
//
// Build: g++ -O2 -std=c++17 -shared -fPIC oracle/fst_compose_oracle.cpp -o oracle/libfst_oracle.so

#include <algorithm>
#include <chrono>
#include <cstdint>
#include <cstring>
#include <unordered_map>
#include <vector>

namespace {

struct InFst {                 // mirrors the ctypes struct in oracle/__init__.py
    int32_t n_states, n_isyms, n_osyms, start;
    int64_t n_arcs;
    const int32_t *src, *ilabel, *olabel, *tgt;
    const float *weight;
    int32_t n_accept;
    const int32_t *accept;
};

struct Arc {                   // one input transition q --outer:inner/p--> r, or q --inner:outer/p--> r
    int32_t inner, outer, tgt;
    double p;
};

// Arcs grouped by source state, each group sorted by inner symbol.
struct Machine {
    int32_t n_states = 0;
    std::vector<int64_t> row;  // row[q]..row[q+1] = arcs leaving q
    std::vector<Arc> arcs;
    std::vector<uint8_t> is_accept;
};

// side 1: inner symbol is the OUTPUT label (M1: Σ -> Γ); side 2: the INPUT label (M2: Γ -> Δ).
Machine load_machine(const InFst &f, int side) {
    Machine m;
    m.n_states = f.n_states;
    std::vector<int64_t> order(f.n_arcs);
    for (int64_t i = 0; i < f.n_arcs; ++i) order[i] = i;
    auto inner_of = [&](int64_t i) { return side == 1 ? f.olabel[i] : f.ilabel[i]; };
    std::stable_sort(order.begin(), order.end(), [&](int64_t x, int64_t y) {
        if (f.src[x] != f.src[y]) return f.src[x] < f.src[y];
        return inner_of(x) < inner_of(y);
    });
    m.arcs.resize(f.n_arcs);
    m.row.assign(f.n_states + 1, 0);
    for (int64_t k = 0; k < f.n_arcs; ++k) {
        int64_t i = order[k];
        Arc a;
        a.inner = inner_of(i);
        a.outer = side == 1 ? f.ilabel[i] : f.olabel[i];
        a.tgt = f.tgt[i];
        a.p = static_cast<double>(f.weight[i]);
        m.arcs[k] = a;
        m.row[f.src[i] + 1] += 1;
    }
    for (int32_t q = 0; q < f.n_states; ++q) m.row[q + 1] += m.row[q];
    m.is_accept.assign(f.n_states, 0);
    for (int32_t i = 0; i < f.n_accept; ++i) m.is_accept[f.accept[i]] = 1;
    return m;
}

// Arcs of state q2 in M2 whose inner symbol is c: [lo, hi) by binary search on the sorted slice.
inline void inner_range(const Machine &m, int32_t q, int32_t c, int64_t &lo, int64_t &hi) {
    const Arc *b = m.arcs.data() + m.row[q], *e = m.arcs.data() + m.row[q + 1];
    auto cmp_lo = [](const Arc &a, int32_t v) { return a.inner < v; };
    auto cmp_hi = [](int32_t v, const Arc &a) { return v < a.inner; };
    lo = std::lower_bound(b, e, c, cmp_lo) - m.arcs.data();
    hi = std::upper_bound(b, e, c, cmp_hi) - m.arcs.data();
}

// raw(q1,q2) = number of arc pairs (e1,e2) leaving (q1,q2) that share the inner symbol (N16).
int64_t raw_count(const Machine &m1, const Machine &m2, int32_t q1, int32_t q2) {
    int64_t n = 0;
    for (int64_t i = m1.row[q1]; i < m1.row[q1 + 1]; ++i) {
        int64_t lo, hi;
        inner_range(m2, q2, m1.arcs[i].inner, lo, hi);
        n += hi - lo;
    }
    return n;
}

struct OutArc {                // one composed transition, target in pair coordinates
    int32_t r1, r2, a, b;
    double w;
};

// Alg. 1 lines 6-8 for ONE popped pair: all (e1,e2) with equal inner symbol, weight p1·p2.
void expand_pair(const Machine &m1, const Machine &m2, int32_t q1, int32_t q2, std::vector<OutArc> &out) {
    out.clear();
    for (int64_t i = m1.row[q1]; i < m1.row[q1 + 1]; ++i) {
        const Arc &e1 = m1.arcs[i];
        int64_t lo, hi;
        inner_range(m2, q2, e1.inner, lo, hi);
        for (int64_t j = lo; j < hi; ++j) {
            const Arc &e2 = m2.arcs[j];
            out.push_back(OutArc{e1.tgt, e2.tgt, e1.outer, e2.outer, e1.p * e2.p});
        }
    }
}

// "merged, adding their weights": sort by (target pair, a, b), sum equal keys in fp64.
void merge_arcs(std::vector<OutArc> &v) {
    std::stable_sort(v.begin(), v.end(), [](const OutArc &x, const OutArc &y) {
        if (x.r1 != y.r1) return x.r1 < y.r1;
        if (x.r2 != y.r2) return x.r2 < y.r2;
        if (x.a != y.a) return x.a < y.a;
        return x.b < y.b;
    });
    size_t n = 0;
    for (size_t i = 0; i < v.size(); ++i) {
        if (n > 0 && v[n - 1].r1 == v[i].r1 && v[n - 1].r2 == v[i].r2 && v[n - 1].a == v[i].a &&
            v[n - 1].b == v[i].b) {
            v[n - 1].w += v[i].w;
        } else {
            v[n++] = v[i];
        }
    }
    v.resize(n);
}

// Visited set Q that is also the pair -> state number map.
struct Visited {
    bool dense = false;
    std::vector<int64_t> table;                       // -1 = not visited
    std::unordered_map<uint64_t, int64_t> map;
    void init(uint64_t n_pairs, bool force_map) {
        dense = !force_map && n_pairs <= (uint64_t(1) << 28);
        if (dense) table.assign(n_pairs, -1);
    }
    int64_t find(uint64_t k) const {
        if (dense) return table[k];
        auto it = map.find(k);
        return it == map.end() ? -1 : it->second;
    }
    void insert(uint64_t k, int64_t id) {
        if (dense) table[k] = id; else map.emplace(k, id);
    }
};

struct Result {
    // states in creation order; state i is the pair (q1[i], q2[i]); state 0 = (s1, s2)
    std::vector<int32_t> q1, q2, level;
    std::vector<uint8_t> expanded;
    // arcs (kept only when keep_arcs): ids refer to the state list above
    std::vector<int64_t> src, tgt;
    std::vector<int32_t> a, b;
    std::vector<double> w;
    std::vector<int64_t> accept;        // ascending ids
    std::vector<int64_t> level_raw;     // R_l of every level that was at least partly expanded
    std::vector<int64_t> level_size;    // |F_l|
    int64_t n_arcs = 0, n_raw = 0, n_expanded = 0;
    int32_t n_levels = 0, truncated = 0;
    double seconds = 0.0;
};

Result *compose(const InFst &f1, const InFst &f2, int merge, int64_t max_raw_arcs, int max_levels,
                int keep_arcs, int force_map) {
    auto t0 = std::chrono::steady_clock::now();
    Machine m1 = load_machine(f1, 1), m2 = load_machine(f2, 2);
    const uint64_t nq2 = static_cast<uint64_t>(f2.n_states);
    Result *res = new Result();
    Result &R = *res;
    Visited Q;
    Q.init(static_cast<uint64_t>(f1.n_states) * nq2, force_map != 0);

    auto key_of = [&](int32_t a, int32_t b) { return static_cast<uint64_t>(a) * nq2 + static_cast<uint64_t>(b); };
    auto new_state = [&](int32_t a, int32_t b, int32_t lvl) {
        int64_t id = static_cast<int64_t>(R.q1.size());
        R.q1.push_back(a); R.q2.push_back(b); R.level.push_back(lvl); R.expanded.push_back(0);
        Q.insert(key_of(a, b), id);
        return id;
    };

    // Alg. 1 lines 1-3
    std::vector<int64_t> frontier{new_state(f1.start, f2.start, 0)};
    std::vector<OutArc> buf;
    int64_t cum = 0;
    for (int32_t lvl = 0; !frontier.empty(); ++lvl) {
        if (max_levels > 0 && lvl == max_levels) { R.truncated = 1; break; }
        // R_l = Σ raw(p), p ∈ F_l
        std::vector<int64_t> raw(frontier.size());
        int64_t Rl = 0;
        for (size_t i = 0; i < frontier.size(); ++i) {
            raw[i] = raw_count(m1, m2, R.q1[frontier[i]], R.q2[frontier[i]]);
            Rl += raw[i];
        }
        std::vector<int64_t> todo;                     // the pairs of this level that get expanded, in order
        bool stop_after = false;
        if (max_raw_arcs == 0 || cum + Rl <= max_raw_arcs) {
            todo = frontier;
        } else {                                       // rule T: key-ordered maximal prefix
            std::vector<size_t> idx(frontier.size());
            for (size_t i = 0; i < idx.size(); ++i) idx[i] = i;
            std::sort(idx.begin(), idx.end(), [&](size_t x, size_t y) {
                return key_of(R.q1[frontier[x]], R.q2[frontier[x]]) < key_of(R.q1[frontier[y]], R.q2[frontier[y]]);
            });
            int64_t c = cum;
            for (size_t i : idx) {
                if (c + raw[i] > max_raw_arcs) break;
                c += raw[i];
                todo.push_back(frontier[i]);
            }
            R.truncated = 1;
            stop_after = true;
        }
        R.level_size.push_back(static_cast<int64_t>(frontier.size()));
        int64_t level_raw = 0;
        std::vector<int64_t> next;
        for (int64_t s : todo) {                       // Alg. 1 line 5: pop
            expand_pair(m1, m2, R.q1[s], R.q2[s], buf);            // lines 6-8
            level_raw += static_cast<int64_t>(buf.size());
            if (merge) merge_arcs(buf);
            R.expanded[s] = 1;
            R.n_expanded += 1;
            for (const OutArc &e : buf) {
                int64_t t = Q.find(key_of(e.r1, e.r2));             // line 9
                if (t < 0) {                                        // lines 10-11
                    t = new_state(e.r1, e.r2, lvl + 1);
                    next.push_back(t);
                }
                if (keep_arcs) {
                    R.src.push_back(s); R.tgt.push_back(t); R.a.push_back(e.a); R.b.push_back(e.b);
                    R.w.push_back(e.w);
                }
                R.n_arcs += 1;
            }
        }
        R.level_raw.push_back(level_raw);
        R.n_raw += level_raw;
        cum += level_raw;
        R.n_levels = lvl + 1;
        if (stop_after) break;
        frontier.swap(next);
    }
    // accept states: F1×F2 restricted to the created states (N5)
    for (size_t i = 0; i < R.q1.size(); ++i)
        if (m1.is_accept[R.q1[i]] && m2.is_accept[R.q2[i]]) R.accept.push_back(static_cast<int64_t>(i));
    R.seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    return res;
}

}  // namespace

extern "C" {

void *fsto_compose(const InFst *m1, const InFst *m2, int merge, int64_t max_raw_arcs, int max_levels,
                   int keep_arcs, int force_map) {
    return compose(*m1, *m2, merge, max_raw_arcs, max_levels, keep_arcs, force_map);
}

// info[0..7] = n_states, n_arcs, n_raw, n_accept, n_levels, truncated, n_expanded, arcs_kept
void fsto_info(void *h, int64_t *info) {
    Result &R = *static_cast<Result *>(h);
    info[0] = static_cast<int64_t>(R.q1.size());
    info[1] = R.n_arcs;
    info[2] = R.n_raw;
    info[3] = static_cast<int64_t>(R.accept.size());
    info[4] = R.n_levels;
    info[5] = R.truncated;
    info[6] = R.n_expanded;
    info[7] = static_cast<int64_t>(R.src.size());
}

double fsto_seconds(void *h) { return static_cast<Result *>(h)->seconds; }

void fsto_get_states(void *h, int32_t *q1, int32_t *q2, int32_t *level, uint8_t *expanded) {
    Result &R = *static_cast<Result *>(h);
    size_t n = R.q1.size();
    std::memcpy(q1, R.q1.data(), n * 4);
    std::memcpy(q2, R.q2.data(), n * 4);
    std::memcpy(level, R.level.data(), n * 4);
    std::memcpy(expanded, R.expanded.data(), n);
}

void fsto_get_arcs(void *h, int64_t *src, int64_t *tgt, int32_t *a, int32_t *b, double *w) {
    Result &R = *static_cast<Result *>(h);
    size_t n = R.src.size();
    std::memcpy(src, R.src.data(), n * 8);
    std::memcpy(tgt, R.tgt.data(), n * 8);
    std::memcpy(a, R.a.data(), n * 4);
    std::memcpy(b, R.b.data(), n * 4);
    std::memcpy(w, R.w.data(), n * 8);
}

void fsto_get_accept(void *h, int64_t *ids) {
    Result &R = *static_cast<Result *>(h);
    std::memcpy(ids, R.accept.data(), R.accept.size() * 8);
}

// out must hold n_levels entries each
void fsto_get_levels(void *h, int64_t *level_raw, int64_t *level_size) {
    Result &R = *static_cast<Result *>(h);
    std::memcpy(level_raw, R.level_raw.data(), R.level_raw.size() * 8);
    std::memcpy(level_size, R.level_size.data(), R.level_size.size() * 8);
}

void fsto_free(void *h) { delete static_cast<Result *>(h); }

// ---- one pair at a time (sampled checks at sizes where the whole result does not fit the host) ----
// A prepared pair of machines, so that many pairs can be expanded without re-sorting the inputs.
struct Prepared { Machine m1, m2; std::vector<OutArc> buf; };

void *fsto_prepare(const InFst *m1, const InFst *m2) {
    Prepared *p = new Prepared();
    p->m1 = load_machine(*m1, 1);
    p->m2 = load_machine(*m2, 2);
    return p;
}

int64_t fsto_raw_count(void *hp, int32_t q1, int32_t q2) {
    Prepared &P = *static_cast<Prepared *>(hp);
    return raw_count(P.m1, P.m2, q1, q2);
}

// Expands (q1,q2) by the definition; returns the number of (merged) arcs and keeps them for fsto_pair_arcs.
int64_t fsto_expand_pair(void *hp, int32_t q1, int32_t q2, int merge) {
    Prepared &P = *static_cast<Prepared *>(hp);
    expand_pair(P.m1, P.m2, q1, q2, P.buf);
    if (merge) merge_arcs(P.buf);
    return static_cast<int64_t>(P.buf.size());
}

void fsto_pair_arcs(void *hp, int32_t *r1, int32_t *r2, int32_t *a, int32_t *b, double *w) {
    Prepared &P = *static_cast<Prepared *>(hp);
    for (size_t i = 0; i < P.buf.size(); ++i) {
        r1[i] = P.buf[i].r1; r2[i] = P.buf[i].r2; a[i] = P.buf[i].a; b[i] = P.buf[i].b; w[i] = P.buf[i].w;
    }
}

void fsto_prepared_free(void *hp) { delete static_cast<Prepared *>(hp); }

}  // extern "C"
