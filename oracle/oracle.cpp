// oracle.cpp — CPU ORACLE for the SymDel hot path.  TEST INFRASTRUCTURE ONLY.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// build, load or call this file.  It shares no code, header, table or constant with the CUDA
// path under paper_2403_09010_b200/csrc/ (no 5-bit packing, no hashing to integers, no radix
// sort, no bit-parallel distance): variants are exact byte strings, the join is a string-keyed
// multi-value hash map, the distance is the full Wagner-Fischer table.
//
// What it computes (the plain definition the method reaches exactly):
//   self (S, d): every (i, j, lev(S_i, S_j)) with 0 <= i < j < n and lev <= d, ascending (i, j)
//   cross(Q, R, d): every (q, r, lev(Q_q, R_r)) with lev <= d, ascending (q, r)
// by two routes:
//   oracle_bruteforce_*  — "Exhaustive search: the brute-force algorithm comparing all pairs of
//                          sequences" (the paper's own validation reference,
//                          PAPER.md:166).  OpenMP over the OUTER loop only.
//   oracle_symdel_*      — Appendix F.1 "SymDel lookup", step by step, with a
//                          multi-value hash map.  Single-threaded.
//
// Readings of the paper adopted here: A-1 the 0-deletion original is a
// variant; A-3 self-search reports i < j once, never (i, i); A-4 any depth <= d on either side may
// match; A-5 the distance returned is the exact Levenshtein distance; A-7 exact duplicates are
// reported at distance 0; A-8 the empty string is a legal variant and a legal sequence.
//
// Pins (tests/test_oracle_pins.py, none of which calls back into this file for its expected
// value): 55 deletion variants and 79,745 neighbours, CAT/COAT,
// m(m-1)/2, hand-worked Fig. 1 categories, a pure-Python recursive definition of
// the edit distance, symdel == bruteforce on 5,000 sequences at d = 1, 2, 3,
// the bag-of-amino-acids bound.
// Unpinned (data-, key-dependent; reported only): n_variants, n_matched, n_unique counters.

#include <algorithm>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <string>
#include <unordered_map>
#include <vector>

#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

struct Triple {
    int32_t i, j, dist;
};

struct Result {
    std::vector<Triple> out;
    int64_t n_variants = 0;  // number of (v_ij, i) tuples generated (Table S1 "DeletionVariants")
    int64_t n_matched = 0;   // pairs found by step 3 before dedup, distinct ids only
    int64_t n_unique = 0;    // pairs after step 4
};

// Unit-cost Levenshtein distance, textbook Wagner-Fischer recurrence, FULL table, no band, no
// early exit (SURVEY.md §8(c) definition):
//   D[i][0] = i, D[0][j] = j, D[i][j] = min(D[i-1][j-1] + [a_i != b_j], D[i-1][j] + 1, D[i][j-1] + 1)
int lev_full(const int8_t* a, int la, const int8_t* b, int lb) {
    std::vector<int> D((size_t)(la + 1) * (lb + 1));
    auto at = [&](int i, int j) -> int& { return D[(size_t)i * (lb + 1) + j]; };
    for (int i = 0; i <= la; ++i) at(i, 0) = i;
    for (int j = 0; j <= lb; ++j) at(0, j) = j;
    for (int i = 1; i <= la; ++i)
        for (int j = 1; j <= lb; ++j) {
            int sub = at(i - 1, j - 1) + (a[i - 1] != b[j - 1] ? 1 : 0);
            int del = at(i - 1, j) + 1;
            int ins = at(i, j - 1) + 1;
            at(i, j) = std::min(sub, std::min(del, ins));
        }
    return at(la, lb);
}

// Step 1 of App. F.1: all deletion variants of s up to depth d, as strings, one per
// deletion SET (so a variant reachable through several sets appears several times — reading A-2).
// `only_k` >= 0 restricts to deletion sets of exactly that size (used to slice the map by variant
// length, which keeps memory bounded without changing what matches: variants of different lengths
// can never be equal).
void variants_rec(const int8_t* s, int L, int start, int left, std::string& cur, std::vector<bool>& del,
                  std::vector<std::string>& out) {
    if (left == 0) {
        std::string v;
        for (int p = 0; p < L; ++p)
            if (!del[p]) v.push_back((char)s[p]);
        out.push_back(v);
        return;
    }
    for (int p = start; p <= L - left; ++p) {
        del[p] = true;
        variants_rec(s, L, p + 1, left - 1, cur, del, out);
        del[p] = false;
    }
}

void deletion_variants(const int8_t* s, int L, int d, int only_k, std::vector<std::string>& out) {
    out.clear();
    std::string cur;
    std::vector<bool> del((size_t)std::max(L, 1), false);
    for (int k = 0; k <= d && k <= L; ++k) {
        if (only_k >= 0 && k != only_k) continue;
        variants_rec(s, L, 0, k, cur, del, out);
    }
}

inline int seq_len(const int64_t* off, int64_t i) { return (int)(off[i + 1] - off[i]); }

// Steps 4-5 of App. F.1: dedup, distance, threshold.
void dedup_and_verify(std::vector<uint64_t>& pairs, const int8_t* sa, const int64_t* oa, const int8_t* sb,
                      const int64_t* ob, int d, Result& res) {
    res.n_matched = (int64_t)pairs.size();
    std::sort(pairs.begin(), pairs.end());
    pairs.erase(std::unique(pairs.begin(), pairs.end()), pairs.end());
    res.n_unique = (int64_t)pairs.size();
    for (uint64_t p : pairs) {
        int32_t i = (int32_t)(p >> 32), j = (int32_t)(p & 0xffffffffu);
        int dist = lev_full(sa + oa[i], seq_len(oa, i), sb + ob[j], seq_len(ob, j));
        if (dist <= d) res.out.push_back({i, j, dist});
    }
}

}  // namespace

extern "C" {

int oracle_lev(const int8_t* a, int la, const int8_t* b, int lb) { return lev_full(a, la, b, lb); }

// Writes the deletion variants of one sequence, each as: 1 length byte + the residues, back to
// back into `buf` (capacity `cap` bytes).  Returns the number of variants (with multiplicity), or
// -1 if the buffer is too small.
int64_t oracle_deletion_variants(const int8_t* s, int L, int d, int8_t* buf, int64_t cap) {
    std::vector<std::string> v;
    deletion_variants(s, L, d, -1, v);
    int64_t pos = 0;
    for (auto& x : v) {
        if (pos + 1 + (int64_t)x.size() > cap) return -1;
        buf[pos++] = (int8_t)x.size();
        std::memcpy(buf + pos, x.data(), x.size());
        pos += (int64_t)x.size();
    }
    return (int64_t)v.size();
}

// ---- exhaustive search ---------------------------------------------------------
void* oracle_bruteforce_self(const int8_t* seqs, const int64_t* off, int64_t n, int d, int threads) {
    auto* res = new Result();
    std::vector<std::vector<Triple>> rows((size_t)std::max<int64_t>(n, 0));
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#endif
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < n; ++i) {
        int li = seq_len(off, i);
        for (int64_t j = i + 1; j < n; ++j) {
            int lj = seq_len(off, j);
            if (std::abs(li - lj) > d) continue;  // lev >= |ΔL| is immediate from the definition
            int dist = lev_full(seqs + off[i], li, seqs + off[j], lj);
            if (dist <= d) rows[(size_t)i].push_back({(int32_t)i, (int32_t)j, dist});
        }
    }
    for (auto& r : rows) res->out.insert(res->out.end(), r.begin(), r.end());
    return res;
}

void* oracle_bruteforce_cross(const int8_t* qs, const int64_t* qo, int64_t nq, const int8_t* rs, const int64_t* ro,
                              int64_t nr, int d, int threads) {
    auto* res = new Result();
    std::vector<std::vector<Triple>> rows((size_t)std::max<int64_t>(nq, 0));
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#endif
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t q = 0; q < nq; ++q) {
        int lq = seq_len(qo, q);
        for (int64_t r = 0; r < nr; ++r) {
            int lr = seq_len(ro, r);
            if (std::abs(lq - lr) > d) continue;
            int dist = lev_full(qs + qo[q], lq, rs + ro[r], lr);
            if (dist <= d) rows[(size_t)q].push_back({(int32_t)q, (int32_t)r, dist});
        }
    }
    for (auto& r : rows) res->out.insert(res->out.end(), r.begin(), r.end());
    return res;
}

// ---- Hamming mode (NEXT-3, Fig. S3 A/C) ---------------------------------
// The paper benchmarks "Hamming distance, d = 1, 2" without restating the definition; reading A-17:
// the Hamming distance is defined for sequences of EQUAL length as the number of positions at which
// they differ; pairs of unequal length are never neighbours.  Plain double loop, same output order.
static int hamming_plain(const int8_t* a, const int8_t* b, int L) {
    int h = 0;
    for (int t = 0; t < L; ++t) h += a[t] != b[t] ? 1 : 0;
    return h;
}

void* oracle_bruteforce_hamming_self(const int8_t* seqs, const int64_t* off, int64_t n, int d) {
    auto* res = new Result();
    for (int64_t i = 0; i < n; ++i) {
        int li = seq_len(off, i);
        for (int64_t j = i + 1; j < n; ++j) {
            if (seq_len(off, j) != li) continue;
            int dist = hamming_plain(seqs + off[i], seqs + off[j], li);
            if (dist <= d) res->out.push_back({(int32_t)i, (int32_t)j, dist});
        }
    }
    return res;
}

void* oracle_bruteforce_hamming_cross(const int8_t* qs, const int64_t* qo, int64_t nq, const int8_t* rs, const int64_t* ro,
                                      int64_t nr, int d) {
    auto* res = new Result();
    for (int64_t q = 0; q < nq; ++q) {
        int lq = seq_len(qo, q);
        for (int64_t r = 0; r < nr; ++r) {
            if (seq_len(ro, r) != lq) continue;
            int dist = hamming_plain(qs + qo[q], rs + ro[r], lq);
            if (dist <= d) res->out.push_back({(int32_t)q, (int32_t)r, dist});
        }
    }
    return res;
}

// Neighbours of ONE probe sequence among a set (used to sample rows at full config sizes).
void* oracle_bruteforce_row(const int8_t* p, int lp, const int8_t* rs, const int64_t* ro, int64_t nr, int d) {
    auto* res = new Result();
    for (int64_t r = 0; r < nr; ++r) {
        int lr = seq_len(ro, r);
        if (std::abs(lp - lr) > d) continue;
        int dist = lev_full(p, lp, rs + ro[r], lr);
        if (dist <= d) res->out.push_back({0, (int32_t)r, dist});
    }
    return res;
}

// ---- SymDel lookup, App. F.1 ------------------------------------------------
void* oracle_symdel_self(const int8_t* seqs, const int64_t* off, int64_t n, int d) {
    auto* res = new Result();
    int maxL = 0;
    for (int64_t i = 0; i < n; ++i) maxL = std::max(maxL, seq_len(off, i));
    std::vector<uint64_t> pairs;
    std::vector<std::string> vars;
    for (int vl = 0; vl <= maxL; ++vl) {  // one variant length at a time (memory relief only)
        // 1-2. generate all deletion variants (v_ij, i); store v_ij -> {i} in a multi-value hash map
        std::unordered_map<std::string, std::vector<int32_t>> map;
        for (int64_t i = 0; i < n; ++i) {
            int L = seq_len(off, i), k = L - vl;
            if (k < 0 || k > d) continue;
            deletion_variants(seqs + off[i], L, d, k, vars);
            res->n_variants += (int64_t)vars.size();
            for (auto& v : vars) map[v].push_back((int32_t)i);
        }
        // 3. for each (v_ij, i) look up the matched sequence indices i' (reading A-3: keep i < i')
        for (int64_t i = 0; i < n; ++i) {
            int L = seq_len(off, i), k = L - vl;
            if (k < 0 || k > d) continue;
            deletion_variants(seqs + off[i], L, d, k, vars);
            for (auto& v : vars) {
                auto it = map.find(v);
                for (int32_t ip : it->second)
                    if (ip > (int32_t)i) pairs.push_back(((uint64_t)i << 32) | (uint32_t)ip);
            }
        }
    }
    // 4-5. deduplicate {(i, i')}; distance; threshold
    dedup_and_verify(pairs, seqs, off, seqs, off, d, *res);
    return res;
}

void* oracle_symdel_cross(const int8_t* qs, const int64_t* qo, int64_t nq, const int8_t* rs, const int64_t* ro,
                          int64_t nr, int d) {
    auto* res = new Result();
    int maxL = 0;
    for (int64_t i = 0; i < nq; ++i) maxL = std::max(maxL, seq_len(qo, i));
    std::vector<uint64_t> pairs;
    std::vector<std::string> vars;
    for (int vl = 0; vl <= maxL; ++vl) {
        std::unordered_map<std::string, std::vector<int32_t>> map;  // built over the QUERY variants
        for (int64_t q = 0; q < nq; ++q) {
            int L = seq_len(qo, q), k = L - vl;
            if (k < 0 || k > d) continue;
            deletion_variants(qs + qo[q], L, d, k, vars);
            res->n_variants += (int64_t)vars.size();
            for (auto& v : vars) map[v].push_back((int32_t)q);
        }
        if (map.empty()) continue;
        for (int64_t r = 0; r < nr; ++r) {  // the reference variants are streamed through it
            int L = seq_len(ro, r), k = L - vl;
            if (k < 0 || k > d) continue;
            deletion_variants(rs + ro[r], L, d, k, vars);
            res->n_variants += (int64_t)vars.size();
            for (auto& v : vars) {
                auto it = map.find(v);
                if (it == map.end()) continue;
                for (int32_t q : it->second) pairs.push_back(((uint64_t)q << 32) | (uint32_t)r);
            }
        }
    }
    dedup_and_verify(pairs, qs, qo, rs, ro, d, *res);
    return res;
}

// ---- result access -----------------------------------------------------------------------------
int64_t oracle_result_size(void* h) { return (int64_t)((Result*)h)->out.size(); }
void oracle_result_counters(void* h, int64_t* c3) {
    auto* r = (Result*)h;
    c3[0] = r->n_variants, c3[1] = r->n_matched, c3[2] = r->n_unique;
}
void oracle_result_copy(void* h, int32_t* i, int32_t* j, int32_t* dist) {
    auto* r = (Result*)h;
    for (size_t t = 0; t < r->out.size(); ++t) i[t] = r->out[t].i, j[t] = r->out[t].j, dist[t] = r->out[t].dist;
}
void oracle_result_free(void* h) { delete (Result*)h; }
int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
