"""Pins for the CPU oracle.  No GPU, no CUDA path.

Every expected value here comes from the paper (tests/golden/paper_values.txt, cited), from a
closed form, from a hand-worked case, or from an independent pure-Python restatement — never
from the oracle itself.
"""
import itertools
import math
from functools import lru_cache
from pathlib import Path

import numpy as np
import pytest

from paper_2403_09010_b200 import synth

GOLD = Path(__file__).parent / "golden"


def paper_values():
    out = {}
    for line in (GOLD / "paper_values.txt").read_text().splitlines():
        line = line.split("#")[0].strip()
        if line:
            k, v = [x.strip() for x in line.split("=")]
            out[k] = v
    return out


def S(*strings):
    return synth.from_strings(list(strings))


def enc(s):
    return S(s).seqs


def as_set(res):
    i, j, d = res[:3]
    return set(zip(i.tolist(), j.tolist(), d.tolist()))


# ---- independent pure-Python definitions -------------------------------------------------
def py_lev(a, b):
    """Recursive definition on suffixes (not Wagner-Fischer's table)."""

    @lru_cache(maxsize=None)
    def f(i, j):
        if i == len(a):
            return len(b) - j
        if j == len(b):
            return len(a) - i
        return min(f(i + 1, j) + 1, f(i, j + 1) + 1, f(i + 1, j + 1) + (a[i] != b[j]))

    return f(0, 0)


def py_edits1(s, alphabet):
    out = set()
    for p in range(len(s) + 1):
        for c in alphabet:
            out.add(s[:p] + (c,) + s[p:])  # insertion
    for p in range(len(s)):
        out.add(s[:p] + s[p + 1:])  # deletion
        for c in alphabet:
            out.add(s[:p] + (c,) + s[p + 1:])  # substitution
    return out


# ---- P-1 variant count ----------------------------------------------------------------------
def test_p1_variant_count_paper(oracle):
    pv = paper_values()
    v = oracle.deletion_variants(np.arange(1, 11, dtype=np.int8), 2)
    assert len(v) - 1 == int(pv["deletion_variants_L10_d2"])  # 55 without the original
    assert len(set(v)) == len(v)  # all-distinct residues: no repeated variant


@pytest.mark.parametrize("L,d", [(0, 2), (1, 1), (1, 3), (5, 0), (8, 1), (15, 2), (12, 3), (9, 4), (24, 2), (30, 3)])
def test_p1_variant_count_formula(oracle, L, d):
    """sum_{i=1..d} C(L, i) deletion variants (+1 for the original, reading A-1)."""
    s = ((np.arange(L) % 20) + 1).astype(np.int8)
    v = oracle.deletion_variants(s, d)
    assert len(v) == sum(math.comb(L, k) for k in range(0, d + 1))
    assert all(len(x) >= L - d for x in v)


def test_variants_are_exactly_the_subsequences(oracle):
    """Brute force on a tiny input: variants == all subsequences of length >= L-d, with
    multiplicity = number of embeddings' deletion sets."""
    s = enc("ABCAB")
    for d in range(0, 4):
        got = sorted(oracle.deletion_variants(s, d))
        exp = []
        for k in range(0, d + 1):
            for dele in itertools.combinations(range(5), k):
                exp.append(bytes(int(s[p]) for p in range(5) if p not in dele))
        assert got == sorted(exp)


def test_p5_repeats_AAAA(oracle):
    v = oracle.deletion_variants(enc("AAAA"), 2)
    assert len(v) == 11 and len(set(v)) == 3


# ---- P-2 neighbourhood size (pins lev + brute force together) ---------------------------------
def test_p2_neighbourhood_79745(oracle):
    pv = paper_values()
    alphabet = tuple(range(1, 21))
    s = tuple(range(1, 11))  # length 10, all-distinct residues
    e1 = py_edits1(s, alphabet)
    e2 = set(e1)
    for t in e1:
        e2 |= py_edits1(t, alphabet)
    e1.discard(s)
    e2.discard(s)
    assert len(e2) == int(pv["neighbours_L10_d2"])  # the paper's 79,745
    assert len(e1) == 410
    cand = sorted(e2)
    cs = synth.from_padded(
        np.array([list(t) + [0] * (12 - len(t)) for t in cand], dtype=np.int8), np.array([len(t) for t in cand])
    )
    probe = np.array(s, dtype=np.int8)
    j, dist = oracle.bruteforce_row(probe, cs.seqs, cs.offsets, 2)
    assert len(j) == 79745
    exp = np.array([1 if t in e1 else 2 for t in cand])
    assert np.array_equal(dist, exp[j]) and np.array_equal(j, np.arange(len(cand)))
    j1, dist1 = oracle.bruteforce_row(probe, cs.seqs, cs.offsets, 1)
    assert len(j1) == 410 and (dist1 == 1).all()
    # strings at exactly 3 edits that are not within 2 must be rejected at d = 2
    far = [t for t in itertools.islice((u for t2 in cand[::977] for u in py_edits1(t2, alphabet)), 20000) if t not in e2 and t != s]
    fs = synth.from_padded(np.array([list(t) + [0] * (13 - len(t)) for t in far], dtype=np.int8), np.array([len(t) for t in far]))
    jf, _ = oracle.bruteforce_row(probe, fs.seqs, fs.offsets, 2)
    assert len(far) > 1000 and len(jf) == 0


# ---- P-10 lev against an independent definition ------------------------------------------------
def test_p10_lev_exhaustive_small_alphabet(oracle):
    strs = [()]
    for L in range(1, 5):
        strs += list(itertools.product((1, 2, 3), repeat=L))
    for a in strs:
        for b in strs:
            assert oracle.lev(np.array(a, np.int8), np.array(b, np.int8)) == py_lev(a, b)


def test_p10_lev_random_long(oracle):
    rng = np.random.default_rng(7)
    for _ in range(1500):
        la, lb = rng.integers(0, 31, 2)
        a = rng.integers(1, 5, la).astype(np.int8)
        b = a.copy()[: lb] if rng.random() < 0.5 else rng.integers(1, 5, lb).astype(np.int8)
        if b.size and rng.random() < 0.7:
            b = b.copy()
            b[rng.integers(0, b.size)] = 4
        assert oracle.lev(a, b) == py_lev(tuple(a.tolist()), tuple(b.tolist()))


def test_lev_textbook_values(oracle):
    assert oracle.lev(enc("KITTEN"), enc("SITTING")) == 3
    assert oracle.lev(enc("SUNDAY"), enc("SATURDAY")) == 3
    assert oracle.lev(enc("FLAW"), enc("LAWN")) == 2
    assert oracle.lev(enc(""), enc("ABC")) == 3 and oracle.lev(enc("ABC"), enc("")) == 3 and oracle.lev(enc(""), enc("")) == 0
    # asymmetric operands / transposed table would break these
    assert oracle.lev(enc("AB"), enc("ABCDE")) == 3 and oracle.lev(enc("ABCDE"), enc("DE")) == 3


# ---- P-4 prefix example ----------------------------------------------------------
def test_p4_cat_coat(oracle):
    pv = paper_values()
    assert oracle.lev(enc("CAT"), enc("COAT")) == int(pv["lev_CAT_COAT"])
    assert oracle.lev(enc("CAT"), enc("COA")) == int(pv["lev_CAT_COA"])
    ca = bytes(enc(pv["shared_variant_CAT_COA"]).view(np.uint8))
    assert ca in oracle.deletion_variants(enc("CAT"), 1) and ca in oracle.deletion_variants(enc("COA"), 1)


@pytest.mark.parametrize("d,P", [(1, 2), (1, 5), (2, 3), (2, 8), (3, 4), (3, 12)])
def test_p4_prefix_lemma_random_pairs(oracle, d, P):
    """App. B: if lev(u, v) <= d and P > d, the prefixes u[:P], v[:P] share a deletion variant
    within depth d.  Random pairs built by <= d edits; the variants come from the oracle's plain enumeration."""
    rng = np.random.default_rng(1000 * d + P)
    n_checked = 0
    for _ in range(300):
        L = int(rng.integers(1, 16))
        u = rng.integers(1, 5, L).astype(np.int8)  # small alphabet: many repeats
        v = list(u)
        for _e in range(int(rng.integers(0, d + 1))):
            op = int(rng.integers(0, 3))
            if op == 0 and v:
                v[int(rng.integers(0, len(v)))] = int(rng.integers(1, 5))
            elif op == 1:
                v.insert(int(rng.integers(0, len(v) + 1)), int(rng.integers(1, 5)))
            elif v:
                del v[int(rng.integers(0, len(v)))]
        v = np.asarray(v, dtype=np.int8)
        if oracle.lev(u, v) > d:
            continue
        n_checked += 1
        assert set(oracle.deletion_variants(u[:P], d)) & set(oracle.deletion_variants(v[:P], d)), (u, v)
    assert n_checked > 200


# ---- P-3 m(m-1)/2 candidates per group -------------------------------------------
@pytest.mark.parametrize("m", [2, 3, 7, 12])
def test_p3_pairs_per_group(oracle, m):
    letters = "HIJKLMNOPQRS"
    s = S(*[letters[k] + "ACDEFG" for k in range(m)])  # share exactly one variant at d = 1: "ACDEFG"
    i, j, d, c = oracle.symdel_self(s.seqs, s.offsets, 1, with_counters=True)
    assert c["n_matched"] == m * (m - 1) // 2 == c["n_unique"] == len(i)
    assert (d == 1).all()


# ---- P-5 hand-worked Fig. 1 categories ------------------------------------
def shared(oracle, a, b, d):
    return set(oracle.deletion_variants(enc(a), d)) & set(oracle.deletion_variants(enc(b), d))


def names(vs):
    return {"".join(chr(ord("A") + c - 1) for c in v) for v in vs}


def test_p5_insertion_deletion(oracle):  # Fig. 1A
    assert names(shared(oracle, "ACDEF", "ACDF", 1)) == {"ACDF"}
    s = S("ACDEF", "ACDF")
    assert as_set(oracle.symdel_self(s.seqs, s.offsets, 1)) == {(0, 1, 1)}


def test_p5_substitution(oracle):  # Fig. 1B
    assert names(shared(oracle, "ACDEF", "ACGEF", 1)) == {"ACEF"}
    s = S("ACDEF", "ACGEF")
    assert as_set(oracle.symdel_self(s.seqs, s.offsets, 1)) == {(0, 1, 1)}


def test_p5_duplicates(oracle):  # Fig. 1C
    assert names(shared(oracle, "ACDEF", "ACGEF", 2)) == {"ACEF", "ACE", "ACF", "AEF", "CEF"}
    s = S("ACDEF", "ACGEF")
    i, j, d, c = oracle.symdel_self(s.seqs, s.offsets, 2, with_counters=True)
    assert c["n_matched"] == 5 and c["n_unique"] == 1 and as_set((i, j, d)) == {(0, 1, 1)}
    s = S("ACCD", "ACD")  # consecutive character repeat
    i, j, d, c = oracle.symdel_self(s.seqs, s.offsets, 1, with_counters=True)
    assert c["n_matched"] == 2 and c["n_unique"] == 1 and as_set((i, j, d)) == {(0, 1, 1)}


def test_p5_false_positive(oracle):  # Fig. 1D
    assert names(shared(oracle, "AB", "BA", 1)) == {"A", "B"}
    s = S("AB", "BA")
    i, j, d, c = oracle.symdel_self(s.seqs, s.offsets, 1, with_counters=True)
    assert len(i) == 0 and c["n_unique"] == 1
    assert as_set(oracle.symdel_self(s.seqs, s.offsets, 2)) == {(0, 1, 2)}
    s = S("ACDEF", "CDEFA")
    assert "CDEF" in names(shared(oracle, "ACDEF", "CDEFA", 1))
    assert as_set(oracle.symdel_self(s.seqs, s.offsets, 1)) == set()
    assert as_set(oracle.symdel_self(s.seqs, s.offsets, 2)) == {(0, 1, 2)}
    assert as_set(oracle.bruteforce_self(s.seqs, s.offsets, 1)) == set()


def test_p5_empty_variant_and_empty_sequence(oracle):  # reading A-8
    s = S("A", "B")
    assert as_set(oracle.symdel_self(s.seqs, s.offsets, 1)) == {(0, 1, 1)}
    s = S("", "A", "AB", "ABC", "")
    exp = {(0, 1, 1), (0, 2, 2), (0, 4, 0), (1, 2, 1), (1, 3, 2), (1, 4, 1), (2, 3, 1), (2, 4, 2)}
    assert as_set(oracle.symdel_self(s.seqs, s.offsets, 2)) == exp
    assert as_set(oracle.bruteforce_self(s.seqs, s.offsets, 2)) == exp


def test_order_and_orientation(oracle):  # readings A-3, A-10
    s = S("AAAA", "AAAB", "AAAA", "AABA", "CCCC")
    for f in (oracle.symdel_self, oracle.bruteforce_self):
        i, j, d = f(s.seqs, s.offsets, 2)[:3]
        assert (i < j).all()
        key = i.astype(np.int64) * 100 + j
        assert (np.diff(key) > 0).all()
        assert (0, 2, 0) in as_set((i, j, d))  # exact duplicates reported at distance 0 (A-7)
        assert as_set((i, j, d)) == {(0, 1, 1), (0, 2, 0), (0, 3, 1), (1, 2, 1), (1, 3, 2), (2, 3, 1)}


def test_cross_orientation_hand_worked(oracle):
    """(q, r) orientation of the two-set form pinned on the oracle itself by an ASYMMETRIC hand-worked case
    ("for both the query and reference sets"; Fig. 1): the first component indexes
    the query set, the second the reference set, sorted by (q, r).  Q = [ACDF], R = [GGGG, ACDEF, ACDF]:
    ACDF -> ACDEF is one insertion, ACDF = ACDF, and GGGG is four substitutions away."""
    q, r = S("ACDF"), S("GGGG", "ACDEF", "ACDF")
    for f in (oracle.symdel_cross, oracle.bruteforce_cross):
        i, j, d = f(q.seqs, q.offsets, r.seqs, r.offsets, 1)[:3]
        assert list(zip(i.tolist(), j.tolist(), d.tolist())) == [(0, 1, 1), (0, 2, 0)]
        # swapped roles: three queries against one reference -> the indices swap sides
        i, j, d = f(r.seqs, r.offsets, q.seqs, q.offsets, 1)[:3]
        assert list(zip(i.tolist(), j.tolist(), d.tolist())) == [(1, 0, 1), (2, 0, 0)]
    # two queries, asymmetric sizes and a query index > every reference index of its matches
    q2, r2 = S("WWWW", "ACDEF", "CDEFA"), S("ACDF", "CDEF")
    exp = [(1, 0, 1), (1, 1, 1), (2, 1, 1)]  # ACDEF-ACDF (del E), ACDEF-CDEF (del A), CDEFA-CDEF (del A); CDEFA-ACDF = 3
    for f in (oracle.symdel_cross, oracle.bruteforce_cross):
        i, j, d = f(q2.seqs, q2.offsets, r2.seqs, r2.offsets, 1)[:3]
        assert list(zip(i.tolist(), j.tolist(), d.tolist())) == exp


# ---- P-6 exactness: symdel == brute force on 5,000 sequences, d = 1, 2, 3 -------
@pytest.mark.parametrize("family", ["tcr", "bcr"])
@pytest.mark.parametrize("d", [1, 2, 3])
def test_p6_symdel_equals_bruteforce_5000(oracle, family, d):
    s = synth.tcr_set(5000, 100) if family == "tcr" else synth.bcr_set(5000, 101, n_lineages=500)
    a = oracle.bruteforce_self(s.seqs, s.offsets, d)
    b = oracle.symdel_self(s.seqs, s.offsets, d)
    assert len(a[0]) > 50
    for x, y in zip(a, b):
        assert np.array_equal(x, y)


def test_p6_cross_equals_bruteforce(oracle):
    q, r = synth.cross_sets(600, 8000, 103)
    for d in (1, 2):
        a = oracle.bruteforce_cross(q.seqs, q.offsets, r.seqs, r.offsets, d)
        b = oracle.symdel_cross(q.seqs, q.offsets, r.seqs, r.offsets, d)
        assert len(a[0]) > 20
        for x, y in zip(a, b):
            assert np.array_equal(x, y)


def test_p6_repeat_heavy(oracle):
    s = synth.repeat_heavy_set(400, 5, alphabet=2, lo=0, hi=9)
    for d in (0, 1, 2, 3):
        a = oracle.bruteforce_self(s.seqs, s.offsets, d)
        b = oracle.symdel_self(s.seqs, s.offsets, d)
        for x, y in zip(a, b):
            assert np.array_equal(x, y)


# ---- P-7 invariants -----------------------------------------------------------------------------
def test_p7_monotone_symmetry_self_cross(oracle):
    s = synth.tcr_set(1500, 11)
    r3 = oracle.symdel_self(s.seqs, s.offsets, 3)
    for d in (0, 1, 2):
        rd = oracle.symdel_self(s.seqs, s.offsets, d)
        assert as_set(rd) == {t for t in as_set(r3) if t[2] <= d}
    a, b = synth.tcr_set(700, 12), synth.tcr_set(900, 11)
    ab = as_set(oracle.symdel_cross(a.seqs, a.offsets, b.seqs, b.offsets, 2))
    ba = as_set(oracle.symdel_cross(b.seqs, b.offsets, a.seqs, a.offsets, 2))
    assert ab == {(j, i, d) for (i, j, d) in ba}
    ss = as_set(oracle.symdel_cross(s.seqs, s.offsets, s.seqs, s.offsets, 2))
    assert {t for t in ss if t[0] < t[1]} == {t for t in as_set(r3) if t[2] <= 2}
    assert all((i, i, 0) in ss for i in range(s.n))
    # every pair: dist <= d, |ΔL| <= dist, dist == 0 <=> equal strings
    L = s.lengths
    for i, j, d in as_set(r3):
        assert d <= 3 and abs(int(L[i]) - int(L[j])) <= d
        assert (d == 0) == np.array_equal(s.seq(i), s.seq(j))


# ---- P-8 permutation invariance --------------------------------------------------
def test_p8_shuffle_invariance(oracle):
    s = synth.tcr_set(3000, 13)
    base = as_set(oracle.symdel_self(s.seqs, s.offsets, 2))
    perm = np.random.default_rng(5).permutation(s.n)
    sp = s.take(perm)
    got = as_set(oracle.symdel_self(sp.seqs, sp.offsets, 2))
    back = {(min(perm[i], perm[j]), max(perm[i], perm[j]), d) for (i, j, d) in got}
    assert back == base


# ---- P-9 bag-of-amino-acids bound --------------------------------------------
def test_p9_bag_bound(oracle):
    s = synth.bcr_set(3000, 14, n_lineages=300)
    i, j, d = oracle.symdel_self(s.seqs, s.offsets, 3)
    rows, lens = synth.to_padded(s)
    bag = np.stack([(rows == c).sum(1) for c in range(1, 21)], 1).astype(np.float64)
    dist = np.linalg.norm(bag[i] - bag[j], axis=1)
    assert len(i) > 100 and (dist <= math.sqrt(2) * d + 1e-9).all()


# ---- P-10 special cases -------------------------------------------------------------------------
def test_p10_d0_is_duplicate_detection(oracle):
    s = synth.repeat_heavy_set(500, 3, alphabet=2, lo=1, hi=6)
    got = as_set(oracle.symdel_self(s.seqs, s.offsets, 0))
    groups = {}
    for t in range(s.n):
        groups.setdefault(bytes(s.seq(t).view(np.uint8)), []).append(t)
    exp = {(a, b, 0) for g in groups.values() for a, b in itertools.combinations(g, 2)}
    assert got == exp and len(exp) > 100


def test_p10_equal_length_substitutions_hamming(oracle):
    """Sequences = one base string with substitutions only and all-distinct residues per position
    class: the Levenshtein distance equals the Hamming distance when it is <= d and every string has
    the same length and no shift can help (alphabet split by position parity prevents shifts)."""
    rng = np.random.default_rng(9)
    n, L = 300, 12
    base = np.array([(p % 2) * 10 + 1 + (p // 2) % 5 for p in range(L)])
    rows = np.tile(base, (n, 1))
    for t in range(n):
        for p in rng.choice(L, size=rng.integers(0, 3), replace=False):
            rows[t, p] = (p % 2) * 10 + 6 + rng.integers(0, 5)  # stays in the parity class of p
    s = synth.from_padded(rows.astype(np.int8), np.full(n, L))
    i, j, d = oracle.symdel_self(s.seqs, s.offsets, 2)
    ham = (rows[:, None, :] != rows[None, :, :]).sum(-1)
    exp = {(a, b, int(ham[a, b])) for a in range(n) for b in range(a + 1, n) if ham[a, b] <= 2}
    assert as_set((i, j, d)) == exp


# ---- NEXT-3 Hamming mode (Fig. S3 A/C; reading A-17) -----------------------------------
def test_hamming_hand_cases(oracle):
    s = S("CASSL", "CASSL", "CATSL", "CTTSL", "CASS", "ACASS", "LSSAC")
    i, j, d = oracle.hamming_self(s.seqs, s.offsets, 2)
    got = {(int(a), int(b)): int(c) for a, b, c in zip(i, j, d)}
    # equal lengths only: CASS (4) pairs with nothing; ACASS vs CASSL: a shift, 4 mismatches (lev 2) -> not a pair
    assert got == {(0, 1): 0, (0, 2): 1, (1, 2): 1, (0, 3): 2, (1, 3): 2, (2, 3): 1}
    i1, j1, d1 = oracle.hamming_self(s.seqs, s.offsets, 1)
    assert {(int(a), int(b)) for a, b in zip(i1, j1)} == {(0, 1), (0, 2), (1, 2), (2, 3)}


def test_hamming_equals_numpy_all_pairs(oracle):
    """Re-derivation with numpy on padded rows: mismatch counts of equal-length rows."""
    s = synth.tcr_set(1200, 61)
    rows, lens = synth.to_padded(s)
    exp = []
    for a in range(s.n):
        same = np.nonzero(lens[a + 1:] == lens[a])[0] + a + 1
        h = (rows[same] != rows[a]).sum(axis=1)
        exp += [(a, int(b), int(x)) for b, x in zip(same, h) if x <= 2]
    i, j, d = oracle.hamming_self(s.seqs, s.offsets, 2)
    assert list(zip(i.tolist(), j.tolist(), d.tolist())) == exp
    assert len(exp) > 50


def test_hamming_vs_levenshtein_relations(oracle):
    """On equal lengths lev <= hamming; so the Hamming neighbours are a subset of the Levenshtein ones, every
    Levenshtein pair of equal length at distance <= 1 is a Hamming pair at the same distance, and cross agrees
    with self."""
    s = synth.tcr_set(1500, 62)
    hi, hj, hd = oracle.hamming_self(s.seqs, s.offsets, 2)
    li, lj, ld = oracle.bruteforce_self(s.seqs, s.offsets, 2)
    lev = {(int(a), int(b)): int(c) for a, b, c in zip(li, lj, ld)}
    ham = {(int(a), int(b)): int(c) for a, b, c in zip(hi, hj, hd)}
    assert set(ham) <= set(lev) and all(lev[k] <= v for k, v in ham.items())
    L = s.lengths
    for (a, b), v in lev.items():
        if v <= 1 and L[a] == L[b]:
            assert ham[(a, b)] == v
    ci, cj, cd = oracle.hamming_cross(s.seqs, s.offsets, s.seqs, s.offsets, 2)
    assert {(int(a), int(b)): int(c) for a, b, c in zip(ci, cj, cd) if a < b} == ham


# ---- NEXT-4 M x M overlap matrix (reading A-18) ----------------------------------------
def test_overlap_matrix_hand_case_and_invariants(oracle):
    # sequences 0..5 in repertoires [0, 0, 1, 1, 2, 2]; pairs (0,1) within rep 0; (0,2), (1,3) between 0 and 1; (2,4) 1-2
    lab = np.array([0, 0, 1, 1, 2, 2], dtype=np.int32)
    i, j = np.array([0, 0, 1, 2]), np.array([1, 2, 3, 4])
    m = oracle.overlap_matrix(i, j, lab, lab, 3, True)
    assert m.tolist() == [[1, 2, 0], [2, 0, 1], [0, 1, 0]]
    assert (m == m.T).all() and np.triu(m).sum() == len(i)
    # cross form: rows = query repertoires, columns = reference repertoires, no mirroring
    mq = oracle.overlap_matrix(np.array([0, 1, 1]), np.array([5, 5, 0]), np.array([1, 0], np.int32), lab, 3, False)
    assert mq.tolist() == [[1, 0, 1], [0, 0, 1], [0, 0, 0]] and mq.sum() == 3
    # against numpy's scatter-add on a real result
    s = synth.tcr_set(3000, 81)
    ri, rj, _ = oracle.symdel_self(s.seqs, s.offsets, 2)
    labs = (np.arange(s.n) % 5).astype(np.int32)
    ref = np.zeros((5, 5), np.int64)
    np.add.at(ref, (labs[ri], labs[rj]), 1)
    ref = ref + ref.T - np.diag(np.diag(ref))
    assert (oracle.overlap_matrix(ri, rj, labs, labs, 5, True) == ref).all()
