"""Parity of the CUDA path (through the C ABI) with the CPU oracle.  All tests need a B200.

Bar: bit-exact — identical pair sets, identical distances, identical order (integer work).
Element-by-element at sizes the oracle finishes in seconds (several tiles + ragged tails); at the
BASELINE.json full sizes by the stored oracle digests (tests/golden/config_*.json, written by
tests/golden/make_golden.py from the oracle alone) plus sampled rows recomputed by brute force.
"""
import hashlib
import json
from pathlib import Path

import numpy as np
import pytest

from paper_2403_09010_b200 import synth

pytestmark = pytest.mark.gpu
GOLD = Path(__file__).parent / "golden"


@pytest.fixture(scope="module")
def torch():
    import torch as t

    assert t.cuda.is_available(), "gpu tests need a CUDA device"
    return t


@pytest.fixture(scope="module")
def sd(torch):
    from paper_2403_09010_b200 import symdel

    symdel.lib()  # must load: there is no fallback
    return symdel


@pytest.fixture()
def ctx(sd):
    c = sd.Context(0)
    yield c
    c.close()


def run_self(sd, ctx, s, d, **kw):
    ds, do = sd.to_device(s)
    return [t.cpu().numpy() for t in ctx.symdel_self(ds, do, d, **kw)]


def run_cross(sd, ctx, q, r, d, **kw):
    qs, qo = sd.to_device(q)
    rs, ro = sd.to_device(r)
    return [t.cpu().numpy() for t in ctx.symdel_cross(qs, qo, rs, ro, d, **kw)]


def assert_same(got, exp):
    assert len(got[0]) == len(exp[0]), (len(got[0]), len(exp[0]))
    for a, b in zip(got, exp[:3]):
        assert a.dtype == np.int32 and np.array_equal(a, b)


def digest(i, j, d):
    h = hashlib.sha256()
    for a in (i, j, d):
        h.update(np.ascontiguousarray(a, dtype=np.int32).tobytes())
    return h.hexdigest()


def assert_matches_golden(g, i, j, dist):
    """Full-size comparison with the oracle's stored digests (tests/golden/*.json, written by make_golden.py from
    the oracle alone).  Equal sha256 of (i, j, dist) <=> identical pairs, distances and order.  On a mismatch the
    per-block digests locate the first differing block of 4096 output rows and its rows are printed."""
    if digest(i, j, dist) == g["out_sha256"] and len(i) == g["n_out"]:
        return
    B = g["block_rows"]
    rows = np.ascontiguousarray(np.stack([np.asarray(a, dtype=np.int32) for a in (i, j, dist)], axis=1))
    got = [hashlib.sha256(rows[t:t + B].tobytes()).hexdigest()[:12] for t in range(0, len(rows), B)]
    first = next((b for b, (x, y) in enumerate(zip(got, g["block_sha"])) if x != y), min(len(got), len(g["block_sha"])))
    lo = first * B
    raise AssertionError(
        f"output differs from the oracle: {len(i)} rows vs {g['n_out']}; dist histogram "
        f"{np.bincount(dist, minlength=g['d'] + 1).tolist()} vs {g['dist_hist']}; first differing block {first} "
        f"(rows {lo}..{lo + B}); its first rows here:\n{rows[lo:lo + 12]}\n(rows before it are identical; the oracle's rows "
        f"of this block start at i >= {int(rows[lo - 1, 0]) if lo else 0})")


# ---- S2/K2: radix sort -----------------------------------------------------------------------------
def _keys(kind, n, seed):
    rng = np.random.default_rng(seed)
    if kind == "rand":
        return rng.integers(0, 2**64, n, dtype=np.uint64)
    if kind == "equal":
        return np.full(n, 0xDEADBEEF12345678, dtype=np.uint64)
    if kind == "few":
        return rng.integers(0, 3, n, dtype=np.uint64) << np.uint64(20)
    if kind == "sorted":
        return np.sort(rng.integers(0, 2**64, n, dtype=np.uint64))
    if kind == "reverse":
        return np.sort(rng.integers(0, 2**64, n, dtype=np.uint64))[::-1].copy()
    if kind == "onebin":  # every key in one bin except a sprinkle: match-any ranking degenerates
        k = np.zeros(n, dtype=np.uint64)
        k[rng.integers(0, max(n, 1), max(n // 100, 1))] = np.uint64(255)
        return k | (rng.integers(0, 2**32, n, dtype=np.uint64) << np.uint64(32))
    raise ValueError(kind)


@pytest.mark.parametrize("n", [0, 1, 31, 4095, 4096, 4097, 12289, 1_000_003])
def test_sort_sizes(torch, sd, ctx, n):
    k = _keys("rand", n, n)
    t = torch.from_numpy(k.view(np.int64).copy()).cuda()
    ctx.symdel_stage_sort_u64(t, 0, 64)
    assert np.array_equal(t.cpu().numpy().view(np.uint64), np.sort(k, kind="stable"))


@pytest.mark.parametrize("kind", ["equal", "few", "sorted", "reverse", "onebin"])
@pytest.mark.parametrize("bits", [(0, 8), (0, 32), (20, 52), (24, 64)])
def test_sort_stability_and_bit_ranges(torch, sd, ctx, kind, bits):
    b, e = bits
    k = _keys(kind, 70_001, 5)
    t = torch.from_numpy(k.view(np.int64).copy()).cuda()
    ctx.symdel_stage_sort_u64(t, b, e)
    field = (k >> np.uint64(b)) & np.uint64((1 << (e - b)) - 1)
    exp = k[np.argsort(field, kind="stable")]  # stable: ties keep input order
    assert np.array_equal(t.cpu().numpy().view(np.uint64), exp)


def test_sort_many_tiny_tiles_stress(torch, sd, ctx):
    """Look-back stress: many tiles, repeated (the ticket/status protocol must never deadlock or mis-sum)."""
    for rep in range(5):
        k = _keys("rand", 3_000_000 + rep, rep) & np.uint64(0xFFFF)
        t = torch.from_numpy(k.view(np.int64).copy()).cuda()
        ctx.symdel_stage_sort_u64(t, 0, 16)
        assert np.array_equal(t.cpu().numpy().view(np.uint64), np.sort(k, kind="stable"))


# ---- S4/K6: bit-parallel distance --------------------------------------------------------------------
def test_lev_exhaustive_small(torch, sd, ctx, oracle):
    import itertools

    strs = [()]
    for L in range(1, 6):
        strs += list(itertools.product((1, 2, 3), repeat=L))
    rows = np.zeros((len(strs), 5), np.int8)
    lens = np.array([len(s) for s in strs])
    for i, s in enumerate(strs):
        rows[i, :len(s)] = s
    ss = synth.from_padded(rows, lens)
    ia, ib = np.meshgrid(np.arange(ss.n, dtype=np.int32), np.arange(ss.n, dtype=np.int32))
    ia, ib = ia.ravel(), ib.ravel()
    ds, do = sd.to_device(ss)
    got = ctx.symdel_stage_lev(ds, do, ds, do, torch.from_numpy(ia).cuda(), torch.from_numpy(ib).cuda()).cpu().numpy()
    # oracle distances through its brute-force routine with an unreachable threshold
    _, j, dist = oracle.bruteforce_cross(ss.seqs, ss.offsets, ss.seqs, ss.offsets, 99)
    exp = dist.reshape(ss.n, ss.n)  # row q, column r
    assert np.array_equal(got.reshape(ss.n, ss.n).T, exp)
    assert len(ia) == 364 * 364


def test_lev_random_up_to_L_MAX(torch, sd, ctx, oracle):
    rng = np.random.default_rng(1)
    n = 3000
    lens = rng.integers(0, 65, n)
    lens[:4] = (0, 64, 32, 33)
    rows = rng.integers(1, 5, (n, 64)).astype(np.int8)
    rows[n // 2:] = rows[: n - n // 2]  # near-duplicates: small distances as well as large
    flip = rng.random((n, 64)) < 0.05
    rows[flip] = rng.integers(1, 32, flip.sum())
    rows[np.arange(64)[None, :] >= lens[:, None]] = 0
    ss = synth.from_padded(rows, lens)
    ia = rng.integers(0, n, 30000).astype(np.int32)
    ib = np.where(rng.random(30000) < 0.5, (ia + n // 2) % n, rng.integers(0, n, 30000)).astype(np.int32)
    ds, do = sd.to_device(ss)
    got = ctx.symdel_stage_lev(ds, do, ds, do, torch.from_numpy(ia).cuda(), torch.from_numpy(ib).cuda()).cpu().numpy()
    exp = np.array([oracle.lev(ss.seq(a), ss.seq(b)) for a, b in zip(ia, ib)])
    assert np.array_equal(got, exp)


# ---- S1/K1: variant generation -----------------------------------------------------------------------
def test_generate_fast_and_general_paths_agree(torch, sd, oracle):
    """The d <= 2 warp-per-batch kernel and the general kernel compute the same hash function and the
    same thinning: identical record multisets per sequence (their enumeration orders differ)."""
    s = synth.SeqSet(*[np.concatenate(x) for x in zip(
        (synth.tcr_set(3000, 5).seqs, synth.tcr_set(3000, 5).offsets[:-1]),
        (synth.repeat_heavy_set(500, 6, alphabet=2, lo=0, hi=32).seqs,
         synth.repeat_heavy_set(500, 6, alphabet=2, lo=0, hi=32).offsets + synth.tcr_set(3000, 5).offsets[-1]))])
    ds, do = sd.to_device(s)
    for d in (0, 1, 2):
        for thinning in (True, False):
            recs = []
            for general in (0, 1):
                c = sd.Context(0)
                c.symdel_set_option(sd.OPT_GENERAL_GENERATE, general)
                r = c.symdel_stage_generate(ds, do, d, 40, 13, thinning, 4_000_000).cpu().numpy().view(np.uint64)
                assert (np.diff((r & np.uint64(8191)).astype(np.int64)) >= 0).all()
                recs.append(np.sort(r))
            assert np.array_equal(recs[0], recs[1]), (d, thinning)


@pytest.mark.parametrize("d", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("thinning", [True, False])
def test_generate_groups_match_oracle_variants(torch, sd, ctx, oracle, d, thinning):
    """The multiset of id-groups sharing a key equals the oracle's groups sharing a variant string
    (hash consistent and collision-free at 48 bits on this input); record count = number of distinct
    (variant, id) with thinning (P-11), = sum C(L, k) without."""
    s = synth.repeat_heavy_set(70, 3, alphabet=3, lo=0, hi=9 if d < 4 else 8)
    ds, do = sd.to_device(s)
    id_bits, hash_bits = 8, 48
    rec = ctx.symdel_stage_generate(ds, do, d, hash_bits, id_bits, thinning, 1 << 20).cpu().numpy().view(np.uint64)
    ids = (rec & np.uint64(255)).astype(np.int64)
    keys = rec >> np.uint64(id_bits)
    assert (np.diff(ids) >= 0).all()  # written in id order
    var = [oracle.deletion_variants(s.seq(i), d) for i in range(s.n)]
    if thinning:
        exp_cnt = np.array([len(set(v)) for v in var])
    else:
        exp_cnt = np.array([len(v) for v in var])
    assert np.array_equal(np.bincount(ids, minlength=s.n), exp_cnt)
    got_groups = {}
    for k, i in zip(keys.tolist(), ids.tolist()):
        got_groups.setdefault(k, []).append(i)
    exp_groups = {}
    for i, v in enumerate(var):
        for x in (set(v) if thinning else v):
            exp_groups.setdefault(x, []).append(i)
    assert sorted(map(tuple, got_groups.values())) == sorted(map(tuple, (sorted(g) for g in exp_groups.values())))


def _fused_records(ctx, ds, do, d, hash_bits, id_bits, thinning, cap, **kw):
    """Records of the fused generator, bin by bin; checks that every record sits in the bin of its top 8 hash bits."""
    bins, counts = ctx.symdel_stage_generate_fused(ds, do, d, hash_bits, id_bits, thinning, cap, **kw)
    bins, counts = bins.cpu().numpy().view(np.uint64), counts.cpu().numpy()
    assert counts.max(initial=0) <= cap
    rec = np.concatenate([bins[b, :counts[b]] for b in range(256)])
    where = np.repeat(np.arange(256, dtype=np.uint64), counts)
    assert np.array_equal((rec >> np.uint64(id_bits + hash_bits - 8)) & np.uint64(255), where)
    return rec


@pytest.mark.parametrize("d", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("thinning", [True, False])
@pytest.mark.parametrize("mode", ["plain", "narrow", "general"])
def test_fused_generate_bins_match_oracle_variants(torch, sd, oracle, d, thinning, mode):
    """Kernel-level pin of the generators of the DEFAULT pipeline (k_gen2_part for d <= 3, k_generate_part for d = 4 or
    on request): the records they push into the level-1 bins, gathered, form the same multiset of id-groups per key as
    the oracle's deletion-variant strings (App. F.1 step 1) — the comparison of
    test_generate_groups_match_oracle_variants, on the fused kernels — and every record lies in the bin of its digit."""
    s = synth.repeat_heavy_set(70, 3, alphabet=3, lo=0, hi=9 if d < 4 else 8)
    ds, do = sd.to_device(s)
    id_bits, hash_bits = (8, 56) if mode == "plain" else (8, 48)
    c = sd.Context(0)
    if mode == "general":
        c.symdel_set_option(sd.OPT_GENERAL_GENERATE, 1)
    rec = _fused_records(c, ds, do, d, hash_bits, id_bits, thinning, 4096)
    c.close()
    ids = (rec & np.uint64(255)).astype(np.int64)
    keys = rec >> np.uint64(id_bits)
    var = [oracle.deletion_variants(s.seq(i), d) for i in range(s.n)]
    exp_cnt = np.array([len(set(v)) if thinning else len(v) for v in var])
    assert np.array_equal(np.bincount(ids, minlength=s.n), exp_cnt)
    got_groups = {}
    for k, i in zip(keys.tolist(), ids.tolist()):
        got_groups.setdefault(k, []).append(i)
    exp_groups = {}
    for i, v in enumerate(var):
        for x in (set(v) if thinning else v):
            exp_groups.setdefault(x, []).append(i)
    assert sorted(tuple(sorted(g)) for g in got_groups.values()) == sorted(tuple(sorted(g)) for g in exp_groups.values())


@pytest.mark.parametrize("family,d,general", [("tcr", 1, 0), ("tcr", 2, 0), ("tcr", 2, 1), ("bcr", 3, 0), ("bcr", 3, 1), ("bcr", 4, 0),
                                              ("long", 2, 0)])
def test_fused_generate_equals_exact_generate_and_chunks_partition_it(torch, sd, family, d, general):
    """Many blocks, rounds and flushes: the fused generators make exactly the records of the exact generator (which the
    oracle pins above), and the key-range-chunk instances (S5) split that set: the chunks are disjoint and their union
    is the whole — for a cut inside a variant length (hash fraction) and for cuts at length boundaries."""
    if family == "tcr":
        s = synth.tcr_set(20000, 5)
    elif family == "bcr":
        s = synth.bcr_set(2500 if d == 3 else 600, 6, n_lineages=300)
    else:  # longer than 32 residues: the 64-residue rows of the general kernel
        rng = np.random.default_rng(8)
        lens = rng.integers(20, 45, size=3000).astype(np.int32)
        rows = rng.integers(1, 21, size=(3000, 44)).astype(np.int8)
        rows[np.arange(44)[None, :] >= lens[:, None]] = 0
        s = synth.from_padded(rows, lens)
    ds, do = sd.to_device(s)
    id_bits, hash_bits = 16, 48
    c = sd.Context(0)
    if general:
        c.symdel_set_option(sd.OPT_GENERAL_GENERATE, 1)
    exact = np.sort(c.symdel_stage_generate(ds, do, d, hash_bits, id_bits, True, 1 << 26).cpu().numpy().view(np.uint64))
    cap = ((len(exact) // 256 * 3) // 2 + 4096) // 32 * 32
    whole = np.sort(_fused_records(c, ds, do, d, hash_bits, id_bits, True, cap))
    assert np.array_equal(whole, exact)
    vl = int(np.median(s.lengths)) - 1
    cuts = [0, (vl - 1) << 32, (vl << 32) | 0x5555_5555, (vl + 1) << 32, (1 << 64) - 1]
    parts = [_fused_records(c, ds, do, d, hash_bits, id_bits, True, cap, n_chunks=4, chunk_lo=lo, chunk_hi=hi)
             for lo, hi in zip(cuts[:-1], cuts[1:])]
    c.close()
    assert all(len(p) for p in parts)
    assert np.array_equal(np.sort(np.concatenate(parts)), exact)  # disjoint (equal multisets) and complete


# ---- full path: small / structured inputs -------------------------------------------------------------
def test_hand_worked_cases(sd, ctx, oracle):
    s = synth.from_strings(["ACDEF", "ACDF", "ACGEF", "AB", "BA", "", "A", "ACCD", "ACD", "AAAA", "AAA", "CDEFA", "B"])
    for d in range(0, 5):
        assert_same(run_self(sd, ctx, s, d), oracle.bruteforce_self(s.seqs, s.offsets, d))


def test_degenerate_inputs(torch, sd, ctx, oracle):
    one = synth.from_strings(["ACD"])
    assert len(run_self(sd, ctx, one, 2)[0]) == 0
    empties = synth.from_strings(["", "", ""])
    assert_same(run_self(sd, ctx, empties, 1), oracle.bruteforce_self(empties.seqs, empties.offsets, 1))
    same = synth.from_strings(["ACDEFGH"] * 40)  # one long run: 780 pairs at distance 0
    got = run_self(sd, ctx, same, 2)
    assert_same(got, oracle.bruteforce_self(same.seqs, same.offsets, 2))
    assert len(got[0]) == 780 and (got[2] == 0).all()
    # n = 0 through the raw ABI
    z8 = torch.zeros(1, dtype=torch.int8, device="cuda")
    z64 = torch.zeros(1, dtype=torch.int64, device="cuda")
    assert len(ctx.symdel_self(z8, z64, 2)[0]) == 0
    # maximum length 64 and d = 4
    rng = np.random.default_rng(3)
    rows = np.tile(rng.integers(1, 21, (1, 64)), (12, 1)).astype(np.int8)
    for t in range(1, 12):
        rows[t, rng.integers(0, 64, t % 5)] = 20 + t
    lens = np.full(12, 64)
    lens[5:] = 63
    big = synth.from_padded(rows, lens)
    assert_same(run_self(sd, ctx, big, 4), oracle.bruteforce_self(big.seqs, big.offsets, 4))


def test_error_codes(torch, sd, ctx):
    s = synth.tcr_set(200, 1)
    ds, do = sd.to_device(s)
    bad = ds.clone()
    bad[5] = 0
    with pytest.raises(sd.SymdelError) as e:
        ctx.symdel_self(bad, do, 1)
    assert e.value.code == sd.E_RESIDUE
    bad_off = do.clone()
    bad_off[3] = bad_off[4] + 1
    with pytest.raises(sd.SymdelError) as e:
        ctx.symdel_self(ds, bad_off, 1)
    assert e.value.code == sd.E_OFFSETS
    long = synth.from_padded(np.ones((2, 70), np.int8), np.array([70, 70]))
    ls, lo = sd.to_device(long)
    with pytest.raises(sd.SymdelError) as e:
        ctx.symdel_self(ls, lo, 1)
    assert e.value.code == sd.E_TOO_LONG
    with pytest.raises(sd.SymdelError) as e:
        ctx.symdel_self(ds, do, 5)
    assert e.value.code == sd.E_ARG
    with pytest.raises(sd.SymdelError) as e:
        ctx.symdel_self(ds, do, 2, capacity=3)
    assert e.value.code == sd.E_CAPACITY and ctx.last_required > 3
    with pytest.raises(sd.SymdelError) as e:
        ctx.symdel_self(ds, do, 2, workspace=torch.empty(4096, dtype=torch.uint8, device="cuda"))
    assert e.value.code == sd.E_WORKSPACE


@pytest.mark.parametrize("d", [0, 1, 2, 3, 4])
def test_repeat_heavy(sd, ctx, oracle, d):
    s = synth.repeat_heavy_set(400, 5, alphabet=2, lo=0, hi=9)
    assert_same(run_self(sd, ctx, s, d), oracle.bruteforce_self(s.seqs, s.offsets, d))


@pytest.mark.parametrize("family", ["tcr", "bcr"])
@pytest.mark.parametrize("d", [1, 2, 3])
def test_validation_protocol_5000(sd, ctx, oracle, family, d):
    """5,000 sequences at d = 1, 2, 3 against the brute-force double loop."""
    s = synth.tcr_set(5000, 100) if family == "tcr" else synth.bcr_set(5000, 101, n_lineages=500)
    assert_same(run_self(sd, ctx, s, d), oracle.bruteforce_self(s.seqs, s.offsets, d))


@pytest.mark.parametrize("opts", [
    {}, {"FORCE_CHUNKS": 4}, {"FORCE_CHUNKS": 16}, {"CAND_CAPACITY": 4999}, {"HASH_BITS": 8}, {"HASH_BITS": 48},
    {"NO_THINNING": 1}, {"FORCE_CHUNKS": 3, "CAND_CAPACITY": 777, "HASH_BITS": 16}, {"GENERAL_GENERATE": 1},
    {"GENERAL_GENERATE": 1, "FORCE_CHUNKS": 5}, {"SORT_VARIANT": 1}, {"SORT_VARIANT": 3},
    {"SORT_BITS": 255}, {"SORT_BITS": 8}, {"SORT_BITS": 24}, {"SORT_BITS": 40}, {"SORT_STABLE": 1},
    {"SORT_BITS": 255, "CAND_CAPACITY": 1500}, {"HASH_BITS": 13, "SORT_BITS": 8},
    {"SORT_BITS": 8, "HASH_BITS": 12, "CAND_CAPACITY": 100000, "FORCE_CHUNKS": 2},
    {"JOIN_GENERAL": 1}, {"JOIN_GENERAL": 1, "FORCE_CHUNKS": 3}, {"JOIN_GENERAL": 1, "SORT_BITS": 255},
    {"EXACT_PIPELINE": 1}, {"EXACT_PIPELINE": 1, "FORCE_CHUNKS": 2},
    {"CAND_FILTER": 1}, {"CAND_FILTER": 2}, {"CAND_FILTER": 1, "FORCE_CHUNKS": 3, "CAND_CAPACITY": 2000},
    {"CAND_FILTER": 1, "EXACT_PIPELINE": 1, "CAND_CAPACITY": 5000}, {"CAND_FILTER": 1, "HASH_BITS": 16},
    {"FORCE_CHUNKS": 4, "FLUSH_PER_CHUNK": 1}, {"FORCE_CHUNKS": 16, "FLUSH_PER_CHUNK": 1},
    {"FORCE_CHUNKS": 3, "CAND_CAPACITY": 777, "FLUSH_PER_CHUNK": 1},
])
def test_output_invariant_under_chunks_windows_and_key_width(sd, oracle, opts):
    """P-11: chunk count, candidate-buffer windows, key width and thinning change memory use and
    candidate counts only, never the result."""
    s = synth.tcr_set(6000, 21)
    exp = oracle.symdel_self(s.seqs, s.offsets, 2)
    c = sd.Context(0)
    for k, v in opts.items():
        c.symdel_set_option(getattr(sd, "OPT_" + k), v)
    try:
        assert_same(run_self(sd, c, s, 2), exp)
    finally:
        c.symdel_set_option(sd.OPT_SORT_VARIANT, 0)  # process-wide hook: restore
    st = c.symdel_get_stats()
    if "FORCE_CHUNKS" in opts:
        assert st["n_chunks"] == opts["FORCE_CHUNKS"]
    if set(opts) == {"FORCE_CHUNKS"}:
        assert st["n_flushes"] == 1  # S5: the chunks append to one candidate window, flushed after the last chunk
    if set(opts) == {"FORCE_CHUNKS", "FLUSH_PER_CHUNK"}:
        assert st["n_flushes"] == st["n_chunks"]
    if "CAND_CAPACITY" in opts:
        assert st["n_flushes"] > 1
        if set(opts) <= {"CAND_CAPACITY", "FORCE_CHUNKS", "CAND_FILTER", "HASH_BITS", "FLUSH_PER_CHUNK"}:
            # the pairs exceed one window: the bucket join runs again over the buckets that did not fit (fused all the way)
            assert st["join_windows"] >= 1 and st["join_general"] == 0 and st["fused_chunks"] == st["n_chunks"]
        else:
            assert st["join_general"] >= 1  # exact pipeline: the fast join kernel hands over to the windowed one
    if "JOIN_GENERAL" in opts:
        assert st["join_general"] == st["n_chunks"]
    if (not opts or set(opts) <= {"FORCE_CHUNKS", "HASH_BITS", "NO_THINNING"}) and opts.get("HASH_BITS", 64) >= 16:
        assert st["join_general"] == 0  # (a hash of 8 bits piles thousands of records on each key: the lists overflow)
        assert st["fused_chunks"] == st["n_chunks"]
    if "EXACT_PIPELINE" in opts or "SORT_BITS" in opts:
        assert st["fused_chunks"] == 0
    if set(opts) <= {"GENERAL_GENERATE", "FORCE_CHUNKS"} and "GENERAL_GENERATE" in opts:
        assert st["fused_chunks"] == st["n_chunks"]  # k_generate_part: the general generator, fused


@pytest.mark.parametrize("copies,sort_bits,general,expect_general", [
    (10, 0, 0, 0),     # dense but inside one window and the list capacity: the fast kernel finishes
    (10, 255, 0, 1),   # one bucket: the first tile lists every record, overflows, hands over
    (40, 0, 0, 1),     # 40 copies overflow the fixed-capacity buckets (exact pipeline); 3.7 M pairs: more than its default window
    (40, 0, 1, 1),
])
def test_join_dense_runs(sd, oracle, copies, sort_bits, general, expect_general):
    """Many sequences under one variant (m(m-1)/2 pairs per shared variant): exact copies of
    each of 200 sequences, d = 1, so nearly every record has partners.  Whichever kernel finishes the
    join, the result is the brute-force one."""
    base = synth.tcr_set(200, 31)
    rep = base.take(np.repeat(np.arange(base.n), copies))
    c = sd.Context(0)
    c.symdel_set_option(sd.OPT_JOIN_GENERAL, general)
    c.symdel_set_option(sd.OPT_SORT_BITS, sort_bits)
    assert_same(run_self(sd, c, rep, 1), oracle.bruteforce_self(rep.seqs, rep.offsets, 1))
    st = c.symdel_get_stats()
    assert st["join_general"] == expect_general
    if copies == 10 and sort_bits == 0:
        assert st["fused_chunks"] == 1  # the bucket join has no candidate list to overflow: dense buckets stay fused


def test_fused_bin_overflow_falls_back(sd, oracle):
    """The fused pipeline sizes its bins for hash-uniform keys.  100 exact copies of each of 600 sequences
    at d = 0 (one record per sequence) pile whole groups of 100 onto single hash values: some bin runs
    full, the chunk is redone by the exact pipeline, the result is the same (reading A-7)."""
    base = synth.tcr_set(600, 33)
    rep = base.take(np.repeat(np.arange(base.n), 100))
    c = sd.Context(0)
    exp = oracle.symdel_self(rep.seqs, rep.offsets, 0)
    assert_same(run_self(sd, c, rep, 0, capacity=4_000_000), exp)
    assert c.symdel_get_stats()["fused_chunks"] == 0
    assert len(exp[0]) == base.n * 100 * 99 // 2


@pytest.mark.parametrize("family,d,P,opts", [
    ("tcr", 1, 2, {}), ("tcr", 2, 3, {}), ("tcr", 2, 8, {}), ("tcr", 2, 12, {"FORCE_CHUNKS": 3}), ("tcr", 2, 18, {"EXACT_PIPELINE": 1}),
    ("tcr", 2, 10, {"EXACT_PIPELINE": 1}), ("bcr", 3, 12, {}), ("bcr", 3, 4, {}), ("bcr", 2, 18, {}), ("bcr", 1, 40, {}),
])
def test_prefix_truncation_is_exact(sd, oracle, family, d, P, opts):
    """NEXT-1 / App. B: generating the variants of the first P > d residues only, and
    verifying on the whole sequences, returns exactly the same pairs — with fewer records."""
    s = synth.tcr_set(6000, 41) if family == "tcr" else synth.bcr_set(4000, 42, n_lineages=400)
    exp = oracle.symdel_self(s.seqs, s.offsets, d)
    c = sd.Context(0)
    assert_same(run_self(sd, c, s, d), exp)
    full = c.symdel_get_stats()["n_records"]
    c.symdel_set_option(sd.OPT_PREFIX_LEN, P)
    for k, v in opts.items():
        c.symdel_set_option(getattr(sd, "OPT_" + k), v)
    assert_same(run_self(sd, c, s, d), exp)
    if P < int(s.lengths.min()):
        assert c.symdel_get_stats()["n_records"] < full


def test_prefix_not_longer_than_threshold_is_rejected(sd, ctx):
    s = synth.tcr_set(100, 43)
    ctx.symdel_set_option(sd.OPT_PREFIX_LEN, 2)
    with pytest.raises(sd.SymdelError) as e:
        run_self(sd, ctx, s, 2)
    assert e.value.code == sd.E_ARG


def test_prefix_truncation_cross(sd, oracle):
    q, r = synth.cross_sets(400, 6000, 44)
    exp = oracle.symdel_cross(q.seqs, q.offsets, r.seqs, r.offsets, 2)
    c = sd.Context(0)
    c.symdel_set_option(sd.OPT_PREFIX_LEN, 9)
    assert_same(run_cross(sd, c, q, r, 2), exp)


@pytest.mark.parametrize("d,fanout,opts", [(1, 64, {}), (2, 64, {}), (2, 16, {"EXACT_PIPELINE": 1}), (2, 200, {}),
                                           (2, 64, {"CAND_CAPACITY": 200000}), (2, 64, {"CAND_FILTER": 1}),
                                           (2, 200, {"CAND_FILTER": 1, "CAND_CAPACITY": 300000})])
def test_dense_neighbourhoods(sd, oracle, d, fanout, opts):
    """NEXT-2: clusters of near-identical sequences (candidates ~ records, long runs of one variant, most records
    with partners: PAPER.md:96, 287-294).  Same bit-exact bar against the oracle's hash-map SymDel."""
    s = synth.dense_set(12000, 51, fanout=fanout)
    exp = oracle.symdel_self(s.seqs, s.offsets, d)
    c = sd.Context(0)
    for k, v in opts.items():
        c.symdel_set_option(getattr(sd, "OPT_" + k), v)
    assert_same(run_self(sd, c, s, d, capacity=len(exp[0]) + 16), exp)
    st = c.symdel_get_stats()
    assert st["n_candidates"] > st["n_records"] // 20


@pytest.mark.parametrize("family,d,opts", [("tcr", 1, {}), ("tcr", 2, {}), ("tcr", 2, {"EXACT_PIPELINE": 1, "FORCE_CHUNKS": 2}),
                                           ("bcr", 3, {}), ("dense", 2, {}), ("tcr", 2, {"PREFIX_LEN": 9})])
def test_hamming_mode(sd, oracle, family, d, opts):
    """NEXT-3 (Fig. S3 A/C): equal-length pairs with <= d mismatches, against the oracle's plain
    double loop."""
    s = {"tcr": lambda: synth.tcr_set(5000, 71), "bcr": lambda: synth.bcr_set(4000, 72, n_lineages=400),
         "dense": lambda: synth.dense_set(5000, 73)}[family]()
    c = sd.Context(0)
    c.symdel_set_option(sd.OPT_METRIC, sd.METRIC_HAMMING)
    for k, v in opts.items():
        c.symdel_set_option(getattr(sd, "OPT_" + k), v)
    exp = oracle.hamming_self(s.seqs, s.offsets, d)
    assert len(exp[0]) > 100
    assert_same(run_self(sd, c, s, d), exp)


def test_hamming_mode_cross_and_long(sd, oracle):
    q, r = synth.cross_sets(500, 5000, 74)
    c = sd.Context(0)
    c.symdel_set_option(sd.OPT_METRIC, sd.METRIC_HAMMING)
    assert_same(run_cross(sd, c, q, r, 2), oracle.hamming_cross(q.seqs, q.offsets, r.seqs, r.offsets, 2))
    s = synth.bcr_set(1500, 75, n_lineages=100, lo=30, hi=60, mean=45.0, sd=6.0)  # 64-bit plane words
    assert_same(run_self(sd, c, s, 2), oracle.hamming_self(s.seqs, s.offsets, 2))


@pytest.mark.parametrize("M", [1, 2, 7, 64, 100])
def test_overlap_matrix(torch, sd, ctx, oracle, M):
    """NEXT-4: M x M repertoire-overlap matrix of the neighbour pairs, self and cross form."""
    s = synth.tcr_set(6000, 91)
    ds, do = sd.to_device(s)
    i, j, _ = ctx.symdel_self(ds, do, 2)
    labs = np.random.default_rng(M).integers(0, M, s.n).astype(np.int32)
    lt = torch.from_numpy(labs).cuda()
    got = ctx.symdel_overlap_matrix(i, j, lt, lt, M, True).cpu().numpy()
    assert (got == oracle.overlap_matrix(i.cpu().numpy(), j.cpu().numpy(), labs, labs, M, True)).all()
    q, r = synth.cross_sets(500, 5000, 92)
    qi, rj, _ = ctx.symdel_cross(*sd.to_device(q), *sd.to_device(r), 2)
    lq = np.random.default_rng(M + 1).integers(0, M, q.n).astype(np.int32)
    lr = np.random.default_rng(M + 2).integers(0, M, r.n).astype(np.int32)
    got = ctx.symdel_overlap_matrix(qi, rj, torch.from_numpy(lq).cuda(), torch.from_numpy(lr).cuda(), M, False).cpu().numpy()
    assert (got == oracle.overlap_matrix(qi.cpu().numpy(), rj.cpu().numpy(), lq, lr, M, False)).all()
    if M > 1:
        with pytest.raises(sd.SymdelError) as e:
            ctx.symdel_overlap_matrix(i, j, lt, lt, M - 1, True)  # some label == M - 1 is out of range
        assert e.value.code == sd.E_ARG


@pytest.mark.parametrize("d,opts", [(2, {}), (3, {}), (4, {}), (4, {"EXACT_PIPELINE": 1}), (3, {"FORCE_CHUNKS": 3}),
                                    (4, {"PREFIX_LEN": 20})])
def test_long_sequences_up_to_the_limits(sd, oracle, d, opts):
    """Edge of the limits: lengths 33..64 = SYMDEL_L_MAX (general generator, 64-bit verifier words) up to
    d = 4 = SYMDEL_D_MAX (V(64, 4) = 679,121 deletion sets per sequence), against brute force."""
    s = synth.bcr_set(60, 95, n_lineages=6, lo=33, hi=64, mean=50.0, sd=10.0, kmax=4)
    assert s.lengths.max() > 56
    c = sd.Context(0)
    for k, v in opts.items():
        c.symdel_set_option(getattr(sd, "OPT_" + k), v)
    exp = oracle.bruteforce_self(s.seqs, s.offsets, d)
    assert len(exp[0]) > 20
    assert_same(run_self(sd, c, s, d), exp)


@pytest.mark.parametrize("family,d", [("tcr", 2), ("bcr", 3), ("dense", 1)])
def test_pipelines_agree_on_stage_counters(sd, family, d):
    """The fused and the exact pipeline use the same hash and the same thinning rule: beyond the identical output,
    the number of records, of candidate pairs and of unique candidates must coincide (they are unpinned against
    the paper, but pinned against each other)."""
    s = {"tcr": lambda: synth.tcr_set(8000, 97), "bcr": lambda: synth.bcr_set(3000, 98, n_lineages=300),
         "dense": lambda: synth.dense_set(8000, 99)}[family]()
    stats, outs = [], []
    for exact in (0, 1):
        c = sd.Context(0)
        c.symdel_set_option(sd.OPT_EXACT_PIPELINE, exact)
        outs.append(run_self(sd, c, s, d))
        stats.append(c.symdel_get_stats())
    assert_same(outs[0], outs[1])
    assert stats[0]["fused_chunks"] == 1 and stats[1]["fused_chunks"] == 0
    for k in ("n_records", "n_candidates", "n_unique", "n_outputs"):
        assert stats[0][k] == stats[1][k], k


def test_small_workspace_forces_chunking(torch, sd, ctx, oracle):
    s = synth.tcr_set(20000, 22)
    exp = oracle.symdel_self(s.seqs, s.offsets, 2)
    ds, do = sd.to_device(s)
    ws = torch.empty(24 << 20, dtype=torch.uint8, device="cuda")  # ~1/3 of the un-chunked need
    got = [t.cpu().numpy() for t in ctx.symdel_self(ds, do, 2, workspace=ws, capacity=200_000)]
    assert_same(got, exp)
    assert ctx.symdel_get_stats()["n_chunks"] > 1


def test_shuffle_invariance(sd, ctx):
    """results invariant under random shuffling of the input."""
    s = synth.tcr_set(8000, 23)
    i, j, d = run_self(sd, ctx, s, 2)
    perm = np.random.default_rng(1).permutation(s.n)
    i2, j2, d2 = run_self(sd, ctx, s.take(perm), 2)
    a = {(int(x), int(y), int(z)) for x, y, z in zip(i, j, d)}
    b = {(int(min(perm[x], perm[y])), int(max(perm[x], perm[y])), int(z)) for x, y, z in zip(i2, j2, d2)}
    assert a == b


@pytest.mark.parametrize("d", [1, 2])
def test_cross_small(sd, ctx, oracle, d):
    q, r = synth.cross_sets(600, 8000, 103)
    assert_same(run_cross(sd, ctx, q, r, d), oracle.bruteforce_cross(q.seqs, q.offsets, r.seqs, r.offsets, d))


@pytest.mark.parametrize("nq,nr,d,opts", [(300, 5000, 2, {}), (2000, 60000, 2, {}), (2000, 60000, 1, {"FORCE_CHUNKS": 3}),
                                          (1500, 40000, 3, {}), (2000, 60000, 2, {"CAND_CAPACITY": 3000}), (5000, 20000, 2, {})])
def test_cross_query_filter(sd, oracle, nq, nr, d, opts):
    """Cross-search with the queries the small side: the level-2 partition drops the reference records whose hash bits no
    query record of their bin has (k_bin_bitmap / k_part2<true>).  Same result with the filter and without it."""
    q, r = synth.cross_sets(nq, nr, 17)
    exp = oracle.symdel_cross(q.seqs, q.offsets, r.seqs, r.offsets, d)
    for off in (0, 1):
        c = sd.Context(0)
        c.symdel_set_option(sd.OPT_NO_QUERY_FILTER, off)
        for k, v in opts.items():
            c.symdel_set_option(getattr(sd, "OPT_" + k), v)
        assert_same(run_cross(sd, c, q, r, d), exp)
        st = c.symdel_get_stats()
        assert st["fused_chunks"] == st["n_chunks"]
        assert (st["query_filter_bits"] > 0) == (off == 0 and q.n * 4 <= r.n), st["query_filter_bits"]
    # the other orientation (references the small side): no filter, same pairs mirrored
    c = sd.Context(0)
    i, j, dist = run_cross(sd, c, r, q, d)
    assert c.symdel_get_stats()["query_filter_bits"] == 0
    order = np.lexsort((i, j))
    assert_same([j[order], i[order], dist[order]], exp)


def test_cross_symmetry_and_self_relation(sd, ctx):
    a, b = synth.tcr_set(3000, 12), synth.tcr_set(4000, 11)
    ab = run_cross(sd, ctx, a, b, 2)
    ba = run_cross(sd, ctx, b, a, 2)
    assert {(x, y, z) for x, y, z in zip(*map(np.ndarray.tolist, ab))} == {(y, x, z) for x, y, z in zip(*map(np.ndarray.tolist, ba))}
    ss = run_cross(sd, ctx, a, a, 2)
    self_ = run_self(sd, ctx, a, 2)
    tri = {(x, y, z) for x, y, z in zip(*map(np.ndarray.tolist, ss)) if x < y}
    assert tri == {(x, y, z) for x, y, z in zip(*map(np.ndarray.tolist, self_))}
    assert sum(1 for x, y, z in zip(*map(np.ndarray.tolist, ss)) if x == y and z == 0) == a.n


def test_cross_chunked_windowed(sd, oracle):
    q, r = synth.cross_sets(600, 8000, 103)
    c = sd.Context(0)
    c.symdel_set_option(sd.OPT_FORCE_CHUNKS, 3)
    c.symdel_set_option(sd.OPT_CAND_CAPACITY, 300)
    assert_same(run_cross(sd, c, q, r, 2), oracle.symdel_cross(q.seqs, q.offsets, r.seqs, r.offsets, 2))


def test_host_entry_points(torch, sd, ctx, oracle):
    s = synth.tcr_set(4000, 31)
    out = tuple(torch.empty(100000, dtype=torch.int32).pin_memory() for _ in range(3))
    hs = torch.from_numpy(s.seqs).pin_memory()
    ho = torch.from_numpy(s.offsets).pin_memory()
    k = ctx.symdel_self_host(hs, ho, 2, out)
    assert_same([o[:k].numpy() for o in out], oracle.symdel_self(s.seqs, s.offsets, 2))
    q, r = synth.cross_sets(300, 5000, 9)
    out2 = tuple(np.empty(100000, np.int32) for _ in range(3))
    k = ctx.symdel_cross_host(q.seqs, q.offsets, r.seqs, r.offsets, 2, out2)
    assert_same([o[:k] for o in out2], oracle.symdel_cross(q.seqs, q.offsets, r.seqs, r.offsets, 2))


@pytest.mark.parametrize("num,pinned", [(2, True), (2, False), (3, True), (5, True)])
def test_host_entry_points_sliced_input(torch, sd, num, pinned):
    """symdel_self_host on a large set: the offsets go first, the residues follow in slices and generation of a slice
    overlaps the copy of the next (include/symdel.h, host entry points).  Same golden digest as the device entry point,
    from pinned and from pageable host memory, three calls in a row on one context (the arena and the events are reused)."""
    g = _golden(f"config_{num}.json")
    kind, d, (s,) = synth.config(num)
    assert s.n >= 65536  # the sliced path
    c = sd.Context(0)
    cap = 1 << 20
    mk = (lambda a: torch.from_numpy(a).pin_memory()) if pinned else (lambda a: a)
    hs, ho = mk(s.seqs), mk(s.offsets)
    out = tuple((torch.empty(cap, dtype=torch.int32).pin_memory() if pinned else np.empty(cap, np.int32)) for _ in range(3))
    for rep in range(3):
        k = c.symdel_self_host(hs, ho, d, out)
        i, j, dist = [(o[:k].numpy() if pinned else o[:k]) for o in out]
        assert_matches_golden(g, i, j, dist)
    st = c.symdel_get_stats()
    assert st["n_chunks"] == 1 and st["fused_chunks"] == 1


def test_host_entry_points_low_arena_estimate_only_chunks(torch, sd, oracle):
    """The host entry points size their arena from the MEAN length; a set whose few long sequences carry most of the
    deletion sets makes that estimate low — the search then runs in key-range chunks, the result is the same."""
    rng = np.random.default_rng(5)
    n = 70000
    lens = np.where(rng.random(n) < 0.03, 60, 6).astype(np.int64)  # 3 % long sequences hold ~70 % of the records at d = 2
    rows = rng.integers(1, 21, size=(n, 60)).astype(np.int8)
    rows[n // 2:] = rows[: n - n // 2]  # second half = first half with one substitution: plenty of pairs
    rows[n // 2:, 2] = rng.integers(1, 21, size=n - n // 2)
    lens[n // 2:] = lens[: n - n // 2]
    s = synth.from_padded(rows, lens)
    exp = oracle.symdel_self(s.seqs, s.offsets, 2)
    c = sd.Context(0)
    out = tuple(np.empty(len(exp[0]) + 64, np.int32) for _ in range(3))
    k = c.symdel_self_host(s.seqs, s.offsets, 2, out)
    assert_same([o[:k] for o in out], exp)
    assert c.symdel_get_stats()["n_chunks"] >= 2


def test_host_entry_points_reject_malformed_offsets(torch, sd):
    """Offsets are validated on the device (k_prepare) after the copy; the slice boundaries the host reads from them
    are clamped to the arena, whatever they say."""
    kind, d, (s,) = synth.config(2)
    c = sd.Context(0)
    out = tuple(np.empty(1 << 18, np.int32) for _ in range(3))
    for where, val, code in ((s.n // 2, -5, sd.E_OFFSETS), (s.n // 3, int(s.offsets[-1]) + 10 ** 9, sd.E_OFFSETS), (100, None, sd.E_TOO_LONG)):
        off = s.offsets.copy()
        if val is None:
            off[where + 1:] += 70  # one sequence of length > 64
            seqs = np.concatenate([s.seqs, np.ones(70, np.int8)])
        else:
            off[where] = val
            seqs = s.seqs
        with pytest.raises(sd.SymdelError) as e:
            c.symdel_self_host(seqs, off, d, out)
        assert e.value.code == code, (where, val)
    k = c.symdel_self_host(s.seqs, s.offsets, d, out)  # the context is still good
    assert k == _golden("config_2.json")["n_out"]


# ---- BASELINE.json configs at full size ---------------------------------------------------------------
def _golden(name):
    p = GOLD / name
    if not p.exists():
        pytest.skip(f"{name} not generated")
    return json.loads(p.read_text())


def _check_sampled_rows(oracle, s, d, i, j, dist, n_rows, seed):
    """Completeness on sampled rows: all neighbours of sequence t by brute force over the whole set."""
    rng = np.random.default_rng(seed)
    hit = np.unique(np.concatenate([i[:: max(1, len(i) // (n_rows // 2))][: n_rows // 2], rng.integers(0, s.n, n_rows // 2)]))
    for t in hit:
        r, dd = oracle.bruteforce_row(s.seq(int(t)), s.seqs, s.offsets, d)
        keep = r != t
        exp = {(int(min(t, x)), int(max(t, x)), int(y)) for x, y in zip(r[keep], dd[keep])}
        m = (i == t) | (j == t)
        got = {(int(a), int(b), int(c)) for a, b, c in zip(i[m], j[m], dist[m])}
        assert got == exp, int(t)


@pytest.mark.parametrize("num", [1, 2, 3, 5])
def test_config_full_size(sd, ctx, oracle, num):
    g = _golden(f"config_{num}.json")
    kind, d, (s,) = synth.config(num)
    assert s.sha256() == g["input_sha256"] and s.n == g["n"]
    i, j, dist = run_self(sd, ctx, s, d)
    assert_matches_golden(g, i, j, dist)  # identical pairs, distances and order as the oracle
    assert np.bincount(dist, minlength=d + 1).tolist() == g["dist_hist"]
    assert (i < j).all() and (np.diff(i.astype(np.int64) * (1 << 31) + j) > 0).all()
    _check_sampled_rows(oracle, s, d, i, j, dist, 24 if num >= 3 else 60, num)
    # every reported distance re-derived by the oracle's full-table recurrence (sample at full size)
    step = max(1, len(i) // 20000)
    for a, b, c in zip(i[::step], j[::step], dist[::step]):
        assert oracle.lev(s.seq(int(a)), s.seq(int(b))) == c


def test_config4_scaled(sd, ctx, oracle):
    g = _golden("config_4_scale0.1.json")
    kind, d, (q, r) = synth.config(4, 0.1)
    assert q.sha256() + r.sha256() == g["input_sha256"]
    i, j, dist = run_cross(sd, ctx, q, r, d)
    assert_matches_golden(g, i, j, dist)


def test_config4_full_size(sd, ctx, oracle):
    g = _golden("config_4.json")
    kind, d, (q, r) = synth.config(4)
    assert q.sha256() + r.sha256() == g["input_sha256"]
    i, j, dist = run_cross(sd, ctx, q, r, d)
    assert_matches_golden(g, i, j, dist)
    assert np.bincount(dist, minlength=d + 1).tolist() == g["dist_hist"]
    rng = np.random.default_rng(4)
    for t in np.unique(np.concatenate([i[:: max(1, len(i) // 10)][:10], rng.integers(0, q.n, 6)])):
        rr, dd = oracle.bruteforce_row(q.seq(int(t)), r.seqs, r.offsets, d)
        m = i == t
        assert np.array_equal(j[m], rr) and np.array_equal(dist[m], dd)


@pytest.mark.parametrize("pinned", [True, False])
def test_config4_full_size_host_entry(torch, sd, pinned):
    """symdel_cross_host at the size where the copies matter most (the two-set form of PAPER.md:43 through HOST buffers:
    98 MB of residues and offsets in, the result out, inside the call): same golden digest as the device entry point,
    from pinned and from pageable memory, two calls in a row on one context (arena reuse)."""
    g = _golden("config_4.json")
    kind, d, (q, r) = synth.config(4)
    assert q.sha256() + r.sha256() == g["input_sha256"]
    c = sd.Context(0)
    cap = 1 << 20
    mk = (lambda a: torch.from_numpy(a).pin_memory()) if pinned else (lambda a: a)
    hq, hqo, hr, hro = mk(q.seqs), mk(q.offsets), mk(r.seqs), mk(r.offsets)
    out = tuple((torch.empty(cap, dtype=torch.int32).pin_memory() if pinned else np.empty(cap, np.int32)) for _ in range(3))
    for rep in range(2):
        k = c.symdel_cross_host(hq, hqo, hr, hro, d, out)
        i, j, dist = [(o[:k].numpy() if pinned else o[:k]) for o in out]
        assert_matches_golden(g, i, j, dist)
    c.close()


# ---- S5 at full size: key-range chunking under a memory budget (BASELINE.json config 5) ------
@pytest.mark.parametrize("num,opts,ws_frac", [
    (5, {"FORCE_CHUNKS": 4}, None), (5, {"FORCE_CHUNKS": 16}, None), (5, {}, 0.1), (5, {"EXACT_PIPELINE": 1}, 0.07),
    (3, {"FORCE_CHUNKS": 4}, None), (3, {"FORCE_CHUNKS": 16}, None), (3, {}, 0.1),
    (5, {"FORCE_CHUNKS": 4, "FLUSH_PER_CHUNK": 1}, None), (3, {"FLUSH_PER_CHUNK": 1}, 0.1),
])
def test_config_full_size_chunked(torch, sd, oracle, num, opts, ws_frac):
    """Config 5 "exercises chunked key-range streaming" (BASELINE.json) — on a 180 GB device only under a budget:
    a forced chunk count, or a workspace that is a fraction of the un-chunked need (the planner then picks P).
    Same golden digest as the un-chunked run: chunking changes memory use only (P-11)."""
    g = _golden(f"config_{num}.json")
    kind, d, (s,) = synth.config(num)
    c = sd.Context(0)
    for k, v in opts.items():
        c.symdel_set_option(getattr(sd, "OPT_" + k), v)
    ds, do = sd.to_device(s)
    cap = 1 << 20
    ws = None
    if ws_frac is not None:
        full = sd.symdel_workspace_bytes(s.n, s.seqs.size, 0, 0, int(s.lengths.max()), d, cap)
        ws = torch.empty(int(full * ws_frac) // 256 * 256, dtype=torch.uint8, device="cuda")
    i, j, dist = [t.cpu().numpy() for t in c.symdel_self(ds, do, d, workspace=ws, capacity=cap)]
    st = c.symdel_get_stats()
    assert_matches_golden(g, i, j, dist)
    if "FORCE_CHUNKS" in opts:
        assert st["n_chunks"] == opts["FORCE_CHUNKS"]
    else:
        assert st["n_chunks"] >= 4, st["n_chunks"]
    if "EXACT_PIPELINE" not in opts:
        assert st["fused_chunks"] == st["n_chunks"]  # every chunk stays on the fused pipeline
    if "EXACT_PIPELINE" in opts or "FLUSH_PER_CHUNK" in opts:
        assert st["n_flushes"] >= st["n_chunks"]
    else:  # S5: dedup + verify when the candidate window fills or after the last chunk, not per chunk
        assert st["n_flushes"] < st["n_chunks"], (st["n_flushes"], st["n_chunks"])


@pytest.mark.parametrize("num,window", [(3, 1_000_000), (5, 3_000_000)])
def test_config_full_size_windowed_bucket_join(torch, sd, num, window):
    """The paper's large regime has more matched pairs than one candidate buffer holds (Table S1: 11.3 B
    pairs from 1.2 B variants).  With the candidate window capped, the fused pipeline joins the buckets that fit, flushes,
    and joins the rest in further passes: same golden digest, no hand-over to the exact pipeline."""
    g = _golden(f"config_{num}.json")
    kind, d, (s,) = synth.config(num)
    c = sd.Context(0)
    c.symdel_set_option(sd.OPT_CAND_CAPACITY, window)
    ds, do = sd.to_device(s)
    i, j, dist = [t.cpu().numpy() for t in c.symdel_self(ds, do, d, capacity=1 << 20)]
    st = c.symdel_get_stats()
    assert_matches_golden(g, i, j, dist)
    assert st["fused_chunks"] == st["n_chunks"] == 1 and st["join_general"] == 0
    assert st["join_windows"] >= st["n_candidates"] // window - 1 >= 2 and st["n_flushes"] == st["join_windows"] + 1


def test_windowed_bucket_join_single_bucket_exceeds_window(sd, oracle):
    """A bucket whose own pairs exceed a whole window cannot be windowed bucket by bucket: the chunk is handed to the exact
    pipeline (windowed join inside a bucket), whatever was flushed before; the final pass removes the repeats."""
    rows, lens = synth.to_padded(synth.tcr_set(1500, 5))
    s = synth.from_padded(np.concatenate([rows] * 30), np.concatenate([lens] * 30))
    exp = oracle.symdel_self(s.seqs, s.offsets, 1)
    c = sd.Context(0)
    c.symdel_set_option(sd.OPT_CAND_CAPACITY, 300)  # 30 copies: 435 pairs on every variant key
    assert_same(run_self(sd, c, s, 1, capacity=len(exp[0]) + 16), exp)
    st = c.symdel_get_stats()
    assert st["join_general"] >= 1


def test_dense_full_size(sd, ctx):
    """NEXT-2 at the size bench.py --dense times: synth.dense_set(1,000,000, seed 11, fanout 64), d = 2 — 14.4 M
    output pairs, candidates ~ records.  Golden written by the oracle alone."""
    g = _golden("dense_1m.json")
    s = synth.dense_set(1_000_000, 11, fanout=64)
    assert s.sha256() == g["input_sha256"]
    i, j, dist = run_self(sd, ctx, s, 2, capacity=g["n_out"] + 1024)
    assert_matches_golden(g, i, j, dist)
    st = ctx.symdel_get_stats()
    assert st["n_candidates"] > st["n_records"] // 2


# ---- run-to-run stability: every protocol built on atomics must give the same bits every time ---------------------
@pytest.mark.parametrize("opts,reps", [({}, 200), ({"EXACT_PIPELINE": 1, "FORCE_CHUNKS": 3}, 50),
                                       ({"FORCE_CHUNKS": 2, "CAND_CAPACITY": 100000}, 30)])
def test_repeat_runs_are_bit_identical(torch, sd, opts, reps):
    """Config 2, repeated in one process on one context and one workspace: claim-mode atomics, tickets, look-back and
    shared overflow lists make the ORDER of intermediate data vary from run to run; the output may not."""
    g = _golden("config_2.json")
    kind, d, (s,) = synth.config(2)
    c = sd.Context(0)
    for k, v in opts.items():
        c.symdel_set_option(getattr(sd, "OPT_" + k), v)
    ds, do = sd.to_device(s)
    cap = 1 << 18
    ws = torch.empty(sd.symdel_workspace_bytes(s.n, s.seqs.size, 0, 0, int(s.lengths.max()), d, cap), dtype=torch.uint8, device="cuda")
    out = tuple(torch.empty(cap, dtype=torch.int32, device="cuda") for _ in range(3))
    for rep in range(reps):
        i, j, dist = [t.cpu().numpy() for t in c.symdel_self(ds, do, d, workspace=ws, out=out)]
        assert digest(i, j, dist) == g["out_sha256"], rep
        if rep % 16 == 0:
            ws.random_(0, 255)  # stale workspace contents must not matter
            for o in out:
                o.fill_(-7)


# ---- boundary: devices, threads, capacity ---------------------------------------------------------------------------
def test_two_contexts_in_one_process(torch, sd, oracle):
    """Per-device state is set up by symdel_create for the context's device (include/symdel.h "Devices and threads"):
    two live contexts, used alternately and from two host threads, and one per visible device."""
    import threading

    s = synth.tcr_set(5000, 61)
    exp = oracle.symdel_self(s.seqs, s.offsets, 2)
    a, b = sd.Context(0), sd.Context(0)
    for c in (a, b, a, b):
        assert_same(run_self(sd, c, s, 2), exp)
    res = {}

    def work(name, c):
        with torch.cuda.stream(torch.cuda.Stream()):
            res[name] = [run_self(sd, c, s, 2) for _ in range(5)]

    ts = [threading.Thread(target=work, args=(n, c)) for n, c in (("a", a), ("b", b))]
    [t.start() for t in ts]
    [t.join() for t in ts]
    for name in ("a", "b"):
        for got in res[name]:
            assert_same(got, exp)
    for dev in range(1, torch.cuda.device_count()):  # a context on every other visible GPU (one GPU on the test box)
        with torch.cuda.device(dev):
            c = sd.Context(dev)
            ds, do = sd.to_device(s, f"cuda:{dev}")
            assert_same([t.cpu().numpy() for t in c.symdel_self(ds, do, 2)], exp)


@pytest.mark.parametrize("opts", [{"FORCE_CHUNKS": 4}, {"FORCE_CHUNKS": 4, "FLUSH_PER_CHUNK": 1}, {"CAND_CAPACITY": 3000},
                                  {"FORCE_CHUNKS": 3, "CAND_CAPACITY": 2000}, {"EXACT_PIPELINE": 1, "FORCE_CHUNKS": 2}])
def test_capacity_error_in_multi_flush_searches(sd, oracle, opts):
    """SYMDEL_E_CAPACITY on the chunked / windowed path (symdel.h): the first `capacity` pairs are valid and the
    required count is reported; a pair found in several chunks is appended once per flush, and the survivor list is
    merged (sorted, deduplicated) instead of running out of room."""
    s = synth.tcr_set(6000, 21)
    exp = oracle.symdel_self(s.seqs, s.offsets, 2)
    n_exp = len(exp[0])
    assert n_exp > 1500
    for surv_cap, capacity in ((0, 1000), (1, 1000), (1, n_exp), (1, n_exp + 5)):
        c = sd.Context(0)
        for k, v in opts.items():
            c.symdel_set_option(getattr(sd, "OPT_" + k), v)
        c.symdel_set_option(sd.OPT_SURV_CAPACITY, surv_cap)  # 1 = the smallest legal survivor list
        ds, do = sd.to_device(s)
        out = tuple(__import__("torch").full((capacity,), -1, dtype=__import__("torch").int32, device="cuda") for _ in range(3))
        if capacity >= n_exp:
            got = [t.cpu().numpy() for t in c.symdel_self(ds, do, 2, out=out)]
            assert_same(got, exp)
            continue
        with pytest.raises(sd.SymdelError) as e:
            c.symdel_self(ds, do, 2, out=out)
        assert e.value.code == sd.E_CAPACITY
        st = c.symdel_get_stats()
        if st["surv_merges"] == 0:
            assert c.last_required == n_exp  # exact count
        else:
            assert capacity < c.last_required <= n_exp  # a lower bound that still exceeds the capacity
        for o, x in zip(out, exp):
            assert np.array_equal(o.cpu().numpy(), x[:capacity])  # the first `capacity` pairs, ascending


@pytest.mark.parametrize("opts", [{"FORCE_CHUNKS": 2, "FLUSH_PER_CHUNK": 1}, {"CAND_CAPACITY": 150000},
                                  {"FORCE_CHUNKS": 3, "CAND_FILTER": 1, "FLUSH_PER_CHUNK": 1}, {"EXACT_PIPELINE": 1, "FORCE_CHUNKS": 2},
                                  {"FORCE_CHUNKS": 3, "CAND_CAPACITY": 400000}])
def test_survivor_list_smaller_than_one_flush(sd, oracle, opts):
    """A flush that yields far more survivors than the room behind the survivor list (capacity + 4096 entries with
    SYMDEL_OPT_SURV_CAPACITY = 1; the dense set gives tens of thousands per flush): the window is verified in slices
    with merges in between — SYMDEL_E_CAPACITY with the first `capacity` pairs and a lower bound of the count when the
    result is larger than `capacity`, the exact result when it fits; never SYMDEL_E_WORKSPACE."""
    import torch

    s = synth.dense_set(12000, 51, fanout=64)
    exp = oracle.symdel_self(s.seqs, s.offsets, 2)
    n_exp = len(exp[0])
    assert n_exp > 100_000
    ds, do = sd.to_device(s)
    for capacity in (1000, n_exp // 3, n_exp):
        c = sd.Context(0)
        for k, v in opts.items():
            c.symdel_set_option(getattr(sd, "OPT_" + k), v)
        c.symdel_set_option(sd.OPT_SURV_CAPACITY, 1)
        out = tuple(torch.full((capacity,), -1, dtype=torch.int32, device="cuda") for _ in range(3))
        if capacity >= n_exp:
            assert_same([t.cpu().numpy() for t in c.symdel_self(ds, do, 2, out=out)], exp)
        else:
            with pytest.raises(sd.SymdelError) as e:
                c.symdel_self(ds, do, 2, out=out)
            assert e.value.code == sd.E_CAPACITY
            assert capacity < c.last_required <= n_exp
            for o, x in zip(out, exp):
                assert np.array_equal(o.cpu().numpy(), x[:capacity])
        st = c.symdel_get_stats()
        assert st["n_flushes"] >= 2 and st["surv_merges"] >= 1
        c.close()


def test_more_than_2_30_records(torch, sd, oracle):
    """The regime the key-range chunking exists for (1.2 B deletion variants at 10 M sequences and
    d = 2, 577 M at 1 M and d = 3): 400,000 BCR-like sequences of 26..30 residues at d = 3 hold about 1.4 x 2^30
    deletion sets, more than one chunk may carry (record counts and bin cursors are 30-bit).  With NO option set the
    planner has to split the search by itself (n_chunks >= 2).  The oracle's hash map would need hours here, so the
    result is pinned in two other ways: it equals, element by element, the result of the same search forced into 8
    chunks (a path the full-size goldens of configs 3 and 5 do pin), and 32 sampled rows are complete and correct
    against the oracle's brute-force row (every neighbour of a sequence over the whole set)."""
    from math import comb

    d = 3
    s = synth.bcr_set(400_000, 77, lo=26, hi=30, mean=28.0, sd=1.0)
    nmax = sum(int(c) * sum(comb(L, k) for k in range(d + 1)) for L, c in enumerate(np.bincount(s.lengths)))
    assert nmax > (1 << 30) + (1 << 28)
    ds, do = sd.to_device(s)
    cap = 1 << 23
    nbytes = sd.symdel_workspace_bytes(s.n, s.seqs.size, 0, 0, int(s.lengths.max()), d, cap)
    ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    out = tuple(torch.empty(cap, dtype=torch.int32, device="cuda") for _ in range(3))
    c = sd.Context(0)
    got = [t.cpu().numpy() for t in c.symdel_self(ds, do, d, workspace=ws, out=out)]
    st = c.symdel_get_stats()
    assert st["n_chunks"] >= 2 and st["n_records"] >= (1 << 30), st
    c.close()
    c = sd.Context(0)
    c.symdel_set_option(sd.OPT_FORCE_CHUNKS, 8)
    ref = [t.cpu().numpy() for t in c.symdel_self(ds, do, d, workspace=ws, out=out)]
    st8 = c.symdel_get_stats()
    assert st8["n_chunks"] == 8 and st8["n_records"] == st["n_records"]
    c.close()
    assert len(got[0]) > 100_000
    assert_same(got, ref)
    i, j, dist = got
    assert np.all(i < j) and np.all(np.diff(i.astype(np.int64) * s.n + j) > 0)  # ascending (i, j), each pair once
    _check_sampled_rows(oracle, s, d, i, j, dist, 32, 5)


def test_out_of_range_indices_are_rejected(torch, sd, ctx):
    """Caller-supplied indices never steer a read out of bounds: symdel_stage_lev and symdel_overlap_matrix."""
    s = synth.tcr_set(300, 5)
    ds, do = sd.to_device(s)
    ia = torch.tensor([0, 5, s.n - 1], dtype=torch.int32, device="cuda")
    assert (ctx.symdel_stage_lev(ds, do, ds, do, ia, ia).cpu().numpy() == 0).all()
    for bad in (s.n, -1, 2**31 - 1):
        ib = torch.tensor([0, bad, 7], dtype=torch.int32, device="cuda")
        with pytest.raises(sd.SymdelError) as e:
            ctx.symdel_stage_lev(ds, do, ds, do, ia, ib)
        assert e.value.code == sd.E_ARG
    labs = torch.zeros(s.n, dtype=torch.int32, device="cuda")
    pi = torch.tensor([1, 2, s.n - 1], dtype=torch.int32, device="cuda")
    assert int(ctx.symdel_overlap_matrix(pi, pi, labs, labs, 2, True).sum()) == 3
    for bad in (s.n, -5):
        pj = torch.tensor([1, bad, 3], dtype=torch.int32, device="cuda")
        with pytest.raises(sd.SymdelError) as e:
            ctx.symdel_overlap_matrix(pi, pj, labs, labs, 2, True)
        assert e.value.code == sd.E_ARG


def test_malformed_offsets_never_steer_a_read(torch, sd, ctx):
    """A garbage offsets array is reported as SYMDEL_E_OFFSETS / _TOO_LONG before any residue is read through it."""
    s = synth.tcr_set(500, 8)
    ds, do = sd.to_device(s)
    for pos, val in ((500, 1 << 40), (250, -3), (0, 1), (499, 1 << 50)):
        bad = do.clone()
        bad[pos] = val
        with pytest.raises(sd.SymdelError) as e:
            ctx.symdel_self(ds, bad, 2)
        assert e.value.code in (sd.E_OFFSETS, sd.E_TOO_LONG), (pos, e.value.code)
    assert len(ctx.symdel_self(ds, do, 1)[0]) >= 0  # the context still works (no sticky CUDA error)
