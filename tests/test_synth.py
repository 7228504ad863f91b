"""Input generator: determinism, shapes and structure of the BASELINE.json workloads (G-rules)."""
import json
from pathlib import Path

import numpy as np

from paper_2403_09010_b200 import synth

GOLD = Path(__file__).parent / "golden"


def test_config1_matches_golden_input_hash():
    kind, d, (s,) = synth.config(1)
    g = json.loads((GOLD / "config_1.json").read_text())
    assert (kind, d) == ("self", 1) and s.n == g["n"] and s.sha256() == g["input_sha256"]


def test_tcr_shape_and_dedup():
    s = synth.tcr_set(20000, 42)
    L = s.lengths
    assert s.offsets[0] == 0 and s.seqs.dtype == np.int8 and s.offsets.dtype == np.int64
    assert L.min() >= 8 and L.max() <= 24 and abs(L.mean() - 15) < 0.3
    assert s.seqs.min() >= 1 and s.seqs.max() <= 20
    rows, lens = synth.to_padded(s, 24)
    assert len({r.tobytes() for r in rows}) == s.n  # exact duplicates removed (G-5)
    assert 0.98 * 20000 < s.n <= 20000
    s2 = synth.tcr_set(20000, 42)
    assert s2.sha256() == s.sha256() and synth.tcr_set(20000, 43).sha256() != s.sha256()


def test_bcr_shape():
    s = synth.bcr_set(20000, 7, n_lineages=2000)
    L = s.lengths
    assert L.min() >= 8 and L.max() <= 30 and 15 < L.mean() < 17.5
    assert 0.95 * 20000 < s.n <= 20000


def test_cross_sets():
    q, r = synth.cross_sets(2000, 30000, 3)
    assert 1900 < q.n <= 2000 and 29000 < r.n <= 30000
    assert q.lengths.min() >= 8 and q.lengths.max() <= 24


def test_take_roundtrip():
    s = synth.tcr_set(500, 1)
    p = np.random.default_rng(0).permutation(s.n)
    t = s.take(p)
    for k in (0, 17, s.n - 1):
        assert np.array_equal(t.seq(k), s.seq(p[k]))


def test_dense_set_shape():
    s = synth.dense_set(5000, 3, fanout=50)
    assert 4000 < s.n <= 5000 and s.lengths.min() >= 8 and s.lengths.max() <= 24
    assert s.seqs.min() >= 1 and s.seqs.max() <= 20
    s2 = synth.dense_set(5000, 3, fanout=50)
    assert np.array_equal(s.seqs, s2.seqs) and np.array_equal(s.offsets, s2.offsets)
