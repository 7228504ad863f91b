"""Seeded synthetic CDR3 repertoires (BASELINE.json configs 1-5; SURVEY.md §8(d) G-rules).

This module is the ONE input generator shared by the CPU oracle (`oracle/`) and the CUDA
path.  It holds none of the method's arithmetic (no deletion variants, no hashing, no
edit distance): it only draws sequences.  The paper measures on Emerson et al. TCRβ and
Briney et al. BCR CDR3s; neither dataset is available here, so
these generators stand in for them with the same shapes (20-letter alphabet, TCRβ CDR3
length ≈ 15 ± 2 aa, BCR CDR3 longer and broader, clonal-lineage structure).

Layout of every set: CSR, ``seqs int8[ΣL]`` (residue codes 1..20) and
``offsets int64[n+1]`` with ``offsets[0] == 0``.

Only numpy is imported; the code is the specification of the workload.
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass

import numpy as np

ALPHABET = 20  # residue codes 1..20 ("amino-acid string"; BASELINE.json config 1)


@dataclass(frozen=True)
class SeqSet:
    """A CSR sequence set."""

    seqs: np.ndarray  # int8[total]
    offsets: np.ndarray  # int64[n+1]

    @property
    def n(self) -> int:
        return int(self.offsets.shape[0] - 1)

    @property
    def lengths(self) -> np.ndarray:
        return np.diff(self.offsets)

    def seq(self, i: int) -> np.ndarray:
        return self.seqs[self.offsets[i]:self.offsets[i + 1]]

    def sha256(self) -> str:
        h = hashlib.sha256()
        h.update(np.ascontiguousarray(self.offsets).tobytes())
        h.update(np.ascontiguousarray(self.seqs).tobytes())
        return h.hexdigest()

    def take(self, idx) -> "SeqSet":
        """Sub-set / permutation by index (used by the shuffle-invariance tests)."""
        idx = np.asarray(idx, dtype=np.int64)
        rows, lens = to_padded(self)
        return from_padded(rows[idx], lens[idx])


# ----------------------------------------------------------------------------------------
# padded <-> CSR helpers
# ----------------------------------------------------------------------------------------
def to_padded(s: SeqSet, width: int | None = None):
    lens = s.lengths.astype(np.int32)
    w = int(lens.max()) if (width is None and s.n) else int(width or 1)
    rows = np.zeros((s.n, max(w, 1)), dtype=np.int8)
    mask = np.arange(rows.shape[1], dtype=np.int32)[None, :] < lens[:, None]
    rows[mask] = s.seqs
    return rows, lens


def from_padded(rows: np.ndarray, lens: np.ndarray) -> SeqSet:
    lens = np.asarray(lens, dtype=np.int64)
    mask = np.arange(rows.shape[1], dtype=np.int64)[None, :] < lens[:, None]
    seqs = np.ascontiguousarray(rows[mask], dtype=np.int8)
    offsets = np.zeros(lens.shape[0] + 1, dtype=np.int64)
    np.cumsum(lens, out=offsets[1:])
    return SeqSet(seqs, offsets)


def from_strings(strings, alphabet: str = "ABCDEFGHIJKLMNOPQRSTUVWXYZ") -> SeqSet:
    """Letters -> codes 1..len(alphabet) in the order of `alphabet` (tests' hand-worked cases;
    the default maps A..Z to 1..26, all representable in the library's 5-bit residue codes)."""
    code = {c: i + 1 for i, c in enumerate(alphabet)}
    lens = np.array([len(s) for s in strings], dtype=np.int64)
    flat = np.array([code[c] for s in strings for c in s], dtype=np.int8)
    offsets = np.zeros(len(strings) + 1, dtype=np.int64)
    np.cumsum(lens, out=offsets[1:])
    return SeqSet(flat, offsets)


def dedup_first(rows: np.ndarray, lens: np.ndarray):
    """G-5: remove exact duplicates, keep the first occurrence, preserve order."""
    if rows.shape[0] == 0:
        return rows, lens
    key = np.ascontiguousarray(rows).view(np.dtype((np.void, rows.shape[1]))).ravel()
    _, first = np.unique(key, return_index=True)
    keep = np.sort(first)
    return rows[keep], lens[keep]


# ----------------------------------------------------------------------------------------
# drawing
# ----------------------------------------------------------------------------------------
def _draw_seeds(rng, n, width, lo, hi, mean, sd):
    """G-2: length = clip(rint(Normal(mean, sd)), lo, hi); residues i.i.d. uniform 1..20."""
    lens = np.clip(np.rint(rng.normal(mean, sd, size=n)), lo, hi).astype(np.int32)
    rows = rng.integers(1, ALPHABET + 1, size=(n, width), dtype=np.int8)
    rows[np.arange(width, dtype=np.int32)[None, :] >= lens[:, None]] = 0
    return rows, lens


def _apply_edit(rows, lens, u_type, u_pos, res, lo, hi):
    """G-4: one random edit per row, in place semantics (returns new arrays).

    The type is uniform over the edit types that keep the length in [lo, hi] (equivalent to
    "redraw the type" of G-4); position uniform (insertion: L+1 slots); residue uniform over
    all 20 letters (a substitution may redraw the same residue).
    """
    b, w = rows.shape
    ins_ok = lens < hi
    del_ok = lens > lo
    n_allowed = 1 + ins_ok.astype(np.int32) + del_ok.astype(np.int32)
    t_idx = np.minimum((u_type * n_allowed).astype(np.int32), n_allowed - 1)
    # ordered list of allowed types [sub, ins?, del?]
    is_sub = t_idx == 0
    is_ins = (t_idx == 1) & ins_ok
    is_del = ~is_sub & ~is_ins
    slots = np.where(is_ins, lens + 1, lens)
    p = np.minimum((u_pos * slots).astype(np.int32), slots - 1)
    j = np.arange(w, dtype=np.int32)[None, :]
    pc = p[:, None]
    src = np.where(is_ins[:, None], j - (j > pc), np.where(is_del[:, None], j + (j >= pc), j))
    new = np.take_along_axis(rows, np.clip(src, 0, w - 1), axis=1)
    put = (is_sub | is_ins)[:, None] & (j == pc)
    new = np.where(put, res[:, None].astype(np.int8), new)
    new_lens = lens + is_ins.astype(np.int32) - is_del.astype(np.int32)
    new[j >= new_lens[:, None]] = 0
    return new.astype(np.int8), new_lens.astype(np.int32)


def _derive(rng, parent_rows, parent_lens, kmax, lo, hi):
    """Copy each parent and apply k ~ U{1..kmax} random edits (G-3/G-4/G-7)."""
    m = parent_rows.shape[0]
    k = rng.integers(1, kmax + 1, size=m)
    u_type = rng.random((m, kmax))
    u_pos = rng.random((m, kmax))
    res = rng.integers(1, ALPHABET + 1, size=(m, kmax))
    rows, lens = parent_rows.copy(), parent_lens.copy()
    for e in range(kmax):
        act = np.nonzero(k > e)[0]
        if act.size == 0:
            break
        r2, l2 = _apply_edit(rows[act], lens[act], u_type[act, e], u_pos[act, e], res[act, e], lo, hi)
        rows[act], lens[act] = r2, l2
    return rows, lens


def tcr_padded(n_nominal: int, seed, lo=8, hi=24, mean=15.0, sd=2.0, kmax=3, dedup=True):
    """G-3: first half seeds; sequence t >= n/2 copies a uniformly chosen EARLIER sequence
    (seed or derived) and applies k ~ U{1,2,3} edits."""
    rng = np.random.default_rng(seed)
    n = int(n_nominal)
    n_seed = n // 2
    m = n - n_seed
    rows = np.zeros((n, hi), dtype=np.int8)
    lens = np.zeros(n, dtype=np.int32)
    rows[:n_seed], lens[:n_seed] = _draw_seeds(rng, n_seed, hi, lo, hi, mean, sd)
    t = np.arange(n_seed, n, dtype=np.int64)
    parent = np.minimum((rng.random(m) * t).astype(np.int64), t - 1) if m else np.zeros(0, np.int64)
    k = rng.integers(1, kmax + 1, size=m)
    u_type = rng.random((m, kmax))
    u_pos = rng.random((m, kmax))
    res = rng.integers(1, ALPHABET + 1, size=(m, kmax))
    # depth of each derived sequence in the copy forest (seeds are depth 0)
    depth = np.zeros(n, dtype=np.int32)
    for ti in range(m):  # cheap integer loop; the sequence edits below are vectorised per level
        depth[n_seed + ti] = depth[parent[ti]] + 1
    for level in range(1, int(depth.max()) + 1 if m else 1):
        idx = np.nonzero(depth[n_seed:] == level)[0]
        if idx.size == 0:
            continue
        r, l = rows[parent[idx]].copy(), lens[parent[idx]].copy()
        for e in range(kmax):
            act = np.nonzero(k[idx] > e)[0]
            if act.size == 0:
                break
            a = idx[act]
            r2, l2 = _apply_edit(r[act], l[act], u_type[a, e], u_pos[a, e], res[a, e], lo, hi)
            r[act], l[act] = r2, l2
        rows[n_seed + idx], lens[n_seed + idx] = r, l
    if dedup:
        rows, lens = dedup_first(rows, lens)
    return rows, lens


def tcr_set(n_nominal: int, seed, **kw) -> SeqSet:
    """BASELINE.json configs 1-3 (seeds 0, 1, 2) and the reference side of config 4 (seed 3)."""
    return from_padded(*tcr_padded(n_nominal, seed, **kw))


def bcr_set(n_total: int, seed, n_lineages: int | None = None, lo=8, hi=30, mean=16.0, sd=4.0,
            kmax=4, p_geom=0.1, dedup=True) -> SeqSet:
    """G-7 (config 5): lineages emitted contiguously: seed, then g ~ Geometric(p) descendants,
    each = the SEED + k ~ U{1..4} edits (star-shaped); concatenated, cut to n_total, deduped."""
    rng = np.random.default_rng(seed)
    if n_lineages is None:
        n_lineages = max(1, n_total // 10)
    srows, slens = _draw_seeds(rng, n_lineages, hi, lo, hi, mean, sd)
    g = rng.geometric(p_geom, size=n_lineages).astype(np.int64)
    sizes = 1 + g
    starts = np.zeros(n_lineages + 1, dtype=np.int64)
    np.cumsum(sizes, out=starts[1:])
    total = int(starts[-1])
    lineage = np.repeat(np.arange(n_lineages, dtype=np.int64), sizes)
    is_seed = np.zeros(total, dtype=bool)
    is_seed[starts[:-1]] = True
    rows = srows[lineage].copy()
    lens = slens[lineage].copy()
    d_idx = np.nonzero(~is_seed)[0]
    drows, dlens = _derive(rng, rows[d_idx], lens[d_idx], kmax, lo, hi)
    rows[d_idx], lens[d_idx] = drows, dlens
    rows, lens = rows[:n_total], lens[:n_total]
    if dedup:
        rows, lens = dedup_first(rows, lens)
    return from_padded(rows, lens)


def dense_set(n_total: int, seed, fanout: int = 64, kmax: int = 2) -> SeqSet:
    """NEXT-2: a dense-neighbourhood repertoire, the regime the paper reports for real
    data (137 M matched pairs from 120 M variants at 1 M sequences).  n_total / fanout TCR-shaped
    seeds, each with a Geometric(1 / fanout) number of descendants = the seed + k ~ U{1..kmax} edits, emitted
    contiguously, cut to n_total, deduplicated: whole clusters lie within distance 2 * kmax of one another."""
    return bcr_set(n_total, seed, n_lineages=max(1, n_total // fanout), lo=8, hi=24, mean=15.0, sd=2.0, kmax=kmax,
                   p_geom=1.0 / fanout)


def cross_sets(n_query: int, n_ref: int, seed: int, p_derived=0.2, lo=8, hi=24, mean=15.0, sd=2.0, kmax=3):
    """G-6 (config 4): reference = TCR set (seed); queries: with prob. 0.2 a uniformly chosen
    reference sequence + k ~ U{1,2,3} edits, else an independent seed; query RNG =
    default_rng([seed, 1]).  Dedup within each set separately (dist-0 cross pairs are legal)."""
    rrows, rlens = tcr_padded(n_ref, seed, lo=lo, hi=hi, mean=mean, sd=sd, kmax=kmax)
    rng = np.random.default_rng([seed, 1])
    derived = rng.random(n_query) < p_derived
    qrows, qlens = _draw_seeds(rng, n_query, hi, lo, hi, mean, sd)
    d_idx = np.nonzero(derived)[0]
    par = rng.integers(0, rrows.shape[0], size=d_idx.size)
    drows, dlens = _derive(rng, rrows[par], rlens[par], kmax, lo, hi)
    qrows[d_idx], qlens[d_idx] = drows, dlens
    qrows, qlens = dedup_first(qrows, qlens)
    return from_padded(qrows, qlens), from_padded(rrows, rlens)


def repeat_heavy_set(n: int, seed: int, alphabet: int = 3, lo=0, hi=12) -> SeqSet:
    """Test-only stress set: tiny alphabet and short lengths (many repeated residues, many
    duplicate variants, long runs, empty sequences when lo == 0).  Duplicates are KEPT."""
    rng = np.random.default_rng(seed)
    lens = rng.integers(lo, hi + 1, size=n).astype(np.int32)
    rows = rng.integers(1, alphabet + 1, size=(n, max(hi, 1)), dtype=np.int8)
    rows[np.arange(rows.shape[1], dtype=np.int32)[None, :] >= lens[:, None]] = 0
    return from_padded(rows, lens)


# ----------------------------------------------------------------------------------------
# BASELINE.json configs by number (1-based, as SURVEY.md §8 names them)
# ----------------------------------------------------------------------------------------
CONFIGS = {
    1: dict(kind="self", d=1, n=10_000, seed=0, family="tcr"),
    2: dict(kind="self", d=2, n=100_000, seed=1, family="tcr"),
    3: dict(kind="self", d=2, n=1_000_000, seed=2, family="tcr"),
    4: dict(kind="cross", d=2, n_query=100_000, n_ref=5_000_000, seed=3, family="tcr"),
    5: dict(kind="self", d=3, n=200_000, seed=4, family="bcr"),
}


def config(num: int, scale: float = 1.0):
    """Return (kind, d, sets) for BASELINE.json config `num`; `scale` < 1 shrinks n (tests)."""
    c = CONFIGS[num]
    if c["kind"] == "cross":
        q, r = cross_sets(max(1, int(c["n_query"] * scale)), max(2, int(c["n_ref"] * scale)), c["seed"])
        return "cross", c["d"], (q, r)
    n = max(2, int(c["n"] * scale))
    if c["family"] == "bcr":
        return "self", c["d"], (bcr_set(n, c["seed"], n_lineages=max(1, n // 10)),)
    return "self", c["d"], (tcr_set(n, c["seed"]),)
