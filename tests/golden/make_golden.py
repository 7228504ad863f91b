"""Writes tests/golden/config_<k>.json: the oracle's result digest for BASELINE.json config k.

Calls ONLY oracle/ and the input generator (never the CUDA path).  Usage:
    python tests/golden/make_golden.py 1 2 3 5        # self configs (3: ~5 min, 5: ~10 min, 1 thread)
    python tests/golden/make_golden.py 4              # cross 100k x 5M (~20+ min)
    python tests/golden/make_golden.py 4@0.1          # config 4 at 1/10 scale
    python tests/golden/make_golden.py dense          # NEXT-2: synth.dense_set(1,000,000, seed 11, fanout 64), d = 2 (~15 min)
Each file stores: the input sha256, n, d, the number of output pairs, the distance histogram, the
sha256 of the concatenated int32 arrays (i, j, dist), the oracle's (unpinned) stage counters, the
oracle wall time on this host, and `block_sha`: a 48-bit digest of every block of BLOCK consecutive
output rows (so that a full-size mismatch can be located: tests print the first differing block).
"""
import hashlib
import json
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parents[2]
sys.path.insert(0, str(ROOT))
from oracle import oracle  # noqa: E402
from paper_2403_09010_b200 import synth  # noqa: E402


def digest(i, j, d):
    h = hashlib.sha256()
    for a in (i, j, d):
        h.update(np.ascontiguousarray(a, dtype=np.int32).tobytes())
    return h.hexdigest()


BLOCK = 4096


def block_digests(i, j, d):
    """sha256[:12] of the int32 rows (i, j, dist) of each block of BLOCK consecutive output rows."""
    rows = np.ascontiguousarray(np.stack([np.asarray(a, dtype=np.int32) for a in (i, j, d)], axis=1))
    return [hashlib.sha256(rows[t:t + BLOCK].tobytes()).hexdigest()[:12] for t in range(0, len(rows), BLOCK)]


def main(args):
    for a in args:
        if a == "dense":  # the workload of `bench.py --dense` (NEXT-2)
            num, scale, sc = "dense_1m", 1.0, ""
            kind, d, sets = "self", 2, (synth.dense_set(1_000_000, 11, fanout=64),)
        else:
            num, _, sc = a.partition("@")
            num, scale = int(num), float(sc) if sc else 1.0
            kind, d, sets = synth.config(num, scale)
        t0 = time.time()
        if kind == "self":
            (s,) = sets
            i, j, dist, c = oracle.symdel_self(s.seqs, s.offsets, d, with_counters=True)
            meta = dict(n=s.n, input_sha256=s.sha256())
        else:
            q, r = sets
            i, j, dist, c = oracle.symdel_cross(q.seqs, q.offsets, r.seqs, r.offsets, d, with_counters=True)
            meta = dict(n_query=q.n, n_ref=r.n, input_sha256=q.sha256() + r.sha256())
        wall = time.time() - t0
        rec = dict(config=num, scale=scale, kind=kind, d=d, **meta, n_out=int(len(i)),
                   dist_hist=np.bincount(dist, minlength=d + 1).tolist(), out_sha256=digest(i, j, dist),
                   block_rows=BLOCK, block_sha=block_digests(i, j, dist),
                   oracle_counters_unpinned=c, oracle_wall_s=round(wall, 2), oracle="oracle_symdel (App. F.1 hash map)")
        name = f"{num}.json" if a == "dense" else f"config_{num}.json" if scale == 1.0 else f"config_{num}_scale{sc}.json"
        txt = json.dumps(rec, indent=1)
        head, _, tail = txt.partition('"block_sha": [')  # the digest list on few lines
        body, _, rest = tail.partition("]")
        txt = head + '"block_sha": [' + " ".join(body.split()) + "]" + rest
        (Path(__file__).parent / name).write_text(txt + "\n")
        print(name, rec["n_out"], rec["dist_hist"], f"{wall:.1f}s", flush=True)


if __name__ == "__main__":
    main(sys.argv[1:] or ["1", "2"])
