"""Writes tests/golden/config_<k>.json: the oracle's result digest for BASELINE.json config k.

Calls ONLY oracle/ and the input generator (never the CUDA path).  Usage:
    python tests/golden/make_golden.py 1 2 3 5        # self configs (3: ~5 min, 5: ~10 min, 1 thread)
    python tests/golden/make_golden.py 4              # cross 100k x 5M (~20+ min)
    python tests/golden/make_golden.py 4@0.1          # config 4 at 1/10 scale
Each file stores: the input sha256, n, d, the number of output pairs, the distance histogram, the
sha256 of the concatenated int32 arrays (i, j, dist), the oracle's (unpinned) stage counters, and
the oracle wall time on this host.
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


def main(args):
    for a in args:
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
                   oracle_counters_unpinned=c, oracle_wall_s=round(wall, 2), oracle="oracle_symdel (App. F.1 hash map)")
        name = f"config_{num}.json" if scale == 1.0 else f"config_{num}_scale{sc}.json"
        (Path(__file__).parent / name).write_text(json.dumps(rec, indent=1) + "\n")
        print(name, rec["n_out"], rec["dist_hist"], f"{wall:.1f}s", flush=True)


if __name__ == "__main__":
    main(sys.argv[1:] or ["1", "2"])
