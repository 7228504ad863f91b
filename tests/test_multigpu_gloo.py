"""N > 1 path of bench.py ("replicas only": DESIGN.md §8): world_size-2 gloo run on CPU of the only
cross-rank exchange there is — barrier + MAX of the per-rank step times — and of the job-level value."""
import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, str(ROOT))
    import torch
    import torch.distributed as dist

    import bench

    dist.init_process_group("gloo", rank=rank, world_size=world)
    dist.barrier()
    ms, e2e = bench.max_over_ranks([3.0 + rank, 5.0 - rank], dist, torch.device("cpu"))
    q.put((rank, ms, e2e, bench.job_value(1000, world, ms)))
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_max_over_ranks_gloo():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, e2e, value in out:
        assert ms == 4.0 and e2e == 5.0  # the slowest rank decides
        assert value == pytest.approx(2 * 1000 / 4e-3)  # whole-job aggregate over both replicas


def test_single_process_passthrough():
    sys.path.insert(0, str(ROOT))
    import torch

    import bench

    assert bench.max_over_ranks([1.5, 2.5], None, torch.device("cpu")) == [1.5, 2.5]


def test_bench_digest_is_the_golden_format():
    """bench.py hashes what it times and compares with tests/golden/*.json: its digest must be the one
    tests/golden/make_golden.py writes (sha256 of the int32 arrays i, j, dist, concatenated)."""
    import hashlib
    import importlib.util

    import numpy as np

    sys.path.insert(0, str(ROOT))
    import bench

    spec = importlib.util.spec_from_file_location("make_golden", ROOT / "tests" / "golden" / "make_golden.py")
    mg = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mg)
    rng = np.random.default_rng(0)
    i, j, d = (rng.integers(0, 1000, 257).astype(np.int64) for _ in range(3))
    want = hashlib.sha256(b"".join(np.asarray(a, dtype=np.int32).tobytes() for a in (i, j, d))).hexdigest()
    assert bench.digest(i, j, d) == mg.digest(i, j, d) == want
    for name in ("config_1.json", "config_2.json", "config_3.json", "config_4.json", "config_5.json", "dense_1m.json"):
        g = bench.golden(name)
        assert g and len(g["out_sha256"]) == 64 and g["n_out"] > 0, name
