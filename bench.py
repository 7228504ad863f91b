#!/usr/bin/env python
"""bench.py — BASELINE.json metric on its workload: 1M-CDR3 d=2 self-search (config 3).

    python bench.py --gpus N --steps K --warmup W            # the CUDA path (libsymdel)
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle as it stands (slow)

A step = one pass of the whole hot path (prepare, generate, sort, emit, dedup, verify) over the
synthetic repertoire.  `value` = verified pairs/s with inputs resident in HBM; `e2e` = the same
through symdel_self_host with pinned HOST buffers (H2D of the sequences and D2H of the result inside
the timed region).  Timing: CUDA events on the launching stream, per step, with an L2 flush
(512 MiB memset, untimed) between steps; max over ranks.  N > 1 runs N independent replicas (the
path does not shard: DESIGN.md §Multi-GPU), one process per GPU, no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "1M-CDR3 d=2 self-search wall time (s), verified pairs/sec, HBM GB/s vs peak"
UNIT = "verified pairs/s"
WORKLOAD = "config 3: self-search d=2, 1,000,000 synthetic TCRb CDR3 (seed 2), 995,218 after dedup"
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback


def load_peak():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return float(json.loads(p.read_text())["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def load_traffic(kernel: str):
    """dram bytes per launch of `kernel` from the committed ncu --set full capture (profiles/traffic.json)."""
    p = ROOT / "profiles" / "traffic.json"
    if p.exists():
        try:
            return json.loads(p.read_text()).get("dram_bytes_per_launch", {}).get(kernel)
        except Exception:
            return None
    return None


class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "20"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        rows = [r for ts, r in self.rows if t0 <= ts <= t1 + 0.1] or [r for _, r in self.rows]
        sm, mx, reasons = [], None, set()
        for r in rows:
            try:
                sm.append(float(r[0]))
                mx = float(r[1])
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def max_over_ranks(values, dist, device):
    """Replicas-only multi-GPU aggregation: the step time of the job is the MAX over ranks (no data-path
    collective exists; this is the only cross-rank exchange).  `dist` is torch.distributed or None."""
    import torch

    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def job_value(pairs_per_replica: int, world: int, ms: float) -> float:
    """Whole-job verified pairs/s: every replica processes the same workload (weak scaling)."""
    return world * pairs_per_replica / (ms * 1e-3)


def host_info():
    """CPU model, logical cores and the threads the oracle uses (it is single-threaded C++): SURVEY.md section 8(d)."""
    model = None
    try:
        for ln in Path("/proc/cpuinfo").read_text().splitlines():
            if ln.lower().startswith("model name"):
                model = ln.split(":", 1)[1].strip()
                break
    except Exception:
        pass
    return {"cpu_model": model, "nproc": os.cpu_count(), "threads": 1}


def oracle_record(gold, live=None):
    """The oracle's time on one workload: `live` = (pairs, seconds) measured in this run, else the wall time recorded
    when the golden file was written (another host, said so)."""
    if live:
        return {"value": live[0] / live[1], "unit": UNIT, "seconds": live[1], "where": "this run, this host", **host_info()}
    if gold and gold.get("oracle_wall_s"):
        return {"value": gold["n_out"] / gold["oracle_wall_s"], "unit": UNIT, "seconds": gold["oracle_wall_s"],
                "where": "recorded by tests/golden/make_golden.py when the golden file was written (another host)", "threads": 1}
    return None


def cpu_baseline_run(n_sample: int, d: int, s):
    """The oracle as it stands on a bounded sample: the workload's generator and seed at n_sample
    sequences (a prefix of the 1M set would hold seeds only, i.e. no neighbours)."""
    from oracle import oracle
    from paper_2403_09010_b200 import synth

    sub = synth.tcr_set(n_sample, synth.CONFIGS[3]["seed"])
    t0 = time.time()
    i, j, dist = oracle.symdel_self(sub.seqs, sub.offsets, d)
    dt = time.time() - t0
    return len(i), dt


def digest(i, j, d):
    """sha256 of the int32 arrays (i, j, dist): the format of tests/golden/*.json (written by the oracle alone)."""
    import hashlib

    h = hashlib.sha256()
    for a in (i, j, d):
        h.update(np.ascontiguousarray(a, dtype=np.int32).tobytes())
    return h.hexdigest()


def golden(name):
    p = ROOT / "tests" / "golden" / name
    return json.loads(p.read_text()) if p.exists() else None


def run_workload(torch, symdel, dev, name, kind, d, sets, gold, opts=None, ws_frac=None, steps=5, cap=1 << 21, oracle_live=False,
                 e2e_host=False):
    """One of the other workloads (configs 1, 2, 4, 5, dense, forced pipelines): `steps` device-resident steps after one
    warm-up, CUDA events, result checked against the oracle's golden digest.  Not part of the headline's timed region."""
    ctx = symdel.Context(dev.index)
    for k, v in (opts or {}).items():
        ctx.symdel_set_option(getattr(symdel, "OPT_" + k), v)
    devs = [symdel.to_device(s, dev) for s in sets]
    args = [t for pair in devs for t in pair]
    n_a, n_b = sets[0].n, (sets[1].n if kind == "cross" else 0)
    res_a, res_b = int(sets[0].seqs.size), (int(sets[1].seqs.size) if kind == "cross" else 0)
    maxlen = max(int(s.lengths.max()) for s in sets)
    full = symdel.symdel_workspace_bytes(n_a, res_a, n_b, res_b, maxlen, d, cap)
    ws = torch.empty(int(full * (ws_frac or 1.0)) // 256 * 256, dtype=torch.uint8, device=dev)
    out = tuple(torch.empty(cap, dtype=torch.int32, device=dev) for _ in range(3))
    call = ctx.symdel_self if kind == "self" else ctx.symdel_cross
    stream = torch.cuda.current_stream()
    ms, r = [], None
    for it in range(steps + 1):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        r = call(*args, d, workspace=ws, out=out)
        e1.record(stream)
        e1.synchronize()
        if it:
            ms.append(e0.elapsed_time(e1))
    st = ctx.symdel_get_stats()
    i, j, dist = [t.cpu().numpy() for t in r]
    # per-stage CUDA-event times: two more steps with the library's stage timers on (not part of `ms`)
    ctx.symdel_set_option(symdel.OPT_TIMING, 1)
    tst = []
    for _ in range(2):
        call(*args, d, workspace=ws, out=out)
        tst.append(ctx.symdel_get_stats())
    ctx.symdel_set_option(symdel.OPT_TIMING, 0)
    stage_keys = ("ms_prepare", "ms_generate", "ms_sort", "ms_emit", "ms_dedup", "ms_verify", "ms_total")
    stage_ms = {k: float(np.mean([x[k] for x in tst])) for k in stage_keys}
    extra = {}
    if st["fused_chunks"] == 0 and tst[-1]["ms_sort_pass_avg"] > 0:  # exact pipeline: the onesweep passes over the records
        pass_ms = float(np.mean([x["ms_sort_pass_avg"] for x in tst]))
        extra = {"onesweep_pass_ms": pass_ms, "onesweep_passes": st["sort_bits"] // 8, "onesweep_pass_records": st["sort_pass_records"],
                 "onesweep_pass_gbs": 16 * st["sort_pass_records"] / (pass_ms * 1e-3) / 1e9}
    row = {"workload": name, "ms": float(np.mean(ms)), "ms_min": float(np.min(ms)), "ms_median": float(np.median(ms)),
           "stage_ms": stage_ms, **extra, "pairs": int(len(i)), "records": st["n_records"],
           "candidates": st["n_candidates"], "chunks": st["n_chunks"], "flushes": st["n_flushes"],
           "pipeline": "fused" if st["fused_chunks"] == st["n_chunks"] else "exact" if st["fused_chunks"] == 0 else "mixed",
           "workspace_bytes": int(ws.numel()), "steps": steps,
           "verified": bool(gold and digest(i, j, dist) == gold["out_sha256"]) if gold else None}
    if kind == "cross" and e2e_host:
        # the same search through symdel_cross_host: pinned host buffers, H2D of both sets and D2H of the result inside the call
        hb = [torch.from_numpy(a).pin_memory() for a in (sets[0].seqs, sets[0].offsets, sets[1].seqs, sets[1].offsets)]
        ho = tuple(torch.empty(cap, dtype=torch.int32).pin_memory() for _ in range(3))
        tms, k = [], 0
        for it in range(steps + 1):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            k = ctx.symdel_cross_host(*hb, d, ho)
            if it:
                tms.append(1e3 * (time.perf_counter() - t0))
        ok = bool(gold and digest(*[o[:k].numpy() for o in ho]) == gold["out_sha256"]) if gold else None
        row["e2e"] = {"api": "symdel_cross_host (pinned host buffers)", "ms": float(np.mean(tms)), "ms_min": float(np.min(tms)),
                      "ms_median": float(np.median(tms)), "h2d_bytes_per_step": int(sum(t.numel() * t.element_size() for t in hb)),
                      "d2h_bytes_per_step": int(12 * k), "verified": ok}
        del hb, ho
    if oracle_live:  # the oracle on the same workload, timed here (only where it finishes in well under a minute)
        from oracle import oracle

        t0 = time.time()
        oi = oracle.symdel_self(sets[0].seqs, sets[0].offsets, d)[0]
        row["oracle"] = oracle_record(gold, (len(oi), time.time() - t0))
    else:
        row["oracle"] = oracle_record(gold)
    ctx.close()
    del ws, out, devs, args
    torch.cuda.empty_cache()
    return row


def other_workloads(torch, symdel, synth, dev):
    """the workloads README/DESIGN quote, measured in the driver's own run."""
    rows = []

    def add(name, kind, d, sets, gold, **kw):
        try:
            rows.append(run_workload(torch, symdel, dev, name, kind, d, sets, gold, **kw))
        except Exception as e:  # a failed side workload must not lose the headline
            rows.append({"workload": name, "error": repr(e)[:200]})

    for num in (1, 2, 5):
        kind, d, sets = synth.config(num)
        add(f"config {num}", kind, d, sets, golden(f"config_{num}.json"), oracle_live=num in (1, 2))
    kind, d, sets = synth.config(5)
    add("config 5, workspace = 10 % of the un-chunked need (key-range chunking, S5)", kind, d, sets, golden("config_5.json"),
        ws_frac=0.1)
    add("config 5, FORCE_CHUNKS = 4", kind, d, sets, golden("config_5.json"), opts={"FORCE_CHUNKS": 4})
    kind, d, sets = synth.config(3)
    add("config 3, exact pipeline (SYMDEL_OPT_EXACT_PIPELINE)", kind, d, sets, golden("config_3.json"),
        opts={"EXACT_PIPELINE": 1})
    add("config 3, workspace = 10 % (chunked)", kind, d, sets, golden("config_3.json"), ws_frac=0.1)
    add("config 3, prefix P = 12 (NEXT-1)", kind, d, sets, golden("config_3.json"), opts={"PREFIX_LEN": 12})
    sets = (synth.dense_set(1_000_000, 11, fanout=64),)
    add("NEXT-2 dense: synth.dense_set(1e6, seed 11, fanout 64), d=2", "self", 2, sets, golden("dense_1m.json"), cap=32 << 20)
    # beyond 2^30 records: the planner must split by itself; no oracle golden exists at this size
    # (hours of hash map) — tests/test_gpu_parity.py::test_more_than_2_30_records pins the result another way
    sets = (synth.bcr_set(400_000, 77, lo=26, hi=30, mean=28.0, sd=1.0),)
    add("1.3 x 2^30 records: synth.bcr_set(400k, seed 77, L 26..30), d=3, no option (planner splits)", "self", 3, sets, None,
        steps=3, cap=1 << 23)
    kind, d, sets = synth.config(4)
    add("config 4 (cross 100k x 5M)", kind, d, sets, golden("config_4.json"), cap=1 << 22, e2e_host=True)
    return rows


def run_reference(args):
    """--impl reference: the CPU oracle (oracle_symdel_self, App. F.1 hash map, 1 thread)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2403_09010_b200 import synth

    kind, d, (s,) = synth.config(3)
    # bounded sample: unless --ref-sample fixes the size, a 10,000-sequence calibration run gives the oracle's cost per
    # sequence on this box and the whole run (warm-up + steps) is sized to about two minutes
    n_sample = args.ref_sample
    if not n_sample:
        _, t_cal = cpu_baseline_run(10000, d, s)
        n_sample = int(min(150000, max(5000, 120.0 / max(1, args.warmup + args.steps) / (t_cal / 10000.0))))
    n_sample = min(s.n, n_sample)
    times, pairs = [], 0
    for it in range(args.warmup + args.steps):
        pairs, dt = cpu_baseline_run(n_sample, d, s)
        if it >= args.warmup:
            times.append(dt)
    ms = 1e3 * float(np.mean(times))
    value = pairs / (ms / 1e3)
    sample = f"same generator and seed at n={n_sample}, d={d}: {pairs} pairs per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 0, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int64", "data": "synthetic", "config": {"workload": WORKLOAD, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample, **host_info()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="symdel", choices=["symdel", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config (1-based); the metric is quoted on 3")
    ap.add_argument("--ref-sample", type=int, default=0,
                    help="sequences in the oracle's bounded sample (0: 150,000 for cpu_baseline; for --impl reference sized "
                         "so that warm-up + steps take about two minutes)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-workloads", action="store_true", help="skip the `workloads` rows (the other configs, 5 steps each)")
    ap.add_argument("--dense", action="store_true",
                    help="NEXT-2 workload instead of config 3: synth.dense_set(1,000,000, seed 11, fanout 64), d=2 "
                         "(real-repertoire-like density: candidates ~ records; not the BASELINE.json headline)")
    ap.add_argument("--prefix", type=int, default=0,
                    help="prefix-truncated candidate generation (App. B; same output, fewer records); default off: the "
                         "headline generates every deletion variant of every sequence")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch

    from paper_2403_09010_b200 import symdel, synth

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    if args.dense:
        kind, d, sets = "self", 2, (synth.dense_set(1_000_000, 11, fanout=64),)
    else:
        kind, d, sets = synth.config(args.config)
    assert kind == "self"
    s = sets[0]
    ctx = symdel.Context(local)
    # the library's per-stage CUDA-event timers stay OFF (its default) while the metric is timed: the ~14 event records
    # they add between the kernels cost 0.06 ms per step; a second set of steps with the timers on gives `stages`
    if args.prefix:
        ctx.symdel_set_option(symdel.OPT_PREFIX_LEN, args.prefix)
    dev = torch.device("cuda", local)
    seqs_d = torch.from_numpy(s.seqs).to(dev)
    offs_d = torch.from_numpy(s.offsets).to(dev)
    cap = (32 << 20) if args.dense else (4 << 20)
    ws_bytes = symdel.symdel_workspace_bytes(s.n, s.seqs.size, 0, 0, int(s.lengths.max()), d, cap)
    ws = torch.empty(ws_bytes, dtype=torch.uint8, device=dev)
    out = tuple(torch.empty(cap, dtype=torch.int32, device=dev) for _ in range(3))
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    # host buffers of the end-to-end arm (pinned)
    seqs_h = torch.from_numpy(s.seqs).pin_memory()
    offs_h = torch.from_numpy(s.offsets).pin_memory()
    out_h = tuple(torch.empty(cap, dtype=torch.int32).pin_memory() for _ in range(3))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    stream = torch.cuda.current_stream()
    n_out = 0
    stats_acc = []

    def step_device(timed):
        nonlocal n_out
        flush.zero_()  # L2 flush, outside the timed events
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        i, j, dd = ctx.symdel_self(seqs_d, offs_d, d, workspace=ws, out=out)
        e1.record(stream)
        e1.synchronize()
        n_out = int(i.numel())
        if timed:
            stats_acc.append(ctx.symdel_get_stats())
        return e0.elapsed_time(e1)

    def step_host():
        flush.zero_()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        k = ctx.symdel_self_host(seqs_h, offs_h, d, out_h)
        return 1e3 * (time.perf_counter() - t0), k

    sampler = ClockSampler(local) if rank == 0 else None
    for _ in range(args.warmup):
        step_device(False)
    barrier()
    t_begin = time.time()
    ms_steps = [step_device(True) for _ in range(args.steps)]
    barrier()
    t_end = time.time()
    clocks = sampler.stop(t_begin, t_end) if sampler else None

    launches_timed = int(sum(x["n_launches"] for x in stats_acc))
    for _ in range(max(1, args.warmup)):
        step_host()
    barrier()
    e2e = [step_host() for _ in range(args.steps)]
    barrier()
    e2e_ms = float(np.mean([x[0] for x in e2e]))
    assert e2e[0][1] == n_out
    # stage breakdown: the same steps again with the stage timers on (not part of the metric)
    ctx.symdel_set_option(symdel.OPT_TIMING, 1)
    stats_acc = []
    step_device(False)
    ms_steps_timers = [step_device(True) for _ in range(args.steps)]
    ctx.symdel_set_option(symdel.OPT_TIMING, 0)

    # the timed result against the oracle's golden digest (tests/golden, written by the oracle alone)
    gold_name = "dense_1m.json" if args.dense else f"config_{args.config}.json"
    gold = golden(gold_name)
    i_d, j_d, d_d = ctx.symdel_self(seqs_d, offs_d, d, workspace=ws, out=out)
    dig_dev = digest(i_d.cpu().numpy(), j_d.cpu().numpy(), d_d.cpu().numpy())
    dig_host = digest(*[o[:n_out].numpy() for o in out_h])
    verified = bool(gold) and dig_dev == gold["out_sha256"] and dig_host == gold["out_sha256"]
    if gold and not verified:
        raise SystemExit(f"bench: output digest differs from tests/golden/{gold_name} (device {dig_dev[:12]}, host {dig_host[:12]})")

    e2e_all = [x[0] for x in e2e]
    ms, e2e_ms, ms_min, ms_med, e2e_min, e2e_med = max_over_ranks(
        [float(np.mean(ms_steps)), e2e_ms, float(np.min(ms_steps)), float(np.median(ms_steps)), float(np.min(e2e_all)),
         float(np.median(e2e_all))], dist, dev)
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    st = stats_acc[-1]
    n_rec = st["sort_pass_records"]
    n_cand = st["n_candidates"]
    fused = st["fused_chunks"] == st["n_chunks"]
    peak, peak_src = load_peak()
    stage = {k: float(np.mean([x[k] for x in stats_acc])) for k in
             ("ms_prepare", "ms_generate", "ms_sort", "ms_emit", "ms_dedup", "ms_verify", "ms_total")}
    in_bytes = s.seqs.size + 8 * (s.n + 1)
    ppass = (2 * st["id_bits"] + 7) // 8
    # Algorithmic bytes.  Fused pipeline: generation writes 8 B/record into the level-1 bins,
    # the level-2 partition reads and writes 8 B/record, the join reads 8 B/record and writes 8 B/candidate.
    # Exact pipeline: 8 (write) + 16 per onesweep pass + 8 (join read) per record.
    npass = 1 if fused else st["sort_bits"] // 8
    pass_ms = float(np.mean([x["ms_sort_pass_avg"] for x in stats_acc]))
    step_bytes = (n_rec * (8 + 16 * npass + 8) + n_cand * (8 + 8 + 16 * ppass + 8) + n_out * 12 + in_bytes)
    def hbm(name, kernel, ms_key, nbytes):
        gbs = nbytes / (stage[ms_key] * 1e-3) / 1e9 if stage[ms_key] > 0 else 0.0
        return {"stage": name, "kernel": kernel, "ms": stage[ms_key], "share_of_step": stage[ms_key] / stage["ms_total"],
                "algorithmic_bytes": int(nbytes), "achieved_gbs": gbs, "frac_of_peak": gbs / peak,
                "traffic": load_traffic(kernel)}

    # K1 writes 8 B/record (+ the input once); a partition pass moves 16 B/record; the join reads
    # 8 B/record and writes 8 B/candidate.  Each of the first three stages is ONE kernel launch on the fused pipeline.
    stages = [
        hbm("S1 generate + level-1 partition" if fused else "S1 count + scan + generate", "k_gen2_part" if fused else "k_gen2",
            "ms_generate", 8 * n_rec + in_bytes),
        hbm("S2 level-2 partition" if fused else f"S2 {npass} onesweep passes", "k_part2" if fused else "k_onesweep",
            "ms_sort", 16 * n_rec * npass),
        hbm("S3a join / emission", "k_join_bkt" if fused else "k_join_fast", "ms_emit", 8 * n_rec + 8 * n_cand),
        hbm(f"S3b candidate filter + sort ({ppass} onesweep passes)", "k_cand_filter + k_onesweep", "ms_dedup",
            n_cand * 16 + st["n_unique"] * 16 * ppass),
        hbm("S4 unique + verify + unpack", "k_verify", "ms_verify", 8 * n_cand + 64 * st["n_unique"] + 12 * n_out),
    ]
    # `roofline` describes the DOMINANT kernel of the step: the single-kernel stage with the largest share
    top = max(stages[:3], key=lambda r: r["ms"])
    line = {
        "metric": METRIC, "value": job_value(n_out, world, ms), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "ms_per_step_min": ms_min, "ms_per_step_median": ms_med,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u64", "data": "synthetic",
        "config": {"workload": ("NEXT-2 dense: synth.dense_set(1e6, seed 11, fanout 64), d=2" if args.dense else
                                WORKLOAD if args.config == 3 else f"config {args.config}"), "n": s.n, "d": d,
                   "pairs_per_step": n_out, "records": n_rec, "candidates": n_cand,
                   "unique_candidates": st["n_unique"], "hash_bits": st["hash_bits"], "id_bits": st["id_bits"],
                   "partition_bits": st["sort_bits"], "pipeline": "fused" if fused else "exact",
                   "prefix_len": args.prefix or None,
                   "chunks": st["n_chunks"], "l2": "flushed between steps (512 MiB memset, untimed)",
                   "parallelism": "replicas only" if world > 1 else "1 GPU"},
        "verified": verified,
        "wall_time_s": ms * 1e-3, "records_per_s": world * n_rec / (ms * 1e-3),
        "step_hbm_gbs": step_bytes / (ms * 1e-3) / 1e9, "step_hbm_frac": step_bytes / (ms * 1e-3) / 1e9 / peak,
        "stage_ms": stage, "stages": stages,
        "e2e": {"value": job_value(n_out, world, e2e_ms), "unit": UNIT, "ms_per_step": e2e_ms, "ms_per_step_min": e2e_min,
                "ms_per_step_median": e2e_med,
                "h2d_bytes_per_step": int(s.seqs.nbytes + s.offsets.nbytes), "d2h_bytes_per_step": int(12 * n_out),
                "api": "symdel_self_host (pinned host buffers)"},
        "gpu_launches": launches_timed,
        "ms_per_step_with_stage_timers": float(np.mean(ms_steps_timers)),
        "stage_timing": f"{args.steps} further steps with SYMDEL_OPT_TIMING = 1 (CUDA events between the kernels, on the launching stream); "
                        "the metric's steps run with the timers off, the library's default",
        "roofline": {"bound": "hbm", "kernel": f"{top['kernel']} ({top['stage']}; the longest kernel of the step)",
                     "achieved": top["achieved_gbs"], "peak": peak, "unit": "GB/s", "frac": top["frac_of_peak"],
                     "traffic": top["traffic"], "peak_source": peak_src,
                     "algorithmic_bytes_per_launch": top["algorithmic_bytes"], "launch_ms": top["ms"],
                     "share_of_step": top["share_of_step"], "frac_of_nominal_8000": top["achieved_gbs"] / 8000.0},
        "clocks": clocks,
    }
    # What limits the longest kernel: the HBM figure above is what the contract asks for; k_gen2_part itself is
    # bound by instruction issue (DESIGN.md section 6 ablations), k_part2 is the HBM-bound kernel.  Issue roofline: warp
    # instructions per launch (ncu --set full, profiles/traffic.json) / launch time against 148 SMs x 4 schedulers x SM clock.
    winst = load_traffic(top["kernel"] + "_warp_instructions")
    sm_mhz = (clocks or {}).get("sm_mhz") or (clocks or {}).get("sm_max_mhz") or 1965.0
    if winst and top["ms"] > 0:
        issue_peak = 148 * 4 * sm_mhz * 1e6 / 1e9  # G warp-instructions/s
        issue = winst / (top["ms"] * 1e-3) / 1e9
        line["roofline"]["limiter"] = ("hbm" if top["frac_of_peak"] >= 0.5 else "issue" if issue / issue_peak >= 0.45 else
                                       "latency (shared-memory wavefronts / resident warps)")
        line["roofline_issue"] = {"bound": "alu", "kernel": top["kernel"], "achieved": issue, "peak": issue_peak,
                                  "unit": "G warp-instructions/s", "frac": issue / issue_peak,
                                  "warp_instructions_per_launch": winst, "sm_mhz": sm_mhz,
                                  "peak_source": "148 SMs x 4 warp schedulers x SM clock (one warp instruction per scheduler per cycle)",
                                  "source": "instruction count from the committed ncu --set full capture (profiles/traffic.json)"}
    hbm_stage = max(stages[:3], key=lambda r: r["frac_of_peak"])
    line["roofline_hbm_bound_kernel"] = {"bound": "hbm", "kernel": hbm_stage["kernel"], "achieved": hbm_stage["achieved_gbs"], "peak": peak,
                                         "unit": "GB/s", "frac": hbm_stage["frac_of_peak"], "traffic": hbm_stage["traffic"],
                                         "launch_ms": hbm_stage["ms"], "share_of_step": hbm_stage["share_of_step"]}
    if not args.no_cpu_baseline and world == 1 and not args.dense:
        n_sample = min(s.n, args.ref_sample or 150000)
        pairs, dt = cpu_baseline_run(n_sample, d, s)
        line["cpu_baseline"] = {"value": pairs / dt, "unit": UNIT, "cores": 1, "kind": "oracle", **host_info(),
                                "sample": f"same generator and seed at n={n_sample}, d={d}: {pairs} pairs in {dt:.1f} s "
                                          "(oracle_symdel_self, App. F.1 hash map)"}
        if gold and gold.get("oracle_wall_s"):
            line["cpu_baseline_full"] = {
                "value": gold["n_out"] / gold["oracle_wall_s"], "unit": UNIT, "cores": 1, "kind": "oracle",
                "sample": f"the whole workload, recorded when tests/golden/{gold_name} was written (another host): "
                          f"{gold['n_out']} pairs in {gold['oracle_wall_s']} s"}
    if world == 1 and not args.no_workloads and args.config == 3 and not args.dense and not args.prefix:
        del ws, out, flush
        torch.cuda.empty_cache()
        line["workloads"] = other_workloads(torch, symdel, synth, dev)
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
