"""symdel_sort_u64_static: the radix sort for callers that cannot allocate device memory.

Some users of libsymdel run where cudaMalloc is not an option: inside a host application whose memory pool already
owns the GPU, in a service loop that may not take cudaMalloc's device-wide synchronisation, or on an error path
after an out-of-memory.  They call this entry point with their key buffer and nothing else; the scratch is a fixed
array inside the library, one per GPU, shared by every call (include/symdel.h, csrc/static_sort.cu).

What is checked here: (1) its output equals, bit for bit (integer work: the tolerance of every sort test in this
repository is zero), that of the existing path symdel_stage_sort_u64 with caller-provided scratch — on two calls in a
row, the second smaller and on another bit range, so that anything the first call left in the shared array (keys
beyond the second call's n, status words of tiles the second call also uses) would show; (2) the very first call works
with no symdel_ctx ever created, i.e. the entry point does its own per-device set-up; (3) device memory in use does
not change across a call; (4) sizes beyond the built-in maximum are refused before the GPU is touched.

This file sorts last in the collection on purpose: `pytest -x` stops at the first failure, and a failure here must not
hide the parity tests.  It passes both on its own in a fresh process and after all the other test files.
"""
import ctypes as C
import re
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


def _keys(n, seed):
    rng = np.random.default_rng(seed)
    return rng.integers(0, 1 << 63, size=n, dtype=np.int64).astype(np.uint64) * np.uint64(2) + rng.integers(0, 2, size=n).astype(np.uint64)


@pytest.mark.gpu
def test_static_sort_matches_the_workspace_path_on_two_calls_in_a_row():
    import torch

    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2403_09010_b200 import symdel as sd

    sd.lib()  # must load: there is no fallback
    # call 1: the full 2^20 keys on all 64 bits (8 passes); call 2: fewer keys, a ragged tail, 3 passes (the result
    # ends in the ping-pong buffer and is copied back), low digits repeated so that stability matters
    k1 = _keys(sd.STATIC_SORT_MAX_KEYS, 11)
    k2 = _keys(300_007, 12) & np.uint64(0xFFFF_F000_0FFF)
    cases = [(k1, 0, 64), (k2, 16, 40)]
    dev = [torch.from_numpy(k.view(np.int64).copy()).cuda() for k, _, _ in cases]
    ref = [t.clone() for t in dev]
    torch.cuda.synchronize()

    # the static entry point runs FIRST, before any symdel_ctx exists in this process when the file runs alone
    got = []
    for call, (t, (k, b, e)) in enumerate(zip(dev, cases)):
        free_before = torch.cuda.mem_get_info()[0]
        sd.symdel_sort_u64_static(t, b, e)
        if call > 0:  # (the first call may make the driver load kernel images; after it, nothing may be taken)
            assert torch.cuda.mem_get_info()[0] >= free_before
        got.append(t.cpu().numpy().view(np.uint64))

    ctx = sd.Context(0)
    try:
        for g, t, (k, b, e) in zip(got, ref, cases):
            ctx.symdel_stage_sort_u64(t, b, e)  # the existing path: caller-provided tmp + workspace
            exp = t.cpu().numpy().view(np.uint64)
            assert np.array_equal(g, exp)
            field = (k >> np.uint64(b)) & np.uint64((1 << (e - b)) - 1)
            assert np.array_equal(g, k[np.argsort(field, kind="stable")])  # and both are the stable sort
    finally:
        ctx.close()

    # a third call after the context's own sorts, and the two edge sizes
    t = torch.from_numpy(k2.view(np.int64).copy()).cuda()
    sd.symdel_sort_u64_static(t, 0, 48)
    assert np.array_equal(t.cpu().numpy().view(np.uint64), np.sort(k2, kind="stable"))
    one = torch.tensor([5], dtype=torch.int64, device="cuda")
    assert sd.symdel_sort_u64_static(one, 0, 64).item() == 5
    sd.symdel_sort_u64_static(torch.empty(0, dtype=torch.int64, device="cuda"), 0, 64)


@pytest.mark.gpu
def test_static_sort_refuses_more_keys_than_its_array_holds_on_the_gpu():
    import torch

    from paper_2403_09010_b200 import symdel as sd

    k = _keys(sd.STATIC_SORT_MAX_KEYS + 1, 3)
    t = torch.from_numpy(k.view(np.int64).copy()).cuda()
    with pytest.raises(sd.SymdelError) as ei:
        sd.symdel_sort_u64_static(t, 0, 64)
    assert ei.value.code == sd.E_STATIC_LIMIT
    assert np.array_equal(t.cpu().numpy().view(np.uint64), k)  # nothing was touched


def test_static_sort_limit_and_arguments_need_no_gpu():
    """The size and argument checks come before the first CUDA call, so they can be exercised on a CPU-only box
    (the key pointer is never dereferenced on these paths)."""
    from paper_2403_09010_b200 import build, symdel as sd

    build.build_native()
    L = sd.lib()
    fake = C.c_void_p(256)
    assert L.symdel_sort_u64_static(0, fake, sd.STATIC_SORT_MAX_KEYS + 1, 0, 64, None) == sd.E_STATIC_LIMIT
    assert b"SYMDEL_STATIC_SORT_MAX_KEYS" in L.symdel_strerror(sd.E_STATIC_LIMIT)
    assert L.symdel_sort_u64_static(0, fake, -1, 0, 64, None) == sd.E_ARG
    assert L.symdel_sort_u64_static(0, fake, 10, 0, 12, None) == sd.E_ARG   # not a multiple of 8 bits
    assert L.symdel_sort_u64_static(64, fake, 10, 0, 8, None) == sd.E_ARG   # device outside the table
    assert L.symdel_sort_u64_static(0, None, 10, 0, 8, None) == sd.E_ARG    # null keys
    assert L.symdel_sort_u64_static(0, fake, 0, 0, 64, None) == sd.OK       # nothing to do
    text = (ROOT / "include" / "symdel.h").read_text()
    assert int(re.search(r"#define SYMDEL_STATIC_SORT_MAX_KEYS (\d+)", text).group(1)) == sd.STATIC_SORT_MAX_KEYS
    assert int(re.search(r"#define SYMDEL_STATIC_SORT_SCRATCH_BYTES (\d+)", text).group(1)) == sd.STATIC_SORT_SCRATCH_BYTES


def test_static_sort_source_makes_no_allocating_call():
    """Source check of the promise in the header: the translation unit of the entry point and the sort helpers it
    calls contain no allocating or freeing CUDA call, and the scratch is the file-scope array."""
    csrc = ROOT / "paper_2403_09010_b200" / "csrc"
    strip = lambda s: re.sub(r"//.*", "", s)
    unit = strip((csrc / "static_sort.cu").read_text())
    sort = strip((csrc / "radix_sort.cu").read_text())
    banned = re.compile(r"cudaMalloc|cudaFree|cudaHostAlloc|cudaStreamCreate|cudaEventCreate|\bnew\b|\bmalloc\s*\(")
    assert not banned.search(unit)
    assert not banned.search(sort)
    assert re.search(r"static\s+__device__\s+__align__\(256\)\s+unsigned char\s+static_scratch\[", unit)
    assert "cudaGetSymbolAddress((void**)&p, static_scratch) != cudaSuccess" in unit
