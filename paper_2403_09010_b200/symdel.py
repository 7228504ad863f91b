"""Thin ctypes binding of libsymdel (include/symdel.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI.  PyTorch is used for device
memory and the current stream; there is no CPU fallback: if `libsymdel.so` is missing or no CUDA
device is present the calls raise.  This module never imports `oracle/`.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SO = _HERE / "libsymdel.so"
_lib = None

OK = 0
E_ARG, E_OFFSETS, E_TOO_LONG, E_RESIDUE, E_TOO_MANY, E_WORKSPACE, E_CAPACITY, E_CUDA, E_INTERNAL = range(-1, -10, -1)
E_STATIC_LIMIT = -10
STATIC_SORT_MAX_KEYS, STATIC_SORT_SCRATCH_BYTES = 1 << 20, 11 << 20
OPT_TIMING, OPT_FORCE_CHUNKS, OPT_CAND_CAPACITY, OPT_HASH_BITS, OPT_NO_THINNING, OPT_SORT_VARIANT, OPT_GENERAL_GENERATE = 1, 2, 3, 4, 5, 6, 7
OPT_SORT_BITS, OPT_SORT_STABLE, OPT_SORT_GROUPING, OPT_JOIN_GENERAL, OPT_EXACT_PIPELINE, OPT_PREFIX_LEN, OPT_METRIC = 8, 9, 10, 11, 12, 13, 14
OPT_SURV_CAPACITY, OPT_CAND_FILTER, OPT_NO_QUERY_FILTER, OPT_FLUSH_PER_CHUNK = 15, 16, 17, 18
METRIC_LEVENSHTEIN, METRIC_HAMMING = 0, 1
D_MAX, L_MAX = 4, 64

EXPORTS = [
    "symdel_create", "symdel_destroy", "symdel_set_option", "symdel_get_stats", "symdel_last_cuda_error",
    "symdel_strerror", "symdel_workspace_bytes", "symdel_self", "symdel_cross", "symdel_self_host",
    "symdel_cross_host", "symdel_stage_sort_workspace_bytes", "symdel_stage_sort_u64", "symdel_stage_generate",
    "symdel_stage_lev", "symdel_overlap_matrix", "symdel_sort_u64_static",
    "symdel_stage_generate_fused",
]


class Stats(C.Structure):
    _fields_ = [
        ("n_records", C.c_int64), ("n_candidates", C.c_int64), ("n_unique", C.c_int64), ("n_outputs", C.c_int64),
        ("n_chunks", C.c_int64), ("n_flushes", C.c_int64), ("n_launches", C.c_int64),
        ("hash_bits", C.c_int32), ("id_bits", C.c_int32), ("sort_bits", C.c_int32), ("join_general", C.c_int32),
        ("ms_prepare", C.c_float), ("ms_generate", C.c_float), ("ms_sort", C.c_float), ("ms_emit", C.c_float),
        ("ms_dedup", C.c_float), ("ms_verify", C.c_float), ("ms_total", C.c_float), ("ms_sort_pass_avg", C.c_float),
        ("sort_pass_records", C.c_int64), ("fused_chunks", C.c_int64), ("join_redo_tiles", C.c_int64),
        ("surv_merges", C.c_int64), ("join_windows", C.c_int64), ("query_filter_bits", C.c_int64),
    ]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class SymdelError(RuntimeError):
    def __init__(self, code, where, extra=""):
        self.code = code
        msg = lib().symdel_strerror(code).decode()
        super().__init__(f"{where}: {msg} (code {code}){extra}")


def lib():
    """Loads libsymdel.so (built by `__graft_entry__.build()` / `build.build_native()`); fails loudly."""
    global _lib
    if _lib is None:
        if not _SO.exists():
            raise RuntimeError(f"{_SO} is missing: build it with `python -m paper_2403_09010_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(str(_SO))
        vp, i64, i32 = C.c_void_p, C.c_int64, C.c_int
        L.symdel_create.argtypes = [C.POINTER(vp), i32]
        L.symdel_destroy.argtypes = [vp]
        L.symdel_destroy.restype = None
        L.symdel_set_option.argtypes = [vp, i32, i64]
        L.symdel_get_stats.argtypes = [vp, C.POINTER(Stats)]
        L.symdel_last_cuda_error.argtypes = [vp]
        L.symdel_strerror.argtypes = [i32]
        L.symdel_strerror.restype = C.c_char_p
        L.symdel_workspace_bytes.argtypes = [i64, i64, i64, i64, i32, i32, i64, C.POINTER(i64)]
        L.symdel_self.argtypes = [vp, vp, vp, i64, i32, vp, i64, vp, vp, vp, i64, C.POINTER(i64), vp]
        L.symdel_cross.argtypes = [vp, vp, vp, i64, vp, vp, i64, i32, vp, i64, vp, vp, vp, i64, C.POINTER(i64), vp]
        L.symdel_self_host.argtypes = [vp, vp, vp, i64, i32, vp, vp, vp, i64, C.POINTER(i64)]
        L.symdel_cross_host.argtypes = [vp, vp, vp, i64, vp, vp, i64, i32, vp, vp, vp, i64, C.POINTER(i64)]
        L.symdel_stage_sort_workspace_bytes.argtypes = [i64]
        L.symdel_stage_sort_workspace_bytes.restype = i64
        L.symdel_stage_sort_u64.argtypes = [vp, vp, vp, i64, i32, i32, vp, i64, vp]
        L.symdel_stage_generate.argtypes = [vp, vp, vp, i64, i32, i32, i32, i32, vp, i64, C.POINTER(i64), vp, i64, vp]
        L.symdel_stage_generate_fused.argtypes = [vp, vp, vp, i64, i32, i32, i32, i32, i32, C.c_uint64, C.c_uint64, vp, i64, vp,
                                                  C.POINTER(i64), vp, i64, vp]
        L.symdel_stage_lev.argtypes = [vp, vp, vp, i64, vp, vp, i64, vp, vp, i64, vp, vp, i64, vp]
        L.symdel_overlap_matrix.argtypes = [vp, vp, vp, i64, vp, i64, vp, i64, i32, i32, vp, vp, i64, vp]
        L.symdel_sort_u64_static.argtypes = [i32, vp, i64, i32, i32, vp]
        _lib = L
    return _lib


def symdel_workspace_bytes(n_a, residues_a, n_b=0, residues_b=0, max_len=L_MAX, d=2, capacity=0) -> int:
    out = C.c_int64(0)
    rc = lib().symdel_workspace_bytes(n_a, residues_a, n_b, residues_b, max_len, d, capacity, C.byref(out))
    if rc:
        raise SymdelError(rc, "symdel_workspace_bytes")
    return int(out.value)


def symdel_sort_u64_static(keys, begin_bit: int, end_bit: int):
    """symdel_sort_u64_static: the stable radix sort of `Context.symdel_stage_sort_u64`, in place on a uint64-as-int64
    CUDA tensor of at most STATIC_SORT_MAX_KEYS keys, for code that may not allocate device memory (a host application
    that owns the whole GPU, a loop where cudaMalloc's device-wide synchronisation is not acceptable).  No Context, no
    workspace and no temporary tensor: the scratch is an 11 MiB array built into libsymdel.so, one per GPU, shared by
    every call — calls on one device must not overlap, and the first call on a device (it does a one-time address
    look-up) belongs before any stream capture.  More keys than the limit raise SymdelError(E_STATIC_LIMIT)."""
    torch = _torch()
    dev = keys.device.index if keys.device.index is not None else torch.cuda.current_device()
    with torch.cuda.device(dev):
        rc = lib().symdel_sort_u64_static(dev, C.c_void_p(keys.data_ptr()), keys.numel(), begin_bit, end_bit, _stream_ptr(torch))
    if rc:
        raise SymdelError(rc, "symdel_sort_u64_static")
    return keys


def _torch():
    import torch

    if not torch.cuda.is_available():
        raise RuntimeError("libsymdel needs a CUDA device (no CPU fallback)")
    return torch


def _stream_ptr(torch):
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


class Context:
    """symdel_ctx wrapper.  Methods carry the names of the C entry points they call."""

    def __init__(self, device: int = 0):
        self._h = C.c_void_p()
        rc = lib().symdel_create(C.byref(self._h), device)
        if rc:
            raise SymdelError(rc, "symdel_create")
        self.device = device

    def close(self):
        if self._h:
            lib().symdel_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def symdel_set_option(self, option: int, value: int):
        rc = lib().symdel_set_option(self._h, option, value)
        if rc:
            raise SymdelError(rc, "symdel_set_option")

    def symdel_get_stats(self) -> dict:
        s = Stats()
        lib().symdel_get_stats(self._h, C.byref(s))
        return s.as_dict()

    def _raise(self, rc, where):
        extra = ""
        if rc == E_CUDA:
            extra = f" cudaError={lib().symdel_last_cuda_error(self._h)}"
        raise SymdelError(rc, where, extra)

    # ---- device-resident entry points (torch CUDA tensors in, torch CUDA tensors out) ----
    def symdel_self(self, seqs, offsets, d: int, workspace=None, capacity: int | None = None, out=None):
        """seqs: int8 CUDA tensor, offsets: int64 CUDA tensor [n+1].  Returns (i, j, dist) int32 CUDA tensors."""
        return self._run(seqs, offsets, None, None, d, workspace, capacity, out)

    def symdel_cross(self, q_seqs, q_offsets, r_seqs, r_offsets, d: int, workspace=None, capacity: int | None = None,
                     out=None):
        return self._run(q_seqs, q_offsets, r_seqs, r_offsets, d, workspace, capacity, out)

    def _run(self, a_seqs, a_off, b_seqs, b_off, d, workspace, capacity, out):
        torch = _torch()
        cross = b_off is not None
        n_a = a_off.numel() - 1
        n_b = b_off.numel() - 1 if cross else 0
        if out is None:
            cap = capacity if capacity is not None else max(1 << 20, 4 * (n_a + n_b))
            out = tuple(torch.empty(cap, dtype=torch.int32, device=a_off.device) for _ in range(3))
        cap = out[0].numel()
        if workspace is None:
            nbytes = symdel_workspace_bytes(n_a, a_seqs.numel(), n_b, b_seqs.numel() if cross else 0, L_MAX, d, cap)
            workspace = torch.empty(nbytes, dtype=torch.uint8, device=a_off.device)
        n_pairs = C.c_int64(0)
        L = lib()
        p = lambda t: C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)
        if cross:
            rc = L.symdel_cross(self._h, p(a_seqs), p(a_off), n_a, p(b_seqs), p(b_off), n_b, d, p(workspace),
                                workspace.numel(), p(out[0]), p(out[1]), p(out[2]), cap, C.byref(n_pairs),
                                _stream_ptr(torch))
        else:
            rc = L.symdel_self(self._h, p(a_seqs), p(a_off), n_a, d, p(workspace), workspace.numel(), p(out[0]), p(out[1]),
                               p(out[2]), cap, C.byref(n_pairs), _stream_ptr(torch))
        if rc:
            self.last_required = int(n_pairs.value)
            self._raise(rc, "symdel_cross" if cross else "symdel_self")
        k = int(n_pairs.value)
        return out[0][:k], out[1][:k], out[2][:k]

    # ---- host-buffer entry points (numpy / pinned torch CPU tensors) ----
    def symdel_self_host(self, seqs, offsets, d: int, out):
        """seqs int8 / offsets int64 host arrays; out = three int32 host arrays of equal length (capacity)."""
        n_pairs = C.c_int64(0)
        rc = lib().symdel_self_host(self._h, _hp(seqs), _hp(offsets), _hlen(offsets) - 1, d, _hp(out[0]), _hp(out[1]),
                                    _hp(out[2]), _hlen(out[0]), C.byref(n_pairs))
        if rc:
            self.last_required = int(n_pairs.value)
            self._raise(rc, "symdel_self_host")
        return int(n_pairs.value)

    def symdel_cross_host(self, q_seqs, q_offsets, r_seqs, r_offsets, d: int, out):
        n_pairs = C.c_int64(0)
        rc = lib().symdel_cross_host(self._h, _hp(q_seqs), _hp(q_offsets), _hlen(q_offsets) - 1, _hp(r_seqs),
                                     _hp(r_offsets), _hlen(r_offsets) - 1, d, _hp(out[0]), _hp(out[1]), _hp(out[2]),
                                     _hlen(out[0]), C.byref(n_pairs))
        if rc:
            self.last_required = int(n_pairs.value)
            self._raise(rc, "symdel_cross_host")
        return int(n_pairs.value)

    # ---- stage-level entry points ----
    def symdel_stage_sort_u64(self, keys, begin_bit: int, end_bit: int):
        """In-place stable LSD radix sort of a uint64-as-int64 CUDA tensor on bits [begin_bit, end_bit)."""
        torch = _torch()
        n = keys.numel()
        tmp = torch.empty_like(keys)
        wsb = lib().symdel_stage_sort_workspace_bytes(n)
        ws = torch.empty(wsb, dtype=torch.uint8, device=keys.device)
        rc = lib().symdel_stage_sort_u64(self._h, C.c_void_p(keys.data_ptr()), C.c_void_p(tmp.data_ptr()), n, begin_bit,
                                         end_bit, C.c_void_p(ws.data_ptr()), wsb, _stream_ptr(torch))
        if rc:
            self._raise(rc, "symdel_stage_sort_u64")
        return keys

    def symdel_stage_generate(self, seqs, offsets, d: int, hash_bits: int, id_bits: int, thinning: bool, capacity: int):
        torch = _torch()
        n = offsets.numel() - 1
        rec = torch.empty(max(capacity, 1), dtype=torch.int64, device=offsets.device)
        wsb = 16 * (n + 4096) + (1 << 16)
        ws = torch.empty(wsb, dtype=torch.uint8, device=offsets.device)
        cnt = C.c_int64(0)
        rc = lib().symdel_stage_generate(self._h, C.c_void_p(seqs.data_ptr()), C.c_void_p(offsets.data_ptr()), n, d,
                                         hash_bits, id_bits, int(thinning), C.c_void_p(rec.data_ptr()), capacity,
                                         C.byref(cnt), C.c_void_p(ws.data_ptr()), wsb, _stream_ptr(torch))
        if rc:
            self._raise(rc, "symdel_stage_generate")
        return rec[: int(cnt.value)]

    def symdel_stage_generate_fused(self, seqs, offsets, d: int, hash_bits: int, id_bits: int, thinning: bool, bin_capacity: int,
                                    n_chunks: int = 1, chunk_lo: int = 0, chunk_hi: int = 0):
        """Returns (bins int64[256, bin_capacity], counts int32[256]) of the fused generator (CUDA tensors)."""
        torch = _torch()
        n = offsets.numel() - 1
        bins = torch.zeros((256, bin_capacity), dtype=torch.int64, device=offsets.device)
        counts = torch.zeros(256, dtype=torch.int32, device=offsets.device)
        ws = torch.empty(1 << 16, dtype=torch.uint8, device=offsets.device)
        cnt = C.c_int64(0)
        rc = lib().symdel_stage_generate_fused(self._h, C.c_void_p(seqs.data_ptr()), C.c_void_p(offsets.data_ptr()), n, d, hash_bits,
                                               id_bits, int(thinning), n_chunks, chunk_lo, chunk_hi, C.c_void_p(bins.data_ptr()),
                                               bin_capacity, C.c_void_p(counts.data_ptr()), C.byref(cnt),
                                               C.c_void_p(ws.data_ptr()), ws.numel(), _stream_ptr(torch))
        if rc:
            self.last_required = int(cnt.value)
            self._raise(rc, "symdel_stage_generate_fused")
        assert int(counts.sum()) == int(cnt.value)
        return bins, counts

    def symdel_stage_lev(self, a_seqs, a_offsets, b_seqs, b_offsets, ia, ib):
        torch = _torch()
        dist = torch.empty(ia.numel(), dtype=torch.int32, device=ia.device)
        q = lambda t: C.c_void_p(t.data_ptr())
        wsb = 1024 + 48 * (a_offsets.numel() + b_offsets.numel())
        ws = torch.empty(wsb, dtype=torch.uint8, device=ia.device)
        rc = lib().symdel_stage_lev(self._h, q(a_seqs), q(a_offsets), a_offsets.numel() - 1, q(b_seqs), q(b_offsets),
                                    b_offsets.numel() - 1, q(ia), q(ib), ia.numel(), q(dist), q(ws), wsb,
                                    _stream_ptr(torch))
        if rc:
            self._raise(rc, "symdel_stage_lev")
        return dist

    def symdel_overlap_matrix(self, out_i, out_j, labels_i, labels_j, n_repertoires: int, symmetric: bool):
        """M x M overlap matrix (int64 CUDA tensor) of result pairs under per-sequence repertoire labels (int32)."""
        torch = _torch()
        m = torch.empty((n_repertoires, n_repertoires), dtype=torch.int64, device=labels_i.device)
        ws = torch.empty(256, dtype=torch.uint8, device=labels_i.device)
        q = lambda t: C.c_void_p(t.data_ptr())
        rc = lib().symdel_overlap_matrix(self._h, q(out_i), q(out_j), out_i.numel(), q(labels_i), labels_i.numel(), q(labels_j),
                                         labels_j.numel(), n_repertoires, 1 if symmetric else 0, q(m), q(ws), 256,
                                         _stream_ptr(torch))
        if rc:
            self._raise(rc, "symdel_overlap_matrix")
        return m


def _hp(a):
    if isinstance(a, np.ndarray):
        return C.c_void_p(a.ctypes.data)
    return C.c_void_p(a.data_ptr())  # torch CPU tensor (pinned or not)


def _hlen(a):
    return int(a.size) if isinstance(a, np.ndarray) else int(a.numel())


def to_device(seqset, device="cuda"):
    """SeqSet (numpy CSR) -> (seqs int8, offsets int64) CUDA tensors; an empty seqs gets one pad byte."""
    torch = _torch()
    seqs = seqset.seqs if seqset.seqs.size else np.zeros(1, np.int8)
    return torch.from_numpy(np.ascontiguousarray(seqs)).to(device), torch.from_numpy(
        np.ascontiguousarray(seqset.offsets)).to(device)
