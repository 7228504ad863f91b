"""ctypes loader for the CPU oracle (oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SO = _HERE / "liboracle.so"
_SRC = _HERE / "oracle.cpp"
_lib = None


def build(force: bool = False) -> Path:
    """g++ -O2 -fopenmp oracle.cpp -> liboracle.so (rebuilt when the source is newer)."""
    if force or not _SO.exists() or _SO.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-shared", "-fPIC", str(_SRC), "-o", str(_SO)]
        subprocess.run(cmd, check=True)
    return _SO


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_SO))
        p8, p64, p32, vp = C.POINTER(C.c_int8), C.POINTER(C.c_int64), C.POINTER(C.c_int32), C.c_void_p
        L.oracle_lev.restype = C.c_int
        L.oracle_lev.argtypes = [p8, C.c_int, p8, C.c_int]
        L.oracle_deletion_variants.restype = C.c_int64
        L.oracle_deletion_variants.argtypes = [p8, C.c_int, C.c_int, p8, C.c_int64]
        L.oracle_bruteforce_self.restype = vp
        L.oracle_bruteforce_self.argtypes = [p8, p64, C.c_int64, C.c_int, C.c_int]
        L.oracle_bruteforce_cross.restype = vp
        L.oracle_bruteforce_cross.argtypes = [p8, p64, C.c_int64, p8, p64, C.c_int64, C.c_int, C.c_int]
        L.oracle_bruteforce_hamming_self.restype = vp
        L.oracle_bruteforce_hamming_self.argtypes = [p8, p64, C.c_int64, C.c_int]
        L.oracle_bruteforce_hamming_cross.restype = vp
        L.oracle_bruteforce_hamming_cross.argtypes = [p8, p64, C.c_int64, p8, p64, C.c_int64, C.c_int]
        L.oracle_bruteforce_row.restype = vp
        L.oracle_bruteforce_row.argtypes = [p8, C.c_int, p8, p64, C.c_int64, C.c_int]
        L.oracle_symdel_self.restype = vp
        L.oracle_symdel_self.argtypes = [p8, p64, C.c_int64, C.c_int]
        L.oracle_symdel_cross.restype = vp
        L.oracle_symdel_cross.argtypes = [p8, p64, C.c_int64, p8, p64, C.c_int64, C.c_int]
        L.oracle_result_size.restype = C.c_int64
        L.oracle_result_size.argtypes = [vp]
        L.oracle_result_counters.argtypes = [vp, p64]
        L.oracle_result_copy.argtypes = [vp, p32, p32, p32]
        L.oracle_result_free.argtypes = [vp]
        L.oracle_max_threads.restype = C.c_int
        _lib = L
    return _lib


def _p8(a):
    return a.ctypes.data_as(C.POINTER(C.c_int8))


def _p64(a):
    return a.ctypes.data_as(C.POINTER(C.c_int64))


def _csr(seqs, offsets):
    seqs = np.ascontiguousarray(seqs, dtype=np.int8)
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    if seqs.size == 0:
        seqs = np.zeros(1, dtype=np.int8)  # keep a valid pointer
    return seqs, offsets


def _take(h, with_counters=False):
    L = lib()
    n = L.oracle_result_size(h)
    i = np.empty(n, np.int32)
    j = np.empty(n, np.int32)
    d = np.empty(n, np.int32)
    p32 = C.POINTER(C.c_int32)
    if n:
        L.oracle_result_copy(h, i.ctypes.data_as(p32), j.ctypes.data_as(p32), d.ctypes.data_as(p32))
    c = np.zeros(3, np.int64)
    L.oracle_result_counters(h, _p64(c))
    L.oracle_result_free(h)
    if with_counters:
        return i, j, d, dict(n_variants=int(c[0]), n_matched=int(c[1]), n_unique=int(c[2]))
    return i, j, d


def lev(a, b) -> int:
    a = np.ascontiguousarray(a, dtype=np.int8)
    b = np.ascontiguousarray(b, dtype=np.int8)
    pa = _p8(a) if a.size else _p8(np.zeros(1, np.int8))
    pb = _p8(b) if b.size else _p8(np.zeros(1, np.int8))
    return int(lib().oracle_lev(pa, int(a.size), pb, int(b.size)))


def deletion_variants(s, d: int):
    """All deletion variants of `s` up to depth d (one per deletion set), as a list of bytes."""
    s = np.ascontiguousarray(s, dtype=np.int8)
    cap = 1 << 24
    buf = np.empty(cap, np.int8)
    n = lib().oracle_deletion_variants(_p8(s) if s.size else _p8(np.zeros(1, np.int8)), int(s.size), int(d), _p8(buf), cap)
    assert n >= 0
    out, pos = [], 0
    for _ in range(n):
        ln = int(buf[pos])
        out.append(bytes(buf[pos + 1:pos + 1 + ln].view(np.uint8)))
        pos += 1 + ln
    return out


def bruteforce_self(seqs, offsets, d: int, threads: int = 0):
    seqs, offsets = _csr(seqs, offsets)
    return _take(lib().oracle_bruteforce_self(_p8(seqs), _p64(offsets), offsets.size - 1, int(d), int(threads)))


def bruteforce_cross(qs, qo, rs, ro, d: int, threads: int = 0):
    qs, qo = _csr(qs, qo)
    rs, ro = _csr(rs, ro)
    return _take(lib().oracle_bruteforce_cross(_p8(qs), _p64(qo), qo.size - 1, _p8(rs), _p64(ro), ro.size - 1, int(d),
                                               int(threads)))


def hamming_self(seqs, offsets, d: int):
    """NEXT-3: every (i, j, hamming) with i < j, equal lengths and <= d mismatches (plain double loop)."""
    seqs, offsets = _csr(seqs, offsets)
    return _take(lib().oracle_bruteforce_hamming_self(_p8(seqs), _p64(offsets), offsets.size - 1, int(d)))


def hamming_cross(qs, qo, rs, ro, d: int):
    qs, qo = _csr(qs, qo)
    rs, ro = _csr(rs, ro)
    return _take(lib().oracle_bruteforce_hamming_cross(_p8(qs), _p64(qo), qo.size - 1, _p8(rs), _p64(ro), ro.size - 1, int(d)))


def bruteforce_row(probe, rs, ro, d: int):
    """(r, dist) for every reference r within distance d of one probe sequence."""
    probe = np.ascontiguousarray(probe, dtype=np.int8)
    rs, ro = _csr(rs, ro)
    pp = _p8(probe) if probe.size else _p8(np.zeros(1, np.int8))
    _, j, dist = _take(lib().oracle_bruteforce_row(pp, int(probe.size), _p8(rs), _p64(ro), ro.size - 1, int(d)))
    return j, dist


def symdel_self(seqs, offsets, d: int, with_counters=False):
    seqs, offsets = _csr(seqs, offsets)
    return _take(lib().oracle_symdel_self(_p8(seqs), _p64(offsets), offsets.size - 1, int(d)), with_counters)


def symdel_cross(qs, qo, rs, ro, d: int, with_counters=False):
    qs, qo = _csr(qs, qo)
    rs, ro = _csr(rs, ro)
    return _take(lib().oracle_symdel_cross(_p8(qs), _p64(qo), qo.size - 1, _p8(rs), _p64(ro), ro.size - 1, int(d)),
                 with_counters)


def overlap_matrix(i, j, labels_i, labels_j, n_repertoires: int, symmetric: bool):
    """NEXT-4: M x M matrix, entry (p, q) = number of neighbour pairs between repertoires p and q.
    Plain loop over the pairs.  symmetric (self-search, reading A-18): a pair with labels p != q counts in
    [p][q] and [q][p]; a within-repertoire pair counts once on the diagonal."""
    m = np.zeros((n_repertoires, n_repertoires), dtype=np.int64)
    for a, b in zip(np.asarray(i).tolist(), np.asarray(j).tolist()):
        p, q = int(labels_i[a]), int(labels_j[b])
        m[p, q] += 1
        if symmetric and p != q:
            m[q, p] += 1
    return m


def max_threads() -> int:
    return int(lib().oracle_max_threads())
