"""CPU oracle for the GPUSparse hot path — TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It is independent of ``paper_2606_26441_b200`` (it imports nothing
from it, and the CUDA path imports nothing from here); both sides merely receive the same numpy
arrays from the seeded workload generator.

The arithmetic lives in ``oracle.c`` (plain C, see its header for the definition it follows:
PAPER.md L106-111 Eq. 4 + top-k over all N docs, ties by lower doc id).  This file is a ctypes
wrapper only.  parity pins: see ``oracle.c`` header and DESIGN.md §3 — every exported function is
pinned by ``tests/test_oracle_pins.py`` (none is "parity unpinned").
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_SO = os.path.join(_HERE, "liboracle.so")
_lib_handle = None

W_F32, W_U8 = 0, 1
_ERR = {1: "invalid argument", 2: "out of range", 3: "duplicate term in a row", 5: "out of memory",
        8: "integer score overflows int32"}


class OracleError(RuntimeError):
    def __init__(self, code: int):
        super().__init__(f"oracle error {code}: {_ERR.get(code, '?')}")
        self.code = code


def build(force: bool = False) -> str:
    """gcc oracle.c -> liboracle.so (building the checker is not using it)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + f".tmp{os.getpid()}"
        subprocess.run(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-Wall", "-o", tmp, _SRC], check=True)
        os.replace(tmp, _SO)
    return _SO


def _lib():
    global _lib_handle
    if _lib_handle is None:
        build()
        L = ctypes.CDLL(_SO)
        vp, i64, i32, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_int
        L.or_rows_create.argtypes = [i64, vp, vp, vp, i32, i32, ci, ctypes.POINTER(vp)]
        L.or_rows_create.restype = ci
        L.or_rows_free.argtypes = [vp]
        L.or_rows_free.restype = None
        L.or_score_pairs.argtypes = [vp, vp, i64, vp, vp, vp, vp]
        L.or_score_pairs.restype = ci
        L.or_search.argtypes = [vp, vp, i64, i64, i32, vp, vp, vp, vp, vp, ci]
        L.or_search.restype = ci
        L.or_max_threads.restype = ci
        _lib_handle = L
    return _lib_handle


def max_threads() -> int:
    return int(_lib().or_max_threads())


def _ptr(a):
    return None if a is None else a.ctypes.data


class Rows:
    """Canonical (term-sorted, validated) copy of a CSR batch: step 1 of the definition."""

    def __init__(self, indptr, terms, weights, vocab: int, nthreads: int = 0):
        self.indptr = np.ascontiguousarray(indptr, dtype=np.int64)
        self.terms = np.ascontiguousarray(terms, dtype=np.int32)
        w = np.ascontiguousarray(weights)
        if w.dtype == np.uint8:
            self.wtype = W_U8
        elif w.dtype == np.float32:
            self.wtype = W_F32
        else:
            raise TypeError("weights must be float32 or uint8")
        self.weights = w
        self.rows = int(self.indptr.shape[0] - 1)
        self.vocab = int(vocab)
        h = ctypes.c_void_p()
        rc = _lib().or_rows_create(self.rows, _ptr(self.indptr), _ptr(self.terms), _ptr(self.weights),
                                   self.wtype, self.vocab, nthreads, ctypes.byref(h))
        if rc:
            raise OracleError(rc)
        self._h = h

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h and _lib_handle is not None:
            _lib_handle.or_rows_free(h)


def as_rows(csr, vocab: int, nthreads: int = 0) -> Rows:
    """Accept anything with .indptr/.terms/.weights (e.g. the workload generator's Csr) or a Rows."""
    return csr if isinstance(csr, Rows) else Rows(csr.indptr, csr.terms, csr.weights, vocab, nthreads)


def score_pairs(queries: Rows, docs: Rows, qb, dd) -> np.ndarray:
    """Eq. 4 for sampled (query, doc) pairs.  float64 in fp32 mode, int64 in integer mode."""
    qb = np.ascontiguousarray(qb, dtype=np.int64)
    dd = np.ascontiguousarray(dd, dtype=np.int64)
    n = int(qb.shape[0])
    f32 = queries.wtype == W_F32
    out = np.empty(n, dtype=np.float64 if f32 else np.int64)
    rc = _lib().or_score_pairs(queries._h, docs._h, n, _ptr(qb), _ptr(dd), _ptr(out) if f32 else None,
                               None if f32 else _ptr(out))
    if rc:
        raise OracleError(rc)
    return out


def search(queries: Rows, docs: Rows, k: int, *, b0: int = 0, b1: int | None = None, all_scores: bool = False,
           nthreads: int = 0):
    """Exhaustive scoring + full sort + first k for queries [b0, b1).

    Returns (ids int32 [B,k], scores [B,k] float64|int32[, all [B,N] float64|int32]).
    """
    b1 = queries.rows if b1 is None else b1
    nb = b1 - b0
    f32 = queries.wtype == W_F32
    ids = np.empty((nb, k), dtype=np.int32)
    sc = np.empty((nb, k), dtype=np.float64 if f32 else np.int32)
    al = np.empty((nb, docs.rows), dtype=np.float64 if f32 else np.int32) if all_scores else None
    rc = _lib().or_search(queries._h, docs._h, b0, b1, k, _ptr(ids),
                          _ptr(sc) if f32 else None, None if f32 else _ptr(sc),
                          _ptr(al) if (f32 and all_scores) else None,
                          _ptr(al) if (not f32 and all_scores) else None, nthreads)
    if rc:
        raise OracleError(rc)
    return (ids, sc, al) if all_scores else (ids, sc)
