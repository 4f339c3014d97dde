"""Seeded synthetic workloads — the ONLY module shared by the oracle and the CUDA path.

It draws inputs; it contains none of the method's arithmetic (no scoring, no
top-k, no index layout).  The C generator in ``gen.c`` is compiled with gcc into
``libworkload.so`` next to this file (by ``__graft_entry__.build()`` or on first
use) and called through ctypes.

The synthetic rows stand in for MS MARCO passages / dev queries encoded with
SPLADE (§6.1), which are not available offline; the
distribution parameters are the ones ``BASELINE.json:configs`` fixes.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen.c")
_SO = os.path.join(_HERE, "libworkload.so")
_lib_handle = None


def build(force: bool = False) -> str:
    """Compile gen.c -> libworkload.so (gcc, OpenMP)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + f".tmp{os.getpid()}"
        subprocess.run(
            ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-Wall", "-o", tmp, _SRC, "-lm"],
            check=True,
        )
        os.replace(tmp, _SO)
    return _SO


class _Params(ctypes.Structure):
    _fields_ = [
        ("seed", ctypes.c_uint64),
        ("stream", ctypes.c_uint64),
        ("vocab", ctypes.c_int32),
        ("zipf_s", ctypes.c_double),
        ("nnz_law", ctypes.c_int32),
        ("nnz_mu", ctypes.c_double),
        ("nnz_sigma", ctypes.c_double),
        ("nnz_lo", ctypes.c_int32),
        ("nnz_hi", ctypes.c_int32),
    ]


def _lib():
    global _lib_handle
    if _lib_handle is None:
        build()
        L = ctypes.CDLL(_SO)
        L.wl_indptr.argtypes = [ctypes.POINTER(_Params), ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int]
        L.wl_indptr.restype = ctypes.c_int
        L.wl_fill.argtypes = [ctypes.POINTER(_Params), ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p,
                              ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]
        L.wl_fill.restype = ctypes.c_int
        L.wl_quantize_u8.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int]
        L.wl_quantize_u8.restype = None
        L.wl_checksum.argtypes = [ctypes.c_void_p, ctypes.c_int64]
        L.wl_checksum.restype = ctypes.c_uint64
        L.wl_max_threads.restype = ctypes.c_int
        _lib_handle = L
    return _lib_handle


STREAM_DOCS = 0
STREAM_QUERIES = 1
NNZ_NORMAL = 0
NNZ_UNIFORM = 1


@dataclass
class Csr:
    """A batch of sparse rows: row r holds terms[indptr[r]:indptr[r+1]] with the matching weights."""
    indptr: np.ndarray   # int64 [rows+1]
    terms: np.ndarray    # int32 [nnz], unique within a row, draw order (not sorted)
    weights: np.ndarray  # float32 [nnz] or uint8 [nnz]

    @property
    def rows(self) -> int:
        return int(self.indptr.shape[0] - 1)

    @property
    def nnz(self) -> int:
        return int(self.indptr[-1])

    def row(self, r: int):
        a, b = int(self.indptr[r]), int(self.indptr[r + 1])
        return self.terms[a:b], self.weights[a:b]

    def slice_rows(self, r0: int, r1: int) -> "Csr":
        a, b = int(self.indptr[r0]), int(self.indptr[r1])
        return Csr((self.indptr[r0:r1 + 1] - self.indptr[r0]).copy(), self.terms[a:b].copy(), self.weights[a:b].copy())

    def to_u8(self) -> "Csr":
        return Csr(self.indptr, self.terms, quantize_u8(self.weights))


def make_rows(rows: int, *, seed: int, stream: int, vocab: int = 30522, zipf_s: float = 1.1,
              nnz_law: int = NNZ_NORMAL, mu: float = 120.0, sigma: float = 40.0, lo: int = 20, hi: int = 400,
              row0: int = 0, nthreads: int = 0, alloc=None) -> Csr:
    """Generate rows [row0, row0+rows).  ``alloc(shape, dtype)`` may supply (e.g. pinned) output buffers."""
    L = _lib()
    p = _Params(seed, stream, vocab, zipf_s, nnz_law, mu, sigma, lo, hi)
    alloc = alloc or (lambda shape, dtype: np.empty(shape, dtype=dtype))
    indptr = alloc((rows + 1,), np.int64)
    rc = L.wl_indptr(ctypes.byref(p), row0, rows, indptr.ctypes.data, nthreads)
    if rc:
        raise RuntimeError(f"wl_indptr failed: {rc}")
    nnz = int(indptr[rows])
    terms = alloc((nnz,), np.int32)
    weights = alloc((nnz,), np.float32)
    rc = L.wl_fill(ctypes.byref(p), row0, rows, indptr.ctypes.data, terms.ctypes.data, weights.ctypes.data, nthreads)
    if rc:
        raise RuntimeError(f"wl_fill failed: {rc}")
    return Csr(indptr, terms, weights)


def quantize_u8(w: np.ndarray, nthreads: int = 0) -> np.ndarray:
    """BASELINE.json config 4: uint8 = clamp(round(100*w), 1, 255) (round-half-even), done once, here."""
    w = np.ascontiguousarray(w, dtype=np.float32)
    out = np.empty(w.shape, dtype=np.uint8)
    _lib().wl_quantize_u8(w.ctypes.data, w.size, out.ctypes.data, nthreads)
    return out


def checksum(a: np.ndarray) -> int:
    a = np.ascontiguousarray(a)
    return int(_lib().wl_checksum(a.ctypes.data, a.nbytes))


def max_threads() -> int:
    return int(_lib().wl_max_threads())


# --------------------------------------------------------------------------------------
# BASELINE.json configs.  Docs of every config with the same Zipf exponent are a prefix of
# the 8.8M-doc collection (counter-based RNG), so "mid" == first 1M docs of "paper".
# --------------------------------------------------------------------------------------
VOCAB = 30522
_DOC = dict(nnz_law=NNZ_NORMAL, mu=120.0, sigma=40.0, lo=20, hi=400)
_QRY = dict(nnz_law=NNZ_NORMAL, mu=25.0, sigma=8.0, lo=5, hi=64)
_QRY_SKEW = dict(nnz_law=NNZ_UNIFORM, mu=0.0, sigma=0.0, lo=5, hi=256)   # DESIGN.md reading R7: nnz ~ U{5..256}

CONFIGS = {
    #  name        N          B    k     zipf  wtype  query law
    "tiny":       dict(N=10_000,    B=16,  k=10,   s=1.1, wtype="f32", qlaw=_QRY),       # configs[0]
    "mid":        dict(N=1_000_000, B=64,  k=1000, s=1.1, wtype="f32", qlaw=_QRY),       # configs[1]
    "paper":      dict(N=8_800_000, B=500, k=1000, s=1.1, wtype="f32", qlaw=_QRY),       # configs[2]
    "paper_u8":   dict(N=8_800_000, B=500, k=10,   s=1.1, wtype="u8",  qlaw=_QRY),       # configs[3]
    "skew_b1":    dict(N=8_800_000, B=1,   k=10,   s=1.3, wtype="f32", qlaw=_QRY_SKEW),  # configs[4]
    "skew_b32":   dict(N=8_800_000, B=32,  k=10,   s=1.3, wtype="f32", qlaw=_QRY_SKEW),  # configs[4]
}


@dataclass
class Workload:
    name: str
    vocab: int
    k: int
    wtype: str          # "f32" | "u8"
    docs: Csr
    queries: Csr


def make_docs(name: str, *, n_docs: Optional[int] = None, seed: int = 0, nthreads: int = 0, alloc=None,
              row0: int = 0) -> Csr:
    c = CONFIGS[name]
    n = c["N"] if n_docs is None else int(n_docs)
    d = make_rows(n, seed=seed, stream=STREAM_DOCS, vocab=VOCAB, zipf_s=c["s"], row0=row0,
                  nthreads=nthreads, alloc=alloc, **_DOC)
    return d.to_u8() if c["wtype"] == "u8" else d


def make_queries(name: str, *, n_queries: Optional[int] = None, seed: int = 0, row0: int = 0,
                 nthreads: int = 0) -> Csr:
    c = CONFIGS[name]
    b = c["B"] if n_queries is None else int(n_queries)
    q = make_rows(b, seed=seed, stream=STREAM_QUERIES, vocab=VOCAB, zipf_s=c["s"], row0=row0,
                  nthreads=nthreads, **c["qlaw"])
    return q.to_u8() if c["wtype"] == "u8" else q


def make_workload(name: str, *, n_docs: Optional[int] = None, n_queries: Optional[int] = None,
                  seed: int = 0, nthreads: int = 0) -> Workload:
    """One of BASELINE.json's configs (optionally with fewer docs/queries: a prefix of the same collection)."""
    c = CONFIGS[name]
    return Workload(name, VOCAB, c["k"], c["wtype"],
                    make_docs(name, n_docs=n_docs, seed=seed, nthreads=nthreads),
                    make_queries(name, n_queries=n_queries, seed=seed, nthreads=nthreads))
