"""Thin ctypes binding over the C ABI in include/gpusparse.h — argument marshalling only.

Every step of the hot path runs inside ``libgpusparse.so`` (hand-written CUDA for sm_100a).  PyTorch is
used for device memory and streams.  There is NO fallback: if the library is missing, cannot be loaded,
or the device is not sm_100, the calls raise.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgpusparse.so")

GS_W_F32, GS_W_U8 = 0, 1
GS_ALGO_AUTO, GS_ALGO_TERM_PARALLEL, GS_ALGO_DOC_PARALLEL = 0, 1, 2
GS_FLAG_VALIDATE_QUERIES, GS_FLAG_FORCE_DENSE_TOPK, GS_FLAG_NO_HEAD_STRIPS, GS_FLAG_TENSOR_CORE_HEAD = 1, 2, 4, 8
GS_MAX_K = 4096
ALGOS = {"auto": GS_ALGO_AUTO, "term": GS_ALGO_TERM_PARALLEL, "doc": GS_ALGO_DOC_PARALLEL}

EXPORTS = [
    "gs_index_build", "gs_index_info", "gs_index_free", "gs_index_copy_meta", "gs_index_copy_list",
    "gs_index_copy_head_terms",
    "gs_search_workspace_bytes", "gs_search", "gs_search_finish", "gs_search_host", "gs_search_stats", "gs_score_dense",
    "gs_topk_workspace_bytes", "gs_topk_dense", "gs_topk_dense_static", "gs_merge_topk_workspace_bytes", "gs_merge_topk", "gs_strerror", "gs_version", "gs_abi_version",
    "gs_last_cuda_error", "gs_last_launch_count", "gs_profile_enable", "gs_profile_read", "gs_kclass_name", "gs_dispatch_model",
]
GS_PROF_CLASSES = 8


class GsError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"gpusparse error {code}: {msg}")
        self.code = code


class gs_csr_t(ctypes.Structure):
    _fields_ = [("rows", ctypes.c_int64), ("nnz", ctypes.c_int64), ("indptr", ctypes.c_void_p),
                ("term_ids", ctypes.c_void_p), ("weights", ctypes.c_void_p), ("wtype", ctypes.c_int32)]


class gs_build_opts_t(ctypes.Structure):
    _fields_ = [("tile_docs", ctypes.c_int32), ("head_max", ctypes.c_int32), ("head_density", ctypes.c_float),
                ("validate", ctypes.c_int32), ("pack_postings", ctypes.c_int32)]


class gs_info_t(ctypes.Structure):
    _fields_ = [("num_docs", ctypes.c_int64), ("vocab_size", ctypes.c_int32), ("wtype", ctypes.c_int32),
                ("nnz", ctypes.c_int64), ("padded_nnz", ctypes.c_int64), ("nonempty_terms", ctypes.c_int64),
                ("tile_docs", ctypes.c_int32), ("num_tiles", ctypes.c_int32), ("head_terms", ctypes.c_int32),
                ("bytes_inverted", ctypes.c_int64), ("bytes_inverted_meta", ctypes.c_int64),
                ("bytes_forward", ctypes.c_int64), ("bytes_head", ctypes.c_int64), ("bytes_total", ctypes.c_int64),
                ("forward_tail_nnz", ctypes.c_int64), ("head_terms_term_parallel", ctypes.c_int32), ("packed_layout", ctypes.c_int32),
                ("forward_padded_nnz", ctypes.c_int64)]


class gs_alloc_t(ctypes.Structure):
    _fields_ = [("alloc", ctypes.c_void_p), ("free", ctypes.c_void_p), ("user", ctypes.c_void_p)]


class gs_search_opts_t(ctypes.Structure):
    _fields_ = [("algo", ctypes.c_int32), ("flags", ctypes.c_uint32), ("query_group", ctypes.c_int32),
                ("doc_query_tile", ctypes.c_int32), ("sample_shift", ctypes.c_int32)]


class gs_stats_t(ctypes.Structure):
    _fields_ = [("candidates", ctypes.c_int64), ("overflow_queries", ctypes.c_int32), ("launches", ctypes.c_int32),
                ("algo_used", ctypes.c_int32), ("sample_tiles", ctypes.c_int32), ("doc_query_tile", ctypes.c_int32),
                ("doc_passes", ctypes.c_int32), ("query_group", ctypes.c_int32)]


class gs_profile_t(ctypes.Structure):
    _fields_ = [("launches", ctypes.c_int32 * GS_PROF_CLASSES), ("ms", ctypes.c_float * GS_PROF_CLASSES)]


_lib_handle = None


def lib():
    """Load libgpusparse.so (fails loudly when it has not been built)."""
    global _lib_handle
    if _lib_handle is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(
                f"{LIB_PATH} is missing: build it with `python -m paper_2606_26441_b200.build` "
                "(there is no CPU or PyTorch fallback for the hot path)")
        L = ctypes.CDLL(LIB_PATH)
        vp, i32, i64, sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_size_t
        P = ctypes.POINTER
        L.gs_index_build.argtypes = [P(gs_csr_t), i32, P(gs_build_opts_t), vp, vp, P(vp)]
        L.gs_index_info.argtypes = [vp, P(gs_info_t)]
        L.gs_index_free.argtypes = [vp]
        L.gs_index_free.restype = None
        L.gs_index_copy_meta.argtypes = [vp, vp, vp]
        L.gs_index_copy_list.argtypes = [vp, i32, i64, vp, vp, P(i64)]
        L.gs_index_copy_head_terms.argtypes = [vp, i32, vp, P(i32)]
        L.gs_search_workspace_bytes.argtypes = [vp, i64, i64, i32, P(gs_search_opts_t), P(sz)]
        L.gs_search.argtypes = [vp, P(gs_csr_t), i32, P(gs_search_opts_t), vp, vp, vp, sz, vp]
        L.gs_search_finish.argtypes = [vp, P(gs_csr_t), i32, P(gs_search_opts_t), vp, vp, vp, sz, vp, P(i32)]
        L.gs_search_host.argtypes = [vp, P(gs_csr_t), i32, P(gs_search_opts_t), vp, vp, vp]
        L.gs_search_stats.argtypes = [vp, vp, P(gs_stats_t)]
        L.gs_score_dense.argtypes = [vp, P(gs_csr_t), P(gs_search_opts_t), vp, i64, vp, sz, vp]
        L.gs_topk_workspace_bytes.argtypes = [i64, i64, i32, P(sz)]
        L.gs_topk_dense.argtypes = [vp, i32, i64, i64, i64, i32, vp, vp, vp, sz, vp]
        L.gs_topk_dense_static.argtypes = [vp, i32, i64, i64, i64, i32, vp, vp, vp]
        L.gs_merge_topk_workspace_bytes.argtypes = [i32, i64, i32, i32, P(sz)]
        L.gs_merge_topk.argtypes = [i32, i32, i64, i32, i32, vp, vp, P(i64), vp, vp, vp, sz, vp]
        L.gs_strerror.argtypes = [ctypes.c_int]
        L.gs_strerror.restype = ctypes.c_char_p
        L.gs_version.restype = ctypes.c_char_p
        L.gs_profile_enable.argtypes = [i32]
        L.gs_profile_enable.restype = None
        L.gs_profile_read.argtypes = [P(gs_profile_t)]
        L.gs_kclass_name.argtypes = [i32]
        L.gs_kclass_name.restype = ctypes.c_char_p
        for name in EXPORTS:
            getattr(L, name)            # every symbol the header declares must be exported
        _lib_handle = L
    return _lib_handle


def _check(code: int):
    if code != 0:
        L = lib()
        msg = L.gs_strerror(code).decode()
        if code == 6:
            msg += f" (cudaError {L.gs_last_cuda_error()})"
        raise GsError(code, msg)


def dispatch_model(num_docs: int, tile_docs: int, stream_bytes: int, num_queries: int, query_nnz: int):
    """Cost model behind algo="auto" (gpusparse.h: gs_dispatch_model; host arithmetic, no GPU needed).
    Returns (algo name, estimated term-parallel ms, estimated document-parallel ms)."""
    t, d = ctypes.c_double(0.0), ctypes.c_double(0.0)
    L = lib()
    L.gs_dispatch_model.restype = ctypes.c_int32
    L.gs_dispatch_model.argtypes = [ctypes.c_int64, ctypes.c_int32, ctypes.c_int64, ctypes.c_int64, ctypes.c_int64,
                                    ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    a = L.gs_dispatch_model(num_docs, tile_docs, stream_bytes, num_queries, query_nnz, ctypes.byref(t), ctypes.byref(d))
    return ("doc" if a == GS_ALGO_DOC_PARALLEL else "term"), t.value, d.value


def version() -> str:
    return lib().gs_version().decode()


def last_launch_count() -> int:
    return int(lib().gs_last_launch_count())


def profile_enable(on: bool) -> None:
    """gs_profile_enable: bracket every kernel launch of this thread's following calls with CUDA events."""
    lib().gs_profile_enable(1 if on else 0)


def profile_read() -> dict:
    """gs_profile_read -> {kernel class: {"launches": n, "ms": summed device time}} (clears the record)."""
    L = lib()
    pr = gs_profile_t()
    _check(L.gs_profile_read(ctypes.byref(pr)))
    out = {}
    for c in range(GS_PROF_CLASSES):
        name = L.gs_kclass_name(c).decode()
        if name and pr.launches[c]:
            out[name] = {"launches": int(pr.launches[c]), "ms": float(pr.ms[c])}
    return out


def _torch():
    import torch
    return torch


def _stream_ptr(stream=None) -> int:
    torch = _torch()
    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


def _wtype_of(t) -> int:
    torch = _torch()
    if t.dtype == torch.float32:
        return GS_W_F32
    if t.dtype == torch.uint8:
        return GS_W_U8
    raise TypeError("weights must be float32 or uint8")


def _dev_csr(indptr, terms, weights) -> gs_csr_t:
    torch = _torch()
    assert indptr.dtype == torch.int64 and terms.dtype == torch.int32
    assert indptr.is_cuda and terms.is_cuda and weights.is_cuda
    assert indptr.is_contiguous() and terms.is_contiguous() and weights.is_contiguous()
    return gs_csr_t(indptr.numel() - 1, terms.numel(), indptr.data_ptr(), terms.data_ptr(), weights.data_ptr(),
                    _wtype_of(weights))


def _opts(algo="auto", flags=0, query_group=0, doc_query_tile=0, sample_shift=0) -> gs_search_opts_t:
    a = ALGOS[algo] if isinstance(algo, str) else int(algo)
    return gs_search_opts_t(a, flags, query_group, doc_query_tile, sample_shift)


class Index:
    """gs_index_build / gs_index_free: a GPU-resident inverted + forward index (§3)."""

    def __init__(self, indptr, terms, weights, vocab_size: int, *, tile_docs: int = 0, head_max: int = 0,
                 head_density: float = 0.0, validate: bool = True, pack_postings: bool = True, stream=None, allocator=None):
        """``allocator``: optional pair of ctypes callbacks (alloc(bytes, stream, user) -> ptr, free(ptr, stream, user))
        passed as gs_alloc_t; everything the handle owns then comes from it (default: cudaMalloc).
        ``pack_postings`` (integer-impact mode): one 32-bit word per posting where the sizes allow it (gs_build_opts_t)."""
        L = lib()
        csr = _dev_csr(indptr, terms, weights)
        bo = gs_build_opts_t(tile_docs, head_max, head_density, 1 if validate else 0, 0 if pack_postings else -1)
        h = ctypes.c_void_p()
        self._h = None
        self._alloc = None
        if allocator is not None:
            self._cb = allocator                       # keep the callbacks alive as long as the handle
            self._alloc = gs_alloc_t(ctypes.cast(allocator[0], ctypes.c_void_p), ctypes.cast(allocator[1], ctypes.c_void_p), None)
        _check(L.gs_index_build(ctypes.byref(csr), vocab_size, ctypes.byref(bo),
                                ctypes.byref(self._alloc) if self._alloc is not None else None, _stream_ptr(stream),
                                ctypes.byref(h)))
        self._h = h
        self.wtype = csr.wtype
        self.vocab_size = int(vocab_size)
        self.device = indptr.device
        self._ws = None
        inf = self.info()
        self.num_docs = inf["num_docs"]

    @classmethod
    def from_numpy(cls, csr, vocab_size: int, device="cuda:0", **kw) -> "Index":
        """csr: anything with .indptr/.terms/.weights numpy arrays (e.g. workload.Csr)."""
        torch = _torch()
        d = torch.device(device)
        return cls(torch.from_numpy(np.ascontiguousarray(csr.indptr)).to(d),
                   torch.from_numpy(np.ascontiguousarray(csr.terms)).to(d),
                   torch.from_numpy(np.ascontiguousarray(csr.weights)).to(d), vocab_size, **kw)

    def close(self):
        h, self._h = self._h, None
        if h:
            lib().gs_index_free(h)
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def info(self) -> dict:
        inf = gs_info_t()
        _check(lib().gs_index_info(self._h, ctypes.byref(inf)))
        return {k: getattr(inf, k) for k, _ in gs_info_t._fields_}

    def meta(self) -> Tuple[np.ndarray, np.ndarray]:
        """(padded list offsets int64 [V+1], true list lengths int32 [V]) copied to the host."""
        off = np.empty(self.vocab_size + 1, np.int64)
        ln = np.empty(self.vocab_size, np.int32)
        _check(lib().gs_index_copy_meta(self._h, off.ctypes.data, ln.ctypes.data))
        return off, ln

    def head_terms(self) -> np.ndarray:
        """Term ids whose lists are also kept as dense strips, densest first."""
        n = ctypes.c_int32()
        out = np.empty(64, np.int32)
        _check(lib().gs_index_copy_head_terms(self._h, 64, out.ctypes.data, ctypes.byref(n)))
        return out[:n.value].copy()

    def posting_list(self, term: int) -> Tuple[np.ndarray, np.ndarray]:
        """The padded posting list of ``term`` (doc ids incl. -1 sentinels, weights incl. 0 padding)."""
        n = ctypes.c_int64()
        _check(lib().gs_index_copy_list(self._h, term, 0, None, None, ctypes.byref(n)))
        ids = np.empty(n.value, np.int32)
        w = np.empty(n.value, np.float32 if self.wtype == GS_W_F32 else np.uint8)
        _check(lib().gs_index_copy_list(self._h, term, n.value, ids.ctypes.data, w.ctypes.data, ctypes.byref(n)))
        return ids, w

    # ------------------------------------------------------------------ search
    def workspace_bytes(self, num_queries: int, query_nnz: int, k: int, **opt) -> int:
        o = _opts(**opt)
        out = ctypes.c_size_t()
        _check(lib().gs_search_workspace_bytes(self._h, num_queries, query_nnz, k, ctypes.byref(o), ctypes.byref(out)))
        return int(out.value)

    def _workspace(self, nbytes: int):
        torch = _torch()
        if self._ws is None or self._ws.numel() < nbytes:
            self._ws = None
            self._ws = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        return self._ws

    def search(self, q_indptr, q_terms, q_weights, k: int, *, out_ids=None, out_scores=None, workspace=None,
               stream=None, finish: bool = True, **opt):
        """gs_search on DEVICE tensors -> (ids int32 [B,k], scores float32|int32 [B,k]) device tensors.

        ``finish=True`` (default) follows it with gs_search_finish (one stream synchronisation; re-runs the queries
        whose candidate list overflowed, so the result is always exact).  ``finish=False`` only enqueues the search
        (asynchronous, capturable into a CUDA graph); call :meth:`finish` or check ``stats()["overflow_queries"]``."""
        torch = _torch()
        csr = _dev_csr(q_indptr, q_terms, q_weights)
        o = _opts(**opt)
        B = csr.rows
        if workspace is None:
            workspace = self._workspace(self.workspace_bytes(B, csr.nnz, k, **opt))
        sdt = torch.float32 if self.wtype == GS_W_F32 else torch.int32
        if out_ids is None:
            out_ids = torch.empty((B, k), dtype=torch.int32, device=self.device)
        if out_scores is None:
            out_scores = torch.empty((B, k), dtype=sdt, device=self.device)
        _check(lib().gs_search(self._h, ctypes.byref(csr), k, ctypes.byref(o), out_ids.data_ptr(), out_scores.data_ptr(),
                               workspace.data_ptr(), workspace.numel(), _stream_ptr(stream)))
        self._last_ws = workspace
        self.last_resolved = 0
        if finish:
            r = ctypes.c_int32()
            _check(lib().gs_search_finish(self._h, ctypes.byref(csr), k, ctypes.byref(o), out_ids.data_ptr(),
                                          out_scores.data_ptr(), workspace.data_ptr(), workspace.numel(),
                                          _stream_ptr(stream), ctypes.byref(r)))
            self.last_resolved = int(r.value)
        return out_ids, out_scores

    def finish(self, q_indptr, q_terms, q_weights, k: int, out_ids, out_scores, workspace, stream=None, **opt) -> int:
        """gs_search_finish for a search enqueued with ``finish=False``; returns the number of queries re-run."""
        csr = _dev_csr(q_indptr, q_terms, q_weights)
        o = _opts(**opt)
        r = ctypes.c_int32()
        _check(lib().gs_search_finish(self._h, ctypes.byref(csr), k, ctypes.byref(o), out_ids.data_ptr(),
                                      out_scores.data_ptr(), workspace.data_ptr(), workspace.numel(),
                                      _stream_ptr(stream), ctypes.byref(r)))
        return int(r.value)

    def search_host(self, q_indptr: np.ndarray, q_terms: np.ndarray, q_weights: np.ndarray, k: int, *,
                    out_ids: Optional[np.ndarray] = None, out_scores: Optional[np.ndarray] = None, stream=None, **opt):
        """gs_search_host on HOST (numpy) buffers; copies are inside the call."""
        B = int(q_indptr.shape[0] - 1)
        wt = GS_W_F32 if q_weights.dtype == np.float32 else GS_W_U8
        csr = gs_csr_t(B, int(q_terms.shape[0]), q_indptr.ctypes.data, q_terms.ctypes.data, q_weights.ctypes.data, wt)
        o = _opts(**opt)
        if out_ids is None:
            out_ids = np.empty((B, k), np.int32)
        if out_scores is None:
            out_scores = np.empty((B, k), np.float32 if self.wtype == GS_W_F32 else np.int32)
        _check(lib().gs_search_host(self._h, ctypes.byref(csr), k, ctypes.byref(o), out_ids.ctypes.data,
                                    out_scores.ctypes.data, _stream_ptr(stream)))
        return out_ids, out_scores

    def stats(self, workspace=None, stream=None) -> dict:
        ws = workspace if workspace is not None else getattr(self, "_last_ws", None)
        st = gs_stats_t()
        _check(lib().gs_search_stats(ws.data_ptr(), _stream_ptr(stream), ctypes.byref(st)))
        return {k: getattr(st, k) for k, _ in gs_stats_t._fields_}

    def score_dense(self, q_indptr, q_terms, q_weights, *, algo="term", stream=None, **opt):
        """gs_score_dense -> [B, ld] device tensor of all scores (columns >= N are undefined)."""
        torch = _torch()
        csr = _dev_csr(q_indptr, q_terms, q_weights)
        o = _opts(algo=algo, **opt)
        inf = self.info()
        ld = inf["num_tiles"] * inf["tile_docs"]
        sdt = torch.float32 if self.wtype == GS_W_F32 else torch.int32
        out = torch.zeros((csr.rows, max(ld, 1)), dtype=sdt, device=self.device)
        ws = self._workspace(self.workspace_bytes(csr.rows, csr.nnz, 1, algo=algo, **opt))
        _check(lib().gs_score_dense(self._h, ctypes.byref(csr), ctypes.byref(o), out.data_ptr(), ld, ws.data_ptr(),
                                    ws.numel(), _stream_ptr(stream)))
        return out


def topk_dense(scores, k: int, n: Optional[int] = None, stream=None):
    """gs_topk_dense: rows of a dense device score matrix -> (ids, scores), ties by lower id."""
    torch = _torch()
    assert scores.is_cuda and scores.dim() == 2 and scores.is_contiguous()
    rows, ld = scores.shape
    n = ld if n is None else n
    wt = GS_W_F32 if scores.dtype == torch.float32 else GS_W_U8
    if wt == GS_W_U8:
        assert scores.dtype == torch.int32
    need = ctypes.c_size_t()
    _check(lib().gs_topk_workspace_bytes(rows, n, k, ctypes.byref(need)))
    ws = torch.empty(max(need.value, 256), dtype=torch.uint8, device=scores.device)
    ids = torch.empty((rows, k), dtype=torch.int32, device=scores.device)
    sc = torch.empty((rows, k), dtype=scores.dtype, device=scores.device)
    _check(lib().gs_topk_dense(scores.data_ptr(), wt, rows, n, ld, k, ids.data_ptr(), sc.data_ptr(), ws.data_ptr(),
                               ws.numel(), _stream_ptr(stream)))
    return ids, sc


GS_TOPK_STATIC_SCRATCH_BYTES = 2624000


def topk_dense_static(scores, k: int, out_ids, out_scores, n: Optional[int] = None, stream=None):
    """gs_topk_dense_static: as topk_dense, but the library allocates nothing (scratch = a static device array of
    GS_TOPK_STATIC_SCRATCH_BYTES shared by all calls) and neither does this wrapper: the caller passes the outputs
    ``out_ids`` [rows, k] int32 and ``out_scores`` [rows, k] (dtype of ``scores``).  Raises GsError(2) beyond the maximum."""
    torch = _torch()
    assert scores.is_cuda and scores.dim() == 2 and scores.is_contiguous()
    rows, ld = scores.shape
    n = ld if n is None else n
    wt = GS_W_F32 if scores.dtype == torch.float32 else GS_W_U8
    if wt == GS_W_U8:
        assert scores.dtype == torch.int32
    assert out_ids.is_cuda and out_ids.dtype == torch.int32 and out_ids.shape == (rows, k) and out_ids.is_contiguous()
    assert out_scores.is_cuda and out_scores.dtype == scores.dtype and out_scores.shape == (rows, k) and out_scores.is_contiguous()
    _check(lib().gs_topk_dense_static(scores.data_ptr(), wt, rows, n, ld, k, out_ids.data_ptr(), out_scores.data_ptr(),
                                      _stream_ptr(stream)))
    return out_ids, out_scores


def merge_topk(ids, scores, k_out: int, doc_bases=None, workspace=None, stream=None):
    """gs_merge_topk: partial top-k lists ``ids``/``scores`` [n_lists, B, k_in] (device, shard-local doc ids, -1 padding) ->
    the k_out best of the union per query (global ids = local id + doc_bases[list]), score desc, ties by lower id."""
    torch = _torch()
    assert ids.is_cuda and scores.is_cuda and ids.dim() == 3 and ids.shape == scores.shape
    assert ids.dtype == torch.int32 and ids.is_contiguous() and scores.is_contiguous()
    n_lists, B, k_in = ids.shape
    wt = GS_W_F32 if scores.dtype == torch.float32 else GS_W_U8
    if wt == GS_W_U8:
        assert scores.dtype == torch.int32
    need = ctypes.c_size_t()
    _check(lib().gs_merge_topk_workspace_bytes(n_lists, B, k_in, k_out, ctypes.byref(need)))
    if workspace is None:
        workspace = torch.empty(max(need.value, 256), dtype=torch.uint8, device=ids.device)
    assert workspace.numel() >= need.value
    bases = None
    if doc_bases is not None:
        assert len(doc_bases) == n_lists
        bases = (ctypes.c_int64 * n_lists)(*[int(x) for x in doc_bases])
    out_ids = torch.empty((B, k_out), dtype=torch.int32, device=ids.device)
    out_sc = torch.empty((B, k_out), dtype=scores.dtype, device=ids.device)
    _check(lib().gs_merge_topk(wt, n_lists, B, k_in, k_out, ids.data_ptr(), scores.data_ptr(), bases, out_ids.data_ptr(),
                               out_sc.data_ptr(), workspace.data_ptr(), workspace.numel(), _stream_ptr(stream)))
    return out_ids, out_sc
