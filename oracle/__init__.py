"""ctypes wrapper of the CPU oracle (oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this module; the
product package never does.  Plans are plain Python data (no product types):

    table  = [np.ndarray, ...]                    columns by index (int8 / int32 / int64)
    pred   = (col, "lt|le|gt|ge|eq|ne|range_co|range_cc", lo[, hi])
    expr   = [("col", i) | ("const", v) | ("add",) | ("sub",) | ("mul",), ...]      postfix
    agg    = ("sum|min|max", expr_index) | ("count",)
    build  = dict(table=, preds=[], probes=[(build_index, key_col)], key=col, payload=[cols])
    query  = dict(builds=[], table=, preds=[], probes=[], exprs=[], keys=[], aggs=[], topk=0, topk_agg=0)
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRCS = [os.path.join(_HERE, "oracle.cpp"), os.path.join(_HERE, "oracle.h")]
_lib = None

_DT = {np.dtype(np.int8): 1, np.dtype(np.int32): 2, np.dtype(np.int64): 3}
_CMP = dict(lt=0, le=1, gt=2, ge=3, eq=4, ne=5, range_co=6, range_cc=7)
_XOP = dict(col=0, const=1, add=2, sub=3, mul=4)
_AGG = dict(sum=0, min=1, max=2, count=3)


class _Col(C.Structure):
    _fields_ = [("data", C.c_void_p), ("dtype", C.c_int32)]


class _Table(C.Structure):
    _fields_ = [("cols", C.POINTER(_Col)), ("ncols", C.c_int32), ("nrows", C.c_int64)]


class _SortKey(C.Structure):
    _fields_ = [("col", C.c_int32), ("descending", C.c_int32)]


class _Pred(C.Structure):
    _fields_ = [("col", C.c_int32), ("op", C.c_int32), ("lo", C.c_int64), ("hi", C.c_int64)]


class _Tok(C.Structure):
    _fields_ = [("op", C.c_int32), ("arg", C.c_int64)]


class _Expr(C.Structure):
    _fields_ = [("toks", C.POINTER(_Tok)), ("ntoks", C.c_int32)]


class _Agg(C.Structure):
    _fields_ = [("op", C.c_int32), ("expr", C.c_int32)]


class _Probe(C.Structure):
    _fields_ = [("build", C.c_int32), ("key_col", C.c_int32)]


class _Build(C.Structure):
    _fields_ = [("in_", _Table), ("preds", C.POINTER(_Pred)), ("npred", C.c_int32), ("probes", C.POINTER(_Probe)),
                ("nprobes", C.c_int32), ("key_col", C.c_int32), ("payload_cols", C.POINTER(C.c_int32)),
                ("npayload", C.c_int32)]


class _Query(C.Structure):
    _fields_ = [("builds", C.POINTER(_Build)), ("nbuilds", C.c_int32), ("in_", _Table), ("preds", C.POINTER(_Pred)),
                ("npred", C.c_int32), ("probes", C.POINTER(_Probe)), ("nprobes", C.c_int32),
                ("exprs", C.POINTER(_Expr)), ("nexpr", C.c_int32), ("key_cols", C.POINTER(C.c_int32)),
                ("nkeys", C.c_int32), ("aggs", C.POINTER(_Agg)), ("naggs", C.c_int32), ("topk", C.c_int32),
                ("topk_agg", C.c_int32)]


def build(force: bool = False) -> str:
    """Compile liboracle.so with g++ (building the checker is not using it)."""
    newest = max(os.path.getmtime(s) for s in _SRCS)
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < newest:
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", _SRCS[0], "-o", _SO])
    return _SO


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.ocl_run_query.restype = C.c_void_p
        L.ocl_run_query.argtypes = [C.POINTER(_Query)]
        L.ocl_filter_project.restype = C.c_void_p
        L.ocl_filter_project.argtypes = [C.POINTER(_Table), C.POINTER(_Pred), C.c_int32, C.POINTER(_Expr), C.c_int32]
        for nm in ("ocl_join_pairs", "ocl_join_pairs_bruteforce"):
            f = getattr(L, nm)
            f.restype = C.c_void_p
            f.argtypes = [C.POINTER(_Table), C.POINTER(_Pred), C.c_int32, C.c_int32,
                          C.POINTER(_Table), C.POINTER(_Pred), C.c_int32, C.c_int32]
        L.ocl_hash_partition.restype = C.c_void_p
        L.ocl_hash_partition.argtypes = [C.POINTER(_Table), C.POINTER(C.c_int32), C.c_int32, C.c_int32]
        L.ocl_order_by.restype = C.c_void_p
        L.ocl_order_by.argtypes = [C.POINTER(_Table), C.POINTER(_SortKey), C.c_int32, C.c_int64]
        L.ocl_result_nrows.restype = C.c_int64
        L.ocl_result_nrows.argtypes = [C.c_void_p]
        L.ocl_result_ncols.restype = C.c_int32
        L.ocl_result_ncols.argtypes = [C.c_void_p]
        L.ocl_result_col.restype = C.POINTER(C.c_int64)
        L.ocl_result_col.argtypes = [C.c_void_p, C.c_int32]
        L.ocl_result_input_rows.restype = C.c_int64
        L.ocl_result_input_rows.argtypes = [C.c_void_p]
        L.ocl_result_overflow.restype = C.c_int32
        L.ocl_result_overflow.argtypes = [C.c_void_p]
        L.ocl_avg.restype = C.c_double
        L.ocl_avg.argtypes = [C.c_int64, C.c_int64]
        L.ocl_result_free.argtypes = [C.c_void_p]
        _lib = L
    return _lib


class _Keep(list):
    """Keeps ctypes/numpy objects alive for the duration of a call."""


def _table(cols, keep) -> _Table:
    arrs = [np.ascontiguousarray(c) for c in cols]
    n = arrs[0].shape[0] if arrs else 0
    for a in arrs:
        if a.dtype not in _DT or a.ndim != 1 or a.shape[0] != n:
            raise ValueError("columns must be 1-D int8/int32/int64 arrays of equal length")
    cc = (_Col * max(1, len(arrs)))()
    for i, a in enumerate(arrs):
        cc[i].data = a.ctypes.data
        cc[i].dtype = _DT[a.dtype]
    keep.extend([arrs, cc])
    return _Table(cc, len(arrs), n)


def _preds(preds, keep):
    pp = (_Pred * max(1, len(preds)))()
    for i, p in enumerate(preds):
        pp[i] = _Pred(int(p[0]), _CMP[p[1]], int(p[2]), int(p[3]) if len(p) > 3 else 0)
    keep.append(pp)
    return pp, len(preds)


def _exprs(exprs, keep):
    ee = (_Expr * max(1, len(exprs)))()
    for i, e in enumerate(exprs):
        tt = (_Tok * max(1, len(e)))()
        for j, t in enumerate(e):
            tt[j] = _Tok(_XOP[t[0]], int(t[1]) if len(t) > 1 else 0)
        keep.append(tt)
        ee[i] = _Expr(tt, len(e))
    keep.append(ee)
    return ee, len(exprs)


def _probes(probes, keep):
    pp = (_Probe * max(1, len(probes)))()
    for i, p in enumerate(probes):
        pp[i] = _Probe(int(p[0]), int(p[1]))
    keep.append(pp)
    return pp, len(probes)


def _ints(vals, keep):
    a = (C.c_int32 * max(1, len(vals)))(*[int(v) for v in vals])
    keep.append(a)
    return a, len(vals)


class Result:
    """cols = list of int64 numpy arrays (keys then aggregates / expressions / pair indices)."""

    def __init__(self, handle):
        L = lib()
        if not handle:
            raise ValueError("oracle rejected the plan (malformed)")
        n = L.ocl_result_nrows(handle)
        self.nrows = int(n)
        self.cols = [np.ctypeslib.as_array(L.ocl_result_col(handle, c), shape=(n,)).copy() if n else
                     np.zeros(0, np.int64) for c in range(L.ocl_result_ncols(handle))]
        self.input_rows = int(L.ocl_result_input_rows(handle))
        self.overflow = bool(L.ocl_result_overflow(handle))
        L.ocl_result_free(handle)


def run_query(q: dict) -> Result:
    keep = _Keep()
    bb = (_Build * max(1, len(q.get("builds", []))))()
    for i, b in enumerate(q.get("builds", [])):
        pr, npr = _preds(b.get("preds", []), keep)
        pb, npb = _probes(b.get("probes", []), keep)
        pay, npay = _ints(b.get("payload", []), keep)
        bb[i] = _Build(_table(b["table"], keep), pr, npr, pb, npb, int(b["key"]), pay, npay)
    pr, npr = _preds(q.get("preds", []), keep)
    pb, npb = _probes(q.get("probes", []), keep)
    ee, ne = _exprs(q.get("exprs", []), keep)
    kk, nk = _ints(q.get("keys", []), keep)
    aggs = q.get("aggs", [])
    aa = (_Agg * max(1, len(aggs)))()
    for i, a in enumerate(aggs):
        aa[i] = _Agg(_AGG[a[0]], int(a[1]) if len(a) > 1 and a[1] is not None else 0)
    cq = _Query(bb, len(q.get("builds", [])), _table(q["table"], keep), pr, npr, pb, npb, ee, ne, kk, nk, aa,
                len(aggs), int(q.get("topk", 0)), int(q.get("topk_agg", 0)))
    return Result(lib().ocl_run_query(C.byref(cq)))


def filter_project(table, preds, exprs) -> Result:
    keep = _Keep()
    t = _table(table, keep)
    pr, npr = _preds(preds, keep)
    ee, ne = _exprs(exprs, keep)
    return Result(lib().ocl_filter_project(C.byref(t), pr, npr, ee, ne))


def join_pairs(build_table, bpreds, bkey, probe_table, ppreds, pkey, bruteforce=False) -> Result:
    keep = _Keep()
    bt, pt = _table(build_table, keep), _table(probe_table, keep)
    bp, nbp = _preds(bpreds, keep)
    pp, npp = _preds(ppreds, keep)
    f = lib().ocl_join_pairs_bruteforce if bruteforce else lib().ocl_join_pairs
    return Result(f(C.byref(bt), bp, nbp, int(bkey), C.byref(pt), pp, npp, int(pkey)))


def order_by(table, keys, limit=0) -> Result:
    """keys = [(column, descending)]; -> Result with cols[0] = input row numbers in order, then the gathered columns."""
    keep = _Keep()
    t = _table(table, keep)
    kk = (_SortKey * max(1, len(keys)))()
    for i, (c, d) in enumerate(keys):
        kk[i] = _SortKey(int(c), 1 if d else 0)
    return Result(lib().ocl_order_by(C.byref(t), kk, len(keys), int(limit)))


def hash_partition(table, key_cols, nparts) -> Result:
    """-> Result with cols[0] = destination of every output row, cols[1] = input row number, then the columns; rows are
    destination-major, input order inside a destination."""
    keep = _Keep()
    t = _table(table, keep)
    kk = (C.c_int32 * max(1, len(key_cols)))(*[int(c) for c in key_cols])
    return Result(lib().ocl_hash_partition(C.byref(t), kk, len(key_cols), int(nparts)))


def avg(s: int, c: int) -> float:
    return float(lib().ocl_avg(int(s), int(c)))
