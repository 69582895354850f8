"""Thin Python binding of libgq.so (include/gq.h): argument marshalling only — every step runs in the CUDA library.

PyTorch is used for device memory and streams (columns, outputs and workspaces are torch CUDA tensors). There is no
CPU fallback: if libgq.so is missing or a call fails, an exception is raised.

Plan notation (plain Python data, mirrors gq.h):
    pred = (col, "lt|le|gt|ge|eq|ne|range_co|range_cc", lo[, hi])
    expr = [("col", i) | ("const", v) | ("add",) | ("sub",) | ("mul",), ...]        postfix, int64 wrapping
    agg  = ("sum|min|max", expr_index) | ("count",)
    probe = (Table, key_col)
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libgq.so")
_lib = None

I8, I32, I64 = 1, 2, 3
_DT = {torch.int8: I8, torch.int32: I32, torch.int64: I64}
_TORCH_DT = {I8: torch.int8, I32: torch.int32, I64: torch.int64}
_CMP = dict(lt=0, le=1, gt=2, ge=3, eq=4, ne=5, range_co=6, range_cc=7)
_XOP = dict(col=0, const=1, add=2, sub=3, mul=4)
_AGG = dict(sum=0, min=1, max=2, count=3)
F_UNIQUE_KEYS = 1
F_CHECK_DEPENDENT = 2
F_DENSE_KEYS = 4
F_FINAL_MODE = 8
STATUS = ["GQ_OK", "GQ_ERR_INVALID_ARG", "GQ_ERR_UNSUPPORTED", "GQ_ERR_CAPACITY", "GQ_ERR_WORKSPACE_TOO_SMALL",
          "GQ_ERR_CUDA", "GQ_ERR_DUPLICATE_KEY", "GQ_ERR_COMPILE", "GQ_ERR_DEPENDENT_KEY", "GQ_ERR_KEY_RANGE"]

# every symbol include/gq.h declares (tests check that the library exports all of them)
SYMBOLS = ["gq_create", "gq_destroy", "gq_sync", "gq_clear_error", "gq_status_str", "gq_last_cuda_error",
           "gq_last_message", "gq_launch_count", "gq_filter_project", "gq_hash_build_workspace", "gq_hash_build",
           "gq_hash_build_finish", "gq_table_count", "gq_table_destroy", "gq_hash_probe",
           "gq_hash_aggregate_workspace", "gq_hash_aggregate_workspace_for", "gq_hash_aggregate", "gq_topk_scratch_bytes", "gq_hash_aggregate_finish",
           "gq_aggstate_destroy", "gq_pipeline_workspace", "gq_pipeline", "gq_pipeline_host_workspace",
           "gq_pipeline_host", "gq_set_kernel_cache_dir", "gq_precompile_pipeline", "gq_precompile_build", "gq_precompile_materialise",
           "gq_table_describe", "gq_read_probe", "gq_set_option", "gq_hash_build_workspace_dense", "gq_profile", "gq_profile_read", "gq_order_by_workspace", "gq_order_by", "gq_aggstate_merge", "gq_aggstate_count",
           "gq_aggstate_rehash", "gq_order_by_static", "gq_order_by_static_max_rows",
           "gq_hash_partition_workspace", "gq_hash_partition", "gq_hash_partition_count", "gq_hash_partition_scatter_to"]


class GqError(RuntimeError):
    def __init__(self, status: int, msg: str = ""):
        self.status = status
        super().__init__(f"{STATUS[status] if 0 <= status < len(STATUS) else status}: {msg}")


class _Col(C.Structure):
    _fields_ = [("data", C.c_void_p), ("dtype", C.c_int)]


class _Batch(C.Structure):
    _fields_ = [("cols", C.POINTER(_Col)), ("ncols", C.c_int32), ("nrows", C.c_int64)]


class _Pred(C.Structure):
    _fields_ = [("col", C.c_int32), ("op", C.c_int), ("lo", C.c_int64), ("hi", C.c_int64)]


class _Tok(C.Structure):
    _fields_ = [("op", C.c_int), ("arg", C.c_int64)]


class _Expr(C.Structure):
    _fields_ = [("toks", C.POINTER(_Tok)), ("ntoks", C.c_int32)]


class _Agg(C.Structure):
    _fields_ = [("op", C.c_int), ("expr", C.c_int32)]


class _SortKey(C.Structure):
    _fields_ = [("col", C.c_int32), ("descending", C.c_int32)]


class _Probe(C.Structure):
    _fields_ = [("table", C.c_void_p), ("key_col", C.c_int32)]


class _BuildDesc(C.Structure):
    _fields_ = [("preds", C.POINTER(_Pred)), ("npred", C.c_int32), ("probes", C.POINTER(_Probe)),
                ("nprobes", C.c_int32), ("key_col", C.c_int32), ("payload_cols", C.POINTER(C.c_int32)),
                ("npayload", C.c_int32), ("flags", C.c_uint32), ("key_min", C.c_int64), ("key_max", C.c_int64)]


class _AggDesc(C.Structure):
    _fields_ = [("preds", C.POINTER(_Pred)), ("npred", C.c_int32), ("probes", C.POINTER(_Probe)),
                ("nprobes", C.c_int32), ("exprs", C.POINTER(_Expr)), ("nexpr", C.c_int32),
                ("key_cols", C.POINTER(C.c_int32)), ("nkeys", C.c_int32), ("ndependent", C.c_int32),
                ("aggs", C.POINTER(_Agg)), ("naggs", C.c_int32), ("max_groups", C.c_int64), ("flags", C.c_uint32)]


class _Avg(C.Structure):
    _fields_ = [("sum_agg", C.c_int32), ("count_agg", C.c_int32)]


class _Plan(C.Structure):
    _fields_ = [("in_", C.POINTER(_Batch)), ("agg", _AggDesc), ("avgs", C.POINTER(_Avg)), ("navg", C.c_int32),
                ("topk", C.c_int32), ("topk_agg", C.c_int32)]


def lib():
    """Loads libgq.so; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise RuntimeError(f"{_SO} is missing: build it with `python -m paper_2606_24647_b200.build` "
                               "(there is no CPU or PyTorch fallback)")
        L = C.CDLL(_SO)
        L.gq_status_str.restype = C.c_char_p
        L.gq_last_message.restype = C.c_char_p
        L.gq_last_message.argtypes = [C.c_void_p]
        L.gq_launch_count.restype = C.c_int64
        L.gq_launch_count.argtypes = [C.c_void_p]
        L.gq_topk_scratch_bytes.restype = C.c_size_t
        L.gq_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_void_p]
        for nm in ("gq_destroy", "gq_sync", "gq_clear_error", "gq_last_cuda_error"):
            getattr(L, nm).argtypes = [C.c_void_p]
        L.gq_filter_project.argtypes = [C.c_void_p, C.POINTER(_Batch), C.POINTER(_Pred), C.c_int32, C.POINTER(_Expr),
                                        C.c_int32, C.POINTER(C.c_void_p), C.c_int64, C.c_void_p]
        L.gq_hash_build_workspace.argtypes = [C.c_int64, C.c_int32, C.POINTER(C.c_size_t)]
        L.gq_hash_build_workspace_dense.argtypes = [C.c_int64, C.c_int64, C.c_int64, C.c_int32, C.POINTER(C.c_size_t)]
        L.gq_hash_build.argtypes = [C.c_void_p, C.POINTER(C.c_void_p), C.c_void_p, C.c_size_t, C.c_int64,
                                    C.POINTER(_Batch), C.POINTER(_BuildDesc)]
        L.gq_hash_build_finish.argtypes = [C.c_void_p, C.c_void_p]
        L.gq_table_count.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.gq_table_destroy.argtypes = [C.c_void_p]
        L.gq_hash_probe.argtypes = [C.c_void_p, C.POINTER(_Batch), C.POINTER(_Pred), C.c_int32, C.POINTER(_Probe),
                                    C.c_int32, C.POINTER(_Expr), C.c_int32, C.POINTER(C.c_void_p), C.c_int64, C.c_void_p]
        L.gq_hash_aggregate_workspace.argtypes = [C.c_int64, C.c_int32, C.c_int32, C.POINTER(C.c_size_t)]
        L.gq_hash_aggregate_workspace_for.argtypes = [C.POINTER(_Batch), C.POINTER(_AggDesc), C.POINTER(C.c_size_t)]
        L.gq_hash_aggregate.argtypes = [C.c_void_p, C.POINTER(C.c_void_p), C.c_void_p, C.c_size_t, C.POINTER(_Batch),
                                        C.POINTER(_AggDesc)]
        L.gq_hash_aggregate_finish.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p),
                                               C.POINTER(_Avg), C.c_int32, C.POINTER(C.c_void_p), C.c_int64,
                                               C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
        L.gq_aggstate_destroy.argtypes = [C.c_void_p]
        L.gq_pipeline_workspace.argtypes = [C.POINTER(_Plan), C.POINTER(C.c_size_t)]
        L.gq_pipeline.argtypes = [C.c_void_p, C.POINTER(_Plan), C.c_void_p, C.c_size_t, C.POINTER(C.c_void_p),
                                  C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.c_int64, C.c_void_p]
        L.gq_pipeline_host_workspace.argtypes = [C.POINTER(_Plan), C.c_int64, C.POINTER(C.c_size_t)]
        L.gq_pipeline_host.argtypes = [C.c_void_p, C.POINTER(_Plan), C.c_int64, C.c_void_p, C.c_size_t,
                                       C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.c_int64,
                                       C.c_void_p]
        L.gq_set_kernel_cache_dir.argtypes = [C.c_char_p]
        L.gq_precompile_pipeline.argtypes = [C.POINTER(_Plan), C.c_char_p, C.c_size_t]
        L.gq_precompile_build.argtypes = [C.POINTER(_Batch), C.POINTER(_BuildDesc), C.c_char_p, C.c_size_t]
        L.gq_precompile_materialise.argtypes = [C.POINTER(_Batch), C.POINTER(_Pred), C.c_int32, C.POINTER(_Probe), C.c_int32,
                                                C.POINTER(_Expr), C.c_int32, C.c_char_p, C.c_size_t]
        L.gq_table_describe.argtypes = [C.POINTER(C.c_void_p), C.POINTER(C.c_int), C.c_int32, C.c_uint32]
        L.gq_read_probe.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
        L.gq_set_option.argtypes = [C.c_char_p, C.c_int64]
        L.gq_aggstate_merge.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.gq_aggstate_count.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.gq_aggstate_rehash.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t, C.c_int64]
        L.gq_order_by_workspace.argtypes = [C.c_int64, C.POINTER(C.c_size_t)]
        L.gq_order_by.argtypes = [C.c_void_p, C.POINTER(_Batch), C.POINTER(_SortKey), C.c_int32, C.c_int64, C.c_void_p, C.c_size_t,
                                  C.c_void_p, C.POINTER(C.c_void_p)]
        L.gq_hash_partition_workspace.argtypes = [C.c_int32, C.POINTER(C.c_size_t)]
        L.gq_hash_partition.argtypes = [C.c_void_p, C.POINTER(_Batch), C.POINTER(C.c_int32), C.c_int32, C.c_int32, C.c_void_p, C.c_size_t,
                                        C.POINTER(C.c_void_p), C.c_void_p, C.c_void_p]
        L.gq_hash_partition_count.argtypes = [C.c_void_p, C.POINTER(_Batch), C.POINTER(C.c_int32), C.c_int32, C.c_int32, C.c_void_p, C.c_size_t,
                                              C.c_void_p]
        L.gq_hash_partition_scatter_to.argtypes = [C.c_void_p, C.POINTER(_Batch), C.POINTER(C.c_int32), C.c_int32, C.c_int32, C.c_void_p,
                                                   C.c_size_t, C.c_void_p, C.c_void_p]
        L.gq_order_by_static.argtypes = [C.c_void_p, C.POINTER(_Batch), C.POINTER(_SortKey), C.c_int32, C.c_int64,
                                         C.c_void_p, C.POINTER(C.c_void_p)]
        L.gq_order_by_static_max_rows.argtypes = []
        L.gq_order_by_static_max_rows.restype = C.c_int64
        L.gq_profile.argtypes = [C.c_void_p, C.c_int32]
        L.gq_profile_read.argtypes = [C.c_void_p, C.c_char_p, C.c_size_t, C.POINTER(C.c_float), C.c_int32]
        L.gq_profile_read.restype = C.c_int32
        _lib = L
    return _lib


# ------------------------------------------------------------------------------------------------ marshalling
class _M:
    """Marshalled descriptor arrays; keeps every ctypes object (and tensor) alive."""

    def __init__(self):
        self.keep = []

    def batch(self, cols, dtypes=None, nrows=None):
        """cols: tensors (device or pinned host) — or None entries with explicit dtypes for precompilation."""
        n = len(cols)
        cc = (_Col * max(1, n))()
        rows = nrows
        for i, t in enumerate(cols):
            if t is None:
                cc[i].data, cc[i].dtype = None, dtypes[i]
                continue
            if t.dtype not in _DT or t.dim() != 1 or not t.is_contiguous():
                raise ValueError("columns must be contiguous 1-D int8/int32/int64 tensors")
            cc[i].data, cc[i].dtype = t.data_ptr(), _DT[t.dtype]
            rows = t.shape[0] if rows is None else rows
            if t.shape[0] != rows:
                raise ValueError("columns of a batch must have equal length")
        b = _Batch(cc, n, rows or 0)
        self.keep += [cc, b, list(cols)]
        return b

    def preds(self, preds):
        pp = (_Pred * max(1, len(preds)))()
        for i, p in enumerate(preds):
            pp[i] = _Pred(int(p[0]), _CMP[p[1]], int(p[2]), int(p[3]) if len(p) > 3 else 0)
        self.keep.append(pp)
        return pp, len(preds)

    def exprs(self, exprs):
        ee = (_Expr * max(1, len(exprs)))()
        for i, e in enumerate(exprs):
            tt = (_Tok * max(1, len(e)))()
            for j, t in enumerate(e):
                tt[j] = _Tok(_XOP[t[0]], int(t[1]) if len(t) > 1 else 0)
            self.keep.append(tt)
            ee[i] = _Expr(tt, len(e))
        self.keep.append(ee)
        return ee, len(exprs)

    def probes(self, probes):
        pp = (_Probe * max(1, len(probes)))()
        for i, (tbl, key_col) in enumerate(probes):
            pp[i] = _Probe(tbl.handle, int(key_col))
        self.keep += [pp, list(probes)]
        return pp, len(probes)

    def ints(self, vals):
        a = (C.c_int32 * max(1, len(vals)))(*[int(v) for v in vals])
        self.keep.append(a)
        return a, len(vals)

    def ptrs(self, tensors):
        a = (C.c_void_p * max(1, len(tensors)))(*[t.data_ptr() for t in tensors])
        self.keep += [a, list(tensors)]
        return a

    def agg_desc(self, preds, probes, exprs, keys, ndependent, aggs, max_groups, check_dependent=False, final_mode=False):
        pr, npr = self.preds(preds)
        pb, npb = self.probes(probes)
        ee, ne = self.exprs(exprs)
        kk, nk = self.ints(keys)
        aa = (_Agg * max(1, len(aggs)))()
        for i, a in enumerate(aggs):
            aa[i] = _Agg(_AGG[a[0]], int(a[1]) if len(a) > 1 and a[1] is not None else 0)
        self.keep.append(aa)
        return _AggDesc(pr, npr, pb, npb, ee, ne, kk, nk, int(ndependent), aa, len(aggs), int(max_groups),
                        (F_CHECK_DEPENDENT if check_dependent else 0) | (F_FINAL_MODE if final_mode else 0))

    def build_desc(self, preds, probes, key, payload, unique, dense_range=None):
        pr, npr = self.preds(preds)
        pb, npb = self.probes(probes)
        pay, npay = self.ints(payload)
        lo, hi = (int(dense_range[0]), int(dense_range[1])) if dense_range is not None else (0, 0)
        return _BuildDesc(pr, npr, pb, npb, int(key), pay, npay,
                          (F_UNIQUE_KEYS if unique else 0) | (F_DENSE_KEYS if dense_range is not None else 0), lo, hi)

    def avgs(self, avgs):
        aa = (_Avg * max(1, len(avgs)))()
        for i, (s, c) in enumerate(avgs):
            aa[i] = _Avg(int(s), int(c))
        self.keep.append(aa)
        return aa, len(avgs)


class Table:
    """Join hash table: host handle + the workspace tensor it lives in."""

    def __init__(self, handle, workspace=None, payload_dtypes=()):
        self.handle, self.workspace, self.payload_dtypes = handle, workspace, tuple(payload_dtypes)

    def destroy(self):
        if self.handle:
            lib().gq_table_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def describe_table(payload_dtypes=(), unique=False, dense=False) -> Table:
    """Schema-only table handle for ahead-of-time kernel compilation (no device memory)."""
    h = C.c_void_p()
    arr = (C.c_int * max(1, len(payload_dtypes)))(*payload_dtypes)
    st = lib().gq_table_describe(C.byref(h), arr, len(payload_dtypes), (F_UNIQUE_KEYS if unique else 0) | (F_DENSE_KEYS if dense else 0))
    if st:
        raise GqError(st)
    return Table(h, None, payload_dtypes)


class AggState:
    def __init__(self, handle, workspace, key_dtypes, naggs):
        self.handle, self.workspace, self.key_dtypes, self.naggs = handle, workspace, key_dtypes, naggs

    def destroy(self):
        if self.handle:
            lib().gq_aggstate_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def _row_dtypes(cols, probes):
    dts = [_DT[c.dtype] for c in cols]
    for tbl, _ in probes:
        dts += list(tbl.payload_dtypes)
    return dts


class Context:
    """gq_ctx bound to a device and a CUDA stream (default: torch's current stream on that device)."""

    def __init__(self, device: int = 0, stream: torch.cuda.Stream | None = None):
        self.L = lib()
        if not torch.cuda.is_available():
            raise RuntimeError("gq needs a CUDA device (there is no CPU fallback)")
        self.device = torch.device("cuda", device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        self._check(self.L.gq_create(C.byref(h), device, C.c_void_p(self.stream.cuda_stream)), None)
        self.h = h

    def _check(self, st, _unused=None):
        if st != 0:
            msg = self.L.gq_last_message(self.h).decode() if getattr(self, "h", None) else ""
            raise GqError(st, msg)

    def close(self):
        if getattr(self, "h", None):
            self.L.gq_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def sync(self):
        """Host-blocking pipeline boundary; raises on a sticky device error."""
        self._check(self.L.gq_sync(self.h))

    def clear_error(self):
        self._check(self.L.gq_clear_error(self.h))

    def launch_count(self) -> int:
        return int(self.L.gq_launch_count(self.h))

    def _empty(self, n, dtype):
        return torch.empty(max(1, int(n)), dtype=dtype, device=self.device)

    def _ws(self, nbytes):
        return torch.empty(int(nbytes) + 256, dtype=torch.uint8, device=self.device)

    @staticmethod
    def _ws_ptr(ws):
        return (ws.data_ptr() + 255) // 256 * 256

    # ---- FilterProject / HashProbe (materialising) ----
    def filter_project(self, cols, preds, exprs, capacity=None, probes=(), outs=None, count=None):
        """outs / count: optional pre-allocated int64 output columns and a ZEROED int64[1] counter to reuse."""
        with torch.cuda.stream(self.stream):
            m = _M()
            b = m.batch(cols)
            cap = int(capacity) if capacity is not None else int(b.nrows)
            if outs is None:
                outs = [self._empty(cap, torch.int64) for _ in exprs]
            if count is None:
                count = torch.zeros(1, dtype=torch.int64, device=self.device)
            pr, npr = m.preds(preds)
            ee, ne = m.exprs(exprs)
            if probes:
                pb, npb = m.probes(probes)
                st = self.L.gq_hash_probe(self.h, C.byref(b), pr, npr, pb, npb, ee, ne, m.ptrs(outs), cap, count.data_ptr())
            else:
                st = self.L.gq_filter_project(self.h, C.byref(b), pr, npr, ee, ne, m.ptrs(outs), cap, count.data_ptr())
            self._check(st)
        return outs, count

    def hash_probe(self, cols, preds, probes, exprs, capacity, outs=None, count=None):
        return self.filter_project(cols, preds, exprs, capacity=capacity, probes=probes, outs=outs, count=count)

    # ---- HashBuild ----
    def hash_build(self, cols, preds=(), probes=(), key=0, payload=(), unique=False, max_rows=None, table=None,
                   finish=True, workspace=None, dense_range=None):
        """workspace: a uint8 CUDA tensor to (re)use for the table instead of allocating one.
        dense_range=(key_min, key_max): GQ_F_DENSE_KEYS, a direct-address table over that key range."""
        with torch.cuda.stream(self.stream):
            m = _M()
            b = m.batch(cols)
            d = m.build_desc(preds, probes, key, payload, unique, dense_range)
            if table is None:
                max_rows = int(b.nrows if max_rows is None else max_rows)
                nbytes = C.c_size_t()
                if dense_range is not None:
                    self._check(self.L.gq_hash_build_workspace_dense(int(dense_range[0]), int(dense_range[1]), max_rows, len(payload), C.byref(nbytes)))
                else:
                    self._check(self.L.gq_hash_build_workspace(max_rows, len(payload), C.byref(nbytes)))
                ws = workspace if workspace is not None else self._ws(nbytes.value)
                if ws.numel() < nbytes.value + 256:
                    raise ValueError("workspace tensor too small")
                dts = _row_dtypes(cols, probes)
                h = C.c_void_p()
                st = self.L.gq_hash_build(self.h, C.byref(h), self._ws_ptr(ws), nbytes.value, max_rows, C.byref(b), C.byref(d))
                self._check(st)
                table = Table(h, ws, [dts[c] for c in payload])
            else:
                h = C.c_void_p(table.handle.value if isinstance(table.handle, C.c_void_p) else table.handle)
                self._check(self.L.gq_hash_build(self.h, C.byref(h), None, 0, 0, C.byref(b), C.byref(d)))
            if finish:
                self._check(self.L.gq_hash_build_finish(self.h, table.handle))
        return table

    # ---- OrderBy / TopN ----
    def order_by(self, cols, keys, limit=0, gather=True, workspace=None):
        """keys = [(column, descending)]. -> (index int64[n_out], [gathered columns] or None); n_out = min(limit, nrows)."""
        with torch.cuda.stream(self.stream):
            m = _M()
            b = m.batch(cols)
            n = int(b.nrows)
            nout = n if limit <= 0 or limit > n else int(limit)
            kk = (_SortKey * max(1, len(keys)))()
            for i, (c, d) in enumerate(keys):
                kk[i] = _SortKey(int(c), 1 if d else 0)
            m.keep.append(kk)
            nbytes = C.c_size_t()
            self._check(self.L.gq_order_by_workspace(n, C.byref(nbytes)))
            ws = workspace if workspace is not None else self._ws(nbytes.value)
            index = self._empty(nout, torch.int64)
            outs = [self._empty(nout, c.dtype) for c in cols] if gather else None
            self._check(self.L.gq_order_by(self.h, C.byref(b), kk, len(keys), int(limit), self._ws_ptr(ws), nbytes.value,
                                           index.data_ptr(), m.ptrs(outs) if gather else None))
            self._last_ws = ws
        return index[:nout], ([o[:nout] for o in outs] if gather else None)

    def hash_partition(self, cols, key_cols, nparts, want_rows=False, workspace=None, outs=None, offsets=None):
        """gq_hash_partition: -> (out_cols, offsets int64[nparts + 1], rows int64[n] or None); rows of destination d are
        out rows [offsets[d], offsets[d + 1]), in input order."""
        with torch.cuda.stream(self.stream):
            m = _M()
            b = m.batch(cols)
            n = int(b.nrows)
            kk = (C.c_int32 * max(1, len(key_cols)))(*[int(c) for c in key_cols])
            m.keep.append(kk)
            nbytes = C.c_size_t()
            st = self.L.gq_hash_partition_workspace(int(nparts), C.byref(nbytes))
            ws = workspace if workspace is not None else self._ws(nbytes.value if st == 0 else 256)
            outs = outs if outs is not None else [self._empty(n, c.dtype) for c in cols]
            offsets = offsets if offsets is not None else self._empty(max(1, int(nparts)) + 1, torch.int64)
            rows = self._empty(n, torch.int64) if want_rows else None
            self._check(self.L.gq_hash_partition(self.h, C.byref(b), kk, len(key_cols), int(nparts), self._ws_ptr(ws), nbytes.value,
                                                 m.ptrs(outs), rows.data_ptr() if want_rows else None, offsets.data_ptr()))
            self._last_ws = ws
        return outs, offsets, rows

    def hash_partition_count(self, cols, key_cols, nparts, workspace=None):
        """Phase 1 of the fused partition + transfer: -> (counts int64[nparts] on the device, workspace to pass on)."""
        with torch.cuda.stream(self.stream):
            m = _M()
            b = m.batch(cols)
            kk = (C.c_int32 * max(1, len(key_cols)))(*[int(c) for c in key_cols])
            m.keep.append(kk)
            nbytes = C.c_size_t()
            st = self.L.gq_hash_partition_workspace(int(nparts), C.byref(nbytes))
            ws = workspace if workspace is not None else self._ws(nbytes.value if st == 0 else 256)
            counts = self._empty(max(1, int(nparts)), torch.int64)
            self._check(self.L.gq_hash_partition_count(self.h, C.byref(b), kk, len(key_cols), int(nparts), self._ws_ptr(ws), nbytes.value,
                                                       counts.data_ptr()))
        return counts, ws

    def hash_partition_scatter_to(self, cols, key_cols, nparts, workspace, dst_cols, dst_row0):
        """Phase 2: scatter the same batch; dst_cols[d][c] = destination d's buffer for column c (a tensor this GPU can
        write: local or peer-mapped), dst_row0 = int64[nparts] device tensor of first rows."""
        with torch.cuda.stream(self.stream):
            m = _M()
            b = m.batch(cols)
            kk = (C.c_int32 * max(1, len(key_cols)))(*[int(c) for c in key_cols])
            m.keep.append(kk)
            nbytes = C.c_size_t()
            self._check(self.L.gq_hash_partition_workspace(int(nparts), C.byref(nbytes)))
            ptrs = torch.tensor([int(t.data_ptr()) for d in dst_cols for t in d], dtype=torch.int64).to(self.device, non_blocking=False)
            self._check(self.L.gq_hash_partition_scatter_to(self.h, C.byref(b), kk, len(key_cols), int(nparts), self._ws_ptr(workspace),
                                                            nbytes.value, ptrs.data_ptr(), dst_row0.data_ptr()))
            self._last_ptrs = ptrs

    def order_by_static(self, cols, keys, limit, out_index, out_cols=None):
        """gq_order_by_static: order_by that allocates nothing — scratch is a fixed device array inside libgq.so, the
        caller passes the outputs (out_index int64[>= n_out] and/or out_cols, one tensor per input column). At most
        order_by_static_max_rows() rows; calls on one device must not overlap on the GPU. -> n_out."""
        with torch.cuda.stream(self.stream):
            m = _M()
            b = m.batch(cols)
            n = int(b.nrows)
            nout = n if limit <= 0 or limit > n else int(limit)
            kk = (_SortKey * max(1, len(keys)))()
            for i, (c, d) in enumerate(keys):
                kk[i] = _SortKey(int(c), 1 if d else 0)
            m.keep.append(kk)
            if out_index is not None and (out_index.dtype != torch.int64 or out_index.numel() < nout):
                raise ValueError("out_index must be int64 with at least n_out elements")
            if out_cols is not None and (len(out_cols) != len(cols) or any(o.dtype != c.dtype or o.numel() < nout for o, c in zip(out_cols, cols))):
                raise ValueError("out_cols must match the input columns' dtypes and hold n_out rows")
            self._check(self.L.gq_order_by_static(self.h, C.byref(b), kk, len(keys), int(limit),
                                                  out_index.data_ptr() if out_index is not None else None,
                                                  m.ptrs(list(out_cols)) if out_cols is not None else None))
        return nout

    @staticmethod
    def order_by_static_max_rows() -> int:
        return int(lib().gq_order_by_static_max_rows())

    def profile(self, enable=True):
        """gq_profile: bracket every kernel launch of this context with CUDA events (off in timed loops)."""
        self._check(self.L.gq_profile(self.h, 1 if enable else 0))

    def profile_read(self, max_entries=256):
        """-> [(kernel name, ms)] recorded since the last read; waits for the stream."""
        names = C.create_string_buffer(64 * max_entries)
        ms = (C.c_float * max_entries)()
        n = self.L.gq_profile_read(self.h, names, len(names), ms, max_entries)
        if n < 0:
            raise GqError(5, "gq_profile_read")
        return list(zip(names.value.decode().split("\n")[:n], [float(ms[i]) for i in range(n)]))

    def table_count(self, table) -> torch.Tensor:
        out = torch.zeros(1, dtype=torch.int64, device=self.device)
        with torch.cuda.stream(self.stream):
            self._check(self.L.gq_table_count(self.h, table.handle, out.data_ptr()))
        return out

    # ---- HashAggregation (streaming) ----
    def aggregate(self, state, cols, preds=(), probes=(), exprs=(), keys=(), ndependent=0, aggs=(), max_groups=1,
                  plan_aware_workspace=False, check_dependent=False, final_mode=False):
        """plan_aware_workspace: size the state with gq_hash_aggregate_workspace_for (enables direct aggregation).
        final_mode: GQ_F_FINAL_MODE — the rows are intermediate results; ("count", e) sums the partial counts in expr e."""
        with torch.cuda.stream(self.stream):
            m = _M()
            b = m.batch(cols)
            d = m.agg_desc(preds, probes, exprs, keys, ndependent, aggs, max_groups, check_dependent, final_mode)
            if state is None:
                nbytes = C.c_size_t()
                if plan_aware_workspace:
                    self._check(self.L.gq_hash_aggregate_workspace_for(C.byref(b), C.byref(d), C.byref(nbytes)))
                else:
                    self._check(self.L.gq_hash_aggregate_workspace(int(max_groups), len(keys), len(aggs), C.byref(nbytes)))
                ws = self._ws(nbytes.value)
                dts = _row_dtypes(cols, probes)
                h = C.c_void_p()
                self._check(self.L.gq_hash_aggregate(self.h, C.byref(h), self._ws_ptr(ws), nbytes.value, C.byref(b), C.byref(d)))
                state = AggState(h, ws, [dts[k] for k in keys], len(aggs))
            else:
                h = C.c_void_p(state.handle.value)
                self._check(self.L.gq_hash_aggregate(self.h, C.byref(h), None, 0, C.byref(b), C.byref(d)))
        return state

    def aggregate_merge(self, dst, src):
        """gq_aggstate_merge: fold the groups of state `src` into state `dst` (Partial -> Final between states)."""
        with torch.cuda.stream(self.stream):
            self._check(self.L.gq_aggstate_merge(self.h, dst.handle, src.handle))

    def aggregate_count(self, state) -> torch.Tensor:
        out = torch.zeros(1, dtype=torch.int64, device=self.device)
        with torch.cuda.stream(self.stream):
            self._check(self.L.gq_aggstate_count(self.h, state.handle, out.data_ptr()))
        return out

    def aggregate_rehash(self, state, new_max_groups):
        """gq_aggstate_rehash: grow a high-cardinality state into a larger table (new workspace; the old one is kept
        alive by the state object until the next rehash)."""
        with torch.cuda.stream(self.stream):
            nbytes = C.c_size_t()
            self._check(self.L.gq_hash_aggregate_workspace(int(new_max_groups), len(state.key_dtypes), state.naggs, C.byref(nbytes)))
            ws = self._ws(nbytes.value)
            self._check(self.L.gq_aggstate_rehash(self.h, state.handle, self._ws_ptr(ws), nbytes.value, int(new_max_groups)))
            state.old_workspace, state.workspace = state.workspace, ws

    def aggregate_finish(self, state, capacity, avgs=(), topk=0, topk_agg=0):
        with torch.cuda.stream(self.stream):
            m = _M()
            cap = int(capacity)
            keys = [self._empty(cap, _TORCH_DT[dt]) for dt in state.key_dtypes]
            aggs = [self._empty(cap, torch.int64) for _ in range(state.naggs)]
            av = [self._empty(cap, torch.float64) for _ in avgs]
            n = torch.zeros(1, dtype=torch.int64, device=self.device)
            aa, na = m.avgs(avgs)
            scratch = self._ws(self.L.gq_topk_scratch_bytes()) if topk > 0 else None
            st = self.L.gq_hash_aggregate_finish(self.h, state.handle, m.ptrs(keys), m.ptrs(aggs), aa, na, m.ptrs(av), cap,
                                                 int(topk), int(topk_agg), self._ws_ptr(scratch) if topk > 0 else None,
                                                 n.data_ptr())
            self._check(st)
        return dict(keys=keys, aggs=aggs, avgs=av, n=n, _scratch=scratch)

    # ---- fused pipeline ----
    def prepare_pipeline(self, cols, preds=(), probes=(), exprs=(), keys=(), ndependent=0, aggs=(), max_groups=1,
                         avgs=(), topk=0, topk_agg=0, out_capacity=None, check_dependent=False):
        return Pipeline(self, cols, preds, probes, exprs, keys, ndependent, aggs, max_groups, avgs, topk, topk_agg,
                        out_capacity, check_dependent)

    def read_probe(self, t: torch.Tensor) -> torch.Tensor:
        out = torch.zeros(1, dtype=torch.int64, device=self.device)
        nbytes = t.numel() * t.element_size() // 16 * 16
        with torch.cuda.stream(self.stream):
            self._check(self.L.gq_read_probe(self.h, t.data_ptr(), nbytes, out.data_ptr()))
        return out



class Pipeline:
    """A marshalled gq_plan with its workspace and outputs pre-allocated: run() is one gq_pipeline call (enqueue only)."""

    def __init__(self, ctx, cols, preds, probes, exprs, keys, ndependent, aggs, max_groups, avgs, topk, topk_agg,
                 out_capacity, check_dependent=False):
        self.ctx, L = ctx, ctx.L
        m = self.m = _M()
        self.host = not cols[0].is_cuda
        self.batch = m.batch(cols)
        aa, na = m.avgs(avgs)
        self.plan = _Plan(C.pointer(self.batch),
                          m.agg_desc(preds, probes, exprs, keys, ndependent, aggs, max_groups, check_dependent),
                          aa, na, int(topk), int(topk_agg))
        dts = _row_dtypes(cols, probes)
        cap = int(out_capacity if out_capacity is not None else (topk if topk > 0 else max(1, max_groups)))
        self.capacity = cap
        dev = "cpu" if self.host else ctx.device
        mk = (lambda n, dt: torch.empty(max(1, n), dtype=dt).pin_memory()) if self.host else \
             (lambda n, dt: torch.empty(max(1, n), dtype=dt, device=dev))
        self.keys = [mk(cap, _TORCH_DT[dts[k]]) for k in keys]
        self.aggs = [mk(cap, torch.int64) for _ in aggs]
        self.avgs = [mk(cap, torch.float64) for _ in avgs]
        self.n = mk(1, torch.int64)
        self.pk, self.pa, self.pv = m.ptrs(self.keys), m.ptrs(self.aggs), m.ptrs(self.avgs)
        self.chunk_rows = None
        self.ws = None
        if not self.host:
            nbytes = C.c_size_t()
            ctx._check(L.gq_pipeline_workspace(C.byref(self.plan), C.byref(nbytes)))
            self.ws_bytes = nbytes.value
            with torch.cuda.stream(ctx.stream):
                self.ws = ctx._ws(self.ws_bytes)

    def run(self):
        """Enqueue the whole pipeline (device-resident inputs). No host synchronisation."""
        c = self.ctx
        c._check(c.L.gq_pipeline(c.h, C.byref(self.plan), Context._ws_ptr(self.ws), self.ws_bytes, self.pk, self.pa,
                                 self.pv, self.capacity, self.n.data_ptr()))

    def run_host(self, chunk_rows=8 << 20):
        """End-to-end call with HOST (pinned) input columns and HOST outputs; returns after results have landed."""
        c = self.ctx
        if self.ws is None or self.chunk_rows != chunk_rows:
            nbytes = C.c_size_t()
            c._check(c.L.gq_pipeline_host_workspace(C.byref(self.plan), int(chunk_rows), C.byref(nbytes)))
            self.ws_bytes, self.chunk_rows = nbytes.value, chunk_rows
            with torch.cuda.stream(c.stream):
                self.ws = c._ws(self.ws_bytes)
        c._check(c.L.gq_pipeline_host(c.h, C.byref(self.plan), int(chunk_rows), Context._ws_ptr(self.ws), self.ws_bytes,
                                      self.pk, self.pa, self.pv, self.capacity, self.n.data_ptr()))

    def result(self):
        """After ctx.sync(): dict of trimmed output tensors."""
        n = int(self.n.item())
        return dict(n=n, keys=[k[:n] for k in self.keys], aggs=[a[:n] for a in self.aggs], avgs=[v[:n] for v in self.avgs])


def set_option(name: str, value: int) -> None:
    """Planner knob (gq_set_option): e.g. "part_min_rows"; a negative value restores the default."""
    st = lib().gq_set_option(name.encode(), int(value))
    if st:
        raise GqError(st, f"unknown option {name}")


def precompile_pipeline(col_dtypes, nrows, preds=(), probes=(), exprs=(), keys=(), ndependent=0, aggs=(), max_groups=1,
                        check_dependent=False):
    """Compile (or find cached) the fused kernel of a plan shape; needs no GPU. Returns the cubin path."""
    m = _M()
    b = m.batch([None] * len(col_dtypes), dtypes=list(col_dtypes), nrows=int(nrows))
    plan = _Plan(C.pointer(b), m.agg_desc(preds, probes, exprs, keys, ndependent, aggs, max_groups, check_dependent),
                 None, 0, 0, 0)
    buf = C.create_string_buffer(8192)
    st = lib().gq_precompile_pipeline(C.byref(plan), buf, 8192)
    if st:
        raise GqError(st, buf.value.decode(errors="replace"))
    return buf.value.decode()


def precompile_materialise(col_dtypes, nrows, preds=(), probes=(), exprs=()):
    """Kernel of filter_project / hash_probe for this shape; needs no GPU. Returns the cubin path."""
    m = _M()
    b = m.batch([None] * len(col_dtypes), dtypes=list(col_dtypes), nrows=int(nrows))
    pr, npr = m.preds(preds)
    pb, npb = m.probes(probes)
    ee, ne = m.exprs(exprs)
    buf = C.create_string_buffer(8192)
    st = lib().gq_precompile_materialise(C.byref(b), pr, npr, pb, npb, ee, ne, buf, 8192)
    if st:
        raise GqError(st, buf.value.decode(errors="replace"))
    return buf.value.decode()


def precompile_build(col_dtypes, nrows, preds=(), probes=(), key=0, payload=(), unique=False, dense_range=None):
    m = _M()
    b = m.batch([None] * len(col_dtypes), dtypes=list(col_dtypes), nrows=int(nrows))
    d = m.build_desc(preds, probes, key, payload, unique, dense_range)
    buf = C.create_string_buffer(8192)
    st = lib().gq_precompile_build(C.byref(b), C.byref(d), buf, 8192)
    if st:
        raise GqError(st, buf.value.decode(errors="replace"))
    return buf.value.decode()
