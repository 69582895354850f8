"""Seeded synthetic column generator; shared by the oracle tests and the CUDA path.

Holds none of the method's arithmetic: it only draws columns.  ``make_config(n, scale)`` returns the tables of
BASELINE.json config C<n> as ``{table: {column: numpy array}}``; the recipe is restated in DESIGN.md §"Input recipe".
The tables stand in for the dbgen-generated TPC-H-like tables the paper measures on.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libgqgen.so")
_SRC = os.path.join(_HERE, "gqgen.cpp")
_lib = None

BASE_SEED = 26062464700  # seed of config n = BASE_SEED + n


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-pthread", _SRC, "-o", _SO])
    return _SO


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        u64, i64, p, ci = ctypes.c_uint64, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int
        L.gqgen_hw_threads.restype = ci
        for nm in ("gqgen_uniform_i64", "gqgen_uniform_i32", "gqgen_uniform_i8"):
            getattr(L, nm).argtypes = [u64, u64, i64, i64, i64, p, ci]
            getattr(L, nm).restype = None
        L.gqgen_shuffle_i64.argtypes = [u64, u64, i64, p]
        L.gqgen_permutation_i64.argtypes = [u64, u64, i64, p]
        L.gqgen_pick_i64.argtypes = [u64, u64, p, i64, i64, p, ci]
        L.gqgen_fanout_fk.argtypes = [u64, u64, u64, p, i64, i64, ci, p]
        L.gqgen_fanout_fk.restype = ci
        L.gqgen_zipf_keys.argtypes = [u64, u64, i64, i64, p, ci]
        L.gqgen_checksum.argtypes = [p, ci, i64, p]
        _lib = L
    return _lib


def _threads() -> int:
    return max(1, min(64, lib().gqgen_hw_threads()))


_DT = {"i8": np.int8, "i32": np.int32, "i64": np.int64}


def uniform(seed: int, stream: int, lo: int, hi: int, n: int, dtype: str) -> np.ndarray:
    out = np.empty(n, dtype=_DT[dtype])
    getattr(lib(), "gqgen_uniform_" + dtype)(seed, stream, lo, hi, n, out.ctypes.data, _threads())
    return out


def permutation(seed: int, stream: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.int64)
    lib().gqgen_permutation_i64(seed, stream, n, out.ctypes.data)
    return out


def pick(seed: int, stream: int, domain: np.ndarray, n: int) -> np.ndarray:
    domain = np.ascontiguousarray(domain, dtype=np.int64)
    out = np.empty(n, dtype=np.int64)
    lib().gqgen_pick_i64(seed, stream, domain.ctypes.data, domain.size, n, out.ctypes.data, _threads())
    return out


def fanout_fk(seed: int, s_counts: int, s_shuffle: int, dimkeys: np.ndarray, nfact: int, clustered: bool) -> np.ndarray:
    dimkeys = np.ascontiguousarray(dimkeys, dtype=np.int64)
    out = np.empty(nfact, dtype=np.int64)
    rc = lib().gqgen_fanout_fk(seed, s_counts, s_shuffle, dimkeys.ctypes.data, dimkeys.size, nfact, int(clustered),
                               out.ctypes.data)
    if rc != 0:
        raise ValueError("fanout_fk needs ndim <= nfact <= 7*ndim")
    return out


def zipf_keys(seed: int, stream: int, ndistinct: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.int64)
    lib().gqgen_zipf_keys(seed, stream, ndistinct, n, out.ctypes.data, _threads())
    return out


def checksum(a: np.ndarray):
    a = np.ascontiguousarray(a)
    out = (ctypes.c_uint64 * 4)()
    lib().gqgen_checksum(a.ctypes.data, a.dtype.itemsize, a.size, out)
    return [int(out[0]), int(out[1]), int(np.int64(np.uint64(out[2]))), int(np.int64(np.uint64(out[3])))]


# Column streams (fixed ids so a column's bytes do not depend on which other columns are generated).
_S = dict(shipdate=1, quantity=2, price=3, discount=4, tax=5, flagA=6, flagB=7, dimkey=8, orderdate=9, fk_counts=10,
          fk_shuffle=11, custkey_perm=12, segment=13, ord_custkey=14, zipf=15)

# Full row counts of BASELINE.json configs.
ROWS = {1: dict(fact=1_000_000), 2: dict(fact=60_000_000), 3: dict(dim=15_000_000, fact=60_000_000),
        4: dict(cust=1_500_000, orders=15_000_000, fact=60_000_000), 5: dict(fact=600_000_000, keys=50_000_000)}


def _fact_cols(seed: int, n: int, names) -> dict:
    spec = dict(shipdate=(0, 2525, "i32"), quantity=(1, 50, "i64"), price=(90000, 10500000, "i64"),
                discount=(0, 10, "i64"), tax=(0, 8, "i64"), flagA=(0, 2, "i8"), flagB=(0, 1, "i8"))
    return {c: uniform(seed, _S[c], spec[c][0], spec[c][1], n, spec[c][2]) for c in names}


def make_config(cfg: int, scale: float = 1.0, clustered: bool = False, seed: int | None = None) -> dict:
    """Tables of config C<cfg>; ``scale`` multiplies every row count (and the Zipf domain) for small parity cases."""
    seed = BASE_SEED + cfg if seed is None else seed
    r = {k: max(1, int(round(v * scale))) for k, v in ROWS[cfg].items()}
    if cfg == 1:
        return {"fact": _fact_cols(seed, r["fact"], ["shipdate", "quantity", "price", "discount", "tax", "flagA", "flagB"])}
    if cfg == 2:
        return {"fact": _fact_cols(seed, r["fact"], ["shipdate", "discount", "quantity", "price"])}
    if cfg == 3:
        nd = r["dim"]; nf = min(max(r["fact"], nd), 7 * nd)
        key = permutation(seed, _S["dimkey"], nd)
        dim = {"key": key, "orderdate": uniform(seed, _S["orderdate"], 0, 2405, nd, "i32")}
        fact = {"fk": fanout_fk(seed, _S["fk_counts"], _S["fk_shuffle"], key, nf, clustered)}
        fact.update(_fact_cols(seed, nf, ["shipdate", "price", "discount"]))
        return {"dim": dim, "fact": fact}
    if cfg == 4:
        nc, no = r["cust"], r["orders"]; nf = min(max(r["fact"], no), 7 * no)
        ckey = permutation(seed, _S["custkey_perm"], nc)
        cust = {"key": ckey, "segment": uniform(seed, _S["segment"], 0, 4, nc, "i8")}
        okey = permutation(seed, _S["dimkey"], no)
        orders = {"orderkey": okey, "custkey": pick(seed, _S["ord_custkey"], ckey, no),
                  "orderdate": uniform(seed, _S["orderdate"], 0, 2405, no, "i32")}
        fact = {"fk": fanout_fk(seed, _S["fk_counts"], _S["fk_shuffle"], okey, nf, clustered)}
        fact.update(_fact_cols(seed, nf, ["shipdate", "price", "discount"]))
        return {"cust": cust, "orders": orders, "fact": fact}
    if cfg == 5:
        n, nk = r["fact"], r["keys"]
        fact = {"key": zipf_keys(seed, _S["zipf"], nk, n)}
        fact.update(_fact_cols(seed, n, ["shipdate", "price", "quantity"]))
        return {"fact": fact}
    raise ValueError("config must be 1..5")
