"""Runs a neutral plan (tests/plans.py format) through the CUDA library and returns numpy results comparable with the
oracle's: rows sorted by key tuple (or in top-k order). Marshalling only — no arithmetic of the method happens here."""
from __future__ import annotations

import numpy as np
import torch

from paper_2606_24647_b200 import gq


def dev(cols, device="cuda"):
    return [torch.from_numpy(np.ascontiguousarray(c)).to(device) for c in cols]


def build_tables(ctx, plan, device_tables=None, workspaces=None):
    """HashBuild for every plan['builds'] entry, in order (each may probe earlier ones)."""
    tables = []
    for i, b in enumerate(plan.get("builds", [])):
        ws = workspaces[i] if workspaces is not None else None
        cols = device_tables[i] if device_tables is not None else dev(b["table"])
        probes = [(tables[bi], kc) for bi, kc in b.get("probes", [])]
        tables.append(ctx.hash_build(cols, preds=b.get("preds", []), probes=probes, key=b["key"],
                                     payload=b.get("payload", []), unique=b.get("unique", False),
                                     max_rows=b.get("max_rows"), workspace=ws, dense_range=b.get("dense_range")))
    return tables


def prepare(ctx, plan, tables, cols=None, out_capacity=None, avgs=()):
    cols = cols if cols is not None else dev(plan["table"])
    probes = [(tables[bi], kc) for bi, kc in plan.get("probes", [])]
    return ctx.prepare_pipeline(cols, preds=plan.get("preds", []), probes=probes, exprs=plan.get("exprs", []),
                                keys=plan.get("keys", []), ndependent=plan.get("ndependent", 0), aggs=plan["aggs"],
                                max_groups=plan.get("max_groups", 1), avgs=avgs, topk=plan.get("topk", 0),
                                topk_agg=plan.get("topk_agg", 0), out_capacity=out_capacity)


def sort_rows(cols, nkeys):
    """Sort result columns by key tuple ascending (group order is unspecified on the GPU side)."""
    if not cols or len(cols[0]) == 0 or nkeys == 0:
        return cols
    order = np.lexsort(tuple(cols[k] for k in reversed(range(nkeys))))
    return [c[order] for c in cols]


def run_query(plan, ctx=None, avgs=(), out_capacity=None):
    """-> dict(cols=[int64 numpy arrays: keys then aggs], avgs=[float64 arrays], n=int)"""
    ctx = ctx or gq.Context()
    tables = build_tables(ctx, plan)
    p = prepare(ctx, plan, tables, out_capacity=out_capacity, avgs=avgs)
    p.run()
    ctx.sync()
    r = p.result()
    cols = [k.cpu().numpy().astype(np.int64) for k in r["keys"]] + [a.cpu().numpy() for a in r["aggs"]]
    av = [v.cpu().numpy() for v in r["avgs"]]
    nk = len(plan.get("keys", []))
    if plan.get("topk", 0) == 0 and nk:
        order = np.lexsort(tuple(cols[k] for k in reversed(range(nk))))
        cols = [c[order] for c in cols]
        av = [v[order] for v in av]
    return dict(cols=cols, avgs=av, n=r["n"])
