"""Writes tests/golden/fullsize_digests.json: digests of the ORACLE's output for BASELINE.json configs C2-C5 at their
full row counts (SURVEY §8(c) "full table exact").

    python tests/golden/make_fullsize_digests.py [--configs 2,3,4,5] [--jobs 4]

Calls only oracle/ and the seeded generator (paper_2606_24647_b200.datagen); nothing here comes from the CUDA path.
Per config: ngroups, rows fed to GROUP BY, and for every output column (keys, then aggregates), taken in key-tuple
order: wrapping u64 sum, xor, SHA-256 of the little-endian int64 bytes; C3 additionally stores its top-10 rows in
order. The single-threaded oracle cannot hold C5's 34 M groups in one std::map in reasonable time, so C5 (and, for
speed, C3/C4) is evaluated in SHARDS: fact rows are selected by `group key mod nshards` (selecting rows is input
preparation; every group lies in exactly one shard, so the union of the shard results is the oracle's result), each
shard is one oracle.run_query call, and the shard outputs are concatenated and sorted by key tuple.
"""
from __future__ import annotations

import argparse
import json
import multiprocessing as mp
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
for p in (ROOT, os.path.join(ROOT, "tests")):
    if p not in sys.path:
        sys.path.insert(0, p)

import oracle  # noqa: E402
import plans  # noqa: E402
from golden_util import digest_columns  # noqa: E402
from paper_2606_24647_b200 import datagen  # noqa: E402

OUT = os.path.join(HERE, "fullsize_digests.json")
_G = {}


def _shard(args):
    cfg, s, n = args
    plan = _G["plan"]
    key = plan["table"][plan["keys"][0]]
    m = (key % n) == s
    sub = dict(plan, table=[c[m] for c in plan["table"]])
    r = oracle.run_query(sub)
    return s, r.cols, r.input_rows, r.overflow


def run_config(cfg: int, jobs: int, nshards: int):
    t0 = time.time()
    t = datagen.make_config(cfg)
    plan = plans.PLANS[cfg](t)
    print(f"C{cfg}: generated in {time.time() - t0:.1f} s", flush=True)
    t0 = time.time()
    if not plan.get("keys"):
        r = oracle.run_query(plan)
        cols, input_rows, overflow = r.cols, r.input_rows, r.overflow
    else:
        _G["plan"] = plan
        with mp.get_context("fork").Pool(jobs) as pool:
            parts = pool.map(_shard, [(cfg, s, nshards) for s in range(nshards)], chunksize=1)
        ncol = len(parts[0][1])
        cols = [np.concatenate([p[1][c] for p in parts]) for c in range(ncol)]
        nk = len(plan["keys"])
        order = np.lexsort(tuple(cols[k] for k in reversed(range(nk))))
        cols = [c[order] for c in cols]
        input_rows = sum(p[2] for p in parts)
        overflow = any(p[3] for p in parts)
    print(f"C{cfg}: oracle {time.time() - t0:.1f} s, {len(cols[0])} output rows", flush=True)
    d = dict(ngroups=int(len(cols[0])), input_rows=int(input_rows), overflow=bool(overflow), columns=digest_columns(cols),
             nshards=(nshards if plan.get("keys") else 1), seed=datagen.BASE_SEED + cfg)
    if cfg == 3:   # top-10 under S11 from the full table: (sum desc, key asc)
        order = np.lexsort((cols[0], -cols[1]))[:10]
        d["top10"] = [[int(c[i]) for c in cols] for i in order]
        top = oracle.run_query(dict(table=cols, preds=[], exprs=[[("col", 1)], [("col", 2)]], keys=[0],
                                    aggs=[("sum", 0), ("sum", 1)], topk=10, topk_agg=0))   # the oracle's own top-k rule
        assert [[int(c[i]) for c in top.cols] for i in range(top.nrows)] == d["top10"]
    return d


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="2,3,4,5")
    ap.add_argument("--jobs", type=int, default=max(1, min(6, (os.cpu_count() or 2) - 1)))
    args = ap.parse_args()
    out = json.load(open(OUT)) if os.path.exists(OUT) else {}
    out["_how"] = "python tests/golden/make_fullsize_digests.py — oracle/ + datagen only; see the script's docstring"
    for cfg in [int(c) for c in args.configs.split(",")]:
        out[f"C{cfg}"] = run_config(cfg, args.jobs, {2: 1, 3: 16, 4: 16, 5: 96}[cfg])
        with open(OUT, "w") as f:
            json.dump(out, f, indent=1, sort_keys=True)
            f.write("\n")


if __name__ == "__main__":
    main()
