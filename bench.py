#!/usr/bin/env python
"""bench.py — measures the hot path on B200 (contract: prompt §④ / "Maintain bench.py").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--configs 1,1x64,3,4,5,ops]

A step = one pass of the whole fused pipeline (table init -> builds -> fused scan kernel -> finaliser) over one batch
of synthetic input. Headline workload: BASELINE.json configs[1] (C2: selective filter + global SUM over 60 M rows, the
pure scan-bandwidth test the metric's >= 70 % target is quoted on). Every other config is measured in the same run and
reported under "per_config" with the same record: pipeline ms, per-kernel device times (gq_profile), the dominant
kernel's roofline, parity against the oracle (stored oracle-written digests at full size), clocks. Inputs are larger
than L2 (C1: rotated copies), so every timed iteration reads HBM. N > 1 (torchrun): the path does not shard — each
rank runs an independent replica ("replicas only") and value = N * rows / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
for p in (ROOT, os.path.join(ROOT, "tests")):
    if p not in sys.path:
        sys.path.insert(0, p)

import numpy as np  # noqa: E402

METRIC = "input rows/s and achieved HBM GB/s (% of B200 peak) per operator pipeline"
WORKLOAD = "C2 selective filter + global SUM(price*discount), 60M-row fact (BASELINE configs[1])"
ALG_BYTES_PER_ROW = {1: 38, 2: 28, 3: 28, 4: 28, 5: 28}   # referenced fact columns, SURVEY §8(d)
L2_NOTE = "inputs (1.68 GB) are larger than L2: every timed iteration reads HBM (no flush needed)"
MIN_LOAD_MS = 120.0                                      # the clock sampler sees at least this much load per loop


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def host_info():
    model, mem = None, None
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    model = line.split(":", 1)[1].strip()
                    break
        with open("/proc/meminfo") as f:
            for line in f:
                if line.startswith("MemTotal"):
                    mem = line.split(":", 1)[1].strip()
                    break
    except OSError:
        pass
    return dict(nproc=os.cpu_count(), cpu_model=model, mem_total=mem)


class ClockSampler:
    """Samples SM clock and clock-event (throttle) reasons through NVML in a thread while a loop runs."""
    BITS = dict(sw_power_cap=0x4, hw_slowdown=0x8, sw_thermal_slowdown=0x20, hw_thermal_slowdown=0x40)

    def __init__(self, index=0):
        self.index, self.sm, self.reasons, self.max, self.power = index, [], 0, None, []
        self._stop = threading.Event()
        self._t = None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            get_reasons = getattr(pynvml, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
                pynvml.nvmlDeviceGetCurrentClocksThrottleReasons

            def loop():
                while not self._stop.is_set():
                    try:
                        self.sm.append(float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)))
                        self.reasons |= int(get_reasons(h))
                        self.power.append(pynvml.nvmlDeviceGetPowerUsage(h) / 1000.0)
                    except Exception:
                        pass
                    time.sleep(0.002)
            self._t = threading.Thread(target=loop, daemon=True)
            self._t.start()
        except Exception:
            self._t = None
        return self

    def stop(self):
        self._stop.set()
        if self._t:
            self._t.join(timeout=1.0)
        return dict(sm_mhz=float(np.median(self.sm)) if self.sm else None, sm_max_mhz=self.max,
                    reasons=[n for n, b in self.BITS.items() if self.reasons & b], samples=len(self.sm),
                    span="sampled every 2 ms across warm-up + timed loop", power_w_max=max(self.power) if self.power else None)


def dist():
    ws = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    lr = int(os.environ.get("LOCAL_RANK", "0"))
    return ws, rank, lr


def whole_job_value(local_total_ms, rows_per_rank, steps, td=None, device=None):
    """Replicas-only multi-GPU accounting: every rank runs the same pipeline on its own copy of the
    workload; the job's time is the MAX over ranks and value = world_size * rows / that time. td = torch.distributed
    (initialised) or None for a single process. Returns (ms_per_step, rows_per_s)."""
    ws, total = 1, float(local_total_ms)
    if td is not None and td.is_initialized() and td.get_world_size() > 1:
        import torch
        ws = td.get_world_size()
        t = torch.tensor([total], dtype=torch.float64, device=device or "cpu")
        td.all_reduce(t, op=td.ReduceOp.MAX)
        total = float(t.item())
    ms_per_step = total / steps
    return ms_per_step, ws * rows_per_rank / ms_per_step * 1e3


def time_steps(torch, stream, fn, steps, warmup, barrier, min_load_ms=0.0):
    """W untimed calls of fn (plus, when min_load_ms is given, further untimed calls until the GPU has been under load
    that long, so that a clock sampler running beside the loop collects enough samples), then EXACTLY `steps` timed
    calls bracketed by CUDA events on the launching stream; returns the timed total in ms (this rank)."""
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        e0.record(stream)
        for _ in range(warmup):
            fn()
        e1.record(stream)
    torch.cuda.synchronize()
    if min_load_ms > 0:
        per = max(e0.elapsed_time(e1) / max(1, warmup), 1e-3)
        need = min_load_ms - steps * per
        for _ in range(int(min(200_000, max(0.0, need) / per))):
            fn()
    barrier()
    torch.cuda.synchronize()
    with torch.cuda.stream(stream):
        e0.record(stream)
        for _ in range(steps):
            fn()
        e1.record(stream)
    torch.cuda.synchronize()
    barrier()
    return e0.elapsed_time(e1)


def parse_configs(text, c5_scale):
    """'1,1x64,3' -> [(label, cfg, scale)]; 'NxS' = config N at S times its row count (supplementary steady-state rows)."""
    out = []
    for tok in [t for t in text.split(",") if t and t != "ops"]:
        if "x" in tok:
            c, sc = tok.split("x")
            out.append((f"C{c}x{sc}", int(c), float(sc)))
        else:
            out.append((f"C{tok}", int(tok), c5_scale if int(tok) == 5 else 1.0))
    return out


def load_digests():
    with open(os.path.join(ROOT, "tests", "golden", "fullsize_digests.json")) as f:
        return json.load(f)


def load_traffic():
    path = os.path.join(ROOT, "profiles", "traffic.json")   # dram bytes per launch from the committed ncu captures
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f)
    return {}


def result_columns(torch, res, nkeys):
    """Output columns of a pipeline as int64 numpy arrays sorted by the first key (group order is unspecified)."""
    cols = [k.to(torch.int64) for k in res["keys"]] + list(res["aggs"])
    if nkeys and res["n"] > 1:
        order = torch.argsort(cols[0])
        cols = [c[order] for c in cols]
    return [c.cpu().numpy() for c in cols]


def result_rows(torch, res):
    cols = [k.to(torch.int64).cpu().numpy() for k in res["keys"]] + [a.cpu().numpy() for a in res["aggs"]]
    return [[int(c[i]) for c in cols] for i in range(res["n"])]


def check_parity(torch, cfg, scale, plan, res, digests):
    """The timed configuration's output against the oracle: C1 (any scale the oracle finishes in seconds) by running
    the oracle on the same plan; C2-C5 at full size against the oracle-written digests of tests/golden/ (whole table;
    C3's timed plan is the top-10, compared row by row)."""
    import golden_util
    import oracle
    nkeys = len(plan.get("keys", []))
    if cfg == 1 and scale <= 4.0:
        exp = oracle.run_query(plan)
        got = result_columns(torch, res, nkeys)
        if nkeys > 1:
            order = np.lexsort(tuple(got[k] for k in reversed(range(nkeys))))
            got = [c[order] for c in got]
        return dict(ok=bool(res["n"] == exp.nrows and all(np.array_equal(g, e) for g, e in zip(got, exp.cols))),
                    how="oracle.run_query on the same plan, every output row")
    if scale != 1.0 or f"C{cfg}" not in digests:
        return dict(ok=None, how="no stored digest for this scale")
    d = digests[f"C{cfg}"]
    if plan.get("topk", 0):
        return dict(ok=bool(result_rows(torch, res) == d["top10"]), how="top-10 rows == oracle's (tests/golden/fullsize_digests.json)")
    got = result_columns(torch, res, nkeys)
    ok = res["n"] == d["ngroups"] and golden_util.digest_columns(got) == d["columns"]
    return dict(ok=bool(ok), how=f"whole table ({d['ngroups']} groups): per-column sum/xor/SHA-256 == oracle-written digests "
                                 "(tests/golden/fullsize_digests.json)")


def run_config(cfg, gq, ctx, torch, datagen, plans, gqrun, steps, warmup, scale=1.0, peak=6548.2, dense=True, hinted=True,
               detail=False, digests=None, traffic=None, dev=None):
    """Device-resident timing of one config: whole pipeline (builds + fused scan + finalise). detail=True adds the
    per-kernel device times of one profiled step, the dominant kernel's roofline, parity and clocks."""
    t0 = time.time()
    tabs = datagen.make_config(cfg, scale=scale)
    plan = plans.PLANS[cfg](tabs, topk=10) if cfg == 3 else plans.PLANS[cfg](tabs)
    gen_s = time.time() - t0
    nrows = len(plan["table"][0])
    l2 = float(dev["l2_bytes"]) if dev else 126e6
    ncopies = 1
    fact_bytes = sum(c.nbytes for c in plan["table"])
    if fact_bytes < 2 * l2:                  # C1: rotate copies so every timed rep reads cold HBM
        ncopies = int(np.ceil(3 * l2 / fact_bytes)) + 1
    sizing = "n/a"
    if plan.get("builds"):
        # Table sizing (DESIGN D2). "dense": the planner's column statistics (min/max of every build key) select
        # direct-address tables. "hinted": expected surviving build rows from the predicates' selectivities (uniform
        # columns: orderdate < 1200 of 2406 values, segment == 1 of 5 values), + 10 %. "upper bound": max_rows = input rows.
        sel = {3: [1200 / 2406], 4: [1 / 5, (1200 / 2406) * (1 / 5)]}[cfg]
        if dense:
            sizing = ("direct-address tables (GQ_F_DENSE_KEYS): key range from min/max statistics of the build keys, "
                      "rows from predicate selectivities + 10 %")
            for b, s in zip(plan["builds"], sel):
                k = b["table"][b["key"]]
                b["dense_range"] = (int(k.min()), int(k.max()))
                b["max_rows"] = int(len(k) * s * 1.1) + 1024
            plan["max_groups"] = plan["builds"][-1]["max_rows"]
        elif hinted:
            sizing = "hash tables sized from predicate selectivities + 10 %"
            for b, s in zip(plan["builds"], sel):
                b["max_rows"] = int(len(b["table"][0]) * s * 1.1) + 1024
            plan["max_groups"] = plan["builds"][-1]["max_rows"]
        else:
            sizing = "hash tables sized for every build input row (no selectivity knowledge)"
    if cfg == 5:
        plan["max_groups"] = int(datagen.ROWS[5]["keys"] * scale)
    build_cols = [gqrun.dev(b["table"]) for b in plan.get("builds", [])]
    fact = [gqrun.dev(plan["table"]) for _ in range(ncopies)]
    torch.cuda.synchronize()
    build_bytes = sum(c.nbytes for b in plan.get("builds", []) for c in b["table"])
    state = {"i": 0, "tables": None, "pipes": None}

    def make():
        state["tables"] = gqrun.build_tables(ctx, plan, device_tables=build_cols)
        state["ws"] = [t.workspace for t in state["tables"]]      # table workspaces are reused by every timed step
        state["pipes"] = [gqrun.prepare(ctx, plan, state["tables"], cols=f,
                                        out_capacity=(10 if cfg == 3 else plan["max_groups"])) for f in fact]
    make()

    def step():
        if plan.get("builds"):
            state["tables"] = gqrun.build_tables(ctx, plan, device_tables=build_cols, workspaces=state["ws"])   # re-init + rebuild: timed
            probes = [(state["tables"][bi], kc) for bi, kc in plan["probes"]]
            for p in state["pipes"]:
                pp, _ = p.m.probes(probes)
                p.plan.agg.probes = pp
        state["pipes"][state["i"] % ncopies].run()
        state["i"] += 1
    l0 = ctx.launch_count()
    step(); ctx.sync()
    launches_per_step = ctx.launch_count() - l0
    sampler = ClockSampler(dev["index"] if dev else 0).start() if detail else None
    ms = time_steps(torch, ctx.stream, step, steps, warmup, lambda: None, MIN_LOAD_MS if detail else 0.0) / steps
    clocks = sampler.stop() if sampler else None
    ctx.sync()
    alg = ALG_BYTES_PER_ROW[cfg] * nrows + build_bytes
    out = dict(rows=nrows, ms_per_step=ms, rows_per_s=nrows / ms * 1e3, alg_gb=alg / 1e9, gbs=alg / ms / 1e6,
               frac_of_measured=alg / ms / 1e6 / peak, frac_of_8000=alg / ms / 1e6 / 8000.0,
               launches_per_step=launches_per_step, scale=scale, cold_copies=ncopies, gen_s=round(gen_s, 2), table_sizing=sizing)
    if detail:
        out["clocks"] = clocks
        # one profiled step: every kernel (group) bracketed by CUDA events on the context's stream
        ctx.profile(True)
        step()
        kernels = ctx.profile_read()
        ctx.profile(False)
        out["kernels_ms"] = [[n, round(t, 5)] for n, t in kernels]
        scans = [(t, n) for n, t in kernels if n.startswith("gq_scan") or n == "gq_psa"]
        dom_ms, dom_name = max(scans) if scans else max((t, n) for n, t in kernels)
        how = "CUDA events around the launch (gq_profile), one step after the timed loop"
        if len(kernels) == 1:   # a one-launch step: the timed loop IS the kernel back to back (event brackets would add ~5 us)
            dom_ms, how = ms, "the step is this one launch: CUDA events around the timed loop / steps"
        tot_ms = max(sum(t for _, t in kernels), dom_ms)
        # algorithmic bytes of the dominant kernel's launch: the fact batch it streams (B/row x rows)
        dom_alg = ALG_BYTES_PER_ROW[cfg] * nrows
        tr = (traffic or {}).get(f"C{cfg}") if scale == 1.0 else None
        out["roofline"] = dict(bound="hbm", kernel=dom_name, kernel_ms=dom_ms, kernel_share_of_step=dom_ms / tot_ms,
                               algorithmic_bytes_per_launch=dom_alg, achieved=dom_alg / dom_ms / 1e6, peak=peak, unit="GB/s",
                               frac=dom_alg / dom_ms / 1e6 / peak, frac_of_nominal_8000=dom_alg / dom_ms / 1e6 / 8000.0,
                               traffic=tr, how=how)
        res = state["pipes"][(state["i"] - 1) % ncopies].result()
        out["parity_vs_oracle"] = check_parity(torch, cfg, scale, plan, res, digests or {})
    if cfg == 1:   # L2-warm figure, labelled as such
        def warm():
            state["pipes"][0].run()
        out["ms_l2_warm"] = time_steps(torch, ctx.stream, warm, steps, warmup, lambda: None) / steps
        if detail and ncopies > 1:
            # The 17 us step is a latency, not a bandwidth, figure: the same launches replayed from a CUDA graph (no host
            # enqueue cost between kernels), and the same kernel on two tiles = launch + set-up + merge tail alone.
            side = torch.cuda.Stream()
            with torch.cuda.stream(side):
                c2 = gq.Context(dev["index"] if dev else 0, stream=side)
                pipes2 = [gqrun.prepare(c2, plan, [], cols=f, out_capacity=plan["max_groups"]) for f in fact]
                small = gqrun.prepare(c2, plan, [], cols=[c[:2048] for c in fact[0]], out_capacity=plan["max_groups"])
                for p in pipes2 + [small]:
                    p.run()
                c2.sync()
                for name, seq in (("ms_cuda_graph_replay", pipes2), ("ms_fixed_cost_2048_rows_cuda_graph", [small] * len(pipes2))):
                    g = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(g, stream=side):
                        for p in seq:
                            p.run()
                    g.replay(); torch.cuda.synchronize()
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(side)
                    for _ in range(10):
                        g.replay()
                    e1.record(side)
                    torch.cuda.synchronize()
                    out[name] = e0.elapsed_time(e1) / (10 * len(seq))
                del pipes2, small, c2
    return out, plan, state


def run_standalone_ops(gq, ctx, torch, datagen, plans, gqrun, steps, warmup):
    """The standalone entry points on the C2 / C3 tables: gq_filter_project (ballot/popc compaction), gq_hash_partition,
    gq_order_by, gq_hash_build, gq_hash_probe (inner join materialised as output columns)."""
    out = {}
    t2 = datagen.make_config(2)
    p2 = plans.plan_c2(t2)
    cols = gqrun.dev(p2["table"])
    n = len(p2["table"][0])
    exprs = [[("col", 3), ("col", 1), ("mul",)], [("col", 0)]]
    cap = n // 20
    outs = [torch.empty(cap, dtype=torch.int64, device="cuda") for _ in exprs]
    count = torch.zeros(1, dtype=torch.int64, device="cuda")

    def fp():
        count.zero_()
        ctx.filter_project(cols, p2["preds"], exprs, capacity=cap, outs=outs, count=count)
    ms = time_steps(torch, ctx.stream, fp, steps, warmup, lambda: None) / steps
    ctx.sync()
    out["filter_project_c2"] = dict(rows=n, out_rows=int(count.item()), ms=ms, rows_per_s=n / ms * 1e3,
                                    gbs=(28 * n + 16 * int(count.item())) / ms / 1e6)
    del outs
    # gq_hash_partition (PartitionedOutput): the C2 table to 8 / 64 destinations by its int64 price
    # column (column 3: > 10^6 distinct values); algorithmic bytes = key column once (histogram) + every column read and written once (scatter)
    pouts = [torch.empty_like(c) for c in cols]
    for nparts in (8, 64):
        _, poff, _ = ctx.hash_partition(cols, [3], nparts, outs=pouts)
        pws = ctx._last_ws

        def part():
            ctx.hash_partition(cols, [3], nparts, workspace=pws, outs=pouts, offsets=poff)
        ms = time_steps(torch, ctx.stream, part, steps, warmup, lambda: None) / steps
        ctx.sync()
        sizes = (poff[1:] - poff[:-1]).cpu().tolist()
        out[f"hash_partition_c2_{nparts}"] = dict(rows=n, destinations=nparts, ms=ms, rows_per_s=n / ms * 1e3,
                                                  algorithmic_bytes=(8 + 2 * 28) * n, gbs=(8 + 2 * 28) * n / ms / 1e6,
                                                  rows_min=int(min(sizes)), rows_max=int(max(sizes)), rows_total=int(sum(sizes)))
    del pouts
    # gq_order_by (OrderBy / TopN) on the same table: full stable sort by the int64 price column (row
    # numbers only / all four columns gathered), by (date desc, price asc), and TopN 100 with the columns gathered
    for label, keys, limit, gather in (("order_by_c2_int64_index", [(3, False)], 0, False), ("order_by_c2_int64_gather", [(3, False)], 0, True),
                                       ("order_by_c2_date_desc_price", [(0, True), (3, False)], 0, False),
                                       ("top100_c2_int64_gather", [(3, True)], 100, True)):
        ctx.order_by(cols, keys, limit=limit, gather=gather)
        ows = ctx._last_ws
        l0 = ctx.launch_count()
        ctx.order_by(cols, keys, limit=limit, gather=gather, workspace=ows)
        nl = ctx.launch_count() - l0

        def sort():
            ctx.order_by(cols, keys, limit=limit, gather=gather, workspace=ows)
        ms = time_steps(torch, ctx.stream, sort, max(2, steps // 2), 2, lambda: None) / max(2, steps // 2)
        ctx.sync()
        out[label] = dict(rows=n, keys=[[c, "desc" if d else "asc"] for c, d in keys], limit=limit, gathered_columns=4 if gather else 0,
                          ms=ms, rows_per_s=n / ms * 1e3, launches=nl)
    # ORDER BY at the end of a query: a small group table (2048 rows, two keys, columns gathered) - one launch
    scols = [c[:2048].contiguous() for c in cols]
    ctx.order_by(scols, [(0, True), (3, False)], limit=0, gather=True)
    sws = ctx._last_ws

    def small_sort():
        ctx.order_by(scols, [(0, True), (3, False)], limit=0, gather=True, workspace=sws)
    ms = time_steps(torch, ctx.stream, small_sort, 50, 5, lambda: None) / 50
    ctx.sync()
    out["order_by_2048_rows_two_keys_gather"] = dict(rows=2048, ms=ms, rows_per_s=2048 / ms * 1e3, launches=1)
    del cols, scols
    torch.cuda.empty_cache()
    t3 = datagen.make_config(3)
    p3 = plans.plan_c3(t3)
    b = p3["builds"][0]
    bcols = gqrun.dev(b["table"])
    nb = len(b["table"][0])
    fcols = gqrun.dev(p3["table"])
    nf = len(p3["table"][0])
    pexprs = [[("col", 0)], p3["exprs"][0]]
    pcap = nf // 3
    pouts = [torch.empty(pcap, dtype=torch.int64, device="cuda") for _ in pexprs]
    for label, kw in (("hashed", dict(max_rows=int(nb * 1200 / 2406 * 1.1) + 1024)),
                      ("dense", dict(dense_range=(int(b["table"][0].min()), int(b["table"][0].max())), max_rows=int(nb * 1200 / 2406 * 1.1) + 1024))):
        tb = ctx.hash_build(bcols, preds=b["preds"], key=0, unique=True, **kw)
        ws = tb.workspace

        def build():
            return ctx.hash_build(bcols, preds=b["preds"], key=0, unique=True, workspace=ws, **kw)
        ms = time_steps(torch, ctx.stream, build, steps, warmup, lambda: None) / steps
        out[f"hash_build_c3_dim_{label}"] = dict(rows=nb, ms=ms, rows_per_s=nb / ms * 1e3, gbs=12 * nb / ms / 1e6,
                                                 note="table init + scan + inserts (7.48 M of 15 M rows pass the filter)")
        tb = build()

        def probe():
            count.zero_()
            ctx.hash_probe(fcols, p3["preds"], [(tb, 0)], pexprs, capacity=pcap, outs=pouts, count=count)
        ms = time_steps(torch, ctx.stream, probe, steps, warmup, lambda: None) / steps
        ctx.sync()
        out[f"hash_probe_c3_fact_{label}"] = dict(rows=nf, out_rows=int(count.item()), ms=ms, rows_per_s=nf / ms * 1e3,
                                                  gbs=(28 * nf + 16 * int(count.item())) / ms / 1e6)
    return out


# ---------------------------------------------------------------------------------------------- CPU baselines
def oracle_rate(plans, datagen, cfg, sample_rows, reps=1):
    """The oracle as it stands, single thread, on a bounded sample of the workload (rows/s)."""
    import oracle
    scale = sample_rows / datagen.ROWS[cfg]["fact"]
    plan = plans.PLANS[cfg](datagen.make_config(cfg, scale=scale))
    n = len(plan["table"][0])
    best = None
    for _ in range(reps):
        t0 = time.perf_counter()
        oracle.run_query(plan)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return n / best, n, best


def oracle_rate_threads(plans, datagen, nthreads):
    """The same oracle sharded over the host cores: C2's 60 M rows cut into `nthreads` row ranges, one oracle call per
    range on its own thread (the C call releases the GIL), the partial (SUM, COUNT) rows added — Partial -> Final of a
    key-less aggregation. Its result must equal the single-thread oracle's before its time is reported."""
    import oracle
    from concurrent.futures import ThreadPoolExecutor
    plan = plans.PLANS[2](datagen.make_config(2))
    n = len(plan["table"][0])
    whole = oracle.run_query(plan)
    cuts = [n * i // nthreads for i in range(nthreads + 1)]
    parts = [dict(plan, table=[np.ascontiguousarray(c[a:b]) for c in plan["table"]]) for a, b in zip(cuts, cuts[1:])]
    best, res = None, None
    with ThreadPoolExecutor(nthreads) as ex:
        for _ in range(3):
            t0 = time.perf_counter()
            rs = list(ex.map(oracle.run_query, parts))
            dt = time.perf_counter() - t0
            if best is None or dt < best:
                best, res = dt, rs
    tot = [int(np.sum(np.array([int(r.cols[c][0]) for r in res], dtype=np.int64))) for c in range(len(whole.cols))]
    equal = all(tot[c] == int(whole.cols[c][0]) for c in range(len(whole.cols)))
    return n / best, best, equal


def main_reference(args):
    """--impl reference: the CPU oracle (this tier's reference arm) on the box's host cores, rank 0 only. Same config
    as the repo's arm (C2, 60 M rows); each step runs the oracle over a bounded sample of those rows sized so that the
    whole --steps K run ends within a few minutes (all 60 M rows when K is small enough)."""
    ws, rank, _ = dist()
    if rank != 0:
        return
    import oracle
    import plans
    from paper_2606_24647_b200 import datagen
    full = datagen.ROWS[2]["fact"]
    plan = plans.PLANS[2](datagen.make_config(2))
    calib = dict(plan, table=[np.ascontiguousarray(c[:2_000_000]) for c in plan["table"]])
    t0 = time.perf_counter()
    oracle.run_query(calib)
    rate0 = 2_000_000 / (time.perf_counter() - t0)
    sample = int(min(full, max(1_000_000, rate0 * 150.0 / max(1, args.steps + args.warmup))))
    sub = plan if sample == full else dict(plan, table=[np.ascontiguousarray(c[:sample]) for c in plan["table"]])
    for _ in range(args.warmup):
        oracle.run_query(sub)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.run_query(sub)
    total = time.perf_counter() - t0
    rate = sample * args.steps / total
    what = f"first {sample} of the 60000000 rows of the seeded C2 table per step" if sample < full else "all 60000000 rows per step"
    line = dict(impl="reference", metric=METRIC, value=rate, unit="rows/s", n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=total / args.steps * 1e3, higher_is_better=True, scaling="weak",
                vs_baseline=None, dtype="int64", data="synthetic",
                config=dict(workload=WORKLOAD, rows=full, l2=L2_NOTE),
                cpu_baseline=dict(value=rate, unit="rows/s", cores=1, kind="oracle", sample=what),
                e2e=dict(value=rate, unit="rows/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0,
                host=host_info())
    print(json.dumps(line))


def main():
    global MIN_LOAD_MS
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=400)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--configs", default="1,1x64,3,4,5,ops", help="extra configs reported under per_config ('' = none); "
                    "ops = the standalone materialising entry points (filter_project, hash_build, hash_probe); "
                    "NxS = config N at S times its rows (C1x64: the low-cardinality pipeline at steady state)")
    ap.add_argument("--c5-scale", type=float, default=1.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--min-load-ms", type=float, default=MIN_LOAD_MS, help="untimed warm-up is extended until the GPU has been "
                    "under load this long (clock samples); 0 keeps launch lists under ncu short")
    ap.add_argument("--only-configs", action="store_true", help="skip the C2 headline: print only the --configs records "
                    "(the ncu captures under profiles/ name this command)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    MIN_LOAD_MS = args.min_load_ms
    if args.impl == "reference":
        return main_reference(args)

    import torch
    import gqrun
    import plans
    from paper_2606_24647_b200 import build as gqbuild, datagen
    ws, rank, lr = dist()
    if ws > 1:
        import torch.distributed as td
        torch.cuda.set_device(lr)
        td.init_process_group("nccl", device_id=torch.device("cuda", lr))
        flag = torch.zeros(1, device="cuda")

        def barrier():
            td.all_reduce(flag)
            torch.cuda.synchronize()
    else:
        def barrier():
            pass
    if rank == 0:
        gqbuild.build()
    barrier()
    from paper_2606_24647_b200 import gq
    dev_index = lr if ws > 1 else 0
    ctx = gq.Context(dev_index)
    peak, peak_src = peaks()
    props = torch.cuda.get_device_properties(dev_index)
    dev = dict(index=dev_index, name=props.name, sms=int(props.multi_processor_count), l2_bytes=int(props.L2_cache_size),
               mem_bytes=int(props.total_memory))
    digests, traffic = load_digests(), load_traffic()
    cfg_steps = max(5, min(20, args.steps))

    def extra_configs():
        per_config = {}
        for label, cfg, sc in parse_configs(args.configs, args.c5_scale):
            try:
                out, _, _ = run_config(cfg, gq, ctx, torch, datagen, plans, gqrun, cfg_steps, 3, scale=sc, peak=peak, detail=True,
                                       digests=digests, traffic=traffic, dev=dev)
                per_config[label] = out
                torch.cuda.empty_cache()
                if cfg in (3, 4) and sc == 1.0:   # the same pipeline on hash tables: sized from selectivities, and for every input row
                    alt = {}
                    for name, kw in (("hashed_hinted", dict(dense=False, hinted=True)), ("hashed_upper_bound", dict(dense=False, hinted=False))):
                        o2, _, _ = run_config(cfg, gq, ctx, torch, datagen, plans, gqrun, 5, 3, scale=sc, peak=peak, dev=dev, **kw)
                        alt[name] = dict(ms_per_step=o2["ms_per_step"], table_sizing=o2["table_sizing"], launches_per_step=o2["launches_per_step"])
                        torch.cuda.empty_cache()
                    out["other_table_sizings"] = alt
            except Exception as e:  # a failing extra config must not hide the headline number
                per_config[label] = dict(error=str(e)[:300])
            torch.cuda.empty_cache()
        if "ops" in args.configs.split(","):
            try:
                per_config["standalone_ops"] = run_standalone_ops(gq, ctx, torch, datagen, plans, gqrun, 10, 3)
            except Exception as e:
                per_config["standalone_ops"] = dict(error=str(e)[:300])
            torch.cuda.empty_cache()
        return per_config

    if args.only_configs:
        print(json.dumps(dict(per_config=extra_configs(), device=dev)))
        return

    # ---------------- headline: C2, device-resident ----------------
    tabs = datagen.make_config(2)
    plan = plans.plan_c2(tabs)
    nrows = len(plan["table"][0])
    cols = gqrun.dev(plan["table"], device=f"cuda:{dev_index}")
    pipe = gqrun.prepare(ctx, plan, [], cols=cols)
    l0 = ctx.launch_count()
    pipe.run(); ctx.sync()
    launches_per_step = ctx.launch_count() - l0
    parity = check_parity(torch, 2, 1.0, plan, pipe.result(), digests) if rank == 0 else None
    sampler = ClockSampler(dev_index).start()
    total_ms = time_steps(torch, ctx.stream, pipe.run, args.steps, args.warmup, barrier, MIN_LOAD_MS)
    clocks = sampler.stop()
    # dominant kernel alone: further batches into an existing aggregation state launch only the fused scan kernel
    st = ctx.aggregate(None, cols, preds=plan["preds"], exprs=plan["exprs"], keys=[], aggs=plan["aggs"], max_groups=1)
    scan = lambda: ctx.aggregate(st, cols, preds=plan["preds"], exprs=plan["exprs"], keys=[], aggs=plan["aggs"], max_groups=1)
    scan_ms = time_steps(torch, ctx.stream, scan, args.steps, args.warmup, lambda: None) / args.steps
    # read-only roofline probe of this box (same bytes)
    probe_t = torch.empty(1 << 30, dtype=torch.uint8, device=f"cuda:{dev_index}")
    probe_ms = time_steps(torch, ctx.stream, lambda: ctx.read_probe(probe_t), 10, 3, lambda: None) / 10
    ms_per_step, value = whole_job_value(total_ms, nrows, args.steps, td if ws > 1 else None, "cuda")
    alg_bytes = ALG_BYTES_PER_ROW[2] * nrows + 16
    achieved = alg_bytes / scan_ms / 1e6
    roofline = dict(bound="hbm", kernel="gq_scan:global (C2 fused filter+project+global aggregate; the step's only launch)",
                    achieved=achieved, peak=peak, unit="GB/s", frac=achieved / peak, traffic=traffic.get("C2"), peak_source=peak_src,
                    algorithmic_bytes_per_launch=alg_bytes, kernel_ms=scan_ms, frac_of_nominal_8000=achieved / 8000.0,
                    read_probe_gbs=(1 << 30) / probe_ms / 1e6,
                    traffic_source="dram__bytes_read.sum + dram__bytes_write.sum of this kernel, committed ncu capture (profiles/traffic.json)")

    # ---------------- end to end: HOST buffers through the C ABI ----------------
    e2e = None
    if rank == 0 or ws > 1:
        hcols = [torch.from_numpy(np.ascontiguousarray(c)).pin_memory() for c in plan["table"]]
        hp = gqrun.prepare(ctx, plan, [], cols=hcols)
        hp.run_host(); hp.run_host()
        k = max(3, min(args.steps, 5))
        t0 = time.perf_counter()
        for _ in range(k):
            hp.run_host()
        e2e_ms = (time.perf_counter() - t0) / k * 1e3     # run_host returns after the results landed on the host
        if parity is not None and parity["ok"]:
            parity["ok"] = bool(result_rows(torch, hp.result()) == result_rows(torch, pipe.result()))   # e2e path: same row
        e2e = dict(value=ws * nrows / e2e_ms * 1e3, unit="rows/s", h2d_bytes_per_step=int(sum(c.nbytes for c in plan["table"])),
                   d2h_bytes_per_step=8 * (1 + len(plan["aggs"])), ms_per_step=e2e_ms,
                   how="gq_pipeline_host: pinned host columns, 8 Mi-row chunks, H2D overlapped with the scan")
        del hcols, hp

    # ---------------- other configs (device-resident), rank 0 of a 1-GPU run only ----------------
    per_config = {}
    if ws == 1 and args.configs:
        del cols, pipe, st, probe_t
        torch.cuda.empty_cache()
        per_config = extra_configs()
        # end to end for a join pipeline too: C3 with its build side device-resident, the 60 M-row fact table on the host
        if "C3" in per_config:
            try:
                t3 = datagen.make_config(3)
                p3 = plans.plan_c3(t3, topk=10)
                for b in p3["builds"]:
                    kk = b["table"][b["key"]]
                    b["dense_range"] = (int(kk.min()), int(kk.max()))
                    b["max_rows"] = int(len(kk) * (1200 / 2406) * 1.1) + 1024
                tables = gqrun.build_tables(ctx, p3)
                h3 = [torch.from_numpy(np.ascontiguousarray(c)).pin_memory() for c in p3["table"]]
                hp3 = gqrun.prepare(ctx, p3, tables, cols=h3, out_capacity=10)
                hp3.run_host(); hp3.run_host()
                t0 = time.perf_counter()
                for _ in range(3):
                    hp3.run_host()
                ms3 = (time.perf_counter() - t0) / 3 * 1e3
                per_config["C3"]["e2e"] = dict(
                    value=len(p3["table"][0]) / ms3 * 1e3, unit="rows/s", ms_per_step=ms3,
                    h2d_bytes_per_step=int(sum(c.nbytes for c in p3["table"])), d2h_bytes_per_step=8 + 10 * 8 * 3,
                    parity_vs_oracle=bool(result_rows(torch, hp3.result()) == digests["C3"]["top10"]),
                    how="gq_pipeline_host: fact columns in pinned host memory, build-side table device-resident")
                del h3, hp3, tables
                torch.cuda.empty_cache()
            except Exception as e:
                per_config["C3"]["e2e"] = dict(error=str(e)[:300])

        # ... and for the high-cardinality group-by: C5's 16.8 GB of columns in pinned host memory (the host path
        # streams 8 Mi-row chunks into the global-table aggregation; the partitioned path needs the whole batch in HBM)
        if "C5" in per_config and per_config["C5"].get("scale", 1.0) == 1.0:
            try:
                p5 = plans.plan_c5(datagen.make_config(5))
                h5 = [torch.from_numpy(np.ascontiguousarray(c)).pin_memory() for c in p5["table"]]
                hp5 = gqrun.prepare(ctx, p5, [], cols=h5)
                hp5.run_host()
                t0 = time.perf_counter()
                hp5.run_host()
                ms5 = (time.perf_counter() - t0) * 1e3
                r5 = hp5.result()
                per_config["C5"]["e2e"] = dict(
                    value=len(p5["table"][0]) / ms5 * 1e3, unit="rows/s", ms_per_step=ms5,
                    h2d_bytes_per_step=int(sum(c.nbytes for c in p5["table"])),
                    d2h_bytes_per_step=8 + int(r5["n"]) * 8 * (len(p5["keys"]) + len(p5["aggs"])),
                    parity_vs_oracle=check_parity(torch, 5, 1.0, p5, r5, digests)["ok"],
                    how="gq_pipeline_host: all columns in pinned host memory, 8 Mi-row chunks into the global-table "
                        "aggregation, the whole result table copied back to host buffers")
                del h5, hp5, r5
                torch.cuda.empty_cache()
            except Exception as e:
                per_config["C5"]["e2e"] = dict(error=str(e)[:300])

    # ---------------- CPU baselines: the oracle on this box's host cores ----------------
    cpu, cpu_threads, host = None, None, host_info()
    if rank == 0 and not args.no_cpu_baseline:
        rate, n, dt = oracle_rate(plans, datagen, 2, 60_000_000, reps=3)
        cpu = dict(value=rate, unit="rows/s", cores=1, kind="oracle", sample=f"all {n} rows of C2, best of 3 ({dt:.2f} s each)",
                   host_cores=os.cpu_count())
        nt = os.cpu_count() or 1
        trate, tdt, equal = oracle_rate_threads(plans, datagen, nt)
        cpu_threads = dict(value=trate if equal else None, unit="rows/s", cores=nt,
                           kind="oracle sharded over row ranges, one thread each; partial rows added",
                           sample=f"all {n} rows of C2, best of 3 ({tdt:.2f} s each)", equals_single_thread_oracle=bool(equal))
    if rank == 0:
        line = dict(metric=METRIC, value=value, unit="rows/s", n_gpus=ws, steps=args.steps, warmup=args.warmup,
                    ms_per_step=ms_per_step, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="int64",
                    data="synthetic", config=dict(workload=WORKLOAD, rows=nrows, l2=L2_NOTE),
                    parallelism="replicas only" if ws > 1 else "1 GPU", parity_vs_oracle=parity,
                    roofline=roofline, cpu_baseline=cpu, cpu_baseline_threads=cpu_threads, host=host, device=dev, e2e=e2e,
                    gpu_launches=launches_per_step * args.steps, launches_per_step=launches_per_step, clocks=clocks,
                    per_config=per_config)
        print(json.dumps(line))
    if ws > 1:
        td.destroy_process_group()


if __name__ == "__main__":
    main()
