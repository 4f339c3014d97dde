#!/usr/bin/env python
"""bench.py — QPS of exact batched sparse top-k search on the seeded synthetic stand-in for BASELINE.json's
paper-scale config (8.8M docs, batch 500, top-1000, fp32), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config paper] [--docs N] [--queries B] [--k K] [--algo auto|term|doc]

A "step" is one gs_search call (S1 ingest -> S2 scoring -> S3 top-k -> S4 output) over one batch
of B queries.  `value` is measured with queries/outputs resident in HBM (CUDA events on the launching
stream, barrier + synchronize on both sides, max over ranks); `e2e` goes through gs_search_host with pinned
HOST buffers (H2D + D2H inside the timed region).  Inputs (index 8.45 GB per layout) are far larger than
the 126 MB L2, so no explicit flush is needed between iterations (stated in config.l2).
The forward and inverted index are built once before the timed region (the paper does not time the build
either).

--gpus N > 1 (torchrun): the path does not shard (BASELINE.json north_star: one GPU, no collectives), so
every rank is an independent replica with its own index and its own query batch ("replicas only",
DESIGN.md §8); value = all ranks' queries / max-over-ranks time.

--impl reference: times the CPU oracle (oracle/) as it stands on the host cores, on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "QPS @8.8M docs batch 500 top-1000"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="paper")
    ap.add_argument("--docs", type=int, default=None, help="use the first N docs of the collection (debug)")
    ap.add_argument("--queries", type=int, default=None)
    ap.add_argument("--k", type=int, default=None)
    ap.add_argument("--algo", default="auto", choices=["auto", "term", "doc"])
    ap.add_argument("--also", default="term,doc", help="extra algos timed after the main one ('' = none)")
    ap.add_argument("--doc-query-tile", type=int, default=0)
    ap.add_argument("--query-group", type=int, default=0)
    ap.add_argument("--sample-shift", type=int, default=0, help="threshold sample = 1/2^shift of the doc tiles (0 = auto)")
    ap.add_argument("--tile-docs", type=int, default=0)
    ap.add_argument("--head-max", type=int, default=0, help="dense strips kept by the index (0 = default 64, -1 = none)")
    ap.add_argument("--head-density", type=float, default=0.0, help="list density from which a strip is kept (0 = default)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cpu-sample-queries", type=int, default=0, help="oracle sample size (0 = one per core)")
    ap.add_argument("--latency-queries", type=int, default=200, help="single-query searches timed for the batch-1 latency leg (0 = skip)")
    ap.add_argument("--no-suite", action="store_true", help="skip the other BASELINE.json configs (1, 2, 4, 5: QPS, p50/p99, roofline) in the line's `suite` key")
    ap.add_argument("--sweeps", action="store_true", help="also run the batch-size sweep and the sparsity sweep (PAPER.md Tables 3 / 5 analogues)")
    return ap.parse_args()


# ---------------------------------------------------------------------------------------------------------
# clocks: sample nvidia-smi DURING the timed region
# ---------------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.samples, self._stop, self._t = index, [], threading.Event(), None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.samples.append([x.strip() for x in out.splitlines()[0].split(",")])
            except Exception:
                pass
            self._stop.wait(0.05)

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=10)

    def summary(self) -> dict:
        sm, mx, reasons, pw = [], [], set(), []
        for s in self.samples:
            try:
                sm.append(float(s[0])); mx.append(float(s[1])); pw.append(float(s[2]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), s[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "reasons": sorted(reasons), "samples": len(sm)}


def measured_peaks() -> dict:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": float(d["hbm_gbs"]), "source": "measured (MEASURED_PEAKS.json)",
                "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0))}
    return {"hbm_gbs": 6650.0, "source": "fallback (B200_PROFILING.md)", "sm_max_mhz": 1965.0}


def workload_for(args, rank: int):
    from paper_2606_26441_b200 import workload as wl
    c = wl.CONFIGS[args.config]
    n_docs = args.docs or c["N"]
    B = args.queries or c["B"]
    k = args.k or c["k"]
    return wl, c, n_docs, B, k


# ---------------------------------------------------------------------------------------------------------
# the oracle timed on the host cores (cpu_baseline leg and --impl reference)
# ---------------------------------------------------------------------------------------------------------
def time_oracle(docs, queries, vocab, k, n_sample: int, steps: int = 1, warmup: int = 0, R_d=None):
    import oracle
    cores = oracle.max_threads()
    n = n_sample or cores
    n = max(1, min(n, queries.rows))
    t0 = time.perf_counter()
    if R_d is None:
        R_d = oracle.as_rows(docs, vocab)
    t_rows = time.perf_counter() - t0
    R_q = oracle.as_rows(queries.slice_rows(0, n), vocab)
    times = []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        oracle.search(R_q, R_d, k, nthreads=0)
        if it >= warmup:
            times.append(time.perf_counter() - t0)
    dt = float(np.mean(times))
    return {"value": n / dt, "unit": "queries/s", "cores": min(cores, n), "kind": "oracle",
            "sample": f"first {n} of {queries.rows} queries against all {docs.rows} docs, exhaustive merge scoring + full sort "
                      f"(oracle.search, OpenMP over queries); {dt:.2f} s per pass; doc canonicalisation {t_rows:.1f} s not counted",
            "ms_per_query": 1e3 * dt / n * min(cores, n), "seconds_per_pass": dt}, R_d


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl, c, n_docs, B, k = workload_for(args, 0)
    docs = wl.make_docs(args.config, n_docs=n_docs)
    queries = wl.make_queries(args.config, n_queries=B)
    base, _ = time_oracle(docs, queries, wl.VOCAB, k, args.cpu_sample_queries, steps=max(1, args.steps), warmup=min(args.warmup, 1))
    dt = base["seconds_per_pass"]
    line = {"impl": "reference", "metric": METRIC, "value": base["value"], "unit": "queries/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64" if c["wtype"] == "f32" else "int64", "data": "synthetic",
            "config": config_dict(args, c, n_docs, B, k, "oracle"),
            "cpu_baseline": {k_: base[k_] for k_ in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": base["value"], "unit": "queries/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


BJ_INDEX = {"tiny": 0, "mid": 1, "paper": 2, "paper_u8": 3, "skew_b1": 4, "skew_b32": 4}


def workload_label(name, c, n_docs, B, k):
    qlaw = "nnz~U{5..256}" if c["qlaw"]["nnz_law"] == 1 else "nnz~N(25,8) clip [5,64]"
    return (f"BASELINE.json configs[{BJ_INDEX.get(name, '?')}] '{name}': V=30522, N={n_docs} docs (nnz~N(120,40) clip [20,400], "
            f"Zipf s={c['s']}, LogNormal(0,0.5) {c['wtype']} weights), B={B} queries ({qlaw}, Zipf s={c['s']}), top-k={k}, seed 0")


def config_dict(args, c, n_docs, B, k, algo):
    return {"workload": workload_label(args.config, c, n_docs, B, k),
            "num_docs": n_docs, "batch": B, "k": k, "vocab": 30522, "wtype": c["wtype"], "algo": algo,
            "l2": "index arrays (GBs) exceed the 126 MB L2; no explicit flush between iterations",
            "parallelism": "replicas only (no sharding, no collectives)"}


# ---------------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------------
def timed_steps(torch, dist, fn, steps, warmup, world):
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    s = torch.cuda.current_stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(s)
    for _ in range(steps):
        fn()
    e1.record(s)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    from paper_2606_26441_b200 import replicas
    return replicas.max_over_ranks(e0.elapsed_time(e1), dist if world > 1 else None, "cuda")


def latency_leg(torch, ix, queries, k, n, algo, batch=1, **opt):
    """Per-call latency of gs_search for `n` distinct batches of `batch` queries (device-resident CSR slices),
    CUDA events around each call plus a stream synchronise per call (SURVEY §8d timing protocol)."""
    dev = ix.device
    n = max(1, min(n, queries.rows // batch))
    slices = []
    for i in range(n):
        q = queries.slice_rows(i * batch, (i + 1) * batch)
        slices.append(([torch.from_numpy(a).to(dev) for a in (q.indptr, q.terms, q.weights)], q.nnz))
    max_nnz = max(z for _, z in slices)
    ws = torch.empty(ix.workspace_bytes(batch, max_nnz, k, algo=algo, **opt), dtype=torch.uint8, device=dev)
    sdt = torch.float32 if queries.weights.dtype == np.float32 else torch.int32
    out_ids = torch.empty((batch, k), dtype=torch.int32, device=dev)
    out_sc = torch.empty((batch, k), dtype=sdt, device=dev)
    s = torch.cuda.current_stream()
    for (q, _) in slices[:3]:
        ix.search(*q, k, out_ids=out_ids, out_scores=out_sc, workspace=ws, algo=algo, **opt)
    torch.cuda.synchronize()
    ms = []
    for (q, _) in slices:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(s)
        ix.search(*q, k, out_ids=out_ids, out_scores=out_sc, workspace=ws, algo=algo, **opt)
        e1.record(s)
        e1.synchronize()
        ms.append(e0.elapsed_time(e1))
    st = ix.stats(ws)
    ms = np.array(ms)
    out = {"batch": batch, "calls": int(n), "algo": algo, "algo_used": {1: "term", 2: "doc"}.get(st["algo_used"], "?"),
           "p50_ms": float(np.percentile(ms, 50)), "p99_ms": float(np.percentile(ms, 99)), "mean_ms": float(ms.mean()),
           "p50_ms_per_query": float(np.percentile(ms, 50)) / batch,
           "protocol": "per call: CUDA event, gs_search + gs_search_finish (stream sync + 64 B read-back), CUDA event"}
    # the same search captured ONCE into a CUDA graph (gs_search is asynchronous) and replayed for every query: the new
    # query is copied into the captured buffers before the first event, so the timed region is the graph replay alone
    if st["algo_used"] == 1 and batch <= 32:
        try:
            cap = max_nnz
            g_ip = torch.zeros(batch + 1, dtype=torch.int64, device=dev)
            g_t = torch.zeros(max(cap, 1), dtype=torch.int32, device=dev)
            g_w = torch.zeros(max(cap, 1), dtype=slices[0][0][2].dtype, device=dev)

            def put(q):
                g_ip.copy_(q[0]); g_t[:q[1].numel()].copy_(q[1]); g_w[:q[2].numel()].copy_(q[2])

            put(slices[0][0])
            side = torch.cuda.Stream()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                ix.search(g_ip, g_t, g_w, k, out_ids=out_ids, out_scores=out_sc, workspace=ws, algo=algo, finish=False, **opt)
            torch.cuda.current_stream().wait_stream(side)
            torch.cuda.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph):
                ix.search(g_ip, g_t, g_w, k, out_ids=out_ids, out_scores=out_sc, workspace=ws, algo=algo, finish=False, **opt)
            gms, n_ov = [], 0
            for (q, _) in slices:
                put(q)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(s)
                graph.replay()
                e1.record(s)
                e1.synchronize()
                gms.append(e0.elapsed_time(e1))
                n_ov += ix.stats(ws)["overflow_queries"]
            gms = np.array(gms)
            out.update({"graph_p50_ms": float(np.percentile(gms, 50)), "graph_p99_ms": float(np.percentile(gms, 99)),
                        "graph_overflow_queries": int(n_ov)})
            del graph
        except Exception as e:                                   # report, never hide
            out["graph_error"] = repr(e)[:200]
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device: there is no CPU fallback for the hot path"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    from paper_2606_26441_b200 import binding as gs
    from paper_2606_26441_b200 import build as gsbuild
    if rank == 0 and not os.path.exists(gs.LIB_PATH):
        gsbuild.build_all()
    if world > 1:
        dist.barrier()
    gs.lib()
    wl, c, n_docs, B, k = workload_for(args, rank)
    dev = torch.device(f"cuda:{local}")
    peaks = measured_peaks()

    t0 = time.perf_counter()
    docs = wl.make_docs(args.config, n_docs=n_docs)                  # every replica indexes the same collection
    from paper_2606_26441_b200 import replicas
    queries = wl.make_queries(args.config, n_queries=B, row0=replicas.query_rows(rank, B)[0])   # ... and searches its own batch
    t_gen = time.perf_counter() - t0
    t0 = time.perf_counter()
    ix = gs.Index.from_numpy(docs, wl.VOCAB, device=dev, tile_docs=args.tile_docs, head_max=args.head_max,
                             head_density=args.head_density)
    torch.cuda.synchronize()
    t_build = time.perf_counter() - t0
    info = ix.info()
    lens = ix.meta()[1].astype(np.int64)
    head_terms = ix.head_terms()
    q_dev = [torch.from_numpy(a).to(dev) for a in (queries.indptr, queries.terms, queries.weights)]
    sdt = torch.float32 if c["wtype"] == "f32" else torch.int32
    out_ids = torch.empty((B, k), dtype=torch.int32, device=dev)
    out_sc = torch.empty((B, k), dtype=sdt, device=dev)
    opt_common = dict(doc_query_tile=args.doc_query_tile, query_group=args.query_group, sample_shift=args.sample_shift)

    def measure(algo):
        ws_bytes = ix.workspace_bytes(B, queries.nnz, k, algo=algo, **opt_common)
        ws = torch.empty(ws_bytes, dtype=torch.uint8, device=dev)

        def step():      # asynchronous gs_search; the overflow count of the (identical) steps is read after the timed region
            ix.search(*q_dev, k, out_ids=out_ids, out_scores=out_sc, workspace=ws, algo=algo, finish=False, **opt_common)

        with ClockSampler(local) as cs:
            ms = timed_steps(torch, dist, step, args.steps, args.warmup, world)
        launches = gs.last_launch_count()
        st = ix.stats(ws)
        # per-kernel device time, measured live with CUDA events on the launching stream (same K steps again)
        gs.profile_enable(True)
        torch.cuda.synchronize()
        for _ in range(args.steps):
            step()
        torch.cuda.synchronize()
        prof = gs.profile_read()
        gs.profile_enable(False)
        res = {"algo": algo, "algo_used": {1: "term", 2: "doc"}.get(st["algo_used"], "?"), "ms_per_step": ms / args.steps,
               "qps": replicas.aggregate_qps(world, B, args.steps, ms), "ms_per_query": ms / args.steps / B,
               "launches_per_step": launches, "candidates_per_query": st["candidates"] / max(B, 1),
               "overflow_queries": st["overflow_queries"], "workspace_bytes": ws_bytes, "clocks": cs.summary(),
               "kernels": {n: {"launches_per_step": v["launches"] / args.steps, "ms_per_step": v["ms"] / args.steps}
                           for n, v in prof.items()}}
        res["roofline"] = roofline(res, st, info, lens, head_terms, queries, B, k, peaks, c["wtype"])
        del ws
        return res

    main = measure(args.algo)
    others = {}
    for a in [x for x in args.also.split(",") if x]:
        if a != args.algo and a != main["algo_used"]:
            others[a] = measure(a)
        elif a == main["algo_used"] and a != args.algo:
            others[a] = "same as the main line (auto dispatch chose it)"

    # ---- e2e: HOST buffers through gs_search_host (pinned), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        pin = [torch.from_numpy(a).pin_memory() for a in (queries.indptr, queries.terms, queries.weights)]
        h_ids = torch.empty((B, k), dtype=torch.int32).pin_memory()
        h_sc = torch.empty((B, k), dtype=sdt).pin_memory()
        pn = [t.numpy() for t in pin]

        def step_host():
            ix.search_host(pn[0], pn[1], pn[2], k, out_ids=h_ids.numpy(), out_scores=h_sc.numpy(), algo=args.algo, **opt_common)

        for _ in range(args.warmup):
            step_host()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            step_host()          # synchronous: returns after the D2H copy of the results
        dt = time.perf_counter() - t0
        dt = replicas.max_over_ranks(dt, dist if world > 1 else None, "cuda")
        e2e = {"value": replicas.aggregate_qps(world, B, args.steps, 1e3 * dt), "unit": "queries/s", "ms_per_step": 1e3 * dt / args.steps,
               "h2d_bytes_per_step": int(sum(a.nbytes for a in pn)), "d2h_bytes_per_step": int(h_ids.numel() * 4 + h_sc.numel() * 4),
               "api": "gs_search_host (pinned host buffers; H2D + search + D2H + stream sync per step, host wall clock)"}

    # ---- batch-1 latency (BASELINE.json metric: "batch-1 p50 ms/query"), both kernels, on the same index
    latency = None
    if world == 1 and args.latency_queries > 0:
        latency = {a: latency_leg(torch, ix, queries, k, args.latency_queries, a, **opt_common) for a in ("term", "doc")}

    # ---- batch-size sweep on the same index (Table 3 L262-271 analogue), with --suite
    sweep = None
    if world == 1 and args.sweeps:
        sweep = []
        for Bs in (1, 2, 4, 8, 16, 32, 64, 128, 256, B):
            if Bs > B:
                continue
            qb_ = queries.slice_rows(0, Bs)
            qd_ = [torch.from_numpy(a).to(dev) for a in (qb_.indptr, qb_.terms, qb_.weights)]
            row = {"batch": Bs}
            for a in ("term", "doc"):
                ws_ = torch.empty(ix.workspace_bytes(Bs, qb_.nnz, k, algo=a), dtype=torch.uint8, device=dev)
                oi = torch.empty((Bs, k), dtype=torch.int32, device=dev)
                osc = torch.empty((Bs, k), dtype=sdt, device=dev)
                ms_ = timed_steps(torch, None, lambda: ix.search(*qd_, k, out_ids=oi, out_scores=osc, workspace=ws_, algo=a), 5, 3, 1)
                row[a] = {"ms_per_batch": ms_ / 5, "qps": Bs * 5 / (ms_ * 1e-3)}
                del ws_
            sweep.append(row)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        full, _ = time_oracle(docs, queries, wl.VOCAB, k, args.cpu_sample_queries)
        cpu = {k_: full[k_] for k_ in ("value", "unit", "cores", "kind", "sample")}

    if rank == 0:
        line = {"metric": METRIC, "value": main["qps"], "unit": "queries/s", "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": main["ms_per_step"], "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32" if c["wtype"] == "f32" else "u8", "data": "synthetic",
                "config": config_dict(args, c, n_docs, B, k, f"{args.algo}->{main['algo_used']}"),
                "ms_per_query": main["ms_per_query"], "clocks": main["clocks"], "e2e": e2e, "latency_b1": latency, "batch_sweep": sweep,
                "gpu_launches": int(main["launches_per_step"] * args.steps), "roofline": main["roofline"],
                "cpu_baseline": cpu, "kernels": main["kernels"], "candidates_per_query": main["candidates_per_query"],
                "overflow_queries": main["overflow_queries"], "other_algos": others,
                "index": {"postings": info["nnz"], "padded_postings": info["padded_nnz"], "bytes_inverted": info["bytes_inverted"],
                          "bytes_forward": info["bytes_forward"], "bytes_head": info["bytes_head"],
                          "bytes_meta": info["bytes_inverted_meta"], "head_terms": info["head_terms"], "head_terms_term_parallel": info["head_terms_term_parallel"],
                          "forward_tail_postings": info["forward_tail_nnz"], "forward_padded_postings": info["forward_padded_nnz"], "tile_docs": info["tile_docs"],
                          "build_s": t_build, "generate_s": t_gen},
                "data_checksums": {"docs_indptr": f"{wl.checksum(docs.indptr):016x}", "docs_terms": f"{wl.checksum(docs.terms):016x}",
                                   "docs_weights": f"{wl.checksum(docs.weights):016x}", "query_terms": f"{wl.checksum(queries.terms):016x}",
                                   "query_weights": f"{wl.checksum(queries.weights):016x}",
                                   "note": "64-bit checksums of the generated arrays (workload.checksum): same seed -> same inputs on every box"},
                "context": {"paper_h100_qps": 787, "paper_h100_doc_parallel_hbm_frac": 0.626,
                            "note": "paper numbers are H100 + MS MARCO/SPLADE (PAPER.md L292, L340): context, not a baseline"}}
    ix.close()
    del ix, q_dev, out_ids, out_sc
    if rank == 0:
        if not args.no_suite and world == 1 and args.config == "paper" and args.docs is None:
            line["suite"] = run_suite(torch, gs, wl, args, peaks)
        if args.sweeps and world == 1:
            line["sparsity_sweep"] = sparsity_sweep(torch, gs, wl)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def sparsity_sweep(torch, gs, wl):
    """Analogue of the paper's synthetic sparsity sweep (Table 5: 500K docs, 64 queries, mean doc nnz
    10..500; the paper does not state its generator, so only the shape is comparable): ms per 64-query batch of both kernels,
    top-10, docs from the seeded generator with nnz ~ N(m, m/3) clipped to [m/6, 4m]."""
    dev = torch.device("cuda:0")
    queries = wl.make_queries("mid", n_queries=64)
    q_dev = [torch.from_numpy(a).to(dev) for a in (queries.indptr, queries.terms, queries.weights)]
    out = []
    for m in (10, 50, 120, 250, 500):
        docs = wl.make_rows(500_000, seed=0, stream=wl.STREAM_DOCS, vocab=wl.VOCAB, zipf_s=1.1, nnz_law=wl.NNZ_NORMAL,
                            mu=float(m), sigma=m / 3.0, lo=max(1, m // 6), hi=4 * m)
        ix = gs.Index.from_numpy(docs, wl.VOCAB, device=dev)
        row = {"mean_doc_nnz": m, "postings": int(docs.indptr[-1])}
        for algo in ("term", "doc"):
            ws = torch.empty(ix.workspace_bytes(64, queries.nnz, 10, algo=algo), dtype=torch.uint8, device=dev)
            oi = torch.empty((64, 10), dtype=torch.int32, device=dev)
            osc = torch.empty((64, 10), dtype=torch.float32, device=dev)
            ms = timed_steps(torch, None, lambda: ix.search(*q_dev, 10, out_ids=oi, out_scores=osc, workspace=ws, algo=algo), 5, 3, 1)
            row[algo + "_ms_per_batch"] = ms / 5
            del ws
        ix.close()
        out.append(row)
    return out


def suite_entry(torch, gs, wl, name, args, peaks, docs, ix):
    """One BASELINE.json config other than the headline one, compact: QPS of both kernels (CUDA events, queries resident),
    scoring-kernel time and roofline fraction, overflow count, per-call p50/p99 for the latency configs (B <= 32).
    Parity of these configs is the business of tests/ (test_gpu_golden.py, test_gpu_parity.py)."""
    c = wl.CONFIGS[name]
    dev = torch.device("cuda:0")
    B, k = c["B"], c["k"]
    n_lat = (200 if B == 1 else 50) if (B <= 32 and args.latency_queries > 0) else 0
    queries = wl.make_queries(name, n_queries=max(B, n_lat * B))
    batch = queries.slice_rows(0, B)
    info, lens, head_terms = ix.info(), ix.meta()[1].astype(np.int64), ix.head_terms()
    q_dev = [torch.from_numpy(a).to(dev) for a in (batch.indptr, batch.terms, batch.weights)]
    sdt = torch.float32 if c["wtype"] == "f32" else torch.int32
    out_ids = torch.empty((B, k), dtype=torch.int32, device=dev)
    out_sc = torch.empty((B, k), dtype=sdt, device=dev)
    res = {"workload": workload_label(name, c, docs.rows, B, k), "dtype": c["wtype"], "algos": {}}
    steps = max(args.steps, 5)
    for algo in ("auto", "term", "doc"):
        ws = torch.empty(ix.workspace_bytes(B, batch.nnz, k, algo=algo), dtype=torch.uint8, device=dev)

        def step():
            ix.search(*q_dev, k, out_ids=out_ids, out_scores=out_sc, workspace=ws, algo=algo, finish=False)

        ms = timed_steps(torch, None, step, steps, max(args.warmup, 3), 1)
        st = ix.stats(ws)
        used = {1: "term", 2: "doc"}.get(st["algo_used"], "?")
        if algo == "auto":
            res["auto_dispatch"] = used
            if used in ("term", "doc"):
                del ws
                continue
        gs.profile_enable(True)
        for _ in range(steps):
            step()
        torch.cuda.synchronize()
        prof = gs.profile_read()
        gs.profile_enable(False)
        r = {"algo_used": used, "ms_per_step": ms / steps, "qps": B * steps / (ms * 1e-3), "ms_per_query": ms / steps / B,
             "overflow_queries": st["overflow_queries"], "launches_per_step": gs.last_launch_count(),
             "kernels": {n: {"launches_per_step": v["launches"] / steps, "ms_per_step": v["ms"] / steps} for n, v in prof.items()}}
        rl = roofline(r, st, info, lens, head_terms, batch, B, k, peaks, c["wtype"])
        del r["kernels"]
        if rl:
            r["roofline"] = {kk: rl.get(kk) for kk in ("kernel", "bound", "achieved", "peak", "unit", "frac", "kernel_ms_per_step",
                                                       "share_of_step", "hbm_frac", "frac_one_pass", "doc_query_tile")
                             if rl.get(kk) is not None}
        if n_lat:
            lat = latency_leg(torch, ix, queries, k, n_lat, algo, batch=B)
            r["latency"] = {kk: lat[kk] for kk in ("calls", "p50_ms", "p99_ms", "p50_ms_per_query", "graph_p50_ms", "graph_p99_ms") if kk in lat}
        res["algos"][algo] = r
        del ws
    if c["wtype"] == "u8" and B >= 64:
        # the same term-parallel search with the head contraction on the tensor cores (tcgen05.mma kind::i8, opt-in flag):
        # bit-identical results (tests/test_gpu_parity.py::test_tensor_core_head_contraction_is_bit_exact)
        ws = torch.empty(ix.workspace_bytes(B, batch.nnz, k, algo="term", flags=gs.GS_FLAG_TENSOR_CORE_HEAD), dtype=torch.uint8, device=dev)
        ms = timed_steps(torch, None, lambda: ix.search(*q_dev, k, out_ids=out_ids, out_scores=out_sc, workspace=ws, algo="term",
                                                        flags=gs.GS_FLAG_TENSOR_CORE_HEAD, finish=False), steps, max(args.warmup, 3), 1)
        res["algos"]["term_tensor_core_head"] = {"ms_per_step": ms / steps, "qps": B * steps / (ms * 1e-3),
                                                 "kernel": "k_score_term_mma (tcgen05.mma kind::i8, uint8 x uint8 -> int32, exact)"}
        del ws
    return res


def run_suite(torch, gs, wl, args, peaks):
    """BASELINE.json configs 1, 2, 4 and 5 beside the headline config 3 (north_star: QPS, batch-1 p50 latency and roofline
    fraction for every config).  Collections that share documents are generated and indexed once."""
    dev = torch.device("cuda:0")
    out = {}
    groups = [("tiny", ["tiny"]), ("mid", ["mid"]), ("paper_u8", ["paper_u8"]), ("skew_b32", ["skew_b1", "skew_b32"])]
    for doc_cfg, names in groups:
        docs = wl.make_docs(doc_cfg)
        ix = gs.Index.from_numpy(docs, wl.VOCAB, device=dev, tile_docs=args.tile_docs, head_max=args.head_max,
                                 head_density=args.head_density)
        for name in names:
            out[name] = suite_entry(torch, gs, wl, name, args, peaks, docs, ix)
        inf = ix.info()
        out[names[0]]["index_bytes"] = {kk: inf[kk] for kk in ("bytes_inverted", "bytes_inverted_meta", "bytes_forward", "bytes_head", "bytes_total")}
        ix.close()
        del docs, ix
    return out


def measured_traffic(kernel: str, info, B: int):
    """DRAM bytes per launch of a scoring kernel from the committed ncu capture (profiles/traffic.csv), for the headline
    workload only (8.8M docs, B=500); None otherwise."""
    import csv
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    if info["num_docs"] != 8_800_000 or B != 500 or not os.path.exists(path):
        return None
    for r in csv.DictReader(open(path)):
        if r["kernel"] == kernel and r["workload"] == "paper":
            return {"bytes_per_launch": int(r["dram_bytes_per_launch"]), "launch": r["launch"], "source": r["source"]}
    return None


def roofline(res, st, info, lens, head_terms, queries, B, k, peaks, wtype):
    """Roofline of the dominant scoring kernel of the step (SURVEY §8d byte models).

    doc-parallel (bound hbm): algorithmic bytes per step = sum over passes of bytes(forward index) * (1 + sample
      share): the forward index (indptr + tail CSR + the dense strips the pass's queries use) is streamed once
      per tile of `doc_query_tile` queries (PAPER.md L174 streams it once per QUERY: B*N*kbar*12 bytes); the
      threshold sample re-reads 1/2^shift of it.
    term-parallel: algorithmic bytes per step = (4 + w) * U, U = postings of the batch's distinct terms
      (each read once; the paper's model B*qbar*Lbar*8 of L172 counts them once per query: `bytes_paper_model`).
      The kernel is bound by shared-memory read-modify-writes, so its `mac_per_s` is reported too.
    """
    from paper_2606_26441_b200 import roofline as rf
    kern = res["kernels"]
    name = "score_doc" if res["algo_used"] == "doc" else "score_term"
    if name not in kern:
        return None
    kms, nl = kern[name]["ms_per_step"], kern[name]["launches_per_step"]
    ntiles = max(info["num_tiles"], 1)
    share = st["sample_tiles"] / ntiles if st["sample_tiles"] < ntiles else 0.0
    ts = rf.batch_term_stats(lens, queries.terms)
    tr = measured_traffic(name, info, B) if wtype == "f32" else None
    out = {"kernel": name, "kernel_ms_per_step": kms, "launches_per_step": nl, "share_of_step": kms / res["ms_per_step"],
           "bound": "hbm", "unit": "GB/s", "peak": peaks["hbm_gbs"], "peak_source": peaks["source"],
           # `traffic` (ncu dram bytes per launch) cannot be measured inside an un-profiled run: the figure of the committed ncu
           # capture of the same kernel and workload is quoted under its own name
           "traffic": None, "traffic_static_from_profiles": tr,
           "useful_mac_per_step": ts["W"], "mac_per_s": ts["W"] / (kms * 1e-3)}
    if name == "score_doc":
        sp = rf.strips_per_pass(queries.indptr, queries.terms, head_terms, st["doc_query_tile"])
        alg = rf.doc_parallel_bytes(info["num_docs"], info["forward_padded_nnz"], wtype, B, st["doc_query_tile"], share, sp)
        one = rf.forward_index_bytes(info["num_docs"], info["forward_padded_nnz"], wtype, len(head_terms))
        out.update({"doc_query_tile": st["doc_query_tile"], "passes": st["doc_passes"], "bytes_per_step": alg,
                    "bytes_model": "sum_passes(8*(N/32+1)+(4+w)*P_fwd+w*N*strips_used(pass))*(1+sample share), P_fwd = tail postings padded per 32-doc block",
                    "strips_used_per_pass_mean": float(np.mean(sp)) if sp else 0.0, "bytes_one_pass": one,
                    "frac_one_pass": rf.effective_gbps(one, kms) / peaks["hbm_gbs"]})
    else:
        # not HBM bound by construction: the roof is the shared-memory pipeline.  HBM figures kept beside it.
        hbm = rf.term_parallel_bytes(ts["U"], wtype, share)
        # batch kernel: the second tier of dense strips is read in full (w bytes per document per strip) on top of the postings
        x_strips = info["head_terms_term_parallel"] - info["head_terms"] if st["query_group"] >= 32 else 0
        hbm += rf.weight_bytes(wtype) * float(info["num_docs"]) * x_strips * (1.0 + share)
        ht = rf.head_tail_work(lens, queries.terms, head_terms)
        alg = rf.term_parallel_smem_bytes(ht["W_head"], ht["W_tail"], info["num_tiles"] * B, info["tile_docs"], share)
        peak = rf.smem_peak_gbs(peaks["sm_max_mhz"])
        out.update({"bound": "alu", "peak": peak,
                    "peak_source": f"derived: 148 SMs x 128 B/clk shared memory x {peaks['sm_max_mhz']:.0f} MHz (B200_PROFILING.md unit counts and clocks)",
                    "cell_rows_per_cta": st["query_group"], "bytes_per_step": alg, "W_head": ht["W_head"], "W_tail": ht["W_tail"],
                    "bytes_model": "shared-memory traffic: (4*W_head + 8*W_tail + 8*Ts*tiles*B)*(1+sample share)",
                    "hbm_bytes_per_step": hbm, "hbm_bytes_model": "((4+w)*U + w*N*x_strips)*(1+sample share), U=postings of distinct batch terms, x_strips=second-tier strips (batch kernel)", "x_strips": x_strips,
                    "hbm_achieved": rf.effective_gbps(hbm, kms), "hbm_frac": rf.effective_gbps(hbm, kms) / peaks["hbm_gbs"],
                    "hbm_bytes_paper_model": rf.term_parallel_bytes(ts["W"], wtype)})
        out["achieved"] = rf.effective_gbps(alg, kms)
        out["frac"] = out["achieved"] / peak
        return out
    out["achieved"] = rf.effective_gbps(alg, kms)
    out["frac"] = out["achieved"] / peaks["hbm_gbs"]
    # context: the nominal HBM3e figure of B200_PROFILING.md (7.7 TB/s, HGX); the fraction that counts is of the measured peak
    out["peak_nominal"] = 7700.0
    out["frac_of_nominal"] = out["achieved"] / 7700.0
    return out


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
