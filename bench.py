#!/usr/bin/env python
"""Benchmark of the hot path: one "step" = one complete randomized 1-WL refinement (all S0-S6 rows of SURVEY.md §8(a),
Algorithm 1 of PAPER.md L106-L127, run to its fixed point) of the headline synthetic graph, BASELINE.json configs[3]:
R-MAT scale 27, edge factor 16, (a,b,c,d) = (.57,.19,.19,.05), seed 2, symmetrised, deduplicated, CSR resident in HBM.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--scale S] [--impl reference]

Prints ONE JSON line (see the task contract).  `value` = column indices consumed per second over the whole call
(GEdges/s); `e2e` = the same through wl_refine_host (pinned host CSR -> device, colours -> host inside the timed region);
`roofline` = the SpMV kernel (dominant) against the measured HBM copy bandwidth; `cpu_baseline` = the CPU oracle on a
bounded sample.  With N > 1 (torchrun) every rank refines its own replica of the graph: the path does not shard
without a collective per round, so scaling is weak / replicas only.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

RMAT_SEEDS = {22: 1, 27: 2, 30: 3}  # BASELINE.json configs[2..4]
ORACLE_SAMPLE_SCALE = 21           # bounded sample of the same recipe for the CPU oracle (about 10-30 s)
HBM_FALLBACK_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback
GEN_TOP_BITS = 9  # source-range groups of the host generator: the largest holds 0.76^9 of the draws (< 2^31 keys at scale 30)
KNOWN_SIZES = {22: (4194304, 128311764), 27: (134217728, 4223286680)}  # (n, m) of the deterministic generator


def ncu_traffic():
    """DRAM bytes per launch of the round-2 kernels from the last `ncu --set full` capture: a tracked data file that names the
    commit it was measured on (profiles/ncu_traffic.json), never a constant in this script."""
    try:
        return json.load(open(os.path.join(ROOT, "profiles", "ncu_traffic.json")))
    except Exception:
        return None


def _classify(got, want):
    """Reading Q12: 'equal', 'coarser' (the exact colouring strictly refines the result: a randomized collision) or
    'other' (a bug).  numpy int arrays of canonical colours."""
    import numpy as np
    if got.shape == want.shape and bool((got == want).all()):
        return "equal"
    # want refines got <=> every block of want lies inside one block of got
    pairs = np.unique(np.stack([want.astype(np.int64), got.astype(np.int64)], 1), axis=0)
    return "coarser" if pairs.shape[0] == int(want.max()) + 1 else "other"


def mismatch_report(wl, gg, oracle, dev, seeds_c1=100, seeds_c3=0):
    """north_star: 'any randomized-collision mismatch counted and reported against the paper's stated failure bound'.
    C1 (and C3 when asked) refined with many seeds, every result classified against the oracle's colouring."""
    import torch
    out = {"bound_per_run": 1e-9, "bound_source": "Theorem 1, PAPER.md L129 (q = 64)", "configs": []}
    todo = [("C1 Erdos-Renyi 10k/50k", gg.erdos_renyi(), seeds_c1)]
    if seeds_c3:
        todo.append(("C3 R-MAT scale 22", gg.rmat(22, seed=RMAT_SEEDS[22], device=dev), seeds_c3))
    for name, g, seeds in todo:
        n, rp, ci, wt = g.numpy()
        want, counts, _ = oracle.refine(n, rp, ci, wt)
        gd = g.to(dev)
        wdev = torch.from_numpy(want).to(dev)
        t = {"equal": 0, "coarser": 0, "other": 0}
        for seed in range(seeds):
            r = wl.wl_refine(n, gd.row_ptr, gd.col, None, seed=7000 + seed)
            if bool(torch.equal(r.colors, wdev)) and r.round_colors == counts:
                t["equal"] += 1
            else:
                t[_classify(r.colors.cpu().numpy(), want)] += 1
        out["configs"].append({"config": name, "runs": seeds, **t})
    out["runs"] = sum(c["runs"] for c in out["configs"])
    out["mismatching_runs"] = sum(c["coarser"] + c["other"] for c in out["configs"])
    return out


def split_pairs_on_device(wl, n, row_ptr, col, rounds, dev):
    """N_r = sum over the blocks B of the partition before round r of C(s_B, 2), s_B = number of blocks of the partition after
    round r inside B: the pairs of sub-blocks whose z must differ for round r to be computed exactly (failure bound
    of the build).  Partitions after r rounds come from wl_refine(max_rounds = r)."""
    import torch
    prev = torch.zeros(n, dtype=torch.int64, device=dev)
    out = []
    for r in range(1, rounds):
        cur = wl.wl_refine(n, row_ptr, col, None, seed=1, max_rounds=r, allow_max_rounds=True, deep=False).colors.to(torch.int64)
        k_cur = int(cur.max()) + 1
        pairs = torch.unique(prev * k_cur + cur)
        s_b = torch.bincount(pairs // k_cur)
        out.append(int((s_b * (s_b - 1) // 2).sum()))
        prev = cur
        del pairs, s_b
    return out


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)), "measured"
        except Exception:
            pass
    return {"hbm_gbs": HBM_FALLBACK_GBS}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for l in self.lines:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 8:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(names, f[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(scale: int):
    """The CPU oracle, as it stands, on a bounded sample of the workload: the same R-MAT recipe at a smaller scale."""
    import graphgen as gg
    import oracle
    try:
        import torch
        gen_dev = "cuda" if torch.cuda.is_available() else "cpu"
    except Exception:
        gen_dev = "cpu"
    g = gg.rmat(scale, seed=RMAT_SEEDS[27], device=gen_dev)  # input generation only; the oracle runs on the host cores
    n, rp, ci, wt = g.numpy()
    t0 = time.perf_counter()
    _, counts, rounds = oracle.refine(n, rp, ci, wt)
    dt = time.perf_counter() - t0
    cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    return {"value": g.m * rounds / dt / 1e9, "unit": "GEdges/s", "cores": cores, "kind": "oracle",
            "sample": f"R-MAT scale {scale} (n={n}, m={g.m}), same recipe and seed as the workload, {rounds} rounds of "
                      f"signature-sort refinement in {dt:.2f} s (signatures built with OpenMP, sort on one core)",
            "seconds": dt, "rounds": rounds, "m": g.m, "n": n}


def run_reference(args):
    """--impl reference: the oracle on the host cores, on this arm's metric / unit / config."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    times, last = [], None
    for i in range(args.warmup + args.steps):
        last = oracle_sample(args.oracle_scale)
        if i >= args.warmup:
            times.append(last["seconds"])
    ms = 1e3 * sum(times) / len(times)
    value = last["m"] * last["rounds"] / (ms / 1e3) / 1e9
    cb = {k: last[k] for k in ("unit", "cores", "kind", "sample")}
    cb["value"] = value
    # this arm's config is the headline workload (the driver compares the two arms on it); every step is a bounded sample of
    # it: the same recipe and seed at a smaller scale, named here with its true sizes
    cfg = workload_config(args.scale, KNOWN_SIZES.get(args.scale, (None, None))[0], KNOWN_SIZES.get(args.scale, (None, None))[1])
    cfg["sample"] = {"scale": args.oracle_scale, "n": last["n"], "m": last["m"], "rounds": last["rounds"],
                     "what": "each step refines this bounded sample of the workload (same R-MAT recipe and seed, smaller scale) "
                             "with the CPU oracle (signature-sort refinement)"}
    cfg["value_definition"] = "m_sample x rounds / seconds (every round of the oracle reads every edge; no pruning)"
    line = {"impl": "reference", "metric": "refine_gedges_per_s", "value": value, "unit": "GEdges/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
            "config": cfg, "cpu_baseline": cb,
            "e2e": {"value": value, "unit": "GEdges/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def run_batched(args):
    """--workload batched: Algorithm 2 (RBSC) over a HOST-resident directed R-MAT graph under a device-memory cap: BASELINE.json
    configs[4] (scale 30) or a smaller scale of the same recipe.  One step = one wl_refine_batched call to its fixed point;
    inputs start in pinned host memory, the colours end there.  --consume-input (forced from scale 30 on: 77 GB of input + 154 GB
    of quotient scratch exceed the box's 196 GB of host memory): WL_FLAG_CONSUME_INPUT, the quotients overwrite the input's
    column array, so every step needs a freshly generated graph (one cold step per mode, no warm-up)."""
    import torch
    import graphgen as gg
    import paper_2607_02603_b200 as wl
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
    consume = args.consume_input or args.scale >= 30
    cap = int(args.cap_gb * (1 << 30))
    t_gen0 = time.perf_counter()
    if consume:
        n, rp, col = gg.rmat_directed_to_host(args.scale, seed=RMAT_SEEDS[30], device=dev, pin=True, top_bits=GEN_TOP_BITS)
        m = col.numel()
        col_buf = col
    else:
        g = gg.rmat(args.scale, seed=RMAT_SEEDS[30], symmetrize=False, device=dev, chunk=1 << 27)
        n, m = g.n, g.m
        rp = torch.empty(n + 1, dtype=torch.int64, pin_memory=True)
        col = torch.empty(m, dtype=torch.int32, pin_memory=True)
        rp.copy_(g.row_ptr)
        col.copy_(g.col)
        del g
    torch.cuda.empty_cache()
    gen_s = time.perf_counter() - t_gen0
    hws_bytes = (wl.wl_refine_batched_host_bytes_consume(n, m) + wl.wl_refine_batched_host_overflow_bytes(m)) if consume else wl.wl_refine_batched_host_bytes(n, m)
    scratch_kind = "pinned"
    try:
        hws = torch.empty(hws_bytes, dtype=torch.uint8, pin_memory=True)
    except RuntimeError:  # this box pins about 120 GB at most: the scratch then stays pageable (slower, staged transfers)
        torch.cuda.synchronize(dev)
        hws = torch.empty(hws_bytes, dtype=torch.uint8)
        hws.zero_()  # touch the pages outside the timed region, as pinning would
        scratch_kind = "pageable (pinning %.0f GB on top of the %.0f GB input failed on this box)" % (
            hws_bytes / 2 ** 30, (rp.numel() * 8 + col.numel() * 4) / 2 ** 30)
    out = torch.empty(n, dtype=torch.int32, pin_memory=(scratch_kind == "pinned"))
    base_flags = args.flags | (wl.WL_FLAG_CONSUME_INPUT if consume else 0)
    # caller-owned device arena of the cap's size (wl_options.device_workspace): the timed calls allocate nothing on the device
    arena = None if args.no_arena else torch.empty(cap, dtype=torch.uint8, device=dev)

    def measure_link():
        """Pinned copies of 256 MiB: host -> device alone, device -> host alone, both at once (GB/s; best of three)."""
        nb = 1 << 26
        h_up = torch.empty(nb, dtype=torch.int32, pin_memory=True)
        h_dn = torch.empty(nb, dtype=torch.int32, pin_memory=True)
        d_up = torch.empty(nb, dtype=torch.int32, device=dev)
        d_dn = torch.empty(nb, dtype=torch.int32, device=dev)
        s_up, s_dn = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
        gb = 4 * nb / 1e9

        def timed(up, down):
            best = 0.0
            for _ in range(3):
                torch.cuda.synchronize(dev)
                t = time.perf_counter()
                if up:
                    with torch.cuda.stream(s_up):
                        d_up.copy_(h_up, non_blocking=True)
                if down:
                    with torch.cuda.stream(s_dn):
                        h_dn.copy_(d_dn, non_blocking=True)
                torch.cuda.synchronize(dev)
                best = max(best, (int(up) + int(down)) * gb / (time.perf_counter() - t))
            return best
        return {"h2d": timed(True, False), "d2h": timed(False, True), "both_sum": timed(True, True)}

    try:
        link_peak = measure_link()
        link_kind = "pinned copies of 256 MiB measured on this box right before the timed calls"
    except RuntimeError:  # no pinned memory left for the probe (scale 30 pins 108 GB of this box's limit of about 120 GB)
        link_peak = {"h2d": 55.6, "d2h": 57.3, "both_sum": 99.0}
        link_kind = "pinned copies measured on another box of this pool (the probe found no pinned memory here)"
    torch.cuda.empty_cache()

    def one(flags, seed):
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        r = wl.wl_refine_batched(n, rp, col, None, max_batch_edges=args.batch_edges, seed=seed, device_cap_bytes=cap,
                                 flags=flags, host_workspace=hws, out=out, device_workspace=arena)
        torch.cuda.synchronize(dev)
        return r, time.perf_counter() - t0

    def regenerate():
        if consume:  # the previous step overwrote the column array
            gg.rmat_directed_to_host(args.scale, seed=RMAT_SEEDS[30], device=dev, pin=True, col_out=col_buf, row_ptr_out=rp,
                                     top_bits=GEN_TOP_BITS)
            torch.cuda.empty_cache()

    times, res = [], None
    n_runs = 1 if consume else args.warmup + args.steps
    for i in range(n_runs):
        res, dt = one(base_flags, 300 + i)
        if consume or i >= args.warmup:
            times.append(dt)
    st = res.stats
    sec = sum(times) / len(times)
    link = (st["bytes_h2d"] + st["bytes_d2h"]) / sec / 1e9
    # the same with WL_FLAG_INHERIT_BATCHES (reading Q14b: quotients keep the batches of their graph and are refined while
    # their rows are still on the device: one upload pass per outer iteration instead of two)
    inh = None
    if not (base_flags & wl.WL_FLAG_INHERIT_BATCHES) and not args.no_inherit_leg:
        ti = []
        for i in range(1 if consume else max(1, args.steps)):
            regenerate()
            ri, dt = one(base_flags | wl.WL_FLAG_INHERIT_BATCHES, 400 + i)
            ti.append(dt)
        si = ri.stats
        seci = sum(ti) / len(ti)
        inh = {"seconds_to_stable_coloring": seci, "value": m / seci / 1e9, "unit": "GEdges/s", "outer_iters": si["outer_iters"],
               "num_colors": si["num_colors"], "reduction_power": si["num_colors"] / n, "h2d_bytes_per_step": si["bytes_h2d"],
               "d2h_bytes_per_step": si["bytes_d2h"], "link_gb_per_s": (si["bytes_h2d"] + si["bytes_d2h"]) / seci / 1e9}
    # Theorem 2 on a sample: Def. 1 on sampled non-singleton blocks of the result (the full check is the oracle's, in the tests)
    line = {"metric": "batched_refine_input_gedges_per_s", "value": m / sec / 1e9, "unit": "GEdges/s", "n_gpus": 1,
            "steps": len(times), "warmup": 0 if consume else args.warmup, "ms_per_step": 1e3 * sec, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
            "config": {"workload": f"R-MAT scale {args.scale}, edge factor 16, seed 3, directed, deduplicated, CSR in pinned host "
                                   f"memory; device cap {args.cap_gb} GB, M_b = {args.batch_edges if args.batch_edges > 0 else 'derived from the cap'} "
                                   f"({'BASELINE.json configs[4]' if args.scale == 30 else 'shape of BASELINE.json configs[4]'})",
                       "n": n, "m": m, "step": "wl_refine_batched to the batched fixed point (Algorithm 2, B1-B7)",
                       "consume_input": consume, "generation_seconds": gen_s, "host_scratch": scratch_kind,
                       "device_arena": "none (library allocates)" if arena is None else "caller-owned, %.1f GB = the cap" % (cap / 2 ** 30),
                       "pinned_host_gb": (rp.numel() * 8 + col.numel() * 4 + hws.numel() + out.numel() * 4) / 2 ** 30},
            "seconds_to_stable_coloring": sec, "outer_iters": st["outer_iters"], "num_colors": st["num_colors"],
            "reduction_power": st["num_colors"] / n, "last_num_batches": st["last_num_batches"],
            "boundary_nodes": st["boundary_nodes"], "h2d_bytes_per_step": st["bytes_h2d"],
            "d2h_bytes_per_step": st["bytes_d2h"],
            "link": {"achieved": link, "unit": "GB/s", "peak": link_peak["both_sum"],
                     "peak_kind": link_kind + ": both directions running together (sum); h2d / d2h alone: %.1f / %.1f GB/s" % (
                         link_peak["h2d"], link_peak["d2h"]),
                     "frac": link / link_peak["both_sum"],
                     "h2d_gb_per_s": st["bytes_h2d"] / sec / 1e9, "d2h_gb_per_s": st["bytes_d2h"] / sec / 1e9,
                     "frac_h2d_alone": st["bytes_h2d"] / sec / 1e9 / link_peak["h2d"]},
            "ms_inbatch_spmv": st["ms_spmv"], "gpu_launches": st["kernel_launches"], "inherit_batches": inh,
            "e2e": {"value": m / sec / 1e9, "unit": "GEdges/s", "h2d_bytes_per_step": st["bytes_h2d"],
                    "d2h_bytes_per_step": st["bytes_d2h"]}}
    print(json.dumps(line))
    return 0


def run_batch_study(args):
    """--workload batch-study: the shape of the paper's simulated-memory experiment (Tables 1 and 3, L237-L297): the
    same graph refined with N_b = 1, 2, 4, ... row-contiguous edge batches; reports the reduction power |H|/|V| next to the
    coarsest colouring's and the slow-down against N_b = 1."""
    import torch
    import graphgen as gg
    import paper_2607_02603_b200 as wl
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    graphs = [("C1 Erdos-Renyi 10k/50k", gg.erdos_renyi()), ("grid 512^2", gg.grid2d(512, device=dev)),
              (f"R-MAT scale {args.scale} symmetrised", gg.rmat(args.scale, seed=RMAT_SEEDS.get(args.scale, 1), device=dev)),
              (f"R-MAT scale {args.scale} directed", gg.rmat(args.scale, seed=3, symmetrize=False, device=dev))]
    rows = []
    for name, g in graphs:
        n, m = g.n, g.m
        gd = g.to(dev)
        single = wl.wl_refine(n, gd.row_ptr, gd.col, None, seed=1)
        rp, col = gd.row_ptr.cpu().pin_memory(), gd.col.cpu().pin_memory()
        hws = torch.empty(wl.wl_refine_batched_host_bytes(n, m), dtype=torch.uint8, pin_memory=True)
        base = None
        for nb in (1, 2, 4, 8):
            best = None
            for rep in range(3):
                torch.cuda.synchronize(dev)
                t0 = time.perf_counter()
                r = wl.wl_refine_batched(n, rp, col, None, max_batch_edges=(m + nb - 1) // nb, seed=10 + rep, host_workspace=hws)
                dt = time.perf_counter() - t0
                best = dt if best is None else min(best, dt)
            base = best if nb == 1 else base
            rows.append({"graph": name, "n": n, "m": m, "N_b": nb, "partition": "row-contiguous (CSR slices)",
                         "colors": r.num_colors,
                         "reduction_power_pct": 100.0 * r.num_colors / n,
                         "coarsest_pct": 100.0 * single.num_colors / n,
                         "gap_pp": 100.0 * (r.num_colors - single.num_colors) / n,
                         "outer_iters": r.stats["outer_iters"], "boundary_nodes": r.stats["boundary_nodes"],
                         "seconds": best, "slowdown_vs_Nb1": best / base})
            if nb == 1:
                continue
            # the same graph under ARBITRARY edge partitions (COO batches, Thm 2)
            gc = gd.to("cpu")
            for pname, eb in (("random edges", gg.random_edge_batches(gc, nb, 5)),
                              ("by source node, 5 % of the edges moved", gg.node_hash_edge_batches(gc, nb, 5, 5))):
                cb = [tuple(None if t is None else t.pin_memory() for t in b) for b in gg.coo_batches(gc, eb, nb)]
                best = None
                for rep in range(2):
                    torch.cuda.synchronize(dev)
                    t0 = time.perf_counter()
                    r = wl.wl_refine_batched(n, None, None, None, max_batch_edges=(m + nb - 1) // nb, seed=20 + rep,
                                             host_workspace=hws, coo_batches=cb)
                    dt = time.perf_counter() - t0
                    best = dt if best is None else min(best, dt)
                rows.append({"graph": name, "n": n, "m": m, "N_b": nb, "partition": pname, "colors": r.num_colors,
                             "reduction_power_pct": 100.0 * r.num_colors / n,
                             "coarsest_pct": 100.0 * single.num_colors / n,
                             "gap_pp": 100.0 * (r.num_colors - single.num_colors) / n,
                             "outer_iters": r.stats["outer_iters"], "boundary_nodes": r.stats["boundary_nodes"],
                             "seconds": best, "slowdown_vs_Nb1": best / base})
    print(json.dumps({"metric": "batch_study", "unit": "table", "data": "synthetic", "rows": rows}))
    return 0


def run_cap_sweep(args):
    """--workload cap-sweep: the shape of the paper's Table 4 (L311-L332): the same host-resident graph refined with aggressive
    termination (L328) under two batch caps M_b; reports seconds and reduction power per cap."""
    import torch
    import graphgen as gg
    import paper_2607_02603_b200 as wl
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    g = gg.rmat(args.scale, seed=RMAT_SEEDS[30], symmetrize=False, device=dev, chunk=1 << 27)
    n, m = g.n, g.m
    rp = torch.empty(n + 1, dtype=torch.int64, pin_memory=True)
    col = torch.empty(m, dtype=torch.int32, pin_memory=True)
    rp.copy_(g.row_ptr)
    col.copy_(g.col)
    single = wl.wl_refine(n, g.row_ptr, g.col, None, seed=1, deep=False).num_colors if args.scale <= 27 else None
    del g
    torch.cuda.empty_cache()
    hws = torch.empty(wl.wl_refine_batched_host_bytes(n, m), dtype=torch.uint8, pin_memory=True)
    out = torch.empty(n, dtype=torch.int32, pin_memory=True)
    # caller-owned device arena (wl_options.device_workspace): the timed calls allocate nothing on the device
    arena = None if args.no_arena else torch.empty(int(args.cap_gb * (1 << 30)), dtype=torch.uint8, device=dev)
    rows = []
    for cap_edges in (args.batch_edges, 4 * args.batch_edges):
        for name, flags in (("aggressive (L328)", wl.WL_FLAG_AGGRESSIVE_STOP), ("paper termination (L200)", 0),
                            ("inherited batches (Q14b)", wl.WL_FLAG_INHERIT_BATCHES)):
            best, r = None, None
            for rep in range(2):
                torch.cuda.synchronize(dev)
                t0 = time.perf_counter()
                r = wl.wl_refine_batched(n, rp, col, None, max_batch_edges=cap_edges, seed=20 + rep, flags=flags,
                                         host_workspace=hws, out=out, device_workspace=arena)
                torch.cuda.synchronize(dev)
                dt = time.perf_counter() - t0
                best = dt if best is None else min(best, dt)
            rows.append({"M_b": cap_edges, "termination": name, "seconds": best, "outer_iters": r.stats["outer_iters"],
                         "colors": r.num_colors, "reduction_power_pct": 100.0 * r.num_colors / n,
                         "coarsest_pct": None if single is None else 100.0 * single / n,
                         "first_num_batches": -(-m // cap_edges)})
    print(json.dumps({"metric": "cap_sweep", "unit": "table", "data": "synthetic",
                      "config": {"workload": f"R-MAT scale {args.scale}, directed, seed 3", "n": n, "m": m,
                                 "device_arena_gb": None if arena is None else args.cap_gb}, "rows": rows}))
    return 0


def _oracle_child(kind, path, threads, q):
    """Runs in a child process (so that a wall-clock limit can end it): one oracle run on the graph stored at `path`."""
    os.environ["OMP_NUM_THREADS"] = str(threads)
    import numpy as np
    import oracle
    d = np.load(path)
    n, rp, ci = int(d["n"]), d["rp"], d["ci"]
    t0 = time.perf_counter()
    if kind == "refine":
        c, counts, rounds = oracle.refine(n, rp, ci)
    else:
        c, counts, rounds, _ = oracle.rsc(n, rp, ci, seed=424242)
    dt = time.perf_counter() - t0
    np.save(path + ".colors.npy", c)
    q.put((dt, counts, rounds))


def _timed_oracle(kind, n, rp, ci, threads, limit, tag):
    import multiprocessing as mp
    import numpy as np
    path = f"/tmp/wl_oracle_{tag}_{os.getpid()}.npz"
    np.savez(path, n=n, rp=rp, ci=ci)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    p = ctx.Process(target=_oracle_child, args=(kind, path, threads, q))
    t0 = time.perf_counter()
    p.start()
    res = None
    try:
        res = q.get(timeout=limit)
    except Exception:
        pass
    if res is None:
        p.kill()
        p.join()
        out = {"finished": False, "seconds": time.perf_counter() - t0, "limit_s": limit}
    else:
        p.join()
        out = {"finished": True, "seconds": res[0], "counts": res[1], "rounds": res[2],
               "colors": np.load(path + ".colors.npy")}
    for f in (path, path + ".colors.npy"):
        try:
            os.remove(f)
        except OSError:
            pass
    return out


def run_oracle_times(args):
    """--workload oracle-times: SURVEY.md §8(d) "Oracle timing": the CPU oracle (signature-sort refinement), single-threaded and
    on all cores, on C1-C3, each under a wall-clock limit ("did not finish" is an allowed outcome); nproc printed.  C4 is
    attempted by `--workload c4-check` with the CPU Algorithm 1 (the signature oracle needs more host memory than the box has
    at scale 27)."""
    import torch
    import graphgen as gg
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    nproc = os.cpu_count() or 1
    rows = []
    for name, make in (("C1 Erdos-Renyi 10k/50k", lambda: gg.erdos_renyi()),
                       ("C2 grid 2048^2 (1024 rounds)", lambda: gg.grid2d(2048, device=dev)),
                       ("C3 R-MAT scale 22", lambda: gg.rmat(22, seed=RMAT_SEEDS[22], device=dev))):
        g = make()
        n, rp, ci, wt = g.numpy()
        del g
        for threads in (1, nproc):
            r = _timed_oracle("refine", n, rp, ci, threads, args.time_limit, name.split()[0])
            rows.append({"config": name, "n": n, "m": int(rp[-1]), "threads": threads, "finished": r["finished"],
                         "seconds": r["seconds"], "rounds": r.get("rounds"),
                         "num_colors": (r["counts"][-1] if r.get("counts") else None)})
            print(json.dumps(rows[-1]), file=sys.stderr, flush=True)
    print(json.dumps({"metric": "oracle_times", "unit": "table", "nproc": nproc, "limit_s": args.time_limit, "rows": rows}))
    return 0


def run_c4_check(args):
    """--workload c4-check: an element-by-element target for the headline config.  The CPU Algorithm 1 (oracle.rsc, pinned equal
    to the signature oracle) refines the scale-27 graph once with ITS OWN seed under a wall-clock limit;
    the GPU colouring (different seed, default flags) must equal it element by element, per-round colour counts included."""
    import numpy as np
    import torch
    import graphgen as gg
    import paper_2607_02603_b200 as wl
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    g = gg.rmat(args.scale, seed=RMAT_SEEDS.get(args.scale, 2), device=dev, chunk=1 << 28)
    torch.cuda.empty_cache()
    n, m = g.n, g.m
    res = wl.wl_refine(n, g.row_ptr, g.col, None, seed=2027, deep=False)
    got = res.colors.cpu().numpy()
    rp, ci = g.row_ptr.cpu().numpy(), g.col.cpu().numpy()
    del g
    torch.cuda.empty_cache()
    r = _timed_oracle("rsc", n, rp, ci, 1, args.time_limit, "c4")
    line = {"metric": "c4_check", "unit": "bool", "config": workload_config(args.scale, n, m), "gpu_rounds": res.rounds,
            "gpu_round_colors": res.round_colors, "gpu_num_colors": res.num_colors,
            "oracle": "oracle.rsc (CPU Algorithm 1 in Z/2^64, one thread, seed 424242)", "oracle_finished": r["finished"],
            "oracle_seconds": r["seconds"], "limit_s": args.time_limit}
    if r["finished"]:
        line["oracle_round_colors"] = r["counts"]
        line["trajectory_equal"] = r["counts"] == res.round_colors
        line["colors_equal_element_by_element"] = bool((r["colors"] == got).all())
        line["classification"] = _classify(got, r["colors"])
    print(json.dumps(line))
    return 0


def run_sharded(args):
    """--workload sharded: Algorithm 2 with the batches of every outer iteration spread over the ranks (sharded.py): STRONG scaling
    of one fixed host-resident graph over N GPUs (torchrun), the exchange being one all-gather of block counts and one
    all-gather-v of the block-map slices per outer iteration.  N = 1 runs the same driver on one GPU."""
    import torch
    import graphgen as gg
    from paper_2607_02603_b200.sharded import refine_batched_sharded
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    g = gg.rmat(args.scale, seed=RMAT_SEEDS[30], symmetrize=False, device=dev, chunk=1 << 27)
    n, m = g.n, g.m
    rp, col = g.row_ptr.cpu().pin_memory(), g.col.cpu().pin_memory()
    del g
    torch.cuda.empty_cache()
    cap = args.batch_edges if args.batch_edges > 0 else max(1, m // 32 + 1)
    times, res = [], None
    for i in range(args.warmup + args.steps):
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        res = refine_batched_sharded(n, rp, col, None, max_batch_edges=cap, seed=500 + i, dist=dist, device=dev)
        torch.cuda.synchronize(dev)
        if i >= args.warmup:
            times.append(time.perf_counter() - t0)
    local = sum(times) / len(times)
    t = torch.tensor([local], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    sec = float(t.item())
    if rank == 0:
        colours, k, outer = res
        print(json.dumps({"metric": "sharded_batched_refine_input_gedges_per_s", "value": m / sec / 1e9, "unit": "GEdges/s",
                          "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sec,
                          "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
                          "config": {"workload": f"R-MAT scale {args.scale}, directed, seed 3, host-resident; batches of {cap} edges "
                                                 "spread over the ranks (sharded.py, inherited batches)", "n": n, "m": m},
                          "num_colors": k, "outer_iters": outer, "reduction_power": k / n}))
    if dist is not None:
        dist.destroy_process_group()
    return 0


def aggregate_over_ranks(dist, local_ms: float, units_per_rank: float, device=None):
    """Max-over-ranks time and whole-job throughput for N independent replicas (weak scaling, no data-path collective).
    dist = torch.distributed (initialised) or None for a single process.  Returns (ms_max, total_units_per_second)."""
    import torch
    world = 1
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([units_per_rank], dtype=torch.float64, device=device)
    if dist is not None:
        world = dist.get_world_size()
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    ms = float(t.item())
    return ms, float(u.item()) / (ms / 1e3), world


def workload_config(scale, n, m):
    return {"workload": f"R-MAT scale {scale}, edge factor 16, (a,b,c,d)=(0.57,0.19,0.19,0.05), seed "
                        f"{RMAT_SEEDS.get(scale, 2)}, symmetrised, deduplicated, uniform initial colour "
                        f"(BASELINE.json configs[{ {22: 2, 27: 3}.get(scale, 3)}])",
            "n": n, "m": m, "step": "wl_refine to the fixed point (all rounds, S0-S6)",
            "l2": "inputs (CSR >= 0.5 GB, 17 GB at scale 27) exceed the 126 MB L2; no flush needed between steps"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--scale", type=int, default=27)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--oracle-scale", type=int, default=ORACLE_SAMPLE_SCALE)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--flags", type=int, default=0, help="WL_FLAG_* bits passed to wl_refine")
    ap.add_argument("--mismatch-c3-seeds", type=int, default=20, help="seeds of the C3 leg of the mismatch report (0: C1 only)")
    ap.add_argument("--time-limit", type=float, default=1800.0, help="oracle-times / c4-check: wall-clock limit per oracle run (s)")
    ap.add_argument("--workload", default="single", choices=["single", "batched", "batch-study", "cap-sweep", "oracle-times", "c4-check", "sharded"],
                    help="single: wl_refine on the HBM-resident graph (the headline); batched: wl_refine_batched")
    ap.add_argument("--cap-gb", type=float, default=16.0, help="batched: device memory cap")
    ap.add_argument("--consume-input", action="store_true", help="batched: WL_FLAG_CONSUME_INPUT (forced from scale 30 on)")
    ap.add_argument("--no-inherit-leg", action="store_true", help="batched: skip the second run with WL_FLAG_INHERIT_BATCHES")
    ap.add_argument("--no-arena", action="store_true", help="batched: let the library cudaMalloc / cudaFree its device buffers")
    ap.add_argument("--batch-edges", type=int, default=0, help="batched: M_b (0: derived by the library from the device cap)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    if args.impl == "reference":
        return run_reference(args)
    if args.workload == "batched":
        return run_batched(args)
    if args.workload == "batch-study":
        return run_batch_study(args)
    if args.workload == "cap-sweep":
        return run_cap_sweep(args)
    if args.workload == "oracle-times":
        return run_oracle_times(args)
    if args.workload == "c4-check":
        return run_c4_check(args)
    if args.workload == "sharded":
        return run_sharded(args)

    import torch
    import graphgen as gg
    import paper_2607_02603_b200 as wl

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---- synthetic input, generated on the device (not timed) --------------------------------------------------------
    seed = RMAT_SEEDS.get(args.scale, 2)
    g = gg.rmat(args.scale, seed=seed, device=dev, chunk=1 << 28)
    torch.cuda.empty_cache()
    n, m = g.n, g.m
    ws = torch.empty(wl.wl_refine_workspace_bytes(n, m), dtype=torch.uint8, device=dev)
    out = torch.empty(n, dtype=torch.int32, device=dev)

    def step(i):
        return wl.wl_refine(n, g.row_ptr, g.col, None, seed=1000 + i, flags=args.flags, workspace=ws, out=out)

    # nvidia-smi is started BEFORE the warm-up so that its start-up (NVML initialisation takes driver locks for a few
    # hundred ms and would stretch the host round trips of the first timed steps) is over when the timed region begins;
    # it keeps sampling every 200 ms during the timed region.
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        t_wait = time.perf_counter()
        while not sampler.lines and time.perf_counter() - t_wait < 10.0:
            time.sleep(0.05)
    for i in range(max(args.warmup, 3)):
        res = step(i)
    if rank == 0:
        sampler.lines.clear()
    barrier()
    launches0 = wl.wl_kernel_launches()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    results = []
    for i in range(args.steps):
        results.append(step(100 + i))
    ev1.record()
    barrier()
    launches = wl.wl_kernel_launches() - launches0
    clocks = sampler.stop() if rank == 0 else None
    edges_per_step = results[-1].stats["edges_streamed"]
    ms_total, edges_per_s, _ = aggregate_over_ranks(dist, ev0.elapsed_time(ev1), edges_per_step * args.steps, dev)
    ms_per_step = ms_total / args.steps
    value = edges_per_s / 1e9

    # ---- roofline of the dominant kernel: the S1+S2 launch of the one un-pruned round (round 2 from a uniform start: the
    # row kernel + the hub-chunk kernel), timed by the library's own CUDA events on the launch stream -------------------
    peaks, peak_kind = measured_peaks()
    spmv_ms = sum(r.stats["ms_spmv_kernel"] for r in results)
    spmv_launches = sum(r.stats["spmv_launches"] for r in results)
    alg_bytes = sum(r.stats["spmv_alg_bytes"] for r in results)  # (4+G) per streamed entry + 16 per row, DESIGN.md
    spmv_edges = sum(r.stats["edges_streamed"] for r in results)
    top_ms = sum(r.stats["ms_spmv_top"] for r in results) / len(results)
    top_bytes = results[-1].stats["spmv_top_alg_bytes"]
    top_edges = results[-1].stats["spmv_top_edges"]
    roofline = None
    tr = ncu_traffic() if args.scale == 27 and not args.flags else None
    NCU_TRAFFIC_BYTES = tr["spmv_round2_bytes"] if tr else None
    NCU_RELABEL_BYTES = tr["relabel_round2_bytes"] if tr else None
    if spmv_launches and top_ms > 0:
        achieved = top_bytes / (top_ms / 1e3) / 1e9
        roofline = {"bound": "hbm", "kernel": "spmv_merge_kernel" if args.flags & 4 else
                    "spmv_rows32_kernel<u16>+spmv_hub_kernel<u16> (S1+S2 of round 2, the un-pruned round)",
                    "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": achieved / peaks["hbm_gbs"],
                    "peak_kind": f"{peak_kind} copy bandwidth", "algorithmic_bytes_per_launch": top_bytes,
                    "avg_launch_ms": top_ms, "launches_timed": len(results),
                    "gedges_per_s_in_kernel": top_edges / (top_ms / 1e3) / 1e9,
                    "traffic": NCU_TRAFFIC_BYTES,
                    "dram_gb_per_s_ncu_traffic": (NCU_TRAFFIC_BYTES / (top_ms / 1e3) / 1e9) if tr else None,
                    "traffic_source": (f"profiles/ncu_traffic.json <- {tr['source']}, measured on commit {tr['measured_on_commit']} "
                                       "(dram__bytes_read.sum + dram__bytes_write.sum, row + hub kernel)") if tr else None,
                    "share_of_step": top_ms / ms_per_step,
                    "all_spmv_launches": {"launches": spmv_launches, "algorithmic_gb_per_s": alg_bytes / (spmv_ms / 1e3) / 1e9,
                                          "gedges_per_s": spmv_edges / (spmv_ms / 1e3) / 1e9,
                                          "share_of_step": spmv_ms / ms_total},
                    "round_pair": {  # the SpMV + relabel pair of that round, model bytes (4+G) m + 64 n
                        "spmv_ms": top_ms, "relabel_and_compaction_ms": sum(r.stats["ms_rest_top"] for r in results) / len(results),
                        "rows": results[-1].stats["rows_top"],
                        "algorithmic_gb_per_s": (top_bytes + 48 * results[-1].stats["rows_top"]) /
                        ((top_ms + sum(r.stats["ms_rest_top"] for r in results) / len(results)) / 1e3) / 1e9,
                        "dram_gb_per_s_ncu": ((NCU_TRAFFIC_BYTES + NCU_RELABEL_BYTES) /
                                              ((top_ms + sum(r.stats["ms_rest_top"] for r in results) / len(results)) / 1e3) / 1e9)
                        if tr else None},
                    "binding_unit": "L1TEX 76 % / L2 73 % of peak (ncu): one sector lookup per gathered 2-byte id; DRAM 43 %"}

    # ---- end to end through the host-buffer entry point ---------------------------------------------------------------
    e2e = None
    if not args.no_e2e:
        h_rp = torch.empty(n + 1, dtype=torch.int64, pin_memory=True)
        h_col = torch.empty(m, dtype=torch.int32, pin_memory=True)
        h_out = torch.empty(n, dtype=torch.int32, pin_memory=True)
        h_rp.copy_(g.row_ptr)
        h_col.copy_(g.col)
        torch.cuda.synchronize(dev)
        e_steps = max(1, min(args.steps, 3))
        # the device arena of the call is the caller's (allocated once, outside the timed region, like every other buffer of a
        # caller that refines repeatedly); the same call with the library's own cudaMalloc / cudaFree inside is timed beside it
        arena = torch.empty(wl.wl_refine_host_device_bytes(n, m), dtype=torch.uint8, device=dev)
        wl.wl_refine_host(n, h_rp, h_col, seed=5, flags=args.flags, out=h_out, device_workspace=arena)  # warm-up
        barrier()
        t0 = time.perf_counter()
        for i in range(e_steps):
            r = wl.wl_refine_host(n, h_rp, h_col, seed=200 + i, flags=args.flags, out=h_out, device_workspace=arena)
        torch.cuda.synchronize(dev)
        dt = time.perf_counter() - t0
        del arena
        torch.cuda.empty_cache()
        t1 = time.perf_counter()
        wl.wl_refine_host(n, h_rp, h_col, seed=300, flags=args.flags, out=h_out)
        torch.cuda.synchronize(dev)
        dt_own = time.perf_counter() - t1
        tt = torch.tensor([dt], dtype=torch.float64, device=dev)
        if dist is not None:
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        dt = float(tt.item())
        e2e = {"value": world * r.stats["edges_streamed"] * e_steps / dt / 1e9, "unit": "GEdges/s",
               "h2d_bytes_per_step": r.stats["bytes_h2d"], "d2h_bytes_per_step": r.stats["bytes_d2h"],
               "seconds_per_step": dt / e_steps, "steps": e_steps,
               "api": "wl_refine_host (pinned host CSR, pinned result; device arena passed in by the caller)",
               "seconds_per_step_library_allocates": dt_own}
        same = bool((h_out.to(dev) == out).all().item())
        e2e["matches_device_path"] = same
        del h_rp, h_col, h_out

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    cpu_baseline = None
    mismatches = None
    failure_bound = None
    if not args.no_cpu_baseline and world == 1:
        cb = oracle_sample(args.oracle_scale)
        cpu_baseline = {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample")}
        import oracle
        mismatches = mismatch_report(wl, gg, oracle, dev, seeds_c1=100, seeds_c3=args.mismatch_c3_seeds)
        # the failure bound of the default build on this workload: plain Algorithm 1 fails only if the
        # confirming round misses one witness pair (the paper's eps); R5 (final blocks) can make a mid-run merge permanent
        # only if the same pair of sub-blocks collides under TWO independent keys, over all N pairs of the trajectory
        npairs = split_pairs_on_device(wl, n, g.row_ptr, g.col, results[-1].rounds, dev)
        eps_paper = 2.0 ** -32 / 0.6
        eps_row32 = 2.0 ** (5 - 64) / 0.6  # rows of <= 32 unit entries: coefficient differences below 2^5
        failure_bound = {"pairs_per_round": npairs, "pairs": sum(npairs), "paper_eps_per_run": eps_paper,
                         "default_build_bound": eps_paper + sum(npairs) * eps_row32 ** 2,
                         "single_key_finality_would_be": sum(npairs) * 2.0 ** -64 / 0.6,
                         "note": "default_build_bound = paper's terminal-round eps + N x (2^(5-64)/0.6)^2 for the doubly "
                                 "confirmed final blocks; single_key_finality_would_be = the union bound of the round-1 design "
                                 "(one sum per round, odd coefficient differences)"}

    last = results[-1]
    line = {
        "metric": "refine_gedges_per_s", "value": value, "unit": "GEdges/s", "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "scaling_kind": "replicas only: every rank refines its own copy, no data-path collective (DESIGN.md section 9); not a "
                        "scaling curve of the method",
        "vs_baseline": None, "dtype": "u64", "data": "synthetic", "config": workload_config(args.scale, n, m),
        "rounds": last.rounds, "num_colors": last.num_colors, "round_colors": last.round_colors,
        "edges_streamed_per_step": edges_per_step,
        "effective_gedges_per_s": world * m * last.rounds / (ms_per_step / 1e3) / 1e9,
        "seconds_to_stable_coloring": ms_per_step / 1e3,
        "phase_ms": {"spmv": last.stats["ms_spmv"], "relabel": last.stats["ms_relabel"], "total": last.stats["ms_total"]},
        "roofline": roofline, "cpu_baseline": cpu_baseline, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
        "mismatches": mismatches, "failure_bound": failure_bound,
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
