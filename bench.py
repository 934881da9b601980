#!/usr/bin/env python
"""Benchmark of the hits -> edge-scores hot path (BASELINE.json metric: events/s per B200).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config c2]

A step is one pass of the whole path (etx_embed, etx_build_graph, etx_gnn_forward, etx_edge_scores)
over one batch of synthetic events.  `value` is measured with the inputs resident in HBM; `e2e` is
the same metric through etx_infer_host with pinned HOST buffers (H2D of the hits and D2H of the edge
list and scores inside the timed region).  Rank 0 prints ONE JSON line.

Multi-GPU (torchrun): events are independent, so every rank runs its own batch of the same
config (rank r takes event ids r*n .. (r+1)*n-1): weak scaling, no data-path collective; only the
timing is reduced (max over ranks).

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample per step.
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
sys.path.insert(0, ROOT)

from paper_2508_07423_b200 import synth  # noqa: E402

METRIC = "events/s per B200 (GNN graph build + message passing); % of tensor/HBM roofline"
NAMES = {"c2": "c2: 1000 independent events, Poisson(150) tracks, 5% noise, fp32, emb 3-128-128-128-4, "
               "GNN H=128, 6 iterations, G=3, mean out-degree 6",
         "c3": "c3: c2 inputs with bf16 MLP operands, fp32 accumulate and state",
         "c4": "c4: 1000 events, Poisson(300) tracks, 10% noise, out-degree 10, H=128, 8 iterations, fp32",
         "c1": "c1: single Run-3-occupancy event", "c0": "c0: tiny single event"}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": d["hbm_gbs"], "bf16_tflops": d["bf16_tflops"],
                "bf16_tflops_sustained": d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                "sm_max_mhz": d.get("sm_max_mhz", 1965.0), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": 1965.0,
            "source": "fallback"}


def measured_alu_peaks(local: int):
    """ALU denominators measured live by the library's microbenchmark (etx_measure_alu_peak, include/etx.h): unfused
    fp32 add+mul as scalar and as packed-pair instructions (operations/s) and FFMA (flop/s)."""
    from paper_2508_07423_b200 import binding
    return {"scalar_ops": binding.etx_measure_alu_peak(local, 0), "packed_ops": binding.etx_measure_alu_peak(local, 1),
            "ffma_flops": binding.etx_measure_alu_peak(local, 2)}


def measured_tf32_peak(dev, seconds: float = 1.5):
    """Dense TF32 tensor peak measured the way MEASURED_PEAKS.json's bf16 figure is: cuBLAS (torch.matmul on fp32 inputs
    with TF32 allowed) 8192^3, best of 10 launches (burst) and back to back for `seconds` (sustained, power-capped)."""
    import torch
    old = torch.backends.cuda.matmul.allow_tf32
    torch.backends.cuda.matmul.allow_tf32 = True
    try:
        n = 8192
        a = torch.randn(n, n, device=dev)
        b = torch.randn(n, n, device=dev)
        c = torch.empty(n, n, device=dev)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.matmul(a, b, out=c)
        best = float("inf")
        for _ in range(10):
            e0.record(); torch.matmul(a, b, out=c); e1.record(); e1.synchronize()
            best = min(best, e0.elapsed_time(e1))
        reps, t_start = 0, time.perf_counter()
        e0.record()
        while time.perf_counter() - t_start < seconds:
            for _ in range(10):
                torch.matmul(a, b, out=c)
            reps += 10
            torch.cuda.synchronize()
        e1.record(); e1.synchronize()
        sus = e0.elapsed_time(e1) / max(reps, 1)
        return {"burst": 2 * n ** 3 / (best * 1e-3) / 1e12, "sustained": 2 * n ** 3 / (sus * 1e-3) / 1e12}
    finally:
        torch.backends.cuda.matmul.allow_tf32 = old


def shard_event_ids(cfg, rank: int, n_ev: int):
    """Events are independent: rank r takes event ids r*n_ev .. (r+1)*n_ev - 1 of the config's
    stream (weak scaling, no data-path collective)."""
    return range(rank * n_ev, (rank + 1) * n_ev)


def reduce_max(value: float, device=None) -> float:
    """Max over ranks of a per-rank time (the only collective of a multi-GPU run)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_events_per_s(world: int, n_ev_per_rank: int, ms_step_max: float) -> float:
    """Whole-job throughput: all ranks' events over the slowest rank's step time."""
    return world * n_ev_per_rank / (ms_step_max * 1e-3)


def flops_mlp(dims):
    return sum(2 * dims[i] * dims[i + 1] for i in range(len(dims) - 1))


def path_flops(cfg, N, E):
    """Algorithmic FLOP of one step by kernel class."""
    H, L = cfg.gnn_hidden, cfg.gnn_mlp_hidden_layers
    hid = (H,) * L
    return {"embed": N * flops_mlp(cfg.emb_widths),
            "node_enc": N * flops_mlp((3,) + hid + (H,)),
            "edge_enc": E * flops_mlp((2 * H,) + hid + (H,)),
            "node_net": cfg.n_iter * N * flops_mlp((3 * H,) + hid + (H,)),
            "edge_net": cfg.n_iter * E * flops_mlp((3 * H,) + hid + (H,)),
            "cls": E * flops_mlp((H,) + hid + (1,)),
            "scatter": cfg.n_iter * 2 * E * H,
            "edge_proj": (cfg.n_iter + 1) * N * 2 * H * 2 * H}


def pair_tests(batch, gap):
    """Candidate pairs of the windowed search: sum over events and planes p of n_p x (n_{p+1} + .. + n_{p+gap})
    (= the edge count at r -> infinity, SURVEY 8(c) closed form)."""
    n_ev = len(batch["event_ptr"]) - 1
    if len(batch["plane"]) == 0:
        return 0
    n_pl = int(batch["plane"].max()) + 1
    ev_of = np.repeat(np.arange(n_ev), np.diff(batch["event_ptr"]))
    cnt = np.bincount(ev_of * n_pl + batch["plane"].astype(np.int64), minlength=n_ev * n_pl).reshape(n_ev, n_pl)
    return sum(int((cnt[:, :n_pl - k].astype(np.int64) * cnt[:, k:]).sum()) for k in range(1, gap + 1))


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([t.strip() for t in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()
            self.thread.join(timeout=2)

    def summary(self):
        mhz, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                mhz.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not mhz:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(mhz)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                "samples": len(mhz)}


# --------------------------------------------------------------------------------------------------
# reference arm: the oracle as it stands, on the host cores
# --------------------------------------------------------------------------------------------------
def oracle_events_per_s(cfg, event_ids, keep=None):
    from oracle import etx_oracle as orc
    batch = synth.generate_events(cfg, event_ids)
    blob = synth.generate_weights(cfg)
    layout = {s.name: (s.dims, s.offset) for s in synth.model_layout(cfg)}
    t = time.perf_counter()
    out = orc.run_path(batch, blob, layout, cfg.gnn_hidden, cfg.n_iter, synth.r2_max(cfg), cfg.max_plane_gap,
                       synth.NORM_CENTER, synth.NORM_SCALE)
    dt = time.perf_counter() - t
    if keep is not None:
        keep.update(batch=batch, out=out)
    return len(event_ids) / dt, dt, len(batch["r"]), len(out["src"])


CDF_AT = [1e-7, 1e-6, 1e-5, 1e-4, 1e-3, 1e-2, 2e-2, 5e-2]


def compare_with_oracle(gpu, ora, event_ptr=None):
    """End-to-end comparison of one GPU run with the oracle's on the same events (reading Q16): the edge sets
    (symmetric difference: the two embeddings decide pairs near the radius differently) and the score error on the common edges
    with its CDF and the oracle's score histogram (reading Q14)."""
    n = int(max(gpu["src"].max(initial=0), gpu["dst"].max(initial=0), ora["src"].max(initial=0), ora["dst"].max(initial=0))) + 1
    kg = gpu["src"].astype(np.int64) * n + gpu["dst"]
    ko = ora["src"].astype(np.int64) * n + ora["dst"]
    common, ig, io = np.intersect1d(kg, ko, assume_unique=True, return_indices=True)
    d = np.abs(gpu["scores"][ig].astype(np.float64) - np.asarray(ora["scores"], np.float64)[io])
    hist, _ = np.histogram(np.asarray(ora["scores"], np.float64), bins=10, range=(0.0, 1.0))
    same = {}
    if event_ptr is not None:
        # the tolerance is defined on identical graphs: the events in which both sides found exactly the same edges
        ep = np.asarray(event_ptr, np.int64)
        ev_of = lambda hits: np.searchsorted(ep, hits, side="right") - 1
        only = np.concatenate([np.setdiff1d(kg, common), np.setdiff1d(ko, common)]) // n
        bad = np.unique(ev_of(only)) if len(only) else np.zeros(0, np.int64)
        keep = ~np.isin(ev_of(common // n), bad)
        same = {"events_with_identical_graphs": int(len(ep) - 1 - len(bad)),
                "score_err_on_identical_graphs": {"edges": int(keep.sum()), "max": float(d[keep].max(initial=0.0)),
                                                  "p99": float(np.quantile(d[keep], 0.99)) if keep.any() else 0.0}}
    return {**same, "edges_gpu": int(len(kg)), "edges_oracle": int(len(ko)), "common": int(len(common)),
            "only_gpu": int(len(kg) - len(common)), "only_oracle": int(len(ko) - len(common)),
            "score_err_on_common": {"max": float(d.max(initial=0.0)), "p99": float(np.quantile(d, 0.99)) if len(d) else 0.0,
                                    "median": float(np.median(d)) if len(d) else 0.0},
            "score_err_cdf": {f"{t:g}": float(np.mean(d <= t)) if len(d) else 1.0 for t in CDF_AT},
            "oracle_score_hist_0_to_1_by_0.1": [float(x) / max(len(ko), 1) for x in hist]}


def oracle_single_thread(config: str):
    """The same oracle on event 0 alone with ONE OpenMP thread (a fresh process: the thread count is read at load)."""
    code = ("import json, bench, sys; from paper_2508_07423_b200 import synth; "
            f"v, dt, nh, ne = bench.oracle_events_per_s(synth.CONFIGS[{config!r}], [0]); "
            "print(json.dumps({'value': v, 'unit': 'events/s', 'cores': 1, 'sample': f'event 0 ({nh} hits, {ne} edges) in {dt:.1f} s'}))")
    try:
        out = subprocess.run([sys.executable, "-c", code], cwd=ROOT, env=dict(os.environ, OMP_NUM_THREADS="1"),
                             capture_output=True, text=True, timeout=600)
        return json.loads(out.stdout.strip().splitlines()[-1])
    except Exception as e:  # noqa: BLE001
        return {"unavailable": str(e)[:200]}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import etx_oracle as orc
    cfg = synth.CONFIGS[args.config]
    per_step = 2
    for w in range(args.warmup):
        oracle_events_per_s(cfg, [w * per_step + i for i in range(per_step)])
    t_tot, n_ev = 0.0, 0
    for k in range(args.steps):
        _, dt, _, _ = oracle_events_per_s(cfg, [(args.warmup + k) * per_step + i for i in range(per_step)])
        t_tot += dt
        n_ev += per_step
    v = n_ev / t_tot
    sample = f"{per_step} events of {args.config} per step ({n_ev} timed), oracle/etx_oracle.cpp, OpenMP over rows"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": "events/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_tot / max(args.steps, 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": NAMES[args.config], "sample": sample},
        "cpu_baseline": {"value": v, "unit": "events/s", "cores": orc.n_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


# --------------------------------------------------------------------------------------------------
# our arm
# --------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2508_07423_b200 import binding, build

    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    build.build()

    cfg = synth.CONFIGS[args.config]
    if args.tracks_mean > 0:
        import dataclasses
        cfg = dataclasses.replace(cfg, tracks_mean=args.tracks_mean)
    n_ev = args.events or cfg.n_events
    batch = synth.generate_events(cfg, shard_event_ids(cfg, rank, n_ev))
    blob = synth.generate_weights(cfg)
    etx = binding.Etx(binding.make_desc(cfg, precision=args.precision if args.precision is not None else cfg.precision),
                      blob, device=local)
    if int(etx.desc.precision) in (synth.PREC_INT8, synth.PREC_FP8):     # next row NEXT-3 as the whole step: needs the stored calibrated ranges
        etx.etx_set_int8_ranges(synth.int8_gnn_alpha(cfg))
    r2, gap, H = synth.r2_max(cfg), cfg.max_plane_gap, cfg.gnn_hidden
    N = len(batch["r"])
    cap = int(N * (cfg.target_degree * (1.25 if args.tracks_mean <= 0 else 4.0) + 2))   # r^2 is calibrated at the config's occupancy
    db = binding.DeviceBatch(batch, dev)
    etx.ensure_workspace(db.n_events, N, cap, with_host_path=True)
    g = binding.DeviceGraph(N, cap, dev)
    emb = torch.empty(N, etx.emb_dim, device=dev)
    enc = torch.empty(cap, H, device=dev)
    scores = torch.empty(cap, device=dev)

    def step():
        etx.etx_embed(db, emb)
        E = etx.etx_build_graph(db, emb, r2, gap, g)
        etx.etx_gnn_forward(db, g, enc)
        etx.etx_edge_scores(g, enc, scores)
        return E

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        E = step()
    barrier()
    etx.profile_enable(True)
    etx.profile_read()
    l0 = etx.launch_count()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clk:
        barrier()
        t0.record()
        for _ in range(args.steps):
            E = step()
        t1.record()
        barrier()
    ms = t0.elapsed_time(t1)
    launches = etx.launch_count() - l0
    prof = etx.profile_read()
    etx.profile_enable(False)
    ms = reduce_max(ms, dev)
    ms_step = ms / args.steps
    value = aggregate_events_per_s(world, n_ev, ms_step)

    # ---- next rows beyond the step (reported separately, not part of `value`)
    next_rows = {}

    def time3(fn):
        fn()
        barrier()
        t0.record()
        for _ in range(3):
            r = fn()
        t1.record()
        barrier()
        return t0.elapsed_time(t1) / 3, r

    if not args.no_next_rows:
        # NEXT-1: score cut + WCC tracks
        labels = torch.empty(max(N, 1), dtype=torch.int32, device=dev)
        wcc_ms, _ = time3(lambda: etx.etx_build_tracks(db, g, scores, 0.5, labels))
        sizes = torch.bincount(labels[:N].long(), minlength=1)
        next_rows["wcc_tracks"] = {"ms": wcc_ms, "events_per_s": n_ev / (wcc_ms * 1e-3), "score_min": 0.5,
                                   "components_ge3_hits": int((sizes >= 3).sum().item())}
        # NEXT-4 (triplet part): triplet building on the same purified graph
        tr = etx.etx_build_triplets(db, g, scores, 0.5)
        n_tr = [int(tr[k].shape[0]) for k in ("articulation", "left_elbow", "right_elbow")]
        del tr
        tms, _ = time3(lambda: etx.etx_build_triplets(db, g, scores, 0.5, capacity=sum(n_tr)) and None)
        next_rows["triplets"] = {"ms": tms, "events_per_s": n_ev / (tms * 1e-3), "score_min": 0.5,
                                 "articulations": n_tr[0], "left_elbows": n_tr[1], "right_elbows": n_tr[2],
                                 "rows_per_s": sum(n_tr) / (tms * 1e-3)}
        # NEXT-2: k_max-capped search (the thesis' k_max = 50, which rarely binds, and a cap that does)
        g2 = binding.DeviceGraph(N, cap, dev)
        for kk in (50, 4):
            kms, Ek = time3(lambda: etx.etx_build_graph(db, emb, r2, gap, g2, k_max=kk))
            next_rows[f"graph_kmax_{kk}"] = {"ms": kms, "events_per_s": n_ev / (kms * 1e-3), "n_edges": int(Ek)}
        del g2
        # NEXT-3 (embedding part): INT8 embedding MLP with the stored calibrated ranges, and the graph it gives
        al = synth.int8_act_alpha(cfg)
        emb8 = torch.empty_like(emb)
        ims, _ = time3(lambda: etx.etx_embed_int8(db, al, emb8))
        g3 = binding.DeviceGraph(N, int(cap * 1.5), dev)
        E8 = etx.etx_build_graph(db, emb8, r2, gap, g3)
        next_rows["embed_int8"] = {"ms": ims, "events_per_s": n_ev / (ims * 1e-3), "fp32_embed_ms": stages_embed_ms(prof, args.steps),
                                   "n_edges": int(E8), "edges_vs_fp32": E8 / max(int(E), 1)}
        del g3, emb8
        # NEXT-4 (rest): triplet classifiers on the final edge encodings, then track building from triplets
        etx.etx_set_triplet_classifiers(synth.generate_triplet_weights(cfg))
        tr = etx.etx_build_triplets(db, g, scores, 0.5)
        cms, ts = time3(lambda: etx.etx_triplet_scores(g, enc, tr))
        n_rows = sum(int(x) for x in tr["c"].n)
        next_rows["triplet_scores"] = {"ms": cms, "events_per_s": n_ev / (cms * 1e-3), "triplets": n_rows,
                                       "triplets_per_s": n_rows / (cms * 1e-3), "kept_at_0.5": int((ts["all"][:n_rows] >= 0.5).sum().item())}
        ws_before = etx._ws_bytes
        tms, tk = time3(lambda: etx.etx_build_tracks_from_triplets(db, g, scores, 0.5, tr, ts["all"], 0.5))
        next_rows["tracks_from_triplets"] = {"ms": tms, "events_per_s": n_ev / (tms * 1e-3), "score_min": 0.5, "triplet_min": 0.5,
                                             "tracks": int(tk["track_ptr"].numel() - 1), "joins": int(tk["joins"].shape[0]),
                                             "hit_entries": int(tk["track_hits"].numel()),
                                             "note": "two calls per run (count, then fill) as the binding sizes its buffers"}
        del tr, ts, tk
        if etx._ws_bytes != ws_before:                 # the track building may have grown (and clobbered) the workspace
            etx.ensure_workspace(db.n_events, N, cap, with_host_path=True)

    if not args.no_next_rows and H == 128:
        # NEXT-3 (GNN part): the same graph through the quantised GNNs -- INT8 (ETX_PREC_INT8, tcgen05.mma.kind::i8) and FP8 e4m3
        # (ETX_PREC_FP8, kind::f8f6f4) -- with the stored calibrated ranges; the default mode's scores of this run are the comparison
        ref_scores = scores[:E].clone()
        default_gnn_ms = sum(prof[k][0] for k in ("node_enc", "edge_enc", "scatter", "node_net", "edge_net", "edge_proj", "cls")) / args.steps
        for row, qprec in (("gnn_int8", synth.PREC_INT8), ("gnn_fp8", synth.PREC_FP8)):
            q = binding.Etx(binding.make_desc(cfg, precision=qprec), blob, device=local)
            q.etx_set_int8_ranges(synth.int8_gnn_alpha(cfg))
            q.ensure_workspace(db.n_events, N, cap)
            sc8 = torch.empty(cap, device=dev)

            def q_step():
                q.etx_gnn_forward(db, g, enc)
                q.etx_edge_scores(g, enc, sc8)

            q.profile_enable(True)
            q.profile_read()
            qms, _ = time3(q_step)
            qprof = q.profile_read()
            d8 = (sc8[:E] - ref_scores).abs()
            next_rows[row] = {"ms": qms, "events_per_s": n_ev / (qms * 1e-3), "default_mode_gnn_ms": default_gnn_ms,
                              "speed_vs_default_mode": default_gnn_ms / qms,
                              "edge_net_ms_per_launch": qprof["edge_net"][0] / max(qprof["edge_net"][1], 1),
                              "stages_ms": {k: v[0] / 4 for k, v in qprof.items() if v[1]},
                              "score_err_vs_default_mode": {"max": float(d8.max()), "median": float(d8.median()),
                                                            "p99": float(torch.quantile(d8[::16].float(), 0.99))},
                              "kept_edges_at_0.5": {row[4:]: int((sc8[:E] >= 0.5).sum()), "default": int((ref_scores >= 0.5).sum())}}
            del q, sc8
        del ref_scores

    # ---- end to end through the host-buffer entry point
    host = binding.pinned_host_batch(batch)
    o_src = torch.empty(cap, dtype=torch.int32).pin_memory()
    o_dst = torch.empty(cap, dtype=torch.int32).pin_memory()
    o_sc = torch.empty(cap, dtype=torch.float32).pin_memory()
    etx.etx_infer_host(host, r2, gap, cap, o_src, o_dst, o_sc)
    barrier()
    e2e_steps = args.steps                       # the same number of timed steps as `value`
    w0 = time.perf_counter()
    t0.record()
    for _ in range(e2e_steps):
        E2 = etx.etx_infer_host(host, r2, gap, cap, o_src, o_dst, o_sc)
    t1.record()
    barrier()
    e2e_ms = max(t0.elapsed_time(t1), 1e3 * (time.perf_counter() - w0)) / e2e_steps
    e2e_ms = reduce_max(e2e_ms, dev)
    h2d = sum(host[k].numel() * host[k].element_size() for k in host)
    d2h = E2 * 12

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    pk = peaks()
    fl = path_flops(cfg, N, E)
    stages = {}
    for k, (kms, kn) in prof.items():
        per = kms / args.steps
        stages[k] = {"ms": per, "launches": kn // max(args.steps, 1),
                     "events_per_s": (n_ev / (per * 1e-3)) if per > 0 else None}
        if k in fl and per > 0:
            stages[k]["tflops"] = fl[k] / (per * 1e-3) / 1e12
    # scatter-sum algorithmic bytes (e read once when both sums come from one pass -- the second
    # use of a row is an L2 hit by construction, scatter.cu) + in_perm + write of m, per iteration
    sc_bytes = cfg.n_iter * (E * H * 4 + 4 * E + N * 2 * H * 4 + 8 * (N + 1))
    if stages["scatter"]["ms"] > 0:
        stages["scatter"]["gbs"] = sc_bytes / (stages["scatter"]["ms"] * 1e-3) / 1e9
        stages["scatter"]["hbm_frac"] = stages["scatter"]["gbs"] / pk["hbm_gbs"]
    # graph build (a2): the windowed all-pairs test is bound by plain fp32 ALU work, not by HBM: report
    # both.  Pair tests = sum over events and planes p of n_p x (n_{p+1} + .. + n_{p+G}); 3d flop each (d subtractions,
    # d multiplications, d-1 additions and the comparison, individually rounded: no FMA); the kernels sweep the
    # candidates twice (count pass, fill pass).  Bytes: embeddings + plane ids read, both CSR structures written.
    if stages["graph"]["ms"] > 0:
        pairs = pair_tests(batch, gap)
        d_emb = cfg.emb_widths[-1]
        t_s = stages["graph"]["ms"] * 1e-3
        alu = measured_alu_peaks(local)
        alu_peak = alu["packed_ops"] if d_emb == 4 else alu["scalar_ops"]     # unfused fp32 operations per second, measured
        g_bytes = N * (4 * d_emb + 1) + 2 * (4 * (N + 1) + 8 * E)
        stages["graph"].update({"pair_tests": pairs, "pair_tests_per_s": pairs / t_s,
                                "alu_frac": pairs * 3 * d_emb / t_s / alu_peak,
                                "alu_frac_executed": 2 * pairs * 3 * d_emb / t_s / alu_peak,
                                "gbs": g_bytes / t_s / 1e9, "hbm_frac": g_bytes / t_s / 1e9 / pk["hbm_gbs"],
                                "alu_peak_ops_per_s": alu_peak,
                                "bound": "alu (fp32 add/mul, unfused, %s): measured by etx_measure_alu_peak; nominal 148 SM x 128 lanes x "
                                         "%.0f MHz = %.3g/s" % ("packed pairs" if d_emb == 4 else "scalar", pk["sm_max_mhz"],
                                                                148 * 128 * pk["sm_max_mhz"] * 1e6)})
    gnn_ms = sum(stages[k]["ms"] for k in ("node_enc", "edge_enc", "scatter", "node_net", "edge_net", "edge_proj"))
    stages["message_passing_total"] = {"ms": gnn_ms, "events_per_s": n_ev / (gnn_ms * 1e-3) if gnn_ms else None}

    # ---- roofline of the dominant kernel: the edge network (a6)
    # achieved = ALGORITHMIC flop (10 H^2 per edge and step) / mean launch duration.  The
    # tensor-core modes execute a different count: the first layer is factorised (per-hit projections
    # run in the edge_proj launches, the edge kernel keeps 6 H^2 per edge) and the split modes issue 3
    # MMAs per product; that executed rate is reported next to it as `executed`.
    en = prof["edge_net"]
    per_launch_ms = en[0] / max(en[1], 1)
    per_launch_flop = fl["edge_net"] / cfg.n_iter
    achieved = per_launch_flop / (per_launch_ms * 1e-3) / 1e12 if per_launch_ms > 0 else 0.0
    prec = int(etx.desc.precision)
    L = cfg.gnn_mlp_hidden_layers
    mma_flop = E * flops_mlp((H,) + (H,) * L + (H,))          # per launch, factorised first layer
    if prec == synth.PREC_FP32:
        # FFMA: measured by the library's microbenchmark (nominal: 148 SMs x 128 fp32 lanes x 2 FLOP x max SM clock)
        peak = measured_alu_peaks(local)["ffma_flops"] / 1e12
        roof = {"bound": "alu", "unit": "TFLOP/s", "peak": peak,
                "peak_source": "measured FFMA microbenchmark (etx_measure_alu_peak); nominal 148 SM x 128 lanes x 2 x %.0f MHz = %.1f"
                               % (pk["sm_max_mhz"], 148 * 128 * 2 * pk["sm_max_mhz"] * 1e6 / 1e12)}
        dtype, passes, mma_flop = "f32", 1, per_launch_flop
    elif prec == synth.PREC_TF32X3:
        tf = measured_tf32_peak(dev)
        peak = tf["sustained"]
        roof = {"bound": "tensor", "unit": "TFLOP/s", "peak": peak,
                "peak_source": "measured in this run: cuBLAS TF32 8192^3 sustained (burst %.0f; bf16 sustained x 0.5 nominal ratio = %.0f)"
                               % (tf["burst"], pk["bf16_tflops_sustained"] * 0.5)}
        dtype, passes = "tf32x3", 3
    elif prec == synth.PREC_BF16X3:
        peak = pk["bf16_tflops_sustained"]
        roof = {"bound": "tensor", "unit": "TFLOP/s", "peak": peak, "peak_source": f"{pk['source']} bf16 sustained"}
        dtype, passes = "bf16x3", 3
    elif prec in (synth.PREC_INT8, synth.PREC_FP8):
        peak = pk["bf16_tflops_sustained"] * 2.0
        roof = {"bound": "tensor", "unit": "TOP/s" if prec == synth.PREC_INT8 else "TFLOP/s", "peak": peak,
                "peak_source": f"{pk['source']} bf16 sustained x 2 (8-bit nominal ratio)"}
        dtype, passes = ("i8" if prec == synth.PREC_INT8 else "f8e4m3"), 1
    else:
        peak = pk["bf16_tflops_sustained"]
        roof = {"bound": "tensor", "unit": "TFLOP/s", "peak": peak, "peak_source": f"{pk['source']} bf16 sustained"}
        dtype, passes = "bf16", 1
    executed = passes * mma_flop / (per_launch_ms * 1e-3) / 1e12 if per_launch_ms > 0 else 0.0
    # Algorithmic bytes of one edge-network launch: e read + reduce-add into e, the src/dst indices,
    # every row of the per-hit projections p once.  Single-pass bf16 with fp32 state sits below the ridge
    # ("bf16 MMA + fp32 state is HBM-bound"), so that mode reports the HBM roofline; the tensor figures
    # stay under `executed` / `tensor`.
    alg_bytes = 2 * E * H * 4 + 8 * E + N * 2 * H * 4
    gbs = alg_bytes / (per_launch_ms * 1e-3) / 1e9 if per_launch_ms > 0 else 0.0
    roof["hbm"] = {"algorithmic_bytes": alg_bytes, "gbs": gbs, "frac": gbs / pk["hbm_gbs"]}
    if prec == synth.PREC_BF16:
        roof["tensor"] = {"achieved": achieved, "peak": peak, "frac": achieved / peak, "peak_source": roof["peak_source"]}
        roof.update({"bound": "hbm", "unit": "GB/s", "peak_source": f"{pk['source']} HBM"})
        achieved, peak_t, peak = gbs, peak, pk["hbm_gbs"]
        roof["peak"] = peak
    else:
        peak_t = peak
    roof.update({"kernel": "edge network (a6)", "achieved": achieved, "frac": achieved / peak,
                 "ms_per_launch": per_launch_ms,
                 # the committed capture is of config c2, full size, default precision: null for anything else
                 "traffic": read_traffic() if (args.config == "c2" and not args.events and args.tracks_mean <= 0
                                               and prec == synth.PREC_BF16X3) else None,
                 "executed": {"tflops": executed, "frac": executed / peak_t,
                              "note": "flop the kernel issues: %d MMA pass(es) x %s" %
                                      (passes, "10 H^2 per edge" if prec == synth.PREC_FP32 else
                                       "6 H^2 per edge (first layer factorised; the per-hit part runs in edge_proj)")}})

    # ---- CPU baseline: the oracle on a bounded sample, rank 0, N=1 only
    cpu, parity = None, None
    if world == 1 and not args.no_cpu_baseline:
        from oracle import etx_oracle as orc
        _, dt1, _, _ = oracle_events_per_s(cfg, [0])
        n_s = int(min(32, max(2, round(15.0 / max(dt1, 1e-3)))))
        kept = {}
        v, dt, nh, ne = oracle_events_per_s(cfg, list(range(n_s)), keep=kept)
        # parity on the same sample, end to end (the GPU's own embedding and graph): every config / mode that is benched
        # carries its comparison with the oracle in the line
        gpu_s = binding.run_path(etx, kept["batch"], r2, gap, edge_capacity=int(nh * (cfg.target_degree * 1.25 + 2)))
        parity = {"sample": f"first {n_s} events of {args.config}, end to end (GPU embedding and graph) against the oracle",
                  "note": "the gate is defined on identical graphs (tests/, profiles/r02_parity.md); end to end the few edges only one "
                          "side has (pairs within 1e-5 of the radius) also move the scores of their neighbours, which is what the "
                          "maximum shows when only_gpu + only_oracle > 0",
                  "gate": {synth.PREC_BF16: 2e-2, synth.PREC_INT8: None, synth.PREC_FP8: None}.get(int(etx.desc.precision), 1e-4),
                  **compare_with_oracle(gpu_s, kept["out"], kept["batch"]["event_ptr"])}
        if H == 128 and int(etx.desc.precision) != synth.PREC_FP32:
            # reading Q16's report: the same events with a bf16 EMBEDDING (etx_embed_bf16) -- which edges change, and the
            # score error on the edges both graphs have
            gpu_b = binding.run_path(etx, kept["batch"], r2, gap, edge_capacity=int(nh * (cfg.target_degree * 1.25 + 2) * 2),
                                     embed="etx_embed_bf16")
            next_rows["bf16_embedding_end_to_end"] = {
                "note": "report only (reading Q16): the step with etx_embed_bf16 instead of the 3xTF32 embedding, same radius",
                **compare_with_oracle(gpu_b, kept["out"], kept["batch"]["event_ptr"])}
        cpu = {"value": v, "unit": "events/s", "cores": orc.n_threads(), "kind": "oracle",
               "sample": f"first {n_s} events of {args.config} ({nh} hits, {ne} edges) in {dt:.1f} s",
               "note": "the oracle is deliberately unoptimised (per-neuron loops, double accumulators, no BLAS/SIMD, OpenMP "
                       "over rows): a reported baseline, not a tuned CPU implementation",
               "single_thread": oracle_single_thread(args.config)}

    print(json.dumps({
        "metric": METRIC, "value": value, "unit": "events/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": dtype, "data": "synthetic",
        "config": {"workload": NAMES[args.config] + (f" [tracks_mean overridden to {args.tracks_mean:g}]" if args.tracks_mean > 0 else ""),
                   "n_events_per_gpu": n_ev, "n_hits": N, "n_edges": int(E),
                   "mean_out_degree": E / max(N, 1), "r2_max": r2, "hits_per_s": world * N / (ms_step * 1e-3),
                   "l2": "state larger than L2 (edge encodings %.1f GB), no flush needed" % (E * H * 4 / 1e9),
                   "parallelism": "events sharded across GPUs, no collective" if world > 1 else "single GPU",
                   **({"precision_note": "per-edge MLP chains single-pass bf16; per-hit MLPs and the classifier run the bf16x3 split "
                                         "(every edge of c3 then holds the 2e-2 gate, DESIGN.md section 6)"} if dtype == "bf16" else {})},
        "roofline": roof, "cpu_baseline": cpu, "parity": parity,
        "e2e": {"value": aggregate_events_per_s(world, n_ev, e2e_ms), "unit": "events/s", "h2d_bytes_per_step": int(h2d),
                "d2h_bytes_per_step": int(d2h), "ms_per_step": e2e_ms},
        "gpu_launches": int(launches), "clocks": clk.summary(), "stages": stages, "next_rows": next_rows}))
    if world > 1:
        dist.destroy_process_group()


def stages_embed_ms(prof, steps):
    return prof["embed"][0] / max(steps, 1)


def read_traffic():
    """DRAM bytes per launch of the dominant kernel from the committed ncu summary (or null)."""
    p = os.path.join(ROOT, "profiles", "edge_net_traffic.txt")
    if not os.path.exists(p):
        return None
    for line in open(p):
        if line.startswith("dram_bytes_per_launch"):
            try:
                return float(line.split("=")[1])
            except ValueError:
                return None
    return None


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="c2", choices=sorted(synth.CONFIGS))
    ap.add_argument("--events", type=int, default=0, help="events per GPU (default: the config's)")
    ap.add_argument("--precision", type=int, default=None, help="override etx_precision (0 fp32, 1 tf32x3, 2 bf16, 3 bf16x3, 4 int8, 5 fp8 e4m3)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-next-rows", action="store_true", help="skip the next-row timings (launch lists of the step only)")
    ap.add_argument("--tracks-mean", type=float, default=0.0,
                    help="override the config's mean tracks per event (occupancy sweep, cf. thesis Figs. 9.11-9.13)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
