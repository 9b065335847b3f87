#!/usr/bin/env python
"""bench.py -- candidates scored/sec of the FusionANNS GPU stage on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl ours|reference]

A step = one pass of the whole hot path (lookup table + dedup + code gather/ADC + top-k)
over one batch of synthetic queries.  Prints ONE JSON line.
The path does not shard (north star: one GPU, no collectives): with --gpus N > 1 every
rank runs an independent replica on its own batch ("replicas only").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

DEFAULT_WORKLOAD = "u8_1b_m64"          # BASELINE.json configs[4]: the largest 1B-vector config, fits one B200
METRIC = "candidates scored/sec (dedup+ADC+top-k)"
UNIT = "candidates/s"
L2_BYTES = 126 << 20


def measured_peak_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.rows, self.proc, self.thread = [], None, None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20",
                 "-i", str(gpu_index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for t, r in self.rows if t0 <= t <= t1 + 0.2] or [r for _, r in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); smax = float(f[1])
            except Exception:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": smax, "reasons": sorted(reasons),
                "samples": len(sm)}


def sample_inputs(w, n_queries: int, codes_dev):
    """Host-side inputs of the first n_queries queries for the CPU oracle.  The code rows the sample touches
    are fetched to the host and the IDs relabelled monotonically onto that compact array (the oracle's
    (dist, id) order is unchanged; tests/test_oracle_pins.py pins this relabelling).  `used` maps back."""
    import numpy as np
    import torch
    off = w.cand_offsets[: n_queries + 1].cpu().numpy()
    ids_dev = w.cand_ids[: int(off[-1])]
    used = torch.unique(ids_dev)                                   # ascending int32 (IDs < 2^31)
    rows = codes_dev[used.long()].cpu().numpy()
    rel = torch.searchsorted(used, ids_dev).to(torch.int32).cpu().numpy().view(np.uint32)
    return {"q": w.queries[:n_queries].cpu().numpy(), "cb": w.codebooks.cpu().numpy(), "rows": rows, "off": off,
            "rel": rel, "used": used.cpu().numpy().view(np.uint32)}


def oracle_sample(w, n_queries: int, codes_dev, nthreads: int = 0):
    """Run the CPU oracle on the first n_queries queries.
    Returns (seconds, result dict with ids mapped back, units scored)."""
    import oracle
    s = sample_inputs(w, n_queries, codes_dev)
    t0 = time.perf_counter()
    r = oracle.search(s["q"], s["cb"], s["rows"], s["off"], s["rel"], w.cfg.k, N=s["rows"].shape[0], nthreads=nthreads)
    dt = time.perf_counter() - t0
    ids = r["ids"].copy()
    valid = ids != 0xFFFFFFFF
    ids[valid] = s["used"][ids[valid]]
    r["ids"] = ids
    return dt, r, int(r["uniq"].sum())


def band_check_sample(w, n_queries: int, codes_dev, gpu_out):
    """Tolerance-regime parity (oracle/parity.py check_band) of the first n_queries queries of a batch the
    GPU has answered; gpu_out = (ids, dists, counts, uniq) device tensors.  Returns how many needed the band."""
    import numpy as np
    import oracle
    from oracle.parity import check_band
    s = sample_inputs(w, n_queries, codes_dev)
    gi = gpu_out[0][:n_queries].cpu().numpy().view(np.uint32)
    gd = gpu_out[1][:n_queries].cpu().numpy()
    gc = gpu_out[2][:n_queries].cpu().numpy().view(np.uint32)
    gu = gpu_out[3][:n_queries].cpu().numpy().view(np.uint32)
    needed = 0
    for b in range(n_queries):
        ai, ad = oracle.query_all(s["q"][b], s["cb"], s["rows"], s["rel"][s["off"][b]:s["off"][b + 1]], N=s["rows"].shape[0])
        assert gu[b] == ai.size, f"query {b}: {gu[b]} distinct candidates, the oracle has {ai.size}"
        needed += int(check_band(gi[b], gd[b], gc[b], s["used"][ai], ad, w.cfg.k))
    return needed


def aggregate_over_ranks(total_ms: float, units: float, inputs: float, device=None):
    """Replicas only: the job's time is the MAX over ranks, its work the SUM.  Uses the
    default process group if one is initialised (nccl on GPUs; gloo in the CPU test), else passes through."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(total_ms), float(units), float(inputs)
    t = torch.tensor([total_ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    u = torch.tensor([units, inputs], dtype=torch.float64, device=device)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u[0].item()), float(u[1].item())


def rank_seed(base_seed: int, rank: int) -> int:
    """Every replica scores its own batch: rank r draws its workload from seed base + r."""
    return base_seed + rank


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD)
    ap.add_argument("--cpu-queries", type=int, default=0, help="oracle sample size (0 = auto, ~10-30 s)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--id-map", default=None, choices=["feistel", "lattice"],
                    help="vector -> ID map of the generator (default: the config's, 'feistel')")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)

    import numpy as np
    import torch
    from workloads import CONFIGS, DEFAULT_SEED, make_workload

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    cfg = CONFIGS[args.workload]
    if args.id_map:
        cfg = cfg.scaled(id_map=args.id_map)

    if args.impl == "reference":
        return reference_arm(args, cfg, rank, world)

    assert torch.cuda.is_available(), "bench.py needs a CUDA device: there is no CPU fallback"
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(dev))
    import paper_2409_16576_b200 as fann
    from paper_2409_16576_b200.build import build
    build()

    t_gen = time.time()
    w = make_workload(cfg, seed=rank_seed(DEFAULT_SEED, rank), device=dev)     # each replica: its own batch
    torch.cuda.synchronize()
    t_gen = time.time() - t_gen
    B, k, M, dsub = cfg.B, cfg.k, cfg.M, cfg.dsub
    total = int(w.cand_ids.numel())

    ix = fann.FannIndex(local_rank)
    ix.load_codes(w.codes)
    lut = torch.empty((B, M, 256), dtype=torch.float32, device=dev)
    out = (torch.empty((B, k), dtype=torch.int32, device=dev), torch.empty((B, k), dtype=torch.float32, device=dev),
           torch.empty(B, dtype=torch.int32, device=dev), torch.empty(B, dtype=torch.int32, device=dev))
    ws = ix.workspace(B, total, k)
    stream = torch.cuda.current_stream().cuda_stream

    def step():
        fann.fann_build_lut(ix.handle, w.queries, B, w.codebooks, dsub, lut, stream)
        fann.fann_dedup_scan_topk(ix.handle, lut, B, w.cand_offsets, w.cand_ids, total, k,
                                  out[0], out[1], out[2], out[3], ws, ws.numel(), stream)

    # working set per step vs L2: flush between timed iterations when it could stay resident
    U_guess_bytes = total * 4 + B * M * 1024
    flush = None
    if U_guess_bytes + total * M < 4 * L2_BYTES:
        flush = torch.empty(2 * L2_BYTES, dtype=torch.uint8, device=dev)

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    fann.fann_workspace_status(ix.handle, ws, stream)
    U_total = int(out[3].sum().item())

    fann.fann_set_timing(ix.handle, True)
    launches0 = ix.info()["kernel_launches"]
    sampler = ClockSampler(local_rank) if rank == 0 else None
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kern = {"lut_ms": [], "plan_ms": [], "dedup_ms": [], "scan_ms": []}
    barrier()
    t0 = time.time()
    for i in range(args.steps):
        if flush is not None:
            flush.fill_(i & 0xFF)
        ev[i][0].record()
        step()
        ev[i][1].record()
        ev[i][1].synchronize()
        for kk, v in fann.fann_last_timing(ix.handle).items():
            kern[kk].append(v)
    barrier()
    t1 = time.time()
    fann.fann_workspace_status(ix.handle, ws, stream)               # raises if any timed step overflowed a table
    launches = ix.info()["kernel_launches"] - launches0
    fann.fann_set_timing(ix.handle, False)
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = float(sum(step_ms))
    clocks = sampler.stop(t0, t1) if sampler else None
    total_ms, U_all, C_all = aggregate_over_ranks(total_ms, U_total, total, device=dev)
    ms_per_step = total_ms / args.steps
    value = U_all / (ms_per_step * 1e-3)

    # ---- roofline of the dominant kernel (scan: dedup + gather + ADC + local top-k)
    peak, peak_src = measured_peak_gbs()
    # scan kernel's own algorithmic bytes: code rows + distinct IDs + tables + outputs
    algo_bytes = M * U_total + 4 * U_total + 1024 * M * B + 8 * k * B
    path_bytes = algo_bytes + 4 * total + 4 * U_total                          # + dedup: IDs read, distinct IDs written
    scan_ms = float(np.mean(kern["scan_ms"]))
    achieved = algo_bytes / (scan_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": "scan_kernel", "achieved": round(achieved, 1), "peak": peak,
                "unit": "GB/s", "frac": round(achieved / peak, 4),
                # dram__bytes_read+write of this kernel per gathered row, measured by ncu on this very workload
                # (profiles/r1k_launches_u8_1b_m64.md: 50.56 GB for 7.322e8 rows of 64 bytes = 69.05 B/row); the
                # figure is per launch like `achieved`; null for other row sizes (not captured)
                "traffic": int(69.05 * U_total) if M > 32 else None,
                "peak_source": peak_src, "algorithmic_bytes": algo_bytes, "kernel_ms": round(scan_ms, 4),
                "code_bytes_only_frac": round(M * U_total / (scan_ms * 1e-3) / 1e9 / peak, 4),
                "share_of_step": round(scan_ms / ms_per_step, 4),
                "kernels_ms": {kk: round(float(np.mean(v)), 4) for kk, v in kern.items()}}

    if rank != 0:
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        return

    # ---- e2e: same metric through the C ABI with HOST buffers (copies inside the timed region)
    e2e = None
    if not args.no_e2e:
        need = fann.fann_search_host_scratch_bytes(ix.handle, B, dsub, total, k)
        del ws
        ix._ws = None
        torch.cuda.empty_cache()
        scratch = torch.empty(need, dtype=torch.uint8, device=dev)
        q_h, off_h, ids_h = w.queries.cpu().pin_memory(), w.cand_offsets.cpu().pin_memory(), w.cand_ids.cpu().pin_memory()
        oi = torch.empty((B, k), dtype=torch.int32).pin_memory()
        od = torch.empty((B, k), dtype=torch.float32).pin_memory()
        oc = torch.empty(B, dtype=torch.int32).pin_memory()

        def host_step():
            fann.fann_search_host(ix.handle, q_h, B, w.codebooks, dsub, off_h, ids_h, k, oi, od, oc, scratch, need, stream)

        for _ in range(2):
            host_step()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(args.steps):
            host_step()
        b.record()
        b.synchronize()
        e_ms = a.elapsed_time(b) / args.steps
        same = bool(np.array_equal(oi.numpy(), out[0].cpu().numpy()))
        e2e = {"value": U_total / (e_ms * 1e-3), "unit": UNIT, "ms_per_step": round(e_ms, 3),
               "h2d_bytes_per_step": int(q_h.numel() * 4 + off_h.numel() * 8 + ids_h.numel() * 4),
               "d2h_bytes_per_step": int(oi.numel() * 4 + od.numel() * 4 + oc.numel() * 4),
               "matches_device_path": same}
        del scratch, q_h, ids_h

    # ---- CPU baseline: the oracle as it stands on a bounded sample, plus parity on that sample
    cpu = None
    if not args.no_cpu:
        import oracle
        nq = args.cpu_queries
        if nq <= 0:
            dt, _, _ = oracle_sample(w, min(B, 8), w.codes)
            nq = int(max(8, min(B, 8 * 15.0 / max(dt, 1e-3))))
        dt, r, units = oracle_sample(w, nq, w.codes)
        gi = out[0][:nq].cpu().numpy().view(np.uint32)
        gu = out[3][:nq].cpu().numpy().view(np.uint32)
        if cfg.integer_exact:
            parity = bool(np.array_equal(gi, r["ids"]) and np.array_equal(gu, r["uniq"]) and
                          np.array_equal(out[1][:nq].cpu().numpy(), r["dists"]))
        else:
            try:                                                    # tolerance regime: oracle/parity.py check_band
                band_check_sample(w, min(nq, 64), w.codes, out)
                parity = bool(np.array_equal(gu, r["uniq"]))
            except AssertionError:
                parity = False
        cpu = {"value": units / dt, "unit": UNIT, "cores": r["threads"], "kind": "oracle",
               "sample": f"first {nq} of {B} queries of {cfg.name} ({units} distinct candidates, {dt:.2f} s)",
               "batch_qps": nq / dt, "gpu_matches_oracle_on_sample": parity}

    line = {
        "path_algorithmic_bytes": path_bytes, "path_hbm_frac": round(path_bytes / (ms_per_step * 1e-3) / 1e9 / peak, 4),
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": round(ms_per_step, 4), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": cfg.name, "N": cfg.N, "d": cfg.d, "M": M, "B": B, "nprobe": cfg.nprobe, "k": k,
                   "id_map": cfg.id_map, "parallelism": "single GPU" if world == 1 else f"{world} independent replicas",
                   "l2": "flushed between timed steps" if flush is not None else "inputs larger than L2",
                   "C_total": total, "U_total": U_total, "distinct_fraction": round(U_total / max(total, 1), 4),
                   "C_mean": w.stats["C_mean"], "C_max": w.stats["C_max"], "gen_seconds": round(t_gen, 1)},
        "batch_qps": B * world / (ms_per_step * 1e-3),
        "input_ids_per_s": C_all / (ms_per_step * 1e-3),
        "hbm_frac_nominal_8TBs": round(achieved / 8000.0, 4),
        "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches),
        "clocks": clocks, "geometry": {kk: v for kk, v in ix.info().items() if kk.startswith(("scan_", "dedup_", "table_", "row_", "chunks"))},
    }
    print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def reference_arm(args, cfg, rank, world):
    """--impl reference: the CPU oracle, as it stands, on the box's host cores.  Each step is a
    bounded sample of the workload.  Rank 0 alone runs; other ranks exit 0."""
    if rank != 0:
        return
    import numpy as np
    import torch
    import oracle
    from workloads import DEFAULT_SEED, make_workload
    dev = "cuda:0" if torch.cuda.is_available() else "cpu"
    w = make_workload(cfg, seed=DEFAULT_SEED, device=dev)
    nq = args.cpu_queries
    if nq <= 0:
        dt, _, _ = oracle_sample(w, min(cfg.B, 8), w.codes)
        per_step = 60.0 / (args.steps + args.warmup)                    # whole run ~1 minute of oracle time
        nq = int(max(4, min(cfg.B, 8 * per_step / max(dt, 1e-3))))
    times, units = [], 0
    for i in range(args.warmup + args.steps):
        dt, r, units = oracle_sample(w, nq, w.codes)
        if i >= args.warmup:
            times.append(dt)
    ms = 1e3 * float(np.mean(times))
    v = units / (ms * 1e-3)
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": round(ms, 3), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "N": cfg.N, "d": cfg.d, "M": cfg.M, "B": cfg.B, "nprobe": cfg.nprobe,
                       "k": cfg.k, "parallelism": "host cores (OpenMP over queries)"},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle",
                             "sample": f"first {nq} of {cfg.B} queries of {cfg.name} per step"},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


if __name__ == "__main__":
    main()
