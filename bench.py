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


def traffic_from_profiles(workload: str, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of `kernel` per launch at this workload, from the ncu capture
    committed as profiles/r2_traffic.json (written from the ncu CSV named there); None if not captured."""
    p = os.path.join(ROOT, "profiles", "r2_traffic.json")
    try:
        t = json.load(open(p))
        return int(t["workloads"][workload][kernel]), f"profiles/r2_traffic.json ({t.get('source', 'ncu')})"
    except Exception:
        return None, None


def gather_ceiling(fann, ix, w, dev, nq_groups: int = 4):
    """MEASUREMENT ONLY (include/fann_probe.h, built into its own libfann_probe.so): how fast this part reads the
    code rows the scan kernel reads, in the scan kernel's own order and launch shape (one 512-thread CTA per SM,
    each sweeping one query's distinct list as the dedup kernel leaves it), with none of its arithmetic.  The
    distinct lists come from fann_dedup_only on the first queries of the timed batch.  Returns rows/s of the
    scan kernel's fill path (cp.async ring), of the sm_100 TMA gather4 flavour and of the same rows shuffled."""
    import torch
    lib = _probe_lib()
    info = ix.info()
    sms, row_bytes, N = info["num_sms"], info["row_bytes"], info["N"]
    nq = min(w.cfg.B, nq_groups * sms) // sms * sms
    if nq == 0:
        return None
    off = w.cand_offsets[: nq + 1]
    total = int(off[-1])
    uniq, counts = ix.dedup_only(off, w.cand_ids[:total], total)
    rps = 2048 // row_bytes                                   # rows per ring stage
    unit = 16 * rps                                           # rows one CTA consumes per stage step
    flats, shuffled = [], []
    gen = torch.Generator(device=dev)
    gen.manual_seed(7)
    for g in range(nq // sms):
        c = counts[g * sms:(g + 1) * sms].long()
        L = int(c.min()) // unit * unit
        if L == 0:
            continue
        starts = off[g * sms:(g + 1) * sms]
        idx = starts[:, None] + torch.arange(L, device=dev)[None, :]
        q = uniq[idx]                                         # [sms, L]: every CTA's list, in the dedup's order
        flats.append(q.view(sms, L // unit, 16, rps).permute(1, 0, 2, 3).reshape(-1))
        perm = torch.argsort(torch.rand((sms, L), device=dev, generator=gen), dim=1)
        shuffled.append(torch.gather(q, 1, perm).view(sms, L // unit, 16, rps).permute(1, 0, 2, 3).reshape(-1))
    if not flats:
        return None
    own, rnd = torch.cat(flats).contiguous(), torch.cat(shuffled).contiguous()
    sink = torch.zeros(4, dtype=torch.int32, device=dev)
    stream = torch.cuda.current_stream().cuda_stream

    def rate(ids, flavor):
        best = None
        for it in range(4):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            rc = lib.fann_probe_gather(info["codes_device_ptr"], row_bytes, N, ids.data_ptr(), ids.numel(),
                                       sink.data_ptr(), flavor, 1, stream)
            b.record()
            b.synchronize()
            if rc != 0:
                return None
            if it:
                t = a.elapsed_time(b)
                best = t if best is None else min(best, t)
        return ids.numel() / (best * 1e-3)

    return {"rows": int(own.numel()), "queries": nq,
            "own_order_cp_async_ring": rate(own, 3), "own_order_tma_gather4": rate(own, 4),
            "shuffled_cp_async_ring": rate(rnd, 3)}


def same_ids(cfg, a, b) -> bool:
    """Two runs of the path on one batch: the same bytes on integer data; on real-valued data a row's fp32 sum depends
    on the lane that scores it, so neighbours a rounding apart may swap places (tolerance regime): the
    runs must agree on at least 99.9 % of the output slots."""
    import numpy as np
    a, b = np.asarray(a).view(np.int32), np.asarray(b).view(np.int32)
    if cfg.integer_exact:
        return bool(np.array_equal(a, b))
    return bool(a.shape == b.shape and np.mean(a == b) >= 0.999)


def _probe_lib():
    import ctypes as C
    from paper_2409_16576_b200.build import build_probe
    lib = C.CDLL(build_probe())
    lib.fann_probe_gather.restype = C.c_int
    lib.fann_probe_gather.argtypes = [C.c_void_p, C.c_uint32, C.c_uint64, C.c_void_p, C.c_uint64, C.c_void_p,
                                      C.c_uint32, C.c_uint32, C.c_void_p]
    lib.fann_probe_last_error.restype = C.c_char_p
    return lib


def probe_sweep(args, cfg):
    """--probe-sweep: MEASUREMENT ONLY (include/fann_probe.h).  What bounds a gather of code rows on this part, on a
    synthetic code array of the workload's size (contents are irrelevant to a read): every issue flavour of the probe
    x {random, ascending inside each CTA's list} x {1, 2 CTAs per SM}, and the address-translation test -- random rows
    confined to K random 2 MB pages of the array.  One JSON line; profiles/r2_gather_ceiling.md is written from it."""
    import torch
    lib = _probe_lib()
    dev = "cuda:0"
    torch.cuda.set_device(0)
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    N, M = cfg.N, cfg.M
    row_bytes = 16 if M <= 16 else (32 if M <= 32 else 64)
    codes = torch.empty(N * row_bytes, dtype=torch.uint8, device=dev)
    codes.view(torch.int64)[:] = 0x0102030405060708
    sink = torch.zeros(4, dtype=torch.int32, device=dev)
    gen = torch.Generator(device=dev)
    gen.manual_seed(1)
    stream = torch.cuda.current_stream().cuda_stream
    rps = 2048 // row_bytes
    unit = 16 * rps
    U = max(unit, int(0.58 * cfg.nprobe * cfg.mean_list) // unit * unit)        # rows of one query's distinct list
    groups = max(1, min(8, 40_000_000 // (sms * U)))

    def lists(order):
        out = []
        for _ in range(groups):
            ids = torch.randint(0, N, (sms, U), device=dev, generator=gen, dtype=torch.int64)
            if order == "ascending":
                ids = ids.sort(dim=1).values
            out.append(ids.view(sms, U // unit, 16, rps).permute(1, 0, 2, 3).reshape(-1))
        return torch.cat(out).to(torch.int32).contiguous()

    def rate(ids, flavor, cps):
        best = None
        for it in range(4):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            rc = lib.fann_probe_gather(codes.data_ptr(), row_bytes, N, ids.data_ptr(), ids.numel(), sink.data_ptr(),
                                       flavor, cps, stream)
            b.record()
            b.synchronize()
            if rc != 0:
                return None
            if it:
                t = a.elapsed_time(b)
                best = t if best is None else min(best, t)
        return round(ids.numel() / best / 1e6, 2)                               # G rows/s

    names = {0: "ldg16", 1: "ldg16_l2_64", 2: "ldg32", 3: "cp_async_ring", 4: "tma_gather4"}
    flavors = [f for f in (0, 1, 2, 3, 4) if not (f == 2 and row_bytes < 32)]
    sweep = []
    for order in ("random", "ascending"):
        ids = lists(order)
        for f in flavors:
            for cps in (1, 2):
                sweep.append({"order": order, "flavor": names[f], "ctas_per_sm": cps, "rows": int(ids.numel()),
                              "G_rows_per_s": rate(ids, f, cps)})
    # address translation: random rows confined to K random 2 MB pages of the array
    page_rows = (2 << 20) // row_bytes
    npages = N // page_rows
    n = groups * sms * U
    pages_test = []
    for K in (256, 1024, 4096, 16384, npages):
        if K > npages:
            continue
        pg = torch.randperm(npages, device=dev, generator=gen)[:K]
        ids = (pg[torch.randint(0, K, (n,), device=dev, generator=gen)] * page_rows +
               torch.randint(0, page_rows, (n,), device=dev, generator=gen)).to(torch.int32)
        pages_test.append({"pages_2MB": int(K), "footprint_GB": round(K * (2 << 20) / 1e9, 2),
                           "G_rows_per_s": rate(ids, 3, 1)})
    # what about the order matters: the same kind of lists (one per CTA, U random rows), cp.async ring, 1 CTA per SM
    n_st = U // unit

    def rnd_perm(*shape):
        return torch.argsort(torch.rand(shape, device=dev, generator=gen), dim=-1)

    def ordered(variant):
        out = []
        for _ in range(groups):
            ids = torch.randint(0, N, (sms, U), device=dev, generator=gen, dtype=torch.int64).sort(dim=1).values
            if variant == "ascending_each_cta_at_another_phase":
                sh = (torch.arange(sms, device=dev) * n_st // sms) * unit
                ids = torch.gather(ids, 1, (torch.arange(U, device=dev)[None, :] + sh[:, None]) % U)
            elif variant == "cta_steps_shuffled_ascending_inside":          # a step = the 16 warps' stages: `unit` rows
                p = rnd_perm(sms, n_st)
                ids = torch.gather(ids.view(sms, n_st, unit), 1, p[:, :, None].expand(-1, -1, unit)).reshape(sms, U)
            elif variant == "cta_steps_ascending_shuffled_inside":
                ids = torch.gather(ids.view(sms, n_st, unit), 2, rnd_perm(sms, n_st, unit)).reshape(sms, U)
            elif variant == "warp_stage_rows_in_random_lane_order":
                ids = torch.gather(ids.view(sms, U // rps, rps), 2, rnd_perm(sms, U // rps, rps)).reshape(sms, U)
            elif variant == "rows_of_a_step_dealt_round_robin_to_warps":
                ids = ids.view(sms, n_st, rps, 16).permute(0, 1, 3, 2).reshape(sms, U)
            elif variant.startswith("warp_stage_random_in_window_MB_"):     # a stage's rows random inside a window at a random place
                X = int(variant.rsplit("_", 1)[1]) << 20
                base = torch.randint(0, (N * row_bytes - X) // row_bytes, (sms, U // rps), device=dev, generator=gen)
                ids = base.repeat_interleave(rps, dim=1) + torch.randint(0, X // row_bytes, (sms, U), device=dev, generator=gen)
            elif variant == "each_warp_instruction_in_its_own_random_2MB_page":
                per = 512 // row_bytes                                      # rows one 32-lane 16-byte instruction covers
                pg = torch.randint(0, npages, (sms, U // per), device=dev, generator=gen)
                ids = pg.repeat_interleave(per, dim=1) * page_rows + torch.randint(0, page_rows, (sms, U), device=dev, generator=gen)
            elif variant.startswith("share_with_neighbour_cta_pct_"):       # L2: a part of every list is the next CTA's rows too
                kk = U * int(variant.rsplit("_", 1)[1]) // 100
                nb = torch.gather(torch.roll(ids, 1, 0), 1, rnd_perm(sms, U)[:, :kk])
                ids = torch.cat([torch.gather(ids, 1, rnd_perm(sms, U)[:, : U - kk]), nb], 1).sort(dim=1).values
            elif variant == "random":
                ids = torch.gather(ids, 1, rnd_perm(sms, U))
            out.append(ids.view(sms, n_st, 16, rps).permute(1, 0, 2, 3).reshape(-1))
        return torch.cat(out).to(torch.int32).contiguous()

    order_study = []
    for variant in ("ascending", "ascending_each_cta_at_another_phase", "cta_steps_shuffled_ascending_inside",
                    "cta_steps_ascending_shuffled_inside", "warp_stage_rows_in_random_lane_order",
                    "rows_of_a_step_dealt_round_robin_to_warps", "each_warp_instruction_in_its_own_random_2MB_page",
                    "warp_stage_random_in_window_MB_8", "warp_stage_random_in_window_MB_128",
                    "warp_stage_random_in_window_MB_512", "warp_stage_random_in_window_MB_2048",
                    "share_with_neighbour_cta_pct_30", "share_with_neighbour_cta_pct_60", "random"):
        order_study.append({"order": variant, "G_rows_per_s": rate(ordered(variant), 3, 1)})
    print(json.dumps({"probe_sweep": {"workload": cfg.name, "N": N, "row_bytes": row_bytes, "array_GB": round(N * row_bytes / 1e9, 1),
                                      "rows_per_cta_list": U, "sms": sms, "order_x_flavor": sweep,
                                      "random_rows_in_K_pages": pages_test, "order_study": order_study}}))


def time_device_path(fann, cfg, args, rank, local_rank, world, dev, keep_lists=False, sample_clocks=False):
    """Generate the workload, load it, warm up, time K steps of fann_build_lut + fann_dedup_scan_topk with
    everything resident in HBM.  Returns (result dict, live objects for the legs that follow)."""
    import numpy as np
    import torch
    from workloads import DEFAULT_SEED, make_workload
    t_gen = time.time()
    by_window = getattr(args, "query_order", "generated") == "window"
    lists_sorted = getattr(args, "list_order", "generated") == "ascending"
    w = make_workload(cfg, seed=rank_seed(DEFAULT_SEED, rank), device=dev,
                      keep_lists=keep_lists or by_window or lists_sorted)   # each replica: its own batch
    if lists_sorted:
        # measurement variant: every posting list stored in ascending ID order (a list's order carries no meaning,
        # PAPER.md:L150; fann_load_lists does the same to its own copy): 32 consecutive candidates then fall into
        # few ID-range classes, which is what the class split's MATCH instruction pays for
        from workloads.generate import PostingLists, make_candidates
        n_lists = w.list_offsets.numel() - 1
        step = max(1, n_lists // 16)                               # a sixteenth of the lists at a time: bounded scratch
        for l0 in range(0, n_lists, step):
            l1 = min(n_lists, l0 + step)
            e0, e1 = int(w.list_offsets[l0]), int(w.list_offsets[l1])
            lens = w.list_offsets[l0 + 1:l1 + 1] - w.list_offsets[l0:l1]
            seg = torch.repeat_interleave(torch.arange(l1 - l0, device=dev), lens)
            key = (seg << 32) | (w.list_ids[e0:e1].long() & 0xFFFFFFFF)
            w.list_ids[e0:e1] = (torch.sort(key).values & 0xFFFFFFFF).to(torch.int32)
            del key, seg, lens
        w.cand_offsets, w.cand_ids = make_candidates(cfg, PostingLists(w.list_offsets, w.list_ids, 0), w.probes.long())
        torch.cuda.empty_cache()                                   # the library allocates outside torch's pool
    if by_window:
        # measurement variant: the same queries, ordered by the position of their probed window, so that queries
        # which share posting lists -- and code rows -- are scanned at about the same time (L2 reuse)
        from workloads.generate import PostingLists, make_candidates
        perm = torch.argsort(w.probes.long().median(dim=1).values)
        w.probes, w.queries = w.probes[perm].contiguous(), w.queries[perm].contiguous()
        w.cand_offsets, w.cand_ids = make_candidates(cfg, PostingLists(w.list_offsets, w.list_ids, 0), w.probes.long())
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
    flush = None
    if total * 4 + B * M * 1024 + total * M < 4 * L2_BYTES:
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
    sampler = ClockSampler(local_rank) if sample_clocks else None
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kern = {}
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
            kern.setdefault(kk, []).append(v)
    barrier()
    t1 = time.time()
    fann.fann_workspace_status(ix.handle, ws, stream)               # raises if any timed step overflowed a table
    modes = fann.fann_workspace_modes(ix.handle, ws, B, total, k, stream)
    launches = ix.info()["kernel_launches"] - launches0
    fann.fann_set_timing(ix.handle, False)
    total_ms = float(sum(a.elapsed_time(b) for a, b in ev))
    clocks = sampler.stop(t0, t1) if sampler else None
    total_ms, U_all, C_all = aggregate_over_ranks(total_ms, U_total, total, device=dev)
    ms_per_step = total_ms / args.steps

    # ---- roofline of the dominant kernel (scan: code-row gather + ADC + top-k), DESIGN.md 7
    peak, peak_src = measured_peak_gbs()
    # the scan kernel's algorithmic bytes: code rows + the distinct IDs it reads + tables + outputs
    algo_bytes = M * U_total + 4 * U_total + 1024 * M * B + 8 * k * B
    # the whole step: + candidate IDs read by the dedup stage + tables written
    path_bytes = algo_bytes + 4 * total + 1024 * M * B
    scan_ms = float(np.mean(kern["scan_ms"]))
    achieved = algo_bytes / (scan_ms * 1e-3) / 1e9
    traffic, traffic_src = traffic_from_profiles(cfg.name, "scan_kernel")
    roofline = {"bound": "hbm", "kernel": "scan_kernel", "achieved": round(achieved, 1), "peak": peak,
                "unit": "GB/s", "frac": round(achieved / peak, 4), "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": peak_src, "algorithmic_bytes": algo_bytes, "kernel_ms": round(scan_ms, 4),
                "code_bytes_only_frac": round(M * U_total / (scan_ms * 1e-3) / 1e9 / peak, 4),
                "rows_per_s": U_total / (scan_ms * 1e-3),
                "share_of_step": round(scan_ms / ms_per_step, 4),
                "kernels_ms": {kk: round(float(np.mean(v)), 4) for kk, v in kern.items()},
                "dedup_placement": modes}
    res = {"ms_per_step": ms_per_step, "value": U_all / (ms_per_step * 1e-3), "U_all": U_all, "C_all": C_all,
           "U_total": U_total, "C_total": total, "roofline": roofline, "launches": int(launches), "clocks": clocks,
           "path_algorithmic_bytes": path_bytes, "path_hbm_frac": round(path_bytes / (ms_per_step * 1e-3) / 1e9 / peak, 4),
           "l2": "flushed between timed steps" if flush is not None else "inputs larger than L2",
           "gen_seconds": round(t_gen, 1), "stats": w.stats}
    return res, {"w": w, "ix": ix, "out": out, "ws": ws, "lut": lut}


def small_batch_leg(fann, ix, w, cfg, dev, ref_ids):
    """the path one small batch at a time through the block pool
    (fann_search_small_lists: queries and probed-list indices from HOST buffers, results back on the host).
    Latency is the host's wall clock around the synchronous call; throughput is queries answered per second by
    T host threads calling at the same time on one handle."""
    import threading
    import numpy as np
    k, dsub, nprobe = cfg.k, cfg.dsub, cfg.nprobe
    nq = min(cfg.B, 512)
    per_q = int((w.cand_offsets[1:nq + 1] - w.cand_offsets[:nq]).max())
    max_B = min(64, cfg.B)
    pool = fann.fann_pool_create(ix.handle, 8, max_B, per_q * max_B, dsub, nprobe, k)
    q_h = w.queries[:nq].cpu().pin_memory()
    p_h = w.probes[:nq].cpu().contiguous().pin_memory()
    res = {"entry": "fann_search_small_lists", "pool_blocks": 8, "timing": "host wall clock around the synchronous call"}
    ok = True
    for B in (1, 8, max_B):
        oi = np.zeros((B, k), np.uint32); od = np.zeros((B, k), np.float32); oc = np.zeros(B, np.uint32)
        ts = []
        for it in range(24):
            b0 = (it * B) % (nq - B + 1)
            t0 = time.perf_counter()
            fann.fann_search_small_lists(ix.handle, pool, q_h[b0:b0 + B], B, w.codebooks, dsub, p_h[b0:b0 + B], nprobe, k, oi, od, oc)
            ts.append(time.perf_counter() - t0)
            ok = ok and same_ids(cfg, oi, ref_ids[b0:b0 + B])
        ts = sorted(ts[4:])
        res[f"B{B}"] = {"latency_us_p50": round(1e6 * ts[len(ts) // 2], 1), "latency_us_p90": round(1e6 * ts[int(len(ts) * 0.9)], 1),
                        "qps_one_thread": round(B / ts[len(ts) // 2], 1)}
    for T in (4, 8):
        done = [0] * T
        stop = time.perf_counter() + 0.6

        def worker(t):
            oi = np.zeros((1, k), np.uint32); od = np.zeros((1, k), np.float32); oc = np.zeros(1, np.uint32)
            b = t
            while time.perf_counter() < stop:
                fann.fann_search_small_lists(ix.handle, pool, q_h[b:b + 1], 1, w.codebooks, dsub, p_h[b:b + 1], nprobe, k, oi, od, oc)
                done[t] += 1
                b = (b + T) % nq
        t0 = time.perf_counter()
        th = [threading.Thread(target=worker, args=(t,)) for t in range(T)]
        for x in th:
            x.start()
        for x in th:
            x.join()
        res[f"threads{T}_B1_qps"] = round(sum(done) / (time.perf_counter() - t0), 1)
    res["matches_device_path"] = ok
    res["pool"] = fann.fann_pool_stats(pool)
    fann.fann_pool_destroy(pool)
    return res


def list_major_leg(fann, ix, w, cfg, args, dev, ref_ids, U_total, C_total):
    """EXPERIMENT, not the paper's layout (fann.h "EXPERIMENT"): a second copy of the codes in posting-list order,
    replicas included, streamed list by list instead of gathered by ID; every candidate is scored and the repeats
    leave where the top-k buffer is pruned, so no dedup pass runs.  Same batch, same outputs; timed like the step."""
    import numpy as np
    import torch
    B, k, M, dsub = cfg.B, cfg.k, cfg.M, cfg.dsub
    info = ix.info()
    w.codes = None                                              # the library has its own copy; nothing below reads this one
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    need_copy = int(w.list_ids.numel()) * info["row_bytes"]
    if free < need_copy + (8 << 30):
        return {"skipped": f"{free >> 30} GB free, the list-major copy needs {need_copy >> 30} GB"}
    stream = torch.cuda.current_stream().cuda_stream
    t0 = torch.cuda.Event(enable_timing=True); t1 = torch.cuda.Event(enable_timing=True)
    t0.record()
    fann.fann_build_list_codes(ix.handle, stream)
    t1.record(); t1.synchronize()
    build_ms = t0.elapsed_time(t1)
    lut = torch.empty((B, M, 256), dtype=torch.float32, device=dev)
    oi = torch.empty((B, k), dtype=torch.int32, device=dev)
    od = torch.empty((B, k), dtype=torch.float32, device=dev)
    oc = torch.empty(B, dtype=torch.int32, device=dev)
    need = fann.fann_search_lists_stream_workspace_bytes(ix.handle, B, C_total)
    ws = torch.empty(need, dtype=torch.uint8, device=dev)
    probes = w.probes

    def step():
        fann.fann_build_lut(ix.handle, w.queries, B, w.codebooks, dsub, lut, stream)
        fann.fann_search_lists_stream(ix.handle, lut, B, probes, cfg.nprobe, C_total, k, oi, od, oc, ws, need, stream)

    for _ in range(args.warmup):
        step()
    fann.fann_search_lists_stream_status(ix.handle, ws, stream)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(args.steps):
        step()
    b.record(); b.synchronize()
    ms = a.elapsed_time(b) / args.steps
    peak, _ = measured_peak_gbs()
    # rows + their vector-IDs (read from the lists) + the (row, ID) pairs (written by the expansion, read by the scan)
    # + tables (written, read) + outputs
    bytes_ = C_total * (info["row_bytes"] + 4 + 16) + 2 * 1024 * M * B + 8 * k * B
    return {"what": "list-major copy of the codes streamed list by list (fann_search_lists_stream); NOT the paper's ID-indexed layout",
            "ms_per_step": round(ms, 4), "value": U_total / (ms * 1e-3), "unit": UNIT,
            "rows_scored_per_s": C_total / (ms * 1e-3), "extra_hbm_bytes": need_copy, "build_ms": round(build_ms, 1),
            "algorithmic_bytes": bytes_, "hbm_frac": round(bytes_ / (ms * 1e-3) / 1e9 / peak, 4),
            "matches_device_path": same_ids(cfg, oi.cpu().numpy(), ref_ids)}


def next_rows_leg(fann, cfg, live, dev, args, with_oracle: bool):
    """SURVEY.md 8(f) NEXT-1 and NEXT-4 measured where the raw vectors fit beside the codes (configs[1], the
    paper's SIFT-shaped case): Algorithm 1 re-ranks the GPU stage's top-n of every query of
    the batch just timed, then Fig. 8's page plan (L198) for the mini-batches Algorithm 1 executed.  CUDA events
    around fann_rerank / fann_page_reads; algorithmic bytes of the re-ranking = raw vectors read + tasks +
    queries + outputs.  The kernels wait on one dependent row gather per mini-batch (the stop rule decides
    whether the next mini-batch is read at all), so this is a latency-bound step: the HBM fraction says so."""
    import numpy as np
    import torch
    from workloads import DEFAULT_SEED, make_page_table, make_raw_vectors
    w, ix, out = live["w"], live["ix"], live["out"]
    B, n = out[0].shape
    vec = make_raw_vectors(cfg, DEFAULT_SEED, device=dev)
    page_of, n_pages = make_page_table(cfg, DEFAULT_SEED, device=dev, elem_bytes=vec.element_size())
    ix.load_vectors(vec)
    ix.load_page_table(page_of, n_pages)
    tasks = out[0]
    peak, _ = measured_peak_gbs()
    flush = torch.empty(2 * L2_BYTES, dtype=torch.uint8, device=dev)

    def timed(fn):
        for _ in range(max(3, args.warmup)):
            r = fn()
        ms = 0.0
        for i in range(args.steps):
            flush.fill_(i & 0xFF)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            r = fn()
            b.record()
            b.synchronize()
            ms += a.elapsed_time(b)
        return ms / args.steps, r

    legs = []
    for bs, k, eps, beta in ((10, 10, 0.15, 2), (10, 10, 0.0, 1)):
        ms, got = timed(lambda: ix.rerank(w.queries, tasks, bs, k, eps, beta))
        reads = int(got[4].sum().item())
        byts = reads * cfg.d * vec.element_size() + tasks.numel() * 4 + B * cfg.d * 4 + B * k * 8
        leg = {"n": n, "batch_size": bs, "k": k, "eps": eps, "beta": beta, "ms": round(ms, 4),
               "queries_per_s": B / (ms * 1e-3), "raw_vectors_read_per_query": reads / B,
               "mini_batches_per_query": float(got[3].float().mean().item()),
               "algorithmic_bytes": byts, "GB_per_s": round(byts / ms / 1e6, 1), "hbm_frac": round(byts / ms / 1e6 / peak, 4)}
        if with_oracle:
            import oracle
            nq = min(B, 32)
            used, rel = torch.unique(tasks[:nq].reshape(-1), return_inverse=True)
            rows = vec[used.long()].cpu().numpy().astype(np.float32)
            ref = oracle.rerank(w.queries[:nq].cpu().numpy(), rows, rel.view(nq, n).cpu().numpy().astype(np.uint32), bs, k, eps, beta)
            ids = used.cpu().numpy().view(np.uint32)[ref["ids"]]
            leg["matches_oracle_on_sample"] = bool(
                np.array_equal(got[0][:nq].cpu().numpy().view(np.uint32), ids) and
                np.array_equal(got[3][:nq].cpu().numpy().view(np.uint32), ref["batches"]) and
                np.allclose(got[1][:nq].cpu().numpy(), ref["dists"], rtol=1e-5, atol=0))
        pms, pr = timed(lambda: ix.page_reads(tasks, bs, batches_run=got[3]))
        leg["page_reads"] = {"ms": round(pms, 4), "queries_per_s": B / (pms * 1e-3),
                             "pages_per_query": float(pr[2].float().mean().item()),
                             "tasks_per_s": reads / (pms * 1e-3)}
        if with_oracle:
            pg, br, tot = oracle.page_reads(page_of.cpu().numpy().view(np.uint32), tasks[:nq].cpu().numpy().view(np.uint32),
                                            bs, max_batches=ref["batches"])
            leg["page_reads"]["matches_oracle_on_sample"] = bool(
                np.array_equal(pr[2][:nq].cpu().numpy().view(np.uint32), tot) and
                np.array_equal(pr[1][:nq].cpu().numpy().view(np.uint32), br))
        legs.append(leg)
    del vec, page_of, flush
    return {"workload": cfg.name, "raw_vectors": f"[{cfg.N}][{cfg.d}] {cfg.values} in HBM", "l2": "flushed between timed calls",
            "entries": "fann_rerank (Algorithm 1), fann_page_reads (Fig. 8)", "runs": legs}


def sample_parity(w, cfg, out, nq):
    """GPU output of the first nq queries against the CPU oracle (bytes for integer data, the 1e-5 band else).
    Returns (parity flag, seconds the oracle took, oracle result, distinct candidates scored)."""
    import numpy as np
    dt, r, units = oracle_sample(w, nq, w.codes)
    gi = out[0][:nq].cpu().numpy().view(np.uint32)
    gu = out[3][:nq].cpu().numpy().view(np.uint32)
    if cfg.integer_exact:
        parity = bool(np.array_equal(gi, r["ids"]) and np.array_equal(gu, r["uniq"]) and
                      np.array_equal(out[1][:nq].cpu().numpy(), r["dists"]))
    else:
        try:                                                        # tolerance regime: oracle/parity.py check_band
            band_check_sample(w, min(nq, 64), w.codes, out)
            parity = bool(np.array_equal(gu, r["uniq"]))
        except AssertionError:
            parity = False
    return parity, dt, r, units


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
    ap.add_argument("--no-ceiling", action="store_true", help="skip the gather-ceiling probe leg")
    ap.add_argument("--no-configs", action="store_true", help="skip the block with the other large workloads")
    ap.add_argument("--no-experiment", action="store_true", help="skip the list-major streaming experiment")
    ap.add_argument("--probe-sweep", action="store_true",
                    help="measurement only: the row-gather ceiling sweep on a synthetic array of the workload's size")
    ap.add_argument("--query-order", default="generated", choices=["generated", "window"],
                    help="measurement variant: 'window' orders the batch's queries by the position of their probed lists")
    ap.add_argument("--list-order", default="generated", choices=["generated", "ascending"],
                    help="measurement variant: 'ascending' stores every posting list in ascending ID order")
    ap.add_argument("--id-map", default=None, choices=["feistel", "lattice"],
                    help="vector -> ID map of the generator (default: the config's, 'feistel')")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)

    import numpy as np
    import torch
    from workloads import CONFIGS

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    cfg = CONFIGS[args.workload]
    if args.id_map:
        cfg = cfg.scaled(id_map=args.id_map)

    if args.impl == "reference":
        return reference_arm(args, cfg, rank, world)
    if args.probe_sweep:
        if rank == 0:
            probe_sweep(args, cfg)
        return

    assert torch.cuda.is_available(), "bench.py needs a CUDA device: there is no CPU fallback"
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(dev))
    import paper_2409_16576_b200 as fann
    from paper_2409_16576_b200.build import build
    build()

    B, k, M, dsub = cfg.B, cfg.k, cfg.M, cfg.dsub
    want_lists = not args.no_e2e and rank == 0
    res, live = time_device_path(fann, cfg, args, rank, local_rank, world, dev, keep_lists=want_lists,
                                 sample_clocks=rank == 0)
    w, ix, out = live["w"], live["ix"], live["out"]
    total, U_total = res["C_total"], res["U_total"]
    roofline = res["roofline"]
    stream = torch.cuda.current_stream().cuda_stream

    if rank != 0:
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        return

    # ---- the gather ceiling of this part for the rows of this very batch (measurement only)
    if not args.no_ceiling:
        try:
            gc = gather_ceiling(fann, ix, w, dev)
        except Exception as e:                                      # the probe must never take the bench line down
            gc = {"error": str(e)[:200]}
        if gc and gc.get("own_order_cp_async_ring"):
            roofline["gather_ceiling_rows_per_s"] = gc["own_order_cp_async_ring"]
            roofline["frac_of_gather_ceiling"] = round(roofline["rows_per_s"] / gc["own_order_cp_async_ring"], 4)
        roofline["gather_probe"] = gc

    # ---- CPU baseline: the oracle as it stands on a bounded sample, plus parity on that sample
    cpu = None
    if not args.no_cpu:
        nq = args.cpu_queries
        if nq <= 0:
            dt, _, _ = oracle_sample(w, min(B, 8), w.codes)
            nq = int(max(8, min(B, 8 * 15.0 / max(dt, 1e-3))))
        parity, dt, r, units = sample_parity(w, cfg, out, nq)
        cpu = {"value": units / dt, "unit": UNIT, "cores": r["threads"], "kind": "oracle",
               "sample": f"first {nq} of {B} queries of {cfg.name} ({units} distinct candidates, {dt:.2f} s)",
               "batch_qps": nq / dt, "gpu_matches_oracle_on_sample": parity}

    # ---- e2e: the same metric through the C ABI with HOST buffers (copies inside the timed region).
    # `e2e`: posting lists resident in HBM (fann_search_lists_host): queries and probed-list indices go up.
    # `e2e_candidate_ids`: the paper's step (4) (fann_search_host): the candidate IDs themselves go up.
    e2e, e2e_ids, small, experiment = None, None, None, None
    if not args.no_e2e:
        ref_ids = out[0].cpu().numpy()
        del live["ws"], live["lut"]
        ix._ws = None
        torch.cuda.empty_cache()

        def timed(fn):
            for _ in range(2):
                fn()
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(args.steps):
                fn()
            b.record()
            b.synchronize()
            return a.elapsed_time(b) / args.steps

        oi = torch.empty((B, k), dtype=torch.int32).pin_memory()
        od = torch.empty((B, k), dtype=torch.float32).pin_memory()
        oc = torch.empty(B, dtype=torch.int32).pin_memory()
        q_h = w.queries.cpu().pin_memory()
        d2h = int(oi.numel() * 4 + od.numel() * 4 + oc.numel() * 4)

        ix.load_lists(w.list_offsets, w.list_ids)
        p_h = w.probes.cpu().contiguous().pin_memory()
        need = fann.fann_search_lists_host_scratch_bytes(ix.handle, B, dsub, cfg.nprobe, total, k)
        scratch = torch.empty(need, dtype=torch.uint8, device=dev)
        e_ms = timed(lambda: fann.fann_search_lists_host(ix.handle, q_h, B, w.codebooks, dsub, p_h, cfg.nprobe, total, k,
                                                         oi, od, oc, scratch, need, stream))
        e2e = {"value": U_total / (e_ms * 1e-3), "unit": UNIT, "ms_per_step": round(e_ms, 3),
               "entry": "fann_search_lists_host (posting lists resident in HBM, PAPER.md:L125 step 3 on the GPU)",
               "h2d_bytes_per_step": int(q_h.numel() * 4 + p_h.numel() * 4), "d2h_bytes_per_step": d2h,
               "matches_device_path": same_ids(cfg, oi.numpy(), ref_ids)}
        del scratch, p_h
        torch.cuda.empty_cache()
        try:
            small = small_batch_leg(fann, ix, w, cfg, dev, ref_ids)
        except Exception as e:                                      # never take the bench line down
            small = {"error": str(e)[:200]}
        if not args.no_experiment:
            try:
                experiment = list_major_leg(fann, ix, w, cfg, args, dev, ref_ids, U_total, total)
            except Exception as e:
                experiment = {"error": str(e)[:200]}

        need = fann.fann_search_host_scratch_bytes(ix.handle, B, dsub, total, k)
        scratch = torch.empty(need, dtype=torch.uint8, device=dev)
        off_h, ids_h = w.cand_offsets.cpu().pin_memory(), w.cand_ids.cpu().pin_memory()
        e_ms = timed(lambda: fann.fann_search_host(ix.handle, q_h, B, w.codebooks, dsub, off_h, ids_h, k, oi, od, oc,
                                                   scratch, need, stream))
        e2e_ids = {"value": U_total / (e_ms * 1e-3), "unit": UNIT, "ms_per_step": round(e_ms, 3),
                   "entry": "fann_search_host (candidate IDs from the host, PAPER.md:L125 step 4)",
                   "h2d_bytes_per_step": int(q_h.numel() * 4 + off_h.numel() * 8 + ids_h.numel() * 4),
                   "d2h_bytes_per_step": d2h, "matches_device_path": same_ids(cfg, oi.numpy(), ref_ids)}
        del scratch, q_h, ids_h, off_h

    ms_per_step = res["ms_per_step"]
    geometry = {kk: v for kk, v in ix.info().items() if kk.startswith(("scan_", "dedup_", "table_", "row_", "chunks"))}
    stats = res["stats"]

    # ---- the other large workloads ("report both" 1B configs), same process, one after another
    others, next_rows = None, None
    if world == 1 and not args.no_configs and args.workload == DEFAULT_WORKLOAD:
        live.clear()
        ix.close()
        del w, ix, out
        torch.cuda.empty_cache()
        others = []
        for name in ("i8_1b_m25", "f32_100m_m48", "u8_10m_m32"):
            c2 = CONFIGS[name]
            if args.id_map:
                c2 = c2.scaled(id_map=args.id_map)
            r2, l2 = time_device_path(fann, c2, args, rank, local_rank, world, dev)
            entry = {"workload": name, "N": c2.N, "M": c2.M, "B": c2.B, "nprobe": c2.nprobe, "k": c2.k,
                     "ms_per_step": round(r2["ms_per_step"], 4), "value": r2["value"], "unit": UNIT,
                     "batch_qps": c2.B / (r2["ms_per_step"] * 1e-3), "C_total": r2["C_total"], "U_total": r2["U_total"],
                     "l2": r2["l2"], "roofline": r2["roofline"]}
            if not args.no_cpu:
                par, dt, _, units = sample_parity(l2["w"], c2, l2["out"], min(c2.B, 48))
                entry["gpu_matches_oracle_on_sample"] = par
                entry["oracle_sample"] = f"first {min(c2.B, 48)} queries, {units} distinct candidates, {dt:.2f} s"
            if name == "u8_10m_m32":
                try:
                    next_rows = next_rows_leg(fann, c2, l2, dev, args, with_oracle=not args.no_cpu)
                except Exception as e:                              # never take the bench line down
                    next_rows = {"error": str(e)[:200]}
            others.append(entry)
            l2["ix"].close()
            l2.clear()
            del l2
            torch.cuda.empty_cache()

    line = {
        "path_algorithmic_bytes": res["path_algorithmic_bytes"], "path_hbm_frac": res["path_hbm_frac"],
        "metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": round(ms_per_step, 4), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": cfg.name, "N": cfg.N, "d": cfg.d, "M": M, "B": B, "nprobe": cfg.nprobe, "k": k,
                   "id_map": cfg.id_map, "query_order": args.query_order, "list_order": args.list_order, "parallelism": "single GPU" if world == 1 else f"{world} independent replicas",
                   "l2": res["l2"], "C_total": total, "U_total": U_total,
                   "distinct_fraction": round(U_total / max(total, 1), 4),
                   "C_mean": stats["C_mean"], "C_max": stats["C_max"], "gen_seconds": res["gen_seconds"]},
        "batch_qps": B * world / (ms_per_step * 1e-3),
        "input_ids_per_s": res["C_all"] / (ms_per_step * 1e-3),
        "hbm_frac_nominal_8TBs": round(roofline["achieved"] / 8000.0, 4),
        "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "e2e_candidate_ids": e2e_ids, "small_batch": small,
        "experiment_list_major": experiment, "next_rows": next_rows,
        "gpu_launches": res["launches"], "clocks": res["clocks"], "geometry": geometry, "configs": others,
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
