"""Row-gather ceiling of step (6) on this GPU (DESIGN.md 6.3 / 6.4, profiles/r1_gather_ceiling.md).

    python -m paper_2409_16576_b200.gather_ceiling [--M 64] [--N 1000000000] [--rows 40000000]

Times `fann_gather_probe` -- the scan kernel's code-row access pattern with none of its arithmetic --
over a code array of N rows, for row IDs in three orders:

    random        uniformly random IDs (what a hashed dedup table hands to the scan kernel)
    sorted_100k   the same IDs sorted inside consecutive blocks of 100,000 (one query's distinct list in
                  ascending order: what the order-preserving dedup table produces)
    paged_100k    blocks of 100,000 whose IDs are grouped by 2 MB page but shuffled inside a page and
                  with the pages in random order (is it order, or only page locality?)

and prints one JSON line per (order, load flavour).  The array contents do not matter (random bytes).
Measurement only; nothing on the product path imports this module.
"""
from __future__ import annotations

import argparse
import json


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--M", type=int, default=64, help="PQ bytes per row (stored row = 16/32/64 bytes)")
    ap.add_argument("--N", type=int, default=1_000_000_000)
    ap.add_argument("--rows", type=int, default=40_000_000)
    ap.add_argument("--flavors", default="1,257",
                    help="bits 0-7: 0 = 16-byte nc loads, 1 = same with a 64-byte L2 fetch (scan kernel); bits 8+: CTAs per SM (0 = 2)")
    ap.add_argument("--reps", type=int, default=3)
    args = ap.parse_args()

    import torch
    from . import binding as fann
    from .build import build
    build()
    dev = "cuda:0"
    ix = fann.FannIndex(0)
    step = 1 << 24
    first = 0
    while first < args.N:                                  # load in chunks: no second N x M copy in HBM
        n = min(step * 16, args.N - first)
        chunk = torch.empty((n, args.M), dtype=torch.uint8, device=dev).random_(0, 256)
        ix.load_codes(chunk, first=first, N_total=args.N)
        first += n
        del chunk
    rb = ix.info()["row_bytes"]
    blk = 100_000
    nblk = args.rows // blk
    n = nblk * blk
    g = torch.Generator(device=dev)
    g.manual_seed(1)
    ids = torch.randint(0, args.N, (n,), dtype=torch.int64, device=dev, generator=g)
    rows_per_page = (2 << 20) // rb
    orders = {"random": ids}
    orders["sorted_100k"] = torch.sort(ids.view(nblk, blk), dim=1).values.reshape(-1)
    page = ids // rows_per_page
    scramble = (page * 2654435761) % (1 << 31)             # pages in a pseudo-random order, IDs of a page adjacent
    key = scramble * 4 + torch.randint(0, 4, (n,), device=dev, generator=g)
    orders["paged_100k"] = torch.gather(ids.view(nblk, blk), 1, torch.argsort(key.view(nblk, blk), dim=1)).reshape(-1)
    sink = torch.zeros(4, dtype=torch.int32, device=dev)
    st = torch.cuda.current_stream().cuda_stream
    for name, arr64 in orders.items():
        arr = arr64.to(torch.int32).contiguous()           # IDs < 2^31 here
        for f in [int(x) for x in args.flavors.split(",")]:
            fann.fann_gather_probe(ix.handle, arr, n, sink, f, st)
            torch.cuda.synchronize()
            best = 1e30
            for _ in range(args.reps):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                fann.fann_gather_probe(ix.handle, arr, n, sink, f, st)
                b.record()
                b.synchronize()
                best = min(best, a.elapsed_time(b))
            print(json.dumps({"N": args.N, "M": args.M, "row_bytes": rb, "array_GB": round(args.N * rb / 1e9, 2),
                              "order": name, "flavor": f & 255, "ctas_per_sm": (f >> 8) or 2, "rows": n, "ms": round(best, 3),
                              "Grows_per_s": round(n / best / 1e6, 2),
                              "GBps_row_bytes": round(n * rb / best / 1e6, 1)}), flush=True)
    ix.close()


if __name__ == "__main__":
    main()
