"""CUDA path vs CPU oracle for the low-latency small-batch mode,
through the C ABI: several scan CTAs per query, the block pool, concurrent host threads on one handle."""
import threading

import numpy as np
import pytest
import torch

import oracle
from oracle.parity import check_band, check_exact
from workloads import CONFIGS, make_workload, mini

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


@pytest.fixture(scope="module")
def fann():
    import paper_2409_16576_b200 as f
    from paper_2409_16576_b200.build import build
    build()
    f.load_library()
    return f


def np_u32(t):
    return t.cpu().numpy().view(np.uint32)


@pytest.fixture(scope="module")
def wl():
    """configs[1] structure at N = 1 M: 40 queries of ~32 k candidates (k = 100), integer data: bytes must match."""
    return make_workload(mini("u8_10m_m32", N=1_000_000, n_lists=2_000, B=40, codes_mode="histogram"), keep_lists=True)


@pytest.fixture(scope="module")
def ref(wl):
    w = wl
    return oracle.search(w.queries.numpy(), w.codebooks.numpy(), w.codes.numpy(), w.cand_offsets.numpy(),
                         w.cand_ids.numpy().view(np.uint32), w.cfg.k)


def _sub(w, b0, b1):
    off = w.cand_offsets[b0:b1 + 1]
    return w.queries[b0:b1].contiguous(), (off - off[0]).contiguous(), w.cand_ids[int(off[0]):int(off[-1])].contiguous()


def _ref_rows(ref, b0, b1):
    return {k: v[b0:b1] for k, v in ref.items() if isinstance(v, np.ndarray)}


@pytest.mark.parametrize("B,k", [(1, 100), (3, 100), (9, 1000), (40, 10), (40, 1024)])
def test_split_scan_gives_the_oracles_bytes(fann, wl, B, k):
    """Batches smaller than half the SMs take several scan CTAs per query (each on a slice of the query's distinct
    list, merged on the device): same bytes as the oracle, and as one CTA per query (FANN_SPLIT_SCAN=0 in
    test_every_code_path_gives_the_same_bytes)."""
    w = wl
    q, off, ids = _sub(w, 0, B)
    ix = fann.FannIndex(0)
    ix.load_codes(w.codes.to(DEV))
    lut = ix.build_lut(q.to(DEV), w.codebooks.to(DEV))
    o = ix.dedup_scan_topk(lut, off.to(DEV), ids.to(DEV), k, check=True)
    torch.cuda.synchronize()
    r = oracle.search(q.numpy(), w.codebooks.numpy(), w.codes.numpy(), off.numpy(), ids.numpy().view(np.uint32), k)
    check_exact((np_u32(o[0]), o[1].cpu().numpy(), np_u32(o[2]), np_u32(o[3])), r)
    ix.close()


def test_split_scan_edge_lists(fann):
    """Empty lists, lists shorter than k and than one slice, all-duplicate lists, with several CTAs per query."""
    rng = np.random.default_rng(5)
    N, M, dsub = 50_000, 16, 4
    codes = rng.integers(0, 256, size=(N, M), dtype=np.uint8)
    cb = rng.integers(0, 256, size=(M, 256, dsub)).astype(np.float32)
    q = rng.integers(0, 256, size=(5, M * dsub)).astype(np.float32)
    lists = [np.empty(0, np.uint32), rng.integers(0, N, 7).astype(np.uint32), np.full(3000, 123, np.uint32),
             rng.integers(0, N, 5000).astype(np.uint32), np.array([0xFFFFFFFF, N + 3, 5, 5], np.uint32)]
    off = np.zeros(6, np.int64)
    off[1:] = np.cumsum([len(x) for x in lists])
    ids = np.concatenate(lists)
    ix = fann.FannIndex(0)
    ix.load_codes(torch.from_numpy(codes).to(DEV))
    for k in (1, 50, 1000):
        lut = ix.build_lut(torch.from_numpy(q).to(DEV), torch.from_numpy(cb).to(DEV))
        o = ix.dedup_scan_topk(lut, torch.from_numpy(off).to(DEV), torch.from_numpy(ids.view(np.int32)).to(DEV), k, check=True)
        torch.cuda.synchronize()
        check_exact((np_u32(o[0]), o[1].cpu().numpy(), np_u32(o[2]), np_u32(o[3])), oracle.search(q, cb, codes, off, ids, k))
    ix.close()


@pytest.mark.parametrize("B", [1, 9, 20, 40])
def test_split_scan_distance_follows_the_id(fann, B):
    """The slices of a query's distinct list are ID ranges (ordered dedup placement).  Here the distance is a monotone
    function of the ID with 780 equal distances in a row, so the top-k sits in ONE slice (the lowest IDs for query 0,
    the highest for query 1, the middle for query 2): the merge's bound from the parts' m-th keys is then far above
    the k-th key, its selection does not apply and it falls back to merging the parts pairwise; ties are decided by ID
    across slice borders.  16, 16, 4 and 2 scan CTAs per query."""
    rng = np.random.default_rng(11)
    N, M, dsub = 200_000, 16, 4
    codes = np.repeat((np.arange(N, dtype=np.int64) * 256 // N).astype(np.uint8)[:, None], M, axis=1)
    cb = np.repeat(np.arange(256, dtype=np.float32)[None, :, None], M, axis=0).repeat(dsub, axis=2)   # centroid j = (j, j, j, j)
    q = np.zeros((B, M * dsub), dtype=np.float32)
    q[1::3] = 255.0
    q[2::3] = 128.0
    lists = [rng.integers(0, N, 60_000 + 1000 * b).astype(np.uint32) for b in range(B)]
    off = np.zeros(B + 1, np.int64)
    off[1:] = np.cumsum([len(x) for x in lists])
    ids = np.concatenate(lists)
    ix = fann.FannIndex(0)
    ix.load_codes(torch.from_numpy(codes).to(DEV))
    lut = ix.build_lut(torch.from_numpy(q).to(DEV), torch.from_numpy(cb).to(DEV))
    for k in (1000, 64, 1):
        o = ix.dedup_scan_topk(lut, torch.from_numpy(off).to(DEV), torch.from_numpy(ids.view(np.int32)).to(DEV), k, check=True)
        torch.cuda.synchronize()
        check_exact((np_u32(o[0]), o[1].cpu().numpy(), np_u32(o[2]), np_u32(o[3])), oracle.search(q, cb, codes, off, ids, k))
    ix.close()


def test_split_scan_fp32_band(fann):
    w = make_workload(CONFIGS["tiny_local"])
    ix = fann.FannIndex(0)
    ix.load_codes(w.codes.to(DEV))
    B = 5
    q, off, ids = _sub(w, 0, B)
    lut = ix.build_lut(q.to(DEV), w.codebooks.to(DEV))
    o = ix.dedup_scan_topk(lut, off.to(DEV), ids.to(DEV), w.cfg.k, check=True)
    torch.cuda.synchronize()
    cand = ids.numpy().view(np.uint32)
    for b in range(B):
        ai, ad = oracle.query_all(q.numpy()[b], w.codebooks.numpy(), w.codes.numpy(), cand[off[b]:off[b + 1]])
        assert np_u32(o[3])[b] == ai.size
        check_band(np_u32(o[0])[b], o[1].cpu().numpy()[b], np_u32(o[2])[b], ai, ad, w.cfg.k)
    ix.close()


def _pool(fann, ix, w, n_blocks, max_B):
    per_q = int((w.cand_offsets[1:] - w.cand_offsets[:-1]).max())
    return fann.fann_pool_create(ix.handle, n_blocks, max_B, per_q * max_B, w.cfg.dsub, w.cfg.nprobe, w.cfg.k)


@pytest.mark.parametrize("graphs", ["1", "0"])
def test_pool_entries_match_the_oracle(fann, wl, ref, monkeypatch, graphs):
    """Both entry forms on a pool block; the posting-list form replays one CUDA graph per call shape
    (FANN_SMALL_GRAPH=0: plain launches) -- the second call of a shape is a pure replay."""
    monkeypatch.setenv("FANN_SMALL_GRAPH", graphs)
    w = wl
    ix = fann.FannIndex(0)
    ix.load_codes(w.codes.to(DEV))
    ix.load_lists(w.list_offsets.to(DEV), w.list_ids.to(DEV))
    pool = _pool(fann, ix, w, 2, 4)
    cb = w.codebooks.to(DEV)
    k = w.cfg.k
    for b0, b1 in ((0, 1), (1, 4), (4, 8), (39, 40), (7, 8), (20, 23)):
        B = b1 - b0
        q, off, ids = _sub(w, b0, b1)
        for form in ("ids", "lists"):
            oi, od = np.zeros((B, k), np.uint32), np.zeros((B, k), np.float32)
            oc = np.zeros(B, np.uint32)
            if form == "ids":
                fann.fann_search_small(ix.handle, pool, q.numpy(), B, cb, w.cfg.dsub, off.numpy(), ids.numpy(), k, oi, od, oc)
            else:
                P = np.ascontiguousarray(w.probes[b0:b1].numpy())
                fann.fann_search_small_lists(ix.handle, pool, q.numpy(), B, cb, w.cfg.dsub, P, w.cfg.nprobe, k, oi, od, oc)
            r = _ref_rows(ref, b0, b1)
            assert np.array_equal(oi, r["ids"]) and np.array_equal(od.view(np.uint32), r["dists"].view(np.uint32))
            assert np.array_equal(oc, r["counts"])
    st = fann.fann_pool_stats(pool)
    assert st["calls"] == 12 and st["in_use"] == 0 and st["n_blocks"] == 2 and st["high_water"] == 1
    # other posting lists loaded under a live pool: graphs captured for the old arrays must not be replayed
    ids2 = torch.flip(w.list_ids, dims=[0]).contiguous()
    ix.load_lists(w.list_offsets.to(DEV), ids2.to(DEV))
    P = np.ascontiguousarray(w.probes[:3].numpy())
    oi, od, oc = np.zeros((3, k), np.uint32), np.zeros((3, k), np.float32), np.zeros(3, np.uint32)
    fann.fann_search_small_lists(ix.handle, pool, w.queries[:3].contiguous().numpy(), 3, cb, w.cfg.dsub, P, w.cfg.nprobe, k, oi, od, oc)
    r2 = oracle.search_lists(w.queries[:3].numpy(), w.codebooks.numpy(), w.codes.numpy(), w.list_offsets.numpy(),
                             ids2.numpy(), P.view(np.uint32), k)
    assert np.array_equal(oi, r2["ids"]) and np.array_equal(oc, r2["counts"])
    ix.load_lists(w.list_offsets.to(DEV), w.list_ids.to(DEV))
    # what the pool was not created for
    q, off, ids = _sub(w, 0, 5)
    oi, od, oc = np.zeros((5, k), np.uint32), np.zeros((5, k), np.float32), np.zeros(5, np.uint32)
    with pytest.raises(fann.FannError):
        fann.fann_search_small(ix.handle, pool, q.numpy(), 5, cb, w.cfg.dsub, off.numpy(), ids.numpy(), k, oi, od, oc)
    with pytest.raises(fann.FannError):
        fann.fann_search_small(ix.handle, pool, q.numpy()[:1], 1, cb, w.cfg.dsub, off.numpy()[:2], ids.numpy(), 2 * k, oi, od, oc)
    fann.fann_pool_destroy(pool)
    ix.close()


def test_pool_block_holds_every_batch_size_up_to_max_b(fann, wl, ref):
    """The workspace of a call is not largest at max_B: small batches take several scan CTAs per query (partial top-k
    lists) and up to 32 dedup classes per query.  A pool created for max_B must serve every B <= max_B, through both
    forms, with the oracle's bytes."""
    w = wl
    ix = fann.FannIndex(0)
    ix.load_codes(w.codes.to(DEV))
    ix.load_lists(w.list_offsets.to(DEV), w.list_ids.to(DEV))
    max_B = w.cfg.B
    pool = _pool(fann, ix, w, 1, max_B)
    cb = w.codebooks.to(DEV)
    k = w.cfg.k
    for B in list(range(1, 12)) + [16, 18, 19, 24, 30, 37, 38, max_B]:
        q, off, ids = _sub(w, 0, B)
        P = np.ascontiguousarray(w.probes[:B].numpy())
        r = _ref_rows(ref, 0, B)
        for form in ("lists", "ids"):
            oi, od, oc = np.zeros((B, k), np.uint32), np.zeros((B, k), np.float32), np.zeros(B, np.uint32)
            if form == "lists":
                fann.fann_search_small_lists(ix.handle, pool, q.numpy(), B, cb, w.cfg.dsub, P, w.cfg.nprobe, k, oi, od, oc)
            else:
                fann.fann_search_small(ix.handle, pool, q.numpy(), B, cb, w.cfg.dsub, off.numpy(), ids.numpy(), k, oi, od, oc)
            assert np.array_equal(oi, r["ids"]) and np.array_equal(od.view(np.uint32), r["dists"].view(np.uint32)), (B, form)
            assert np.array_equal(oc, r["counts"])
    fann.fann_pool_destroy(pool)
    ix.close()


def test_concurrent_host_threads_one_handle(fann, wl, ref):
    """PAPER.md:L204 "each CPU thread handles an individual query": 8 host threads, one handle, a pool of 3 blocks
    (so calls also wait for a block), every query answered once through both entry forms; the bytes are the
    oracle's, whatever the interleaving."""
    w = wl
    ix = fann.FannIndex(0)
    ix.load_codes(w.codes.to(DEV))
    ix.load_lists(w.list_offsets.to(DEV), w.list_ids.to(DEV))
    pool = _pool(fann, ix, w, 3, 2)
    cb = w.codebooks.to(DEV)
    k, B_all = w.cfg.k, w.cfg.B
    got_ids = np.zeros((2, B_all, k), np.uint32)
    got_d = np.zeros((2, B_all, k), np.float32)
    errors = []

    def worker(t, n_threads):
        try:
            for b0 in range(2 * t, B_all, 2 * n_threads):
                b1 = min(b0 + 2, B_all)
                B = b1 - b0
                q, off, ids = _sub(w, b0, b1)
                oi, od, oc = np.zeros((B, k), np.uint32), np.zeros((B, k), np.float32), np.zeros(B, np.uint32)
                fann.fann_search_small(ix.handle, pool, q.numpy(), B, cb, w.cfg.dsub, off.numpy(), ids.numpy(), k, oi, od, oc)
                got_ids[0, b0:b1], got_d[0, b0:b1] = oi, od
                P = np.ascontiguousarray(w.probes[b0:b1].numpy())
                fann.fann_search_small_lists(ix.handle, pool, q.numpy(), B, cb, w.cfg.dsub, P, w.cfg.nprobe, k, oi, od, oc)
                got_ids[1, b0:b1], got_d[1, b0:b1] = oi, od
        except Exception as e:                                     # noqa: BLE001
            errors.append(repr(e))

    threads = [threading.Thread(target=worker, args=(t, 8)) for t in range(8)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors
    for form in (0, 1):
        assert np.array_equal(got_ids[form], ref["ids"])
        assert np.array_equal(got_d[form].view(np.uint32), ref["dists"].view(np.uint32))
    st = fann.fann_pool_stats(pool)
    assert st["calls"] == 2 * (B_all // 2) and st["in_use"] == 0 and 1 <= st["high_water"] <= 3
    fann.fann_pool_destroy(pool)
    ix.close()
