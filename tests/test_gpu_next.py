"""CUDA path vs CPU oracle for the rows SURVEY.md 8(f) adds around the hot path, through the C ABI:
posting lists resident in HBM (NEXT-2), heuristic re-ranking / Algorithm 1 (NEXT-1), page-level I/O dedup /
Fig. 8 (NEXT-4)."""
import json
import os

import numpy as np
import pytest
import torch

import oracle
from oracle.parity import NONE, check_band, check_exact
from workloads import CONFIGS, DEFAULT_SEED, make_page_table, make_raw_vectors, make_workload, mini

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


@pytest.fixture(scope="module")
def fann():
    import paper_2409_16576_b200 as f
    from paper_2409_16576_b200.build import build
    build()
    f.load_library()
    return f


def np_u32(t):
    return t.cpu().numpy().view(np.uint32)


def as_dev_u32(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.uint32).view(np.int32)).to(DEV)


# ------------------------------------------------------------------ NEXT-2: posting lists resident in HBM

@pytest.fixture(scope="module")
def wl_int():
    return make_workload(mini("u8_10m_m32", N=400_000, n_lists=800, B=24, codes_mode="histogram"), keep_lists=True)


@pytest.fixture(scope="module")
def wl_tiny():
    return make_workload(CONFIGS["tiny_local"], keep_lists=True)


def _index_with_lists(fann, w):
    ix = fann.FannIndex(0)
    ix.load_codes(w.codes.to(DEV))
    ix.load_lists(w.list_offsets.to(DEV), w.list_ids.to(DEV))
    return ix


def _search_lists(fann, w, probes_np, k=None, cap=None):
    k = k or w.cfg.k
    ix = _index_with_lists(fann, w)
    B = probes_np.shape[0]
    lut = ix.build_lut(w.queries[:B].contiguous().to(DEV), w.codebooks.to(DEV))
    if cap is None:
        cap = int(oracle.expand_lists(w.list_offsets.numpy(), w.list_ids.numpy(), probes_np)[0][-1])
    o = ix.search_lists(lut, as_dev_u32(probes_np), k, cap, check=True)
    torch.cuda.synchronize()
    return ix, (np_u32(o[0]), o[1].cpu().numpy(), np_u32(o[2]), np_u32(o[3]))


@pytest.mark.parametrize("direct", ["1", "0"])
def test_search_lists_equals_oracle_and_the_id_path(fann, wl_int, wl_tiny, monkeypatch, direct):
    """direct = 1: the lists are sorted and indexed at load and the dedup kernel reads every ID-range class straight
    from the probed lists; 0 (FANN_LISTS_DIRECT=0, also the path of lists too long to sort): the candidate array is
    written out and split first.  Same bytes either way."""
    monkeypatch.setenv("FANN_LISTS_DIRECT", direct)
    for w in (wl_int, wl_tiny):
        P = w.probes.numpy().view(np.uint32)
        ix, res = _search_lists(fann, w, P)
        ref = oracle.search_lists(w.queries.numpy(), w.codebooks.numpy(), w.codes.numpy(), w.list_offsets.numpy(),
                                  w.list_ids.numpy(), P, w.cfg.k)
        if w.cfg.integer_exact:
            check_exact(res, ref)
        else:
            off, ids = oracle.expand_lists(w.list_offsets.numpy(), w.list_ids.numpy(), P)
            for b in range(w.cfg.B):
                ai, ad = oracle.query_all(w.queries.numpy()[b], w.codebooks.numpy(), w.codes.numpy(), ids[off[b]:off[b + 1]])
                assert res[3][b] == ai.size
                check_band(res[0][b], res[1][b], res[2][b], ai, ad, w.cfg.k)
        # the same batch as explicit candidate IDs (fann_dedup_scan_topk): same bytes
        lut = ix.build_lut(w.queries.to(DEV), w.codebooks.to(DEV))
        o = ix.dedup_scan_topk(lut, w.cand_offsets.to(DEV), w.cand_ids.to(DEV), w.cfg.k, check=True)
        torch.cuda.synchronize()
        assert np.array_equal(np_u32(o[3]), res[3])
        if w.cfg.integer_exact:
            assert np.array_equal(np_u32(o[0]), res[0]) and np.array_equal(o[1].cpu().numpy(), res[1])
        else:
            # fp32 data: a row's summation order depends on the lane that scores it, and the order of the distinct
            # list on which store wins a slot, so two runs agree within the band, not byte for byte
            assert np.array_equal(np_u32(o[0]), res[0])
            assert np.allclose(o[1].cpu().numpy(), res[1], rtol=2e-6, atol=0)
        ix.close()


@pytest.mark.parametrize("env", [{}, {"FANN_DEDUP_MODE": "1"}, {"FANN_DEDUP_THREADS": "1024"}, {"FANN_LISTS_DIRECT": "0"}])
def test_search_lists_padding_unknown_lists_and_capacity(fann, wl_int, monkeypatch, env):
    """Also with hash classes forced (the direct path then reads whole lists and filters) and with the one-CTA shape."""
    for key, val in env.items():
        monkeypatch.setenv(key, val)
    w = wl_int
    P = w.probes.numpy().view(np.uint32).copy()
    P[0, ::2] = NONE                                             # padding probes
    P[1, :5] = w.cfg.n_lists + 7                                 # names no list
    P[2, :] = NONE                                               # a query with no list at all
    P[3, 1] = P[3, 0]                                            # the same list twice
    _, res = _search_lists(fann, w, P, cap=w.cand_ids.numel() + 1000)
    ref = oracle.search_lists(w.queries.numpy(), w.codebooks.numpy(), w.codes.numpy(), w.list_offsets.numpy(),
                              w.list_ids.numpy(), P, w.cfg.k)
    check_exact(res, ref)
    assert res[2][2] == 0 and res[3][2] == 0
    # a workspace sized for fewer candidates than the batch has: refused, with the count that was needed
    need = int(oracle.expand_lists(w.list_offsets.numpy(), w.list_ids.numpy(), P)[0][-1])
    with pytest.raises(fann.FannError) as err:
        _search_lists(fann, w, P, cap=need - 1)
    assert err.value.code == -5 and err.value.total_cands == need


@pytest.mark.parametrize("outputs", ["pinned", "pageable", "pinned_copied"])
def test_search_lists_host_entry(fann, wl_int, monkeypatch, outputs):
    """Pinned output arrays are written by the kernels themselves, pageable ones through a staged copy
    (FANN_HOST_DIRECT=0: always the copy): the same bytes."""
    if outputs == "pinned_copied":
        monkeypatch.setenv("FANN_HOST_DIRECT", "0")
    w = wl_int
    ix, res = _search_lists(fann, w, w.probes.numpy().view(np.uint32))
    B, k, nprobe = w.cfg.B, w.cfg.k, w.cfg.nprobe
    cap = w.cand_ids.numel()
    need = fann.fann_search_lists_host_scratch_bytes(ix.handle, B, w.cfg.dsub, nprobe, cap, k)
    scratch = torch.empty(need, dtype=torch.uint8, device=DEV)
    q_h, p_h = w.queries.pin_memory(), w.probes.contiguous().pin_memory()
    oi = torch.empty((B, k), dtype=torch.int32)
    od = torch.empty((B, k), dtype=torch.float32)
    oc = torch.empty(B, dtype=torch.int32)
    if outputs != "pageable":
        oi, od, oc = oi.pin_memory(), od.pin_memory(), oc.pin_memory()
    for _ in range(2):
        oi.fill_(0)
        fann.fann_search_lists_host(ix.handle, q_h, B, w.codebooks.to(DEV), w.cfg.dsub, p_h, nprobe, cap, k, oi, od, oc,
                                    scratch, need, torch.cuda.current_stream().cuda_stream)
        assert np.array_equal(oi.numpy().view(np.uint32), res[0]) and np.array_equal(od.numpy(), res[1])
        assert np.array_equal(oc.numpy().view(np.uint32), res[2])
    ix.close()


def test_search_lists_full_size_equals_id_path(fann):
    """configs[1] at full size: the list entry gives the bytes of the candidate-ID entry for the whole batch and
    the oracle's on the first queries."""
    import bench
    cfg = CONFIGS["u8_10m_m32"]
    w = make_workload(cfg, device=DEV, keep_lists=True)
    ix = fann.FannIndex(0)
    ix.load_codes(w.codes)
    ix.load_lists(w.list_offsets, w.list_ids)
    lut = ix.build_lut(w.queries, w.codebooks)
    a = ix.search_lists(lut, w.probes, cfg.k, w.cand_ids.numel(), check=True)
    a = [t.clone() for t in a]
    b = ix.dedup_scan_topk(lut, w.cand_offsets, w.cand_ids, cfg.k, check=True)
    torch.cuda.synchronize()
    for x, y in zip(a, b):
        assert torch.equal(x, y)
    nq = 24
    _, r, _ = bench.oracle_sample(w, nq, w.codes)
    check_exact((np_u32(a[0][:nq]), a[1][:nq].cpu().numpy(), np_u32(a[2][:nq]), np_u32(a[3][:nq])), r)
    ix.close()


# ------------------------------------------------------------------ experiment: list-major code copy, streamed

def _search_stream(fann, ix, w, probes_np, k, cap):
    B = probes_np.shape[0]
    lut = ix.build_lut(w.queries[:B].contiguous().to(DEV), w.codebooks.to(DEV))
    need = fann.fann_search_lists_stream_workspace_bytes(ix.handle, B, cap)
    ws = torch.empty(need, dtype=torch.uint8, device=DEV)
    oi = torch.empty((B, k), dtype=torch.int32, device=DEV)
    od = torch.empty((B, k), dtype=torch.float32, device=DEV)
    oc = torch.empty(B, dtype=torch.int32, device=DEV)
    st = torch.cuda.current_stream().cuda_stream
    fann.fann_search_lists_stream(ix.handle, lut, B, as_dev_u32(probes_np), probes_np.shape[1], cap, k, oi, od, oc, ws, need, st)
    total = fann.fann_search_lists_stream_status(ix.handle, ws, st)
    return np_u32(oi), od.cpu().numpy(), np_u32(oc), total


@pytest.mark.parametrize("k", [1, 100, 1000])
def test_list_major_stream_gives_the_oracles_bytes(fann, wl_int, k):
    """Every candidate is scored, repeats included, and the repeats leave where the top-k buffer is pruned: same
    ids / dists / counts as the oracle (integer data: bytes), also with padding probes, a list named twice (every ID
    of it twice), unknown lists and an empty query."""
    w = wl_int
    ix = _index_with_lists(fann, w)
    fann.fann_build_list_codes(ix.handle)
    P = w.probes.numpy().view(np.uint32).copy()
    P[0, ::2] = NONE
    P[1, :5] = w.cfg.n_lists + 7
    P[2, :] = NONE
    P[3, 1::2] = P[3, 0::2]                                      # every second probe repeats its neighbour
    cap = w.cand_ids.numel() + 1000
    gi, gd, gc, total = _search_stream(fann, ix, w, P, k, cap)
    ref = oracle.search_lists(w.queries.numpy(), w.codebooks.numpy(), w.codes.numpy(), w.list_offsets.numpy(),
                              w.list_ids.numpy(), P, k)
    assert np.array_equal(gi, ref["ids"]) and np.array_equal(gd.view(np.uint32), ref["dists"].view(np.uint32))
    assert np.array_equal(gc, ref["counts"]) and gc[2] == 0
    assert total == int(oracle.expand_lists(w.list_offsets.numpy(), w.list_ids.numpy(), P)[0][-1])
    with pytest.raises(fann.FannError) as err:                   # a workspace sized for fewer candidates: refused
        _search_stream(fann, ix, w, P, k, total - 1)
    assert err.value.code == -5 and err.value.total_cands == total
    ix.close()


def test_list_major_stream_fp32_band(fann, wl_tiny):
    w = wl_tiny
    ix = _index_with_lists(fann, w)
    fann.fann_build_list_codes(ix.handle)
    P = w.probes.numpy().view(np.uint32)
    gi, gd, gc, _ = _search_stream(fann, ix, w, P, w.cfg.k, w.cand_ids.numel())
    off, ids = oracle.expand_lists(w.list_offsets.numpy(), w.list_ids.numpy(), P)
    for b in range(w.cfg.B):
        ai, ad = oracle.query_all(w.queries.numpy()[b], w.codebooks.numpy(), w.codes.numpy(), ids[off[b]:off[b + 1]])
        check_band(gi[b], gd[b], gc[b], ai, ad, w.cfg.k)
    ix.close()


def test_list_major_stream_heavy_repeats(fann):
    """Few distinct vectors, each many times: one short list probed 300 times, k below and above the distinct count
    (the buffer fills with repeats many times over and must still end with each vector once)."""
    rng = np.random.default_rng(11)
    N, M, dsub = 5_000, 32, 4
    codes = rng.integers(0, 256, size=(N, M), dtype=np.uint8)
    cb = rng.integers(0, 256, size=(M, 256, dsub)).astype(np.float32)
    q = rng.integers(0, 256, size=(2, M * dsub)).astype(np.float32)
    lists = [rng.choice(N, 40, replace=False).astype(np.uint32), rng.choice(N, 2000, replace=False).astype(np.uint32)]
    loff = np.array([0, 40, 2040], np.int64)
    lids = np.concatenate(lists)
    P = np.zeros((2, 300), np.uint32)
    P[1, ::3] = 1                                                # query 1: both lists, 200 and 100 times
    ix = fann.FannIndex(0)
    ix.load_codes(torch.from_numpy(codes).to(DEV))
    ix.load_lists(torch.from_numpy(loff).to(DEV), torch.from_numpy(lids.view(np.int32)).to(DEV))
    fann.fann_build_list_codes(ix.handle)

    class W:                                                     # what _search_stream reads
        queries, codebooks = torch.from_numpy(q), torch.from_numpy(cb)
    for k in (10, 64, 1024):
        gi, gd, gc, total = _search_stream(fann, ix, W, P, k, 300 * 2040)
        ref = oracle.search_lists(q, cb, codes, loff, lids, P, k)
        assert np.array_equal(gi, ref["ids"]) and np.array_equal(gd.view(np.uint32), ref["dists"].view(np.uint32))
        assert np.array_equal(gc, ref["counts"])
    ix.close()


# ------------------------------------------------------------------ NEXT-1: heuristic re-ranking (Algorithm 1)

def _pq_stage_tasks(fann, w, n):
    """Top-n candidate IDs of every query in ascending PQ order (the GPU stage's output)."""
    ix = fann.FannIndex(0)
    ix.load_codes(w.codes.to(DEV))
    lut = ix.build_lut(w.queries.to(DEV), w.codebooks.to(DEV))
    o = ix.dedup_scan_topk(lut, w.cand_offsets.to(DEV), w.cand_ids.to(DEV), n, check=True)
    torch.cuda.synchronize()
    return ix, o[0].clone()


def _check_rerank(got, ref, exact):
    ids, dists, counts, batches, reads = got
    assert np.array_equal(np_u32(counts), ref["counts"]), "counts"
    assert np.array_equal(np_u32(batches), ref["batches"]), "mini-batches executed"
    assert np.array_equal(np_u32(reads), ref["reads"]), "vectors read"
    assert np.array_equal(np_u32(ids), ref["ids"]), "ids"
    g = dists.cpu().numpy()
    if exact:
        assert np.array_equal(g.view(np.uint32), ref["dists"].view(np.uint32))
    else:
        fin = np.isfinite(ref["dists64"])
        assert np.all(np.abs(g[fin] - ref["dists64"][fin]) <= 1e-5 * ref["dists64"][fin])
        assert np.all(np.isposinf(g[~fin]))


@pytest.mark.parametrize("bs,k,eps,beta", [(8, 10, 0.15, 2), (16, 10, 0.0, 1), (10, 5, 0.3, 1), (7, 33, 0.1, 3), (200, 10, 0.5, 1)])
def test_rerank_tiny_fp32(fann, tiny_local, bs, k, eps, beta):
    """configs[0]: raw fp32 vectors in HBM, tasks = the GPU stage's top-64 in ascending PQ order."""
    w = tiny_local
    vec = make_raw_vectors(w.cfg, DEFAULT_SEED)
    ix, tasks = _pq_stage_tasks(fann, w, 64)
    ix.load_vectors(vec.to(DEV))
    got = ix.rerank(w.queries.to(DEV), tasks, bs, k, eps, beta)
    torch.cuda.synchronize()
    ref = oracle.rerank(w.queries.numpy(), vec.numpy(), np_u32(tasks), bs, k, eps, beta)
    _check_rerank(got, ref, exact=False)
    if eps > 0 and beta == 1 and bs < 64:
        assert ref["batches"].min() < -(-64 // bs)               # the heuristic really stops early somewhere
    ix.close()


@pytest.mark.parametrize("dtype", [torch.uint8, torch.float32])
def test_rerank_integer_data_bytes(fann, dtype):
    """configs[1] structure (uint8 vectors, codes = true nearest-centroid codes): every distance is an integer
    < 2^24, so ids, distances, stop points compare byte for byte; raw vectors stored as uint8 and as fp32."""
    w = make_workload(mini("u8_10m_m32", N=200_000, n_lists=400, B=32, codes_mode="encode"))
    vec = make_raw_vectors(w.cfg, DEFAULT_SEED)
    assert vec.dtype == torch.uint8
    ix, tasks = _pq_stage_tasks(fann, w, 100)
    ix.load_vectors(vec.to(dtype).to(DEV))
    for bs, k, eps, beta in ((10, 10, 0.15, 2), (25, 10, 0.0, 1), (10, 40, 0.08, 2), (1, 3, 0.5, 4)):
        got = ix.rerank(w.queries.to(DEV), tasks, bs, k, eps, beta)
        torch.cuda.synchronize()
        ref = oracle.rerank(w.queries.numpy(), vec.numpy().astype(np.float32), np_u32(tasks), bs, k, eps, beta)
        _check_rerank(got, ref, exact=True)
    ix.close()


def test_rerank_edge_cases(fann):
    rng = np.random.default_rng(77)
    N, d, B, n = 500, 20, 6, 40
    vec = rng.integers(-128, 128, size=(N, d)).astype(np.int8)
    q = rng.integers(-128, 128, size=(B, d)).astype(np.float32)
    tasks = np.stack([rng.permutation(N)[:n] for _ in range(B)]).astype(np.uint32)
    tasks[0, 10:] = NONE                                          # short list
    tasks[1, :] = NONE                                            # empty list
    tasks[2, 3] = N + 5                                           # IDs outside the array are skipped
    tasks[2, 4] = 2 ** 31
    vec[tasks[3, 5]] = vec[tasks[3, 2]]                           # an exact tie: the earlier task keeps its place
    ix = fann.FannIndex(0)
    ix.load_vectors(torch.from_numpy(vec).to(DEV))
    for bs, k, eps, beta in ((4, 6, 0.2, 2), (100, 50, 0.0, 1), (3, 1, 0.9, 1), (5, 40, 2.0, 1)):
        got = ix.rerank(torch.from_numpy(q).to(DEV), as_dev_u32(tasks), bs, k, eps, beta)
        torch.cuda.synchronize()
        ref = oracle.rerank(q, vec.astype(np.float32), tasks, min(bs, n), k, eps, beta)
        _check_rerank(got, ref, exact=True)
    with pytest.raises(fann.FannError):
        ix.rerank(torch.from_numpy(q).to(DEV), as_dev_u32(tasks), 4, 2000, 0.1, 1)       # k above the maximum
    with pytest.raises(fann.FannError):
        ix.rerank(torch.from_numpy(q).to(DEV), as_dev_u32(tasks), 4, 5, 0.1, 0)          # beta == 0
    ix.close()


def test_rerank_full_size_config1(fann):
    """configs[1] at full size: 10 M raw uint8 vectors in HBM, 1,024 queries, the GPU stage's top-100 re-ranked to
    top-10; the oracle gets the touched rows only (tasks relabelled onto them: Algorithm 1 never looks at an ID's value)."""
    cfg = CONFIGS["u8_10m_m32"]
    w = make_workload(cfg, device=DEV)
    vec = make_raw_vectors(cfg, DEFAULT_SEED, device=DEV)
    ix = fann.FannIndex(0)
    ix.load_codes(w.codes)
    ix.load_vectors(vec)
    lut = ix.build_lut(w.queries, w.codebooks)
    tasks = ix.dedup_scan_topk(lut, w.cand_offsets, w.cand_ids, cfg.k, check=True)[0]
    got = ix.rerank(w.queries, tasks, 10, 10, 0.15, 2)
    torch.cuda.synchronize()
    used, rel = torch.unique(tasks.view(-1), return_inverse=True)
    rows = vec[used.long()].cpu().numpy().astype(np.float32)
    ref = oracle.rerank(w.queries.cpu().numpy(), rows, rel.view(tasks.shape).cpu().numpy().astype(np.uint32), 10, 10, 0.15, 2)
    ref["ids"] = np_u32(used)[ref["ids"]]
    _check_rerank(got, ref, exact=True)
    assert 1 < ref["batches"].mean() < 10                         # early stops happen, and not at once
    ix.close()


# ------------------------------------------------------------------ NEXT-4: page-level I/O dedup (Fig. 8)

def _check_pages(got, want, bs):
    pages, br, tot = (np_u32(t) for t in got)
    wp, wbr, wt = want
    assert np.array_equal(tot, wt) and np.array_equal(br, wbr)
    for b in range(pages.shape[0]):
        pos = 0
        for t in range(br.shape[1]):                              # inside a mini-batch the order is free
            assert np.array_equal(np.sort(pages[b][pos:pos + br[b, t]]), np.sort(wp[b][pos:pos + br[b, t]]))
            pos += br[b, t]
        assert np.all(pages[b][tot[b]:] == NONE)


def test_page_reads_paper_fig8_example(fann):
    g = json.load(open(os.path.join(GOLDEN, "fig8_io_dedup.json")))
    for p8, p9 in g["page_of_v8_v9_either"]:
        page_of = np.arange(100, 110, dtype=np.uint32)
        for vid, pg in g["page_of"].items():
            page_of[int(vid)] = pg
        page_of[8], page_of[9] = p8, p9
        ix = fann.FannIndex(0)
        ix.load_page_table(as_dev_u32(page_of), 200)
        pages, br, tot = ix.page_reads(as_dev_u32(np.array([g["tasks"]])), g["batch_size"])
        torch.cuda.synchronize()
        assert np_u32(br)[0].tolist() == g["reads_per_mini_batch"] and int(tot[0]) == 4
        assert sorted(np_u32(pages)[0][:2].tolist()) == g["pages_read_mini_batch_0"]
        assert sorted(np_u32(pages)[0][2:4].tolist()) == g["pages_read_mini_batch_1"]
        ix.close()


def test_page_reads_equal_the_oracle(fann, tiny_local):
    w = tiny_local
    page_of, n_pages = make_page_table(w.cfg, DEFAULT_SEED, elem_bytes=4)         # 8 fp32 vectors of 128 dims per 4 KB page
    ix, tasks = _pq_stage_tasks(fann, w, 64)
    ix.load_page_table(page_of.to(DEV), n_pages)
    t_np = np_u32(tasks)
    rng = np.random.default_rng(3)
    resident = np.zeros((n_pages + 31) // 32, dtype=np.uint32)
    for pg in rng.integers(0, n_pages, size=n_pages // 4):
        resident[pg >> 5] |= np.uint32(1 << (pg & 31))
    limits = rng.integers(0, 9, size=w.cfg.B).astype(np.uint32)
    for bs in (8, 5, 64, 1):
        got = ix.page_reads(tasks, bs)
        torch.cuda.synchronize()
        _check_pages(got, oracle.page_reads(page_of.numpy().view(np.uint32), t_np, bs), bs)
        got = ix.page_reads(tasks, bs, batches_run=as_dev_u32(limits), resident_bits=as_dev_u32(resident))
        torch.cuda.synchronize()
        _check_pages(got, oracle.page_reads(page_of.numpy().view(np.uint32), t_np, bs, max_batches=limits,
                                            resident=resident, n_pages=n_pages), bs)
    # clustered layout: vectors of one query share pages, so fewer page reads than vectors (the point of L190-L198)
    tot = np_u32(ix.page_reads(tasks, 8)[2])
    assert tot.mean() < 0.9 * 64
    ix.close()


def test_rerank_then_page_reads_pipeline(fann, tiny_local):
    """Steps (7) -> (8) -> I/O plan chained on the device: top-n IDs, Algorithm 1's stop point, the pages of exactly
    the mini-batches it executed."""
    w = tiny_local
    vec = make_raw_vectors(w.cfg, DEFAULT_SEED)
    page_of, n_pages = make_page_table(w.cfg, DEFAULT_SEED, elem_bytes=4)
    ix, tasks = _pq_stage_tasks(fann, w, 64)
    ix.load_vectors(vec.to(DEV))
    ix.load_page_table(page_of.to(DEV), n_pages)
    rr = ix.rerank(w.queries.to(DEV), tasks, 8, 10, 0.15, 1)
    got = ix.page_reads(tasks, 8, batches_run=rr[3])
    torch.cuda.synchronize()
    ref = oracle.rerank(w.queries.numpy(), vec.numpy(), np_u32(tasks), 8, 10, 0.15, 1)
    _check_pages(got, oracle.page_reads(page_of.numpy().view(np.uint32), np_u32(tasks), 8, max_batches=ref["batches"]), 8)
    ix.close()
