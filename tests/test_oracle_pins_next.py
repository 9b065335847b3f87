"""Pins of the oracle functions for the rows SURVEY.md 8(f) adds around the hot path: list expansion (NEXT-2),
heuristic re-ranking / Algorithm 1 (NEXT-1), page-level I/O dedup / Fig. 8 (NEXT-4).

As in test_oracle_pins.py, every expected value comes from the paper (Fig. 8), hand arithmetic (tests/golden), a
numpy / textbook routine, brute force or an invariant -- never from the oracle and never from the CUDA path."""
import json
import os

import numpy as np
import pytest
import torch

import oracle
from workloads import DEFAULT_SEED, make_candidates, make_lists, make_probes, mini

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
NONE = 0xFFFFFFFF
rng = np.random.default_rng(4321)


# ------------------------------------------------------------------ NEXT-2: list expansion, PAPER.md:L125 (3)

def _random_lists(n_lists=50, max_len=40, N=5000):
    lens = rng.integers(0, max_len, size=n_lists)
    off = np.zeros(n_lists + 1, dtype=np.int64)
    off[1:] = np.cumsum(lens)
    ids = rng.integers(0, N, size=int(off[-1])).astype(np.uint32)
    return off, ids


def test_expand_equals_python_concatenation():
    off, ids = _random_lists()
    probes = rng.integers(0, 50, size=(7, 9)).astype(np.uint32)
    co, ci = oracle.expand_lists(off, ids, probes)
    want = [np.concatenate([ids[off[l]:off[l + 1]] for l in row] + [np.empty(0, np.uint32)]) for row in probes]
    assert co.tolist() == [0] + np.cumsum([w.size for w in want]).tolist()
    assert np.array_equal(ci, np.concatenate(want))


def test_expand_skips_padding_and_unknown_lists():
    off, ids = _random_lists()
    probes = np.array([[3, NONE, 7, 50, 2 ** 31, 3]], dtype=np.uint32)      # 50 and 2^31 name no list; 3 twice
    co, ci = oracle.expand_lists(off, ids, probes)
    want = np.concatenate([ids[off[3]:off[4]], ids[off[7]:off[8]], ids[off[3]:off[4]]])
    assert np.array_equal(ci, want) and co.tolist() == [0, want.size]
    co, ci = oracle.expand_lists(off, ids, np.full((2, 4), NONE, dtype=np.uint32))
    assert co.tolist() == [0, 0, 0] and ci.size == 0


def test_expand_equals_the_generators_own_expansion():
    """workloads.make_candidates builds the same CSR with torch index arithmetic (a different routine)."""
    cfg = mini("u8_10m_m32", N=300_000, n_lists=600, B=5)
    L = make_lists(cfg, DEFAULT_SEED)
    P = make_probes(cfg, DEFAULT_SEED)
    off, ids = make_candidates(cfg, L, P)
    co, ci = oracle.expand_lists(L.offsets.numpy(), L.ids.numpy(), P.numpy().astype(np.uint32))
    assert np.array_equal(co, off.numpy()) and np.array_equal(ci, ids.numpy().view(np.uint32))


def test_search_lists_is_search_on_the_concatenation_and_ignores_probe_order(tiny_local):
    w = tiny_local
    cfg = w.cfg
    L = make_lists(cfg, DEFAULT_SEED)
    P = make_probes(cfg, DEFAULT_SEED).numpy().astype(np.uint32)
    q, cb, codes = w.queries.numpy(), w.codebooks.numpy(), w.codes.numpy()
    a = oracle.search_lists(q, cb, codes, L.offsets.numpy(), L.ids.numpy(), P, cfg.k)
    b = oracle.search(q, cb, codes, w.cand_offsets.numpy(), w.cand_ids.numpy(), cfg.k)
    for key in ("ids", "dists", "counts", "uniq"):
        assert np.array_equal(a[key], b[key])
    P2 = np.stack([rng.permutation(row) for row in P])
    c = oracle.search_lists(q, cb, codes, L.offsets.numpy(), L.ids.numpy(), P2, cfg.k)
    assert np.array_equal(a["ids"], c["ids"]) and np.array_equal(a["uniq"], c["uniq"])


# ------------------------------------------------------------------ NEXT-1: Algorithm 1

@pytest.fixture(scope="module")
def rr():
    return json.load(open(os.path.join(GOLDEN, "rerank_hand.json")))


def test_rerank_golden_hand_example(rr):
    q = np.array([rr["query"]], dtype=np.float32)
    v = np.array(rr["vectors"], dtype=np.float32)
    tasks = np.array([rr["tasks"]], dtype=np.uint32)
    for case in rr["cases"]:
        r = oracle.rerank(q, v, tasks, rr["batch_size"], rr["k"], case["eps"], case["beta"])
        assert r["batches"][0] == case["batches"], case
        assert r["reads"][0] == case["reads"], case
        assert r["ids"][0].tolist() == case["ids"], case
        assert r["dists"][0].tolist() == case["dists"], case
        assert r["counts"][0] == len(case["ids"])


def _problem(B=6, N=400, d=12, n=96, integer=False):
    if integer:
        v = rng.integers(0, 256, size=(N, d)).astype(np.float32)
        q = rng.integers(0, 256, size=(B, d)).astype(np.float32)
    else:
        v = rng.standard_normal((N, d)).astype(np.float32)
        q = rng.standard_normal((B, d)).astype(np.float32)
    tasks = np.stack([rng.permutation(N)[:n] for _ in range(B)]).astype(np.uint32)
    return q, v, tasks


def _brute_topk(q, v, task_row, k):
    """k smallest of the given tasks under (fp32 distance, position), straight from the raw vectors."""
    d64 = ((q.astype(np.float64)[None, :] - v[task_row].astype(np.float64)) ** 2).sum(1)
    d32 = d64.astype(np.float32)
    order = np.lexsort((np.arange(task_row.size), d32))[:k]
    return task_row[order], d32[order], d64[order]


@pytest.mark.parametrize("integer", [False, True])
def test_rerank_eps_zero_never_stops_and_equals_brute_force_topk(integer):
    """eps = 0: Delta < 0 never holds, every mini-batch runs, Q = exact top-k of all n tasks (textbook kNN)."""
    q, v, tasks = _problem(integer=integer)
    for bs, k in ((8, 10), (96, 5), (7, 33), (200, 96)):
        r = oracle.rerank(q, v, tasks, bs, k, 0.0, 1)
        for b in range(q.shape[0]):
            ids, d32, d64 = _brute_topk(q[b], v, tasks[b], k)
            assert r["batches"][b] == -(-tasks.shape[1] // bs) and r["reads"][b] == tasks.shape[1]
            assert np.array_equal(r["ids"][b][:ids.size], ids)
            assert np.array_equal(r["dists"][b][:ids.size], d32)
            assert np.allclose(r["dists64"][b][:ids.size], d64, rtol=1e-12)


def test_rerank_stop_state_is_topk_of_the_prefix_it_read():
    """Whenever it stops, Q is the exact top-k of the tasks read so far (the heap invariant), and the stop
    obeys the rule: the last beta mini-batches each changed fewer than eps*k members of Q, and no earlier
    run of beta such mini-batches exists."""
    q, v, tasks = _problem(B=8, n=120)
    bs, k = 10, 8
    for eps, beta in ((0.2, 1), (0.3, 2), (0.13, 3), (1.1, 2)):
        r = oracle.rerank(q, v, tasks, bs, k, eps, beta)
        for b in range(q.shape[0]):
            t = int(r["batches"][b])
            ids, d32, _ = _brute_topk(q[b], v, tasks[b][: t * bs], k)
            assert np.array_equal(r["ids"][b], ids) and np.array_equal(r["dists"][b], d32)
            # replay Delta from brute-force prefixes
            prev, run, stop_at = set(), 0, None
            for n_b in range(1, -(-tasks.shape[1] // bs) + 1):
                cur = set(_brute_topk(q[b], v, tasks[b][: n_b * bs], k)[0].tolist())
                delta = len(cur - prev) / k
                run = run + 1 if delta < np.float32(eps) else 0
                prev = cur
                if run >= beta:
                    stop_at = n_b
                    break
            assert t == (stop_at if stop_at is not None else -(-tasks.shape[1] // bs))


def test_rerank_beta_one_stops_after_the_first_quiet_batch():
    """Tasks already in exact-distance order and k <= BatchSize: the first mini-batch fills Q with the true top-k,
    the second changes nothing, so with beta = 1 exactly two mini-batches run."""
    q, v, tasks = _problem(B=4, n=64)
    for b in range(4):
        d = ((q[b][None, :].astype(np.float64) - v[tasks[b]].astype(np.float64)) ** 2).sum(1)
        tasks[b] = tasks[b][np.argsort(d, kind="stable")]
    r = oracle.rerank(q, v, tasks, 16, 10, 0.05, 1)
    assert r["batches"].tolist() == [2] * 4 and r["reads"].tolist() == [32] * 4
    assert np.array_equal(r["ids"], tasks[:, :10])


def test_rerank_ties_padding_and_bad_ids():
    v = np.array([[1.0], [1.0], [1.0], [2.0], [0.0]], dtype=np.float32)       # ids 0,1,2 tie at distance 1
    q = np.array([[0.0]], dtype=np.float32)
    r = oracle.rerank(q, v, np.array([[2, 0, 1, 3]], dtype=np.uint32), 1, 2, 0.0, 1)
    assert r["ids"][0].tolist() == [2, 0]                       # equal distance: the earlier task stays (strict <)
    r = oracle.rerank(q, v, np.array([[3, 7, 4, NONE, 0]], dtype=np.uint32), 2, 3, 0.0, 1)
    assert r["ids"][0].tolist() == [4, 3, NONE] and r["counts"][0] == 2        # 7 >= N skipped, padding ends the list
    assert r["reads"][0] == 2 and np.isposinf(r["dists"][0][2])
    r = oracle.rerank(q, v, np.full((1, 4), NONE, dtype=np.uint32), 2, 3, 0.5, 1)
    assert r["counts"][0] == 0 and r["batches"][0] == 0 and r["ids"][0].tolist() == [NONE] * 3


def test_rerank_is_exact_squared_l2():
    """GetDistance = the textbook squared Euclidean distance (numpy), also for M-dimensional integer data."""
    q, v, tasks = _problem(B=3, N=50, d=128, n=50, integer=True)
    r = oracle.rerank(q, v, tasks, 50, 50, 0.0, 1)
    for b in range(3):
        want = ((q[b][None, :] - v[r["ids"][b]]) ** 2).sum(1)           # exact in fp32: integers < 2^24
        assert np.array_equal(r["dists"][b], want)


# ------------------------------------------------------------------ NEXT-4: Fig. 8

def test_page_reads_paper_fig8_example():
    g = json.load(open(os.path.join(GOLDEN, "fig8_io_dedup.json")))
    tasks = np.array([g["tasks"]], dtype=np.uint32)
    for p8, p9 in g["page_of_v8_v9_either"]:
        page_of = np.arange(100, 110, dtype=np.uint32)           # vectors the example does not mention: pages of their own
        for vid, pg in g["page_of"].items():
            page_of[int(vid)] = pg
        page_of[8], page_of[9] = p8, p9
        pages, br, tot = oracle.page_reads(page_of, tasks, g["batch_size"])
        assert br[0].tolist() == g["reads_per_mini_batch"] and tot[0] == 4
        assert sorted(pages[0][:2].tolist()) == g["pages_read_mini_batch_0"]
        assert sorted(pages[0][2:4].tolist()) == g["pages_read_mini_batch_1"]
        assert np.all(pages[0][4:] == NONE)


def test_page_reads_equal_numpy_unique_and_respect_buffer_and_limits():
    N, n_pages, B, n, bs = 3000, 200, 5, 90, 8
    page_of = rng.integers(0, n_pages, size=N).astype(np.uint32)
    tasks = np.stack([rng.permutation(N)[:n] for _ in range(B)]).astype(np.uint32)
    tasks[1, 70:] = NONE                                          # a shorter list
    tasks[2, 5] = N + 3                                           # an ID outside the table
    pages, br, tot = oracle.page_reads(page_of, tasks, bs)
    for b in range(B):
        valid = tasks[b][(tasks[b] != NONE) & (tasks[b] < N)] if b != 1 else tasks[b][:70]
        want = np.unique(page_of[valid])
        got = pages[b][: tot[b]]
        assert np.array_equal(np.sort(got), want) and br[b].sum() == tot[b]          # every needed page read once
        seen, pos = set(), 0
        for t in range(br.shape[1]):                             # a mini-batch reads only pages no earlier one read
            cur = got[pos: pos + br[b, t]].tolist()
            pos += br[b, t]
            batch_tasks = tasks[b][t * bs:(t + 1) * bs]
            batch_tasks = batch_tasks[(batch_tasks != NONE) & (batch_tasks < N)]
            if b == 1:
                batch_tasks = batch_tasks[: max(0, 70 - t * bs)]
            need = set(page_of[batch_tasks].tolist())
            assert set(cur) == need - seen and len(cur) == len(set(cur))
            seen |= need
    # batch size 1: one read per first occurrence of a page
    pages1, br1, tot1 = oracle.page_reads(page_of, tasks[:1], 1)
    first = [i for i, t in enumerate(tasks[0]) if page_of[t] not in set(page_of[tasks[0][:i]].tolist())]
    assert np.flatnonzero(br1[0]).tolist() == first
    # pages already in the DRAM buffer are never read; a limit on mini-batches cuts the list
    resident = np.zeros((n_pages + 31) // 32, dtype=np.uint32)
    for pg in range(0, n_pages, 3):
        resident[pg >> 5] |= np.uint32(1 << (pg & 31))
    pages_r, _, tot_r = oracle.page_reads(page_of, tasks, bs, resident=resident, n_pages=n_pages)
    for b in range(B):
        full = set(pages[b][: tot[b]].tolist())
        assert set(pages_r[b][: tot_r[b]].tolist()) == {pg for pg in full if pg % 3 != 0}
    lim = np.array([1, 2, 3, 4, 12], dtype=np.uint32)
    pages_l, br_l, tot_l = oracle.page_reads(page_of, tasks, bs, max_batches=lim)
    for b in range(B):
        assert np.array_equal(br_l[b][: lim[b]], br[b][: lim[b]]) and br_l[b][lim[b]:].sum() == 0
        assert np.array_equal(pages_l[b][: tot_l[b]], pages[b][: tot_l[b]])
