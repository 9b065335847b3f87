"""Pins of the CPU oracle (oracle/fann_oracle.c) to things other than itself.

Every expected value below comes from hand arithmetic (tests/golden), a closed
form, an invariant, a numpy/textbook routine or brute force -- never from the
oracle and never from the CUDA path.  Citations are PAPER.md lines.
"""
import itertools
import json
import os

import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
NONE = 0xFFFFFFFF
rng = np.random.default_rng(1234)


# ------------------------------------------------------------------ golden (hand arithmetic)

@pytest.fixture(scope="module")
def hand():
    g = json.load(open(os.path.join(GOLDEN, "lut_adc_hand.json")))
    M, dsub = g["M"], g["dsub"]
    cb = np.full((M, 256, dsub), 100.0, dtype=np.float32)
    cb[0, :4] = np.array(g["centroids"]["sub0"], dtype=np.float32)
    cb[1, :4] = np.array(g["centroids"]["sub1"], dtype=np.float32)
    q = np.array([g["query"]], dtype=np.float32)
    codes = np.zeros((7, M), dtype=np.uint8)
    for i in range(7):
        codes[i] = g["codes"][str(i)]
    return g, q, cb, codes


def test_golden_lut(hand):
    g, q, cb, _ = hand
    lut = oracle.build_lut(q, cb)
    assert lut.shape == (1, 2, 256)
    assert lut[0, 0, :4].tolist() == g["lut"]["sub0"]
    assert lut[0, 1, :4].tolist() == g["lut"]["sub1"]
    assert np.all(lut[0, 0, 4:] == g["lut"]["sub0_other"])
    assert np.all(lut[0, 1, 4:] == g["lut"]["sub1_other"])


def test_golden_adc_and_topk(hand):
    g, q, cb, codes = hand
    lut = oracle.build_lut(q, cb)[0]
    for i in range(7):
        assert oracle.adc(lut, codes, i) == g["adc"][str(i)]
    cand = np.array(g["candidates"], dtype=np.uint32)
    assert oracle.dedup(cand, N=7).tolist() == g["distinct"]
    off = np.array([0, cand.size], dtype=np.int64)
    r = oracle.search(q, cb, codes, off, cand, k=4)
    assert r["ids"][0].tolist() == g["top4_ids"]
    assert r["dists"][0].tolist() == g["top4_dists"]
    assert r["counts"][0] == 4 and r["uniq"][0] == 7
    r = oracle.search(q, cb, codes, off, cand, k=10)
    assert r["ids"][0].tolist() == g["top10_ids"]
    assert r["counts"][0] == g["top10_count"]
    assert np.all(np.isinf(r["dists"][0][7:])) and np.all(r["dists"][0][7:] > 0)


# ------------------------------------------------------------------ (1) lookup table

def _rand_problem(B=3, M=5, dsub=3, integer=False):
    if integer:
        q = rng.integers(-128, 256, size=(B, M * dsub)).astype(np.float32)
        cb = rng.integers(-128, 256, size=(M, 256, dsub)).astype(np.float32)
    else:
        q = rng.standard_normal((B, M * dsub)).astype(np.float32)
        cb = rng.standard_normal((M, 256, dsub)).astype(np.float32)
    return q, cb


def test_lut_zero_query_is_centroid_norm():
    q, cb = _rand_problem()
    q[:] = 0
    lut = oracle.build_lut(q, cb)
    want = (cb.astype(np.float64) ** 2).sum(-1)                    # [M, 256]
    np.testing.assert_allclose(lut, np.broadcast_to(want, lut.shape), rtol=1e-15)


def test_lut_query_equal_to_centroid_gives_exact_zero_and_row_min():
    q, cb = _rand_problem(B=4, M=6, dsub=2)
    js = [7, 0, 255, 100]
    for b, j in enumerate(js):
        q[b] = cb[:, j, :].reshape(-1)
    lut = oracle.build_lut(q, cb)
    for b, j in enumerate(js):
        assert np.all(lut[b, :, j] == 0.0)
        assert np.all(lut[b].min(axis=1) == 0.0)
    assert np.all(lut >= 0)


def test_lut_integer_inputs_match_int64_expansion_exactly():
    # independent formula: |q|^2 - 2 q.c + |c|^2 in exact integer arithmetic
    q, cb = _rand_problem(B=5, M=4, dsub=4, integer=True)
    lut = oracle.build_lut(q, cb)
    qi = q.astype(np.int64).reshape(5, 4, 4)
    ci = cb.astype(np.int64)
    want = ((qi ** 2).sum(-1)[:, :, None] - 2 * np.einsum("bmt,mjt->bmj", qi, ci)
            + (ci ** 2).sum(-1)[None])
    assert np.array_equal(lut, want.astype(np.float64))
    assert lut.max() < 2 ** 24


def test_lut_symmetric_under_swapping_query_and_centroid():
    q, cb = _rand_problem(B=1, M=3, dsub=4)
    lut = oracle.build_lut(q, cb)
    j = 17
    q2 = cb[:, j, :].reshape(1, -1).copy()
    cb2 = cb.copy()
    cb2[:, j, :] = q.reshape(3, 4)
    lut2 = oracle.build_lut(q2, cb2)
    assert np.array_equal(lut[0, :, j], lut2[0, :, j])


def test_lut_indexing_not_transposed():
    # sub-space m uses query dims [m*dsub, (m+1)*dsub) and codebook [m]: one-hot probes
    M, dsub = 3, 2
    cb = np.zeros((M, 256, dsub), dtype=np.float32)
    q = np.zeros((1, M * dsub), dtype=np.float32)
    q[0, 3] = 2.0                                                    # sub-space 1, t = 1
    lut = oracle.build_lut(q, cb)
    assert np.all(lut[0, 1] == 4.0) and np.all(lut[0, 0] == 0) and np.all(lut[0, 2] == 0)
    cb[2, 9, 0] = 3.0
    lut = oracle.build_lut(q, cb)
    assert lut[0, 2, 9] == 9.0 and lut[0, 2, 8] == 0.0 and lut[0, 1, 9] == 4.0


# ------------------------------------------------------------------ (5) dedup

def _brute_distinct(ids, N):
    out = []
    for x in ids:                                                    # O(C^2) textbook
        if x == NONE or x >= N:
            continue
        if not any(x == y for y in out):
            out.append(int(x))
    return sorted(out)


def test_dedup_bruteforce_small():
    for _ in range(20):
        n = int(rng.integers(0, 65))
        ids = rng.integers(0, 40, size=n).astype(np.uint32)
        ids[rng.random(n) < 0.1] = NONE
        assert oracle.dedup(ids, N=30).tolist() == _brute_distinct(ids.tolist(), 30)


def test_dedup_equals_numpy_unique_and_invariants():
    N = 1_000_000
    ids = rng.integers(0, 5000, size=20000).astype(np.uint32) * 199 % N
    ids = ids.astype(np.uint32)
    u = oracle.dedup(ids, N)
    assert np.array_equal(u, np.unique(ids))
    assert u.size <= ids.size and np.all(np.isin(u, ids))
    assert np.array_equal(oracle.dedup(u, N), u)                                 # idempotent
    assert np.array_equal(oracle.dedup(rng.permutation(ids), N), u)              # order-free
    assert np.array_equal(oracle.dedup(np.concatenate([ids, ids]), N), u)        # list twice
    assert np.array_equal(oracle.dedup(np.concatenate([ids, [NONE] * 7]).astype(np.uint32), N), u)


def test_dedup_degenerate():
    assert oracle.dedup(np.array([], dtype=np.uint32), 10).size == 0
    assert oracle.dedup(np.full(100, 7, dtype=np.uint32), 10).tolist() == [7]
    a = np.arange(100, dtype=np.uint32)[::-1].copy()
    assert oracle.dedup(a, 1000).tolist() == list(range(100))
    assert oracle.dedup(np.array([5, 9, 10, 11, NONE, 0], dtype=np.uint32), 10).tolist() == [0, 5, 9]
    # ids near 2^32 are compared as unsigned
    assert oracle.dedup(np.array([0xFFFFFFFE, 1, 0x80000000], dtype=np.uint32), 2 ** 32).tolist() == \
        [1, 0x80000000, 0xFFFFFFFE]


# ------------------------------------------------------------------ (6) ADC, Eq. 1

def test_adc_equals_distance_to_pq_reconstruction():
    B, M, dsub, N = 2, 7, 3, 50
    q, cb = _rand_problem(B, M, dsub)
    codes = rng.integers(0, 256, size=(N, M)).astype(np.uint8)
    lut = oracle.build_lut(q, cb)
    for b in range(B):
        for v in range(N):
            recon = np.concatenate([cb[m, codes[v, m]] for m in range(M)]).astype(np.float64)
            want = ((q[b].astype(np.float64) - recon) ** 2).sum()
            got = oracle.adc(lut[b], codes, v)
            assert abs(got - want) <= 1e-12 * max(1.0, want)


def test_adc_special_cases():
    q, cb = _rand_problem(B=1, M=1, dsub=4)
    codes = rng.integers(0, 256, size=(10, 1)).astype(np.uint8)
    lut = oracle.build_lut(q, cb)
    for v in range(10):                                              # M = 1: one table read
        assert oracle.adc(lut[0], codes, v) == lut[0, 0, codes[v, 0]]
    q, cb = _rand_problem(B=1, M=4, dsub=2)
    cb[:] = 0                                                        # zero codebook: |q|^2
    lut = oracle.build_lut(q, cb)
    codes = rng.integers(0, 256, size=(10, 4)).astype(np.uint8)
    qq = (q.astype(np.float64).reshape(4, 2) ** 2).sum(1)            # per sub-space, summed in order
    want = ((qq[0] + qq[1]) + qq[2]) + qq[3]
    for v in range(10):
        assert oracle.adc(lut[0], codes, v) == want


# ------------------------------------------------------------------ (7) top-n

def test_topk_equals_full_sort_prefix():
    for U, k in [(1000, 10), (1000, 1), (50, 100), (0, 5), (64, 64)]:
        ids = rng.permutation(100000)[:U].astype(np.uint32)
        d = rng.integers(0, 40, size=U).astype(np.float32)           # many ties
        oi, od, cnt = oracle.topk(ids, d, k)
        order = np.lexsort((ids, d))                                 # dist, then id
        c = min(U, k)
        assert cnt == c
        assert np.array_equal(oi[:c], ids[order][:c])
        assert np.array_equal(od[:c], d[order][:c])
        assert np.all(oi[c:] == NONE) and np.all(np.isposinf(od[c:]))
        assert np.all(np.diff(od[:c]) >= 0)
        assert np.unique(oi[:c]).size == c
    ids = np.array([9, 3, 5], dtype=np.uint32)
    d = np.array([2.0, 1.0, 1.0], dtype=np.float32)
    oi, od, _ = oracle.topk(ids, d, 1)
    assert oi[0] == 3 and od[0] == 1.0                                # argmin, tie -> lower id


# ------------------------------------------------------------------ whole path

def _lossless_problem(N=400, M=4, dsub=3, B=6):
    """Every sub-vector of every data vector IS one of the 256 centroids, so the
    PQ reconstruction is the vector itself and Eq. 1 is the exact squared L2."""
    cb = rng.integers(0, 64, size=(M, 256, dsub)).astype(np.float32)
    codes = rng.integers(0, 256, size=(N, M)).astype(np.uint8)
    raw = np.stack([np.concatenate([cb[m, codes[v, m]] for m in range(M)]) for v in range(N)])
    q = rng.integers(0, 64, size=(B, M * dsub)).astype(np.float32)
    return q, cb, codes, raw


def test_lossless_pq_equals_bruteforce_exact_knn():
    q, cb, codes, raw = _lossless_problem()
    N, B, k = raw.shape[0], q.shape[0], 15
    lens = rng.integers(0, 300, size=B)
    lens[2] = 0                                                      # an empty list
    lens[3] = 8                                                      # fewer than k
    off = np.zeros(B + 1, dtype=np.int64)
    off[1:] = np.cumsum(lens)
    cand = rng.integers(0, N, size=off[-1]).astype(np.uint32)
    r = oracle.search(q, cb, codes, off, cand, k)
    for b in range(B):
        c = cand[off[b]:off[b + 1]]
        dist = {int(v): float(((raw[v].astype(np.float64) - q[b]) ** 2).sum()) for v in set(c.tolist())}
        want = sorted(dist.items(), key=lambda kv: (kv[1], kv[0]))[:k]
        cnt = len(want)
        assert r["counts"][b] == cnt and r["uniq"][b] == len(dist)
        assert r["ids"][b, :cnt].tolist() == [v for v, _ in want]
        assert r["dists64"][b, :cnt].tolist() == [dv for _, dv in want]
        assert r["dists"][b, :cnt].tolist() == [np.float32(dv) for _, dv in want]
        assert np.all(r["ids"][b, cnt:] == NONE) and np.all(np.isposinf(r["dists"][b, cnt:]))


def test_metamorphic_permute_duplicate_pad_relabel(tiny_local):
    w = tiny_local
    q = w.queries.numpy()[:8]
    cb = w.codebooks.numpy()
    codes = w.codes.numpy()
    off0 = w.cand_offsets.numpy()
    ids0 = w.cand_ids.numpy().view(np.uint32)
    lists = [ids0[off0[b]:off0[b + 1]] for b in range(8)]
    k = 10

    def run(ls, cds=codes):
        off = np.zeros(len(ls) + 1, dtype=np.int64)
        off[1:] = np.cumsum([len(x) for x in ls])
        return oracle.search(q, cb, cds, off, np.concatenate(ls).astype(np.uint32), k)

    base = run(lists)
    assert np.all(base["uniq"] < [len(x) for x in lists])            # duplicates do occur
    for variant in (
        [rng.permutation(x) for x in lists],
        [np.concatenate([x, x]) for x in lists],
        [np.concatenate([x[:5], [NONE, NONE], x[5:], [NONE]]).astype(np.uint32) for x in lists],
    ):
        r = run(variant)
        for key in ("ids", "dists", "counts", "uniq"):
            assert np.array_equal(r[key], base[key])
    # monotone relabelling of IDs onto a compacted code array (the harness uses
    # this to run the oracle on sampled queries of the 1B-vector configs)
    used = np.unique(np.concatenate(lists))
    rel = [np.searchsorted(used, x).astype(np.uint32) for x in lists]
    r = run(rel, codes[used])
    assert np.array_equal(used[r["ids"]], base["ids"])
    assert np.array_equal(r["dists"], base["dists"]) and np.array_equal(r["uniq"], base["uniq"])


def test_query_all_consistent_with_definitions(tiny_local):
    w = tiny_local
    off = w.cand_offsets.numpy()
    ids = w.cand_ids.numpy().view(np.uint32)
    cb = w.codebooks.numpy().astype(np.float64)
    codes = w.codes.numpy()
    b = 3
    c = ids[off[b]:off[b + 1]]
    ai, ad = oracle.query_all(w.queries.numpy()[b], w.codebooks.numpy(), codes, c)
    assert np.array_equal(ai, np.unique(c))
    qv = w.queries.numpy()[b].astype(np.float64)
    M = cb.shape[0]
    recon = cb[np.arange(M)[None, :], codes[ai].astype(np.int64)].reshape(ai.size, -1)
    want = ((recon - qv) ** 2).sum(1)
    np.testing.assert_allclose(ad, want, rtol=1e-12)
