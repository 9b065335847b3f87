"""CUDA path vs CPU oracle, through the C ABI (python binding = marshalling only).

Integer-valued workloads: byte equality.  Real-valued workloads: the tolerance rules of
DESIGN.md "Parity rules" (1e-5 relative, ties within the band may permute)."""
import numpy as np
import pytest
import torch

import oracle
from oracle.parity import NONE, check_band, check_exact, check_lut
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


def gpu_search(fann, w, k=None, cand=None, check=True, queries=None):
    """Run the whole path on the GPU.  cand = (offsets int64 np, ids uint32 np) overrides w's lists."""
    k = k or w.cfg.k
    ix = fann.FannIndex(0)
    ix.load_codes(w.codes.to(DEV))
    q, cb = (w.queries if queries is None else queries).to(DEV), w.codebooks.to(DEV)
    if cand is None:
        off, ids = w.cand_offsets.to(DEV), w.cand_ids.to(DEV)
    else:
        off = torch.from_numpy(np.ascontiguousarray(cand[0], dtype=np.int64)).to(DEV)
        ids = torch.from_numpy(np.ascontiguousarray(cand[1], dtype=np.uint32).view(np.int32)).to(DEV)
        q = q[: off.numel() - 1].contiguous()
    lut = ix.build_lut(q, cb)
    o = ix.dedup_scan_topk(lut, off, ids, k, check=check)
    torch.cuda.synchronize()
    res = (np_u32(o[0]), o[1].cpu().numpy(), np_u32(o[2]), np_u32(o[3]))
    return ix, lut, res


def orc_search(w, k=None, cand=None, queries=None):
    k = k or w.cfg.k
    q = (w.queries if queries is None else queries).numpy()
    if cand is None:
        off, ids = w.cand_offsets.numpy(), w.cand_ids.numpy().view(np.uint32)
    else:
        off, ids = cand
        q = q[: len(off) - 1]
    return oracle.search(q, w.codebooks.numpy(), w.codes.numpy(), off, ids, k)


def band_all(w, res, k=None, cand=None):
    k = k or w.cfg.k
    if cand is None:
        off, ids = w.cand_offsets.numpy(), w.cand_ids.numpy().view(np.uint32)
    else:
        off, ids = cand
    needed = 0
    for b in range(len(off) - 1):
        ai, ad = oracle.query_all(w.queries.numpy()[b], w.codebooks.numpy(), w.codes.numpy(), ids[off[b]:off[b + 1]])
        assert res[3][b] == ai.size, f"query {b}: uniq {res[3][b]} != {ai.size}"
        needed += check_band(res[0][b], res[1][b], res[2][b], ai, ad, k)
    return needed


# ------------------------------------------------------------------ workloads

@pytest.fixture(scope="module")
def w_int():
    """configs[1] structure (uint8 data, M=32, k=100) at a size the oracle finishes in seconds;
    ~32k candidates per query -> several table partitions, ragged tails."""
    return make_workload(mini("u8_10m_m32", N=400_000, n_lists=800, B=24, codes_mode="histogram"))


@pytest.fixture(scope="module")
def w_i8():
    """configs[3] structure (int8, M=25 -> rows padded to 32 bytes, power-law lists)."""
    return make_workload(mini("i8_1b_m25", N=300_000, n_lists=600, B=16))


@pytest.fixture(scope="module")
def w_k1000():
    """configs[4] structure (M=64, nprobe=256, k=1000): ~128k candidates per query."""
    return make_workload(mini("u8_1b_m64", N=600_000, n_lists=1_200, B=6))


@pytest.fixture(scope="module")
def w_f32():
    """configs[2] structure (fp32 Gaussian normalised, M=48): tolerance regime."""
    return make_workload(mini("f32_100m_m48", N=300_000, n_lists=600, B=8))


# ------------------------------------------------------------------ (1) lookup table

@pytest.mark.parametrize("name", ["tiny", "tiny_local"])
def test_lut_tiny(fann, name, request):
    w = request.getfixturevalue(name)
    ix = fann.FannIndex(0)
    ix.load_codes(w.codes.to(DEV))
    lut = ix.build_lut(w.queries.to(DEV), w.codebooks.to(DEV)).cpu().numpy()
    check_lut(lut, oracle.build_lut(w.queries.numpy(), w.codebooks.numpy()))


def test_lut_integer_exact_and_fp32(fann, w_int, w_f32, w_i8):
    for w in (w_int, w_i8, w_f32):
        ix = fann.FannIndex(0)
        ix.load_codes(w.codes[:1000].contiguous().to(DEV))
        lut = ix.build_lut(w.queries.to(DEV), w.codebooks.to(DEV)).cpu().numpy()
        lut64 = oracle.build_lut(w.queries.numpy(), w.codebooks.numpy())
        check_lut(lut, lut64)
        if w.cfg.integer_exact:
            assert np.array_equal(lut.astype(np.float64), lut64)


@pytest.mark.parametrize("M,dsub", [(5, 3), (7, 1), (16, 8), (25, 4), (3, 2), (64, 2), (6, 5)])
def test_lut_any_shape(fann, M, dsub):
    """Sub-space counts that do not fill a block of 4, and dsub with and without the float4 codebook path."""
    rng = np.random.default_rng(M * 100 + dsub)
    B = 37
    q = torch.from_numpy(rng.normal(size=(B, M * dsub)).astype(np.float32))
    cb = torch.from_numpy(rng.normal(size=(M, 256, dsub)).astype(np.float32))
    ix = fann.FannIndex(0)
    ix.load_codes(torch.zeros((8, M), dtype=torch.uint8, device=DEV))
    lut = ix.build_lut(q.to(DEV), cb.to(DEV)).cpu().numpy()
    check_lut(lut, oracle.build_lut(q.numpy(), cb.numpy()))


def test_lut_query_on_centroid_is_exact_zero(fann, tiny):
    w = tiny
    q = w.queries.clone()
    q[0] = w.codebooks[:, 17, :].reshape(-1)
    ix = fann.FannIndex(0)
    ix.load_codes(w.codes[:100].contiguous().to(DEV))
    lut = ix.build_lut(q.to(DEV), w.codebooks.to(DEV)).cpu().numpy()
    assert np.all(lut[0, :, 17] == 0.0) and np.all(lut >= 0)


# ------------------------------------------------------------------ (5) dedup

def _dedup_check(fann, w, off, ids, ascending=None):
    """ascending: query indices whose distinct list must come out in ascending order (ordered placement),
    up to the shuffle inside a compaction step, the few IDs displaced by probing and the partition seams."""
    ix = fann.FannIndex(0)
    ix.load_codes(w.codes.to(DEV))
    o = torch.from_numpy(np.ascontiguousarray(off, dtype=np.int64)).to(DEV)
    i = torch.from_numpy(np.ascontiguousarray(ids, dtype=np.uint32).view(np.int32)).to(DEV)
    uids, ucnt = ix.dedup_only(o, i)
    torch.cuda.synchronize()
    uids, ucnt = np_u32(uids), np_u32(ucnt)
    for b in range(len(off) - 1):
        want = oracle.dedup(ids[off[b]:off[b + 1]], w.cfg.N)
        got = uids[off[b]:off[b] + ucnt[b]]
        assert ucnt[b] == want.size, f"query {b}: {ucnt[b]} != {want.size}"
        assert np.array_equal(np.sort(got), want), f"query {b}: distinct sets differ"
        if ascending and b in ascending and got.size > 1:
            g64 = got.astype(np.int64)                         # ascending beyond the 128-slot compaction step
            far = np.count_nonzero(g64[512:] < g64[:-512])
            # each partition of the query (at most 16) contributes one ascending segment, in any order
            assert far <= 0.01 * got.size + 16 * 512, f"query {b}: {far} of {got.size} ids descend over a distance of 512"


def test_dedup_sets_bit_exact(fann, tiny_local, w_int, w_k1000):
    for w in (tiny_local, w_int, w_k1000):
        _dedup_check(fann, w, w.cand_offsets.numpy(), w.cand_ids.numpy().view(np.uint32))


def test_dedup_adversarial(fann, tiny_local):
    w = tiny_local
    N = w.cfg.N
    rng = np.random.default_rng(5)
    lists = [
        np.full(5000, 4242, dtype=np.uint32),                                   # all duplicates
        np.arange(3000, dtype=np.uint32),                                       # no duplicate
        np.array([], dtype=np.uint32),                                          # empty
        np.full(100, NONE, dtype=np.uint32),                                    # only padding
        np.array([N, N + 1, 2 ** 31, NONE - 1, 5], dtype=np.uint32),            # out of range except one
        rng.integers(0, 50, size=40_000).astype(np.uint32),                     # 50 ids, long list
        np.concatenate([rng.permutation(N)[:60_000].astype(np.uint32)] * 2),    # 120k, each twice
        rng.permutation(N)[:41_500].astype(np.uint32),      # no repeat, fills one table to 74 %: many store races
        rng.permutation(N)[:20_900].astype(np.uint32),      # the same for the two-CTA shape's half table
    ]
    off = np.zeros(len(lists) + 1, dtype=np.int64)
    off[1:] = np.cumsum([len(x) for x in lists])
    _dedup_check(fann, w, off, np.concatenate(lists))


def _bunched_lists(N, rng):
    """Candidate lists whose IDs are NOT spread evenly over [0, N): the order-preserving table
    would pile them up, so the library must fall back to hashed placement."""
    runs = np.concatenate([np.arange(s, s + 400, dtype=np.uint32) for s in rng.integers(0, N - 400, size=60)])
    dense = rng.integers(N // 3, N // 3 + 30_000, size=45_000).astype(np.uint32)         # one narrow range
    half = np.concatenate([rng.integers(0, N // 64, size=20_000), rng.integers(0, N, size=5_000)]).astype(np.uint32)
    spread = rng.permutation(N)[:30_000].astype(np.uint32)                               # evenly spread: ordered
    return [np.concatenate([runs, runs[::-1]]), dense, rng.permutation(half), spread]


@pytest.mark.parametrize("force", [None, "0", "1"])
def test_dedup_placement_modes(fann, tiny_local, monkeypatch, force):
    """Ordered, hashed and per-query placement give the same distinct sets; evenly spread lists come
    out ascending when the placement is ordered (what the scan kernel's gather relies on for speed)."""
    if force is None:
        monkeypatch.delenv("FANN_DEDUP_MODE", raising=False)
    else:
        monkeypatch.setenv("FANN_DEDUP_MODE", force)
    w = tiny_local
    lists = _bunched_lists(w.cfg.N, np.random.default_rng(11))
    off = np.zeros(len(lists) + 1, dtype=np.int64)
    off[1:] = np.cumsum([len(x) for x in lists])
    _dedup_check(fann, w, off, np.concatenate(lists), ascending=None if force == "1" else {3})


# ------------------------------------------------------------------ whole path

def test_tiny_configs_tolerance_regime(fann, tiny, tiny_local):
    for w in (tiny, tiny_local):
        _, _, res = gpu_search(fann, w)
        band_all(w, res)


def test_integer_exact_configs_bytes(fann, w_int, w_i8):
    for w in (w_int, w_i8):
        ix, _, res = gpu_search(fann, w)
        check_exact(res, orc_search(w))
        assert ix.info()["kernel_launches"] >= 4


def test_k1000_partitions_bytes(fann, w_k1000):
    w = w_k1000
    _, _, res = gpu_search(fann, w)
    ref = orc_search(w)
    check_exact(res, ref)
    assert ref["uniq"].min() > 1000                      # k < U: selection really happens
    # integer data: exact ties inside the top-1000 exist and are ordered by id
    ties = sum(int(np.sum(np.diff(ref["dists"][b]) == 0)) for b in range(w.cfg.B))
    assert ties > 0


@pytest.mark.parametrize("env", [
    {"FANN_DEDUP_THREADS": "512"},                       # two dedup CTAs per SM, half tables
    {"FANN_DEDUP_THREADS": "1024"},                      # one dedup CTA per SM
    {"FANN_PARTITION": "0"},                             # dedup passes filter the whole list themselves
    {"FANN_DEDUP_MODE": "1"},                            # hashed placement and hash classes
    {"FANN_DEDUP_MODE": "1", "FANN_PARTITION": "0"},
    {"FANN_SCAN_RING": "0"},                             # code rows through registers
    {"FANN_CHUNKS": "4"},                                # dedup of chunk i+1 on a second stream beside the scan of chunk i
    {"FANN_SPLIT_SCAN": "0"},                            # one scan CTA per query even when the batch is smaller than the machine
])
def test_every_code_path_gives_the_same_bytes(fann, w_k1000, w_i8, monkeypatch, env):
    """The library picks CTA shapes, placement and staging by itself; each alternative (also the
    fallbacks it takes on bunched IDs or refused splits) must give the oracle's bytes."""
    for key in ("FANN_DEDUP_THREADS", "FANN_PARTITION", "FANN_DEDUP_MODE", "FANN_SCAN_RING", "FANN_CHUNKS", "FANN_SPLIT_SCAN"):
        monkeypatch.delenv(key, raising=False)
    for key, val in env.items():
        monkeypatch.setenv(key, val)
    for w in (w_k1000, w_i8):
        _, _, res = gpu_search(fann, w)
        check_exact(res, orc_search(w))


def test_fp32_config_band(fann, w_f32):
    _, _, res = gpu_search(fann, w_f32)
    band_all(w_f32, res)


@pytest.mark.parametrize("d,M", [(15, 5), (7, 7), (40, 40), (34, 17), (130, 26)])
def test_odd_geometries_band(fann, d, M):
    """PQ shapes outside BASELINE's five: M that does not fill a stored row (padding bytes must not
    contribute), dsub without the float4 table path, rows of 16, 32 and 64 bytes."""
    cfg = CONFIGS["tiny_local"].scaled(name=f"odd_d{d}_M{M}", N=60_000, n_lists=600, B=10, d=d, M=M, k=50)
    w = make_workload(cfg)
    _, lut, res = gpu_search(fann, w)
    check_lut(lut.cpu().numpy(), oracle.build_lut(w.queries.numpy(), w.codebooks.numpy()))
    band_all(w, res)


def _hash_round1(x):
    """First round of the library's slot hash (fann.h: "IDs chosen to collide under the library's hash")."""
    x = x.astype(np.uint64)
    return ((x ^ (x >> np.uint64(16))) * np.uint64(0x7feb352d)) & np.uint64(0xFFFFFFFF)


def test_table_overflow_is_reported_not_silent(fann):
    """IDs CHOSEN to collide: 100,000 distinct IDs whose hash falls into class 0 whatever the number of classes
    (top four hash bits zero, up to 16 classes).  Neither ID-range classes (the IDs sit in part of [0, N)) nor hash
    classes can split them, so one table must overflow: the call has to say so through fann_workspace_status,
    never return a quiet wrong answer."""
    import paper_2409_16576_b200 as f
    N, M = 4_000_000, 16
    allv = np.arange(2_400_000, dtype=np.uint32)
    ids = allv[(_hash_round1(allv) >> np.uint64(28)) == 0][:100_000]
    assert ids.size == 100_000
    ix = f.FannIndex(0)
    ix.load_codes(torch.zeros((N, M), dtype=torch.uint8, device=DEV))
    lut = torch.zeros((1, M, 256), dtype=torch.float32, device=DEV)
    o = torch.from_numpy(np.array([0, ids.size], dtype=np.int64)).to(DEV)
    i = torch.from_numpy(ids.view(np.int32)).to(DEV)
    with pytest.raises(f.FannError) as err:
        ix.dedup_scan_topk(lut, o, i, 10, check=True)
    assert err.value.code == -6                               # FANN_EOVERFLOW
    assert ix.info()["table_slots"] < 100_000                 # the premise: one table cannot hold them
    ix.close()


@pytest.mark.parametrize("frac,count", [(0.4, 80_000), (0.5, 160_000), (0.35, 120_000), (0.06, 60_000)])
def test_dedup_ids_concentrated_in_part_of_the_range(fann, frac, count):
    """IDs spread evenly over only [0, frac N): no fine-grained bunching for mode_kernel's sample to see, but an
    ID-range class of the lower part receives far more than its share.  The partition kernel counts the classes
    exactly and must fall back to hash classes by itself (no FANN_DEDUP_MODE): distinct sets equal the oracle's."""
    N, M = 2_000_000, 16
    rng = np.random.default_rng(int(frac * 100) + count)
    lists = [rng.integers(0, int(frac * N), size=count).astype(np.uint32),
             rng.permutation(int(frac * N))[:count // 2].astype(np.uint32),
             rng.integers(0, N, size=count).astype(np.uint32)]                  # an evenly spread list beside them
    off = np.zeros(len(lists) + 1, dtype=np.int64)
    off[1:] = np.cumsum([len(x) for x in lists])
    ids = np.concatenate(lists)
    ix = fann.FannIndex(0)
    ix.load_codes(torch.zeros((N, M), dtype=torch.uint8, device=DEV))
    o = torch.from_numpy(off).to(DEV)
    i = torch.from_numpy(ids.view(np.int32)).to(DEV)
    uids, ucnt = ix.dedup_only(o, i)                          # raises on FANN_EOVERFLOW
    torch.cuda.synchronize()
    uids, ucnt = np_u32(uids), np_u32(ucnt)
    for b in range(len(lists)):
        want = oracle.dedup(ids[off[b]:off[b + 1]], N)
        assert ucnt[b] == want.size
        assert np.array_equal(np.sort(uids[off[b]:off[b] + ucnt[b]]), want)
    ix.close()


def test_understated_total_cands_is_refused_not_corrupting(fann, w_int):
    """total_cands is the caller's promise that sized the workspace.  If it does not equal cand_offsets[B] the
    library must not touch the lists (it would write past its arrays): fann_workspace_status says FANN_EINVAL and
    every query reports zero candidates."""
    import paper_2409_16576_b200 as f
    w = w_int
    ix = f.FannIndex(0)
    ix.load_codes(w.codes.to(DEV))
    lut = ix.build_lut(w.queries.to(DEV), w.codebooks.to(DEV))
    off, ids = w.cand_offsets.to(DEV), w.cand_ids.to(DEV)
    B, k = w.cfg.B, 10
    total = ids.numel()
    for claimed in (total // 2, total - 1, 1):
        ws = torch.empty(f.fann_workspace_bytes(ix.handle, B, claimed, k) + 4096, dtype=torch.uint8, device=DEV)
        ws[-4096:] = 0xAB                                      # canary behind the workspace proper
        out = (torch.zeros((B, k), dtype=torch.int32, device=DEV), torch.zeros((B, k), device=DEV),
               torch.full((B,), 77, dtype=torch.int32, device=DEV), torch.full((B,), 77, dtype=torch.int32, device=DEV))
        f.fann_dedup_scan_topk(ix.handle, lut, B, off, ids, claimed, k, out[0], out[1], out[2], out[3],
                               ws, ws.numel() - 4096, torch.cuda.current_stream().cuda_stream)
        with pytest.raises(f.FannError) as err:
            f.fann_workspace_status(ix.handle, ws, torch.cuda.current_stream().cuda_stream)
        assert err.value.code == -1                           # FANN_EINVAL
        assert bool((ws[-4096:] == 0xAB).all())
        assert bool((out[2] == 0).all()) and bool((out[3] == 0).all()) and bool((out[0] == -1).all())
    ix.close()


def test_misaligned_pointers_are_refused(fann, tiny):
    import paper_2409_16576_b200 as f
    w = tiny
    ix = f.FannIndex(0)
    ix.load_codes(w.codes.to(DEV))
    B, M = w.cfg.B, w.cfg.M
    q, cb = w.queries.to(DEV), w.codebooks.to(DEV)
    raw = torch.empty(B * M * 256 + 8, dtype=torch.float32, device=DEV)
    lut_bad = raw[1:1 + B * M * 256]                          # 4-byte aligned only
    with pytest.raises(f.FannError) as err:
        f.fann_build_lut(ix.handle, q, B, cb, w.cfg.dsub, lut_bad, None)
    assert err.value.code == -1
    lut = ix.build_lut(q, cb)
    off, ids = w.cand_offsets.to(DEV), w.cand_ids.to(DEV)
    out = [torch.empty((B, 10), dtype=torch.int32, device=DEV), torch.empty((B, 10), device=DEV)]
    ws = ix.workspace(B, ids.numel(), 10)
    torch.cuda.synchronize()
    lut_copy = raw[1:1 + B * M * 256].copy_(lut.view(-1))
    with pytest.raises(f.FannError) as err:
        f.fann_dedup_scan_topk(ix.handle, lut_copy, B, off, ids, ids.numel(), 10, out[0], out[1], None, None,
                               ws, ws.numel(), None)
    assert err.value.code == -1
    ix.close()


def test_edge_cases(fann, w_int):
    w = w_int
    N = w.cfg.N
    rng = np.random.default_rng(9)
    base = w.cand_ids.numpy().view(np.uint32)[: int(w.cand_offsets[1])]
    lists = [
        np.array([], dtype=np.uint32),                                          # empty list -> count 0
        base[:37],                                                              # fewer than k distinct
        np.full(2000, base[3], dtype=np.uint32),                                # one distinct id
        np.concatenate([[NONE] * 5, base[:500], [N, N + 7], [NONE] * 3]).astype(np.uint32),
        base,                                                                   # a normal list
        np.concatenate([base, base]),                                           # appended to itself
        rng.permutation(base),                                                  # permuted
        rng.permutation(N)[:150_000].astype(np.uint32),                         # max-skew: 150k distinct
    ]
    off = np.zeros(len(lists) + 1, dtype=np.int64)
    off[1:] = np.cumsum([len(x) for x in lists])
    cand = (off, np.concatenate(lists))
    q = w.queries.clone()
    q[5] = q[4]                                                                 # same query for the
    q[6] = q[4]                                                                 # metamorphic triple
    for k in (100, 1, 1024, 7):
        _, _, res = gpu_search(fann, w, k=k, cand=cand, queries=q)
        ref = orc_search(w, k=k, cand=cand, queries=q)
        check_exact(res, ref)
        assert res[2][0] == 0 and np.all(res[0][0] == NONE) and np.all(np.isposinf(res[1][0]))
        assert res[2][2] == 1
        for a, b in ((4, 5), (4, 6)):                                           # metamorphic
            assert np.array_equal(res[0][a], res[0][b]) and np.array_equal(res[1][a], res[1][b])


@pytest.mark.parametrize("seed", range(40))
def test_random_shapes_differential(fann, seed):
    """Differential test on random problem shapes nobody chose: M, dsub, N, batch size (also below half the SMs: several
    scan CTAs per query), list lengths from 0 to 150 k with a random share of repeats, invalid IDs sprinkled in, k from
    1 to 1024, IDs either spread over [0, N) or bunched.  Integer data, so the oracle's bytes are the bar; the lookup
    table is checked too."""
    rng = np.random.default_rng(1000 + seed)
    M = int(rng.choice([1, 3, 8, 16, 17, 25, 32, 33, 48, 64]))
    dsub = int(rng.choice([1, 2, 4, 8]))
    N = int(rng.choice([300, 5_000, 70_000, 400_000]))
    B = int(rng.choice([1, 2, 5, 13, 40, 75, 150, 300]))
    k = int(rng.choice([1, 2, 10, 100, 257, 1000, 1024]))
    codes = rng.integers(0, 256, size=(N, M), dtype=np.uint8)
    cb = rng.integers(0, 16, size=(M, 256, dsub)).astype(np.float32)
    q = rng.integers(0, 16, size=(B, M * dsub)).astype(np.float32)
    lists = []
    budget = 1_500_000
    for b in range(B):
        kind = rng.integers(0, 6)
        n = int(min(budget // B * 2, rng.choice([0, 1, 30, 700, 9_000, 40_000, 150_000])))
        if kind == 0:
            x = rng.integers(0, N, n)                                               # spread, natural repeats
        elif kind == 1:
            x = rng.integers(0, max(1, N // 50), n)                                 # bunched at the bottom: heavy repeats
        elif kind == 2:
            x = N - 1 - rng.integers(0, max(1, N // 7), n)                          # bunched at the top
        elif kind == 3:
            x = np.repeat(rng.integers(0, N, max(1, n // 5)), 5)[:n]                # every ID five times in a row
        elif kind == 4:
            x = np.sort(rng.integers(0, N, n))                                      # ascending
        else:
            x = np.concatenate([rng.integers(0, N, n // 2), rng.integers(N, 2 ** 32 - 1, n - n // 2)])   # half invalid
        x = x.astype(np.uint32)
        if n and kind != 5 and rng.random() < 0.5:
            x[rng.integers(0, n, max(1, n // 100))] = NONE                          # padding entries
        lists.append(x)
    off = np.zeros(B + 1, dtype=np.int64)
    off[1:] = np.cumsum([len(x) for x in lists])
    ids = np.concatenate(lists) if off[-1] else np.zeros(0, np.uint32)
    ix = fann.FannIndex(0)
    ix.load_codes(torch.from_numpy(codes).to(DEV))
    lut = ix.build_lut(torch.from_numpy(q).to(DEV), torch.from_numpy(cb).to(DEV))
    assert np.array_equal(lut.cpu().numpy(), oracle.build_lut(q, cb).astype(np.float32)), "integer tables must be exact"
    ids_dev = torch.from_numpy(ids.view(np.int32)).to(DEV) if ids.size else torch.zeros(1, dtype=torch.int32, device=DEV)
    o = ix.dedup_scan_topk(lut, torch.from_numpy(off).to(DEV), ids_dev, k, total_cands=int(off[-1]), check=True)
    torch.cuda.synchronize()
    ref = oracle.search(q, cb, codes, off, ids, k)
    check_exact((np_u32(o[0]), o[1].cpu().numpy(), np_u32(o[2]), np_u32(o[3])), ref)
    ix.close()


def test_argument_errors(fann, tiny):
    w = tiny
    ix = fann.FannIndex(0)
    with pytest.raises(fann.FannError):                                         # no codes yet
        fann.fann_workspace_bytes(ix.handle, 4, 100, 10)
    ix.load_codes(w.codes[:1000].contiguous().to(DEV))
    lut = ix.build_lut(w.queries.to(DEV), w.codebooks.to(DEV))
    off, ids = w.cand_offsets.to(DEV), w.cand_ids.to(DEV)
    with pytest.raises(fann.FannError) as e:
        ix.dedup_scan_topk(lut, off, ids, k=fann.FANN_MAX_K + 1)
    assert e.value.code in (-1, -4)
    B = w.cfg.B
    out = [torch.empty((B, 10), dtype=torch.int32, device=DEV), torch.empty((B, 10), device=DEV)]
    small = torch.empty(256, dtype=torch.uint8, device=DEV)
    with pytest.raises(fann.FannError) as e:
        fann.fann_dedup_scan_topk(ix.handle, lut, B, off, ids, ids.numel(), 10, out[0], out[1], None, None,
                                  small, small.numel())
    assert e.value.code == -5
    with pytest.raises(fann.FannError):
        ix.load_codes(w.codes[:10, :8].contiguous().to(DEV))                    # M changed


@pytest.mark.parametrize("outputs", ["pinned", "pageable"])
def test_host_entry_matches_device_entry(fann, w_i8, outputs):
    """Pinned host outputs are written by the kernels directly, pageable ones by a copy after them."""
    w = w_i8
    ix, _, res = gpu_search(fann, w)
    B, k, total = w.cfg.B, w.cfg.k, w.cand_ids.numel()
    need = fann.fann_search_host_scratch_bytes(ix.handle, B, w.cfg.dsub, total, k)
    scratch = torch.empty(need, dtype=torch.uint8, device=DEV)
    q_h, off_h, ids_h = w.queries.pin_memory(), w.cand_offsets.pin_memory(), w.cand_ids.pin_memory()
    oi = torch.empty((B, k), dtype=torch.int32)
    od = torch.empty((B, k), dtype=torch.float32)
    oc = torch.empty(B, dtype=torch.int32)
    if outputs == "pinned":
        oi, od, oc = oi.pin_memory(), od.pin_memory(), oc.pin_memory()
    fann.fann_search_host(ix.handle, q_h, B, w.codebooks.to(DEV), w.cfg.dsub, off_h, ids_h, k, oi, od, oc,
                          scratch, need, torch.cuda.current_stream().cuda_stream)
    assert np.array_equal(oi.numpy().view(np.uint32), res[0])
    assert np.array_equal(od.numpy(), res[1]) and np.array_equal(oc.numpy().view(np.uint32), res[2])


def test_host_entry_in_chunks_matches_device_entry_and_oracle(fann):
    """A batch large enough (> 4 M candidate IDs) for fann_search_host to send the IDs up in 8 chunks of
    queries behind which the path runs chunk by chunk: same bytes as the one-call device path, and the
    first queries equal the oracle."""
    w = make_workload(mini("u8_10m_m32", N=1_000_000, n_lists=2_000, B=160, codes_mode="histogram"))
    assert w.cand_ids.numel() > (4 << 20)
    ix, _, res = gpu_search(fann, w)
    B, k, total = w.cfg.B, w.cfg.k, w.cand_ids.numel()
    need = fann.fann_search_host_scratch_bytes(ix.handle, B, w.cfg.dsub, total, k)
    scratch = torch.empty(need, dtype=torch.uint8, device=DEV)
    q_h, off_h, ids_h = w.queries.pin_memory(), w.cand_offsets.pin_memory(), w.cand_ids.pin_memory()
    oi = torch.empty((B, k), dtype=torch.int32).pin_memory()
    od = torch.empty((B, k), dtype=torch.float32).pin_memory()
    oc = torch.empty(B, dtype=torch.int32).pin_memory()
    for _ in range(2):                                        # twice: the scratch is reused across batches
        oi.fill_(0)
        fann.fann_search_host(ix.handle, q_h, B, w.codebooks.to(DEV), w.cfg.dsub, off_h, ids_h, k, oi, od, oc,
                              scratch, need, torch.cuda.current_stream().cuda_stream)
        assert np.array_equal(oi.numpy().view(np.uint32), res[0])
        assert np.array_equal(od.numpy(), res[1]) and np.array_equal(oc.numpy().view(np.uint32), res[2])
    nq = 12
    off = w.cand_offsets.numpy()[: nq + 1]
    ref = oracle.search(w.queries.numpy()[:nq], w.codebooks.numpy(), w.codes.numpy(), off,
                        w.cand_ids.numpy().view(np.uint32)[: off[-1]], k)
    assert np.array_equal(oi.numpy().view(np.uint32)[:nq], ref["ids"]) and np.array_equal(od.numpy()[:nq], ref["dists"])


@pytest.mark.parametrize("name,nq", [("u8_10m_m32", 48), ("f32_100m_m48", 24), ("i8_1b_m25", 24), ("u8_1b_m64", 12)])
def test_full_size_configs_sampled_against_oracle(fann, name, nq):
    """BASELINE's configs at full size, in the launch configuration bench.py times (same calls, same
    workspace sizing): the first nq queries are compared with the oracle -- lookup tables to 1e-5, results byte
    for byte in the integer-exact regime and by the tolerance rules for the real-valued config -- and every query
    with properties that hold at any size."""
    import bench
    cfg = CONFIGS[name]
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 2 * cfg.N * max(cfg.M, 32) + (40 << 30):     # workload's codes + the library's copy + per-batch arrays
        pytest.skip("not enough free device memory for this config")
    w = make_workload(cfg, device=DEV)
    B, k = cfg.B, cfg.k
    ix = fann.FannIndex(0)
    ix.load_codes(w.codes)
    lut = ix.build_lut(w.queries, w.codebooks)
    o = ix.dedup_scan_topk(lut, w.cand_offsets, w.cand_ids, k, check=True)
    torch.cuda.synchronize()
    ids, dists, counts, uniq = o
    # any size: counts = min(k, U), U <= C, distances ascending, no ID twice in a row of results
    C = (w.cand_offsets[1:] - w.cand_offsets[:-1])
    assert bool((uniq.long() <= C).all()) and bool((counts.long() == torch.clamp(uniq.long(), max=k)).all())
    assert bool((dists[:, 1:] >= dists[:, :-1]).all())
    srt = torch.sort(ids.long() & 0xFFFFFFFF, dim=1).values
    assert bool(((srt[:, 1:] != srt[:, :-1]) | (srt[:, 1:] == 0xFFFFFFFF)).all())
    # sampled: the lookup tables of the first nq queries
    lut64 = oracle.build_lut(w.queries[:nq].cpu().numpy(), w.codebooks.cpu().numpy())
    check_lut(lut[:nq].cpu().numpy(), lut64)
    if cfg.integer_exact:
        assert np.array_equal(lut[:nq].cpu().numpy().astype(np.float64), lut64)
        _, r, _ = bench.oracle_sample(w, nq, w.codes)
        check_exact((np_u32(ids[:nq]), dists[:nq].cpu().numpy(), np_u32(counts[:nq]), np_u32(uniq[:nq])), r)
    else:
        bench.band_check_sample(w, nq, w.codes, o)
    ix.close()
    del w, lut, o
    torch.cuda.empty_cache()


@pytest.fixture(scope="module")
def w_m16():
    """16-byte code rows (M = 16) on integer data: uint8 values, dsub = 8; every ADC sum < 2^24, so bytes compare."""
    cfg = mini("u8_10m_m32", N=400_000, n_lists=800, B=6, codes_mode="histogram", M=16)
    assert cfg.M * cfg.dsub * 255 ** 2 < 2 ** 24
    return make_workload(cfg)


@pytest.mark.parametrize("k", [1, 100, 1000, 1024])
@pytest.mark.parametrize("rows", [16, 32, 64])
def test_row_bytes_times_k_matrix_bytes(fann, w_m16, w_int, w_k1000, rows, k):
    """Every stored row size (16 / 32 / 64 bytes: 128 / 64 / 32 rows per ring stage, different buffer margins)
    against every k regime up to the compiled maximum, U >> k, integer-exact: byte equality with the oracle."""
    w = {16: w_m16, 32: w_int, 64: w_k1000}[rows]
    ix, _, res = gpu_search(fann, w, k=k)
    assert ix.info()["row_bytes"] == rows
    ref = orc_search(w, k=k)
    assert ref["uniq"].min() > 4 * k or k >= 1000
    check_exact(res, ref)


def test_two_host_threads_on_one_handle(fann, w_int, w_i8):
    """PAPER.md:L204 "each CPU thread handles an individual query": two host threads call the path on ONE handle
    at the same time, each with its own stream, workspace and outputs (fann.h "Threads").  Bytes equal the serial run."""
    import threading
    import paper_2409_16576_b200 as f
    w = w_int
    ix, _, serial = gpu_search(fann, w)
    q, cb = w.queries.to(DEV), w.codebooks.to(DEV)
    off, ids = w.cand_offsets.to(DEV), w.cand_ids.to(DEV)
    B, k, total = w.cfg.B, w.cfg.k, w.cand_ids.numel()
    need = f.fann_workspace_bytes(ix.handle, B, total, k)
    results, errors = {}, []

    def worker(t):
        try:
            torch.cuda.set_device(0)
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                ws = torch.empty(need, dtype=torch.uint8, device=DEV)
                lut = torch.empty((B, w.cfg.M, 256), dtype=torch.float32, device=DEV)
                out = (torch.empty((B, k), dtype=torch.int32, device=DEV), torch.empty((B, k), device=DEV),
                       torch.empty(B, dtype=torch.int32, device=DEV), torch.empty(B, dtype=torch.int32, device=DEV))
                for _ in range(20):
                    f.fann_build_lut(ix.handle, q, B, cb, w.cfg.dsub, lut, st.cuda_stream)
                    f.fann_dedup_scan_topk(ix.handle, lut, B, off, ids, total, k, out[0], out[1], out[2], out[3],
                                           ws, need, st.cuda_stream)
                f.fann_workspace_status(ix.handle, ws, st.cuda_stream)
                st.synchronize()
                results[t] = (np_u32(out[0]), out[1].cpu().numpy(), np_u32(out[2]), np_u32(out[3]))
        except Exception as e:                                 # noqa: BLE001
            errors.append(e)

    th = [threading.Thread(target=worker, args=(t,)) for t in range(2)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    assert not errors, errors
    for t in range(2):
        for a, b in zip(results[t], serial):
            assert np.array_equal(a, b)
    ix.close()


def test_load_codes_from_host_and_in_chunks(fann, w_i8):
    w = w_i8
    ix = fann.FannIndex(0)
    N = w.cfg.N
    half = N // 2
    ix.load_codes(w.codes[:half].contiguous(), first=0, N_total=N)             # host source, padded rows
    ix.load_codes(w.codes[half:].contiguous().to(DEV), first=half, N_total=N)  # device source
    lut = ix.build_lut(w.queries.to(DEV), w.codebooks.to(DEV))
    o = ix.dedup_scan_topk(lut, w.cand_offsets.to(DEV), w.cand_ids.to(DEV), w.cfg.k, check=True)
    torch.cuda.synchronize()
    check_exact((np_u32(o[0]), o[1].cpu().numpy(), np_u32(o[2]), np_u32(o[3])), orc_search(w))
