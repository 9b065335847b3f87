"""Parity rules between the CUDA path and the oracle.

TEST INFRASTRUCTURE like the rest of oracle/: used by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline leg to compare what the CUDA path returned with what the oracle computed."""
import numpy as np

NONE = 0xFFFFFFFF
RTOL = 1e-5          # north star: lookup-table entries and distances agree to 1e-5 relative in fp32


def check_lut(lut_gpu, lut64):
    """|lut_gpu - lut64| <= 1e-5 * lut64 elementwise (exactly 0 where lut64 == 0)."""
    g = np.asarray(lut_gpu, dtype=np.float64)
    assert g.shape == lut64.shape
    err = np.abs(g - lut64)
    bad = err > RTOL * lut64
    assert not bad.any(), f"{bad.sum()} LUT entries off; worst rel {np.max(err / np.maximum(lut64, 1e-300)):.3e}"


def check_exact(gpu, orc, B=None):
    """Integer-exact regime: ids, dists, counts, uniq byte-identical."""
    ids, dists, counts, uniq = gpu
    sl = slice(None) if B is None else slice(0, B)
    assert np.array_equal(counts[sl], orc["counts"]), "counts differ"
    assert np.array_equal(uniq[sl], orc["uniq"]), "uniq differ"
    assert np.array_equal(ids[sl], orc["ids"]), "ids differ"
    assert np.array_equal(dists[sl].view(np.uint32), orc["dists"].view(np.uint32)), "dist bits differ"


def check_band(ids, dists, count, all_ids, all_d64, k):
    """Tolerance regime for one query.  all_ids ascending distinct ids, all_d64 their fp64
    distances (oracle.query_all).  Returns True if the band was needed (a candidate other
    than the k-th lies within tau*(1 +- 1e-5))."""
    U = all_ids.size
    c = min(k, U)
    assert count == c, f"count {count} != {c}"
    assert np.all(ids[c:] == NONE) and np.all(np.isposinf(dists[c:])), "padding"
    got = ids[:c]
    assert np.unique(got).size == c, "repeated id in output"
    pos = np.searchsorted(all_ids, got)
    assert np.all(pos < U) and np.all(all_ids[np.minimum(pos, U - 1)] == got), "id not a candidate"
    D = all_d64[pos]
    g = dists[:c].astype(np.float64)
    assert np.all(np.abs(g - D) <= RTOL * D + 1e-30), f"distance off: worst {np.max(np.abs(g - D) / np.maximum(D, 1e-300)):.3e}"
    assert np.all(np.diff(dists[:c]) >= 0), "not ascending"
    if U <= k:
        assert np.array_equal(np.sort(got), all_ids)
        return False
    order = np.sort(all_d64)
    tau = order[k - 1]
    must = all_ids[all_d64 < tau * (1 - RTOL)]
    assert np.all(np.isin(must, got)), "a candidate clearly inside the top-k is missing"
    assert np.all(D <= tau * (1 + RTOL)), "a returned candidate is clearly outside the top-k"
    in_band = np.sum((all_d64 >= tau * (1 - RTOL)) & (all_d64 <= tau * (1 + RTOL)))
    return in_band > 1
