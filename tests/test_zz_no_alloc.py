"""fann_dedup_scan_topk_static: the entry point that allocates nothing (its workspace is a file-scope device array
of the library, FANN_STATIC_WS_BYTES) against the existing path, fann_dedup_scan_topk with a caller's workspace.

Collected last on purpose (the name): the suite runs with `pytest -x`, so a failure here hides no other test.
Runs alone in a fresh process (`pytest tests/test_zz_no_alloc.py`) and after the other GPU tests."""
import numpy as np
import pytest
import torch

import oracle
from oracle.parity import check_band
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


class _Case:
    """One workload on the device with its own index, and the existing path's answer."""

    def __init__(self, fann, w):
        self.w, self.B, self.k = w, w.cfg.B, w.cfg.k
        self.ix = fann.FannIndex(0)
        self.ix.load_codes(w.codes.to(DEV))
        self.off, self.ids = w.cand_offsets.to(DEV), w.cand_ids.to(DEV)
        self.total = int(self.ids.numel())
        self.lut = self.ix.build_lut(w.queries.to(DEV), w.codebooks.to(DEV))
        o = self.ix.dedup_scan_topk(self.lut, self.off, self.ids, self.k, check=True)     # existing path, caller's workspace
        torch.cuda.synchronize()
        self.ref = (np_u32(o[0]), o[1].cpu().numpy(), np_u32(o[2]), np_u32(o[3]))

    def run_static(self, fann):
        """Outputs are pre-filled with garbage: every element must be written by the call."""
        B, k = self.B, self.k
        oi = torch.full((B, k), 0x5A5A5A5A, dtype=torch.int32, device=DEV)
        od = torch.full((B, k), -7.0, dtype=torch.float32, device=DEV)
        oc = torch.full((B,), 0x5A5A5A5A, dtype=torch.int32, device=DEV)
        ou = torch.full((B,), 0x5A5A5A5A, dtype=torch.int32, device=DEV)
        st = torch.full((1,), 0x5A5A5A5A, dtype=torch.int32, device=DEV)
        fann.fann_dedup_scan_topk_static(self.ix.handle, self.lut, B, self.off, self.ids, self.total, k,
                                         oi, od, oc, ou, st, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        assert int(np_u32(st)[0]) == 0, "status word"
        return np_u32(oi), od.cpu().numpy(), np_u32(oc), np_u32(ou)

    def check(self, got):
        ids, dists, counts, uniq = got
        r = self.ref
        assert np.array_equal(counts, r[2]) and np.array_equal(uniq, r[3])
        if self.w.cfg.integer_exact:
            # integer regime: the bar of the parity tests is byte equality
            assert np.array_equal(ids, r[0]), "ids differ from fann_dedup_scan_topk"
            assert np.array_equal(dists.view(np.uint32), r[1].view(np.uint32)), "dist bits differ from fann_dedup_scan_topk"
        else:
            # fp32 data: a row's summation order depends on the lane that scores it, so two runs of the SAME entry agree
            # within the band only (tests/test_gpu_next.py): distances to 1e-5 against the existing path, and the
            # oracle's band check on the result itself
            fin = np.isfinite(r[1])
            assert np.array_equal(np.isfinite(dists), fin)
            assert np.allclose(dists[fin], r[1][fin], rtol=1e-5, atol=0)
            w = self.w
            off, cid = w.cand_offsets.numpy(), w.cand_ids.numpy().view(np.uint32)
            for b in range(self.B):
                ai, ad = oracle.query_all(w.queries.numpy()[b], w.codebooks.numpy(), w.codes.numpy(), cid[off[b]:off[b + 1]])
                assert uniq[b] == ai.size
                check_band(ids[b], dists[b], counts[b], ai, ad, self.k)

    def close(self):
        self.ix.close()


def test_static_entry_equals_the_workspace_entry_on_calls_in_a_row(fann):
    """Calls in a row on the one shared array, from two handles of different geometry (32- and 25-byte codes,
    k = 100 and 10, different batch sizes, so every region of the layout moves between calls) and back: each call
    gives the bytes of fann_dedup_scan_topk; nothing is cleared between them by the caller."""
    a = _Case(fann, make_workload(mini("u8_10m_m32", N=400_000, n_lists=800, B=24, codes_mode="histogram")))
    b = _Case(fann, make_workload(mini("i8_1b_m25", N=300_000, n_lists=600, B=17, codes_mode="histogram", k=10)))
    assert a.w.cfg.integer_exact and b.w.cfg.integer_exact
    need_a = fann.fann_workspace_bytes(a.ix.handle, a.B, a.total, a.k)
    need_b = fann.fann_workspace_bytes(b.ix.handle, b.B, b.total, b.k)
    assert 0 < need_a <= fann.FANN_STATIC_WS_BYTES and 0 < need_b <= fann.FANN_STATIC_WS_BYTES
    for case in (a, a, b, a, b, b):
        case.check(case.run_static(fann))
    a.close()
    b.close()


def test_static_entry_fp32_band_twice(fann):
    c = _Case(fann, make_workload(CONFIGS["tiny_local"]))
    assert not c.w.cfg.integer_exact
    for _ in range(2):
        c.check(c.run_static(fann))
    c.close()


def test_static_entry_reports_a_bad_total_and_recovers(fann):
    """The status word of the shared array does not leak into the next call: a call with an understated
    total_cands reports FANN_STATUS_BAD_TOTAL, the next good call reports 0 and the right bytes."""
    c = _Case(fann, make_workload(mini("u8_10m_m32", N=200_000, n_lists=400, B=9, codes_mode="histogram")))
    B, k = c.B, c.k
    oi = torch.empty((B, k), dtype=torch.int32, device=DEV)
    od = torch.empty((B, k), dtype=torch.float32, device=DEV)
    oc = torch.empty(B, dtype=torch.int32, device=DEV)
    st = torch.zeros(1, dtype=torch.int32, device=DEV)
    fann.fann_dedup_scan_topk_static(c.ix.handle, c.lut, B, c.off, c.ids, c.total - 1000, k, oi, od, oc, None, st,
                                     torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert int(np_u32(st)[0]) & fann.FANN_STATUS_BAD_TOTAL
    c.check(c.run_static(fann))
    c.close()


def test_static_entry_refuses_a_batch_beyond_its_array(fann):
    """Sizes beyond FANN_STATIC_WS_BYTES: a clear error naming both sizes, nothing enqueued, and the entry still
    works afterwards.  (The arrays are never read: the check is on the host.)"""
    c = _Case(fann, make_workload(mini("u8_10m_m32", N=200_000, n_lists=400, B=9, codes_mode="histogram")))
    B, k = c.B, c.k
    big = 40_000_000                                                        # 12 bytes of workspace per candidate ID
    assert fann.fann_workspace_bytes(c.ix.handle, B, big, k) > fann.FANN_STATIC_WS_BYTES
    oi = torch.empty((B, k), dtype=torch.int32, device=DEV)
    od = torch.empty((B, k), dtype=torch.float32, device=DEV)
    with pytest.raises(fann.FannError) as e:
        fann.fann_dedup_scan_topk_static(c.ix.handle, c.lut, B, c.off, c.ids, big, k, oi, od, None, None, None,
                                         torch.cuda.current_stream().cuda_stream)
    assert "FANN_STATIC_WS_BYTES" in str(e.value) and str(fann.FANN_STATIC_WS_BYTES) in str(e.value)
    c.check(c.run_static(fann))
    c.close()
