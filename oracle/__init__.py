"""ctypes wrapper of the CPU oracle (oracle/fann_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs import this package.  It does
not import the CUDA package and the CUDA package does not import it.
Inputs and outputs are numpy arrays on the host.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fann_oracle.c")
_LIB = os.path.join(_HERE, "libfann_oracle.so")
ID_NONE = 0xFFFFFFFF

_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp the oracle into oracle/libfann_oracle.so."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        p = C.c_void_p
        lib.oracle_build_lut.argtypes = [p, p, C.c_uint32, C.c_uint32, C.c_uint32, p]
        lib.oracle_build_lut.restype = None
        lib.oracle_dedup.argtypes = [p, C.c_uint64, C.c_uint64, p]
        lib.oracle_dedup.restype = C.c_uint64
        lib.oracle_adc.argtypes = [p, p, C.c_uint32, C.c_uint64]
        lib.oracle_adc.restype = C.c_double
        lib.oracle_topk.argtypes = [p, p, C.c_uint64, C.c_uint32, p, p, p]
        lib.oracle_topk.restype = None
        lib.oracle_search.argtypes = [p, p, p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32,
                                      p, p, C.c_uint32, p, p, p, p, p, C.c_int]
        lib.oracle_search.restype = C.c_int
        lib.oracle_query_all.argtypes = [p, p, p, C.c_uint64, C.c_uint32, C.c_uint32,
                                         p, C.c_uint64, p, p]
        lib.oracle_query_all.restype = C.c_uint64
        lib.oracle_max_threads.restype = C.c_int
        lib.oracle_expand_lists.argtypes = [p, p, C.c_uint64, p, C.c_uint32, C.c_uint32, p, p]
        lib.oracle_expand_lists.restype = C.c_uint64
        lib.oracle_rerank.argtypes = [p, p, C.c_uint64, C.c_uint32, p, C.c_uint32, C.c_uint32, C.c_uint32,
                                      C.c_float, C.c_uint32, p, p, p, p, p]
        lib.oracle_rerank.restype = C.c_uint32
        lib.oracle_page_reads.argtypes = [p, C.c_uint64, p, C.c_uint32, C.c_uint32, C.c_uint32, p, C.c_uint64, p, p]
        lib.oracle_page_reads.restype = C.c_uint32
        _lib = lib
    return _lib


def _arr(a, dtype):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def build_lut(queries, codebooks) -> np.ndarray:
    """queries [B, d] f32, codebooks [M, 256, dsub] f32 -> lut64 [B, M, 256] f64."""
    q = _arr(queries, np.float32)
    cb = _arr(codebooks, np.float32)
    M, n256, dsub = cb.shape
    assert n256 == 256 and q.shape[1] == M * dsub
    out = np.empty((q.shape[0], M, 256), dtype=np.float64)
    _load().oracle_build_lut(_ptr(q), _ptr(cb), q.shape[0], M, dsub, _ptr(out))
    return out


def dedup(ids, N) -> np.ndarray:
    """distinct valid IDs, ascending (uint32)."""
    a = _arr(ids, np.uint32)
    out = np.empty(max(1, a.size), dtype=np.uint32)
    u = _load().oracle_dedup(_ptr(a), a.size, int(N), _ptr(out))
    return out[:u].copy()


def adc(lut64_q, codes, vid) -> float:
    """lut64_q [M, 256] f64, codes [N, M] u8 -> Eq. 1 distance of vector `vid`."""
    lut = _arr(lut64_q, np.float64)
    cd = _arr(codes, np.uint8)
    return float(_load().oracle_adc(_ptr(lut), _ptr(cd), lut.shape[0], int(vid)))


def topk(ids, dists, k):
    """(ids [U] u32, dists [U] f32) -> (out_ids [k], out_dists [k], count)."""
    a = _arr(ids, np.uint32)
    d = _arr(dists, np.float32)
    oi = np.empty(k, dtype=np.uint32)
    od = np.empty(k, dtype=np.float32)
    cnt = C.c_uint32(0)
    _load().oracle_topk(_ptr(a), _ptr(d), a.size, k, _ptr(oi), _ptr(od), C.byref(cnt))
    return oi, od, int(cnt.value)


def search(queries, codebooks, codes, cand_offsets, cand_ids, k, N=None, nthreads=0):
    """The whole GPU stage on the CPU.  Returns a dict with ids [B,k] u32,
    dists [B,k] f32, dists64 [B,k] f64, counts [B] u32, uniq [B] u32, threads."""
    q = _arr(queries, np.float32)
    cb = _arr(codebooks, np.float32)
    cd = _arr(codes, np.uint8)
    off = _arr(cand_offsets, np.int64)
    ids = _arr(np.asarray(cand_ids).view(np.uint32) if np.asarray(cand_ids).dtype == np.int32
               else cand_ids, np.uint32)
    M, _, dsub = cb.shape
    B = q.shape[0]
    if N is None:
        N = cd.shape[0]
    assert cd.ndim == 2 and cd.shape[1] == M and off.size == B + 1
    oi = np.empty((B, k), dtype=np.uint32)
    od = np.empty((B, k), dtype=np.float32)
    od64 = np.empty((B, k), dtype=np.float64)
    cnt = np.empty(B, dtype=np.uint32)
    uq = np.empty(B, dtype=np.uint32)
    thr = _load().oracle_search(_ptr(q), _ptr(cb), _ptr(cd), int(N), M, dsub, B, _ptr(off), _ptr(ids),
                                k, _ptr(oi), _ptr(od), _ptr(od64), _ptr(cnt), _ptr(uq), int(nthreads))
    return {"ids": oi, "dists": od, "dists64": od64, "counts": cnt, "uniq": uq, "threads": int(thr)}


def query_all(query, codebooks, codes, ids, N=None):
    """One query: (distinct IDs ascending [U] u32, fp64 distances [U])."""
    q = _arr(query, np.float32).reshape(-1)
    cb = _arr(codebooks, np.float32)
    cd = _arr(codes, np.uint8)
    a = np.asarray(ids)
    a = _arr(a.view(np.uint32) if a.dtype == np.int32 else a, np.uint32)
    M, _, dsub = cb.shape
    if N is None:
        N = cd.shape[0]
    ai = np.empty(max(1, a.size), dtype=np.uint32)
    ad = np.empty(max(1, a.size), dtype=np.float64)
    u = _load().oracle_query_all(_ptr(q), _ptr(cb), _ptr(cd), int(N), M, dsub, _ptr(a), a.size,
                                 _ptr(ai), _ptr(ad))
    return ai[:u].copy(), ad[:u].copy()


def expand_lists(list_offsets, list_ids, probes):
    """PAPER.md:L125 step (3): probes [B, nprobe] u32 (list indices) -> (cand_offsets [B+1] i64, cand_ids u32),
    each query's candidates = its probed lists' IDs concatenated in probe order."""
    lo = _arr(list_offsets, np.int64)
    li = _arr(np.asarray(list_ids).view(np.uint32) if np.asarray(list_ids).dtype == np.int32 else list_ids, np.uint32)
    pr = np.asarray(probes)
    pr = _arr(pr.view(np.uint32) if pr.dtype == np.int32 else pr, np.uint32)
    B, nprobe = pr.shape
    off = np.empty(B + 1, dtype=np.int64)
    total = _load().oracle_expand_lists(_ptr(lo), _ptr(li), lo.size - 1, _ptr(pr), B, nprobe, _ptr(off), None)
    ids = np.empty(max(1, total), dtype=np.uint32)
    _load().oracle_expand_lists(_ptr(lo), _ptr(li), lo.size - 1, _ptr(pr), B, nprobe, _ptr(off), _ptr(ids))
    return off, ids[:total]


def search_lists(queries, codebooks, codes, list_offsets, list_ids, probes, k, N=None, nthreads=0):
    """Steps (3)(1)(5)(6)(7): expand the probed lists, then the whole GPU stage on the CPU."""
    off, ids = expand_lists(list_offsets, list_ids, probes)
    return search(queries, codebooks, codes, off, ids, k, N=N, nthreads=nthreads)


def rerank(queries, vectors, tasks, batch_size, k, eps, beta):
    """Algorithm 1 for every query.  queries [B, d] f32, vectors [N, d] f32 raw vectors,
    tasks [B, n] u32 candidate IDs in ascending PQ order (0xFFFFFFFF padded).  Returns a dict: ids [B,k] u32,
    dists [B,k] f32, dists64 [B,k] f64, counts [B], batches [B] (mini-batches executed), reads [B] (vectors read)."""
    q = _arr(queries, np.float32)
    v = _arr(vectors, np.float32)
    t = np.asarray(tasks)
    t = _arr(t.view(np.uint32) if t.dtype == np.int32 else t, np.uint32)
    B, n = t.shape
    N, d = v.shape
    assert q.shape == (B, d)
    oi = np.empty((B, k), dtype=np.uint32)
    od = np.empty((B, k), dtype=np.float32)
    od64 = np.empty((B, k), dtype=np.float64)
    cnt = np.zeros(B, dtype=np.uint32)
    bat = np.zeros(B, dtype=np.uint32)
    reads = np.zeros(B, dtype=np.uint32)
    lib = _load()
    for b in range(B):
        c, nb = C.c_uint32(0), C.c_uint32(0)
        reads[b] = lib.oracle_rerank(_ptr(q[b]), _ptr(v), N, d, _ptr(t[b]), n, batch_size, k, eps, beta,
                                     _ptr(oi[b]), _ptr(od[b]), _ptr(od64[b]), C.byref(c), C.byref(nb))
        cnt[b], bat[b] = c.value, nb.value
    return {"ids": oi, "dists": od, "dists64": od64, "counts": cnt, "batches": bat, "reads": reads}


def page_reads(page_of, tasks, batch_size, max_batches=None, resident=None, n_pages=0):
    """Fig. 8 for every query.  page_of [N] u32, tasks [B, n] u32, max_batches [B] or None,
    resident: uint32 bitmap over pages or None.  Returns (pages [B, n] u32 padded with 0xFFFFFFFF,
    batch_reads [B, nb] u32, total [B] u32)."""
    po = _arr(page_of, np.uint32)
    t = np.asarray(tasks)
    t = _arr(t.view(np.uint32) if t.dtype == np.int32 else t, np.uint32)
    B, n = t.shape
    nb = (n + batch_size - 1) // batch_size
    pages = np.full((B, n), ID_NONE, dtype=np.uint32)
    br = np.zeros((B, nb), dtype=np.uint32)
    tot = np.zeros(B, dtype=np.uint32)
    res = None if resident is None else _arr(resident, np.uint32)
    lib = _load()
    for b in range(B):
        mb = 0 if max_batches is None else int(max_batches[b])
        row = np.empty(n, dtype=np.uint32)
        tot[b] = lib.oracle_page_reads(_ptr(po), po.size, _ptr(t[b]), n, batch_size, mb,
                                       None if res is None else _ptr(res), n_pages, _ptr(row), _ptr(br[b]))
        pages[b, :tot[b]] = row[:tot[b]]
    return pages, br, tot
