"""ctypes binding of include/fann.h -- argument marshalling only.

The module-level ``fann_*`` functions mirror the C entry points one to one and take raw
addresses (ints) or torch tensors (their ``data_ptr()`` is passed).  ``FannIndex`` is a small
convenience wrapper that allocates outputs / workspace through torch (device memory and
streams are the only things torch is used for) and calls the same entry points.

There is no CPU fallback: if libfann.so is absent or no CUDA device exists, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(HERE, "libfann.so")

FANN_ID_NONE = 0xFFFFFFFF
FANN_MAX_M = 64
FANN_MAX_K = 1024
FANN_MAX_NPROBE = 8192
FANN_ELEM_F32, FANN_ELEM_U8, FANN_ELEM_I8 = 0, 1, 2
FANN_OK = 0
FANN_STATIC_WS_BYTES = 32 * 1024 * 1024      # fann_dedup_scan_topk_static: the static workspace (fann.h)
FANN_STATUS_TABLE_FULL, FANN_STATUS_BAD_TOTAL = 1, 2

_lib = None


class FannError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"fann error {code}: {msg}")
        self.code = code


class _Info(C.Structure):
    _fields_ = [("N", C.c_uint64), ("M", C.c_uint32), ("row_bytes", C.c_uint32), ("num_sms", C.c_uint32),
                ("dedup_threads", C.c_uint32), ("dedup_ctas", C.c_uint32), ("dedup_smem_bytes", C.c_uint32),
                ("table_slots", C.c_uint32), ("scan_threads", C.c_uint32), ("scan_ctas", C.c_uint32),
                ("scan_smem_bytes", C.c_uint32), ("scan_buffer_keys", C.c_uint32), ("chunks", C.c_uint32),
                ("reserved", C.c_uint32), ("kernel_launches", C.c_uint64), ("codes_device_ptr", C.c_uint64)]


class _PoolInfo(C.Structure):
    _fields_ = [("block_bytes", C.c_uint64), ("calls", C.c_uint64), ("waits", C.c_uint64), ("n_blocks", C.c_uint32),
                ("in_use", C.c_uint32), ("high_water", C.c_uint32), ("reserved", C.c_uint32)]


def library_path() -> str:
    return _LIB_PATH


def load_library():
    """dlopen libfann.so (built in-tree by paper_2409_16576_b200.build).  Raises if missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise FileNotFoundError(
            f"{_LIB_PATH} not found: build it with `python -m paper_2409_16576_b200.build` "
            "(there is no CPU or PyTorch fallback)")
    lib = C.CDLL(_LIB_PATH)
    p, u32, u64, sz, i = C.c_void_p, C.c_uint32, C.c_uint64, C.c_size_t, C.c_int
    sig = {
        "fann_create": (i, [C.POINTER(p), i]),
        "fann_destroy": (None, [p]),
        "fann_last_error": (C.c_char_p, []),
        "fann_version": (C.c_char_p, []),
        "fann_load_codes": (i, [p, p, u64, u64, u64, u32, i, p]),
        "fann_build_lut": (i, [p, p, u32, p, u32, p, p]),
        "fann_workspace_bytes": (sz, [p, u32, u64, u32]),
        "fann_dedup_scan_topk": (i, [p, p, u32, p, p, u64, u32, p, p, p, p, p, sz, p]),
        "fann_dedup_scan_topk_static": (i, [p, p, u32, p, p, u64, u32, p, p, p, p, p, p]),
        "fann_dedup_only": (i, [p, u32, p, p, u64, p, p, p, sz, p]),
        "fann_workspace_status": (i, [p, p, p]),
        "fann_workspace_modes": (i, [p, p, u32, u64, u32, C.POINTER(u32), C.POINTER(u32), p]),
        "fann_search_host_scratch_bytes": (sz, [p, u32, u32, u64, u32]),
        "fann_search_host": (i, [p, p, u32, p, u32, p, p, u32, p, p, p, p, sz, p]),
        "fann_load_lists": (i, [p, p, p, u64, u64, i, p]),
        "fann_search_lists_workspace_bytes": (sz, [p, u32, u64, u32]),
        "fann_search_lists": (i, [p, p, u32, p, u32, u64, u32, p, p, p, p, p, sz, p]),
        "fann_search_lists_status": (i, [p, p, u32, u64, u32, C.POINTER(u64), p]),
        "fann_search_lists_host_scratch_bytes": (sz, [p, u32, u32, u32, u64, u32]),
        "fann_search_lists_host": (i, [p, p, u32, p, u32, p, u32, u64, u32, p, p, p, p, sz, p]),
        "fann_build_list_codes": (i, [p, p]),
        "fann_search_lists_stream_workspace_bytes": (sz, [p, u32, u64]),
        "fann_search_lists_stream": (i, [p, p, u32, p, u32, u64, u32, p, p, p, p, sz, p]),
        "fann_search_lists_stream_status": (i, [p, p, C.POINTER(u64), p]),
        "fann_pool_create": (i, [p, u32, u32, u64, u32, u32, u32, C.POINTER(p)]),
        "fann_pool_destroy": (None, [p]),
        "fann_pool_stats": (i, [p, C.POINTER(_PoolInfo)]),
        "fann_search_small": (i, [p, p, p, u32, p, u32, p, p, u32, p, p, p]),
        "fann_search_small_lists": (i, [p, p, p, u32, p, u32, p, u32, u32, p, p, p]),
        "fann_load_vectors": (i, [p, p, u64, u64, u64, u32, i, i, p]),
        "fann_rerank": (i, [p, p, u32, p, u32, u32, u32, C.c_float, u32, p, p, p, p, p, p]),
        "fann_load_page_table": (i, [p, p, u64, u64, i, p]),
        "fann_page_reads": (i, [p, p, u32, u32, u32, p, p, p, p, p, p]),
        "fann_get_info": (i, [p, C.POINTER(_Info)]),
        "fann_set_timing": (i, [p, i]),
        "fann_last_timing": (i, [p] + [C.POINTER(C.c_float)] * 5),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    _lib = lib
    return lib


def _addr(x) -> Optional[int]:
    """raw address of a torch tensor / numpy array / int / None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if hasattr(x, "ctypes"):
        return x.ctypes.data
    raise TypeError(type(x))


def _check(rc: int):
    if rc != FANN_OK:
        raise FannError(rc, fann_last_error())


# ---- one-to-one mirrors of the C entry points --------------------------------

def fann_last_error() -> str:
    return load_library().fann_last_error().decode()


def fann_version() -> str:
    return load_library().fann_version().decode()


def fann_create(device: int = 0) -> int:
    h = C.c_void_p()
    _check(load_library().fann_create(C.byref(h), device))
    return h.value


def fann_destroy(ix: int) -> None:
    load_library().fann_destroy(ix)


def fann_load_codes(ix, codes, first, n, N_total, M, src_is_device, stream=None) -> None:
    _check(load_library().fann_load_codes(ix, _addr(codes), first, n, N_total, M, int(src_is_device), stream))


def fann_build_lut(ix, queries, B, codebooks, dsub, lut, stream=None) -> None:
    _check(load_library().fann_build_lut(ix, _addr(queries), B, _addr(codebooks), dsub, _addr(lut), stream))


def fann_workspace_bytes(ix, B, total_cands, k) -> int:
    n = load_library().fann_workspace_bytes(ix, B, total_cands, k)
    if n == 0:
        raise FannError(-1, fann_last_error())
    return n


def fann_dedup_scan_topk(ix, lut, B, cand_offsets, cand_ids, total_cands, k, out_ids, out_dists,
                         out_counts, out_uniq, workspace, workspace_bytes, stream=None) -> None:
    _check(load_library().fann_dedup_scan_topk(ix, _addr(lut), B, _addr(cand_offsets), _addr(cand_ids),
                                               total_cands, k, _addr(out_ids), _addr(out_dists),
                                               _addr(out_counts), _addr(out_uniq), _addr(workspace),
                                               workspace_bytes, stream))


def fann_dedup_scan_topk_static(ix, lut, B, cand_offsets, cand_ids, total_cands, k, out_ids, out_dists,
                                out_counts, out_uniq, out_status, stream=None) -> None:
    """No allocation anywhere: the workspace is a device array of the library (FANN_STATIC_WS_BYTES)."""
    _check(load_library().fann_dedup_scan_topk_static(ix, _addr(lut), B, _addr(cand_offsets), _addr(cand_ids),
                                                      total_cands, k, _addr(out_ids), _addr(out_dists),
                                                      _addr(out_counts), _addr(out_uniq), _addr(out_status), stream))


def fann_dedup_only(ix, B, cand_offsets, cand_ids, total_cands, uniq_ids, uniq_counts, workspace,
                    workspace_bytes, stream=None) -> None:
    _check(load_library().fann_dedup_only(ix, B, _addr(cand_offsets), _addr(cand_ids), total_cands,
                                          _addr(uniq_ids), _addr(uniq_counts), _addr(workspace),
                                          workspace_bytes, stream))


def fann_workspace_status(ix, workspace, stream=None) -> None:
    _check(load_library().fann_workspace_status(ix, _addr(workspace), stream))


def fann_search_host_scratch_bytes(ix, B, dsub, total_cands, k) -> int:
    n = load_library().fann_search_host_scratch_bytes(ix, B, dsub, total_cands, k)
    if n == 0:
        raise FannError(-1, fann_last_error())
    return n


def fann_search_host(ix, queries_h, B, codebooks_d, dsub, cand_offsets_h, cand_ids_h, k, out_ids_h,
                     out_dists_h, out_counts_h, device_scratch, scratch_bytes, stream=None) -> None:
    _check(load_library().fann_search_host(ix, _addr(queries_h), B, _addr(codebooks_d), dsub,
                                           _addr(cand_offsets_h), _addr(cand_ids_h), k, _addr(out_ids_h),
                                           _addr(out_dists_h), _addr(out_counts_h), _addr(device_scratch),
                                           scratch_bytes, stream))


def fann_load_lists(ix, list_offsets, list_ids, n_lists, n_entries, src_is_device, stream=None) -> None:
    _check(load_library().fann_load_lists(ix, _addr(list_offsets), _addr(list_ids), n_lists, n_entries,
                                          int(src_is_device), stream))


def fann_search_lists_workspace_bytes(ix, B, max_total_cands, k) -> int:
    n = load_library().fann_search_lists_workspace_bytes(ix, B, max_total_cands, k)
    if n == 0:
        raise FannError(-1, fann_last_error())
    return n


def fann_search_lists(ix, lut, B, probes, nprobe, max_total_cands, k, out_ids, out_dists, out_counts, out_uniq,
                      workspace, workspace_bytes, stream=None) -> None:
    _check(load_library().fann_search_lists(ix, _addr(lut), B, _addr(probes), nprobe, max_total_cands, k,
                                            _addr(out_ids), _addr(out_dists), _addr(out_counts), _addr(out_uniq),
                                            _addr(workspace), workspace_bytes, stream))


def fann_search_lists_status(ix, workspace, B, max_total_cands, k, stream=None) -> int:
    """Raises on a bad status; returns the batch's candidate count."""
    total = C.c_uint64(0)
    rc = load_library().fann_search_lists_status(ix, _addr(workspace), B, max_total_cands, k, C.byref(total), stream)
    if rc != FANN_OK:
        err = FannError(rc, fann_last_error())
        err.total_cands = int(total.value)
        raise err
    return int(total.value)


def fann_search_lists_host_scratch_bytes(ix, B, dsub, nprobe, max_total_cands, k) -> int:
    n = load_library().fann_search_lists_host_scratch_bytes(ix, B, dsub, nprobe, max_total_cands, k)
    if n == 0:
        raise FannError(-1, fann_last_error())
    return n


def fann_search_lists_host(ix, queries_h, B, codebooks_d, dsub, probes_h, nprobe, max_total_cands, k, out_ids_h,
                           out_dists_h, out_counts_h, device_scratch, scratch_bytes, stream=None) -> None:
    _check(load_library().fann_search_lists_host(ix, _addr(queries_h), B, _addr(codebooks_d), dsub, _addr(probes_h),
                                                 nprobe, max_total_cands, k, _addr(out_ids_h), _addr(out_dists_h),
                                                 _addr(out_counts_h), _addr(device_scratch), scratch_bytes, stream))


def fann_build_list_codes(ix, stream=None) -> None:
    _check(load_library().fann_build_list_codes(ix, stream))


def fann_search_lists_stream_workspace_bytes(ix, B, max_total_cands) -> int:
    n = load_library().fann_search_lists_stream_workspace_bytes(ix, B, max_total_cands)
    if n == 0:
        raise FannError(-1, fann_last_error())
    return n


def fann_search_lists_stream(ix, lut, B, probes, nprobe, max_total_cands, k, out_ids, out_dists, out_counts,
                             workspace, workspace_bytes, stream=None) -> None:
    _check(load_library().fann_search_lists_stream(ix, _addr(lut), B, _addr(probes), nprobe, max_total_cands, k,
                                                   _addr(out_ids), _addr(out_dists), _addr(out_counts),
                                                   _addr(workspace), workspace_bytes, stream))


def fann_search_lists_stream_status(ix, workspace, stream=None) -> int:
    """Raises on a bad status; returns the batch's candidate count."""
    total = C.c_uint64(0)
    rc = load_library().fann_search_lists_stream_status(ix, _addr(workspace), C.byref(total), stream)
    if rc != FANN_OK:
        err = FannError(rc, fann_last_error())
        err.total_cands = int(total.value)
        raise err
    return int(total.value)


def fann_pool_create(ix, n_blocks, max_B, max_cands, dsub, max_nprobe, k_max) -> int:
    h = C.c_void_p()
    _check(load_library().fann_pool_create(ix, n_blocks, max_B, max_cands, dsub, max_nprobe, k_max, C.byref(h)))
    return h.value


def fann_pool_destroy(pool) -> None:
    load_library().fann_pool_destroy(pool)


def fann_pool_stats(pool) -> dict:
    info = _PoolInfo()
    _check(load_library().fann_pool_stats(pool, C.byref(info)))
    return {name: int(getattr(info, name)) for name, _ in _PoolInfo._fields_ if name != "reserved"}


def fann_search_small(ix, pool, queries_h, B, codebooks_d, dsub, cand_offsets_h, cand_ids_h, k, out_ids_h, out_dists_h,
                      out_counts_h) -> None:
    """ctypes releases the GIL during the call, so Python threads really run their calls side by side."""
    _check(load_library().fann_search_small(ix, pool, _addr(queries_h), B, _addr(codebooks_d), dsub,
                                            _addr(cand_offsets_h), _addr(cand_ids_h), k, _addr(out_ids_h),
                                            _addr(out_dists_h), _addr(out_counts_h)))


def fann_search_small_lists(ix, pool, queries_h, B, codebooks_d, dsub, probes_h, nprobe, k, out_ids_h, out_dists_h,
                            out_counts_h) -> None:
    _check(load_library().fann_search_small_lists(ix, pool, _addr(queries_h), B, _addr(codebooks_d), dsub,
                                                  _addr(probes_h), nprobe, k, _addr(out_ids_h), _addr(out_dists_h),
                                                  _addr(out_counts_h)))


def fann_load_vectors(ix, vectors, first, n, N_total, d, elem_type, src_is_device, stream=None) -> None:
    _check(load_library().fann_load_vectors(ix, _addr(vectors), first, n, N_total, d, elem_type,
                                            int(src_is_device), stream))


def fann_rerank(ix, queries, B, task_ids, n, batch_size, k, eps, beta, out_ids, out_dists, out_counts,
                out_batches=None, out_reads=None, stream=None) -> None:
    _check(load_library().fann_rerank(ix, _addr(queries), B, _addr(task_ids), n, batch_size, k, float(eps), beta,
                                      _addr(out_ids), _addr(out_dists), _addr(out_counts), _addr(out_batches),
                                      _addr(out_reads), stream))


def fann_load_page_table(ix, page_of, N, n_pages, src_is_device, stream=None) -> None:
    _check(load_library().fann_load_page_table(ix, _addr(page_of), N, n_pages, int(src_is_device), stream))


def fann_page_reads(ix, task_ids, B, n, batch_size, batches_run, resident_bits, out_pages, out_batch_reads,
                    out_total, stream=None) -> None:
    _check(load_library().fann_page_reads(ix, _addr(task_ids), B, n, batch_size, _addr(batches_run),
                                          _addr(resident_bits), _addr(out_pages), _addr(out_batch_reads),
                                          _addr(out_total), stream))


def fann_get_info(ix) -> dict:
    info = _Info()
    _check(load_library().fann_get_info(ix, C.byref(info)))
    return {name: int(getattr(info, name)) for name, _ in _Info._fields_}


def fann_set_timing(ix, enable: bool) -> None:
    _check(load_library().fann_set_timing(ix, int(enable)))


def fann_workspace_modes(ix, workspace, B, total_cands, k, stream=None) -> dict:
    a, b = C.c_uint32(0), C.c_uint32(0)
    _check(load_library().fann_workspace_modes(ix, _addr(workspace), B, total_cands, k, C.byref(a), C.byref(b), stream))
    return {"ordered": int(a.value), "hashed": int(b.value)}


def fann_last_timing(ix) -> dict:
    v = [C.c_float(-1.0) for _ in range(5)]
    _check(load_library().fann_last_timing(ix, *[C.byref(x) for x in v]))
    return dict(zip(("lut_ms", "plan_ms", "partition_ms", "dedup_ms", "scan_ms"), (float(x.value) for x in v)))


# ---- convenience wrapper (torch for device memory and streams only) ----------

class FannIndex:
    """Owns a fann_index handle; allocates outputs and workspace with torch."""

    def __init__(self, device: int = 0):
        import torch
        self._torch = torch
        self.device = device
        self.handle = fann_create(device)
        self._ws = None
        self.M = 0
        self.N = 0

    def close(self):
        if self.handle:
            fann_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _stream(self):
        return self._torch.cuda.current_stream(self.device).cuda_stream

    def load_codes(self, codes, first: int = 0, N_total: Optional[int] = None):
        """codes: uint8 [n, M] torch tensor (cuda or cpu) or numpy array."""
        n, M = codes.shape
        N_total = n if N_total is None else N_total
        is_dev = bool(getattr(codes, "is_cuda", False))
        if hasattr(codes, "is_contiguous"):
            assert codes.is_contiguous()
        fann_load_codes(self.handle, codes, first, n, N_total, M, is_dev, self._stream())
        self.M, self.N = M, N_total

    def build_lut(self, queries, codebooks, out=None):
        torch = self._torch
        B = queries.shape[0]
        M, n256, dsub = codebooks.shape
        assert n256 == 256 and M == self.M and queries.shape[1] == M * dsub
        assert queries.is_cuda and codebooks.is_cuda and queries.is_contiguous() and codebooks.is_contiguous()
        assert queries.dtype == torch.float32 and codebooks.dtype == torch.float32
        if out is None:
            out = torch.empty((B, M, 256), dtype=torch.float32, device=queries.device)
        fann_build_lut(self.handle, queries, B, codebooks, dsub, out, self._stream())
        return out

    def workspace(self, B, total_cands, k):
        torch = self._torch
        need = fann_workspace_bytes(self.handle, B, total_cands, k)
        if self._ws is None or self._ws.numel() < need:
            self._ws = None
            self._ws = torch.empty(need, dtype=torch.uint8, device=f"cuda:{self.device}")
        return self._ws

    def dedup_scan_topk(self, lut, cand_offsets, cand_ids, k, total_cands=None, out=None, check=False):
        """Returns (ids int32 view of uint32 [B,k], dists f32 [B,k], counts int32 [B], uniq int32 [B])."""
        torch = self._torch
        B = cand_offsets.numel() - 1
        if total_cands is None:
            total_cands = int(cand_ids.numel())
        dev = lut.device
        if out is None:
            out = (torch.empty((B, k), dtype=torch.int32, device=dev),
                   torch.empty((B, k), dtype=torch.float32, device=dev),
                   torch.empty(B, dtype=torch.int32, device=dev),
                   torch.empty(B, dtype=torch.int32, device=dev))
        ws = self.workspace(B, total_cands, k)
        fann_dedup_scan_topk(self.handle, lut, B, cand_offsets, cand_ids, total_cands, k,
                             out[0], out[1], out[2], out[3], ws, ws.numel(), self._stream())
        if check:
            fann_workspace_status(self.handle, ws, self._stream())
        return out

    def dedup_only(self, cand_offsets, cand_ids, total_cands=None):
        torch = self._torch
        B = cand_offsets.numel() - 1
        if total_cands is None:
            total_cands = int(cand_ids.numel())
        dev = cand_offsets.device
        uniq_ids = torch.full((max(1, total_cands),), -1, dtype=torch.int32, device=dev)
        uniq_counts = torch.empty(B, dtype=torch.int32, device=dev)
        ws = self.workspace(B, total_cands, 1)
        fann_dedup_only(self.handle, B, cand_offsets, cand_ids, total_cands, uniq_ids, uniq_counts,
                        ws, ws.numel(), self._stream())
        fann_workspace_status(self.handle, ws, self._stream())
        return uniq_ids, uniq_counts

    def search(self, queries, codebooks, cand_offsets, cand_ids, k, check=False):
        lut = self.build_lut(queries, codebooks)
        return self.dedup_scan_topk(lut, cand_offsets, cand_ids, k, check=check)

    def load_lists(self, list_offsets, list_ids):
        """CSR of all posting lists: int64 [n_lists + 1], int32/uint32 [entries] (torch, cuda or cpu)."""
        is_dev = bool(getattr(list_offsets, "is_cuda", False))
        assert bool(getattr(list_ids, "is_cuda", False)) == is_dev
        fann_load_lists(self.handle, list_offsets, list_ids, list_offsets.numel() - 1, list_ids.numel(), is_dev,
                        self._stream())

    def search_lists(self, lut, probes, k, max_total_cands, out=None, check=False):
        """probes: int32 view of uint32 [B, nprobe] on the device.  Returns (ids, dists, counts, uniq)."""
        torch = self._torch
        B, nprobe = probes.shape
        dev = lut.device
        if out is None:
            out = (torch.empty((B, k), dtype=torch.int32, device=dev),
                   torch.empty((B, k), dtype=torch.float32, device=dev),
                   torch.empty(B, dtype=torch.int32, device=dev),
                   torch.empty(B, dtype=torch.int32, device=dev))
        need = fann_search_lists_workspace_bytes(self.handle, B, max_total_cands, k)
        if self._ws is None or self._ws.numel() < need:
            self._ws = None
            self._ws = torch.empty(need, dtype=torch.uint8, device=f"cuda:{self.device}")
        fann_search_lists(self.handle, lut, B, probes, nprobe, max_total_cands, k, out[0], out[1], out[2], out[3],
                          self._ws, self._ws.numel(), self._stream())
        if check:
            fann_search_lists_status(self.handle, self._ws, B, max_total_cands, k, self._stream())
        return out

    def load_vectors(self, vectors, first: int = 0, N_total: Optional[int] = None):
        """Raw vectors [n, d]: float32, uint8 or int8 torch tensor (cuda or cpu)."""
        torch = self._torch
        n, d = vectors.shape
        elem = {torch.float32: FANN_ELEM_F32, torch.uint8: FANN_ELEM_U8, torch.int8: FANN_ELEM_I8}[vectors.dtype]
        assert vectors.is_contiguous()
        fann_load_vectors(self.handle, vectors, first, n, n if N_total is None else N_total, d, elem,
                          bool(vectors.is_cuda), self._stream())

    def rerank(self, queries, task_ids, batch_size, k, eps, beta):
        """Returns (ids [B,k], dists [B,k], counts [B], batches [B], reads [B])."""
        torch = self._torch
        B, n = task_ids.shape
        dev = queries.device
        out = (torch.empty((B, k), dtype=torch.int32, device=dev), torch.empty((B, k), dtype=torch.float32, device=dev),
               torch.empty(B, dtype=torch.int32, device=dev), torch.empty(B, dtype=torch.int32, device=dev),
               torch.empty(B, dtype=torch.int32, device=dev))
        fann_rerank(self.handle, queries, B, task_ids, n, batch_size, k, eps, beta, *out, stream=self._stream())
        return out

    def load_page_table(self, page_of, n_pages):
        fann_load_page_table(self.handle, page_of, page_of.numel(), n_pages, bool(page_of.is_cuda), self._stream())

    def page_reads(self, task_ids, batch_size, batches_run=None, resident_bits=None):
        """Returns (pages [B,n], batch_reads [B,nb], total [B])."""
        torch = self._torch
        B, n = task_ids.shape
        bs = min(batch_size, n)
        nb = (n + bs - 1) // bs
        dev = task_ids.device
        out = (torch.empty((B, n), dtype=torch.int32, device=dev), torch.empty((B, nb), dtype=torch.int32, device=dev),
               torch.empty(B, dtype=torch.int32, device=dev))
        fann_page_reads(self.handle, task_ids, B, n, batch_size, batches_run, resident_bits, *out, stream=self._stream())
        return out

    def info(self) -> dict:
        return fann_get_info(self.handle)
