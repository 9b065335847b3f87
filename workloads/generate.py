"""Seeded synthetic inputs for the FusionANNS GPU stage.

Everything here is *input construction*: vectors, PQ codebooks and codes (the
offline stage, which is outside the hot path), posting lists
with boundary replication (the *shape* of PAPER.md:L145-L148, not Eq. 2
itself) and the per-query candidate-ID lists the CPU would send to the GPU
(PAPER.md:L125 steps 2-4).  None of the hot path's arithmetic (lookup table,
dedup, ADC, top-k) lives here; both the oracle tests and the CUDA tests feed
from this module and from nothing else in common.

All randomness is a counter-based hash (splitmix64 finaliser) of
(seed, stream label, element index) evaluated with torch integer ops, so any
piece can be regenerated independently, in chunks, on CPU or on a GPU.
Floating-point pieces (Gaussian vectors) are deterministic per device type
only; tests always generate once and hand the same tensors to both sides.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Dict, Optional

import torch

from .configs import WorkloadConfig

DEFAULT_SEED = 20240916
ID_NONE = 0xFFFFFFFF          # padding value of the boundary (as int32: -1)
_ID_MULT = 2654435761         # prime; coprime to every N used here

_U64 = (1 << 64) - 1


def _s64(v: int) -> int:
    v &= _U64
    return v - (1 << 64) if v >= (1 << 63) else v


def _py_mix64(x: int) -> int:
    x = (x + 0x9E3779B97F4A7C15) & _U64
    x = ((x ^ (x >> 30)) * 0xBF58476D1CE4E5B9) & _U64
    x = ((x ^ (x >> 27)) * 0x94D049BB133111EB) & _U64
    return x ^ (x >> 31)


def stream_key(seed: int, *labels) -> int:
    """64-bit key of a named random stream."""
    k = _py_mix64(seed & _U64)
    for lab in labels:
        if isinstance(lab, str):
            for ch in lab.encode():
                k = _py_mix64(k ^ ch)
        else:
            k = _py_mix64(k ^ (int(lab) & _U64))
    return k


def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    return (x >> s) & ((1 << (64 - s)) - 1)


def hash64(key: int, ctr: torch.Tensor) -> torch.Tensor:
    """splitmix64 finaliser of (ctr xor key); ctr is an int64 tensor."""
    x = ctr ^ _s64(key)
    x = x + _s64(0x9E3779B97F4A7C15)
    x = (x ^ _lsr(x, 30)) * _s64(0xBF58476D1CE4E5B9)
    x = (x ^ _lsr(x, 27)) * _s64(0x94D049BB133111EB)
    return x ^ _lsr(x, 31)


def _uniform24(h: torch.Tensor) -> torch.Tensor:
    """float32 in [0,1) from the top 24 bits."""
    return _lsr(h, 40).to(torch.float32) * (2.0 ** -24)


def _uniform53(h: torch.Tensor) -> torch.Tensor:
    return _lsr(h, 11).to(torch.float64) * (2.0 ** -53)


def _randint(h: torch.Tensor, n: int) -> torch.Tensor:
    """int64 in [0, n), n < 2^31."""
    return (_lsr(h, 33) * n) >> 31


# --------------------------------------------------------------------------
# vectors, codebooks, codes
# --------------------------------------------------------------------------

def draw_vectors(cfg: WorkloadConfig, key: int, first: int, count: int,
                 device="cpu") -> torch.Tensor:
    """`count` vectors [count, d] fp32 of the config's value distribution."""
    d = cfg.d
    ctr = (torch.arange(first * d, (first + count) * d, dtype=torch.int64, device=device))
    h = hash64(key, ctr)
    if cfg.values == "uniform01":
        x = _uniform24(h)
    elif cfg.values == "u8":
        x = _lsr(h, 56).to(torch.float32)
    elif cfg.values == "i8":
        x = (_lsr(h, 56) - 128).to(torch.float32)
    elif cfg.values == "gauss_norm":
        u1 = (_lsr(h, 40).to(torch.float64) + 1.0) * (2.0 ** -24)       # (0, 1]
        u2 = _uniform53(hash64(key ^ 0x5851F42D4C957F2D, ctr))
        z = torch.sqrt(-2.0 * torch.log(u1)) * torch.cos(2.0 * math.pi * u2)
        z = z.view(count, d)
        z = z / z.norm(dim=1, keepdim=True)
        return z.to(torch.float32)
    else:
        raise ValueError(cfg.values)
    return x.view(count, d)


def make_codebooks(cfg: WorkloadConfig, seed: int, device="cpu") -> torch.Tensor:
    """[M, 256, dsub] fp32: centroid (m, j) = sub-vector m of the j-th of 256
    fresh draws of the vector distribution ("drawn from the data")."""
    v = draw_vectors(cfg, stream_key(seed, cfg.name, "codebook"), 0, 256, device)
    return v.view(256, cfg.M, cfg.dsub).permute(1, 0, 2).contiguous()


def make_queries(cfg: WorkloadConfig, seed: int, device="cpu") -> torch.Tensor:
    return draw_vectors(cfg, stream_key(seed, cfg.name, "queries"), 0, cfg.B, device).contiguous()


def encode_nearest(x: torch.Tensor, codebooks: torch.Tensor, chunk: int = 0) -> torch.Tensor:
    """Offline PQ encode: nearest centroid per sub-space,
    squared L2, ties -> lowest centroid index.  x [n, d] -> uint8 [n, M]."""
    M, _, dsub = codebooks.shape
    n = x.shape[0]
    if chunk <= 0:
        chunk = max(1, (1 << 24) // (M * 256))
    out = torch.empty((n, M), dtype=torch.uint8, device=x.device)
    cb = codebooks.unsqueeze(0)                                  # [1, M, 256, dsub]
    for a in range(0, n, chunk):
        xs = x[a:a + chunk].view(-1, M, 1, dsub)
        d2 = ((xs - cb) ** 2).sum(-1)                            # [c, M, 256]
        out[a:a + chunk] = d2.argmin(dim=2).to(torch.uint8)
    return out


def make_codes(cfg: WorkloadConfig, seed: int, codebooks: torch.Tensor,
               device="cpu", n_hist: int = 1 << 17) -> torch.Tensor:
    """uint8 [N, M] PQ codes.

    'encode'    : encode all N vectors of the 'data' stream.
    'histogram' : encode n_hist vectors of the 'data' stream, take each
                  sub-space's 256-way code histogram and draw the N x M codes
                  i.i.d. from it (coordinates are i.i.d., so codes are too).
    """
    N, M = cfg.N, cfg.M
    kdata = stream_key(seed, cfg.name, "data")
    if cfg.codes_mode == "encode":
        out = torch.empty((N, M), dtype=torch.uint8, device=device)
        step = 1 << 16
        for a in range(0, N, step):
            n = min(step, N - a)
            out[a:a + n] = encode_nearest(draw_vectors(cfg, kdata, a, n, device), codebooks)
        return out
    if cfg.codes_mode != "histogram":
        raise ValueError(cfg.codes_mode)
    sample = encode_nearest(draw_vectors(cfg, kdata, 0, n_hist, device), codebooks)   # [n_hist, M]
    hist = torch.zeros((M, 256), dtype=torch.float64, device=device)
    hist.scatter_add_(1, sample.t().to(torch.int64),
                      torch.ones((M, n_hist), dtype=torch.float64, device=device))
    cdf = torch.cumsum(hist / hist.sum(1, keepdim=True), dim=1)                     # [M, 256]
    # 16-bit inverse-CDF table: table[m][u] = code for u/65536
    u = (torch.arange(65536, dtype=torch.float64, device=device) + 0.5) / 65536.0
    table = torch.searchsorted(cdf.contiguous(), u.expand(M, -1).contiguous()).clamp_(max=255).to(torch.uint8)
    kcodes = stream_key(seed, cfg.name, "codes")
    out = torch.empty((N, M), dtype=torch.uint8, device=device)
    flat = out.view(-1)
    total = N * M
    assert total % 4 == 0
    step = 1 << 27                                         # elements per chunk (multiple of 4)
    table_flat = table.view(-1)
    for e0 in range(0, total, step):
        ne = min(step, total - e0)
        h = hash64(kcodes, torch.arange(e0 // 4, (e0 + ne) // 4, dtype=torch.int64, device=device))
        f = torch.stack([(h >> s) & 0xFFFF for s in (0, 16, 32, 48)], dim=1).view(-1)   # [ne]
        m_idx = torch.arange(e0, e0 + ne, dtype=torch.int64, device=device) % M
        flat[e0:e0 + ne] = table_flat[m_idx * 65536 + f]
    return out


# --------------------------------------------------------------------------
# vector -> ID maps
# --------------------------------------------------------------------------

_FEISTEL_ROUNDS = 4


def feistel_permute(x: torch.Tensor, N: int, key: int) -> torch.Tensor:
    """Seeded bijection of [0, N) (int64 in, int64 out): a 4-round unbalanced Feistel network on
    ceil(log2 N) bits -- round i xors one half with a hash of the other half, so every round is
    invertible -- with cycle-walking: a value that lands in [N, 2^bits) goes through the network
    again until it falls below N.  A list's IDs then behave like uniformly random distinct
    positions of the code array (SURVEY.md 8(d) "Vector -> ID")."""
    bits = max(2, (N - 1).bit_length())
    a = bits // 2                      # low half
    b = bits - a                       # high half
    ma, mb = (1 << a) - 1, (1 << b) - 1
    keys = [stream_key(key, "feistel", r) for r in range(_FEISTEL_ROUNDS)]

    def network(v):
        lo, hi = v & ma, (v >> a) & mb
        for r in range(_FEISTEL_ROUNDS):
            if r % 2 == 0:
                hi = hi ^ (_lsr(hash64(keys[r], lo), 20) & mb)
            else:
                lo = lo ^ (_lsr(hash64(keys[r], hi), 20) & ma)
        return (hi << a) | lo

    y = network(x)
    while True:
        out = y >= N
        if not bool(out.any()):
            return y
        y = torch.where(out, network(y), y)


def vector_ids(cfg: WorkloadConfig, seed: int, t: torch.Tensor) -> torch.Tensor:
    """IDs (int64) of the distinct vectors with indices t (int64, < N)."""
    if cfg.id_map == "lattice":
        # Kronecker lattice: very evenly spread (three gap lengths) -- the friendliest case for an
        # order-preserving dedup table; kept for A/B measurements only
        return (t * _ID_MULT + stream_key(seed, cfg.name, "id_add") % cfg.N) % cfg.N
    if cfg.id_map == "feistel":
        return feistel_permute(t, cfg.N, stream_key(seed, cfg.name, "id_map"))
    raise ValueError(cfg.id_map)


# --------------------------------------------------------------------------
# posting lists with boundary replication
# --------------------------------------------------------------------------

def _mean_replicas(cfg: WorkloadConfig) -> float:
    rbar = (2 + cfg.r_max) / 2.0
    return 1.0 + cfg.p_rep * (rbar - 1.0)


def list_home_sizes(cfg: WorkloadConfig, seed: int, device="cpu") -> torch.Tensor:
    """int64 [n_lists]: number of 'home' (non-replica) vectors of each list,
    scaled so that the final mean list length (with replicas) is cfg.mean_list."""
    L = cfg.n_lists
    mean_home = cfg.mean_list / _mean_replicas(cfg)
    h = hash64(stream_key(seed, cfg.name, "list_sizes"), torch.arange(L, dtype=torch.int64, device=device))
    if cfg.size_law == "const":
        s = torch.full((L,), mean_home, dtype=torch.float64, device=device)
    elif cfg.size_law == "lognormal":
        sigma = 0.5
        u1 = (_lsr(h, 40).to(torch.float64) + 1.0) * (2.0 ** -24)
        u2 = _uniform53(hash64(stream_key(seed, cfg.name, "list_sizes2"),
                               torch.arange(L, dtype=torch.int64, device=device)))
        z = torch.sqrt(-2.0 * torch.log(u1)) * torch.cos(2.0 * math.pi * u2)
        s = mean_home * torch.exp(sigma * z - 0.5 * sigma * sigma)
    elif cfg.size_law == "powerlaw":
        # bounded power law p(s) ~ s^-1.1 on [16, 4096], rescaled to the mean
        a, lo, hi = 1.1, 16.0, 4096.0
        u = _uniform53(h)
        s = (lo ** (1 - a) + u * (hi ** (1 - a) - lo ** (1 - a))) ** (1.0 / (1 - a))
        mean_law = ((hi ** (2 - a) - lo ** (2 - a)) / (2 - a)) / ((hi ** (1 - a) - lo ** (1 - a)) / (1 - a))
        s = s * (mean_home / mean_law)
    else:
        raise ValueError(cfg.size_law)
    return torch.clamp(torch.round(s), min=1).to(torch.int64)


def _replica_count(cfg: WorkloadConfig, key: int, t: torch.Tensor):
    """(r, sigma) for distinct-vector indices t: r = number of lists holding the
    vector (1 = home only), sigma = +-1 side on which the nearest replica sits."""
    h = hash64(key, t)
    rep = _uniform24(h) < cfg.p_rep
    r = 2 + _randint(hash64(key ^ 0x2545F4914F6CDD1D, t), cfg.r_max - 1)     # U{2..r_max}
    r = torch.where(rep, r, torch.ones_like(r))
    sigma = torch.where((h & 1) == 1, 1, -1)
    return r, sigma


def _sources(cfg: WorkloadConfig):
    """Ring offsets a replica can sit at: 0 (home), +-1 .. +-ceil((r_max-1)/2)."""
    mmax = cfg.r_max // 2
    offs = [0]
    for m in range(1, mmax + 1):
        offs += [m, -m]
    return offs


def _has_offset(r: torch.Tensor, sigma: torch.Tensor, delta: int) -> torch.Tensor:
    """Vector with (r, sigma) has a copy at ring offset delta.  Extra copy j
    (1 <= j <= r-1) sits at sigma * (+1, -1, +2, -2, ...)[j-1]: the nearest
    adjacent lists first, as boundary vectors are assigned to the closest
    clusters."""
    if delta == 0:
        return torch.ones_like(r, dtype=torch.bool)
    m = abs(delta)
    same_side = (sigma > 0) == (delta > 0)
    return torch.where(same_side, r >= 2 * m, r >= 2 * m + 1)


@dataclass
class PostingLists:
    offsets: torch.Tensor      # int64 [n_lists + 1]
    ids: torch.Tensor          # int32 [entries] (vector IDs, all < 2^31)
    n_distinct: int            # distinct vectors referenced


def make_lists(cfg: WorkloadConfig, seed: int, device="cpu",
               lists_per_chunk: int = 1 << 16) -> PostingLists:
    L, N = cfg.n_lists, cfg.N
    home_sz = list_home_sizes(cfg, seed, device)
    home_start = torch.zeros(L + 1, dtype=torch.int64, device=device)
    home_start[1:] = torch.cumsum(home_sz, 0)
    T = int(home_start[-1])
    assert T <= N, f"{T} distinct vectors > N={N}"
    krep = stream_key(seed, cfg.name, "replicas")
    srcs = _sources(cfg)

    def chunk_attrs(l0, l1):
        t0, t1 = int(home_start[l0]), int(home_start[l1])
        t = torch.arange(t0, t1, dtype=torch.int64, device=device)
        home = torch.repeat_interleave(torch.arange(l0, l1, dtype=torch.int64, device=device),
                                       home_sz[l0:l1])
        r, sigma = _replica_count(cfg, krep, t)
        return t, home, r, sigma

    # pass 1: per (source, home list) counts
    cnt_home = torch.zeros((len(srcs), L), dtype=torch.int64, device=device)
    for l0 in range(0, L, lists_per_chunk):
        l1 = min(L, l0 + lists_per_chunk)
        t, home, r, sigma = chunk_attrs(l0, l1)
        for si, delta in enumerate(srcs):
            mask = _has_offset(r, sigma, delta)
            cnt_home[si, l0:l1] = torch.bincount(home[mask] - l0, minlength=l1 - l0)
    cnt_tgt = torch.stack([torch.roll(cnt_home[si], shifts=delta) for si, delta in enumerate(srcs)])
    sizes = cnt_tgt.sum(0)
    offsets = torch.zeros(L + 1, dtype=torch.int64, device=device)
    offsets[1:] = torch.cumsum(sizes, 0)
    base = torch.cumsum(cnt_tgt, 0) - cnt_tgt                     # [src, L] exclusive over sources
    E = int(offsets[-1])
    ids = torch.empty(E, dtype=torch.int32, device=device)

    # pass 2: scatter
    for l0 in range(0, L, lists_per_chunk):
        l1 = min(L, l0 + lists_per_chunk)
        t, home, r, sigma = chunk_attrs(l0, l1)
        vid = vector_ids(cfg, seed, t).to(torch.int32)
        for si, delta in enumerate(srcs):
            mask = _has_offset(r, sigma, delta)
            idx = torch.nonzero(mask, as_tuple=False).squeeze(1)
            if idx.numel() == 0:
                continue
            h_of = home[idx]
            c = cnt_home[si, l0:l1]
            seg_first = torch.cumsum(c, 0) - c
            rank = torch.arange(idx.numel(), dtype=torch.int64, device=device) - seg_first[h_of - l0]
            tgt = (h_of + delta) % L
            ids[offsets[tgt] + base[si, tgt] + rank] = vid[idx]
    return PostingLists(offsets=offsets, ids=ids, n_distinct=T)


# --------------------------------------------------------------------------
# per-query candidate lists (what the CPU sends to the GPU, PAPER.md:L125 (3)(4))
# --------------------------------------------------------------------------

def make_probes(cfg: WorkloadConfig, seed: int, device="cpu") -> torch.Tensor:
    """int64 [B, nprobe]: the posting lists each query probes, in probe order."""
    B, L, P = cfg.B, cfg.n_lists, cfg.nprobe
    kq = stream_key(seed, cfg.name, "probes")
    if cfg.probe_mode == "random":
        W = L
        start = torch.zeros(B, dtype=torch.int64, device=device)
    elif cfg.probe_mode == "window":
        W = min(L, cfg.window_factor * P)
        centre = _randint(hash64(kq, torch.arange(B, dtype=torch.int64, device=device)), L)
        start = centre - W // 2
    else:
        raise ValueError(cfg.probe_mode)
    assert P <= W
    keys = hash64(kq ^ 0x9E3779B97F4A7C15,
                  torch.arange(B * W, dtype=torch.int64, device=device)).view(B, W)
    keys = _lsr(keys, 1)                                          # non-negative, order = random
    sel = torch.topk(keys, P, dim=1, largest=False, sorted=True).indices
    return (start.unsqueeze(1) + sel) % L


def make_candidates(cfg: WorkloadConfig, lists: PostingLists, probes: torch.Tensor,
                    max_chunk_ids: int = 1 << 26):
    """CSR candidate lists: (cand_offsets int64 [B+1], cand_ids int32 [total]).
    Query b's candidates are its probed lists' IDs concatenated in probe order."""
    device = probes.device
    B, P = probes.shape
    lens = (lists.offsets[1:] - lists.offsets[:-1])[probes]         # [B, P]
    starts = lists.offsets[:-1][probes]
    per_q = lens.sum(1)
    cand_offsets = torch.zeros(B + 1, dtype=torch.int64, device=device)
    cand_offsets[1:] = torch.cumsum(per_q, 0)
    total = int(cand_offsets[-1])
    cand_ids = torch.empty(total, dtype=torch.int32, device=device)
    b0 = 0
    per_q_cpu = per_q.cpu()
    csum = torch.cumsum(per_q_cpu, 0)
    while b0 < B:
        # queries [b0, b1) with at most max_chunk_ids IDs (at least one query)
        base = int(csum[b0 - 1]) if b0 > 0 else 0
        b1 = int(torch.searchsorted(csum, torch.tensor(base + max_chunk_ids), right=True))
        b1 = max(b1, b0 + 1)
        b1 = min(b1, B)
        ln = lens[b0:b1].reshape(-1)
        st = starts[b0:b1].reshape(-1)
        n = int(ln.sum())
        if n:
            excl = torch.cumsum(ln, 0) - ln
            src = torch.repeat_interleave(st - excl, ln) + torch.arange(n, dtype=torch.int64, device=device)
            o = int(cand_offsets[b0])
            cand_ids[o:o + n] = lists.ids[src]
        b0 = b1
    return cand_offsets, cand_ids


@dataclass
class Workload:
    cfg: WorkloadConfig
    seed: int
    queries: torch.Tensor                  # [B, d] fp32
    codebooks: torch.Tensor                # [M, 256, dsub] fp32
    codes: Optional[torch.Tensor]          # [N, M] uint8 (None if not requested)
    cand_offsets: torch.Tensor             # [B+1] int64
    cand_ids: torch.Tensor                 # [total] int32 holding uint32 bit patterns
    stats: Dict[str, float] = field(default_factory=dict)
    list_offsets: Optional[torch.Tensor] = None   # [n_lists + 1] int64  (keep_lists=True)
    list_ids: Optional[torch.Tensor] = None       # [entries] int32
    probes: Optional[torch.Tensor] = None         # [B, nprobe] int32: the lists each query probes, in probe order


def make_raw_vectors(cfg: WorkloadConfig, seed: int, device="cpu", dtype=None) -> torch.Tensor:
    """The N raw vectors the codes were encoded from ('data' stream; only meaningful for codes_mode == 'encode',
    where code i is the nearest-centroid code of vector i), as fp32 or -- for integer-valued data -- uint8 / int8."""
    kdata = stream_key(seed, cfg.name, "data")
    want = dtype or {"u8": torch.uint8, "i8": torch.int8}.get(cfg.values, torch.float32)
    out = torch.empty((cfg.N, cfg.d), dtype=want, device=device)
    step = 1 << 16
    for a in range(0, cfg.N, step):
        n = min(step, cfg.N - a)
        out[a:a + n] = draw_vectors(cfg, kdata, a, n, device).to(want)
    return out


def make_page_table(cfg: WorkloadConfig, seed: int, device="cpu", page_bytes: int = 4096, elem_bytes: int = 1):
    """Vector -> SSD page in the *shape* of the paper's optimised layout: the raw vectors of a
    posting list's home members are stored together, page after page, so vectors of one cluster share pages.
    Distinct vector t (ordered by home list) sits in page t // per_page; IDs no list references follow.
    Returns (page_of int32 [N], n_pages)."""
    per_page = max(1, page_bytes // (cfg.d * elem_bytes))
    home_sz = list_home_sizes(cfg, seed, device)
    T = int(home_sz.sum())
    page_of = torch.full((cfg.N,), -1, dtype=torch.int32, device=device)
    step = 1 << 24
    for a in range(0, T, step):
        t = torch.arange(a, min(T, a + step), dtype=torch.int64, device=device)
        page_of[vector_ids(cfg, seed, t)] = (t // per_page).to(torch.int32)
    rest = torch.nonzero(page_of < 0, as_tuple=False).squeeze(1)
    first_free = (T + per_page - 1) // per_page
    page_of[rest] = (first_free + torch.arange(rest.numel(), dtype=torch.int64, device=device) // per_page).to(torch.int32)
    n_pages = first_free + (rest.numel() + per_page - 1) // per_page
    return page_of, int(n_pages)


def make_workload(cfg: WorkloadConfig, seed: int = DEFAULT_SEED, device="cpu",
                  with_codes: bool = True, keep_lists: bool = False) -> Workload:
    codebooks = make_codebooks(cfg, seed, device)
    queries = make_queries(cfg, seed, device)
    lists = make_lists(cfg, seed, device)
    probes = make_probes(cfg, seed, device)
    cand_offsets, cand_ids = make_candidates(cfg, lists, probes)
    sizes = (lists.offsets[1:] - lists.offsets[:-1]).to(torch.float64)
    per_q = (cand_offsets[1:] - cand_offsets[:-1]).to(torch.float64)
    stats = {
        "list_entries": int(lists.offsets[-1]),
        "distinct_vectors": lists.n_distinct,
        "list_mean": float(sizes.mean()),
        "list_p50": float(sizes.quantile(0.5)) if sizes.numel() <= (1 << 24) else float("nan"),
        "list_max": float(sizes.max()),
        "C_total": int(cand_offsets[-1]),
        "C_mean": float(per_q.mean()), "C_min": float(per_q.min()), "C_max": float(per_q.max()),
    }
    kept = (lists.offsets, lists.ids, probes.to(torch.int32)) if keep_lists else (None, None, None)
    del lists
    codes = make_codes(cfg, seed, codebooks, device) if with_codes else None
    return Workload(cfg, seed, queries, codebooks, codes, cand_offsets, cand_ids, stats, *kept)
