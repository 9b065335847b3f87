"""Named synthetic workloads (BASELINE.json `configs`).

This module only *describes* inputs.  It holds none of the method's
arithmetic (no lookup table, no dedup, no ADC, no top-k) and is imported by
the oracle tests, the GPU tests and bench.py alike.

The paper measures on SIFT1B / SPACEV1B / DEEP1B (PAPER.md:L224-L229,
Table 1).  Those datasets are not available here; the configs below take
their shapes (d, dtype) and BASELINE.json's value distributions and stand
in for them.
"""
from __future__ import annotations

from dataclasses import dataclass, replace


@dataclass(frozen=True)
class WorkloadConfig:
    name: str
    N: int                 # vectors (rows of the PQ code array)
    d: int                 # vector dimension
    M: int                 # PQ sub-spaces (bytes per code)
    values: str            # 'uniform01' | 'u8' | 'i8' | 'gauss_norm'
    n_lists: int           # posting lists
    mean_list: int         # final mean posting-list length (IDs incl. replicas)
    size_law: str          # 'const' | 'lognormal' | 'powerlaw'
    p_rep: float           # fraction of vectors replicated into >1 list
    r_max: int             # max lists per replicated vector (<= 8)
    B: int                 # queries per batch
    nprobe: int            # probed posting lists per query (paper's top-m)
    k: int                 # candidates returned (paper's top-n)
    probe_mode: str        # 'window' (adjacent lists) | 'random'
    window_factor: int     # window = window_factor * nprobe lists around a centre
    codes_mode: str        # 'encode' (true nearest-centroid) | 'histogram'
    integer_exact: bool    # all fp32 arithmetic exact (integers < 2^24)
    id_map: str = "feistel"  # distinct vector -> ID: 'feistel' (seeded random bijection of [0, N)) | 'lattice' ((A t + c) mod N)

    @property
    def dsub(self) -> int:
        return self.d // self.M

    def scaled(self, **kw) -> "WorkloadConfig":
        """A smaller workload with the same structure (tests)."""
        return replace(self, **kw)


CONFIGS = {
    # configs[0]: tiny, literal reading ("8 random lists")
    "tiny": WorkloadConfig(
        name="tiny", N=100_000, d=128, M=16, values="uniform01",
        n_lists=1_000, mean_list=100, size_law="const", p_rep=0.10, r_max=2,
        B=64, nprobe=8, k=10, probe_mode="random", window_factor=2,
        codes_mode="encode", integer_exact=False),
    # configs[0] with adjacent probes, so that duplicates actually occur
    "tiny_local": WorkloadConfig(
        name="tiny_local", N=100_000, d=128, M=16, values="uniform01",
        n_lists=1_000, mean_list=100, size_law="const", p_rep=0.10, r_max=2,
        B=64, nprobe=8, k=10, probe_mode="window", window_factor=2,
        codes_mode="encode", integer_exact=False),
    # configs[1]: 10M x 128 uint8 (SIFT-shaped), M=32
    "u8_10m_m32": WorkloadConfig(
        name="u8_10m_m32", N=10_000_000, d=128, M=32, values="u8",
        n_lists=20_000, mean_list=500, size_law="lognormal", p_rep=0.20, r_max=4,
        B=1024, nprobe=64, k=100, probe_mode="window", window_factor=2,
        codes_mode="encode", integer_exact=True),
    # configs[2]: 100M x 96 fp32 (DEEP-shaped), M=48
    "f32_100m_m48": WorkloadConfig(
        name="f32_100m_m48", N=100_000_000, d=96, M=48, values="gauss_norm",
        n_lists=200_000, mean_list=500, size_law="lognormal", p_rep=0.25, r_max=8,
        B=4096, nprobe=128, k=100, probe_mode="window", window_factor=2,
        codes_mode="histogram", integer_exact=False),
    # configs[3]: 1B x 100 int8 (SPACEV-shaped), M=25
    "i8_1b_m25": WorkloadConfig(
        name="i8_1b_m25", N=1_000_000_000, d=100, M=25, values="i8",
        n_lists=2_000_000, mean_list=500, size_law="powerlaw", p_rep=0.30, r_max=8,
        B=10_000, nprobe=64, k=100, probe_mode="window", window_factor=2,
        codes_mode="histogram", integer_exact=True),
    # configs[4]: 1B x 128 uint8 (SIFT1B-shaped), M=64, k=1000
    "u8_1b_m64": WorkloadConfig(
        name="u8_1b_m64", N=1_000_000_000, d=128, M=64, values="u8",
        n_lists=2_000_000, mean_list=500, size_law="powerlaw", p_rep=0.30, r_max=8,
        B=10_000, nprobe=256, k=1000, probe_mode="window", window_factor=2,
        codes_mode="histogram", integer_exact=True),
}

# BASELINE.json order
BASELINE_ORDER = ["tiny", "u8_10m_m32", "f32_100m_m48", "i8_1b_m25", "u8_1b_m64"]


def mini(name: str, N: int, n_lists: int, B: int, **kw) -> WorkloadConfig:
    """Structure of a big config at a size the CPU oracle finishes in seconds."""
    c = CONFIGS[name]
    return c.scaled(name=f"{name}@mini", N=N, n_lists=n_lists, B=B,
                    codes_mode=kw.pop("codes_mode", c.codes_mode), **kw)
