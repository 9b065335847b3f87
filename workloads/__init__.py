"""Seeded synthetic inputs shared by the oracle tests, the CUDA tests and bench.py.
Holds input construction only; none of the hot path's arithmetic."""
from .configs import CONFIGS, BASELINE_ORDER, WorkloadConfig, mini
from .generate import (DEFAULT_SEED, ID_NONE, Workload, make_workload, make_codebooks,
                       make_queries, make_codes, make_lists, make_probes, make_candidates,
                       encode_nearest, draw_vectors, stream_key, hash64, feistel_permute, vector_ids, make_raw_vectors, make_page_table)
