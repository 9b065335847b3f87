"""B200-native GPU stage of FusionANNS (arxiv 2409.16576): thin Python binding of the
C-ABI library declared in include/fann.h.  Every step of the path runs in the CUDA
kernels of csrc/; this package only marshals arguments.  Importing it does not load
the library; the first call does, and fails loudly if libfann.so is missing."""
from .binding import (FANN_ID_NONE, FANN_MAX_K, FANN_MAX_M, FannError, FannIndex, fann_build_lut,
                      fann_create, fann_dedup_only, fann_dedup_scan_topk, fann_destroy, fann_gather_probe, fann_get_info,
                      fann_last_error, fann_last_timing, fann_load_codes, fann_search_host, fann_search_host_scratch_bytes, fann_set_timing,
                      fann_version, fann_workspace_bytes, fann_workspace_status, library_path, load_library)
