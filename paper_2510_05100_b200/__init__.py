"""B200-native batched matrix-element reweighting (arxiv 2510.05100: Rex / teaRex / MadtRex hot path).

Thin ctypes binding over the C ABI of include/rex_trex.h (librex_trex.so, hand-written CUDA for sm_100a).
Every step of the path runs in the library's kernels; this package only marshals arguments. PyTorch is
used for device memory and streams. There is no CPU fallback: importing works without a GPU (so that the
exported symbols can be checked), any compute call without the built library or a CUDA device raises.
"""
from .binding import (  # noqa: F401
    lib, library_path, exported_symbols, TrexError,
    rex_pack_key, rex_pack_key_filtered, rex_keys, rex_keys_filtered, rex_bucket, rex_bucket_keys, rex_gather, rex_scatter,
    trex_subproc_id, trex_npar, trex_ncolor, trex_nhel, trex_colour_matrix,
    trex_reweight, trex_run, trex_run_multi, trex_run_alphas, trex_run_pdg, trex_run_host, trex_debug_flow_amps, trex_debug_xtile, trex_debug_helicity_me2, trex_probe_fma, trex_xsec_moments, trex_xsec_moments_noalloc, TREX_XSEC_NOALLOC_MAX_EVENTS, trex_xsec_finish,
    trex_set_stream, trex_set_precision, trex_get_precision, trex_set_algorithm, trex_set_poly_multi, trex_set_helicity_symmetry, trex_launch_count, trex_graph_replays, trex_kernel_timing, trex_kernel_time, trex_last_error, trex_shutdown,
    REX_MAX_BUCKETS, REX_NPOS, TREX_NTHETA, SUBPROCESS_IDS,
)
