"""B200-native L.A.Cosmic hot path (arxiv/paper_2602_17938, dfcosmic): thin Python binding.

The product is liblacosmic_b200.so (hand-written sm_100a CUDA kernels behind the C ABI declared in
include/lacosmic.h).  This package only marshals arguments; torch is used for device memory and
streams.  There is no CPU fallback: every call raises if the CUDA library cannot be loaded.
"""
from .binding import (  # noqa: F401
    MAX_NITER,
    MODE_DENSE,
    MODE_LAZY,
    FS_ADU,
    FS_NORMALISED,
    LacosmicError,
    Params,
    lacosmic_bitplane_pitch_words,
    lacosmic_clean,
    lacosmic_dilate3,
    lacosmic_estimate_gain,
    lacosmic_host_workspace_bytes,
    lacosmic_kernel_timing_enable,
    lacosmic_kernel_timing_read,
    lacosmic_last_launch_count,
    lacosmic_lplus,
    lacosmic_masked_median,
    lacosmic_medfilt,
    lacosmic_pack_bits,
    lacosmic_probe_minmax_rate,
    lacosmic_run,
    lacosmic_run_batch,
    lacosmic_run_host,
    lacosmic_run_ws,
    lacosmic_run_ex,
    lacosmic_run_sepmed_compare,
    lacosmic_sepmed_workspace_bytes,
    lacosmic_sepmedfilt,
    lacosmic_satstar_mask,
    lacosmic_masked_median_bpm,
    lacosmic_strerror,
    lacosmic_unpack_bits,
    lacosmic_version,
    lacosmic_workspace_bytes,
    lacosmic_batch_workspace_bytes,
    lacosmic_host_batch_workspace_bytes,
    lacosmic_run_host_batch,
    lacosmic_run_host_sparse,
    lacosmic_run_host_stream_sparse,
    library_path,
    load_library,
)

__all__ = [n for n in dir() if n.startswith("lacosmic_")] + ["LacosmicError", "Params",
                                                              "library_path", "load_library",
                                                              "MODE_LAZY", "MODE_DENSE", "MAX_NITER",
                                                              "FS_ADU", "FS_NORMALISED"]
