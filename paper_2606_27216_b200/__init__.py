"""B200-native HiMuon hot path (arxiv/paper_2606_27216): tiled Newton-Schulz optimizer update.

The product is the C-ABI shared library `libhimuon.so` (include/himuon.h), built in-tree from
`csrc/` by `paper_2606_27216_b200.build`.  This package is its thin Python binding.
"""
from .binding import (  # noqa: F401
    HIMUON_BF16, HIMUON_F32, HIMUON_PATH_AUTO, HIMUON_PATH_FP32, HIMUON_PATH_FP8, HParams, HimuonError, NS_COEFFS, Plan,
    himuon_launch_count, himuon_layer, himuon_mat, himuon_ns_tiles, himuon_ns_tiles_static,
    himuon_ns_tiles_static_max_tiles, himuon_plan_chunks,
    himuon_supported_tile_sizes, mat_of, shape_mat,
)
