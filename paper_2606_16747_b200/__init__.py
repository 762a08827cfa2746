"""B200-native neural-OIT resolve (STAR-NT hot path, arxiv/paper_2606_16747).

`Noit` is the thin binding over the C ABI in include/noit.h (libnoit.so, hand-written CUDA for
sm_100a).  No CPU fallback: loading fails loudly when the library is missing.
"""
from .binding import (ABSENT, EXPORTS, MLP_BF16, MLP_FP32, MLP_PARAMS, QT_CORNER, QT_VARIANCE,  # noqa: F401
                      RGBA_F16, RGBA_F32, DeviceFragBuf, Noit, NoitError, lib, lib_path)
from .sharding import (balance_band, band_matrix, exchange_halo_rows, extended_band, gather_rows, halo_rows,  # noqa: F401
                       shard_rows, slice_rows)
