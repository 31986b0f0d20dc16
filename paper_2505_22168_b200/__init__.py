"""B200-native (sm_100a) GMNN energy-and-force path of arxiv 2505.22168 behind a C ABI.

    from paper_2505_22168_b200 import Model, System

Importing this package loads libgmnn_b200.so (build it with `python -m paper_2505_22168_b200.build`).
It never imports oracle/ and has no CPU fallback.
"""
from .binding import (  # noqa: F401
    EXPORTS, LIB_PATH, GmnnError, Model, System, launch_count, n_features,
    GMNN_OK, GMNN_INVALID_ARG, GMNN_UNSUPPORTED, GMNN_NEIGHBOR_OVERFLOW, GMNN_STALE_NEIGHBORS,
    GMNN_CUDA_ERROR, GMNN_OOM, GMNN_OUT_OF_BOX, GMNN_MLP_FP32, GMNN_MLP_3XTF32, GMNN_MLP_TF32,
    GMNN_FORCE_GATHER, GMNN_FORCE_PAIRBUF,
)
