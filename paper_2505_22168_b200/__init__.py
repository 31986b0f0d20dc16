"""B200-native (sm_100a) GMNN energy-and-force path of arxiv 2505.22168 behind a C ABI.

    from paper_2505_22168_b200 import Model, System

The binding (and with it libgmnn_b200.so) is loaded on first use of any name below, so that
`python -m paper_2505_22168_b200.build` can run before the library exists.  If the shared object
is missing it is built in-tree with nvcc; if that is impossible the import fails.  The package
never imports oracle/ and has no CPU fallback.
"""
_NAMES = (
    "EXPORTS", "LIB_PATH", "GmnnError", "Model", "System", "launch_count", "measure_fp32_peak", "n_features", "lib", "sum_energies_static", "STATIC_SUM_MAX_ATOMS",
    "GMNN_OK", "GMNN_INVALID_ARG", "GMNN_UNSUPPORTED", "GMNN_NEIGHBOR_OVERFLOW", "GMNN_STALE_NEIGHBORS",
    "GMNN_CUDA_ERROR", "GMNN_OOM", "GMNN_OUT_OF_BOX", "GMNN_MLP_FP32", "GMNN_MLP_3XTF32", "GMNN_MLP_TF32", "GMNN_MLP_3XF16",
    "GMNN_FORCE_GATHER", "GMNN_FORCE_PAIRBUF",
)


def __getattr__(name):
    if name in _NAMES:
        from . import binding

        return getattr(binding, name)
    raise AttributeError("module %r has no attribute %r" % (__name__, name))


def __dir__():
    return sorted(list(globals()) + list(_NAMES))
