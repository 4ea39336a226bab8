"""paper_2007_03143_b200: B200-native XC integration (arxiv 2007.03143 hot path) -- Python binding of
the C-ABI library libxc_b200.so.

The binding is loaded on first use (so that `python -m paper_2007_03143_b200.build` can run before the
library exists); any use of the API without the built CUDA library raises ImportError -- there is no
CPU fallback."""

_API = ("EXPORTED", "LIB_PATH", "Plan", "XC_SPEC_SPLIT_CLASS1", "XC_STATIC_MAX_POINTS", "XcError", "XcGridSpec", "functional", "functional_uks_static", "grid_spec",
        "measure_fp64_peak", "partition_weights", "xc_integrate")


def __getattr__(name):
    if name in _API or name == "binding":
        import importlib
        b = importlib.import_module(".binding", __name__)
        return b if name == "binding" else getattr(b, name)
    raise AttributeError(name)
