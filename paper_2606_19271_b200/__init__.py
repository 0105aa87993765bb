"""B200-native coalesced chunk processing (the hot path of TurboServe, arxiv/paper_2606_19271).

The product is the C-ABI library `libturbochunk.so` (include/turbochunk.h); this package is the thin
Python binding with the same names (argument marshalling only).  PyTorch is used for device memory,
pinned host memory and streams.  There is no CPU fallback: importing the binding fails loudly when the
library is missing, and every compute call fails with TS_ERR_CUDA without an sm_100 GPU.
"""
import importlib

__all__ = ["TurboChunkError", "TurboChunkPool", "TurboSched", "StepPlan", "lib", "lib_path", "TS_COMMIT", "TS_RUN_APPEND", "TS_OK", "TS_ERR_INVALID",
           "TS_ERR_STATE", "TS_ERR_NO_PAGES", "TS_ERR_NO_HOST", "TS_ERR_CAPACITY", "TS_ERR_CUDA",
           "TS_SESSION_RESIDENT", "TS_SESSION_SUSPENDED", "EXPORTED_SYMBOLS"]


def __getattr__(name):
    # Lazy (PEP 562) so that `python -m paper_2606_19271_b200.build` can run before the library exists; the
    # first use of any binding name loads libturbochunk.so and raises ImportError if it is missing.
    if name in __all__ or name == "binding":
        mod = importlib.import_module(".binding", __name__)
        return mod if name == "binding" else getattr(mod, name)
    raise AttributeError(f"module {__name__!r} has no attribute {name!r}")
