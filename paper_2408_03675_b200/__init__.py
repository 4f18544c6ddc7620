"""B200-native NACL one-shot encoding-phase KV-cache eviction (arXiv 2408.03675).

The product is the C-ABI library `libnacl_evict.so` (include/nacl_evict.h) built from
csrc/*.cu for sm_100a; `binding` is argument marshalling only.  `configs` / `inputs`
are host-side workload description shared with the tests.  Nothing here imports the
CPU oracle.
"""
from .configs import CONFIGS, EvictConfig, budget_counts  # noqa: F401

__all__ = ["CONFIGS", "EvictConfig", "budget_counts", "nacl_evict", "binding"]


def __getattr__(name):  # lazy: importing the package must not need the CUDA library
    if name == "binding":
        import importlib

        return importlib.import_module(".binding", __name__)
    if name in ("nacl_evict", "nacl_evict_ex", "nacl_workspace_bytes", "nacl_evict_host", "nacl_evict_generation"):
        from . import binding

        return getattr(binding, name)
    raise AttributeError(name)
