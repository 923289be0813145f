"""KVarN hot path for B200 (sm_100a): C-ABI CUDA library + thin ctypes binding.

`from paper_2606_03458_b200 import kvarn` loads the CUDA library (and fails
loudly if it has not been built); `workloads` is importable without it.
"""
__all__ = ["kvarn", "workloads"]


def __getattr__(name):
    if name in ("kvarn", "workloads", "build"):
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
