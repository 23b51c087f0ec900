"""B200-native (sm_100a) decode-stage hot path of Prefilling-dLLM (arxiv/paper_2606_10537).

`binding` is the thin ctypes layer over the C-ABI library declared in include/pdllm.h;
`workloads` is the seeded synthetic-input generator.  Nothing here computes the
method on the CPU: without the compiled CUDA library the binding raises.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "binding"]


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
