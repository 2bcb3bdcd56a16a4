"""B200-native (sm_100a) Lookahead Sparse Attention decode hot path (arxiv/paper_2606_09079).

`paper_2606_09079_b200.lsa`       - thin ctypes binding of the C-ABI library (liblsa.so)
`paper_2606_09079_b200.workloads` - seeded synthetic inputs (no method arithmetic)

The binding is imported lazily so that `workloads` stays usable without the CUDA build;
touching any LSA entry point without the built library raises immediately (no CPU fallback).
"""

__all__ = ["lsa", "workloads"]


def __getattr__(name):
    if name in ("lsa", "workloads"):
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
