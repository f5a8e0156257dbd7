"""B200-native FP8 attention forward with the paper's kernel-faithful P-cast semantics.

The CUDA library is loaded lazily (first use of `fp8attn`), so that importing
`paper_2606_06521_b200.workloads` never touches it.
"""
__all__ = ["fp8attn", "workloads", "sharding"]


def __getattr__(name):
    if name == "fp8attn":
        import importlib
        return importlib.import_module(".fp8attn", __name__)
    raise AttributeError(name)
