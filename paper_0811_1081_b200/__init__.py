"""B200-native (sm_100a) hot path of Andrecut's iterative PCA (arxiv 0811.1081).

  * `paper_0811_1081_b200.csrc`    hand-written CUDA kernels + the C ABI of include/pca.h
  * `paper_0811_1081_b200.binding` thin ctypes binding with the same names (argument marshalling only)
  * `paper_0811_1081_b200.sharded` calling sequence of the row-sharded multi-GPU entry points (places the one all-reduce per pass)
  * `paper_0811_1081_b200.inputs`  seeded synthetic inputs (no method arithmetic; shared with the oracle's tests)

The binding is imported lazily so that `inputs` can be used without torch or the CUDA library.
"""
__all__ = ["binding", "inputs", "sharded"]


def __getattr__(name):
    if name in ("binding", "inputs", "sharded"):
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
