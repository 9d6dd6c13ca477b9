"""B200-native AutoDDL strategy-search hot path (arxiv 2301.06813): SBP cost tables, chain DP, Coordinate Descent.

`binding` (the ctypes layer over the C-ABI library) is imported lazily so that the input
generators in `configs` can be used without torch or the CUDA library.
"""


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
