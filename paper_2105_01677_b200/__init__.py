"""B200-native MPS time-step particle-interaction path (arXiv 2105.01677).

`scenes` (seeded inputs) imports nothing native.  `binding` loads the C-ABI
CUDA library `libmps_b200.so` and raises if it is missing: there is no CPU
fallback anywhere in this package.
"""
from . import scenes  # noqa: F401


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
