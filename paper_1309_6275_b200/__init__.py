"""B200-native Hough-transform trigger hot path (arXiv:1309.6275): vote -> peaks -> tracks -> phi-cone jets.

The product is the C-ABI library built from csrc/ (include/hough.h) plus this thin binding.  Importing the
package does not load CUDA; `Hough` (binding.py) loads libhough_b200.so on first use and fails loudly if it
is missing -- there is no CPU fallback.  `workloads` holds the seeded synthetic input generators only.
"""
from . import workloads  # noqa: F401  (numpy only)


def __getattr__(name):
    if name in ("Hough", "HoughError"):
        import importlib
        return getattr(importlib.import_module(__name__ + ".binding"), name)
    raise AttributeError(name)
