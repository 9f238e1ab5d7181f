"""libshaken: B200-native (sm_100a) shaken-dynamics PCA half-step (arXiv 1908.07341).

Importing the package is cheap; the CUDA library is loaded by ``paper_1908_07341_b200.shaken.lib()`` on first
use and fails loudly if it has not been built (``python -m paper_1908_07341_b200.build``).  No CPU fallback."""
__all__ = ["workloads", "shaken", "build"]
