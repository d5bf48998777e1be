"""paper_1001_0599_b200 -- B200-native (sm_100a) hot path of Jia et al.'s TV-regularised
cone-beam CT reconstruction (arxiv 1001.0599): cone-beam forward projector, exact-transpose
back-projector, TV-prox (ROF by Armijo gradient descent) and the multi-grid
forward-backward-splitting driver, behind the C ABI of include/cbct.h.

  cbct    -- ctypes binding of libcbct.so (argument marshalling only; no CPU fallback)
  inputs  -- seeded synthetic problem descriptions and input arrays (numpy only)
  build   -- nvcc build of libcbct.so
"""
from . import inputs  # noqa: F401

__all__ = ["inputs", "cbct", "build"]
