"""B200-native mixed-batch paged attention for chunked-prefill serving (libcp).

The package is deliberately thin: `workloads` (seeded synthetic inputs, numpy only),
`build` (nvcc driver) and `binding` (ctypes marshalling over the C-ABI of
include/cp.h).  Importing the package loads nothing native; `binding.load()` fails
loudly when libcp.so is missing -- there is no CPU fallback.
"""
__all__ = ["workloads", "build", "binding"]
