"""paper_1711_07663_b200 -- B200-native direct-cut hole cutting (arxiv 1711.07663, section 4.2).

The product is libdc.so (hand-written sm_100a CUDA behind the C ABI of include/dc.h).  This
package is a thin ctypes binding with the same names: argument marshalling only.  PyTorch is
used by callers for device memory and streams; nothing here computes on the CPU and there is
no fallback: importing `binding` without the built library, or calling it without an sm_100
GPU, fails loudly.
"""
from ._build import build_lib, LIB  # noqa: F401

__all__ = ["build_lib", "LIB", "binding"]
