"""B200-native (sm_100a) intranuclear-cascade + evaporation Monte Carlo (arXiv:1309.7963).

The product is the C-ABI library built from csrc/ (declared in include/inc.h); this
package is a thin ctypes binding.  See DESIGN.md.
"""
__all__ = ["workloads"]
