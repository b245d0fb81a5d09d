"""paper_2606_28952_b200 -- B200-native operator-state multiplication (H|psi>, <psi|H|psi>, grouped
Pauli rotations, Taylor propagation) for Pauli sums in binary symplectic form on (N_alpha, N_beta)
sectors.  All compute is in csrc/*.cu behind the C ABI of include/bs.h (libbs.so); `bs` is the thin
ctypes binding, `jw_terms` emits the raw Jordan-Wigner term lists that bs_group_xmask consumes.
"""
from . import build as _build  # noqa: F401  (build script; does not compile on import)


def load():
    """Import the binding (raises ImportError if libbs.so has not been built)."""
    from . import bs
    return bs
