"""ORACLE package — test infrastructure, NOT the product.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code, header, table or
constant with the CUDA library in ``paper_2107_14008_b200/`` and never imports it.

Contents
  p2p_oracle.c   plain fp64 minimum-image direct sum of the truncated P2P force (§2, Eq. 1)
  binding.py     builds p2p_oracle.c with gcc and calls it through ctypes (marshalling only)
  table.py       Eq. 2 written out in numpy fp64: the Taylor interpolation of T
  m2l.py         truncated M2L: the prefactors f_(n), the derivative tensors D_n, P2M / M2L / L2P
"""
from .binding import build, oracle_T, p2p, p2p_sampled, num_threads  # noqa: F401
from .table import make_table, eval_table  # noqa: F401
from . import m2l  # noqa: F401
