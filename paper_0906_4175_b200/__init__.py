"""gwmf — matched filter + chi^2 veto hot path of arxiv/paper_0906_4175 on one B200.

Sub-modules
  gwmf   : thin ctypes binding over the C-ABI library ``libgwmf.so`` (include/gwmf.h).
  build  : compiles the library in-tree with nvcc for sm_100a.

The seeded synthetic workloads used by the tests and bench.py live in ``workloads.py`` at the
repository root: they are test/bench inputs, not part of the shipped library.
"""

__all__ = ["gwmf", "build"]
