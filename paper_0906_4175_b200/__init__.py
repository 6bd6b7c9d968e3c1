"""gwmf — matched filter + chi^2 veto hot path of arxiv/paper_0906_4175 on one B200.

Sub-modules
  inputs : seeded synthetic workloads (noise, injections, banks).  Pure numpy, no
           method arithmetic shared with either the oracle or the CUDA path.
  gwmf   : thin ctypes binding over the C-ABI library ``libgwmf.so`` (include/gwmf.h).
           Imported lazily so that the CPU-only test tier can import ``inputs``
           on a box without the CUDA runtime being initialised.
"""

__all__ = ["inputs", "gwmf"]
