"""Parallel-tempering diagnostics of PAPER.md:197 and Fig. 3: a thin front end of the C ABI's
``hsg_pt_diag_reset`` / ``hsg_pt_diag_get``.  The counters are accumulated on the device by the parallel-tempering kernel
itself (``pt_swap_kernel``); nothing is computed here.

* ``p_diff[t]``  — probability that, after a parallel-tempering pass, the copy of the system at ``T_t`` has moved to a
  neighbouring temperature (Fig. 3, main panel), averaged over samples and replicas.
* ``n_tunnel``   — per configuration, the number of closed loops between the end points ``T_1`` and ``T_{R_T}``
  ("A tunneling event occurs when a replica travels a closed loop between the temperature end points"):
  ``traversals // 2``, where every arrival at one end point after the last touch of the other one is a traversal.
"""
from __future__ import annotations


class PtDiagnostics:
    def __init__(self, eng):
        """Starts counting on ``eng`` (an ``Hsg`` engine): every later ``eng.pt_swap()`` is included."""
        self.eng = eng
        eng.pt_diag_reset()

    def p_diff(self):
        """[T] numpy array."""
        return self.eng.pt_diag_get()[2].cpu().numpy()

    def n_tunnel(self):
        """[D][O][T] closed loops per configuration slot (numpy)."""
        return (self.eng.pt_diag_get()[1] // 2).cpu().numpy()

    def n_pass(self) -> int:
        return self.eng.pt_diag_get()[3]
