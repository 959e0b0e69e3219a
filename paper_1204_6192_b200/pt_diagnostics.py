"""Parallel-tempering diagnostics of PAPER.md:197 and Fig. 3, from what the C ABI already returns.

Nothing here is on the hot path: ``hsg_pt_swap`` reports its accept flags and ``hsg_get_state`` the permutation
``slot_of_temp`` (which configuration slot holds which temperature); this module only accumulates them, with torch
tensor ops on the engine's device (plumbing, no kernels of its own).

* ``p_diff[t]``  — probability that, after a parallel-tempering pass, the configuration that held temperature ``T_t``
  has moved to a neighbouring temperature (Fig. 3, main panel), averaged over samples and replicas.
* ``n_tunnel``   — per configuration, the number of closed loops between the end points ``T_1`` and ``T_{R_T}``
  ("A tunneling event occurs when a replica travels a closed loop between the temperature end points",
  PAPER.md:234): every arrival at one end point after the other one counts half a loop.
"""
from __future__ import annotations


class PtDiagnostics:
    def __init__(self, eng=None, perm=None):
        """``eng``: an hsg engine (its permutation is read with ``get_state``), or ``perm``: the initial
        ``slot_of_temp[D][O][T]`` as a torch tensor when the permutations are fed by hand (``after_pt_swap(perm)``)."""
        import torch as t
        self.eng, self.torch = eng, t
        self._perm = (eng.get_state()[0] if perm is None else perm).to(t.int64)
        D, O, T = self._perm.shape
        self.T, dev = T, self._perm.device
        self.n_pass = 0
        self.moved = t.zeros((D, O, T), dtype=t.int64, device=dev)       # by temperature index
        self.last_end = t.zeros((D, O, T), dtype=t.int8, device=dev)     # by slot: 0 none, +1 cold end, -1 hot end
        self.traversals = t.zeros((D, O, T), dtype=t.int64, device=dev)  # by slot: end-to-end traversals
        self._touch(self._perm)

    def _touch(self, perm):
        """Configurations now sitting at an end point: count a traversal if they last touched the other one."""
        t, T = self.torch, self.T
        for t_end, tag in ((0, 1), (T - 1, -1)):
            slot = perm[..., t_end:t_end + 1]                                    # [D][O][1]
            last = self.last_end.gather(2, slot)
            crossed = (last == -tag).to(t.int64)
            self.traversals.scatter_add_(2, slot, crossed)
            self.last_end.scatter_(2, slot, t.full_like(last, tag))

    def after_pt_swap(self, perm=None):
        """Call once after every parallel-tempering pass (``eng.pt_swap()``), or pass the new permutation by hand."""
        t = self.torch
        if perm is None:
            with t.cuda.stream(self.eng.stream):
                return self.after_pt_swap(self.eng.get_state()[0])
        perm = perm.to(t.int64)
        self.moved += (perm != self._perm).to(t.int64)                          # the slot that held T_t holds another one now
        self._perm = perm
        self.n_pass += 1
        self._touch(perm)

    def p_diff(self):
        """[T] probability per temperature, averaged over samples and replicas."""
        return (self.moved.to(self.torch.float64).mean(dim=(0, 1)) / max(self.n_pass, 1)).cpu().numpy()

    def n_tunnel(self):
        """[D][O][T] closed loops per configuration slot."""
        return (self.traversals // 2).cpu().numpy()
