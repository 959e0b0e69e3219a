"""The band clause of BASELINE.json for parallel-tempering decisions ("identical except where |dbeta*dE| lies within
1e-4 of the acceptance threshold"), as a helper of the lockstep parity tests; checked on its own in test_pt_band.py."""
import numpy as np

from tests import philox_np as pnp


def excuse_or_fail(acc_g, acc_o, E_pre, beta, seed, k_pt, O, sample_offset=0):
    """BASELINE.json: swap decisions identical except where |dbeta*dE - ln u| lies within 1e-4 of the threshold.  For every
    chain (d, o) with a mismatch, walk the ladder as the oracle did (energies by temperature index BEFORE the pass, swapped
    along with every accepted exchange) up to the FIRST differing pair and require that this very pair sat inside the band;
    later differences of the same chain are consequences of the first."""
    for d, o in sorted({(d, o) for d, o, _ in zip(*np.nonzero(acc_g != acc_o))}):
        e = np.array(E_pre[d, o], dtype=np.float64)
        for t in range(len(e) - 1):
            x = (beta[t + 1] - beta[t]) * (e[t + 1] - e[t])
            if acc_g[d, o, t] != acc_o[d, o, t]:
                u = float(pnp.u01(pnp.draw(pnp.DOMAIN_PT, t, k_pt, (sample_offset + d) * O + o, seed)[0]))
                assert x < 0 and abs(x - np.log(u)) < 1e-4, f"PT decision differs outside the band: d={d} o={o} t={t} x={x} ln u={np.log(u)}"
                break
            if acc_o[d, o, t]:
                e[[t, t + 1]] = e[[t + 1, t]]
