"""NumPy ``einsum`` twin of the oracle -- TEST INFRASTRUCTURE (pin P11).

The same definition as oracle_elph.c's header (Eq. 13 + Eq. 7 of PAPER.md,
L133 / L98, readings R1-R7), written as library tensor contractions so the C
loops are pinned to a textbook routine.  Shares no code with the CUDA path.
"""
from __future__ import annotations

import numpy as np


def phases(kpts: np.ndarray, R: np.ndarray, deg: np.ndarray | None) -> np.ndarray:
    """exp(2 pi i k.R)/deg, shape [..., nR]."""
    x = np.tensordot(np.asarray(kpts, dtype=np.float64), np.asarray(R, dtype=np.float64).T, axes=1)
    ph = np.exp(2j * np.pi * x)
    return ph if deg is None else ph / deg


def elph_einsum(gW, Re, Rp, deg_e, deg_p, k, Uk, q, Ukq, ev, omega) -> np.ndarray:
    phe = phases(k, Re, deg_e)                      # [nRe]
    php = phases(q, Rp, deg_p)                      # [nq, nRp]
    # G[q,b1,b2,nu] = sum phe[e] php[q,p] Uk[w1,b1] conj(Ukq[q,w2,b2]) ev[q,ka,nu] gW[p,e,w1,w2,ka]
    G = np.einsum("e,qp,ab,qcd,qkn,peack->qbdn", phe, php, Uk, np.conj(Ukq), ev, gW, optimize=True)
    w = np.asarray(omega)[:, None, None, :]
    with np.errstate(divide="ignore", invalid="ignore"):
        out = np.where(w > 0, (G.real ** 2 + G.imag ** 2) / (2.0 * w), 0.0)
    return out
