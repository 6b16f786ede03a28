"""CPU oracle for the el-ph Wannier->Bloch |g|^2 hot path -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
``--impl reference`` legs may import this package.  It shares no code with the
CUDA path (paper_2111_14999_b200/csrc, binding) and neither imports the other.

``oracle.direct / setk / setk_slab / qbatch`` are thin ctypes wrappers around
oracle_elph.c (plain C99; see its header for the paper passages it follows).
``oracle.oracle_einsum`` is the independent NumPy twin (pin P11).
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build.build())
        _lib.oracle_num_threads.restype = ctypes.c_int
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _c(a, dtype, shape=None):
    a = np.ascontiguousarray(a, dtype=dtype)
    if shape is not None:
        assert a.shape == tuple(shape), (a.shape, tuple(shape))
    return a


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def direct(gW, Re, Rp, deg_e, deg_p, k, Uk, q, Ukq, ev, omega):
    """Plain double sum over (Re,Rp), Eq. 13 + Eq. 7.  Returns out[nq][nb1][nb2][nm]."""
    nRp, nRe, nw, _, nm = gW.shape
    nb1 = Uk.shape[1]
    nq, _, nb2 = Ukq.shape
    gW = _c(gW, np.complex128); Re = _c(Re, np.float64, (nRe, 3)); Rp = _c(Rp, np.float64, (nRp, 3))
    deg_e = None if deg_e is None else _c(deg_e, np.float64, (nRe,))
    deg_p = None if deg_p is None else _c(deg_p, np.float64, (nRp,))
    k = _c(k, np.float64, (3,)); Uk = _c(Uk, np.complex128, (nw, nb1))
    q = _c(q, np.float64, (nq, 3)); Ukq = _c(Ukq, np.complex128, (nq, nw, nb2))
    ev = _c(ev, np.complex128, (nq, nm, nm)); omega = _c(omega, np.float64, (nq, nm))
    out = np.empty((nq, nb1, nb2, nm), dtype=np.float64)
    rc = _load().oracle_direct(nRe, nRp, nw, nm, nb1, nb2, nq, _p(gW), _p(Re), _p(Rp), _p(deg_e),
                               _p(deg_p), _p(k), _p(Uk), _p(q), _p(Ukq), _p(ev), _p(omega), _p(out))
    assert rc == 0
    return out


def setk_slab(gW_p, Re, deg_e, k, Uk):
    """Eq. 71 for one phonon lattice vector: g1_p[nb1][nw][nm]."""
    nRe, nw, _, nm = gW_p.shape
    nb1 = Uk.shape[1]
    gW_p = _c(gW_p, np.complex128); Re = _c(Re, np.float64, (nRe, 3))
    deg_e = None if deg_e is None else _c(deg_e, np.float64, (nRe,))
    k = _c(k, np.float64, (3,)); Uk = _c(Uk, np.complex128, (nw, nb1))
    g1 = np.empty((nb1, nw, nm), dtype=np.complex128)
    rc = _load().oracle_setk_slab(nRe, nw, nm, nb1, _p(gW_p), _p(Re), _p(deg_e), _p(k), _p(Uk), _p(g1))
    assert rc == 0
    return g1


def setk(gW, Re, deg_e, k, Uk):
    """Eq. 71 (steps a1+a2): g1[nRp][nb1][nw][nm]."""
    nRp, nRe, nw, _, nm = gW.shape
    nb1 = Uk.shape[1]
    gW = _c(gW, np.complex128); Re = _c(Re, np.float64, (nRe, 3))
    deg_e = None if deg_e is None else _c(deg_e, np.float64, (nRe,))
    k = _c(k, np.float64, (3,)); Uk = _c(Uk, np.complex128, (nw, nb1))
    g1 = np.empty((nRp, nb1, nw, nm), dtype=np.complex128)
    rc = _load().oracle_setk(nRe, nRp, nw, nm, nb1, _p(gW), _p(Re), _p(deg_e), _p(k), _p(Uk), _p(g1))
    assert rc == 0
    return g1


def qbatch(g1, Rp, deg_p, q, Ukq, ev, omega):
    """Rest of Eq. 70 + Eq. 7 (steps a3..a7): out[nq][nb1][nb2][nm]."""
    nRp, nb1, nw, nm = g1.shape
    nq, _, nb2 = Ukq.shape
    g1 = _c(g1, np.complex128); Rp = _c(Rp, np.float64, (nRp, 3))
    deg_p = None if deg_p is None else _c(deg_p, np.float64, (nRp,))
    q = _c(q, np.float64, (nq, 3)); Ukq = _c(Ukq, np.complex128, (nq, nw, nb2))
    ev = _c(ev, np.complex128, (nq, nm, nm)); omega = _c(omega, np.float64, (nq, nm))
    out = np.empty((nq, nb1, nb2, nm), dtype=np.float64)
    rc = _load().oracle_qbatch(nRp, nw, nm, nb1, nb2, nq, _p(g1), _p(Rp), _p(deg_p), _p(q), _p(Ukq),
                               _p(ev), _p(omega), _p(out))
    assert rc == 0
    return out


def elph(gW, Re, Rp, deg_e, deg_p, k, Uk, q, Ukq, ev, omega):
    """setk followed by qbatch (the factorised two-step form, Eq. 71 then Eq. 70)."""
    return qbatch(setk(gW, Re, deg_e, k, Uk), Rp, deg_p, q, Ukq, ev, omega)


# ---- linewidths from |g|^2 (Eq. 29 + Eq. 61) -------------------------------
def _dbl(name, nargs):
    f = getattr(_load(), name)
    f.restype = ctypes.c_double
    f.argtypes = [ctypes.c_double] * nargs
    return f


def fermi(eps, mu, kT):
    return float(_dbl("oracle_fermi", 3)(eps, mu, kT))


def bose(omega, kT):
    return float(_dbl("oracle_bose", 2)(omega, kT))


def delta_gauss(x, sigma):
    """Eq. 61: exp(-x^2/sigma^2)/(sqrt(pi) sigma)."""
    return float(_dbl("oracle_delta_gauss", 2)(x, sigma))


def rate_weight(eps_kb, eps_kqb, omega, kT, mu, sigma):
    """The square bracket of Eq. 29 for one (b, b', nu) term."""
    return float(_dbl("oracle_rate_weight", 6)(eps_kb, eps_kqb, omega, kT, mu, sigma))


def rates(out, eps_k, eps_kq, omega, kT, mu, sigma, pref, rate=None):
    """rate[b1] (+)= pref * sum_{q,b2,nu} out[q][b1][b2][nu] * W   (Eq. 29 with the Gaussian delta of Eq. 61)."""
    nq, nb1, nb2, nm = out.shape
    out = _c(out, np.float64); eps_k = _c(eps_k, np.float64, (nb1,)); eps_kq = _c(eps_kq, np.float64, (nq, nb2))
    omega = _c(omega, np.float64, (nq, nm))
    rate = np.zeros(nb1) if rate is None else rate
    assert rate.dtype == np.float64 and rate.shape == (nb1,) and rate.flags.c_contiguous
    f = _load().oracle_rates
    f.argtypes = [ctypes.c_int] * 4 + [ctypes.c_void_p] * 4 + [ctypes.c_double] * 4 + [ctypes.c_void_p]
    rc = f(nq, nb1, nb2, nm, _p(out), _p(eps_k), _p(eps_kq), _p(omega), kT, mu, sigma, pref, _p(rate))
    assert rc == 0
    return rate


# ---- polar long-range term (Eq. 14-15) ---------------------------------------------------------------
def polar_amplitude(q, ev, recip, G, Zstar, eps_inf, coeff):
    """P[nq][nm] = i coeff sum_G (Q.Zeff_nu)/(Q.eps_inf.Q): the (q, nu)-only factor of Eq. 15 (readings R20-R24)."""
    nq, nm, _ = ev.shape
    q = _c(q, np.float64, (nq, 3)); ev = _c(ev, np.complex128, (nq, nm, nm))
    recip = _c(recip, np.float64, (3, 3)); G = _c(G, np.float64).reshape(-1, 3)
    Zstar = _c(Zstar, np.float64, (nm // 3, 3, 3)); eps_inf = _c(eps_inf, np.float64, (3, 3))
    P = np.empty((nq, nm), dtype=np.complex128)
    f = _load().oracle_polar_amplitude
    f.argtypes = [ctypes.c_int] * 3 + [ctypes.c_void_p] * 6 + [ctypes.c_double, ctypes.c_void_p]
    rc = f(nq, nm, len(G), _p(q), _p(ev), _p(recip), _p(G), _p(Zstar), _p(eps_inf), float(coeff), _p(P))
    assert rc == 0
    return P


def qbatch_polar(g1, Rp, deg_p, q, Ukq, ev, omega, Uk, P):
    """qbatch with the long-range amplitude P[q][nu] [U_kq^dagger U_k]_{b2 b1} added before |.|^2 (Eq. 14)."""
    nRp, nb1, nw, nm = g1.shape
    nq, _, nb2 = Ukq.shape
    g1 = _c(g1, np.complex128); Rp = _c(Rp, np.float64, (nRp, 3))
    deg_p = None if deg_p is None else _c(deg_p, np.float64, (nRp,))
    q = _c(q, np.float64, (nq, 3)); Ukq = _c(Ukq, np.complex128, (nq, nw, nb2))
    ev = _c(ev, np.complex128, (nq, nm, nm)); omega = _c(omega, np.float64, (nq, nm))
    Uk = _c(Uk, np.complex128, (nw, nb1)); P = _c(P, np.complex128, (nq, nm))
    out = np.empty((nq, nb1, nb2, nm), dtype=np.float64)
    rc = _load().oracle_qbatch_polar(nRp, nw, nm, nb1, nb2, nq, _p(g1), _p(Rp), _p(deg_p), _p(q), _p(Ukq), _p(ev),
                                     _p(omega), _p(Uk), _p(P), _p(out))
    assert rc == 0
    return out


# ---- three-phonon coupling (Eq. 5), the second workload with the Eq. 70 shape ----------------------
def v3sq(V3, R, R2, q, z, q1, z1, z2):
    """|bare three-phonon contraction|^2 of Eq. 5 (readings R25-R27): out[nq][n0][n1][nm].
    V3 [nR2][nR][nm][nm][nm]; z [nm][n0] at q; z1 [nq][nm][n1] at q'; z2 [nq][nm][nm] at q''."""
    nR2, nR, nm = V3.shape[:3]
    n0 = z.shape[1]
    nq, _, n1 = z1.shape
    V3 = _c(V3, np.complex128, (nR2, nR, nm, nm, nm)); R = _c(R, np.float64, (nR, 3)); R2 = _c(R2, np.float64, (nR2, 3))
    q = _c(q, np.float64, (3,)); z = _c(z, np.complex128, (nm, n0)); q1 = _c(q1, np.float64, (nq, 3))
    z1 = _c(z1, np.complex128, (nq, nm, n1)); z2 = _c(z2, np.complex128, (nq, nm, nm))
    out = np.empty((nq, n0, n1, nm), dtype=np.float64)
    rc = _load().oracle_v3sq(nR, nR2, nm, n0, n1, nq, _p(V3), _p(R), _p(R2), _p(q), _p(z), _p(q1), _p(z1), _p(z2), _p(out))
    assert rc == 0
    return out
