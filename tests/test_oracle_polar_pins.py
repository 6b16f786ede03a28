"""Pins of the polar (long-range) oracle: PAPER.md Eq. 14-15 (L139-L147) in the readings R20-R24
(DESIGN.md).  None of them retypes the oracle's loops:

  PP1  coeff = 0 or Z* = 0: qbatch_polar == qbatch (Eq. 14 with g^L = 0).
  PP2  hand-computed closed forms (tests/golden/polar_closed_forms.txt: isotropic eps_inf and Z*, ev = identity, one G).
  PP3  the overlap factor is [U_kq^dagger U_k]_{b2 b1}: identity for U_kq = U_k (orthonormal columns), a pure phase
       for a re-phased U_kq, and equal to a NumPy matmul for general rectangular U (pins conj and index order).
  PP4  interference with the short-range amplitude: pins the factor i of Eq. 15 and its sign (golden polar_out_c).
  PP5  q -> q + G0 with the G list shifted by -G0 leaves P unchanged (the sum is over q + G only).
  PP6  the G = -q term is skipped, and only that one.
  PP7  anisotropic eps_inf / Z*, several atoms, complex ev: equals a NumPy einsum evaluation.
  PP8  scalings: P is linear in coeff and Z*, inversely linear in eps_inf, and of degree -1 in the reciprocal lattice.
"""
import os

import numpy as np
import pytest

import oracle
from paper_2111_14999_b200 import workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "polar_closed_forms.txt")


def _golden(name):
    for line in open(GOLDEN):
        f = line.split()
        if f and f[0] == name:
            return np.array([float(x) for x in f[1:]])
    raise KeyError(name)


ISO = dict(recip=np.eye(3), G=np.zeros((1, 3)), Zstar=2.0 * np.eye(3)[None], eps_inf=4.0 * np.eye(3), coeff=0.5)


def _grid(h):
    r = np.arange(-h, h + 1)
    return np.array([[a, b, c] for a in r for b in r for c in r], dtype=np.float64)


def _rand_setup(seed, nat=2, nq=5):
    rng = np.random.default_rng(seed)
    nm = 3 * nat
    q = rng.random((nq, 3))
    ev = wl.haar_unitary(rng, nm, nq)
    recip = rng.normal(size=(3, 3)) + 2.0 * np.eye(3)
    Z = rng.normal(size=(nat, 3, 3))
    A = rng.normal(size=(3, 3))
    eps = A @ A.T + 3.0 * np.eye(3)
    return q, ev, recip, Z, eps


@pytest.mark.parametrize("name", ["polar_P_a", "polar_P_b"])
def test_PP2_closed_forms(name):
    g = _golden(name)
    q, want = g[:3], g[3::2] + 1j * g[4::2]
    P = oracle.polar_amplitude(q[None], np.eye(3, dtype=complex)[None], **ISO)
    assert np.allclose(P[0], want, rtol=1e-15, atol=1e-16)


def _tiny_problem(seed, nw=3, nb1=2, nb2=2, nm=3, nq=4):
    w = wl.custom(nw=nw, nb1=nb1, nb2=nb2, nm=nm, grid_e=(2, 1, 1), grid_p=(2, 2, 1), nq=nq, cfg_id=40 + seed)
    g1 = oracle.setk(wl.gW_full(w), wl.Re_vectors(w), None, wl.k_points(w)[0], wl.U_k(w))
    q, Ukq, ev, om = wl.q_inputs(w)
    return w, g1, wl.Rp_vectors(w), wl.U_k(w), q, Ukq, ev, om


def test_PP1_vanishing_polar_term_gives_back_qbatch():
    w, g1, Rp, Uk, q, Ukq, ev, om = _tiny_problem(1)
    ref = oracle.qbatch(g1, Rp, None, q, Ukq, ev, om)
    _, _, recip, Z, eps = _rand_setup(2, nat=1)
    P0 = oracle.polar_amplitude(q, ev, recip, _grid(1), Z, eps, 0.0)
    assert np.all(P0 == 0)
    assert np.allclose(oracle.qbatch_polar(g1, Rp, None, q, Ukq, ev, om, Uk, P0), ref, rtol=1e-13, atol=0)
    Pz = oracle.polar_amplitude(q, ev, recip, _grid(1), 0.0 * Z, eps, 1.3)
    assert np.all(Pz == 0)


def test_PP3_overlap_is_Ukq_dagger_Uk():
    w, g1, Rp, Uk, q, Ukq, ev, om = _tiny_problem(2, nw=4, nb1=3, nb2=2, nq=3)
    g0 = np.zeros_like(g1)
    P = np.random.default_rng(0).normal(size=(3, 3)) + 1j * np.random.default_rng(1).normal(size=(3, 3))
    out = oracle.qbatch_polar(g0, Rp, None, q, Ukq, ev, om, Uk, P)
    O = np.einsum("qwb,wa->qab", Ukq.conj(), Uk)                       # [q][b1][b2] via a library contraction
    want = (np.abs(P)[:, None, None, :] * np.abs(O)[..., None]) ** 2 / (2 * om[:, None, None, :])
    assert np.allclose(out, want, rtol=1e-13, atol=0)
    # U_kq = U_k (same orthonormal columns): the overlap is the identity -> only b1 == b2 survives
    Uk3 = wl.haar_unitary(np.random.default_rng(3), 4)[:, :3]
    same = np.broadcast_to(Uk3, (3, 4, 3)).copy()
    out = oracle.qbatch_polar(np.zeros((g1.shape[0], 3, 4, 3), complex), Rp, None, q, same, ev, om, Uk3, P)
    diag = np.abs(P) ** 2 / (2 * om)
    for b1 in range(3):
        for b2 in range(3):
            assert np.allclose(out[:, b1, b2, :], diag if b1 == b2 else 0.0, rtol=1e-13, atol=1e-28)
    # re-phasing the columns of U_kq changes the overlap by a phase only
    ph = np.exp(1j * np.array([0.3, -1.1, 2.0]))
    out2 = oracle.qbatch_polar(np.zeros((g1.shape[0], 3, 4, 3), complex), Rp, None, q, same * ph, ev, om, Uk3, P)
    assert np.allclose(out2, out, rtol=1e-13, atol=1e-28)


def test_PP4_interference_pins_the_factor_i_and_its_sign():
    want = _golden("polar_out_c")
    gW = np.array([1.0, 2.0j, 0.0]).reshape(1, 1, 1, 1, 3)
    one = np.ones((1, 1), complex)
    g1 = oracle.setk(gW, np.zeros((1, 3)), None, np.array([0.2, 0.1, 0.7]), one)
    q = np.array([[0.3, 0.4, 0.0]])
    ev = np.eye(3, dtype=complex)[None]
    P = oracle.polar_amplitude(q, ev, **ISO)
    out = oracle.qbatch_polar(g1, np.zeros((1, 3)), None, q, one[None], ev, np.full((1, 3), 0.5), one, P)
    assert np.allclose(out[0, 0, 0], want, rtol=1e-14, atol=1e-16)


def test_PP5_shift_of_q_and_G_list():
    q, ev, recip, Z, eps = _rand_setup(5)
    G = _grid(2)
    G0 = np.array([1.0, -2.0, 1.0])
    a = oracle.polar_amplitude(q, ev, recip, G, Z, eps, 0.7)
    b = oracle.polar_amplitude(q + G0, ev, recip, G - G0, Z, eps, 0.7)
    assert np.allclose(a, b, rtol=1e-12, atol=0)


def test_PP6_only_the_G_equal_minus_q_term_is_skipped():
    _, ev, recip, Z, eps = _rand_setup(6, nq=2)
    G = _grid(1)
    q = np.array([[0.0, 0.0, 0.0], [1.0, 0.0, -1.0]])                  # q + G = 0 for G = 0 and for G = (-1, 0, 1)
    a = oracle.polar_amplitude(q, ev, recip, G, Z, eps, 1.0)
    assert np.all(np.isfinite(a.view(float)))
    for i, drop in enumerate(([0.0, 0.0, 0.0], [-1.0, 0.0, 1.0])):
        keep = G[~np.all(G == np.array(drop), axis=1)]
        assert len(keep) == len(G) - 1
        b = oracle.polar_amplitude(q[i:i + 1], ev[i:i + 1], recip, keep, Z, eps, 1.0)
        assert np.allclose(a[i], b[0], rtol=1e-14, atol=0)
    # a tiny but non-zero q is NOT skipped: the G = 0 term dominates like 1/|q|
    tiny = oracle.polar_amplitude(np.array([[1e-6, 0.0, 0.0]]), ev[:1], recip, G, Z, eps, 1.0)
    assert np.max(np.abs(tiny)) > 1e3 * np.max(np.abs(a[0]))


def test_PP7_numpy_einsum_twin():
    q, ev, recip, Z, eps = _rand_setup(7, nat=3, nq=6)
    G = _grid(2)
    got = oracle.polar_amplitude(q, ev, recip, G, Z, eps, 0.31)
    nat = 3
    Q = (q[:, None, :] + G[None, :, :]) @ recip                        # [q][G][3] Cartesian
    den = np.einsum("qga,ab,qgb->qg", Q, eps, Q)
    V = np.einsum("qga,qg->qa", Q, 1.0 / den)                           # the q-only real vector sum_G Q / (Q eps Q)
    zeff = np.einsum("sab,qsbn->qan", Z, ev.reshape(6, nat, 3, 3 * nat))
    want = 1j * 0.31 * np.einsum("qa,qan->qn", V, zeff)
    assert np.allclose(got, want, rtol=1e-12, atol=0)


def test_PP8_scalings():
    q, ev, recip, Z, eps = _rand_setup(8)
    G = _grid(1)
    base = oracle.polar_amplitude(q, ev, recip, G, Z, eps, 0.5)
    assert np.allclose(oracle.polar_amplitude(q, ev, recip, G, Z, eps, 1.5), 3 * base, rtol=1e-14)
    assert np.allclose(oracle.polar_amplitude(q, ev, recip, G, -2 * Z, eps, 0.5), -2 * base, rtol=1e-14)
    assert np.allclose(oracle.polar_amplitude(q, ev, recip, G, Z, 4 * eps, 0.5), base / 4, rtol=1e-14)
    assert np.allclose(oracle.polar_amplitude(q, ev, 2 * recip, G, Z, eps, 0.5), base / 2, rtol=1e-14)
    # Z* acts with its ROW index on the wavevector (R24): transposing a non-symmetric Z* changes P
    assert not np.allclose(oracle.polar_amplitude(q, ev, recip, G, Z.transpose(0, 2, 1), eps, 0.5), base, rtol=1e-3)
