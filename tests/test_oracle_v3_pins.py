"""Pins of the three-phonon oracle (Eq. 5 L82 in the readings R25-R27 of DESIGN.md):

  VP1  closed forms with one lattice vector at the origin: identity eigenvectors give |V3[a][b][c]|^2; a rank-1 tensor
       x (x) y (x) w gives |z^dagger x|^2 |z1^dagger y|^2 |z2^dagger w|^2 -- all three eigenvectors CONJUGATED (complex
       x, y, w make conj vs plain visible).
  VP2  the phases carry a MINUS sign: a tensor A at R = 0 and iA at R0 gives |A|^2 (2 + 2 sin(2 pi q.R0)) (Eq. 13's plus
       sign would give 2 - 2 sin); same for R' with q'.
  VP3  equals a NumPy einsum of Eq. 5.
  VP4  q -> q + G, q' -> q' + G' for integer G leave it unchanged (integer lattice vectors).
"""
import numpy as np

import oracle
from paper_2111_14999_b200 import workloads as wl


def _rand(seed, nm=3, nR=4, nR2=3, nq=3, n0=2, n1=3):
    rng = np.random.default_rng(seed)
    V3 = rng.normal(size=(nR2, nR, nm, nm, nm)) + 1j * rng.normal(size=(nR2, nR, nm, nm, nm))
    R = rng.integers(-2, 3, size=(nR, 3)).astype(float); R2 = rng.integers(-2, 3, size=(nR2, 3)).astype(float)
    z = wl.haar_unitary(rng, nm)[:, :n0]
    z1 = wl.haar_unitary(rng, nm, nq)[:, :, :n1]
    z2 = wl.haar_unitary(rng, nm, nq)
    return V3, R, R2, rng.random(3), np.ascontiguousarray(z), rng.random((nq, 3)), np.ascontiguousarray(z1), z2


def test_VP1_closed_forms_at_the_origin():
    rng = np.random.default_rng(0)
    nm = 3
    V3 = rng.normal(size=(1, 1, nm, nm, nm)) + 1j * rng.normal(size=(1, 1, nm, nm, nm))
    O = np.zeros((1, 3)); I = np.eye(nm, dtype=complex)
    out = oracle.v3sq(V3, O, O, rng.random(3), I, rng.random((1, 3)), I[None], I[None])
    assert np.allclose(out[0], np.abs(V3[0, 0]) ** 2, rtol=1e-14, atol=0)
    x, y, w = [rng.normal(size=nm) + 1j * rng.normal(size=nm) for _ in range(3)]
    z = wl.haar_unitary(rng, nm); z1 = wl.haar_unitary(rng, nm); z2 = wl.haar_unitary(rng, nm)
    T = np.einsum("a,b,c->abc", x, y, w)[None, None]
    out = oracle.v3sq(T, O, O, rng.random(3), z, rng.random((1, 3)), z1[None], z2[None])
    want = np.einsum("n,m,l->nml", np.abs(z.conj().T @ x) ** 2, np.abs(z1.conj().T @ y) ** 2, np.abs(z2.conj().T @ w) ** 2)
    assert np.allclose(out[0], want, rtol=1e-13, atol=0)
    plain = np.einsum("n,m,l->nml", np.abs(z.T @ x) ** 2, np.abs(z1.T @ y) ** 2, np.abs(z2.T @ w) ** 2)
    assert not np.allclose(out[0], plain, rtol=1e-3)


def test_VP2_minus_sign_of_both_phases():
    A = 0.7 - 0.4j
    one = np.ones((1, 1), complex)
    R0 = np.array([1.0, 0.0, 2.0])
    q, q1 = np.array([0.13, 0.4, 0.21]), np.array([[0.3, 0.9, 0.05]])
    two, O = np.stack([np.zeros(3), R0]), np.zeros((1, 3))
    V_R = np.array([A, 1j * A]).reshape(1, 2, 1, 1, 1)          # two vectors R (paired with q)
    out = oracle.v3sq(V_R, two, O, q, one, q1, one[None], one[None])[0, 0, 0, 0]
    assert abs(out - abs(A) ** 2 * (2 + 2 * np.sin(2 * np.pi * q @ R0))) < 1e-14
    V_R2 = np.array([A, 1j * A]).reshape(2, 1, 1, 1, 1)         # two vectors R' (paired with q')
    out = oracle.v3sq(V_R2, O, two, q, one, q1, one[None], one[None])[0, 0, 0, 0]
    assert abs(out - abs(A) ** 2 * (2 + 2 * np.sin(2 * np.pi * q1[0] @ R0))) < 1e-14


def test_VP3_numpy_einsum_twin():
    V3, R, R2, q, z, q1, z1, z2 = _rand(3)
    got = oracle.v3sq(V3, R, R2, q, z, q1, z1, z2)
    ph = np.exp(-2j * np.pi * (R @ q))                           # [R]
    ph1 = np.exp(-2j * np.pi * (q1 @ R2.T))                      # [q][R']
    amp = np.einsum("r,qs,srabc,an,qbm,qcl->qnml", ph, ph1, V3, z.conj(), z1.conj(), z2.conj())
    assert np.allclose(got, np.abs(amp) ** 2, rtol=1e-12, atol=0)


def test_VP4_periodicity():
    V3, R, R2, q, z, q1, z1, z2 = _rand(4)
    base = oracle.v3sq(V3, R, R2, q, z, q1, z1, z2)
    assert np.allclose(oracle.v3sq(V3, R, R2, q + [1, -2, 0], z, q1 + [0, 3, -1], z1, z2), base, rtol=1e-11, atol=0)
