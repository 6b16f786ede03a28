"""Pins for the CPU oracle: the oracle is checked
against what the paper's equations and the mathematics fix -- closed forms,
invariants, brute force, a library routine -- never against itself alone and
never against the CUDA path.  CPU only.
"""
import os

import numpy as np
import pytest

import oracle
from oracle import oracle_einsum
from paper_2111_14999_b200 import workloads as wl

HERE = os.path.dirname(os.path.abspath(__file__))


def _inputs(w, ik=0, nq=None):
    gW = wl.gW_full(w)
    Re, Rp = wl.Re_vectors(w), wl.Rp_vectors(w)
    k = wl.k_points(w)[ik]
    Uk = wl.U_k(w, ik)
    q, Ukq, ev, om = wl.q_inputs(w, ik)
    if nq is not None:
        q, Ukq, ev, om = q[:nq], Ukq[:nq], ev[:nq], om[:nq]
    return dict(gW=gW, Re=Re, Rp=Rp, deg_e=None, deg_p=None, k=k, Uk=Uk, q=q, Ukq=Ukq, ev=ev, omega=om)


def _relerr(a, b):
    return np.max(np.abs(a - b)) / np.max(np.abs(b))


SMALL = [
    wl.custom(nw=2, nm=3, grid_e=(3, 3, 3), nq=5, cfg_id=50),
    wl.custom(nw=3, nb1=2, nb2=1, nm=2, grid_e=(2, 1, 1), grid_p=(1, 3, 2), nq=4, cfg_id=51),
    wl.custom(nw=4, nb1=3, nb2=2, nm=3, grid_e=(1, 2, 3), grid_p=(2, 2, 1), nq=3, cfg_id=52),
    wl.custom(nw=1, nm=1, grid_e=(1, 1, 1), grid_p=(1, 1, 1), nq=2, cfg_id=53),
]


# ---- P1: direct double sum == factorised two-step form ----------------------
@pytest.mark.parametrize("w", SMALL, ids=lambda w: f"cfg{w.cfg_id}")
def test_P1_direct_equals_factorised(w):
    a = _inputs(w)
    rng = np.random.default_rng(w.cfg_id)
    a["deg_e"] = rng.integers(1, 4, w.nRe).astype(np.float64)
    a["deg_p"] = rng.integers(1, 4, w.nRp).astype(np.float64)
    ref = oracle.direct(**a)
    got = oracle.elph(**a)
    assert ref.shape == (w.nq, w.nb1, w.nb2, w.nm)
    assert _relerr(got, ref) < 1e-13


def test_P1_tiny_config_first_q():
    w = wl.CONFIGS["tiny"]
    a = _inputs(w, nq=3)
    assert _relerr(oracle.elph(**a), oracle.direct(**a)) < 1e-13


# ---- P2: periodicity, Eq. 87 --------------------------------
def test_P2_q_plus_G_invariance():
    w = wl.custom(nw=3, nb1=2, nb2=3, nm=3, grid_e=(3, 3, 3), nq=6, cfg_id=54)
    a = _inputs(w)
    ref = oracle.elph(**a)
    for G in [(1, 0, 0), (0, -2, 0), (0, 0, 2), (-1, 2, -2)]:
        b = dict(a)
        b["q"] = a["q"] + np.array(G, dtype=np.float64)
        assert _relerr(oracle.elph(**b), ref) < 1e-12
        c = dict(a)
        c["k"] = a["k"] + np.array(G, dtype=np.float64)
        assert _relerr(oracle.elph(**c), ref) < 1e-12
    # a half-integer shift is NOT a symmetry (guards against a missing factor 2 in 2*pi)
    b = dict(a)
    b["q"] = a["q"] + np.array([0.5, 0, 0])
    assert _relerr(oracle.elph(**b), ref) > 1e-3


# ---- P3: Frobenius-norm identity under unitary rotations --------------------
def test_P3_frobenius_identity():
    w = wl.custom(nw=4, nm=6, grid_e=(3, 2, 3), grid_p=(2, 3, 3), nq=5, cfg_id=55)
    a = _inputs(w)
    out = oracle.elph(**a)
    lhs = np.einsum("qabn,qn->q", out, 2.0 * a["omega"])
    # right side: no rotations at all, plain numpy Fourier sums
    phe = np.exp(2j * np.pi * (a["Re"] @ a["k"]))
    php = np.exp(2j * np.pi * (a["q"] @ a["Rp"].T))
    F = np.einsum("e,qp,peabk->qabk", phe, php, a["gW"])
    rhs = np.sum(np.abs(F) ** 2, axis=(1, 2, 3))
    assert np.max(np.abs(lhs - rhs) / rhs) < 1e-12


# ---- P4: closed forms with one lattice vector at the origin -----------------
def test_P4_identity_rotations():
    w = wl.custom(nw=3, nm=2, grid_e=(1, 1, 1), nq=3, cfg_id=56)
    a = _inputs(w)
    a["Uk"] = np.eye(3, dtype=np.complex128)
    a["Ukq"] = np.broadcast_to(np.eye(3, dtype=np.complex128), (3, 3, 3)).copy()
    a["ev"] = np.broadcast_to(np.eye(2, dtype=np.complex128), (3, 2, 2)).copy()
    out = oracle.elph(**a)
    g = a["gW"][0, 0]                                   # [w1][w2][kappa]
    expect = np.abs(g)[None] ** 2 / (2.0 * a["omega"][:, None, None, :])
    assert _relerr(out, expect) < 1e-14


def test_P4_rank_one_separates_conjugations():
    nw, nm, nq = 4, 3, 4
    w = wl.custom(nw=nw, nb1=3, nb2=2, nm=nm, grid_e=(1, 1, 1), nq=nq, cfg_id=57)
    a = _inputs(w)
    rng = np.random.default_rng(7)
    va = rng.standard_normal(nw) + 1j * rng.standard_normal(nw)
    vb = rng.standard_normal(nw) + 1j * rng.standard_normal(nw)
    vc = rng.standard_normal(nm) + 1j * rng.standard_normal(nm)
    a["gW"] = np.einsum("a,b,c->abc", va, vb, vc)[None, None].copy()
    out = oracle.elph(**a)
    f1 = np.abs(a["Uk"].T @ va) ** 2                                  # plain U_k on w1
    f2 = np.abs(np.einsum("qwb,w->qb", np.conj(a["Ukq"]), vb)) ** 2   # conj(U_kq) on w2
    f3 = np.abs(np.einsum("qkn,k->qn", a["ev"], vc)) ** 2             # plain ev on kappa
    expect = f1[None, :, None, None] * f2[:, None, :, None] * f3[:, None, None, :] / (2 * a["omega"][:, None, None, :])
    assert _relerr(out, expect) < 1e-13
    # with the wrong conjugation on U_kq the value differs (the pin has teeth)
    f2_wrong = np.abs(np.einsum("qwb,w->qb", a["Ukq"], vb)) ** 2
    wrong = f1[None, :, None, None] * f2_wrong[:, None, :, None] * f3[:, None, None, :] / (2 * a["omega"][:, None, None, :])
    assert _relerr(wrong, expect) > 1e-3


def test_P4_which_wannier_index_is_the_ket():
    """R5: first Wannier index of g_W pairs with U_k (b1), second with U_kq (b2)."""
    nw, nm = 3, 1
    w = wl.custom(nw=nw, nb1=nw, nb2=nw, nm=nm, grid_e=(1, 1, 1), nq=1, cfg_id=58)
    a = _inputs(w)
    g = np.zeros((1, 1, nw, nw, nm), dtype=np.complex128)
    g[0, 0, 0, 2, 0] = 2.0            # only w1=0, w2=2
    a["gW"] = g
    a["Uk"] = np.eye(nw, dtype=np.complex128)
    a["Ukq"] = np.eye(nw, dtype=np.complex128)[None].copy()
    a["ev"] = np.ones((1, 1, 1), dtype=np.complex128)
    a["omega"] = np.full((1, 1), 0.5)
    out = oracle.elph(**a)
    expect = np.zeros((1, nw, nw, 1))
    expect[0, 0, 2, 0] = 4.0
    assert np.array_equal(out, expect)


# ---- golden closed forms (hand-computed, tests/golden/closed_forms.txt) ------
def _golden_rows():
    rows = []
    with open(os.path.join(HERE, "golden", "closed_forms.txt")) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append(line.split())
    return rows


@pytest.mark.parametrize("row", _golden_rows(), ids=lambda r: r[0])
def test_golden_closed_forms(row):
    name, g0r, g0i, g1r, g1i, which = row[:6]
    R0 = np.array([float(x) for x in row[6:9]])
    k = np.array([float(x) for x in row[9:12]])
    q = np.array([float(x) for x in row[12:15]])
    om, expect = float(row[15]), float(row[16])
    A, B = complex(float(g0r), float(g0i)), complex(float(g1r), float(g1i))
    two = np.stack([np.zeros(3), R0])
    one = np.zeros((1, 3))
    if which == "Rp":
        Rp, Re = two, one
        gW = np.array([A, B], dtype=np.complex128).reshape(2, 1, 1, 1, 1)
    else:
        Rp, Re = one, two
        gW = np.array([A, B], dtype=np.complex128).reshape(1, 2, 1, 1, 1)
    I1 = np.ones((1, 1), dtype=np.complex128)
    args = dict(gW=gW, Re=Re, Rp=Rp, deg_e=None, deg_p=None, k=k, Uk=I1, q=q[None], Ukq=I1[None],
                ev=I1[None], omega=np.array([[om]]))
    for fn in (oracle.direct, oracle.elph, oracle_einsum.elph_einsum):
        got = float(fn(**args)[0, 0, 0, 0])
        assert abs(got - expect) < 1e-12 * max(1.0, expect), (name, fn.__name__, got, expect)


# ---- P5: single lattice-vector support --------------------------------------
def test_P5_single_vector_support_and_degeneracies():
    w = wl.custom(nw=2, nm=2, grid_e=(3, 1, 2), grid_p=(2, 2, 1), nq=4, cfg_id=59)
    a = _inputs(w)
    e0, p0 = 4, 2
    g = np.zeros_like(a["gW"])
    g[p0, e0] = a["gW"][p0, e0]
    a["gW"] = g
    # same rotations at every q so only the phases could make out depend on q
    for key in ("Ukq", "ev", "omega"):
        a[key] = np.broadcast_to(a[key][0], a[key].shape).copy()
    de = np.ones(w.nRe); de[e0] = 2.0
    dp = np.ones(w.nRp); dp[p0] = 3.0
    a["deg_e"], a["deg_p"] = de, dp
    out = oracle.elph(**a)
    assert _relerr(out[1:], np.broadcast_to(out[0], out[1:].shape)) < 1e-13     # independent of q
    b = dict(a); b["k"] = a["k"] + np.array([0.123, -0.4, 0.77])
    assert _relerr(oracle.elph(**b), out) < 1e-13                                # independent of k
    # equals the one-vector closed form divided by (deg_e*deg_p)^2
    G = np.einsum("ab,cd,kn,ack->bdn", a["Uk"], np.conj(a["Ukq"][0]), a["ev"][0], g[p0, e0])
    expect = np.abs(G) ** 2 / (2 * a["omega"][0][None, None, :]) / (2.0 * 3.0) ** 2
    assert _relerr(out[0], expect) < 1e-13


# ---- P6: two-vector interference fixes the SIGN of the phase -----------------
def test_P6_phase_sign():
    nw, nm, nq = 2, 2, 6
    w = wl.custom(nw=nw, nm=nm, grid_e=(1, 1, 1), grid_p=(1, 1, 1), nq=nq, cfg_id=60)
    a = _inputs(w)
    A = a["gW"][0, 0]
    R0 = np.array([1.0, -2.0, 1.0])
    base = oracle.elph(**a)                                    # out_A
    # phonon side
    b = dict(a)
    b["Rp"] = np.stack([np.zeros(3), R0])
    b["gW"] = np.stack([A, 1j * A])[:, None].copy()            # [2][1][...]
    got = oracle.elph(**b)
    fac = 2.0 - 2.0 * np.sin(2 * np.pi * (a["q"] @ R0))
    assert _relerr(got, base * fac[:, None, None, None]) < 1e-12
    # electron side
    c = dict(a)
    c["Re"] = np.stack([np.zeros(3), R0])
    c["gW"] = np.stack([A, 1j * A])[None].copy()               # [1][2][...]
    got = oracle.elph(**c)
    fac = 2.0 - 2.0 * np.sin(2 * np.pi * (a["k"] @ R0))
    assert _relerr(got, base * fac) < 1e-12


# ---- P7: scaling --------------------------------------------------------------
def test_P7_scaling():
    a = _inputs(SMALL[1])
    ref = oracle.elph(**a)
    c = 0.3 - 1.7j
    b = dict(a); b["gW"] = a["gW"] * c
    assert _relerr(oracle.elph(**b), ref * abs(c) ** 2) < 1e-13
    b = dict(a); b["omega"] = a["omega"] * 3.5
    assert _relerr(oracle.elph(**b), ref / 3.5) < 1e-13


def test_R7_nonpositive_omega_gives_zero():
    a = _inputs(SMALL[0])
    om = a["omega"].copy(); om[1, 2] = 0.0; om[2, 0] = -0.01
    a["omega"] = om
    for fn in (oracle.elph, oracle.direct, oracle_einsum.elph_einsum):
        out = fn(**a)
        assert np.all(out[1, :, :, 2] == 0.0) and np.all(out[2, :, :, 0] == 0.0)
        assert np.all(np.isfinite(out)) and np.all(out[0] > 0)


# ---- P8: gauge freedom ---------------------------------------------------------
def test_P8_gauge():
    w = wl.custom(nw=3, nm=3, grid_e=(2, 2, 1), nq=3, cfg_id=61)
    a = _inputs(w)
    ref = oracle.elph(**a)
    b = dict(a)
    b["Uk"] = a["Uk"] * np.exp(1j * np.array([0.3, -1.1, 2.0]))[None, :]
    b["Ukq"] = a["Ukq"] * np.exp(1j * np.array([1.3, 0.1, -2.0]))[None, None, :]
    b["ev"] = a["ev"] * np.exp(1j * np.array([-0.7, 0.9, 0.2]))[None, None, :]
    assert _relerr(oracle.elph(**b), ref) < 1e-13
    # mixing two degenerate columns by a 2x2 unitary keeps the SUM of the two slices
    th = 0.6
    M = np.array([[np.cos(th), -np.sin(th) * np.exp(0.4j)], [np.sin(th) * np.exp(-0.4j), np.cos(th)]])
    c = dict(a)
    Uk2 = a["Uk"].copy(); Uk2[:, :2] = a["Uk"][:, :2] @ M
    c["Uk"] = Uk2
    got = oracle.elph(**c)
    assert _relerr(got[:, 0] + got[:, 1], ref[:, 0] + ref[:, 1]) < 1e-13
    assert _relerr(got[:, 2], ref[:, 2]) < 1e-13


# ---- P9: rectangular U (band windows) -----------------------------------------
def test_P9_rectangular_consistency():
    w = wl.custom(nw=4, nm=3, grid_e=(2, 2, 2), nq=3, cfg_id=62)
    a = _inputs(w)
    full = oracle.elph(**a)
    S1, S2 = [0, 2], [3, 1, 2]
    b = dict(a)
    b["Uk"] = np.ascontiguousarray(a["Uk"][:, S1])
    b["Ukq"] = np.ascontiguousarray(a["Ukq"][:, :, S2])
    assert _relerr(oracle.elph(**b), full[:, S1][:, :, S2]) < 1e-14


# ---- P10: ordering of the lattice-vector lists ---------------------------------
def test_P10_permutation_of_R_lists():
    w = wl.custom(nw=2, nm=3, grid_e=(3, 2, 2), grid_p=(2, 3, 2), nq=3, cfg_id=63)
    a = _inputs(w)
    ref = oracle.elph(**a)
    rng = np.random.default_rng(3)
    pe, pp = rng.permutation(w.nRe), rng.permutation(w.nRp)
    b = dict(a)
    b["Re"], b["Rp"] = a["Re"][pe], a["Rp"][pp]
    b["gW"] = np.ascontiguousarray(a["gW"][pp][:, pe])
    assert _relerr(oracle.elph(**b), ref) < 1e-13


# ---- P11: NumPy einsum twin ------------------------------------------------------
def test_P11_einsum_twin_tiny():
    w = wl.CONFIGS["tiny"]
    a = _inputs(w)
    assert _relerr(oracle.elph(**a), oracle_einsum.elph_einsum(**a)) < 1e-13


def test_P11_einsum_twin_rectangular_with_degeneracies():
    w = SMALL[2]
    a = _inputs(w)
    rng = np.random.default_rng(11)
    a["deg_e"] = rng.integers(1, 5, w.nRe).astype(np.float64)
    a["deg_p"] = rng.integers(1, 5, w.nRp).astype(np.float64)
    e = oracle_einsum.elph_einsum(**a)
    assert _relerr(oracle.elph(**a), e) < 1e-13
    assert _relerr(oracle.direct(**a), e) < 1e-13


def test_P11_einsum_twin_si_like_64q():
    """Si-like shapes (nw=8, nm=6, 343x343 lattice vectors), first 64 q."""
    w = wl.CONFIGS["si-like"]
    a = _inputs(w, nq=64)
    got = oracle.elph(**a)
    # the twin, done in two library contractions to keep memory small
    phe = oracle_einsum.phases(a["k"], a["Re"], None)
    T = np.tensordot(phe, a["gW"], axes=([0], [1]))                 # [p][w1][w2][ka]
    php = oracle_einsum.phases(a["q"], a["Rp"], None)               # [q][p]
    F = np.tensordot(php, T, axes=([1], [0]))                       # [q][w1][w2][ka]
    G = np.einsum("ab,qcd,qkn,qack->qbdn", a["Uk"], np.conj(a["Ukq"]), a["ev"], F, optimize=True)
    expect = np.abs(G) ** 2 / (2 * a["omega"][:, None, None, :])
    assert _relerr(got, expect) < 1e-12


# ---- P12: Gamma point ---------------------------------------------------------------
def test_P12_zero_wavevectors_are_plain_sums():
    w = wl.custom(nw=2, nm=2, grid_e=(3, 3, 1), grid_p=(1, 2, 3), nq=2, cfg_id=64)
    a = _inputs(w)
    a["k"] = np.zeros(3)
    a["q"] = np.zeros((2, 3))
    out = oracle.elph(**a)
    S = a["gW"].sum(axis=(0, 1))
    G = np.einsum("ab,qcd,qkn,ack->qbdn", a["Uk"], np.conj(a["Ukq"]), a["ev"], S)
    assert _relerr(out, np.abs(G) ** 2 / (2 * a["omega"][:, None, None, :])) < 1e-13


def test_setk_slab_matches_setk():
    w = SMALL[2]
    a = _inputs(w)
    g1 = oracle.setk(a["gW"], a["Re"], None, a["k"], a["Uk"])
    for p in range(w.nRp):
        assert np.array_equal(oracle.setk_slab(a["gW"][p], a["Re"], None, a["k"], a["Uk"]), g1[p])
