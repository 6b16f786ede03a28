"""Pins of the linewidth oracle (Eq. 29 L229 with the Gaussian delta of Eq. 61)
against what the paper and the mathematics fix -- none of them retypes the oracle's own formula:

  RP1  Eq. 61 is a nascent delta: it integrates to 1 and has second moment sigma^2/2 (exponent x^2/sigma^2,
       NOT x^2/(2 sigma^2)); its peak is 1/(sqrt(pi) sigma).
  RP2  f and n are the Fermi-Dirac / Bose-Einstein functions: f(mu) = 1/2, f(mu+x) + f(mu-x) = 1,
       n(w) (e^{w/kT} - 1) = 1, 1 + n(w) + n(-w) = 0.
  RP3  the paper's own symmetrisation (Eq. 30 -> Eq. 31): ON the energy shell of either delta the
       occupation bracket of Eq. 28/29 times sqrt(f(1-f) / (f'(1-f'))) equals 1/(2 sinh(omega / 2 kT)), the
       factor Eq. 31 prints (f = f_kb, f' = f_k'b').  Reading R19: Eq. 30 prints the square root the other way
       up; with the bracket exactly as Eq. 28 prints it, only this orientation reproduces Eq. 31 -- for BOTH
       deltas, whatever eps, omega, mu, T -- and any swap of the occupation factors or sign inside them breaks it.
       With sigma << omega a single-term rate isolates each bracket, so this pins which occupation factor goes
       with which delta and every sign inside them.
  RP4  zero-temperature limit: emission only into empty states, absorption only ... (step functions).
  RP5  linear in out and in pref, additive over q batches (accumulation), independent of q order.
  RP6  a vectorised NumPy evaluation (library exp, broadcasting) == the C loops.
"""
import numpy as np
import pytest

import oracle


def test_RP1_gaussian_delta_is_normalised_with_variance_sigma2_over_2():
    for sigma in (0.004, 0.012, 0.3):
        x = np.linspace(-12 * sigma, 12 * sigma, 48001)
        d = np.array([oracle.delta_gauss(v, sigma) for v in x])
        h = x[1] - x[0]
        assert abs(np.sum(d) * h - 1.0) < 1e-11
        assert abs(np.sum(d * x * x) * h - sigma ** 2 / 2) < 1e-11 * sigma ** 2
        assert abs(oracle.delta_gauss(0.0, sigma) * np.sqrt(np.pi) * sigma - 1.0) < 1e-15
        assert oracle.delta_gauss(0.3 * sigma, sigma) == oracle.delta_gauss(-0.3 * sigma, sigma)


def test_RP2_occupation_functions():
    kT, mu = 0.02585, 0.07
    assert oracle.fermi(mu, mu, kT) == 0.5
    for x in (0.001, 0.03, 0.4):
        assert abs(oracle.fermi(mu + x, mu, kT) + oracle.fermi(mu - x, mu, kT) - 1.0) < 1e-15
        assert abs(oracle.bose(x, kT) * np.expm1(x / kT) - 1.0) < 1e-13
        assert abs(1.0 + oracle.bose(x, kT) + oracle.bose(-x, kT)) < 1e-12 * (1 + oracle.bose(x, kT))
    assert oracle.fermi(mu + 2.0, mu, kT) < 1e-30 and oracle.fermi(mu - 2.0, mu, kT) == 1.0


@pytest.mark.parametrize("shell", [-1, +1], ids=["emission_eps2=eps-w", "absorption_eps2=eps+w"])
def test_RP3_symmetrised_bracket_equals_inverse_2sinh(shell):
    """Eq. 30-31: on shell, bracket * sqrt(f(1-f)/(f'(1-f'))) = 1 / (2 sinh(w / 2kT))."""
    kT, mu, sigma, pref = 0.02585, 0.013, 1e-4, 0.37
    rng = np.random.default_rng(5)
    for _ in range(20):
        eps = rng.uniform(-0.1, 0.1)
        om = rng.uniform(0.01, 0.06)            # >> sigma: the other delta is e^{-(2 om/sigma)^2} = 0
        eps2 = eps + shell * om
        out = np.array([[[[2.5]]]])
        rate = oracle.rates(out, np.array([eps]), np.array([[eps2]]), np.array([[om]]), kT, mu, sigma, pref)[0]
        bracket = rate * np.sqrt(np.pi) * sigma / (pref * 2.5)
        f = 1.0 / (np.exp((eps - mu) / kT) + 1.0)
        f2 = 1.0 / (np.exp((eps2 - mu) / kT) + 1.0)
        sym = bracket * np.sqrt(f * (1 - f) / (f2 * (1 - f2)))
        assert abs(sym * 2.0 * np.sinh(om / (2 * kT)) - 1.0) < 1e-12


def test_RP4_zero_temperature_limit():
    kT, mu, sigma = 1e-5, 0.0, 1e-3
    om = 0.03
    peak = 1.0 / (np.sqrt(np.pi) * sigma)
    # emission (eps2 = eps - om): allowed only if the final state is empty (eps2 > mu); n -> 0
    assert abs(oracle.rate_weight(0.05, 0.02, om, kT, mu, sigma) / peak - 1.0) < 1e-12
    assert oracle.rate_weight(0.01, -0.02, om, kT, mu, sigma) / peak < 1e-12
    # absorption-like term (eps2 = eps + om) carries f' + n: needs the state at eps2 occupied
    assert abs(oracle.rate_weight(-0.05, -0.02, om, kT, mu, sigma) / peak - 1.0) < 1e-12
    assert oracle.rate_weight(0.01, 0.04, om, kT, mu, sigma) / peak < 1e-12
    # R18: omega <= 0 contributes nothing
    assert oracle.rate_weight(0.0, 0.0, 0.0, 0.02, 0.0, 0.01) == 0.0
    assert oracle.rate_weight(0.0, 0.0, -0.01, 0.02, 0.0, 0.01) == 0.0


def _random_case(seed, nq=37, nb1=3, nb2=4, nm=5):
    rng = np.random.default_rng(seed)
    out = rng.random((nq, nb1, nb2, nm))
    eps_k = rng.uniform(-0.15, 0.15, nb1)
    eps_kq = rng.uniform(-0.15, 0.15, (nq, nb2))
    om = rng.uniform(0.005, 0.06, (nq, nm))
    return out, eps_k, eps_kq, om


def test_RP5_linearity_additivity_order():
    out, eps_k, eps_kq, om = _random_case(1)
    P = dict(kT=0.02585, mu=0.01, sigma=0.012)
    r = oracle.rates(out, eps_k, eps_kq, om, pref=0.3, **P)
    assert np.all(r > 0)
    assert np.allclose(oracle.rates(3.0 * out, eps_k, eps_kq, om, pref=0.3, **P), 3.0 * r, rtol=1e-14, atol=0)
    assert np.allclose(oracle.rates(out, eps_k, eps_kq, om, pref=0.6, **P), 2.0 * r, rtol=1e-14, atol=0)
    # accumulate two q batches into the same array == one batch
    acc = np.zeros(3)
    oracle.rates(out[:20], eps_k, eps_kq[:20], om[:20], pref=0.3, rate=acc, **P)
    oracle.rates(out[20:], eps_k, eps_kq[20:], om[20:], pref=0.3, rate=acc, **P)
    assert np.allclose(acc, r, rtol=1e-14, atol=0)
    perm = np.random.default_rng(2).permutation(len(out))
    assert np.allclose(oracle.rates(out[perm], eps_k, eps_kq[perm], om[perm], pref=0.3, **P), r, rtol=1e-14, atol=0)
    # a band b1 only sees its own slice of out
    out2 = out.copy(); out2[:, 1] = 0.0
    r2 = oracle.rates(out2, eps_k, eps_kq, om, pref=0.3, **P)
    assert r2[1] == 0.0 and r2[0] == r[0] and r2[2] == r[2]


def test_RP6_numpy_broadcast_twin():
    out, eps_k, eps_kq, om = _random_case(3, nq=64, nb1=4, nb2=3, nm=6)
    om[7, 2] = 0.0
    om[9, 1] = -0.02
    out[7, :, :, 2] = 0.0
    out[9, :, :, 1] = 0.0
    kT, mu, sigma, pref = 0.02585, -0.02, 0.02, 1.7
    f = 1.0 / (np.exp((eps_kq - mu) / kT) + 1.0)                      # [q, b2]
    with np.errstate(divide="ignore", over="ignore", invalid="ignore"):
        n = np.where(om > 0, 1.0 / np.expm1(np.where(om > 0, om, 1.0) / kT), 0.0)    # [q, nu]
    e1 = eps_k[None, :, None, None]; e2 = eps_kq[:, None, :, None]; w = om[:, None, None, :]
    fb = f[:, None, :, None]; nb = n[:, None, None, :]
    d = lambda x: np.exp(-(x / sigma) ** 2) / (np.sqrt(np.pi) * sigma)
    W = np.where(w > 0, (1 - fb + nb) * d(e1 - w - e2) + (fb + nb) * d(e1 + w - e2), 0.0)
    ref = pref * np.einsum("qabn,qabn->a", out, W)
    got = oracle.rates(out, eps_k, eps_kq, om, kT, mu, sigma, pref)
    assert np.allclose(got, ref, rtol=1e-13, atol=0)
