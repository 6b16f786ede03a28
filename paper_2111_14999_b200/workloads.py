"""Seeded synthetic inputs for the el-ph Wannier->Bloch |g|^2 hot path.

This module is the ONE piece of code shared by the CPU oracle's tests and the
CUDA path's tests / bench.  It holds none of the method's arithmetic: it only
draws random tensors with the shapes, distributions and structure of the five
workloads named in BASELINE.json (recipe: SURVEY.md section 8(d), restated in
DESIGN.md "Input recipe").  NumPy only; it imports neither ``oracle`` nor the
CUDA binding.

The workloads stand in for the paper's GaN runs (14
Wannier functions, 12 phonon modes, coarse grids 7x7x4 .. 12x12x7), whose
ab-initio data are not available here.

Every tensor is drawn from ``numpy.random.default_rng([seed, cfg_id,
tensor_id, index])`` (PCG64), so any slab / k-point can be regenerated on its
own, bit for bit, without materialising the rest (the "large" g_W is 57.8 GB).
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Tuple

import numpy as np

# tensor ids used in the seed sequence
_T_GW, _T_K, _T_Q, _T_UK, _T_UKQ, _T_EV, _T_OMEGA = range(7)


@dataclass(frozen=True)
class Workload:
    """One synthetic workload (all sizes in the paper's notation)."""

    name: str
    cfg_id: int
    nw: int                      # Wannier functions
    nb1: int                     # bands kept at k      (columns of U_k)
    nb2: int                     # bands kept at k+q    (columns of U_{k+q})
    nm: int                      # phonon modes = 3 * atoms
    grid_e: Tuple[int, int, int]  # electron lattice-vector box (counts per axis)
    grid_p: Tuple[int, int, int]  # phonon lattice-vector box
    lam: float                   # decay length of g_W in |Re|+|Rp|
    nk: int
    nq: int
    k_rule: str                  # "random" | "grid8_even"
    q_rule: str                  # "random" | "grid16"
    omega_lo: float
    omega_hi: float
    seed: int = 0

    @property
    def nRe(self) -> int:
        return int(np.prod(self.grid_e))

    @property
    def nRp(self) -> int:
        return int(np.prod(self.grid_p))

    @property
    def X(self) -> int:
        """complex elements of g_W per (Rp, Re) pair."""
        return self.nw * self.nw * self.nm

    @property
    def N(self) -> int:
        """columns of the Rp contraction = nb1*nw*nm."""
        return self.nb1 * self.nw * self.nm

    @property
    def gW_bytes(self) -> int:
        return 16 * self.nRp * self.nRe * self.X

    def with_(self, **kw) -> "Workload":
        return replace(self, **kw)


def _w(name, cfg_id, nw, nb1, nb2, nm, g, lam, nk, nq, k_rule, q_rule, lo, hi):
    return Workload(name, cfg_id, nw, nb1, nb2, nm, (g, g, g), (g, g, g), lam,
                    nk, nq, k_rule, q_rule, lo, hi, 0)


#: BASELINE.json "configs", in order.
CONFIGS = {
    "tiny":        _w("tiny",        0,  2,  2,  2,  3, 3, 1.5,   1,    64, "random",     "random", 0.01,  0.1),
    "si-like":     _w("si-like",     1,  8,  8,  8,  6, 7, 2.0,   1,  4096, "random",     "grid16", 0.005, 0.06),
    "4-atom":      _w("4-atom",      2, 16, 16, 16, 12, 9, 2.0,  16,  8192, "random",     "random", 0.005, 0.06),
    "band-window": _w("band-window", 3,  8,  4,  4,  6, 7, 2.0, 256,  4096, "grid8_even", "random", 0.005, 0.06),
    "large":       _w("large",       4, 32, 32, 32, 30, 7, 2.0,   4, 16384, "random",     "random", 0.002, 0.05),
}
CONFIG_ORDER = ["tiny", "si-like", "4-atom", "band-window", "large"]


def custom(name="custom", *, nw, nb1=None, nb2=None, nm, grid_e, grid_p=None,
           lam=2.0, nk=1, nq=8, omega=(0.01, 0.1), seed=0, cfg_id=99,
           k_rule="random", q_rule="random") -> Workload:
    """A small ad-hoc workload for tests (asymmetric grids, nb1 != nb2 != nw)."""
    grid_e = tuple(int(x) for x in grid_e)
    grid_p = grid_e if grid_p is None else tuple(int(x) for x in grid_p)
    return Workload(name, cfg_id, nw, nw if nb1 is None else nb1,
                    nw if nb2 is None else nb2, nm, grid_e, grid_p, lam, nk, nq,
                    k_rule, q_rule, omega[0], omega[1], seed)


def _rng(w: Workload, tensor_id: int, index: int = 0) -> np.random.Generator:
    return np.random.default_rng([w.seed, w.cfg_id, tensor_id, index])


def lattice_vectors(grid: Tuple[int, int, int]) -> np.ndarray:
    """Integer lattice vectors of a box centred at the origin, crystal
    coordinates, x slowest / z fastest.  An axis with n points
    spans -(n//2) .. -(n//2)+n-1.  Returns float64 [n, 3]."""
    axes = [np.arange(-(n // 2), -(n // 2) + n, dtype=np.float64) for n in grid]
    X, Y, Z = np.meshgrid(*axes, indexing="ij")
    return np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1).copy()


def Re_vectors(w: Workload) -> np.ndarray:
    return lattice_vectors(w.grid_e)


def Rp_vectors(w: Workload) -> np.ndarray:
    return lattice_vectors(w.grid_p)


def degeneracies(w: Workload):
    """Wigner-Seitz degeneracy weights; all 1 in BASELINE.json's configs."""
    return np.ones(w.nRe), np.ones(w.nRp)


def _cnormal(rng: np.random.Generator, shape) -> np.ndarray:
    """Standard complex Gaussian N(0,1) + i N(0,1), complex128."""
    out = np.empty(shape, dtype=np.complex128)
    v = out.view(np.float64)
    rng.standard_normal(out=v)
    return out


def gW_slab(w: Workload, p: int, out: np.ndarray | None = None) -> np.ndarray:
    """g_W[p] : complex128 [nRe][nw][nw][nm] for phonon lattice vector p.
    (N(0,1)+iN(0,1)) * exp(-(|Re|+|Rp|)/lam)."""
    shape = (w.nRe, w.nw, w.nw, w.nm)
    if out is None:
        out = np.empty(shape, dtype=np.complex128)
    assert out.shape == shape and out.dtype == np.complex128 and out.flags.c_contiguous
    _rng(w, _T_GW, p).standard_normal(out=out.view(np.float64))
    re_norm = np.linalg.norm(Re_vectors(w), axis=1)
    rp_norm = float(np.linalg.norm(Rp_vectors(w)[p]))
    decay = np.exp(-(re_norm + rp_norm) / w.lam)
    out *= decay[:, None, None, None]
    return out


def gW_full(w: Workload) -> np.ndarray:
    """g_W : complex128 [nRp][nRe][nw][nw][nm]. Only for configs that fit host RAM."""
    out = np.empty((w.nRp, w.nRe, w.nw, w.nw, w.nm), dtype=np.complex128)
    for p in range(w.nRp):
        gW_slab(w, p, out[p])
    return out


def k_points(w: Workload) -> np.ndarray:
    """float64 [nk][3], fractional (crystal) coordinates."""
    if w.k_rule == "random":
        return _rng(w, _T_K).random((w.nk, 3))
    if w.k_rule == "grid8_even":
        idx = np.arange(0, 512, 2)[: w.nk]          # even linear indices, z fastest
        i, j, l = idx // 64, (idx // 8) % 8, idx % 8
        return np.stack([i, j, l], axis=1).astype(np.float64) / 8.0
    raise ValueError(w.k_rule)


def q_points(w: Workload, ik: int = 0) -> np.ndarray:
    """float64 [nq][3]; fresh random list per k unless the rule is a grid."""
    if w.q_rule == "random":
        return _rng(w, _T_Q, ik).random((w.nq, 3))
    if w.q_rule == "grid16":
        idx = np.arange(w.nq)
        i, j, l = idx // 256, (idx // 16) % 16, idx % 16
        return np.stack([i, j, l], axis=1).astype(np.float64) / 16.0
    raise ValueError(w.q_rule)


def haar_unitary(rng: np.random.Generator, n: int, batch: int | None = None) -> np.ndarray:
    """Haar-distributed unitary matrices: Q of the QR of a complex Gaussian,
    columns re-phased by conj(diag R)/|diag R|.  [batch, n, n] or [n, n]."""
    shape = (n, n) if batch is None else (batch, n, n)
    z = _cnormal(rng, shape)
    q, r = np.linalg.qr(z)
    d = np.diagonal(r, axis1=-2, axis2=-1)
    ph = d / np.abs(d)
    return np.ascontiguousarray(q * ph[..., None, :])


def U_k(w: Workload, ik: int = 0) -> np.ndarray:
    """complex128 [nw][nb1]: orthonormal columns (first nb1 of a Haar unitary)."""
    return np.ascontiguousarray(haar_unitary(_rng(w, _T_UK, ik), w.nw)[:, : w.nb1])


def U_kq(w: Workload, ik: int = 0) -> np.ndarray:
    """complex128 [nq][nw][nb2], independent per (k, q)."""
    return np.ascontiguousarray(haar_unitary(_rng(w, _T_UKQ, ik), w.nw, w.nq)[:, :, : w.nb2])


def ph_eigvecs(w: Workload, ik: int = 0) -> np.ndarray:
    """complex128 [nq][nm][nm] (row kappa, column nu), Haar per (k, q)."""
    return haar_unitary(_rng(w, _T_EV, ik), w.nm, w.nq)


def omega(w: Workload, ik: int = 0) -> np.ndarray:
    """float64 [nq][nm], iid uniform [omega_lo, omega_hi)."""
    return _rng(w, _T_OMEGA, ik).uniform(w.omega_lo, w.omega_hi, (w.nq, w.nm))


def q_inputs(w: Workload, ik: int = 0):
    """(q, Ukq, ev, omega) for k-point ik."""
    return q_points(w, ik), U_kq(w, ik), ph_eigvecs(w, ik), omega(w, ik)


def sample_indices(n: int, count: int, seed: int = 12345) -> np.ndarray:
    """A seeded, sorted sample of `count` distinct indices of range(n) (parity
    subsets at full size; covers every tile position with high probability)."""
    count = min(count, n)
    return np.sort(np.random.default_rng(seed).permutation(n)[:count])


# ---- inputs of the fused linewidth accumulation (Eq. 29, Eq. 61) ----------
_T_EPS_K, _T_EPS_KQ = 7, 8

#: k_B T (300 K in eV), chemical potential, Gaussian smearing sigma (Eq. 61), prefactor 2 pi/(N_k V) of Eq. 29.
#: Energies are in eV-like units on the scale of omega (0.005 .. 0.06) so that both delta functions of
#: Eq. 29 have support inside the band window.
RATE_PARAMS = dict(kT=0.02585, mu=0.0, sigma=0.012, pref=2.0 * np.pi / 4096.0)


def band_energies(w: Workload, ik: int = 0):
    """(eps_k [nb1], eps_kq [nq][nb2]): band energies at k and at every k+q, iid uniform in
    [-0.15, 0.15) around mu = 0 (a band window a few phonon energies wide)."""
    eps_k = _rng(w, _T_EPS_K, ik).uniform(-0.15, 0.15, w.nb1)
    eps_kq = _rng(w, _T_EPS_KQ, ik).uniform(-0.15, 0.15, (w.nq, w.nb2))
    return eps_k, eps_kq


# ---- inputs of the polar long-range term (Eq. 14-15) --------------------------------------
_T_POLAR = 9


def polar_inputs(w: Workload, h: int = 2):
    """dict(recip [3][3], G [(2h+1)^3][3], Zstar [nm/3][3][3], eps_inf [3][3], coeff): a slightly sheared reciprocal
    lattice, the integer box {-h..h}^3 of G vectors, random Born charges of order 1 (not symmetric), a symmetric
    positive-definite high-frequency dielectric tensor, and a coefficient that makes the long-range amplitude
    comparable to the short-range one of the recipe."""
    assert w.nm % 3 == 0
    rng = _rng(w, _T_POLAR)
    recip = 2.0 * np.pi * (np.eye(3) + 0.1 * rng.normal(size=(3, 3)))
    A = rng.normal(size=(3, 3))
    return dict(recip=recip, G=lattice_vectors((2 * h + 1,) * 3), Zstar=rng.normal(size=(w.nm // 3, 3, 3)),
                eps_inf=A @ A.T + 3.0 * np.eye(3), coeff=2.0)
