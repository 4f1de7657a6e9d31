"""Pins for oracle/philox.py, oracle/nm.py and oracle/constants.py (CPU only)."""
import math
import os

import numpy as np
import pytest

from oracle import constants, nm, philox

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _golden_table(name):
    rows = {}
    for line in open(os.path.join(GOLDEN, name)):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split()[:2]
            rows[k] = float(v)
    return rows


# ---------------------------------------------------------------- constants
def test_constants_match_paper():
    g = _golden_table("paper_constants.txt")
    assert constants.H_PLANCK == g["h_eV_ps"]
    assert constants.MVV2E == g["mvv2e"]
    assert abs(constants.HBAR - g["h_eV_ps"] / (2 * math.pi)) < 1e-18
    # L244: dt = 0.5 fs, 1 s/step -> 86400 steps/day * 0.5e-6 ns = 0.0432 ns/day, printed 0.043
    assert abs(86400 * 0.5e-6 - g["ns_per_day_at_1s_per_step"]) < 5e-4
    # Appendix C example (L458): printed 0.600; its printed inputs give 0.5906 -> loose pin only
    lam = g["h_eV_ps"] / (g["neon_sigma_A"] * math.sqrt(g["neon_mass"] * g["neon_eps_eV"]) * math.sqrt(g["mvv2e"]))
    assert abs(lam - g["neon_lambda_star_printed"]) < 0.02


def test_beta_hbar_at_300K():
    # beta*hbar at 300 K is 25.46 fs (textbook value hbar/(k_B 300 K)); omega_P = P/(beta hbar), Eq. 2
    bh = constants.HBAR / (constants.KB * 300.0)
    assert abs(bh - 25.46e-3) < 0.01e-3
    assert abs(nm.omega_P(32, 300.0) - 32 / bh) < 1e-9


# ---------------------------------------------------------------- Philox
def test_philox_known_answers():
    n = 0
    for line in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")):
        line = line.split("#")[0].strip()
        if not line:
            continue
        w = [int(t, 16) for t in line.split()]
        out = philox.philox4x32_10(*w[:6])
        assert [int(o) for o in out] == w[6:]
        n += 1
    assert n == 3


def test_philox_vectorised_equals_scalar():
    rng = np.random.default_rng(5)
    c = rng.integers(0, 2 ** 32, size=(6, 17), dtype=np.uint64)
    vec = philox.philox4x32_10(*c)
    for t in range(17):
        sc = philox.philox4x32_10(*[int(c[a, t]) for a in range(6)])
        assert [int(v[t]) for v in vec] == [int(s) for s in sc]


def test_keying_is_injective_in_every_field():
    base = [int(w) for w in philox.words_for(7, 3, 2, 5, 1)]
    for other in [(8, 3, 2, 5, 1), (7, 4, 2, 5, 1), (7, 3, 4, 5, 1), (7, 3, 2, 6, 1), (7, 3, 2, 5, 2),
                  (7 + 2 ** 32, 3, 2, 5, 1), (7, 3 + 2 ** 32, 2, 5, 1)]:
        assert [int(w) for w in philox.words_for(*other)] != base
    # counter word 3 is 4*(k//2) + alpha: (k=2, alpha=0) must differ from (k=0, alpha=3) + 1 etc.
    assert [int(w) for w in philox.words_for(7, 3, 2, 5, 0)] != [int(w) for w in philox.words_for(7, 3, 0, 5, 3)]
    # modes 2q and 2q+1 share the draw (same words) and take different Box-Muller branches
    assert [int(w) for w in philox.words_for(7, 3, 3, 5, 1)] == base
    e2, e3 = float(philox.normal(7, 3, 2, 5, 1)), float(philox.normal(7, 3, 3, 5, 1))
    w = base
    u1 = float(philox.uniform53(w[0], w[1])) + 2.0 ** -53
    u2 = float(philox.uniform53(w[2], w[3]))
    assert abs(e2 * e2 + e3 * e3 - (-2.0 * math.log(u1))) < 1e-12          # cos^2 + sin^2 = 1
    assert abs(math.atan2(e3, e2) % (2 * math.pi) - 2 * math.pi * u2) < 1e-12


def test_uniform_grid_and_normal_finite_at_extremes():
    assert philox.uniform53(0, 0) == 0.0
    assert philox.uniform53(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 2.0 ** -53        # exact, < 1
    assert philox.uniform53(1 << 5, 0) == 2.0 ** -27 and philox.uniform53(0, 1 << 6) == 2.0 ** -53
    # u1 = grid + 2^-53 lies in (0, 1]: the Box-Muller radius is finite, at most sqrt(2*53 ln 2)
    assert math.sqrt(-2.0 * math.log(2.0 ** -53)) < 8.58


def test_normal_moments():
    k, i, a = np.meshgrid(np.arange(8), np.arange(5000), np.arange(3), indexing="ij")
    eta = philox.normal(1234, 17, k, i, a).ravel()
    n = eta.size                                   # 120000
    assert abs(eta.mean()) < 4.0 / math.sqrt(n)
    assert abs(eta.var() - 1.0) < 4.0 * math.sqrt(2.0 / n)
    assert abs((eta ** 4).mean() - 3.0) < 4.0 * math.sqrt(96.0 / n)
    assert abs((eta ** 3).mean()) < 4.0 * math.sqrt(15.0 / n)
    # different steps are uncorrelated
    eta2 = philox.normal(1234, 18, k, i, a).ravel()
    assert abs(np.mean(eta * eta2)) < 4.0 / math.sqrt(n)
    # the two branches of one draw (modes 2q, 2q+1) are uncorrelated, also in their squares
    ev = philox.normal(1234, 17, k, i, a)
    c, s_ = ev[0::2].ravel(), ev[1::2].ravel()
    assert abs(np.mean(c * s_)) < 4.0 / math.sqrt(c.size)
    assert abs(np.mean((c * c - 1.0) * (s_ * s_ - 1.0))) < 4.0 * 2.0 / math.sqrt(c.size)


# ---------------------------------------------------------------- normal modes (PAPER.md B1-B3)
@pytest.mark.parametrize("P", [1, 2, 3, 4, 5, 8, 32, 64])
def test_nm_matrix_orthogonal_and_diagonalises_ring(P):
    M = nm.nm_matrix(P)
    assert np.abs(M @ M.T - np.eye(P)).max() < 1e-13                   # B3 (L446-448)
    # ring Laplacian of Eq. 1 (L53): sum_k (r_k - r_{k+1})^2 = r^T A r, A = 2I - S - S^T
    S = np.roll(np.eye(P), 1, axis=1)
    A = 2 * np.eye(P) - S - S.T
    lam = nm.lambdas(P)
    assert np.abs(M @ A @ M.T - np.diag(lam)).max() < 1e-13            # B2 (L443), same row index k
    assert lam[0] == 0.0


def test_nm_first_row_is_centroid_and_p4_explicit():
    M = nm.nm_matrix(4)
    expect = np.array([[0.5, 0.5, 0.5, 0.5],
                       [math.sqrt(0.5), 0.0, -math.sqrt(0.5), 0.0],
                       [0.5, -0.5, 0.5, -0.5],
                       [0.0, -math.sqrt(0.5), 0.0, math.sqrt(0.5)]])
    assert np.abs(M - expect).max() < 1e-15
    x = np.random.default_rng(0).standard_normal((4, 3, 3))
    assert np.allclose(nm.to_nm(M, x)[0], x.mean(axis=0) * 2.0)       # sqrt(P) * centroid
    assert np.allclose(nm.from_nm(M, nm.to_nm(M, x)), x, atol=1e-15)


def test_spring_energy_cartesian_equals_normal_mode():
    # Eq. 1 spring term vs Eq. A3 (DESIGN R-1: omega_n^2): sum_k 1/2 m w_P^2 |r_k - r_{k+1}|^2 = sum_k 1/2 m w_k^2 x~_k^2
    P, T = 32, 300.0
    rng = np.random.default_rng(1)
    x = rng.standard_normal((P, 7, 3))
    M = nm.nm_matrix(P)
    wP, wk = nm.omega_P(P, T), nm.omegas(P, T)
    cart = 0.5 * wP ** 2 * np.sum((x - np.roll(x, -1, axis=0)) ** 2)
    xt = nm.to_nm(M, x)
    nmode = 0.5 * np.sum(wk[:, None, None] ** 2 * xt ** 2)
    assert abs(cart - nmode) < 1e-12 * abs(cart)
    assert abs(wk[P // 2] - 2 * wP) < 1e-9
