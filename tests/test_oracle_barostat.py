"""Pins of oracle/barostat.py and of the NpH / NpT step of oracle/pimd.py against what the paper and the
mathematics fix (Appendix A Eq. A10-A17, Appendix E Eq. E1, E4-E7, L196):
  * E1 equals the time integral of the cell force over the B kick it is paired with (quadrature);
  * E4/E5 solve dx/dt = v_W x + v, dv/dt = -v_W v (numerical ODE), with the v_W -> 0 limit;
  * the NpH step conserves the enthalpy of Eq. A17 with second-order drift -- this fails for a wrong sign
    or factor in any of E1's first-order terms, E4, E5, E6, and for the printed "1/(n k_B T)" (R-20);
  * A12 = A11 at n = 1; ideal-gas and harmonic closed forms of A12; A10 from the spring energy;
  * E7 keeps <K_W> = n k_B T / 2 and draws the documented Philox normal.
"""
import numpy as np
import pytest
from scipy.integrate import solve_ivp

from oracle import barostat, integrator, nm, philox
from oracle.constants import KB, MVV2E
from oracle.pimd import OraclePIMD


def _state(P, N, seed, T=300.0, spread=0.05):
    rng = np.random.default_rng(seed)
    masses = rng.choice([15.9994, 1.008], size=N)
    xc = rng.uniform(-3.0, 3.0, size=(1, N, 3))
    x = xc + spread * rng.standard_normal((P, N, 3))
    v = rng.standard_normal((P, N, 3)) * np.sqrt(P * KB * T / (masses[None, :, None] * MVV2E))
    return masses, x, v


def test_constants_and_mass():
    assert barostat.BAR_PER_EV_A3 == pytest.approx(1.602176634e-19 / 1e-30 / 1e5, rel=1e-15)
    assert barostat.barostat_mass(4, 10, 300.0, 0.5) == pytest.approx(3 * 4 * 10 * KB * 300.0 * 0.25, rel=1e-15)


def test_E1_is_the_integral_of_the_cell_force_over_the_kick():
    """d(W v_W)/dt = sum m v~0(t)^2 - S_cv + sum Tr Xi - 3 n V P_ext + 3 n k_B T with v~0(t) = v~0 + t F~0/m."""
    P, N = 4, 7
    masses, x, v = _state(P, N, 1)
    M = nm.nm_matrix(P)
    vt = nm.to_nm(M, v)
    k_spring = 0.8
    f = -k_spring * x
    ft = nm.to_nm(M, f)
    Xi = np.stack([x[k].T @ f[k] for k in range(P)])
    V, T, W, p_ext, h, vW0 = 512.0, 300.0, 7.3, 2.0e-5, 0.013, 0.021
    got = barostat.press_v_step(vW0, x, vt, ft, Xi, masses, V, T, W, p_ext, h)
    rc = x.mean(axis=0, keepdims=True)
    const = -np.sum((x - rc) * f) + np.trace(Xi, axis1=1, axis2=2).sum() - 3 * P * V * p_ext + 3 * P * KB * T
    ts, ws = np.polynomial.legendre.leggauss(8)
    ts = 0.5 * h * (ts + 1.0)
    ws = 0.5 * h * ws
    integral = 0.0
    for t, w in zip(ts, ws):
        v0t = vt[0] + t * ft[0] / (masses[:, None] * MVV2E)
        integral += w * (np.sum(masses[:, None] * v0t * v0t) * MVV2E + const)
    assert got == pytest.approx(vW0 + integral / W, rel=1e-13)


@pytest.mark.parametrize("vW", [0.0, 1e-9, 0.9e-4 / 0.01, 1.1e-4 / 0.01, 0.7, -1.3])
def test_E4_E5_solve_the_cell_coupled_drift(vW):
    h = 0.01
    xt = np.zeros((2, 1, 3)); vt = np.zeros((2, 1, 3))
    xt[0, 0] = [1.0, -2.0, 0.5]; vt[0, 0] = [3.0, 0.25, -1.0]
    xt[1, 0] = [9.0, 9.0, 9.0]; vt[1, 0] = [7.0, 7.0, 7.0]
    xn, vn, box = barostat.qc_step(xt, vt, [10.0, 11.0, 12.0], vW, h)
    sol = solve_ivp(lambda t, y: np.concatenate([vW * y[:3] + y[3:], -vW * y[3:]]), (0.0, h),
                    np.concatenate([xt[0, 0], vt[0, 0]]), rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(xn[0, 0], sol.y[:3, -1], rtol=1e-10)
    np.testing.assert_allclose(vn[0, 0], sol.y[3:, -1], rtol=1e-10)
    np.testing.assert_array_equal(xn[1], xt[1])          # internal modes untouched (R-21)
    np.testing.assert_array_equal(vn[1], vt[1])
    np.testing.assert_allclose(box, np.array([10.0, 11.0, 12.0]) * np.exp(h * vW), rtol=1e-15)   # E6
    if vW == 0.0:
        np.testing.assert_array_equal(xn[0], xt[0] + h * vt[0])


def test_E4_group_property():
    xt = np.random.default_rng(0).standard_normal((1, 3, 3)); vt = np.random.default_rng(1).standard_normal((1, 3, 3))
    a1, b1, L1 = barostat.qc_step(xt, vt, [5.0, 5.0, 5.0], 0.37, 0.2)
    a2, b2, L2 = barostat.qc_step(a1, b1, L1, 0.37, 0.3)
    a3, b3, L3 = barostat.qc_step(xt, vt, [5.0, 5.0, 5.0], 0.37, 0.5)
    np.testing.assert_allclose(a2, a3, rtol=1e-13); np.testing.assert_allclose(b2, b3, rtol=1e-13)
    np.testing.assert_allclose(L2, L3, rtol=1e-15)


def _nph(dt, n_steps, P=4, N=6, gamma=0.0, seed=3, integ="baoab", aniso=False):
    masses_t = [15.9994, 1.008]
    rng = np.random.default_rng(seed)
    types = rng.integers(0, 2, size=N)
    m = np.asarray(masses_t)[types]
    x = 0.23 * rng.standard_normal((1, N, 3)) + 0.05 * rng.standard_normal((P, N, 3))   # thermal width of the trap
    p = rng.standard_normal((P, N, 3)) * np.sqrt(P * KB * 300.0 * m[None, :, None] / MVV2E)   # (g/mol) A/ps
    sim = OraclePIMD(types, masses_t, [10.0, 10.0, 10.0], P, 300.0, dt, gamma, 11, integrator=integ)
    sim.set_barostat(KB * 300.0 / 1000.0 * barostat.BAR_PER_EV_A3, 0.05, aniso=aniso)   # trapped gas: <V> = k_B T / P_ext
    sim.set_state(x, p)
    sim.set_model_harmonic(0.5)
    h0 = sim.barostat_state()["enthalpy"]
    hs = []
    for _ in range(n_steps):
        sim.step(1)
        hs.append(sim.barostat_state()["enthalpy"] - h0)
    return sim, np.asarray(hs)


def test_obabo_equals_baoab_in_nph():
    """Without thermostats both splittings are B A B with the same cell sub-steps: A(dt) = A(dt/2) A(dt/2) and
    E4-E6 compose (group property), so the trajectories agree to rounding."""
    a, _ = _nph(1.0e-3, 20, integ="baoab")
    b, _ = _nph(1.0e-3, 20, integ="obabo")
    np.testing.assert_allclose(a.positions(), b.positions(), rtol=0, atol=1e-11)
    assert a.vW == pytest.approx(b.vW, rel=1e-10)
    np.testing.assert_allclose(a.box, b.box, rtol=1e-13)


def test_obabo_npt_draws_both_half_step_streams():
    sim, _ = _nph(1.0e-3, 3, gamma=20.0, integ="obabo")
    ref, _ = _nph(1.0e-3, 3, gamma=20.0, integ="baoab")
    assert np.isfinite(sim.barostat_state()["enthalpy"]) and sim.vW != ref.vW


@pytest.mark.parametrize("integ", ["baoab", "obabo"])
def test_nph_conserves_the_enthalpy_A17_to_second_order(integ):
    sim1, d1 = _nph(1.0e-3, 400, integ=integ)
    sim2, d2 = _nph(0.5e-3, 800, integ=integ)
    st = sim1.barostat_state()
    assert abs(st["V"] / 1000.0 - 1.0) > 0.02 and abs(st["v_W"]) > 0           # the cell really moved
    assert np.abs(d1).max() < 5e-4 * abs(st["enthalpy"])
    assert np.abs(d2).max() < 0.3 * np.abs(d1).max()                          # ~ dt^2


def test_printed_reciprocal_in_E1_would_break_A17(monkeypatch):
    """R-20: with 1/(n k_B T) in place of n k_B T the same run drifts by orders of magnitude more."""
    _, good = _nph(1.0e-3, 400)
    orig = barostat.press_v_step

    def printed(vW, x, vt, ft, Xi, masses, V, T, W, p_ext, h):
        P = x.shape[0]
        return orig(vW, x, vt, ft, Xi, masses, V, T, W, p_ext, h) + (3.0 * h / W) * (1.0 / (P * KB * T) - P * KB * T)

    monkeypatch.setattr(barostat, "press_v_step", printed)
    _, bad = _nph(1.0e-3, 400)
    assert np.abs(bad).max() > 100.0 * np.abs(good).max()


def test_pcv_special_cases():
    # n = 1: A12 = A11 (no r - r_c term, v~0 = v)
    masses, x, v = _state(1, 9, 4)
    M = nm.nm_matrix(1)
    vt = nm.to_nm(M, v)
    f = np.random.default_rng(5).standard_normal(x.shape)
    Xi = np.random.default_rng(6).standard_normal((1, 3, 3))
    V = 321.0
    K_ring = 0.5 * np.sum(masses[None, :, None] * vt * vt) * MVV2E
    assert barostat.p_cv(x, vt, nm.to_nm(M, f), Xi, masses, V) == pytest.approx(barostat.p_md(K_ring, Xi, V), rel=1e-13)
    # ideal gas, all beads moving together with velocity u: v~0 = sqrt(n) u -> P_CV = sum m u^2 / (3V)
    P, N = 8, 5
    masses, x, _ = _state(P, N, 7)
    u = np.random.default_rng(8).standard_normal((N, 3))
    vt = nm.to_nm(nm.nm_matrix(P), np.broadcast_to(u, (P, N, 3)).copy())
    z = np.zeros((P, N, 3))
    got = barostat.p_cv(x, vt, z, np.zeros((P, 3, 3)), masses, V)
    assert got == pytest.approx(np.sum(masses[:, None] * u * u) * MVV2E / (3.0 * V), rel=1e-12)
    # harmonic trap: -S_cv + sum Tr Xi = sum_k r_c.F_k
    f = -0.7 * x
    Xi = np.stack([x[k].T @ f[k] for k in range(P)])
    rc = x.mean(axis=0)
    got = barostat.p_cv(x, z, nm.to_nm(nm.nm_matrix(P), f), Xi, masses, V)
    assert got == pytest.approx(np.sum(rc[None] * f) / (3.0 * P * V), rel=1e-12)


def test_p_pr_from_cartesian_springs():
    P, N, T, V = 8, 5, 250.0, 400.0
    masses, x, _ = _state(P, N, 9)
    M = nm.nm_matrix(P)
    om = nm.omegas(P, T)
    e = integrator.estimators(x, np.zeros_like(x), np.zeros_like(x), np.zeros(P), masses, M, om, T)
    wP = nm.omega_P(P, T)
    dr = x - np.roll(x, -1, axis=0)
    direct = (3 * P * N * KB * T - np.sum(masses[None, :, None] * wP * wP * dr * dr) * MVV2E / P) / (3 * V)
    assert barostat.p_pr(e["S_ring"], P, N, T, V) == pytest.approx(direct, rel=1e-12)
    assert barostat.p_pr(e["S_ring"], P, N, T, V) == pytest.approx(2.0 * e["K_PR"] / (3 * V), rel=1e-12)   # A10 = (2/3V) A7


def test_p_pr_of_the_free_ring_polymer_is_the_ideal_gas_pressure():
    """Pin of the 1/n in A10 (DESIGN R-6 / R-25): normal-mode coordinates of a FREE ring polymer drawn from their exact
    Gaussians at the ring temperature nT, <x~_k^2> = n k_B T / (m omega_k^2 mvv2e), give <S_ring> = 3N(n-1) n k_B T / 2,
    hence <P_PR> = N k_B T / V.  Without the 1/n the mean would be -n(n-2) N k_B T / V."""
    P, N, T, V = 16, 40, 300.0, 5000.0
    rng = np.random.default_rng(2)
    masses = rng.uniform(1.0, 16.0, N)
    om = nm.omegas(P, T)
    sig = np.zeros((P, N))
    sig[1:] = np.sqrt(P * KB * T / (masses[None, :] * om[1:, None] ** 2 * MVV2E))
    acc = []
    for _ in range(400):
        xt = sig[:, :, None] * rng.standard_normal((P, N, 3))
        S = 0.5 * np.sum(masses[None, :, None] * om[:, None, None] ** 2 * xt * xt) * MVV2E
        acc.append(barostat.p_pr(S, P, N, T, V))
    ideal = N * KB * T / V
    err = np.std(acc) / np.sqrt(len(acc))
    assert abs(np.mean(acc) - ideal) < 4 * err and err < 0.1 * ideal


def test_E7_keeps_the_barostat_temperature_and_uses_the_documented_normal():
    P, N, T, W, g, h, seed = 4, 12, 300.0, 3.0, 5.0, 0.01, 77
    c1 = np.exp(-h * g)
    v1 = barostat.press_o_step(0.4, P, N, T, W, g, h, seed, 5)
    eta = float(philox.normal(seed, 5, 0, N, 0))
    assert v1 == pytest.approx(c1 * 0.4 + np.sqrt(1 - c1 * c1) * np.sqrt(P * KB * T / W) * eta, rel=1e-14)
    vW, acc = 0.0, []
    for s in range(40000):
        vW = barostat.press_o_step(vW, P, N, T, W, g, 0.2, seed, s)
        acc.append(0.5 * W * vW * vW)
    assert np.mean(acc[100:]) == pytest.approx(0.5 * P * KB * T, rel=0.04)


def test_npt_run_is_finite_and_thermostats_the_cell():
    sim, _ = _nph(1.0e-3, 50, gamma=20.0)
    st = sim.barostat_state()
    assert np.isfinite(st["enthalpy"]) and st["V"] > 0
    assert st["P_CV"] != st["P_MD"] and np.isfinite(st["P_PR"])


# ---- anisotropic variant (Eq. A14, E2, E3) ----------------------------------------------------------------------

def test_E3_diagonal_averages_to_A12_and_mass_A14():
    P, N = 4, 7
    masses, x, v = _state(P, N, 21)
    M = nm.nm_matrix(P)
    vt = nm.to_nm(M, v)
    f = np.random.default_rng(22).standard_normal(x.shape)
    ft = nm.to_nm(M, f)
    Xi = np.random.default_rng(23).standard_normal((P, 3, 3))
    d = barostat.p_cv_diag(x, vt, ft, Xi, masses, 300.0)
    assert d.mean() == pytest.approx(barostat.p_cv(x, vt, ft, Xi, masses, 300.0), rel=1e-13)
    assert len(set(np.round(d, 12))) == 3
    assert barostat.barostat_mass_aniso(4, 10, 300.0, 0.5) == pytest.approx(barostat.barostat_mass(4, 10, 300.0, 0.5) / 3)


def test_E2_is_the_integral_of_the_cell_force_per_component():
    P, N = 4, 7
    masses, x, v = _state(P, N, 31)
    M = nm.nm_matrix(P)
    vt = nm.to_nm(M, v)
    f = -0.8 * x * np.array([1.0, 0.5, 2.0])
    ft = nm.to_nm(M, f)
    Xi = np.stack([x[k].T @ f[k] for k in range(P)])
    V, T, W, p_ext, h = 512.0, 300.0, 2.1, 2.0e-5, 0.013
    vW0 = np.array([0.02, -0.01, 0.005])
    got = barostat.press_v_step_aniso(vW0, x, vt, ft, Xi, masses, V, T, W, p_ext, h)
    rc = x.mean(axis=0, keepdims=True)
    ts, ws = np.polynomial.legendre.leggauss(8)
    ts = 0.5 * h * (ts + 1.0)
    ws = 0.5 * h * ws
    for a in range(3):
        const = -np.sum(((x - rc) * f)[:, :, a]) + Xi[:, a, a].sum() - P * V * p_ext + P * KB * T
        integral = sum(w * (np.sum(masses * (vt[0][:, a] + t * ft[0][:, a] / (masses * MVV2E)) ** 2) * MVV2E + const)
                       for t, w in zip(ts, ws))
        assert got[a] == pytest.approx(vW0[a] + integral / W, rel=1e-13)


@pytest.mark.parametrize("integ", ["baoab", "obabo"])
def test_anisotropic_nph_conserves_the_enthalpy_with_A14(integ):
    sim1, d1 = _nph(1.0e-3, 400, integ=integ, aniso=True)
    sim2, d2 = _nph(0.5e-3, 800, integ=integ, aniso=True)
    st = sim1.barostat_state()
    assert np.ptp(st["box"]) > 0.05 and np.ptp(st["v_W3"]) > 0            # the three cell vectors went their own ways
    assert np.abs(d1).max() < 5e-4 * abs(st["enthalpy"])
    assert np.abs(d2).max() < 0.3 * np.abs(d1).max()


def test_anisotropic_E7_draws_one_normal_per_component():
    P, N, T, W, g, h, seed = 4, 12, 300.0, 3.0, 5.0, 0.01, 77
    c1 = np.exp(-h * g)
    v1 = barostat.press_o_step_aniso(np.array([0.4, 0.1, -0.2]), P, N, T, W, g, h, seed, 5, half=1)
    eta = np.array([float(philox.normal(seed, 5, 0, N, a, 1)) for a in range(3)])
    np.testing.assert_allclose(v1, c1 * np.array([0.4, 0.1, -0.2]) + np.sqrt(1 - c1 * c1) * np.sqrt(P * KB * T / W) * eta,
                               rtol=1e-14)
    assert len(set(eta)) == 3
