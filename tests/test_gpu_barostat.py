"""GPU parity of the isotropic BZP barostat (Appendix E, Eq. A10-A17) through the
C ABI against oracle/barostat.py + oracle/pimd.py, on the same seeded inputs.  Tolerances: x, p, cell and v_W
<= 1e-10 relative after one step with FP64 forces (harmonic model), <= 1e-6 after 10 steps (north_star's integrator
bar); with the se_e2_a model the FP32-level forces and virial set the bar (1e-6 on x, p after 10 steps;
pressures to 1e-4 of their largest term)."""
import numpy as np
import pytest

import workloads
from oracle.constants import KB, MVV2E
from oracle.pimd import OraclePIMD

pytestmark = pytest.mark.gpu

BAR = 1.602176634e6


@pytest.fixture(scope="module")
def pk():
    import paper_2602_13553_b200 as pk
    pk.lib()
    return pk


def _rel(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


def _trap_system(N, P, seed, T=300.0):
    """A gas at the thermal width of a harmonic trap k = 0.5 eV/A^2 (the system of the oracle's NpH pin)."""
    rng = np.random.default_rng(seed)
    types = rng.integers(0, 2, size=N).astype(np.int32)
    masses = np.array([15.9994, 1.008])
    m = masses[types]
    x = 0.23 * rng.standard_normal((1, N, 3)) + 0.05 * rng.standard_normal((P, N, 3))
    p = rng.standard_normal((P, N, 3)) * np.sqrt(P * KB * T * m[None, :, None] / MVV2E)
    return types, masses, x, p


def _compare_state(bs, bo, tol):
    for key in ("v_W", "V", "P_CV", "P_PR", "P_MD", "K_W", "U_W", "J_W", "enthalpy"):
        scale = max(abs(bo[key]), abs(bo["P_MD"]) if key.startswith("P_") else 0.0, 1e-3 if key == "v_W" else 0.0)
        assert abs(bs[key] - bo[key]) <= tol * max(scale, 1e-12), (key, bs[key], bo[key])
    assert _rel(bs["box"], bo["box"]) <= tol


@pytest.mark.parametrize("P", [1, 4, 32, 64])
@pytest.mark.parametrize("gamma", [0.0, 20.0])
def test_barostat_parity_harmonic(pk, P, gamma):
    N = 43                                           # 129 dofs: one full 128-thread block and a tail of one
    types, masses, x, p = _trap_system(N, P, seed=20 + P)
    box = [10.0, 11.0, 12.0]
    p_ext = 2.0 * KB * 300.0 / 1320.0 * BAR
    args = (types, masses, box, P, 300.0, 1.0e-3, gamma)
    sim = pk.PIMD(*args, seed=5)
    sim.set_state(x, p)
    sim.set_model_harmonic(0.5)
    sim.set_barostat(p_ext, 0.05)
    orc = OraclePIMD(*args, seed=5)
    orc.set_barostat(p_ext, 0.05)
    orc.set_state(x, p)
    orc.set_model_harmonic(0.5)
    _compare_state(sim.barostat_state(), orc.barostat_state(), 1e-11)
    sim.step(1)
    orc.step(1)
    assert _rel(sim.positions(), orc.positions()) < 1e-10
    assert _rel(sim.momenta(), orc.momenta()) < 1e-10
    _compare_state(sim.barostat_state(), orc.barostat_state(), 1e-10)
    sim.step(9)
    orc.step(9)
    assert _rel(sim.positions(), orc.positions()) < 1e-9
    assert _rel(sim.momenta(), orc.momenta()) < 1e-9
    bs, bo = sim.barostat_state(), orc.barostat_state()
    _compare_state(bs, bo, 1e-9)
    assert abs(bo["V"] / 1320.0 - 1.0) > 1e-3 and bo["v_W"] != 0.0          # the cell really moved
    e, o = sim.estimators(), orc.estimators()
    for key in ("K_PR", "K_CV", "H", "K_ring", "S_ring", "U_sum"):
        assert abs(e[key] - o[key]) <= 1e-9 * max(1.0, abs(o[key])), key
    sim.close()


def test_nph_enthalpy_is_conserved_on_the_gpu(pk):
    """Eq. A17 over 2000 steps of the CUDA path alone (a property that holds at any size)."""
    P, N = 8, 64
    types, masses, x, p = _trap_system(N, P, seed=3)
    sim = pk.PIMD(types, masses, [10.0] * 3, P, 300.0, 0.5e-3, 0.0, seed=1)
    sim.set_state(x, p)
    sim.set_model_harmonic(0.5)
    sim.set_barostat(KB * 300.0 / 1000.0 * BAR, 0.05)
    h0 = sim.barostat_state()["enthalpy"]
    dev = []
    for _ in range(20):
        sim.step(100)
        dev.append(sim.barostat_state()["enthalpy"] - h0)
    assert np.abs(dev).max() < 5e-4 * abs(h0)
    assert abs(sim.barostat_state()["V"] / 1000.0 - 1.0) > 0.01
    sim.close()


def test_split_calls_agree_with_one_call_under_the_barostat(pk):
    """step(6) against step(1)+step(2)+step(3).  Not bitwise: a call boundary re-reads the kicked velocities where
    the single call advances the two velocity sums analytically (barostat.cu), a rounding-level difference."""
    N, P = 50, 8
    types, masses, x, p = _trap_system(N, P, seed=9)
    out = []
    for chunks in ((6,), (1, 2, 3)):
        sim = pk.PIMD(types, masses, [10.0] * 3, P, 300.0, 1e-3, 20.0, seed=4)
        sim.set_state(x, p)
        sim.set_model_harmonic(0.5)
        sim.set_barostat(40.0, 0.05)
        for c in chunks:
            sim.step(c)
        out.append((sim.positions(), sim.momenta(), sim.barostat_state()))
        sim.close()
    assert _rel(out[0][0], out[1][0]) < 1e-12 and _rel(out[0][1], out[1][1]) < 1e-12
    assert abs(out[0][2]["v_W"] - out[1][2]["v_W"]) < 1e-12 * abs(out[1][2]["v_W"])
    assert _rel(out[0][2]["box"], out[1][2]["box"]) < 1e-14


def test_full_npt_step_parity_config0(pk):
    """configs[0] geometry and model under NpT at 1 bar (configs[4]'s ensemble at the size the oracle finishes):
    multi-image neighbours from a cell that changes every step."""
    cfg, wb, desc, w = workloads.make_config(0)
    args = (wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"])
    sim = pk.PIMD(*args, seed=11, model_desc=desc)
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    sim.set_barostat(1.0, 0.02)
    orc = OraclePIMD(*args, seed=11)
    orc.set_barostat(1.0, 0.02)
    orc.set_state(wb["x"], wb["p"])
    orc.set_model(desc, w)

    def pressures_close(bs, bo):
        # A12's three terms nearly cancel; the FP32-level virial bounds the error by 1e-4 of the largest term
        trXi = np.trace(orc.virial(), axis1=1, axis2=2).sum()
        big = abs(trXi) / (3.0 * bo["V"]) * BAR
        for key in ("P_CV", "P_MD"):
            assert abs(bs[key] - bo[key]) <= 1e-4 * max(big, abs(bo[key])), (key, bs[key], bo[key], big)
        assert abs(bs["P_PR"] - bo["P_PR"]) <= 1e-6 * abs(bo["P_PR"])

    pressures_close(sim.barostat_state(), orc.barostat_state())
    sim.step(1)
    orc.step(1)
    ex1, ep1 = _rel(sim.positions(), orc.positions()), _rel(sim.momenta(), orc.momenta())
    assert ex1 <= 1e-10 and ep1 <= 1e-7, (ex1, ep1)
    sim.step(9)
    orc.step(9)
    ex, ep = _rel(sim.positions(), orc.positions()), _rel(sim.momenta(), orc.momenta())
    assert ex <= 1e-6 and ep <= 1e-6, (ex, ep)
    bs, bo = sim.barostat_state(), orc.barostat_state()
    # the cell integrates the FP32-level virial: its bar is that of the positions it scales
    assert _rel(bs["box"], bo["box"]) <= 1e-6
    assert abs(bs["v_W"] - bo["v_W"]) <= 1e-4 * max(abs(bo["v_W"]), 1e-3)
    assert bo["V"] != float(np.prod(wb["box"]))
    pressures_close(bs, bo)
    assert abs(bs["enthalpy"] - bo["enthalpy"]) <= 1e-6 * sim.N * sim.P
    sim.close()


def test_barostat_argument_errors(pk):
    types, masses, x, p = _trap_system(5, 4, seed=1)
    sim = pk.PIMD(types, masses, [10.0] * 3, 4, 300.0, 1e-3, 0.0, seed=1)
    with pytest.raises(pk.PimdError):
        sim.barostat_state()                         # no barostat set
    with pytest.raises(pk.PimdError):
        sim.set_barostat(1.0, 0.0)                   # tau_p <= 0
    sim.set_barostat(1.0, 0.1)
    with pytest.raises(pk.PimdError):
        pk.pimd_set_integrator(sim.ctx, "obabo")     # BAOAB only (R-24)
    with pytest.raises(pk.PimdError):
        pk.pimd_set_fixcom(sim.ctx, True)
    sim.close()
    sim = pk.PIMD(types, masses, [10.0] * 3, 4, 300.0, 1e-3, 0.0, seed=1, integrator="obabo")
    with pytest.raises(pk.PimdError):
        sim.set_barostat(1.0, 0.1)
    sim.close()
