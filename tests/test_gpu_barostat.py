"""GPU parity of the isotropic BZP barostat (Appendix E, Eq. A10-A17) through the
C ABI against oracle/barostat.py + oracle/pimd.py, on the same seeded inputs.  Tolerances: x, p, cell and v_W
<= 1e-10 relative after one step with FP64 forces (harmonic model), <= 1e-6 after 10 steps (north_star's integrator
bar); with the se_e2_a model the FP32-level forces and virial set the bar (1e-6 on x, p after 10 steps;
pressures to 1e-4 of their largest term)."""
import numpy as np
import pytest

import workloads
from oracle import barostat, nm, se_e2_a
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
    assert np.abs(bs["v_W3"] - bo["v_W3"]).max() <= tol * max(np.abs(bo["v_W3"]).max(), 1e-3)
    assert np.abs(bs["P_CV3"] - bo["P_CV3"]).max() <= tol * max(np.abs(bo["P_CV3"]).max(), abs(bo["P_MD"]))


@pytest.mark.parametrize("aniso", [False, True])
@pytest.mark.parametrize("integ", ["baoab", "obabo"])
@pytest.mark.parametrize("P", [1, 4, 32, 64])
@pytest.mark.parametrize("gamma", [0.0, 20.0])
def test_barostat_parity_harmonic(pk, P, gamma, integ, aniso):
    N = 43                                           # 129 dofs: one full 128-thread block and a tail of one
    types, masses, x, p = _trap_system(N, P, seed=20 + P)
    box = [10.0, 11.0, 12.0]
    p_ext = 2.0 * KB * 300.0 / 1320.0 * BAR
    args = (types, masses, box, P, 300.0, 1.0e-3, gamma)
    sim = pk.PIMD(*args, seed=5, integrator=integ)
    sim.set_state(x, p)
    sim.set_model_harmonic(0.5)
    sim.set_barostat(p_ext, 0.05, aniso=aniso)
    orc = OraclePIMD(*args, seed=5, integrator=integ)
    orc.set_barostat(p_ext, 0.05, aniso=aniso)
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
    assert (np.ptp(bo["v_W3"]) > 0) == aniso
    e, o = sim.estimators(), orc.estimators()
    for key in ("K_PR", "K_CV", "H", "K_ring", "S_ring", "U_sum"):
        assert abs(e[key] - o[key]) <= 1e-9 * max(1.0, abs(o[key])), key
    sim.close()


@pytest.mark.parametrize("aniso", [False, True])
@pytest.mark.parametrize("integ", ["baoab", "obabo"])
def test_nph_enthalpy_is_conserved_on_the_gpu(pk, integ, aniso):
    """Eq. A17 over 2000 steps of the CUDA path alone (a property that holds at any size)."""
    P, N = 8, 64
    types, masses, x, p = _trap_system(N, P, seed=3)
    sim = pk.PIMD(types, masses, [10.0] * 3, P, 300.0, 0.5e-3, 0.0, seed=1, integrator=integ)
    sim.set_state(x, p)
    sim.set_model_harmonic(0.5)
    sim.set_barostat(KB * 300.0 / 1000.0 * BAR, 0.05, aniso=aniso)
    h0 = sim.barostat_state()["enthalpy"]
    dev = []
    for _ in range(20):
        sim.step(100)
        dev.append(sim.barostat_state()["enthalpy"] - h0)
    assert np.abs(dev).max() < 5e-4 * abs(h0)
    assert abs(sim.barostat_state()["V"] / 1000.0 - 1.0) > 0.01
    sim.close()


@pytest.mark.parametrize("integ", ["baoab", "obabo"])
def test_npt_ideal_gas_samples_the_isobaric_volume_distribution(pk, integ):
    """Free particles (harmonic model with k = 0) under NpT: the cell force is sum m v~0^2 - 3 n V P_ext + 3 n k_B T,
    whose stationary volume distribution is V^N exp(-P_ext V / k_B T), so <V> = (N + 1) k_B T / P_ext and
    <K_W> = n k_B T / 2 -- a statistical check of E1's n k_B T term (R-20), E4-E7 and the thermostats together
    (N rather than N + 1 would be 12.5 % off at N = 8; the tolerance is 4 sigma of the measured block error)."""
    N, P, T = 8, 4, 300.0
    rng = np.random.default_rng(0)
    types = np.zeros(N, dtype=np.int32)
    masses = np.array([15.9994])
    x = rng.uniform(0.0, 10.0, size=(1, N, 3)) + 0.05 * rng.standard_normal((P, N, 3))
    p = rng.standard_normal((P, N, 3)) * np.sqrt(P * KB * T * masses[0] / MVV2E)
    p_ext = (N + 1) * KB * T / 1000.0                                  # eV/A^3: <V> = 1000 A^3
    sim = pk.PIMD(types, masses, [10.0] * 3, P, T, 2.0e-3, 20.0, seed=7, integrator=integ)
    sim.set_state(x, p)
    sim.set_model_harmonic(0.0)
    sim.set_barostat(p_ext * BAR, 0.05)
    sim.step(2000)
    V, KW = [], []
    for _ in range(3000):
        sim.step(100)
        b = sim.barostat_state()
        V.append(b["V"]); KW.append(b["K_W"])
    V, KW = np.asarray(V), np.asarray(KW)
    blocks = V.reshape(30, 100).mean(axis=1)
    err = blocks.std(ddof=1) / np.sqrt(len(blocks))
    assert err < 0.02 * 1000.0
    assert abs(V.mean() - 1000.0) < 4.0 * err, (V.mean(), err)
    kb = KW.reshape(30, 100).mean(axis=1)
    assert abs(KW.mean() - 0.5 * P * KB * T) < 4.0 * kb.std(ddof=1) / np.sqrt(len(kb)), KW.mean()
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


@pytest.mark.parametrize("integ,aniso", [("baoab", False), ("obabo", False), ("baoab", True), ("obabo", True)])
def test_full_npt_step_parity_config0(pk, integ, aniso):
    """configs[0] geometry and model under NpT at 1 bar (configs[4]'s ensemble at the size the oracle finishes):
    multi-image neighbours from a cell that changes every step.  OBABO + npt is the paper's own example command
    (PAPER.md:L82)."""
    cfg, wb, desc, w = workloads.make_config(0)
    args = (wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"])
    sim = pk.PIMD(*args, seed=11, model_desc=desc, integrator=integ)
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    sim.set_barostat(1.0, 0.02, aniso=aniso)
    orc = OraclePIMD(*args, seed=11, integrator=integ)
    orc.set_barostat(1.0, 0.02, aniso=aniso)
    orc.set_state(wb["x"], wb["p"])
    orc.set_model(desc, w)

    def pressures_close(bs, bo):
        # A12's three terms nearly cancel; the FP32-level virial bounds the error by 1e-4 of the largest term
        trXi = np.trace(orc.virial(), axis1=1, axis2=2).sum()
        big = abs(trXi) / (3.0 * bo["V"]) * BAR
        for key in ("P_CV", "P_MD"):
            assert abs(bs[key] - bo[key]) <= 1e-4 * max(big, abs(bo[key])), (key, bs[key], bo[key], big)
        assert np.abs(bs["P_CV3"] - bo["P_CV3"]).max() <= 1e-4 * max(big, np.abs(bo["P_CV3"]).max())
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
    assert np.abs(bs["v_W3"] - bo["v_W3"]).max() <= 1e-4 * max(np.abs(bo["v_W3"]).max(), 1e-3)
    assert bo["V"] != float(np.prod(wb["box"])) and (np.ptp(bo["box"]) > 0) == aniso
    pressures_close(bs, bo)
    assert abs(bs["enthalpy"] - bo["enthalpy"]) <= 1e-6 * sim.N * sim.P
    sim.close()


@pytest.mark.parametrize("squeeze", [False, True])
def test_neighbour_lists_bit_exact_in_the_rescaled_cell(pk, squeeze):
    """After the barostat has moved the cell (expanding at 1 bar under the random-weight model's pressure, or
    squeezed by a target far above it), the neighbour rows of the last force evaluation are exactly the brute-force
    rows of the oracle at the positions and cell the getters return (wrap, images and cutoff all use the new L)."""
    cfg, wb, desc, w = workloads.make_config(0)
    sim = pk.PIMD(wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"], seed=2,
                  model_desc=desc)
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    sim.set_barostat(1.0, 0.02)
    if squeeze:
        sim.set_barostat(sim.barostat_state()["P_CV"] + 1.0e5, 0.02)
    for _ in range(12):                               # stop between 0.5 % and a few % of linear change
        sim.step(2)
        bs = sim.barostat_state()
        if abs(bs["box"][0] / wb["box"][0] - 1.0) > 5e-3:
            break
    assert (bs["box"][0] < wb["box"][0] * 0.995) if squeeze else (bs["box"][0] > wb["box"][0] * 1.005)
    x = sim.positions()
    for k in (0, 3):
        count, j, shift = sim.neighbors(k)
        ri, rj, rn, _ = se_e2_a.neighbours_bruteforce(x[k], bs["box"], desc["rcut"])
        tj = np.asarray(wb["types"])[rj]
        order = np.lexsort((rn[:, 2], rn[:, 1], rn[:, 0], rj, tj, ri))
        assert np.array_equal(count, np.bincount(ri, minlength=sim.N))
        assert np.array_equal(j, rj[order])
        assert np.array_equal(shift.astype(np.int64), rn[order])
    sim.close()


def _squeezed_config1(pk, seed):
    cfg, wb, desc, w = workloads.make_config(1, n_beads=4)      # L = 12.42: two cells of 6.21 A per side, R = 1
    sim = pk.PIMD(wb["types"], wb["masses"], wb["box"], 4, cfg["T"], cfg["dt"], cfg["gamma"], seed=seed, model_desc=desc)
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    sim.set_barostat(1.0, 0.02)
    sim.set_barostat(sim.barostat_state()["P_CV"] + 1.0e5, 0.02)
    return sim, wb, desc


def test_cell_grid_follows_a_shrinking_cell_across_calls(pk):
    """The cell grid is fixed at pimd_set_model; once the cell is below 2 x 6 A the walk range must grow to two
    cells (refit at every API call): rows stay bit-exact."""
    sim, wb, desc = _squeezed_config1(pk, 3)
    for _ in range(200):
        sim.step(2)
        bs = sim.barostat_state()
        if bs["box"][0] < 11.9:
            break
    assert bs["box"][0] < 11.9
    x = sim.positions()
    count, j, shift = sim.neighbors(1)
    ri, rj, rn, _ = se_e2_a.neighbours_bruteforce(x[1], bs["box"], desc["rcut"])
    order = np.lexsort((rn[:, 2], rn[:, 1], rn[:, 0], rj, np.asarray(wb["types"])[rj], ri))
    assert np.array_equal(count, np.bincount(ri, minlength=sim.N))
    assert np.array_equal(j, rj[order]) and np.array_equal(shift.astype(np.int64), rn[order])
    sim.close()


def test_cell_shrinking_past_the_grid_margin_inside_one_call_is_an_error(pk):
    """... and the failed call is undone as a whole (positions, momenta, cell, step counter), so the caller can go on
    with fewer steps per call."""
    sim, wb, desc = _squeezed_config1(pk, 3)
    x0, p0, b0 = sim.positions(), sim.momenta(), sim.barostat_state()
    with pytest.raises(pk.PimdError, match="cell shrank|more neighbours") as ei:
        sim.step(400)
    assert "rolled back" in str(ei.value)
    b1 = sim.barostat_state()
    assert np.array_equal(sim.positions(), x0) and np.array_equal(sim.momenta(), p0)
    assert np.array_equal(b1["box"], b0["box"]) and b1["v_W"] == b0["v_W"] and sim.estimators()["step"] == 0
    sim.step(2)
    assert sim.estimators()["step"] == 2
    sim.close()


def test_npt_config4_full_size_sampled(pk):
    """BASELINE.json configs[4] (6144 atoms x 64 beads, NpT) in the launch configuration bench.py times, with a
    fast cell (tau_p 0.02 ps) so that it moves in three steps.  The oracle cannot step this size; it (a) recomputes
    Eq. A12 from the state the getters return, (b) evaluates one sampled bead at the RESCALED cell."""
    cfg, wb, desc, w = workloads.make_config(4)
    P = cfg["P"]
    sim = pk.PIMD(wb["types"], wb["masses"], wb["box"], P, cfg["T"], cfg["dt"], cfg["gamma"], seed=0, model_desc=desc)
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    sim.set_barostat(cfg["p_ext_bar"], 0.02)
    sim.step(3)
    bs = sim.barostat_state()
    assert abs(bs["box"][0] / wb["box"][0] - 1.0) > 1e-5 and np.isfinite(bs["enthalpy"])
    np.testing.assert_allclose(bs["V"], np.prod(bs["box"]), rtol=1e-15)
    x, p, f, Xi = sim.positions(), sim.momenta(), sim.forces(), sim.virial().reshape(P, 3, 3)
    m = wb["masses"][wb["types"]]
    M = nm.nm_matrix(P)
    vt, ft = nm.to_nm(M, p / m[None, :, None]), nm.to_nm(M, f)
    pcv = barostat.p_cv(x, vt, ft, Xi, m, bs["V"]) * BAR
    big = abs(np.trace(Xi, axis1=1, axis2=2).sum()) / (3.0 * P * bs["V"]) * BAR
    assert abs(bs["P_CV"] - pcv) <= 1e-9 * max(big, abs(pcv)), (bs["P_CV"], pcv, big)
    e = sim.estimators()
    assert abs(bs["P_MD"] - barostat.p_md(e["K_ring"], Xi, bs["V"]) * BAR) <= 1e-9 * max(big * P, abs(bs["P_MD"]))
    assert abs(bs["P_PR"] - barostat.p_pr(e["S_ring"], P, sim.N, cfg["T"], bs["V"]) * BAR) <= 1e-9 * abs(bs["P_PR"])
    # forces and virial of a sampled bead at the cell the barostat produced
    model = se_e2_a.Model(desc, w)
    k = 37
    Eo, Fo, Xio, parts = se_e2_a.energy_forces(x[k], wb["types"], bs["box"], model, return_parts=True)
    frms = np.sqrt((Fo ** 2).mean())
    err = np.abs(f[k] - Fo) / np.maximum(np.abs(Fo), frms)
    assert err.max() <= 1e-4, "force error %.3e" % err.max()
    assert np.abs(Xi[k] - Xio).max() <= 1e-4 * np.abs(Xio).max()
    assert abs(sim.energies()[k] - Eo.sum()) / sim.N <= 1e-6
    # the neighbour rows of that bead in the moved cell (6 cells per side, the cell read from the device), row for
    # row against the brute-force rows the oracle has just used (all 6144 centres)
    count, j, shift = sim.neighbors(k)
    ri, rj, rn = parts["ri"], parts["rj"], parts["rn"]
    order = np.lexsort((rn[:, 2], rn[:, 1], rn[:, 0], rj, np.asarray(wb["types"])[rj], ri))
    assert np.array_equal(count, np.bincount(ri, minlength=sim.N))
    assert np.array_equal(j, rj[order]) and np.array_equal(shift.astype(np.int64), rn[order])
    sim.close()


@pytest.mark.parametrize("aniso", [False, True])
def test_checkpoint_resume_under_the_barostat(pk, aniso):
    """{x, p, f, U, step} + {cell, v_W, virials} restored into a fresh context continue the NpT trajectory (to the
    rounding of a call boundary): counter-based noise for atoms and cell alike."""
    N, P = 50, 8
    types, masses, x, p = _trap_system(N, P, seed=9)
    args = (types, masses, [10.0, 10.5, 11.0], P, 300.0, 1e-3, 20.0)
    ref = pk.PIMD(*args, seed=4)
    ref.set_state(x, p)
    ref.set_model_harmonic(0.5)
    ref.set_barostat(40.0, 0.05, aniso=aniso)
    ref.step(3)
    ck = dict(x=ref.positions(), p=ref.momenta(), f=ref.forces(), U=ref.energies(), xi=ref.virial(),
              b=ref.barostat_state())
    ref.step(3)
    sim = pk.PIMD(*args, seed=4)
    sim.set_model_harmonic(0.5)
    sim.set_barostat(40.0, 0.05, aniso=aniso)
    sim.restore_cell(ck["b"]["box"], ck["b"]["v_W3"], ck["xi"])
    pk.pimd_restore(sim.ctx, ck["x"], ck["p"], ck["f"], ck["U"], 3)
    b0 = sim.barostat_state()
    assert abs(b0["P_CV"] - ck["b"]["P_CV"]) <= 1e-12 * abs(ck["b"]["P_MD"])
    assert abs(b0["enthalpy"] - ck["b"]["enthalpy"]) <= 1e-12 * abs(ck["b"]["enthalpy"])
    sim.step(3)
    assert _rel(sim.positions(), ref.positions()) < 1e-12 and _rel(sim.momenta(), ref.momenta()) < 1e-12
    bs, br = sim.barostat_state(), ref.barostat_state()
    assert _rel(bs["box"], br["box"]) < 1e-14 and np.abs(bs["v_W3"] - br["v_W3"]).max() < 1e-12 * np.abs(br["v_W3"]).max()
    assert sim.estimators()["step"] == 6
    ref.close(); sim.close()


@pytest.mark.parametrize("integ,aniso", [("baoab", False), ("obabo", True)])
def test_barostat_history_every_step(pk, integ, aniso):
    """Appendix A outputs 8-15 of EVERY step of one pimd_step call against the oracle stepped one by one."""
    N, P = 30, 4
    types, masses, x, p = _trap_system(N, P, seed=12)
    args = (types, masses, [10.0, 10.5, 11.0], P, 300.0, 1e-3, 20.0)
    sim = pk.PIMD(*args, seed=6, integrator=integ)
    sim.set_state(x, p)
    sim.set_model_harmonic(0.5)
    sim.set_barostat(40.0, 0.05, aniso=aniso)
    orc = OraclePIMD(*args, seed=6, integrator=integ)
    orc.set_barostat(40.0, 0.05, aniso=aniso)
    orc.set_state(x, p)
    orc.set_model_harmonic(0.5)
    sim.step(7)
    hist = sim.barostat_history()
    assert len(hist) == 7
    for q in range(7):
        orc.step(1)
        _compare_state(hist[q], orc.barostat_state(), 1e-9)
    last = sim.barostat_state()
    for key in ("v_W", "V", "P_CV", "P_PR", "P_MD", "K_W", "U_W", "J_W", "enthalpy"):
        assert hist[-1][key] == last[key], key
    assert len(sim.barostat_history(cap=3)) == 3
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
        pk.pimd_set_fixcom(sim.ctx, True)            # not with a barostat (R-24)
    sim.close()
    sim = pk.PIMD(types, masses, [10.0] * 3, 4, 300.0, 1e-3, 0.0, seed=1, fixcom=True)
    with pytest.raises(pk.PimdError):
        sim.set_barostat(1.0, 0.1)
    sim.close()
