"""GPU parity of the compressed (tabulated) embedding path -- SURVEY 8(f) NEXT-3, PAPER.md:L76 / L262, DESIGN R-28 --
against the oracle's compressed model (oracle/compress.py), through the C ABI.  Same tolerances as the MLP path
(north_star: force 1e-4 with the bead's F_rms as floor, energy 1e-6 eV/atom, x and p 1e-10 after one step, 1e-6 after
ten), now RELATIVE TO THE COMPRESSED ORACLE: the table is an approximation of the MLP, so the MLP oracle is not the
reference here (the distance between the two models is checked separately)."""
import numpy as np
import pytest

import workloads
from oracle import compress, se_e2_a
from oracle.pimd import OraclePIMD

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pk():
    import paper_2602_13553_b200 as pk
    pk.lib()
    return pk


def _rel(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


def _sim(pk, cfg, wb, desc, w, seed=0, **kw):
    sim = pk.PIMD(wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"], seed=seed,
                  model_desc=desc, **kw)
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    sim.set_compressed(True)
    return sim


@pytest.mark.parametrize("scale", [1.0, 1.0e3])
def test_compressed_force_energy_virial_parity_config0_all_beads(pk, scale):
    cfg, wb, desc, _ = workloads.make_config(0)
    w = workloads.model_weights(desc, cfg["weight_seed"], last_layer_scale=scale)
    sim = _sim(pk, cfg, wb, desc, w)
    model = compress.compress(se_e2_a.Model(desc, w))
    P, N = cfg["P"], sim.N
    f, U, Xi, E = sim.forces(), sim.energies(), sim.virial(), sim.atom_energies()
    for k in range(P):
        Eo, Fo, Xio = se_e2_a.energy_forces(wb["x"][k], wb["types"], wb["box"], model)
        frms = np.sqrt((Fo ** 2).mean())
        err = np.abs(f[k] - Fo) / np.maximum(np.abs(Fo), frms)
        assert err.max() <= 1e-4, "bead %d force error %.3e" % (k, err.max())
        assert abs(U[k] - Eo.sum()) / N <= 1e-6 * scale
        assert np.abs(E[k] - Eo).max() <= 1e-6 * scale
        assert np.abs(Xi[k] - Xio).max() <= 1e-4 * np.abs(Xio).max()
    assert np.abs(f.sum(axis=1)).max() <= 1e-6 * np.abs(f).max() * N ** 0.5       # Newton's third law
    sim.close()


def test_compressed_force_parity_config2_sampled_beads(pk):
    """The headline size in the launch configuration bench.py --compressed times; x1000 model so the force matters."""
    cfg, wb, desc, _ = workloads.make_config(2)
    w = workloads.model_weights(desc, cfg["weight_seed"], last_layer_scale=1.0e3)
    sim = _sim(pk, cfg, wb, desc, w)
    model = compress.compress(se_e2_a.Model(desc, w))
    f, U, Xi, E = sim.forces(), sim.energies(), sim.virial().reshape(-1, 3, 3), sim.atom_energies()
    for k in (0, 31):
        Eo, Fo, Xio = se_e2_a.energy_forces(wb["x"][k], wb["types"], wb["box"], model)
        frms = np.sqrt((Fo ** 2).mean())
        err = np.abs(f[k] - Fo) / np.maximum(np.abs(Fo), frms)
        assert err.max() <= 1e-4, "force error %.3e" % err.max()
        assert abs(U[k] - Eo.sum()) / sim.N <= 1e-6 * 1.0e3
        assert np.abs(E[k] - Eo).max() <= 1e-6 * 1.0e3
        assert np.abs(Xi[k] - Xio).max() <= 1e-4 * np.abs(Xio).max()
    assert np.abs(f.sum(axis=1)).max() <= 1e-6 * np.abs(f).max() * sim.N ** 0.5
    sim.close()


def test_compressed_full_step_parity_config0(pk):
    cfg, wb, desc, w = workloads.make_config(0)
    sim = _sim(pk, cfg, wb, desc, w, seed=11)
    args = (wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"])
    orc = OraclePIMD(*args, seed=11)
    orc.set_state(wb["x"], wb["p"])
    orc.set_model(desc, w, compressed=True)
    sim.step(1)
    orc.step(1)
    ex1, ep1 = _rel(sim.positions(), orc.positions()), _rel(sim.momenta(), orc.momenta())
    assert ex1 <= 1e-10 and ep1 <= 1e-10, (ex1, ep1)
    sim.step(9)
    orc.step(9)
    ex, ep = _rel(sim.positions(), orc.positions()), _rel(sim.momenta(), orc.momenta())
    assert ex <= 1e-6 and ep <= 1e-6, (ex, ep)
    e, o = sim.estimators(), orc.estimators()
    assert e["step"] == 10
    assert abs(e["K_CV"] - o["K_CV"]) <= 1e-6 * abs(o["K_CV"])
    assert abs(e["H"] - o["H"]) <= 1e-6 * sim.N * sim.P
    sim.close()


def test_compressed_model_is_close_to_the_mlp_model_and_switches_back(pk):
    """R-28's table error (|G~ - G| <= 3e-8) shows up as a force difference far below the parity tolerance; switching the
    table off returns exactly the MLP path's forces."""
    cfg, wb, desc, _ = workloads.make_config(0)
    w = workloads.model_weights(desc, cfg["weight_seed"], last_layer_scale=1.0e3)
    sim = pk.PIMD(wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"], seed=0,
                  model_desc=desc)
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    f_mlp, E_mlp = sim.forces(), sim.atom_energies()
    sim.set_compressed(True)
    f_tab, E_tab = sim.forces(), sim.atom_energies()
    frms = np.sqrt((f_mlp ** 2).mean())
    assert 0 < np.abs(f_tab - f_mlp).max() <= 3e-5 * frms          # both FP32-class; the table itself adds ~1e-6
    assert np.abs(E_tab - E_mlp).max() <= 1e-6 * 1.0e3
    sim.set_compressed(False)
    assert np.abs(sim.forces() - f_mlp).max() <= 5e-6 * frms        # the MLP path again (FP32 / FP64 atomics order only)
    sim.close()


def test_compressed_degenerate_inputs_and_dilute_gas(pk):
    """Atoms without neighbours, a centre type with no rows of one neighbour type, tiles that are almost empty; and a
    dilute gas (few rows per centre: most moment buckets empty, the k-step skipping of the forward kernel)."""
    desc = workloads.model_desc()
    w = workloads.model_weights(desc, 3, last_layer_scale=50.0)
    model = compress.compress(se_e2_a.Model(desc, w))
    box = np.array([60.0, 60.0, 60.0])
    x1 = np.array([[5.0, 5.0, 5.0], [5.9, 5.2, 5.0], [4.8, 5.9, 5.1],
                   [30.0, 30.0, 30.0], [32.5, 30.0, 30.5],
                   [50.0, 10.0, 10.0], [10.0, 50.0, 10.0], [10.0, 10.0, 50.0]])
    types = np.array([0, 1, 1, 0, 0, 1, 1, 0], dtype=np.int32)
    for P in (1, 4):
        rng = np.random.default_rng(P)
        x = x1[None] + 0.01 * rng.standard_normal((P, 8, 3))
        p = rng.standard_normal((P, 8, 3))
        sim = pk.PIMD(types, [15.9994, 1.008], box, P, 300.0, 0.5e-3, 1.0, seed=1, model_desc=desc)
        sim.set_state(x, p)
        sim.set_model(w)
        sim.set_compressed(True)
        f, U, E = sim.forces(), sim.energies(), sim.atom_energies()
        for k in range(P):
            Eo, Fo, _ = se_e2_a.energy_forces(x[k], types, box, model)
            assert np.abs(E[k] - Eo).max() <= 1e-6 * 50.0
            assert np.abs(f[k] - Fo).max() <= 1e-4 * max(np.abs(Fo).max(), 1e-30)
            assert np.all(f[k, 5:] == 0.0)
        sim.step(2)
        assert np.all(np.isfinite(sim.positions()))
        sim.close()
    # dilute gas
    w = workloads.model_weights(desc, 5)
    model = compress.compress(se_e2_a.Model(desc, w))
    rng = np.random.default_rng(17)
    N, L = 320, 40.0
    pts = []
    while len(pts) < N:
        c = rng.uniform(0, L, 3)
        if all(np.linalg.norm((c - q + L / 2) % L - L / 2) > 1.1 for q in pts):
            pts.append(c)
    x = np.array(pts)[None] + 0.01 * rng.standard_normal((2, N, 3))
    types = (np.arange(N) % 3 != 0).astype(np.int32)
    sim = pk.PIMD(types, [15.9994, 1.008], [L] * 3, 2, 300.0, 0.5e-3, 1.0, seed=1, model_desc=desc)
    sim.set_state(x, rng.standard_normal((2, N, 3)))
    sim.set_model(w)
    sim.set_compressed(True)
    f, E = sim.forces(), sim.atom_energies()
    for k in range(2):
        Eo, Fo, _ = se_e2_a.energy_forces(x[k], types, [L] * 3, model)
        frms = np.sqrt((Fo ** 2).mean())
        assert (np.abs(f[k] - Fo) / np.maximum(np.abs(Fo), frms)).max() <= 1e-4
        assert np.abs(E[k] - Eo).max() <= 1e-6
    sim.close()


def test_compressed_row_outside_the_table_is_an_error(pk):
    """Two atoms 0.4 A apart: s = 1/r = 2.5 > 2.  The oracle raises; the library returns PIMD_ETABLE_RANGE."""
    desc = workloads.model_desc()
    w = workloads.model_weights(desc, 3)
    x = np.array([[[5.0, 5.0, 5.0], [5.4, 5.0, 5.0], [9.0, 9.0, 9.0]]])
    types = np.array([0, 1, 1], dtype=np.int32)
    model = compress.compress(se_e2_a.Model(desc, w))
    with pytest.raises(OverflowError):
        se_e2_a.energy_forces(x[0], types, [40.0] * 3, model)
    sim = pk.PIMD(types, [15.9994, 1.008], [40.0] * 3, 1, 300.0, 0.5e-3, 1.0, seed=1, model_desc=desc)
    sim.set_state(x, np.zeros_like(x))
    sim.set_model(w)                                    # the MLP path accepts the pair (s = 1/r below r_s)
    with pytest.raises(pk.PimdError) as ei:
        sim.set_compressed(True)
    assert ei.value.code == pk.PIMD_ETABLE_RANGE
    sim.close()
    sim = pk.PIMD(types, [15.9994, 1.008], [40.0] * 3, 1, 300.0, 0.5e-3, 1.0, seed=1)
    with pytest.raises(pk.PimdError) as ei:
        sim.set_compressed(True)                        # no model yet
    assert ei.value.code == pk.PIMD_ENOMODEL
    sim.close()
