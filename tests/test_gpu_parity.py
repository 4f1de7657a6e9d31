"""GPU parity: the CUDA path (through the C ABI) against the oracle, element by element, on the same
seeded inputs.  Tolerances are north_star's: neighbour lists and Philox words bit-exact; force error
<= 1e-4 relative per component with the bead's F_rms as floor (DESIGN R-17); energy/atom <= 1e-6 eV;
x, p <= 1e-10 relative (max-norm) after one step with identical FP64 forces (harmonic model) and <= 1e-6
after 10 steps."""
import numpy as np
import pytest

import workloads
from oracle import philox, se_e2_a
from oracle.pimd import OraclePIMD

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pk():
    import paper_2602_13553_b200 as pk
    pk.lib()
    return pk


def _rel(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


def _random_system(N, P, seed, T=300.0):
    rng = np.random.default_rng(seed)
    types = rng.integers(0, 2, size=N).astype(np.int32)
    masses = np.array([15.9994, 1.008])
    x = rng.standard_normal((P, N, 3)) * 0.3
    p = rng.standard_normal((P, N, 3)) * np.sqrt(masses[types])[None, :, None] * 5.0
    return types, masses, x, p


# ---------------------------------------------------------------------------------------------
# Philox stream: bit-exact
# ---------------------------------------------------------------------------------------------
def test_philox_words_bit_exact_and_normals(pk):
    sim = pk.PIMD(np.zeros(4, np.int32), [1.0], [10.0] * 3, 4, 300.0, 1e-3, 1.0, seed=0x123456789ABCDEF)
    rng = np.random.default_rng(3)
    idx = np.stack([rng.integers(0, 64, 4096), rng.integers(0, 1 << 22, 4096), rng.integers(0, 3, 4096)], axis=1)
    for step in (0, 1, 12345678901):
        words, eta = pk.pimd_debug_noise(sim.ctx, step, idx)
        w = philox.words_for(0x123456789ABCDEF, step, idx[:, 0], idx[:, 1], idx[:, 2])
        for q in range(4):
            assert np.array_equal(words[:, q].astype(np.uint64), w[q])
        ref = philox.normal(0x123456789ABCDEF, step, idx[:, 0], idx[:, 1], idx[:, 2])
        assert np.abs(eta - ref).max() < 1e-13
    sim.close()


# ---------------------------------------------------------------------------------------------
# integrator alone (harmonic model: identical FP64 forces on both sides)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("P", [1, 2, 4, 8, 16, 32, 64])
@pytest.mark.parametrize("gamma", [0.0, 5.0])
def test_integrator_parity_harmonic(pk, P, gamma):
    N = 37                                           # 111 dofs: ragged tail of the 128-thread blocks
    types, masses, x, p = _random_system(N, P, seed=10 + P)
    ks = 2.5
    sim = pk.PIMD(types, masses, [30.0] * 3, P, 300.0, 0.25e-3, gamma, seed=99)
    sim.set_state(x, p)
    sim.set_model_harmonic(ks)
    orc = OraclePIMD(types, masses, [30.0] * 3, P, 300.0, 0.25e-3, gamma, seed=99)
    orc.set_state(x, p)
    orc.set_model_harmonic(ks)
    assert _rel(sim.momenta(), orc.momenta()) < 1e-13          # p -> v~ -> p round trip
    e0, o0 = sim.estimators(), orc.estimators()
    for key in ("K_PR", "K_CV", "H", "K_ring", "S_ring", "U_sum", "T_ring"):
        assert abs(e0[key] - o0[key]) <= 1e-11 * max(1.0, abs(o0[key])), key
    sim.step(1)
    orc.step(1)
    assert _rel(sim.positions(), orc.positions()) < 1e-10
    assert _rel(sim.momenta(), orc.momenta()) < 1e-10
    sim.step(9)
    orc.step(9)
    assert _rel(sim.positions(), orc.positions()) < 1e-6
    assert _rel(sim.momenta(), orc.momenta()) < 1e-6
    assert _rel(sim.positions(), orc.positions()) < 1e-11      # what the FP64 kernel actually reaches
    e, o = sim.estimators(), orc.estimators()
    assert e["step"] == 10
    for key in ("K_PR", "K_CV", "H", "K_ring", "S_ring", "U_sum", "T_ring"):
        assert abs(e[key] - o[key]) <= 1e-9 * max(1.0, abs(o[key])), key
    assert _rel(sim.forces(), orc.forces()) < 1e-11
    assert np.abs(sim.virial() - orc.virial()).max() < 1e-9 * np.abs(orc.virial()).max()
    sim.close()


@pytest.mark.parametrize("P", [1, 4, 32, 64])
@pytest.mark.parametrize("gamma", [0.0, 5.0])
def test_integrator_parity_harmonic_obabo(pk, P, gamma):
    """OBABO splitting in the same fused kernel: two half-step O's per
    launch, each with its own Philox stream; also split calls and a switch of the splitting mid-run."""
    N = 37
    types, masses, x, p = _random_system(N, P, seed=20 + P)
    ks = 2.5
    sim = pk.PIMD(types, masses, [30.0] * 3, P, 300.0, 0.25e-3, gamma, seed=99, integrator="obabo")
    sim.set_state(x, p)
    sim.set_model_harmonic(ks)
    orc = OraclePIMD(types, masses, [30.0] * 3, P, 300.0, 0.25e-3, gamma, seed=99, integrator="obabo")
    orc.set_state(x, p)
    orc.set_model_harmonic(ks)
    sim.step(1)
    orc.step(1)
    assert _rel(sim.positions(), orc.positions()) < 1e-10
    assert _rel(sim.momenta(), orc.momenta()) < 1e-10
    sim.step(4)
    sim.step(5)
    orc.step(9)
    assert _rel(sim.positions(), orc.positions()) < 1e-11
    assert _rel(sim.momenta(), orc.momenta()) < 1e-10
    e, o = sim.estimators(), orc.estimators()
    assert e["step"] == 10
    for key in ("K_PR", "K_CV", "H", "K_ring", "S_ring", "U_sum", "T_ring"):
        assert abs(e[key] - o[key]) <= 1e-9 * max(1.0, abs(o[key])), key
    # back to BAOAB for two steps: the oracle follows
    pk.pimd_set_integrator(sim.ctx, "baoab")
    orc.integrator = "baoab"
    sim.step(2)
    orc.step(2)
    assert _rel(sim.positions(), orc.positions()) < 1e-11
    assert _rel(sim.momenta(), orc.momenta()) < 1e-10
    with pytest.raises(pk.PimdError):
        pk.pimd_set_integrator(sim.ctx, 7)
    sim.close()


@pytest.mark.parametrize("integ", ["baoab", "obabo"])
@pytest.mark.parametrize("P", [1, 8, 32])
def test_fixcom_parity_and_zero_centroid_momentum(pk, integ, P):
    """fixcom (DESIGN R-19): two integrator launches per step (close + accumulate, subtract +
    estimators + open); trajectories follow the oracle and the total bead momentum vanishes after every step."""
    N = 301                                          # several 128-thread blocks and a ragged tail
    types, masses, x, p = _random_system(N, P, seed=40 + P)
    ks = 2.5
    args = (types, masses, [30.0] * 3, P, 300.0, 0.25e-3, 5.0)
    sim = pk.PIMD(*args, seed=7, integrator=integ, fixcom=True)
    sim.set_state(x, p)
    sim.set_model_harmonic(ks)
    orc = OraclePIMD(*args, seed=7, integrator=integ, fixcom=True)
    orc.set_state(x, p)
    orc.set_model_harmonic(ks)
    sim.step(1)
    orc.step(1)
    assert _rel(sim.positions(), orc.positions()) < 1e-10
    assert _rel(sim.momenta(), orc.momenta()) < 1e-10
    ptot = sim.momenta().sum(axis=(0, 1))
    assert np.abs(ptot).max() < 1e-10 * np.abs(sim.momenta()).max() * N ** 0.5
    sim.step(3)
    sim.step(2)
    orc.step(5)
    assert _rel(sim.positions(), orc.positions()) < 1e-10
    assert _rel(sim.momenta(), orc.momenta()) < 1e-9
    ptot = sim.momenta().sum(axis=(0, 1))
    assert np.abs(ptot).max() < 1e-10 * np.abs(sim.momenta()).max() * N ** 0.5
    e, o = sim.estimators(), orc.estimators()
    for key in ("K_PR", "K_CV", "H", "K_ring", "S_ring", "U_sum", "T_ring"):
        assert abs(e[key] - o[key]) <= 1e-9 * max(1.0, abs(o[key])), key
    sim.close()


def test_full_step_parity_config0_obabo(pk):
    cfg, wb, desc, w = workloads.make_config(0)
    args = (wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"])
    sim = pk.PIMD(*args, seed=11, model_desc=desc, integrator="obabo")
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    orc = OraclePIMD(*args, seed=11, integrator="obabo")
    orc.set_state(wb["x"], wb["p"])
    orc.set_model(desc, w)
    sim.step(1)
    orc.step(1)
    ex1, ep1 = _rel(sim.positions(), orc.positions()), _rel(sim.momenta(), orc.momenta())
    assert ex1 <= 1e-10 and ep1 <= 1e-10, (ex1, ep1)
    sim.step(4)
    orc.step(4)
    ex, ep = _rel(sim.positions(), orc.positions()), _rel(sim.momenta(), orc.momenta())
    assert ex <= 1e-6 and ep <= 1e-6, (ex, ep)
    sim.close()


@pytest.mark.parametrize("P", [16, 32, 64])
def test_four_lane_integrator_variant_parity(pk, P, monkeypatch):
    """north_star's layout (a group of four lanes owns the beads of an atom-dimension, shuffles for the transforms;
    integrator4.cu) is the measured A/B partner of the default kernel: same parity bar."""
    monkeypatch.setenv("PIMD_INT4", "1")
    N = 37
    types, masses, x, p = _random_system(N, P, seed=70 + P)
    args = (types, masses, [30.0] * 3, P, 300.0, 0.25e-3, 5.0)
    sim = pk.PIMD(*args, seed=99)
    sim.set_state(x, p)
    sim.set_model_harmonic(2.5)
    orc = OraclePIMD(*args, seed=99)
    orc.set_state(x, p)
    orc.set_model_harmonic(2.5)
    sim.step(1)
    orc.step(1)
    assert _rel(sim.positions(), orc.positions()) < 1e-10 and _rel(sim.momenta(), orc.momenta()) < 1e-10
    sim.step(9)
    orc.step(9)
    assert _rel(sim.positions(), orc.positions()) < 1e-11 and _rel(sim.momenta(), orc.momenta()) < 1e-10
    e, o = sim.estimators(), orc.estimators()
    for key in ("K_PR", "K_CV", "H", "K_ring", "S_ring"):
        assert abs(e[key] - o[key]) <= 1e-9 * max(1.0, abs(o[key])), key
    sim.close()


def test_estimator_history_every_step(pk):
    N, P = 50, 8
    types, masses, x, p = _random_system(N, P, seed=5)
    sim = pk.PIMD(types, masses, [30.0] * 3, P, 300.0, 0.25e-3, 2.0, seed=1)
    sim.set_state(x, p)
    sim.set_model_harmonic(1.0)
    orc = OraclePIMD(types, masses, [30.0] * 3, P, 300.0, 0.25e-3, 2.0, seed=1)
    orc.set_state(x, p)
    orc.set_model_harmonic(1.0)
    sim.step(5)
    hist = sim.estimator_history()
    assert [h["step"] for h in hist] == [1, 2, 3, 4, 5]
    for h in hist:
        orc.step(1)
        o = orc.estimators()
        for key in ("K_PR", "K_CV", "H"):
            assert abs(h[key] - o[key]) <= 1e-9 * max(1.0, abs(o[key]))
    sim.close()


def test_step_loop_is_replayed_as_a_cuda_graph_and_matches_plain_launches(pk):
    """pimd_step(n >= 3) with the se_e2_a model replays one captured {integrator, force evaluation} sequence; the
    trajectory and the per-step estimator history equal those of step(1) calls (plain launches) to rounding."""
    cfg, wb, desc, w = workloads.make_config(0)
    args = (wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"])
    a = pk.PIMD(*args, seed=3, model_desc=desc)
    a.set_state(wb["x"], wb["p"])
    a.set_model(w)
    assert pk.pimd_debug_graph_state(a.ctx) == 0
    a.step(6)
    assert pk.pimd_debug_graph_state(a.ctx) == 1
    b = pk.PIMD(*args, seed=3, model_desc=desc)
    b.set_state(wb["x"], wb["p"])
    b.set_model(w)
    hb = []
    for _ in range(6):
        b.step(1)
        hb.append(b.estimators())
    assert pk.pimd_debug_graph_state(b.ctx) == 0
    # Two runs of the same kernels differ by the order of their FP32 / FP64 atomic sums (T_i, F_j): ~1e-6 relative on a force
    # of ~2e-4 eV/A, i.e. ~1e-9 on a momentum of 10..100 per kick -- a few 1e-11 relative after six steps (1.1e-11 seen).  The
    # bound leaves a factor ten for that noise and stays four orders under north_star's 1e-6 for ten steps.
    assert _rel(a.positions(), b.positions()) < 1e-11 and _rel(a.momenta(), b.momenta()) < 1e-10
    ha = a.estimator_history()
    assert [h["step"] for h in ha] == [1, 2, 3, 4, 5, 6]
    for x, y in zip(ha, hb):
        assert abs(x["K_CV"] - y["K_CV"]) <= 1e-9 * abs(y["K_CV"])
        assert abs(x["H"] - y["H"]) <= 1e-7 * abs(y["H"])          # U is an FP32-network sum accumulated by atomics
    a.step(4)                                             # the graph is reused by the next call
    assert a.estimators()["step"] == 10
    a.close()
    b.close()


def test_split_calls_equal_one_call_bitwise(pk):
    """step(3)+step(4) == step(7): the noise is keyed by the absolute step counter (R-10)."""
    N, P = 20, 4
    types, masses, x, p = _random_system(N, P, seed=8)
    outs = []
    for plan in ((7,), (3, 4)):
        sim = pk.PIMD(types, masses, [30.0] * 3, P, 300.0, 0.5e-3, 1.0, seed=4)
        sim.set_state(x, p)
        sim.set_model_harmonic(3.0)
        for n in plan:
            sim.step(n)
        outs.append((sim.positions(), sim.momenta()))
        sim.close()
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])


# ---------------------------------------------------------------------------------------------
# neighbour lists: bit-exact sets
# ---------------------------------------------------------------------------------------------
def _oracle_rows(x, types, box, rcut):
    ri, rj, rn, _ = se_e2_a.neighbours_bruteforce(x, box, rcut)
    tj = np.asarray(types)[rj]
    order = np.lexsort((rn[:, 2], rn[:, 1], rn[:, 0], rj, tj, ri))
    return ri[order], rj[order], rn[order]


@pytest.mark.parametrize("cfg_idx,beads", [(0, (0, 1, 2, 3)), (1, (0, 31))])
def test_neighbour_lists_bit_exact(pk, cfg_idx, beads):
    cfg, wb, desc, w = workloads.make_config(cfg_idx)
    sim = pk.PIMD(wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"], seed=0,
                  model_desc=desc)
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    for k in beads:
        count, j, shift = sim.neighbors(k)
        ri, rj, rn = _oracle_rows(wb["x"][k], wb["types"], wb["box"], desc["rcut"])
        assert np.array_equal(count, np.bincount(ri, minlength=sim.N))
        assert np.array_equal(j, rj)
        assert np.array_equal(shift.astype(np.int64), rn)
    if cfg_idx == 0:
        assert (np.abs(shift).max() == 1)             # multi-image rows exist (box < 2 r_c)
    sim.close()


def test_neighbour_lists_bit_exact_config2_full_cell_grid(pk):
    """BASELINE.json configs[2] (the headline size): 4 cells per side, so the pruning of cells outside the cut-off
    sphere, the compacted non-empty-cell list and the flat candidate walk of neighbor_env_kernel all discriminate
    between cells.  Beads 0 and 31, every row (1536^2 x 27 FP64 distance tests per bead in the oracle)."""
    cfg, wb, desc, w = workloads.make_config(2)
    sim = pk.PIMD(wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"], seed=0,
                  model_desc=desc)
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    for k in (0, 31):
        count, j, shift = sim.neighbors(k)
        ri, rj, rn = _oracle_rows(wb["x"][k], wb["types"], wb["box"], desc["rcut"])
        assert np.array_equal(count, np.bincount(ri, minlength=sim.N))
        assert np.array_equal(j, rj)
        assert np.array_equal(shift.astype(np.int64), rn)
        assert np.abs(shift).max() == 1 and count.sum() > 120000
    sim.close()


def _rows_of_centres(count, j, shift, centres):
    """Slices of the library's concatenated canonical rows that belong to the given centres."""
    start = np.concatenate([[0], np.cumsum(count)])
    idx = np.concatenate([np.arange(start[i], start[i + 1]) for i in centres])
    return np.concatenate([np.full(count[i], i) for i in centres]), j[idx], shift[idx].astype(np.int64)


def test_neighbour_lists_bit_exact_config3_sampled_centres(pk):
    """configs[3] (12288 atoms, 8 cells per side): 96 sampled centres of beads 0 and 17 -- among them the atoms
    closest to the cell faces and box corners -- each compared with the brute-force rows of that centre."""
    cfg, wb, desc, w = workloads.make_config(3)
    sim = pk.PIMD(wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"], seed=0,
                  model_desc=desc)
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    rng = np.random.default_rng(33)
    L = wb["box"][0]
    for k in (0, 17):
        wk = wb["x"][k] - L * np.floor(wb["x"][k] / L)
        cw = L / 8.0
        face_dist = np.abs(((wk / cw) + 0.5) % 1.0 - 0.5).min(axis=1)           # distance to the nearest cell face
        near = np.argsort(face_dist)[:16]
        corner = np.argsort(np.abs(wk - L / 2).min(axis=1) * -1.0)[:16]            # closest to a box face
        centres = np.unique(np.concatenate([near, corner, rng.choice(sim.N, size=64, replace=False)]))
        count, j, shift = sim.neighbors(k)
        ri, rj, rn, _ = se_e2_a.neighbours_bruteforce(wb["x"][k], wb["box"], desc["rcut"], centres=centres)
        tj = np.asarray(wb["types"])[rj]
        order = np.lexsort((rn[:, 2], rn[:, 1], rn[:, 0], rj, tj, ri))
        gi, gj, gs = _rows_of_centres(count, j, shift, centres)
        assert np.array_equal(gi, ri[order]) and np.array_equal(gj, rj[order]) and np.array_equal(gs, rn[order])
    sim.close()


def test_neighbour_lists_bit_exact_orthorhombic_3x4x5_cells(pk):
    """A non-cubic box with a different number of cells per side (3, 4, 5) and different cell widths: the index
    arithmetic of the cell walk (strides, per-axis wrap and image code) is exercised per axis.  Jittered lattice of
    O/H sites at liquid-water number density; every row of both beads."""
    desc = workloads.model_desc()
    w = workloads.model_weights(desc, 4)
    box = np.array([3 * 6.2, 4 * 6.4, 5 * 6.05])
    g = np.array([9, 12, 14])                                # ~0.105 atoms / A^3
    rng = np.random.default_rng(12)
    idx = np.array([(a, b, c) for a in range(g[0]) for b in range(g[1]) for c in range(g[2])], dtype=np.float64)
    x1 = (idx + 0.5) * (box / g) + rng.uniform(-0.35, 0.35, size=idx.shape)
    N = x1.shape[0]
    types = (np.arange(N) % 3 != 0).astype(np.int32)
    rng.shuffle(types)
    P = 2
    x = x1[None] + 0.02 * rng.standard_normal((P, N, 3))
    x[1] += np.array([2 * box[0], -3 * box[1], box[2]])      # bead 1 sits several boxes away (unwrapped state)
    p = rng.standard_normal((P, N, 3))
    sim = pk.PIMD(types, [15.9994, 1.008], box, P, 300.0, 0.25e-3, 1.0, seed=1, model_desc=desc)
    sim.set_state(x, p)
    sim.set_model(w)
    for k in range(P):
        count, j, shift = sim.neighbors(k)
        ri, rj, rn = _oracle_rows(x[k], types, box, desc["rcut"])
        assert np.array_equal(count, np.bincount(ri, minlength=N))
        assert np.array_equal(j, rj) and np.array_equal(shift.astype(np.int64), rn)
        assert set(np.unique(shift[:, 0])) == {-1, 0, 1} and set(np.unique(shift[:, 2])) == {-1, 0, 1}
    # and the force path runs on that grid: forces of bead 0 against the oracle
    model = se_e2_a.Model(desc, w)
    Eo, Fo, Xio = se_e2_a.energy_forces(x[0], types, box, model)
    f = sim.forces()
    frms = np.sqrt((Fo ** 2).mean())
    assert (np.abs(f[0] - Fo) / np.maximum(np.abs(Fo), frms)).max() <= 1e-4
    sim.close()


def test_neighbours_atoms_far_outside_the_box_and_on_faces(pk):
    """Unwrapped coordinates several boxes away, and atoms exactly on the faces x = 0, x = L."""
    cfg, wb, desc, w = workloads.make_config(0)
    x = wb["x"].copy()
    L = wb["box"][0]
    x[:, 0::7] += np.array([3 * L, -2 * L, 5 * L])
    x[0, 3] = [0.0, L, 2 * L]
    x[0, 4] = [-1e-300, 0.5 * L, 0.25 * L]
    sim = pk.PIMD(wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"], seed=0,
                  model_desc=desc)
    sim.set_state(x, wb["p"])
    sim.set_model(w)
    count, j, shift = sim.neighbors(0)
    ri, rj, rn = _oracle_rows(x[0], wb["types"], wb["box"], desc["rcut"])
    assert np.array_equal(count, np.bincount(ri, minlength=sim.N))
    assert np.array_equal(j, rj) and np.array_equal(shift.astype(np.int64), rn)
    sim.close()


def test_isolated_atoms_empty_pair_types_and_single_atom_beads(pk):
    """Degenerate inputs of the force path: atoms with no neighbour at all (energy = the fitting net at D = 0,
    zero force), a centre type with no rows of one neighbour type, row tiles that are almost empty, P = 1."""
    desc = workloads.model_desc()
    w = workloads.model_weights(desc, 3, last_layer_scale=50.0)
    model = se_e2_a.Model(desc, w)
    box = np.array([60.0, 60.0, 60.0])
    # one water (3 atoms inside r_c of each other), one O-O pair, three isolated atoms (H, H, O)
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
        f, U, E = sim.forces(), sim.energies(), sim.atom_energies()
        for k in range(P):
            Eo, Fo, Xio = se_e2_a.energy_forces(x[k], types, box, model)
            assert np.abs(E[k] - Eo).max() <= 1e-6 * 50.0
            assert abs(U[k] - Eo.sum()) / 8 <= 1e-6 * 50.0
            scale = max(np.abs(Fo).max(), 1e-30)
            assert np.abs(f[k] - Fo).max() <= 1e-4 * scale
            assert np.all(f[k, 5:] == 0.0) and np.all(Fo[5:] == 0.0)          # isolated atoms feel nothing
        count, j, shift = sim.neighbors(0)
        assert list(count) == [2, 2, 2, 1, 1, 0, 0, 0]
        sim.step(2)                                                          # and the step runs on it
        assert np.all(np.isfinite(sim.positions()))
        sim.close()


def test_dilute_gas_many_centres_per_row_tile(pk):
    """A dilute system (about 4 neighbours per atom): a 128-row tile of the embedding kernels then spans ~30 centres,
    which takes the backward kernel's un-staged dT path and many short centre segments in the forward kernel."""
    desc = workloads.model_desc()
    w = workloads.model_weights(desc, 5)
    model = se_e2_a.Model(desc, w)
    rng = np.random.default_rng(17)
    N, L = 320, 40.0
    pts = []
    while len(pts) < N:                                  # random positions at least 1.1 A apart
        c = rng.uniform(0, L, 3)
        if all(np.linalg.norm((c - q + L / 2) % L - L / 2) > 1.1 for q in pts):
            pts.append(c)
    x1 = np.array(pts)
    types = (np.arange(N) % 3 != 0).astype(np.int32)     # O, H, H, ...
    P = 2
    x = x1[None] + 0.01 * rng.standard_normal((P, N, 3))
    p = rng.standard_normal((P, N, 3))
    box = np.array([L, L, L])
    sim = pk.PIMD(types, [15.9994, 1.008], box, P, 300.0, 0.5e-3, 1.0, seed=1, model_desc=desc)
    sim.set_state(x, p)
    sim.set_model(w)
    f, U, E = sim.forces(), sim.energies(), sim.atom_energies()
    counts = pk.pimd_get_neighbor_counts(sim.ctx, P, N, 2)
    assert counts.sum() / (P * N) < 12                   # dilute indeed
    for k in range(P):
        Eo, Fo, Xio = se_e2_a.energy_forces(x[k], types, box, model)
        frms = np.sqrt((Fo ** 2).mean())
        assert (np.abs(f[k] - Fo) / np.maximum(np.abs(Fo), frms)).max() <= 1e-4
        assert np.abs(E[k] - Eo).max() <= 1e-6
        assert abs(U[k] - Eo.sum()) / N <= 1e-6
    sim.close()


@pytest.mark.parametrize("N,sel,L", [(256, [46, 92], 15.0), (128, [32, 64], 14.0), (250, [40, 85], 15.5)])
def test_force_parity_power_of_two_atom_counts_and_other_sel(pk, N, sel, L):
    """The embedding kernels divide a slot index by N_sel and a bead-atom index by N with a host-made multiply-shift pair
    (embedding_tc.cu `fastdiv`); every BASELINE config has N = 3 x molecules and N_sel = 138.  Powers of two take the other
    branch of the constant's construction (m = 2^31), other N_sel other constants: forces and energies against the oracle."""
    desc = dict(workloads.model_desc(), sel=sel)
    w = workloads.model_weights(desc, 11)
    model = se_e2_a.Model(desc, w)
    rng = np.random.default_rng(N)
    pts = []                                             # box sizes keep the largest neighbour count under sel (asserted below)
    while len(pts) < N:                                  # random positions at least 1.3 A apart
        c = rng.uniform(0, L, 3)
        if all(np.linalg.norm((c - q + L / 2) % L - L / 2) > 1.3 for q in pts):
            pts.append(c)
    x1 = np.array(pts)
    types = (np.arange(N) % 3 != 0).astype(np.int32)
    P = 4
    x = x1[None] + 0.02 * rng.standard_normal((P, N, 3))
    p = rng.standard_normal((P, N, 3))
    box = np.array([L, L, L])
    sim = pk.PIMD(types, [15.9994, 1.008], box, P, 300.0, 0.5e-3, 1.0, seed=1, model_desc=desc)
    sim.set_state(x, p)
    sim.set_model(w, desc)
    f, U, E = sim.forces(), sim.energies(), sim.atom_energies()
    counts = pk.pimd_get_neighbor_counts(sim.ctx, P, N, 2)
    assert counts[..., 0].max() <= sel[0] and counts[..., 1].max() <= sel[1] and counts.sum() / (P * N) > 20
    for k in (0, P - 1):
        Eo, Fo, Xio = se_e2_a.energy_forces(x[k], types, box, model)
        frms = np.sqrt((Fo ** 2).mean())
        assert (np.abs(f[k] - Fo) / np.maximum(np.abs(Fo), frms)).max() <= 1e-4
        assert np.abs(E[k] - Eo).max() <= 1e-6
        assert abs(U[k] - Eo.sum()) / N <= 1e-6
    sim.close()


def test_sel_overflow_is_an_error(pk):
    cfg, wb, desc, w = workloads.make_config(0)
    small = dict(desc, sel=[8, 16])
    sim = pk.PIMD(wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"], seed=0,
                  model_desc=small)
    sim.set_state(wb["x"], wb["p"])
    with pytest.raises(pk.PimdError) as ei:
        sim.set_model(w, small)
    assert ei.value.code == pk.PIMD_ESEL_OVERFLOW
    sim.close()


def test_sel_overflow_inside_a_call_rolls_the_call_back(pk):
    """sel set to the largest neighbour counts of the initial configuration (32 O / 67 H): the oracle's trajectory
    overflows at step 2 (atom 17 gains a 33rd O neighbour).  pimd_step(5) must report that step and undo the WHOLE
    call -- not leave steps 3..5 integrated on truncated rows: x, p, f and the step counter are those at entry."""
    cfg, wb, desc, w = workloads.make_config(0)
    tight = dict(desc, sel=[32, 67])
    args = (wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"])
    orc = OraclePIMD(*args, seed=11)
    orc.set_state(wb["x"], wb["p"])
    orc.set_model(tight, w)
    orc.step(1)
    x1_oracle = orc.positions()
    with pytest.raises(OverflowError):
        orc.step(1)
    sim = pk.PIMD(*args, seed=11, model_desc=tight)
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w, tight)
    x0, p0, f0, U0 = sim.positions(), sim.momenta(), sim.forces(), sim.energies()
    with pytest.raises(pk.PimdError, match="step 2 of this call of 5 = absolute step 2") as ei:
        sim.step(5)
    assert ei.value.code == pk.PIMD_ESEL_OVERFLOW
    assert np.array_equal(sim.positions(), x0) and np.array_equal(sim.momenta(), p0)
    assert np.array_equal(sim.forces(), f0) and np.array_equal(sim.energies(), U0)
    assert sim.estimators()["step"] == 0
    sim.step(1)                                           # step 1 is fine and follows the oracle
    assert sim.estimators()["step"] == 1
    assert _rel(sim.positions(), x1_oracle) <= 1e-10
    x1 = sim.positions()
    with pytest.raises(pk.PimdError, match="step 1 of this call of 1 = absolute step 2"):
        sim.step(1)
    assert np.array_equal(sim.positions(), x1) and sim.estimators()["step"] == 1
    sim.close()


def test_operands_outside_the_fp16_split_range_are_errors_not_nans(pk):
    """The tensor-core kernels split operands into FP16 hi / lo pairs with fixed scales: a weight beyond +-1000 (or a
    non-finite one) is refused by pimd_set_model, and a pair of atoms closer than 0.01 A (s = 1/r > 100) is reported
    as PIMD_ECONTACT instead of producing inf / NaN forces."""
    desc = workloads.model_desc()
    w = workloads.model_weights(desc, 3)
    types = np.array([0, 1, 1], dtype=np.int32)
    x = np.array([[[5.0, 5.0, 5.0], [5.9, 5.2, 5.0], [4.8, 5.9, 5.1]]])
    for bad in (2.0e3, np.inf, np.nan):
        wb = w.copy()
        wb[30000] = bad
        sim = pk.PIMD(types, [15.9994, 1.008], [40.0] * 3, 1, 300.0, 0.5e-3, 1.0, seed=1, model_desc=desc)
        sim.set_state(x, np.zeros_like(x))
        with pytest.raises(pk.PimdError) as ei:
            sim.set_model(wb)
        assert ei.value.code == pk.PIMD_EINVAL and "weight 30000" in str(ei.value)
        sim.close()
    xc = x.copy()
    xc[0, 1] = xc[0, 0] + np.array([0.004, 0.0, 0.0])
    sim = pk.PIMD(types, [15.9994, 1.008], [40.0] * 3, 1, 300.0, 0.5e-3, 1.0, seed=1, model_desc=desc)
    sim.set_model(w)
    with pytest.raises(pk.PimdError) as ei:
        sim.set_state(xc, np.zeros_like(xc))
    assert ei.value.code == pk.PIMD_ECONTACT
    sim.set_state(x, np.zeros_like(x))                    # a sane configuration afterwards is accepted
    assert np.all(np.isfinite(sim.forces()))
    sim.close()


def test_binding_refuses_device_tensors_of_the_wrong_kind(pk):
    import torch
    types, masses, x, p = _random_system(10, 4, seed=2)
    sim = pk.PIMD(types, masses, [30.0] * 3, 4, 300.0, 1e-3, 1.0, seed=1)
    xd, pd = torch.from_numpy(x).cuda(), torch.from_numpy(p).cuda()
    with pytest.raises(ValueError, match="float64"):
        sim.set_state(xd.float(), pd)
    with pytest.raises(ValueError, match="contiguous"):
        sim.set_state(xd.transpose(0, 1), pd)
    with pytest.raises(ValueError, match="elements"):
        sim.set_state(xd[:2], pd)
    with pytest.raises(ValueError):
        sim.set_state(x[:2], p)
    sim.set_state(xd, pd)
    sim.set_model_harmonic(1.0)
    sim.step(1)
    sim.close()


# ---------------------------------------------------------------------------------------------
# force model
# ---------------------------------------------------------------------------------------------
def _force_checks(f, fo, U, Uo, Xi, Xio, E, Eo, N):
    frms = np.sqrt((fo ** 2).mean(axis=(1, 2), keepdims=True))
    err = np.abs(f - fo) / np.maximum(np.abs(fo), frms)
    assert err.max() <= 1e-4, "force error %.3e" % err.max()
    assert np.abs(U - Uo).max() / N <= 1e-6
    assert np.abs(E - Eo).max() <= 1e-6
    assert np.abs(Xi - Xio).max() <= 1e-4 * np.abs(Xio).max()
    return err.max()


@pytest.mark.parametrize("scale", [1.0, 1.0e3])
def test_force_energy_virial_parity_config0(pk, scale):
    cfg, wb, desc, _ = workloads.make_config(0)
    w = workloads.model_weights(desc, cfg["weight_seed"], last_layer_scale=scale)
    sim = pk.PIMD(wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"], seed=0,
                  model_desc=desc)
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    model = se_e2_a.Model(desc, w)
    P, N = cfg["P"], sim.N
    fo, Uo, Xio, Eo = np.zeros((P, N, 3)), np.zeros(P), np.zeros((P, 3, 3)), np.zeros((P, N))
    for k in range(P):
        E, F, Xi = se_e2_a.energy_forces(wb["x"][k], wb["types"], wb["box"], model)
        fo[k], Uo[k], Xio[k], Eo[k] = F, E.sum(), Xi, E
    tol_scale = scale                                   # energies scale with the last layer
    f, U, Xi, E = sim.forces(), sim.energies(), sim.virial(), sim.atom_energies()
    frms = np.sqrt((fo ** 2).mean(axis=(1, 2), keepdims=True))
    err = np.abs(f - fo) / np.maximum(np.abs(fo), frms)
    assert err.max() <= 1e-4, "force error %.3e" % err.max()
    assert np.abs(U - Uo).max() / N <= 1e-6 * tol_scale
    assert np.abs(E - Eo).max() <= 1e-6 * tol_scale
    assert np.abs(Xi - Xio).max() <= 1e-4 * np.abs(Xio).max()
    assert np.abs(f.sum(axis=1)).max() <= 1e-6 * np.abs(fo).max() * N ** 0.5     # Newton's third law
    sim.close()


def test_force_parity_config1_sampled_beads(pk):
    cfg, wb, desc, w = workloads.make_config(1)
    sim = pk.PIMD(wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"], seed=0,
                  model_desc=desc)
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    model = se_e2_a.Model(desc, w)
    f, U, Xi, E = sim.forces(), sim.energies(), sim.virial(), sim.atom_energies()
    for k in (0, 13, 31):
        Eo, Fo, Xio = se_e2_a.energy_forces(wb["x"][k], wb["types"], wb["box"], model)
        _force_checks(f[k:k + 1], Fo[None], U[k:k + 1], np.array([Eo.sum()]), Xi[k:k + 1], Xio[None], E[k], Eo, sim.N)
    sim.close()


def test_force_parity_config2_headline_size_sampled_beads(pk):
    """BASELINE.json's headline configuration (1536 atoms x 32 beads), in the launch configuration bench.py
    times; the oracle evaluates two sampled beads (a few seconds each)."""
    cfg, wb, desc, w = workloads.make_config(2)
    sim = pk.PIMD(wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"], seed=0,
                  model_desc=desc)
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    model = se_e2_a.Model(desc, w)
    f, U, Xi, E = sim.forces(), sim.energies(), sim.virial(), sim.atom_energies()
    for k in (0, 31):
        Eo, Fo, Xio = se_e2_a.energy_forces(wb["x"][k], wb["types"], wb["box"], model)
        _force_checks(f[k:k + 1], Fo[None], U[k:k + 1], np.array([Eo.sum()]), Xi[k:k + 1], Xio[None], E[k], Eo, sim.N)
    # properties that hold for every bead at any size: Newton's third law, symmetric virial
    assert np.abs(f.sum(axis=1)).max() <= 1e-6 * np.abs(f).max() * sim.N ** 0.5
    X3 = Xi.reshape(-1, 3, 3)
    assert np.abs(X3 - np.swapaxes(X3, 1, 2)).max() <= 1e-5 * np.abs(X3).max()
    sim.close()


def test_force_parity_config2_strong_model_one_bead(pk):
    """configs[2] with the last fitting layer scaled by 10^3 (forces ~0.2 eV/A: every term of the backward pass
    matters; the x1 random-init model gives 2e-4 eV/A).  Energies scale with the layer, so their bound is the
    relative one of DESIGN R-17: 1e-6 eV/atom per unit of last-layer scale."""
    cfg, wb, desc, _ = workloads.make_config(2)
    w = workloads.model_weights(desc, cfg["weight_seed"], last_layer_scale=1.0e3)
    sim = pk.PIMD(wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"], seed=0,
                  model_desc=desc)
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    model = se_e2_a.Model(desc, w)
    f, U, Xi, E = sim.forces(), sim.energies(), sim.virial().reshape(-1, 3, 3), sim.atom_energies()
    k = 19
    Eo, Fo, Xio = se_e2_a.energy_forces(wb["x"][k], wb["types"], wb["box"], model)
    frms = np.sqrt((Fo ** 2).mean())
    assert frms > 0.05                                    # the force matters
    err = np.abs(f[k] - Fo) / np.maximum(np.abs(Fo), frms)
    assert err.max() <= 1e-4, "force error %.3e" % err.max()
    assert abs(U[k] - Eo.sum()) / sim.N <= 1e-6 * 1.0e3
    assert np.abs(E[k] - Eo).max() <= 1e-6 * 1.0e3
    assert np.abs(Xi[k] - Xio).max() <= 1e-4 * np.abs(Xio).max()
    sim.close()


@pytest.mark.slow
def test_config1_as_specified_100_steps_estimators_every_step(pk):
    """BASELINE.json configs[1] as north_star states it: 64 H2O x 32 beads, the se_e2_a model, 100 steps in ONE
    pimd_step(100) call, and the primitive (Eq. A7) and centroid-virial (Eq. A9) kinetic-energy
    estimators of EVERY step (L86-88) against the oracle's (3200 bead evaluations of 192 atoms on the CPU).
    x, p <= 1e-6 at step 10 (north_star) and at step 100."""
    cfg, wb, desc, w = workloads.make_config(1)
    assert cfg["P"] == 32 and cfg["steps"] == 100
    args = (wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"])
    sim = pk.PIMD(*args, seed=5, model_desc=desc)
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    from _parallel_oracle import ParallelOraclePIMD     # the oracle, one bead per worker process
    orc = ParallelOraclePIMD(*args, seed=5)
    orc.set_state(wb["x"], wb["p"])
    orc.set_model(desc, w)
    # the first ten steps in a call of their own: positions and momenta at step 10
    sim10 = pk.PIMD(*args, seed=5, model_desc=desc)
    sim10.set_state(wb["x"], wb["p"])
    sim10.set_model(w)
    sim10.step(10)
    sim.step(100)
    hist = sim.estimator_history()
    assert [h["step"] for h in hist] == list(range(1, 101))
    worst = {"K_PR": 0.0, "K_CV": 0.0, "H": 0.0}
    for n, h in enumerate(hist, start=1):
        orc.step(1)
        o = orc.estimators()
        for key in ("K_PR", "K_CV"):
            rel = abs(h[key] - o[key]) / abs(o[key])
            worst[key] = max(worst[key], rel)
            assert rel <= 1e-6, (n, key, h[key], o[key])
        dH = abs(h["H"] - o["H"]) / (sim.N * sim.P)
        worst["H"] = max(worst["H"], dH)
        assert dH <= 1e-6, (n, h["H"], o["H"])                              # eV per bead-atom
        assert abs(h["T_ring"] - o["T_ring"]) <= 1e-6 * o["T_ring"]
        if n == 10:
            ex, ep = _rel(sim10.positions(), orc.positions()), _rel(sim10.momenta(), orc.momenta())
            assert ex <= 1e-6 and ep <= 1e-6, (ex, ep)
            print("configs[1] step 10: rel err x %.2e p %.2e" % (ex, ep))
    ex, ep = _rel(sim.positions(), orc.positions()), _rel(sim.momenta(), orc.momenta())
    print("configs[1] step 100: rel err x %.2e p %.2e; worst per-step K_PR %.2e K_CV %.2e H/bead-atom %.2e eV"
          % (ex, ep, worst["K_PR"], worst["K_CV"], worst["H"]))
    assert ex <= 1e-6 and ep <= 1e-6, (ex, ep)
    e, o = sim.estimators(), orc.estimators()
    assert e["step"] == 100 and abs(e["K_CV"] - o["K_CV"]) <= 1e-6 * abs(o["K_CV"])
    orc.close()
    sim.close()
    sim10.close()


# ---------------------------------------------------------------------------------------------
# the whole step, configs[0]
# ---------------------------------------------------------------------------------------------
def test_full_step_parity_config0(pk):
    cfg, wb, desc, w = workloads.make_config(0)
    args = (wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"])
    sim = pk.PIMD(*args, seed=11, model_desc=desc)
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    orc = OraclePIMD(*args, seed=11)
    orc.set_state(wb["x"], wb["p"])
    orc.set_model(desc, w)
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
    assert abs(e["K_PR"] - o["K_PR"]) <= 1e-6 * abs(o["K_PR"])
    assert abs(e["H"] - o["H"]) <= 1e-6 * sim.N * sim.P
    sim.close()


# ---------------------------------------------------------------------------------------------
# tensor-core GEMM kernel alone (3xTF32 on tcgen05) against the FP64 product
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("M,N,K", [(256, 240, 16), (300, 240, 1600), (1000, 240, 240), (417, 1600, 240), (5, 160, 48)])
def test_tc_gemm_3xtf32_matches_fp64_product(pk, M, N, K):
    rng = np.random.default_rng(M + N + K)
    A = rng.standard_normal((M, K)).astype(np.float32)
    Bt = (rng.standard_normal((N, K)) / np.sqrt(K)).astype(np.float32)
    sim = pk.PIMD(np.zeros(4, np.int32), [1.0], [10.0] * 3, 4, 300.0, 1e-3, 1.0, seed=0)
    C = pk.pimd_debug_gemm(sim.ctx, A, Bt)
    ref = A.astype(np.float64) @ Bt.astype(np.float64).T
    err = np.abs(C - ref).max() / np.abs(ref).max()
    assert err < 3e-5, err          # FP32-class (K = 1600: 1.1e-5); single-pass TF32 gives ~1e-3
    sim.close()


def test_tensor_core_and_cuda_core_fitting_paths_agree(pk):
    cfg, wb, desc, w = workloads.make_config(0)
    w = workloads.model_weights(desc, cfg["weight_seed"], last_layer_scale=1.0e3)
    out = []
    for use_tc in (1, 0):
        sim = pk.PIMD(wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"], seed=0,
                      model_desc=desc)
        sim.set_model(w)
        pk.pimd_set_fitting_path(sim.ctx, use_tc)
        sim.set_state(wb["x"], wb["p"])
        out.append((sim.forces(), sim.atom_energies()))
        sim.close()
    frms = np.sqrt((out[1][0] ** 2).mean())
    assert np.abs(out[0][0] - out[1][0]).max() <= 2e-5 * frms
    assert np.abs(out[0][1] - out[1][1]).max() <= 1e-6 * 1e3


def test_tensor_core_and_cuda_core_embedding_paths_agree(pk):
    """embedding_tc.cu (tcgen05, 3xTF32, fast tanh) against the FP32 CUDA-core embedding kernels: forces, atom
    energies and virial of configs[0] (multi-image neighbours, ragged last tiles of all four type pairs)."""
    cfg, wb, desc, w = workloads.make_config(0)
    w = workloads.model_weights(desc, cfg["weight_seed"], last_layer_scale=1.0e3)
    out = []
    for use_tc in (1, 0):
        sim = pk.PIMD(wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"], seed=0,
                      model_desc=desc)
        sim.set_model(w)
        pk.pimd_set_embedding_path(sim.ctx, use_tc)
        sim.set_state(wb["x"], wb["p"])
        out.append((sim.forces(), sim.atom_energies(), sim.virial()))
        sim.close()
    frms = np.sqrt((out[1][0] ** 2).mean())
    assert np.abs(out[0][0] - out[1][0]).max() <= 5e-5 * frms
    assert np.abs(out[0][1] - out[1][1]).max() <= 1e-6 * 1e3
    assert np.abs(out[0][2] - out[1][2]).max() <= 5e-5 * np.abs(out[1][2]).max()


# ---------------------------------------------------------------------------------------------
# `method pimd`: integration in Cartesian coordinates (Eq. D3)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("integ", ["baoab", "obabo"])
@pytest.mark.parametrize("P", [1, 2, 8, 32, 64])
@pytest.mark.parametrize("gamma", [0.0, 5.0])
def test_cartesian_method_parity_harmonic(pk, P, gamma, integ):
    N = 37
    types, masses, x, p = _random_system(N, P, seed=40 + P)
    ks = 2.5
    args = (types, masses, [30.0] * 3, P, 300.0, 0.1e-3, gamma)
    sim = pk.PIMD(*args, seed=99, integrator=integ, method="pimd")
    sim.set_state(x, p)
    sim.set_model_harmonic(ks)
    orc = OraclePIMD(*args, seed=99, integrator=integ, method="pimd")
    orc.set_state(x, p)
    orc.set_model_harmonic(ks)
    assert _rel(sim.momenta(), orc.momenta()) < 1e-15
    e0, o0 = sim.estimators(), orc.estimators()
    for key in ("K_PR", "K_CV", "H", "K_ring", "S_ring", "U_sum", "T_ring"):
        assert abs(e0[key] - o0[key]) <= 1e-11 * max(1.0, abs(o0[key])), key
    sim.step(1)
    orc.step(1)
    assert _rel(sim.positions(), orc.positions()) < 1e-10
    assert _rel(sim.momenta(), orc.momenta()) < 1e-10
    sim.step(9)
    orc.step(9)
    assert _rel(sim.positions(), orc.positions()) < 1e-10
    assert _rel(sim.momenta(), orc.momenta()) < 1e-9
    e, o = sim.estimators(), orc.estimators()
    assert e["step"] == 10
    for key in ("K_PR", "K_CV", "H", "K_ring", "S_ring", "U_sum", "T_ring"):
        assert abs(e[key] - o[key]) <= 1e-9 * max(1.0, abs(o[key])), key
    sim.close()


def test_cartesian_method_full_step_parity_config0(pk):
    cfg, wb, desc, w = workloads.make_config(0)
    args = (wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], 0.1e-3, cfg["gamma"])
    sim = pk.PIMD(*args, seed=11, model_desc=desc, method="pimd")
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    orc = OraclePIMD(*args, seed=11, method="pimd")
    orc.set_state(wb["x"], wb["p"])
    orc.set_model(desc, w)
    sim.step(1)
    orc.step(1)
    ex1, ep1 = _rel(sim.positions(), orc.positions()), _rel(sim.momenta(), orc.momenta())
    assert ex1 <= 1e-10 and ep1 <= 1e-10, (ex1, ep1)
    sim.step(9)
    orc.step(9)
    ex, ep = _rel(sim.positions(), orc.positions()), _rel(sim.momenta(), orc.momenta())
    assert ex <= 1e-6 and ep <= 1e-6, (ex, ep)
    e, o = sim.estimators(), orc.estimators()
    assert abs(e["K_CV"] - o["K_CV"]) <= 1e-6 * abs(o["K_CV"])
    assert abs(e["H"] - o["H"]) <= 1e-6 * sim.N * sim.P
    sim.close()


@pytest.mark.parametrize("integ", ["baoab", "obabo"])
@pytest.mark.parametrize("P", [1, 8, 32])
def test_cartesian_method_fixcom_removes_every_beads_momentum(pk, integ, P):
    """fixcom under `method pimd` ("for each bead individually"): trajectories follow the oracle and the
    total momentum of every bead vanishes after every step."""
    N = 301
    types, masses, x, p = _random_system(N, P, seed=60 + P)
    args = (types, masses, [30.0] * 3, P, 300.0, 0.1e-3, 5.0)
    sim = pk.PIMD(*args, seed=7, integrator=integ, fixcom=True, method="pimd")
    sim.set_state(x, p)
    sim.set_model_harmonic(2.5)
    orc = OraclePIMD(*args, seed=7, integrator=integ, fixcom=True, method="pimd")
    orc.set_state(x, p)
    orc.set_model_harmonic(2.5)
    sim.step(1)
    orc.step(1)
    assert _rel(sim.positions(), orc.positions()) < 1e-10 and _rel(sim.momenta(), orc.momenta()) < 1e-10
    pb = sim.momenta().sum(axis=1)
    assert np.abs(pb).max() < 1e-10 * np.abs(sim.momenta()).max() * N ** 0.5
    sim.step(3)
    sim.step(2)
    orc.step(5)
    assert _rel(sim.positions(), orc.positions()) < 1e-10 and _rel(sim.momenta(), orc.momenta()) < 1e-9
    pb = sim.momenta().sum(axis=1)
    assert np.abs(pb).max() < 1e-10 * np.abs(sim.momenta()).max() * N ** 0.5
    e, o = sim.estimators(), orc.estimators()
    for key in ("K_PR", "K_CV", "H", "K_ring", "S_ring"):
        assert abs(e[key] - o[key]) <= 1e-9 * max(1.0, abs(o[key])), key
    sim.close()


def test_cartesian_method_argument_rules(pk):
    types, masses, x, p = _random_system(5, 4, seed=1)
    sim = pk.PIMD(types, masses, [30.0] * 3, 4, 300.0, 1e-4, 1.0, seed=1)
    sim.set_state(x, p)
    sim.set_model_harmonic(1.0)
    pk.pimd_set_method(sim.ctx, "pimd")
    with pytest.raises(pk.PimdError):
        sim.step(1)                                  # the change of representation dropped the state
    with pytest.raises(pk.PimdError):
        sim.set_barostat(1.0, 0.1)
    with pytest.raises(pk.PimdError):
        pk.pimd_set_method(sim.ctx, 7)
    sim.set_state(x, p)
    sim.step(2)
    sim.close()


# ---------------------------------------------------------------------------------------------
# the largest configuration: outputs of sampled atoms, one by one
# ---------------------------------------------------------------------------------------------
def _cluster_energy_force(xb, types, box, model, i, rcut):
    """E_i and F_i of atom i of one bead from the oracle on the cluster of all atom images within 2 r_c of it
    (E_j of every j within r_c of i then has its complete environment, so F_i = -dU/dx_i is exact), placed in
    the middle of a huge non-periodic cell."""
    L = np.asarray(box, dtype=np.float64)
    w = xb - L * np.floor(xb / L)
    shifts = np.array([(a, b, c) for a in (-1, 0, 1) for b in (-1, 0, 1) for c in (-1, 0, 1)], dtype=np.float64) * L
    rel = (w[:, None, :] - w[i][None, None, :]) + shifts[None, :, :]          # [N, 27, 3]
    r2 = (rel ** 2).sum(axis=2)
    jj, ss = np.nonzero(r2 < (2.0 * rcut) ** 2)
    order = np.argsort(r2[jj, ss], kind="stable")                              # the centre itself (r = 0) first
    jj, ss = jj[order], ss[order]
    assert jj[0] == i and r2[jj[0], ss[0]] == 0.0
    E, F, _ = se_e2_a.energy_forces(rel[jj, ss] + 500.0, np.asarray(types)[jj], [1000.0] * 3, model)
    return E[0], F[0], len(jj)


def test_force_parity_config3_largest_size_sampled_atoms(pk):
    """BASELINE.json configs[3] (12288 atoms x 32 beads = 393,216 bead-atoms, the largest NVT configuration, in the
    launch configuration bench.py --config 3 times): E_i and F_i of sampled atoms of two beads against the oracle."""
    cfg, wb, desc, w = workloads.make_config(3)
    sim = pk.PIMD(wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"], seed=0,
                  model_desc=desc)
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    model = se_e2_a.Model(desc, w)
    f, E = sim.forces(), sim.atom_energies()
    rng = np.random.default_rng(3)
    for k in (0, 31):
        frms = np.sqrt((f[k] ** 2).mean())
        for i in rng.choice(sim.N, size=4, replace=False):
            Eo, Fo, n_cluster = _cluster_energy_force(wb["x"][k], wb["types"], wb["box"], model, int(i), desc["rcut"])
            assert n_cluster > 500
            assert abs(E[k, i] - Eo) <= 1e-6
            err = np.abs(f[k, i] - Fo) / np.maximum(np.abs(Fo), frms)
            assert err.max() <= 1e-4, "force error %.3e" % err.max()
    assert np.abs(f.sum(axis=1)).max() <= 1e-6 * np.abs(f).max() * sim.N ** 0.5     # Newton's third law, every bead
    X3 = sim.virial().reshape(-1, 3, 3)
    assert np.abs(X3 - np.swapaxes(X3, 1, 2)).max() <= 1e-5 * np.abs(X3).max()
    sim.close()
