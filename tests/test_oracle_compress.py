"""Pins of oracle/compress.py (tabulated embedding, PAPER.md:L76 / ref. 41; DESIGN R-28)."""
import numpy as np
import pytest

import workloads
from oracle import compress, se_e2_a


@pytest.fixture(scope="module")
def c0():
    cfg, wb, desc, w = workloads.make_config(0)
    return wb, desc, w


def test_forward_mode_derivatives_match_finite_differences(c0):
    _, desc, w = c0
    layers = se_e2_a.Model(desc, w).emb[(0, 1)]
    s = np.array([0.013, 0.4, 0.77, 1.3, 1.95])
    G, G1, G2 = compress.mlp_value_d1_d2(layers, s)
    Gref, _ = se_e2_a._mlp_forward(layers, s[:, None], se_e2_a._embed_rule)
    np.testing.assert_allclose(G, Gref, rtol=1e-14, atol=1e-15)
    e = 1e-4
    Gp, _, _ = compress.mlp_value_d1_d2(layers, s + e)
    Gm, _, _ = compress.mlp_value_d1_d2(layers, s - e)
    np.testing.assert_allclose(G1, (Gp - Gm) / (2 * e), rtol=0, atol=1e-7 * np.abs(G1).max())
    np.testing.assert_allclose(G2, (Gp - 2 * G + Gm) / (e * e), rtol=0, atol=2e-6 * max(np.abs(G2).max(), 1.0))


def test_table_matches_value_and_two_derivatives_at_both_nodes(c0):
    _, desc, w = c0
    layers = se_e2_a.Model(desc, w).emb[(1, 0)]
    tab = compress.build_table(layers)
    assert tab["n"] == 40 and tab["coef"].shape == (40, 6, 100)
    nodes = tab["s_lo"] + tab["h"] * np.arange(tab["n"] + 1)
    y, y1, y2 = compress.mlp_value_d1_d2(layers, nodes)
    c, h = tab["coef"], tab["h"]
    np.testing.assert_allclose(c[:, 0], y[:-1], rtol=0, atol=1e-15)
    np.testing.assert_allclose(c[:, 1], y1[:-1], rtol=0, atol=1e-15)
    np.testing.assert_allclose(2 * c[:, 2], y2[:-1], rtol=0, atol=1e-14)
    p = np.array([h ** k for k in range(6)])
    np.testing.assert_allclose(np.einsum("npm,p->nm", c, p), y[1:], rtol=0, atol=1e-13)
    dp = np.array([k * h ** (k - 1) if k else 0.0 for k in range(6)])
    np.testing.assert_allclose(np.einsum("npm,p->nm", c, dp), y1[1:], rtol=0, atol=1e-12)
    ddp = np.array([k * (k - 1) * h ** (k - 2) if k > 1 else 0.0 for k in range(6)])
    np.testing.assert_allclose(np.einsum("npm,p->nm", c, ddp), y2[1:], rtol=0, atol=1e-10)


def test_table_error_is_sixth_order_and_small(c0):
    _, desc, w = c0
    layers = se_e2_a.Model(desc, w).emb[(0, 0)]
    s = np.random.default_rng(0).uniform(0.0, 2.0, size=4000)
    G, G1, _ = compress.mlp_value_d1_d2(layers, s)
    errs = []
    for h in (0.1, 0.05):
        Gt, Gpt = compress.table_eval(compress.build_table(layers, h=h), s)
        errs.append(np.abs(Gt - G).max())
        assert np.abs(Gpt - G1).max() < 50 * errs[-1] / h
    assert errs[1] < 6e-8                                  # at the stride of R-28: below FP32 rounding of an O(1) value
    assert errs[1] < errs[0] / 30.0                        # ~ 2^6


def test_rows_outside_the_table_are_an_error(c0):
    _, desc, w = c0
    tab = compress.build_table(se_e2_a.Model(desc, w).emb[(0, 0)])
    with pytest.raises(OverflowError):
        compress.table_eval(tab, np.array([2.0001]))
    with pytest.raises(OverflowError):
        compress.table_eval(tab, np.array([-1e-9]))
    G, _ = compress.table_eval(tab, np.array([0.0, 2.0]))   # both ends belong to the table
    assert np.isfinite(G).all()


def test_compressed_model_is_close_to_the_mlp_and_its_forces_are_its_own_gradient(c0):
    wb, desc, w = c0
    w = workloads.model_weights(desc, 0, last_layer_scale=1.0e3)
    x = wb["x"][0]
    full = se_e2_a.Model(desc, w)
    comp = compress.compress(se_e2_a.Model(desc, w))
    E0, F0, Xi0 = se_e2_a.energy_forces(x, wb["types"], wb["box"], full)
    E1, F1, Xi1 = se_e2_a.energy_forces(x, wb["types"], wb["box"], comp)
    assert np.abs(E1 - E0).max() < 1e-6 * max(1.0, np.abs(E0).max())
    assert np.abs(F1 - F0).max() < 1e-6 * np.abs(F0).max()
    # forces = -dU/dx of the COMPRESSED energy (central differences)
    for (i, a) in [(0, 0), (17, 2), (55, 1)]:
        xp, xm = x.copy(), x.copy()
        xp[i, a] += 1e-5
        xm[i, a] -= 1e-5
        Up = se_e2_a.energy_forces(xp, wb["types"], wb["box"], comp)[0].sum()
        Um = se_e2_a.energy_forces(xm, wb["types"], wb["box"], comp)[0].sum()
        assert F1[i, a] == pytest.approx(-(Up - Um) / 2e-5, rel=2e-6, abs=1e-7 * np.abs(F1).max())
