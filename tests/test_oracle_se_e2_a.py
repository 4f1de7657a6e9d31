"""Pins for oracle/se_e2_a.py (CPU only).

The paper prints no equation for the Deep-Potential model, so the forward
architecture is "parity unpinned" against physics (DESIGN R-11..R-16).  What CAN be pinned, and is
here: the neighbour search against an independent k-d tree over explicit replicas; the analytic
backward against central finite differences and against torch float64 autograd of a dense,
differently organised forward; the invariances the descriptor must have; the virial of
PAPER.md:L372 against -dU/d(strain); continuity at r_c; a two-atom case computed by hand.
"""
import math

import numpy as np
import pytest

import workloads as wl
from oracle import se_e2_a


@pytest.fixture(scope="module")
def c0():
    cfg, wb, desc, w = wl.make_config(0)
    # last fitting layer x1e3 so that forces are eV/A-scale and every term of the backward matters
    w = wl.model_weights(desc, cfg["weight_seed"], last_layer_scale=1.0e3)
    model = se_e2_a.Model(desc, w)
    x = wb["x"][0]
    E, F, Xi, parts = se_e2_a.energy_forces(x, wb["types"], wb["box"], model, return_parts=True)
    return dict(cfg=cfg, wb=wb, desc=desc, w=w, model=model, x=x, E=E, F=F, Xi=Xi, parts=parts)


# ------------------------------------------------------------------------------- weights / packing
def test_weight_count_matches_the_architecture():
    desc = wl.model_desc()
    # 4 embedding nets (1*25+25 + 25*50+50 + 50*100+100 = 6450) + 2 fitting nets (500,161)
    assert se_e2_a.Model.n_weights(desc) == 4 * 6450 + 2 * 500161 == 1026122
    with pytest.raises(ValueError):
        se_e2_a.Model(desc, np.zeros(10))


def test_packing_order_embedding_then_fitting():
    desc = wl.model_desc()
    w = np.arange(se_e2_a.Model.n_weights(desc), dtype=np.float64)
    m = se_e2_a.Model(desc, w)
    W1, b1 = m.emb[(0, 0)][0]
    assert W1.shape == (1, 25) and W1[0, 0] == 0.0 and b1[0] == 25.0
    W1, _ = m.emb[(0, 1)][0]
    assert W1[0, 0] == 6450.0                       # second ordered type pair follows the first
    W1, _ = m.emb[(1, 0)][0]
    assert W1[0, 0] == 2 * 6450.0
    Wf, bf = m.fitnet[0][0]
    assert Wf.shape == (1600, 240) and Wf[0, 0] == 4 * 6450.0 and Wf[0, 1] == 4 * 6450.0 + 1   # row-major in x out
    W4, b4 = m.fitnet[1][3]
    assert W4.shape == (240, 1) and b4[0] == w.size - 1


# ------------------------------------------------------------------------------- neighbours
def _kdtree_rows(x, L, rcut):
    """Independent neighbour search: replicate the wrapped box explicitly and use scipy's k-d tree."""
    from scipy.spatial import cKDTree
    N = x.shape[0]
    w = x - L * np.floor(x / L)
    s = int(math.ceil(rcut / L))
    shifts = [(a, b, c) for a in range(-s, s + 1) for b in range(-s, s + 1) for c in range(-s, s + 1)]
    rep = np.concatenate([w + np.array(sh) * L for sh in shifts])
    tree = cKDTree(rep)
    rows = set()
    for i in range(N):
        for q in tree.query_ball_point(w[i], rcut * (1 + 1e-9)):
            j, n = q % N, shifts[q // N]
            if j == i and n == (0, 0, 0):
                continue
            d = (w[j] - w[i]) + np.array(n) * L
            if (d[0] * d[0] + d[1] * d[1]) + d[2] * d[2] < rcut * rcut:
                rows.add((i, j) + n)
    return rows


@pytest.mark.parametrize("idx", [0, 1])
def test_neighbours_match_kdtree_over_replicas(idx):
    cfg, wb, desc, w = wl.make_config(idx, n_beads=1)
    x, L = wb["x"][0], cfg["box"]
    ri, rj, rn, d = se_e2_a.neighbours_bruteforce(x, wb["box"], desc["rcut"])
    got = set(zip(ri.tolist(), rj.tolist(), rn[:, 0].tolist(), rn[:, 1].tolist(), rn[:, 2].tolist()))
    assert len(got) == ri.size
    assert got == _kdtree_rows(x, L, desc["rcut"])
    # symmetric: (i, j, n) present <=> (j, i, -n) present
    assert got == {(j, i, -a, -b, -c) for (i, j, a, b, c) in got}
    if idx == 0:
        # L = 9.86 < 2 r_c: some ordered pairs see each other through several images
        pairs = {}
        for (i, j, a, b, c) in got:
            pairs[(i, j)] = pairs.get((i, j), 0) + 1
        assert sum(1 for v in pairs.values() if v >= 2) > 500
    else:
        assert len({(i, j) for (i, j, *_n) in got}) == len(got)        # L > 2 r_c: one image per pair
    # mean rows per atom of the synthetic liquid: 84-92
    assert 80.0 < ri.size / x.shape[0] < 95.0


def test_neighbours_rows_sorted_and_displacements_consistent(c0):
    p = c0["parts"]
    key = np.stack([p["ri"], p["rj"], p["rn"][:, 0], p["rn"][:, 1], p["rn"][:, 2]], axis=1)
    assert all(tuple(key[a]) < tuple(key[a + 1]) for a in range(0, len(key) - 1, 7))
    x, L = c0["x"], c0["wb"]["box"]
    w = x - L * np.floor(x / L)
    assert np.array_equal(p["d"], (w[p["rj"]] - w[p["ri"]]) + p["rn"] * L)
    r = np.linalg.norm(p["d"], axis=1)
    assert r.max() < 6.0 and r.min() > 0.8


def test_sel_overflow_raises():
    desc = dict(wl.model_desc())
    desc["sel"] = [46, 20]                       # water at 1 g/cm3 has ~60 H inside 6 A
    w = np.zeros(se_e2_a.Model.n_weights(desc))
    cfg, wb, _, _ = wl.make_config(0, n_beads=1)
    with pytest.raises(OverflowError):
        se_e2_a.energy_forces(wb["x"][0], wb["types"], wb["box"], se_e2_a.Model(desc, w))


# ------------------------------------------------------------------------------- switch function
def test_switch_values_and_derivative():
    rs, rc = 0.5, 6.0
    r = np.array([0.3, 0.5, 1.0, 3.25, 5.9, 5.999999, 6.0, 7.0])
    s, ds = se_e2_a.switch(r, rs, rc)
    assert s[0] == 1.0 / 0.3 and abs(ds[0] + 1.0 / 0.09) < 1e-14           # 1/r inside r_s
    assert abs(s[1] - 2.0) < 1e-15                                          # continuous at r_s
    assert abs(s[3] - 0.5 / 3.25) < 1e-15                                   # u = 1/2 -> polynomial = 1/2
    assert s[6] == 0.0 and s[7] == 0.0 and ds[6] == 0.0
    assert abs(s[5]) < 1e-15                                                # C2-smooth at r_c
    h = 1e-6
    rr = np.array([0.4, 0.8, 2.0, 4.0, 5.5])
    num = (se_e2_a.switch(rr + h, rs, rc)[0] - se_e2_a.switch(rr - h, rs, rc)[0]) / (2 * h)
    assert np.abs(num - se_e2_a.switch(rr, rs, rc)[1]).max() < 1e-8


# ------------------------------------------------------------------------------- two-atom hand case
def test_two_atom_case_by_hand():
    """One O and one H at distance r along a tilted axis in a huge box: each atom has one row, so
    T = G(s) (x) R / 138 and D = T T[:16]^T can be written out with scalar loops."""
    desc = wl.model_desc()
    w = wl.model_weights(desc, 3)
    m = se_e2_a.Model(desc, w)
    dvec = np.array([1.1, -0.7, 0.4])
    x = np.array([[50.0, 50.0, 50.0], [50.0, 50.0, 50.0] + dvec])
    types = np.array([0, 1])
    E, F, Xi = se_e2_a.energy_forces(x, types, np.array([200.0] * 3), m)
    r = math.sqrt(float(dvec @ dvec))
    u = (r - 0.5) / 5.5
    s = (u ** 3 * (-6 * u * u + 15 * u - 10) + 1) / r
    for (ti, tj, sign) in [(0, 1, 1.0), (1, 0, -1.0)]:
        (W1, b1), (W2, b2), (W3, b3) = m.emb[(ti, tj)]
        h1 = [math.tanh(s * W1[0, a] + b1[a]) for a in range(25)]
        h2 = [h1[a % 25] + math.tanh(sum(h1[c] * W2[c, a] for c in range(25)) + b2[a]) for a in range(50)]
        G = [h2[a % 50] + math.tanh(sum(h2[c] * W3[c, a] for c in range(50)) + b3[a]) for a in range(100)]
        R = [s] + [s * sign * dvec[c] / r for c in range(3)]
        T = np.array([[G[a] * R[c] / 138.0 for c in range(4)] for a in range(100)])
        D = np.array([[sum(T[a, c] * T[b, c] for c in range(4)) for b in range(16)] for a in range(100)]).reshape(-1)
        (F1, c1), (F2, c2), (F3, c3), (F4, c4) = m.fitnet[ti]
        y1 = np.tanh(D @ F1 + c1)
        y2 = y1 + np.tanh(y1 @ F2 + c2)
        y3 = y2 + np.tanh(y2 @ F3 + c3)
        e = float(y3 @ F4[:, 0] + c4[0])
        assert abs(E[0 if ti == 0 else 1] - e) < 1e-14
    assert np.abs(F[0] + F[1]).max() < 1e-18
    # central force: F parallel to d
    assert np.abs(np.cross(F[0], dvec)).max() < 1e-16 * max(1.0, np.abs(F[0]).max() * 1e6)


# ------------------------------------------------------------------------------- backward: finite differences
def test_forces_equal_minus_dE_dx_by_central_differences(c0):
    x, types, box, model, F = c0["x"], c0["wb"]["types"], c0["wb"]["box"], c0["model"], c0["F"]
    h = 1e-4
    frms = math.sqrt(float(np.mean(F * F)))
    assert frms > 0.05                       # the x1e3 model has forces that matter
    for (i, a) in [(0, 0), (5, 2), (50, 1), (95, 0)]:
        xp, xm = x.copy(), x.copy()
        xp[i, a] += h
        xm[i, a] -= h
        Ep = se_e2_a.energy_forces(xp, types, box, model)[0].sum()
        Em = se_e2_a.energy_forces(xm, types, box, model)[0].sum()
        assert abs(-(Ep - Em) / (2 * h) - F[i, a]) < 2e-6 * frms


def test_total_force_vanishes_and_virial_is_symmetric(c0):
    F, Xi = c0["F"], c0["Xi"]
    assert np.abs(F.sum(axis=0)).max() < 1e-13 * np.abs(F).max() * F.shape[0]
    assert np.abs(Xi - Xi.T).max() < 1e-12 * np.abs(Xi).max()


# ------------------------------------------------------------------------------- backward: torch autograd, dense forward
def _torch_dense_energy(x, L, types, model, eps=None):
    """Independent forward in torch float64: every (i, j, image) triple is a row of a dense tensor,
    masked by r < r_c.  Organised per ordered type pair, not per row list.  With `eps` (3x3 strain,
    requires_grad) positions and cell are deformed x -> x(1+eps), so that autograd gives dU/d(eps)."""
    import torch
    N = x.shape[0]
    tt = torch.as_tensor(types)
    s_max = int(math.ceil(model.rcut / float(L.min())))
    sh = torch.tensor([(a, b, c) for a in range(-s_max, s_max + 1) for b in range(-s_max, s_max + 1)
                       for c in range(-s_max, s_max + 1)], dtype=torch.float64)
    w = x - L * torch.floor(x / L)                                  # wrap in the undeformed cell
    d = w[None, :, None, :] - w[:, None, None, :] + (sh * L)[None, None, :, :]      # [i, j, n, 3]
    if eps is not None:
        d = d + d @ eps.T
    self_mask = torch.eye(N, dtype=torch.bool)[:, :, None] & (sh.abs().sum(-1) == 0)[None, None, :]
    r2 = (d * d).sum(-1)
    r = torch.sqrt(torch.where(self_mask, torch.ones_like(r2), r2))     # sqrt'(0) would poison autograd
    mask = (r < model.rcut) & ~self_mask
    rs, rc = model.rcut_smth, model.rcut
    rsafe = torch.where(mask, r, torch.ones_like(r))
    u = (rsafe - rs) / (rc - rs)
    sw = torch.where(rsafe < rs, torch.ones_like(u), u ** 3 * (-6 * u ** 2 + 15 * u - 10) + 1)
    s = torch.where(mask, sw / rsafe, torch.zeros_like(r))
    R = torch.cat([s[..., None], (s / rsafe)[..., None] * d], dim=-1)              # [i, j, n, 4]
    T = torch.zeros(N, model.embed[-1], 4, dtype=torch.float64)
    for ti in range(model.ntypes):
        for tj in range(model.ntypes):
            ii = torch.nonzero(tt == ti).ravel()
            jj = torch.nonzero(tt == tj).ravel()
            sij = s[ii][:, jj]                                                       # [ni, nj, n]
            h = sij[..., None]
            for (W, b) in model.emb[(ti, tj)]:
                W, b = torch.as_tensor(W), torch.as_tensor(b)
                t = torch.tanh(h @ W + b)
                h = torch.cat([h, h], dim=-1) + t if W.shape[1] == 2 * W.shape[0] else t
            h = h * mask[ii][:, jj][..., None]                                       # padded rows: exactly 0
            T[ii] = T[ii] + torch.einsum("ijnm,ijnc->imc", h, R[ii][:, jj])
    T = T / model.nsel
    D = torch.einsum("imc,ikc->imk", T, T[:, :model.axis, :]).reshape(N, -1)
    E = torch.zeros(N, dtype=torch.float64)
    for t_ in range(model.ntypes):
        at = torch.nonzero(tt == t_).ravel()
        y = D[at]
        for li, (W, b) in enumerate(model.fitnet[t_]):
            W, b = torch.as_tensor(W), torch.as_tensor(b)
            if li == len(model.fitnet[t_]) - 1:
                y = y @ W + b
            else:
                z = torch.tanh(y @ W + b)
                y = y + z if W.shape[0] == W.shape[1] else z
        E[at] = y[:, 0]
    return E


def test_forces_and_virial_match_torch_autograd(c0):
    import torch
    x = torch.tensor(c0["x"], dtype=torch.float64, requires_grad=True)
    L = torch.tensor(c0["wb"]["box"], dtype=torch.float64)
    eps = torch.zeros(3, 3, dtype=torch.float64, requires_grad=True)
    E = _torch_dense_energy(x, L, c0["wb"]["types"], c0["model"], eps)
    assert np.abs(E.detach().numpy() - c0["E"]).max() < 1e-11 * max(1.0, np.abs(c0["E"]).max())
    gx, geps = torch.autograd.grad(E.sum(), [x, eps])
    F = -gx.numpy()
    assert np.abs(F - c0["F"]).max() < 1e-10 * np.abs(c0["F"]).max()
    # Xi_ab = -sum_g dU/dh_ag h_gb; for the strain d -> (1+eps) d this is -dU/d(eps_ab)
    Xi = -geps.numpy()
    assert np.abs(Xi - c0["Xi"]).max() < 1e-10 * np.abs(c0["Xi"]).max()


# ------------------------------------------------------------------------------- invariances
def test_translation_and_permutation_invariance(c0):
    x, types, box, model = c0["x"], c0["wb"]["types"], c0["wb"]["box"], c0["model"]
    E0 = c0["E"].sum()
    # translation, including across the periodic boundary (atoms re-wrap, images change)
    E1, F1, Xi1 = se_e2_a.energy_forces(x + np.array([3.7, -12.1, 0.33]), types, box, model)
    assert abs(E1.sum() - E0) < 1e-10 * abs(E0)
    assert np.abs(F1 - c0["F"]).max() < 1e-9 * np.abs(c0["F"]).max()
    assert np.abs(Xi1 - c0["Xi"]).max() < 1e-9 * np.abs(c0["Xi"]).max()
    # a lattice translation of single atoms (unwrapped coordinates may leave the box)
    x2 = x.copy()
    x2[7] += box * np.array([1, -2, 0])
    assert abs(se_e2_a.energy_forces(x2, types, box, model)[0].sum() - E0) < 1e-10 * abs(E0)
    # permutation of atoms
    perm = np.random.default_rng(5).permutation(x.shape[0])
    Ep, Fp, _ = se_e2_a.energy_forces(x[perm], types[perm], box, model)
    assert np.abs(Ep - c0["E"][perm]).max() < 1e-11 * np.abs(c0["E"]).max()
    assert np.abs(Fp - c0["F"][perm]).max() < 1e-9 * np.abs(c0["F"]).max()


def test_rotation_invariance_on_isolated_cluster(c0):
    model, types = c0["model"], c0["wb"]["types"][:24]
    box = np.array([400.0, 400.0, 400.0])
    xc = c0["x"][:24] - c0["x"][:24].mean(axis=0)
    q = np.array([0.3, -0.5, 0.7, 0.41])
    q /= np.linalg.norm(q)
    a, b, c, d = q
    Rm = np.array([[a * a + b * b - c * c - d * d, 2 * (b * c - a * d), 2 * (b * d + a * c)],
                   [2 * (b * c + a * d), a * a - b * b + c * c - d * d, 2 * (c * d - a * b)],
                   [2 * (b * d - a * c), 2 * (c * d + a * b), a * a - b * b - c * c + d * d]])
    E0, F0, Xi0 = se_e2_a.energy_forces(xc + 200.0, types, box, model)
    E1, F1, Xi1 = se_e2_a.energy_forces(xc @ Rm.T + 200.0, types, box, model)
    assert np.abs(E1 - E0).max() < 1e-11 * np.abs(E0).max()
    assert np.abs(F1 - F0 @ Rm.T).max() < 1e-10 * np.abs(F0).max()
    assert np.abs(Xi1 - Rm @ Xi0 @ Rm.T).max() < 1e-10 * np.abs(Xi0).max()


def test_energy_continuous_when_a_neighbour_crosses_rcut(c0):
    """s, s', s'' vanish at r_c, so E changes by O(delta^3) when a pair distance crosses r_c."""
    model = c0["model"]
    types = np.array([0, 1, 1, 0])
    box = np.array([300.0] * 3)
    base = np.array([[100.0, 100.0, 100.0], [100.9, 100.2, 100.1], [99.6, 100.8, 100.0], [0, 0, 0]])
    Es = []
    for delta in (-1e-5, 1e-5):
        x = base.copy()
        x[3] = base[0] + np.array([0.0, 0.0, 6.0 + delta])
        Es.append(se_e2_a.energy_forces(x, types, box, model)[0].sum())
    assert abs(Es[0] - Es[1]) < 1e-12 * abs(Es[0])


def test_padded_slots_contribute_nothing_descriptor_scales_with_nsel(c0):
    """T is divided by N_sel = sum(sel) (138), not by the real neighbour count (DESIGN R-14)."""
    p = c0["parts"]
    i = 3
    rows = np.flatnonzero(p["ri"] == i)
    model = c0["model"]
    types = c0["wb"]["types"]
    acc = np.zeros((100, 4))
    for r_ in rows:
        layers = model.emb[(int(types[i]), int(types[p["rj"][r_]]))]
        h = np.array([[p["R"][r_, 0]]])
        for (W, b) in layers:
            t = np.tanh(h @ W + b)
            h = np.concatenate([h, h], axis=1) + t if W.shape[1] == 2 * W.shape[0] else t
        acc += np.outer(h[0], p["R"][r_])
    assert np.abs(acc / 138.0 - p["T"][i]).max() < 1e-15


def test_bruteforce_neighbours_restricted_to_centres_are_the_same_rows():
    """`centres=` (used by the sampled GPU parity checks at configs[3]) returns exactly the rows of those centres."""
    cfg, wb, desc, w = wl.make_config(0)
    full = se_e2_a.neighbours_bruteforce(wb["x"][1], wb["box"], desc["rcut"])
    centres = np.array([0, 5, 17, 95])
    part = se_e2_a.neighbours_bruteforce(wb["x"][1], wb["box"], desc["rcut"], centres=centres)
    keep = np.isin(full[0], centres)
    assert keep.sum() > 300
    for a, b in zip(full, part):
        assert np.array_equal(a[keep], b)
