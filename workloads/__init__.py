"""Seeded synthetic inputs shared by the oracle's tests and the CUDA path's tests / bench.

This module holds NO arithmetic of the method (no transform, integrator, descriptor or network);
it only draws the inputs: water boxes shaped like the paper's DP-water workloads
(PAPER.md:L76, L232, L252-254 -- 128/512/4096 H2O x 32 beads; the paper's own configurations and
its trained model are not available offline) and random-init network weights, following the
recipe of BASELINE.json `configs` spelled out in DESIGN.md section 4.

Draw order for one box (numpy default_rng(seed), PCG64): lattice jitter -> orientation
quaternions -> bead noise -> momenta.  Weights use their own default_rng(weight_seed).
"""
import math
import numpy as np

# input-distribution constants (Maxwell-Boltzmann width of the momenta); values as in DESIGN R-9
_KB = 8.617333262e-5        # eV/K
_MVV2E = 1.0364269e-4       # eV / ((g/mol)(A/ps)^2)

MASS_O, MASS_H = 15.9994, 1.008
R_OH, ANGLE_HOH = 0.9572, 104.52

# BASELINE.json configs[0..4]
CONFIGS = [
    dict(name="c0_32h2o_p4", n_mol=32, box=9.86, P=4, T=300.0, dt=0.5e-3, gamma=1.0, lattice="fcc",
         steps=10, geom_seed=0, weight_seed=0),
    dict(name="c1_64h2o_p32", n_mol=64, box=12.42, P=32, T=300.0, dt=0.25e-3, gamma=1.0, lattice="sc",
         steps=100, geom_seed=1, weight_seed=1),
    dict(name="c2_512h2o_p32", n_mol=512, box=24.83, P=32, T=300.0, dt=0.25e-3, gamma=1.0, lattice="sc",
         steps=200, geom_seed=2, weight_seed=1),
    dict(name="c3_4096h2o_p32", n_mol=4096, box=49.67, P=32, T=300.0, dt=0.25e-3, gamma=1.0, lattice="sc",
         steps=50, geom_seed=3, weight_seed=1),
    dict(name="c4_2048h2o_p64_npt", n_mol=2048, box=39.42, P=64, T=300.0, dt=0.25e-3, gamma=1.0,
         lattice="fcc", steps=50, geom_seed=4, weight_seed=1, p_ext_bar=1.0, tau_p=0.5),   # NpT: PAPER.md:L76
]


def model_desc():
    """se_e2_a architecture of BASELINE.json configs[0]."""
    return dict(rcut=6.0, rcut_smth=0.5, sel=[46, 92], embed=[25, 50, 100], axis=16, fit=[240, 240, 240])


def n_model_weights(desc):
    nt = len(desc["sel"])
    n_emb, n_in = 0, 1
    for n_out in desc["embed"]:
        n_emb += n_in * n_out + n_out
        n_in = n_out
    n_fit, n_in = 0, desc["embed"][-1] * desc["axis"]
    for n_out in list(desc["fit"]) + [1]:
        n_fit += n_in * n_out + n_out
        n_in = n_out
    return nt * nt * n_emb + nt * n_fit


def model_weights(desc, seed, last_layer_scale=1.0):
    """Flat float64 weight vector in the C-ABI packing order: W ~ N(0,1)/sqrt(fan_in), b ~ 0.1 N(0,1)
    ("N(0, 1/fan_in)", "N(0, 0.01)" read as variances).  `last_layer_scale` multiplies the final
    fitting layer (weights and bias), for tests that need forces that matter."""
    rng = np.random.default_rng(seed)
    nt = len(desc["sel"])
    out = []

    def layer(n_in, n_out, scale=1.0):
        out.append(scale * rng.standard_normal(n_in * n_out) / math.sqrt(n_in))
        out.append(scale * 0.1 * rng.standard_normal(n_out))

    for _ti in range(nt):
        for _tj in range(nt):
            n_in = 1
            for n_out in desc["embed"]:
                layer(n_in, n_out)
                n_in = n_out
    for _ti in range(nt):
        n_in = desc["embed"][-1] * desc["axis"]
        for n_out in desc["fit"]:
            layer(n_in, n_out)
            n_in = n_out
        layer(n_in, 1, last_layer_scale)
    w = np.concatenate(out)
    assert w.size == n_model_weights(desc)
    return w


def _lattice_sites(n_mol, L, kind):
    if kind == "sc":
        g = round(n_mol ** (1.0 / 3.0))
        assert g ** 3 == n_mol, "simple-cubic lattice needs a cube number of molecules"
        idx = np.array([(a, b, c) for a in range(g) for b in range(g) for c in range(g)], dtype=np.float64)
        return (idx + 0.5) * (L / g)
    if kind == "fcc":
        c = round((n_mol / 4) ** (1.0 / 3.0))
        assert 4 * c ** 3 == n_mol, "fcc lattice needs 4*c^3 molecules"
        basis = np.array([(0, 0, 0), (0.5, 0.5, 0), (0.5, 0, 0.5), (0, 0.5, 0.5)])
        cells = np.array([(a, b, d) for a in range(c) for b in range(c) for d in range(c)], dtype=np.float64)
        return ((cells[:, None, :] + basis[None, :, :] + 0.25).reshape(-1, 3)) * (L / c)
    raise ValueError(kind)


def water_box(n_mol, L, P, T, seed, lattice="sc", bead_sigma=0.01, jitter=0.2):
    """Returns dict(types[N] int32, masses[2], box[3], x[P,N,3], p[P,N,3]).  Atom order O,H,H per
    molecule; types 0 (O), 1 (H).  x is unwrapped (atoms may stick out of the box); p are Cartesian
    bead momenta drawn at the ring temperature P*T."""
    rng = np.random.default_rng(seed)
    sites = _lattice_sites(n_mol, L, lattice)
    sites = sites + rng.uniform(-jitter, jitter, size=sites.shape)
    q = rng.standard_normal((n_mol, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    a, b, c, d = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    Rm = np.stack([
        np.stack([a * a + b * b - c * c - d * d, 2 * (b * c - a * d), 2 * (b * d + a * c)], axis=1),
        np.stack([2 * (b * c + a * d), a * a - b * b + c * c - d * d, 2 * (c * d - a * b)], axis=1),
        np.stack([2 * (b * d - a * c), 2 * (c * d + a * b), a * a - b * b - c * c + d * d], axis=1),
    ], axis=1)                                                   # [n_mol, 3, 3]
    half = 0.5 * math.radians(ANGLE_HOH)
    h_local = R_OH * np.array([[math.sin(half), 0.0, math.cos(half)],
                               [-math.sin(half), 0.0, math.cos(half)]])
    N = 3 * n_mol
    x0 = np.empty((N, 3))
    x0[0::3] = sites
    x0[1::3] = sites + np.einsum("nab,b->na", Rm, h_local[0])
    x0[2::3] = sites + np.einsum("nab,b->na", Rm, h_local[1])
    types = np.tile(np.array([0, 1, 1], dtype=np.int32), n_mol)
    masses = np.array([MASS_O, MASS_H])
    x = x0[None, :, :] + bead_sigma * rng.standard_normal((P, N, 3))
    m_atom = masses[types]
    sig_p = np.sqrt(m_atom * P * _KB * T / _MVV2E)
    p = sig_p[None, :, None] * rng.standard_normal((P, N, 3))
    return dict(types=types, masses=masses, box=np.array([L, L, L], dtype=np.float64), x=x, p=p)


def make_config(idx, n_beads=None):
    """Inputs of BASELINE.json configs[idx]: (cfg dict, box dict, model desc, weights)."""
    cfg = dict(CONFIGS[idx])
    if n_beads is not None:
        cfg["P"] = n_beads
    wb = water_box(cfg["n_mol"], cfg["box"], cfg["P"], cfg["T"], cfg["geom_seed"], cfg["lattice"])
    desc = model_desc()
    w = model_weights(desc, cfg["weight_seed"])
    return cfg, wb, desc, w
