"""Deep-Potential `se_e2_a` energy, forces and virial of ONE bead -- oracle (test infrastructure;
see oracle/__init__.py).  FP64 numpy, brute-force neighbours, hand-written analytic backward.

The paper only cites the Deep Potential model and prints no equation
for it; the definition below is BASELINE.json's north_star / configs[0] plus the readings
DESIGN R-11 .. R-16 (PARITY UNPINNED against physics; backward pinned against the forward).
The bead virial follows PAPER.md:L372: Xi_ab = -sum_g dU/dh_ag h_gb.

Weight vector layout (C-ABI `pimd_set_model`): row-major W[in][out] then bias,
  for t_i in types: for t_j in types: embedding layers 1..3
  then for t_i in types: fitting layers 1..4 (the last one has out = 1).
"""
import math
import numpy as np


class Model:
    """Unpacked se_e2_a parameters.  desc: dict(rcut, rcut_smth, sel, embed, axis, fit)."""

    def __init__(self, desc, weights):
        self.rcut = float(desc["rcut"])
        self.rcut_smth = float(desc["rcut_smth"])
        self.sel = [int(s) for s in desc["sel"]]
        self.ntypes = len(self.sel)
        self.embed = [int(w) for w in desc["embed"]]
        self.axis = int(desc["axis"])
        self.fit = [int(w) for w in desc["fit"]]
        self.nsel = sum(self.sel)
        w = np.asarray(weights, dtype=np.float64)
        pos = 0

        def take(n_in, n_out):
            nonlocal pos
            W = w[pos:pos + n_in * n_out].reshape(n_in, n_out)
            pos += n_in * n_out
            b = w[pos:pos + n_out]
            pos += n_out
            return W, b

        self.emb = {}
        for ti in range(self.ntypes):
            for tj in range(self.ntypes):
                layers, n_in = [], 1
                for n_out in self.embed:
                    layers.append(take(n_in, n_out))
                    n_in = n_out
                self.emb[(ti, tj)] = layers
        self.fitnet = []
        m1 = self.embed[-1]
        for ti in range(self.ntypes):
            layers, n_in = [], m1 * self.axis
            for n_out in self.fit + [1]:
                layers.append(take(n_in, n_out))
                n_in = n_out
            self.fitnet.append(layers)
        if pos != w.size:
            raise ValueError("weight vector has %d entries, the architecture needs %d" % (w.size, pos))
        self.tables = None       # set by oracle.compress.compress(): tabulated embedding

    @staticmethod
    def n_weights(desc):
        nt = len(desc["sel"])
        n, n_in = 0, 1
        for n_out in desc["embed"]:
            n += n_in * n_out + n_out
            n_in = n_out
        n_emb = n
        n, n_in = 0, desc["embed"][-1] * desc["axis"]
        for n_out in list(desc["fit"]) + [1]:
            n += n_in * n_out + n_out
            n_in = n_out
        return nt * nt * n_emb + nt * n


# ----------------------------------------------------------------------------------------------
# neighbours
# ----------------------------------------------------------------------------------------------

def neighbours_bruteforce(x, box, rcut, i_block=128, centres=None):
    """All rows (i, j, n) with |(w_j - w_i) + n*L| < rcut, (j, n) != (i, 0), by brute force over
    every pair and every periodic image n in {-s..s}^3, s = ceil(rcut/L) (DESIGN R-11; PAPER.md:
    L200-202 for the wrap).  w = x - L*floor(x/L).  The squared distance is evaluated as
    (dx*dx + dy*dy) + dz*dz in FP64 with no fused multiply-add, compared strictly (< rcut*rcut).
    Returns i[M], j[M], n[M,3] (int) and d[M,3] sorted by (i, j, n_x, n_y, n_z).
    `centres` (sorted atom indices) restricts the rows to those centres i -- the sampled parity checks at sizes
    where all N^2 x images distance tests would take minutes; the arithmetic per row is unchanged."""
    x = np.asarray(x, dtype=np.float64)
    L = np.asarray(box, dtype=np.float64)
    N = x.shape[0]
    if centres is not None:
        centres = np.asarray(centres, dtype=np.int64)
        w = x - L * np.floor(x / L)
        s = [int(math.ceil(rcut / L[a])) for a in range(3)]
        shifts = np.array([(a, b, c) for a in range(-s[0], s[0] + 1)
                           for b in range(-s[1], s[1] + 1)
                           for c in range(-s[2], s[2] + 1)], dtype=np.int64)
        shift_vec = shifts.astype(np.float64) * L
        self_img = np.flatnonzero((shifts == 0).all(axis=1))[0]
        oi, oj, on, od = [], [], [], []
        for i in centres:
            d = (w[:, None, :] - w[i][None, None, :]) + shift_vec[None, :, :]
            r2 = (d[..., 0] * d[..., 0] + d[..., 1] * d[..., 1]) + d[..., 2] * d[..., 2]
            mask = r2 < rcut * rcut
            mask[i, self_img] = False
            bj, bs = np.nonzero(mask)
            oi.append(np.full(bj.size, i, dtype=np.int64))
            oj.append(bj)
            on.append(shifts[bs])
            od.append(d[bj, bs])
        return (np.concatenate(oi), np.concatenate(oj), np.concatenate(on).reshape(-1, 3),
                np.concatenate(od).reshape(-1, 3))
    w = x - L * np.floor(x / L)
    s = [int(math.ceil(rcut / L[a])) for a in range(3)]
    shifts = np.array([(a, b, c) for a in range(-s[0], s[0] + 1)
                       for b in range(-s[1], s[1] + 1)
                       for c in range(-s[2], s[2] + 1)], dtype=np.int64)
    shift_vec = shifts.astype(np.float64) * L                  # n o L
    rc2 = rcut * rcut
    out_i, out_j, out_n, out_d = [], [], [], []
    for i0 in range(0, N, i_block):
        i1 = min(N, i0 + i_block)
        # d[i, j, image, :] = (w_j - w_i) + n*L
        d = (w[None, :, None, :] - w[i0:i1, None, None, :]) + shift_vec[None, None, :, :]
        r2 = (d[..., 0] * d[..., 0] + d[..., 1] * d[..., 1]) + d[..., 2] * d[..., 2]
        mask = r2 < rc2
        self_img = np.flatnonzero((shifts == 0).all(axis=1))[0]
        ii = np.arange(i0, i1)
        mask[ii - i0, ii, self_img] = False
        bi, bj, bs = np.nonzero(mask)                          # already sorted by (i, j, image)
        out_i.append(bi + i0)
        out_j.append(bj)
        out_n.append(shifts[bs])
        out_d.append(d[bi, bj, bs])
    return (np.concatenate(out_i), np.concatenate(out_j),
            np.concatenate(out_n).reshape(-1, 3), np.concatenate(out_d).reshape(-1, 3))


# ----------------------------------------------------------------------------------------------
# pieces of the model
# ----------------------------------------------------------------------------------------------

def switch(r, rs, rc):
    """s(r) and s'(r) (DESIGN R-12): s = 1/r for r < r_s; [u^3(-6u^2+15u-10)+1]/r for r_s <= r < r_c,
    u = (r-r_s)/(r_c-r_s); 0 beyond."""
    u = (r - rs) / (rc - rs)
    poly = u * u * u * (-6.0 * u * u + 15.0 * u - 10.0) + 1.0
    dpoly = -30.0 * u * u * (u - 1.0) * (u - 1.0) / (rc - rs)
    inner = r < rs
    sw = np.where(inner, 1.0, poly)
    dsw = np.where(inner, 0.0, dpoly)
    outside = r >= rc
    sw = np.where(outside, 0.0, sw)
    dsw = np.where(outside, 0.0, dsw)
    s = sw / r
    ds = dsw / r - sw / (r * r)
    return s, ds


def _segment_sum(values, seg, n_seg):
    """out[a] = sum of values[rows with seg == a]; `seg` is sorted ascending (rows are sorted by i)."""
    out = np.zeros((n_seg,) + values.shape[1:])
    if values.shape[0] == 0:
        return out
    present, starts = np.unique(seg, return_index=True)
    out[present] = np.add.reduceat(values, starts, axis=0)
    return out


def _scatter_add(n, idx, values):
    """out[idx[r], c] += values[r, c] for unsorted idx."""
    return np.stack([np.bincount(idx, weights=values[:, c], minlength=n) for c in range(values.shape[1])], axis=1)


def _mlp_forward(layers, h, skip_rule):
    """Generic tanh MLP.  Returns output and the list of tanh values t_l per layer (for backward).
    skip_rule(n_in, n_out) in {"none", "id", "double"}."""
    tanhs = []
    for (W, b) in layers:
        n_in, n_out = W.shape
        t = np.tanh(h @ W + b)
        rule = skip_rule(n_in, n_out)
        if rule == "double":
            h = np.concatenate([h, h], axis=1) + t
        elif rule == "id":
            h = h + t
        else:
            h = t
        tanhs.append(t)
    return h, tanhs


def _mlp_backward(layers, tanhs, dh, skip_rule):
    """Back-propagate dU/d(output) = dh through the tanh MLP to dU/d(input)."""
    for (W, b), t in zip(reversed(layers), reversed(tanhs)):
        n_in, n_out = W.shape
        da = dh * (1.0 - t * t)
        dprev = da @ W.T
        rule = skip_rule(n_in, n_out)
        if rule == "double":
            dprev = dprev + dh[:, :n_in] + dh[:, n_in:]
        elif rule == "id":
            dprev = dprev + dh
        dh = dprev
    return dh


def _embed_rule(n_in, n_out):
    # DESIGN R-13: G-net layers with out = 2*in carry the doubling skip h <- [h,h] + tanh(.)
    if n_out == 2 * n_in:
        return "double"
    if n_out == n_in:
        return "id"
    return "none"


def _fit_rule(n_in, n_out):
    # DESIGN R-15: identity skip where widths match, no timestep factor
    return "id" if n_out == n_in else "none"


def energy_forces(x, types, box, model, return_parts=False, row_block=32768):
    """E_i[N], F[N,3] (eV/A), virial Xi[3,3] (eV) of one bead at unwrapped positions x[N,3].

    1. rows = neighbours_bruteforce;  2. s(r), R_row = (s, s dx/r, s dy/r, s dz/r)  (R-12);
    3. G_row = embedding net of the ordered type pair (t_i, t_j) applied to s      (R-13);
    4. T_i = (1/N_sel) sum_rows G_row (x) R_row in R^{M1 x 4};  D_i = T_i T_i[:axis]^T (R-14);
    5. E_i = fitting net of t_i applied to D_i flattened m1-major                   (R-15);
    6. analytic backward to g = dU/dd per row;  F_i += g, F_j -= g;  Xi_ab = -sum d_a g_b (R-16).
    Raises OverflowError when an atom has more neighbours of a type than sel allows (R-11)."""
    types = np.asarray(types, dtype=np.int64)
    N = x.shape[0]
    ri, rj, rn, d = neighbours_bruteforce(x, box, model.rcut)
    tj = types[rj]
    ti = types[ri]
    for t in range(model.ntypes):
        cnt = np.bincount(ri[tj == t], minlength=N)
        if cnt.size and cnt.max() > model.sel[t]:
            raise OverflowError("atom %d has %d neighbours of type %d > sel %d"
                                % (int(cnt.argmax()), int(cnt.max()), t, model.sel[t]))
    Mrows = ri.size
    r = np.sqrt((d[:, 0] * d[:, 0] + d[:, 1] * d[:, 1]) + d[:, 2] * d[:, 2])
    s, ds = switch(r, model.rcut_smth, model.rcut)
    R = np.empty((Mrows, 4))
    R[:, 0] = s
    R[:, 1:] = (s / r)[:, None] * d
    M1, M2 = model.embed[-1], model.axis
    inv_nsel = 1.0 / model.nsel

    # ---- forward: embedding and T ----
    pair_id = ti * model.ntypes + tj
    T = np.zeros((N, M1, 4))
    for b0 in range(0, Mrows, row_block):
        b1 = min(Mrows, b0 + row_block)
        G = np.empty((b1 - b0, M1))
        for p in range(model.ntypes ** 2):
            sel_rows = np.flatnonzero(pair_id[b0:b1] == p)
            if sel_rows.size:
                pair = (p // model.ntypes, p % model.ntypes)
                if model.tables is not None:
                    from . import compress
                    G[sel_rows], _ = compress.table_eval(model.tables[pair], s[b0:b1][sel_rows])
                else:
                    G[sel_rows], _ = _mlp_forward(model.emb[pair], s[b0:b1][sel_rows, None], _embed_rule)
        T += _segment_sum(G[:, :, None] * R[b0:b1, None, :], ri[b0:b1], N)
    T *= inv_nsel

    # ---- descriptor, fitting net forward and backward (per centre type) ----
    D = np.einsum("imc,inc->imn", T, T[:, :M2, :]).reshape(N, M1 * M2)
    E = np.zeros(N)
    dD = np.zeros((N, M1 * M2))
    for t in range(model.ntypes):
        at = np.flatnonzero(types == t)
        if at.size == 0:
            continue
        hidden, (W4, b4) = model.fitnet[t][:-1], model.fitnet[t][-1]
        y, tanhs = _mlp_forward(hidden, D[at], _fit_rule)
        E[at] = (y @ W4 + b4)[:, 0]                              # last layer is linear: E_i = y3.w4 + b4
        dy = np.broadcast_to(W4[:, 0], y.shape)                 # dU/dy3 = w4
        dD[at] = _mlp_backward(hidden, tanhs, dy, _fit_rule)
    dD3 = dD.reshape(N, M1, M2)
    # dT[m,c] = sum_{m2<M2} dD[m,m2] T[m2,c]  +  [m<M2] sum_{m1} dD[m1,m] T[m1,c]
    dT = np.einsum("imn,inc->imc", dD3, T[:, :M2, :])
    dT[:, :M2, :] += np.einsum("imn,imc->inc", dD3, T)

    # ---- backward through T, the embedding net and the environment row ----
    F = np.zeros((N, 3))
    Xi = np.zeros((3, 3))
    g_all = np.empty((Mrows, 3)) if return_parts else None
    for b0 in range(0, Mrows, row_block):
        b1 = min(Mrows, b0 + row_block)
        sb, dsb, rb, db, Rb = s[b0:b1], ds[b0:b1], r[b0:b1], d[b0:b1], R[b0:b1]
        dTi = dT[ri[b0:b1]]                                     # [rows, M1, 4]
        G = np.empty((b1 - b0, M1))
        dsG = np.empty(b1 - b0)                                  # dU/ds through the embedding input
        dG = np.einsum("rmc,rc->rm", dTi, Rb) * inv_nsel
        for p in range(model.ntypes ** 2):
            sel_rows = np.flatnonzero(pair_id[b0:b1] == p)
            if sel_rows.size:
                pair = (p // model.ntypes, p % model.ntypes)
                if model.tables is not None:
                    from . import compress
                    G[sel_rows], Gp = compress.table_eval(model.tables[pair], sb[sel_rows])
                    dsG[sel_rows] = np.einsum("rm,rm->r", dG[sel_rows], Gp)
                    continue
                layers = model.emb[pair]
                G[sel_rows], tanhs = _mlp_forward(layers, sb[sel_rows, None], _embed_rule)
                dsG[sel_rows] = _mlp_backward(layers, tanhs, dG[sel_rows], _embed_rule)[:, 0]
        dR = np.einsum("rmc,rm->rc", dTi, G) * inv_nsel          # [rows, 4]
        # g = (ds_G + dR_0) s' d/r + sum_c dR_c [ (s'/r - s/r^2) d_c d/r + (s/r) e_c ]
        dhat = db / rb[:, None]
        radial = (dsG + dR[:, 0]) * dsb + (dsb / rb - sb / (rb * rb)) * np.einsum("rc,rc->r", dR[:, 1:], db)
        g = radial[:, None] * dhat + (sb / rb)[:, None] * dR[:, 1:]
        F += _scatter_add(N, ri[b0:b1], g)
        F -= _scatter_add(N, rj[b0:b1], g)
        Xi -= db.T @ g
        if return_parts:
            g_all[b0:b1] = g
    if return_parts:
        return E, F, Xi, {"ri": ri, "rj": rj, "rn": rn, "d": d, "R": R, "T": T, "D": D, "dT": dT, "g": g_all}
    return E, F, Xi


def harmonic_energy_forces(x, k_spring):
    """Test model (C-ABI `pimd_set_model_harmonic`): U = sum_i 1/2 k |r_i|^2 about the origin on the
    unwrapped coordinates; F = -k r; virial Xi_ab = -sum_i r_a dU/dr_b... reported as sum_i r_a F_b."""
    E = 0.5 * k_spring * np.sum(x * x, axis=1)
    F = -k_spring * x
    Xi = x.T @ F
    return E, F, Xi
