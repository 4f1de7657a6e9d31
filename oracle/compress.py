"""Tabulated ("compressed") embedding net of the oracle (test infrastructure; see oracle/__init__.py).

The paper's benchmarks run a *compressed* DP model (ref. 41, "DP Compress", is only cited): the
embedding net G(s) of each ordered type pair -- a function of ONE scalar -- is replaced by a piecewise polynomial
table.  SURVEY 8(f) NEXT-3.  DESIGN R-28 fixes what the paper does not print:
  * uniform grid s_n = s_lo + n h on [s_lo, s_hi] = [0, 2] (s = 1/r for r < r_s = 0.5 A, so r >= 0.5 A is covered;
    a row outside the table is an error, not an extrapolation), stride h = 0.05;
  * on [s_n, s_n + h] the quintic Hermite polynomial in t = s - s_n that matches G, G', G'' at both nodes
    (C^2 across nodes); G', G'' by forward-mode differentiation of the tanh net;
  * the backward pass uses the derivative of the SAME polynomial (so forces stay the exact gradient of the
    compressed energy).
It is an approximation of the MLP: |G~ - G| <= h^6 max|G^(6)| / 46080 (quintic Hermite remainder), pinned in
tests/test_oracle_compress.py together with the node conditions and the energy / force consistency.
This round holds the oracle only; the CUDA kernel of NEXT-3 is not built yet.
"""
import numpy as np

S_LO, S_HI, STRIDE = 0.0, 2.0, 0.05


def mlp_value_d1_d2(layers, s):
    """G(s), dG/ds, d2G/ds2 of the embedding net (DESIGN R-13: h <- [h,h] + tanh(hW+b) where the width doubles,
    h <- tanh(.) on the first layer) by forward-mode differentiation; s[R] -> three arrays [R, M1]."""
    s = np.asarray(s, dtype=np.float64)
    h = s[:, None]
    h1 = np.ones_like(h)
    h2 = np.zeros_like(h)
    for (W, b) in layers:
        n_in, n_out = W.shape
        z, z1, z2 = h @ W + b, h1 @ W, h2 @ W
        t = np.tanh(z)
        u = 1.0 - t * t                                   # tanh'
        t1 = u * z1
        t2 = u * z2 - 2.0 * t * u * z1 * z1               # (tanh z)'' = tanh'(z) z'' + tanh''(z) z'^2
        if n_out == 2 * n_in:
            h = np.concatenate([h, h], axis=1) + t
            h1 = np.concatenate([h1, h1], axis=1) + t1
            h2 = np.concatenate([h2, h2], axis=1) + t2
        elif n_out == n_in:
            h, h1, h2 = h + t, h1 + t1, h2 + t2
        else:
            h, h1, h2 = t, t1, t2
    return h, h1, h2


def build_table(layers, s_lo=S_LO, s_hi=S_HI, h=STRIDE):
    """coef[n, p, m]: G~_m(s) = sum_p coef[n, p, m] t^p on interval n, t = s - (s_lo + n h)."""
    n_int = int(round((s_hi - s_lo) / h))
    nodes = s_lo + h * np.arange(n_int + 1)
    y, y1, y2 = mlp_value_d1_d2(layers, nodes)
    M = y.shape[1]
    coef = np.empty((n_int, 6, M))
    coef[:, 0] = y[:-1]
    coef[:, 1] = y1[:-1]
    coef[:, 2] = 0.5 * y2[:-1]
    # the cubic..quintic part q(t) = a3 t^3 + a4 t^4 + a5 t^5 takes what is left at the right node
    d0 = y[1:] - (y[:-1] + h * y1[:-1] + 0.5 * h * h * y2[:-1])
    d1 = y1[1:] - (y1[:-1] + h * y2[:-1])
    d2 = y2[1:] - y2[:-1]
    A = np.array([[h ** 3, h ** 4, h ** 5],
                  [3 * h ** 2, 4 * h ** 3, 5 * h ** 4],
                  [6 * h, 12 * h ** 2, 20 * h ** 3]])
    sol = np.linalg.solve(A, np.stack([d0.ravel(), d1.ravel(), d2.ravel()]))      # [3, n_int*M]
    coef[:, 3:] = sol.reshape(3, n_int, M).transpose(1, 0, 2)
    return {"s_lo": float(s_lo), "h": float(h), "n": n_int, "coef": coef}


def table_eval(tab, s):
    """G~(s) and dG~/ds, [R, M1] each.  Raises when a row lies outside the table (R-28)."""
    s = np.asarray(s, dtype=np.float64)
    u = (s - tab["s_lo"]) / tab["h"]
    if s.size and (u.min() < 0.0 or u.max() > tab["n"]):
        raise OverflowError("environment value s outside the compression table")
    iv = np.minimum(np.floor(u).astype(np.int64), tab["n"] - 1)
    t = (s - (tab["s_lo"] + tab["h"] * iv))[:, None]
    c = tab["coef"][iv]                                   # [R, 6, M]
    G = ((((c[:, 5] * t + c[:, 4]) * t + c[:, 3]) * t + c[:, 2]) * t + c[:, 1]) * t + c[:, 0]
    Gp = (((5.0 * c[:, 5] * t + 4.0 * c[:, 4]) * t + 3.0 * c[:, 3]) * t + 2.0 * c[:, 2]) * t + c[:, 1]
    return G, Gp


def compress(model, s_lo=S_LO, s_hi=S_HI, h=STRIDE):
    """Attach the tables of all ordered type pairs to an oracle Model: se_e2_a.energy_forces then evaluates the
    embedding through them."""
    model.tables = {pair: build_table(layers, s_lo, s_hi, h) for pair, layers in model.emb.items()}
    return model
