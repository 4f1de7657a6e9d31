"""BAOAB PIMD/Langevin integrator and estimators of the oracle (test infrastructure; see
oracle/__init__.py).  Everything is FP64 numpy, one statement per step of the method.

Sources: PAPER.md:L165 (B = velocity update, A = position update, O = thermostat; BAOAB),
L190-194 (normal-mode EOMs "as i-PI"; three transforms per step; thermostat target n*T),
Appendix A L319-365 (estimators), Appendix B (transform), Appendix D L464-476 (PILE_L).
Readings of garbled / silent passages: DESIGN R-1 .. R-8.

State convention: Cartesian coordinates x[P,N,3] (Angstrom, unwrapped),
normal-mode velocities vt[P,N,3] (A/ps), normal-mode forces ft[P,N,3] (eV/A).
"""
import numpy as np

from .constants import KB, MVV2E
from . import nm, philox


def b_step(vt, ft, masses, h):
    """B: velocity update over time h from the normal-mode forces:
    v~ <- v~ + h f~ / m_i, with f~/(m_i * mvv2e) the acceleration in A/ps^2 (DESIGN R-9)."""
    return vt + h * ft / (masses[None, :, None] * MVV2E)


def a_step(xt, vt, om, h):
    """A: exact free ring-polymer propagation over time h in normal-mode space (PAPER.md:L190-192
    prints no formula; DESIGN R-5 = north_star's "exact free ring-polymer propagation").
    Mode k is a harmonic oscillator of frequency omega_k (Eq. A3 spring energy, L330):
      k = 0 : x~ <- x~ + h v~
      k > 0 : x~' = cos(w h) x~ + sin(w h)/w v~ ;  v~' = -w sin(w h) x~ + cos(w h) v~ ."""
    xn = np.empty_like(xt)
    vn = np.empty_like(vt)
    for k in range(xt.shape[0]):
        w = om[k]
        if w == 0.0:
            xn[k] = xt[k] + h * vt[k]
            vn[k] = vt[k]
        else:
            c, s = np.cos(w * h), np.sin(w * h)
            xn[k] = c * xt[k] + (s / w) * vt[k]
            vn[k] = -w * s * xt[k] + c * vt[k]
    return xn, vn


def pile_l_coefficients(om, gamma0, h):
    """c1_k = exp(-h/tau_k), c2_k = sqrt(1 - c1_k^2) (Eq. D2 text) with
    tau_0 = 1/gamma0 (the `tau` keyword, L174, L464) and tau_k = 1/(2 omega_k), k >= 1 (Eq. D1)."""
    gam = 2.0 * np.asarray(om, dtype=np.float64)
    gam[0] = gamma0
    c1 = np.exp(-h * gam)
    c2 = np.sqrt(1.0 - c1 * c1)
    return c1, c2


def o_step(vt, masses, T, om, gamma0, h, seed, step, half=0):
    """O: PILE_L thermostat, Eq. D2 verbatim:
      v~_k <- c1_k v~_k + c2_k sqrt(n/(m_i beta)) eta,   eta(seed; step, k, i, alpha) from Philox.
    sqrt(n k_B T / m_i) is converted to A/ps with mvv2e.  gamma0 == 0 means NVE: the whole O step
    is skipped for every mode (DESIGN R-4)."""
    if gamma0 == 0.0:
        return vt.copy()
    P, N, _ = vt.shape
    c1, c2 = pile_l_coefficients(om, gamma0, h)
    kk, ii, aa = np.meshgrid(np.arange(P), np.arange(N), np.arange(3), indexing="ij")
    eta = philox.normal(seed, step, kk, ii, aa, half)
    sigma = np.sqrt(P * KB * T / (masses * MVV2E))            # [N]
    return c1[:, None, None] * vt + c2[:, None, None] * sigma[None, :, None] * eta


def baoab_positions_half(x, vt, ft, masses, M, om, T, gamma0, dt, seed, step):
    """First part of one BAOAB step: B(dt/2), transform x, A(dt/2), O(dt),
    A(dt/2), inverse transform (L192: "forward and inverse normal mode transformations of the
    coordinates before and after propagating the atomic positions").  O takes the full dt
    because BAOAB has a single O (DESIGN R-3).  Returns the new Cartesian x and v~."""
    vt = b_step(vt, ft, masses, 0.5 * dt)
    xt = nm.to_nm(M, x)
    xt, vt = a_step(xt, vt, om, 0.5 * dt)
    vt = o_step(vt, masses, T, om, gamma0, dt, seed, step)
    xt, vt = a_step(xt, vt, om, 0.5 * dt)
    x = nm.from_nm(M, xt)
    return x, vt


def baoab_finish(vt, f, masses, M, dt):
    """Second part: "a normal mode transformation of the forces following the force evaluation"
    (PAPER.md:L192), then the closing B(dt/2).  Returns (v~, f~)."""
    ft = nm.to_nm(M, f)
    vt = b_step(vt, ft, masses, 0.5 * dt)
    return vt, ft


def obabo_positions_half(x, vt, ft, masses, M, om, T, gamma0, dt, seed, step):
    """First part of one OBABO step (PAPER.md:L165 lists OBABO as the default Trotter splitting; L84):
    O(dt/2), B(dt/2), transform x, A(dt), inverse transform.  Each of the two O's of the step takes dt/2
    (DESIGN R-3) and its own normals (`half` = 0 here, 1 in obabo_finish)."""
    vt = o_step(vt, masses, T, om, gamma0, 0.5 * dt, seed, step, half=0)
    vt = b_step(vt, ft, masses, 0.5 * dt)
    xt = nm.to_nm(M, x)
    xt, vt = a_step(xt, vt, om, dt)
    x = nm.from_nm(M, xt)
    return x, vt


def obabo_finish(vt, f, masses, M, om, T, gamma0, dt, seed, step):
    """Second part: transform of the new forces, B(dt/2), O(dt/2).  Returns (v~, f~)."""
    ft = nm.to_nm(M, f)
    vt = b_step(vt, ft, masses, 0.5 * dt)
    vt = o_step(vt, masses, T, om, gamma0, 0.5 * dt, seed, step, half=1)
    return vt, ft


# ---- `method pimd`: integration in Cartesian coordinates (Eq. D3) ------------------------

def spring_force_cart(x, masses, wP):
    """-dS/dx of the ring springs of Eq. 1 (omega_n squared by DESIGN R-1), Cartesian:
    F^spring_k = -m omega_n^2 (2 x_k - x_{k-1} - x_{k+1}), beads cyclic; eV/A via mvv2e."""
    m = masses[None, :, None]
    return -m * wP * wP * MVV2E * (2.0 * x - np.roll(x, 1, axis=0) - np.roll(x, -1, axis=0))


def o_step_cart(v, masses, T, wP, gamma0, h, seed, step, half=0):
    """Eq. D3: v_k <- c1 v_k + c2 sqrt(n/(m beta)) eta for EVERY bead k with the same
    c1 = exp(-h/tau_0), tau_0 = 1/(2 omega_n) (L478: "the default damping time is tau_k = 1/(2 omega_n),
    k = 0..n-1"; DESIGN R-27: the `tau` keyword does not enter, gamma0 == 0 still means no thermostat).
    eta(seed; step, k, i, alpha) is the stream of Eq. D2 with the bead index in place of the mode index."""
    if gamma0 == 0.0:
        return v.copy()
    P, N, _ = v.shape
    c1 = np.exp(-h * 2.0 * wP)
    c2 = np.sqrt(1.0 - c1 * c1)
    kk, ii, aa = np.meshgrid(np.arange(P), np.arange(N), np.arange(3), indexing="ij")
    eta = philox.normal(seed, step, kk, ii, aa, half)
    sigma = np.sqrt(P * KB * T / (masses * MVV2E))
    return c1 * v + c2 * sigma[None, :, None] * eta


def cart_kick(v, x, f, masses, wP, h):
    """B in Cartesian coordinates: the bead force plus the ring-spring force (both terms of Eq. 1's potential)."""
    return v + h * (f + spring_force_cart(x, masses, wP)) / (masses[None, :, None] * MVV2E)


def cart_positions_half(x, v, f, masses, T, wP, gamma0, dt, seed, step, obabo):
    """First part of one Cartesian step (DESIGN R-27; A is the plain drift x += h v, L165 "position update"):
    BAOAB: B(dt/2) A(dt/2) O(dt) A(dt/2);  OBABO: O(dt/2) B(dt/2) A(dt)."""
    if obabo:
        v = o_step_cart(v, masses, T, wP, gamma0, 0.5 * dt, seed, step, half=0)
        v = cart_kick(v, x, f, masses, wP, 0.5 * dt)
        return x + dt * v, v
    v = cart_kick(v, x, f, masses, wP, 0.5 * dt)
    x = x + 0.5 * dt * v
    v = o_step_cart(v, masses, T, wP, gamma0, dt, seed, step)
    x = x + 0.5 * dt * v
    return x, v


def cart_finish(x, v, f, masses, T, wP, gamma0, dt, seed, step, obabo):
    """Second part: B(dt/2) with the new bead forces and the springs at the new positions (+ O(dt/2) for OBABO)."""
    v = cart_kick(v, x, f, masses, wP, 0.5 * dt)
    if obabo:
        v = o_step_cart(v, masses, T, wP, gamma0, 0.5 * dt, seed, step, half=1)
    return v


def remove_centroid_com(vt, masses):
    """`fixcom yes`: "the center-of-mass velocity is removed in every timestep for the
    centroid mode" (nmpimd).  v~_0,i <- v~_0,i - sum_j m_j v~_0,j / sum_j m_j, per Cartesian component;
    applied once per step after its last velocity update (DESIGN R-19: the paper does not say where)."""
    out = vt.copy()
    vcom = np.sum(masses[:, None] * vt[0], axis=0) / np.sum(masses)
    out[0] = vt[0] - vcom[None, :]
    return out


def remove_bead_com(v, masses):
    """`fixcom yes` under `method pimd`: the center-of-mass velocity is removed "for each bead
    individually".  v_k,i <- v_k,i - sum_j m_j v_k,j / sum_j m_j for every bead k, per Cartesian component; applied once
    per step after its last velocity update, like the centroid variant (DESIGN R-19).  v[P,N,3] Cartesian."""
    vcom = np.sum(masses[None, :, None] * v, axis=1) / np.sum(masses)          # [P, 3]
    return v - vcom[:, None, :]


def estimators(x, vt, f, U, masses, M, om, T):
    """Appendix A outputs that the hot path reports, on unwrapped coordinates
    (L202).  x, f Cartesian [P,N,3]; vt normal-mode velocities; U[P] bead potential energies.

      K^(k)  = sum_i 1/2 m_i v~_i^(k)2                       (A1, L319)
      S^(k)  = sum_i 1/2 m_i omega_k^2 x~_i^(k)2             (A3, L330; omega_n lambda_k printed
                                                              without the square: DESIGN R-1)
      H      = sum_k K + S + U                               (A6, L350)
      K_PR   = 3 n N k_B T/2 - (1/n) sum_k sum_i 1/2 m_i omega_n^2 |r^(k)-r^(k+1)|^2
                                                             (A7, L354; the 1/n and the square are
                                                              DESIGN R-6, pinned by the HO test)
      K_CV   = 3 N k_B T/2 - 1/(2n) sum_k sum_i (r^(k)-r^c).F^(k)       (A9, L365)
      T_ring = 2 sum_k K^(k) / (3 n N k_B)  -- averages n*T (L194, Fig. 2 caption L120)
    """
    P, N, _ = x.shape
    m = masses[None, :, None]
    xt = nm.to_nm(M, x)
    K_k = 0.5 * np.sum(m * vt * vt, axis=(1, 2)) * MVV2E
    S_k = 0.5 * np.sum(m * (om[:, None, None] ** 2) * xt * xt, axis=(1, 2)) * MVV2E
    wP = nm.omega_P(P, T)
    dr = x - np.roll(x, -1, axis=0)                      # r^(k) - r^(k+1), r^(n) = r^(0)
    spring_cart = 0.5 * np.sum(m * wP * wP * dr * dr) * MVV2E
    K_PR = 1.5 * P * N * KB * T - spring_cart / P
    rc = np.mean(x, axis=0, keepdims=True)
    K_CV = 1.5 * N * KB * T - np.sum((x - rc) * f) / (2.0 * P)
    K_ring = float(np.sum(K_k))
    S_ring = float(np.sum(S_k))
    U_sum = float(np.sum(U))
    return {
        "K_PR": float(K_PR), "K_CV": float(K_CV), "H": K_ring + S_ring + U_sum,
        "K_ring": K_ring, "S_ring": S_ring, "U_sum": U_sum,
        "T_ring": 2.0 * K_ring / (3.0 * P * N * KB), "K_k": K_k, "S_k": S_k,
        "spring_cart": float(spring_cart),
    }
