"""The whole hot path, step by step -- oracle (test infrastructure; see oracle/__init__.py).

`OraclePIMD` mirrors the problem statement of the C-ABI (create with types, masses, box, P, T,
dt, gamma, seed; set_state; set_model; step(n); getters) but shares nothing with it.
One step = PAPER.md:L165 BAOAB with the three normal-mode transforms of L192 and one force
evaluation per step placed after the second A (DESIGN R-7); estimators (Appendix A) are taken
after the closing B with x, f consistent.
"""
import numpy as np

from .constants import KB, MVV2E
from . import nm, integrator, se_e2_a, barostat


class OraclePIMD:
    def __init__(self, types, masses_per_type, box, n_beads, T, dt, gamma_centroid, seed, integrator="baoab", fixcom=False,
                 method="nmpimd"):
        self.types = np.asarray(types, dtype=np.int64)
        self.N = self.types.size
        self.masses = np.asarray(masses_per_type, dtype=np.float64)[self.types]   # per atom
        self.box = np.asarray(box, dtype=np.float64)
        self.P = int(n_beads)
        self.T = float(T)
        self.dt = float(dt)
        self.gamma0 = float(gamma_centroid)
        self.seed = int(seed)
        assert integrator in ("baoab", "obabo")
        self.integrator = integrator
        self.fixcom = bool(fixcom)
        assert method in ("nmpimd", "pimd")
        self.method = method                             # PAPER.md:L164; "pimd" = Cartesian (DESIGN R-27)
        self.M = nm.nm_matrix(self.P)
        self.om = nm.omegas(self.P, self.T)
        self.step_count = 0
        self.model = None
        self.k_spring = None
        self.x = None
        self.vt = None
        self.f = None
        self.ft = None
        self.U = np.zeros(self.P)
        self.Xi = np.zeros((self.P, 3, 3))
        self.only_beads = None       # bench.py's bounded cpu_baseline sample: evaluate these beads only
        self.baro = False            # isotropic BZP barostat (NpH; NpT when gamma0 > 0)
        self.aniso = False
        self.vW = 0.0
        self.p_ext = 0.0
        self.W = 0.0

    # ---- inputs ----
    def set_state(self, x, p):
        """x[P,N,3] unwrapped Cartesian (A); p[P,N,3] Cartesian bead momenta ((g/mol) A/ps).
        Internally v~ = M (p/m) (velocities live in normal-mode form)."""
        self.x = np.array(x, dtype=np.float64).reshape(self.P, self.N, 3)
        v = np.asarray(p, dtype=np.float64).reshape(self.P, self.N, 3) / self.masses[None, :, None]
        self.vt = v.copy() if self.method == "pimd" else nm.to_nm(self.M, v)     # `pimd`: vt holds Cartesian v
        self.step_count = 0
        if self.model is not None or self.k_spring is not None:
            self._forces()

    def set_model(self, desc, weights, compressed=False):
        """compressed=True: the tabulated embedding net of oracle/compress.py (DESIGN R-28)."""
        self.model = se_e2_a.Model(desc, weights)
        if compressed:
            from . import compress
            compress.compress(self.model)
        self.k_spring = None
        if self.x is not None:
            self._forces()

    def set_model_harmonic(self, k_spring):
        self.k_spring = float(k_spring)
        self.model = None
        if self.x is not None:
            self._forces()

    def set_barostat(self, p_ext_bar, tau_p, aniso=False):
        """`iso p_ext barostat BZP taup tau_p`: isotropic target pressure in bar,
        barostat mass W = 3 n N k_B T tau_p^2 (L389); v_W starts at 0.  Sub-step order: DESIGN R-24."""
        assert not self.fixcom and self.method == "nmpimd"
        self.baro = True
        self.p_ext = float(p_ext_bar) / barostat.BAR_PER_EV_A3
        self.aniso = bool(aniso)                     # PAPER.md:L176 `aniso`: one v_W per cell vector (Eq. E2-E3, A14)
        if self.aniso:
            self.W = barostat.barostat_mass_aniso(self.P, self.N, self.T, float(tau_p))
            self.vW = np.zeros(3)
        else:
            self.W = barostat.barostat_mass(self.P, self.N, self.T, float(tau_p))
            self.vW = 0.0

    def _press_v(self, h):
        fn = barostat.press_v_step_aniso if self.aniso else barostat.press_v_step
        self.vW = fn(self.vW, self.x, self.vt, self.ft, self.Xi, self.masses, float(np.prod(self.box)), self.T,
                     self.W, self.p_ext, h)

    def _press_o(self, h, half=0):
        if self.gamma0 != 0.0:
            fn = barostat.press_o_step_aniso if self.aniso else barostat.press_o_step
            self.vW = fn(self.vW, self.P, self.N, self.T, self.W, self.gamma0, h, self.seed, self.step_count, half)

    # ---- the path ----
    def _forces(self):
        f = np.zeros((self.P, self.N, 3))
        beads = range(self.P) if self.only_beads is None else self.only_beads
        for k in beads:
            if self.k_spring is not None:
                E, F, Xi = se_e2_a.harmonic_energy_forces(self.x[k], self.k_spring)
            else:
                E, F, Xi = se_e2_a.energy_forces(self.x[k], self.types, self.box, self.model)
            f[k] = F
            self.U[k] = E.sum()
            self.Xi[k] = Xi
        self.f = f
        self.ft = nm.to_nm(self.M, f)

    def _drift_half(self, xt, h):
        """A(h) (h = dt/2 in BAOAB, dt in OBABO) with the cell: centroid by Eq. E4-E6, modes k >= 1 by the free ring-polymer rotation (R-21)."""
        xq, vq, self.box = (barostat.qc_step_aniso if self.aniso else barostat.qc_step)(xt, self.vt, self.box, self.vW, h)
        xa, va = integrator.a_step(xt, self.vt, self.om, h)
        xa[0], va[0] = xq[0], vq[0]
        self.vt = va
        return xa

    def _npt_step(self):
        """One BAOAB step with the BZP barostat (DESIGN R-24; the paper prints the sub-steps, Appendix E, but not
        their order): [E1(dt/2), B(dt/2)], [E4-E6 + A](dt/2), [O(dt), E7(dt)], [E4-E6 + A](dt/2), forces at the new
        positions and cell, [E1(dt/2), B(dt/2)] -- every barostat sub-step sits next to the atomic sub-step of
        the same letter and takes its length."""
        h = 0.5 * self.dt
        self._press_v(h)
        self.vt = integrator.b_step(self.vt, self.ft, self.masses, h)
        xt = nm.to_nm(self.M, self.x)
        xt = self._drift_half(xt, h)
        self.vt = integrator.o_step(self.vt, self.masses, self.T, self.om, self.gamma0, self.dt, self.seed,
                                    self.step_count)
        self._press_o(self.dt)
        xt = self._drift_half(xt, h)
        self.x = nm.from_nm(self.M, xt)
        self._forces()
        self._press_v(h)
        self.vt = integrator.b_step(self.vt, self.ft, self.masses, h)
        self.step_count += 1

    def _npt_step_obabo(self):
        """One OBABO step (the fix's default splitting, PAPER.md:L82-84 runs it with `ensemble npt`) with the BZP
        barostat, DESIGN R-24: [O, E7](dt/2), [E1, B](dt/2), [E4-E6 + A](dt), forces, [E1, B](dt/2), [O, E7](dt/2)."""
        h = 0.5 * self.dt
        self.vt = integrator.o_step(self.vt, self.masses, self.T, self.om, self.gamma0, h, self.seed,
                                    self.step_count, half=0)
        self._press_o(h, half=0)
        self._press_v(h)
        self.vt = integrator.b_step(self.vt, self.ft, self.masses, h)
        xt = nm.to_nm(self.M, self.x)
        xt = self._drift_half(xt, self.dt)
        self.x = nm.from_nm(self.M, xt)
        self._forces()
        self._press_v(h)
        self.vt = integrator.b_step(self.vt, self.ft, self.masses, h)
        self.vt = integrator.o_step(self.vt, self.masses, self.T, self.om, self.gamma0, h, self.seed,
                                    self.step_count, half=1)
        self._press_o(h, half=1)
        self.step_count += 1

    def _cart_step(self):
        wP = nm.omega_P(self.P, self.T)
        ob = self.integrator == "obabo"
        self.x, self.vt = integrator.cart_positions_half(self.x, self.vt, self.f, self.masses, self.T, wP,
                                                         self.gamma0, self.dt, self.seed, self.step_count, ob)
        self._forces()
        self.vt = integrator.cart_finish(self.x, self.vt, self.f, self.masses, self.T, wP, self.gamma0, self.dt,
                                         self.seed, self.step_count, ob)
        if self.fixcom:
            self.vt = integrator.remove_bead_com(self.vt, self.masses)      # L180: "for each bead individually"
        self.step_count += 1

    def step(self, n_steps=1):
        for _ in range(int(n_steps)):
            if self.method == "pimd":
                self._cart_step()
                continue
            if self.baro:
                if self.integrator == "obabo":
                    self._npt_step_obabo()
                else:
                    self._npt_step()
                continue
            if self.integrator == "obabo":
                self.x, self.vt = integrator.obabo_positions_half(
                    self.x, self.vt, self.ft, self.masses, self.M, self.om, self.T, self.gamma0,
                    self.dt, self.seed, self.step_count)
                self._forces()
                self.vt, _ = integrator.obabo_finish(self.vt, self.f, self.masses, self.M, self.om, self.T,
                                                     self.gamma0, self.dt, self.seed, self.step_count)
                if self.fixcom:
                    self.vt = integrator.remove_centroid_com(self.vt, self.masses)
                self.step_count += 1
                continue
            self.x, self.vt = integrator.baoab_positions_half(
                self.x, self.vt, self.ft, self.masses, self.M, self.om, self.T, self.gamma0,
                self.dt, self.seed, self.step_count)
            self._forces()                                   # one force evaluation per step
            self.vt, _ = integrator.baoab_finish(self.vt, self.f, self.masses, self.M, self.dt)
            if self.fixcom:
                self.vt = integrator.remove_centroid_com(self.vt, self.masses)
            self.step_count += 1

    # ---- outputs ----
    def positions(self):
        return self.x.copy()

    def momenta(self):
        """Cartesian bead momenta p = m M^T v~."""
        if self.method == "pimd":
            return self.vt * self.masses[None, :, None]
        return nm.from_nm(self.M, self.vt) * self.masses[None, :, None]

    def forces(self):
        return self.f.copy()

    def virial(self):
        return self.Xi.copy()

    def energies(self):
        return self.U.copy()

    def estimators(self):
        vt = nm.to_nm(self.M, self.vt) if self.method == "pimd" else self.vt      # Appendix A is written in v~
        e = integrator.estimators(self.x, vt, self.f, self.U, self.masses, self.M, self.om, self.T)
        e["step"] = self.step_count
        return e

    def barostat_state(self):
        """Outputs 8-15 of Appendix A; pressures in bar."""
        e = self.estimators()
        V = float(np.prod(self.box))
        KW, UW, JW = barostat.extended_terms(self.vW, V, self.P, self.T, self.W, self.p_ext)
        bar = barostat.BAR_PER_EV_A3
        return {
            "v_W": float(np.mean(self.vW)), "v_W3": np.broadcast_to(self.vW, (3,)).copy(), "box": self.box.copy(), "V": V,
            "P_CV3": barostat.p_cv_diag(self.x, self.vt, self.ft, self.Xi, self.masses, V) * bar,
            "P_CV": barostat.p_cv(self.x, self.vt, self.ft, self.Xi, self.masses, V) * bar,
            "P_PR": barostat.p_pr(e["S_ring"], self.P, self.N, self.T, V) * bar,
            "P_MD": barostat.p_md(e["K_ring"], self.Xi, V) * bar,
            "K_W": KW, "U_W": UW, "J_W": JW, "enthalpy": e["H"] + KW + UW + JW,     # A17
        }
