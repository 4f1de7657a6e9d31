"""Physical constants of the oracle (test infrastructure; see oracle/__init__.py).

Units are LAMMPS "metal": Angstrom, ps, eV, g/mol, K.  Two of the three constants are
printed in the paper's worked example, PAPER.md:L458 (Appendix C):
  h      = 4.135667403e-3 eV*ps
  mvv2e  = 1.0364269e-4   eV per (g/mol)(A/ps)^2
k_B is not printed anywhere in the paper; DESIGN R-9 takes the CODATA value.
"""
import math

H_PLANCK = 4.135667403e-3            # eV ps
HBAR = H_PLANCK / (2.0 * math.pi)    # eV ps
MVV2E = 1.0364269e-4                 # eV / ((g/mol) (A/ps)^2)
KB = 8.617333262e-5                  # eV / K       DESIGN R-9
