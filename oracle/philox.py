"""Counter-based random numbers of the oracle (test infrastructure; see oracle/__init__.py).

The paper's thermostat needs one standard normal eta per (mode k, atom i, component alpha)
and step (Eq. D2); the paper itself seeds one LAMMPS generator per fix
(PAPER.md:L84).  BASELINE.json's north_star replaces that by counter-based Philox normals
keyed by (seed, step, bead, atom, dim); the keying below is DESIGN R-10.

Philox4x32-10 is restated here from its published definition (Salmon et al., SC'11):
ten rounds of two 32x32->64 multiplies with the key bumped by Weyl constants between rounds.
"""
import numpy as np

_M0 = np.uint64(0xD2511F53)
_M1 = np.uint64(0xCD9E8D57)
_W0 = np.uint64(0x9E3779B9)
_W1 = np.uint64(0xBB67AE85)
_MASK = np.uint64(0xFFFFFFFF)
_S32 = np.uint64(32)


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """Philox4x32 with 10 rounds.  All arguments: integer arrays (broadcastable) holding 32-bit
    words.  Returns the four output words as uint64 arrays with values < 2**32."""
    c0, c1, c2, c3, k0, k1 = np.broadcast_arrays(
        *[np.asarray(a, dtype=np.uint64) & _MASK for a in (c0, c1, c2, c3, k0, k1)])
    c0, c1, c2, c3, k0, k1 = (a.copy() for a in (c0, c1, c2, c3, k0, k1))
    for rnd in range(10):
        if rnd > 0:                      # key schedule: bump before every round but the first
            k0 = (k0 + _W0) & _MASK
            k1 = (k1 + _W1) & _MASK
        p0 = _M0 * c0                    # 64-bit products (operands < 2**32: no overflow)
        p1 = _M1 * c2
        hi0, lo0 = p0 >> _S32, p0 & _MASK
        hi1, lo1 = p1 >> _S32, p1 & _MASK
        c0, c1, c2, c3 = hi1 ^ c1 ^ k0, lo1, hi0 ^ c3 ^ k1, lo0
    return c0, c1, c2, c3


def words_for(seed, step, k, i, alpha, half=0):
    """The four Philox words behind thermostat normal (step, mode k, atom i, component alpha).
    DESIGN R-10: key = (seed_lo32, seed_hi32); counter = (step_lo32, step_hi32, i, 4*(k//2) + alpha):
    modes 2q and 2q+1 share one call and take the two Box-Muller branches (see `normal`).
    `half` = 1 selects the second thermostat half-step of an OBABO step (bit 31 of counter word 1;
    steps are < 2**63); BAOAB's single O uses half = 0."""
    seed = int(seed) & 0xFFFFFFFFFFFFFFFF
    step = int(step) & 0xFFFFFFFFFFFFFFFF
    k = np.asarray(k, dtype=np.uint64)
    i = np.asarray(i, dtype=np.uint64)
    alpha = np.asarray(alpha, dtype=np.uint64)
    return philox4x32_10(step & 0xFFFFFFFF, (step >> 32) | (int(half) << 31), i, np.uint64(4) * (k >> np.uint64(1)) + alpha,
                         seed & 0xFFFFFFFF, seed >> 32)


def uniform53(wa, wb):
    """53-bit uniform on the grid {0, 1, .., 2^53-1} * 2^-53 in [0,1):
    ((wa>>5)*2^26 + (wb>>6)) * 2^-53, exact in FP64 (DESIGN R-10)."""
    wa = np.asarray(wa, dtype=np.uint64)
    wb = np.asarray(wb, dtype=np.uint64)
    n = (wa >> np.uint64(5)) * np.uint64(1 << 26) + (wb >> np.uint64(6))   # < 2**53, exact
    return n.astype(np.float64) * (2.0 ** -53)


def normal(seed, step, k, i, alpha, half=0):
    """eta ~ N(0,1) of Eq. D2 by Box-Muller (DESIGN R-10):
    u1 = uniform53(w0,w1) + 2^-53 in (0,1] (so the logarithm is finite; the sum is exact),
    u2 = uniform53(w2,w3) in [0,1);  r = sqrt(-2 ln u1);
    eta = r cos(2 pi u2) for even k, r sin(2 pi u2) for odd k -- the two branches of one draw are
    independent standard normals, so one Philox call serves the mode pair (2q, 2q+1)."""
    w0, w1, w2, w3 = words_for(seed, step, k, i, alpha, half)
    u1 = uniform53(w0, w1) + 2.0 ** -53
    u2 = uniform53(w2, w3)
    r = np.sqrt(-2.0 * np.log(u1))
    odd = (np.asarray(k, dtype=np.uint64) & np.uint64(1)).astype(bool)
    return np.where(odd, r * np.sin(2.0 * np.pi * u2), r * np.cos(2.0 * np.pi * u2))
