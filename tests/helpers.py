"""Independent re-derivations used to pin the oracle (mpmath / exact rationals / numpy).

Nothing here calls the oracle or the CUDA path.
"""
from fractions import Fraction

import mpmath as mp
import numpy as np

mp.mp.dps = 50
K = mp.mpf("1.267")          # phase constant, R1


def fma_exact(a: float, b: float, c: float) -> float:
    """Correctly rounded a*b+c (what std::fma / __fma_rn return) via exact rationals."""
    return float(Fraction(a) * Fraction(b) + Fraction(c))


def escale_exact(a0, a1, a2, v):
    return fma_exact(fma_exact(a2, v, a1), v, a0)


def angles(s2_2theta):
    """theta in the first octant from sin^2(2 theta) (R4)."""
    return mp.asin(mp.sqrt(mp.mpf(s2_2theta))) / 2


def pee_eq1_mp(s13, mee, s12, m21, L, E):
    """PAPER.md:34 Eq. 1 typed directly from the paper with angles, 50 digits."""
    t13, t12 = angles(s13), angles(s12)
    x = mp.mpf(L) / mp.mpf(E)
    return (1 - mp.sin(2 * t13) ** 2 * mp.sin(K * mp.mpf(mee) * x) ** 2
            - mp.cos(t13) ** 4 * mp.sin(2 * t12) ** 2 * mp.sin(K * mp.mpf(m21) * x) ** 2)


def pee_full3_mp(s13, mee, s12, m21, L, E, ordering=+1):
    """Textbook 3-flavour vacuum survival probability from the PMNS elements
    |U_e1|^2 = c12^2 c13^2, |U_e2|^2 = s12^2 c13^2, |U_e3|^2 = s13^2:
        P = 1 - 4 sum_{i<j} |U_ei|^2 |U_ej|^2 sin^2(D_ij)
    with dm31, dm32 from inverting PAPER.md:39 Eq. 2."""
    t13, t12 = angles(s13), angles(s12)
    c12, s12_, c13, s13_ = mp.cos(t12), mp.sin(t12), mp.cos(t13), mp.sin(t13)
    U1, U2, U3 = (c12 * c13) ** 2, (s12_ * c13) ** 2, s13_ ** 2
    o = 1 if ordering >= 0 else -1
    m21 = mp.mpf(m21)
    mee = mp.mpf(mee)
    # Eq. 2: mee = c12^2 |dm31| + s12^2 |dm32|, and | |dm31| - |dm32| | = dm21 with the sign set by the ordering
    m31 = mee + o * s12_ ** 2 * m21
    m32 = mee - o * c12 ** 2 * m21
    x = mp.mpf(L) / mp.mpf(E)
    return (1 - 4 * U1 * U2 * mp.sin(K * m21 * x) ** 2
            - 4 * U1 * U3 * mp.sin(K * m31 * x) ** 2
            - 4 * U2 * U3 * mp.sin(K * m32 * x) ** 2)


def pee_eq10_repaired_mp(s13, mee, s12, m21, L, E, ordering=+1):
    """PAPER.md:219-226 Eq. 10 after the repair of DESIGN.md R2 (the printed form is garbled):
        P = 1 - 1/2 s13 [1 - sqrt(1 - s12 sin^2 D21) cos(2 D_ee +- phi)] - c13^4 s12 sin^2 D21,
        phi = atan2(cos(2th12) sin D21 ... ) on the continuous branch; evaluated here through
        sin(phi), cos(phi) so that no branch choice is needed:
        sqrt(1 - s12 sin^2 D21) cos(phi_full) = c12^2 cos(2 s12^2 D21) + s12^2 cos(2 c12^2 D21)
        sqrt(1 - s12 sin^2 D21) sin(phi_full) = c12^2 sin(2 s12^2 D21) - s12^2 sin(2 c12^2 D21)
    (Parke 2016, ref. [8] of the paper, re-derived)."""
    t13, t12 = angles(s13), angles(s12)
    c12sq, s12sq = mp.cos(t12) ** 2, mp.sin(t12) ** 2
    x = mp.mpf(L) / mp.mpf(E)
    D21 = K * mp.mpf(m21) * x
    Dee = K * mp.mpf(mee) * x
    o = 1 if ordering >= 0 else -1
    Rc = c12sq * mp.cos(2 * s12sq * D21) + s12sq * mp.cos(2 * c12sq * D21)
    Rs = c12sq * mp.sin(2 * s12sq * D21) - s12sq * mp.sin(2 * c12sq * D21)
    # sqrt(.) cos(2 Dee +- phi) = cos(2Dee) Rc -+ sin(2Dee) Rs
    amp_cos = mp.cos(2 * Dee) * Rc - o * mp.sin(2 * Dee) * Rs
    assert abs(Rc ** 2 + Rs ** 2 - (1 - mp.mpf(s12) * mp.sin(D21) ** 2)) < mp.mpf("1e-40")
    return (1 - mp.mpf(s13) / 2 * (1 - amp_cos)
            - mp.cos(t13) ** 4 * mp.mpf(s12) * mp.sin(D21) ** 2)


def hist_right(values, weights, edges):
    """Plain weighted histogram, half-open bins [e_b, e_b+1), outside dropped (R7)."""
    values = np.asarray(values, dtype=np.float64)
    idx = np.searchsorted(edges, values, side="right") - 1
    ok = (values >= edges[0]) & (values < edges[-1])
    return np.bincount(idx[ok], weights=np.asarray(weights, dtype=np.float64)[ok],
                       minlength=len(edges) - 1)[: len(edges) - 1]
