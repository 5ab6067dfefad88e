"""O2 — image-plane taper (oracle, test infrastructure only).

The paper does not print a taper (PAPER.md:30 only says the visibilities are
convolved "with a new convolution kernel function"); north_star fixes it as
"prolate-spheroidal taper x w-screen".  Reading R2: the angular
prolate spheroidal wave function of order zero, S_00(c, nu), with
c = pi*m_t/2, m_t = 6, normalised psi(0) = 1 and psi(nu) := 0 for |nu| >= 1.
T(l, m) = psi(2l/FoV) * psi(2m/FoV).

The routine is the library one: scipy.special.pro_ang1(0, 0, c, nu).  It is
pinned in tests/test_oracle_taper.py against an independent Legendre-series
recipe (written in the test, not here) and against printed values.
"""
import numpy as np
from scipy import special

M_T = 6                      # taper width parameter m_t (reading R2)
C_PSWF = np.pi * M_T / 2.0   # c = 3*pi


def psi(nu):
    """psi(nu) = S_00(c, nu)/S_00(c, 0) for |nu| < 1, else 0.  fp64."""
    nu = np.asarray(nu, dtype=np.float64)
    out = np.zeros(nu.shape, dtype=np.float64)
    inside = np.abs(nu) < 1.0
    s0 = special.pro_ang1(0, 0, C_PSWF, 0.0)[0]
    out[inside] = special.pro_ang1(0, 0, C_PSWF, nu[inside])[0] / s0
    return out


def taper2d(l, m, fov):
    """T(l, m) = psi(2l/FoV) psi(2m/FoV) on the outer product m (rows) x l (cols)."""
    return np.outer(psi(2.0 * np.asarray(m) / fov), psi(2.0 * np.asarray(l) / fov))
