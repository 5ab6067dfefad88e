"""O3 — oversampled W-kernel stack, K1-K6 (oracle, test infrastructure only).

The paper cites the method to Cornwell, Golap & Bhatnagar 2008
and gives only the parameters (23 planes, full support 9).
Every choice below is a DESIGN.md reading (R1-R7); the steps are written in
the order and notation of SURVEY.md §8(c):

K1  w_p = -w_max + (p + 1/2) * dw,  dw = 2 w_max / Nw
K2  Nk = max(32, next_pow2(4 S));  l_a = (a - Nk/2) FoV / Nk
    F_p[b][a] = T(l_a, m_b) exp(+2 pi i w_p (n_ab - 1)),
    n - 1 = -r^2 / (1 + sqrt(1 - r^2)),  F := 0 where r^2 >= 1
K3  C_p[t_v][t_u] = sum_b sum_a F_p[b][a]
                    exp(-2 pi i (t_u (a - Nk/2) + t_v (b - Nk/2)) / (Q Nk)),
    t in [-S Q/2 + 1, S Q/2]           (written as E F E^T, a library matmul)
K4  K[p][ov][ou][iv][iu] = C_p[t(iv, ov)][t(iu, ou)] / s,
    t(i, o) = (i + 1) Q - S Q / 2 - o
K5  s = Re sum of the S x S slice at the on-cell offset o* (0 for even S,
    Q/2 for odd S) of the table built with w = 0
K6  ragged: S_p = clamp(2 ceil(sqrt((m_t/2)^2 + (|w_p| FoV^2 / 2)^2)),
    S_min, S_max); K2-K4 per plane with its own S_p, Nk; K5 uses S_min.
"""
from dataclasses import dataclass
import math
import numpy as np

from .taper import psi, M_T


@dataclass
class KernelStack:
    data: np.ndarray          # flat complex128, planes concatenated
    support: np.ndarray       # [Nw] int32, S_p
    plane_offset: np.ndarray  # [Nw+1] int64, element offsets into data
    Nw: int
    oversample: int
    grid_N: int
    cell: float
    w_max: float

    def plane(self, p):
        """View K[p] as [Q][Q][S_p][S_p]."""
        S, Q = int(self.support[p]), self.oversample
        return self.data[self.plane_offset[p]:self.plane_offset[p + 1]].reshape(Q, Q, S, S)

    @property
    def uniform(self):
        return bool(np.all(self.support == self.support[0]))

    def as_array(self):
        """Uniform stacks only: K[Nw][Q][Q][S][S]."""
        assert self.uniform
        S, Q = int(self.support[0]), self.oversample
        return self.data.reshape(self.Nw, Q, Q, S, S)


def plane_centres(Nw, w_max):
    """K1."""
    dw = 2.0 * w_max / Nw
    return -w_max + (np.arange(Nw) + 0.5) * dw


def nk_of(S):
    """K2: image-plane sample count per axis."""
    return max(32, 1 << int(math.ceil(math.log2(4 * S))))


def ragged_support(Nw, w_max, grid_N, cell, S_min, S_max):
    """K6: per-plane full support."""
    fov = grid_N * cell
    wp = plane_centres(Nw, w_max)
    S = 2 * np.ceil(np.sqrt((M_T / 2.0) ** 2 + (np.abs(wp) * fov * fov / 2.0) ** 2))
    return np.clip(S, S_min, S_max).astype(np.int32)


def image_plane_samples(w, S, fov):
    """K2: F[b][a] (rows m_b, columns l_a) for one w value."""
    Nk = nk_of(S)
    a = np.arange(Nk)
    l = (a - Nk / 2) * fov / Nk
    T = np.outer(psi(2.0 * l / fov), psi(2.0 * l / fov))
    r2 = l[None, :] ** 2 + l[:, None] ** 2
    ok = r2 < 1.0
    r2c = np.where(ok, r2, 0.0)
    nm1 = -r2c / (1.0 + np.sqrt(1.0 - r2c))
    F = T * np.exp(2j * np.pi * w * nm1)
    return np.where(ok, F, 0.0)


def uv_table(F, S, Q):
    """K3: C[t_v][t_u], index 0 is t = -S Q/2 + 1."""
    Nk = F.shape[0]
    assert (S * Q) % 2 == 0
    t = np.arange(-S * Q // 2 + 1, S * Q // 2 + 1)
    a = np.arange(Nk) - Nk // 2
    E = np.exp(-2j * np.pi * np.outer(t, a) / (Q * Nk))   # E[t][a]
    return E @ F @ E.T


def slice_table(C, S, Q):
    """K4 without the normalisation: K[ov][ou][iv][iu] = C[t(iv,ov)][t(iu,ou)]."""
    i = np.arange(S)
    o = np.arange(Q)
    t = (i[None, :] + 1) * Q - S * Q // 2 - o[:, None]      # t[o][i]
    idx = t + S * Q // 2 - 1                                # row/col of C
    return C[idx[:, None, :, None], idx[None, :, None, :]]  # [ov][ou][iv][iu]


def norm_scalar(S, Q, fov):
    """K5."""
    C0 = uv_table(image_plane_samples(0.0, S, fov), S, Q)
    o_star = 0 if S % 2 == 0 else Q // 2
    return float(np.real(np.sum(slice_table(C0, S, Q)[o_star, o_star])))


def build_stack(Nw, w_max, support, oversample, grid_N, cell, plane_w=None):
    """K1-K6.  `support` is an int (uniform) or a length-Nw sequence (ragged).

    `plane_w` overrides the K1 plane centres (used by the pin that sets all
    w_p := 0 and must fail the DFT comparison)."""
    Q = int(oversample)
    fov = grid_N * cell
    if np.isscalar(support):
        Sp = np.full(Nw, int(support), dtype=np.int32)
    else:
        Sp = np.asarray(support, dtype=np.int32)
        assert Sp.shape == (Nw,)
    wp = plane_centres(Nw, w_max) if plane_w is None else np.asarray(plane_w, float)
    s = norm_scalar(int(Sp.min()), Q, fov)
    sizes = Q * Q * Sp.astype(np.int64) ** 2
    off = np.zeros(Nw + 1, dtype=np.int64)
    off[1:] = np.cumsum(sizes)
    data = np.empty(off[-1], dtype=np.complex128)
    for p in range(Nw):
        S = int(Sp[p])
        C = uv_table(image_plane_samples(wp[p], S, fov), S, Q)
        data[off[p]:off[p + 1]] = (slice_table(C, S, Q) / s).ravel()
    return KernelStack(data, Sp, off, Nw, Q, grid_N, float(cell), float(w_max))
