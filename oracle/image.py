"""O5 dirty image and O6 brute-force 3-D DFT (oracle, test infrastructure only).

O5 ("the master node performs an IFFT on the ... gridding
result to obtain the final image"; the grid correction is reading R11, the
paper never mentions it):
    img = fftshift(ifft2(ifftshift(g))) * N^2
    I[jm][jl] = Re(img[jm][jl]) / sum(wt) / (psi(2 l_j/FoV) psi(2 m_j/FoV)),
    l_j = (j - N/2) cell;  pixels whose taper product is < TAPER_FLOOR are 0.

O6 (the measurement model O1 inverted term by term; "the effect
of the w-term cannot be neglected"):
    I_D(l, m) = (1/sum wt) Re sum_k wt_k V_k exp(+2 pi i [u_k l + v_k m + w_k (n - 1)]),
    n - 1 = -r^2/(1 + sqrt(1 - r^2)).
"""
import numpy as np

from .taper import psi

TAPER_FLOOR = 1e-3


def dirty_image(grid, cell, weight_sum):
    """O5.  grid [N][N] complex (v slow axis) -> image [N][N] float64 (m slow axis)."""
    g = np.asarray(grid, dtype=np.complex128)
    N = g.shape[0]
    fov = N * cell
    img = np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(g))) * (N * N)
    l = (np.arange(N) - N // 2) * cell
    t1 = psi(2.0 * l / fov)
    tap = np.outer(t1, t1)
    out = np.zeros((N, N), dtype=np.float64)
    ok = tap >= TAPER_FLOOR
    out[ok] = img.real[ok] / weight_sum / tap[ok]
    return out


def dft_image(u, v, w, vis, weight, l, m):
    """O6.  u, v, w in wavelengths [nvis]; l, m direction cosines [npix] -> I_D [npix]."""
    u = np.asarray(u, np.float64); v = np.asarray(v, np.float64); w = np.asarray(w, np.float64)
    vis = np.asarray(vis, np.complex128); weight = np.asarray(weight, np.float64)
    l = np.asarray(l, np.float64); m = np.asarray(m, np.float64)
    out = np.empty(l.shape, dtype=np.float64)
    wsum = weight.sum()
    wv = weight * vis
    for i in range(l.size):
        r2 = l.flat[i] ** 2 + m.flat[i] ** 2
        nm1 = -r2 / (1.0 + np.sqrt(1.0 - r2))
        ph = u * l.flat[i] + v * m.flat[i] + w * nm1
        out.flat[i] = np.real(np.sum(wv * np.exp(2j * np.pi * ph))) / wsum
    return out
