"""Pins of the oracle degridder (oracle_degrid): adjointness with the pinned gridder, single-cell grids, and
the physics — degridding the transform of a model image predicts the measurement model O1."""
import numpy as np

from oracle import gridder, wkernel
from oracle.taper import psi
from paper_1905_03213_b200 import synth

N, FOV, WABS = 64, 0.08, 60.0


def test_adjoint_of_gridding():
    """<grid(v), g> = <v, degrid(g)> for every v, g: ties plane, window, sub-cell and conjugation conventions of
    the degridder to the gridder's (which P6-P12 pin)."""
    rng = np.random.default_rng(2)
    for S, Q in ((7, 8), (8, 4)):
        cell = FOV / N
        st = wkernel.build_stack(6, WABS, S, Q, N, cell)
        n = 500
        du = 1.0 / FOV
        uvw = np.stack([rng.uniform(-34, 34, n) * du, rng.uniform(-34, 34, n) * du, rng.uniform(-80, 80, n)], 1)
        freq = np.array([0.9, 1.1]) * synth.C0
        v = (rng.standard_normal((n, 2)) + 1j * rng.standard_normal((n, 2))).astype(np.complex64)
        g = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
        Av, stats = gridder.grid(uvw, v, np.ones((n, 2), np.float32), freq, st)
        AHg, cnt = gridder.degrid(uvw, freq, st, g)
        assert cnt["n_predicted"] == stats["n_gridded"] and cnt["n_outside"] == stats["n_skipped_oob"] > 0
        lhs = np.vdot(g, Av)                   # sum conj(g) * Av
        rhs = np.vdot(AHg, v.astype(np.complex128))
        assert abs(lhs - rhs) <= 1e-12 * abs(lhs)


def test_single_cell_grid_returns_conjugate_coefficient():
    cell = FOV / N
    S, Q = 8, 8
    st = wkernel.build_stack(4, WABS, S, Q, N, cell)
    du = 1.0 / FOV
    uvw = np.array([[3.25 * du, -5.5 * du, 20.0], [25.0 * du, 0.0, -50.0]])
    freq = np.array([synth.C0])
    j0u, ou = gridder.index_map(uvw[0, 0], N, cell, S, Q); j0v, ov = gridder.index_map(uvw[0, 1], N, cell, S, Q)
    p, _ = gridder.plane_of(20.0, WABS, 4)
    Kp = st.data[st.plane_offset[p]:st.plane_offset[p + 1]].reshape(Q, Q, S, S)
    for iv, iu in ((0, 0), (3, 5), (7, 7)):
        g = np.zeros((N, N), complex); g[j0v + iv, j0u + iu] = 2.0 - 1.0j
        out, _ = gridder.degrid(uvw, freq, st, g)
        assert out[0, 0] == (2.0 - 1.0j) * np.conj(Kp[ov, ou, iv, iu])
        assert out[1, 0] == 0.0                                   # the other window does not contain the cell


def test_predicts_the_measurement_model():
    """Model image of point sources on pixel centres -> grid = centred FFT of (image / taper) -> degrid: the
    visibilities of O1, V = sum S exp(-2 pi i (u l + v m + w (n - 1))), to ~1e-4 with u, v on oversample
    points and w on plane centres (the same error budget as P9), and clearly worse without the w-term."""
    cell = FOV / N
    du = 1.0 / FOV
    S, Q, Nw = 12, 8, 8
    case = synth.tiny_dft_case(N=N, fov=FOV, nvis=300, w_abs=WABS, snap_uv_step=du / Q,
                               snap_w_values=wkernel.plane_centres(Nw, WABS))
    uvw = case["uvw"]
    pix = [(40, 29, 1.0), (25, 37, 0.6), (33, 33, 0.3)]          # (jl, jm, flux) within the inner half
    img = np.zeros((N, N))
    t1 = psi(2.0 * (np.arange(N) - N // 2) / N)
    for jl, jm, fl in pix:
        img[jm, jl] = fl / (t1[jl] * t1[jm])
    g = np.fft.fftshift(np.fft.fft2(np.fft.ifftshift(img)))
    l = np.array([(jl - N // 2) * cell for jl, _, _ in pix]); m = np.array([(jm - N // 2) * cell for _, jm, _ in pix])
    ref = synth.predict_vis(uvw[:, 0], uvw[:, 1], uvw[:, 2], [p[2] for p in pix], l, m)
    errs = {}
    for name, plane_w in (("w", None), ("now", np.zeros(Nw))):
        st = wkernel.build_stack(Nw, WABS, S, Q, N, cell, plane_w=plane_w)
        out, cnt = gridder.degrid(uvw, np.array([synth.C0]), st, g)
        assert cnt["n_outside"] == 0
        errs[name] = np.max(np.abs(out[:, 0] - ref)) / np.max(np.abs(ref))
    assert errs["w"] <= 3e-4, errs
    assert errs["now"] > 10 * errs["w"], errs
