"""P9 — the whole oracle chain (stack O3 -> gridder O4 -> dirty image O5) against the
brute-force direct 3-D DFT O6 on tiny inputs, plus the w-term sanity check of PAPER.md:104
(an off-centre source is wrong without the w-term and right with w-projection)."""
import numpy as np
import pytest

from oracle import gridder, image, wkernel
from paper_1905_03213_b200 import synth

N, FOV, WABS = 64, 0.08, 60.0


def run_case(S, Q, Nw, snap_uv, snap_w, zero_w=False, seed=synth.SEED0):
    cell = FOV / N
    du = 1.0 / FOV
    case = synth.tiny_dft_case(seed=seed, N=N, fov=FOV, nvis=300, w_abs=WABS,
                               snap_uv_step=(du / Q) if snap_uv else None,
                               snap_w_values=wkernel.plane_centres(Nw, WABS) if snap_w else None)
    st = wkernel.build_stack(Nw, WABS, S, Q, N, cell, plane_w=np.zeros(Nw) if zero_w else None)
    uvw = case["uvw"]
    vis = case["vis"].astype(np.complex64)[:, None]
    wt = np.ones((uvw.shape[0], 1), np.float32)
    g, stats = gridder.grid(uvw, vis, wt, np.array([synth.C0]), st)
    assert stats["n_gridded"] == 300
    img = image.dirty_image(g, cell, float(wt.sum()))
    j = np.arange(N // 4, 3 * N // 4)                        # inner half of the image
    jj, ii = np.meshgrid(j, j, indexing="ij")
    l = (ii.ravel() - N // 2) * cell
    m = (jj.ravel() - N // 2) * cell
    ref = image.dft_image(uvw[:, 0], uvw[:, 1], uvw[:, 2], vis[:, 0], wt[:, 0], l, m)
    got = img[jj.ravel(), ii.ravel()]
    return np.max(np.abs(got - ref)) / np.max(np.abs(ref))


def test_p9_snapped_matches_dft():
    e8 = run_case(8, 8, 8, True, True)
    e12 = run_case(12, 8, 8, True, True)
    assert e8 <= 2e-4 and e12 <= 2e-4, (e8, e12)


def test_p9_without_w_term_fails():
    good = run_case(8, 8, 8, True, True)
    bad = run_case(8, 8, 8, True, True, zero_w=True)
    assert bad > 10 * good and bad > 2e-3, (good, bad)


def test_p9_error_scales_with_oversample_and_planes():
    eq = [run_case(8, Q, 8, False, True) for Q in (8, 16, 32)]       # only u, v free
    assert eq[0] > 1.5 * eq[1] > 1.5 * 1.5 * eq[2] and eq[0] < 3e-2, eq
    ew = [run_case(8, 8, Nw, True, False) for Nw in (8, 32, 128)]    # only w free
    assert ew[0] > 2 * ew[1] > 2 * ew[2] and ew[0] < 5e-3, ew


def test_p9_config1_image_vs_dft():
    wl = synth.config1()
    st = wkernel.build_stack(wl.Nw, wl.w_max, wl.support, wl.oversample, wl.grid_N, wl.cell)
    g, stats = gridder.grid(wl.uvw, wl.vis, wl.weight, wl.freq, st)
    assert stats["n_gridded"] == wl.nvis and stats["n_skipped_oob"] == 0
    img = image.dirty_image(g, wl.cell, float(wl.weight.sum()))
    rng = np.random.default_rng(11)
    Nn = wl.grid_N
    jl = rng.integers(Nn // 4, 3 * Nn // 4, 300); jm = rng.integers(Nn // 4, 3 * Nn // 4, 300)
    # add the pixels nearest the five sources
    jl = np.concatenate([jl, np.round(wl.sources["l"] / wl.cell).astype(int) + Nn // 2])
    jm = np.concatenate([jm, np.round(wl.sources["m"] / wl.cell).astype(int) + Nn // 2])
    l = (jl - Nn // 2) * wl.cell; m = (jm - Nn // 2) * wl.cell
    ref = image.dft_image(wl.uvw[:, 0], wl.uvw[:, 1], wl.uvw[:, 2], wl.vis[:, 0], wl.weight[:, 0], l, m)
    err = np.max(np.abs(img[jm, jl] - ref)) / np.max(np.abs(ref))
    assert err <= 1e-2, err
    # the brightest source shows up at its nearest pixel with roughly its flux (the source
    # sits between pixels and the other four contribute sidelobes, hence the loose bound)
    k = int(np.argmax(wl.sources["flux"]))
    assert abs(ref[300 + k] - wl.sources["flux"][k]) < 0.2


def test_o5_point_grid_gives_flat_over_taper():
    """A single unit cell at the grid centre transforms to a constant image / taper."""
    Nn, cell = 32, 0.004
    g = np.zeros((Nn, Nn), complex); g[Nn // 2, Nn // 2] = 2.0
    img = image.dirty_image(g, cell, 2.0)
    from oracle.taper import psi
    t = psi(2.0 * (np.arange(Nn) - Nn // 2) / Nn)
    ok = np.outer(t, t) >= image.TAPER_FLOOR
    assert np.allclose(img[ok] * np.outer(t, t)[ok], 1.0, atol=1e-13)
    assert np.all(img[~ok] == 0.0) and img[0, 5] == 0.0
    # shift theorem: a cell one step off centre in u gives cos(2 pi l du) in l, constant in m
    g = np.zeros((Nn, Nn), complex); g[Nn // 2, Nn // 2 + 1] = 1.0
    img = image.dirty_image(g, cell, 1.0) * np.outer(t, t)
    l = (np.arange(Nn) - Nn // 2) * cell
    assert np.allclose(img[Nn // 2, 1:], np.cos(2 * np.pi * l / (Nn * cell))[1:], atol=1e-12)
