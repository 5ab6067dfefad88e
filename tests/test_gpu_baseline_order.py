"""GPU parity of the paper's own data order (Eqs. 1-2) through the C ABI: the re-order is
integer work and must match the oracle bit for bit; the grid must match the oracle's grid within the gridding
tolerances (the sum does not depend on the order)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import baseline_order as obo
from oracle import gridder as ogrid
from oracle import wkernel as owk
from paper_1905_03213_b200 import synth, wpgrid

TOL = {wpgrid.F32: 1e-4, wpgrid.F64: 1e-10}


@pytest.fixture(scope="module")
def ctx():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    c = wpgrid.Context(0)
    yield c
    c.close()


def check_reorder(ctx, a1, a2, n_ant):
    bstart, perm = ctx.baseline_reorder(torch.from_numpy(a1).cuda(), torch.from_numpy(a2).cuda(), n_ant)
    C, B = obo.start_index(a1, a2, n_ant)
    assert np.array_equal(bstart.cpu().numpy().astype(np.int64), B)                      # Eq. (2), exact
    assert np.array_equal(perm.cpu().numpy().astype(np.int64), obo.reorder(a1, a2, n_ant))   # stable order, exact


def test_reorder_matches_oracle_bit_for_bit(ctx):
    rng = np.random.default_rng(3)
    # random pairs incl. autocorrelations and swapped order, ragged counts, a baseline with thousands of rows
    n_ant, nrow = 13, 40_000
    a1 = rng.integers(0, n_ant, nrow).astype(np.int32); a2 = rng.integers(0, n_ant, nrow).astype(np.int32)
    a1[:6000] = 2; a2[:6000] = 9
    check_reorder(ctx, a1, a2, n_ant)
    # time-major tracks with rows deleted at random (RFI flags)
    a1, a2 = synth.track_antennas(40, 780 * 50)
    keep = rng.uniform(size=a1.size) > 0.1
    check_reorder(ctx, a1[keep], a2[keep], 40)
    # one antenna, one row; empty input
    check_reorder(ctx, np.zeros(1, np.int32), np.zeros(1, np.int32), 1)
    check_reorder(ctx, np.zeros(0, np.int32), np.zeros(0, np.int32), 5)


def test_bad_antenna_ids_and_oversized_baselines_are_errors(ctx):
    a1 = torch.tensor([0, 1, 7], dtype=torch.int32).cuda(); a2 = torch.tensor([1, 2, 3], dtype=torch.int32).cuda()
    with pytest.raises(wpgrid.WpgError) as e:
        ctx.baseline_reorder(a1, a2, 4)
    assert e.value.code == wpgrid.EINVAL
    a = torch.zeros(9000, dtype=torch.int32).cuda()
    with pytest.raises(wpgrid.WpgError) as e:
        ctx.baseline_reorder(a, a + 1, 3)
    assert e.value.code == wpgrid.EINVAL


def test_grid_in_baseline_order_matches_oracle(ctx):
    """Config-2-like tracks (400k rows) in both precisions, and a two-channel case with flagged rows and
    visibilities off the grid (they stay in the time series as zero-valued records)."""
    wl = synth.config2(nvis=400_000)
    a1, a2 = synth.track_antennas(wl.notes["n_ant"], wl.uvw.shape[0])
    st = owk.build_stack(wl.Nw, wl.w_max, wl.support, wl.oversample, wl.grid_N, wl.cell)
    ref, rstats = ogrid.grid(wl.uvw, wl.vis, wl.weight, wl.freq, st, threads=4)
    d = [torch.from_numpy(x).cuda() for x in (wl.vis, wl.uvw, wl.weight, wl.freq, a1, a2)]
    for prec in (wpgrid.F32, wpgrid.F64):
        ks = ctx.stack_from_host(st.data, st.Nw, st.w_max, wl.support, st.oversample, st.grid_N, st.cell, prec)
        g, s = ctx.grid_baseline_order(*d, wl.notes["n_ant"], ks, stats=True)
        assert s == rstats
        err = float(np.max(np.abs(g.cpu().numpy() - ref)) / np.max(np.abs(ref)))
        assert err <= TOL[prec], (prec, err)
    rng = np.random.default_rng(11)
    N, cell, Q, S, Nw, w_max = 256, 0.1 / 256, 8, 8, 8, 100.0
    n_ant, n_dump, nchan = 12, 300, 2
    a1, a2 = synth.track_antennas(n_ant, 66 * n_dump)
    nrow = a1.size
    b = np.arange(nrow) % 66; t = np.arange(nrow) // 66
    uvw = np.stack([(b - 33) * 18.0 + 0.6 * t, (b % 7 - 3) * 150.0 + 0.3 * t, rng.uniform(-120, 120, 66)[b]], 1)
    freq = np.array([1.0, 1.03]) * synth.C0 / 0.5
    vis = (rng.standard_normal((nrow, nchan)) + 1j * rng.standard_normal((nrow, nchan))).astype(np.complex64)
    wt = rng.uniform(0.0, 2.0, (nrow, nchan)).astype(np.float32)
    wt[rng.uniform(size=wt.shape) < 0.07] = 0.0
    st = owk.build_stack(Nw, w_max, S, Q, N, cell)
    ref, rstats = ogrid.grid(uvw, vis, wt, freq, st)
    assert rstats["n_skipped_zero_weight"] > 0 and rstats["n_skipped_oob"] > 0 and rstats["n_clamped_w"] > 0
    d = [torch.from_numpy(x).cuda() for x in (vis, uvw, wt, freq, a1, a2)]
    for prec in (wpgrid.F32, wpgrid.F64):
        ks = ctx.stack_from_host(st.data, Nw, w_max, S, Q, N, cell, prec)
        g, s = ctx.grid_baseline_order(*d, n_ant, ks, stats=True)
        assert s == rstats
        err = float(np.max(np.abs(g.cpu().numpy() - ref)) / np.max(np.abs(ref)))
        assert err <= TOL[prec], (prec, err)
    # NaN / Inf values under zero weight (RFI-flagged samples) and in samples off the grid: skipped
    # outright by the oracle and by wpg_grid, and they must not leak through the zero-valued place-holder records
    vis_bad = vis.copy()
    flagged = wt == 0.0
    vis_bad[flagged] = np.complex64(complex(np.nan, np.inf))
    fscale = freq / synth.C0
    off_grid = np.zeros_like(flagged)
    for c in range(nchan):
        for k in range(nrow):
            j0u, _ = ogrid.index_map(uvw[k, 0] * fscale[c], N, cell, S, Q)
            j0v, _ = ogrid.index_map(uvw[k, 1] * fscale[c], N, cell, S, Q)
            off_grid[k, c] = j0u < 0 or j0v < 0 or j0u + S > N or j0v + S > N
    assert off_grid.sum() == rstats["n_skipped_oob"] + (off_grid & flagged).sum()
    vis_bad[off_grid] = np.complex64(complex(-np.inf, np.nan))
    ref_bad, rstats_bad = ogrid.grid(uvw, vis_bad, wt, freq, st)
    assert rstats_bad == rstats and np.array_equal(ref_bad, ref)
    d_bad = [torch.from_numpy(vis_bad).cuda()] + d[1:]
    for prec in (wpgrid.F32, wpgrid.F64):
        ks = ctx.stack_from_host(st.data, Nw, w_max, S, Q, N, cell, prec)
        g, s = ctx.grid_baseline_order(*d_bad, n_ant, ks, stats=True)
        g2, s2 = ctx.grid(*d_bad[:4], ks, stats=True)
        assert s == rstats and s2 == rstats
        for gg in (g, g2):
            gh = gg.cpu().numpy()
            assert np.isfinite(gh).all()
            assert float(np.max(np.abs(gh - ref)) / np.max(np.abs(ref))) <= TOL[prec]
    # ragged stack on the same tracks: the order is partitioned by support class (stably), one gridder launch per class
    sup = np.array([8, 8, 10, 10, 12, 12, 8, 9], np.int32)
    st_r = owk.build_stack(Nw, w_max, sup, Q, N, cell)
    ref_r, rstats_r = ogrid.grid(uvw, vis, wt, freq, st_r)
    for prec in (wpgrid.F32, wpgrid.F64):
        ks = ctx.stack_from_host(st_r.data, Nw, w_max, sup, Q, N, cell, prec)
        g, s = ctx.grid_baseline_order(*d, n_ant, ks, stats=True)
        assert s == rstats_r
        err = float(np.max(np.abs(g.cpu().numpy() - ref_r)) / np.max(np.abs(ref_r)))
        assert err <= TOL[prec], (prec, err)


def test_baseline_order_ragged_config4_layout(ctx):
    """The paper's order on config 4's layout (512 SKA-low-like stations, 8 channels, N = 8192, w-dependent support —
    PAPER.md:192 (6) names SKA-size images as the case to keep in mind): 2 dumps, every support class of the input."""
    wl = synth.config4(n_dump=2, values="random")
    sup = owk.ragged_support(wl.Nw, wl.w_max, wl.grid_N, wl.cell, 8, 32)
    st = owk.build_stack(wl.Nw, wl.w_max, sup, wl.oversample, wl.grid_N, wl.cell)
    assert len(set(sup.tolist())) >= 4
    ref, rstats = ogrid.grid(wl.uvw, wl.vis, wl.weight, wl.freq, st, threads=4)
    a1, a2 = synth.track_antennas(wl.notes["n_ant"], wl.uvw.shape[0])
    d = [torch.from_numpy(x).cuda() for x in (wl.vis, wl.uvw, wl.weight, wl.freq, a1, a2)]
    ks = ctx.stack_from_host(st.data, st.Nw, st.w_max, sup, st.oversample, st.grid_N, st.cell, wpgrid.F32)
    g, s = ctx.grid_baseline_order(*d, wl.notes["n_ant"], ks, stats=True)
    assert s == rstats
    err = float(np.max(np.abs(g.cpu().numpy() - ref)) / np.max(np.abs(ref)))
    assert err <= TOL[wpgrid.F32], err
