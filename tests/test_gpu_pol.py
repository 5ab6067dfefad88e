"""Polarised gridder (wpg_grid_pol) against the oracle: by definition it is npol independent griddings that
share positions, weights and coefficients, so every polarisation plane must equal the oracle's gridding of that
polarisation's visibilities (tolerance as for fp32 gridding), and the counters must match."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import gridder as ogrid
from oracle import wkernel as owk
from paper_1905_03213_b200 import synth, wpgrid


@pytest.fixture(scope="module")
def ctx():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    c = wpgrid.Context(0)
    yield c
    c.close()


TOL = {wpgrid.F32: 1e-4, wpgrid.F64: 1e-10}


def check_pol(ctx, uvw, freq, vis, wt, st, row_blocks=(0,), precs=(wpgrid.F32, wpgrid.F64)):
    npol = vis.shape[2]
    refs = [ogrid.grid(uvw, np.ascontiguousarray(vis[:, :, p]), wt, freq, st, threads=4) for p in range(npol)]
    d = (torch.from_numpy(vis).cuda(), torch.from_numpy(uvw).cuda(), torch.from_numpy(wt).cuda(), torch.from_numpy(freq).cuda())
    for prec in precs:
        sup = int(st.support[0]) if st.uniform else st.support
        ks = ctx.stack_from_host(st.data, st.Nw, st.w_max, sup, st.oversample, st.grid_N, st.cell, prec)
        for rb in row_blocks:
            ctx.set_option("row_block", rb)
            g, s = ctx.grid_pol(*d, ks, stats=True)
            gh = g.cpu().numpy()
            for p in range(npol):
                ref, rstats = refs[p]
                assert s == rstats
                err = float(np.max(np.abs(gh[p] - ref)) / np.max(np.abs(ref)))
                assert err <= TOL[prec], (prec, rb, p, err)
        ctx.set_option("row_block", 0)
        # accumulation into a non-zero grid, and tiny work items
        ctx.set_option("segment", 3)
        g2, _ = ctx.grid_pol(*d, ks, grid=g.clone())
        ctx.set_option("segment", 0)
        assert float((g2 - 2 * g).abs().max() / g.abs().max()) <= 10 * TOL[prec]


@pytest.mark.parametrize("S,npol", [(8, 4), (8, 2), (16, 4), (16, 2)])
def test_pol_planes_match_single_pol_oracle(ctx, S, npol):
    """Uniform supports 8 and 16: fp32 takes the pair gridders, fp64 the general cell gridder; with and without the
    rows-per-time-step hint (record compression active)."""
    rng = np.random.default_rng(S * 10 + npol)
    wl = synth.config2(nvis=150_001)
    nrow = wl.uvw.shape[0]
    nchan = 2
    freq = np.array([150e6, 151e6])
    vis = (rng.standard_normal((nrow, nchan, npol)) + 1j * rng.standard_normal((nrow, nchan, npol))).astype(np.complex64)
    wt = rng.uniform(0.0, 2.0, (nrow, nchan)).astype(np.float32)
    wt[rng.uniform(size=wt.shape) < 0.05] = 0.0
    st = owk.build_stack(wl.Nw, wl.w_max, S, wl.oversample, wl.grid_N, wl.cell)
    check_pol(ctx, wl.uvw, freq, vis, wt, st, row_blocks=(0, wl.notes["row_block"]))


@pytest.mark.parametrize("S,npol", [(4, 4), (7, 2), (9, 4), (12, 2), (12, 4), (21, 2), (32, 4)])
def test_pol_general_supports_both_precisions(ctx, S, npol):
    """The general polarised cell gridder: supports that are odd, not a power of two, or need the window split over
    several work items (S = 21, 32), fp32 and fp64, plane by plane against the oracle."""
    rng = np.random.default_rng(500 + S + npol)
    N, cell, Q, Nw, w_max, n = 128, 0.06 / 128, 4, 6, 80.0, 5000
    du = 1.0 / 0.06
    uvw = np.stack([rng.uniform(-40, 40, n) * du, rng.uniform(-40, 40, n) * du, rng.uniform(-90, 90, n)], 1)
    uvw[: n // 3, :2] = np.round(uvw[: n // 3, :2] / du) * du
    freq = np.array([synth.C0])
    vis = (rng.standard_normal((n, 1, npol)) + 1j * rng.standard_normal((n, 1, npol))).astype(np.complex64)
    wt = rng.uniform(0.5, 1.5, (n, 1)).astype(np.float32)
    st = owk.build_stack(Nw, w_max, S, Q, N, cell)
    check_pol(ctx, uvw, freq, vis, wt, st)


@pytest.mark.parametrize("npol", [2, 4])
def test_pol_ragged_stack_config4_layout(ctx, npol):
    """Ragged stack (w-dependent support, config 4's layout: SKA-low-like stations, 8 channels, N = 8192): one launch of
    the general gridder per support class, fp32 and fp64."""
    rng = np.random.default_rng(40 + npol)
    wl = synth.config4(n_dump=1, nchan=2, values="random")
    sup = owk.ragged_support(wl.Nw, wl.w_max, wl.grid_N, wl.cell, 8, 32)
    st = owk.build_stack(wl.Nw, wl.w_max, sup, wl.oversample, wl.grid_N, wl.cell)
    assert len(set(sup.tolist())) >= 4
    nrow, nchan = wl.uvw.shape[0], wl.freq.size
    vis = (rng.standard_normal((nrow, nchan, npol)) + 1j * rng.standard_normal((nrow, nchan, npol))).astype(np.complex64)
    check_pol(ctx, wl.uvw, wl.freq, vis, wl.weight, st, precs=(wpgrid.F32, wpgrid.F64) if npol == 2 else (wpgrid.F32,))


def test_pol_argument_errors(ctx):
    st = owk.build_stack(4, 50.0, 12, 8, 128, 0.001)
    ks = ctx.stack_from_host(st.data, 4, 50.0, 12, 8, 128, 0.001, wpgrid.F32)
    v = torch.zeros((10, 1, 3), dtype=torch.complex64).cuda()          # three correlations: refused
    with pytest.raises(wpgrid.WpgError):
        ctx.grid_pol(v, torch.zeros((10, 3), dtype=torch.float64).cuda(), torch.ones((10, 1)).cuda(),
                     torch.tensor([synth.C0], dtype=torch.float64).cuda(), ks)
