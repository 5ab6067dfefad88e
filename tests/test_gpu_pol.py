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


@pytest.mark.parametrize("S,npol", [(8, 4), (8, 2), (16, 4), (16, 2)])
def test_pol_planes_match_single_pol_oracle(ctx, S, npol):
    rng = np.random.default_rng(S * 10 + npol)
    wl = synth.config2(nvis=150_001)
    nrow = wl.uvw.shape[0]
    nchan = 2
    freq = np.array([150e6, 151e6])
    vis = (rng.standard_normal((nrow, nchan, npol)) + 1j * rng.standard_normal((nrow, nchan, npol))).astype(np.complex64)
    wt = rng.uniform(0.0, 2.0, (nrow, nchan)).astype(np.float32)
    wt[rng.uniform(size=wt.shape) < 0.05] = 0.0
    st = owk.build_stack(wl.Nw, wl.w_max, S, wl.oversample, wl.grid_N, wl.cell)
    ks = ctx.stack_from_host(st.data, st.Nw, st.w_max, S, st.oversample, st.grid_N, st.cell, wpgrid.F32)
    d = (torch.from_numpy(vis).cuda(), torch.from_numpy(wl.uvw).cuda(), torch.from_numpy(wt).cuda(), torch.from_numpy(freq).cuda())
    for rb in (0, wl.notes["row_block"]):
        ctx.set_option("row_block", rb)
        g, s = ctx.grid_pol(*d, ks, stats=True)
        gh = g.cpu().numpy()
        for p in range(npol):
            ref, rstats = ogrid.grid(wl.uvw, np.ascontiguousarray(vis[:, :, p]), wt, freq, st, threads=4)
            assert s == rstats
            err = float(np.max(np.abs(gh[p] - ref)) / np.max(np.abs(ref)))
            assert err <= 1e-4, (p, err)
    ctx.set_option("row_block", 0)
    # accumulation into a non-zero grid, and tiny work items
    ctx.set_option("segment", 3)
    g2, _ = ctx.grid_pol(*d, ks, grid=g.clone())
    ctx.set_option("segment", 0)
    assert float((g2 - 2 * g).abs().max() / g.abs().max()) <= 1e-4


def test_pol_argument_errors(ctx):
    st = owk.build_stack(4, 50.0, 12, 8, 128, 0.001)
    ks = ctx.stack_from_host(st.data, 4, 50.0, 12, 8, 128, 0.001, wpgrid.F32)
    v = torch.zeros((10, 1, 4), dtype=torch.complex64).cuda()
    with pytest.raises(wpgrid.WpgError):
        ctx.grid_pol(v, torch.zeros((10, 3), dtype=torch.float64).cuda(), torch.ones((10, 1)).cuda(),
                     torch.tensor([synth.C0], dtype=torch.float64).cuda(), ks)
