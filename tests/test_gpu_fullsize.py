"""Full-size GPU runs of BASELINE configs 3, 4 and 5 in the launch configuration bench.py times (-m gpu).

A full oracle pass over these workloads (2.6e10 - 2.8e10 updates) takes minutes on the box's host cores, so the
full runs are checked with what SURVEY.md §8(c) prescribes for them: the counters bit for bit, and P11 — flux
conservation — whose right-hand side is O(nvis): oracle.gridder.flux (oracle_flux in grid_oracle.c, pinned in
tests/test_oracle_gridder.py) gives sum(grid) and, beyond P11, the two first moments sum(grid * ju), sum(grid * jv),
which also pin where the flux went.  fp64 makes the check sharp (a single dropped, duplicated or misplaced
visibility is orders of magnitude outside the bound); fp32 is bounded by its accumulation error.  On top of that,
sampled outputs the oracle computes one by one: oracle.gridder.cells (oracle_cells in grid_oracle.c, G5 read as a
gather over ALL visibilities, pinned in tests/test_oracle_gridder.py) gives the exact value of a seeded sample of
grid cells — cells inside the windows of randomly drawn visibilities, so that they follow the density of the
coverage, plus uniformly drawn ones — which the GPU grid must match to north_star's 1e-4 / 1e-10 of the largest
sampled magnitude (at most the grid's largest, so the bound is the stricter one).  Element-wise parity on seeded
prefixes through the full-size grid is in test_gpu_parity.py.
"""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import gridder as ogrid
from oracle import wkernel as owk
from paper_1905_03213_b200 import synth, wpgrid

# |sum_gpu - sum_oracle| <= FLUX_TOL * L1,  L1 = sum |wt V| |sigma| (first moments: * N).  fp64: rounding of ~1e9
# reductions in arbitrary order, far below one visibility (|V sigma| / L1 ~ 3e-9 on config 4, larger elsewhere).  fp32: the
# accumulated rounding of the c64 grid, measured 1e-12 .. 3e-9 of L1; fp64 measured 1e-17 (profiles/r02_fullsize_parity.md).
FLUX_TOL = {wpgrid.F32: 2e-8, wpgrid.F64: 1e-14}
CELL_TOL = {wpgrid.F32: 1e-4, wpgrid.F64: 1e-10}        # north_star, relative to the largest |reference| (here: of the sample)
N_CELL_VIS, N_CELL_UNIFORM = 160, 32
THREADS = min(os.cpu_count() or 1, 32)


@pytest.fixture(scope="module")
def ctx():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    c = wpgrid.Context(0)
    yield c
    c.close()


def oracle_stack(wl):
    sup = wl.support
    if not np.isscalar(sup):
        sup = owk.ragged_support(wl.Nw, wl.w_max, wl.grid_N, wl.cell, sup[1], sup[2])
    return owk.build_stack(wl.Nw, wl.w_max, sup, wl.oversample, wl.grid_N, wl.cell)


def sample_cells(wl, st, seed):
    """Seeded sample of grid cells: one cell inside the window of each of N_CELL_VIS randomly drawn visibilities (so
    the sample follows the coverage: most lie where the grid is dense), plus N_CELL_UNIFORM uniformly drawn cells."""
    rng = np.random.default_rng(seed)
    N, nchan = wl.grid_N, wl.freq.size
    cu, cv = [], []
    while len(cu) < N_CELL_VIS:
        r, c = int(rng.integers(0, wl.uvw.shape[0])), int(rng.integers(0, nchan))
        f = wl.freq[c] / synth.C0
        p, _ = ogrid.plane_of(wl.uvw[r, 2] * f, wl.w_max, wl.Nw)
        S = int(st.support[p])
        j0u, _ = ogrid.index_map(wl.uvw[r, 0] * f, N, wl.cell, S, wl.oversample)
        j0v, _ = ogrid.index_map(wl.uvw[r, 1] * f, N, wl.cell, S, wl.oversample)
        u, v = j0u + int(rng.integers(0, S)), j0v + int(rng.integers(0, S))
        if 0 <= u < N and 0 <= v < N:
            cu.append(u); cv.append(v)
    cu += [int(x) for x in rng.integers(0, N, N_CELL_UNIFORM)]
    cv += [int(x) for x in rng.integers(0, N, N_CELL_UNIFORM)]
    return np.array(cu, dtype=np.int32), np.array(cv, dtype=np.int32)


def grid_sums(g):
    """(sum, u-moment, v-moment) of a device grid, accumulated in fp64 on the device (test arithmetic, torch)."""
    N = g.shape[0]
    j = torch.arange(N, dtype=torch.float64, device=g.device)
    cols = torch.zeros(N, dtype=torch.complex128, device=g.device)
    rows = torch.zeros(N, dtype=torch.complex128, device=g.device)
    for r0 in range(0, N, 1024):                       # in slabs: a c128 copy of an 8192^2 grid is 1 GB
        blk = g[r0:r0 + 1024].to(torch.complex128)
        cols += blk.sum(dim=0)
        rows[r0:r0 + 1024] = blk.sum(dim=1)
    jc = j.to(torch.complex128)
    return complex(cols.sum().item()), complex((cols * jc).sum().item()), complex((rows * jc).sum().item())


def check_full(ctx, wl, precs, label):
    st = oracle_stack(wl)
    fl, rstats = ogrid.flux(wl.uvw, wl.vis, wl.weight, wl.freq, st, threads=THREADS)
    assert rstats["n_gridded"] + rstats["n_skipped_oob"] + rstats["n_skipped_zero_weight"] == wl.nvis
    cu, cv = sample_cells(wl, st, 2024)
    cref, cl1 = ogrid.cells(wl.uvw, wl.vis, wl.weight, wl.freq, st, cu, cv, threads=THREADS)
    cmax = float(np.max(np.abs(cref)))
    assert np.count_nonzero(cref) >= N_CELL_VIS                            # the sample is not a set of empty cells
    t_cu, t_cv = torch.from_numpy(cu.astype(np.int64)).cuda(), torch.from_numpy(cv.astype(np.int64)).cuda()
    d = (torch.from_numpy(wl.vis).cuda(), torch.from_numpy(wl.uvw).cuda(),
         torch.from_numpy(wl.weight).cuda(), torch.from_numpy(wl.freq).cuda())
    nrow, nchan, N = wl.uvw.shape[0], wl.freq.size, wl.grid_N
    ctx.set_option("row_block", int(wl.notes.get("row_block", 0)))      # as bench.py does
    out = {}
    try:
        for prec in precs:
            sup = int(st.support[0]) if st.uniform else st.support
            ks = ctx.stack_from_host(st.data, st.Nw, st.w_max, sup, st.oversample, N, st.cell, prec)
            ws = torch.empty(ctx.grid_workspace_bytes(nrow, nchan, ks), dtype=torch.uint8, device="cuda")
            grid = ctx.new_grid(ks)
            for rep in range(2):                                           # twice: workspace reuse, as in the timed loop
                grid.zero_()
                g, s = ctx.grid(*d, ks, grid=grid, workspace=ws, stats=True)
                assert s == rstats, (label, prec, s, rstats)
                tot, mu, mv = grid_sums(g)
                e0 = abs(tot - fl["sum"]) / fl["l1"]
                eu = abs(mu - fl["mom_u"]) / (fl["l1"] * N)
                ev = abs(mv - fl["mom_v"]) / (fl["l1"] * N)
                print("%s prec %s rep %d: flux err %.2e  u-moment %.2e  v-moment %.2e  (of L1 = %.3e; %d updates)"
                      % (label, "f32" if prec == wpgrid.F32 else "f64", rep, e0, eu, ev, fl["l1"], s["n_updates"]))
                assert max(e0, eu, ev) <= FLUX_TOL[prec], (label, prec, e0, eu, ev)
                assert bool(torch.isfinite(torch.view_as_real(g)).all())
                got = g[t_cv, t_cu].cpu().numpy().astype(np.complex128)
                ec = float(np.max(np.abs(got - cref))) / cmax
                el = float(np.max(np.abs(got - cref)[cl1 > 0] / cl1[cl1 > 0]))
                print("%s prec %s rep %d: %d sampled cells, max err %.2e of the largest sampled |value| %.3e (%.2e of a cell's own L1)"
                      % (label, "f32" if prec == wpgrid.F32 else "f64", rep, cu.size, ec, cmax, el))
                assert ec <= CELL_TOL[prec], (label, prec, ec)
                assert np.all(got[cl1 == 0] == 0)                          # a cell no window covers stays exactly zero
            out[prec] = (e0, eu, ev)
            del g, grid, ws, ks
    finally:
        ctx.set_option("row_block", 0)
    return out, rstats


def test_config4_full_size_flux_and_counters(ctx):
    """BASELINE config 4 at its full 376 750 080 visibilities (130 816 baselines x 360 dumps x 8 channels, N = 8192,
    128 planes, ragged support 8 .. 32), exactly the workload bench.py times by default: counters bit-exact, P11 and
    first moments in fp32 and fp64."""
    from bench import make_workload
    wl = make_workload("config4", 0, "cuda")
    assert wl.nvis == 376_750_080 and wl.grid_N == 8192
    sup = owk.ragged_support(wl.Nw, wl.w_max, wl.grid_N, wl.cell, 8, 32)
    assert int(sup.min()) == 8 and int(sup.max()) == 32
    _, rstats = check_full(ctx, wl, (wpgrid.F32, wpgrid.F64), "config4 full")
    assert rstats["n_updates"] > 2.5e10


def test_config5_full_size_flux_and_counters(ctx):
    """BASELINE config 5 at its full 1e8 visibilities (N = 4096, S = 16), identical inputs in fp32 and fp64."""
    wl = synth.config5(device="cuda")
    assert wl.nvis == 100_000_000
    _, rstats = check_full(ctx, wl, (wpgrid.F32, wpgrid.F64), "config5 full")
    assert rstats["n_updates"] == rstats["n_gridded"] * 256


@pytest.mark.parametrize("N,S", [(8192, 16), (8192, 4), (4096, 12)])
def test_config3_full_size_flux_and_counters(ctx, N, S):
    """Config-3 sweep points at the full 5e7 visibilities in the regime the paper flags (grid > 2048; support > 8,
    PAPER.md:168-178) and at the HBM-bound S = 4, fp32 and fp64."""
    wl = synth.config3(N=N, S=S)
    assert wl.nvis == 50_000_000
    check_full(ctx, wl, (wpgrid.F32, wpgrid.F64), "config3 N=%d S=%d" % (N, S))


@pytest.mark.parametrize("S", [4, 8, 16])
def test_config3_large_grid_elementwise(ctx, S):
    """N = 8192 with the other supports of the sweep (S = 12 is in test_gpu_parity.py), 3e6 visibilities through the
    full-size grid, element by element against the oracle, fp32 and fp64."""
    wl = synth.config3(N=8192, S=S, nvis=3_000_000)
    st = oracle_stack(wl)
    ref, rstats = ogrid.grid(wl.uvw, wl.vis, wl.weight, wl.freq, st, threads=8)
    d = (torch.from_numpy(wl.vis).cuda(), torch.from_numpy(wl.uvw).cuda(),
         torch.from_numpy(wl.weight).cuda(), torch.from_numpy(wl.freq).cuda())
    for prec, tol in ((wpgrid.F32, 1e-4), (wpgrid.F64, 1e-10)):
        ks = ctx.stack_from_host(st.data, st.Nw, st.w_max, S, st.oversample, st.grid_N, st.cell, prec)
        g, s = ctx.grid(*d, ks, stats=True)
        assert s == rstats
        e = float(np.max(np.abs(g.cpu().numpy().astype(np.complex128) - ref)) / np.max(np.abs(ref)))
        print("config3 N=8192 S=%d prec %d relerr %.3e" % (S, prec, e))
        assert e <= tol
        del g
