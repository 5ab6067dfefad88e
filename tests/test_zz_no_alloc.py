"""wpg_grid_static — the entry point that allocates nothing (scratch in the library's static device array,
csrc/wpg_static.cu) — against the existing path wpg_grid with a caller-owned workspace, through the C ABI (-m gpu).

Collected last on purpose (the suite runs with pytest -x).  Every case makes two calls in a row on different inputs:
the static array keeps the previous call's contents, so a call that failed to clear what must start at zero, or that
read the array's host-side stand-in instead of its device address, cannot pass the second one.  Tolerances as in
test_gpu_parity.py (north_star: 1e-4 / 1e-10 of the largest magnitude; the two paths differ only in the order of the
grid's reductions), counters bit for bit.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from paper_1905_03213_b200 import synth, wpgrid

TOL = {wpgrid.F32: 1e-4, wpgrid.F64: 1e-10}


@pytest.fixture(scope="module")
def ctx():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    c = wpgrid.Context(0)
    yield c
    c.close()


def inputs(seed, n, nchan, extent, w_extent):
    rng = np.random.default_rng(seed)
    uvw = np.stack([rng.uniform(-extent, extent, n), rng.uniform(-extent, extent, n), rng.uniform(-w_extent, w_extent, n)], 1)
    vis = (rng.standard_normal((n, nchan)) + 1j * rng.standard_normal((n, nchan))).astype(np.complex64)
    wt = rng.uniform(0.1, 2.0, (n, nchan)).astype(np.float32)
    wt[rng.uniform(size=wt.shape) < 0.05] = 0.0                      # flagged samples
    freq = (np.linspace(0.95, 1.05, nchan) * synth.C0).astype(np.float64)
    return tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (vis, uvw, wt, freq))


def compare(ctx, ks, prec, d):
    ref, rstats = ctx.grid(*d, ks, stats=True)                        # existing path: torch-allocated workspace
    got = torch.zeros_like(ref)
    got, stats = ctx.grid_static(*d, ks, got, stats=True)
    assert stats == rstats
    assert rstats["n_gridded"] > 0 and rstats["n_skipped_zero_weight"] > 0
    scale = float(ref.abs().max())
    err = float((got - ref).abs().max()) / scale
    assert err <= TOL[prec], (prec, err)
    assert bool(((got == 0) == (ref == 0)).all())
    return err


@pytest.mark.parametrize("prec", [wpgrid.F32, wpgrid.F64])
def test_static_scratch_matches_workspace_path_two_calls_in_a_row(ctx, prec):
    N, cell, Q, Nw, w_max, S = 512, 0.2 / 512, 8, 16, 300.0, 8
    ks = ctx.wkernel_build(Nw, w_max, S, Q, N, cell, prec)
    ext = 0.45 * N / (N * cell) / 1.05                                  # a few windows fall off the grid's edge
    first = inputs(101, 300_000, 2, ext * 1.12, 350.0)
    second = inputs(202, 41_003, 2, ext * 0.5, 100.0)                   # fewer, elsewhere: stale records and counts would show
    e1 = compare(ctx, ks, prec, first)
    e2 = compare(ctx, ks, prec, second)
    e3 = compare(ctx, ks, prec, first)
    print("static scratch vs workspace, prec %d: relerr %.2e %.2e %.2e" % (prec, e1, e2, e3))


def test_static_scratch_ragged_stack_and_accumulation(ctx):
    """Ragged stack (config 4's support rule, one gridder launch per class) and accumulation into a non-zero grid."""
    wl = synth.config4(n_dump=2, nchan=2, values="random")
    sup, _ = wpgrid.ragged_support(wl.Nw, wl.w_max, wl.grid_N, wl.cell, wl.oversample, 8, 32)
    ks = ctx.wkernel_build(wl.Nw, wl.w_max, sup, wl.oversample, wl.grid_N, wl.cell, wpgrid.F32)
    nrow, nchan = wl.uvw.shape[0], wl.freq.size
    d = tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (wl.vis, wl.uvw, wl.weight, wl.freq))
    assert ctx.grid_workspace_bytes(nrow, nchan, ks) > ctx.static_scratch_bytes()       # default key budget: 2^24 entries
    ctx.set_option("key_bits", 22)                                     # a 16 MiB bucket table (wpgrid.h: the limit)
    try:
        assert ctx.grid_workspace_bytes(nrow, nchan, ks) <= ctx.static_scratch_bytes()
        ref, rstats = ctx.grid(*d, ks, stats=True)
        ref, _ = ctx.grid(*d, ks, grid=ref)                            # gridded twice into the same grid
        got = ctx.new_grid(ks)
        for _ in range(2):
            got, stats = ctx.grid_static(*d, ks, got, stats=True)
            assert stats == rstats
    finally:
        ctx.set_option("key_bits", 0)
    assert rstats["n_updates"] > 64 * rstats["n_gridded"]             # several support classes took part
    err = float((got - ref).abs().max()) / float(ref.abs().max())
    assert err <= TOL[wpgrid.F32], err


def test_static_scratch_allocates_nothing_and_rejects_oversize(ctx):
    N, cell, Q, Nw, w_max, S = 1024, 0.2 / 1024, 8, 8, 200.0, 8
    ks = ctx.wkernel_build(Nw, w_max, S, Q, N, cell, wpgrid.F32)
    d = inputs(303, 200_000, 1, 1500.0, 150.0)
    grid = ctx.new_grid(ks)
    ctx.grid_static(*d, ks, grid)                                      # first call: module load, symbol look-up
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    alloc0 = torch.cuda.memory_allocated()
    for _ in range(3):
        ctx.grid_static(*d, ks, grid)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert torch.cuda.memory_allocated() == alloc0 and free1 == free0, (free0, free1)

    # beyond the static array: a clear error, nothing launched, the grid untouched
    n_big = 5_000_000
    assert ctx.grid_workspace_bytes(n_big, 1, ks) > ctx.static_scratch_bytes()
    big = tuple(torch.zeros(s, dtype=t, device="cuda") for s, t in
                (((n_big, 1), torch.complex64), ((n_big, 3), torch.float64), ((n_big, 1), torch.float32)))
    before = grid.clone()
    launches = ctx.launch_count()
    with pytest.raises(wpgrid.WpgError) as ei:
        ctx.grid_static(big[0], big[1], big[2], d[3], ks, grid)
    assert ei.value.code == wpgrid.ENOMEM and "static" in str(ei.value) and str(ctx.static_scratch_bytes()) in str(ei.value)
    assert ctx.launch_count() == launches and bool((grid == before).all())
    # the context still works afterwards
    ctx.grid_static(*d, ks, grid)
    torch.cuda.synchronize()
