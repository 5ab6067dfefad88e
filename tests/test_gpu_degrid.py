"""GPU degridder (wpg_degrid) against the oracle degridder through the C ABI: element by element on the same
seeded inputs, counts exact; tolerances as for gridding, relative to the largest predicted visibility."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

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


def check(ctx, uvw, freq, st, g, support):
    ref, rcnt = ogrid.degrid(uvw, freq, st, g)
    du, df = torch.from_numpy(uvw).cuda(), torch.from_numpy(freq).cuda()
    for prec in (wpgrid.F32, wpgrid.F64):
        ks = ctx.stack_from_host(st.data, st.Nw, st.w_max, support, st.oversample, st.grid_N, st.cell, prec)
        dg = torch.from_numpy(g.astype(np.complex64 if prec == wpgrid.F32 else np.complex128)).cuda()
        for general in (0, 1):            # 0: degrid_fast_kernel where it applies (S = 4, 8, 16); 1: degrid_kernel always
            ctx.set_option("no_pairs", general)
            out, cnt = ctx.degrid(dg, du, df, ks, counts=True)
            ctx.set_option("no_pairs", 0)
            assert cnt == rcnt
            o = out.cpu().numpy().astype(np.complex128)
            err = float(np.max(np.abs(o - ref)) / np.max(np.abs(ref)))
            assert err <= TOL[prec], (prec, general, err)
            assert np.array_equal(o == 0, ref == 0) or prec == wpgrid.F32


@pytest.mark.parametrize("S", [4, 7, 8, 12, 16, 32])
def test_degrid_matches_oracle_uniform_stacks(ctx, S):
    rng = np.random.default_rng(40 + S)
    N, cell, Q, Nw, w_max = 256, 0.1 / 256, 8 if S != 7 else 8, 6, 90.0
    n, nchan = 20_001, 2                      # not a multiple of 32: ragged last warp batch
    dul = 1.0 / 0.1
    uvw = np.stack([rng.uniform(-135, 135, n) * dul, rng.uniform(-135, 135, n) * dul, rng.uniform(-100, 100, n)], 1)
    freq = np.array([0.95, 1.05]) * synth.C0
    st = owk.build_stack(Nw, w_max, S, Q, N, cell)
    g = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    check(ctx, uvw, freq, st, g, S)


def test_degrid_ragged_stack_and_empty_input(ctx):
    wl = synth.config4(n_dump=1, nchan=2, values="random")
    sup = owk.ragged_support(wl.Nw, wl.w_max, wl.grid_N, wl.cell, 8, 32)
    st = owk.build_stack(wl.Nw, wl.w_max, sup, wl.oversample, wl.grid_N, wl.cell)
    rng = np.random.default_rng(1)
    N = wl.grid_N
    g = (rng.standard_normal((N, N), dtype=np.float32) + 1j * rng.standard_normal((N, N), dtype=np.float32)).astype(np.complex128)
    check(ctx, wl.uvw[:60_000], wl.freq, st, g, sup)
    ks = ctx.stack_from_host(st.data, st.Nw, st.w_max, sup, st.oversample, N, st.cell, wpgrid.F32)
    out, cnt = ctx.degrid(torch.zeros((N, N), dtype=torch.complex64).cuda(), torch.zeros((0, 3), dtype=torch.float64).cuda(),
                          torch.from_numpy(wl.freq).cuda(), ks, counts=True)
    assert out.shape == (0, 2) and cnt == {"n_predicted": 0, "n_outside": 0}


def test_degrid_is_the_adjoint_of_the_gpu_gridder(ctx):
    """<wpg_grid(v), g> = <v, wpg_degrid(g)> on the device, fp64, config-2-like tracks."""
    wl = synth.config2(nvis=200_000)
    ks = ctx.wkernel_build(wl.Nw, wl.w_max, wl.support, wl.oversample, wl.grid_N, wl.cell, wpgrid.F64)
    d = [torch.from_numpy(x).cuda() for x in (wl.vis, wl.uvw, wl.weight, wl.freq)]
    Av, _ = ctx.grid(*d, ks)
    gen = torch.Generator(device="cuda").manual_seed(5)
    g = torch.randn((wl.grid_N, wl.grid_N), dtype=torch.complex128, device="cuda", generator=gen)
    AHg, _ = ctx.degrid(g, d[1], d[3], ks)
    lhs = torch.vdot(g.flatten(), Av.flatten()); rhs = torch.vdot(AHg.flatten(), d[0].flatten().to(torch.complex128))
    assert abs(lhs - rhs) <= 1e-10 * abs(lhs)
