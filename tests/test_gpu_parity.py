"""GPU <-> oracle parity (-m gpu).  Everything goes through the C ABI (libwpgrid.so) via the
thin binding.  Tolerances (north_star / DESIGN.md R17): max|g - g_oracle| <= 1e-4 max|g_oracle|
for fp32 and <= 1e-10 max|g_oracle| for fp64; integer outputs (counters, records) bit-exact."""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import gridder as ogrid
from oracle import image as oimage
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


def dev(wl):
    return (torch.from_numpy(wl.vis).cuda(), torch.from_numpy(wl.uvw).cuda(),
            torch.from_numpy(wl.weight).cuda(), torch.from_numpy(wl.freq).cuda())


def oracle_stack(wl):
    sup = wl.support
    if not np.isscalar(sup):
        sup = owk.ragged_support(wl.Nw, wl.w_max, wl.grid_N, wl.cell, sup[1], sup[2])
    return owk.build_stack(wl.Nw, wl.w_max, sup, wl.oversample, wl.grid_N, wl.cell)


def classes_exercised(wl, st):
    """{support: number of visibilities whose plane has that support} (which gridder instantiations a ragged stack
    reaches; w -> plane as in G2, used only for this coverage assertion)."""
    w = (wl.uvw[:, 2:3] * (wl.freq / synth.C0)[None, :]).ravel()
    p = np.clip(np.floor((w + wl.w_max) / (2.0 * wl.w_max / wl.Nw)), 0, wl.Nw - 1).astype(np.int64)
    cls, cnt = np.unique(st.support[p], return_counts=True)
    return dict(zip(cls.tolist(), cnt.tolist()))


def upload(ctx, st, prec):
    sup = int(st.support[0]) if st.uniform else st.support
    return ctx.stack_from_host(st.data, st.Nw, st.w_max, sup, st.oversample, st.grid_N, st.cell, prec)


def relerr(g, ref):
    return float(np.max(np.abs(g.astype(np.complex128) - ref)) / np.max(np.abs(ref)))


def check_all_paths(ctx, wl, st, ref, rstats, precs=(wpgrid.F32, wpgrid.F64), key_bits=(0,), segments=(0,)):
    d = dev(wl)
    for prec in precs:
        ks = upload(ctx, st, prec)
        g, s = ctx.grid_naive(*d, ks, stats=True)
        assert s == rstats
        assert relerr(g.cpu().numpy(), ref) <= TOL[prec], ("naive", prec)
        for kb in key_bits:
            for seg in segments:
                ctx.set_option("key_bits", kb); ctx.set_option("segment", seg)
                g, s = ctx.grid(*d, ks, stats=True)
                assert s == rstats, (kb, seg)
                e = relerr(g.cpu().numpy(), ref)
                assert e <= TOL[prec], ("runs", prec, kb, seg, e)
    ctx.set_option("key_bits", 0); ctx.set_option("segment", 0)


# ------------------------------------------------------------------ config 1 (full size)
@pytest.fixture(scope="module")
def cfg1():
    wl = synth.config1()
    st = oracle_stack(wl)
    ref, rstats = ogrid.grid(wl.uvw, wl.vis, wl.weight, wl.freq, st)
    return wl, st, ref, rstats


def test_config1_gridder_parity(ctx, cfg1):
    wl, st, ref, rstats = cfg1
    check_all_paths(ctx, wl, st, ref, rstats, key_bits=(0, 12, 8), segments=(0, 1, 7, 100, 100000))


def test_config1_wkernel_build_parity(ctx, cfg1):
    wl, st, _, _ = cfg1
    K = st.data
    k64 = ctx.wkernel_build(wl.Nw, wl.w_max, wl.support, wl.oversample, wl.grid_N, wl.cell, wpgrid.F64)
    assert np.max(np.abs(k64.data.cpu().numpy() - K)) <= 1e-10 * np.max(np.abs(K))
    k32 = ctx.wkernel_build(wl.Nw, wl.w_max, wl.support, wl.oversample, wl.grid_N, wl.cell, wpgrid.F32)
    assert np.max(np.abs(k32.data.cpu().numpy() - K)) <= 1e-6 * np.max(np.abs(K))


def test_config1_end_to_end_image(ctx, cfg1):
    """wkernel_build -> grid -> dirty_image entirely in the library vs the oracle chain."""
    wl, st, ref, _ = cfg1
    d = dev(wl)
    wsum = float(wl.weight.sum())
    ref_img = oimage.dirty_image(ref, wl.cell, wsum)
    for prec, tol in ((wpgrid.F32, 1e-4), (wpgrid.F64, 1e-10)):           # north_star's bounds, end to end
        ks = ctx.wkernel_build(wl.Nw, wl.w_max, wl.support, wl.oversample, wl.grid_N, wl.cell, prec)
        g, _ = ctx.grid(*d, ks)
        assert relerr(g.cpu().numpy(), ref) <= tol
        img = ctx.dirty_image(g, ks, wsum).cpu().numpy().astype(np.float64)
        assert np.max(np.abs(img - ref_img)) <= tol * np.max(np.abs(ref_img))
        # the image step alone, fed the oracle's grid
        gi = torch.from_numpy(ref.astype(np.complex64 if prec == wpgrid.F32 else np.complex128)).cuda()
        img = ctx.dirty_image(gi, ks, wsum).cpu().numpy().astype(np.float64)
        # (fp32: the division by a taper as small as 1e-3 amplifies the FFT's rounding near the edge)
        assert np.max(np.abs(img - ref_img)) <= (1e-4 if prec == wpgrid.F32 else 1e-12) * np.max(np.abs(ref_img))
        assert np.array_equal(img == 0.0, ref_img == 0.0)


def test_grid_host_variant_matches(ctx, cfg1):
    wl, st, ref, rstats = cfg1
    ks = upload(ctx, st, wpgrid.F32)
    out, s = ctx.grid_host(wl.vis, wl.uvw, wl.weight, wl.freq, ks, stats=True)
    assert s == rstats and relerr(out, ref) <= 1e-4
    out2, _ = ctx.grid_host(wl.vis, wl.uvw, wl.weight, wl.freq, ks)       # grid is overwritten, not accumulated
    assert relerr(out2, ref) <= 1e-4


# ------------------------------------------------------------------ binning (bit-exact)
def test_binning_records_match_oracle_index_map(ctx):
    wl = synth.config1(nvis=20000)
    st = oracle_stack(wl)
    ks = upload(ctx, st, wpgrid.F32)
    d = dev(wl)
    S, Q, N = 7, 8, wl.grid_N
    exp = []
    for k in range(wl.uvw.shape[0]):
        j0u, ou = ogrid.index_map(wl.uvw[k, 0], N, wl.cell, S, Q)
        j0v, ov = ogrid.index_map(wl.uvw[k, 1], N, wl.cell, S, Q)
        p, _ = ogrid.plane_of(wl.uvw[k, 2], wl.w_max, wl.Nw)
        exp.append((j0u | (j0v << 16), (p * Q * Q + ov * Q + ou) * S * S,
                    np.float32(wl.vis[k, 0].real).view(np.uint32), np.float32(wl.vis[k, 0].imag).view(np.uint32)))
    exp = sorted(exp)
    ctx.set_option("compress", 0)              # one record per gridded visibility (compression: test_record_compression)
    for kb in (0, 12):
        ctx.set_option("key_bits", kb)
        ws, info, stats = ctx.bin(*d, ks)
        assert info["n_records"] == 20000 and info["n_classes"] == 1 and info["record_bytes"] == 16
        ksh = info["key_shift"]
        nkg = (N + (1 << ksh) - 1) >> ksh
        assert ksh == (0 if kb == 0 else 4) and info["keys_per_class"] == N * nkg
        raw = ws.cpu().numpy()
        rec = raw[info["off_records"]:info["off_records"] + 16 * 20000].view(np.uint32).reshape(-1, 4)
        got = sorted((int(r[2]), int(r[3]), int(r[0]), int(r[1])) for r in rec)
        assert got == [tuple(int(x) for x in e) for e in exp]
        # records are ordered by key = j0u * ceil(N / 2^ksh) + (j0v >> ksh); bucket_start matches that order
        ju = (rec[:, 2] & 0xFFFF).astype(np.int64); jv = (rec[:, 2] >> 16).astype(np.int64)
        key = ju * nkg + (jv >> ksh)
        assert np.all(np.diff(key) >= 0)
        bs = raw[info["off_bucket_start"]:info["off_bucket_start"] + 4 * (info["n_keys"] + 1)].view(np.uint32)
        assert bs[0] == 0 and bs[-1] == 20000
        assert np.array_equal(bs.astype(np.int64), np.searchsorted(key, np.arange(info["n_keys"] + 1)))
    ctx.set_option("key_bits", 0); ctx.set_option("compress", 1)


def test_record_compression(ctx):
    """Record compression: with the rows-per-time-step hint a binning thread
    holds consecutive samples of one baseline and channel; those with the same window start and coefficient slice
    share one record carrying the sum of their weight * vis.  Checked on slowly drifting tracks: fewer records than
    gridded visibilities; every record is an oracle (window, slice) pair; per pair the record values sum to the
    oracle-side sum of weight * vis; counters count visibilities, not records; the grid is unchanged."""
    rng = np.random.default_rng(17)
    N, cell, Q, S, Nw, w_max = 256, 0.1 / 256, 8, 8, 8, 100.0
    nbl, ndump, nchan = 97, 200, 2
    nrow = nbl * ndump
    b = np.arange(nrow) % nbl; t = np.arange(nrow) // nbl
    uvw = np.stack([(b - 48) * 11.0 + 0.05 * t, (b % 9 - 4) * 95.0 + 0.03 * t, rng.uniform(-90, 90, nbl)[b]], 1)
    freq = np.array([1.0, 1.01]) * synth.C0 / 0.5
    vis = (rng.standard_normal((nrow, nchan)) + 1j * rng.standard_normal((nrow, nchan))).astype(np.complex64)
    wt = rng.uniform(0.5, 2.0, (nrow, nchan)).astype(np.float32)
    wt[rng.uniform(size=wt.shape) < 0.05] = 0.0
    st = owk.build_stack(Nw, w_max, S, Q, N, cell)
    ref, rstats = ogrid.grid(uvw, vis, wt, freq, st)
    wl = synth.Workload("drift", uvw, freq, vis, wt, N, cell, Nw, w_max, S, Q)
    d = dev(wl)
    expect = {}
    fs = freq / synth.C0
    for k in range(nrow):
        for c in range(nchan):
            if wt[k, c] == 0.0:
                continue
            j0u, ou = ogrid.index_map(uvw[k, 0] * fs[c], N, cell, S, Q)
            j0v, ov = ogrid.index_map(uvw[k, 1] * fs[c], N, cell, S, Q)
            if j0u < 0 or j0v < 0 or j0u + S > N or j0v + S > N:
                continue
            p, _ = ogrid.plane_of(uvw[k, 2] * fs[c], w_max, Nw)
            kk = (j0u | (j0v << 16), (p * Q * Q + ov * Q + ou) * S * S)
            expect[kk] = expect.get(kk, 0j) + complex(np.float32(wt[k, c])) * complex(vis[k, c])
    for prec, rb_bytes in ((wpgrid.F32, 16), (wpgrid.F64, 24)):
        ks = upload(ctx, st, prec)
        n_rec = {}
        for rb, comp in ((nbl, 1), (nbl, 0), (0, 1)):
            ctx.set_option("row_block", rb); ctx.set_option("compress", comp)
            ws, info, stats = ctx.bin(*d, ks)
            assert stats == rstats and info["record_bytes"] == rb_bytes
            n = info["n_records"]
            n_rec[(rb, comp)] = n
            raw = ws.cpu().numpy()[info["off_records"]:info["off_records"] + rb_bytes * n]
            got = {}
            if prec == wpgrid.F32:
                r = raw.view(np.uint32).reshape(-1, 4)
                vals = r[:, :2].copy().view(np.float32).astype(np.float64); keys = r[:, 2:]
            else:
                vals = raw.view(np.float64).reshape(-1, 3)[:, :2]; keys = raw.view(np.uint32).reshape(-1, 6)[:, 4:]
            for (re, im), (ps, ko) in zip(vals, keys):
                kk = (int(ps), int(ko))
                got[kk] = got.get(kk, 0j) + complex(re, im)
            assert set(got) == set(expect)
            tol = 2e-6 if prec == wpgrid.F32 else 1e-13
            assert max(abs(got[k] - expect[k]) for k in expect) <= tol * max(abs(x) for x in expect.values())
            g, s = ctx.grid(*d, ks, stats=True)
            assert s == rstats and relerr(g.cpu().numpy(), ref) <= TOL[prec]
        assert n_rec[(nbl, 0)] == rstats["n_gridded"]
        assert n_rec[(nbl, 1)] < 0.6 * rstats["n_gridded"]        # consecutive samples drift by ~0.005 cells: runs of 4 merge
        assert n_rec[(nbl, 1)] >= len(expect)
    ctx.set_option("row_block", 0); ctx.set_option("compress", 1)


# ------------------------------------------------------------------ edge cases
def test_edge_cases(ctx):
    N, cell, Q, S, Nw, w_max = 64, 0.08 / 64, 8, 8, 4, 50.0
    st = owk.build_stack(Nw, w_max, S, Q, N, cell)
    du = 1.0 / 0.08
    uvw = np.array([[0.0, 0.0, 0.0], [40 * du, 0.0, 0.0], [-29 * du, 0.0, 0.0], [-29.1 * du, 0.0, 0.0],
                    [0.0, 28.4 * du, 10.0], [0.0, 27.4 * du, 10.0], [du, du, 80.0], [du, du, -80.0],
                    [1e30, 0.0, 0.0], [0.0, -1e30, 1e30]])
    n = uvw.shape[0]
    vis = (np.arange(n) + 1 + 1j * np.arange(n)).astype(np.complex64)[:, None]
    wt = np.ones((n, 1), np.float32); wt[5, 0] = 0.0
    freq = np.array([synth.C0])
    ref, rstats = ogrid.grid(uvw, vis, wt, freq, st)
    wl = synth.Workload("edge", uvw, freq, vis, wt, N, cell, Nw, w_max, S, Q)
    check_all_paths(ctx, wl, st, ref, rstats)
    # empty input: nothing happens, counters are zero
    ks = upload(ctx, st, wpgrid.F32)
    z = (torch.zeros((0, 1), dtype=torch.complex64).cuda(), torch.zeros((0, 3), dtype=torch.float64).cuda(),
         torch.zeros((0, 1), dtype=torch.float32).cuda(), torch.from_numpy(freq).cuda())
    g, s = ctx.grid(*z, ks, stats=True)
    assert not g.any() and all(v == 0 for v in s.values())
    # everything flagged
    d = dev(wl)
    g, s = ctx.grid(d[0], d[1], torch.zeros_like(d[2]), d[3], ks, stats=True)
    assert not g.any() and s["n_skipped_zero_weight"] == n and s["n_gridded"] == 0
    # accumulation into a non-zero grid (chunking, P12)
    g0 = torch.from_numpy(ref.astype(np.complex64)).cuda()
    g, _ = ctx.grid(*d, ks, grid=g0.clone())
    assert relerr(g.cpu().numpy(), 2 * ref) <= 1e-4


def test_errors_cross_the_abi_as_codes(ctx):
    st = owk.build_stack(2, 10.0, 8, 8, 64, 0.001)
    ks = upload(ctx, st, wpgrid.F32)
    wl = synth.config1(nvis=16)
    d = dev(wl)
    with pytest.raises(wpgrid.WpgError) as e:
        ctx.grid(*d, ks, workspace=torch.empty(16, dtype=torch.uint8, device="cuda"))
    assert e.value.code == wpgrid.ENOMEM
    with pytest.raises(wpgrid.WpgError) as e:
        ctx.wkernel_build(4, 10.0, 7, 3, 64, 0.001)        # S*Q odd
    assert e.value.code == wpgrid.EINVAL
    with pytest.raises(wpgrid.WpgError) as e:
        ctx.set_option("nonsense", 1)
    assert e.value.code == wpgrid.EINVAL


def test_multichannel_and_weights(ctx):
    rng = np.random.default_rng(21)
    N, cell, Q, S, Nw = 256, 0.1 / 256, 8, 8, 8
    nrow, nchan = 3000, 4
    uvw = np.stack([rng.uniform(-600, 600, nrow), rng.uniform(-600, 600, nrow), rng.uniform(-40, 40, nrow)], 1)
    freq = np.linspace(0.9, 1.3, nchan) * synth.C0 / 0.5          # wavelengths 0.5/0.9 ... m
    w_max = 100.0
    vis = (rng.standard_normal((nrow, nchan)) + 1j * rng.standard_normal((nrow, nchan))).astype(np.complex64)
    wt = rng.uniform(0.0, 2.0, (nrow, nchan)).astype(np.float32)
    wt[rng.uniform(size=wt.shape) < 0.1] = 0.0
    st = owk.build_stack(Nw, w_max, S, Q, N, cell)
    ref, rstats = ogrid.grid(uvw, vis, wt, freq, st)
    assert rstats["n_skipped_zero_weight"] > 0 and rstats["n_skipped_oob"] > 0 and rstats["n_clamped_w"] > 0
    wl = synth.Workload("mc", uvw, freq, vis, wt, N, cell, Nw, w_max, S, Q)
    check_all_paths(ctx, wl, st, ref, rstats)


# ------------------------------------------------------------------ the other configs, scaled
@pytest.mark.parametrize("S", [4, 7, 8, 12, 16])
def test_config3_supports(ctx, S):
    """Config-3 sweep points at reduced visibility count (N = 1024, every support of the sweep
    plus the odd 7): several tiles, ragged tails, fp32 and fp64, both sort orders."""
    wl = synth.config3(N=1024, S=S, nvis=150_000)
    st = oracle_stack(wl)
    ref, rstats = ogrid.grid(wl.uvw, wl.vis, wl.weight, wl.freq, st, threads=4)
    assert rstats["n_gridded"] == 150_000
    check_all_paths(ctx, wl, st, ref, rstats)


def test_config2_scaled(ctx):
    wl = synth.config2(nvis=400_000)
    st = oracle_stack(wl)
    ref, rstats = ogrid.grid(wl.uvw, wl.vis, wl.weight, wl.freq, st, threads=4)
    check_all_paths(ctx, wl, st, ref, rstats, precs=(wpgrid.F32,))
    ks = ctx.wkernel_build(wl.Nw, wl.w_max, wl.support, wl.oversample, wl.grid_N, wl.cell, wpgrid.F64)
    assert np.max(np.abs(ks.data.cpu().numpy() - st.data)) <= 1e-10 * np.max(np.abs(st.data))


def test_config4_ragged_scaled(ctx):
    """SKA-low-like layout, ragged support 8..32, 8 channels, N = 8192; 2 dumps (2.1e6 visibilities)."""
    wl = synth.config4(n_dump=2, values="random")
    st = oracle_stack(wl)
    # the support classes this input sends visibilities to (each is one gridder launch of its own instantiation)
    assert sorted(classes_exercised(wl, st)) == [8, 10, 12, 14, 16, 18]
    ref, rstats = ogrid.grid(wl.uvw, wl.vis, wl.weight, wl.freq, st, threads=4)
    sup, off = wpgrid.ragged_support(wl.Nw, wl.w_max, wl.grid_N, wl.cell, wl.oversample, 8, 32)
    assert np.array_equal(sup, st.support) and np.array_equal(off, st.plane_offset)
    check_all_paths(ctx, wl, st, ref, rstats, precs=(wpgrid.F32,))
    # the library's own ragged stack
    ks = ctx.wkernel_build(wl.Nw, wl.w_max, sup, wl.oversample, wl.grid_N, wl.cell, wpgrid.F64)
    assert np.max(np.abs(ks.data.cpu().numpy() - st.data)) <= 1e-10 * np.max(np.abs(st.data))


def test_config5_scaled_both_precisions(ctx):
    wl = synth.config5(nvis=300_000)
    st = oracle_stack(wl)
    ref, rstats = ogrid.grid(wl.uvw, wl.vis, wl.weight, wl.freq, st, threads=4)
    check_all_paths(ctx, wl, st, ref, rstats)


# ------------------------------------------------------------------ full size, bench.py's launch configuration
def test_config2_full_size_as_benchmarked(ctx):
    """BASELINE config 2 at its full 1e7 visibilities, in the configuration bench.py times (preallocated
    workspace, default options, the library's own stack): the whole 2048^2 grid element by element against the
    oracle (the C oracle with all host cores finishes 6.4e8 updates in about a second), the counters bit-exact,
    and flux conservation (P11) on the GPU grid."""
    import os
    wl = synth.config2(device="cuda")
    assert wl.nvis == 10_000_000
    st = oracle_stack(wl)
    ref, rstats = ogrid.grid(wl.uvw, wl.vis, wl.weight, wl.freq, st, threads=min(os.cpu_count() or 1, 32))
    assert rstats["n_updates"] == 640_000_000
    d = dev(wl)
    ks = ctx.wkernel_build(wl.Nw, wl.w_max, wl.support, wl.oversample, wl.grid_N, wl.cell, wpgrid.F32)
    ws = torch.empty(ctx.grid_workspace_bytes(wl.uvw.shape[0], 1, ks), dtype=torch.uint8, device="cuda")
    grid = ctx.new_grid(ks)
    ctx.set_option("row_block", wl.notes["row_block"])  # as bench.py does for track-based workloads
    for _ in range(2):                                  # twice: workspace reuse, as in the timed loop
        grid.zero_()
        g, s = ctx.grid(*d, ks, grid=grid, workspace=ws, stats=True)
        assert s == rstats
        gh = g.cpu().numpy()
        print("config2 full size fp32 relerr %.3e" % relerr(gh, ref))          # (-s shows it; profiles/r01_precision.md)
        assert relerr(gh, ref) <= TOL[wpgrid.F32]
        assert abs(gh.sum(dtype=np.complex128) - ref.sum()) <= 1e-5 * abs(ref.sum())
    # the host-buffer entry point pipelines four row chunks (copy of chunk k + 1 under the gridding of chunk k)
    out, s_host = ctx.grid_host(wl.vis, wl.uvw, wl.weight, wl.freq, ks, stats=True)
    assert s_host == rstats and relerr(out, ref) <= TOL[wpgrid.F32]
    ctx.set_option("row_block", 0)
    out, s_host = ctx.grid_host(wl.vis[:1_300_001], wl.uvw[:1_300_001], wl.weight[:1_300_001], wl.freq, ks, stats=True)
    ref13, rstats13 = ogrid.grid(wl.uvw[:1_300_001], wl.vis[:1_300_001], wl.weight[:1_300_001], wl.freq, st, threads=8)
    assert s_host == rstats13 and relerr(out, ref13) <= TOL[wpgrid.F32]
    # dirty image of the full grid
    wsum = float(wl.weight.sum())
    img = ctx.dirty_image(g, ks, wsum).cpu().numpy().astype(np.float64)
    ref_img = oimage.dirty_image(ref, wl.cell, wsum)
    ierr = float(np.max(np.abs(img - ref_img)) / np.max(np.abs(ref_img)))
    print("config2 full size fp32 dirty image relerr %.3e" % ierr)
    assert ierr <= 1e-4


def test_config5_1e7_both_precisions_full_grid(ctx):
    """Config 5 (N = 4096, S = 16, 256-station tracks) on its first 1e7 visibilities through the full-size
    grid, fp32 and fp64 from identical inputs, errors against the fp64 oracle (2.56e9 updates)."""
    import os
    wl = synth.config5(nvis=10_000_000, device="cuda")
    st = oracle_stack(wl)
    ref, rstats = ogrid.grid(wl.uvw, wl.vis, wl.weight, wl.freq, st, threads=min(os.cpu_count() or 1, 32))
    d = dev(wl)
    for prec in (wpgrid.F32, wpgrid.F64):
        ks = upload(ctx, st, prec)
        g, s = ctx.grid(*d, ks, stats=True)
        assert s == rstats
        e = relerr(g.cpu().numpy(), ref)
        print("config5 1e7 prec %d relerr %.3e" % (prec, e))
        assert e <= TOL[prec], (prec, e)
        del g


def test_config3_large_grid_uniform(ctx):
    """Config-3 sweep point in the regime the paper flags as slow (N = 8192 > 2048, S = 12 > 8), 4e6
    visibilities through the full-size grid, fp32 and fp64."""
    wl = synth.config3(N=8192, S=12, nvis=4_000_000)
    st = oracle_stack(wl)
    ref, rstats = ogrid.grid(wl.uvw, wl.vis, wl.weight, wl.freq, st, threads=8)
    d = dev(wl)
    for prec in (wpgrid.F32, wpgrid.F64):
        ks = upload(ctx, st, prec)
        g, s = ctx.grid(*d, ks, stats=True)
        assert s == rstats
        e = relerr(g.cpu().numpy(), ref)
        print("config3 N=8192 S=12 prec %d relerr %.3e" % (prec, e))
        assert e <= TOL[prec], (prec, e)
        del g


# ------------------------------------------------------------------ code paths added with the pair / cell gridders
def _support_case(S, seed):
    rng = np.random.default_rng(seed)
    N, cell, Q, Nw, w_max, n = 128, 0.06 / 128, 4, 6, 80.0, 6000
    du = 1.0 / 0.06
    uvw = np.stack([rng.uniform(-40, 40, n) * du, rng.uniform(-40, 40, n) * du, rng.uniform(-90, 90, n)], 1)
    uvw[: n // 3, :2] = np.round(uvw[: n // 3, :2] / du) * du          # long runs of equal windows as well
    vis = (rng.standard_normal((n, 1)) + 1j * rng.standard_normal((n, 1))).astype(np.complex64)
    wt = rng.uniform(0.5, 1.5, (n, 1)).astype(np.float32)
    freq = np.array([synth.C0])
    st = owk.build_stack(Nw, w_max, S, Q, N, cell)
    ref, rstats = ogrid.grid(uvw, vis, wt, freq, st)
    assert rstats["n_gridded"] > 5000
    return synth.Workload("S%d" % S, uvw, freq, vis, wt, N, cell, Nw, w_max, S, Q), st, ref, rstats


@pytest.mark.parametrize("S", [2, 4, 6, 8, 10, 12, 14, 16, 18, 20, 22, 24, 26, 28, 30, 32])
def test_even_supports_segments_and_tails(ctx, S):
    """Every instantiation of the pair gridder (lane groups at S = 4 and 8, power-of-two and generic supports with
    1..4 lane-slot sets, the window split over two to four work items from S = 16 up) and of the fp64 cell gridder
    (window split over 2..8 work items), with work-item lengths that leave ragged tails in the look-ahead ring
    (1, 5, 17 records) and one item for everything.  launch_class (csrc/wpg_grid.cu) picks the instantiation from S
    alone for a uniform stack, so this list reaches every even-support line of it in both precisions."""
    wl, st, ref, rstats = _support_case(S, 100 + S)
    check_all_paths(ctx, wl, st, ref, rstats, segments=(0, 1, 5, 17, 100000))
    ctx.set_option("no_pairs", 1)                                       # the run gridder on the same input
    check_all_paths(ctx, wl, st, ref, rstats)
    ctx.set_option("no_pairs", 0)


@pytest.mark.parametrize("S", [3, 5, 7, 9, 11, 13, 15, 17, 19, 21, 23, 27, 31])
def test_odd_supports_segments_and_tails(ctx, S):
    """Odd supports (the paper's own experiments use full support 9): fp32 goes through the cell
    gridder with one cell per lane-slot (2 slot sets up to S = 7, 4 at S = 9 / 11, the window split over 2 / 4 / 8
    work items at S = 13-15 / 17-21 / 23-31), fp64 through its 5-slot and window-split lines (S = 9 ... 27).  Same
    ragged work-item lengths as the even supports, and the run gridder on the same input."""
    wl, st, ref, rstats = _support_case(S, 300 + S)
    check_all_paths(ctx, wl, st, ref, rstats, segments=(0, 1, 5, 17, 100000))
    ctx.set_option("no_pairs", 1)
    check_all_paths(ctx, wl, st, ref, rstats)
    ctx.set_option("no_pairs", 0)


def test_ragged_stack_key_budgets_both_precisions(ctx):
    """Ragged stack (per-class sort keys planned on the device from the class census): the result must not
    depend on the key budget — from one key per grid column (key_bits = 8 is below the minimum and is raised
    to it) to ample — in fp32 and fp64."""
    wl = synth.config4(n_dump=1, nchan=2, values="random")
    st = oracle_stack(wl)
    ref, rstats = ogrid.grid(wl.uvw, wl.vis, wl.weight, wl.freq, st, threads=4)
    assert sorted(classes_exercised(wl, st)) == [8, 10, 12, 14, 16, 18]
    check_all_paths(ctx, wl, st, ref, rstats, key_bits=(0, 8, 20, 27))


def test_row_block_hint_changes_nothing_but_speed(ctx):
    """The rows-per-time-step hint only re-maps binning threads to visibilities (same baseline at consecutive
    times, one bucket-counter update per run of equal keys): counters bit-exact, grid within tolerance, for a
    track-based workload, for a block size that does not divide the row count, and with several channels."""
    wl = synth.config2(nvis=400_001)
    st = oracle_stack(wl)
    ref, rstats = ogrid.grid(wl.uvw, wl.vis, wl.weight, wl.freq, st, threads=4)
    for rb in (wl.notes["row_block"], 1, 777):
        ctx.set_option("row_block", rb)
        check_all_paths(ctx, wl, st, ref, rstats, precs=(wpgrid.F32,))
    rng = np.random.default_rng(5)
    N, cell, Q, S, Nw, w_max = 256, 0.1 / 256, 8, 8, 8, 100.0
    nrow, nchan = 40_000, 2
    # slowly drifting tracks: 123 "baselines", consecutive time steps move by a fraction of a cell
    b = np.arange(nrow) % 123; t = np.arange(nrow) // 123
    uvw = np.stack([(b - 60) * 9.0 + 0.7 * t, (b % 11 - 5) * 80.0 + 0.4 * t, rng.uniform(-90, 90, 123)[b]], 1)
    freq = np.array([1.0, 1.02]) * synth.C0 / 0.5
    vis = (rng.standard_normal((nrow, nchan)) + 1j * rng.standard_normal((nrow, nchan))).astype(np.complex64)
    wt = rng.uniform(0.0, 2.0, (nrow, nchan)).astype(np.float32)
    wt[rng.uniform(size=wt.shape) < 0.05] = 0.0
    st = owk.build_stack(Nw, w_max, S, Q, N, cell)
    ref, rstats = ogrid.grid(uvw, vis, wt, freq, st)
    assert rstats["n_gridded"] > 50_000
    wl2 = synth.Workload("tracks", uvw, freq, vis, wt, N, cell, Nw, w_max, S, Q)
    for rb in (123, 0):
        ctx.set_option("row_block", rb)
        check_all_paths(ctx, wl2, st, ref, rstats)
    ctx.set_option("row_block", 0)


def test_binning_exactness_on_ties_and_near_ties(ctx):
    """Exactness rule G6 under the constant-divisor fast path: visibilities whose oversampled coordinate
    x*Q + 1/2 lands exactly on an integer (rounding ties), one ulp to either side, and whose w sits on plane
    boundaries, for cell sizes whose reciprocal is not a power of two.  Every record (window start, coefficient
    slice) must equal the oracle's integer decisions bit for bit."""
    rng = np.random.default_rng(99)
    for N, fov, S, Q, Nw, w_max in ((256, 0.1, 8, 8, 16, 77.7), (1000, 0.0731, 7, 8, 9, 310.0), (512, 0.0509, 12, 4, 5, 55.5)):
        cell = fov / N
        du = 1.0 / fov
        n = 6000
        # coordinates in cells at multiples of 1/(2Q) (ties of the nearest-oversample-point rule) -> wavelengths,
        # then nudged by 0, +-1, +-2 ulps
        k = rng.integers(-int(0.4 * N) * 2 * Q, int(0.4 * N) * 2 * Q, size=(n, 2))
        uv = (k / (2.0 * Q)) * du
        nudge = rng.integers(-2, 3, size=(n, 2))
        for _ in range(2):
            uv = np.where(nudge > 0, np.nextafter(uv, np.inf), np.where(nudge < 0, np.nextafter(uv, -np.inf), uv))
            nudge = nudge - np.sign(nudge)
        dw = 2.0 * w_max / Nw
        w = -w_max + dw * rng.integers(0, Nw + 1, n)                  # plane boundaries
        wn = rng.integers(-1, 2, n)
        w = np.where(wn > 0, np.nextafter(w, np.inf), np.where(wn < 0, np.nextafter(w, -np.inf), w))
        uvw = np.ascontiguousarray(np.stack([uv[:, 0], uv[:, 1], w], 1))
        vis = (np.arange(n) + 1j).astype(np.complex64)[:, None]
        wt = np.ones((n, 1), np.float32)
        freq = np.array([synth.C0])
        st = owk.build_stack(Nw, w_max, S, Q, N, cell)
        ks = upload(ctx, st, wpgrid.F32)
        exp = []
        for i in range(n):
            j0u, ou = ogrid.index_map(uvw[i, 0], N, cell, S, Q)
            j0v, ov = ogrid.index_map(uvw[i, 1], N, cell, S, Q)
            p, _ = ogrid.plane_of(uvw[i, 2], w_max, Nw)
            if j0u < 0 or j0v < 0 or j0u + S > N or j0v + S > N:
                continue
            exp.append((j0u | (j0v << 16), (p * Q * Q + ov * Q + ou) * S * S, i))
        d = (torch.from_numpy(vis).cuda(), torch.from_numpy(uvw).cuda(), torch.from_numpy(wt).cuda(), torch.from_numpy(freq).cuda())
        ctx.set_option("compress", 0)
        for rb in (0, 7):
            ctx.set_option("row_block", rb)
            ws, info, stats = ctx.bin(*d, ks)
            assert info["n_records"] == len(exp)
            raw = ws.cpu().numpy()
            rec = raw[info["off_records"]:info["off_records"] + 16 * len(exp)].view(np.uint32).reshape(-1, 4)
            got = sorted((int(r[2]), int(r[3]), int(round(float(np.array([r[0]], np.uint32).view(np.float32)[0])))) for r in rec)
            assert got == sorted(exp)
        ctx.set_option("row_block", 0); ctx.set_option("compress", 1)


def test_odd_grid_size_and_small_grids(ctx):
    """Grid sizes that are odd, not a multiple of the support, or barely larger than the window."""
    rng = np.random.default_rng(77)
    for N, S, Q in ((255, 7, 8), (101, 8, 4), (12, 8, 8), (9, 4, 2)):
        cell = 0.05 / N
        du = 1.0 / 0.05
        n = 4000
        uvw = np.stack([rng.uniform(-0.55, 0.55, n) * N * du, rng.uniform(-0.55, 0.55, n) * N * du, rng.uniform(-30, 30, n)], 1)
        vis = (rng.standard_normal((n, 1)) + 1j * rng.standard_normal((n, 1))).astype(np.complex64)
        wt = np.ones((n, 1), np.float32)
        freq = np.array([synth.C0])
        st = owk.build_stack(3, 25.0, S, Q, N, cell)
        ref, rstats = ogrid.grid(uvw, vis, wt, freq, st)
        assert rstats["n_gridded"] > 100 and rstats["n_skipped_oob"] > 100
        wl = synth.Workload("odd%d" % N, uvw, freq, vis, wt, N, cell, 3, 25.0, S, Q)
        check_all_paths(ctx, wl, st, ref, rstats)


def test_sharded_gridding_one_rank_nccl(ctx):
    """paper_1905_03213_b200/sharded.py on the GPU with a one-rank NCCL group (the box has one GPU): the rank's shard
    is everything, the reduce is the identity; the multi-rank logic is covered on CPU (tests/test_sharded_gloo.py)."""
    import torch.distributed as dist
    from paper_1905_03213_b200 import sharded
    wl = synth.config2(nvis=2016 * 70 + 3)
    st = oracle_stack(wl)
    ref, rstats = ogrid.grid(wl.uvw, wl.vis, wl.weight, wl.freq, st, threads=4)
    ks = upload(ctx, st, wpgrid.F32)
    dist.init_process_group("nccl", init_method="tcp://127.0.0.1:%d" % (33000 + os.getpid() % 2000), rank=0, world_size=1,
                            device_id=torch.device("cuda", 0))
    try:
        g, s = sharded.grid_sharded(ctx, *dev(wl), ks, dist, rows="all", row_block=wl.notes["row_block"], stats=True)
        assert s == rstats and relerr(g.cpu().numpy(), ref) <= TOL[wpgrid.F32]
    finally:
        dist.destroy_process_group()
        ctx.set_option("row_block", 0)


def test_microbenchmarks_run_and_order_sensibly(ctx):
    """wpg_microbench (the machine limits bench.py reads its rooflines against): every pattern runs, rejects a bad
    selector, and the measured rates keep the order the hardware fixes — L1-resident loads beat L1-missing ones,
    packed fp32 FMAs beat fp64 FMAs, row-segment reductions beat scattered ones."""
    r = {w: ctx.microbench(w, 200, 32 << 20)[0] for w in range(10)}
    assert all(v > 0 for v in r.values())
    assert r[2] > 1.3 * r[9]                   # L1-resident vs L2-resident, L1-missing 16-byte loads
    assert r[3] * 2 > r[4]                     # f32x2 (two FMAs each) vs f64 FMAs
    assert r[0] > r[1]                         # a warp per row segment vs every lane its own cell
    assert r[8] > r[7]                         # plain tile updates vs shared-memory atomics
    with pytest.raises(wpgrid.WpgError):
        ctx.microbench(10, 10)
    with pytest.raises(wpgrid.WpgError):
        ctx.microbench(2, 10, 1 << 20)         # needs a 16 MiB buffer
