"""P2-P5, P8 — the W-kernel stack O3 pinned by two routes, symmetries, the w=0
special case, Poisson summation and stored values."""
import numpy as np
import pytest

from oracle import wkernel
from oracle.taper import psi


def test_k1_plane_centres():
    wp = wkernel.plane_centres(4, 100.0)
    assert np.allclose(wp, [-75, -25, 25, 75])
    assert np.allclose(wkernel.plane_centres(16, 200.0)[8], 12.5)


def test_k2_nk():
    assert [wkernel.nk_of(S) for S in (4, 7, 8, 9, 12, 16, 17, 32)] == [32, 32, 32, 64, 64, 64, 128, 128]


@pytest.mark.parametrize("S,Q,w,fov", [(7, 8, 37.5, 0.125), (8, 4, -80.0, 0.08), (4, 2, 75.0, 0.128)])
def test_p2_direct_sum_vs_padded_fft(S, Q, w, fov):
    """K3 by the written double sum (E F E^T) vs zero-pad + fftshift(fft2(ifftshift))."""
    F = wkernel.image_plane_samples(w, S, fov)
    Nk = F.shape[0]
    C = wkernel.uv_table(F, S, Q)
    big = np.zeros((Q * Nk, Q * Nk), complex)
    lo = Q * Nk // 2 - Nk // 2
    big[lo:lo + Nk, lo:lo + Nk] = F
    full = np.fft.fftshift(np.fft.fft2(np.fft.ifftshift(big)))
    t = np.arange(-S * Q // 2 + 1, S * Q // 2 + 1) + Q * Nk // 2
    ref = full[np.ix_(t, t)]
    assert np.max(np.abs(C - ref)) <= 1e-13 * np.max(np.abs(ref))


def test_k3_brute_force_double_sum_tiny():
    """The matmul form equals the literally written double sum at a few table points."""
    S, Q, fov, w = 4, 2, 0.128, 75.0
    F = wkernel.image_plane_samples(w, S, fov)
    Nk = F.shape[0]
    C = wkernel.uv_table(F, S, Q)
    for tv, tu in [(-3, -3), (0, 0), (4, -1), (2, 3)]:
        acc = 0j
        for b in range(Nk):
            for a in range(Nk):
                acc += F[b, a] * np.exp(-2j * np.pi * (tu * (a - Nk / 2) + tv * (b - Nk / 2)) / (Q * Nk))
        assert abs(C[tv + S * Q // 2 - 1, tu + S * Q // 2 - 1] - acc) <= 1e-12 * abs(acc)


def test_k4_slice_index():
    """t(i, o) = (i+1) Q - S Q/2 - o covers the table exactly."""
    S, Q = 7, 8
    C = np.arange((S * Q) ** 2).reshape(S * Q, S * Q).astype(complex)
    K = wkernel.slice_table(C, S, Q)
    assert K.shape == (Q, Q, S, S)
    for ov, ou, iv, iu in [(0, 0, 0, 0), (7, 7, 0, 0), (0, 0, 6, 6), (3, 5, 2, 4)]:
        tv = (iv + 1) * Q - S * Q // 2 - ov
        tu = (iu + 1) * Q - S * Q // 2 - ou
        assert K[ov, ou, iv, iu] == C[tv + S * Q // 2 - 1, tu + S * Q // 2 - 1]
    assert K[Q - 1, Q - 1, 0, 0] == C[0, 0] and K[0, 0, S - 1, S - 1] == C[-1, -1]


@pytest.fixture(scope="module")
def stack_cfg1():
    return wkernel.build_stack(16, 200.0, 7, 8, 256, 2.0 ** -11)


def test_p3_symmetries(stack_cfg1):
    K = stack_cfg1.as_array()
    Nw, Q, _, S, _ = K.shape
    assert np.max(np.abs(K[::-1] - np.conj(K))) <= 1e-15
    for o in range(1, Q):
        assert np.max(np.abs(K[:, o, o] - K[:, Q - o, Q - o, ::-1, ::-1])) <= 1e-15
    # o = 0: i <-> S-2-i (row/col S-1 has no partner)
    A = K[:, 0, 0, :S - 1, :S - 1]
    assert np.max(np.abs(A - A[:, ::-1, ::-1])) <= 1e-15


def test_p4_w0_is_real_and_separable():
    st = wkernel.build_stack(4, 0.0, 8, 8, 64, 0.08 / 64)
    K = st.as_array()
    assert np.max(np.abs(K.imag)) <= 1e-16
    assert np.max(np.abs(K - K[0])) == 0.0            # every plane is the same (w_p = 0)
    # ordinary 2-D PSWF gridding: K = k1[ov] (x) k1[ou], k1 = 1-D transform of psi
    S, Q, Nk = 8, 8, 32
    a = np.arange(Nk) - Nk // 2
    t = np.arange(-S * Q // 2 + 1, S * Q // 2 + 1)
    c1 = np.exp(-2j * np.pi * np.outer(t, a) / (Q * Nk)) @ psi(2.0 * a / Nk)
    i = np.arange(S)[None, :]; o = np.arange(Q)[:, None]
    k1 = c1[(i + 1) * Q - S * Q // 2 - o + S * Q // 2 - 1].real      # [o][i]
    sep = k1[:, None, :, None] * k1[None, :, None, :]
    sep /= sep[0, 0].sum()
    assert np.max(np.abs(K[0].real - sep)) <= 1e-14


def test_p5_slice_sums_near_one(stack_cfg1):
    K = stack_cfg1.as_array()
    sums = K.sum(axis=(3, 4))
    # deviation = energy thrown away by the S x S crop (cfg1 <= 8e-3)
    assert np.max(np.abs(sums - 1.0)) <= 8e-3
    assert abs(sums[8, 4, 4].real - 1.0) <= 1e-3
    st16 = wkernel.build_stack(2, 10.0, 16, 8, 64, 0.05 / 64)
    assert np.max(np.abs(st16.as_array().sum(axis=(3, 4)) - 1.0)) <= 5e-6   # SURVEY P5 quotes "<= 4e-6 (S=16)" for its own (unstated) parameters
    # K5: the on-cell w=0 slice sums to exactly 1 by construction
    s0 = wkernel.build_stack(1, 0.0, 7, 8, 256, 2.0 ** -11).as_array()
    assert abs(s0[0, 4, 4].sum() - 1.0) <= 1e-14


def test_p8_stored_values(golden, stack_cfg1):
    A = wkernel.build_stack(4, 100.0, 4, 2, 64, 0.002).as_array()
    B = stack_cfg1.as_array()
    for row in golden("p8_kernel_values.txt"):
        case = row[0]
        val = float(row[6]) + 1j * float(row[7])
        if case in ("A", "B"):
            p, ov, ou, iv, iu = (int(x) for x in row[1:6])
            got = (A if case == "A" else B)[p, ov, ou, iv, iu]
        elif case == "A_sum":
            got = A[0, 0, 0].sum()
        elif case == "B_maxabs":
            got = np.max(np.abs(B))
        assert abs(got - val) <= 2e-14, (row, got)


def test_k6_ragged_support_and_layout():
    N, cell, Nw, w_max = 8192, 1.0e-5, 128, 5.0e3
    sup = wkernel.ragged_support(Nw, w_max, N, cell, 8, 32)
    assert sup.min() == 8 and sup.max() == 32 and np.all(sup % 2 == 0)
    assert np.all(sup == sup[::-1])                        # |w_p| symmetric
    # hand value: plane 0, |w_p| = 5000 - 39.0625, FoV = 0.08192
    wp0 = 5000.0 - 5000.0 / 128
    s0 = 2 * np.ceil(np.sqrt(9.0 + (wp0 * 0.08192 ** 2 / 2) ** 2))
    assert sup[0] == min(32, s0)
    st = wkernel.build_stack(4, 3000.0, wkernel.ragged_support(4, 3000.0, 512, 0.08192 / 512, 8, 32),
                             2, 512, 0.08192 / 512)
    assert not st.uniform
    assert np.all(np.diff(st.plane_offset) == 4 * st.support.astype(np.int64) ** 2)
    # a ragged plane equals the same plane of a uniform stack up to the common scalar s (K5 uses S_min)
    p = 0
    S = int(st.support[p])
    uni = wkernel.build_stack(4, 3000.0, S, 2, 512, 0.08192 / 512)
    ratio = st.plane(p) / uni.plane(p)
    assert np.max(np.abs(ratio - ratio.flat[0])) <= 1e-12
