"""O4 — ctypes front end of grid_oracle.c (oracle, test infrastructure only).

The C file is compiled on first use with
``gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC`` (G6: no FMA contraction)
into ``oracle/libgridoracle.so`` (git-ignored build artefact).
``__graft_entry__.build()`` calls :func:`build` too.
"""
import ctypes
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "grid_oracle.c")
_LIB = os.path.join(_HERE, "libgridoracle.so")
_lib = None

STAT_NAMES = ("n_gridded", "n_skipped_oob", "n_skipped_zero_weight", "n_clamped_w", "n_updates")


def build(force=False):
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                               _SRC, "-o", tmp, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i64, dbl, cint = ctypes.c_int64, ctypes.c_double, ctypes.c_int
        vp = ctypes.c_void_p
        lib.oracle_index_map.argtypes = [dbl, cint, dbl, cint, cint,
                                         ctypes.POINTER(i64), ctypes.POINTER(cint)]
        lib.oracle_index_map.restype = None
        lib.oracle_plane.argtypes = [dbl, dbl, cint, ctypes.POINTER(cint)]
        lib.oracle_plane.restype = cint
        lib.oracle_grid.argtypes = [vp, vp, vp, vp, i64, cint, vp, vp, vp, cint, cint, cint,
                                    dbl, dbl, vp, vp, cint]
        lib.oracle_grid.restype = cint
        lib.oracle_degrid.argtypes = [vp, vp, i64, cint, vp, vp, vp, cint, cint, cint, dbl, dbl, vp, vp, vp]
        lib.oracle_degrid.restype = cint
        lib.oracle_flux.argtypes = [vp, vp, vp, vp, i64, cint, vp, vp, cint, cint, cint, dbl, dbl, vp, vp, cint]
        lib.oracle_flux.restype = cint
        lib.oracle_cells.argtypes = [vp, vp, vp, vp, i64, cint, vp, vp, vp, cint, cint, cint, dbl, dbl, vp, vp, cint, vp, vp, cint]
        lib.oracle_cells.restype = cint
        lib.oracle_max_threads.restype = cint
        _lib = lib
    return _lib


def max_threads():
    return int(_load().oracle_max_threads())


def index_map(x_lambda, N, cell, S, Q):
    """G3 for one axis: (j0, o)."""
    j0, o = ctypes.c_int64(), ctypes.c_int()
    _load().oracle_index_map(float(x_lambda), int(N), float(cell), int(S), int(Q),
                             ctypes.byref(j0), ctypes.byref(o))
    return int(j0.value), int(o.value)


def plane_of(w, w_max, Nw):
    """G2: (p, clamped)."""
    cl = ctypes.c_int()
    p = _load().oracle_plane(float(w), float(w_max), int(Nw), ctypes.byref(cl))
    return int(p), bool(cl.value)


def grid(uvw, vis, weight, freq, stack, grid=None, threads=1):
    """O4.  uvw [nrow][3] f64 metres, vis [nrow][nchan] c64, weight [nrow][nchan] f32,
    freq [nchan] f64 Hz, stack an oracle.wkernel.KernelStack.
    Returns (grid [N][N] complex128 — accumulated into `grid` if given, stats dict)."""
    uvw = np.ascontiguousarray(uvw, dtype=np.float64)
    vis = np.ascontiguousarray(vis, dtype=np.complex64)
    weight = np.ascontiguousarray(weight, dtype=np.float32)
    freq = np.ascontiguousarray(freq, dtype=np.float64)
    nrow = uvw.shape[0]
    nchan = freq.shape[0]
    vis = vis.reshape(nrow, nchan)
    weight = weight.reshape(nrow, nchan)
    N = stack.grid_N
    if grid is None:
        grid = np.zeros((N, N), dtype=np.complex128)
    assert grid.shape == (N, N) and grid.dtype == np.complex128 and grid.flags.c_contiguous
    K = np.ascontiguousarray(stack.data, dtype=np.complex128)
    sup = np.ascontiguousarray(stack.support, dtype=np.int32)
    off = np.ascontiguousarray(stack.plane_offset, dtype=np.int64)
    st = np.zeros(5, dtype=np.int64)
    rc = _load().oracle_grid(uvw.ctypes.data, vis.ctypes.data, weight.ctypes.data, freq.ctypes.data,
                             nrow, nchan, K.ctypes.data, sup.ctypes.data, off.ctypes.data,
                             stack.Nw, stack.oversample, N, stack.cell, stack.w_max,
                             grid.ctypes.data, st.ctypes.data, int(threads))
    if rc != 0:
        raise RuntimeError("oracle_grid failed rc=%d" % rc)
    return grid, dict(zip(STAT_NAMES, (int(x) for x in st)))


def degrid(uvw, freq, stack, grid):
    """Adjoint of :func:`grid` with unit weights (oracle_degrid in grid_oracle.c):
    vis[r][c] = sum over the window of grid * conj(K slice); 0 where the window leaves the grid.
    Returns (vis [nrow][nchan] complex128, {"n_predicted", "n_outside"})."""
    uvw = np.ascontiguousarray(uvw, dtype=np.float64)
    freq = np.ascontiguousarray(freq, dtype=np.float64)
    grid = np.ascontiguousarray(grid, dtype=np.complex128)
    nrow, nchan, N = uvw.shape[0], freq.shape[0], stack.grid_N
    assert grid.shape == (N, N)
    K = np.ascontiguousarray(stack.data, dtype=np.complex128)
    sup = np.ascontiguousarray(stack.support, dtype=np.int32)
    off = np.ascontiguousarray(stack.plane_offset, dtype=np.int64)
    out = np.zeros((nrow, nchan), dtype=np.complex128)
    cnt = np.zeros(2, dtype=np.int64)
    rc = _load().oracle_degrid(uvw.ctypes.data, freq.ctypes.data, nrow, nchan, K.ctypes.data, sup.ctypes.data,
                               off.ctypes.data, stack.Nw, stack.oversample, N, stack.cell, stack.w_max,
                               grid.ctypes.data, out.ctypes.data, cnt.ctypes.data)
    if rc != 0:
        raise RuntimeError("oracle_degrid failed rc=%d" % rc)
    return out, {"n_predicted": int(cnt[0]), "n_outside": int(cnt[1])}


def slice_moments(stack):
    """[Nw * Q * Q][3] complex128: (sigma, sigma_u, sigma_v) of every slice K[p][ov][ou] — its sum and its first
    moments over the window columns iu and rows iv (P11)."""
    Q = stack.oversample
    out = np.empty((stack.Nw * Q * Q, 3), dtype=np.complex128)
    for p in range(stack.Nw):
        Kp = stack.plane(p)                                  # [Q][Q][S][S]
        S = Kp.shape[-1]
        i = np.arange(S, dtype=np.float64)
        blk = out[p * Q * Q:(p + 1) * Q * Q].reshape(Q, Q, 3)
        blk[..., 0] = Kp.sum(axis=(2, 3))
        blk[..., 1] = (Kp * i[None, None, None, :]).sum(axis=(2, 3))
        blk[..., 2] = (Kp * i[None, None, :, None]).sum(axis=(2, 3))
    return out


def flux(uvw, vis, weight, freq, stack, threads=1):
    """P11 without a grid, O(nvis) (oracle_flux in grid_oracle.c): what sum(grid), sum(grid * ju) and sum(grid * jv)
    of the gridded result must be.  Returns ({"sum", "mom_u", "mom_v": complex, "l1": float}, stats dict)."""
    uvw = np.ascontiguousarray(uvw, dtype=np.float64)
    vis = np.ascontiguousarray(vis, dtype=np.complex64)
    weight = np.ascontiguousarray(weight, dtype=np.float32)
    freq = np.ascontiguousarray(freq, dtype=np.float64)
    nrow, nchan = uvw.shape[0], freq.shape[0]
    assert vis.size == nrow * nchan and weight.size == nrow * nchan
    sig = np.ascontiguousarray(slice_moments(stack))
    sup = np.ascontiguousarray(stack.support, dtype=np.int32)
    out = np.zeros(8, dtype=np.float64)
    st = np.zeros(5, dtype=np.int64)
    rc = _load().oracle_flux(uvw.ctypes.data, vis.ctypes.data, weight.ctypes.data, freq.ctypes.data, nrow, nchan,
                             sig.ctypes.data, sup.ctypes.data, stack.Nw, stack.oversample, stack.grid_N,
                             stack.cell, stack.w_max, out.ctypes.data, st.ctypes.data, int(threads))
    if rc != 0:
        raise RuntimeError("oracle_flux failed rc=%d" % rc)
    return ({"sum": complex(out[0], out[1]), "mom_u": complex(out[2], out[3]), "mom_v": complex(out[4], out[5]),
             "l1": float(out[6])}, dict(zip(STAT_NAMES, (int(x) for x in st))))


def cells(uvw, vis, weight, freq, stack, cu, cv, threads=1):
    """Gridded value of the single cells (cv[k], cu[k]), one by one (oracle_cells in grid_oracle.c: G5 read as a
    gather, every visibility tested against every requested cell) — what a full-size GPU run is checked against on
    sampled outputs.  Returns (values complex128 [ncell], l1 float64 [ncell] = sum |wt V| |K| per cell)."""
    uvw = np.ascontiguousarray(uvw, dtype=np.float64)
    vis = np.ascontiguousarray(vis, dtype=np.complex64)
    weight = np.ascontiguousarray(weight, dtype=np.float32)
    freq = np.ascontiguousarray(freq, dtype=np.float64)
    cu = np.ascontiguousarray(cu, dtype=np.int32)
    cv = np.ascontiguousarray(cv, dtype=np.int32)
    nrow, nchan = uvw.shape[0], freq.shape[0]
    assert vis.size == nrow * nchan and weight.size == nrow * nchan and cu.shape == cv.shape and cu.ndim == 1
    K = np.ascontiguousarray(stack.data, dtype=np.complex128)
    sup = np.ascontiguousarray(stack.support, dtype=np.int32)
    off = np.ascontiguousarray(stack.plane_offset, dtype=np.int64)
    out = np.zeros(cu.size, dtype=np.complex128)
    l1 = np.zeros(cu.size, dtype=np.float64)
    rc = _load().oracle_cells(uvw.ctypes.data, vis.ctypes.data, weight.ctypes.data, freq.ctypes.data, nrow, nchan,
                              K.ctypes.data, sup.ctypes.data, off.ctypes.data, stack.Nw, stack.oversample,
                              stack.grid_N, stack.cell, stack.w_max, cu.ctypes.data, cv.ctypes.data, int(cu.size),
                              out.ctypes.data, l1.ctypes.data, int(threads))
    if rc != 0:
        raise RuntimeError("oracle_cells failed rc=%d" % rc)
    return out, l1
