"""Thin ctypes binding over libwpgrid.so (include/wpgrid.h) — argument marshalling only.

Every step of the path runs inside the library's CUDA kernels; torch is used for device
memory and the stream.  There is no fallback: if the library is missing, or no CUDA device
is present, the calls raise.
"""
import ctypes
import os
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("WPGRID_LIB") or os.path.join(_HERE, "libwpgrid.so")   # override: an alternative build

F32, F64 = 0, 1
OK, EINVAL, ENOMEM, ECUDA = 0, -1, -2, -3

EXPORTS = (
    "wpg_create", "wpg_destroy", "wpg_last_error", "wpg_version", "wpg_set_option", "wpg_taper",
    "wpg_ragged_support", "wpg_wkernel_elems", "wpg_wkernel_workspace_bytes", "wpg_wkernel_build", "wpg_grid_workspace_bytes",
    "wpg_grid", "wpg_grid_naive", "wpg_grid_host", "wpg_bin", "wpg_dirty_image_workspace_bytes",
    "wpg_dirty_image", "wpg_launch_count", "wpg_phase_ms", "wpg_microbench",
    "wpg_baseline_workspace_bytes", "wpg_baseline_reorder", "wpg_grid_baseline_order",
    "wpg_degrid_workspace_bytes", "wpg_degrid", "wpg_grid_pol_workspace_bytes", "wpg_grid_pol", "wpg_shard_rows",
    "wpg_static_scratch_bytes", "wpg_grid_static",
)


class WpgError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("libwpgrid error %d: %s" % (code, text))
        self.code = code


class KDesc(ctypes.Structure):
    _fields_ = [("Nw", ctypes.c_int), ("oversample", ctypes.c_int), ("grid_N", ctypes.c_int),
                ("w_max", ctypes.c_double), ("cell", ctypes.c_double), ("support_max", ctypes.c_int),
                ("support", ctypes.POINTER(ctypes.c_int)), ("plane_offset", ctypes.POINTER(ctypes.c_int64))]


class Stats(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int64) for n in
                ("n_gridded", "n_skipped_oob", "n_skipped_zero_weight", "n_clamped_w", "n_updates")]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


class BinInfo(ctypes.Structure):
    _fields_ = [("n_records", ctypes.c_int64), ("n_keys", ctypes.c_int64), ("n_classes", ctypes.c_int32),
                ("key_shift", ctypes.c_int32), ("record_bytes", ctypes.c_int32), ("keys_per_class", ctypes.c_int32),
                ("off_records", ctypes.c_int64), ("off_bucket_start", ctypes.c_int64)]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


_lib = None


def load():
    """Load libwpgrid.so (fails loudly if it has not been built)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("%s not found: build it with `python -m paper_1905_03213_b200.build` "
                          "(there is no CPU fallback)" % LIB_PATH)
    lib = ctypes.CDLL(LIB_PATH)
    vp, i64, cint, dbl, sz = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
    kd, stp = ctypes.POINTER(KDesc), ctypes.POINTER(Stats)
    lib.wpg_create.argtypes = [ctypes.POINTER(vp), cint, vp]; lib.wpg_create.restype = cint
    lib.wpg_destroy.argtypes = [vp]; lib.wpg_destroy.restype = None
    lib.wpg_last_error.argtypes = [vp]; lib.wpg_last_error.restype = ctypes.c_char_p
    lib.wpg_version.argtypes = []; lib.wpg_version.restype = cint
    lib.wpg_set_option.argtypes = [vp, ctypes.c_char_p, i64]; lib.wpg_set_option.restype = cint
    lib.wpg_taper.argtypes = [vp, i64, vp]; lib.wpg_taper.restype = cint
    lib.wpg_ragged_support.argtypes = [cint, dbl, cint, dbl, cint, cint, cint, vp, vp]
    lib.wpg_ragged_support.restype = cint
    lib.wpg_wkernel_elems.argtypes = [cint, cint, cint]; lib.wpg_wkernel_elems.restype = i64
    lib.wpg_wkernel_workspace_bytes.argtypes = [kd]; lib.wpg_wkernel_workspace_bytes.restype = sz
    lib.wpg_wkernel_build.argtypes = [vp, kd, cint, vp, vp, sz]; lib.wpg_wkernel_build.restype = cint
    lib.wpg_grid_workspace_bytes.argtypes = [vp, i64, cint, kd, cint]; lib.wpg_grid_workspace_bytes.restype = sz
    lib.wpg_grid.argtypes = [vp, vp, vp, vp, vp, i64, cint, vp, kd, cint, vp, vp, sz, stp]
    lib.wpg_grid.restype = cint
    lib.wpg_static_scratch_bytes.argtypes = []; lib.wpg_static_scratch_bytes.restype = sz
    lib.wpg_grid_static.argtypes = [vp, vp, vp, vp, vp, i64, cint, vp, kd, cint, vp, stp]
    lib.wpg_grid_static.restype = cint
    lib.wpg_grid_naive.argtypes = [vp, vp, vp, vp, vp, i64, cint, vp, kd, cint, vp, stp]
    lib.wpg_grid_naive.restype = cint
    lib.wpg_grid_host.argtypes = [vp, vp, vp, vp, vp, i64, cint, vp, kd, cint, vp, stp, vp, dbl]
    lib.wpg_grid_host.restype = cint
    lib.wpg_bin.argtypes = [vp, vp, vp, vp, vp, i64, cint, kd, cint, vp, sz, ctypes.POINTER(BinInfo), stp]
    lib.wpg_bin.restype = cint
    lib.wpg_dirty_image_workspace_bytes.argtypes = [cint, cint]; lib.wpg_dirty_image_workspace_bytes.restype = sz
    lib.wpg_dirty_image.argtypes = [vp, vp, kd, dbl, cint, vp, vp, sz]; lib.wpg_dirty_image.restype = cint
    lib.wpg_launch_count.argtypes = [vp]; lib.wpg_launch_count.restype = i64
    lib.wpg_phase_ms.argtypes = [vp, ctypes.POINTER(dbl)]; lib.wpg_phase_ms.restype = cint
    lib.wpg_baseline_workspace_bytes.argtypes = [i64, cint, cint, cint]; lib.wpg_baseline_workspace_bytes.restype = sz
    lib.wpg_baseline_reorder.argtypes = [vp, vp, vp, cint, i64, vp, vp, vp, sz]; lib.wpg_baseline_reorder.restype = cint
    lib.wpg_grid_baseline_order.argtypes = [vp, vp, vp, vp, vp, vp, vp, cint, i64, cint, vp, kd, cint, vp, vp, sz, stp]
    lib.wpg_grid_baseline_order.restype = cint
    lib.wpg_degrid_workspace_bytes.argtypes = [cint]; lib.wpg_degrid_workspace_bytes.restype = sz
    lib.wpg_degrid.argtypes = [vp, vp, vp, vp, i64, cint, vp, kd, cint, vp, vp, sz, ctypes.POINTER(i64)]
    lib.wpg_degrid.restype = cint
    lib.wpg_grid_pol_workspace_bytes.argtypes = [vp, i64, cint, cint, kd, cint]; lib.wpg_grid_pol_workspace_bytes.restype = sz
    lib.wpg_grid_pol.argtypes = [vp, vp, vp, vp, vp, i64, cint, cint, vp, kd, cint, vp, vp, sz, stp]; lib.wpg_grid_pol.restype = cint
    lib.wpg_microbench.argtypes = [vp, cint, cint, vp, sz, ctypes.POINTER(dbl)]; lib.wpg_microbench.restype = cint
    lib.wpg_shard_rows.argtypes = [i64, i64, cint, cint, ctypes.POINTER(i64), ctypes.POINTER(i64)]; lib.wpg_shard_rows.restype = cint
    _lib = lib
    return lib


def taper(nu):
    """psi(nu), the library's own evaluation (host)."""
    nu = np.ascontiguousarray(nu, dtype=np.float64)
    out = np.empty_like(nu)
    rc = load().wpg_taper(nu.ctypes.data, nu.size, out.ctypes.data)
    if rc:
        raise WpgError(rc, "wpg_taper")
    return out


def ragged_support(Nw, w_max, grid_N, cell, oversample, S_min, S_max):
    sup = np.zeros(Nw, dtype=np.int32)
    off = np.zeros(Nw + 1, dtype=np.int64)
    rc = load().wpg_ragged_support(Nw, w_max, grid_N, cell, oversample, S_min, S_max,
                                   sup.ctypes.data, off.ctypes.data)
    if rc:
        raise WpgError(rc, "wpg_ragged_support: bad argument")
    return sup, off


@dataclass
class Stack:
    """A kernel stack on the device plus its descriptor (keeps the host arrays alive)."""
    data: object            # torch tensor, complex64 | complex128, flat
    desc: KDesc
    prec: int
    support: np.ndarray     # [Nw] int32
    plane_offset: np.ndarray  # [Nw+1] int64
    uniform: bool


def make_desc(Nw, w_max, support, oversample, grid_N, cell):
    """support: int (uniform) or int array [Nw] (ragged).  Returns (KDesc, support, plane_offset)."""
    Q = int(oversample)
    if np.isscalar(support):
        sup = np.full(Nw, int(support), dtype=np.int32)
        uniform = True
    else:
        sup = np.ascontiguousarray(support, dtype=np.int32)
        uniform = False
    off = np.zeros(Nw + 1, dtype=np.int64)
    off[1:] = np.cumsum(Q * Q * sup.astype(np.int64) ** 2)
    d = KDesc()
    d.Nw, d.oversample, d.grid_N, d.w_max, d.cell = int(Nw), Q, int(grid_N), float(w_max), float(cell)
    d.support_max = int(sup.max()) if Nw > 0 else 0
    if uniform:
        d.support = None
        d.plane_offset = None
    else:
        d.support = sup.ctypes.data_as(ctypes.POINTER(ctypes.c_int))
        d.plane_offset = off.ctypes.data_as(ctypes.POINTER(ctypes.c_int64))
    return d, sup, off, uniform


class Context:
    """wpg_ctx bound to a torch CUDA device and stream."""

    def __init__(self, device=0, stream=None):
        import torch
        self.torch = torch
        self.lib = load()
        if not torch.cuda.is_available():
            raise WpgError(ECUDA, "no CUDA device; libwpgrid has no CPU fallback")
        self.device = torch.device("cuda", device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = ctypes.c_void_p()
        rc = self.lib.wpg_create(ctypes.byref(h), device, ctypes.c_void_p(self.stream.cuda_stream))
        if rc:
            raise WpgError(rc, self.lib.wpg_last_error(None).decode())
        self.h = h

    def close(self):
        if getattr(self, "h", None):
            self.lib.wpg_destroy(self.h)
            self.h = None

    __del__ = close

    def _check(self, rc):
        if rc:
            raise WpgError(rc, self.lib.wpg_last_error(self.h).decode())

    def set_option(self, name, value):
        self._check(self.lib.wpg_set_option(self.h, name.encode(), int(value)))

    def launch_count(self):
        return int(self.lib.wpg_launch_count(self.h))

    def phase_ms(self):
        """(binning ms, gridder ms) of the last wpg_grid call made with option "timing" = 1."""
        out = (ctypes.c_double * 2)()
        self._check(self.lib.wpg_phase_ms(self.h, out))
        return float(out[0]), float(out[1])

    def microbench(self, which, iters=2000, buf_bytes=1 << 25):
        """(operations/s, ms) of machine-limit microbenchmark `which` (see wpg_microbench in wpgrid.h)."""
        t = self.torch
        buf = t.zeros(buf_bytes, dtype=t.uint8, device=self.device)
        out = (ctypes.c_double * 2)()
        self._check(self.lib.wpg_microbench(self.h, int(which), int(iters), buf.data_ptr(), buf.numel(), out))
        return float(out[0]), float(out[1])

    # ---- a0
    def wkernel_build(self, Nw, w_max, support, oversample, grid_N, cell, prec=F32):
        t = self.torch
        d, sup, off, uniform = make_desc(Nw, w_max, support, oversample, grid_N, cell)
        K = t.empty(int(off[-1]), dtype=t.complex64 if prec == F32 else t.complex128, device=self.device)
        need = int(self.lib.wpg_wkernel_workspace_bytes(ctypes.byref(d)))
        if need == 0:
            raise WpgError(EINVAL, "wpg_wkernel_workspace_bytes: bad kernel descriptor")
        ws = self._temp(need)
        self._check(self.lib.wpg_wkernel_build(self.h, ctypes.byref(d), prec, K.data_ptr(), ws.data_ptr(), ws.numel()))
        return Stack(K, d, prec, sup, off, uniform)

    def stack_from_host(self, data, Nw, w_max, support, oversample, grid_N, cell, prec=F32):
        """Upload a stack computed elsewhere (tests feed the oracle's stack to the gridder)."""
        t = self.torch
        d, sup, off, uniform = make_desc(Nw, w_max, support, oversample, grid_N, cell)
        arr = np.ascontiguousarray(data, dtype=np.complex64 if prec == F32 else np.complex128).ravel()
        assert arr.size == off[-1]
        return Stack(t.from_numpy(arr).to(self.device), d, prec, sup, off, uniform)

    # ---- a1 + a2
    def grid_workspace_bytes(self, nrow, nchan, stack):
        n = self.lib.wpg_grid_workspace_bytes(self.h, nrow, nchan, ctypes.byref(stack.desc), stack.prec)
        if n == 0:
            raise WpgError(EINVAL, "wpg_grid_workspace_bytes: bad arguments")
        return int(n)

    def _inputs(self, vis, uvw, weight, freq):
        t = self.torch
        assert vis.dtype == t.complex64 and uvw.dtype == t.float64 and weight.dtype == t.float32 \
            and freq.dtype == t.float64
        for x in (vis, uvw, weight, freq):
            assert x.is_cuda and x.is_contiguous()
        nrow, nchan = uvw.shape[0], freq.shape[0]
        assert vis.numel() == nrow * nchan and weight.numel() == nrow * nchan and uvw.shape[1] == 3
        return nrow, nchan

    def _check_grid(self, grid, stack, lead=()):
        """A caller-supplied grid goes to the C ABI as a raw pointer: refuse anything but a contiguous device
        tensor of the stack's precision and shape."""
        t = self.torch
        N = stack.desc.grid_N
        want = t.complex64 if stack.prec == F32 else t.complex128
        if not (grid.is_cuda and grid.device == self.device and grid.is_contiguous()
                and grid.dtype == want and tuple(grid.shape) == tuple(lead) + (N, N)):
            raise WpgError(EINVAL, "grid must be a contiguous %s tensor of shape %s on %s (got %s %s on %s)"
                           % (want, tuple(lead) + (N, N), self.device, grid.dtype, tuple(grid.shape), grid.device))

    def _temp(self, nbytes):
        """Temporary workspace, allocated on the context's stream (torch's caching allocator ties a block to the
        stream it was allocated on: a block from another stream could be handed out again while the library's
        kernels are still queued)."""
        t = self.torch
        with t.cuda.stream(self.stream):
            return t.empty(int(nbytes), dtype=t.uint8, device=self.device)

    def new_grid(self, stack):
        t = self.torch
        N = stack.desc.grid_N
        return t.zeros((N, N), dtype=t.complex64 if stack.prec == F32 else t.complex128, device=self.device)

    def grid(self, vis, uvw, weight, freq, stack, grid=None, workspace=None, stats=False):
        """grid += gridding(vis).  Returns (grid, stats dict or None)."""
        t = self.torch
        nrow, nchan = self._inputs(vis, uvw, weight, freq)
        if grid is None:
            grid = self.new_grid(stack)
        self._check_grid(grid, stack)
        if workspace is None:
            workspace = self._temp(self.grid_workspace_bytes(nrow, nchan, stack))
        st = Stats()
        self._check(self.lib.wpg_grid(self.h, vis.data_ptr(), uvw.data_ptr(), weight.data_ptr(), freq.data_ptr(),
                                      nrow, nchan, stack.data.data_ptr(), ctypes.byref(stack.desc), stack.prec,
                                      grid.data_ptr(), workspace.data_ptr(), workspace.numel(),
                                      ctypes.byref(st) if stats else None))
        return grid, (st.as_dict() if stats else None)

    def grid_static(self, vis, uvw, weight, freq, stack, grid, stats=False):
        """grid += gridding(vis) through wpg_grid_static: no workspace argument and no device allocation — the scratch
        is the library's static device array (static_scratch_bytes(); larger problems raise WpgError ENOMEM).  The
        caller supplies the grid.  Calls on one device share the array: do not overlap them on the GPU."""
        nrow, nchan = self._inputs(vis, uvw, weight, freq)
        self._check_grid(grid, stack)
        st = Stats()
        self._check(self.lib.wpg_grid_static(self.h, vis.data_ptr(), uvw.data_ptr(), weight.data_ptr(), freq.data_ptr(),
                                             nrow, nchan, stack.data.data_ptr(), ctypes.byref(stack.desc), stack.prec,
                                             grid.data_ptr(), ctypes.byref(st) if stats else None))
        return grid, (st.as_dict() if stats else None)

    def static_scratch_bytes(self):
        return int(self.lib.wpg_static_scratch_bytes())

    def grid_naive(self, vis, uvw, weight, freq, stack, grid=None, stats=False):
        nrow, nchan = self._inputs(vis, uvw, weight, freq)
        if grid is None:
            grid = self.new_grid(stack)
        self._check_grid(grid, stack)
        st = Stats()
        self._check(self.lib.wpg_grid_naive(self.h, vis.data_ptr(), uvw.data_ptr(), weight.data_ptr(),
                                            freq.data_ptr(), nrow, nchan, stack.data.data_ptr(),
                                            ctypes.byref(stack.desc), stack.prec, grid.data_ptr(),
                                            ctypes.byref(st) if stats else None))
        return grid, (st.as_dict() if stats else None)

    def grid_host(self, vis, uvw, weight, freq, stack, out=None, stats=False, image_out=None, weight_sum=0.0):
        """Host numpy (or pinned torch CPU) inputs -> host grid (and, if image_out is given, the
        dirty image); H2D/D2H copies happen inside the call."""
        def ptr(x):
            return x.data_ptr() if hasattr(x, "data_ptr") else x.ctypes.data
        nrow, nchan = int(uvw.shape[0]), int(freq.shape[0])
        N = stack.desc.grid_N
        cdt = np.complex64 if stack.prec == F32 else np.complex128
        if out is None:
            out = np.empty((N, N), dtype=cdt)

        def host_ok(x, dtype, size):
            """C-contiguous host array (numpy or CPU torch) of the given element type and size"""
            if hasattr(x, "data_ptr"):
                return (not x.is_cuda) and x.is_contiguous() and x.numel() == size and \
                    np.dtype(str(x.dtype).replace("torch.", "")) == np.dtype(dtype)
            return isinstance(x, np.ndarray) and x.flags.c_contiguous and x.size == size and x.dtype == np.dtype(dtype)

        checks = [(vis, np.complex64, nrow * nchan, "vis"), (uvw, np.float64, nrow * 3, "uvw"),
                  (weight, np.float32, nrow * nchan, "weight"), (freq, np.float64, nchan, "freq"), (out, cdt, N * N, "out")]
        if image_out is not None:
            checks.append((image_out, np.float32 if stack.prec == F32 else np.float64, N * N, "image_out"))
        for x, dtype, size, name in checks:
            if not host_ok(x, dtype, size):
                raise WpgError(EINVAL, "grid_host: %s must be a C-contiguous host array of %d %s elements"
                               % (name, size, np.dtype(dtype).name))
        st = Stats()
        self._check(self.lib.wpg_grid_host(self.h, ptr(vis), ptr(uvw), ptr(weight), ptr(freq), nrow, nchan,
                                           stack.data.data_ptr(), ctypes.byref(stack.desc), stack.prec,
                                           ptr(out), ctypes.byref(st) if stats else None,
                                           ptr(image_out) if image_out is not None else None, float(weight_sum)))
        return out, (st.as_dict() if stats else None)

    # ---- the paper's baseline-then-time order (Eqs. 1-2)
    def baseline_reorder(self, ant1, ant2, n_ant):
        """(B_start_index [nb + 1], perm [nrow]) as torch int32-sized unsigned tensors (values < 2^31 here)."""
        t = self.torch
        assert ant1.dtype == t.int32 and ant2.dtype == t.int32 and ant1.is_cuda and ant2.is_cuda
        nrow = ant1.numel()
        nb = n_ant * (n_ant + 1) // 2
        bstart = t.empty(nb + 1, dtype=t.int32, device=self.device)
        perm = t.empty(max(nrow, 1), dtype=t.int32, device=self.device)
        need = int(self.lib.wpg_baseline_workspace_bytes(nrow, 1, n_ant, F32))
        ws = self._temp(need)
        self._check(self.lib.wpg_baseline_reorder(self.h, ant1.data_ptr(), ant2.data_ptr(), n_ant, nrow,
                                                  bstart.data_ptr(), perm.data_ptr(), ws.data_ptr(), ws.numel()))
        return bstart, perm[:nrow]

    def grid_baseline_order(self, vis, uvw, weight, freq, ant1, ant2, n_ant, stack, grid=None, workspace=None, stats=False):
        """grid += gridding(vis) with the records in the paper's baseline-then-time order."""
        t = self.torch
        nrow, nchan = self._inputs(vis, uvw, weight, freq)
        assert ant1.dtype == t.int32 and ant2.dtype == t.int32 and ant1.numel() == nrow and ant2.numel() == nrow
        if grid is None:
            grid = self.new_grid(stack)
        self._check_grid(grid, stack)
        if workspace is None:
            workspace = self._temp(self.lib.wpg_baseline_workspace_bytes(nrow, nchan, n_ant, stack.prec))
        st = Stats()
        self._check(self.lib.wpg_grid_baseline_order(
            self.h, vis.data_ptr(), uvw.data_ptr(), weight.data_ptr(), freq.data_ptr(), ant1.data_ptr(), ant2.data_ptr(),
            n_ant, nrow, nchan, stack.data.data_ptr(), ctypes.byref(stack.desc), stack.prec, grid.data_ptr(),
            workspace.data_ptr(), workspace.numel(), ctypes.byref(st) if stats else None))
        return grid, (st.as_dict() if stats else None)

    # ---- polarisation axis
    def grid_pol(self, vis, uvw, weight, freq, stack, grid=None, workspace=None, stats=False):
        """vis [nrow][nchan][npol] complex64 -> grid [npol][N][N] (accumulated into), in the stack's precision."""
        t = self.torch
        assert vis.dtype == t.complex64 and vis.dim() == 3 and vis.is_cuda and vis.is_contiguous()
        nrow, nchan, npol = vis.shape
        assert uvw.shape == (nrow, 3) and weight.numel() == nrow * nchan and freq.shape[0] == nchan
        N = stack.desc.grid_N
        if grid is None:
            grid = t.zeros((npol, N, N), dtype=t.complex64 if stack.prec == F32 else t.complex128, device=self.device)
        self._check_grid(grid, stack, lead=(npol,))
        if workspace is None:
            need = int(self.lib.wpg_grid_pol_workspace_bytes(self.h, nrow, nchan, npol, ctypes.byref(stack.desc), stack.prec))
            if need == 0:
                raise WpgError(EINVAL, "wpg_grid_pol_workspace_bytes: bad arguments (npol must be 2 or 4)")
            workspace = self._temp(need)
        st = Stats()
        self._check(self.lib.wpg_grid_pol(self.h, vis.data_ptr(), uvw.data_ptr(), weight.data_ptr(), freq.data_ptr(),
                                          nrow, nchan, npol, stack.data.data_ptr(), ctypes.byref(stack.desc), stack.prec,
                                          grid.data_ptr(), workspace.data_ptr(), workspace.numel(),
                                          ctypes.byref(st) if stats else None))
        return grid, (st.as_dict() if stats else None)

    # ---- degridding (adjoint of grid with unit weights)
    def degrid(self, grid, uvw, freq, stack, out=None, counts=False):
        """vis[r][c] = sum over the window of grid * conj(kernel slice).  Returns (vis, counts dict or None)."""
        t = self.torch
        N = stack.desc.grid_N
        cdt = t.complex64 if stack.prec == F32 else t.complex128
        assert grid.is_cuda and grid.is_contiguous() and grid.shape == (N, N) and grid.dtype == cdt
        assert uvw.dtype == t.float64 and freq.dtype == t.float64 and uvw.is_cuda and freq.is_cuda
        nrow, nchan = uvw.shape[0], freq.shape[0]
        if out is None:
            out = t.empty((nrow, nchan), dtype=cdt, device=self.device)
        ws = self._temp(self.lib.wpg_degrid_workspace_bytes(nchan))
        c2 = (ctypes.c_int64 * 2)()
        self._check(self.lib.wpg_degrid(self.h, grid.data_ptr(), uvw.data_ptr(), freq.data_ptr(), nrow, nchan,
                                        stack.data.data_ptr(), ctypes.byref(stack.desc), stack.prec, out.data_ptr(),
                                        ws.data_ptr(), ws.numel(), c2 if counts else None))
        return out, ({"n_predicted": int(c2[0]), "n_outside": int(c2[1])} if counts else None)

    def bin(self, vis, uvw, weight, freq, stack, workspace=None):
        """Step a1 alone.  Returns (workspace tensor, BinInfo dict, stats dict)."""
        t = self.torch
        nrow, nchan = self._inputs(vis, uvw, weight, freq)
        if workspace is None:
            workspace = self._temp(self.grid_workspace_bytes(nrow, nchan, stack))
        info, st = BinInfo(), Stats()
        self._check(self.lib.wpg_bin(self.h, vis.data_ptr(), uvw.data_ptr(), weight.data_ptr(), freq.data_ptr(),
                                     nrow, nchan, ctypes.byref(stack.desc), stack.prec, workspace.data_ptr(),
                                     workspace.numel(), ctypes.byref(info), ctypes.byref(st)))
        return workspace, info.as_dict(), st.as_dict()

    # ---- a3
    def dirty_image(self, grid, stack, weight_sum, workspace=None):
        t = self.torch
        N = stack.desc.grid_N
        assert grid.is_cuda and grid.is_contiguous() and grid.shape == (N, N)
        need = int(self.lib.wpg_dirty_image_workspace_bytes(N, stack.prec))
        if workspace is None:
            workspace = self._temp(need)
        img = t.empty((N, N), dtype=t.float32 if stack.prec == F32 else t.float64, device=self.device)
        self._check(self.lib.wpg_dirty_image(self.h, grid.data_ptr(), ctypes.byref(stack.desc), float(weight_sum),
                                             stack.prec, img.data_ptr(), workspace.data_ptr(), workspace.numel()))
        return img
