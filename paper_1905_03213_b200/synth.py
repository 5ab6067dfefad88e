"""Seeded synthetic workloads (the five BASELINE.json configs) — input generators only.

This module serves both the oracle (tests, cpu_baseline) and the CUDA path
with the SAME arrays.  It holds none of the method's arithmetic: no index
mapping, no kernels, no gridding — only array layouts, the interferometer
measurement equation that defines the inputs and noise.
It imports neither ``oracle`` nor the CUDA binding.

The paper measures on the JVLA G55.7+3.4 Measurement Set, which
is not available; these inputs stand in for it (recipe: SURVEY.md §8(d),
restated in DESIGN.md).  RNG: numpy PCG64, seed 1905032130 + config number.
"""
from dataclasses import dataclass, field
import math
import numpy as np

C0 = 299792458.0
SEED0 = 1905032130
SIDEREAL_DAY_S = 86164.0905
LAT_DEG = -26.7
DEC_DEG = -30.0


@dataclass
class Workload:
    name: str
    uvw: np.ndarray        # [nrow][3] float64, metres
    freq: np.ndarray       # [nchan] float64, Hz
    vis: np.ndarray        # [nrow][nchan] complex64
    weight: np.ndarray     # [nrow][nchan] float32
    grid_N: int
    cell: float            # rad
    Nw: int
    w_max: float           # wavelengths
    support: object        # int (uniform) or ("ragged", S_min, S_max): each side applies rule K6 itself
    oversample: int
    sources: dict = field(default_factory=dict)   # flux, l, m
    notes: dict = field(default_factory=dict)     # e.g. row_block: rows per time step (rows are dump-major)

    @property
    def nvis(self):
        return self.vis.shape[0] * self.vis.shape[1]

    @property
    def fov(self):
        return self.grid_N * self.cell

    def uvw_lambda(self):
        """[nrow][nchan][3] in wavelengths (for the DFT pin and diagnostics)."""
        return self.uvw[:, None, :] * (self.freq / C0)[None, :, None]


# --------------------------------------------------------------------------- O1
def predict_vis(u, v, w, flux, l, m, chunk=1 << 20, device=None):
    """Measurement model O1: V = sum_s S_s exp(-2 pi i [u l_s + v m_s + w (n_s - 1)]).

    u, v, w: wavelengths, any shape; returns complex128 of that shape.
    `device`: optional torch device for the bulk (fp64 either way)."""
    shape = np.shape(u)
    u = np.ravel(u); v = np.ravel(v); w = np.ravel(w)
    flux = np.asarray(flux, np.float64); l = np.asarray(l, np.float64); m = np.asarray(m, np.float64)
    r2 = l * l + m * m
    nm1 = -r2 / (1.0 + np.sqrt(1.0 - r2))
    out = np.empty(u.size, dtype=np.complex128)
    if device is None:
        for i0 in range(0, u.size, chunk):
            s = slice(i0, i0 + chunk)
            ph = np.outer(u[s], l) + np.outer(v[s], m) + np.outer(w[s], nm1)
            out[s] = np.exp(-2j * np.pi * ph) @ flux
    else:
        import torch
        tl = torch.as_tensor(l, device=device); tm = torch.as_tensor(m, device=device)
        tn = torch.as_tensor(nm1, device=device); tf = torch.as_tensor(flux, device=device)
        for i0 in range(0, u.size, chunk):
            s = slice(i0, i0 + chunk)
            tu = torch.as_tensor(u[s], device=device); tv = torch.as_tensor(v[s], device=device)
            tw = torch.as_tensor(w[s], device=device)
            ph = torch.outer(tu, tl) + torch.outer(tv, tm) + torch.outer(tw, tn)
            ang = (-2.0 * math.pi) * ph
            re = torch.cos(ang) @ tf
            im = torch.sin(ang) @ tf
            out[s] = (re + 1j * im).cpu().numpy()
    return out.reshape(shape)


def _sources(rng, n, half_width):
    flux = rng.uniform(0.1, 1.0, n)
    l = rng.uniform(-half_width, half_width, n)
    m = rng.uniform(-half_width, half_width, n)
    return dict(flux=flux, l=l, m=m)


def _noise(rng, shape, sigma=0.1):
    # "N(0, 0.01)": variance 0.01 => sigma 0.1 on each of re and im (reading R16)
    return rng.normal(0.0, sigma, shape) + 1j * rng.normal(0.0, sigma, shape)


# ------------------------------------------------------------ earth rotation
def earth_rotation_uvw(E, N, n_dump, dt=10.0, dec_deg=DEC_DEG, lat_deg=LAT_DEG, max_rows=None):
    """uvw [n_dump * n_bl][3] metres, rows dump-major then baseline (i < j)."""
    phi = math.radians(lat_deg); dec = math.radians(dec_deg)
    X = -N * math.sin(phi); Y = E.copy(); Z = N * math.cos(phi)
    i, j = np.triu_indices(E.size, k=1)
    Lx = X[j] - X[i]; Ly = Y[j] - Y[i]; Lz = Z[j] - Z[i]
    n_bl = Lx.size
    if max_rows is not None:
        n_dump_eff = min(n_dump, -(-max_rows // n_bl))
    else:
        n_dump_eff = n_dump
    d = np.arange(n_dump_eff)
    # the track is centred on transit for the FULL n_dump; a truncated run keeps its first dumps
    H = (d + 0.5 - n_dump / 2.0) * dt * 2.0 * math.pi / SIDEREAL_DAY_S
    sH = np.sin(H)[:, None]; cH = np.cos(H)[:, None]
    sd, cd = math.sin(dec), math.cos(dec)
    out = np.empty((n_dump_eff, n_bl, 3), dtype=np.float64)
    out[:, :, 0] = sH * Lx + cH * Ly
    out[:, :, 1] = -sd * cH * Lx + sd * sH * Ly + cd * Lz
    out[:, :, 2] = cd * cH * Lx - cd * sH * Ly + sd * Lz
    out = out.reshape(-1, 3)
    if max_rows is not None:
        out = out[:max_rows]
    return np.ascontiguousarray(out)


def track_antennas(n_ant, nrow):
    """Antenna IDs (int32) of the rows earth_rotation_uvw produces: dump-major, baselines (i < j) in
    np.triu_indices order within a dump."""
    i, j = np.triu_indices(n_ant, k=1)
    reps = -(-nrow // i.size)
    return (np.tile(i, reps)[:nrow].astype(np.int32), np.tile(j, reps)[:nrow].astype(np.int32))


def _disc_layout(rng, n, radius):
    r = radius * np.sqrt(rng.uniform(0, 1, n)); th = rng.uniform(0, 2 * math.pi, n)
    return r * np.cos(th), r * np.sin(th)


def _cell_and_wmax(uvw, freq):
    fmax = float(np.max(freq)) / C0
    r_max = float(np.sqrt(np.max(uvw[:, 0] ** 2 + uvw[:, 1] ** 2))) * fmax
    w_max = float(np.max(np.abs(uvw[:, 2]))) * fmax
    return 0.4 / r_max, w_max


def _fill_vis(rng, uvw, freq, src, device, noise=True):
    nrow, nchan = uvw.shape[0], freq.size
    vis = np.empty((nrow, nchan), dtype=np.complex64)
    for c in range(nchan):
        f = freq[c] / C0
        v = predict_vis(uvw[:, 0] * f, uvw[:, 1] * f, uvw[:, 2] * f,
                        src["flux"], src["l"], src["m"], device=device)
        if noise:
            v = v + _noise(rng, nrow)
        vis[:, c] = v.astype(np.complex64)
    return vis


# ------------------------------------------------------------------ configs
def config1(nvis=65536, seed=SEED0 + 1):
    """Tiny: N=256, cell=2^-11, uv uniform disc 0.4 N cells, w U[-200,200], Nw=16, S=7, Q=8."""
    rng = np.random.default_rng(seed)
    N, cell = 256, 2.0 ** -11
    du = 1.0 / (N * cell)
    rr = 0.4 * N * du * np.sqrt(rng.uniform(0, 1, nvis)); th = rng.uniform(0, 2 * math.pi, nvis)
    uvw = np.stack([rr * np.cos(th), rr * np.sin(th), rng.uniform(-200.0, 200.0, nvis)], axis=1)
    src = _sources(rng, 5, 0.05)
    vis = predict_vis(uvw[:, 0], uvw[:, 1], uvw[:, 2], src["flux"], src["l"], src["m"])
    vis = (vis + _noise(rng, nvis)).astype(np.complex64)[:, None]
    return Workload("config1", np.ascontiguousarray(uvw), np.array([C0]), vis,
                    np.ones((nvis, 1), np.float32), N, cell, 16, 200.0, 7, 8, src)


def config2(nvis=10_000_000, seed=SEED0 + 2, device=None, n_dump=4961, noise=True):
    """N=2048, 64 stations in a 5 km disc, 150 MHz, 10 s dumps, Nw=32, S=8, Q=8, fp32.
    Primary reading: 4961 dumps truncated to 1e7 rows (the config's "4 h" gives only 2.9e6)."""
    rng = np.random.default_rng(seed)
    E, Nn = _disc_layout(rng, 64, 5000.0)
    uvw = earth_rotation_uvw(E, Nn, n_dump, max_rows=nvis)
    freq = np.array([150e6])
    cell, w_max = _cell_and_wmax(uvw, freq)
    N = 2048
    src = _sources(rng, 20, 0.3 * N * cell)
    vis = _fill_vis(rng, uvw, freq, src, device, noise)
    return Workload("config2", uvw, freq, vis, np.ones(vis.shape, np.float32),
                    N, cell, 32, w_max, 8, 8, src, notes={"row_block": E.size * (E.size - 1) // 2, "n_ant": int(E.size)})


def config3(N=2048, S=8, nvis=50_000_000, seed=SEED0 + 3):
    """Sweep point: uniform-disc u,v (radius 0.4 N cells), w U[-1000,1000], Nw=64, Q=8,
    vis ~ N(0,1) + i N(0,1), FoV 0.05."""
    rng = np.random.default_rng(seed)
    cell = 0.05 / N
    du = 1.0 / 0.05
    rr = 0.4 * N * du * np.sqrt(rng.uniform(0, 1, nvis)); th = rng.uniform(0, 2 * math.pi, nvis)
    uvw = np.empty((nvis, 3)); uvw[:, 0] = rr * np.cos(th); uvw[:, 1] = rr * np.sin(th)
    del rr, th
    uvw[:, 2] = rng.uniform(-1000.0, 1000.0, nvis)
    vis = np.empty((nvis, 1), np.complex64)
    vis.real[:, 0] = rng.standard_normal(nvis, dtype=np.float32)
    vis.imag[:, 0] = rng.standard_normal(nvis, dtype=np.float32)
    return Workload("config3_N%d_S%d" % (N, S), uvw, np.array([C0]), vis,
                    np.ones((nvis, 1), np.float32), N, cell, 64, 1000.0, int(S), 8)


def ska_low_layout(rng):
    """512 stations: 256 Gaussian core (sigma 500 m, r < 1.5 km) + 3 log-spiral arms to 40 km."""
    E = np.empty(512); Nn = np.empty(512)
    k = 0
    while k < 256:
        x, y = rng.normal(0, 500.0, 2)
        if x * x + y * y < 1500.0 ** 2:
            E[k], Nn[k] = x, y; k += 1
    for a, n in enumerate((86, 85, 85)):
        i = np.arange(n)
        r = 1500.0 * (40.0 / 1.5) ** ((i + 0.5) / n)
        th = 2 * math.pi * a / 3 + 3 * math.pi * np.log(r / 1500.0) / math.log(40.0 / 1.5)
        r = r * (1.0 + 0.03 * rng.standard_normal(n)); th = th + 0.05 * rng.standard_normal(n)
        E[k:k + n] = r * np.cos(th); Nn[k:k + n] = r * np.sin(th); k += n
    return E, Nn


def _fill_vis_blocks(seed, uvw, freq, src, device, noise=True, block_rows=1 << 20):
    """vis[row][chan] = O1 model + noise, generated in row blocks with the noise drawn row-major from its own
    stream, so that the first k rows of a workload are the same whatever the total row count (a prefix of the
    workload can be generated on its own)."""
    nrow, nchan = uvw.shape[0], freq.size
    vis = np.empty((nrow, nchan), dtype=np.complex64)
    f = freq / C0
    nrng = np.random.default_rng([seed, 7])
    for r0 in range(0, nrow, block_rows):
        blk = uvw[r0:r0 + block_rows]
        v = predict_vis(blk[:, 0:1] * f[None, :], blk[:, 1:2] * f[None, :], blk[:, 2:3] * f[None, :],
                        src["flux"], src["l"], src["m"], device=device)
        if noise:
            nz = nrng.normal(0.0, 0.1, (blk.shape[0], nchan, 2))        # R16: sigma 0.1 on re and im
            v = v + (nz[..., 0] + 1j * nz[..., 1])
        vis[r0:r0 + block_rows] = v.astype(np.complex64)
    return vis


def config4(n_dump=360, nchan=8, seed=SEED0 + 4, device=None, max_rows=None, noise=True,
            values="model", prefix_rows=None):
    """SKA1-low-like: 512 stations, 130 816 baselines x n_dump x nchan (150-160 MHz),
    N=8192, Nw=128, ragged support 8..32 (rule K6), Q=8, fp32.
    values="model": 50 sources + noise; values="random": N(0,1) (same throughput, cheap).
    prefix_rows: keep only the first rows of the workload (cell, w_max and every value are those of the full
    n_dump workload: a bounded sample of the same workload for the CPU legs)."""
    rng = np.random.default_rng(seed)
    E, Nn = ska_low_layout(rng)
    uvw = earth_rotation_uvw(E, Nn, n_dump, max_rows=max_rows)
    freq = np.linspace(150e6, 160e6, nchan)
    cell, w_max = _cell_and_wmax(uvw, freq)
    if prefix_rows is not None:
        uvw = np.ascontiguousarray(uvw[:prefix_rows])
    N, Nw = 8192, 128
    src = _sources(rng, 50, 0.3 * N * cell)
    if values == "model":
        vis = _fill_vis_blocks(seed, uvw, freq, src, device, noise)
    else:
        vis = np.empty((uvw.shape[0], nchan), np.complex64)
        for part, sub in ((vis.real, 1), (vis.imag, 2)):
            prng = np.random.default_rng([seed, sub])
            for r0 in range(0, uvw.shape[0], 1 << 22):
                part[r0:r0 + (1 << 22)] = prng.standard_normal((min(1 << 22, uvw.shape[0] - r0), nchan), dtype=np.float32)
    return Workload("config4", uvw, freq, vis, np.ones(vis.shape, np.float32),
                    N, cell, Nw, w_max, ("ragged", 8, 32), 8, src,
                    notes={"row_block": E.size * (E.size - 1) // 2, "n_ant": int(E.size), "n_dump": int(n_dump),
                           "full_rows": int(n_dump * (E.size * (E.size - 1) // 2)) if max_rows is None else int(max_rows)})


def config5(nvis=100_000_000, seed=SEED0 + 5, device=None, n_dump=3064, noise=True):
    """N=4096, 256 stations in a 10 km disc, 150 MHz, 10 s dumps (3064 dumps truncated),
    Nw=64, S=16, Q=8; gridded in fp32 and fp64."""
    rng = np.random.default_rng(seed)
    E, Nn = _disc_layout(rng, 256, 10000.0)
    uvw = earth_rotation_uvw(E, Nn, n_dump, max_rows=nvis)
    freq = np.array([150e6])
    cell, w_max = _cell_and_wmax(uvw, freq)
    N = 4096
    src = _sources(rng, 20, 0.3 * N * cell)
    vis = _fill_vis(rng, uvw, freq, src, device, noise)
    return Workload("config5", uvw, freq, vis, np.ones(vis.shape, np.float32),
                    N, cell, 64, w_max, 16, 8, src, notes={"row_block": E.size * (E.size - 1) // 2, "n_ant": int(E.size)})


def tiny_dft_case(seed=SEED0, N=64, fov=0.08, nvis=300, w_abs=60.0, nsrc=3, src_half=0.02,
                  snap_uv_step=None, snap_w_values=None):
    """P9 input: nvis in a disc of 0.35 N cells, |w| <= w_abs, sources within +-src_half.
    snap_uv_step: round u, v to multiples of this step (wavelengths);
    snap_w_values: replace each w by the nearest of these values.  (The caller picks the
    step / values, e.g. the oversample step and the plane centres.)"""
    rng = np.random.default_rng(seed)
    cell = fov / N
    du = 1.0 / fov
    rr = 0.35 * N * du * np.sqrt(rng.uniform(0, 1, nvis)); th = rng.uniform(0, 2 * math.pi, nvis)
    u = rr * np.cos(th); v = rr * np.sin(th); w = rng.uniform(-w_abs, w_abs, nvis)
    if snap_uv_step is not None:
        u = np.round(u / snap_uv_step) * snap_uv_step
        v = np.round(v / snap_uv_step) * snap_uv_step
    if snap_w_values is not None:
        wv = np.asarray(snap_w_values, float)
        w = wv[np.argmin(np.abs(w[:, None] - wv[None, :]), axis=1)]
    src = _sources(rng, nsrc, src_half)
    vis = predict_vis(u, v, w, src["flux"], src["l"], src["m"])
    uvw = np.ascontiguousarray(np.stack([u, v, w], axis=1))
    return dict(uvw=uvw, vis=vis, N=N, cell=cell, fov=fov, w_max=w_abs, src=src)
