"""Seeded synthetic workloads for the gridding / degridding path.

This module is the ONE piece shared by the CUDA path's tests, bench.py and the CPU oracle.  It only
makes inputs: antenna layouts, uvw tracks, visibilities, weights, convolution-function (CF) tables
and the caller-side ``cf_index``.  It holds none of the method's arithmetic: no pixel rounding, no
sub-pixel phase, no tap loop, no binning (those live in ``csrc/`` and, independently, in ``oracle/``).

The paper's workload is VLA A-array, 2-4 GHz, wide-band AW-projection on the Hubble Ultra Deep Field
(Sec. 6).  That data is not available; the five configurations below take its shapes
(BASELINE.json ``configs``) and stand in for it.  Table 1 of the paper
 fixes which terms make up a CF: PS (Standard), PS*W (W-Projection), PS*A*W
(AW-Projection).

Random numbers: numpy's counter-based Philox generator, key = (BASE_SEED, stream), where the stream
encodes (config, purpose, chunk) so that any part can be regenerated alone and in parallel.
"""
from __future__ import annotations

import math
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field, replace
from typing import Optional

import numpy as np

BASE_SEED = 250817187
C_LIGHT = 299792458.0
N_ANT = 27
N_BL = N_ANT * (N_ANT - 1) // 2  # 351
VLA_LAT_DEG = 34.08
DEC_DEG = -27.8
NU0_HZ = 3.0e9  # reference frequency of the Taylor-term weights


def _rng(cfg_id: int, purpose: int, chunk: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[BASE_SEED, (cfg_id << 40) | (purpose << 32) | chunk]))


# --------------------------------------------------------------------------------------------------
# configuration presets
# --------------------------------------------------------------------------------------------------
@dataclass(frozen=True)
class Config:
    """Shape of one synthetic workload."""

    cfg_id: int
    name: str
    ntimes: int
    nchan: int
    ncorr: int
    nterms: int
    nx: int
    ny: int
    oversampling: int
    cf_kind: str            # "ps" | "w" | "aw"
    s_min: int              # smallest / only CF support
    s_max: int
    n_w: int = 1            # w planes
    n_pa: int = 1           # parallactic-angle bins (aw)
    n_fb: int = 1           # frequency bins (aw)
    ha_hours: float = 4.0   # hour angle spans -ha..+ha
    dt_s: float = 2.0
    kind: str = "vla"       # "disk" (cfg1) | "vla"
    time_stride_of: int = 0  # cfg5: take ntimes samples out of this many, 0 = off
    degrid: bool = False    # cfg5: model grid + degrid + residual gridding
    n_sources: int = 0
    tile: int = 8           # uv tiles of the bucket sort: tile_x wide (u) by tile tall (v); 8 x 8 is the library's default.
    tile_x: int = 8         # cfg2-4 use 4 wide x 8 tall tiles (dense data, narrower regions), cfg1 and cfg5 the default

    @property
    def nrow(self) -> int:
        return N_BL * self.ntimes

    @property
    def npoints(self) -> int:
        return self.nrow * self.nchan

    @property
    def n_cf(self) -> int:
        return self.n_w * self.n_pa * self.n_fb


def full_config(n: int) -> Config:
    """The five BASELINE.json configurations at full size."""
    if n == 1:
        return Config(1, "cfg1-tiny-ps", 60, 1, 1, 1, 256, 256, 20, "ps", 7, 7, kind="disk")
    if n == 2:
        return Config(2, "cfg2-vla-continuum-ps", 14400, 64, 2, 1, 4096, 4096, 20, "ps", 9, 9, ha_hours=4.0, tile_x=4)
    if n == 3:
        return Config(3, "cfg3-wprojection", 7200, 16, 2, 1, 8192, 8192, 8, "w", 9, 65, n_w=128, ha_hours=2.0, tile_x=4)
    if n == 4:
        return Config(4, "cfg4-awprojection-fullpol", 7200, 16, 4, 1, 4096, 4096, 8, "aw", 17, 49,
                      n_w=32, n_pa=8, n_fb=4, ha_hours=2.0, tile_x=4)
    if n == 5:
        return Config(5, "cfg5-degrid-multiterm", 1157, 16, 2, 2, 8192, 8192, 8, "w", 9, 65, n_w=128,
                      ha_hours=2.0, time_stride_of=7200, degrid=True, n_sources=200)
    raise ValueError(n)


def small_config(n: int) -> Config:
    """Reduced variants of the same structure, sized so that the oracle finishes in seconds while the
    data still spans many tiles, several support classes and a ragged tail."""
    c = full_config(n)
    if n == 1:
        return c
    if n == 2:
        return replace(c, name=c.name + "-small", ntimes=40, nchan=8, nx=512, ny=512)
    if n == 3:
        return replace(c, name=c.name + "-small", ntimes=24, nchan=4, nx=1024, ny=1024, n_w=16, s_max=33)
    if n == 4:
        return replace(c, name=c.name + "-small", ntimes=16, nchan=4, nx=512, ny=512, n_w=4, n_pa=2,
                       n_fb=2, s_min=9, s_max=21)
    if n == 5:
        return replace(c, name=c.name + "-small", ntimes=19, nchan=4, nx=1024, ny=1024, n_w=16,
                       s_max=33, time_stride_of=120, n_sources=20)
    raise ValueError(n)


# --------------------------------------------------------------------------------------------------
# prolate-spheroidal function from its textbook definition
# --------------------------------------------------------------------------------------------------
class Prolate:
    """Zero-order prolate spheroidal wave function psi_c on [-1, 1]: the dominant eigenfunction of the
    band-limiting operator  int_{-1}^{1} sin(c(x-y)) / (pi (x-y)) psi(y) dy = lambda psi(x)
    (SURVEY.md Sec. 8(d)), with c = pi*S/2 for a support of S pixels.

    For c of a few pi the leading eigenvalues of that integral operator all sit within 1e-10 of 1, so
    power iteration on it cannot separate psi_0.  The same functions are the eigenfunctions of the
    commuting differential operator  d/dx[(1 - x^2) psi'] - c^2 x^2 psi = -chi psi  (Slepian & Pollak),
    whose eigenvalues are well separated; psi_0 belongs to the smallest chi.  Expanding psi in normalised
    Legendre polynomials of even order turns it into a symmetric tridiagonal eigenproblem, solved here
    with numpy.  `integral_residual()` checks the result against the integral definition above."""

    def __init__(self, support: int, n_terms: int = 0):
        self.c = c = math.pi * support / 2.0
        n = n_terms or (2 * int(c) + 40)
        k = 2.0 * np.arange(n)                                  # even orders
        diag = k * (k + 1) + c * c * (2 * k * (k + 1) - 1) / ((2 * k + 3) * (2 * k - 1))
        off = c * c * (k + 2) * (k + 1) / ((2 * k + 3) * np.sqrt((2 * k + 1) * (2 * k + 5)))
        A = np.diag(diag) + np.diag(off[:-1], 1) + np.diag(off[:-1], -1)
        w, v = np.linalg.eigh(A)
        self.beta = v[:, 0] * np.sqrt(k + 0.5)                  # coefficients of plain P_k
        self.orders = k.astype(int)
        self.norm0 = 1.0
        self.norm0 = float(self(np.array([0.0]))[0])
        if self.norm0 < 0:
            self.beta, self.norm0 = -self.beta, -self.norm0

    def __call__(self, x: np.ndarray) -> np.ndarray:
        x = np.asarray(x, dtype=np.float64)
        coef = np.zeros(self.orders[-1] + 1)
        coef[self.orders] = self.beta
        out = np.polynomial.legendre.legval(np.clip(x, -1.0, 1.0), coef)
        return np.where(np.abs(x) > 1.0, 0.0, out)

    def integral_residual(self, n_nodes: int = 256):
        """(lambda, max |K psi - lambda psi| / max |psi|) for the sinc-kernel integral operator."""
        y, w = np.polynomial.legendre.leggauss(n_nodes)
        d = y[:, None] - y[None, :]
        K = (self.c / math.pi) * np.sinc(self.c * d / math.pi) * w[None, :]
        psi = self(y)
        kp = K @ psi
        lam = float(kp @ (w * psi) / (psi @ (w * psi)))
        return lam, float(np.abs(kp - lam * psi).max() / np.abs(psi).max())


def _kernel_sample_offsets(S: int, os_: int) -> np.ndarray:
    """Pixel offsets of the S*os samples of an oversampled kernel.  Storage convention handed to the
    library: sample m sits at offset (m - c0)/os pixels, c0 = h*os + (os - 1 - os//2)
    (= h*os + os/2 - 1 for even os)."""
    h = (S - 1) // 2
    c0 = h * os_ + (os_ - 1 - os_ // 2)
    return (np.arange(S * os_) - c0) / float(os_)


def ps_kernel(S: int, os_: int) -> np.ndarray:
    """(S*os)^2 complex64 'Standard' CF (Table 1 row Standard): outer product of psi."""
    psi = Prolate(S)
    off = _kernel_sample_offsets(S, os_)
    k1 = psi(off / (S / 2.0)) / psi.norm0
    k = np.outer(k1, k1)
    k *= os_ * os_ / k.sum()  # sum(all samples)/os^2 = 1
    return k.astype(np.complex64)


def _dft_crop(img: np.ndarray, S: int, os_: int) -> np.ndarray:
    """Samples of the 2-D forward DFT of `img` (N x N raster spanning the field, centre at N/2) at
    the (S*os)^2 oversampled uv positions of the storage convention.  Mathematically the zero-padded
    (x os) FFT cropped about the centre, evaluated as two small matrix
    products instead of a large padded FFT."""
    N = img.shape[0]
    off = _kernel_sample_offsets(S, os_)              # uv offset in grid pixels
    n = np.arange(N) - N // 2                           # image pixel index about the centre
    E = np.exp(-2j * np.pi * np.outer(off, n) / N)      # [S*os, N]
    return E @ img @ E.T


@dataclass
class CFTable:
    """Caller-side CF table exactly as handed to ``lra_plan_create``."""

    support: np.ndarray   # int32 [n_cf]
    offset: np.ndarray    # int64 [n_cf] element offsets into data
    data: np.ndarray      # complex64 flat
    oversampling: int

    def kernel(self, i: int) -> np.ndarray:
        n = int(self.support[i]) * self.oversampling
        return self.data[self.offset[i]: self.offset[i] + n * n].reshape(n, n)


def _pack(kernels, os_) -> CFTable:
    sup = np.array([k.shape[0] // os_ for k in kernels], dtype=np.int32)
    sizes = np.array([k.size for k in kernels], dtype=np.int64)
    off = np.concatenate([[0], np.cumsum(sizes)[:-1]]).astype(np.int64)
    data = np.concatenate([k.reshape(-1) for k in kernels]).astype(np.complex64)
    return CFTable(sup, off, data, os_)


def w_plane_support(cfg: Config, p: int) -> int:
    """S_p = S_min + 2*round((S_max - S_min)/2 * p/(Nw-1))."""
    if cfg.n_w == 1:
        return cfg.s_min
    return cfg.s_min + 2 * int(round((cfg.s_max - cfg.s_min) / 2.0 * p / (cfg.n_w - 1)))


def make_cf_table(cfg: Config, fov_rad: float, w_max: float, n_img: int = 0) -> CFTable:
    """CF table per Table 1: 'ps' -> PS; 'w' -> PS*W; 'aw' -> PS*A*W, where the
    convolution in the uv plane is a product in the image plane followed by a Fourier transform."""
    os_ = cfg.oversampling
    if cfg.cf_kind == "ps":
        return _pack([ps_kernel(cfg.s_min, os_)], os_)
    if n_img == 0:
        n_img = 128 if cfg.s_max > 33 else 64
    assert n_img >= cfg.s_max + 1
    taper1 = Prolate(cfg.s_min)
    x = (np.arange(n_img) - n_img // 2) / (n_img / 2.0)       # [-1, 1)
    t1 = taper1(x) / taper1.norm0
    taper = np.outer(t1, t1)
    l = x * (fov_rad / 2.0)
    ll, mm = np.meshgrid(l, l)                               # mm varies along axis 0 (v), ll along axis 1 (u)
    r2 = ll * ll + mm * mm
    nterm = np.sqrt(np.maximum(0.0, 1.0 - r2)) - 1.0
    kernels = []
    if cfg.cf_kind == "aw":
        apertures = _aw_apertures(cfg, n_img, fov_rad)
    for wp in range(cfg.n_w):
        w_c = (wp + 0.5) * w_max / cfg.n_w              # plane centre
        S = w_plane_support(cfg, wp)
        wphase = np.exp(2j * np.pi * w_c * nterm)
        if cfg.cf_kind == "w":
            k = _dft_crop(taper * wphase, S, os_)
            k *= os_ * os_ / k.sum()
            kernels.append(k.astype(np.complex64))
        else:
            for pa in range(cfg.n_pa):
                for fb in range(cfg.n_fb):
                    k = _dft_crop(taper * apertures[pa][fb] * wphase, S, os_)
                    k *= os_ * os_ / k.sum()
                    kernels.append(k.astype(np.complex64))
    return _pack(kernels, os_)


def w_kernel(S: int, os_: int, s_taper: int, w_lambda: float, fov_rad: float, n_img: int = 64) -> np.ndarray:
    """One PS*W kernel at an explicit w (used by the generator pins, P10)."""
    taper1 = Prolate(s_taper)
    x = (np.arange(n_img) - n_img // 2) / (n_img / 2.0)
    t1 = taper1(x) / taper1.norm0
    l = x * (fov_rad / 2.0)
    ll, mm = np.meshgrid(l, l)
    nterm = np.sqrt(np.maximum(0.0, 1.0 - ll * ll - mm * mm)) - 1.0
    k = _dft_crop(np.outer(t1, t1) * np.exp(2j * np.pi * w_lambda * nterm), S, os_)
    k *= os_ * os_ / k.sum()
    return k.astype(np.complex64)


def _aw_apertures(cfg: Config, n_img: int, fov_rad: float):
    """A-term: image-plane power pattern |FT(aperture)|^2 of one tapered circular aperture with
    seeded smooth phase errors, rotated by the parallactic-angle bin centre and scaled by the
    frequency bin centre."""
    rng = _rng(cfg.cfg_id, 7)
    n_ap = 64
    # smooth aperture phase errors: a few low-order 2-D cosine modes with seeded amplitudes
    modes = [(a, b) for a in range(3) for b in range(3) if a + b > 0]
    amp = rng.normal(0.0, 0.15, size=len(modes))
    pha = rng.uniform(0.0, 2 * np.pi, size=len(modes))
    out = []
    pa_lo, pa_hi = -1.2, 1.2  # nominal range of bin centres (radians); the index bins use the data range
    for pa in range(cfg.n_pa):
        ang = pa_lo + (pa + 0.5) * (pa_hi - pa_lo) / cfg.n_pa
        row = []
        for fb in range(cfg.n_fb):
            nu = 2.0e9 + (fb + 0.5) * 2.0e9 / cfg.n_fb
            # aperture plane sampled so that the primary beam (lambda/D, D = 25 m) spans the field
            d_lambda = 25.0 * nu / C_LIGHT
            # image raster l in [-fov/2, fov/2): aperture coordinate conjugate to l, in wavelengths
            a = (np.arange(n_ap) - n_ap // 2) / (n_ap / 2.0)  # [-1, 1) aperture radius units
            ax, ay = np.meshgrid(a, a)
            rx = np.cos(ang) * ax + np.sin(ang) * ay
            ry = -np.sin(ang) * ax + np.cos(ang) * ay
            rr = np.sqrt(rx * rx + ry * ry)
            illum = np.where(rr <= 1.0, (1.0 - 0.75 * rr * rr), 0.0)
            ph = np.zeros_like(rr)
            for (ma, mb), am, p0 in zip(modes, amp, pha):
                ph += am * np.cos(np.pi * (ma * rx + mb * ry) + p0)
            ap = illum * np.exp(1j * ph)
            # far-field voltage pattern at image raster points: direct DFT, aperture radius d_lambda/2
            l = (np.arange(n_img) - n_img // 2) * (fov_rad / n_img)
            pos = a * (d_lambda / 2.0)
            E = np.exp(-2j * np.pi * np.outer(l, pos))
            volt = E @ ap @ E.T
            power = np.abs(volt) ** 2
            power /= power[n_img // 2, n_img // 2]
            # keep the (weak) asymmetry from the phase errors in a complex pattern so that the CF is
            # not Hermitian-symmetric: A = power * exp(i * small odd phase)
            odd = np.angle(volt * np.conj(volt[::-1, ::-1]))
            row.append(power * np.exp(0.5j * odd))
        out.append(row)
    return out


# --------------------------------------------------------------------------------------------------
# geometry
# --------------------------------------------------------------------------------------------------
def antenna_xyz(cfg_id: int) -> np.ndarray:
    """27 antennas, 9 per arm, arms at azimuth 5, 125, 245 deg, radius 21 km * xi, xi ~ U(0.02, 1);
    local ENU -> equatorial XYZ at latitude 34.08 N."""
    rng = _rng(2, 1)  # one array layout for all VLA-like configs
    xi = rng.uniform(0.02, 1.0, size=N_ANT)
    az = np.deg2rad(np.repeat([5.0, 125.0, 245.0], 9))
    r = 21000.0 * xi
    e, n, u = r * np.sin(az), r * np.cos(az), np.zeros(N_ANT)
    lat = math.radians(VLA_LAT_DEG)
    X = -math.sin(lat) * n + math.cos(lat) * u
    Y = e
    Z = math.cos(lat) * n + math.sin(lat) * u
    return np.stack([X, Y, Z], axis=1)


def hour_angles(cfg: Config) -> np.ndarray:
    if cfg.time_stride_of:
        k = np.arange(cfg.ntimes)
        idx = np.floor(k * cfg.time_stride_of / cfg.ntimes)
        n_all = cfg.time_stride_of
    else:
        idx = np.arange(cfg.ntimes, dtype=np.float64)
        n_all = cfg.ntimes
    # samples centred in their 2 s (or stretched, for reduced configs) slots over [-ha, +ha]
    span = 2.0 * cfg.ha_hours * 3600.0
    t = -cfg.ha_hours * 3600.0 + (idx + 0.5) * span / n_all
    return t * (2.0 * math.pi / 86164.0905)


def uvw_metres(cfg: Config) -> np.ndarray:
    """uvw[nrow][3] in metres, row = time * 351 + baseline (Measurement-Set order), textbook rotation:
    u = sinH X + cosH Y; v = -sin(d) cosH X + sin(d) sinH Y + cos(d) Z; w = cos(d) cosH X - cos(d) sinH Y + sin(d) Z."""
    xyz = antenna_xyz(cfg.cfg_id)
    i, j = np.triu_indices(N_ANT, 1)
    b = xyz[j] - xyz[i]                                      # [351, 3]
    H = hour_angles(cfg)[:, None]
    sd, cd = math.sin(math.radians(DEC_DEG)), math.cos(math.radians(DEC_DEG))
    X, Y, Z = b[None, :, 0], b[None, :, 1], b[None, :, 2]
    u = np.sin(H) * X + np.cos(H) * Y
    v = -sd * np.cos(H) * X + sd * np.sin(H) * Y + cd * Z
    w = cd * np.cos(H) * X - cd * np.sin(H) * Y + sd * Z
    return np.stack([u, v, w], axis=-1).reshape(-1, 3)


def parallactic_angle(cfg: Config) -> np.ndarray:
    """Textbook parallactic angle per time sample."""
    H = hour_angles(cfg)
    lat, dec = math.radians(VLA_LAT_DEG), math.radians(DEC_DEG)
    return np.arctan2(np.cos(lat) * np.sin(H), np.sin(lat) * math.cos(dec) - np.cos(lat) * math.sin(dec) * np.cos(H))


def channel_freqs(cfg: Config) -> np.ndarray:
    if cfg.kind == "disk":
        return np.array([C_LIGHT], dtype=np.float64)         # lambda = 1 m
    return 2.0e9 + (np.arange(cfg.nchan) + 0.5) * (2.0e9 / cfg.nchan)


# --------------------------------------------------------------------------------------------------
# random payloads (parallel, chunked, each chunk its own counter stream)
# --------------------------------------------------------------------------------------------------
_CHUNK = 1 << 22


def _parallel_fill(n: int, fn, dtype) -> np.ndarray:
    out = np.empty(n, dtype=dtype)
    nch = (n + _CHUNK - 1) // _CHUNK

    def work(c):
        lo, hi = c * _CHUNK, min(n, (c + 1) * _CHUNK)
        out[lo:hi] = fn(c, hi - lo)

    if nch <= 1:
        for c in range(nch):
            work(c)
    else:
        with ThreadPoolExecutor(max_workers=min(32, nch)) as ex:
            list(ex.map(work, range(nch)))
    return out


def complex_normal(cfg_id: int, purpose: int, n: int) -> np.ndarray:
    """complex64 with re, im ~ N(0,1) independently ('CN(0,1)' in SURVEY.md Sec. 8(d))."""
    f = _parallel_fill(2 * n, lambda c, m: _rng(cfg_id, purpose, c).standard_normal(m, dtype=np.float32), np.float32)
    return f.view(np.complex64)


def uniform_f32(cfg_id: int, purpose: int, n: int, lo: float, hi: float) -> np.ndarray:
    return _parallel_fill(n, lambda c, m: (lo + (hi - lo) * _rng(cfg_id, purpose, c).random(m, dtype=np.float32)), np.float32)


# --------------------------------------------------------------------------------------------------
# the workload object
# --------------------------------------------------------------------------------------------------
@dataclass
class Workload:
    cfg: Config
    uvw: np.ndarray                  # float64 [nrow, 3] metres
    freq: np.ndarray                 # float64 [nchan] Hz
    vis: np.ndarray                  # complex64 [nrow, nchan, ncorr]
    wt: np.ndarray                   # float32 [nrow, nchan, ncorr]
    cf: CFTable
    cf_index: Optional[np.ndarray]   # int32 [nrow, nchan] or None
    tau: Optional[np.ndarray]        # float32 [nchan, nterms] or None
    scale_u: float
    scale_v: float
    model_grid: Optional[np.ndarray] = None  # complex64 [1, ncorr, ny, nx] (cfg5)
    info: dict = field(default_factory=dict)

    def sum_s2(self) -> int:
        """Sum over all points of S^2 (the tap count per correlation and term before validity)."""
        if self.cf_index is None:
            return int(self.cfg.npoints) * int(self.cf.support[0]) ** 2
        s = self.cf.support.astype(np.int64)
        cnt = np.bincount(self.cf_index.reshape(-1), minlength=len(s)).astype(np.int64)
        return int((cnt * s * s).sum())


def make_workload(cfg: Config, with_payload: bool = True) -> Workload:
    if cfg.kind == "disk":
        return _make_disk(cfg)
    uvw = uvw_metres(cfg)
    freq = channel_freqs(cfg)
    # conjugate-flip rows with w < 0 so that only w >= 0 planes are needed
    neg = uvw[:, 2] < 0.0
    uvw[neg] *= -1.0
    lam_inv = freq / C_LIGHT
    r_m = np.sqrt(uvw[:, 0] ** 2 + uvw[:, 1] ** 2).max()
    r_lambda_max = r_m * lam_inv.max()
    scale = 0.4 * cfg.nx / r_lambda_max                          # SURVEY R15, pixels per wavelength
    fov = scale                                                   # = 1 / uv cell, radians (R1: scale = nx * dl)
    w_max = float(np.abs(uvw[:, 2]).max() * lam_inv.max())
    info = {"scale_px_per_lambda": scale, "cell_lambda": 1.0 / scale, "fov_rad": fov, "w_max_lambda": w_max}

    cf_index = None
    if cfg.cf_kind in ("w", "aw"):
        w_l = np.abs(uvw[:, 2])[:, None] * lam_inv[None, :]
        wp = np.minimum(cfg.n_w - 1, np.floor(w_l / w_max * cfg.n_w).astype(np.int64))
        if cfg.cf_kind == "w":
            cf_index = wp.astype(np.int32)
        else:
            pa_t = parallactic_angle(cfg)
            lo, hi = pa_t.min(), pa_t.max()
            pa_bin = np.minimum(cfg.n_pa - 1, np.floor((pa_t - lo) / max(hi - lo, 1e-30) * cfg.n_pa).astype(np.int64))
            pa_row = np.repeat(pa_bin, N_BL)[:, None]
            fb = np.minimum(cfg.n_fb - 1, np.floor((freq - 2.0e9) / 2.0e9 * cfg.n_fb).astype(np.int64))[None, :]
            cf_index = ((wp * cfg.n_pa + pa_row) * cfg.n_fb + fb).astype(np.int32)
        cf_index = np.ascontiguousarray(cf_index)
    cf = make_cf_table(cfg, fov, w_max)

    vis = wt = None
    if with_payload:
        n = cfg.npoints * cfg.ncorr
        vis = complex_normal(cfg.cfg_id, 2, n).reshape(cfg.nrow, cfg.nchan, cfg.ncorr)
        wt = uniform_f32(cfg.cfg_id, 3, n, 0.5, 1.0).reshape(cfg.nrow, cfg.nchan, cfg.ncorr)
        # R8 payload part of the flip: V -> V*, and RL <-> LR for four correlations
        if neg.any():
            vis[neg] = np.conj(vis[neg])
            if cfg.ncorr == 4:
                vis[neg] = vis[neg][:, :, [0, 2, 1, 3]]
                wt[neg] = wt[neg][:, :, [0, 2, 1, 3]]
    tau = None
    if cfg.nterms > 1:
        x = (freq - NU0_HZ) / NU0_HZ
        tau = np.stack([x ** t for t in range(cfg.nterms)], axis=1).astype(np.float32)
    wl = Workload(cfg, np.ascontiguousarray(uvw), freq, vis, wt, cf, cf_index, tau, scale, scale, info=info)
    if cfg.degrid:
        wl.model_grid = _model_grid(cfg, fov)
    return wl


def _make_disk(cfg: Config) -> Workload:
    """cfg1: (u, v) in pixels uniform in a disk of radius 0.4*N about the centre, lambda = 1 m, scale = 1."""
    rng = _rng(cfg.cfg_id, 1)
    n = cfg.nrow
    r = 0.4 * cfg.nx * np.sqrt(rng.random(n))
    th = 2.0 * np.pi * rng.random(n)
    uvw = np.stack([r * np.cos(th), r * np.sin(th), np.zeros(n)], axis=1)
    vis = complex_normal(cfg.cfg_id, 2, n * cfg.nchan * cfg.ncorr).reshape(n, cfg.nchan, cfg.ncorr)
    wt = np.ones((n, cfg.nchan, cfg.ncorr), dtype=np.float32)
    cf = make_cf_table(cfg, 0.0, 0.0)
    return Workload(cfg, uvw, channel_freqs(cfg), vis, wt, cf, None, None, 1.0, 1.0,
                    info={"scale_px_per_lambda": 1.0})


def _model_grid(cfg: Config, fov: float) -> np.ndarray:
    """cfg5 model: point sources at seeded positions within the inner 80 % of the field, flux ~ U(0.1, 1);
    the model *grid* is their analytic Fourier transform sampled at the uv pixel centres (the 2-D FFT of the delta
    functions, evaluated directly; host-side, not timed).  NO inverse taper is applied (reading R20: the
    taper correction is an input-side choice that does not touch the path; lra_model_grid takes it as corr_x / corr_y).
    Same grid for every correlation."""
    rng = _rng(cfg.cfg_id, 5)
    ns = cfg.n_sources
    # integer image-pixel positions so that the transform is an exact DFT harmonic
    px = rng.integers(int(0.1 * cfg.nx), int(0.9 * cfg.nx), size=ns) - cfg.nx // 2
    py = rng.integers(int(0.1 * cfg.ny), int(0.9 * cfg.ny), size=ns) - cfg.ny // 2
    flux = rng.uniform(0.1, 1.0, size=ns)
    ku = (np.arange(cfg.nx) - cfg.nx // 2)
    kv = (np.arange(cfg.ny) - cfg.ny // 2)
    # sum over sources of flux * exp(-2 pi i (ku*px/nx + kv*py/ny)), as one [ny, ns] x [ns, nx] product
    eu = np.exp(-2j * np.pi * np.outer(px, ku) / cfg.nx)
    ev = np.exp(-2j * np.pi * np.outer(kv, py) / cfg.ny) * flux[None, :]
    g = (ev.astype(np.complex64) @ eu.astype(np.complex64)).astype(np.complex64)
    return np.ascontiguousarray(np.broadcast_to(g, (1, cfg.ncorr, cfg.ny, cfg.nx)))
