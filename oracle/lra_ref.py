"""ctypes front end of the CPU oracle ``oracle/lra_ref.c``.  TEST INFRASTRUCTURE ONLY.

Only tests/, ``__graft_entry__.smoke()`` and bench.py's ``cpu_baseline`` / ``--impl reference`` legs
import this module; nothing under ``paper_2508_17187_b200/`` does.  The functions marshal numpy
arrays into the C calls and do no arithmetic of their own.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liblra_ref.so")
_SRC = os.path.join(_HERE, "lra_ref.c")
_SRCS = [_SRC, os.path.join(_HERE, "lra_ref_image.c"), os.path.join(_HERE, "lra_ref_gain.c"),
         os.path.join(_HERE, "lra_ref_cf.c")]

SORT_TILE, SORT_TILE_CF = 0, 1


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off -fopenmp: no FMA contraction, so each * and + rounds once (R2)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < max(os.path.getmtime(f) for f in _SRCS):
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
                               "-o", _SO] + _SRCS + ["-lm"])
    return _SO


class _Desc(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("ncorr", C.c_int32), ("nterms", C.c_int32),
                ("oversampling", C.c_int32), ("tile", C.c_int32), ("sort_mode", C.c_int32),
                ("scale_u", C.c_double), ("scale_v", C.c_double), ("n_cf", C.c_int32),
                ("cf_support", C.c_void_p), ("cf_offset", C.c_void_p), ("cf_data", C.c_void_p),
                ("tile_x", C.c_int32)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
    return _lib


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def max_threads() -> int:
    return int(lib().lra_ref_max_threads())


class RefPlan:
    """Holds the descriptor (grid dims, CF table, oversampling) the oracle calls share."""

    def __init__(self, nx, ny, ncorr, nterms, oversampling, scale_u, scale_v, cf_support, cf_offset, cf_data,
                 tile=32, sort_mode=SORT_TILE, tile_x=0):
        self.cf_support = np.ascontiguousarray(cf_support, dtype=np.int32)
        self.cf_offset = np.ascontiguousarray(cf_offset, dtype=np.int64)
        self.cf_data = np.ascontiguousarray(cf_data, dtype=np.complex64)
        self.nx, self.ny, self.ncorr, self.nterms, self.os, self.tile = nx, ny, ncorr, nterms, oversampling, tile
        self.tile_x = tile_x or tile      # R5: tiles are tile_x wide (u) by tile tall (v)
        self.d = _Desc(nx, ny, ncorr, nterms, oversampling, tile, sort_mode, float(scale_u), float(scale_v),
                       len(self.cf_support), _p(self.cf_support), _p(self.cf_offset), _p(self.cf_data), tile_x)

    @property
    def ntiles(self):
        return ((self.nx + self.tile_x - 1) // self.tile_x) * ((self.ny + self.tile - 1) // self.tile)

    def _geom(self, uvw, freq, cf_index):
        uvw = np.ascontiguousarray(uvw, dtype=np.float64)
        freq = np.ascontiguousarray(freq, dtype=np.float64)
        if cf_index is not None:
            cf_index = np.ascontiguousarray(cf_index, dtype=np.int32)
        return uvw, freq, cf_index, uvw.shape[0], freq.shape[0]

    def bin(self, uvw, freq, cf_index=None):
        uvw, freq, cf_index, nrow, nchan = self._geom(uvw, freq, cf_index)
        n = nrow * nchan
        out = dict(ix=np.empty(n, np.int32), iy=np.empty(n, np.int32), fx=np.empty(n, np.int8),
                   fy=np.empty(n, np.int8), key=np.empty(n, np.uint64), perm=np.empty(n, np.uint32),
                   tile_start=np.empty(self.ntiles + 1, np.uint32))
        nv = C.c_int64(0)
        rc = lib().lra_ref_bin(C.byref(self.d), C.c_int64(nrow), C.c_int32(nchan), _p(uvw), _p(freq), _p(cf_index),
                               _p(out["ix"]), _p(out["iy"]), _p(out["fx"]), _p(out["fy"]), _p(out["key"]),
                               _p(out["perm"]), _p(out["tile_start"]), C.byref(nv))
        assert rc == 0
        out["n_valid"] = int(nv.value)
        out["perm"] = out["perm"][: out["n_valid"]]
        return out

    def grid(self, uvw, freq, cf_index, vis, wt, tau=None, grid=None, sumwt=None, nthreads=0):
        uvw, freq, cf_index, nrow, nchan = self._geom(uvw, freq, cf_index)
        vis = np.ascontiguousarray(vis, dtype=np.complex64)
        wt = np.ascontiguousarray(wt, dtype=np.float32)
        tau = None if tau is None else np.ascontiguousarray(tau, dtype=np.float32)
        if grid is None:
            grid = np.zeros((self.nterms, self.ncorr, self.ny, self.nx), dtype=np.complex128)
        if sumwt is None:
            sumwt = np.zeros((self.nterms, self.ncorr), dtype=np.float64)
        rc = lib().lra_ref_grid(C.byref(self.d), C.c_int64(nrow), C.c_int32(nchan), _p(uvw), _p(freq), _p(cf_index),
                                _p(vis), _p(wt), _p(tau), _p(grid), _p(sumwt), C.c_int32(nthreads or max_threads()))
        assert rc == 0
        return grid, sumwt

    def degrid(self, uvw, freq, cf_index, grid, tau=None, vis_in=None, nthreads=0):
        uvw, freq, cf_index, nrow, nchan = self._geom(uvw, freq, cf_index)
        grid = np.ascontiguousarray(grid, dtype=np.complex128)
        tau = None if tau is None else np.ascontiguousarray(tau, dtype=np.float32)
        vis_in = None if vis_in is None else np.ascontiguousarray(vis_in, dtype=np.complex64)
        out = np.empty((nrow, nchan, self.ncorr), dtype=np.complex128)
        rc = lib().lra_ref_degrid(C.byref(self.d), C.c_int64(nrow), C.c_int32(nchan), _p(uvw), _p(freq), _p(cf_index),
                                  _p(grid), _p(tau), _p(vis_in), _p(out), C.c_int32(nthreads or max_threads()))
        assert rc == 0
        return out

    def _awp(self, elems, cf_indices, po_table, po_index):
        eg = np.ascontiguousarray([e[0] for e in elems], dtype=np.int32)
        ec = np.ascontiguousarray([e[1] for e in elems], dtype=np.int32)
        keep = [None if a is None else np.ascontiguousarray(a, dtype=np.int32) for a in (cf_indices or [None] * len(elems))]
        ptrs = (C.c_void_p * len(elems))(*[None if a is None else a.ctypes.data for a in keep])
        po_table = None if po_table is None else np.ascontiguousarray(po_table, dtype=np.float64).reshape(-1, 3)
        po_index = None if po_index is None else np.ascontiguousarray(po_index, dtype=np.int32)
        return eg, ec, keep, ptrs, po_table, po_index

    def grid_awp(self, uvw, freq, elems, cf_indices, vis, wt, tau=None, po_table=None, po_index=None):
        """lra_ref_grid_awp (Eq. 27 + Mueller elements).  elems: [(grid plane, visibility correlation)]; cf_indices: one
        int32 [nrow, nchan] (or None) per element; vis, wt: [nrow, nchan, ncorr_vis]; -> (grid, sumwt)."""
        uvw, freq, _, nrow, nchan = self._geom(uvw, freq, None)
        eg, ec, keep, ptrs, po_table, po_index = self._awp(elems, cf_indices, po_table, po_index)
        vis = np.ascontiguousarray(vis, dtype=np.complex64)
        wt = np.ascontiguousarray(wt, dtype=np.float32)
        tau = None if tau is None else np.ascontiguousarray(tau, dtype=np.float32)
        grid = np.zeros((self.nterms, self.ncorr, self.ny, self.nx), dtype=np.complex128)
        sumwt = np.zeros((self.nterms, self.ncorr), dtype=np.float64)
        rc = lib().lra_ref_grid_awp(C.byref(self.d), C.c_int64(nrow), C.c_int32(nchan), _p(uvw), _p(freq), C.c_int32(len(eg)),
                                    _p(eg), _p(ec), ptrs, C.c_int32(vis.shape[2]), _p(vis), _p(wt), _p(tau), _p(po_table),
                                    _p(po_index), _p(grid), _p(sumwt))
        assert rc == 0
        return grid, sumwt

    def degrid_awp(self, uvw, freq, elems, cf_indices, ncorr_vis, grid, tau=None, po_table=None, po_index=None, vis_in=None):
        """lra_ref_degrid_awp -> complex128 [nrow, nchan, ncorr_vis]."""
        uvw, freq, _, nrow, nchan = self._geom(uvw, freq, None)
        eg, ec, keep, ptrs, po_table, po_index = self._awp(elems, cf_indices, po_table, po_index)
        grid = np.ascontiguousarray(grid, dtype=np.complex128)
        tau = None if tau is None else np.ascontiguousarray(tau, dtype=np.float32)
        vis_in = None if vis_in is None else np.ascontiguousarray(vis_in, dtype=np.complex64)
        out = np.empty((nrow, nchan, ncorr_vis), dtype=np.complex128)
        rc = lib().lra_ref_degrid_awp(C.byref(self.d), C.c_int64(nrow), C.c_int32(nchan), _p(uvw), _p(freq), C.c_int32(len(eg)),
                                      _p(eg), _p(ec), ptrs, C.c_int32(ncorr_vis), _p(grid), _p(tau), _p(po_table),
                                      _p(po_index), _p(vis_in), _p(out))
        assert rc == 0
        return out

    def phase_gradient(self, src, f, dl, dm, conjugate=False, dst=None):
        """lra_ref_phase_gradient: dst (+)= f e^{+-2 pi i (dl u + dm v)} src over all planes of src [..., ny, nx]."""
        src = np.ascontiguousarray(src, dtype=np.complex128)
        nplanes = int(np.prod(src.shape[:-2], dtype=np.int64)) if src.ndim > 2 else 1
        acc = dst is not None
        out = np.ascontiguousarray(dst, dtype=np.complex128).copy() if acc else np.empty_like(src)
        rc = lib().lra_ref_phase_gradient(C.byref(self.d), C.c_int32(nplanes), _p(src), C.c_double(f), C.c_double(dl),
                                          C.c_double(dm), C.c_int32(1 if conjugate else 0), C.c_int32(1 if acc else 0), _p(out))
        assert rc == 0
        return out

    def grid_pixels(self, uvw, freq, cf_index, vis, wt, tau, pix, nthreads=0):
        uvw, freq, cf_index, nrow, nchan = self._geom(uvw, freq, cf_index)
        vis = np.ascontiguousarray(vis, dtype=np.complex64)
        wt = np.ascontiguousarray(wt, dtype=np.float32)
        tau = None if tau is None else np.ascontiguousarray(tau, dtype=np.float32)
        pix = np.ascontiguousarray(pix, dtype=np.int32).reshape(-1, 4)
        out = np.empty(len(pix), dtype=np.complex128)
        rc = lib().lra_ref_grid_pixels(C.byref(self.d), C.c_int64(nrow), C.c_int32(nchan), _p(uvw), _p(freq),
                                       _p(cf_index), _p(vis), _p(wt), _p(tau), C.c_int32(len(pix)), _p(pix), _p(out),
                                       C.c_int32(nthreads or max_threads()))
        assert rc == 0
        return out

    def degrid_points(self, uvw, freq, cf_index, grid_c64, tau, vis_in, sel):
        uvw, freq, cf_index, nrow, nchan = self._geom(uvw, freq, cf_index)
        grid_c64 = np.ascontiguousarray(grid_c64, dtype=np.complex64)
        tau = None if tau is None else np.ascontiguousarray(tau, dtype=np.float32)
        vis_in = None if vis_in is None else np.ascontiguousarray(vis_in, dtype=np.complex64)
        sel = np.ascontiguousarray(sel, dtype=np.int64)
        out = np.empty((len(sel), self.ncorr), dtype=np.complex128)
        rc = lib().lra_ref_degrid_points(C.byref(self.d), C.c_int64(nrow), C.c_int32(nchan), _p(uvw), _p(freq),
                                         _p(cf_index), _p(grid_c64), _p(tau), _p(vis_in), C.c_int32(len(sel)),
                                         _p(sel), _p(out))
        assert rc == 0
        return out


def plan_for(wl, nterms=None, sort_mode=SORT_TILE, tile=None, tile_x=0) -> RefPlan:
    """RefPlan for a ``workloads.Workload`` (argument marshalling only)."""
    c = wl.cfg
    if tile is None:
        tile, tile_x = c.tile, tile_x or c.tile_x
    return RefPlan(c.nx, c.ny, c.ncorr, c.nterms if nterms is None else nterms, c.oversampling, wl.scale_u,
                   wl.scale_v, wl.cf.support, wl.cf.offset, wl.cf.data, tile=tile, sort_mode=sort_mode,
                   tile_x=tile_x)


def image(grid, sumwt=None, corr_x=None, corr_y=None) -> np.ndarray:
    """lra_ref_image: grid [..., ny, nx] complex -> real image of the same leading shape (oracle/lra_ref_image.c)."""
    grid = np.ascontiguousarray(grid, dtype=np.complex128)
    ny, nx = grid.shape[-2:]
    ng = int(np.prod(grid.shape[:-2], dtype=np.int64)) if grid.ndim > 2 else 1
    sumwt = None if sumwt is None else np.ascontiguousarray(sumwt, dtype=np.float64).reshape(ng)
    corr_x = None if corr_x is None else np.ascontiguousarray(corr_x, dtype=np.float64)
    corr_y = None if corr_y is None else np.ascontiguousarray(corr_y, dtype=np.float64)
    out = np.empty(grid.shape, dtype=np.float64)
    rc = lib().lra_ref_image(C.c_int32(ng), C.c_int32(ny), C.c_int32(nx), _p(grid), _p(sumwt), _p(corr_x), _p(corr_y), _p(out))
    assert rc == 0
    return out


def model_grid(img, corr_x=None, corr_y=None) -> np.ndarray:
    """lra_ref_model_grid: real image [..., ny, nx] -> complex grid of the same shape (oracle/lra_ref_image.c)."""
    img = np.ascontiguousarray(img, dtype=np.float64)
    ny, nx = img.shape[-2:]
    ng = int(np.prod(img.shape[:-2], dtype=np.int64)) if img.ndim > 2 else 1
    corr_x = None if corr_x is None else np.ascontiguousarray(corr_x, dtype=np.float64)
    corr_y = None if corr_y is None else np.ascontiguousarray(corr_y, dtype=np.float64)
    out = np.empty(img.shape, dtype=np.complex128)
    rc = lib().lra_ref_model_grid(C.c_int32(ng), C.c_int32(ny), C.c_int32(nx), _p(img), _p(corr_x), _p(corr_y), _p(out))
    assert rc == 0
    return out


def gain_accumulate(vis, model, wt, nbl, bl_index=None, xsum=None, wsum=None):
    """lra_ref_gain_accumulate (Eq. 19): -> (xsum complex [nbl, ncorr], wsum [nbl, ncorr]), accumulated into if given."""
    vis = np.ascontiguousarray(vis, dtype=np.complex64)
    model = np.ascontiguousarray(model, dtype=np.complex64)
    wt = np.ascontiguousarray(wt, dtype=np.float32)
    nrow, nchan, ncorr = vis.shape
    bl_index = None if bl_index is None else np.ascontiguousarray(bl_index, dtype=np.int32)
    xsum = np.zeros((nbl, ncorr), np.complex128) if xsum is None else xsum
    wsum = np.zeros((nbl, ncorr), np.float64) if wsum is None else wsum
    rc = lib().lra_ref_gain_accumulate(C.c_int64(nrow), C.c_int32(nchan), C.c_int32(ncorr), C.c_int32(nbl), _p(bl_index),
                                       _p(vis), _p(model), _p(wt), _p(xsum), _p(wsum))
    assert rc == 0
    return xsum, wsum


def gain_solve(nant, ant1, ant2, xsum, wsum, alpha, delta, max_iter, gains0):
    """lra_ref_gain_solve (Eq. 20, 21): -> (gains complex [nant, ncorr], iterations)."""
    ant1 = np.ascontiguousarray(ant1, dtype=np.int32)
    ant2 = np.ascontiguousarray(ant2, dtype=np.int32)
    xsum = np.ascontiguousarray(xsum, dtype=np.complex128)
    wsum = np.ascontiguousarray(wsum, dtype=np.float64)
    g = np.array(gains0, dtype=np.complex128, copy=True, order="C")
    it = C.c_int32(0)
    rc = lib().lra_ref_gain_solve(C.c_int32(nant), C.c_int32(len(ant1)), C.c_int32(xsum.shape[1]), _p(ant1), _p(ant2), _p(xsum),
                                  _p(wsum), C.c_double(alpha), C.c_double(delta), C.c_int32(max_iter), _p(g), C.byref(it))
    assert rc == 0
    return g, int(it.value)


def cf(n_img, oversampling, fov_rad, support, taper=None, w_lambda=0.0, aterm=None, normalise=True) -> np.ndarray:
    """lra_ref_cf (Table 1): one CF of `support` pixels as complex128 [(S os), (S os)] (oracle/lra_ref_cf.c)."""
    taper = None if taper is None else np.ascontiguousarray(taper, dtype=np.float64)
    aterm = None if aterm is None else np.ascontiguousarray(aterm, dtype=np.complex128)
    assert taper is None or taper.shape == (n_img,)
    assert aterm is None or aterm.shape == (n_img, n_img)
    so = support * oversampling
    out = np.empty((so, so), dtype=np.complex128)
    rc = lib().lra_ref_cf(C.c_int32(n_img), C.c_int32(oversampling), C.c_double(fov_rad), _p(taper), C.c_double(w_lambda),
                          _p(aterm), C.c_int32(support), C.c_int32(1 if normalise else 0), _p(out))
    if rc != 0:
        raise RuntimeError(f"lra_ref_cf rc={rc}")
    return out
