"""Thin Python binding of liblra.so (include/lra.h).  Argument marshalling only: every step of the path
runs in the CUDA kernels behind the C ABI.  PyTorch supplies device memory and streams, nothing else.

The functions carry the names of the C entry points and take torch CUDA tensors (device pointers) or
numpy arrays (host pointers) exactly where lra.h says "device" or "host".  There is no CPU fallback: if the
shared library cannot be loaded, importing this module's `lib()` raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

from . import _build

LRA_OK, LRA_EINVAL, LRA_ENOMEM, LRA_ECUDA, LRA_ESTATE = 0, 1, 2, 3, 4
LRA_SORT_TILE, LRA_SORT_TILE_CF = 0, 1
LRA_STATIC_MAX_AXES = 65536   # lra.h: largest nx + ny lra_phase_gradient_static accepts


class LraError(RuntimeError):
    pass


class lra_plan_desc(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("ncorr", C.c_int32), ("nterms", C.c_int32),
                ("oversampling", C.c_int32), ("tile", C.c_int32), ("sort_mode", C.c_int32),
                ("scale_u", C.c_double), ("scale_v", C.c_double), ("n_cf", C.c_int32),
                ("cf_support", C.c_void_p), ("cf_offset", C.c_void_p), ("cf_data", C.c_void_p),
                ("device", C.c_int32), ("stream", C.c_void_p), ("tile_x", C.c_int32)]


class lra_cf_desc(C.Structure):
    _fields_ = [("n_img", C.c_int32), ("oversampling", C.c_int32), ("fov_rad", C.c_double), ("taper", C.c_void_p),
                ("n_aterm", C.c_int32), ("aterm", C.c_void_p), ("n_cf", C.c_int32), ("cf_support", C.c_void_p),
                ("cf_offset", C.c_void_p), ("cf_w", C.c_void_p), ("cf_aterm", C.c_void_p), ("normalise", C.c_int32),
                ("device", C.c_int32), ("stream", C.c_void_p)]


_lib = None


def lib() -> C.CDLL:
    """Loads liblra.so (building it in-tree with nvcc if sources are newer).  Fails loudly otherwise."""
    global _lib
    if _lib is None:
        path = _build.SO_PATH
        if _build.needs_build():
            path = _build.build()
        if not os.path.exists(path):
            raise LraError(f"liblra.so not found at {path}; the CUDA extension is required (no CPU fallback)")
        L = C.CDLL(path)
        vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
        L.lra_plan_create.argtypes = [C.POINTER(vp), C.POINTER(lra_plan_desc)]
        L.lra_plan_destroy.argtypes = [vp]
        L.lra_bin.argtypes = [vp, i64, i32, vp, vp, vp]
        L.lra_bin_export.argtypes = [vp] * 8 + [C.POINTER(i64)]
        L.lra_grid.argtypes = [vp] * 6
        L.lra_degrid.argtypes = [vp] * 5
        L.lra_image.argtypes = [vp] * 6
        L.lra_model_grid.argtypes = [vp] * 5
        L.lra_gain_accumulate.argtypes = [i32, vp, i64, i32, i32, i32, vp, vp, vp, vp, vp, vp]
        L.lra_gain_solve.argtypes = [i32, vp, i32, i32, i32, vp, vp, vp, vp, C.c_double, C.c_double, i32, vp, vp]
        L.lra_cf_generate.argtypes = [C.POINTER(lra_cf_desc), vp]
        L.lra_phase_gradient.argtypes = [vp, vp, C.c_double, C.c_double, C.c_double, i32, i32, vp]
        L.lra_phase_gradient_static.argtypes = [i32, i32, i32, C.c_double, C.c_double, vp, C.c_double, C.c_double, C.c_double,
                                                i32, i32, vp, vp]
        L.lra_static_last_error.restype = C.c_char_p
        L.lra_grid_po.argtypes = [vp, vp, vp, vp, i32, vp, vp, vp, vp]
        L.lra_degrid_po.argtypes = [vp, vp, vp, i32, vp, vp, vp, vp]
        L.lra_grid_mueller.argtypes = [vp, i64, i32, vp, vp, i32, vp, vp, vp, i32, vp, vp, vp, i32, vp, vp, i32, vp, vp]
        L.lra_degrid_mueller.argtypes = [vp, i64, i32, vp, vp, i32, vp, vp, vp, i32, i32, vp, vp, i32, vp, vp, vp, vp]
        L.lra_cf_last_cuda_error.restype = C.c_int
        L.lra_launch_count.argtypes = [vp]
        L.lra_launch_count.restype = i64
        L.lra_tap_count.argtypes = [vp, C.POINTER(i64), C.POINTER(i64)]
        L.lra_set_variant.argtypes = [vp, i32, i32]
        L.lra_diag_fma_tflops.argtypes = [i32, C.POINTER(C.c_double)]
        L.lra_diag_l2_gbs.argtypes = [i32, i32, C.POINTER(C.c_double)]
        L.lra_strerror.argtypes = [C.c_int]
        L.lra_strerror.restype = C.c_char_p
        L.lra_last_cuda_error.argtypes = [vp]
        L.lra_last_cuda_error.restype = C.c_char_p
        _lib = L
    return _lib


EXPORTED = ["lra_plan_create", "lra_plan_destroy", "lra_bin", "lra_bin_export", "lra_grid", "lra_degrid", "lra_image",
            "lra_model_grid", "lra_gain_accumulate", "lra_gain_solve", "lra_cf_generate", "lra_cf_last_cuda_error",
            "lra_phase_gradient", "lra_phase_gradient_static", "lra_static_last_error", "lra_grid_po", "lra_degrid_po", "lra_grid_mueller", "lra_degrid_mueller",
            "lra_launch_count", "lra_tap_count", "lra_set_variant", "lra_strerror", "lra_last_cuda_error",
            "lra_diag_fma_tflops", "lra_diag_l2_gbs"]


def _check(rc: int, plan=None):
    if rc != LRA_OK:
        msg = lib().lra_strerror(rc).decode()
        if plan:
            detail = lib().lra_last_cuda_error(plan).decode()
            if detail:
                msg += f" ({detail})"
        raise LraError(f"liblra: {msg} [code {rc}]")


_plan_device = {}   # plan handle -> CUDA device index (argument checks only)


def _dev(t, dtype=None, plan=None) -> Optional[int]:
    """Device pointer of a contiguous CUDA tensor on the plan's device (None passes NULL)."""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise LraError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise LraError(f"expected dtype {dtype}, got {t.dtype}")
    if plan is not None and plan in _plan_device and t.device.index != _plan_device[plan]:
        raise LraError(f"tensor on cuda:{t.device.index}, plan on cuda:{_plan_device[plan]}")
    return t.data_ptr()


def _host(a: np.ndarray, dtype) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=dtype)


def lra_plan_create(nx, ny, ncorr, nterms, oversampling, scale_u, scale_v, cf_support, cf_offset, cf_data,
                    tile=0, sort_mode=LRA_SORT_TILE_CF, device=0, stream=None, tile_x=0) -> int:
    """-> opaque plan handle (int).  cf_support / cf_offset are HOST numpy arrays; cf_data is a HOST numpy array or a
    CUDA complex64 tensor (e.g. lra_cf_generate's output) (lra.h: lra_plan_desc).  tile = 0: the library's
    default 8 x 8 tiles; tile_x = 0 with tile != 0: square tiles.  stream: a CUDA stream handle (int), 0 / None = the
    default stream."""
    sup = _host(cf_support, np.int32)
    off = _host(cf_offset, np.int64)
    if isinstance(cf_data, np.ndarray):
        dat = _host(cf_data, np.complex64)
        dat_ptr = dat.ctypes.data
    else:
        import torch
        if cf_data.device.index != int(device):
            raise LraError(f"cf_data on cuda:{cf_data.device.index}, plan on cuda:{int(device)}")
        dat_ptr = _dev(cf_data, torch.complex64)
    d = lra_plan_desc(nx, ny, ncorr, nterms, oversampling, tile, sort_mode, float(scale_u), float(scale_v), len(sup),
                      sup.ctypes.data, off.ctypes.data, dat_ptr, device, stream or 0, tile_x)
    h = C.c_void_p()
    _check(lib().lra_plan_create(C.byref(h), C.byref(d)))
    _plan_device[h.value] = int(device)
    return h.value


def lra_plan_destroy(plan: int):
    _check(lib().lra_plan_destroy(plan))
    _plan_device.pop(plan, None)


def lra_bin(plan: int, uvw_m, freq_hz, cf_index=None):
    """uvw_m: CUDA float64 [nrow, 3]; freq_hz: HOST float64 [nchan]; cf_index: CUDA int32 [nrow, nchan] or None."""
    import torch
    f = _host(freq_hz, np.float64)
    nrow, nchan = int(uvw_m.shape[0]), len(f)
    if tuple(uvw_m.shape) != (nrow, 3):
        raise LraError(f"uvw_m must be [nrow, 3], got {tuple(uvw_m.shape)}")
    if cf_index is not None and tuple(cf_index.shape) != (nrow, nchan):
        raise LraError(f"cf_index must be [nrow, nchan] = {(nrow, nchan)}, got {tuple(cf_index.shape)}")
    _check(lib().lra_bin(plan, nrow, nchan, _dev(uvw_m, torch.float64, plan), f.ctypes.data,
                         _dev(cf_index, torch.int32, plan)), plan)


def lra_bin_export(plan: int, ix=None, iy=None, fx=None, fy=None, key=None, perm=None, tile_start=None) -> int:
    """Copies the bin arrays into the given CUDA tensors (None skips); returns n_valid."""
    nv = C.c_int64(0)
    _check(lib().lra_bin_export(plan, _dev(ix), _dev(iy), _dev(fx), _dev(fy), _dev(key), _dev(perm), _dev(tile_start),
                                C.byref(nv)), plan)
    return int(nv.value)


def lra_grid(plan: int, vis, wt, tau, grid, sumwt=None):
    import torch
    _check(lib().lra_grid(plan, _dev(vis, torch.complex64, plan), _dev(wt, torch.float32, plan), _dev(tau, torch.float32, plan),
                          _dev(grid, torch.complex64, plan), _dev(sumwt, torch.float64, plan)), plan)


def lra_degrid(plan: int, grid, tau, vis_in, vis_out):
    import torch
    _check(lib().lra_degrid(plan, _dev(grid, torch.complex64, plan), _dev(tau, torch.float32, plan),
                            _dev(vis_in, torch.complex64, plan), _dev(vis_out, torch.complex64, plan)), plan)


def lra_image(plan: int, grid, sumwt, corr_x, corr_y, image):
    """grid complex64 [nterms, ncorr, ny, nx] -> image float32 of the same shape (lra.h: lra_image)."""
    import torch
    _check(lib().lra_image(plan, _dev(grid, torch.complex64, plan), _dev(sumwt, torch.float64, plan),
                           _dev(corr_x, torch.float32, plan), _dev(corr_y, torch.float32, plan),
                           _dev(image, torch.float32, plan)), plan)


def lra_model_grid(plan: int, image, corr_x, corr_y, grid):
    """image float32 [nterms, ncorr, ny, nx] -> grid complex64 of the same shape (lra.h: lra_model_grid)."""
    import torch
    _check(lib().lra_model_grid(plan, _dev(image, torch.float32, plan), _dev(corr_x, torch.float32, plan),
                                _dev(corr_y, torch.float32, plan), _dev(grid, torch.complex64, plan)), plan)


def lra_gain_accumulate(vis, model, wt, nbl, xsum, wsum, bl_index=None, stream=None):
    """Eq. 19: xsum complex128 [nbl, ncorr] and wsum float64 [nbl, ncorr] are accumulated into (lra.h)."""
    import torch
    nrow, nchan, ncorr = (int(x) for x in vis.shape)
    if tuple(model.shape) != (nrow, nchan, ncorr) or tuple(wt.shape) != (nrow, nchan, ncorr):
        raise LraError("vis, model and wt must share the shape [nrow, nchan, ncorr]")
    if tuple(xsum.shape) != (nbl, ncorr) or tuple(wsum.shape) != (nbl, ncorr):
        raise LraError("xsum / wsum must be [nbl, ncorr]")
    _check(lib().lra_gain_accumulate(vis.device.index, stream or 0, nrow, nchan, ncorr, nbl, _dev(bl_index, torch.int32),
                                     _dev(vis, torch.complex64), _dev(model, torch.complex64), _dev(wt, torch.float32),
                                     _dev(xsum, torch.complex128), _dev(wsum, torch.float64)))


def lra_gain_solve(ant1, ant2, xsum, wsum, alpha, delta, max_iter, gains, iters=None, stream=None):
    """Eq. 20 / 21: gains complex128 [nant, ncorr] updated in place; iters: int32 CUDA tensor of one element or None."""
    import torch
    nant, ncorr = (int(x) for x in gains.shape)
    _check(lib().lra_gain_solve(gains.device.index, stream or 0, nant, int(ant1.shape[0]), ncorr, _dev(ant1, torch.int32),
                                _dev(ant2, torch.int32), _dev(xsum, torch.complex128), _dev(wsum, torch.float64), float(alpha),
                                float(delta), int(max_iter), _dev(gains, torch.complex128), _dev(iters, torch.int32)))


def lra_cf_generate(cf_data, n_img, oversampling, fov_rad, cf_support, cf_offset, taper=None, aterm=None, cf_w=None,
                    cf_aterm=None, normalise=True, stream=None):
    """Table 1 / PreCompute (lra.h: lra_cf_generate).  cf_data: CUDA complex64 flat tensor written at cf_offset;
    taper: CUDA float64 [n_img] or None; aterm: CUDA complex64 [n_aterm, n_img, n_img] or None; cf_support, cf_offset,
    cf_w (or None), cf_aterm (or None): HOST arrays [n_cf]."""
    import torch
    sup = _host(cf_support, np.int32)
    off = _host(cf_offset, np.int64)
    w = None if cf_w is None else _host(cf_w, np.float64)
    ia = None if cf_aterm is None else _host(cf_aterm, np.int32)
    n_cf = len(sup)
    if len(off) != n_cf or (w is not None and len(w) != n_cf) or (ia is not None and len(ia) != n_cf):
        raise LraError("cf_support, cf_offset, cf_w and cf_aterm must have one entry per kernel")
    if n_cf and int((off + (sup.astype(np.int64) * oversampling) ** 2).max()) > cf_data.numel():
        raise LraError("cf_data is too small for the offsets given")
    dev = cf_data.device.index
    for t in (taper, aterm):
        if t is not None and t.device.index != dev:
            raise LraError("taper / aterm must be on cf_data's device")
    if taper is not None and tuple(taper.shape) != (n_img,):
        raise LraError(f"taper must be [n_img], got {tuple(taper.shape)}")
    if aterm is not None and (aterm.dim() != 3 or tuple(aterm.shape[1:]) != (n_img, n_img)):
        raise LraError(f"aterm must be [n_aterm, n_img, n_img], got {tuple(aterm.shape)}")
    d = lra_cf_desc(n_img, oversampling, float(fov_rad), _dev(taper, torch.float64), 0 if aterm is None else int(aterm.shape[0]),
                    _dev(aterm, torch.complex64), n_cf, sup.ctypes.data, off.ctypes.data, None if w is None else w.ctypes.data,
                    None if ia is None else ia.ctypes.data, 1 if normalise else 0, dev, stream or 0)
    rc = lib().lra_cf_generate(C.byref(d), _dev(cf_data, torch.complex64))
    if rc != LRA_OK:
        raise LraError(f"{lib().lra_strerror(rc).decode()} (cudaError {lib().lra_cf_last_cuda_error()})")


def _po(po_table, po_index, plan, nrow=None):
    import torch
    t = _host(po_table, np.float64).reshape(-1, 3)
    if po_index is not None and nrow is not None and tuple(po_index.shape) != (nrow,):
        raise LraError(f"po_index must be [nrow], got {tuple(po_index.shape)}")
    return t, len(t), _dev(po_index, torch.int32, plan)


def lra_phase_gradient(plan: int, src, f, dl, dm, dst, conjugate=False, accumulate=False):
    """dst (+)= f e^{+-2 pi i (dl u_X + dm v_Y)} src over all planes (lra.h: lra_phase_gradient)."""
    import torch
    if src.shape != dst.shape:
        raise LraError("src and dst must have the same shape")
    _check(lib().lra_phase_gradient(plan, _dev(src, torch.complex64, plan), float(f), float(dl), float(dm),
                                    1 if conjugate else 0, 1 if accumulate else 0, _dev(dst, torch.complex64, plan)), plan)


def lra_phase_gradient_static(src, scale_u, scale_v, f, dl, dm, dst, conjugate=False, accumulate=False, stream=None):
    """lra_phase_gradient without a plan and without any allocation (lra.h: lra_phase_gradient_static): src, dst CUDA
    complex64 [..., ny, nx] on the current device; enqueued on `stream` (a torch.cuda.Stream; default: the current one)."""
    import torch
    if src.shape != dst.shape or src.dim() < 2:
        raise LraError("src and dst must have the same shape [..., ny, nx]")
    if src.device != dst.device or src.device.index != torch.cuda.current_device():
        raise LraError("src and dst must live on the current CUDA device")
    ny, nx = int(src.shape[-2]), int(src.shape[-1])
    nplanes = int(src.numel() // (nx * ny)) if nx * ny else 0
    s = stream if stream is not None else torch.cuda.current_stream()
    rc = lib().lra_phase_gradient_static(nx, ny, nplanes, float(scale_u), float(scale_v), _dev(src, torch.complex64), float(f),
                                         float(dl), float(dm), 1 if conjugate else 0, 1 if accumulate else 0,
                                         _dev(dst, torch.complex64), s.cuda_stream)
    if rc != LRA_OK:
        raise LraError(f"liblra: {lib().lra_strerror(rc).decode()} ({lra_static_last_error()}) [code {rc}]")


def lra_static_last_error() -> str:
    """Description of this thread's last lra_phase_gradient_static failure ("" after a success)."""
    return lib().lra_static_last_error().decode()


def lra_grid_po(plan: int, vis, wt, tau, po_table, po_index, grid, sumwt=None):
    """lra_grid with the pointing term of Eq. 27: po_table HOST [n_po, 3] = (f, dl, dm); po_index CUDA int32 [nrow] or None."""
    import torch
    t, n_po, pi = _po(po_table, po_index, plan, int(vis.shape[0]))
    _check(lib().lra_grid_po(plan, _dev(vis, torch.complex64, plan), _dev(wt, torch.float32, plan), _dev(tau, torch.float32, plan),
                             n_po, t.ctypes.data, pi, _dev(grid, torch.complex64, plan), _dev(sumwt, torch.float64, plan)), plan)


def lra_degrid_po(plan: int, grid, tau, po_table, po_index, vis_in, vis_out):
    import torch
    t, n_po, pi = _po(po_table, po_index, plan, int(vis_out.shape[0]))
    _check(lib().lra_degrid_po(plan, _dev(grid, torch.complex64, plan), _dev(tau, torch.float32, plan), n_po, t.ctypes.data, pi,
                               _dev(vis_in, torch.complex64, plan), _dev(vis_out, torch.complex64, plan)), plan)


def _mueller(plan, elems, cf_indices):
    import torch
    eg = _host([e[0] for e in elems], np.int32)
    ec = _host([e[1] for e in elems], np.int32)
    if len(cf_indices) != len(elems):
        raise LraError("one cf_index (or None) per element")
    ptrs = (C.c_void_p * len(elems))(*[_dev(a, torch.int32, plan) for a in cf_indices])
    return eg, ec, ptrs


def lra_grid_mueller(plan: int, uvw_m, freq_hz, elems, cf_indices, vis, wt, tau, grid, sumwt=None, po_table=None, po_index=None):
    """Sparse Mueller gridding (lra.h: lra_grid_mueller).  elems: [(grid plane, visibility correlation)]; cf_indices: one
    CUDA int32 [nrow, nchan] (or None) per element; vis, wt CUDA [nrow, nchan, ncorr_vis]; grid CUDA complex64 [ngrid, ny, nx]."""
    import torch
    f = _host(freq_hz, np.float64)
    nrow, nchan = int(uvw_m.shape[0]), len(f)
    if tuple(vis.shape[:2]) != (nrow, nchan) or vis.shape != wt.shape or grid.dim() != 3:
        raise LraError("vis / wt must be [nrow, nchan, ncorr_vis], grid [ngrid, ny, nx]")
    eg, ec, ptrs = _mueller(plan, elems, cf_indices)
    t, n_po, pi = (None, 0, None) if po_table is None else _po(po_table, po_index, plan, nrow)
    _check(lib().lra_grid_mueller(plan, nrow, nchan, _dev(uvw_m, torch.float64, plan), f.ctypes.data, len(eg), eg.ctypes.data,
                                  ec.ctypes.data, ptrs, int(vis.shape[2]), _dev(vis, torch.complex64, plan),
                                  _dev(wt, torch.float32, plan), _dev(tau, torch.float32, plan), n_po,
                                  None if t is None else t.ctypes.data, pi, int(grid.shape[0]), _dev(grid, torch.complex64, plan),
                                  _dev(sumwt, torch.float64, plan)), plan)


def lra_degrid_mueller(plan: int, uvw_m, freq_hz, elems, cf_indices, grid, tau, vis_in, vis_out, po_table=None, po_index=None):
    import torch
    f = _host(freq_hz, np.float64)
    nrow, nchan = int(uvw_m.shape[0]), len(f)
    if tuple(vis_out.shape[:2]) != (nrow, nchan) or grid.dim() != 3 or (vis_in is not None and vis_in.shape != vis_out.shape):
        raise LraError("vis must be [nrow, nchan, ncorr_vis], grid [ngrid, ny, nx]")
    eg, ec, ptrs = _mueller(plan, elems, cf_indices)
    t, n_po, pi = (None, 0, None) if po_table is None else _po(po_table, po_index, plan, nrow)
    _check(lib().lra_degrid_mueller(plan, nrow, nchan, _dev(uvw_m, torch.float64, plan), f.ctypes.data, len(eg), eg.ctypes.data,
                                    ec.ctypes.data, ptrs, int(vis_out.shape[2]), int(grid.shape[0]),
                                    _dev(grid, torch.complex64, plan), _dev(tau, torch.float32, plan), n_po,
                                    None if t is None else t.ctypes.data, pi, _dev(vis_in, torch.complex64, plan),
                                    _dev(vis_out, torch.complex64, plan)), plan)


def lra_cf_last_cuda_error() -> int:
    """cudaError_t of the calling thread's last lra_cf_generate failure (0 = none)."""
    return int(lib().lra_cf_last_cuda_error())


def lra_launch_count(plan: int) -> int:
    return int(lib().lra_launch_count(plan))


def lra_tap_count(plan: int):
    """-> (n_valid, sum over valid points of S^2)."""
    a, b = C.c_int64(0), C.c_int64(0)
    _check(lib().lra_tap_count(plan, C.byref(a), C.byref(b)), plan)
    return int(a.value), int(b.value)


def lra_set_variant(plan: int, grid_variant: int = 0, degrid_variant: int = 0):
    _check(lib().lra_set_variant(plan, grid_variant, degrid_variant), plan)


def lra_diag_fma_tflops(device: int = 0) -> float:
    v = C.c_double(0)
    _check(lib().lra_diag_fma_tflops(device, C.byref(v)))
    return float(v.value)


def lra_diag_l2_gbs(device: int = 0, mbytes: int = 64) -> float:
    v = C.c_double(0)
    _check(lib().lra_diag_l2_gbs(device, mbytes, C.byref(v)))
    return float(v.value)


def lra_strerror(code: int) -> str:
    return lib().lra_strerror(code).decode()
