"""Thin Python binding of libapic (include/apic.h): argument marshalling only.

Every step of the reconstruction runs in the CUDA kernels of ``libapic.so``; PyTorch supplies
device memory and streams.  There is no CPU fallback: importing works without a GPU (so the
symbol table and the host-only geometry can be tested), but ``Plan(...)`` raises ``ApicError``
when no CUDA device is usable, and a missing ``libapic.so`` raises at ``load()``.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path
from typing import Optional, Sequence

import numpy as np

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libapic.so"

APIC_OK, APIC_EINVAL, APIC_ECUDA, APIC_ENOMEM, APIC_EBATCH, APIC_ESCRATCH = 0, -1, -2, -3, -4, -5
TILE_OK, TILE_BACKGROUND, TILE_BAD_INPUT, TILE_SOLVE_FAILED = 0, 1, 2, 3
DBG_SUBSPECTRA, DBG_OBJECT_SPECTRUM, DBG_DF_ITERS = 0, 1, 2

EXPORTS = ("apic_params_default", "apic_plan_create", "apic_plan_destroy", "apic_plan_info",
           "apic_geometry_info", "apic_geometry_dark_grids", "apic_plan_dark_sets", "apic_reconstruct", "apic_reconstruct_host", "apic_reconstruct_u16", "apic_reconstruct_host_u16",
           "apic_submit_host", "apic_submit_host_u16", "apic_wait_host",
           "apic_debug_buffer", "apic_debug_copy", "apic_fft2d", "apic_fft2d_xy", "apic_last_launch_count", "apic_strerror",
           "apic_last_cuda_error", "apic_version", "apic_profile_categories", "apic_profile_category_name",
           "apic_profile_begin", "apic_profile_end", "apic_profile_work", "apic_measure_peak", "apic_reassemble",
           "apic_reassemble_work_bytes", "apic_reassemble_static", "apic_reassemble_static_max_tiles",
           "apic_pupil_field_fit", "apic_reconstruct_prior")


class ApicError(RuntimeError):
    pass


class ApicParams(C.Structure):
    _fields_ = [("tile_n", C.c_int), ("upsample", C.c_int), ("wavelength_um", C.c_double),
                ("pixel_um", C.c_double), ("na_obj", C.c_double), ("n_bright", C.c_int),
                ("k_bright", C.POINTER(C.c_double)), ("n_dark", C.c_int), ("k_dark", C.POINTER(C.c_double)),
                ("n_zernike", C.c_int), ("noll", C.POINTER(C.c_int)), ("kk_pad", C.c_int),
                ("refine_iters", C.c_int), ("df_iters", C.c_int), ("df_tol", C.c_float),
                ("intensity_floor", C.c_float), ("bg_mode", C.c_int), ("bg_threshold", C.c_float),
                ("max_batch", C.c_int), ("chunk_tiles", C.c_int), ("df_mode", C.c_int), ("df_team", C.c_int),
                ("df_order", C.c_int)]


class PlanInfo(C.Structure):
    _fields_ = [("tile_n", C.c_int), ("upsample", C.c_int), ("out_n", C.c_int), ("n_bright", C.c_int),
                ("n_dark", C.c_int), ("n_zernike", C.c_int), ("n_pairs", C.c_int), ("n_rows", C.c_int),
                ("n_grad_rows", C.c_int), ("n_union", C.c_int), ("n_known", C.c_int), ("n_dark_used", C.c_int),
                ("max_unknown", C.c_int), ("max_equations", C.c_int), ("chunk_tiles", C.c_int),
                ("table_bytes", C.c_size_t), ("workspace_bytes", C.c_size_t), ("radius_bins", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None


def load() -> C.CDLL:
    """dlopen libapic.so (built by ``python -m paper_2407_20469_b200.build``)."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise ApicError(f"{LIB_PATH} is missing: build it with `python -m paper_2407_20469_b200.build` "
                        "(CUDA-only library, no CPU fallback)")
    lib = C.CDLL(str(LIB_PATH))
    lib.apic_params_default.argtypes = [C.POINTER(ApicParams)]
    lib.apic_params_default.restype = None
    lib.apic_plan_create.argtypes = [C.POINTER(ApicParams), C.POINTER(C.c_void_p)]
    lib.apic_plan_destroy.argtypes = [C.c_void_p]
    lib.apic_plan_info.argtypes = [C.c_void_p, C.POINTER(PlanInfo)]
    lib.apic_geometry_info.argtypes = [C.POINTER(ApicParams), C.POINTER(PlanInfo), C.POINTER(C.c_int),
                                       C.POINTER(C.c_int), C.POINTER(C.c_int), C.c_int]
    lib.apic_geometry_dark_grids.argtypes = [C.POINTER(ApicParams), C.POINTER(C.c_int), C.POINTER(C.c_int), C.c_int]
    lib.apic_plan_dark_sets.argtypes = [C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int)]
    lib.apic_reconstruct.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_void_p, C.c_void_p]
    lib.apic_reconstruct_host.argtypes = lib.apic_reconstruct.argtypes
    lib.apic_reconstruct_u16.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                                         C.c_void_p, C.c_void_p]
    lib.apic_reconstruct_host_u16.argtypes = lib.apic_reconstruct_u16.argtypes
    lib.apic_submit_host.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.apic_submit_host_u16.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p,
                                         C.c_void_p, C.c_void_p]
    lib.apic_wait_host.argtypes = [C.c_void_p, C.c_int]
    lib.apic_debug_buffer.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_void_p), C.POINTER(C.c_size_t)]
    lib.apic_debug_copy.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_void_p]
    lib.apic_fft2d.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p]
    lib.apic_fft2d_xy.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p]
    lib.apic_last_launch_count.argtypes = [C.c_void_p]
    for name in ("apic_strerror", "apic_last_cuda_error", "apic_version"):
        getattr(lib, name).restype = C.c_char_p
    lib.apic_strerror.argtypes = [C.c_int]
    lib.apic_profile_category_name.restype = C.c_char_p
    lib.apic_profile_category_name.argtypes = [C.c_int]
    lib.apic_profile_begin.argtypes = [C.c_void_p, C.c_int, C.c_int]
    lib.apic_profile_end.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_longlong),
                                     C.POINTER(C.c_longlong)]
    lib.apic_profile_work.argtypes = [C.c_void_p, C.POINTER(C.c_ulonglong)]
    lib.apic_measure_peak.argtypes = [C.c_int, C.POINTER(C.c_double), C.c_void_p]
    lib.apic_pupil_field_fit.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p,
                                         C.c_void_p]
    lib.apic_reconstruct_prior.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                                           C.c_void_p, C.c_void_p]
    lib.apic_reassemble_work_bytes.argtypes = [C.c_int, C.c_int]
    lib.apic_reassemble_work_bytes.restype = C.c_size_t
    lib.apic_reassemble.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                                    C.c_void_p]
    lib.apic_reassemble_static_max_tiles.argtypes = []
    lib.apic_reassemble_static.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p,
                                           C.c_void_p]
    _lib = lib
    return lib


def _check(rc: int, what: str):
    if rc != APIC_OK:
        lib = load()
        msg = lib.apic_strerror(rc).decode()
        if rc == APIC_ECUDA:
            msg += ": " + lib.apic_last_cuda_error().decode()
        raise ApicError(f"{what} failed ({rc}): {msg}")


def make_params(tile_n: int, upsample: int, wavelength_um: float, pixel_um: float, na_obj: float,
                k_bright, k_dark, noll: Sequence[int], **opts):
    """Returns (ApicParams, keep-alive tuple).  ``opts``: kk_pad, refine_iters, df_iters, df_tol,
    intensity_floor, bg_mode, bg_threshold, max_batch, chunk_tiles, df_mode, df_team, df_order."""
    lib = load()
    p = ApicParams()
    lib.apic_params_default(C.byref(p))
    kb = np.ascontiguousarray(np.asarray(k_bright, dtype=np.float64).reshape(-1, 2))
    kd = np.ascontiguousarray(np.asarray(k_dark if k_dark is not None else [], dtype=np.float64).reshape(-1, 2))
    nl = np.ascontiguousarray(np.asarray(list(noll), dtype=np.int32))
    p.tile_n, p.upsample = int(tile_n), int(upsample)
    p.wavelength_um, p.pixel_um, p.na_obj = float(wavelength_um), float(pixel_um), float(na_obj)
    p.n_bright, p.k_bright = kb.shape[0], kb.ctypes.data_as(C.POINTER(C.c_double))
    p.n_dark = kd.shape[0]
    p.k_dark = kd.ctypes.data_as(C.POINTER(C.c_double)) if kd.shape[0] else None
    p.n_zernike, p.noll = nl.shape[0], nl.ctypes.data_as(C.POINTER(C.c_int))
    for k, v in opts.items():
        if not hasattr(p, k):
            raise TypeError(f"unknown apic_params field {k!r}")
        setattr(p, k, v)
    return p, (kb, kd, nl)


def geometry_info(params: ApicParams, max_dark: int = 256):
    """Host-only geometry counts (no GPU needed): (info dict, [(led, |U|, |Q|), ...])."""
    lib = load()
    info = PlanInfo()
    led = (C.c_int * max_dark)()
    nu = (C.c_int * max_dark)()
    nq = (C.c_int * max_dark)()
    _check(lib.apic_geometry_info(C.byref(params), C.byref(info), led, nu, nq, max_dark), "apic_geometry_info")
    n = min(info.n_dark_used, max_dark)
    return info.as_dict(), [(led[i], nu[i], nq[i]) for i in range(n)]


def geometry_dark_grids(params: ApicParams, max_dark: int = 256):
    """Host-only: [(mx, my), ...] reduced cyclic grids of the used darkfield LEDs, processing order."""
    lib = load()
    info, dark = geometry_info(params, max_dark)
    mx, my = (C.c_int * max_dark)(), (C.c_int * max_dark)()
    _check(lib.apic_geometry_dark_grids(C.byref(params), mx, my, max_dark), "apic_geometry_dark_grids")
    return [(mx[i], my[i]) for i in range(len(dark))]


class Plan:
    """apic_plan wrapper.  Tensors are torch CUDA tensors; the current torch stream is used."""

    def __init__(self, tile_n, upsample, wavelength_um, pixel_um, na_obj, k_bright, k_dark, noll, **opts):
        self._lib = load()
        self.params, self._keep = make_params(tile_n, upsample, wavelength_um, pixel_um, na_obj, k_bright,
                                              k_dark, noll, **opts)
        self._h = C.c_void_p()
        _check(self._lib.apic_plan_create(C.byref(self.params), C.byref(self._h)), "apic_plan_create")
        info = PlanInfo()
        _check(self._lib.apic_plan_info(self._h, C.byref(info)), "apic_plan_info")
        self.info = info.as_dict()
        self.n, self.u, self.out_n = info.tile_n, info.upsample, info.out_n
        self.n_img = info.n_bright + info.n_dark
        self.nz = info.n_zernike

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.apic_plan_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def dark_sets(self):
        n = self.info["n_dark_used"]
        led, nu, nq = (C.c_int * max(n, 1))(), (C.c_int * max(n, 1))(), (C.c_int * max(n, 1))()
        _check(self._lib.apic_plan_dark_sets(self._h, led, nu, nq), "apic_plan_dark_sets")
        return [(led[i], nu[i], nq[i]) for i in range(n)]

    def reconstruct(self, intensity, want_pupil: bool = True, out=None, zernike_init=None):
        """intensity: float32 CUDA tensor [B][n_img][N][N].  Returns (field complex64 [B][uN][uN],
        zernike float32 [B][nz], pupil complex64 [B][N][N] | None, status int32 [B]).
        zernike_init: float32 CUDA tensor [B][nz], a prior that replaces the start of the aberration fit
        (apic_reconstruct_prior)."""
        import torch
        if not (intensity.is_cuda and intensity.dtype == torch.float32 and intensity.is_contiguous()):
            raise ApicError("intensity must be a contiguous float32 CUDA tensor")
        b = intensity.shape[0]
        if tuple(intensity.shape[1:]) != (self.n_img, self.n, self.n):
            raise ApicError(f"intensity shape {tuple(intensity.shape)} != [B,{self.n_img},{self.n},{self.n}]")
        dev = intensity.device
        if out is None:
            field = torch.empty((b, self.out_n, self.out_n), dtype=torch.complex64, device=dev)
            zern = torch.empty((b, self.nz), dtype=torch.float32, device=dev)
            pupil = torch.empty((b, self.n, self.n), dtype=torch.complex64, device=dev) if want_pupil else None
            status = torch.empty((b,), dtype=torch.int32, device=dev)
        else:
            field, zern, pupil, status = out
        stream = torch.cuda.current_stream(dev).cuda_stream
        if zernike_init is not None:
            if not (zernike_init.is_cuda and zernike_init.dtype == torch.float32 and zernike_init.is_contiguous()
                    and tuple(zernike_init.shape) == (b, self.nz)):
                raise ApicError(f"zernike_init must be a contiguous float32 CUDA tensor [{b},{self.nz}]")
            _check(self._lib.apic_reconstruct_prior(self._h, intensity.data_ptr(), zernike_init.data_ptr(), b, field.data_ptr(),
                                                    zern.data_ptr(), pupil.data_ptr() if pupil is not None else None,
                                                    status.data_ptr(), C.c_void_p(stream)), "apic_reconstruct_prior")
            return field, zern, pupil, status
        _check(self._lib.apic_reconstruct(self._h, intensity.data_ptr(), b, field.data_ptr(), zern.data_ptr(),
                                          pupil.data_ptr() if pupil is not None else None, status.data_ptr(),
                                          C.c_void_p(stream)), "apic_reconstruct")
        return field, zern, pupil, status

    def reconstruct_u16(self, raw, scale, want_pupil: bool = True, out=None):
        """raw: uint16 CUDA tensor [B][n_img][N][N] (camera counts), scale: float32 CUDA tensor [B][n_img]
        (intensity = count * scale).  Returns the same tuple as ``reconstruct``."""
        import torch
        if not (raw.is_cuda and raw.dtype == torch.uint16 and raw.is_contiguous()):
            raise ApicError("raw must be a contiguous uint16 CUDA tensor")
        b = raw.shape[0]
        if tuple(raw.shape[1:]) != (self.n_img, self.n, self.n):
            raise ApicError(f"raw shape {tuple(raw.shape)} != [B,{self.n_img},{self.n},{self.n}]")
        if not (scale.is_cuda and scale.dtype == torch.float32 and scale.is_contiguous()
                and tuple(scale.shape) == (b, self.n_img)):
            raise ApicError(f"scale must be a contiguous float32 CUDA tensor [{b},{self.n_img}]")
        dev = raw.device
        if out is None:
            field = torch.empty((b, self.out_n, self.out_n), dtype=torch.complex64, device=dev)
            zern = torch.empty((b, self.nz), dtype=torch.float32, device=dev)
            pupil = torch.empty((b, self.n, self.n), dtype=torch.complex64, device=dev) if want_pupil else None
            status = torch.empty((b,), dtype=torch.int32, device=dev)
        else:
            field, zern, pupil, status = out
        stream = torch.cuda.current_stream(dev).cuda_stream
        _check(self._lib.apic_reconstruct_u16(self._h, raw.data_ptr(), scale.data_ptr(), b, field.data_ptr(),
                                              zern.data_ptr(), pupil.data_ptr() if pupil is not None else None,
                                              status.data_ptr(), C.c_void_p(stream)), "apic_reconstruct_u16")
        return field, zern, pupil, status

    def _host_ptrs(self, b, named):
        """Checks dtype, C-contiguity and exact shape of every host buffer before its raw pointer crosses the ABI."""
        import torch
        np_of = {torch.float32: np.float32, torch.complex64: np.complex64, torch.int32: np.int32, torch.uint16: np.uint16}
        out = []
        for name, a, dtype, shape in named:
            if a is None:
                out.append(None)
                continue
            if isinstance(a, np.ndarray):
                ok = a.dtype == dtype and a.flags["C_CONTIGUOUS"] and tuple(a.shape) == shape
                p = a.ctypes.data
            elif isinstance(a, torch.Tensor):
                ok = (not a.is_cuda and np_of.get(a.dtype) == dtype and a.is_contiguous() and tuple(a.shape) == shape)
                p = a.data_ptr()
            else:
                ok, p = False, None
            if not ok:
                raise ApicError(f"{name} must be a C-contiguous host array of dtype {np.dtype(dtype).name} and shape {shape}")
            out.append(p)
        return out

    def _host_outputs(self, b, field, zern, pupil, status):
        return [("field", field, np.complex64, (b, self.out_n, self.out_n)), ("zernike", zern, np.float32, (b, self.nz)),
                ("pupil", pupil, np.complex64, (b, self.n, self.n)), ("status", status, np.int32, (b,))]

    def reconstruct_host_u16(self, raw, scale, field, zern, pupil, status, stream: int = 0):
        """Host buffers (numpy arrays or CPU torch tensors, ideally pinned); blocking."""
        b = int(raw.shape[0])
        p = self._host_ptrs(b, [("raw", raw, np.uint16, (b, self.n_img, self.n, self.n)),
                                ("scale", scale, np.float32, (b, self.n_img))] + self._host_outputs(b, field, zern, pupil, status))
        _check(self._lib.apic_reconstruct_host_u16(self._h, p[0], p[1], b, p[2], p[3], p[4], p[5], C.c_void_p(stream)),
               "apic_reconstruct_host_u16")

    def reconstruct_host(self, intensity, field, zern, pupil, status, stream: int = 0):
        """Host buffers (numpy arrays or CPU torch tensors, ideally pinned); blocking."""
        b = int(intensity.shape[0])
        p = self._host_ptrs(b, [("intensity", intensity, np.float32, (b, self.n_img, self.n, self.n))]
                            + self._host_outputs(b, field, zern, pupil, status))
        _check(self._lib.apic_reconstruct_host(self._h, p[0], b, p[1], p[2], p[3], p[4], C.c_void_p(stream)),
               "apic_reconstruct_host")

    def submit_host(self, slot: int, intensity, field, zern, pupil, status):
        """Streaming form of reconstruct_host: enqueues upload, kernels and download of one batch in pipeline slot
        0 or 1 and returns; wait_host(slot) blocks until the results are in the (pinned) host buffers."""
        b = int(intensity.shape[0])
        p = self._host_ptrs(b, [("intensity", intensity, np.float32, (b, self.n_img, self.n, self.n))]
                            + self._host_outputs(b, field, zern, pupil, status))
        _check(self._lib.apic_submit_host(self._h, slot, p[0], b, p[1], p[2], p[3], p[4]), "apic_submit_host")

    def submit_host_u16(self, slot: int, raw, scale, field, zern, pupil, status):
        b = int(raw.shape[0])
        p = self._host_ptrs(b, [("raw", raw, np.uint16, (b, self.n_img, self.n, self.n)),
                                ("scale", scale, np.float32, (b, self.n_img))] + self._host_outputs(b, field, zern, pupil, status))
        _check(self._lib.apic_submit_host_u16(self._h, slot, p[0], p[1], b, p[2], p[3], p[4], p[5]), "apic_submit_host_u16")

    def wait_host(self, slot: int):
        _check(self._lib.apic_wait_host(self._h, slot), "apic_wait_host")

    def debug_buffer(self, which: int, tiles: int):
        """Stage-level buffers of the last chunk as torch tensors (copies)."""
        import torch
        p, nbytes = C.c_void_p(), C.c_size_t()
        _check(self._lib.apic_debug_buffer(self._h, which, C.byref(p), C.byref(nbytes)), "apic_debug_buffer")
        total = nbytes.value * tiles
        out = torch.empty(total, dtype=torch.uint8, device="cuda")
        stream = torch.cuda.current_stream().cuda_stream
        _check(self._lib.apic_debug_copy(self._h, which, out.data_ptr(), tiles, C.c_void_p(stream)),
               "apic_debug_copy")
        if which == DBG_DF_ITERS:
            return out.view(torch.int32).view(tiles, -1)
        return out.view(torch.complex64).view(tiles, -1)

    def profile_begin(self, stride: int = 1, max_samples: int = 8192):
        _check(self._lib.apic_profile_begin(self._h, stride, max_samples), "apic_profile_begin")

    def profile_end(self):
        """{kernel: (ms summed over the sampled launches, sampled launches, all launches)}"""
        n = self._lib.apic_profile_categories()
        ms, sm, la = (C.c_double * n)(), (C.c_longlong * n)(), (C.c_longlong * n)()
        _check(self._lib.apic_profile_end(self._h, ms, sm, la), "apic_profile_end")
        return {self._lib.apic_profile_category_name(i).decode(): (ms[i], sm[i], la[i]) for i in range(n)}

    def profile_work(self) -> int:
        """N-point line transforms executed by the persistent darkfield kernels since profile_begin."""
        v = C.c_ulonglong()
        _check(self._lib.apic_profile_work(self._h, C.byref(v)), "apic_profile_work")
        return int(v.value)

    @property
    def last_launch_count(self) -> int:
        return int(self._lib.apic_last_launch_count(self._h))


def measure_peak(what: int) -> float:
    """apic_measure_peak on the current device: 0 fp32 FFMA flop/s, 1 fp32 FADD flop/s, 2 shared-memory bytes/s."""
    import torch
    v = C.c_double()
    _check(load().apic_measure_peak(int(what), C.byref(v), C.c_void_p(torch.cuda.current_stream().cuda_stream)),
           "apic_measure_peak")
    return float(v.value)


def pupil_field_fit(zernike, status, xy, order: int = 2):
    """apic_pupil_field_fit: zernike float32 CUDA [T][nz], status int32 CUDA [T], xy float32 CUDA [T][2].
    Returns (fit float32 [T][nz], poly float32 [6][nz])."""
    import torch
    t, nz = int(zernike.shape[0]), int(zernike.shape[1])
    if not (zernike.is_cuda and zernike.dtype == torch.float32 and zernike.is_contiguous()
            and status.is_cuda and status.dtype == torch.int32 and status.is_contiguous() and tuple(status.shape) == (t,)
            and xy.is_cuda and xy.dtype == torch.float32 and xy.is_contiguous() and tuple(xy.shape) == (t, 2)):
        raise ApicError("zernike float32 [T][nz], status int32 [T], xy float32 [T][2]: contiguous CUDA tensors")
    fit = torch.empty_like(zernike)
    poly = torch.empty((6, nz), dtype=torch.float32, device=zernike.device)
    stream = torch.cuda.current_stream(zernike.device).cuda_stream
    _check(load().apic_pupil_field_fit(zernike.data_ptr(), status.data_ptr(), xy.data_ptr(), t, nz, int(order), fit.data_ptr(),
                                       poly.data_ptr(), C.c_void_p(stream)), "apic_pupil_field_fit")
    return fit, poly


def reassemble(fields, overlap: int, align: bool = True, out=None):
    """apic_reassemble: fields = complex64 CUDA tensor [tiles_y][tiles_x][T][T] (reconstructed tiles on a regular grid
    sharing `overlap` pixels).  Returns (fov complex64 [H][W], factors complex64 [tiles_y][tiles_x])."""
    import torch
    if not (fields.is_cuda and fields.dtype == torch.complex64 and fields.is_contiguous() and fields.dim() == 4
            and fields.shape[2] == fields.shape[3]):
        raise ApicError("fields must be a contiguous complex64 CUDA tensor [tiles_y][tiles_x][T][T]")
    ty, tx, t = int(fields.shape[0]), int(fields.shape[1]), int(fields.shape[2])
    overlap = int(overlap)
    if overlap < 0 or 2 * overlap > t:
        raise ApicError("overlap must satisfy 0 <= 2 overlap <= T")
    lib = load()
    h, w = ty * (t - overlap) + overlap, tx * (t - overlap) + overlap
    fov = out if out is not None else torch.empty((h, w), dtype=torch.complex64, device=fields.device)
    if not (fov.is_cuda and fov.dtype == torch.complex64 and fov.is_contiguous() and tuple(fov.shape) == (h, w)):
        raise ApicError("out must be a contiguous complex64 CUDA tensor [H][W]")
    factors = torch.empty((ty, tx), dtype=torch.complex64, device=fields.device)
    work = torch.empty((max(1, lib.apic_reassemble_work_bytes(ty, tx)),), dtype=torch.uint8, device=fields.device)
    stream = torch.cuda.current_stream(fields.device).cuda_stream
    _check(lib.apic_reassemble(fields.data_ptr(), ty, tx, t, overlap, int(bool(align)), fov.data_ptr(), factors.data_ptr(),
                               work.data_ptr(), C.c_void_p(stream)), "apic_reassemble")
    return fov, factors


def reassemble_static(fields, overlap: int, align: bool = True, out=None, factors=None):
    """apic_reassemble_static: ``reassemble`` for callers that must not allocate device memory where they reassemble
    (a process whose GPU memory is already handed out in full, or a loop that cannot afford the stall of an
    allocation).  The library keeps the scratch in a fixed array inside its own device image, so the FOV is limited
    to ``reassemble_static_max_tiles()`` tiles (ApicError with APIC_ESCRATCH beyond that), all calls on a device share
    that array (do not let two of them overlap on the GPU), and the first call on a device does a one-off, host-side
    address look-up: make it at start-up.  Pass preallocated ``out`` [H][W] and ``factors`` [tiles_y][tiles_x]
    (complex64, CUDA, contiguous) and this wrapper allocates nothing either; left out, they are created with torch
    for convenience.  Returns (fov, factors), bit-identical to ``reassemble``."""
    import torch
    if not (fields.is_cuda and fields.dtype == torch.complex64 and fields.is_contiguous() and fields.dim() == 4
            and fields.shape[2] == fields.shape[3]):
        raise ApicError("fields must be a contiguous complex64 CUDA tensor [tiles_y][tiles_x][T][T]")
    ty, tx, t = int(fields.shape[0]), int(fields.shape[1]), int(fields.shape[2])
    overlap = int(overlap)
    if overlap < 0 or 2 * overlap > t:
        raise ApicError("overlap must satisfy 0 <= 2 overlap <= T")
    h, w = ty * (t - overlap) + overlap, tx * (t - overlap) + overlap
    fov = out if out is not None else torch.empty((h, w), dtype=torch.complex64, device=fields.device)
    if not (fov.is_cuda and fov.dtype == torch.complex64 and fov.is_contiguous() and tuple(fov.shape) == (h, w)
            and fov.device == fields.device):
        raise ApicError("out must be a contiguous complex64 CUDA tensor [H][W] on the device of fields")
    u = factors if factors is not None else torch.empty((ty, tx), dtype=torch.complex64, device=fields.device)
    if not (u.is_cuda and u.dtype == torch.complex64 and u.is_contiguous() and tuple(u.shape) == (ty, tx)
            and u.device == fields.device):
        raise ApicError("factors must be a contiguous complex64 CUDA tensor [tiles_y][tiles_x] on the device of fields")
    lib = load()
    with torch.cuda.device(fields.device):      # the address look-up and the launches need the buffers' device current
        stream = torch.cuda.current_stream(fields.device).cuda_stream
        _check(lib.apic_reassemble_static(fields.data_ptr(), ty, tx, t, overlap, int(bool(align)), fov.data_ptr(),
                                          u.data_ptr(), C.c_void_p(stream)), "apic_reassemble_static")
    return fov, u


def reassemble_static_max_tiles() -> int:
    """Largest tiles_y * tiles_x that ``reassemble_static`` accepts (the size of the built-in scratch)."""
    return int(load().apic_reassemble_static_max_tiles())


def fft2d(x, inverse: bool = False):
    """In-place batched 2-D FFT of a complex64 CUDA tensor [B][n][n] by the library's own kernels."""
    import torch
    if not (x.is_cuda and x.dtype == torch.complex64 and x.is_contiguous() and x.dim() == 3
            and x.shape[1] == x.shape[2]):
        raise ApicError("x must be a contiguous complex64 CUDA tensor [B][n][n]")
    lib = load()
    stream = torch.cuda.current_stream(x.device).cuda_stream
    _check(lib.apic_fft2d(x.data_ptr(), x.shape[1], x.shape[0], int(inverse), C.c_void_p(stream)), "apic_fft2d")
    return x


def fft2d_xy(x, mode: int = 0):
    """In-place batched transform of a complex64 CUDA tensor [B][my][mx] by the reduced-grid line
    FFTs (apic_fft2d_xy: mode 0 forward, 1 inverse, 2 / 3 X-then-Y identity round trips)."""
    import torch
    if not (x.is_cuda and x.dtype == torch.complex64 and x.is_contiguous() and x.dim() == 3):
        raise ApicError("x must be a contiguous complex64 CUDA tensor [B][my][mx]")
    lib = load()
    stream = torch.cuda.current_stream(x.device).cuda_stream
    _check(lib.apic_fft2d_xy(x.data_ptr(), x.shape[2], x.shape[1], x.shape[0], int(mode), C.c_void_p(stream)),
           "apic_fft2d_xy")
    return x
