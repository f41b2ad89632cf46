"""Thin ctypes binding of libobem.so (include/obem.h).  Argument marshalling only: every step of the
path runs in the library's CUDA kernels.  torch is used for device memory and streams.

There is NO CPU fallback: if libobem.so is missing or does not load, importing this module raises;
if there is no CUDA device, `Context()` raises (obem_create -> OBEM_ECUDA).
"""
from __future__ import annotations

import ctypes
import os

from . import build as _build

NBODY = 1   # OBEM_NBODY  -- Eq (3.8)
PANELS = 2  # OBEM_PANELS -- Eq (2.13)/(2.14)
PANELS_EXACT = 4  # OBEM_PANELS_EXACT -- with PANELS: closed-form cell integrals near the target (NEXT-3)
NO_PHI = 8  # OBEM_NO_PHI -- E only (Eq 3.8 / 2.14 are field sums); the phi lane of the result is 0

_c_fp = ctypes.c_void_p  # device or host float* passed as an address
_i64 = ctypes.c_int64
_c_dp3 = ctypes.POINTER(ctypes.c_double)  # host double[3]

# every symbol include/obem.h declares: name -> (restype, argtypes)
SIGNATURES = {
    "obem_create": (ctypes.c_int, [ctypes.POINTER(ctypes.c_void_p), ctypes.c_int]),
    "obem_destroy": (ctypes.c_int, [ctypes.c_void_p]),
    "obem_reserve": (ctypes.c_int, [ctypes.c_void_p, _i64, _i64]),
    "obem_set_softening": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_float, ctypes.c_float]),
    "obem_set_panels": (ctypes.c_int, [ctypes.c_void_p, _c_fp, _c_fp, _i64, ctypes.c_void_p]),
    "obem_set_sigma": (ctypes.c_int, [ctypes.c_void_p, _c_fp, _i64, ctypes.c_void_p]),
    "obem_set_charges": (ctypes.c_int, [ctypes.c_void_p, _c_fp, _i64, ctypes.c_void_p]),
    "obem_eval_at_charges": (ctypes.c_int, [ctypes.c_void_p, _c_fp, ctypes.c_uint, ctypes.c_void_p]),
    "obem_eval_at_charges_range": (ctypes.c_int, [ctypes.c_void_p, _i64, _i64, _c_fp, ctypes.c_uint,
                                                  ctypes.c_void_p]),
    "obem_eval_at_points": (ctypes.c_int, [ctypes.c_void_p, _c_fp, _i64, _c_fp, ctypes.c_uint, ctypes.c_void_p]),
    "obem_field_at_charges_host": (ctypes.c_int, [ctypes.c_void_p, _c_fp, _i64, _c_fp, _c_fp, _i64, _c_fp,
                                                  ctypes.c_uint]),
    "obem_field_at_points_host": (ctypes.c_int, [ctypes.c_void_p, _c_fp, _i64, _c_fp, _c_fp, _i64, _c_fp,
                                                 ctypes.c_uint]),
    "obem_nbody_at_points_static": (ctypes.c_int, [_c_fp, _i64, _c_fp, _i64, ctypes.c_float, _c_fp, ctypes.c_void_p]),
    "obem_n_charges": (_i64, [ctypes.c_void_p]),
    "obem_n_panels": (_i64, [ctypes.c_void_p]),
    "obem_sm_count": (ctypes.c_int, [ctypes.c_void_p]),
    "obem_grid_size": (ctypes.c_int, [ctypes.c_void_p]),
    "obem_kernel_launches": (_i64, [ctypes.c_void_p]),
    "obem_last_cuda_error": (ctypes.c_int, [ctypes.c_void_p]),
    "obem_status_string": (ctypes.c_char_p, [ctypes.c_int]),
    "obem_get_panel_sources": (ctypes.c_int, [ctypes.c_void_p, _c_fp, ctypes.c_void_p]),
    "obem_fma_peak_probe": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, _i64, ctypes.POINTER(ctypes.c_double),
                                           ctypes.c_void_p]),
    # adjacent steps
    "obem_influence_on_panels": (ctypes.c_int, [ctypes.c_void_p, _c_fp, _c_fp, ctypes.c_void_p]),
    "obem_rhs_from_influence": (ctypes.c_int, [ctypes.c_void_p, _c_fp, _c_fp, _c_fp, _c_fp, _c_fp, _c_fp, _i64,
                                               ctypes.c_void_p]),
    "obem_apply_inverse": (ctypes.c_int, [ctypes.c_void_p, _c_fp, _i64, _i64, _c_fp, _c_fp, ctypes.c_void_p]),
    "obem_update_sigma_dynamic": (ctypes.c_int, [ctypes.c_void_p, _c_fp, _c_fp, _c_fp, _c_fp, _i64, _c_fp,
                                                 ctypes.c_void_p]),
    "obem_get_panel_normals": (ctypes.c_int, [ctypes.c_void_p, _c_fp, ctypes.c_void_p]),
    "obem_eval_panels_multi": (ctypes.c_int, [ctypes.c_void_p, _c_fp, ctypes.c_int, _c_fp, _i64, _c_fp, ctypes.c_void_p]),
    "obem_ramo_current": (ctypes.c_int, [ctypes.c_void_p, _c_fp, _c_fp, _c_fp, ctypes.c_int, _i64, _c_fp, ctypes.c_void_p]),
    # NEXT-2: recombination by-product of the N-body pass
    "obem_eval_at_charges_partners": (ctypes.c_int, [ctypes.c_void_p, _c_fp, _c_fp, _c_fp, ctypes.c_uint,
                                                     ctypes.c_void_p]),
    "obem_eval_at_charges_partners_range": (ctypes.c_int, [ctypes.c_void_p, _i64, _i64, _c_fp, _c_fp, _c_fp,
                                                           ctypes.c_uint, ctypes.c_void_p]),
    "obem_recombination_radius": (ctypes.c_double, [ctypes.c_double]),
    # NEXT-2: integrators
    "obem_push_drift": (ctypes.c_int, [ctypes.c_void_p, _c_fp, _c_fp, _i64, ctypes.c_float, ctypes.c_void_p]),
    "obem_push_kick": (ctypes.c_int, [ctypes.c_void_p, _c_fp, _c_fp, _c_fp, _i64, ctypes.c_float, ctypes.c_void_p]),
    "obem_step_euler": (ctypes.c_int, [ctypes.c_void_p, _c_fp, _c_fp, _i64, ctypes.c_float, ctypes.c_uint,
                                       ctypes.c_void_p]),
    "obem_step_pefrl": (ctypes.c_int, [ctypes.c_void_p, _c_fp, _c_fp, _i64, ctypes.c_float, ctypes.c_uint,
                                       ctypes.c_void_p]),
    # NEXT-3: near-field-accurate panels
    "obem_set_near_field": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_float]),
    "obem_near_list_size": (_i64, [ctypes.c_void_p]),
    "obem_near_cells": (_i64, [ctypes.c_void_p]),
    "obem_set_panels_cells": (ctypes.c_int, [ctypes.c_void_p, _c_fp, _c_fp, _c_fp, _i64, ctypes.c_void_p]),
    "obem_set_sigma_cells": (ctypes.c_int, [ctypes.c_void_p, _c_fp, _i64, ctypes.c_void_p]),
    "obem_set_symmetry": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.POINTER(ctypes.c_int), _c_dp3,
                                         ctypes.POINTER(ctypes.c_int)]),
    # NEXT-4: NN approximation of the N-body sum
    "obem_set_nn_theta": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_float]),
    "obem_eval_at_charges_nn": (ctypes.c_int, [ctypes.c_void_p, _c_fp, ctypes.c_uint, ctypes.c_void_p]),
    "obem_nn_last_units": (_i64, [ctypes.c_void_p, ctypes.c_void_p]),
    # NEXT-4: static field option (map + trilinear interpolation)
    "obem_field_map": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, _c_dp3, _c_dp3,
                                      _c_fp, ctypes.c_uint, ctypes.c_void_p]),
    "obem_interp_map": (ctypes.c_int, [ctypes.c_void_p, _c_fp, ctypes.c_int, ctypes.c_int, ctypes.c_int, _c_dp3,
                                       _c_dp3, _c_fp, _i64, _c_fp, ctypes.c_int, ctypes.c_void_p]),
}

LIB_PATH = _build.LIB


def load_library(path: str = LIB_PATH) -> ctypes.CDLL:
    """dlopen libobem.so and bind every declared symbol; raises if the library or a symbol is missing."""
    if not os.path.exists(path):
        raise ImportError(
            "libobem.so not found at %s: build it with `python -m paper_2110_09214_b200.build` "
            "(__graft_entry__.build()).  There is no CPU fallback." % path)
    lib = ctypes.CDLL(path)
    for name, (res, args) in SIGNATURES.items():
        fn = getattr(lib, name)  # AttributeError if the symbol is not exported
        fn.restype = res
        fn.argtypes = args
    return lib


_lib = load_library()


class ObemError(RuntimeError):
    def __init__(self, status: int, where: str, cuda_error: int = 0):
        self.status = status
        self.cuda_error = cuda_error
        msg = _lib.obem_status_string(status).decode()
        if cuda_error:
            msg += " [cudaError_t %d]" % cuda_error
        super().__init__("%s: %s" % (where, msg))


def status_string(status: int) -> str:
    return _lib.obem_status_string(int(status)).decode()


def _torch():
    import torch
    return torch


def _dev_f32(t, what, last=None):
    torch = _torch()
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous():
        raise TypeError("%s must be a contiguous float32 CUDA tensor" % what)
    if last is not None and (t.dim() < 1 or tuple(t.shape[-len(last):]) != tuple(last)):
        raise ValueError("%s must have trailing shape %r, got %r" % (what, last, tuple(t.shape)))
    return t


def _stream_ptr(stream):
    torch = _torch()
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


class Context:
    """One obem_ctx on one CUDA device.  Methods mirror the C entry points one to one."""

    def __init__(self, device: int = 0):
        self._h = ctypes.c_void_p()
        self.device = int(device)
        rc = _lib.obem_create(ctypes.byref(self._h), self.device)
        if rc != 0:
            self._h = ctypes.c_void_p()
            raise ObemError(rc, "obem_create(device=%d)" % device)

    # -- lifetime ---------------------------------------------------------------------------------
    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h:
            _lib.obem_destroy(self._h)
            self._h = ctypes.c_void_p()

    close = destroy

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    def _check(self, rc, where):
        if rc != 0:
            raise ObemError(rc, where, _lib.obem_last_cuda_error(self._h))

    # -- setters ----------------------------------------------------------------------------------
    def reserve(self, n_charges: int, n_panels: int):
        self._check(_lib.obem_reserve(self._h, int(n_charges), int(n_panels)), "obem_reserve")

    def set_softening(self, eps_pp: float, eps_panel: float = 0.0):
        self._check(_lib.obem_set_softening(self._h, float(eps_pp), float(eps_panel)), "obem_set_softening")

    def set_panels(self, verts, sigma, stream=None):
        """verts [Np,3,3], sigma [Np] float32 CUDA tensors."""
        n = int(sigma.shape[0])
        if n:
            _dev_f32(verts, "verts", (3, 3))
            _dev_f32(sigma, "sigma")
            if verts.shape[0] != n:
                raise ValueError("verts and sigma disagree on the number of panels")
        self._check(_lib.obem_set_panels(self._h, verts.data_ptr() if n else None, sigma.data_ptr() if n else None,
                                         n, _stream_ptr(stream)), "obem_set_panels")

    def set_sigma(self, sigma, stream=None):
        n = int(sigma.shape[0])
        if n:
            _dev_f32(sigma, "sigma")
        self._check(_lib.obem_set_sigma(self._h, sigma.data_ptr() if n else None, n, _stream_ptr(stream)),
                    "obem_set_sigma")

    def set_charges(self, xyzq, stream=None):
        """xyzq [N,4] float32 CUDA tensor (x, y, z [m], q [C]) -- Eq (3.8)'s particles."""
        n = int(xyzq.shape[0])
        if n:
            _dev_f32(xyzq, "xyzq", (4,))
        self._check(_lib.obem_set_charges(self._h, xyzq.data_ptr() if n else None, n, _stream_ptr(stream)),
                    "obem_set_charges")

    # -- evaluation -------------------------------------------------------------------------------
    def eval_at_charges(self, out=None, flags: int = NBODY | PANELS, stream=None):
        torch = _torch()
        n = self.n_charges
        if n < 0:
            self._check(-2, "obem_eval_at_charges")
        if out is None:
            out = torch.empty((n, 4), dtype=torch.float32, device="cuda:%d" % self.device)
        elif n:
            _dev_f32(out, "out", (4,))
            if out.shape[0] != n:
                raise ValueError("out must be [n_charges, 4]")
        self._check(_lib.obem_eval_at_charges(self._h, out.data_ptr() if n else None, int(flags), _stream_ptr(stream)),
                    "obem_eval_at_charges")
        return out

    def eval_at_charges_range(self, first: int, count: int, out=None, flags: int = NBODY | PANELS, stream=None):
        torch = _torch()
        if out is None:
            out = torch.empty((max(count, 0), 4), dtype=torch.float32, device="cuda:%d" % self.device)
        elif count > 0:
            _dev_f32(out, "out", (4,))
            if out.shape[0] != count:
                raise ValueError("out must be [count, 4]")
        self._check(_lib.obem_eval_at_charges_range(self._h, int(first), int(count),
                                                    out.data_ptr() if count > 0 else None, int(flags),
                                                    _stream_ptr(stream)), "obem_eval_at_charges_range")
        return out

    def eval_at_points(self, pts, out=None, flags: int = PANELS, stream=None):
        torch = _torch()
        m = int(pts.shape[0])
        if m:
            _dev_f32(pts, "pts", (4,))
        if out is None:
            out = torch.empty((m, 4), dtype=torch.float32, device="cuda:%d" % self.device)
        elif m:
            _dev_f32(out, "out", (4,))
            if out.shape[0] != m:
                raise ValueError("out must be [m, 4]")
        self._check(_lib.obem_eval_at_points(self._h, pts.data_ptr() if m else None, m,
                                             out.data_ptr() if m else None, int(flags), _stream_ptr(stream)),
                    "obem_eval_at_points")
        return out

    # -- host-buffer entry points (synchronous) ------------------------------------------------------
    @staticmethod
    def _host_ptr(a, what, shape_tail):
        import numpy as np
        if a is None:
            return None, 0
        if not isinstance(a, np.ndarray) or a.dtype != np.float32 or not a.flags["C_CONTIGUOUS"]:
            raise TypeError("%s must be a C-contiguous float32 numpy array" % what)
        if a.size and tuple(a.shape[1:]) != tuple(shape_tail):
            raise ValueError("%s must have shape [n%s]" % (what, "".join(",%d" % s for s in shape_tail)))
        return (a.ctypes.data if a.size else None), int(a.shape[0])

    def field_at_charges_host(self, xyzq, verts=None, sigma=None, out=None, flags: int = NBODY | PANELS):
        """Whole path through host (numpy) buffers: H2D, set_panels (if verts given), set_charges,
        eval_at_charges, D2H.  Returns out [N,4] float32 numpy."""
        import numpy as np
        px, n = self._host_ptr(xyzq, "xyzq", (4,))
        pv, npan = self._host_ptr(verts, "verts", (3, 3))
        ps, ns = self._host_ptr(sigma, "sigma", ())
        if verts is not None and ns != npan:
            raise ValueError("verts and sigma disagree on the number of panels")
        if out is None:
            out = np.empty((n, 4), dtype=np.float32)
        po, no = self._host_ptr(out, "out", (4,))
        if no != n:
            raise ValueError("out must be [n, 4]")
        if verts is not None and npan == 0:
            pv = ctypes.addressof(ctypes.c_float())  # non-NULL marker: "set an empty panel set"
        self._check(_lib.obem_field_at_charges_host(self._h, px, n, pv, ps, npan, po, int(flags)),
                    "obem_field_at_charges_host")
        return out

    def field_at_points_host(self, pts, verts=None, sigma=None, out=None, flags: int = PANELS):
        import numpy as np
        pp, m = self._host_ptr(pts, "pts", (4,))
        pv, npan = self._host_ptr(verts, "verts", (3, 3))
        ps, ns = self._host_ptr(sigma, "sigma", ())
        if verts is not None and ns != npan:
            raise ValueError("verts and sigma disagree on the number of panels")
        if out is None:
            out = np.empty((m, 4), dtype=np.float32)
        po, mo = self._host_ptr(out, "out", (4,))
        if mo != m:
            raise ValueError("out must be [m, 4]")
        if verts is not None and npan == 0:
            pv = ctypes.addressof(ctypes.c_float())
        self._check(_lib.obem_field_at_points_host(self._h, pp, m, pv, ps, npan, po, int(flags)),
                    "obem_field_at_points_host")
        return out

    # -- introspection ----------------------------------------------------------------------------
    @property
    def n_charges(self) -> int:
        return int(_lib.obem_n_charges(self._h))

    @property
    def n_panels(self) -> int:
        return int(_lib.obem_n_panels(self._h))

    @property
    def sm_count(self) -> int:
        return int(_lib.obem_sm_count(self._h))

    @property
    def grid_size(self) -> int:
        return int(_lib.obem_grid_size(self._h))

    @property
    def kernel_launches(self) -> int:
        return int(_lib.obem_kernel_launches(self._h))

    def get_panel_sources(self, stream=None):
        torch = _torch()
        n = max(self.n_panels, 0)
        out = torch.empty((n * 7, 4), dtype=torch.float32, device="cuda:%d" % self.device)
        self._check(_lib.obem_get_panel_sources(self._h, out.data_ptr() if n else None, _stream_ptr(stream)),
                    "obem_get_panel_sources")
        return out

    def fma_peak_probe(self, mode: int, iters: int, stream=None) -> float:
        """Enqueue the FP32-pipe probe; returns the flop count it executes (time it with events)."""
        fl = ctypes.c_double(0.0)
        self._check(_lib.obem_fma_peak_probe(self._h, int(mode), int(iters), ctypes.byref(fl), _stream_ptr(stream)),
                    "obem_fma_peak_probe")
        return fl.value

    # -- adjacent steps: Eq (3.3)-(3.6), sigma = M^-1 b ---------------------------
    def _new(self, shape):
        torch = _torch()
        return torch.empty(shape, dtype=torch.float32, device="cuda:%d" % self.device)

    def influence_on_panels(self, want_en: bool = True, stream=None):
        """Eq (3.3)/(3.4): returns (infl [Np,4] = Ebar_xyz, Vbar; en [Np] = Ebar.n or None)."""
        n = max(self.n_panels, 0)
        infl = self._new((n, 4))
        en = self._new((n,)) if want_en else None
        self._check(_lib.obem_influence_on_panels(self._h, infl.data_ptr() if n else None,
                                                  en.data_ptr() if (want_en and n) else None, _stream_ptr(stream)),
                    "obem_influence_on_panels")
        return infl, en

    def rhs_from_influence(self, kind, bc, deps, infl, en, stream=None):
        """Eq (3.5)/(3.6): kind int32 [Np] (0 = ed, 1 = dd), bc/deps float32 [Np] -> b [Np]."""
        torch = _torch()
        n = int(kind.shape[0])
        if n:
            if not (kind.is_cuda and kind.dtype == torch.int32 and kind.is_contiguous()):
                raise TypeError("kind must be a contiguous int32 CUDA tensor")
            _dev_f32(bc, "bc"), _dev_f32(deps, "deps"), _dev_f32(infl, "infl", (4,)), _dev_f32(en, "en")
        b = self._new((n,))
        self._check(_lib.obem_rhs_from_influence(self._h, kind.data_ptr() if n else None, bc.data_ptr() if n else None,
                                                 deps.data_ptr() if n else None, infl.data_ptr() if n else None,
                                                 en.data_ptr() if n else None, b.data_ptr() if n else None, n,
                                                 _stream_ptr(stream)), "obem_rhs_from_influence")
        return b

    def apply_inverse(self, minv, b, out=None, stream=None):
        """sigma = M^-1 b: minv [n, n] (or a row-major view with stride(0) >= n), b [n] -> sigma [n]."""
        torch = _torch()
        n = int(b.shape[0])
        ld = n
        if n:
            _dev_f32(b, "b")
            if not (isinstance(minv, torch.Tensor) and minv.is_cuda and minv.dtype == torch.float32 and minv.dim() == 2
                    and minv.shape == (n, n) and minv.stride(1) == 1 and minv.stride(0) >= n):
                raise TypeError("minv must be a float32 CUDA [n, n] tensor with unit column stride")
            ld = int(minv.stride(0))
        if out is None:
            out = self._new((n,))
        self._check(_lib.obem_apply_inverse(self._h, minv.data_ptr() if n else None, n, ld, b.data_ptr() if n else None,
                                            out.data_ptr() if n else None, _stream_ptr(stream)), "obem_apply_inverse")
        return out

    def update_sigma_dynamic(self, kind, bc, deps, minv, stream=None):
        """influence -> rhs -> M^-1 b -> set_sigma on one stream; returns the new sigma [Np]."""
        n = max(self.n_panels, 0)
        sigma = self._new((n,))
        ld = int(minv.stride(0)) if n else 0
        self._check(_lib.obem_update_sigma_dynamic(self._h, kind.data_ptr() if n else None, bc.data_ptr() if n else None,
                                                   deps.data_ptr() if n else None, minv.data_ptr() if n else None, ld,
                                                   sigma.data_ptr() if n else None, _stream_ptr(stream)),
                    "obem_update_sigma_dynamic")
        return sigma

    def eval_panels_multi(self, sigmas, pts, out=None, stream=None):
        """Eq (2.13)/(2.14) for several density vectors on the current cells (weighting fields, Eq 3.13):
        sigmas [K, Np], pts [M, 4] -> out [K, M, 4]."""
        torch = _torch()
        k, m = int(sigmas.shape[0]), int(pts.shape[0])
        npan = max(self.n_panels, 0)
        if k and npan:
            _dev_f32(sigmas, "sigmas")
            if sigmas.dim() != 2 or sigmas.shape[1] != npan:
                raise ValueError("sigmas must be [K, n_panels]")
        if m:
            _dev_f32(pts, "pts", (4,))
        if out is None:
            out = torch.empty((k, m, 4), dtype=torch.float32, device="cuda:%d" % self.device)
        elif k and m:
            _dev_f32(out, "out", (4,))
            if tuple(out.shape) != (k, m, 4):
                raise ValueError("out must be [K, M, 4]")
        self._check(_lib.obem_eval_panels_multi(self._h, sigmas.data_ptr() if (k and npan) else None, k,
                                                pts.data_ptr() if m else None, m,
                                                out.data_ptr() if (k and m) else None, _stream_ptr(stream)),
                    "obem_eval_panels_multi")
        return out

    def ramo_current(self, xyzq, vel, ew, stream=None):
        """Eq (3.13): xyzq [N,4], vel [N,4], ew [K,N,4] float32 -> [K,2] float64 (electrons, ions) [A]."""
        torch = _torch()
        n, k = int(xyzq.shape[0]), int(ew.shape[0])
        if n and k:
            _dev_f32(xyzq, "xyzq", (4,)), _dev_f32(vel, "vel", (4,)), _dev_f32(ew, "ew", (4,))
            if vel.shape[0] != n or tuple(ew.shape) != (k, n, 4):
                raise ValueError("vel must be [N, 4] and ew [K, N, 4]")
        out = torch.empty((k, 2), dtype=torch.float64, device="cuda:%d" % self.device)
        ok = n > 0 and k > 0
        self._check(_lib.obem_ramo_current(self._h, xyzq.data_ptr() if ok else None, vel.data_ptr() if ok else None,
                                           ew.data_ptr() if ok else None, k, n, out.data_ptr() if k else None,
                                           _stream_ptr(stream)), "obem_ramo_current")
        return out

    def get_panel_normals(self, stream=None):
        n = max(self.n_panels, 0)
        out = self._new((n, 4))
        self._check(_lib.obem_get_panel_normals(self._h, out.data_ptr() if n else None, _stream_ptr(stream)),
                    "obem_get_panel_normals")
        return out

    # -- NEXT-2: integrators; xyzq [N,4] and vel [N,4] = (vx, vy, vz, m) are updated IN PLACE ----
    def _state(self, xyzq, vel):
        n = int(xyzq.shape[0])
        if n:
            _dev_f32(xyzq, "xyzq", (4,)), _dev_f32(vel, "vel", (4,))
            if vel.shape[0] != n:
                raise ValueError("xyzq and vel disagree on the number of particles")
        return n

    def push_drift(self, xyzq, vel, h: float, stream=None):
        n = self._state(xyzq, vel)
        self._check(_lib.obem_push_drift(self._h, xyzq.data_ptr() if n else None, vel.data_ptr() if n else None, n,
                                         float(h), _stream_ptr(stream)), "obem_push_drift")

    def push_kick(self, xyzq, vel, field, h: float, stream=None):
        n = self._state(xyzq, vel)
        if n:
            _dev_f32(field, "field", (4,))
        self._check(_lib.obem_push_kick(self._h, xyzq.data_ptr() if n else None, vel.data_ptr() if n else None,
                                        field.data_ptr() if n else None, n, float(h), _stream_ptr(stream)),
                    "obem_push_kick")

    def step_euler(self, xyzq, vel, dt: float, flags: int = NBODY | PANELS, stream=None):
        n = self._state(xyzq, vel)
        self._check(_lib.obem_step_euler(self._h, xyzq.data_ptr() if n else None, vel.data_ptr() if n else None, n,
                                         float(dt), int(flags), _stream_ptr(stream)), "obem_step_euler")

    def step_pefrl(self, xyzq, vel, dt: float, flags: int = NBODY | PANELS, stream=None):
        n = self._state(xyzq, vel)
        self._check(_lib.obem_step_pefrl(self._h, xyzq.data_ptr() if n else None, vel.data_ptr() if n else None, n,
                                         float(dt), int(flags), _stream_ptr(stream)), "obem_step_pefrl")

    # -- NEXT-2: recombination by-product ---------------------------------------------
    def eval_at_charges_partners(self, flags: int = NBODY | PANELS, first: int = 0, count=None, stream=None):
        """Returns (out [count,4], partner_d [count] float32, partner_j [count] int32) for charges [first, first+count)."""
        torch = _torch()
        n = self.n_charges
        if n < 0:
            self._check(-2, "obem_eval_at_charges_partners")
        if count is None:
            count = n - first
        dev = "cuda:%d" % self.device
        out = torch.empty((max(count, 0), 4), dtype=torch.float32, device=dev)
        pd = torch.empty((max(count, 0),), dtype=torch.float32, device=dev)
        pj = torch.empty((max(count, 0),), dtype=torch.int32, device=dev)
        ok = count > 0
        self._check(_lib.obem_eval_at_charges_partners_range(
            self._h, int(first), int(count), out.data_ptr() if ok else None, pd.data_ptr() if ok else None,
            pj.data_ptr() if ok else None, int(flags), _stream_ptr(stream)), "obem_eval_at_charges_partners_range")
        return out, pd, pj

    # -- NEXT-3: near-field-accurate panels -------------------------------------------
    def set_near_field(self, near_factor: float = 3.0):
        self._check(_lib.obem_set_near_field(self._h, float(near_factor)), "obem_set_near_field")

    @property
    def near_list_size(self) -> int:
        return int(_lib.obem_near_list_size(self._h))

    @property
    def near_cells(self) -> int:
        return int(_lib.obem_near_cells(self._h))

    def set_panels_cells(self, verts4, sigma, nvert=None, stream=None):
        """verts4 [Nc,4,3] float32, sigma [Nc] float32, nvert [Nc] int32 (3 or 4; None = all quadrilaterals)."""
        torch = _torch()
        nc = int(sigma.shape[0])
        if nc:
            _dev_f32(verts4, "verts4", (4, 3)), _dev_f32(sigma, "sigma")
            if verts4.shape[0] != nc:
                raise ValueError("verts4 and sigma disagree on the number of cells")
            if nvert is not None and (not nvert.is_cuda or nvert.dtype != torch.int32 or nvert.shape != (nc,)):
                raise TypeError("nvert must be an int32 CUDA tensor of shape [n_cells]")
        self._check(_lib.obem_set_panels_cells(self._h, verts4.data_ptr() if nc else None,
                                               nvert.data_ptr() if (nc and nvert is not None) else None,
                                               sigma.data_ptr() if nc else None, nc, _stream_ptr(stream)),
                    "obem_set_panels_cells")

    def set_sigma_cells(self, sigma, stream=None):
        nc = int(sigma.shape[0])
        if nc:
            _dev_f32(sigma, "sigma")
        self._check(_lib.obem_set_sigma_cells(self._h, sigma.data_ptr() if nc else None, nc, _stream_ptr(stream)),
                    "obem_set_sigma_cells")

    def set_symmetry(self, planes=()):
        """planes: iterable of (axis 0|1|2, coordinate [m], parity +1|-1); at most one per axis; () removes them."""
        planes = list(planes)
        n = len(planes)
        ax = (ctypes.c_int * max(n, 1))(*[int(p[0]) for p in planes])
        co = (ctypes.c_double * max(n, 1))(*[float(p[1]) for p in planes])
        pa = (ctypes.c_int * max(n, 1))(*[int(p[2]) for p in planes])
        self._check(_lib.obem_set_symmetry(self._h, n, ax, co, pa), "obem_set_symmetry")

    # -- NEXT-4: NN approximation of the N-body sum -----------------------------------
    def set_nn_theta(self, theta: float = 2.0):
        self._check(_lib.obem_set_nn_theta(self._h, float(theta)), "obem_set_nn_theta")

    def eval_at_charges_nn(self, out=None, flags: int = NBODY, stream=None):
        n = self.n_charges
        if n < 0:
            self._check(-2, "obem_eval_at_charges_nn")
        if out is None:
            out = self._new((n, 4))
        elif n:
            _dev_f32(out, "out", (4,))
            if out.shape[0] != n:
                raise ValueError("out must be [n_charges, 4]")
        self._check(_lib.obem_eval_at_charges_nn(self._h, out.data_ptr() if n else None, int(flags),
                                                 _stream_ptr(stream)), "obem_eval_at_charges_nn")
        return out

    def nn_last_units(self, stream=None) -> int:
        return int(_lib.obem_nn_last_units(self._h, _stream_ptr(stream)))

    # -- NEXT-4: static field option ------------------------------------------------------
    def field_map(self, shape, origin, spacing, flags: int = PANELS, out=None, stream=None):
        """Fill a [nx, ny, nz, 4] map (Ex, Ey, Ez, phi at the nodes origin + i*spacing)."""
        nx, ny, nz = (int(v) for v in shape)
        if out is None:
            out = self._new((nx, ny, nz, 4))
        else:
            _dev_f32(out, "out", (nx, ny, nz, 4))
        o = (ctypes.c_double * 3)(*[float(v) for v in origin])
        d = (ctypes.c_double * 3)(*[float(v) for v in spacing])
        self._check(_lib.obem_field_map(self._h, nx, ny, nz, o, d, out.data_ptr(), int(flags), _stream_ptr(stream)),
                    "obem_field_map")
        return out

    def interp_map(self, fmap, origin, spacing, pts, out=None, accumulate: bool = False, stream=None):
        """Trilinear interpolation of fmap [nx, ny, nz, 4] at pts [M, 4] -> [M, 4] (added to `out` if accumulate)."""
        _dev_f32(fmap, "fmap", (4,))
        if fmap.dim() != 4:
            raise ValueError("fmap must be [nx, ny, nz, 4]")
        nx, ny, nz = (int(v) for v in fmap.shape[:3])
        m = int(pts.shape[0])
        if m:
            _dev_f32(pts, "pts", (4,))
        if out is None:
            if accumulate:
                raise ValueError("accumulate needs an `out` to add to")
            out = self._new((m, 4))
        elif m:
            _dev_f32(out, "out", (4,))
            if out.shape[0] != m:
                raise ValueError("out and pts disagree on the number of positions")
        o = (ctypes.c_double * 3)(*[float(v) for v in origin])
        d = (ctypes.c_double * 3)(*[float(v) for v in spacing])
        self._check(_lib.obem_interp_map(self._h, fmap.data_ptr(), nx, ny, nz, o, d, pts.data_ptr() if m else None,
                                         m, out.data_ptr() if m else None, 1 if accumulate else 0,
                                         _stream_ptr(stream)), "obem_interp_map")
        return out


STATIC_MAX_POINTS = 16384  # OBEM_STATIC_MAX_POINTS


def nbody_at_points_static(xyzq, pts, eps_pp: float, out, stream=None):
    """obem_nbody_at_points_static: the N-body sum of xyzq [N,4] at pts [M,4] into out [M,4] (all float32 CUDA tensors
    of the current device) with NO allocation anywhere -- no context, scratch in a fixed static device array; M <=
    STATIC_MAX_POINTS.  `out` is required (allocating it here would defeat the purpose)."""
    n, m = int(xyzq.shape[0]), int(pts.shape[0])
    if n:
        _dev_f32(xyzq, "xyzq", (4,))
    if m:
        _dev_f32(pts, "pts", (4,))
        _dev_f32(out, "out", (4,))
        if out.shape[0] != m:
            raise ValueError("out must be [M, 4]")
    rc = _lib.obem_nbody_at_points_static(xyzq.data_ptr() if n else None, n, pts.data_ptr() if m else None, m,
                                          float(eps_pp), out.data_ptr() if m else None, _stream_ptr(stream))
    if rc != 0:
        raise ObemError(rc, "obem_nbody_at_points_static")
    return out


def recombination_radius(e_ioni_ev: float) -> float:
    """Eq (3.12): k_e e / (2 E_ioni) [m], E_ioni in eV."""
    return float(_lib.obem_recombination_radius(float(e_ioni_ev)))
