"""ctypes loader for the fp64 CPU oracle (oracle/obem_ref.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports nothing from
paper_2110_09214_b200 and shares no code with the CUDA path.

The arithmetic lives in obem_ref.c (each function cites the PAPER.md passage it follows); this file
only compiles it with gcc and marshals numpy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "obem_ref.c")
_LIB = os.path.join(_HERE, "libobem_ref.so")

NBODY = 1
PANELS = 2

_lib = None


def build(force: bool = False) -> str:
    """Compile obem_ref.c -> libobem_ref.so (gcc -O2, no fast-math, OpenMP over targets)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(
            ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        c_fp = ctypes.POINTER(ctypes.c_float)
        c_dp = ctypes.POINTER(ctypes.c_double)
        c_ip = ctypes.POINTER(ctypes.c_int64)
        lib.obem_ref_eval.restype = ctypes.c_int
        lib.obem_ref_eval.argtypes = [
            c_fp, ctypes.c_int64, c_fp, c_fp, ctypes.c_int64, ctypes.c_double, ctypes.c_double,
            c_fp, c_ip, ctypes.c_int64, ctypes.c_uint, c_dp, c_dp, ctypes.c_int,
        ]
        lib.obem_ref_panel_sources.restype = ctypes.c_int
        lib.obem_ref_panel_sources.argtypes = [c_fp, c_fp, ctypes.c_int64, c_dp]
        lib.obem_ref_quad_rule.restype = None
        lib.obem_ref_quad_rule.argtypes = [c_dp, c_dp]
        lib.obem_ref_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _f32(a, shape_tail):
    a = np.ascontiguousarray(a, dtype=np.float32)
    if a.size == 0:
        return a.reshape((0,) + shape_tail)
    return a.reshape((-1,) + shape_tail)


def _ptr(a, ctype):
    if a is None or a.size == 0:
        return None
    return a.ctypes.data_as(ctypes.POINTER(ctype))


def quad_rule():
    """(l[7,3], w[7]) of the 7-point degree-5 triangle rule the oracle uses."""
    l = np.zeros((7, 3), dtype=np.float64)
    w = np.zeros(7, dtype=np.float64)
    _load().obem_ref_quad_rule(_ptr(l, ctypes.c_double), _ptr(w, ctypes.c_double))
    return l, w


def panel_sources(verts, sigma):
    """fp64 quadrature sources [np*7, 4] = (x, y, z, sigma*A*w_k) of every panel."""
    verts = _f32(verts, (3, 3))
    sigma = _f32(sigma, ())
    npan = verts.shape[0]
    assert sigma.shape[0] == npan
    out = np.zeros((npan * 7, 4), dtype=np.float64)
    rc = _load().obem_ref_panel_sources(
        _ptr(verts, ctypes.c_float), _ptr(sigma, ctypes.c_float), npan, _ptr(out, ctypes.c_double)
    )
    if rc != 0:
        raise ValueError("obem_ref_panel_sources: bad argument")
    return out


def max_threads() -> int:
    return int(_load().obem_ref_max_threads())


def eval_field(xyzq=None, verts=None, sigma=None, targets=None, self_index=None,
               eps_pp: float = 0.0, eps_panel: float = 0.0, flags: int = NBODY | PANELS,
               n_threads: int = 0):
    """Oracle evaluation.  Returns (out_nbody[T,4], out_panel[T,4]) in float64: (Ex, Ey, Ez, phi).

    targets=None means "at the charges" with self_index = arange(N) (Eq 3.8's p != p')."""
    xyzq = _f32(xyzq if xyzq is not None else [], (4,))
    verts = _f32(verts if verts is not None else [], (3, 3))
    sigma = _f32(sigma if sigma is not None else [], ())
    n, npan = xyzq.shape[0], verts.shape[0]
    assert sigma.shape[0] == npan
    if targets is None:
        targets = xyzq
        if self_index is None:
            self_index = np.arange(n, dtype=np.int64)
    targets = _f32(targets, (4,))
    nt = targets.shape[0]
    if self_index is not None:
        self_index = np.ascontiguousarray(self_index, dtype=np.int64)
        assert self_index.shape == (nt,)
    out_n = np.zeros((nt, 4), dtype=np.float64)
    out_p = np.zeros((nt, 4), dtype=np.float64)
    # keep 1-element placeholders alive so pointers are never NULL when nt == 0 is not the reason
    rc = _load().obem_ref_eval(
        _ptr(xyzq, ctypes.c_float), n, _ptr(verts, ctypes.c_float), _ptr(sigma, ctypes.c_float), npan,
        float(eps_pp), float(eps_panel), _ptr(targets, ctypes.c_float),
        _ptr(self_index, ctypes.c_int64) if self_index is not None else None, nt, int(flags),
        _ptr(out_n, ctypes.c_double), _ptr(out_p, ctypes.c_double), int(n_threads),
    )
    if rc != 0:
        raise ValueError("obem_ref_eval: bad argument")
    return out_n, out_p
