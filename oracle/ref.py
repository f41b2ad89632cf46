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
_SRCS = [_SRC, os.path.join(_HERE, "obem_ref_next.c"),   # hot path; adjacent steps
         os.path.join(_HERE, "obem_ref_analytic.c")]       # NEXT-3: exact cell integrals
_LIB = os.path.join(_HERE, "libobem_ref.so")

NBODY = 1
PANELS = 2

_lib = None


def build(force: bool = False) -> str:
    """Compile obem_ref.c -> libobem_ref.so (gcc -O2, no fast-math, OpenMP over targets)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(f) for f in _SRCS):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(
            ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", tmp] + _SRCS + ["-lm"]
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
        c_i32p = ctypes.POINTER(ctypes.c_int32)
        lib.obem_ref_influence.restype = ctypes.c_int
        lib.obem_ref_influence.argtypes = [c_fp, ctypes.c_int64, c_fp, ctypes.c_int64, ctypes.c_double,
                                           c_dp, c_dp, c_dp, ctypes.c_int]
        lib.obem_ref_rhs.restype = ctypes.c_int
        lib.obem_ref_rhs.argtypes = [c_i32p, c_fp, c_fp, c_dp, c_dp, ctypes.c_int64, c_dp]
        lib.obem_ref_nearest_opposite.restype = ctypes.c_int
        lib.obem_ref_nearest_opposite.argtypes = [c_fp, ctypes.c_int64, c_dp, c_ip, ctypes.c_int]
        lib.obem_ref_nearest_opposite_subset.restype = ctypes.c_int
        lib.obem_ref_nearest_opposite_subset.argtypes = [c_fp, ctypes.c_int64, c_ip, ctypes.c_int64, c_dp, c_ip,
                                                         ctypes.c_int]
        lib.obem_ref_recombination_radius.restype = ctypes.c_double
        lib.obem_ref_recombination_radius.argtypes = [ctypes.c_double]
        lib.obem_ref_matvec.restype = ctypes.c_int
        lib.obem_ref_matvec.argtypes = [c_fp, ctypes.c_int64, ctypes.c_int64, c_fp, c_dp, ctypes.c_int]
        lib.obem_ref_tri_integrals.restype = None
        lib.obem_ref_tri_integrals.argtypes = [c_dp, c_dp, c_dp, c_dp, c_dp, c_dp]
        lib.obem_ref_eval_panels_analytic.restype = ctypes.c_int
        lib.obem_ref_eval_panels_analytic.argtypes = [c_fp, c_fp, ctypes.c_int64, c_fp, ctypes.c_int64, c_dp,
                                                      ctypes.c_int]
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


# --------------------------------------------------------------------------------------------------
# NEXT-1: influence of the particles on the cells, Eq (3.3)-(3.6); sigma = M^-1 b
# --------------------------------------------------------------------------------------------------
def influence(xyzq, verts, eps: float = 0.0, n_threads: int = 0):
    """Eq (3.3)/(3.4).  Returns (infl[Np,4] = (Ebar_x, Ebar_y, Ebar_z, Vbar), en[Np] = Ebar.n, na[Np,4] = (n, A))."""
    xyzq = _f32(xyzq if xyzq is not None else [], (4,))
    verts = _f32(verts if verts is not None else [], (3, 3))
    n, npan = xyzq.shape[0], verts.shape[0]
    out = np.zeros((npan, 4), dtype=np.float64)
    en = np.zeros(npan, dtype=np.float64)
    na = np.zeros((npan, 4), dtype=np.float64)
    rc = _load().obem_ref_influence(_ptr(xyzq, ctypes.c_float), n, _ptr(verts, ctypes.c_float), npan, float(eps),
                                    _ptr(out, ctypes.c_double), _ptr(en, ctypes.c_double),
                                    _ptr(na, ctypes.c_double), int(n_threads))
    if rc != 0:
        raise ValueError("obem_ref_influence: bad argument")
    return out, en, na


def rhs(kind, bc, deps, infl, en):
    """Eq (3.5)/(3.6): b[Np] float64."""
    kind = np.ascontiguousarray(kind, dtype=np.int32)
    bc = _f32(bc, ())
    deps = _f32(deps, ())
    infl = np.ascontiguousarray(infl, dtype=np.float64)
    en = np.ascontiguousarray(en, dtype=np.float64)
    npan = kind.shape[0]
    assert bc.shape[0] == npan and deps.shape[0] == npan and infl.shape == (npan, 4) and en.shape == (npan,)
    b = np.zeros(npan, dtype=np.float64)
    rc = _load().obem_ref_rhs(_ptr(kind, ctypes.c_int32), _ptr(bc, ctypes.c_float), _ptr(deps, ctypes.c_float),
                              _ptr(infl, ctypes.c_double), _ptr(en, ctypes.c_double), npan, _ptr(b, ctypes.c_double))
    if rc != 0:
        raise ValueError("obem_ref_rhs: bad argument (kind must be 0 or 1)")
    return b


def matvec(minv, b, n_threads: int = 0):
    """sigma = M^-1 b with a stored fp32 inverse [n, n] (row-major) and fp32 b; float64 result."""
    minv = np.ascontiguousarray(minv, dtype=np.float32)
    b = _f32(b, ())
    n = b.shape[0]
    assert minv.shape == (n, n)
    out = np.zeros(n, dtype=np.float64)
    rc = _load().obem_ref_matvec(_ptr(minv, ctypes.c_float), n, n, _ptr(b, ctypes.c_float),
                                 _ptr(out, ctypes.c_double), int(n_threads))
    if rc != 0:
        raise ValueError("obem_ref_matvec: bad argument")
    return out


# --------------------------------------------------------------------------------------------------
# NEXT-2: recombination by-product of the N-body pass, Eq (3.12)
# --------------------------------------------------------------------------------------------------
def nearest_opposite(xyzq, idx=None, n_threads: int = 0):
    """(d, j): distance to and index of the nearest charge of opposite sign (-1 / inf if none), for every charge
    or for the charges idx only (candidates are always all charges)."""
    xyzq = _f32(xyzq if xyzq is not None else [], (4,))
    n = xyzq.shape[0]
    if idx is not None:
        idx = np.ascontiguousarray(idx, dtype=np.int64)
        assert idx.ndim == 1 and (idx.size == 0 or (idx.min() >= 0 and idx.max() < n))
    m = n if idx is None else idx.shape[0]
    d = np.zeros(m, dtype=np.float64)
    j = np.zeros(m, dtype=np.int64)
    rc = _load().obem_ref_nearest_opposite_subset(_ptr(xyzq, ctypes.c_float), n,
                                                  _ptr(idx, ctypes.c_int64) if idx is not None else None, m,
                                                  _ptr(d, ctypes.c_double), _ptr(j, ctypes.c_int64), int(n_threads))
    if rc != 0:
        raise ValueError("obem_ref_nearest_opposite: bad argument")
    return d, j


def recombination_radius(e_ioni_ev: float) -> float:
    """Eq (3.12): k_e e / (2 E_ioni) in metres, E_ioni in eV."""
    return float(_load().obem_ref_recombination_radius(float(e_ioni_ev)))


# --------------------------------------------------------------------------------------------------
# NEXT-3: exact cell integrals of Eq (2.13)/(2.14) over flat triangles (obem_ref_analytic.c)
# --------------------------------------------------------------------------------------------------
def tri_integrals(v0, v1, v2, r):
    """(I_phi, I_E[3]) = (Int dS/R, Int (r - r')/R^3 dS) over the flat triangle (v0, v1, v2) at r; float64."""
    a = [np.ascontiguousarray(x, dtype=np.float64).reshape(3) for x in (v0, v1, v2, r)]
    iphi = np.zeros(1, dtype=np.float64)
    ie = np.zeros(3, dtype=np.float64)
    _load().obem_ref_tri_integrals(*[_ptr(x, ctypes.c_double) for x in a], _ptr(iphi, ctypes.c_double),
                                   _ptr(ie, ctypes.c_double))
    return float(iphi[0]), ie


def eval_panels_analytic(verts, sigma, targets, n_threads: int = 0):
    """k_e sum_p sigma_p (I_E, I_phi) at every target: [T, 4] float64 = Ex, Ey, Ez, phi."""
    verts = _f32(verts, (3, 3))
    sigma = _f32(sigma, ())
    targets = _f32(targets, (4,))
    npan, nt = verts.shape[0], targets.shape[0]
    assert sigma.shape[0] == npan
    out = np.zeros((nt, 4), dtype=np.float64)
    rc = _load().obem_ref_eval_panels_analytic(_ptr(verts, ctypes.c_float), _ptr(sigma, ctypes.c_float), npan,
                                               _ptr(targets, ctypes.c_float), nt, _ptr(out, ctypes.c_double),
                                               int(n_threads))
    if rc != 0:
        raise ValueError("obem_ref_eval_panels_analytic: bad argument")
    return out
