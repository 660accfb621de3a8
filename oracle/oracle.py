"""ctypes front-end of oracle/hb_oracle.c -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  It shares nothing with paper_2402_17248_b200 (the CUDA path) and never imports it.

`push(lattice, coords)` walks a lattice description (see workloads/__init__.py) element by
element in fp64: R2/R3/R4 maps, and for a surrogate  [R6 to_t] -> R8 normalise -> R9 MLP ->
R8 de-normalise -> [R7 subtract z_ref, R6 to_s about the new reference]; a monitor takes the
R10 moments.  Citations as in hb_oracle.c.
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hb_oracle.c")
_SO = os.path.join(_HERE, "liboracle.so")

ACT = {"identity": 0, "relu": 1, "prelu": 2, "tanh": 3}


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c99",
                               "-o", _SO, _SRC, "-lm"])
    return _SO


_lib = None
_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int)


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.orc_num_threads.restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(n: int) -> None:
    lib().orc_set_num_threads(ctypes.c_int(int(n)))


def _p(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_dp)


def _rows(c: np.ndarray):
    assert c.dtype == np.float64 and c.ndim == 2 and c.shape[0] == 6 and c.flags["C_CONTIGUOUS"]
    return [_p(c[j]) for j in range(6)]


def reference(kinetic_MeV: float, rest_MeV: float):
    g, bg, b = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    lib().orc_reference(ctypes.c_double(kinetic_MeV), ctypes.c_double(rest_MeV),
                        ctypes.byref(g), ctypes.byref(bg), ctypes.byref(b))
    return g.value, bg.value, b.value


def drift(c, L, bg0):
    lib().orc_drift(*_rows(c), ctypes.c_long(c.shape[1]), ctypes.c_double(L), ctypes.c_double(bg0))


def drift_exact(c, L, bg0):
    lib().orc_drift_exact(*_rows(c), ctypes.c_long(c.shape[1]), ctypes.c_double(L), ctypes.c_double(bg0))


def quad_chromatic(c, L, k, bg0):
    lib().orc_quad_chromatic(*_rows(c), ctypes.c_long(c.shape[1]), ctypes.c_double(L), ctypes.c_double(k),
                             ctypes.c_double(bg0))


def multipole(c, order, kn, ks):
    lib().orc_multipole(*_rows(c), ctypes.c_long(c.shape[1]), ctypes.c_int(int(order)), ctypes.c_double(kn),
                        ctypes.c_double(ks))


def quad(c, L, k, bg0):
    lib().orc_quad(*_rows(c), ctypes.c_long(c.shape[1]), ctypes.c_double(L), ctypes.c_double(k),
                   ctypes.c_double(bg0))


def plens(c, L, k, bg0):
    lib().orc_plens(*_rows(c), ctypes.c_long(c.shape[1]), ctypes.c_double(L), ctypes.c_double(k),
                    ctypes.c_double(bg0))


def sbend(c, L, theta, bg0):
    lib().orc_sbend(*_rows(c), ctypes.c_long(c.shape[1]), ctypes.c_double(L), ctypes.c_double(theta),
                    ctypes.c_double(bg0))


def to_t(c, bg0):
    """s-coordinates [6,n] -> new array (x_t, y_t, z_t, ux, uy, uz)."""
    out = np.empty_like(c)
    lib().orc_to_t(*_rows(c), ctypes.c_long(c.shape[1]), ctypes.c_double(bg0), *_rows(out))
    return out


def to_s(v, bg1):
    """(x_t, y_t, z_t, ux, uy, uz) [6,n] -> new array of s-coordinates about reference bg1."""
    out = np.empty_like(v)
    lib().orc_to_s(*_rows(v), ctypes.c_long(v.shape[1]), ctypes.c_double(bg1), *_rows(out))
    return out


def mlp_normalised(v, sur):
    """In place on v [6,n]: R8 normalise -> R9 MLP -> R8 de-normalise."""
    widths = np.asarray(sur["widths"], dtype=np.int32)
    nl = len(widths) - 1
    W = np.concatenate([np.asarray(w, dtype=np.float32).astype(np.float64).ravel() for w in sur["W"]])
    b = np.concatenate([np.asarray(x, dtype=np.float32).astype(np.float64).ravel() for x in sur["b"]])
    for l in range(nl):
        assert sur["W"][l].shape == (widths[l + 1], widths[l])
    a = sur.get("prelu_a")
    a64 = None if a is None else np.ascontiguousarray(np.asarray(a, dtype=np.float32).astype(np.float64))
    if sur["act"] == "prelu":
        assert a64 is not None and a64.size == nl - 1
    stats = [np.ascontiguousarray(np.asarray(sur[k], dtype=np.float64)) for k in
             ("in_mean", "in_std", "out_mean", "out_std")]
    lib().orc_surrogate(*_rows(v), ctypes.c_long(v.shape[1]), ctypes.c_int(nl),
                        widths.ctypes.data_as(_ip), _p(W), _p(b), ctypes.c_int(ACT[sur["act"]]),
                        _p(a64) if a64 is not None else None, *[_p(s) for s in stats])


def moments(c) -> np.ndarray:
    out = np.empty(27, dtype=np.float64)
    lib().orc_moments(*_rows(c), ctypes.c_long(c.shape[1]), _p(out))
    return out


def surrogate_reference_out(sur, bg0):
    """R7: reference (beta gamma) and z after a COORD_T surrogate.  Given values are used as is;
    NaN -> the net is evaluated in fp64 on the reference input (0,0,0,0,0,bg0)."""
    bg1, z1 = sur["ref_bg_out"], sur["ref_z_out"]
    if math.isnan(bg1) or math.isnan(z1):
        r = np.zeros((6, 1), dtype=np.float64)
        r[5, 0] = bg0
        mlp_normalised(r, sur)
        if math.isnan(bg1):
            bg1 = float(r[5, 0])
        if math.isnan(z1):
            z1 = float(r[2, 0])
    return bg1, z1


class Tracker:
    """Element-by-element fp64 push with reference tracking (R1, R5, R7)."""

    def __init__(self, lattice):
        self.gamma0, self.bg, self.beta0 = reference(lattice["kinetic_MeV"], lattice["rest_MeV"])
        self.records = []

    def apply(self, el, c):
        """Apply one element to c [6,n] float64 (C-contiguous) in place."""
        kind = el["kind"]
        if kind == "drift":
            drift(c, el["L"], self.bg)
        elif kind == "drift_exact":
            drift_exact(c, el["L"], self.bg)
        elif kind == "quad_chromatic":
            quad_chromatic(c, el["L"], el["k"], self.bg)
        elif kind == "multipole":
            multipole(c, el["order"], el["kn"], el["ks"])
        elif kind == "quad":
            quad(c, el["L"], el["k"], self.bg)
        elif kind == "plens":
            plens(c, el["L"], el["k"], self.bg)
        elif kind == "sbend":
            sbend(c, el["L"], el["theta"], self.bg)
        elif kind == "monitor":
            self.records.append(moments(c))
        elif kind == "surrogate":
            if el["coord"] == "s":
                mlp_normalised(c, el)
            else:
                bg1, z1 = surrogate_reference_out(el, self.bg)
                v = to_t(c, self.bg)
                mlp_normalised(v, el)
                v[2] -= z1
                c[...] = to_s(v, bg1)
                self.bg = bg1
        else:
            raise ValueError(kind)


def push(lattice, coords, on_element=None):
    """coords: [6,n] float32 or float64.  Returns (coords_out float64 [6,n], moment records [m,27]).
    on_element(index, element, coords64) is called after each element (tests use it to grab states)."""
    c = np.ascontiguousarray(np.asarray(coords).astype(np.float64))
    tr = Tracker(lattice)
    for i, el in enumerate(lattice["elements"]):
        tr.apply(el, c)
        if on_element is not None:
            on_element(i, el, c)
    rec = np.array(tr.records, dtype=np.float64).reshape(-1, 27)
    return c, rec
