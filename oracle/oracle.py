"""ctypes wrapper around oracle/pact_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` leg may
import this.  It never imports the CUDA path.  See pact_oracle.c's header for what is computed and
which passages of the paper each function follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "pact_oracle.c"
_LIB = _HERE / "liboracle.so"

FIELD_IDS = dict(u1=0, u2=1, u3=2, s11=3, s22=4, s33=5, s23=6, s13=7, s12=8)


class OracleParams(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("h", C.c_double),
                ("dt", C.c_double), ("nt", C.c_int), ("npml", C.c_int), ("pml_R", C.c_double),
                ("pml_cref", C.c_double), ("pml_beta_max", C.c_double)]


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (plain C, fp64, OpenMP loops, -O2)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", str(_LIB), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        vp, dp, fp, ip, lp = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_float), C.c_int, C.POINTER(C.c_long)
        L.oracle_create.restype = vp
        L.oracle_create.argtypes = [C.POINTER(OracleParams), fp, fp, fp, fp, dp, ip]
        L.oracle_destroy.argtypes = [vp]
        L.oracle_field.restype = dp
        L.oracle_field.argtypes = [vp, ip]
        L.oracle_threads.restype = ip
        L.oracle_set_p0.argtypes = [vp, dp]
        L.oracle_sample.argtypes = [vp, dp]
        L.oracle_step.argtypes = [vp]
        L.oracle_forward.restype = ip
        L.oracle_forward.argtypes = [vp, dp, dp]
        L.oracle_adj_begin.argtypes = [vp]
        L.oracle_adj_source.argtypes = [vp, dp]
        L.oracle_adj_step.argtypes = [vp]
        L.oracle_adj_image.argtypes = [vp, dp]
        L.oracle_adjoint.restype = ip
        L.oracle_adjoint.argtypes = [vp, dp, dp]
        L.oracle_coef.restype = C.c_double
        L.oracle_coef.argtypes = [vp, ip, ip, ip, ip, ip, ip]
        L.oracle_pml_tables.argtypes = [vp, ip, dp]
        L.oracle_memvar_energy.restype = C.c_double
        L.oracle_memvar_energy.argtypes = [vp, ip]
        L.oracle_receiver_row.argtypes = [vp, ip, lp, dp]
        _lib = L
    return _lib


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _fptr(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_float))


class Oracle:
    """fp64 CPU H / H^T for one medium + receiver set.  Arrays are [nz][ny][nx]."""

    def __init__(self, prm, lam, mu, rho, alpha, rcv):
        L = lib()
        self.prm = prm
        self.shape = (prm.nz, prm.ny, prm.nx)
        self._keep = [np.ascontiguousarray(a, dtype=np.float32) if a is not None else None
                      for a in (lam, mu, rho, alpha)]
        for a in self._keep:
            if a is not None and a.shape != self.shape:
                raise ValueError("material volume has the wrong shape")
        self.rcv = np.ascontiguousarray(rcv, dtype=np.float64).reshape(-1, 3)
        self.L = int(self.rcv.shape[0])
        self._p = OracleParams(prm.nx, prm.ny, prm.nz, prm.h, prm.dt, prm.nt, prm.npml, prm.pml_R,
                               prm.pml_cref, prm.pml_beta_max)
        self._h = L.oracle_create(C.byref(self._p), *[_fptr(a) for a in self._keep],
                                  _dptr(self.rcv), self.L)
        if not self._h:
            raise ValueError("oracle_create rejected the inputs")

    @classmethod
    def from_problem(cls, prob, nt=None):
        prm = prob.prm
        if nt is not None:
            from dataclasses import replace
            prm = replace(prm, nt=nt)
        return cls(prm, prob.lam, prob.mu, prob.rho, prob.alpha, prob.rcv)

    def close(self):
        if getattr(self, "_h", None):
            lib().oracle_destroy(self._h)
            self._h = None

    __del__ = close

    # ---- whole operators
    def forward(self, p0):
        p0 = np.ascontiguousarray(p0, dtype=np.float64).reshape(self.shape)
        data = np.zeros((self.prm.nt, self.L), dtype=np.float64)
        rc = lib().oracle_forward(self._h, _dptr(p0), _dptr(data))
        assert rc == 0
        return data

    def adjoint(self, data):
        data = np.ascontiguousarray(data, dtype=np.float64).reshape(self.prm.nt, self.L)
        img = np.zeros(self.shape, dtype=np.float64)
        rc = lib().oracle_adjoint(self._h, _dptr(data), _dptr(img))
        assert rc == 0
        return img

    # ---- steppers (for invariants)
    def set_p0(self, p0):
        p0 = np.ascontiguousarray(p0, dtype=np.float64).reshape(self.shape)
        lib().oracle_set_p0(self._h, _dptr(p0))

    def step(self):
        lib().oracle_step(self._h)

    def sample(self):
        out = np.zeros(self.L, dtype=np.float64)
        lib().oracle_sample(self._h, _dptr(out))
        return out

    def field(self, name):
        """Live view (no copy) of a state field."""
        p = lib().oracle_field(self._h, FIELD_IDS[name])
        n = self.prm.nx * self.prm.ny * self.prm.nz
        return np.ctypeslib.as_array(p, shape=(n,)).reshape(self.shape)

    def adj_begin(self):
        lib().oracle_adj_begin(self._h)

    def adj_source(self, pm):
        pm = np.ascontiguousarray(pm, dtype=np.float64)
        lib().oracle_adj_source(self._h, _dptr(pm))

    def adj_step(self):
        lib().oracle_adj_step(self._h)

    def adj_image(self):
        img = np.zeros(self.shape, dtype=np.float64)
        lib().oracle_adj_image(self._h, _dptr(img))
        return img

    # ---- introspection
    def coef(self, kind, b, c, x, y, z):
        return lib().oracle_coef(self._h, kind, b, c, x, y, z)

    def pml_tables(self, axis):
        n = (self.prm.nx, self.prm.ny, self.prm.nz)[axis]
        out = np.zeros(4 * n, dtype=np.float64)
        lib().oracle_pml_tables(self._h, axis, _dptr(out))
        return dict(a_int=out[:n], b_int=out[n:2 * n], a_half=out[2 * n:3 * n], b_half=out[3 * n:])

    def memvar_energy(self, which):
        return lib().oracle_memvar_energy(self._h, 0 if which == "phi" else 1)

    def receiver_row(self, l):
        nodes = np.zeros(8, dtype=np.int64)
        w = np.zeros(8, dtype=np.float64)
        lib().oracle_receiver_row(self._h, l, nodes.ctypes.data_as(C.POINTER(C.c_long)), _dptr(w))
        return nodes, w


def threads() -> int:
    return int(lib().oracle_threads())
