"""ctypes front end of the CPU oracle (oracle/fp_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module; the
product package never does.  It marshals numpy arrays into the plain-C oracle and nothing else: every formula lives
in fp_oracle.c next to the PAPER.md / SURVEY.md passage it follows.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "fp_oracle.c"
_LIB = _HERE / "libfp_oracle.so"


def build(force: bool = False) -> Path:
    """gcc -O2 -ffp-contract=off -fopenmp (the filter decision must not be FMA-contracted)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared", "-std=c11",
               "-o", str(_LIB), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Setup(C.Structure):
    _fields_ = [
        ("natoms", C.c_int32), ("mesh", C.c_int32 * 3), ("lattvec", C.c_double * 9),
        ("masses", C.c_void_p), ("omega", C.c_void_p), ("eig", C.c_void_p), ("vg", C.c_void_p),
        ("n3", C.c_int64), ("atoms3", C.c_void_p), ("cells3", C.c_void_p), ("phi3", C.c_void_p),
        ("n4", C.c_int64), ("atoms4", C.c_void_p), ("cells4", C.c_void_p), ("phi4", C.c_void_p),
        ("T", C.c_double), ("scale", C.c_double), ("ncut", C.c_double), ("sigma_const", C.c_double),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(str(build()))
        _lib.orc_sigma.restype = C.c_double
        _lib.orc_be.restype = C.c_double
        _lib.orc_be.argtypes = [C.c_double, C.c_double]
        _lib.orc_allowed.argtypes = [C.c_void_p, C.c_double, C.c_double]
        _lib.orc_list3.restype = C.c_int64
        _lib.orc_list3.argtypes = [C.c_void_p, C.c_int32, C.c_int, C.c_void_p, C.c_int64]
        _lib.orc_list4.restype = C.c_int64
        _lib.orc_list4.argtypes = [C.c_void_p, C.c_int32, C.c_int, C.c_int32, C.c_int32, C.c_void_p, C.c_int64]
        _lib.orc_rates3.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
        _lib.orc_rates4.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p,
                                    C.c_void_p, C.c_int]
        _lib.orc_v3.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p]
        _lib.orc_v4.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p]
        _lib.orc_kappa.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    return _lib


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


class Oracle:
    """Holds contiguous copies of one Inputs (fp_inputs.Inputs) and exposes the oracle entry points."""

    def __init__(self, inp, T=None, scale=None, ncut=2.0, sigma_const=0.0):
        self.lib = lib()
        self.nb = inp.nb
        self.N = inp.nq
        self._keep = []

        def own(a, dt):
            a = np.ascontiguousarray(a, dtype=dt)
            self._keep.append(a)
            return a
        s = _Setup()
        s.natoms = inp.crystal.natoms
        s.mesh = (C.c_int32 * 3)(*[int(x) for x in inp.mesh])
        s.lattvec = (C.c_double * 9)(*[float(x) for x in np.asarray(inp.crystal.lattvec).reshape(-1)])
        s.masses = _ptr(own(inp.crystal.masses, np.float64))
        s.omega = _ptr(own(inp.omega, np.float64))
        eig = np.ascontiguousarray(inp.eig, dtype=np.complex128)
        s.eig = _ptr(own(eig.view(np.float64), np.float64))
        s.vg = _ptr(own(inp.vg, np.float64))
        if inp.ifc3 is not None:
            s.n3 = inp.ifc3[0].shape[0]
            s.atoms3 = _ptr(own(inp.ifc3[0], np.int32)); s.cells3 = _ptr(own(inp.ifc3[1], np.int32))
            s.phi3 = _ptr(own(inp.ifc3[2], np.float64))
        if inp.ifc4 is not None:
            s.n4 = inp.ifc4[0].shape[0]
            s.atoms4 = _ptr(own(inp.ifc4[0], np.int32)); s.cells4 = _ptr(own(inp.ifc4[1], np.int32))
            s.phi4 = _ptr(own(inp.ifc4[2], np.float64))
        s.T = float(inp.T if T is None else T)
        s.scale = float(inp.scale if scale is None else scale)
        s.ncut = float(ncut)
        s.sigma_const = float(sigma_const)
        self.s = s
        self.sp = C.cast(C.pointer(s), C.c_void_p)

    # -- scalar helpers ------------------------------------------------------------------------------------------------
    @staticmethod
    def constants():
        out = np.zeros(4)
        lib().orc_constants(_ptr(out))
        return {"C3": out[0], "C4": out[1], "Ckappa": out[2], "hbar_over_kb": out[3]}

    @staticmethod
    def recip(lattvec, mesh):
        B = np.zeros(9)
        lib().orc_recip(_ptr(np.ascontiguousarray(lattvec, dtype=np.float64)),
                        _ptr(np.ascontiguousarray(mesh, dtype=np.int32)), _ptr(B))
        return B.reshape(3, 3)

    def sigma(self, va, vb):
        va = np.ascontiguousarray(va, dtype=np.float64); vb = np.ascontiguousarray(vb, dtype=np.float64)
        self.lib.orc_sigma.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        return float(self.lib.orc_sigma(self.sp, _ptr(va), _ptr(vb)))

    def allowed(self, delta, sigma):
        return bool(self.lib.orc_allowed(self.sp, float(delta), float(sigma)))

    @staticmethod
    def be(omega, T):
        return float(lib().orc_be(float(omega), float(T)))

    def v3(self, lam, lam1, lam2, sign):
        out = np.zeros(2)
        self.lib.orc_v3(self.sp, int(lam), int(lam1), int(lam2), int(sign), _ptr(out))
        return complex(out[0], out[1])

    def v4(self, lam, lam1, lam2, lam3, s1, s2):
        out = np.zeros(2)
        self.lib.orc_v4(self.sp, int(lam), int(lam1), int(lam2), int(lam3), int(s1), int(s2), _ptr(out))
        return complex(out[0], out[1])

    # -- rates -----------------------------------------------------------------------------------------------------------
    def rates3(self, targets, weights_only=False):
        t = np.ascontiguousarray(targets, dtype=np.int32)
        g = np.zeros((t.size, 2)); w = np.zeros((t.size, 2)); c = np.zeros((t.size, 2), dtype=np.int64)
        rc = self.lib.orc_rates3(self.sp, _ptr(t), t.size, _ptr(g), _ptr(w), _ptr(c), int(weights_only))
        if rc != 0:
            raise MemoryError("oracle rates3")
        return g, w, c

    def rates4(self, targets, qp_begin=0, qp_end=None, weights_only=False):
        t = np.ascontiguousarray(targets, dtype=np.int32)
        qp_end = self.N if qp_end is None else qp_end
        g = np.zeros((t.size, 3)); w = np.zeros((t.size, 3)); c = np.zeros((t.size, 3), dtype=np.int64)
        rc = self.lib.orc_rates4(self.sp, _ptr(t), t.size, int(qp_begin), int(qp_end), _ptr(g), _ptr(w), _ptr(c),
                                 int(weights_only))
        if rc == -2:
            raise ValueError("oracle rates4: q' range outside the mesh")
        if rc != 0:
            raise MemoryError("oracle rates4")
        return g, w, c

    def list3(self, lam, ch):
        n = self.lib.orc_list3(self.sp, int(lam), int(ch), None, 0)
        pairs = np.zeros((max(n, 1), 2), dtype=np.int32)
        self.lib.orc_list3(self.sp, int(lam), int(ch), _ptr(pairs), n)
        return pairs[:n]

    def list4(self, lam, ch, qp_begin=0, qp_end=None):
        qp_end = self.N if qp_end is None else qp_end
        n = self.lib.orc_list4(self.sp, int(lam), int(ch), int(qp_begin), int(qp_end), None, 0)
        if n < 0:
            raise ValueError("oracle list4: q' range outside the mesh")
        tr = np.zeros((max(n, 1), 3), dtype=np.int32)
        self.lib.orc_list4(self.sp, int(lam), int(ch), int(qp_begin), int(qp_end), _ptr(tr), n)
        return tr[:n]

    def kappa(self, gamma_total):
        g = np.ascontiguousarray(gamma_total, dtype=np.float64).reshape(-1)
        assert g.size == self.N * self.nb
        k = np.zeros(9)
        self.lib.orc_kappa(self.sp, _ptr(g), _ptr(k))
        return k.reshape(3, 3)

    @staticmethod
    def num_threads():
        return int(lib().orc_num_threads())
