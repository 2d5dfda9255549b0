"""ctypes loader for the ORACLE (oracle/pbref.c) -- test infrastructure, not product code.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this module.  It imports nothing from paper_1704_02745_b200/ and vice versa.
See pbref.c for what is computed and which passage of PAPER.md each step follows.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pbref.c")
_LIB = os.path.join(_HERE, "libpbref.so")

OK, INVALID, ALLOC, NOT_SPD, BREAKDOWN, MAXITER = 0, 1, 2, 4, 5, 6


def build(force: bool = False) -> str:
    """Compile pbref.c with gcc (plain C11 + OpenMP) into oracle/libpbref.so."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None
_dp = ctypes.POINTER(ctypes.c_double)


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        lib.pbref_create.argtypes = [ctypes.POINTER(vp), ci, ci, ci, cd, _dp, _dp, _dp, _dp, _dp, _dp]
        lib.pbref_set_rhs.argtypes = [vp, _dp, _dp]
        lib.pbref_apply.argtypes = [vp, _dp, _dp]
        lib.pbref_get_b.argtypes = [vp, _dp]
        lib.pbref_get_diag.argtypes = [vp, _dp]
        lib.pbref_solve.argtypes = [vp, cd, ci, ci, _dp, ctypes.POINTER(ci), _dp, _dp, _dp, _dp]
        lib.pbref_destroy.argtypes = [vp]
        lib.pbref_set_periodic.argtypes = [vp, ci]
        lib.pbref_num_threads.restype = ci
        lib.pbref_set_num_threads.argtypes = [ci]
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().pbref_num_threads())


def set_num_threads(n: int) -> None:
    """OpenMP threads of later oracle calls (timing only: results are bit-identical for any count)."""
    _load().pbref_set_num_threads(int(n))


def _ptr(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


class PBRef:
    """One operator (Eq. 3) + right-hand side (Eq. 4) held by the C oracle."""

    def __init__(self, nx, ny, nz, h, eps_x, eps_y, eps_z, kbar2=None, rhs=None, bc=None):
        lib = _load()
        self.nx, self.ny, self.nz, self.h = int(nx), int(ny), int(nz), float(h)
        ex, ey, ez = _f64(eps_x), _f64(eps_y), _f64(eps_z)
        assert ex.size == nz * ny * (nx + 1) and ey.size == nz * (ny + 1) * nx and ez.size == (nz + 1) * ny * nx
        kb, rh, bcv = _f64(kbar2), _f64(rhs), _f64(bc)
        self._h = ctypes.c_void_p()
        st = lib.pbref_create(ctypes.byref(self._h), nx, ny, nz, h, _ptr(ex), _ptr(ey), _ptr(ez),
                              _ptr(kb), _ptr(rh), _ptr(bcv))
        if st != OK:
            self._h = None
            raise RuntimeError(f"pbref_create failed: status {st}")

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)

    def set_rhs(self, rhs, bc):
        rh, bcv = _f64(rhs), _f64(bc)
        st = _load().pbref_set_rhs(self._h, _ptr(rh), _ptr(bcv))
        assert st == OK

    def set_periodic(self, flag=True):
        """Periodic boundary condition; call set_rhs afterwards to drop the ghost fold-in."""
        assert _load().pbref_set_periodic(self._h, 1 if flag else 0) == OK

    def apply(self, x):
        """y = A x (Eq. 3 left-hand side, 1/h^2 included, ghost x = 0)."""
        x = _f64(x).reshape(-1)
        y = np.empty_like(x)
        st = _load().pbref_apply(self._h, _ptr(x), _ptr(y))
        assert st == OK
        return y.reshape(self.shape)

    def b(self):
        out = np.empty(self.nx * self.ny * self.nz)
        _load().pbref_get_b(self._h, _ptr(out))
        return out.reshape(self.shape)

    def diag(self):
        out = np.empty(self.nx * self.ny * self.nz)
        _load().pbref_get_diag(self._h, _ptr(out))
        return out.reshape(self.shape)

    def solve(self, tol, maxiter, precond=True, history=False, phi0=None):
        """Jacobi-PCG.  Returns dict(phi, iters, relres, true_relres, status)."""
        phi = np.empty(self.nx * self.ny * self.nz)
        it = ctypes.c_int(0)
        rel = ctypes.c_double(0.0)
        trel = ctypes.c_double(0.0)
        hist = np.zeros(maxiter + 1) if history else None
        x0 = None if phi0 is None else _f64(phi0).reshape(-1)
        st = _load().pbref_solve(self._h, float(tol), int(maxiter), 1 if precond else 0, _ptr(phi),
                                 ctypes.byref(it), ctypes.byref(rel), ctypes.byref(trel), _ptr(hist), _ptr(x0))
        if st not in (OK, MAXITER, BREAKDOWN):
            raise RuntimeError(f"pbref_solve failed: status {st}")
        out = dict(phi=phi.reshape(self.shape), iters=it.value, relres=rel.value,
                   true_relres=trel.value, status=st)
        if history:
            out["history"] = hist[: it.value + 1]
        return out

    def close(self):
        if getattr(self, "_h", None):
            _load().pbref_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def from_inputs(inp) -> PBRef:
    """Build the oracle for a workloads.PBInputs."""
    return PBRef(*inp.args())
