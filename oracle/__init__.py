"""oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes access to oracle/vmg_oracle.c, the plain CPU multigrid the CUDA path is checked against.
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import this
package; nothing under paper_2507_08200_b200/ does, and this package imports nothing from there.

Arrays are numpy fp64, C-order, indexed [k, j, i] (x fastest); see the header of vmg_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "vmg_oracle.c")
_SRC_AMR = os.path.join(_HERE, "amr_oracle.c")     # the two-level composite solve (N4, second half), same library
# VMG_ORACLE_LIB: another build of the same source (e.g. with -fsanitize=address,undefined, profiles/r2_sanitizers.md)
_LIB = os.environ.get("VMG_ORACLE_LIB") or os.path.join(_HERE, "libvmg_oracle.so")

STATUS = {0: "OK", 1: "MAXCYCLES", 2: "STALLED", -1: "ERR_ARG", -2: "ERR_SIZE", -3: "ERR_STATE",
          -4: "ERR_SINGULAR", -5: "ERR_DIVERGED"}


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain flags, no contraction, OpenMP over k-planes)."""
    if os.environ.get("VMG_ORACLE_LIB"):
        return _LIB
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_AMR)):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-Wall",
               "-o", _LIB, _SRC, _SRC_AMR, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.ovmg_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int,
                                     C.c_double, C.c_double, C.c_double]
        _lib.ovmg_destroy.argtypes = [C.c_void_p]
        _lib.ovmg_set_coeffs.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, C.c_double, C.c_double]
        _lib.ovmg_set_bc.argtypes = [C.c_void_p, C.POINTER(C.c_int), C.POINTER(_dp)]
        _lib.ovmg_set_option.argtypes = [C.c_void_p, C.c_char_p, C.c_double]
        _lib.ovmg_solve.argtypes = [C.c_void_p, _dp, _dp, C.c_double, C.c_int]
        _lib.ovmg_set_mask.argtypes = [C.c_void_p, C.c_void_p, C.c_int, _dp]
        _lib.ovmg_solve_pcg.argtypes = [C.c_void_p, _dp, _dp, C.c_double, C.c_int]
        _lib.ovmg_get_info.argtypes = [C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_double), _dp]
        _lib.ovmg_num_levels.argtypes = [C.c_void_p]
        _lib.ovmg_level_dims.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int)]
        _lib.ovmg_get_level_coeffs.argtypes = [C.c_void_p, C.c_int, _dp, _dp, _dp, _dp]
        _lib.ovmg_get_level_adiag.argtypes = [C.c_void_p, C.c_int, _dp]
        _lib.ovmg_apply.argtypes = [C.c_void_p, C.c_int, _dp, _dp]
        _lib.ovmg_fold_bc.argtypes = [C.c_void_p, _dp, _dp]
        _lib.ovmg_smooth.argtypes = [C.c_void_p, C.c_int, _dp, _dp, C.c_int]
        _lib.ovmg_residual.argtypes = [C.c_void_p, C.c_int, _dp, _dp, _dp]
        _lib.ovmg_restrict.argtypes = [C.c_void_p, C.c_int, _dp, _dp]
        _lib.ovmg_prolong_add.argtypes = [C.c_void_p, C.c_int, _dp, _dp]
        _lib.ovmg_vcycle.argtypes = [C.c_void_p, _dp, _dp]
        _ip = C.POINTER(C.c_int)
        _lib.oamr_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int, _ip, _ip]
        _lib.oamr_destroy.argtypes = [C.c_void_p]
        _pp = C.POINTER(_dp)
        _lib.oamr_set_coeffs.argtypes = [C.c_void_p] + [_dp] * 4 + [_pp] * 4 + [C.c_double, C.c_double]
        _lib.oamr_set_bc.argtypes = [C.c_void_p, _ip, C.POINTER(_dp)]
        _lib.oamr_set_option.argtypes = [C.c_void_p, C.c_char_p, C.c_double]
        _lib.oamr_fine_dims.argtypes = [C.c_void_p, C.c_int, _ip]
        _lib.oamr_apply.argtypes = [C.c_void_p, _dp, _pp, _dp, _pp]
        _lib.oamr_average_down.argtypes = [C.c_void_p, _dp, _pp]
        _lib.oamr_solve.argtypes = [C.c_void_p, _dp, _pp, _dp, _pp, C.c_double, C.c_int]
        _lib.oamr_get_info.argtypes = [C.c_void_p, _ip, C.POINTER(C.c_double), _dp]
    return _lib


def _p(arr: Optional[np.ndarray]):
    if arr is None:
        return None
    assert arr.dtype == np.float64 and arr.flags["C_CONTIGUOUS"]
    return arr.ctypes.data_as(_dp)


def _c(arr) -> Optional[np.ndarray]:
    return None if arr is None else np.ascontiguousarray(arr, dtype=np.float64)


class OracleError(RuntimeError):
    def __init__(self, code: int, where: str):
        super().__init__(f"oracle {where}: {STATUS.get(code, code)}")
        self.code = code


class Oracle:
    """One multigrid hierarchy on an nx x ny x nz box (nz == 1: 2-D)."""

    def __init__(self, nx: int, ny: int, nz: int, dx: float, dy: float, dz: float):
        self._h = C.c_void_p()
        rc = lib().ovmg_create(C.byref(self._h), nx, ny, nz, dx, dy, dz)
        if rc != 0:
            self._h = None
            raise OracleError(rc, "create")
        self.nx, self.ny, self.nz = nx, ny, nz

    @classmethod
    def from_problem(cls, p) -> "Oracle":
        o = cls(p.nx, p.ny, p.nz, p.dx, p.dy, p.dz)
        o.set_coeffs(p.a, p.bx, p.by, p.bz, p.alpha, p.beta)
        o.set_bc(p.bc_type, p.bc_value)
        return o

    def close(self):
        if getattr(self, "_h", None):
            lib().ovmg_destroy(self._h)
            self._h = None

    __del__ = close

    def _chk(self, rc: int, where: str):
        if rc < 0:
            raise OracleError(rc, where)
        return rc

    # -- boundary ---------------------------------------------------------------------------------
    def set_coeffs(self, a, bx, by, bz, alpha: float, beta: float):
        a, bx, by, bz = _c(a), _c(bx), _c(by), _c(bz)
        self._chk(lib().ovmg_set_coeffs(self._h, _p(a), _p(bx), _p(by), _p(bz), alpha, beta), "set_coeffs")

    def set_bc(self, types: Sequence[int], values: Optional[List[Optional[np.ndarray]]] = None):
        t = (C.c_int * 6)(*[int(v) for v in types])
        keep = [_c(v) for v in (values or [None] * 6)]
        arr = (_dp * 6)(*[_p(v) for v in keep])
        self._chk(lib().ovmg_set_bc(self._h, t, arr), "set_bc")

    def set_mask(self, mask, kind: int, cval=None):
        """Cell mask (1 valid, 0 covered), BC kind at the covered-valid interfaces, Dirichlet values of covered cells.
        Call set_coeffs afterwards (it applies the mask)."""
        m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
        cv = None if cval is None else _c(cval)
        self._keep_mask = (m, cv)
        self._chk(lib().ovmg_set_mask(self._h, None if m is None else m.ctypes.data_as(C.c_void_p), int(kind),
                                      None if cv is None else _p(cv)), "set_mask")

    def set_option(self, key: str, v: float):
        self._chk(lib().ovmg_set_option(self._h, key.encode(), float(v)), "set_option")

    def solve_pcg(self, rhs, phi0=None, rtol: float = 1e-12, max_iter: int = 50):
        """MG-preconditioned conjugate gradients. Returns (phi, status, iterations, relres, history)."""
        return self.solve(rhs, phi0, rtol, max_iter, _fn="ovmg_solve_pcg")

    def solve(self, rhs, phi0=None, rtol: float = 1e-12, max_vcycles: int = 50, _fn: str = "ovmg_solve"):
        """Returns (phi, status, cycles, relres, history)."""
        rhs = _c(rhs)
        phi = np.zeros_like(rhs) if phi0 is None else np.array(phi0, dtype=np.float64, order="C")
        status = getattr(lib(), _fn)(self._h, _p(rhs), _p(phi), rtol, max_vcycles)
        self._chk(status, "solve") if status not in (-5,) else None
        cyc, rr = C.c_int(), C.c_double()
        hist = np.zeros(max_vcycles + 1)
        lib().ovmg_get_info(self._h, C.byref(cyc), C.byref(rr), _p(hist))
        return phi, status, cyc.value, rr.value, hist[:cyc.value + 1].copy()

    # -- per-step entry points ----------------------------------------------------------------------
    @property
    def num_levels(self) -> int:
        return lib().ovmg_num_levels(self._h)

    def level_dims(self, lev: int):
        d = (C.c_int * 3)()
        self._chk(lib().ovmg_level_dims(self._h, lev, d), "level_dims")
        return d[0], d[1], d[2]

    def _zeros(self, lev: int):
        nx, ny, nz = self.level_dims(lev)
        return np.zeros((nz, ny, nx))

    def level_coeffs(self, lev: int):
        nx, ny, nz = self.level_dims(lev)
        a, bx = np.zeros((nz, ny, nx)), np.zeros((nz, ny, nx + 1))
        by, bz = np.zeros((nz, ny + 1, nx)), np.zeros((nz + 1, ny, nx))
        self._chk(lib().ovmg_get_level_coeffs(self._h, lev, _p(a), _p(bx), _p(by), _p(bz)), "level_coeffs")
        return a, bx, by, bz

    def level_adiag(self, lev: int):
        """Masking: the extra diagonal of a level (reading N4)."""
        out = self._zeros(lev)
        self._chk(lib().ovmg_get_level_adiag(self._h, lev, _p(out)), "level_adiag")
        return out

    def apply(self, phi, lev: int = 0):
        phi = _c(phi)
        out = np.zeros_like(phi)
        self._chk(lib().ovmg_apply(self._h, lev, _p(phi), _p(out)), "apply")
        return out

    def fold_bc(self, rhs):
        rhs = _c(rhs)
        out = np.zeros_like(rhs)
        self._chk(lib().ovmg_fold_bc(self._h, _p(rhs), _p(out)), "fold_bc")
        return out

    def smooth(self, phi, rhs, nsweeps: int, lev: int = 0):
        phi = np.array(phi, dtype=np.float64, order="C")
        rhs = _c(rhs)
        self._chk(lib().ovmg_smooth(self._h, lev, _p(phi), _p(rhs), nsweeps), "smooth")
        return phi

    def residual(self, phi, rhs, lev: int = 0):
        phi, rhs = _c(phi), _c(rhs)
        out = np.zeros_like(phi)
        self._chk(lib().ovmg_residual(self._h, lev, _p(phi), _p(rhs), _p(out)), "residual")
        return out

    def restrict(self, rfine, lev: int = 0):
        rfine = _c(rfine)
        out = self._zeros(lev + 1)
        self._chk(lib().ovmg_restrict(self._h, lev, _p(rfine), _p(out)), "restrict")
        return out

    def prolong_add(self, phifine, ecoarse, lev: int = 0):
        phi = np.array(phifine, dtype=np.float64, order="C")
        e = _c(ecoarse)
        self._chk(lib().ovmg_prolong_add(self._h, lev, _p(phi), _p(e)), "prolong_add")
        return phi

    def vcycle(self, phi, btilde):
        phi = np.array(phi, dtype=np.float64, order="C")
        bt = _c(btilde)
        self._chk(lib().ovmg_vcycle(self._h, _p(phi), _p(bt)), "vcycle")
        return phi


class AmrOracle:
    """Two-level composite solve (amr_oracle.c): an nx x ny x nz coarse box with patches of coarse cells [lo, hi) refined
    by 2.  lo, hi: one triple (a single patch: fine arrays are then passed and returned bare) or lists of triples (fine
    arrays as lists, one entry per patch).  Coarse arrays [k, j, i] on the box, fine arrays [K, J, I] on a patch."""

    def __init__(self, nx, ny, nz, dx, dy, dz, lo, hi):
        self._h = C.c_void_p()
        self._single = not isinstance(lo[0], (list, tuple, np.ndarray))
        los = [lo] if self._single else list(lo)
        his = [hi] if self._single else list(hi)
        self.np = len(los)
        flat = lambda v: (C.c_int * (3 * self.np))(*[int(x) for t in v for x in t])
        rc = lib().oamr_create(C.byref(self._h), nx, ny, nz, dx, dy, dz, self.np, flat(los), flat(his))
        if rc != 0:
            self._h = None
            raise OracleError(rc, "amr create")
        self.coarse_shape = (nz, ny, nx)
        self.fine_shapes = []
        for q in range(self.np):
            d = (C.c_int * 3)()
            lib().oamr_fine_dims(self._h, q, d)
            self.fine_shapes.append((d[2], d[1], d[0]))
        self.fine_shape = self.fine_shapes[0]

    def close(self):
        if getattr(self, "_h", None):
            lib().oamr_destroy(self._h)
            self._h = None

    __del__ = close

    def _chk(self, rc, where):
        if rc < 0:
            raise OracleError(rc, where)
        return rc

    def _list(self, x):
        return [x] if self._single else list(x)

    def _ptrs(self, arrs):
        """array of np pointers (NULL entries allowed) + the arrays kept alive"""
        keep = [_c(x) for x in arrs]
        return (_dp * self.np)(*[_p(x) for x in keep]), keep

    def set_coeffs(self, coarse, fine, alpha: float, beta: float):
        """coarse: (a, bx, by, bz); fine: the same per patch (entries may be None: a = 0, b = 1)."""
        cc = [_c(x) for x in coarse]
        per = self._list(fine)
        cols = [self._ptrs([f[i] for f in per]) for i in range(4)]
        self._chk(lib().oamr_set_coeffs(self._h, *[_p(x) for x in cc], *[c[0] for c in cols], alpha, beta), "amr set_coeffs")

    def set_bc(self, types, values=None):
        t = (C.c_int * 6)(*[int(v) for v in types])
        keep = [_c(v) for v in (values or [None] * 6)]
        arr = (_dp * 6)(*[_p(v) for v in keep])
        self._chk(lib().oamr_set_bc(self._h, t, arr), "amr set_bc")

    def set_option(self, key: str, v: float):
        self._chk(lib().oamr_set_option(self._h, key.encode(), float(v)), "amr set_option")

    def apply(self, phic, phif):
        phic = _c(phic)
        pf, keep = self._ptrs(self._list(phif))
        oc = np.zeros_like(phic)
        of = [np.zeros_like(x) for x in keep]
        po, _ = self._ptrs(of)
        self._chk(lib().oamr_apply(self._h, _p(phic), pf, _p(oc), po), "amr apply")
        return oc, (of[0] if self._single else of)

    def average_down(self, phic, phif):
        phic = np.array(phic, dtype=np.float64, order="C")
        pf, keep = self._ptrs(self._list(phif))
        self._chk(lib().oamr_average_down(self._h, _p(phic), pf), "amr average_down")
        return phic

    def solve(self, rhsc, rhsf, phic0=None, phif0=None, rtol: float = 1e-12, max_cycles: int = 50):
        """Returns (phic, phif, status, cycles, relres, history)."""
        rhsc = _c(rhsc)
        pr, rkeep = self._ptrs(self._list(rhsf))
        phic = np.zeros_like(rhsc) if phic0 is None else np.array(phic0, dtype=np.float64, order="C")
        phif = [np.zeros_like(x) for x in rkeep] if phif0 is None else \
            [np.array(x, dtype=np.float64, order="C") for x in self._list(phif0)]
        pp, _ = self._ptrs(phif)
        status = lib().oamr_solve(self._h, _p(rhsc), pr, _p(phic), pp, rtol, max_cycles)
        if status != -5:
            self._chk(status, "amr solve")
        cyc, rr = C.c_int(), C.c_double()
        hist = np.zeros(max_cycles + 1)
        lib().oamr_get_info(self._h, C.byref(cyc), C.byref(rr), _p(hist))
        return phic, (phif[0] if self._single else phif), status, cyc.value, rr.value, hist[:cyc.value + 1].copy()
