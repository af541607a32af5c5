"""Thin Python binding of libvmg.so (include/vmg.h): argument marshalling only.

torch is used for device memory (tensors' data_ptr) and streams; every step of the path runs in the CUDA
kernels of libvmg.so.  There is NO CPU fallback: if the library is missing or no CUDA device is present the
calls raise.  Arrays are torch fp64 CUDA tensors indexed [k, j, i] (x fastest), see paper_2507_08200_b200.inputs.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import List, Optional, Sequence

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libvmg.so")

STATUS = {0: "OK", 1: "MAXCYCLES", 2: "STALLED", -1: "ERR_ARG", -2: "ERR_SIZE", -3: "ERR_STATE",
          -4: "ERR_SINGULAR", -5: "ERR_DIVERGED", -6: "ERR_CUDA", -7: "ERR_ALLOC"}

# every symbol include/vmg.h declares (checked by tests/test_abi.py)
SYMBOLS = ["vmg_create", "vmg_create_batch", "vmg_set_coeffs", "vmg_set_bc", "vmg_set_mask", "vmg_solve", "vmg_solve_batch", "vmg_solve_pcg", "vmg_get_info", "vmg_set_option",
           "vmg_destroy", "vmg_strerror", "vmg_last_cuda_error", "vmg_num_levels", "vmg_level_dims",
           "vmg_get_level_coeffs", "vmg_step_fold_bc", "vmg_step_smooth", "vmg_step_residual",
           "vmg_step_residual_restrict", "vmg_step_prolong_correct", "vmg_step_down", "vmg_step_up", "vmg_step_vcycle", "vmg_step_norm_inf",
           "vmg_last_launch_count", "vmg_total_launch_count", "vmg_get_profile", "vmg_debug_pad_check",
           "vmg_norm_inf_static", "vmg_amr_create", "vmg_amr_fine_dims", "vmg_amr_set_coeffs", "vmg_amr_set_bc",
           "vmg_amr_set_option", "vmg_amr_solve", "vmg_amr_get_info", "vmg_amr_last_launch_count",
           "vmg_amr_last_cuda_error", "vmg_amr_destroy", "vmg_amr_debug_pad_check", "vmg_amr_num_patches"]

_lib = None
_vp = C.c_void_p


def load():
    """dlopen libvmg.so; raises if it has not been built (python -m paper_2507_08200_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2507_08200_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    lib.vmg_create.argtypes = [C.POINTER(_vp), C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, _vp]
    lib.vmg_create_batch.argtypes = [C.c_int, C.POINTER(_vp), C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, _vp]
    lib.vmg_set_coeffs.argtypes = [_vp, _vp, _vp, _vp, _vp, C.c_double, C.c_double]
    lib.vmg_set_bc.argtypes = [_vp, C.POINTER(C.c_int), C.POINTER(_vp)]
    lib.vmg_set_mask.argtypes = [_vp, _vp, C.c_int, _vp]
    lib.vmg_solve.argtypes = [_vp, _vp, _vp, C.c_double, C.c_int]
    lib.vmg_solve_pcg.argtypes = [_vp, _vp, _vp, C.c_double, C.c_int]
    lib.vmg_solve_batch.argtypes = [C.c_int, C.POINTER(_vp), C.POINTER(_vp), C.POINTER(_vp), C.c_double, C.c_int,
                                    C.POINTER(C.c_int)]
    lib.vmg_get_info.argtypes = [_vp, C.POINTER(C.c_int), C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.vmg_set_option.argtypes = [_vp, C.c_char_p, C.c_double]
    lib.vmg_destroy.argtypes = [_vp]
    lib.vmg_strerror.argtypes = [C.c_int]
    lib.vmg_strerror.restype = C.c_char_p
    lib.vmg_last_cuda_error.argtypes = [_vp]
    lib.vmg_num_levels.argtypes = [_vp]
    lib.vmg_level_dims.argtypes = [_vp, C.c_int, C.POINTER(C.c_int)]
    lib.vmg_get_level_coeffs.argtypes = [_vp, C.c_int, _vp, _vp, _vp, _vp]
    lib.vmg_step_fold_bc.argtypes = [_vp, _vp, _vp]
    lib.vmg_step_smooth.argtypes = [_vp, C.c_int, _vp, _vp, C.c_int]
    lib.vmg_step_residual.argtypes = [_vp, C.c_int, _vp, _vp, _vp]
    lib.vmg_step_residual_restrict.argtypes = [_vp, C.c_int, _vp, _vp, _vp]
    lib.vmg_step_prolong_correct.argtypes = [_vp, C.c_int, _vp, _vp]
    lib.vmg_step_down.argtypes = [_vp, C.c_int, _vp, _vp, _vp]
    lib.vmg_step_up.argtypes = [_vp, C.c_int, _vp, _vp, _vp]
    lib.vmg_step_vcycle.argtypes = [_vp, _vp, _vp]
    lib.vmg_step_norm_inf.argtypes = [_vp, _vp, C.c_longlong, C.POINTER(C.c_double)]
    lib.vmg_last_launch_count.argtypes = [_vp]
    lib.vmg_last_launch_count.restype = C.c_longlong
    lib.vmg_total_launch_count.argtypes = [_vp]
    lib.vmg_total_launch_count.restype = C.c_longlong
    lib.vmg_get_profile.argtypes = [_vp, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
    lib.vmg_debug_pad_check.argtypes = [_vp, C.POINTER(C.c_longlong)]
    lib.vmg_norm_inf_static.argtypes = [_vp, C.c_longlong, _vp, _vp, C.POINTER(C.c_char_p)]
    _ip = C.POINTER(C.c_int)
    lib.vmg_amr_create.argtypes = [C.POINTER(_vp), C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int, _ip, _ip, _vp]
    lib.vmg_amr_num_patches.argtypes = [_vp]
    lib.vmg_amr_fine_dims.argtypes = [_vp, C.c_int, _ip]
    _pv = C.POINTER(_vp)
    lib.vmg_amr_set_coeffs.argtypes = [_vp] + [_vp] * 4 + [_pv] * 4 + [C.c_double, C.c_double]
    lib.vmg_amr_set_bc.argtypes = [_vp, _ip, C.POINTER(_vp)]
    lib.vmg_amr_set_option.argtypes = [_vp, C.c_char_p, C.c_double]
    lib.vmg_amr_solve.argtypes = [_vp, _vp, _pv, _vp, _pv, C.c_double, C.c_int]
    lib.vmg_amr_get_info.argtypes = [_vp, _ip, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.vmg_amr_last_launch_count.argtypes = [_vp]
    lib.vmg_amr_last_launch_count.restype = C.c_longlong
    lib.vmg_amr_last_cuda_error.argtypes = [_vp]
    lib.vmg_amr_destroy.argtypes = [_vp]
    lib.vmg_amr_debug_pad_check.argtypes = [_vp, C.POINTER(C.c_longlong)]
    _lib = lib
    return lib


class VmgError(RuntimeError):
    def __init__(self, code: int, where: str, cuda: int = 0):
        msg = load().vmg_strerror(code).decode()
        super().__init__(f"{where}: {STATUS.get(code, code)} ({msg})" + (f" [cudaError {cuda}]" if cuda else ""))
        self.code = code


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2507_08200_b200 needs a CUDA device (no CPU fallback)")
    return torch


def _ptr(t) -> Optional[int]:
    if t is None:
        return None
    torch = _torch()
    assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous(), "need contiguous fp64 CUDA tensors"
    return t.data_ptr()


def solve_batch(solvers, rhs, phi, rtol: float = 1e-12, max_vcycles: int = 50) -> List[int]:
    """vmg_solve_batch: n independent solves advanced in lock-step (give every Vmg its own torch stream so that they
    overlap).  rhs, phi: lists of tensors; returns the list of status codes; raises on the first negative one."""
    n = len(solvers)
    assert len(rhs) == n and len(phi) == n
    lib = load()
    hs = (_vp * n)(*[s._h for s in solvers])
    r = (_vp * n)(*[_ptr(t) for t in rhs])
    p = (_vp * n)(*[_ptr(t) for t in phi])
    st = (C.c_int * n)()
    lib.vmg_solve_batch(n, hs, r, p, rtol, max_vcycles, st)
    out = [int(v) for v in st]
    for s, v in zip(solvers, out):
        if v < 0:
            raise VmgError(v, "vmg_solve_batch", lib.vmg_last_cuda_error(s._h))
    return out


def create_batch(k: int, nx: int, ny: int, nz: int, dx: float, dy: float, dz: float, stream=None):
    """vmg_create_batch: k handles in one allocation on one stream; solve_batch on exactly these runs the coarser levels of
    all of them as single launches (kernel-level batching).  Returns a list of Vmg."""
    torch = _torch()
    lib = load()
    stream = stream if stream is not None else torch.cuda.current_stream()
    sptr = stream.cuda_stream
    hs = (_vp * k)()
    rc = lib.vmg_create_batch(k, hs, nx, ny, nz, dx, dy, dz, _vp(sptr) if sptr else None)
    if rc != 0:
        raise VmgError(rc, "vmg_create_batch")
    return [Vmg(nx, ny, nz, dx, dy, dz, stream=stream, _handle=_vp(hs[i])) for i in range(k)]


class Vmg:
    """One solver handle (vmg_create ... vmg_destroy). Method names follow include/vmg.h."""

    def __init__(self, nx: int, ny: int, nz: int, dx: float, dy: float, dz: float, stream=None, _handle=None):
        torch = _torch()
        self._lib = load()
        self._h = _vp()
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        sptr = self.stream.cuda_stream
        if _handle is not None:          # a member of a vmg_create_batch group (create_batch below)
            self._h = _handle
        else:
            rc = self._lib.vmg_create(C.byref(self._h), nx, ny, nz, dx, dy, dz, _vp(sptr) if sptr else None)
            if rc != 0:
                self._h = None
                raise VmgError(rc, "vmg_create")
        self.nx, self.ny, self.nz = nx, ny, nz
        self.device = torch.device("cuda", torch.cuda.current_device())

    def _chk(self, rc: int, where: str) -> int:
        if rc < 0:
            raise VmgError(rc, where, self._lib.vmg_last_cuda_error(self._h))
        return rc

    def destroy(self):
        if getattr(self, "_h", None):
            self._lib.vmg_destroy(self._h)
            self._h = None

    __del__ = destroy

    # ---- the boundary ---------------------------------------------------------------------------------
    def set_coeffs(self, a, bx, by, bz, alpha: float, beta: float):
        self._chk(self._lib.vmg_set_coeffs(self._h, _ptr(a), _ptr(bx), _ptr(by), _ptr(bz), alpha, beta), "vmg_set_coeffs")

    def set_bc(self, types: Sequence[int], values: Optional[List] = None):
        t = (C.c_int * 6)(*[int(v) for v in types])
        vals = list(values) if values is not None else [None] * 6
        arr = (_vp * 6)(*[_ptr(v) for v in vals])
        self._chk(self._lib.vmg_set_bc(self._h, t, arr), "vmg_set_bc")

    def set_mask(self, mask, kind: int = 1, cval=None):
        """mask: contiguous uint8 CUDA tensor (1 valid, 0 covered) or None; kind: BC type of the covered/valid interfaces;
        cval: fp64 cell tensor with the Dirichlet value in covered cells.  Call set_coeffs afterwards."""
        mp = None
        if mask is not None:
            torch = _torch()
            assert mask.is_cuda and mask.dtype == torch.uint8 and mask.is_contiguous(), "need a contiguous uint8 CUDA mask"
            mp = mask.data_ptr()
        self._chk(self._lib.vmg_set_mask(self._h, mp, int(kind), _ptr(cval)), "vmg_set_mask")

    def set_option(self, key: str, v: float):
        self._chk(self._lib.vmg_set_option(self._h, key.encode(), float(v)), "vmg_set_option")

    def solve(self, rhs, phi, rtol: float = 1e-12, max_vcycles: int = 50) -> int:
        """phi: initial guess in, solution out (in place). Returns the status code (>= 0)."""
        return self._chk(self._lib.vmg_solve(self._h, _ptr(rhs), _ptr(phi), rtol, max_vcycles), "vmg_solve")

    def solve_pcg(self, rhs, phi, rtol: float = 1e-12, max_iter: int = 50) -> int:
        """MG-preconditioned conjugate gradients; phi: initial guess in, solution out. Returns the status code (>= 0)."""
        return self._chk(self._lib.vmg_solve_pcg(self._h, _ptr(rhs), _ptr(phi), rtol, max_iter), "vmg_solve_pcg")

    def get_info(self):
        cyc, rr = C.c_int(), C.c_double()
        self._lib.vmg_get_info(self._h, C.byref(cyc), C.byref(rr), None)
        hist = (C.c_double * (cyc.value + 1))()
        self._lib.vmg_get_info(self._h, None, None, hist)
        return cyc.value, rr.value, list(hist)

    def last_launch_count(self) -> int:
        return int(self._lib.vmg_last_launch_count(self._h))

    def total_launch_count(self) -> int:
        return int(self._lib.vmg_total_launch_count(self._h))

    PROFILE_CLASSES = ["smooth_l0", "residual_restrict_l0", "prolong_correct_l0", "coarse_levels", "norms",
                       "fold_bc", "phi_copies", "set_coeffs"]

    def get_profile(self):
        """{class: (ms, launches)} accumulated since set_option("profile", 1)."""
        ms, ln = (C.c_double * 8)(), (C.c_longlong * 8)()
        self._chk(self._lib.vmg_get_profile(self._h, ms, ln), "vmg_get_profile")
        return {k: (ms[i], ln[i]) for i, k in enumerate(self.PROFILE_CLASSES)}

    def pad_check(self) -> int:
        """Non-zero elements among the zero pads of the handle's internal arrays (must be 0)."""
        n = C.c_longlong()
        self._chk(self._lib.vmg_debug_pad_check(self._h, C.byref(n)), "vmg_debug_pad_check")
        return n.value

    # ---- introspection / single steps ---------------------------------------------------------------------
    @property
    def num_levels(self) -> int:
        return self._lib.vmg_num_levels(self._h)

    def level_dims(self, level: int):
        d = (C.c_int * 3)()
        self._chk(self._lib.vmg_level_dims(self._h, level, d), "vmg_level_dims")
        return d[0], d[1], d[2]

    def _empty(self, level: int):
        nx, ny, nz = self.level_dims(level)
        return _torch().empty((nz, ny, nx), dtype=_torch().float64, device=self.device)

    def get_level_coeffs(self, level: int):
        torch = _torch()
        nx, ny, nz = self.level_dims(level)
        mk = lambda *s: torch.zeros(s, dtype=torch.float64, device=self.device)
        a, bx, by, bz = mk(nz, ny, nx), mk(nz, ny, nx + 1), mk(nz, ny + 1, nx), mk(nz + 1, ny, nx)
        self._chk(self._lib.vmg_get_level_coeffs(self._h, level, _ptr(a), _ptr(bx), _ptr(by), _ptr(bz)),
                  "vmg_get_level_coeffs")
        return a, bx, by, bz

    def step_fold_bc(self, rhs):
        out = _torch().empty_like(rhs)
        self._chk(self._lib.vmg_step_fold_bc(self._h, _ptr(rhs), _ptr(out)), "vmg_step_fold_bc")
        return out

    def step_smooth(self, level: int, phi, rhs, nsweeps: int):
        phi = phi.clone()
        self._chk(self._lib.vmg_step_smooth(self._h, level, _ptr(phi), _ptr(rhs), nsweeps), "vmg_step_smooth")
        return phi

    def step_residual(self, level: int, phi, rhs):
        out = _torch().empty_like(phi)
        self._chk(self._lib.vmg_step_residual(self._h, level, _ptr(phi), _ptr(rhs), _ptr(out)), "vmg_step_residual")
        return out

    def step_residual_restrict(self, level: int, phi, rhs):
        out = self._empty(level + 1)
        self._chk(self._lib.vmg_step_residual_restrict(self._h, level, _ptr(phi), _ptr(rhs), _ptr(out)),
                  "vmg_step_residual_restrict")
        return out

    def step_prolong_correct(self, level: int, phi, e_coarse):
        phi = phi.clone()
        self._chk(self._lib.vmg_step_prolong_correct(self._h, level, _ptr(phi), _ptr(e_coarse)),
                  "vmg_step_prolong_correct")
        return phi

    def step_down(self, level: int, phi, rhs):
        """nu1 sweeps, then residual + restriction: returns (phi, rhs_coarse)."""
        phi = phi.clone()
        out = self._empty(level + 1)
        self._chk(self._lib.vmg_step_down(self._h, level, _ptr(phi), _ptr(rhs), _ptr(out)), "vmg_step_down")
        return phi, out

    def step_up(self, level: int, phi, rhs, e_coarse):
        """prolongation + correction, then nu2 sweeps: returns phi."""
        phi = phi.clone()
        self._chk(self._lib.vmg_step_up(self._h, level, _ptr(phi), _ptr(rhs), _ptr(e_coarse)), "vmg_step_up")
        return phi

    def step_vcycle(self, phi, btilde):
        phi = phi.clone()
        self._chk(self._lib.vmg_step_vcycle(self._h, _ptr(phi), _ptr(btilde)), "vmg_step_vcycle")
        return phi

    def step_norm_inf(self, v) -> float:
        out = C.c_double()
        self._chk(self._lib.vmg_step_norm_inf(self._h, _ptr(v), v.numel(), C.byref(out)), "vmg_step_norm_inf")
        return out.value


class VmgAmr:
    """Two-level composite solve (vmg_amr_* of include/vmg.h): an nx x ny x nz box with patches of coarse cells [lo, hi)
    refined by 2.  lo, hi: one triple (a single patch: fine tensors are then passed and returned bare) or lists of triples
    (fine tensors as lists, one entry per patch).  Coarse tensors [k, j, i] on the box, fine tensors [K, J, I] on a patch."""

    def __init__(self, nx, ny, nz, dx, dy, dz, lo, hi, stream=None):
        torch = _torch()
        self._lib = load()
        self._h = _vp()
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        sptr = self.stream.cuda_stream
        self._single = not isinstance(lo[0], (list, tuple))
        los = [lo] if self._single else list(lo)
        his = [hi] if self._single else list(hi)
        self.np = len(los)
        flat = lambda v: (C.c_int * (3 * self.np))(*[int(x) for t in v for x in t])
        rc = self._lib.vmg_amr_create(C.byref(self._h), nx, ny, nz, dx, dy, dz, self.np, flat(los), flat(his),
                                      _vp(sptr) if sptr else None)
        if rc != 0:
            self._h = None
            raise VmgError(rc, "vmg_amr_create")
        self.coarse_shape = (nz, ny, nx)
        self.fine_shapes = []
        for q in range(self.np):
            d = (C.c_int * 3)()
            self._lib.vmg_amr_fine_dims(self._h, q, d)
            self.fine_shapes.append((d[2], d[1], d[0]))
        self.fine_shape = self.fine_shapes[0]
        self._keep = None

    def _chk(self, rc, where):
        if rc < 0:
            raise VmgError(rc, where, self._lib.vmg_amr_last_cuda_error(self._h))
        return rc

    def destroy(self):
        if getattr(self, "_h", None):
            self._lib.vmg_amr_destroy(self._h)
            self._h = None

    __del__ = destroy

    def _list(self, x):
        return [x] if self._single else list(x)

    def _ptrs(self, tensors):
        return (_vp * self.np)(*[_ptr(t) for t in tensors])

    def set_coeffs(self, coarse, fine, alpha: float, beta: float):
        """coarse: (a, bx, by, bz) tensors; fine: the same per patch (None: a = 0, b = 1); borrowed until the next call."""
        per = [tuple(f) for f in self._list(fine)]
        self._keep = (tuple(coarse), per)
        cols = [self._ptrs([f[i] for f in per]) for i in range(4)]
        self._chk(self._lib.vmg_amr_set_coeffs(self._h, *[_ptr(t) for t in coarse], *cols, alpha, beta), "vmg_amr_set_coeffs")

    def set_bc(self, types, values=None):
        t = (C.c_int * 6)(*[int(v) for v in types])
        vals = list(values) if values is not None else [None] * 6
        arr = (_vp * 6)(*[_ptr(v) for v in vals])
        self._chk(self._lib.vmg_amr_set_bc(self._h, t, arr), "vmg_amr_set_bc")

    def set_option(self, key: str, v: float):
        self._chk(self._lib.vmg_amr_set_option(self._h, key.encode(), float(v)), "vmg_amr_set_option")

    def solve(self, rhs_c, rhs_f, phi_c=None, phi_f=None, rtol: float = 1e-12, max_cycles: int = 50):
        """Returns (phi_c, phi_f, status, cycles, relres, history); phi_c, phi_f are updated in place when given."""
        torch = _torch()
        rf = self._list(rhs_f)
        phi_c = torch.zeros_like(rhs_c) if phi_c is None else phi_c
        pf = [torch.zeros_like(r) for r in rf] if phi_f is None else self._list(phi_f)
        status = self._lib.vmg_amr_solve(self._h, _ptr(rhs_c), self._ptrs(rf), _ptr(phi_c), self._ptrs(pf), rtol, max_cycles)
        if status != -5:
            self._chk(status, "vmg_amr_solve")
        cyc, rr = C.c_int(), C.c_double()
        hist = (C.c_double * (max_cycles + 2))()
        self._lib.vmg_amr_get_info(self._h, C.byref(cyc), C.byref(rr), hist)
        return phi_c, (pf[0] if self._single else pf), status, cyc.value, rr.value, [hist[i] for i in range(cyc.value + 1)]

    def last_launch_count(self) -> int:
        return int(self._lib.vmg_amr_last_launch_count(self._h))

    def pad_check(self) -> int:
        n = C.c_longlong()
        self._chk(self._lib.vmg_amr_debug_pad_check(self._h, C.byref(n)), "vmg_amr_debug_pad_check")
        return n.value


NORM_INF_STATIC_MAX_N = 134217728   # VMG_NORM_INF_STATIC_MAX_N of include/vmg.h


def norm_inf_static(v, out, stream=None):
    """vmg_norm_inf_static: out[0] = max |v| with no allocation inside the library (static device scratch; calls that
    overlap on the GPU race).  v: fp64 CUDA tensor, out: fp64 CUDA tensor of one element, both caller-owned; asynchronous
    on `stream` (default: torch's current stream).  Returns out."""
    torch = _torch()
    lib = load()
    assert out.is_cuda and out.dtype == torch.float64 and out.numel() >= 1
    stream = stream if stream is not None else torch.cuda.current_stream()
    why = C.c_char_p()
    n = v.numel()
    rc = lib.vmg_norm_inf_static(_ptr(v) if n else None, n, out.data_ptr(), _vp(stream.cuda_stream) if stream.cuda_stream else None,
                                 C.byref(why))
    if rc != 0:
        raise RuntimeError(f"vmg_norm_inf_static: {STATUS.get(rc, rc)} ({(why.value or b'').decode()})")
    return out


def upload(p, device=None):
    """Problem (numpy, paper_2507_08200_b200.inputs) -> dict of fp64 CUDA tensors."""
    torch = _torch()
    dev = device or torch.device("cuda", torch.cuda.current_device())
    t = lambda x: None if x is None else torch.from_numpy(x).to(dev)
    return {"a": t(p.a), "bx": t(p.bx), "by": t(p.by), "bz": t(p.bz), "rhs": t(p.rhs),
            "bc_value": [t(v) for v in p.bc_value]}


def from_problem(p, stream=None):
    """Create a handle for a Problem and load its coefficients and boundary data. Returns (Vmg, tensors)."""
    d = upload(p)
    s = Vmg(p.nx, p.ny, p.nz, p.dx, p.dy, p.dz, stream=stream)
    s.set_coeffs(d["a"], d["bx"], d["by"], d["bz"], p.alpha, p.beta)
    s.set_bc(p.bc_type, d["bc_value"])
    return s, d
