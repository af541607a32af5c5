"""Seeded synthetic inputs for the five BASELINE.json configs (recipe: DESIGN.md "Input recipe").

This module serves BOTH the CPU oracle (oracle/) and the CUDA path, and therefore holds none of the
method's arithmetic: no stencil, no smoother, no transfer operator -- only coefficient fields, boundary
data, right-hand sides and (for the manufactured-solution configs) the analytic solution they were made from.

Array convention (matches include/vmg.h): numpy C-order arrays indexed [k, j, i], x fastest.
  a, rhs, phi : (nz, ny, nx)        bx : (nz, ny, nx+1)     by : (nz, ny+1, nx)     bz : (nz+1, ny, nx)
  BC value planes: x faces (nz, ny), y faces (nz, nx), z faces (ny, nx); None = homogeneous.
Face order: XLO, XHI, YLO, YHI, ZLO, ZHI.  BC types: 0 = Dirichlet (value = phi on the face),
1 = Neumann (value = outward-normal derivative d(phi)/dn).

The paper's own workload (a 15-species Ar-H2 streamer state on 256x128x128, sec. 6.1,
PAPER.md:305-307 sec. 7) exists only inside a Vidyut3d run; these fields take its shapes, sizes and value
structure and stand in for it.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

DIRICHLET = 0
NEUMANN = 1
XLO, XHI, YLO, YHI, ZLO, ZHI = range(6)


@dataclass
class Problem:
    name: str
    nx: int
    ny: int
    nz: int
    dx: float
    dy: float
    dz: float
    alpha: float
    beta: float
    a: Optional[np.ndarray]
    bx: np.ndarray
    by: np.ndarray
    bz: Optional[np.ndarray]
    bc_type: List[int]
    bc_value: List[Optional[np.ndarray]]
    rhs: np.ndarray
    rtol: float = 1e-12
    max_vcycles: int = 50
    exact: Optional[np.ndarray] = None      # analytic solution at cell centres, when there is one
    notes: dict = field(default_factory=dict)

    @property
    def ncells(self) -> int:
        return self.nx * self.ny * self.nz

    def phi0(self) -> np.ndarray:
        """Initial guess: all configs start from zero."""
        return np.zeros((self.nz, self.ny, self.nx))


# --------------------------------------------------------------------------------------------------
# Gaussian random field: g(x) = sigma*sqrt(2/M) * sum_m cos(k_m . x + theta_m), k_m ~ N(0, ell^-2 I),
# theta_m ~ U[0, 2pi).  Covariance sigma^2 exp(-r^2 / (2 ell^2)); analytic, resolution independent,
# with an analytic gradient (needed by the manufactured right-hand side of config 2).
# --------------------------------------------------------------------------------------------------
@dataclass
class GRF:
    k: np.ndarray       # (M, 3)
    theta: np.ndarray   # (M,)
    sigma: float

    @staticmethod
    def draw(seed: int, ell: float, sigma: float, modes: int = 64) -> "GRF":
        rng = np.random.Generator(np.random.PCG64(seed))
        k = rng.standard_normal((modes, 3)) / ell
        theta = rng.uniform(0.0, 2.0 * np.pi, modes)
        return GRF(k=k, theta=theta, sigma=sigma)

    def evaluate(self, xs, ys, zs, grad: bool = False):
        """Field on the tensor grid zs x ys x xs -> (len(zs), len(ys), len(xs)); optionally its gradient."""
        xs, ys, zs = (np.atleast_1d(np.asarray(v, dtype=np.float64)) for v in (xs, ys, zs))
        m = self.k.shape[0]
        c = self.sigma * np.sqrt(2.0 / m)
        ex = np.exp(1j * (np.outer(self.k[:, 0], xs) + self.theta[:, None]))    # (M, nx)
        ey = np.exp(1j * np.outer(self.k[:, 1], ys))                            # (M, ny)
        ez = np.exp(1j * np.outer(self.k[:, 2], zs))                            # (M, nz)
        g = np.empty((len(zs), len(ys), len(xs)))
        if grad:
            gx = np.empty_like(g)
            gy = np.empty_like(g)
            gz = np.empty_like(g)
            kx_ex = self.k[:, 0][:, None] * ex
        for kk in range(len(zs)):
            ayz = ey * ez[:, kk][:, None]                                        # (M, ny)
            g[kk] = c * (ayz.T @ ex).real
            if grad:
                gx[kk] = -c * (ayz.T @ kx_ex).imag
                gy[kk] = -c * ((self.k[:, 1][:, None] * ayz).T @ ex).imag
                gz[kk] = -c * ((self.k[:, 2][:, None] * ayz).T @ ex).imag
        if grad:
            return g, gx, gy, gz
        return g


def _centres(n: int, h: float) -> np.ndarray:
    return (np.arange(n) + 0.5) * h


def _faces(n: int, h: float) -> np.ndarray:
    return np.arange(n + 1) * h


def _ndtr(x: np.ndarray) -> np.ndarray:
    from scipy.special import ndtr
    return ndtr(x)


# --------------------------------------------------------------------------------------------------
# Config 1 (BASELINE.json configs[0]): 2-D Poisson, manufactured sin(pi x) sin(pi y)
# --------------------------------------------------------------------------------------------------
def config1(n: int = 64) -> Problem:
    h = 1.0 / n
    x = _centres(n, h)
    y = _centres(n, h)
    exact = (np.sin(np.pi * y)[:, None] * np.sin(np.pi * x)[None, :])[None, :, :]
    rhs = 2.0 * np.pi ** 2 * exact
    return Problem(
        name=f"config1_2d_poisson_{n}x{n}", nx=n, ny=n, nz=1, dx=h, dy=h, dz=1.0,
        alpha=0.0, beta=1.0, a=None,
        bx=np.ones((1, n, n + 1)), by=np.ones((1, n + 1, n)), bz=None,
        bc_type=[DIRICHLET] * 4 + [NEUMANN] * 2, bc_value=[None] * 6,
        rhs=np.ascontiguousarray(rhs), exact=np.ascontiguousarray(exact))


# --------------------------------------------------------------------------------------------------
# Config 2 (configs[1]): 3-D ABec, b = exp(GRF), manufactured phi = x + 0.1 sin(2 pi y) sin(2 pi z)
# Reading R6: Dirichlet / Neumann data are PLANES sampled from the manufactured solution.
# --------------------------------------------------------------------------------------------------
def config2(n: int = 128, seed: int = 1002) -> Problem:
    h = 1.0 / n
    xc, yc, zc = _centres(n, h), _centres(n, h), _centres(n, h)
    xf, yf, zf = _faces(n, h), _faces(n, h), _faces(n, h)
    grf = GRF.draw(seed, ell=0.1, sigma=1.0)
    a0, alpha, beta = 1.0e3, 1.0, 1.0
    tp = 2.0 * np.pi

    def phi_ex(x, y, z):
        return x[None, None, :] + 0.1 * np.sin(tp * y)[None, :, None] * np.sin(tp * z)[:, None, None]

    bx = np.exp(grf.evaluate(xf, yc, zc))
    by = np.exp(grf.evaluate(xc, yf, zc))
    bz = np.exp(grf.evaluate(xc, yc, zf))
    g, gx, gy, gz = grf.evaluate(xc, yc, zc, grad=True)
    b = np.exp(g)
    sy, cy = np.sin(tp * yc)[None, :, None], np.cos(tp * yc)[None, :, None]
    sz, cz = np.sin(tp * zc)[:, None, None], np.cos(tp * zc)[:, None, None]
    px = np.ones_like(g)
    py = 0.1 * tp * cy * sz * np.ones_like(g)
    pz = 0.1 * tp * sy * cz * np.ones_like(g)
    lap = -2.0 * 0.1 * tp ** 2 * sy * sz * np.ones_like(g)
    exact = phi_ex(xc, yc, zc)
    rhs = alpha * a0 * exact - beta * (b * (gx * px + gy * py + gz * pz) + b * lap)

    z0, z1 = np.zeros(1), np.ones(1)
    val = [None] * 6
    val[XLO] = phi_ex(z0, yc, zc)[:, :, 0]                                        # (nz, ny)
    val[XHI] = phi_ex(z1, yc, zc)[:, :, 0]
    # outward-normal derivatives on the y and z faces
    val[YLO] = np.broadcast_to(-(0.1 * tp * np.cos(tp * 0.0) * np.sin(tp * zc))[:, None], (n, n)).copy()
    val[YHI] = np.broadcast_to(+(0.1 * tp * np.cos(tp * 1.0) * np.sin(tp * zc))[:, None], (n, n)).copy()
    val[ZLO] = np.broadcast_to(-(0.1 * tp * np.sin(tp * yc) * np.cos(tp * 0.0))[:, None], (n, n)).copy()
    val[ZHI] = np.broadcast_to(+(0.1 * tp * np.sin(tp * yc) * np.cos(tp * 1.0))[:, None], (n, n)).copy()
    return Problem(
        name=f"config2_abec_mms_{n}^3", nx=n, ny=n, nz=n, dx=h, dy=h, dz=h,
        alpha=alpha, beta=beta, a=np.full((n, n, n), a0), bx=bx, by=by, bz=bz,
        bc_type=[DIRICHLET, DIRICHLET, NEUMANN, NEUMANN, NEUMANN, NEUMANN], bc_value=val,
        rhs=np.ascontiguousarray(rhs), exact=np.ascontiguousarray(exact),
        notes={"b_min": float(min(bx.min(), by.min(), bz.min())),
               "b_max": float(max(bx.max(), by.max(), bz.max()))})


# --------------------------------------------------------------------------------------------------
# Config 3 (configs[2], headline): electrostatic Poisson on 256x128x128, cubic cells, box 2x1x1 (R14)
# Shapes follow the paper's streamer set-up: Gaussian seed, electrode potentials on the
# two x faces and homogeneous Neumann elsewhere.
# --------------------------------------------------------------------------------------------------
def config3(ny: int = 128, seed: int = 1003, rhs_zero: bool = False) -> Problem:
    nx, nz = 2 * ny, ny
    h = 1.0 / ny
    xc, yc, zc = _centres(nx, h), _centres(ny, h), _centres(nz, h)
    R = 0.05
    xh = (1.2, 0.5, 0.5)
    rng = np.random.Generator(np.random.PCG64(seed))
    u = rng.random((nz, ny, nx))
    r2 = ((xc - xh[0]) ** 2)[None, None, :] + ((yc - xh[1]) ** 2)[None, :, None] \
        + ((zc - xh[2]) ** 2)[:, None, None]
    n_e = np.exp(-r2 / R ** 2) + 0.01 * u
    rho2 = ((yc - 0.5) ** 2)[None, :, None] + ((zc - 0.5) ** 2)[:, None, None]
    n_ion = 0.8 * np.exp(-rho2 / R ** 2) * (0.5 * (1.0 + np.tanh((1.2 - xc) / R)))[None, None, :]
    rhs = n_ion - n_e
    rhs = rhs / np.abs(rhs).max()
    if rhs_zero:
        rhs = np.zeros_like(rhs)
    val = [None] * 6
    val[XLO] = np.ones((nz, ny))
    val[XHI] = np.zeros((nz, ny))
    return Problem(
        name=f"config3_poisson_streamer_{nx}x{ny}x{nz}", nx=nx, ny=ny, nz=nz, dx=h, dy=h, dz=h,
        alpha=0.0, beta=1.0, a=np.zeros((nz, ny, nx)),
        bx=np.ones((nz, ny, nx + 1)), by=np.ones((nz, ny + 1, nx)), bz=np.ones((nz + 1, ny, nx)),
        bc_type=[DIRICHLET, DIRICHLET, NEUMANN, NEUMANN, NEUMANN, NEUMANN], bc_value=val,
        rhs=np.ascontiguousarray(rhs))


# --------------------------------------------------------------------------------------------------
# Config 4 (configs[3]): implicit electron-energy-like solve, b over ~6-7 decades (R17, R19)
# dt from Eq. 20 with C_diff = 10, N_dim = 3, D_med = 1.
# --------------------------------------------------------------------------------------------------
def config4(ny: int = 128, seeds=(1004, 1005, 1006), sheath: bool = False) -> Problem:
    nx, nz = 2 * ny, ny
    h = 1.0 / ny
    xc, yc, zc = _centres(nx, h), _centres(ny, h), _centres(nz, h)
    xf, yf, zf = _faces(nx, h), _faces(ny, h), _faces(nz, h)
    g1 = GRF.draw(seeds[0], ell=0.1, sigma=1.0)
    g2 = GRF.draw(seeds[1], ell=0.1, sigma=1.0)
    dt = 10.0 * h * h / (2.0 * 3.0 * 1.0)
    Lx = nx * h

    def ne(x, y, z):
        v = 10.0 ** (-6.0 + 6.0 * _ndtr(g1.evaluate(x, y, z)))
        if sheath:   # "4b": sheath depletion at both electrodes
            v = v * (1e-4 + (1.0 - 1e-4) * np.sin(np.pi * x / Lx) ** 2)[None, None, :]
        return v

    def bface(x, y, z):
        return (5.0 / 3.0) * np.exp(0.5 * g2.evaluate(x, y, z)) * ne(x, y, z)

    a = ne(xc, yc, zc) / dt
    bx, by, bz = bface(xf, yc, zc), bface(xc, yf, zc), bface(xc, yc, zf)
    rng = np.random.Generator(np.random.PCG64(seeds[2]))
    rhs = rng.standard_normal((nz, ny, nx))
    return Problem(
        name=f"config4_energy_contrast_{nx}x{ny}x{nz}" + ("_sheath" if sheath else ""),
        nx=nx, ny=ny, nz=nz, dx=h, dy=h, dz=h, alpha=1.0, beta=1.0, a=a, bx=bx, by=by, bz=bz,
        bc_type=[DIRICHLET, DIRICHLET, NEUMANN, NEUMANN, NEUMANN, NEUMANN], bc_value=[None] * 6,
        rhs=rhs,
        notes={"dt": dt, "b_min": float(min(bx.min(), by.min(), bz.min())),
               "b_max": float(max(bx.max(), by.max(), bz.max()))})


# --------------------------------------------------------------------------------------------------
# Config 5 (configs[4]): 512^3 variable-coefficient ABec, 20 fixed V-cycles (R20)
# ell scales with 512/n so that reduced sizes keep 25.6 cells per correlation length.
# --------------------------------------------------------------------------------------------------
def config5(n: int = 512, seeds=(1007, 1008), cycles: int = 20) -> Problem:
    h = 1.0 / n
    ell = 0.05 * 512.0 / n
    xc, xf = _centres(n, h), _faces(n, h)
    grf = GRF.draw(seeds[0], ell=ell, sigma=2.0)
    bx = np.exp(grf.evaluate(xf, xc, xc))
    by = np.exp(grf.evaluate(xc, xf, xc))
    bz = np.exp(grf.evaluate(xc, xc, xf))
    rng = np.random.Generator(np.random.PCG64(seeds[1]))
    rhs = rng.standard_normal((n, n, n))
    return Problem(
        name=f"config5_abec_{n}^3", nx=n, ny=n, nz=n, dx=h, dy=h, dz=h, alpha=1.0, beta=1.0,
        a=np.full((n, n, n), 1.0e2), bx=bx, by=by, bz=bz,
        bc_type=[DIRICHLET, NEUMANN, NEUMANN, NEUMANN, NEUMANN, NEUMANN], bc_value=[None] * 6,
        rhs=rhs, rtol=0.0, max_vcycles=cycles,
        notes={"ell": ell, "b_min": float(min(bx.min(), by.min(), bz.min())),
               "b_max": float(max(bx.max(), by.max(), bz.max()))})


# --------------------------------------------------------------------------------------------------
# Small seeded problems for unit / parity tests: smooth positive a and b, any mix of BC types with
# inhomogeneous value planes, arbitrary (also non power-of-two) sizes.
# --------------------------------------------------------------------------------------------------
def random_problem(nx: int, ny: int, nz: int, seed: int = 0, bc_type=None, alpha: float = 1.0,
                   beta: float = 1.0, a_scale: float = 10.0, ell: float = 0.4, sigma: float = 1.0,
                   inhomogeneous: bool = True, spacing=None) -> Problem:
    rng = np.random.Generator(np.random.PCG64(seed))
    if spacing is None:
        h = 1.0 / max(ny, 2)
        spacing = (h, h, h)
    dx, dy, dz = spacing
    xc, yc, zc = _centres(nx, dx), _centres(ny, dy), _centres(nz, dz)
    xf, yf, zf = _faces(nx, dx), _faces(ny, dy), _faces(nz, dz)
    gb = GRF.draw(int(rng.integers(1 << 30)), ell=ell, sigma=sigma, modes=16)
    ga = GRF.draw(int(rng.integers(1 << 30)), ell=ell, sigma=0.5, modes=16)
    a = a_scale * np.exp(ga.evaluate(xc, yc, zc))
    bx = np.exp(gb.evaluate(xf, yc, zc))
    by = np.exp(gb.evaluate(xc, yf, zc))
    bz = np.exp(gb.evaluate(xc, yc, zf)) if nz > 1 else None
    if bc_type is None:
        bc_type = [int(v) for v in rng.integers(0, 2, 6)]
        if alpha == 0.0 or a_scale == 0.0:
            bc_type[XLO] = DIRICHLET
    shapes = [(nz, ny), (nz, ny), (nz, nx), (nz, nx), (ny, nx), (ny, nx)]
    val = [rng.standard_normal(s) if inhomogeneous else None for s in shapes]
    rhs = rng.standard_normal((nz, ny, nx))
    return Problem(
        name=f"random_{nx}x{ny}x{nz}_s{seed}", nx=nx, ny=ny, nz=nz, dx=dx, dy=dy, dz=dz,
        alpha=alpha, beta=beta, a=a, bx=bx, by=by, bz=bz, bc_type=list(bc_type), bc_value=val, rhs=rhs)


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


# --------------------------------------------------------------------------------------------------
# Two-level composite (AMR) inputs, SURVEY.md 8(f) N4 second half: a coarse box and one patch of coarse cells [lo, hi)
# refined by 2 (the paper refines where the reduced field and the electron density are large, i.e. around the streamer
# heads).  Every field is an analytic function (or a seeded GRF) sampled on both levels, so the coarse
# coefficients under the patch are consistent with the fine ones.  Fine arrays: the patch as a box of 2 (hi - lo) cells.
# --------------------------------------------------------------------------------------------------
@dataclass
class AmrProblem:
    name: str
    coarse: Problem                 # the box: coefficients, BC types and value planes, rhs (entries under the patch unused)
    lo: tuple
    hi: tuple
    a_f: Optional[np.ndarray]
    bx_f: Optional[np.ndarray]
    by_f: Optional[np.ndarray]
    bz_f: Optional[np.ndarray]
    rhs_f: np.ndarray
    rtol: float = 1e-12
    max_cycles: int = 50

    # several patches: lo, hi are lists of triples and a_f, bx_f, by_f, bz_f, rhs_f lists with one entry per patch
    @property
    def multi(self) -> bool:
        return isinstance(self.lo[0], (list, tuple))

    @property
    def fine_dims(self):
        c = self.coarse
        nd = 3 if c.nz > 1 else 2
        one = lambda lo, hi: tuple(2 * (hi[d] - lo[d]) if d < nd else 1 for d in range(3))
        return [one(l, u) for l, u in zip(self.lo, self.hi)] if self.multi else one(self.lo, self.hi)

    def coarse_coeffs(self):
        c = self.coarse
        return (c.a, c.bx, c.by, c.bz)

    def fine_coeffs(self):
        if self.multi:
            return [tuple(x) for x in zip(self.a_f, self.bx_f, self.by_f, self.bz_f)]
        return (self.a_f, self.bx_f, self.by_f, self.bz_f)


def _patch_axes(p: Problem, lo, hi):
    """cell-centre and face coordinates of the patch's fine cells along x, y, z"""
    nd = 3 if p.nz > 1 else 2
    h = (p.dx, p.dy, p.dz)
    cen, fac = [], []
    for d in range(3):
        if d < nd:
            m = 2 * (hi[d] - lo[d])
            cen.append(lo[d] * h[d] + _centres(m, h[d] / 2))
            fac.append(lo[d] * h[d] + _faces(m, h[d] / 2))
        else:
            cen.append(_centres(1, h[d]))
            fac.append(_faces(1, h[d]))
    return cen, fac


def amr_random_problem(nx: int, ny: int, nz: int, lo, hi, seed: int = 0, bc_type=None, alpha: float = 1.0,
                       a_scale: float = 10.0, ell: float = 0.4, sigma: float = 1.0, spacing=None) -> AmrProblem:
    """random_problem on the box with the same coefficient fields (GRFs) sampled on the patch's fine cells and faces."""
    rng = np.random.Generator(np.random.PCG64(seed))
    if spacing is None:
        h = 1.0 / max(ny, 2)
        spacing = (h, h, h)
    dx, dy, dz = spacing
    xc, yc, zc = _centres(nx, dx), _centres(ny, dy), _centres(nz, dz)
    xf, yf, zf = _faces(nx, dx), _faces(ny, dy), _faces(nz, dz)
    gb = GRF.draw(int(rng.integers(1 << 30)), ell=ell, sigma=sigma, modes=16)
    ga = GRF.draw(int(rng.integers(1 << 30)), ell=ell, sigma=0.5, modes=16)
    if bc_type is None:
        bc_type = [DIRICHLET, NEUMANN, NEUMANN, DIRICHLET, DIRICHLET, NEUMANN]
    shapes = [(nz, ny), (nz, ny), (nz, nx), (nz, nx), (ny, nx), (ny, nx)]
    val = [rng.standard_normal(s) for s in shapes]
    coarse = Problem(
        name=f"amr_box_{nx}x{ny}x{nz}_s{seed}", nx=nx, ny=ny, nz=nz, dx=dx, dy=dy, dz=dz, alpha=alpha, beta=1.0,
        a=a_scale * np.exp(ga.evaluate(xc, yc, zc)) if alpha > 0.0 else None,
        bx=np.exp(gb.evaluate(xf, yc, zc)), by=np.exp(gb.evaluate(xc, yf, zc)),
        bz=np.exp(gb.evaluate(xc, yc, zf)) if nz > 1 else None,
        bc_type=list(bc_type), bc_value=val, rhs=rng.standard_normal((nz, ny, nx)))
    def patch(lo_, hi_):
        (cx, cy, cz), (fx, fy, fz) = _patch_axes(coarse, lo_, hi_)
        m = tuple(len(v) for v in (cx, cy, cz))
        return (a_scale * np.exp(ga.evaluate(cx, cy, cz)) if alpha > 0.0 else None,
                np.exp(gb.evaluate(fx, cy, cz)), np.exp(gb.evaluate(cx, fy, cz)),
                np.exp(gb.evaluate(cx, cy, fz)) if nz > 1 else None,
                rng.standard_normal((m[2], m[1], m[0])))

    if isinstance(lo[0], (list, tuple)):       # several patches: lists, one entry per patch
        parts = [patch(l, u) for l, u in zip(lo, hi)]
        cols = [list(c) for c in zip(*parts)]
        return AmrProblem(name=f"amr_random_{nx}x{ny}x{nz}_s{seed}_{len(parts)}patches", coarse=coarse,
                          lo=[tuple(l) for l in lo], hi=[tuple(u) for u in hi],
                          a_f=cols[0], bx_f=cols[1], by_f=cols[2], bz_f=cols[3], rhs_f=cols[4])
    a_f, bx_f, by_f, bz_f, rhs_f = patch(lo, hi)
    return AmrProblem(name=f"amr_random_{nx}x{ny}x{nz}_s{seed}", coarse=coarse, lo=tuple(lo), hi=tuple(hi),
                      a_f=a_f, bx_f=bx_f, by_f=by_f, bz_f=bz_f, rhs_f=rhs_f)


def amr_streamer(ny: int = 128, seed: int = 1013, explicit_b: bool = True) -> AmrProblem:
    """Config 3 (Poisson, streamer-shaped space charge) with the region around the streamer head x_h = (1.2, 0.5, 0.5)
    refined: patch [15/16, 23/16] x [3/8, 5/8]^2 in units of L_y, i.e. 64 x 32 x 32 coarse cells of the 256 x 128 x 128
    box -> 128 x 64 x 64 fine cells."""
    base = config3(ny)
    lo = (15 * ny // 16, 3 * ny // 8, 3 * ny // 8)
    hi = (23 * ny // 16, 5 * ny // 8, 5 * ny // 8)
    (cx, cy, cz), _ = _patch_axes(base, lo, hi)
    R, xh = 0.05, (1.2, 0.5, 0.5)
    rng = np.random.Generator(np.random.PCG64(seed))

    def charge(xs, ys, zs):                                  # n_ion - n_e of config 3, with this level's own noise
        r2 = ((xs - xh[0]) ** 2)[None, None, :] + ((ys - xh[1]) ** 2)[None, :, None] + ((zs - xh[2]) ** 2)[:, None, None]
        n_e = np.exp(-r2 / R ** 2) + 0.01 * rng.random((len(zs), len(ys), len(xs)))
        rho2 = ((ys - 0.5) ** 2)[None, :, None] + ((zs - 0.5) ** 2)[:, None, None]
        n_ion = 0.8 * np.exp(-rho2 / R ** 2) * (0.5 * (1.0 + np.tanh((1.2 - xs) / R)))[None, None, :]
        return n_ion - n_e

    nx, nz = base.nx, base.nz
    raw_c = charge(_centres(nx, base.dx), _centres(ny, base.dy), _centres(nz, base.dz))
    scale = np.abs(raw_c).max()                              # one normalisation for both levels
    base.rhs = np.ascontiguousarray(raw_c / scale)
    rhs_f = np.ascontiguousarray(charge(cx, cy, cz) / scale)
    m = (len(cx), len(cy), len(cz))
    ones = lambda shape: np.ones(shape) if explicit_b else None
    if not explicit_b:
        base.bx = base.by = base.bz = None
    base.a = None
    return AmrProblem(
        name=f"amr_streamer_{nx}x{ny}x{nz}_patch{m[0]}x{m[1]}x{m[2]}", coarse=base, lo=lo, hi=hi, a_f=None,
        bx_f=ones((m[2], m[1], m[0] + 1)), by_f=ones((m[2], m[1] + 1, m[0])), bz_f=ones((m[2] + 1, m[1], m[0])),
        rhs_f=rhs_f)


def amr_streamers(ny: int = 128, seed: int = 1014) -> AmrProblem:
    """Three streamer heads side by side (the paper's 3-D case has fourteen): config 3's box and boundary data,
    the space charge of config 3 repeated at y = 3/16, 1/2, 13/16 and a patch of ny/2 x ny/4 x ny/4 coarse cells around every
    head (64 x 32 x 32 at ny = 128 -> 128 x 64 x 64 fine cells each), eight coarse cells apart in y."""
    base = config3(ny)
    yh = (3.0 / 16.0, 0.5, 13.0 / 16.0)
    los = [(15 * ny // 16, int(round(y * ny)) - ny // 8, 3 * ny // 8) for y in yh]
    his = [(23 * ny // 16, int(round(y * ny)) + ny // 8, 5 * ny // 8) for y in yh]
    R, xh, zh = 0.05, 1.2, 0.5
    rng = np.random.Generator(np.random.PCG64(seed))

    def charge(xs, ys, zs):
        out = -0.01 * rng.random((len(zs), len(ys), len(xs)))
        for y0 in yh:
            r2 = ((xs - xh) ** 2)[None, None, :] + ((ys - y0) ** 2)[None, :, None] + ((zs - zh) ** 2)[:, None, None]
            rho2 = ((ys - y0) ** 2)[None, :, None] + ((zs - zh) ** 2)[:, None, None]
            out += 0.8 * np.exp(-rho2 / R ** 2) * (0.5 * (1.0 + np.tanh((xh - xs) / R)))[None, None, :] - np.exp(-r2 / R ** 2)
        return out

    nx, nz = base.nx, base.nz
    raw_c = charge(_centres(nx, base.dx), _centres(ny, base.dy), _centres(nz, base.dz))
    scale = np.abs(raw_c).max()
    base.rhs = np.ascontiguousarray(raw_c / scale)
    base.a = None
    rhs_f, bxs, bys, bzs = [], [], [], []
    for lo, hi in zip(los, his):
        (cx, cy, cz), _ = _patch_axes(base, lo, hi)
        rhs_f.append(np.ascontiguousarray(charge(cx, cy, cz) / scale))
        m = (len(cx), len(cy), len(cz))
        bxs.append(np.ones((m[2], m[1], m[0] + 1))); bys.append(np.ones((m[2], m[1] + 1, m[0]))); bzs.append(np.ones((m[2] + 1, m[1], m[0])))
    return AmrProblem(name=f"amr_streamers_{nx}x{ny}x{nz}_3patches", coarse=base, lo=los, hi=his,
                      a_f=[None] * 3, bx_f=bxs, by_f=bys, bz_f=bzs, rhs_f=rhs_f)
