"""Pins for the CPU oracle (oracle/vmg_oracle.c) against things other than itself.

Each test names the reading (SURVEY.md sec. 8(c) / DESIGN.md) or the paper passage it pins.
CPU only: runs under -m "not gpu".
"""
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import Oracle, OracleError
from paper_2507_08200_b200 import inputs
from paper_2507_08200_b200.inputs import DIRICHLET as D, NEUMANN as N

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def dense_from_apply(o: Oracle, lev: int = 0) -> np.ndarray:
    nx, ny, nz = o.level_dims(lev)
    n = nx * ny * nz
    A = np.zeros((n, n))
    for c in range(n):
        e = np.zeros(n)
        e[c] = 1.0
        A[:, c] = o.apply(e.reshape(nz, ny, nx), lev).ravel()
    return A


def brute_force_matrix(p) -> np.ndarray:
    """The level-0 matrix written directly from the finite-volume statement, cell by cell, as flux
    differences over the cell's faces (FV, second-order central diffusive flux):
        alpha a phi_c h^3 - beta * sum_faces (area * b_f * dphi/dn_f) = f h^3
    with dphi/dn across an interior face = (phi_nb - phi_c)/h, at a Dirichlet face = (0 - phi_c)/(h/2),
    at a Neumann face = 0 (homogeneous part).  Deliberately organised by FACES, not by the oracle's
    per-cell stencil, so a wrong face index or factor in either shows up."""
    nx, ny, nz = p.nx, p.ny, p.nz
    three_d = nz > 1
    h = (p.dx, p.dy, p.dz)
    vol = p.dx * p.dy * (p.dz if three_d else 1.0)
    area = (vol / p.dx, vol / p.dy, vol / p.dz if three_d else 0.0)
    n = nx * ny * nz
    A = np.zeros((n, n))
    idx = lambda i, j, k: i + nx * (j + ny * k)
    a = p.a if p.a is not None else np.zeros((nz, ny, nx))
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                A[idx(i, j, k), idx(i, j, k)] += p.alpha * a[k, j, i] * vol
    # x faces
    for k in range(nz):
        for j in range(ny):
            for f in range(nx + 1):
                b = p.bx[k, j, f]
                t = p.beta * area[0] * b / h[0]
                if 0 < f < nx:
                    l, r = idx(f - 1, j, k), idx(f, j, k)
                    A[l, l] += t; A[l, r] -= t; A[r, r] += t; A[r, l] -= t
                else:
                    c = idx(0, j, k) if f == 0 else idx(nx - 1, j, k)
                    if p.bc_type[0 if f == 0 else 1] == D:
                        A[c, c] += 2.0 * t
    for k in range(nz):
        for f in range(ny + 1):
            for i in range(nx):
                b = p.by[k, f, i]
                t = p.beta * area[1] * b / h[1]
                if 0 < f < ny:
                    l, r = idx(i, f - 1, k), idx(i, f, k)
                    A[l, l] += t; A[l, r] -= t; A[r, r] += t; A[r, l] -= t
                else:
                    c = idx(i, 0, k) if f == 0 else idx(i, ny - 1, k)
                    if p.bc_type[2 if f == 0 else 3] == D:
                        A[c, c] += 2.0 * t
    if three_d:
        for f in range(nz + 1):
            for j in range(ny):
                for i in range(nx):
                    b = p.bz[f, j, i]
                    t = p.beta * area[2] * b / h[2]
                    if 0 < f < nz:
                        l, r = idx(i, j, f - 1), idx(i, j, f)
                        A[l, l] += t; A[l, r] -= t; A[r, r] += t; A[r, l] -= t
                    else:
                        c = idx(i, j, 0) if f == 0 else idx(i, j, nz - 1)
                        if p.bc_type[4 if f == 0 else 5] == D:
                            A[c, c] += 2.0 * t
    return A / vol


MIXED = [D, N, N, D, D, N]


# ---- P1: dense direct solve -------------------------------------------------------------------------
@pytest.mark.parametrize("dims,bc,alpha", [((8, 8, 8), MIXED, 1.0), ((16, 8, 8), [D, D, N, N, N, N], 0.0),
                                           ((8, 8, 1), [D, N, N, D, N, N], 1.0), ((12, 6, 10), MIXED, 1.0)])
def test_p1_multigrid_converges_to_dense_direct_solution(dims, bc, alpha):
    p = inputs.random_problem(*dims, seed=11, bc_type=bc, alpha=alpha)
    o = Oracle.from_problem(p)
    A = dense_from_apply(o)
    bt = o.fold_bc(p.rhs)
    ref = np.linalg.solve(A, bt.ravel()).reshape(p.rhs.shape)
    phi, status, cycles, relres, hist = o.solve(p.rhs, rtol=1e-13, max_vcycles=60)
    assert status == 0 and relres <= 1e-13
    assert np.abs(phi - ref).max() <= 1e-11 * np.abs(ref).max()


@pytest.mark.parametrize("dims,bc", [((6, 4, 4), MIXED), ((4, 6, 1), [D, N, N, D, N, N]), ((5, 3, 4), [N, D, D, N, N, D])])
def test_p1b_apply_and_fold_bc_match_facewise_flux_assembly(dims, bc):
    p = inputs.random_problem(*dims, seed=5, bc_type=bc, spacing=(0.3, 0.2, 0.5))
    try:
        o = Oracle.from_problem(p)
    except OracleError:
        pytest.skip("size not coarsenable")
    A = dense_from_apply(o)
    B = brute_force_matrix(p)
    assert np.abs(A - B).max() <= 1e-13 * np.abs(B).max()
    # inhomogeneous part: A phi = btilde must hold for a field that satisfies the BC data exactly.
    # phi = const c: Dirichlet value c on Dirichlet faces, Neumann derivative 0 => A0*c - (btilde - f) = alpha a c
    c = 1.7
    vals = [np.full(s.shape, c if t == D else 0.0) for s, t in zip(p.bc_value, p.bc_type)]
    o.set_bc(p.bc_type, vals)
    bt0 = o.fold_bc(np.zeros_like(p.rhs))
    lhs = o.apply(np.full_like(p.rhs, c))
    assert np.abs(lhs - bt0 - p.alpha * p.a * c).max() <= 1e-12 * np.abs(lhs).max()


def test_p1c_neumann_value_sign_and_scale_linear_field():
    """phi = q*y is reproduced exactly by a scheme that is exact for linear fields: Neumann derivative -q on
    YLO, +q on YHI (outward normal, R5), Dirichlet planes q*y on the x faces, f = 0, a = 0, b variable in x
    only (so div(b grad phi) = 0 for phi = q*y)."""
    nx, ny, nz, q = 8, 8, 4, 0.7
    h = 1.0 / 8
    p = inputs.random_problem(nx, ny, nz, seed=2, bc_type=[D, D, N, N, N, N], alpha=0.0, spacing=(h, h, h))
    prof = np.exp(np.sin(np.arange(nx + 1) * 0.9))
    p.bx = np.broadcast_to(prof[None, None, :], p.bx.shape).copy()
    pc = 0.5 * (prof[1:] + prof[:-1])
    p.by = np.broadcast_to(pc[None, None, :], p.by.shape).copy()
    p.bz = np.broadcast_to(pc[None, None, :], p.bz.shape).copy()
    y = (np.arange(ny) + 0.5) * h
    exact = np.broadcast_to(q * y[None, :, None], (nz, ny, nx)).copy()
    vals = [np.broadcast_to(q * y[None, :], (nz, ny)).copy(), np.broadcast_to(q * y[None, :], (nz, ny)).copy(),
            np.full((nz, nx), -q), np.full((nz, nx), q), None, None]
    o = Oracle(nx, ny, nz, h, h, h)
    o.set_coeffs(None, p.bx, p.by, p.bz, 0.0, 1.0)
    o.set_bc([D, D, N, N, N, N], vals)
    phi, status, *_ = o.solve(np.zeros((nz, ny, nx)), rtol=1e-13)
    assert status == 0
    assert np.abs(phi - exact).max() <= 1e-11


# ---- P2: symmetry and positive definiteness -------------------------------------------------------------
def test_p2_operator_symmetric_positive_definite_every_level():
    p = inputs.random_problem(16, 8, 8, seed=3, bc_type=MIXED)
    o = Oracle.from_problem(p)
    for lev in range(o.num_levels):
        A = dense_from_apply(o, lev)
        assert np.abs(A - A.T).max() == 0.0
        assert np.linalg.eigvalsh(A).min() > 0.0


def test_p2_symmetry_large_grid_inner_products():
    p = inputs.config4(32)
    o = Oracle.from_problem(p)
    rng = np.random.default_rng(0)
    u, v = rng.standard_normal(p.rhs.shape), rng.standard_normal(p.rhs.shape)
    Au, Av = o.apply(u), o.apply(v)
    assert abs((u * Av).sum() - (Au * v).sum()) <= 1e-12 * abs((u * Av).sum())
    assert (u * Au).sum() > 0 and (v * Av).sum() > 0


def test_r16_pure_neumann_without_absorption_is_rejected():
    p = inputs.random_problem(8, 8, 8, seed=1, bc_type=[N] * 6, alpha=0.0)
    o = Oracle.from_problem(p)
    with pytest.raises(OracleError) as e:
        o.solve(p.rhs)
    assert e.value.code == -4


# ---- P3 / P4: manufactured solutions, second order --------------------------------------------------------
def test_p3_config1_mms_second_order():
    errs = []
    for n in (32, 64, 128):
        p = inputs.config1(n)
        phi, status, cycles, relres, _ = Oracle.from_problem(p).solve(p.rhs, rtol=1e-12)
        assert status == 0
        errs.append(np.abs(phi - p.exact).max())
    assert abs(errs[0] / errs[1] - 4.0) < 0.05 and abs(errs[1] / errs[2] - 4.0) < 0.05
    # closed form of the discrete error for this eigenfunction problem: the 5-point Laplacian with the
    # two-point Dirichlet closure has sin(pi x)sin(pi y) sampled at centres as an eigenvector with eigenvalue
    # 2*(2/h^2)(1 - cos(pi h)), so phi_h = exact * 2 pi^2 / that eigenvalue.
    h = 1.0 / 64
    lam = 2.0 * (2.0 / h ** 2) * (1.0 - np.cos(np.pi * h))
    expect = (2.0 * np.pi ** 2 / lam - 1.0) * np.sin(np.pi * (0.5 - h / 2)) ** 2
    assert abs(errs[1] - expect) <= 1e-9


def test_p4_config2_mms_second_order_variable_coefficients():
    errs = []
    for n in (16, 32, 64):
        p = inputs.config2(n)
        phi, status, cycles, relres, _ = Oracle.from_problem(p).solve(p.rhs, rtol=1e-12)
        assert status == 0
        errs.append(np.abs(phi - p.exact).max())
    orders = [np.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert 1.85 < orders[1] < 2.3 and orders[0] > 1.7, (errs, orders)


# ---- P5: exactness for a linear potential between two electrodes -----------------------------------------
def test_p5_linear_potential_exact():
    p = inputs.config3(16, rhs_zero=True)
    phi, status, cycles, relres, _ = Oracle.from_problem(p).solve(p.rhs, rtol=1e-13)
    x = (np.arange(p.nx) + 0.5) * p.dx
    exact = np.broadcast_to((1.0 - x / (p.nx * p.dx))[None, None, :], phi.shape)
    assert status == 0 and np.abs(phi - exact).max() <= 1e-11


# ---- P6: the closed form the paper prints (Eq. 24-27) -------------------------------------------------------
def test_p6_paper_closed_form_poisson_1d():
    phi_ex = lambda x: (x ** 4 - x) / 12.0
    rows = [l.split() for l in open(os.path.join(GOLDEN, "paper_eq27_poisson_1d.txt")) if not l.startswith("#")]
    for xs, num, den in rows:
        assert abs(phi_ex(float(xs)) - float(Fraction(int(num), int(den)))) < 1e-16
    errs = []
    for n in (32, 64, 128):
        h = 1.0 / n
        x = (np.arange(n) + 0.5) * h
        # pseudo-1-D: an n x n 2-D box, homogeneous Neumann in y, so the solution depends on x only
        rhs = np.broadcast_to(-(x ** 2)[None, None, :], (1, n, n)).copy()     # f = -x^2 (sign reading R1)
        o = Oracle(n, n, 1, h, h, 1.0)
        o.set_coeffs(None, None, None, None, 0.0, 1.0)
        o.set_bc([D, D, N, N, N, N], None)
        phi, status, *_ = o.solve(rhs, rtol=1e-12, max_vcycles=100)
        assert status == 0
        errs.append(np.abs(phi - phi_ex(x)[None, None, :]).max())
    assert abs(errs[0] / errs[1] - 4.0) < 0.1 and abs(errs[1] / errs[2] - 4.0) < 0.1
    assert errs[2] < 2e-5


# ---- P7: contraction factor per V-cycle (R13) ----------------------------------------------------------
def _contraction(hist):
    r = [hist[c] / hist[c - 1] for c in range(2, len(hist)) if hist[c] > 1e-13]
    return max(r), (hist[-1] / hist[0]) ** (1.0 / (len(hist) - 1))


@pytest.mark.parametrize("make", [lambda: inputs.config1(64), lambda: inputs.config2(64),
                                  lambda: inputs.config3(64), lambda: inputs.config4(64),
                                  lambda: inputs.config4(32, sheath=True)])
def test_p7_contraction_below_0p2(make):
    p = make()
    phi, status, cycles, relres, hist = Oracle.from_problem(p).solve(p.rhs, rtol=1e-12)
    assert status == 0 and relres <= 1e-12
    worst, mean = _contraction(hist)
    assert worst < 0.2 and mean < 0.2, (worst, mean, cycles)


@pytest.mark.slow
@pytest.mark.parametrize("make,cycles_expected", [(lambda: inputs.config2(128), (9, 11)),
                                                  (lambda: inputs.config3(128), (9, 12)),
                                                  (lambda: inputs.config4(128), (8, 11))])
def test_p7_contraction_full_size(make, cycles_expected):
    p = make()
    phi, status, cycles, relres, hist = Oracle.from_problem(p).solve(p.rhs, rtol=1e-12)
    worst, mean = _contraction(hist)
    assert status == 0 and worst < 0.2 and cycles_expected[0] <= cycles <= cycles_expected[1], (worst, cycles)


# ---- P8: row sums -------------------------------------------------------------------------------------------
def test_p8_constant_vector_all_neumann():
    p = inputs.random_problem(12, 8, 6, seed=9, bc_type=[N] * 6, alpha=1.0)
    a0 = 3.25
    p.a = np.full_like(p.a, a0)
    o = Oracle.from_problem(p)
    for lev in range(o.num_levels):
        nx, ny, nz = o.level_dims(lev)
        out = o.apply(np.ones((nz, ny, nx)), lev)
        scale = np.abs(o.level_coeffs(lev)[1]).max() / (p.dx * 2 ** lev) ** 2
        assert np.abs(out - a0).max() <= 1e-13 * scale


# ---- P9: invariances ------------------------------------------------------------------------------------------
def _permuted(p, perm):
    """Relabel axes: new axis order perm (tuple over 'xyz' indices of the OLD axes, for new x,y,z)."""
    ax = {0: 2, 1: 1, 2: 0}                                  # physical axis -> numpy axis of [k,j,i]
    tr = tuple(ax[perm[2 - d]] for d in range(3))            # numpy transpose for cell arrays
    n_old = (p.nx, p.ny, p.nz)
    h_old = (p.dx, p.dy, p.dz)
    b_old = (p.bx, p.by, p.bz)
    q = inputs.Problem(name="perm", nx=n_old[perm[0]], ny=n_old[perm[1]], nz=n_old[perm[2]],
                       dx=h_old[perm[0]], dy=h_old[perm[1]], dz=h_old[perm[2]], alpha=p.alpha, beta=p.beta,
                       a=np.ascontiguousarray(p.a.transpose(tr)),
                       bx=np.ascontiguousarray(b_old[perm[0]].transpose(tr)),
                       by=np.ascontiguousarray(b_old[perm[1]].transpose(tr)),
                       bz=np.ascontiguousarray(b_old[perm[2]].transpose(tr)),
                       bc_type=[0] * 6, bc_value=[None] * 6, rhs=np.ascontiguousarray(p.rhs.transpose(tr)))
    for dnew in range(3):
        dold = perm[dnew]
        others_new = [d for d in range(3) if d != dnew]       # plane axes (low axis fastest)
        others_old = [d for d in range(3) if d != dold]
        for side in range(2):
            q.bc_type[2 * dnew + side] = p.bc_type[2 * dold + side]
            v = p.bc_value[2 * dold + side]                   # indexed [hi_old, lo_old]
            # new plane is indexed [hi_new, lo_new] where new axis e corresponds to old axis perm[e]
            if (perm[others_new[0]], perm[others_new[1]]) == (others_old[0], others_old[1]):
                q.bc_value[2 * dnew + side] = np.ascontiguousarray(v)
            else:
                q.bc_value[2 * dnew + side] = np.ascontiguousarray(v.T)
    return q, tr


@pytest.mark.parametrize("perm", [(1, 0, 2), (2, 1, 0), (1, 2, 0), (0, 2, 1)])
def test_p9_axis_permutation_invariance(perm):
    p = inputs.random_problem(8, 12, 16, seed=21, bc_type=[D, N, N, D, N, N], spacing=(0.11, 0.07, 0.05))
    q, tr = _permuted(p, perm)
    phi_p, st_p, cyc_p, _, _ = Oracle.from_problem(p).solve(p.rhs, rtol=1e-12)
    phi_q, st_q, cyc_q, _, _ = Oracle.from_problem(q).solve(q.rhs, rtol=1e-12)
    assert st_p == 0 and st_q == 0 and cyc_p == cyc_q
    assert np.abs(phi_p.transpose(tr) - phi_q).max() <= 1e-12 * np.abs(phi_p).max()


def test_p9_scaling_invariance_pure_diffusion():
    p = inputs.random_problem(16, 8, 8, seed=4, bc_type=[D, D, N, N, N, N], alpha=0.0)
    o1 = Oracle.from_problem(p)
    phi1, *_ = o1.solve(p.rhs, rtol=1e-12)
    s = 2.0 ** 7                       # a power of two: the scaled problem is bit-identical arithmetic
    o2 = Oracle(p.nx, p.ny, p.nz, p.dx, p.dy, p.dz)
    o2.set_coeffs(None, p.bx * s, p.by * s, p.bz * s, 0.0, 1.0)
    o2.set_bc(p.bc_type, p.bc_value)
    phi2, *_ = o2.solve(p.rhs * s, rtol=1e-12)
    assert np.array_equal(phi1, phi2)


def _vcycle_matrix(o, shape):
    nz, ny, nx = shape
    n = nx * ny * nz
    M = np.zeros((n, n))
    for c in range(n):
        e = np.zeros(n)
        e[c] = 1.0
        M[:, c] = o.vcycle(np.zeros(shape), e.reshape(shape)).ravel()
    return M


def test_n2_symmetric_vcycle_is_a_symmetric_positive_definite_operator():
    """the preconditioner of ovmg_solve_pcg -- one V-cycle from zero with the post-smoothing (and the
    second half of the bottom sweeps) in the adjoint colour order -- must be a symmetric positive definite linear map
    r -> z; the default V-cycle (same colour order before and after) is NOT symmetric, which shows the check can fail."""
    p = inputs.random_problem(8, 8, 8, seed=2, bc_type=[D, N, N, D, N, N], inhomogeneous=False)
    o = Oracle.from_problem(p)
    shape = p.rhs.shape
    o.set_option("symmetric", 1)
    M = _vcycle_matrix(o, shape)
    assert np.abs(M - M.T).max() <= 1e-12 * np.abs(M).max()
    assert np.linalg.eigvalsh(0.5 * (M + M.T)).min() > 0.0
    # M approximates A^-1: the preconditioned operator's spectrum is clustered near 1
    A = dense_from_apply(o)
    ev = np.linalg.eigvals(M @ A).real
    assert 0.5 < ev.min() and ev.max() < 1.5
    o.set_option("symmetric", 0)
    M0 = _vcycle_matrix(o, shape)
    assert np.abs(M0 - M0.T).max() > 1e-6 * np.abs(M0).max()
    o.close()


@pytest.mark.parametrize("dims,bc", [((8, 8, 8), [D, N, N, D, N, N]), ((16, 8, 8), [D, D, N, N, N, N]), ((16, 16, 1), [N, D, D, N, N, N])])
def test_n2_pcg_converges_to_dense_direct_solution(dims, bc):
    p = inputs.random_problem(*dims, seed=7, bc_type=bc)
    o = Oracle.from_problem(p)
    A = dense_from_apply(o)
    bt = o.fold_bc(p.rhs).ravel()
    x = np.linalg.solve(A, bt).reshape(p.rhs.shape)
    phi, st, it, rr, hist = o.solve_pcg(p.rhs, rtol=1e-13, max_iter=40)
    assert st == 0 and it <= 12 and len(hist) == it + 1
    assert np.abs(phi - x).max() <= 1e-11 * np.abs(x).max()
    # the history is the true residual's norm (recurrence and definition agree to rounding while above the floor)
    r = bt - A @ phi.ravel()
    assert abs(np.abs(r).max() / np.abs(bt).max() - rr) <= 1e-3 * rr + 1e-15
    o.close()


def test_n2_pcg_converges_where_plain_vcycles_do_not():
    """The regime of R17: strong coefficient contrast (sigma = 2, ~8 decades) at three cells per correlation length,
    diffusion dominated.  The plain V(3,3) iteration does not contract there (it stalls at a relative residual of
    order one); conjugate gradients preconditioned by the symmetric V-cycle converge to 1e-10 in about twenty
    iterations, as the theory of SPD preconditioning promises for any SPD preconditioner."""
    p = inputs.random_problem(32, 32, 32, seed=3, bc_type=[D, N, N, N, N, N], ell=0.06, sigma=2.0, a_scale=1.0, inhomogeneous=False)
    o = Oracle.from_problem(p)
    _, st_v, cyc_v, rr_v, hist_v = o.solve(p.rhs, rtol=1e-10, max_vcycles=150)
    phi, st_c, it_c, rr_c, hist_c = o.solve_pcg(p.rhs, rtol=1e-10, max_iter=150)
    assert st_v != 0 and rr_v > 1e-3
    assert st_c == 0 and it_c <= 30 and rr_c <= 1e-10
    o.close()


def _masked_system_by_faces(p, mask, kind, cval):
    """(A, btilde) of the masked problem written face by face from the finite-volume statement:
    a face between two valid cells couples them; a face between a valid and a covered cell is an interior boundary --
    Dirichlet with the covered cell's value (two-point flux over half a cell) or zero flux; domain faces of valid cells
    as usual; a covered cell is an identity row with zero right-hand side.  Per-cell form (divided by the volume)."""
    nx, ny, nz = p.nx, p.ny, p.nz
    h = (p.dx, p.dy, p.dz)
    n = nx * ny * nz
    idx = lambda i, j, k: i + nx * (j + ny * k)
    A = np.zeros((n, n))
    bt = p.rhs.ravel().copy()
    a = p.a if p.a is not None else np.zeros((nz, ny, nx))
    m = mask.astype(bool)
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                c = idx(i, j, k)
                if m[k, j, i]:
                    A[c, c] += p.alpha * a[k, j, i]
                else:
                    A[c, c] = 1.0
                    bt[c] = 0.0
    barr = (p.bx, p.by, p.bz)
    for d in range(3):
        nd = (nx, ny, nz)[d]
        for k in range(nz):
            for j in range(ny):
                for i in range(nx):
                    pos = (i, j, k)[d]
                    # the LOW face of cell (i,j,k) in direction d, and -- for the last cell -- its high face as well
                    for side in ([0] if pos < nd - 1 else [0, 1]):
                        fi = [i, j, k]; fi[d] += side
                        b = barr[d][fi[2], fi[1], fi[0]]
                        t = p.beta * b / h[d] ** 2
                        c = idx(i, j, k)
                        if side == 0 and pos > 0:                          # interior face between (pos-1) and pos
                            lo = [i, j, k]; lo[d] -= 1
                            l = idx(*lo)
                            vl, vr = m[lo[2], lo[1], lo[0]], m[k, j, i]
                            if vl and vr:
                                A[l, l] += t; A[c, c] += t; A[l, c] -= t; A[c, l] -= t
                            elif vl != vr and kind == D:
                                v, cov = (l, (k, j, i)) if vl else (c, (lo[2], lo[1], lo[0]))
                                A[v, v] += 2 * t
                                bt[v] += 2 * t * (cval[cov] if cval is not None else 0.0)
                        else:                                              # domain face
                            if not m[k, j, i]:
                                continue
                            f = 2 * d + (0 if side == 0 and pos == 0 else 1)
                            val = p.bc_value[f]
                            pl = [(j, k), (i, k), (i, j)][d]
                            g = 0.0 if val is None else val[pl[1], pl[0]]
                            if p.bc_type[f] == D:
                                A[c, c] += 2 * t; bt[c] += 2 * t * g
                            else:
                                bt[c] += t * h[d] * g
    return A, bt


@pytest.mark.parametrize("kind", [D, N], ids=["dirichlet_interfaces", "zero_flux_interfaces"])
def test_n4_masked_operator_and_solution_match_facewise_assembly(kind):
    """SURVEY 8(f) N4 / PAPER.md:136: the masked problem the oracle solves is the one assembled face by face above
    (operator on every level-0 row, folded right-hand side), and multigrid / PCG reach its dense solution."""
    p = inputs.random_problem(8, 8, 8, seed=12, bc_type=[D, N, N, D, N, N])
    rng = np.random.default_rng(1)
    mask = np.ones(p.rhs.shape, dtype=np.uint8)
    mask[2:5, 3:6, 1:4] = 0                     # a covered block (k, j, i ranges) inside the box
    mask[0, 0, :3] = 0                          # and covered cells touching the domain boundary
    cval = np.where(mask == 0, 0.7 + 0.1 * rng.standard_normal(p.rhs.shape), 0.0)
    o = Oracle.from_problem(p)
    o.set_mask(mask, kind, cval if kind == D else None)
    o.set_coeffs(p.a, p.bx, p.by, p.bz, p.alpha, p.beta)
    A, bt = _masked_system_by_faces(p, mask, kind, cval if kind == D else None)
    assert np.abs(dense_from_apply(o) - A).max() <= 1e-12 * np.abs(A).max()
    assert np.abs(o.fold_bc(p.rhs).ravel() - bt).max() <= 1e-12 * np.abs(bt).max()
    x = np.linalg.solve(A, bt).reshape(p.rhs.shape)
    assert np.abs(x[mask == 0]).max() == 0.0
    phi, st, cyc, rr, _ = o.solve(p.rhs, rtol=1e-13, max_vcycles=60)
    assert st == 0 and np.abs(phi - x).max() <= 1e-10 * np.abs(x).max()
    phi, st, it, rr, _ = o.solve_pcg(p.rhs, rtol=1e-13, max_iter=60)
    assert st == 0 and np.abs(phi - x).max() <= 1e-10 * np.abs(x).max()
    o.close()


@pytest.mark.parametrize("kind", [D, N], ids=["dirichlet_interfaces", "zero_flux_interfaces"])
def test_n4_coarse_levels_of_a_masked_hierarchy(kind):
    """Reading N4, coarse levels: the effective coefficients a_eff, b_eff are averaged as R10 and the extra diagonal like a.
    Level-1 adiag = mean of the 8 children of the level-0 adiag written here from the mask and b; and the level-1
    operator is the ordinary face-wise operator of the averaged coefficients plus that diagonal -- a wrong coarse average
    (a dropped child, a wrong factor) fails one of the two."""
    import dataclasses
    p = inputs.random_problem(16, 8, 8, seed=15, bc_type=[D, N, N, D, N, N])
    mask = np.ones(p.rhs.shape, dtype=np.uint8)
    mask[2:5, 3:6, 5:11] = 0                    # a covered block that cuts through coarse cells (odd offsets)
    mask[0, 0, :3] = 0
    o = Oracle.from_problem(p)
    o.set_mask(mask, kind, None)
    o.set_coeffs(p.a, p.bx, p.by, p.bz, p.alpha, p.beta)
    nz, ny, nx = p.rhs.shape
    m = mask.astype(bool)
    # level-0 extra diagonal from its definition: 2 beta b / h^2 per face to a covered neighbour (Dirichlet kind), 1 if covered
    ad0 = np.zeros(p.rhs.shape)
    h = (p.dx, p.dy, p.dz)
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                if not m[k, j, i]:
                    ad0[k, j, i] = 1.0
                    continue
                if kind != D:
                    continue
                for d, (di, dj, dk) in enumerate(((1, 0, 0), (0, 1, 0), (0, 0, 1))):
                    for side in (0, 1):
                        ii, jj, kk = i + (2 * side - 1) * di, j + (2 * side - 1) * dj, k + (2 * side - 1) * dk
                        if 0 <= ii < nx and 0 <= jj < ny and 0 <= kk < nz and not m[kk, jj, ii]:
                            b = (p.bx, p.by, p.bz)[d][k + side * dk, j + side * dj, i + side * di]
                            ad0[k, j, i] += 2.0 * p.beta * b / h[d] ** 2
    assert np.abs(o.level_adiag(0) - ad0).max() <= 1e-13 * np.abs(ad0).max()
    ad1 = ad0.reshape(nz // 2, 2, ny // 2, 2, nx // 2, 2).mean(axis=(1, 3, 5))
    assert np.abs(o.level_adiag(1) - ad1).max() <= 1e-13 * np.abs(ad1).max()
    # level-1 operator = face-wise operator of the level's averaged coefficients (h doubled) + diag(adiag)
    a1, bx1, by1, bz1 = o.level_coeffs(1)
    p1 = dataclasses.replace(p, nx=nx // 2, ny=ny // 2, nz=nz // 2, dx=2 * p.dx, dy=2 * p.dy, dz=2 * p.dz, a=a1, bx=bx1, by=by1, bz=bz1)
    A1 = brute_force_matrix(p1) + np.diag(o.level_adiag(1).ravel())
    assert np.abs(dense_from_apply(o, 1) - A1).max() <= 1e-12 * np.abs(A1).max()
    # the averaged effective coefficients themselves: a_eff = a in valid cells, 0 in covered ones
    a_eff = np.where(m, p.a, 0.0)
    assert np.abs(a1 - a_eff.reshape(nz // 2, 2, ny // 2, 2, nx // 2, 2).mean(axis=(1, 3, 5))).max() <= 1e-13 * np.abs(a_eff).max()
    o.close()


def test_n4_electrode_block_obeys_the_maximum_principle():
    """A covered block at potential 1 inside a grounded box (Laplace, no source): 0 <= phi <= 1 in every valid cell, phi
    decays away from the block, and the solution has the block's mirror symmetry."""
    n = 16
    h = 1.0 / n
    ones = lambda shape: np.ones(shape)
    p = inputs.Problem(name="electrode", nx=n, ny=n, nz=n, dx=h, dy=h, dz=h, alpha=0.0, beta=1.0, a=None,
                       bx=ones((n, n, n + 1)), by=ones((n, n + 1, n)), bz=ones((n + 1, n, n)),
                       bc_type=[D] * 6, bc_value=[None] * 6, rhs=np.zeros((n, n, n)))
    mask = np.ones((n, n, n), dtype=np.uint8)
    mask[6:10, 6:10, 6:10] = 0
    o = Oracle.from_problem(p)
    o.set_mask(mask, D, np.where(mask == 0, 1.0, 0.0))
    o.set_coeffs(None, p.bx, p.by, p.bz, 0.0, 1.0)
    phi, st, cyc, rr, _ = o.solve(p.rhs, rtol=1e-12, max_vcycles=60)
    assert st == 0
    v = phi[mask == 1]
    assert v.min() > 0.0 and v.max() < 1.0
    assert np.abs(phi - phi[::-1, :, :]).max() < 1e-10 and np.abs(phi - phi.transpose(2, 1, 0)).max() < 1e-10
    assert phi[8, 8, 10] > phi[8, 8, 12] > phi[8, 8, 14] > 0.0
    o.close()
