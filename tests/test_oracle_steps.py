"""Pins for the single steps of the oracle's V-cycle (C2-C5 of SURVEY.md sec. 8(c)): smoother colour order,
transfer operators, coefficient averaging, cycle sequencing, solve bookkeeping.  CPU only."""
import numpy as np
import pytest

from oracle import Oracle
from paper_2507_08200_b200 import inputs
from paper_2507_08200_b200.inputs import DIRICHLET as D, NEUMANN as N
from test_oracle_pins import dense_from_apply, brute_force_matrix, MIXED


def test_c2_red_black_sweep_equals_dense_block_gauss_seidel():
    """Red first ((i+j+k) even), then black, each colour solved exactly given the other (C2, R7):
    phi_R = D_R^-1 (b_R - A_RB phi_B);  phi_B = D_B^-1 (b_B - A_BR phi_R_new), with A from the independent
    face-wise assembly."""
    p = inputs.random_problem(6, 4, 4, seed=8, bc_type=MIXED)
    o = Oracle.from_problem(p)
    A = brute_force_matrix(p)
    k, j, i = np.meshgrid(np.arange(p.nz), np.arange(p.ny), np.arange(p.nx), indexing="ij")
    red = (((i + j + k) % 2) == 0).ravel()
    rng = np.random.default_rng(1)
    phi = rng.standard_normal(p.rhs.shape)
    b = rng.standard_normal(p.rhs.shape)
    x = phi.ravel().copy()
    dg = np.diag(A)
    for mask in (red, ~red):
        off = A[mask][:, ~mask] @ x[~mask]
        x[mask] = (b.ravel()[mask] - off) / dg[mask]
    got = o.smooth(phi, b, 1)
    assert np.abs(got.ravel() - x).max() <= 1e-13 * np.abs(x).max()
    # two sweeps = the same map applied twice
    assert np.allclose(o.smooth(phi, b, 2), o.smooth(got, b, 1), rtol=0, atol=0)


def test_c3_restriction_is_child_mean_and_prolongation_its_scaled_adjoint():
    p = inputs.random_problem(8, 12, 4, seed=2)
    o = Oracle.from_problem(p)
    rng = np.random.default_rng(3)
    r = rng.standard_normal((4, 12, 8))
    rc = o.restrict(r)
    expect = r.reshape(2, 2, 6, 2, 4, 2).mean(axis=(1, 3, 5))
    assert np.abs(rc - expect).max() <= 1e-15
    e = rng.standard_normal(rc.shape)
    pe = o.prolong_add(np.zeros_like(r), e)
    assert np.array_equal(pe, np.repeat(np.repeat(np.repeat(e, 2, 0), 2, 1), 2, 2))
    assert abs(8.0 * (rc * e).sum() - (r * pe).sum()) <= 1e-12          # P = 8 R^T
    # 2-D: 4 children
    o2 = Oracle.from_problem(inputs.random_problem(8, 4, 1, seed=2))
    r2 = rng.standard_normal((1, 4, 8))
    assert np.abs(o2.restrict(r2) - r2.reshape(1, 2, 2, 4, 2).mean(axis=(2, 4))).max() <= 1e-15
    pe2 = o2.prolong_add(r2, np.ones((1, 2, 4)))
    assert np.array_equal(pe2, r2 + 1.0)


def test_c3_coefficient_averaging_face_means():
    p = inputs.random_problem(8, 4, 4, seed=6)
    o = Oracle.from_problem(p)
    a1, bx1, by1, bz1 = o.level_coeffs(1)
    assert np.abs(a1 - p.a.reshape(2, 2, 2, 2, 4, 2).mean(axis=(1, 3, 5))).max() <= 1e-15 * np.abs(p.a).max()
    # x faces: only fine faces lying ON the coarse face (even fine index), mean over the 2x2 patch in y,z
    assert np.abs(bx1 - p.bx[:, :, ::2].reshape(2, 2, 2, 2, 5).mean(axis=(1, 3))).max() <= 1e-15 * p.bx.max()
    assert np.abs(by1 - p.by[:, ::2, :].reshape(2, 2, 3, 4, 2).mean(axis=(1, 4))).max() <= 1e-15 * p.by.max()
    assert np.abs(bz1 - p.bz[::2, :, :].reshape(3, 2, 2, 4, 2).mean(axis=(2, 4))).max() <= 1e-15 * p.bz.max()
    # level-0 coefficients are the caller's, untouched
    a0, bx0, by0, bz0 = o.level_coeffs(0)
    assert np.array_equal(a0, p.a) and np.array_equal(bx0, p.bx) and np.array_equal(bz0, p.bz)
    # total flux through a coarse face is preserved for a unit gradient: area-weighted sums agree
    assert abs(bx1.sum() * 4.0 - p.bx[:, :, ::2].sum()) <= 1e-12 * p.bx.sum()


def test_r11_level_count_and_dims():
    for dims, nlev, coarsest in [((256, 128, 128), 7, (4, 2, 2)), ((64, 64, 1), 6, (2, 2, 1)),
                                 ((128, 128, 128), 7, (2, 2, 2)), ((24, 16, 8), 3, (6, 4, 2)), ((12, 6, 10), 2, (6, 3, 5))]:
        o = Oracle(*dims, 1.0, 1.0, 1.0)
        assert o.num_levels == nlev and o.level_dims(nlev - 1) == coarsest
        o.close()


def _py_vcycle(o, lev, phi, rhs, nu1=3, nu2=3, nb=32):
    if lev == o.num_levels - 1:
        return o.smooth(np.zeros_like(phi), rhs, nb, lev)
    phi = o.smooth(phi, rhs, nu1, lev)
    rc = o.restrict(o.residual(phi, rhs, lev), lev)
    e = _py_vcycle(o, lev + 1, np.zeros_like(rc), rc, nu1, nu2, nb)
    phi = o.prolong_add(phi, e, lev)
    return o.smooth(phi, rhs, nu2, lev)


def test_c4_vcycle_is_the_stated_sequence_of_steps():
    p = inputs.random_problem(16, 8, 8, seed=12, bc_type=[D, D, N, N, N, N])
    o = Oracle.from_problem(p)
    bt = o.fold_bc(p.rhs)
    phi0 = np.random.default_rng(0).standard_normal(p.rhs.shape)
    assert np.array_equal(o.vcycle(phi0, bt), _py_vcycle(o, 0, phi0, bt))
    o.set_option("nu1", 2); o.set_option("nu2", 1); o.set_option("bottom_sweeps", 8)
    assert np.array_equal(o.vcycle(phi0, bt), _py_vcycle(o, 0, phi0, bt, 2, 1, 8))


def test_c5_solve_history_norm_and_exit_rules():
    p = inputs.random_problem(16, 8, 8, seed=13, bc_type=[D, D, N, N, N, N])
    o = Oracle.from_problem(p)
    bt = o.fold_bc(p.rhs)
    phi, status, cycles, relres, hist = o.solve(p.rhs, rtol=1e-9)
    # history entries are true relative residuals in the infinity norm w.r.t. ||btilde||_inf (R12)
    assert status == 0 and len(hist) == cycles + 1 and hist[-1] == relres <= 1e-9 < hist[-2]
    assert abs(hist[0] - 1.0) <= 1e-15                                    # zero guess: r0 = btilde
    assert abs(relres - np.abs(bt - o.apply(phi)).max() / np.abs(bt).max()) <= 1e-15
    x = np.zeros_like(p.rhs)
    for c in range(cycles):
        x = o.vcycle(x, bt)
    assert np.array_equal(x, phi)
    # warm start: a converged phi in -> 0 cycles
    phi2, status2, cycles2, *_ = o.solve(p.rhs, phi0=phi, rtol=1e-9)
    assert status2 == 0 and cycles2 == 0 and np.array_equal(phi2, phi)
    # rtol <= 0: exactly max_vcycles cycles, status MAXCYCLES
    phi3, status3, cycles3, _, hist3 = o.solve(p.rhs, rtol=0.0, max_vcycles=4)
    assert status3 == 1 and cycles3 == 4 and len(hist3) == 5
    # unreachable tolerance: stalls on the rounding floor
    phi4, status4, cycles4, relres4, _ = o.solve(p.rhs, rtol=1e-30, max_vcycles=60)
    assert status4 == 2 and cycles4 < 60 and relres4 < 1e-14
    # zero right-hand side and homogeneous data: phi = 0, 0 cycles
    o.set_bc(p.bc_type, None)
    phi5, status5, cycles5, *_ = o.solve(np.zeros_like(p.rhs), phi0=np.ones_like(p.rhs))
    assert status5 == 0 and cycles5 == 0 and not phi5.any()


def test_r9_trilinear_prolongation_is_exact_for_linear_fields_and_honours_the_ghost_rules():
    """R9 option prolong = 1 (cell-centred trilinear, weights 3/4 and 1/4 per direction): pinned by what interpolation
    must do, not by its formula -- (i) a coarse field that is linear in the coarse cell centres comes out linear in the
    fine cell centres wherever no ghost is involved; (ii) with the Neumann ghost (+e) a constant stays a constant
    everywhere; (iii) with the Dirichlet ghost (-e) a field that is linear in the distance from the Dirichlet face and
    vanishes ON the face (half a coarse cell from the first centre) is reproduced exactly in the cells next to it."""
    nx, ny, nz = 16, 8, 8
    p = inputs.random_problem(nx, ny, nz, seed=1, bc_type=[D, N, N, N, N, N], inhomogeneous=False, spacing=(1.0, 1.0, 1.0))
    o = Oracle.from_problem(p)
    o.set_option("prolong", 1)
    H = 2.0                                                     # coarse spacing (fine spacing 1)
    K, J, I = np.meshgrid(np.arange(nz // 2), np.arange(ny // 2), np.arange(nx // 2), indexing="ij")
    xc, yc, zc = (I + 0.5) * H, (J + 0.5) * H, (K + 0.5) * H   # coarse centres
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    xf, yf, zf = i + 0.5, j + 0.5, k + 0.5                      # fine centres
    # (i) linear field, interior cells (fine index 1 .. n-2 in every direction: no ghost in their stencil)
    lin_c = 0.3 + 1.7 * xc - 0.9 * yc + 0.4 * zc
    out = o.prolong_add(np.zeros((nz, ny, nx)), lin_c)
    lin_f = 0.3 + 1.7 * xf - 0.9 * yf + 0.4 * zf
    inner = (slice(1, -1),) * 3
    assert np.abs(out[inner] - lin_f[inner]).max() < 1e-13
    # (ii) constants: exact wherever only Neumann ghosts are involved (everywhere but the cells at the Dirichlet face)
    out = o.prolong_add(np.zeros((nz, ny, nx)), np.full((nz // 2, ny // 2, nx // 2), 2.5))
    assert np.abs(out[:, :, 1:] - 2.5).max() < 1e-14
    # ... and next to the Dirichlet face the ghost -e pulls the value towards the face value 0: 3/4 e - 1/4 e
    assert np.abs(out[:, :, 0] - 1.25).max() < 1e-14
    # (iii) e = c * x (zero on the Dirichlet face x = 0): exact for ALL cells in x, including i = 0
    out = o.prolong_add(np.zeros((nz, ny, nx)), 3.0 * xc)
    assert np.abs(out[:, :, :-1] - 3.0 * xf[:, :, :-1]).max() < 1e-13   # (the far x face is Neumann: last cell not linear)
    # the correction is ADDED
    base = np.random.default_rng(0).standard_normal((nz, ny, nx))
    assert np.allclose(o.prolong_add(base.copy(), lin_c), base + o.prolong_add(np.zeros_like(base), lin_c), atol=1e-14)
    o.close()


def test_r9_trilinear_v22_converges_to_the_same_discrete_solution():
    """The option changes the iteration, not its fixed point: V(2,2) with trilinear prolongation reaches the solution
    V(3,3) with piecewise-constant prolongation reaches (both to 1e-12), in no more cycles on a smooth problem."""
    p = inputs.config3(16)
    o = Oracle.from_problem(p)
    phi_c, st_c, cyc_c, *_ = o.solve(p.rhs, rtol=1e-12)
    for k, v in (("prolong", 1), ("nu1", 2), ("nu2", 2)):
        o.set_option(k, v)
    phi_l, st_l, cyc_l, rr_l, hist = o.solve(p.rhs, rtol=1e-12)
    assert st_c == 0 and st_l == 0 and cyc_l <= cyc_c + 2
    assert np.abs(phi_l - phi_c).max() <= 1e-10 * np.abs(phi_c).max()
    o.close()
