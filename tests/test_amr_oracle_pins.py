"""Pins of oracle/amr_oracle.c (two-level composite solve, SURVEY.md 8(f) N4 second half) against things other than itself.

The paper names "the composite multilevel multigrid solver from within AMReX" and gives no formula, so
the pins are what the mathematics fixes for readings A1-A5 (header of amr_oracle.c):
  * a linear field has zero divergence of b grad phi for b = 1: every cell, the interface cells included, must give 0
    (fails for a wrong 1/8, a wrong sign of the tangential slope, a wrong 1.5 hf, a wrong neighbour index);
  * conservation: with zero-flux box faces and a = 0 the volume-weighted sum of A phi vanishes for ANY phi and b
    (fails if the coarse side does not take exactly the fine fluxes);
  * a dense matrix assembled here FACE BY FACE in flux form (the oracle works cell by cell) gives the same A phi;
  * a manufactured solution with variable b converges at second order in the maximum norm over both levels;
  * the cycle converges to the solution of that dense system, contracting by less than 0.2 per cycle.
"""
import itertools

import numpy as np
import pytest

from oracle import AmrOracle

D, N = 0, 1


def _shapes(n, m):
    """cell and face array shapes ([k, j, i], x fastest) of a box of n = (nx, ny, nz) cells"""
    cell = (n[2], n[1], n[0])
    faces = [(n[2], n[1], n[0] + 1), (n[2], n[1] + 1, n[0]), (n[2] + 1, n[1], n[0])]
    return cell, faces


def _fine_dims(n, lo, hi):
    nd = 3 if n[2] > 1 else 2
    return tuple(2 * (hi[d] - lo[d]) if d < nd else 1 for d in range(3)), nd


def _random_coeffs(rng, n, with_a=True, sigma=1.0):
    cell, faces = _shapes(n, None)
    a = np.exp(rng.standard_normal(cell)) if with_a else None
    return (a,) + tuple(np.exp(sigma * rng.standard_normal(s)) for s in faces)


def _at(arr, idx):
    """arr[k, j, i] for idx = (i, j, k)"""
    return arr[idx[2], idx[1], idx[0]]


def _patches(lo, hi):
    """lo, hi: one triple or lists of triples -> lists of triples"""
    single = not isinstance(lo[0], (list, tuple))
    return ([lo], [hi], True) if single else (list(lo), list(hi), False)


def assemble(n, h, lo, hi, coarse, fine, alpha, beta, bctype):
    """The composite matrix in FLUX form: a loop over faces; a face with transmissibility T (flux = T * difference) adds
    T / volume to the rows of the two cells it separates.  Unknowns: uncovered coarse cells (box order), then the fine
    cells patch by patch (patch order).  lo, hi, fine: one patch or lists.  Returns (A, cnum, fnums) with cnum[k, j, i] = -1
    under a patch and fnums a list of index arrays (a bare array for a single patch)."""
    los, his, single = _patches(lo, hi)
    fines = [fine] if single else list(fine)
    nd = 3 if n[2] > 1 else 2
    ms = [_fine_dims(n, l, u)[0] for l, u in zip(los, his)]
    cnum = -np.ones((n[2], n[1], n[0]), dtype=int)
    cnt = 0
    for k, j, i in itertools.product(range(n[2]), range(n[1]), range(n[0])):
        inside = any(all(l[d] <= (i, j, k)[d] < u[d] for d in range(nd)) for l, u in zip(los, his))
        if not inside:
            cnum[k, j, i] = cnt
            cnt += 1
    fnums = []
    for m in ms:
        fnums.append(cnt + np.arange(m[0] * m[1] * m[2]).reshape(m[2], m[1], m[0]))
        cnt += m[0] * m[1] * m[2]
    size = cnt
    A = np.zeros((size, size))
    volc = float(np.prod(h[:nd]))
    volf = volc / 2 ** nd
    ac, bc = coarse[0], coarse[1:]
    one = lambda arr, idx: 1.0 if arr is None else _at(arr, idx)
    # absorption
    for k, j, i in itertools.product(range(n[2]), range(n[1]), range(n[0])):
        r = cnum[k, j, i]
        if r >= 0 and ac is not None:
            A[r, r] += alpha * ac[k, j, i]
    # coarse faces
    for d in range(nd):
        ext = [n[0], n[1], n[2]]
        ext[d] += 1
        area = volc / h[d]
        for k, j, i in itertools.product(range(ext[2]), range(ext[1]), range(ext[0])):
            face = (i, j, k)
            left = list(face); left[d] -= 1
            right = list(face)
            b = one(bc[d], face)
            if left[d] < 0 or right[d] >= n[d]:                      # a face of the box
                inside = right if left[d] < 0 else left
                if bctype[2 * d + (0 if left[d] < 0 else 1)] == D:
                    r = _at(cnum, inside)
                    A[r, r] += beta * b / (h[d] / 2) * area / volc
                continue
            l, r = _at(cnum, left), _at(cnum, right)
            if l >= 0 and r >= 0:
                T = beta * b / h[d] * area
                A[l, l] += T / volc; A[l, r] -= T / volc
                A[r, r] += T / volc; A[r, l] -= T / volc
            # both covered: no unknowns; one covered: a coarse-fine face, taken from the fine side below
    # fine cells and faces, patch by patch
    for lo_, m, fnum, fcoef in zip(los, ms, fnums, fines):
        af, bf = fcoef[0], fcoef[1:]
        for K, J, I in itertools.product(range(m[2]), range(m[1]), range(m[0])):
            if af is not None:
                A[fnum[K, J, I], fnum[K, J, I]] += alpha * af[K, J, I]
        for d in range(nd):
            ext = [m[0], m[1], m[2]]
            ext[d] += 1
            hf = h[d] / 2
            area = volf / hf
            tang = [t for t in range(nd) if t != d]
            for K, J, I in itertools.product(range(ext[2]), range(ext[1]), range(ext[0])):
                face = (I, J, K)
                left = list(face); left[d] -= 1
                right = list(face)
                b = one(bf[d], face)
                if left[d] >= 0 and right[d] < m[d]:
                    T = beta * b / hf * area
                    l, r = _at(fnum, left), _at(fnum, right)
                    A[l, l] += T / volf; A[l, r] -= T / volf
                    A[r, r] += T / volf; A[r, l] -= T / volf
                    continue
                low_side = left[d] < 0
                fcell = right if low_side else left
                F = _at(fnum, fcell)
                ccell = [lo_[t] + fcell[t] // 2 if t < nd else 0 for t in range(3)]
                ccell[d] += -1 if low_side else 1
                g = {_at(cnum, ccell): 1.0}                                # g = sum of coefficient * coarse unknown
                for t in tang:
                    s = 1.0 if fcell[t] % 2 else -1.0
                    up = list(ccell); up[t] += 1
                    dn = list(ccell); dn[t] -= 1
                    g[_at(cnum, up)] = g.get(_at(cnum, up), 0.0) + s / 8
                    g[_at(cnum, dn)] = g.get(_at(cnum, dn), 0.0) - s / 8
                assert all(c >= 0 for c in g)
                T = beta * b / (1.5 * hf) * area                           # flux out of the fine cell = T (phi_F - g)
                Cn = _at(cnum, ccell)
                A[F, F] += T / volf
                A[Cn, F] -= T / volc
                for c, coef in g.items():
                    A[F, c] -= T * coef / volf
                    A[Cn, c] += T * coef / volc
    return A, cnum, (fnums[0] if single else fnums)


def pack(cnum, fnum, vc, vf):
    fnums = fnum if isinstance(fnum, list) else [fnum]
    vfs = vf if isinstance(vf, list) else [vf]
    out = np.zeros(max(f.max() for f in fnums) + 1)
    out[cnum[cnum >= 0]] = vc[cnum >= 0]
    for f, v in zip(fnums, vfs):
        out[f.ravel()] = v.ravel()
    return out


GEOMS = [((12, 10, 8), (0.1, 0.07, 0.13), (2, 3, 2), (7, 8, 6)),
         ((12, 10, 1), (0.1, 0.07, 1.0), (3, 2, 0), (9, 6, 1))]


def _centres(n, h, lo=None, hi=None):
    """cell-centre coordinates ([k, j, i] arrays) of the coarse box, or of the patch's fine cells when lo is given"""
    if lo is None:
        ax = [(np.arange(n[d]) + 0.5) * h[d] for d in range(3)]
    else:
        m, nd = _fine_dims(n, lo, hi)
        ax = [lo[d] * h[d] + (np.arange(m[d]) + 0.5) * h[d] / 2 if d < nd else np.array([0.5 * h[d]]) for d in range(3)]
    z, y, x = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    return x, y, z


@pytest.mark.parametrize("n,h,lo,hi", GEOMS)
def test_a_linear_field_is_in_the_null_space_at_every_interface_cell(n, h, lo, hi):
    o = AmrOracle(*n, *h, lo, hi)
    o.set_coeffs((None,) * 4, (None,) * 4, 0.0, 1.0)
    o.set_bc([N] * 6)
    three_d = n[2] > 1
    lin = lambda x, y, z: 0.3 + 1.7 * x - 2.2 * y + (0.9 * z if three_d else 0.0)
    phic, phif = lin(*_centres(n, h)), lin(*_centres(n, h, lo, hi))
    oc, of = o.apply(phic, phif)
    scale = 2.2 / min(h[:3 if three_d else 2]) ** 2
    assert np.abs(of).max() <= 1e-13 * scale
    inner = np.zeros(oc.shape, bool)                     # the box's own faces are zero-flux here: leave their cells out
    inner[(slice(1, -1) if three_d else slice(None)), 1:-1, 1:-1] = True
    assert np.abs(oc[inner]).max() <= 1e-13 * scale
    # the interface cells are among the checked ones (the patch keeps two cells from the boundary in this geometry)
    assert inner[(lo[2] if three_d else 0), lo[1], lo[0] - 1] and inner[(lo[2] if three_d else 0), hi[1], lo[0]]
    # and the pin bites: a harmonic quadratic (exact in the interior) is NOT annihilated at the interface cells
    quad = lambda x, y, z: x * x - y * y
    oc2, of2 = o.apply(quad(*_centres(n, h)), quad(*_centres(n, h, lo, hi)))
    assert np.abs(of2).max() > 1e-3


@pytest.mark.parametrize("n,h,lo,hi", GEOMS)
def test_conservation_the_coarse_side_takes_exactly_the_fine_fluxes(n, h, lo, hi):
    rng = np.random.default_rng(11)
    m, nd = _fine_dims(n, lo, hi)
    o = AmrOracle(*n, *h, lo, hi)
    coarse, fine = _random_coeffs(rng, n, with_a=False), _random_coeffs(rng, m, with_a=False)
    o.set_coeffs(coarse, fine, 0.0, 1.3)
    o.set_bc([N] * 6)
    phic, phif = rng.standard_normal(o.coarse_shape), rng.standard_normal(o.fine_shape)
    oc, of = o.apply(phic, phif)
    volc = float(np.prod(h[:nd]))
    total = oc.sum() * volc + of.sum() * volc / 2 ** nd
    assert abs(total) <= 1e-12 * (np.abs(oc).sum() * volc + np.abs(of).sum() * volc / 2 ** nd)


@pytest.mark.parametrize("n,h,lo,hi", GEOMS)
def test_apply_equals_a_dense_matrix_assembled_face_by_face(n, h, lo, hi):
    rng = np.random.default_rng(12)
    m, nd = _fine_dims(n, lo, hi)
    bctype = [D, N, N, D, D, N]
    coarse, fine = _random_coeffs(rng, n), _random_coeffs(rng, m)
    o = AmrOracle(*n, *h, lo, hi)
    o.set_coeffs(coarse, fine, 0.7, 1.3)
    o.set_bc(bctype)
    A, cnum, fnum = assemble(n, h, lo, hi, coarse, fine, 0.7, 1.3, bctype)
    phic, phif = rng.standard_normal(o.coarse_shape), rng.standard_normal(o.fine_shape)
    phic[cnum < 0] = 1e30                                   # values under the patch must not be read
    oc, of = o.apply(phic, phif)
    assert np.all(oc[cnum < 0] == 0.0)
    want = A @ pack(cnum, fnum, np.where(cnum >= 0, phic, 0.0), phif)
    got = pack(cnum, fnum, oc, of)
    assert np.abs(got - want).max() <= 1e-13 * np.abs(want).max()


def test_patches_that_touch_the_boundary_or_are_too_thin_are_rejected():
    from oracle import OracleError
    for lo, hi in (((0, 2, 2), (4, 6, 6)), ((2, 2, 2), (8, 6, 6)), ((2, 2, 2), (3, 6, 6))):
        with pytest.raises(OracleError) as e:
            AmrOracle(8, 8, 8, 0.1, 0.1, 0.1, lo, hi)
        assert e.value.code == -2


# ---- manufactured solution (variable b, absorption, Dirichlet planes on x, Neumann planes elsewhere) -----------------
def _mms(three_d):
    kz = 0.9 if three_d else 0.0
    S = lambda x: np.sin(1.3 * x + 0.4)
    dS = lambda x: 1.3 * np.cos(1.3 * x + 0.4)
    C1 = lambda y: np.cos(1.1 * y - 0.2)
    dC1 = lambda y: -1.1 * np.sin(1.1 * y - 0.2)
    C2 = lambda z: np.cos(kz * z + 0.1)
    dC2 = lambda z: -kz * np.sin(kz * z + 0.1)
    phi = lambda x, y, z: S(x) * C1(y) * C2(z) + 0.5 * x
    grad = lambda x, y, z: (dS(x) * C1(y) * C2(z) + 0.5, S(x) * dC1(y) * C2(z), S(x) * C1(y) * dC2(z))
    lap = lambda x, y, z: -(1.3 ** 2 + 1.1 ** 2 + kz ** 2) * S(x) * C1(y) * C2(z)
    cz = -1.0 if three_d else 0.0
    arg = lambda x, y, z: x + 2.0 * y + cz * z
    b = lambda x, y, z: 1.0 + 0.5 * np.sin(arg(x, y, z))
    gb = lambda x, y, z: (0.5 * np.cos(arg(x, y, z)), 1.0 * np.cos(arg(x, y, z)), 0.5 * cz * np.cos(arg(x, y, z)))
    a = 1.5

    def f(x, y, z):
        g, q = grad(x, y, z), gb(x, y, z)
        return a * phi(x, y, z) - (q[0] * g[0] + q[1] * g[1] + q[2] * g[2] + b(x, y, z) * lap(x, y, z))
    return phi, grad, b, a, f


def _face_coords(n, h, d, origin=(0.0, 0.0, 0.0)):
    ax = [origin[t] + (np.arange(n[t]) + 0.5) * h[t] for t in range(3)]
    ax[d] = origin[d] + np.arange(n[d] + 1) * h[d]
    z, y, x = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    return x, y, z


def _mms_error(nn, three_d):
    n = (2 * nn, nn, nn if three_d else 1)
    h = (1.0 / nn,) * 3
    lo, hi = (nn // 2, nn // 4, nn // 4 if three_d else 0), (3 * nn // 2, 3 * nn // 4, 3 * nn // 4 if three_d else 1)
    m, nd = _fine_dims(n, lo, hi)
    hf = tuple(v / 2 for v in h)
    phi, grad, b, a, f = _mms(three_d)
    origin = tuple(lo[d] * h[d] if d < nd else 0.0 for d in range(3))
    cc, fc = _centres(n, h), _centres(n, h, lo, hi)
    coarse = (np.full(cc[0].shape, a),) + tuple(b(*_face_coords(n, h, d)) for d in range(3))
    fine = (np.full(fc[0].shape, a),) + tuple(b(*_face_coords(m, hf, d, origin)) for d in range(3))
    o = AmrOracle(*n, *h, lo, hi)
    o.set_coeffs(coarse, fine, 1.0, 1.0)
    # boundary planes of the box: x faces Dirichlet (phi), the others Neumann (outward normal derivative)
    vals = []
    for face in range(6):
        d, side = face // 2, face % 2
        ax = [(np.arange(n[t]) + 0.5) * h[t] for t in range(3)]
        ax[d] = np.array([side * n[d] * h[d]])
        z, y, x = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
        v = phi(x, y, z) if d == 0 else (1.0 if side else -1.0) * grad(x, y, z)[d]
        vals.append(np.ascontiguousarray(np.squeeze(v, axis=2 - d)))
    o.set_bc([D, D, N, N, N, N], vals)
    pc, pf, status, cycles, relres, hist = o.solve(f(*cc), f(*fc), rtol=1e-11, max_cycles=40)
    assert status == 0, (status, hist)
    unc = np.ones(pc.shape, bool)
    unc[(slice(lo[2], hi[2]) if three_d else slice(None)), lo[1]:hi[1], lo[0]:hi[0]] = False
    return max(np.abs(pc - phi(*cc))[unc].max(), np.abs(pf - phi(*fc)).max())


@pytest.mark.parametrize("three_d,sizes", [(True, (8, 16, 32)), (False, (16, 32, 64))])
def test_manufactured_solution_converges_at_second_order_on_the_composite_grid(three_d, sizes):
    err = [_mms_error(nn, three_d) for nn in sizes]
    orders = [np.log2(err[i] / err[i + 1]) for i in range(len(err) - 1)]
    assert err[-1] < 2e-4 and min(orders) > 1.75, (err, orders)


@pytest.mark.parametrize("n,lo,hi", [((8, 8, 8), (2, 2, 2), (6, 6, 6)), ((16, 16, 1), (4, 3, 0), (12, 11, 1))])
def test_cycle_converges_to_the_dense_solution_and_contracts_below_0p2(n, lo, hi):
    rng = np.random.default_rng(13)
    h = (1.0 / n[1],) * 3
    m, nd = _fine_dims(n, lo, hi)
    hf = tuple(v / 2 for v in h)
    origin = tuple(lo[d] * h[d] if d < nd else 0.0 for d in range(3))
    bfun = lambda x, y, z: np.exp(0.6 * np.sin(3.0 * x + 1.0) * np.cos(2.0 * y) + (0.3 * np.sin(4.0 * z) if nd == 3 else 0.0))
    coarse = (None,) + tuple(bfun(*_face_coords(n, h, d)) for d in range(3))
    fine = (None,) + tuple(bfun(*_face_coords(m, hf, d, origin)) for d in range(3))
    bctype = [D, D, N, N, N, N]
    o = AmrOracle(*n, *h, lo, hi)
    o.set_coeffs(coarse, fine, 0.0, 1.0)
    o.set_bc(bctype)
    rhsc, rhsf = rng.standard_normal(o.coarse_shape), rng.standard_normal(o.fine_shape)
    pc, pf, status, cycles, relres, hist = o.solve(rhsc, rhsf, rtol=1e-12, max_cycles=40)
    assert status == 0 and hist[0] == 1.0 and relres <= 1e-12
    A, cnum, fnum = assemble(n, h, lo, hi, coarse, fine, 0.0, 1.0, bctype)
    want = np.linalg.solve(A, pack(cnum, fnum, rhsc, rhsf))
    got = pack(cnum, fnum, pc, pf)
    assert np.abs(got - want).max() <= 1e-9 * np.abs(want).max()
    # the coarse cells under the patch hold the means of their children
    np.testing.assert_allclose(pc, o.average_down(pc, pf), rtol=0, atol=1e-15 * np.abs(pc).max())
    ratios = [hist[c] / hist[c - 1] for c in range(2, len(hist)) if hist[c] > 1e-11]
    assert max(ratios) < 0.2, ratios


# ---- several patches (A1: at least two coarse cells apart in some direction) ----------------------------------------
MULTI = [((16, 12, 8), (0.1, 0.07, 0.13), [(2, 2, 2), (9, 3, 2), (2, 8, 3)], [(6, 6, 6), (14, 10, 6), (7, 10, 6)]),
         ((20, 16, 1), (0.1, 0.07, 1.0), [(2, 2, 0), (11, 3, 0), (3, 11, 0)], [(8, 7, 1), (18, 9, 1), (16, 14, 1)])]


@pytest.mark.parametrize("n,h,los,his", MULTI)
def test_several_patches_linear_exactness_conservation_and_dense_assembly(n, h, los, his):
    rng = np.random.default_rng(21)
    nd = 3 if n[2] > 1 else 2
    ms = [_fine_dims(n, l, u)[0] for l, u in zip(los, his)]
    # linear field, b = 1
    o = AmrOracle(*n, *h, los, his)
    o.set_coeffs((None,) * 4, [(None,) * 4] * len(los), 0.0, 1.0)
    o.set_bc([N] * 6)
    lin = lambda x, y, z: 0.3 + 1.7 * x - 2.2 * y + (0.9 * z if nd == 3 else 0.0)
    oc, ofs = o.apply(lin(*_centres(n, h)), [lin(*_centres(n, h, l, u)) for l, u in zip(los, his)])
    scale = 2.2 / min(h[:nd]) ** 2
    inner = np.zeros(oc.shape, bool)
    inner[(slice(1, -1) if nd == 3 else slice(None)), 1:-1, 1:-1] = True
    assert max(np.abs(f).max() for f in ofs) <= 1e-13 * scale and np.abs(oc[inner]).max() <= 1e-13 * scale
    # conservation with random b and phi
    coarse = _random_coeffs(rng, n, with_a=False)
    fines = [_random_coeffs(rng, m, with_a=False) for m in ms]
    o.set_coeffs(coarse, fines, 0.0, 1.3)
    phic, phifs = rng.standard_normal(o.coarse_shape), [rng.standard_normal(sh) for sh in o.fine_shapes]
    oc, ofs = o.apply(phic, phifs)
    volc = float(np.prod(h[:nd]))
    total = oc.sum() * volc + sum(f.sum() for f in ofs) * volc / 2 ** nd
    assert abs(total) <= 1e-12 * (np.abs(oc).sum() * volc + sum(np.abs(f).sum() for f in ofs) * volc / 2 ** nd)
    # dense assembly, absorption and mixed box faces
    bctype = [D, N, N, D, D, N]
    coarse = _random_coeffs(rng, n)
    fines = [_random_coeffs(rng, m) for m in ms]
    o.set_coeffs(coarse, fines, 0.7, 1.3)
    o.set_bc(bctype)
    A, cnum, fnums = assemble(n, h, los, his, coarse, fines, 0.7, 1.3, bctype)
    phic[cnum < 0] = 1e30
    oc, ofs = o.apply(phic, phifs)
    want = A @ pack(cnum, fnums, np.where(cnum >= 0, phic, 0.0), phifs)
    got = pack(cnum, fnums, oc, ofs)
    assert np.all(oc[cnum < 0] == 0.0) and np.abs(got - want).max() <= 1e-13 * np.abs(want).max()


def test_several_patches_cycle_converges_to_the_dense_solution():
    rng = np.random.default_rng(22)
    n, los, his = (16, 8, 8), [(2, 2, 2), (9, 1, 2)], [(6, 6, 6), (14, 5, 7)]
    h = (1.0 / n[1],) * 3
    ms = [_fine_dims(n, l, u)[0] for l, u in zip(los, his)]
    hf = tuple(v / 2 for v in h)
    bfun = lambda x, y, z: np.exp(0.6 * np.sin(3.0 * x + 1.0) * np.cos(2.0 * y) + 0.3 * np.sin(4.0 * z))
    coarse = (None,) + tuple(bfun(*_face_coords(n, h, d)) for d in range(3))
    fines = [(None,) + tuple(bfun(*_face_coords(m, hf, d, tuple(l[t] * h[t] for t in range(3)))) for d in range(3))
             for l, m in zip(los, ms)]
    bctype = [D, D, N, N, N, N]
    o = AmrOracle(*n, *h, los, his)
    o.set_coeffs(coarse, fines, 0.0, 1.0)
    o.set_bc(bctype)
    rhsc, rhsfs = rng.standard_normal(o.coarse_shape), [rng.standard_normal(sh) for sh in o.fine_shapes]
    pc, pfs, status, cycles, relres, hist = o.solve(rhsc, rhsfs, rtol=1e-12, max_cycles=40)
    assert status == 0 and hist[0] == 1.0 and relres <= 1e-12
    A, cnum, fnums = assemble(n, h, los, his, coarse, fines, 0.0, 1.0, bctype)
    want = np.linalg.solve(A, pack(cnum, fnums, rhsc, rhsfs))
    assert np.abs(pack(cnum, fnums, pc, pfs) - want).max() <= 1e-9 * np.abs(want).max()
    ratios = [hist[c] / hist[c - 1] for c in range(2, len(hist)) if hist[c] > 1e-11]
    assert max(ratios) < 0.2, ratios


def test_patches_closer_than_two_coarse_cells_are_rejected():
    from oracle import OracleError
    with pytest.raises(OracleError) as e:
        AmrOracle(16, 8, 8, 0.1, 0.1, 0.1, [(2, 2, 2), (7, 2, 2)], [(6, 6, 6), (12, 6, 6)])     # one cell apart
    assert e.value.code == -2
    AmrOracle(16, 8, 8, 0.1, 0.1, 0.1, [(2, 2, 2), (8, 2, 2)], [(6, 6, 6), (12, 6, 6)]).close()   # two cells apart
