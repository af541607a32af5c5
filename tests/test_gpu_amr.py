"""GPU parity of the two-level composite solve (vmg_amr_*, through the C-ABI) against oracle/amr_oracle.c on the same
seeded inputs.  Bars as for the single-level solve (tests/test_gpu_parity.py): phi within 1e-10 relative L-inf on BOTH
levels after both reach relres 1e-12, equal cycle counts, residual histories equal to rounding while above the floor.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import AmrOracle
from paper_2507_08200_b200 import inputs

pytestmark = pytest.mark.gpu

PHI_TOL = 1e-10


def _binding():
    from paper_2507_08200_b200 import binding
    return binding


def dev(x):
    return None if x is None else torch.from_numpy(np.ascontiguousarray(x)).cuda()


def rel(a, b):
    return np.abs(a - b).max() / max(np.abs(b).max(), 1e-300)


def _oracle(p):
    c = p.coarse
    o = AmrOracle(c.nx, c.ny, c.nz, c.dx, c.dy, c.dz, p.lo, p.hi)
    o.set_coeffs(p.coarse_coeffs(), p.fine_coeffs(), c.alpha, c.beta)
    o.set_bc(c.bc_type, c.bc_value)
    return o


def _dev_fine(p, fine):
    """fine coefficient tuple(s) of an AmrProblem -> tensors (a list of lists for several patches)"""
    return [[dev(x) for x in f] for f in fine] if p.multi else [dev(x) for x in fine]


def _gpu(p, **options):
    b = _binding()
    c = p.coarse
    s = b.VmgAmr(c.nx, c.ny, c.nz, c.dx, c.dy, c.dz, p.lo, p.hi)
    for k, v in options.items():
        s.set_option(k, v)
    s.set_coeffs([dev(x) for x in p.coarse_coeffs()], _dev_fine(p, p.fine_coeffs()), c.alpha, c.beta)
    s.set_bc(c.bc_type, [dev(v) for v in c.bc_value])
    return s


def _compare(p, s, o, phic0=None, phif0=None, rtol=1e-12, max_cycles=40, same_cycles=True):
    c = p.coarse
    pc_o, pf_o, st_o, cyc_o, rr_o, hist_o = o.solve(c.rhs, p.rhs_f, phic0, phif0, rtol=rtol, max_cycles=max_cycles)
    gc = dev(np.zeros_like(c.rhs) if phic0 is None else phic0)
    if p.multi:
        gf = [dev(np.zeros_like(r) if phif0 is None else phif0[q]) for q, r in enumerate(p.rhs_f)]
        rf = [dev(r) for r in p.rhs_f]
    else:
        gf = dev(np.zeros_like(p.rhs_f) if phif0 is None else phif0)
        rf = dev(p.rhs_f)
    pc, pf, st, cyc, rr, hist = s.solve(dev(c.rhs), rf, gc, gf, rtol=rtol, max_cycles=max_cycles)
    assert st == st_o, (st, st_o, hist, hist_o)
    if same_cycles:
        assert cyc == cyc_o, (cyc, cyc_o, hist, hist_o)
    n = min(len(hist), len(hist_o))
    for i in range(n):       # 2e-15: the rounding floor of a residual formed from O(1) fields (the GPU runs the coarse V-cycle in place
        if hist_o[i] > 1e-10:    # on phi_c and differences the covered cells for the patch's correction; the oracle solves for the correction)
            assert abs(hist[i] - hist_o[i]) <= 1e-6 * hist_o[i] + 2e-15, (i, hist[i], hist_o[i])
    for g, w in zip(pf if p.multi else [pf], pf_o if p.multi else [pf_o]):
        assert rel(g.cpu().numpy(), w) <= PHI_TOL
    assert rel(pc.cpu().numpy(), pc_o) <= PHI_TOL          # covered cells included: means of the children on both sides
    return pc, pf, cyc, hist


CASES = [
    dict(n=(32, 16, 16), lo=(8, 4, 4), hi=(24, 12, 12), spacing=None, alpha=1.0),
    dict(n=(40, 24, 16), lo=(6, 5, 3), hi=(20, 13, 9), spacing=(0.1, 0.07, 0.13), alpha=1.0),     # ragged, anisotropic spacing
    dict(n=(48, 40, 1), lo=(8, 6, 0), hi=(32, 26, 1), spacing=None, alpha=1.0),                    # 2-D
    dict(n=(24, 24, 24), lo=(1, 3, 1), hi=(17, 23, 21), spacing=None, alpha=0.0),                  # one cell from the x-low, y-high and z-low faces
    dict(n=(64, 32, 32), lo=(30, 2, 14), hi=(34, 30, 18), spacing=None, alpha=0.0),                # a thin slab of a patch
    dict(n=(48, 32, 32), lo=(5, 3, 9), hi=(28, 25, 20), spacing=None, alpha=1.0),                  # 23 x 22 x 11 coarse cells: no hierarchy of its own
]


@pytest.mark.parametrize("case", CASES)
def test_composite_solve_matches_the_oracle(case):
    n = case["n"]
    p = inputs.amr_random_problem(*n, case["lo"], case["hi"], seed=sum(n), alpha=case["alpha"], sigma=0.7,
                                  spacing=case["spacing"])
    o, s = _oracle(p), _gpu(p)
    rng = np.random.default_rng(5)
    phic0, phif0 = rng.standard_normal(p.coarse.rhs.shape), rng.standard_normal(p.rhs_f.shape)
    pc, pf, cyc, hist = _compare(p, s, o, phic0, phif0)
    assert hist[-1] <= 1e-12 and cyc <= 20
    assert s.pad_check() == 0                 # no kernel of the composite cycle wrote a zero pad of either handle
    ratios = [hist[i] / hist[i - 1] for i in range(2, len(hist)) if hist[i] > 1e-11]
    assert max(ratios) < 0.25, ratios
    # a second solve on the same handles from a zero guess, then with new coefficients (1/D of the patch is rebuilt)
    _compare(p, s, o)
    q = inputs.amr_random_problem(*n, case["lo"], case["hi"], seed=sum(n) + 1, alpha=case["alpha"], sigma=0.7,
                                  spacing=case["spacing"])
    c = q.coarse
    o.set_coeffs(q.coarse_coeffs(), q.fine_coeffs(), c.alpha, c.beta)
    o.set_bc(c.bc_type, c.bc_value)
    s.set_coeffs([dev(x) for x in q.coarse_coeffs()], _dev_fine(q, q.fine_coeffs()), c.alpha, c.beta)
    s.set_bc(c.bc_type, [dev(v) for v in c.bc_value])
    _compare(q, s, o)


MULTI = [
    dict(n=(48, 32, 16), lo=[(4, 4, 2), (28, 6, 4)], hi=[(20, 20, 10), (44, 26, 12)], alpha=1.0),                    # two patches
    dict(n=(64, 48, 1), lo=[(4, 4, 0), (30, 6, 0), (8, 30, 0)], hi=[(24, 24, 1), (60, 26, 1), (56, 44, 1)], alpha=0.0),   # 2-D, three
    dict(n=(32, 32, 32), lo=[(1, 1, 1), (19, 1, 1), (1, 19, 19)], hi=[(17, 17, 17), (31, 29, 17), (29, 31, 31)], alpha=0.0),  # two cells apart, next to the faces
]


@pytest.mark.parametrize("case", MULTI)
def test_composite_solve_with_several_patches_matches_the_oracle(case):
    n = case["n"]
    p = inputs.amr_random_problem(*n, case["lo"], case["hi"], seed=sum(n) + 3, alpha=case["alpha"], sigma=0.7)
    assert p.multi
    o, s = _oracle(p), _gpu(p)
    rng = np.random.default_rng(6)
    phic0 = rng.standard_normal(p.coarse.rhs.shape)
    phif0 = [rng.standard_normal(r.shape) for r in p.rhs_f]
    pc, pf, cyc, hist = _compare(p, s, o, phic0, phif0)
    assert hist[-1] <= 1e-12 and cyc <= 20 and s.pad_check() == 0
    _compare(p, s, o)                                            # again from a zero guess on the same handles
    s2 = _gpu(p, graph=0)                                        # plain launches: bitwise the graphs' result
    pc0, pf0, *_ = s.solve(dev(p.coarse.rhs), [dev(r) for r in p.rhs_f], rtol=1e-12, max_cycles=40)
    pc2, pf2, st2, cyc2, rr2, hist2 = s2.solve(dev(p.coarse.rhs), [dev(r) for r in p.rhs_f], rtol=1e-12, max_cycles=40)
    assert torch.equal(pc0, pc2) and all(torch.equal(x, y) for x, y in zip(pf0, pf2))


def test_plain_launches_fixed_cycle_counts_and_options():
    p = inputs.amr_random_problem(32, 16, 16, (8, 4, 4), (24, 12, 12), seed=9, sigma=0.7)
    o = _oracle(p)
    s = _gpu(p)
    pc, pf, cyc, hist = _compare(p, s, o)
    launches = s.last_launch_count()
    assert launches > 0
    # graph = 0 on the coarse handle: the same kernels as plain launches, bitwise the same result
    s2 = _gpu(p, graph=0)
    pc2, pf2, st2, cyc2, rr2, hist2 = s2.solve(dev(p.coarse.rhs), dev(p.rhs_f), rtol=1e-12, max_cycles=40)
    assert cyc2 == cyc and hist2 == hist
    assert torch.equal(pc2, pc) and torch.equal(pf2, pf)
    # device_loop = 0: one graph replay and one read-back per cycle instead of the conditional-WHILE graph: bitwise the same
    s3 = _gpu(p, device_loop=0)
    pc3, pf3, st3, cyc3, rr3, hist3 = s3.solve(dev(p.coarse.rhs), dev(p.rhs_f), rtol=1e-12, max_cycles=40)
    assert cyc3 == cyc and hist3 == hist and torch.equal(pc3, pc) and torch.equal(pf3, pf)
    # every exit rule through the device-side loop against the host loop: MAXCYCLES short of convergence, unreachable rtol -> STALLED
    for rtol, maxc in ((1e-12, 3), (1e-17, 40), (1e-3, 40)):
        g = s.solve(dev(p.coarse.rhs), dev(p.rhs_f), rtol=rtol, max_cycles=maxc)
        w = s3.solve(dev(p.coarse.rhs), dev(p.rhs_f), rtol=rtol, max_cycles=maxc)
        assert g[2] == w[2] and g[3] == w[3] and g[5] == w[5] and torch.equal(g[0], w[0]) and torch.equal(g[1], w[1]), (rtol, maxc, g[2:4], w[2:4])
    # rtol = 0: exactly max_cycles cycles, status MAXCYCLES, history of max_cycles + 1 entries
    o5 = o.solve(p.coarse.rhs, p.rhs_f, rtol=0.0, max_cycles=5)
    g5 = s.solve(dev(p.coarse.rhs), dev(p.rhs_f), rtol=0.0, max_cycles=5)
    assert g5[2] == 1 and o5[2] == 1 and g5[3] == 5 and len(g5[5]) == 6
    assert rel(g5[1].cpu().numpy(), o5[1]) <= 1e-12 and rel(g5[0].cpu().numpy(), o5[0]) <= 1e-12
    # other sweep counts on both sides
    for key, v in (("nu_f", 3), ("nu1", 2), ("nu2", 2)):
        o.set_option(key, v)
        s.set_option(key, v)
    _compare(p, s, o)
    # zero data: phi = 0 in zero cycles
    z = s.solve(dev(np.zeros_like(p.coarse.rhs)), dev(np.zeros_like(p.rhs_f)), dev(p.coarse.rhs.copy()), dev(p.rhs_f.copy()))
    s.set_bc(p.coarse.bc_type, None)
    z = s.solve(dev(np.zeros_like(p.coarse.rhs)), dev(np.zeros_like(p.rhs_f)), dev(p.coarse.rhs.copy()), dev(p.rhs_f.copy()))
    assert z[2] == 0 and z[3] == 0 and float(z[0].abs().max()) == 0.0 and float(z[1].abs().max()) == 0.0


def test_argument_and_state_errors():
    b = _binding()
    with pytest.raises(b.VmgError) as e:
        b.VmgAmr(16, 16, 16, 0.1, 0.1, 0.1, (0, 4, 4), (8, 12, 12))          # touches the boundary
    assert e.value.code == -2
    with pytest.raises(b.VmgError) as e:
        b.VmgAmr(16, 16, 16, 0.1, 0.1, 0.1, (4, 4, 4), (5, 12, 12))          # one coarse cell wide
    assert e.value.code == -2
    with pytest.raises(b.VmgError) as e:
        b.VmgAmr(32, 16, 16, 0.1, 0.1, 0.1, [(2, 2, 2), (11, 2, 2)], [(10, 10, 10), (20, 10, 10)])   # one coarse cell apart
    assert e.value.code == -2
    s = b.VmgAmr(16, 16, 16, 0.1, 0.1, 0.1, (4, 4, 4), (12, 12, 12))
    with pytest.raises(b.VmgError) as e:
        s.solve(torch.zeros(16, 16, 16, dtype=torch.float64, device="cuda"), torch.zeros(16, 16, 16, dtype=torch.float64, device="cuda"))
    assert e.value.code == -3


def test_streamer_patch_at_full_size_against_the_oracle():
    """config 3 with the streamer head refined: 256 x 128 x 128 box (constant-weight kernels: b == NULL on the box) + a
    128 x 64 x 64 patch with explicit arrays of ones; histories and phi against the oracle."""
    p = inputs.amr_streamer(128)
    p.coarse.bx = p.coarse.by = p.coarse.bz = None
    o, s = _oracle(p), _gpu(p)
    pc, pf, cyc, hist = _compare(p, s, o, max_cycles=30)
    assert hist[-1] <= 1e-12 and cyc <= 14


def test_three_streamer_patches_at_full_size_against_the_oracle():
    """bench.py's amr.three_patches workload: the 256 x 128 x 128 box + three 128 x 64 x 64 patches (parallel graph branches)."""
    p = inputs.amr_streamers(128)
    o, s = _oracle(p), _gpu(p)
    pc, pf, cyc, hist = _compare(p, s, o, max_cycles=30)
    assert hist[-1] <= 1e-12 and cyc <= 14 and s.pad_check() == 0
