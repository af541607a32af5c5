"""GPU parity: the CUDA path (through the C-ABI of libvmg.so) against the CPU oracle on the same seeded inputs.

Bars (BASELINE.json:north_star): relative L-inf difference of phi <= 1e-10 after both reach relative
residual 1e-12, V-cycle counts equal within 1.  Single steps: <= 1e-13 relative (rounding-order only:
the GPU uses pre-multiplied face weights, a reciprocal diagonal and FMAs).
"""
import os

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import Oracle, OracleError
from paper_2507_08200_b200 import inputs
from paper_2507_08200_b200.inputs import DIRICHLET as D, NEUMANN as N

pytestmark = pytest.mark.gpu

STEP_TOL = 1e-13
PHI_TOL = 1e-10


def _binding():
    from paper_2507_08200_b200 import binding
    return binding


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def rel(a, b):
    return np.abs(a - b).max() / max(np.abs(b).max(), 1e-300)


# sizes span several 256-thread blocks / tiles with ragged tails, odd coarse grids and the 2-D path
SIZES = [(40, 24, 16), (72, 40, 24), (16, 8, 8), (48, 40, 1), (88, 56, 24), (5, 3, 4), (144, 80, 48)]
MIXED = [D, N, N, D, D, N]


@pytest.mark.parametrize("dims", SIZES)
def test_single_steps_match_oracle(dims):
    b = _binding()
    p = inputs.random_problem(*dims, seed=sum(dims), bc_type=MIXED, sigma=1.0)
    o = Oracle.from_problem(p)
    s, d = b.from_problem(p)
    assert s.num_levels == o.num_levels
    rng = np.random.default_rng(7)
    for lev in range(o.num_levels):
        assert s.level_dims(lev) == o.level_dims(lev)
        nx, ny, nz = o.level_dims(lev)
        if lev > 0:   # S0 coefficient averaging
            ca = o.level_coeffs(lev)
            ga = s.get_level_coeffs(lev)
            for name, x, y in zip("a bx by bz".split(), ga, ca):
                if name == "bz" and nz == 1 and p.nz == 1:
                    continue
                assert rel(x.cpu().numpy(), y) <= 1e-15, (lev, name)
        phi = rng.standard_normal((nz, ny, nx))
        rhs = rng.standard_normal((nz, ny, nx)) * 50.0
        # S2 smoother, 1 and 3 sweeps
        for ns in (1, 3):
            assert rel(s.step_smooth(lev, dev(phi), dev(rhs), ns).cpu().numpy(), o.smooth(phi, rhs, ns, lev)) <= STEP_TOL
        # residual
        r_o = o.residual(phi, rhs, lev)
        assert rel(s.step_residual(lev, dev(phi), dev(rhs)).cpu().numpy(), r_o) <= STEP_TOL
        if lev + 1 < o.num_levels:
            # S3 fused residual + restriction; S4 fused prolongation + correction
            assert np.abs(s.step_residual_restrict(lev, dev(phi), dev(rhs)).cpu().numpy() - o.restrict(r_o, lev)).max() \
                <= STEP_TOL * np.abs(r_o).max()
            cnx, cny, cnz = o.level_dims(lev + 1)
            e = rng.standard_normal((cnz, cny, cnx))
            assert np.array_equal(s.step_prolong_correct(lev, dev(phi), dev(e)).cpu().numpy(), o.prolong_add(phi, e, lev))
            # whole strokes as vmg_solve runs them (fused blocked passes where the level qualifies)
            phi_d, rc_d = s.step_down(lev, dev(phi), dev(rhs))
            phi_sm = o.smooth(phi, rhs, 3, lev)
            assert rel(phi_d.cpu().numpy(), phi_sm) <= STEP_TOL
            assert np.abs(rc_d.cpu().numpy() - o.restrict(o.residual(phi_sm, rhs, lev), lev)).max() <= STEP_TOL * np.abs(r_o).max()
            phi_u = s.step_up(lev, dev(phi), dev(rhs), dev(e))
            assert rel(phi_u.cpu().numpy(), o.smooth(o.prolong_add(phi, e, lev), rhs, 3, lev)) <= STEP_TOL
    # S1 fold_bc, S6 norm, one whole V-cycle (S7)
    bt_o = o.fold_bc(p.rhs)
    bt_g = s.step_fold_bc(d["rhs"]).cpu().numpy()
    assert rel(bt_g, bt_o) <= STEP_TOL
    assert s.step_norm_inf(dev(bt_o)) == np.abs(bt_o).max()
    phi0 = rng.standard_normal(p.rhs.shape)
    for graph in (0, 1):
        s.set_option("graph", graph)
        assert rel(s.step_vcycle(dev(phi0), dev(bt_o)).cpu().numpy(), o.vcycle(phi0, bt_o)) <= 1e-12
    s.destroy()


def test_schedule_options_do_not_change_a_single_bit():
    """Direction of traversal, L2 carve-out, cache policy of the loads, graph replay and the single-CTA tail only reorder independent work:
    the converged phi and the residual history are bitwise those of the plain in-order launches."""
    b = _binding()
    p = inputs.config4(32)
    ref = None
    for opts in (dict(snake=0, l2_persist=0, graph=0, tail=0), dict(), dict(snake=1, graph=0), dict(tail=0), dict(blocked=1),
                 dict(blocked=2), dict(blocked=3, block_min_cells=0), dict(device_loop=0), dict(device_loop=0, graph=0), dict(cluster=0), dict(cluster=0, device_loop=0),
                 dict(phi_keep_cells=0), dict(phi_keep_cells=0, graph=0, tail=0)):   # cache policy of the largest levels on all levels
        s, d = b.from_problem(p)
        for k, v in opts.items():
            s.set_option(k, v)
        phi = torch.zeros_like(d["rhs"])
        assert s.solve(d["rhs"], phi, rtol=p.rtol, max_vcycles=p.max_vcycles) == 0
        out = (phi.clone(), list(s.get_info()[2]))
        s.destroy()
        if ref is None:
            ref = out
        else:
            assert torch.equal(out[0], ref[0]) and out[1] == ref[1], opts


@pytest.mark.parametrize("rtol,maxc", [(1e-12, 50), (0.0, 7), (1e-12, 3), (1e-17, 40), (1e-3, 50)],
                         ids=["converges", "fixed_cycles", "maxcycles", "stalls_on_the_floor", "two_cycles"])
def test_device_side_solve_loop_applies_the_exit_rules_of_the_host_loop(rtol, maxc):
    """The solve as one graph with a conditional WHILE node (exit rules C5 on the device, the residual norm riding on the
    first half-sweep of the next cycle, option device_loop = 1, default) returns the status, the cycle count, the history and
    phi of the host-driven loop bit for bit -- for every exit rule, from a zero and from a warm start, and it leaves a
    converged iterate untouched although the next cycle's first half-sweep has already run."""
    b = _binding()
    p = inputs.config4(32)
    out = {}
    for loop in (0, 1):
        s, d = b.from_problem(p)
        s.set_option("device_loop", loop)
        res = []
        phi = torch.zeros_like(d["rhs"])
        for rep in range(2):                    # second solve: warm start from the first result (often 0 or 1 cycles)
            st = s.solve(d["rhs"], phi, rtol=rtol, max_vcycles=maxc)
            cyc, rr, hist = s.get_info()
            res.append((st, cyc, list(hist), phi.clone()))
        out[loop] = res
        s.destroy()
    for a, c in zip(out[0], out[1]):
        assert a[0] == c[0] and a[1] == c[1] and a[2] == c[2] and torch.equal(a[3], c[3]), (a[:3], c[:3])
    assert out[1][0][0] == {"converges": 0, "fixed_cycles": 1, "maxcycles": 1, "stalls_on_the_floor": 2, "two_cycles": 0}[
        {(1e-12, 50): "converges", (0.0, 7): "fixed_cycles", (1e-12, 3): "maxcycles", (1e-17, 40): "stalls_on_the_floor", (1e-3, 50): "two_cycles"}[(rtol, maxc)]]


@pytest.mark.parametrize("dims", [(40, 24, 16), (72, 40, 24), (5, 3, 4), (48, 40, 1)])
def test_no_kernel_writes_the_zero_pads(dims):
    """Own memory check (compute-sanitizer is closed on this pool, profiles/r2_sanitizers.md): the zero pads around and inside
    every internal array stand for the neighbours beyond the domain and must never be written.  After every kernel family has
    run on a handle -- per-colour sweeps, the three blocked designs with fused transfers, the single-CTA tail, the device-side
    loop, plain launches, PCG, a masked solve -- not one pad element is non-zero."""
    b = _binding()
    p = inputs.random_problem(*dims, seed=5, bc_type=MIXED, sigma=1.0)
    s, d = b.from_problem(p)
    assert s.pad_check() == 0
    rng = np.random.default_rng(2)
    three_d = p.nz > 1
    for opts in (dict(), dict(device_loop=0), dict(graph=0, tail=0), dict(blocked=1, block_min_cells=0),
                 dict(blocked=2, block_min_cells=0), dict(blocked=3, block_min_cells=0), dict(prolong=1)):
        for k, v in opts.items():
            s.set_option(k, v)
        phi = torch.zeros_like(d["rhs"])
        s.solve(d["rhs"], phi, rtol=1e-12, max_vcycles=30)
        for lev in range(s.num_levels - 1):
            nx, ny, nz = s.level_dims(lev)
            cnx, cny, cnz = s.level_dims(lev + 1)
            f, r = dev(rng.standard_normal((nz, ny, nx))), dev(rng.standard_normal((nz, ny, nx)))
            s.step_smooth(lev, f, r, 3); s.step_down(lev, f, r); s.step_up(lev, f, r, dev(rng.standard_normal((cnz, cny, cnx))))
        assert s.pad_check() == 0, opts
        for k in opts:
            s.set_option(k, dict(device_loop=1, graph=1, tail=1, blocked=0, block_min_cells=4096, prolong=0)[k])
    phi = torch.zeros_like(d["rhs"])
    s.solve_pcg(d["rhs"], phi, 1e-12, 30)
    assert s.pad_check() == 0
    if three_d and min(dims) >= 8:
        mask = torch.ones(p.rhs.shape, dtype=torch.uint8, device="cuda")
        mask[2:5, 3:6, 1:4] = 0
        s.set_mask(mask, D, None)
        s.set_coeffs(d["a"], d["bx"], d["by"], d["bz"], p.alpha, p.beta)
        phi = torch.zeros_like(d["rhs"])
        s.solve(d["rhs"], phi, rtol=1e-10, max_vcycles=60)
        assert s.pad_check() == 0
    s.destroy()


@pytest.mark.parametrize("dims", [(40, 24, 16), (88, 56, 24), (144, 80, 48), (256, 128, 32)])
def test_blocked_passes_equal_plain_launches_bitwise(dims):
    """The temporally blocked passes (with fused prolongation / restriction) relax in the same order with the
    same expression as one launch per colour: bitwise equal on every level with even dimensions, on sizes that
    span several tiles and z-segments with ragged edges."""
    b = _binding()
    p = inputs.random_problem(*dims, seed=11, bc_type=MIXED, sigma=1.0)
    s, d = b.from_problem(p)
    s.set_option("block_min_cells", 0)
    s.set_option("restrict_red_cells", 2.0 ** 40)   # the blocked passes restrict all eight children's residuals: compare like with like
    rng = np.random.default_rng(3)
    for lev in range(s.num_levels - 1):
        nx, ny, nz = s.level_dims(lev)
        if nx % 2 or ny % 2 or nz % 2:
            break
        cnx, cny, cnz = s.level_dims(lev + 1)
        phi, rhs = dev(rng.standard_normal((nz, ny, nx))), dev(rng.standard_normal((nz, ny, nx)) * 50.0)
        e = dev(rng.standard_normal((cnz, cny, cnx)))
        out = {}
        for blocked in (1, 2, 3, 0):   # vmg_block2.cuh; vmg_block3.cuh (TMA-fed): 2 x 2 patches, rows; per-colour launches
            s.set_option("blocked", blocked)
            res = [s.step_smooth(lev, phi, rhs, ns) for ns in (1, 2, 3, 4)]
            for nu in (1, 2, 3):
                s.set_option("nu1", nu)
                s.set_option("nu2", nu)
                res += list(s.step_down(lev, phi, rhs)) + [s.step_up(lev, phi, rhs, e)]
            out[blocked] = res
        for blocked in (1, 2, 3):
            for x, y in zip(out[blocked], out[0]):
                assert torch.equal(x, y), (blocked, lev, (x - y).abs().max().item())
    s.destroy()


def solve_both(p, **opts):
    b = _binding()
    o = Oracle.from_problem(p)
    s, d = b.from_problem(p)
    for k, v in opts.items():
        o.set_option(k, v) if k in ("nu1", "nu2", "bottom_sweeps", "prolong") else None
    for k, v in opts.items():
        s.set_option(k, v)
    phi_o, st_o, cyc_o, rr_o, hist_o = o.solve(p.rhs, rtol=p.rtol, max_vcycles=p.max_vcycles)
    phi_g = torch.zeros_like(d["rhs"])
    st_g = s.solve(d["rhs"], phi_g, rtol=p.rtol, max_vcycles=p.max_vcycles)
    cyc_g, rr_g, hist_g = s.get_info()
    s.destroy()
    return (phi_o, st_o, cyc_o, rr_o, hist_o), (phi_g.cpu().numpy(), st_g, cyc_g, rr_g, np.array(hist_g))


def check_parity(p, **opts):
    (phi_o, st_o, cyc_o, rr_o, hist_o), (phi_g, st_g, cyc_g, rr_g, hist_g) = solve_both(p, **opts)
    assert st_o == st_g, (st_o, st_g)
    assert abs(cyc_o - cyc_g) <= 1, (cyc_o, cyc_g)
    if p.rtol > 0:
        assert rr_o <= p.rtol and rr_g <= p.rtol
    assert rel(phi_g, phi_o) <= PHI_TOL, rel(phi_g, phi_o)
    # residual histories agree while above the rounding floor
    m = min(len(hist_o), len(hist_g))
    live = hist_o[:m] > 1e-11
    assert np.all(np.abs(hist_g[:m][live] / hist_o[:m][live] - 1.0) < 1e-3)
    return cyc_o, cyc_g, rel(phi_g, phi_o)


@pytest.mark.parametrize("make", [lambda: inputs.config1(64), lambda: inputs.config2(32), lambda: inputs.config3(32),
                                  lambda: inputs.config4(32), lambda: inputs.config4(32, sheath=True),
                                  lambda: inputs.config5(64, cycles=20)],
                         ids=["config1", "config2_32", "config3_64x32x32", "config4_64x32x32", "config4b", "config5_64"])
def test_configs_reduced_size_parity(make):
    check_parity(make())


@pytest.mark.parametrize("make", [lambda: inputs.config2(128), lambda: inputs.config3(128), lambda: inputs.config4(128)],
                         ids=["config2_128^3", "config3_256x128x128", "config4_256x128x128"])
def test_configs_full_size_parity(make):
    """BASELINE.json configs[1..3] at full size, in the launch configuration bench.py times (defaults)."""
    p = make()
    cyc_o, cyc_g, err = check_parity(p)
    assert 8 <= cyc_g <= 12


_C5 = {}


def _config5_full():
    """BASELINE.json configs[4] at its full size, generated once for the tests that use it (5.4 GB of host arrays)."""
    if "p" not in _C5:
        _C5["p"] = inputs.config5(512)
    return _C5["p"]


@pytest.mark.parametrize("opts", [dict(nu1=2, nu2=2), dict(nu1=1, nu2=3, bottom_sweeps=8), dict(graph=0), dict(blocked=0),
                                  dict(tail=0), dict(blocked=0, tail=0, graph=0), dict(block_min_cells=0),
                                  dict(block_min_cells=0, graph=0, nu1=2, nu2=4), dict(block_min_cells=0, nu1=1, nu2=2),
                                  dict(block_min_cells=0, nu1=4, nu2=1, tail=0), dict(snake=0), dict(l2_persist=0, snake=0, graph=0),
                                  dict(blocked=1, block_min_cells=0), dict(nu1=3, nu2=1), dict(prolong=1, nu1=2, nu2=2), dict(prolong=1),
                                  dict(prolong=1, blocked=1, block_min_cells=0), dict(prolong=1, tail=0, graph=0)])
def test_options_parity(opts):
    check_parity(inputs.random_problem(48, 24, 48, seed=3, bc_type=[D, D, N, N, N, D]), **opts)


@pytest.mark.parametrize("nu", [(2, 0), (0, 2), (0, 0)])
def test_one_sided_smoothing_matches_oracle_cycle_by_cycle(nu):
    """nu2 = 0 takes the stand-alone prolongation kernel, nu1 = 0 restricts the unsmoothed residual: four fixed
    cycles (these variants converge slowly or not at all), phi and history against the oracle."""
    b = _binding()
    p = inputs.random_problem(48, 24, 48, seed=3, bc_type=[D, D, N, N, N, D])
    o = Oracle.from_problem(p)
    s, d = b.from_problem(p)
    for k, v in zip(("nu1", "nu2"), nu):
        o.set_option(k, v)
        s.set_option(k, v)
    phi_o, st_o, cyc_o, rr_o, hist_o = o.solve(p.rhs, rtol=0.0, max_vcycles=4)
    phi = torch.zeros_like(d["rhs"])
    assert s.solve(d["rhs"], phi, rtol=0.0, max_vcycles=4) == st_o == 1
    assert rel(phi.cpu().numpy(), phi_o) <= 1e-12
    assert np.allclose(np.array(s.get_info()[2]), hist_o, rtol=1e-9)
    s.destroy()


def test_edge_cases_and_status_codes():
    b = _binding()
    p = inputs.random_problem(32, 16, 16, seed=5, bc_type=[D, D, N, N, N, N])
    o = Oracle.from_problem(p)
    s, d = b.from_problem(p)
    phi = torch.zeros_like(d["rhs"])
    assert s.solve(d["rhs"], phi, rtol=1e-9) == 0
    cyc, rr, hist = s.get_info()
    phi_o, st_o, cyc_o, rr_o, hist_o = o.solve(p.rhs, rtol=1e-9)
    assert cyc == cyc_o and len(hist) == cyc + 1 and abs(hist[0] - 1.0) < 1e-15
    assert s.last_launch_count() > 0
    # warm start from the converged field: 0 cycles, phi untouched
    keep = phi.clone()
    assert s.solve(d["rhs"], phi, rtol=1e-9) == 0 and s.get_info()[0] == 0 and torch.equal(phi, keep)
    # rtol <= 0: exactly max_vcycles cycles
    phi.zero_()
    assert s.solve(d["rhs"], phi, rtol=0.0, max_vcycles=3) == 1 and s.get_info()[0] == 3
    phi3_o, *_ = o.solve(p.rhs, rtol=0.0, max_vcycles=3)
    assert rel(phi.cpu().numpy(), phi3_o) <= 1e-12
    # unreachable tolerance stalls on the rounding floor, like the oracle
    phi.zero_()
    assert s.solve(d["rhs"], phi, rtol=1e-30, max_vcycles=60) == 2
    # zero rhs with homogeneous data: phi = 0 after 0 cycles
    s.set_bc(p.bc_type, None)
    phi.fill_(1.0)
    assert s.solve(torch.zeros_like(phi), phi) == 0 and s.get_info()[0] == 0 and not phi.any()
    # NaN in the right-hand side: DIVERGED, handle stays usable
    bad = d["rhs"].clone()
    bad[3, 3, 3] = float("nan")
    with pytest.raises(b.VmgError) as e:
        s.solve(bad, phi)
    assert e.value.code == -5
    phi.zero_()
    assert s.solve(d["rhs"], phi, rtol=1e-9) == 0
    # pure Neumann without absorption: SINGULAR
    s.set_coeffs(None, d["bx"], d["by"], d["bz"], 0.0, 1.0)
    s.set_bc([N] * 6, None)
    with pytest.raises(b.VmgError) as e:
        s.solve(d["rhs"], phi)
    assert e.value.code == -4
    s.destroy()
    # solve before set_coeffs / set_bc: STATE
    s2 = b.Vmg(16, 8, 8, 1.0, 1.0, 1.0)
    with pytest.raises(b.VmgError) as e:
        s2.solve(phi[:8, :8, :16].contiguous(), phi[:8, :8, :16].contiguous())
    assert e.value.code == -3
    s2.destroy()
    with pytest.raises(b.VmgError) as e:
        b.Vmg(1030, 1030, 1030, 1.0, 1.0, 1.0)
    assert e.value.code == -2


def test_null_coefficients_mean_a_zero_b_one_and_bc_order_is_free():
    b = _binding()
    p = inputs.config3(16)
    o = Oracle.from_problem(p)
    phi_o, st_o, cyc_o, *_ = o.solve(p.rhs)
    d = b.upload(p)
    s = b.Vmg(p.nx, p.ny, p.nz, p.dx, p.dy, p.dz)
    s.set_bc(p.bc_type, d["bc_value"])                   # bc before coeffs is legal
    s.set_coeffs(None, None, None, None, 0.0, 1.0)       # NULL a, NULL b
    phi = torch.zeros_like(d["rhs"])
    assert s.solve(d["rhs"], phi) == 0 and abs(s.get_info()[0] - cyc_o) <= 1
    assert rel(phi.cpu().numpy(), phi_o) <= PHI_TOL
    # changing BC types afterwards re-finalises the diagonal
    types = [D, N, N, N, N, N]
    s.set_bc(types, d["bc_value"])
    o.set_bc(types, p.bc_value)
    phi.zero_()
    phi_o2, st2, cyc2, *_ = o.solve(p.rhs)
    assert s.solve(d["rhs"], phi) == st2
    assert rel(phi.cpu().numpy(), phi_o2) <= PHI_TOL
    s.destroy()


def test_user_stream_and_repeatability():
    b = _binding()
    p = inputs.config4(16)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        s, d = b.from_problem(p, stream=st)
        phi1 = torch.zeros_like(d["rhs"])
        phi2 = torch.zeros_like(d["rhs"])
        assert s.solve(d["rhs"], phi1) == 0
        assert s.solve(d["rhs"], phi2) == 0
    st.synchronize()
    assert torch.equal(phi1, phi2)          # red-black updates are order independent: bitwise repeatable
    s.destroy()


def test_batched_solves_are_bitwise_the_single_solves():
    """vmg_solve_batch: different problems on different streams advanced in lock-step
    give bit for bit what vmg_solve gives for each, with their own cycle counts and statuses."""
    b = _binding()
    probs = [inputs.config3(16), inputs.config4(16), inputs.config2(32), inputs.random_problem(40, 24, 16, seed=9, bc_type=MIXED)]
    single = []
    for p in probs:
        s, d = b.from_problem(p)
        phi = torch.zeros_like(d["rhs"])
        st = s.solve(d["rhs"], phi, rtol=1e-12, max_vcycles=30)
        single.append((st, s.get_info(), phi.clone()))
        s.destroy()
    streams = [torch.cuda.Stream() for _ in probs]
    solvers, data = [], []
    for p, stream in zip(probs, streams):
        with torch.cuda.stream(stream):
            s, d = b.from_problem(p, stream=stream)
        solvers.append(s); data.append(d)
    torch.cuda.synchronize()
    phis = [torch.zeros_like(d["rhs"]) for d in data]
    sts = b.solve_batch(solvers, [d["rhs"] for d in data], phis, rtol=1e-12, max_vcycles=30)
    for p, s, st, phi, ref in zip(probs, solvers, sts, phis, single):
        cyc, rr, hist = s.get_info()
        assert st == ref[0] and cyc == ref[1][0] and list(hist) == list(ref[1][2])
        assert torch.equal(phi, ref[2])
        s.destroy()
        # ... and each result of the batch against the oracle's solve of that problem (parity, not self-consistency)
        o = Oracle.from_problem(p)
        phi_o, st_o, cyc_o, rr_o, hist_o = o.solve(p.rhs, rtol=1e-12, max_vcycles=30)
        o.close()
        assert st == st_o and abs(cyc - cyc_o) <= 1, (p.name, st, st_o, cyc, cyc_o)
        assert rel(phi.cpu().numpy(), phi_o) <= PHI_TOL, p.name
        m = min(len(hist), len(hist_o))
        live = hist_o[:m] > 1e-11
        assert np.all(np.abs(np.array(hist)[:m][live] / hist_o[:m][live] - 1.0) < 1e-3), p.name
    # the staggered schedule (three graphs per handle, token events) keeps no state between calls: the same handles again,
    # in another order, one of them switched to constant weights, then alone through vmg_solve
    solvers, data, streams2 = [], [], [torch.cuda.Stream() for _ in probs]
    for p, stream in zip(probs, streams2):
        s, d = b.from_problem(p, stream=stream)
        solvers.append(s); data.append(d)
    torch.cuda.synchronize()
    for rnd in range(3):
        order = [0, 1, 2, 3] if rnd == 0 else [3, 1, 0, 2] if rnd == 1 else [2, 0]
        want = list(single)
        if rnd >= 1:   # problem 0 (b = 1) with b == NULL: bitwise the same solve through the constant-weight kernels
            solvers[0].set_coeffs(data[0]["a"], None, None, None, probs[0].alpha, probs[0].beta)
        phis = [torch.zeros_like(data[i]["rhs"]) for i in order]
        sts = b.solve_batch([solvers[i] for i in order], [data[i]["rhs"] for i in order], phis, rtol=1e-12, max_vcycles=30)
        for i, st, phi in zip(order, sts, phis):
            cyc, rr, hist = solvers[i].get_info()
            assert st == want[i][0] and cyc == want[i][1][0] and list(hist) == list(want[i][1][2]), (rnd, i)
            assert torch.equal(phi, want[i][2]), (rnd, i)
    for i, s in enumerate(solvers):
        phi = torch.zeros_like(data[i]["rhs"])
        with torch.cuda.stream(streams2[i]):
            st = s.solve(data[i]["rhs"], phi, rtol=1e-12, max_vcycles=30)
        assert st == single[i][0] and torch.equal(phi, single[i][2])
        s.destroy()
    # a handle may appear once; an unready handle reports its own error without stopping the others
    s1, d1 = b.from_problem(probs[0])
    s2 = b.Vmg(16, 8, 8, 1.0, 1.0, 1.0)
    with pytest.raises(b.VmgError) as e:
        b.solve_batch([s1, s2], [d1["rhs"], d1["rhs"]], [torch.zeros_like(d1["rhs"]), torch.zeros_like(d1["rhs"])])
    assert e.value.code == -3
    s1.destroy(); s2.destroy()


@pytest.mark.parametrize("full_mb", [400.0, 0.0], ids=["all_levels_batched", "coarse_levels_batched"])
def test_kernel_level_batch_matches_oracle_and_single_solves(full_mb):
    """SURVEY.md 8(f) N1 as written: K problems on one grid INSIDE the kernels -- vmg_create_batch puts the
    members' arenas a constant stride apart, vmg_solve_batch runs the levels problem-major (blockIdx.z = planes x problems,
    K CTAs in the tail, one graph; all levels, or -- option batch_full_mb = 0 -- the coarser levels with level 0 one problem
    at a time).  Four different problems (coefficients, boundary kinds and data, right-hand sides; they need 8-10 cycles, so
    the last cycles run with some members finished): every phi against the ORACLE's solve, and status, cycle count,
    history and phi bitwise against vmg_solve on an ordinary handle; a second call and a changed member afterwards."""
    b = _binding()
    probs = [inputs.config4(32), inputs.config3(32), inputs.random_problem(64, 32, 32, seed=3, bc_type=[D, N, N, D, N, N]),
             inputs.random_problem(64, 32, 32, seed=4, bc_type=[D, D, N, N, N, D])]

    def single(p, d):
        s = b.Vmg(p.nx, p.ny, p.nz, p.dx, p.dy, p.dz)
        s.set_coeffs(d["a"], d["bx"], d["by"], d["bz"], p.alpha, p.beta)
        s.set_bc(p.bc_type, d["bc_value"])
        phi = torch.zeros_like(d["rhs"])
        st = s.solve(d["rhs"], phi, rtol=1e-12, max_vcycles=30)
        out = (st, s.get_info(), phi)
        s.destroy()
        return out

    p0 = probs[0]
    hs = b.create_batch(len(probs), p0.nx, p0.ny, p0.nz, p0.dx, p0.dy, p0.dz)
    hs[0].set_option("batch_full_mb", full_mb)
    ds = [b.upload(p) for p in probs]
    for h, p, d in zip(hs, probs, ds):
        h.set_coeffs(d["a"], d["bx"], d["by"], d["bz"], p.alpha, p.beta)
        h.set_bc(p.bc_type, d["bc_value"])
    refs = [single(p, d) for p, d in zip(probs, ds)]
    assert len({r[1][0] for r in refs}) > 1          # the members do not all stop at the same cycle
    for rep in range(2):
        phis = [torch.zeros_like(d["rhs"]) for d in ds]
        sts = b.solve_batch(hs, [d["rhs"] for d in ds], phis, rtol=1e-12, max_vcycles=30)
        for p, h, st, phi, ref in zip(probs, hs, sts, phis, refs):
            cyc, rr, hist = h.get_info()
            assert st == ref[0] and cyc == ref[1][0] and list(hist) == list(ref[1][2]) and torch.equal(phi, ref[2]), (rep, p.name)
            if rep == 0:
                o = Oracle.from_problem(p)
                phi_o, st_o, cyc_o, rr_o, hist_o = o.solve(p.rhs, rtol=1e-12, max_vcycles=30)
                o.close()
                assert st == st_o and abs(cyc - cyc_o) <= 1 and rel(phi.cpu().numpy(), phi_o) <= PHI_TOL, p.name
    # one member gets other coefficients (its graph epoch moves: the group's graphs are recaptured); a member used alone
    p2 = inputs.random_problem(64, 32, 32, seed=8, bc_type=[D, N, N, D, N, N])
    d2 = b.upload(p2)
    hs[2].set_coeffs(d2["a"], d2["bx"], d2["by"], d2["bz"], p2.alpha, p2.beta)
    hs[2].set_bc(p2.bc_type, d2["bc_value"])
    probs[2], ds[2], refs[2] = p2, d2, single(p2, d2)
    phis = [torch.zeros_like(d["rhs"]) for d in ds]
    sts = b.solve_batch(hs, [d["rhs"] for d in ds], phis, rtol=1e-12, max_vcycles=30)
    for h, st, phi, ref in zip(hs, sts, phis, refs):
        assert st == ref[0] and h.get_info()[0] == ref[1][0] and torch.equal(phi, ref[2])
    phi = torch.zeros_like(ds[1]["rhs"])
    assert hs[1].solve(ds[1]["rhs"], phi, rtol=1e-12, max_vcycles=30) == refs[1][0] and torch.equal(phi, refs[1][2])
    assert all(h.pad_check() == 0 for h in hs)
    for h in hs:
        h.destroy()


def _torch_residual_relres(p, d, phi):
    """||btilde - A phi||_inf / ||btilde||_inf written with plain torch slicing from the definition C1 of DESIGN.md
    (face fluxes, two-point Dirichlet flux, Neumann data) -- no libvmg kernel involved.  3-D problems."""
    a, bx, by, bz, rhs = d["a"], d["bx"], d["by"], d["bz"], d["rhs"]
    hs = (p.dx, p.dy, p.dz)
    r = rhs.clone()
    if a is not None:
        r -= p.alpha * a * phi
    for axis, (b, h) in enumerate(zip((bx, by, bz), hs)):      # axis 0 = x is the LAST tensor dim (arrays are [k, j, i])
        dim = 2 - axis
        n = phi.shape[dim]
        w = p.beta / (h * h)
        bi = b.narrow(dim, 1, n - 1)                            # interior faces
        flux = w * bi * (phi.narrow(dim, 1, n - 1) - phi.narrow(dim, 0, n - 1))   # b (phi_hi - phi_lo) / h^2
        r.narrow(dim, 0, n - 1).add_(flux)                      # + for the low cell
        r.narrow(dim, 1, n - 1).sub_(flux)                      # - for the high cell
        for side, f in ((0, 2 * axis), (n - 1, 2 * axis + 1)):
            bf = b.select(dim, 0 if side == 0 else n)
            val = d["bc_value"][f]
            cell = r.select(dim, side)
            if p.bc_type[f] == D:
                g = 0.0 if val is None else val.reshape(bf.shape)
                cell.add_(2.0 * w * bf * (g - phi.select(dim, side)))
            elif val is not None:
                cell.add_(w * h * bf * val.reshape(bf.shape))
    # btilde = rhs + boundary data terms: the same expression with phi = 0
    if all(v is None for v in d["bc_value"]):
        nb = rhs.abs().max()
    else:
        nb = None
    return r.abs().max().item(), (nb.item() if nb is not None else None)


@pytest.mark.parametrize("make,rho", [(lambda: inputs.config3(128), 0.35), (lambda: _config5_full(), 0.9)],
                         ids=["config3_256x128x128", "config5_512^3"])
def test_full_size_residual_property_without_the_oracle(make, rho):
    """At sizes the oracle needs minutes for: the relative residual vmg_solve reports is the one an independent
    evaluation of the discrete operator gives (plain torch slicing on the GPU), and it contracts every cycle while
    above the rounding floor.  (Config 5 at 512^3 -- sigma = 2, 8 decades of b, diffusion dominated -- contracts by
    only ~0.76 per cycle asymptotically, in the oracle as well: DESIGN.md section 3; the bound for it is monotone decrease.)"""
    b = _binding()
    p = make()
    s, d = b.from_problem(p)
    phi = torch.zeros_like(d["rhs"])
    st = s.solve(d["rhs"], phi, rtol=p.rtol, max_vcycles=min(p.max_vcycles, 12) if p.rtol == 0 else p.max_vcycles)
    cyc, rr, hist = s.get_info()
    assert st in (0, 1) and cyc >= 8
    if all(v is None for v in d["bc_value"]):                  # homogeneous data: btilde = rhs
        r_abs, nb = _torch_residual_relres(p, d, phi)
        assert abs(r_abs / nb - rr) <= 1e-6 * rr + 1e-15, (r_abs / nb, rr)
    else:                                                       # inhomogeneous Dirichlet data: compare absolute residuals
        bt = s.step_fold_bc(d["rhs"])
        r_abs, _ = _torch_residual_relres(p, d, phi)
        assert abs(r_abs / bt.abs().max().item() - rr) <= 1e-6 * rr + 1e-15
    h = np.array(hist)
    live = h[1:] > 1e-11
    assert np.all(h[1:][live] < rho * h[:-1][live])
    s.destroy()


def test_config5_full_size_against_the_oracle_cycle_by_cycle():
    """BASELINE.json configs[4] (512^3, 134 M cells) against the oracle at FULL size, in the default launch configuration:
    six fixed V-cycles (rtol = 0) from the zero guess on both sides -- the iterates, not converged solutions (config 5
    contracts slowly) -- phi element by element and the residual history cycle by cycle.  Bounded so
    that the oracle's share stays under a minute on the GPU box's host cores."""
    b = _binding()
    p = _config5_full()
    ncyc = 6
    o = Oracle.from_problem(p)
    phi_o, st_o, cyc_o, rr_o, hist_o = o.solve(p.rhs, rtol=0.0, max_vcycles=ncyc)
    o.close()
    s, d = b.from_problem(p)
    phi_g = torch.zeros_like(d["rhs"])
    st_g = s.solve(d["rhs"], phi_g, rtol=0.0, max_vcycles=ncyc)
    cyc_g, rr_g, hist_g = s.get_info()
    s.destroy()
    print("config5 512^3 history oracle:", " ".join(f"{v:.6e}" for v in hist_o))
    print("config5 512^3 history gpu   :", " ".join(f"{v:.6e}" for v in hist_g))
    assert st_o == st_g == 1 and cyc_o == cyc_g == ncyc          # VMG_MAXCYCLES: fixed count
    hist_g = np.array(hist_g)
    assert np.all(np.abs(hist_g / hist_o - 1.0) < 1e-6), (hist_o, hist_g)
    assert np.all(hist_o[1:] < hist_o[:-1])                      # monotone; ~0.76 per cycle asymptotically
    err = rel(phi_g.cpu().numpy(), phi_o)
    print("config5 512^3 rel Linf(phi_gpu - phi_oracle) after", ncyc, "cycles:", err)
    assert err <= PHI_TOL, err
    _C5.clear()


@pytest.mark.parametrize("dims", [(40, 24, 16), (48, 40, 1), (72, 40, 24), (5, 3, 4)])
def test_trilinear_prolongation_matches_oracle(dims):
    """Option prolong = 1 (reading R9): the stand-alone kernel on every level, all boundary kinds (MIXED has Dirichlet and
    Neumann faces in every direction), 2-D and odd coarse sizes; then a whole V-cycle, which also runs the shared-memory
    tail's version."""
    b = _binding()
    p = inputs.random_problem(*dims, seed=21, bc_type=MIXED)
    o = Oracle.from_problem(p)
    s, d = b.from_problem(p)
    o.set_option("prolong", 1)
    s.set_option("prolong", 1)
    rng = np.random.default_rng(5)
    for lev in range(o.num_levels - 1):
        nx, ny, nz = o.level_dims(lev)
        cnx, cny, cnz = o.level_dims(lev + 1)
        phi, e = rng.standard_normal((nz, ny, nx)), rng.standard_normal((cnz, cny, cnx))
        got = s.step_prolong_correct(lev, dev(phi), dev(e)).cpu().numpy()
        assert rel(got, o.prolong_add(phi, e, lev)) <= STEP_TOL
    bt = o.fold_bc(p.rhs)
    phi0 = rng.standard_normal(p.rhs.shape)
    assert rel(s.step_vcycle(dev(phi0), dev(bt)).cpu().numpy(), o.vcycle(phi0, bt)) <= 1e-12
    s.destroy()


def test_symmetric_vcycle_matches_oracle():
    """Option symmetric = 1 (the PCG preconditioner): one V-cycle against the oracle's, per-colour path, blocked passes
    and the shared-memory tail."""
    b = _binding()
    p = inputs.random_problem(48, 24, 48, seed=3, bc_type=[D, D, N, N, N, D])
    o = Oracle.from_problem(p)
    o.set_option("symmetric", 1)
    bt = o.fold_bc(p.rhs)
    phi0 = np.random.default_rng(2).standard_normal(p.rhs.shape)
    ref = o.vcycle(phi0, bt)
    for opts in (dict(), dict(blocked=1, block_min_cells=0), dict(tail=0, graph=0)):
        s, d = b.from_problem(p)
        s.set_option("symmetric", 1)
        for k, v in opts.items():
            s.set_option(k, v)
        assert rel(s.step_vcycle(dev(phi0), dev(bt)).cpu().numpy(), ref) <= 1e-12, opts
        s.destroy()


@pytest.mark.parametrize("make", [lambda: inputs.config3(32), lambda: inputs.config4(32), lambda: inputs.config2(32),
                                  lambda: inputs.config1(64),
                                  lambda: inputs.random_problem(32, 32, 32, seed=3, bc_type=[D, N, N, N, N, N], ell=0.06, sigma=2.0,
                                                                a_scale=1.0, inhomogeneous=False)],
                         ids=["config3", "config4", "config2", "config1_2d", "contrast_where_vcycles_stall"])
def test_pcg_parity(make):
    """vmg_solve_pcg against ovmg_solve_pcg: same status, iteration counts within 1, phi within 1e-10
    after both reach the tolerance, histories alike while above the floor.  The last case is the one on which the plain
    V-cycle iteration stalls (tests/test_oracle_pins.py)."""
    b = _binding()
    p = make()
    rtol = 1e-10 if "random" in p.name else 1e-12
    o = Oracle.from_problem(p)
    phi_o, st_o, it_o, rr_o, hist_o = o.solve_pcg(p.rhs, rtol=rtol, max_iter=80)
    s, d = b.from_problem(p)
    phi = torch.zeros_like(d["rhs"])
    st = s.solve_pcg(d["rhs"], phi, rtol=rtol, max_iter=80)
    it, rr, hist = s.get_info()
    assert st == st_o == 0 and abs(it - it_o) <= 1 and rr <= rtol
    assert rel(phi.cpu().numpy(), phi_o) <= PHI_TOL
    m = min(len(hist), len(hist_o))
    live = hist_o[:m] > 1e-9
    assert np.all(np.abs(np.array(hist)[:m][live] / hist_o[:m][live] - 1.0) < 1e-2)
    # the handle still does plain V-cycle solves afterwards, and PCG again
    phi2 = torch.zeros_like(d["rhs"])
    s.solve(d["rhs"], phi2, rtol=1e-6, max_vcycles=60) if "random" not in p.name else None
    phi3 = torch.zeros_like(d["rhs"])
    assert s.solve_pcg(d["rhs"], phi3, rtol=rtol, max_iter=80) == 0 and torch.equal(phi3, phi)
    s.destroy()


@pytest.mark.parametrize("dims,spacing", [((96, 48, 80), (0.5, 0.6, 0.55)), ((512, 256, 1), (1.0, 1.0, 1.0)), ((36, 20, 12), (1.0, 1.2, 0.9)),
                                          ((130, 66, 34), (1.0, 1.0, 1.0))],
                         ids=["96x48x80_unequal_h", "512x256_2d", "36x20x12_odd_coarse", "130x66x34_single_coarsening"])
def test_more_shapes_parity(dims, spacing):
    """Unequal mesh widths, a large 2-D grid, hierarchies that stop at odd sizes (36x20x12 -> 9x5x3; 130x66x34 -> 65x33x17:
    two levels, 36 465 coarsest cells would exceed the bottom limit -> VMG_ERR_SIZE, checked instead)."""
    b = _binding()
    if dims == (130, 66, 34):
        with pytest.raises(b.VmgError) as e:
            b.Vmg(*dims, *spacing)
        assert e.value.code == -2
        return
    p = inputs.random_problem(*dims, seed=17, bc_type=[N, D, D, N, N, D], spacing=spacing)
    check_parity(p)


def _mask_for(p, seed=5):
    """Covered geometry of the paper's kind (electrodes / dielectric bodies inside the box): a ball, a slab that
    touches two domain faces, and a few isolated covered cells, so that coarse cells end up fully, partly and not covered."""
    nz, ny, nx = p.rhs.shape
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    mask = np.ones(p.rhs.shape, dtype=np.uint8)
    r = max(2.0, 0.22 * min(nx, ny, nz if nz > 1 else nx))
    mask[(i - 0.55 * nx) ** 2 + (j - 0.45 * ny) ** 2 + ((k - 0.5 * nz) ** 2 if nz > 1 else 0) < r * r] = 0
    mask[: max(1, nz // 3), : max(1, ny // 5), nx // 8: nx // 8 + 3] = 0
    rng = np.random.default_rng(seed)
    mask[rng.random(p.rhs.shape) < 0.003] = 0
    cval = np.where(mask == 0, 0.5 + 0.2 * rng.standard_normal(p.rhs.shape), 0.0)
    return mask, cval


@pytest.mark.parametrize("kind", [D, N], ids=["dirichlet_interface", "neumann_interface"])
@pytest.mark.parametrize("dims", [(40, 24, 16), (48, 40, 1), (64, 64, 32)])
def test_masked_solve_matches_oracle(dims, kind):
    """vmg_set_mask against ovmg_set_mask: folded right-hand side, V-cycle solve and PCG on a
    domain with covered cells, both interface kinds; covered cells come back exactly 0; removing the mask restores the
    unmasked solve bit for bit."""
    b = _binding()
    p = inputs.random_problem(*dims, seed=23, bc_type=[D, N, N, D, N, N])
    mask, cval = _mask_for(p)
    cv = cval if kind == D else None
    o = Oracle.from_problem(p)
    o.set_mask(mask, kind, cv)
    o.set_coeffs(p.a, p.bx, p.by, p.bz, p.alpha, p.beta)
    s, d = b.from_problem(p)
    phi_plain = torch.zeros_like(d["rhs"])
    s.solve(d["rhs"], phi_plain, rtol=1e-12, max_vcycles=60)
    s.set_mask(dev(mask), kind, None if cv is None else dev(cv))
    with pytest.raises(b.VmgError) as e:                       # the coefficients have to be set again
        s.solve(d["rhs"], torch.zeros_like(d["rhs"]))
    assert e.value.code == -3
    s.set_coeffs(d["a"], d["bx"], d["by"], d["bz"], p.alpha, p.beta)
    bt = s.step_fold_bc(d["rhs"])
    bt_o = o.fold_bc(p.rhs)
    assert np.abs(bt.cpu().numpy() - bt_o).max() <= 1e-13 * np.abs(bt_o).max()
    phi_o, st_o, cyc_o, rr_o, hist_o = o.solve(p.rhs, rtol=1e-12, max_vcycles=60)
    phi = torch.full_like(d["rhs"], 3.0)                       # a guess that is non-zero in covered cells
    phi0 = np.full(p.rhs.shape, 3.0)
    phi_o2, st_o2, cyc_o2, _, _ = o.solve(p.rhs, phi0, rtol=1e-12, max_vcycles=60)
    st = s.solve(d["rhs"], phi, rtol=1e-12, max_vcycles=60)
    cyc, rr, hist = s.get_info()
    assert st == st_o2 == 0 and abs(cyc - cyc_o2) <= 1 and rr <= 1e-12
    g = phi.cpu().numpy()
    assert np.all(g[mask == 0] == 0.0)
    assert rel(g, phi_o2) <= PHI_TOL
    phi = torch.zeros_like(d["rhs"])
    assert s.solve(d["rhs"], phi, rtol=1e-12, max_vcycles=60) == st_o
    cyc, rr, hist = s.get_info()
    assert abs(cyc - cyc_o) <= 1 and rel(phi.cpu().numpy(), phi_o) <= PHI_TOL
    m = min(len(hist), len(hist_o))
    live = hist_o[:m] > 1e-11
    assert np.all(np.abs(np.array(hist)[:m][live] / hist_o[:m][live] - 1.0) < 1e-3)
    phi_po, st_po, it_po, _, _ = o.solve_pcg(p.rhs, rtol=1e-12, max_iter=60)
    phi = torch.zeros_like(d["rhs"])
    assert s.solve_pcg(d["rhs"], phi, rtol=1e-12, max_iter=60) == st_po == 0
    it, rr, _ = s.get_info()
    assert abs(it - it_po) <= 1 and rel(phi.cpu().numpy(), phi_po) <= PHI_TOL
    assert np.all(phi.cpu().numpy()[mask == 0] == 0.0)
    s.set_mask(None)
    s.set_coeffs(d["a"], d["bx"], d["by"], d["bz"], p.alpha, p.beta)
    phi = torch.zeros_like(d["rhs"])
    s.solve(d["rhs"], phi, rtol=1e-12, max_vcycles=60)
    assert torch.equal(phi, phi_plain)
    s.destroy()
    o.close()


def test_masked_electrode_regularises_the_all_neumann_problem():
    """All-Neumann Poisson is singular (VMG_ERR_SINGULAR) until a covered block with a Dirichlet interface pins phi; with a
    zero-flux interface it stays singular; an all-valid Dirichlet mask changes nothing."""
    b = _binding()
    p = inputs.random_problem(32, 32, 16, seed=4, bc_type=[N] * 6, inhomogeneous=False)
    s, d = b.from_problem(p)
    s.set_coeffs(None, d["bx"], d["by"], d["bz"], 0.0, p.beta)
    phi = torch.zeros_like(d["rhs"])
    with pytest.raises(b.VmgError) as e:
        s.solve(d["rhs"], phi)
    assert e.value.code == -4
    mask = np.ones(p.rhs.shape, dtype=np.uint8)
    for kind, ok in ((D, False), (N, False)):                  # no covered cell: still singular
        s.set_mask(dev(mask), kind)
        s.set_coeffs(None, d["bx"], d["by"], d["bz"], 0.0, p.beta)
        with pytest.raises(b.VmgError) as e:
            s.solve(d["rhs"], phi)
        assert e.value.code == -4
    mask[6:10, 12:20, 12:20] = 0
    s.set_mask(dev(mask), N)
    s.set_coeffs(None, d["bx"], d["by"], d["bz"], 0.0, p.beta)
    with pytest.raises(b.VmgError) as e:
        s.solve(d["rhs"], phi)
    assert e.value.code == -4
    cval = np.where(mask == 0, 1.0, 0.0)
    s.set_mask(dev(mask), D, dev(cval))
    s.set_coeffs(None, d["bx"], d["by"], d["bz"], 0.0, p.beta)
    o = Oracle.from_problem(p)
    o.set_mask(mask, D, cval)
    o.set_coeffs(None, p.bx, p.by, p.bz, 0.0, p.beta)
    phi_o, st_o, cyc_o, _, _ = o.solve(p.rhs, rtol=1e-11, max_vcycles=80)
    st = s.solve(d["rhs"], phi, rtol=1e-11, max_vcycles=80)
    cyc, rr, _ = s.get_info()
    assert st == st_o == 0 and abs(cyc - cyc_o) <= 1 and rel(phi.cpu().numpy(), phi_o) <= PHI_TOL
    s.destroy()
    o.close()


@pytest.mark.parametrize("opts", [dict(prolong=1), dict(blocked=1, block_min_cells=0), dict(graph=0, tail=0), dict(snake=0, pdl=0, l2_persist=0),
                                  dict(nu1=2, nu2=1, bottom_sweeps=8)],
                         ids=["trilinear", "blocked", "no_graph_no_tail", "plain_schedule", "v21"])
def test_masked_solve_under_options(opts):
    """The mask lives in the stencil arrays, so every schedule / kernel variant has to solve the same masked problem."""
    b = _binding()
    p = inputs.random_problem(72, 40, 24, seed=31, bc_type=[N, D, D, N, D, N])
    mask, cval = _mask_for(p, seed=9)
    o = Oracle.from_problem(p)
    o.set_mask(mask, D, cval)
    o.set_coeffs(p.a, p.bx, p.by, p.bz, p.alpha, p.beta)
    s, d = b.from_problem(p)
    s.set_mask(dev(mask), D, dev(cval))
    s.set_coeffs(d["a"], d["bx"], d["by"], d["bz"], p.alpha, p.beta)
    for k, v in opts.items():
        if k in ("nu1", "nu2", "bottom_sweeps", "prolong"):
            o.set_option(k, v)
        s.set_option(k, v)
    phi_o, st_o, cyc_o, _, hist_o = o.solve(p.rhs, rtol=1e-12, max_vcycles=60)
    phi = torch.zeros_like(d["rhs"])
    st = s.solve(d["rhs"], phi, rtol=1e-12, max_vcycles=60)
    cyc, rr, hist = s.get_info()
    assert st == st_o == 0 and abs(cyc - cyc_o) <= 1
    assert rel(phi.cpu().numpy(), phi_o) <= PHI_TOL
    assert np.all(phi.cpu().numpy()[mask == 0] == 0.0)
    s.destroy()
    o.close()


def test_masked_full_size_parity():
    """256x128x128 (config 3's grid and coefficients) with an electrode ball and a dielectric-like slab covered: the launch
    configuration bench.py times, element by element against the oracle."""
    b = _binding()
    p = inputs.config3(128)
    mask, cval = _mask_for(p, seed=2)
    o = Oracle.from_problem(p)
    o.set_mask(mask, D, cval)
    o.set_coeffs(p.a, p.bx, p.by, p.bz, p.alpha, p.beta)
    s, d = b.from_problem(p)
    s.set_mask(dev(mask), D, dev(cval))
    s.set_coeffs(d["a"], d["bx"], d["by"], d["bz"], p.alpha, p.beta)
    phi_o, st_o, cyc_o, _, _ = o.solve(p.rhs, rtol=1e-11, max_vcycles=40)
    phi = torch.zeros_like(d["rhs"])
    st = s.solve(d["rhs"], phi, rtol=1e-11, max_vcycles=40)
    cyc, rr, _ = s.get_info()
    assert st == st_o == 0 and abs(cyc - cyc_o) <= 1, (st, st_o, cyc, cyc_o)
    assert rel(phi.cpu().numpy(), phi_o) <= PHI_TOL
    s.destroy()
    o.close()


@pytest.mark.parametrize("make", [lambda: inputs.config3(32), lambda: inputs.config1(64),
                                  lambda: inputs.random_problem(40, 24, 16, seed=8, bc_type=[N, D, D, N, N, D], inhomogeneous=True),
                                  lambda: inputs.random_problem(36, 20, 12, seed=9, bc_type=[D, D, N, N, N, N], spacing=(1.0, 1.2, 0.9)),
                                  lambda: inputs.config3(128)],
                         ids=["config3_64x32x32", "config1_2d", "helmholtz_40x24x16", "unequal_h_odd_coarse", "config3_full"])
@pytest.mark.parametrize("opts", [dict(), dict(prolong=1, symmetric=1)], ids=["default", "trilinear_symmetric"])
def test_constant_weight_kernels_equal_the_general_ones_bitwise(make, opts):
    """b == NULL (b = 1: the Poisson equation PAPER.md:54 Eq. 3, Helmholtz with a variable a) selects kernels that form the six
    face weights from beta/h^2 and the cell's position instead of loading them.  Same numbers, same order: phi and the residual
    history equal, bit for bit, those of the general kernels on explicit arrays of ones and those of the general kernels
    with b == NULL (option const_weights=0); PCG likewise."""
    b = _binding()
    p = make()
    d = b.upload(p)
    nz1 = p.nz + 1 if p.nz > 1 else 1
    ones = [torch.ones(sh, dtype=torch.float64, device="cuda") for sh in ((p.nz, p.ny, p.nx + 1), (p.nz, p.ny + 1, p.nx), (nz1, p.ny, p.nx))]
    out = []
    for variant in ("const", "ones", "null_general"):
        s = b.Vmg(p.nx, p.ny, p.nz, p.dx, p.dy, p.dz)
        for k, v in opts.items():
            s.set_option(k, v)
        if variant == "null_general":
            s.set_option("const_weights", 0)
        if variant == "ones":
            s.set_coeffs(d["a"], ones[0], ones[1], ones[2] if p.nz > 1 else None, p.alpha, p.beta)
        else:
            s.set_coeffs(d["a"], None, None, None, p.alpha, p.beta)
        s.set_bc(p.bc_type, d["bc_value"])
        phi = torch.zeros_like(d["rhs"])
        st = s.solve(d["rhs"], phi, rtol=1e-12, max_vcycles=12)
        info = s.get_info()
        phi2 = torch.zeros_like(d["rhs"])
        st2 = s.solve_pcg(d["rhs"], phi2, rtol=1e-12, max_iter=12)
        out.append((st, info, phi, st2, s.get_info(), phi2))
        s.destroy()
    for o in out[1:]:
        assert o[0] == out[0][0] and o[1] == out[0][1] and torch.equal(o[2], out[0][2])
        assert o[3] == out[0][3] and o[4] == out[0][4] and torch.equal(o[5], out[0][5])


def test_alternating_equation_kinds_on_one_handle_keeps_results():
    """One handle used like a time step does (bench.py timestep_leg): constant-weight and general equations in turn, a changed
    beta on the constant-weight one (its kernels take beta/h^2 by value and the V-cycle is a replayed graph).  Every solve
    must equal the solve of a fresh handle bit for bit."""
    b = _binding()
    p = inputs.random_problem(40, 24, 16, seed=14, bc_type=[D, N, N, D, N, N])
    d = b.upload(p)
    # (const b1, general b2, const b2) with b1 != b2: the general call overwrites the levels' beta/h^2, which must not hide
    # from the following constant-weight call that its captured graph still carries b1
    kinds = [("const", 1.0), ("general", 1.0), ("const", 1.0), ("const", 2.5), ("general", 0.5), ("const", 2.5), ("const", 1.0),
             ("general", 2.5), ("const", 2.5), ("general", 4.0), ("const", 4.0), ("const", 1.0)]

    def run(s, kind, beta, pcg):
        if kind == "const":
            s.set_coeffs(d["a"], None, None, None, p.alpha, beta)
        else:
            s.set_coeffs(d["a"], d["bx"], d["by"], d["bz"], p.alpha, beta)
        phi = torch.zeros_like(d["rhs"])
        (s.solve_pcg if pcg else s.solve)(d["rhs"], phi, 1e-12, 12)
        return phi, s.get_info()

    s = b.Vmg(p.nx, p.ny, p.nz, p.dx, p.dy, p.dz)
    s.set_bc(p.bc_type, d["bc_value"])
    for pcg in (False, True):
        for kind, beta in kinds:
            got = run(s, kind, beta, pcg)
            f = b.Vmg(p.nx, p.ny, p.nz, p.dx, p.dy, p.dz)
            f.set_bc(p.bc_type, d["bc_value"])
            want = run(f, kind, beta, pcg)
            f.destroy()
            assert got[1] == want[1] and torch.equal(got[0], want[0]), (kind, beta, pcg)
    s.destroy()


def test_time_step_sequence_matches_the_oracle_solve_by_solve():
    """SURVEY.md 8(f) N3 (Eq. 9-10): the 20 solves of bench.py's time step (Poisson with
    b == NULL, 15 species that differ in beta, energy, three photoionisation Helmholtz shifts) on ONE handle at 64x32x32,
    two time steps with right-hand sides growing 1 % per step and every solve warm-started from its field of the
    previous step; each phi against the oracle run through the same sequence with the same warm starts."""
    b = _binding()
    p3, p4 = inputs.config3(32), inputs.config4(32)
    d3, d4 = b.upload(p3), b.upload(p4)
    shape = p3.rhs.shape
    ones = np.ones(shape)
    photo_rhs = np.random.default_rng(1234).standard_normal(shape)
    betas = np.logspace(-1.0, 1.0, 15)
    # (name, a, use b arrays?, alpha, beta, problem whose BCs apply, rhs)
    eqs = [("poisson", p3.a, False, p3.alpha, p3.beta, p3, p3.rhs)]
    eqs += [("species", p4.a, True, 1.0, float(bk), p4, p4.rhs) for bk in betas]
    eqs += [("energy", p4.a, True, 1.0, 1.0, p4, p4.rhs)]
    eqs += [("photo", ones, False, l2, 1.0, p4, photo_rhs) for l2 in (1.0e2, 1.0e3, 1.0e4)]
    s = b.Vmg(p3.nx, p3.ny, p3.nz, p3.dx, p3.dy, p3.dz)
    o = Oracle(p3.nx, p3.ny, p3.nz, p3.dx, p3.dy, p3.dz)
    f_g = [torch.zeros_like(d3["rhs"]) for _ in eqs]
    f_o = [np.zeros(shape) for _ in eqs]
    rtol = 1e-10
    worst = 0.0
    for step in range(2):
        scale = 1.0 + 0.01 * step
        for i, (name, a, with_b, alpha, beta, pb, rhs) in enumerate(eqs):
            db = d3 if pb is p3 else d4
            a_g = dev(a)
            if with_b:
                s.set_coeffs(a_g, d4["bx"], d4["by"], d4["bz"], alpha, beta)
                o.set_coeffs(a, p4.bx, p4.by, p4.bz, alpha, beta)
            else:
                s.set_coeffs(a_g, None, None, None, alpha, beta)
                o.set_coeffs(a, None, None, None, alpha, beta)
            s.set_bc(pb.bc_type, db["bc_value"])
            o.set_bc(pb.bc_type, pb.bc_value)
            st_g = s.solve(dev(rhs * scale), f_g[i], rtol=rtol, max_vcycles=50)
            cyc_g = s.get_info()[0]
            phi_o, st_o, cyc_o, rr_o, _ = o.solve(rhs * scale, phi0=f_o[i], rtol=rtol, max_vcycles=50)
            f_o[i] = phi_o
            assert st_g == 0 and st_o == 0, (step, name, st_g, st_o)
            assert abs(cyc_g - cyc_o) <= 1, (step, name, cyc_g, cyc_o)
            # the two sides run the same iteration from warm starts that differ by rounding only: the iterates agree to
            # the whole-solve bar when they stop at the same cycle; one cycle apart they differ by what a cycle at
            # relres ~ 1e-10 still changes
            err = rel(f_g[i].cpu().numpy(), phi_o)
            worst = max(worst, err)
            assert err <= (PHI_TOL if cyc_g == cyc_o else 1e-8), (step, name, err, cyc_g, cyc_o)
    print("time-step sequence: worst rel Linf(phi_gpu - phi_oracle) over 40 solves:", worst)
    s.destroy()
    o.close()


@pytest.mark.parametrize("kind", [D, N], ids=["dirichlet_interface", "neumann_interface"])
@pytest.mark.parametrize("dims", [(40, 24, 16), (48, 40, 1), (64, 64, 32), (256, 128, 32)])
def test_masked_constant_weight_kernels_equal_the_general_ones_bitwise(dims, kind):
    """b == NULL with a mask (the Poisson equation around electrodes): level 0 runs kernels that take a
    face weight to be beta/h^2 when the cells on both sides are valid and 0 otherwise, read from the byte mask instead of
    three weight arrays.  Bitwise the general kernels (const_weights=0) for V-cycles and PCG, and the oracle's solution."""
    b = _binding()
    p = inputs.random_problem(*dims, seed=27, bc_type=[D, N, N, D, N, N])
    mask, cval = _mask_for(p, seed=3)
    cv = cval if kind == D else None
    d = b.upload(p)
    out = []
    for cwopt in (1, 0):
        s = b.Vmg(p.nx, p.ny, p.nz, p.dx, p.dy, p.dz)
        s.set_option("const_weights", cwopt)
        s.set_mask(dev(mask), kind, None if cv is None else dev(cv))
        s.set_coeffs(d["a"], None, None, None, p.alpha, p.beta)
        s.set_bc(p.bc_type, d["bc_value"])
        phi = torch.full_like(d["rhs"], 0.5)
        st = s.solve(d["rhs"], phi, rtol=1e-12, max_vcycles=40)
        info = s.get_info()
        phi2 = torch.zeros_like(d["rhs"])
        st2 = s.solve_pcg(d["rhs"], phi2, rtol=1e-12, max_iter=40)
        out.append((st, info, phi, st2, s.get_info(), phi2))
        s.destroy()
    assert out[0][0] == out[1][0] == 0 and out[0][1] == out[1][1] and torch.equal(out[0][2], out[1][2])
    assert out[0][3] == out[1][3] == 0 and out[0][4] == out[1][4] and torch.equal(out[0][5], out[1][5])
    if p.nx * p.ny * p.nz <= 200000:
        o = Oracle.from_problem(p)
        o.set_mask(mask, kind, cv)
        o.set_coeffs(p.a, None, None, None, p.alpha, p.beta)
        phi_o, st_o, cyc_o, _, _ = o.solve(p.rhs, np.full(p.rhs.shape, 0.5), rtol=1e-12, max_vcycles=40)
        assert st_o == 0 and abs(cyc_o - out[0][1][0]) <= 1 and rel(out[0][2].cpu().numpy(), phi_o) <= PHI_TOL
        o.close()


def test_staggered_batch_at_full_size_is_bitwise_the_single_solves():
    """vmg_solve_batch at 256x128x128, where the staggered schedule really overlaps one handle's coarse levels with another's
    fine level (three handles: config 3, config 4, config 3 with b == NULL): bit for bit the single solves."""
    b = _binding()
    probs = [inputs.config3(128), inputs.config4(128), inputs.config3(128)]
    streams = [torch.cuda.Stream() for _ in probs]
    solvers, data = [], []
    for n, (p, stream) in enumerate(zip(probs, streams)):
        s, d = b.from_problem(p, stream=stream)
        if n == 2:
            s.set_coeffs(d["a"], None, None, None, p.alpha, p.beta)
        solvers.append(s); data.append(d)
    torch.cuda.synchronize()
    single = []
    for s, d, p, stream in zip(solvers, data, probs, streams):
        phi = torch.zeros_like(d["rhs"])
        with torch.cuda.stream(stream):
            st = s.solve(d["rhs"], phi, rtol=p.rtol, max_vcycles=p.max_vcycles)
        single.append((st, s.get_info(), phi))
    for _ in range(2):
        phis = [torch.zeros_like(d["rhs"]) for d in data]
        sts = b.solve_batch(solvers, [d["rhs"] for d in data], phis, rtol=probs[0].rtol, max_vcycles=probs[0].max_vcycles)
        for s, st, phi, ref in zip(solvers, sts, phis, single):
            assert st == ref[0] and s.get_info() == ref[1] and torch.equal(phi, ref[2])
    assert torch.equal(single[0][2], single[2][2])   # constant-weight kernels = arrays of ones
    for s in solvers:
        s.destroy()


def test_changing_the_mask_on_a_handle_equals_fresh_handles():
    """vmg_set_mask twice with different geometry and kind, then removed, with and without explicit b: every solve equals the
    solve of a fresh handle bit for bit (the handle re-allocates the mask arrays and drops its captured graphs)."""
    b = _binding()
    p = inputs.random_problem(40, 24, 16, seed=19, bc_type=[D, N, N, D, N, N])
    d = b.upload(p)
    m1, c1 = _mask_for(p, seed=1)
    m2 = np.ones(p.rhs.shape, dtype=np.uint8)
    m2[4:9, 5:15, 10:30] = 0
    steps = [(m1, D, c1, True), (m2, N, None, True), (m2, D, None, False), (None, D, None, False), (m1, N, None, True), (None, D, None, True)]

    def run(s, mask, kind, cval, explicit_b):
        s.set_mask(None if mask is None else dev(mask), kind, None if cval is None else dev(cval))
        if explicit_b:
            s.set_coeffs(d["a"], d["bx"], d["by"], d["bz"], p.alpha, p.beta)
        else:
            s.set_coeffs(d["a"], None, None, None, p.alpha, p.beta)
        phi = torch.zeros_like(d["rhs"])
        st = s.solve(d["rhs"], phi, rtol=1e-12, max_vcycles=60)
        return st, s.get_info(), phi

    s = b.Vmg(p.nx, p.ny, p.nz, p.dx, p.dy, p.dz)
    s.set_bc(p.bc_type, d["bc_value"])
    for step in steps:
        got = run(s, *step)
        f = b.Vmg(p.nx, p.ny, p.nz, p.dx, p.dy, p.dz)
        f.set_bc(p.bc_type, d["bc_value"])
        want = run(f, *step)
        f.destroy()
        assert got[0] == want[0] == 0 and got[1] == want[1] and torch.equal(got[2], want[2])
    s.destroy()


def test_red_only_restriction_after_presmoothing_is_the_full_restriction_to_rounding():
    """Option restrict_red_cells (reading R12 applied to the transfer): after a black half-sweep the black children's residuals
    are their own rounding error, so restricting the red children only changes the coarse right-hand side by rounding: same
    cycle counts, histories equal to rounding, phi within 1e-13 -- and the oracle (which restricts all eight) within the bar."""
    b = _binding()
    p = inputs.config4(32)
    out = {}
    for thresh in (0.0, 2.0 ** 40):          # every level launched as a kernel of its own / no level
        s, d = b.from_problem(p)
        s.set_option("restrict_red_cells", thresh)
        s.set_option("tail", 0)              # no single-CTA tail: every down-stroke goes through residual_restrict_kernel
        phi = torch.zeros_like(d["rhs"])
        assert s.solve(d["rhs"], phi, rtol=p.rtol, max_vcycles=p.max_vcycles) == 0
        out[thresh] = (phi.cpu().numpy(), s.get_info())
        s.destroy()
    (phi_r, info_r), (phi_a, info_a) = out[0.0], out[2.0 ** 40]
    assert info_r[0] == info_a[0]
    assert not np.array_equal(phi_r, phi_a)                      # the option did take effect
    assert rel(phi_r, phi_a) <= 1e-13
    for x, y in zip(info_r[2], info_a[2]):
        assert abs(x - y) <= 1e-9 * y + 2e-15
    phi_o, st_o, cyc_o, rr_o, _ = Oracle.from_problem(p).solve(p.rhs, rtol=p.rtol, max_vcycles=p.max_vcycles)
    assert cyc_o == info_r[0] and rel(phi_r, phi_o) <= PHI_TOL


@pytest.mark.parametrize("dims", [(64, 32, 32), (48, 40, 1), (40, 24, 16)])
def test_bottom_solve_as_a_matrix_is_the_sweeps_to_rounding(dims):
    """Option bottom_matrix (default on): the single-CTA tail applies the nbottom sweeps from zero as the matrix of that linear
    map (built once per coefficient change by running the sweeps on the unit vectors).  Same map, another rounding order:
    cycle counts equal, histories and phi equal to rounding -- against the sweeps and against the oracle (which sweeps)."""
    b = _binding()
    p = inputs.random_problem(*dims, seed=17, bc_type=MIXED, sigma=1.5)
    out = {}
    for bm in (1, 0):
        s, d = b.from_problem(p)
        s.set_option("bottom_matrix", bm)
        phi = torch.zeros_like(d["rhs"])
        assert s.solve(d["rhs"], phi, rtol=1e-12, max_vcycles=50) == 0
        out[bm] = (phi.cpu().numpy(), s.get_info())
        # new coefficients on the same handle: the matrix is rebuilt
        q = inputs.random_problem(*dims, seed=18, bc_type=MIXED, sigma=1.5)
        dq = b.upload(q)
        s.set_coeffs(dq["a"], dq["bx"], dq["by"], dq["bz"], q.alpha, q.beta)
        s.set_bc(q.bc_type, dq["bc_value"])
        phi2 = torch.zeros_like(dq["rhs"])
        assert s.solve(dq["rhs"], phi2, rtol=1e-12, max_vcycles=50) == 0
        out[(bm, 2)] = (phi2.cpu().numpy(), s.get_info(), q)
        s.destroy()
    for key in (1, (1, 2)):
        ref = out[0] if key == 1 else out[(0, 2)]
        got = out[key]
        assert got[1][0] == ref[1][0] and rel(got[0], ref[0]) <= 1e-12
        for x, y in zip(got[1][2], ref[1][2]):
            assert abs(x - y) <= 1e-9 * y + 2e-15
    phi_o, st_o, cyc_o, rr_o, _ = Oracle.from_problem(p).solve(p.rhs, rtol=1e-12, max_vcycles=50)
    assert cyc_o == out[1][1][0] and rel(out[1][0], phi_o) <= PHI_TOL
    q = out[(1, 2)][2]
    phi_o, st_o, cyc_o, rr_o, _ = Oracle.from_problem(q).solve(q.rhs, rtol=1e-12, max_vcycles=50)
    assert cyc_o == out[(1, 2)][1][0] and rel(out[(1, 2)][0], phi_o) <= PHI_TOL
