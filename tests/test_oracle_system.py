"""System-level pins of the oracle (O2-O6 together): exact Riemann solutions, invariants the
discretisation must satisfy, convergence order, long-double agreement.  CPU only."""
import os

import numpy as np
import pytest

import mfc_workloads as W
from oracle import oracle as O
from exact_riemann import Side, sample, solve_star, wave_speeds
from parity_norm import rel_err

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def run_to_time(case, t_end, recon=O.RECON_WENO5, cfl=0.5):
    orc = O.Oracle(case, recon)
    q = W.initial_state(case)
    t, steps = 0.0, 0
    while t < t_end * (1 - 1e-14):
        dt = min(orc.cfl_dt(q, cfl), t_end - t)
        orc.rk3_step(q, dt)
        assert orc.bad == 0
        t += dt
        steps += 1
    return q, steps


# ------------------------------------------------------------------ the test-side exact solver itself
def test_exact_solver_against_published_sod_star_state():
    vals = {}
    for line in open(os.path.join(GOLDEN, "sod_star_state.txt")):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            vals[k] = float(v)
    L, R = Side(1.0, 0.0, 1.0, 1.4, 0.0), Side(0.125, 0.0, 0.1, 1.4, 0.0)
    ps, us = solve_star(L, R)
    assert ps == pytest.approx(vals["p_star"], abs=6e-6)
    assert us == pytest.approx(vals["u_star"], abs=6e-6)
    assert L.rho_star(ps) == pytest.approx(vals["rho_star_L"], abs=6e-6)
    assert R.rho_star(ps) == pytest.approx(vals["rho_star_R"], abs=6e-6)


# ------------------------------------------------------------------ config 1: Sod (BASELINE.json configs[0])
def _sod_errors(n, recon):
    case = W.config(1, n=n)
    q, steps = run_to_time(case, 0.2, recon)
    w = O.Oracle(case).prim_from_cons(q)
    x = (np.arange(n) + 0.5) / n
    rho, u, p, _ = sample(Side(1.0, 0.0, 1.0, 1.4, 0.0), Side(0.125, 0.0, 0.1, 1.4, 0.0), (x - 0.5) / 0.2)
    return w, x, np.abs(w[0, 0, 0] - rho).mean(), rho, u, p, steps


def test_sod_weno5_hllc_converges_to_exact_solution():
    errs = []
    for n in (250, 500, 1000):
        w, x, e, rho, u, p, steps = _sod_errors(n, O.RECON_WENO5)
        errs.append(e)
        assert np.array_equal(w[3], np.ones_like(w[3])) or np.abs(w[3] - 1).max() < 1e-13   # single fluid: alpha stays 1 (A7)
    rates = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert errs[-1] < 1.5e-3 and (rates > 0.75).all(), (errs, rates)
    # n = 1000 (the configuration itself): plateau values and wave positions
    L, R = Side(1.0, 0.0, 1.0, 1.4, 0.0), Side(0.125, 0.0, 0.1, 1.4, 0.0)
    ws = wave_speeds(L, R)
    ps, us = ws["p_star"], ws["contact"]
    dx = 1.0 / 1000
    xc, xs = 0.5 + 0.2 * us, 0.5 + 0.2 * ws["right_shock"]
    mid = (x > xc + 0.01) & (x < xs - 0.01)           # between contact and shock
    assert np.abs(w[2, 0, 0][mid] - ps).max() < 2e-3 * ps
    assert np.abs(w[1, 0, 0][mid] - us).max() < 2e-3 * us
    assert np.abs(w[0, 0, 0][mid] - R.rho_star(ps)).max() < 2e-3
    # shock position: where density crosses the mean of its two sides, within 2 cells
    r = w[0, 0, 0]
    lvl = 0.5 * (R.rho_star(ps) + 0.125)
    i_sh = np.where((r[:-1] >= lvl) & (r[1:] < lvl) & (x[:-1] > xc + 0.01))[0]
    assert len(i_sh) == 1 and abs(x[i_sh[0]] + 0.5 * dx - xs) <= 2 * dx
    lvl = 0.5 * (L.rho_star(ps) + R.rho_star(ps))
    i_c = np.where((r[:-1] >= lvl) & (r[1:] < lvl) & (np.abs(x[:-1] - xc) < 0.03))[0]
    assert len(i_c) == 1 and abs(x[i_c[0]] + 0.5 * dx - xc) <= 2 * dx
    # rarefaction head: leftmost cell that moved by more than 1e-3
    i_h = np.argmax(np.abs(r - 1.0) > 1e-3)
    assert abs(x[i_h] - (0.5 + 0.2 * ws["left_head"])) <= 8 * dx
    assert 850 <= steps <= 950     # "~880 steps" at CFL 0.5 (A9)


def test_sod_first_order_hllc_converges():
    # piecewise-constant reconstruction isolates the Riemann solver
    errs = [_sod_errors(n, O.RECON_PC)[2] for n in (250, 500, 1000)]
    rates = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert (rates > 0.55).all() and errs[-1] < 6e-3, (errs, rates)


# ------------------------------------------------------------------ config 2: water/air tube
def test_water_air_tube_converges_to_exact_two_fluid_solution():
    L, R = Side(1000.0, 0.0, 1.0e9, 4.4, 6.0e8), Side(1.0, 0.0, 1.0e5, 1.4, 0.0)
    ws = wave_speeds(L, R)
    t_end = 1.0e-4
    errs = []
    for n in (500, 1000, 2000):
        case = W.config(2, n=n)
        q, steps = run_to_time(case, t_end)
        w = O.Oracle(case).prim_from_cons(q)
        x = (np.arange(n) + 0.5) / n
        rho, u, p, left = sample(L, R, (x - 0.5) / t_end)
        rho_num = w[0, 0, 0] + w[1, 0, 0]
        errs.append((np.abs(rho_num - rho).mean() / 1000.0, np.abs(w[2, 0, 0] - u).mean() / ws["contact"],
                     np.abs(w[3, 0, 0] - p).mean() / 1e9))
        assert np.abs(w[4] + w[5] - 1).max() < 1e-9   # each alpha_i is advected with its own nonlinear weights
        assert w[4].min() >= 1e-6 / (1 + 2e-6) and w[5].min() >= 1e-6 / (1 + 2e-6)
    errs = np.array(errs)
    rates = np.log2(errs[:-1] / errs[1:])
    assert (rates > 0.6).all(), (errs, rates)
    assert (errs[-1] < [2e-3, 1.5e-2, 2e-3]).all(), errs
    # plateau between the rarefaction tail and the contact: star pressure and velocity
    xt, xc = 0.5 + t_end * ws["left_tail"], 0.5 + t_end * ws["contact"]
    mid = (x > xt + 0.03) & (x < xc - 0.03)
    assert mid.sum() > 200
    assert np.abs(w[3, 0, 0][mid] - ws["p_star"]).max() < 1e-4 * 1.0e9     # p* = 4.8e5 Pa between states at 1e9 and 1e5
    assert np.abs(w[2, 0, 0][mid] - ws["contact"]).max() < 1e-3 * ws["contact"]
    # contact position from the volume fraction
    i_c = np.argmin(np.abs(w[4, 0, 0] - 0.5))
    assert abs(x[i_c] - xc) <= 3.0 / n


# ------------------------------------------------------------------ invariants
@pytest.mark.parametrize("ndim,nfluids,bc", [(1, 1, W.BC_EXTRAP), (2, 2, W.BC_PERIODIC), (3, 2, W.BC_EXTRAP), (3, 3, W.BC_PERIODIC)])
def test_uniform_state_has_exactly_zero_rhs(ndim, nfluids, bc):
    n = 7
    nn = tuple(n if d < ndim else 1 for d in range(3))
    case = W.Case("u", ndim, nn, (0.1, 0.37, 0.013), nfluids, (1.4, 4.4, 1.67)[:nfluids], (0.0, 6e8, 0.0)[:nfluids], (bc,) * 3, (bc,) * 3)
    sh = case.shape[1:]
    a = np.array([0.2, 0.5, 0.3])[:nfluids]; a = a / a.sum()
    q = W.cons_from_prim(case, [np.full(sh, a[i] * (1.0, 1000.0, 0.138)[i]) for i in range(nfluids)],
                         [np.full(sh, v) for v in (31.0, -7.0, 113.0)[:ndim]], 1.2345e5, [np.full(sh, x) for x in a])
    r = O.Oracle(case).rhs(q)
    assert np.array_equal(r, np.zeros_like(r))


def _kahan_sum(a):
    import math
    return math.fsum(a.ravel().tolist())


@pytest.mark.parametrize("form", ["difference", "textbook"])
@pytest.mark.parametrize("idx,n", [(4, 12), (3, 16)])
def test_conservation_on_periodic_domain(idx, n, form):
    case = W.config(idx, n=n)
    case = W.replace(case, bc_lo=(W.BC_PERIODIC,) * 3, bc_hi=(W.BC_PERIODIC,) * 3)
    q = W.initial_state(case)
    orc = O.Oracle(case, form=form)
    r = orc.rhs(q)
    N, D = case.nfluids, case.ndim
    for v in range(N + D + 1):          # partial densities, momenta, energy (alpha is not conserved)
        assert abs(_kahan_sum(r[v])) <= 1e-13 * np.abs(r[v]).sum() + 1e-300, v
    # totals over RK3 steps (clamp never fires here: checked)
    tot0 = [_kahan_sum(q[v]) for v in range(N + D + 1)]
    scale = [max(np.abs(q[v]).sum(), 1e-300) for v in range(N + D + 1)]
    case_nc = W.replace(case, clamp=False)
    q2 = q.copy()
    dt = orc.cfl_dt(q, 0.5)
    for _ in range(20):
        orc.rk3_step(q, dt)
        O.Oracle(case_nc, form=form).rk3_step(q2, dt)
    assert np.array_equal(q, q2)        # the clamp was a bit-exact no-op
    for v in range(N + D + 1):
        # momentum totals are ~0 by symmetry of the sum; scale with sum |q_v|
        assert abs(_kahan_sum(q[v]) - tot0[v]) <= 2e-13 * max(scale[v], np.abs(q[v]).sum()), v


@pytest.mark.parametrize("form", ["difference", "textbook"])
@pytest.mark.parametrize("fluids,tol", [("gas_gas", 1e-12), ("water_air", 1e-9)])
def test_interface_equilibrium_pressure_velocity(fluids, tol, form):
    # uniform u0, p0 across an advected tanh interface stays uniform (the reason primitives are reconstructed)
    n = 64
    if fluids == "gas_gas":
        gam, pinf, rho0, p0, u0 = (1.4, 1.67), (0.0, 0.0), (1.0, 0.138), 1.0, 0.7
    else:
        gam, pinf, rho0, p0, u0 = (4.4, 1.4), (6.0e8, 0.0), (1000.0, 1.0), 1.0e5, 100.0
    case = W.Case("ie", 2, (n, n, 1), (1.0 / n, 1.0 / n, 1.0), 2, gam, pinf, (W.BC_PERIODIC,) * 3, (W.BC_PERIODIC,) * 3, clamp=False)
    # (clamp off: the A10 epilogue edits alpha_i without touching E, so wherever it fires it perturbs p by
    #  O(floor); the equilibrium is a property of the discretisation a1-a6 proper)
    X, Y, _ = W.centres(case)
    r = np.sqrt((X - 0.5) ** 2 + (Y - 0.5) ** 2)
    a0 = np.clip(0.5 * (1 - np.tanh((r - 0.25) / (2.0 / n))), 1e-6, 1 - 1e-6) * np.ones(case.shape[1:])
    q = W.cons_from_prim(case, [a0 * rho0[0], (1 - a0) * rho0[1]], [u0, -0.5 * u0], p0, [a0, 1 - a0])
    orc = O.Oracle(case, form=form)
    dt = orc.cfl_dt(q, 0.5)
    for _ in range(100):
        orc.rk3_step(q, dt)
    w = orc.prim_from_cons(q)
    assert np.abs(w[4] / p0 - 1).max() <= tol
    assert np.abs(w[2] / u0 - 1).max() <= tol and np.abs(w[3] / (-0.5 * u0) - 1).max() <= tol
    assert np.abs(w[5] - a0).max() > 0.1      # ... while the interface really moved


def test_single_fluid_alpha_stays_one_through_shocks():
    # pins A7: with u_f = S* (the other plausible reading) alpha departs from 1 at O(1e-2) in compressions
    case = W.config(1, n=200)
    q, _ = run_to_time(case, 0.2)
    assert np.abs(q[3] - 1.0).max() <= 1e-13


def test_rhs_truncation_error_is_fifth_order_on_smooth_advection():
    # density wave advected by a uniform flow, single fluid, periodic: d(rho)/dt cell-averaged exactly is
    # -u (rho(x_{i+1/2}) - rho(x_{i-1/2}))/dx.  Brute-force refinement.
    errs = []
    for n in (16, 32, 64, 128):
        case = W.Case("adv", 1, (n, 1, 1), (1.0 / n, 1.0, 1.0), 1, (1.4,), (0.0,), (W.BC_PERIODIC,) * 3, (W.BC_PERIODIC,) * 3, weno_eps=1e-6)
        xe = np.arange(n + 1) / n
        avg = 2.0 + (np.cos(2 * np.pi * xe[:-1]) - np.cos(2 * np.pi * xe[1:])) / (2 * np.pi / n)
        u0, p0 = 1.0, 1.0
        q = W.cons_from_prim(case, [avg.reshape(1, 1, n)], [u0], p0, [np.ones((1, 1, n))])
        r = O.Oracle(case).rhs(q)
        exact = -u0 * (np.sin(2 * np.pi * xe[1:]) - np.sin(2 * np.pi * xe[:-1])) * n
        errs.append(np.abs(r[0, 0, 0] - exact).max())
        assert np.abs(r[3]).max() == 0.0
    rates = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert rates[-1] > 4.8 and rates[-2] > 4.5, (errs, rates)


def test_symmetry_of_shock_bubble_about_midline():
    case = W.config(3, n=48)
    q = W.initial_state(case)
    orc = O.Oracle(case)
    dt = orc.cfl_dt(q, 0.5)
    for _ in range(10):
        orc.rk3_step(q, dt)
    for v in range(case.neq):
        sgn = -1.0 if v == case.nfluids + 1 else 1.0
        assert np.abs(q[v, 0] - sgn * q[v, 0, ::-1]).max() <= 1e-11 * max(np.abs(q[v]).max(), 1e-300), v


@pytest.mark.parametrize("idx,n", [(2, 200), (3, 24), (4, 10), (5, 10)])
def test_fp64_oracle_agrees_with_long_double_oracle(idx, n):
    case = W.config(idx, n=n)
    q = W.initial_state(case)
    orc = O.Oracle(case)
    r, rl = orc.rhs(q), orc.rhs_ld(q)
    # stiff water: p is recovered from E with eps*E/Gamma absolute error (N1); fp64 and 80-bit differ by that
    worst, per = rel_err(r, rl, case.nfluids, case.ndim)
    assert worst <= 2e-9, per


@pytest.mark.parametrize("idx,n", [(2, 200), (3, 24), (4, 10), (5, 10)])
def test_textbook_form_rhs_agrees_with_difference_form_rhs(idx, n):
    """The two instantiations type the same definitions in two evaluation forms: their fp64
    results may differ by what either form loses to rounding, which the 80-bit evaluation of each measures — per variable
    |t64 - d64| <= 4 (|t64 - t80| + |d64 - d80|) + 1e-13 of the variable's scale — and the two 80-bit evaluations, where
    rounding is 2^11 times smaller, agree far inside the parity bar.  A dropped or mis-typed term in either form is an
    O(1) disagreement."""
    case = W.config(idx, n=n)
    q = W.initial_state(case)
    do, to = O.Oracle(case), O.Oracle(case, form="textbook")
    d64, d80, t64, t80 = do.rhs(q), do.rhs_ld(q), to.rhs(q), to.rhs_ld(q)
    assert do.bad == 0 and to.bad == 0
    N, D = case.nfluids, case.ndim
    for v in range(case.neq):
        grp = slice(N, N + D) if N <= v < N + D else slice(v, v + 1)   # momentum components share the group's scale
        scale = max(np.abs(d64[grp]).max(), 1e-300)
        noise = np.abs(t64[v] - t80[v]).max() + np.abs(d64[v] - d80[v]).max()
        assert np.abs(t64[v] - d64[v]).max() <= 4.0 * noise + 1e-13 * scale, (v, noise, scale)
        assert np.abs(t80[v] - d80[v]).max() <= 2e-3 * noise + 1e-15 * scale, (v, noise, scale)
    worst, per = rel_err(t80, d80, N, D)
    assert worst <= 1e-12 or idx in (3, 5), per   # configs 3, 5 at t = 0: the alpha rows are pure rounding noise (T2)


def test_operation_count_is_reported():
    case = W.config(4, n=8)
    c = O.Oracle(case).count_rhs(W.initial_state(case))
    per_cell = {k: v / case.cells for k, v in c.items()}
    # 3 directions x (8 WENO + 1 HLLC + prims) per cell: thousands of operations, two square roots per face
    assert 3000 < per_cell["add"] + per_cell["mul"] + per_cell["div"] < 9000, per_cell
    assert per_cell["sqrt"] == pytest.approx(2 * 3 * (8 + 1) / 8.0)
