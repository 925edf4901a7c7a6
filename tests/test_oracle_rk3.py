"""Pins of the oracle's time integrator Solver::rk3_step (O6) and of its mixture sound speed (A5).

Every system pin of test_oracle_system.py (convergence at rate ~1 on shocks, conservation, interface
equilibrium, uniform state, symmetry) is satisfied by ANY convex three-stage combination; these two are not:
  * the amplification factor of one step on a linear problem must be 1 + z + z^2/2 + z^3/6 (the third-order
    Taylor polynomial every third-order three-stage Runge-Kutta method has) — a wrong stage coefficient
    (3/4 <-> 1/4, 1/3 <-> 2/3, a dropped dt) changes the z^2 or z^3 term;
  * the error of a smooth nonlinear run against a much finer time step, on a FIXED grid, must fall as dt^3.
CPU only."""
import numpy as np
import pytest

import mfc_workloads as W
from oracle import oracle as O


def advection_case(n, recon_eps=1e-6):
    # one ideal gas on [0,1), periodic; uniform u and p: the density profile is advected (PAPER.md:57-61 with K = 0)
    return W.Case("adv", 1, (n, 1, 1), (1.0 / n, 1.0, 1.0), 1, (1.4,), (0.0,), (W.BC_PERIODIC,) * 3, (W.BC_PERIODIC,) * 3,
                  weno_eps=recon_eps, clamp=False)


def density_wave(case, rho):
    one = np.ones(case.shape[1:])
    return np.ascontiguousarray(W.cons_from_prim(case, [rho.reshape(case.shape[1:])], [1.0 * one], 1.0, [one]))


# ------------------------------------------------------------------ amplification polynomial
@pytest.mark.parametrize("k,cfl", [(1, 0.9), (3, 0.5), (5, 0.25)])
def test_rk3_amplification_factor_is_the_cubic_taylor_polynomial(k, cfl):
    """With piecewise-constant reconstruction, uniform u > 0 and uniform p the HLLC flux of the density is
    rho_{i-1} u (the contact is resolved exactly): d rho_i/dt = -u (rho_i - rho_{i-1})/dx, a linear
    circulant system.  Fourier mode theta = 2 pi k/n has the eigenvalue lambda = -(u/dx)(1 - exp(-i theta)); one step of a
    third-order three-stage method multiplies its amplitude by R(z) = 1 + z + z^2/2 + z^3/6, z = lambda dt."""
    n = 32
    case = advection_case(n)
    u, dx = 1.0, 1.0 / n
    theta = 2.0 * np.pi * k / n
    i = np.arange(n)
    amp = 1e-3
    rho0 = 1.0 + amp * np.cos(theta * i)
    q = density_wave(case, rho0)
    dt = cfl * dx / u
    orc = O.Oracle(case, recon=O.RECON_PC)
    orc.rk3_step(q, dt)
    assert orc.bad == 0
    rho1 = q[0, 0, 0]
    # complex amplitude of mode k before and after
    a0 = np.sum((rho0 - 1.0) * np.exp(-1j * theta * i)) * 2.0 / n
    a1 = np.sum((rho1 - 1.0) * np.exp(-1j * theta * i)) * 2.0 / n
    z = -(u / dx) * (1.0 - np.exp(-1j * theta)) * dt
    R = 1.0 + z + z * z / 2.0 + z ** 3 / 6.0
    assert abs(a1 / a0 - R) < 1e-11, (a1 / a0, R)
    # the polynomial distinguishes the method: the second-order (Heun) and the first-order (Euler) factors are far away,
    # and so is R with the stage weights 3/4 <-> 1/4 exchanged (q2 = 1/4 q + 3/4 (q1 + dt L q1) gives 1 + 2z + 3/2 z^2 + 1/2 z^3)
    assert abs(R - (1.0 + z + z * z / 2.0)) > 1e-5
    assert abs(R - (1.0 + 2.0 * z + 1.5 * z * z + 0.5 * z ** 3)) > 1e-3
    # velocity and pressure stay uniform (interface equilibrium), so the linear model is the whole of it
    w = O.Oracle(case).prim_from_cons(q)
    assert np.abs(w[1] - 1.0).max() < 1e-13 and np.abs(w[2] - 1.0).max() < 1e-12


# ------------------------------------------------------------------ order in dt on a fixed grid
def test_rk3_error_falls_as_dt_cubed_on_a_fixed_grid():
    """Smooth nonlinear flow (an acoustic + entropy wave of finite amplitude, WENO5-JS + HLLC), fixed grid of 64 cells, to
    t = 0.04: the difference to a run with a 16 times smaller step is the time-integration error alone; it must fall by
    2^3 per halving of dt (observed order >= 2.8)."""
    n = 64
    case = advection_case(n)
    x = (np.arange(n) + 0.5) / n
    one = np.ones(case.shape[1:])
    rho = (1.0 + 0.2 * np.sin(2 * np.pi * x)).reshape(case.shape[1:])
    vel = (0.5 + 0.1 * np.cos(2 * np.pi * x)).reshape(case.shape[1:])
    p = (1.0 + 0.1 * np.sin(4 * np.pi * x)).reshape(case.shape[1:])
    q0 = np.ascontiguousarray(W.cons_from_prim(case, [rho], [vel], p, [one]))
    orc = O.Oracle(case)
    t_end = 0.04

    def run(nsteps):
        q = q0.copy()
        dt = t_end / nsteps
        for _ in range(nsteps):
            orc.rk3_step(q, dt)
            assert orc.bad == 0
        return q

    ref = run(16 * 32)
    errs = [np.abs(run(m) - ref).max() for m in (8, 16, 32)]   # CFL about 0.6, 0.3, 0.15
    orders = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert errs[0] > 1e-8            # the time error is far above round-off: the slope is measured, not noise
    assert np.all(orders > 2.8) and np.all(orders < 3.3), (errs, orders)


# ------------------------------------------------------------------ mixture sound speed (reading A5)
@pytest.mark.parametrize("alpha_w", [1e-6, 0.02, 0.5, 0.97])
def test_mixture_sound_speed_is_the_isentropic_derivative_of_the_eos(alpha_w):
    """A5: c^2 = ((Gamma+1) p + Pi)/(Gamma rho) at frozen volume fractions.  Pinned without that formula: along an isentrope
    de = (p/rho^2) d rho, so c^2 = dp/drho|_s = dp/drho|_e + (p/rho^2) dp/de|_rho, the partial derivatives taken by central
    differences (with one Richardson step) of the pressure the ORACLE's cons->prim conversion returns for the mixture
    (eq.(4), 117); the oracle's c is read off its CFL time step on a one-cell grid (dt = cfl dx/(|u|+c))."""
    case = W.Case("c", 1, (1, 1, 1), (1.0, 1.0, 1.0), 2, (4.4, 1.4), (6.0e8, 0.0), (W.BC_PERIODIC,) * 3, (W.BC_PERIODIC,) * 3)
    orc = O.Oracle(case)
    a = [alpha_w, 1.0 - alpha_w]
    arho = [a[0] * 1000.0, a[1] * 1.2]
    rho = arho[0] + arho[1]
    p0, u0 = 2.0e5, 3.0

    def state(rho_, e_):  # conservative cell of density rho_ (same mass fractions, same alpha) and specific internal energy e_
        s = rho_ / rho
        q = np.zeros(case.shape)
        q[0], q[1] = arho[0] * s, arho[1] * s
        q[2] = rho_ * u0
        q[3] = rho_ * e_ + 0.5 * rho_ * u0 * u0
        q[4], q[5] = a
        return q

    def pressure(rho_, e_):
        return float(orc.prim_from_cons(state(rho_, e_))[3, 0, 0, 0])

    # e at (rho, p0) from the conservative state the workload builder makes (the inverse of cons->prim, used by neither side)
    one = np.ones(case.shape[1:])
    qc = W.cons_from_prim(case, [arho[0] * one, arho[1] * one], [u0 * one], p0, [a[0] * one, a[1] * one])
    e0 = float((qc[3, 0, 0, 0] - 0.5 * rho * u0 * u0) / rho)
    assert pressure(rho, e0) == pytest.approx(p0, rel=1e-9)

    def dcentral(f, x, h):
        d1 = (f(x + h) - f(x - h)) / (2 * h)
        d2 = (f(x + h / 2) - f(x - h / 2)) / h
        return (4 * d2 - d1) / 3

    dp_drho = dcentral(lambda r: pressure(r, e0), rho, 1e-3 * rho)
    dp_de = dcentral(lambda e: pressure(rho, e), e0, 1e-3 * e0)
    c2_brute = dp_drho + p0 / rho ** 2 * dp_de
    dt = orc.cfl_dt(np.ascontiguousarray(qc), 1.0)
    c_oracle = 1.0 / dt - abs(u0)
    assert c_oracle ** 2 == pytest.approx(c2_brute, rel=1e-6)
    # Wood's formula (equilibrium of pressure and phase entropy, 1/(rho c^2) = sum alpha_i/(rho_i c_i^2)) is a DIFFERENT speed:
    # the frozen-alpha speed of A5 is the larger one for a true mixture
    ci2 = [case.gamma[i] * (p0 + case.pi_inf[i]) / (arho[i] / a[i]) for i in range(2)]
    wood = 1.0 / (rho * sum(a[i] / ((arho[i] / a[i]) * ci2[i]) for i in range(2)))
    assert c_oracle ** 2 >= wood * (1 - 1e-12)


# ------------------------------------------------------------------ what the CFL number of cfl_dt means (reading A9)
def test_cfl_dt_scales_the_step_to_the_stability_limit_of_the_fastest_wave():
    """A9 defines dt = CFL / max sum_d (|u_d| + c)/dx_d; nothing in the paper does.  What can be pinned is its meaning: with
    first-order upwinding (piecewise-constant reconstruction + HLLC) each characteristic field of the linearised 1-D Euler
    equations obeys dw/dt = -lambda (w_i - w_{i-1})/dx, and SSP-RK3 is stable for lambda dt/dx <= 1.2564 (|R(z)| <= 1 on
    z = -nu (1 - exp(-i theta)) up to nu = 1.2564).  The fastest field has lambda = |u| + c, so a small perturbation of a
    uniform state must stay bounded for CFL = 1.15 and blow up for CFL = 1.40.  A cfl_dt that used c alone, |u| alone, or
    half / twice the spacing would fail one of the two."""
    n = 64
    case = advection_case(n)
    rng = np.random.default_rng(5)
    one = np.ones(case.shape[1:])
    pert = lambda: 1e-7 * rng.standard_normal(case.shape[1:])
    q0 = np.ascontiguousarray(W.cons_from_prim(case, [1.0 + pert()], [0.8 + pert()], 1.0 + pert(), [one]))  # u = 0.8, c = 1.18
    orc = O.Oracle(case, recon=O.RECON_PC)
    base = np.ascontiguousarray(W.cons_from_prim(case, [one], [0.8 * one], 1.0, [one]))

    def growth(cfl, nsteps=400):
        q = q0.copy()
        dt = orc.cfl_dt(q, cfl)
        assert dt == pytest.approx(cfl * (1.0 / n) / (0.8 + np.sqrt(1.4)), rel=1e-6)
        for _ in range(nsteps):
            orc.rk3_step(q, dt)
        return np.abs(q - base).max() / np.abs(q0 - base).max()

    assert growth(1.15) < 2.0
    g = growth(1.40)
    assert not (g < 1e3)  # grown beyond 10^3, or overflowed to inf / nan
