"""Pins of the oracle's viscous terms (eqs. (1), (2); reading A22) — no GPU.
The viscous contribution is isolated as rhs(eta) - rhs(0) on states of uniform density and pressure."""
import numpy as np
import pytest

import mfc_workloads as W
from oracle import oracle as O

ETA = 0.37


def case_nd(ndim, n, bc=W.BC_PERIODIC, eta=ETA, L=1.0):
    nn = tuple(n if d < ndim else 1 for d in range(3))
    return W.Case("v", ndim, nn, tuple(L / n if d < ndim else 1.0 for d in range(3)), 1, (1.4,), (0.0,),
                  (bc,) * 3, (bc,) * 3, clamp=False, eta=eta)


def state(case, ufun, rho=1.3, p=2.0):
    """uniform rho, p; velocity ufun(x, y, z) -> tuple of ndim arrays, at cell centres"""
    D = case.ndim
    ax = [(np.arange(case.n[d]) + 0.5) * case.dx[d] if d < D else np.zeros(1) for d in range(3)]
    Z, Y, X = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    u = ufun(X, Y, Z)
    q = np.empty(case.shape)
    q[0] = rho
    ke = 0.0
    for d in range(D):
        q[1 + d] = rho * u[d]
        ke = ke + 0.5 * rho * u[d] ** 2
    q[1 + D] = p / 0.4 + ke
    q[2 + D] = 1.0
    return q, (X, Y, Z), u


def viscous_part(case, q):
    from dataclasses import replace
    return O.Oracle(case).rhs(q) - O.Oracle(replace(case, eta=0.0)).rhs(q)


def test_uniform_shear_has_no_force_and_dissipates_eta_s2():
    # u_x = s y: T_xy = eta s everywhere, so div T = 0 and d/dy (T_xy u_x) = eta s^2; exact for a linear field
    s = 3.0
    case = case_nd(2, 16, bc=W.BC_EXTRAP)
    q, _, _ = state(case, lambda X, Y, Z: (s * Y, 0 * Y))
    v = viscous_part(case, q)
    inner = (slice(None), 0, slice(2, -2), slice(2, -2))
    assert np.abs(v[1][inner[1:]]).max() < 1e-12 and np.abs(v[2][inner[1:]]).max() < 1e-12
    assert v[3][inner[1:]] == pytest.approx(ETA * s * s, rel=1e-12)
    assert np.abs(v[0]).max() == 0.0 and np.abs(v[4]).max() == 0.0       # mass and volume fraction untouched


def _wave_error(ndim, n, kind):
    """max error of the viscous momentum rate against the continuum value for a plane wave along the diagonal"""
    case = case_nd(ndim, n)
    k = 2 * np.pi
    D = ndim
    khat = np.ones(D) / np.sqrt(D)
    if kind == "shear":                      # polarisation perpendicular to the wave vector: div u = 0
        pol = np.array([1.0, -1.0, 0.0][:D]) / np.sqrt(2.0)
        coef = 1.0
    else:                                    # longitudinal: u parallel to the wave vector
        pol = khat
        coef = 4.0 / 3.0
    kvec = k * np.ones(D)                    # wave vector (k, k[, k]): periodic on the unit box
    k2 = float(kvec @ kvec)

    def ufun(X, Y, Z):
        ph = kvec[0] * X + kvec[1] * Y + (kvec[2] * Z if D == 3 else 0.0)
        return tuple(0.2 * pol[d] * np.sin(ph) for d in range(D))

    q, _, u = state(case, ufun)
    v = viscous_part(case, q)
    err = 0.0
    for d in range(D):
        exact = -coef * ETA * k2 * u[d]      # eta lap(u) for the shear wave, (4/3) eta grad(div u) for the longitudinal one
        err = max(err, np.abs(v[1 + d] - exact).max())
    return err, ETA * k2 * 0.2


@pytest.mark.parametrize("kind", ["shear", "longitudinal"])
@pytest.mark.parametrize("ndim", [2, 3])
def test_plane_waves_along_the_diagonal_converge_at_second_order(ndim, kind):
    # the diagonal direction exercises every cross derivative: for the shear wave they must cancel to eta lap(u),
    # for the longitudinal wave they must add up to (4/3) eta grad(div u) — a wrong factor, sign, index or a missing
    # -2/3 div term changes the limit, not just the error
    ns = (8, 16, 32) if ndim == 3 else (16, 32, 64)
    errs, scale = [], None
    for n in ns:
        e, scale = _wave_error(ndim, n, kind)
        errs.append(e)
    rates = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert errs[-1] < 0.02 * scale and (rates > 1.8).all() and 1.93 < rates[-1] < 2.07, (errs, rates)


def test_axis_aligned_waves_one_dimensional_limits():
    # u_x = A sin(k x): (4/3) eta u_xx ; u_y = A sin(k x): eta u_xx — the textbook 1-D limits, and the energy equation gets
    # d/dx (T u): compare with the continuum expression
    n, k, A = 128, 2 * np.pi, 0.1
    case = case_nd(2, n)
    q, (X, Y, Z), u = state(case, lambda X, Y, Z: (A * np.sin(k * X), A * np.sin(k * X)))
    v = viscous_part(case, q)
    assert np.abs(v[1] - (-(4.0 / 3.0) * ETA * k * k * u[0])).max() < 2e-3 * ETA * k * k * A
    assert np.abs(v[2] - (-ETA * k * k * u[1])).max() < 2e-3 * ETA * k * k * A
    Txx = (4.0 / 3.0) * ETA * A * k * np.cos(k * X)
    Tyx = ETA * A * k * np.cos(k * X)
    dTu = (-(4.0 / 3.0) * ETA * A * k * k * np.sin(k * X)) * u[0] + Txx * A * k * np.cos(k * X) \
        + (-ETA * A * k * k * np.sin(k * X)) * u[1] + Tyx * A * k * np.cos(k * X)
    assert np.abs(v[3] - dTu).max() < 5e-3 * np.abs(dTu).max()


@pytest.mark.parametrize("ndim", [1, 2, 3])
def test_viscous_terms_conserve_momentum_and_energy_on_a_periodic_domain(ndim):
    rng = np.random.default_rng(3)
    case = case_nd(ndim, 10)
    ph = rng.uniform(0, 6, (3, 3))

    def ufun(X, Y, Z):
        return tuple(np.sin(2 * np.pi * X + ph[d, 0]) * np.cos(2 * np.pi * Y + ph[d, 1]) * np.cos(2 * np.pi * Z + ph[d, 2])
                     for d in range(ndim))
    q, _, _ = state(case, ufun)
    v = viscous_part(case, q)
    for m in range(1, 2 + ndim):
        assert abs(v[m].sum()) <= 1e-10 * np.abs(v[m]).sum() + 1e-12


def test_rigid_motion_and_zero_viscosity_give_nothing():
    case = case_nd(3, 8)
    q, _, _ = state(case, lambda X, Y, Z: (0 * X + 0.3, 0 * X - 0.1, 0 * X + 0.2))   # uniform translation
    assert np.abs(viscous_part(case, q)).max() < 1e-12
    q, _, _ = state(case_nd(2, 12, bc=W.BC_EXTRAP), lambda X, Y, Z: (-2.0 * Y, 2.0 * X))   # rigid rotation: D = 0
    v = viscous_part(case_nd(2, 12, bc=W.BC_EXTRAP), q)
    assert np.abs(v[:, 0, 2:-2, 2:-2]).max() < 1e-11


def test_taylor_green_vortex_dissipation_rate():
    # the paper's viscous example shape.  For the divergence-free Taylor-Green field the viscous terms take
    # kinetic energy out at the rate  -<u . div T> = eta <|curl u|^2> = (3/4) eta V0^2  (volume mean; closed form of the
    # initial field).  The discrete rate converges to it at second order.
    from dataclasses import replace
    errs = []
    for n in (16, 32):
        case = W.taylor_green(n, mach=0.1, reynolds=100.0)
        q = W.initial_state(case)
        v = O.Oracle(case).rhs(q) - O.Oracle(replace(case, eta=0.0)).rhs(q)
        rho = q[0]
        u = q[1:4] / rho
        rate = (u * v[1:4]).sum() / case.cells
        v0 = 0.1 * np.sqrt(1.4)
        exact = -0.75 * case.eta * v0 * v0
        errs.append(abs(rate - exact) / abs(exact))
        # total energy: the viscous work integrates to zero over the periodic box
        assert abs(v[4].sum()) <= 1e-10 * np.abs(v[4]).sum()
    assert errs[1] < 0.01 and 3.6 < errs[0] / errs[1] < 4.4, errs
