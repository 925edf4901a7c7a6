"""Pins of the oracle's Kapila term K div(u) (eqs. (5), (6); reading A13) — no GPU."""
from dataclasses import replace

import numpy as np
import pytest

import mfc_workloads as W
from oracle import oracle as O

WATER, AIR = (4.4, 6.0e8), (1.4, 0.0)


def case_1d(n=40, fluids=(WATER, AIR), model="kapila", bc=W.BC_EXTRAP):
    return W.Case("k", 1, (n, 1, 1), (1.0 / n, 1.0, 1.0), 2, (fluids[0][0], fluids[1][0]), (fluids[0][1], fluids[1][1]),
                  (bc,) * 3, (bc,) * 3, clamp=False, model=model)


def isentropic_dalpha1(p, a1, fluids, dlnV):
    """brute force: a parcel holding volumes a1 and 1 - a1 of the two stiffened gases at common pressure p is compressed
    to total volume 1 + dlnV, each phase isentropically ((p + pi_i) V_i^gamma_i = const), pressures staying equal;
    returns the change of alpha_1 = V_1 / (V_1 + V_2).  No formula of the paper is used."""
    (g1, pi1), (g2, pi2) = fluids
    V1, V2 = a1, 1.0 - a1
    vol = lambda pn: V1 * ((p + pi1) / (pn + pi1)) ** (1.0 / g1) + V2 * ((p + pi2) / (pn + pi2)) ** (1.0 / g2)
    lo, hi = p * 0.5, p * 2.0 + 1.0
    for _ in range(200):                       # bisection on the new common pressure
        mid = 0.5 * (lo + hi)
        if vol(mid) > 1.0 + dlnV:
            lo = mid
        else:
            hi = mid
    pn = 0.5 * (lo + hi)
    V1n = V1 * ((p + pi1) / (pn + pi1)) ** (1.0 / g1)
    return V1n / (1.0 + dlnV) - a1


@pytest.mark.parametrize("fluids", [(WATER, AIR), (AIR, WATER), ((1.4, 0.0), (1.67, 0.0)), ((2.35, 1.0e9), (1.4, 0.0))])
@pytest.mark.parametrize("a1", [0.02, 0.3, 0.5, 0.9])
def test_K_is_the_isentropic_compression_rate_of_alpha1(fluids, a1):
    # d(alpha_1) = K div(u) dt with div(u) dt = dV/V: compare with the parcel computation for a small compression.
    # The printed "+" of eq. (5) would fail this by a factor of order one.
    p = 3.0e5
    orc = O.Oracle(case_1d(fluids=fluids))
    K = orc.kapila_K(p, a1, 1.0 - a1)
    d = -1e-6
    assert isentropic_dalpha1(p, a1, fluids, d) == pytest.approx(K * d, rel=2e-5, abs=1e-15)


def test_K_limits_and_symmetries():
    orc = O.Oracle(case_1d())
    swapped = O.Oracle(case_1d(fluids=(AIR, WATER)))
    same = O.Oracle(case_1d(fluids=(AIR, AIR)))
    for p in (1e5, 1e9):
        for a1 in (0.1, 0.5, 0.8):
            assert same.kapila_K(p, a1, 1 - a1) == 0.0                        # identical fluids: no relative compression
            assert swapped.kapila_K(p, 1 - a1, a1) == pytest.approx(-orc.kapila_K(p, a1, 1 - a1), rel=1e-14)
        # pure fluid: K -> 0 linearly in the vanishing volume fraction
        assert abs(orc.kapila_K(p, 1e-9, 1.0)) < 2e-9
        assert orc.kapila_K(p, 1.0, 1e-9) == pytest.approx(1e3 * orc.kapila_K(p, 1.0, 1e-12), rel=1e-3)
        assert abs(orc.kapila_K(p, 1.0, 1e-12)) < 1e-7
        assert orc.kapila_K(p, 0.0, 1.0) == 0.0 and orc.kapila_K(p, 1.0, 0.0) == 0.0


def uniform_mixture_with_linear_velocity(case, a1, p, s):
    n = case.n[0]
    x = (np.arange(n) + 0.5) / n
    rho = np.array([1000.0, 1.0])
    al = np.array([a1, 1.0 - a1])
    u = s * (x - 0.5)
    q = np.empty(case.shape)
    q[0], q[1] = al[0] * rho[0], al[1] * rho[1]
    r = q[0] + q[1]
    q[2] = r * u
    Gam = sum(al[i] / (case.gamma[i] - 1) for i in range(2))
    Pi = sum(al[i] * case.gamma[i] * case.pi_inf[i] / (case.gamma[i] - 1) for i in range(2))
    q[3] = Gam * p + Pi + 0.5 * r * u * u
    q[4], q[5] = al[0], al[1]
    return q


def test_uniform_mixture_under_uniform_dilatation():
    # uniform alpha, rho, p and u = s x: WENO reproduces the linear velocity, the Riemann problem of two equal states
    # returns it, so d(alpha_1)/dt = K s in the interior (the flux and alpha div(u) parts cancel), -K s for alpha_2,
    # and 0 for the Allaire model
    a1, p, s = 0.3, 2.0e5, 7.0
    ck, ca = case_1d(), case_1d(model="allaire")
    q = uniform_mixture_with_linear_velocity(ck, a1, p, s)
    ok, oa = O.Oracle(ck), O.Oracle(ca)
    rk, ra = ok.rhs(q), oa.rhs(q)
    K = ok.kapila_K(p, a1, 1 - a1)
    inner = slice(4, -4)
    assert np.abs(ra[4, 0, 0, inner]).max() < 1e-9 * abs(K * s)
    assert rk[4, 0, 0, inner] == pytest.approx(K * s, rel=1e-9)
    assert rk[5, 0, 0, inner] == pytest.approx(-K * s, rel=1e-9)
    assert np.array_equal(rk[:4], ra[:4])                                # the conservative equations are untouched


def test_K_term_vanishes_for_an_advected_interface_and_keeps_sum_alpha():
    # uniform p and u across a smeared interface: div(u) = 0, Kapila and Allaire agree; in a flow with div(u) != 0 the
    # two alpha equations get opposite K terms, so their sum is the Allaire one
    n = 64
    ck, ca = case_1d(n, bc=W.BC_PERIODIC), case_1d(n, model="allaire", bc=W.BC_PERIODIC)
    x = (np.arange(n) + 0.5) / n
    a1 = 0.5 * (1 + np.tanh((0.25 - np.abs(x - 0.5)) * 20)) * (1 - 2e-6) + 1e-6
    al = np.array([a1, 1 - a1])
    rho = np.array([1000.0, 1.0])
    for u in (np.full(n, 30.0), 30.0 * np.sin(2 * np.pi * x)):
        q = np.empty(ck.shape)
        q[0, 0, 0], q[1, 0, 0] = al[0] * rho[0], al[1] * rho[1]
        r = q[0, 0, 0] + q[1, 0, 0]
        q[2, 0, 0] = r * u
        Gam = sum(al[i] / (ck.gamma[i] - 1) for i in range(2))
        Pi = sum(al[i] * ck.gamma[i] * ck.pi_inf[i] / (ck.gamma[i] - 1) for i in range(2))
        q[3, 0, 0] = Gam * 1e5 + Pi + 0.5 * r * u * u
        q[4, 0, 0], q[5, 0, 0] = al
        rk, ra = O.Oracle(ck).rhs(q), O.Oracle(ca).rhs(q)
        scale = np.abs(ra[4:]).max()
        if u[0] == u[1]:
            assert np.abs(rk - ra)[4:].max() <= 1e-9 * scale
        else:
            assert np.abs(rk - ra)[4:].max() > 1e-3 * scale                  # the term is there
        assert np.abs((rk[4] + rk[5]) - (ra[4] + ra[5])).max() <= 1e-12 * scale
