"""Pins of the oracle's WENO-M and WENO-Z weights (oracle/mfc_oracle.hpp: weno5_weights, weno5) against what the paper
and the mathematics fix — no GPU.  PAPER.md:165 ("mapped weights, following Henrick et al."), 562-566 (WENO-Z, q = 1)."""
from fractions import Fraction as Fr

import numpy as np
import pytest

from oracle import oracle as O

JS, M, Z = O.RECON_WENO5, O.RECON_WENO5_M, O.RECON_WENO5_Z
D_LEFT = np.array([0.1, 0.6, 0.3])
D_RIGHT = np.array([0.3, 0.6, 0.1])


def test_general_routine_with_js_weights_is_the_pinned_js_routine():
    # the general routine shares candidates, smoothness indicators and evaluation form with weno5_js (pinned in
    # test_oracle_units.py); only two roundings are ordered differently
    rng = np.random.default_rng(11)
    for _ in range(200):
        s = rng.normal(size=5) * 10.0 ** rng.integers(-3, 4)
        for eps in (1e-6, 1e-16, 1e-40):
            a, b = O.weno5(JS, s, eps), O.weno5_js(s, eps)
            scale = np.abs(s).max()
            assert abs(a[0] - b[0]) <= 4e-16 * scale and abs(a[1] - b[1]) <= 4e-16 * scale


@pytest.mark.parametrize("recon", [M, Z])
def test_weights_sum_to_one_and_are_positive(recon):
    rng = np.random.default_rng(5)
    for _ in range(200):
        beta = 10.0 ** rng.uniform(-12, 6, 3)
        for dr in (D_LEFT, D_RIGHT):
            om = O.weno5_weights(recon, dr, beta, 1e-16)
            assert abs(om.sum() - 1.0) < 4e-16 and (om > 0).all()


@pytest.mark.parametrize("recon", [M, Z])
def test_linear_and_quadratic_data_exact(recon):
    # every candidate reproduces quadratics, the weights sum to one -> any convex combination is exact
    x = np.arange(-2, 3, dtype=float)
    for coef in [(3.0, -2.0, 0.0), (1.0, 0.5, 0.25), (-7.0, 0.0, 1.5)]:
        avg = np.array([coef[0] + coef[1] * xi + coef[2] * (xi * xi + 1.0 / 12.0) for xi in x])  # cell means, h = 1
        l, r = O.weno5(recon, avg, 1e-16)
        f = lambda t: coef[0] + coef[1] * t + coef[2] * t * t
        assert abs(l - f(0.5)) < 1e-14 and abs(r - f(-0.5)) < 1e-14


@pytest.mark.parametrize("recon", [M, Z])
def test_equal_smoothness_gives_ideal_weights(recon):
    # beta_0 = beta_1 = beta_2: JS weights are the ideal ones; Henrick's map fixes d_r; tau = 0
    for dr in (D_LEFT, D_RIGHT):
        om = O.weno5_weights(recon, dr, np.array([0.37, 0.37, 0.37]), 1e-16)
        assert np.abs(om - dr).max() < 3e-16


def test_wenoz_symmetric_stencil_is_the_linear_fifth_order_value():
    # stencil (a,b,c,b,a): beta_0 = beta_2 -> tau = 0 -> ideal weights -> the linear 5th-order scheme
    # (2a - 13b + 47c + 27d - 3e)/60, evaluated exactly in rationals; JS on the same stencil does not give it
    a, b, c = Fr(3, 8), Fr(5, 4), Fr(2)
    s = [a, b, c, b, a]
    lin = (2 * s[0] - 13 * s[1] + 47 * s[2] + 27 * s[3] - 3 * s[4]) / 60
    sf = np.array([float(v) for v in s])
    lz, rz = O.weno5(Z, sf, 1e-16)
    assert abs(lz - float(lin)) < 4e-16 and abs(rz - float(lin)) < 4e-16  # symmetric: both faces alike
    assert abs(O.weno5(JS, sf, 1e-16)[0] - float(lin)) > 1e-3


def test_wenoz_weights_worked_example_in_rationals():
    # PAPER.md:562-566 evaluated in exact arithmetic for one set of indicators
    beta = [Fr(1, 4), Fr(2), Fr(5, 2)]
    eps = Fr(1, 1000)
    for dr in ([Fr(1, 10), Fr(6, 10), Fr(3, 10)], [Fr(3, 10), Fr(6, 10), Fr(1, 10)]):
        tau = abs(beta[0] - beta[2])
        al = [d * (1 + tau / (b + eps)) for d, b in zip(dr, beta)]
        ex = [float(x / sum(al)) for x in al]
        om = O.weno5_weights(Z, [float(d) for d in dr], [float(b) for b in beta], float(eps))
        assert np.abs(om - np.array(ex)).max() < 3e-16


def test_mapped_weights_worked_example_in_rationals():
    # Henrick's map g_r(w) = w (d + d^2 - 3 d w + w^2)/(d^2 + w (1 - 2 d)) applied to the JS weights, renormalised
    beta = [Fr(1, 4), Fr(2), Fr(5, 2)]
    eps = Fr(1, 1000)
    for dr in ([Fr(1, 10), Fr(6, 10), Fr(3, 10)], [Fr(3, 10), Fr(6, 10), Fr(1, 10)]):
        al = [d / (b + eps) ** 2 for d, b in zip(dr, beta)]
        w = [x / sum(al) for x in al]
        g = [wi * (d + d * d - 3 * d * wi + wi * wi) / (d * d + wi * (1 - 2 * d)) for wi, d in zip(w, dr)]
        ex = [float(x / sum(g)) for x in g]
        om = O.weno5_weights(M, [float(d) for d in dr], [float(b) for b in beta], float(eps))
        assert np.abs(om - np.array(ex)).max() < 3e-16


def test_mapping_is_flat_to_second_order_at_the_ideal_weights():
    # g_r(d_r) = d_r, g_r'(d_r) = g_r''(d_r) = 0: a perturbation delta of the indicators moves the JS weights by
    # O(delta) and the mapped ones by O(delta^3).  A wrong coefficient in the map leaves a linear or quadratic term.
    devs_js, devs_m = [], []
    for delta in (1e-1, 1e-2, 1e-3):
        beta = np.array([1.0 + delta, 1.0 - 0.5 * delta, 1.0 + 0.25 * delta])
        devs_js.append(np.abs(O.weno5_weights(JS, D_LEFT, beta, 1e-40) - D_LEFT).max())
        devs_m.append(np.abs(O.weno5_weights(M, D_LEFT, beta, 1e-40) - D_LEFT).max())
    r_js = np.log10(np.array(devs_js[:-1]) / np.array(devs_js[1:]))
    r_m = np.log10(np.array(devs_m[:-1]) / np.array(devs_m[1:]))
    assert (np.abs(r_js - 1.0) < 0.15).all(), (devs_js, r_js)
    assert (np.abs(r_m - 3.0) < 0.35).all(), (devs_m, r_m)


@pytest.mark.parametrize("recon", [M, Z])
def test_eno_property_at_a_step(recon):
    # stencil with a jump between cells i+1 and i+2: the candidate that crosses it gets (almost) no weight, the value
    # stays within the smooth data; the mirrored stencil gives the mirrored result
    s = np.array([1.0, 1.0 + 1e-3, 1.0 + 2e-3, 1.0 + 3e-3, 50.0])
    l, r = O.weno5(recon, s, 1e-16)
    assert 1.0 + 2e-3 < l < 1.0 + 3e-3 + 1e-9 and 1.0 + 1e-3 < r < 1.0 + 2e-3
    lm, rm = O.weno5(recon, s[::-1].copy(), 1e-16)
    assert lm == r and rm == l


def _critical_point_orders(recon):
    """order of (f^_{i+1/2} - f^_{i-1/2})/h at the critical point x = 0 of f = x^3 + cos x (f' = 0, f'' != 0), brute
    force refinement in 80-bit arithmetic with eps = 1e-40"""
    f = lambda x: x ** 3 + np.cos(x)
    F = lambda x: x ** 4 / 4 + np.sin(x)
    errs = []
    for k in range(4, 9):
        h = 2.0 ** -k
        avg = lambda i: (F((i + 0.5) * h) - F((i - 0.5) * h)) / h
        L = lambda i: O.weno5(recon, np.array([avg(i + j) for j in range(-2, 3)]), 1e-40, ld=True)[0]
        e = 0.0
        for i in (-1, 0, 1):
            e = max(e, abs(((L(i) - f((i + 0.5) * h)) - (L(i - 1) - f((i - 0.5) * h))) / h))
        errs.append(e)
    errs = np.array(errs)
    return np.log2(errs[:-1] / errs[1:])


def test_order_at_a_critical_point_distinguishes_the_three_weights():
    # JS drops to third order at a critical point; the mapped weights restore fifth (Henrick et al., the reason the
    # paper uses them); WENO-Z with q = 1 gives fourth (q "influences the convergence
    # rate at the critical points")
    r_js, r_m, r_z = (_critical_point_orders(r) for r in (JS, M, Z))
    assert (r_js > 2.8).all() and (r_js < 3.8).all(), r_js
    assert (r_m[1:] > 4.8).all(), r_m
    assert (r_z > 3.9).all() and (r_z < 4.7).all(), r_z


@pytest.mark.parametrize("recon", [M, Z])
def test_fp64_form_agrees_with_80_bit(recon):
    rng = np.random.default_rng(3)
    for _ in range(300):
        s = rng.normal(size=5) * 10.0 ** rng.integers(-2, 6)
        a, b = O.weno5(recon, s, 1e-16), O.weno5(recon, s, 1e-16, ld=True)
        scale = np.abs(s).max()
        assert abs(a[0] - b[0]) <= 8e-16 * scale and abs(a[1] - b[1]) <= 8e-16 * scale


# ------------------------------------------------------------------ system level: the variants inside the whole path
@pytest.mark.parametrize("recon", [M, Z])
def test_sod_with_variant_weights_converges_to_the_exact_solution(recon):
    from test_oracle_system import _sod_errors
    errs = [_sod_errors(n, recon)[2] for n in (250, 500)]
    e_js = _sod_errors(500, JS)[2]
    assert errs[1] < errs[0] * 0.62 and errs[1] < 3e-3, errs
    # sharper weights resolve the contact at least as well as JS on the same grid (less dissipative: PAPER.md:562)
    assert errs[1] <= e_js * 1.02, (errs, e_js)


@pytest.mark.parametrize("recon", [M, Z])
def test_uniform_state_and_conservation_with_variant_weights(recon):
    import mfc_workloads as W
    case = W.config(4, n=10)
    q = W.initial_state(case)
    orc = O.Oracle(case, recon)
    r = orc.rhs(q)
    N, D = case.nfluids, case.ndim
    tot = np.abs(r).reshape(case.neq, -1).sum(axis=1)
    s = r.reshape(case.neq, -1).sum(axis=1)
    assert (np.abs(s[:N + D + 1]) <= 1e-12 * tot[:N + D + 1]).all()   # telescoping flux sums on a periodic domain
    qu = np.empty_like(q)
    qu[...] = q.reshape(case.neq, -1)[:, :1].reshape(case.neq, 1, 1, 1)
    assert np.array_equal(orc.rhs(qu), np.zeros_like(qu))
