"""Pins of the oracle's building blocks (O1-O4, A9, A10) against closed forms, invariants,
textbook forms and brute force.  CPU only."""
import numpy as np
import pytest

import mfc_workloads as W
from oracle import oracle as O


def small_case(ndim=1, nfluids=2, n=8, bc=W.BC_PERIODIC, gamma=(1.4, 4.4, 1.67), pi_inf=(0.0, 6.0e8, 0.0)):
    nn = tuple(n if d < ndim else 1 for d in range(3))
    return W.Case("unit", ndim, nn, tuple(1.0 / n if d < ndim else 1.0 for d in range(3)), nfluids,
                  tuple(gamma[:nfluids]), tuple(pi_inf[:nfluids]), (bc,) * 3, (bc,) * 3, builder="")


# ------------------------------------------------------------------ O1 ghost cells
def test_ghost_index_bruteforce():
    for n in (1, 2, 3, 5, 8):
        for g in range(-3, n + 3):
            assert O.ghost_index(g, n, W.BC_EXTRAP, W.BC_EXTRAP) == min(max(g, 0), n - 1)
            # periodic: the ghost value equals the value of an infinitely repeated line
            rep = list(range(n)) * 9
            assert O.ghost_index(g, n, W.BC_PERIODIC, W.BC_PERIODIC) == rep[g + 4 * n]


# ------------------------------------------------------------------ O2 primitives
@pytest.mark.parametrize("ndim,nfluids", [(1, 1), (1, 2), (2, 2), (3, 2), (3, 3)])
def test_prim_round_trip(ndim, nfluids):
    case = small_case(ndim, nfluids, n=6)
    rng = np.random.default_rng(7)
    sh = case.shape[1:]
    alpha = rng.uniform(0.05, 1.0, (nfluids,) + sh)
    alpha /= alpha.sum(0)
    arho = alpha * np.array([1.0, 1000.0, 0.138])[:nfluids].reshape(-1, 1, 1, 1) * rng.uniform(0.8, 1.2, (nfluids,) + sh)
    u = rng.uniform(-300, 300, (ndim,) + sh)
    p = rng.uniform(1e4, 1e9, sh)
    q = W.cons_from_prim(case, list(arho), list(u), p, list(alpha))   # independent numpy statement of the EOS
    w = O.Oracle(case).prim_from_cons(q)
    N, D = nfluids, ndim
    # E carries p in its trailing digits when Pi >> p: the recoverable accuracy is eps*E/Gamma
    tol_p = 8 * np.finfo(float).eps * np.abs(q[N + D]).max() / (alpha[0] * 0 + sum(alpha[i] / (case.gamma[i] - 1) for i in range(N))).min()
    assert np.abs(w[N + D] - p).max() <= max(tol_p, 1e-13 * p.max())
    assert np.abs(w[N:N + D] - u).max() <= 1e-13 * 300
    assert np.array_equal(w[:N], q[:N]) and np.array_equal(w[N + D + 1:], q[N + D + 1:])


def test_prim_pure_fluid_closed_form():
    # pure stiffened gas: p = (gamma-1)(E - ke) - gamma*pi_inf   (PAPER.md:117 solved for p)
    g, pinf = 4.4, 6.0e8
    case = small_case(1, 1, n=5, gamma=(g,), pi_inf=(pinf,))
    rho = np.array([1000.0, 990.0, 1010.0, 1000.0, 5.0]).reshape(1, 1, 5)
    u = np.array([0.0, 10.0, -300.0, 1500.0, 3.0]).reshape(1, 1, 5)
    E = np.array([8.0e8, 9.0e8, 2.0e9, 4.0e9, 7.8e8]).reshape(1, 1, 5)
    q = np.stack([rho, rho * u, E, np.ones_like(rho)])
    w = O.Oracle(case).prim_from_cons(np.ascontiguousarray(q))
    p_ref = (g - 1.0) * (E - 0.5 * rho * u * u) - g * pinf
    assert np.allclose(w[2], p_ref, rtol=1e-12, atol=1e-6)
    assert np.allclose(w[1], u, rtol=1e-15)


# Every pin of O3 (JS weights) and O4 below runs on BOTH instantiations of the reference: the difference form (readings N2 /
# N3, what the parity bars are measured against) and the textbook form (PAPER.md:163 f = sum omega_r f^(r); PAPER.md:197,
# 668 F = F_K + S_K (q*_K - q_K)) — the second exists to make the parity claim independent of the evaluation form, so it
# must stand on the same pins as the first, not on the CUDA path.
@pytest.fixture(params=["difference", "textbook"])
def form(request):
    return request.param


# ------------------------------------------------------------------ O3 WENO5-JS
def test_weno_linear_data_exact(form):
    l, r = O.weno5_js([1, 2, 3, 4, 5], 1e-16, form=form)
    assert l == pytest.approx(3.5, abs=1e-14) and r == pytest.approx(2.5, abs=1e-14)
    l, r = O.weno5_js([7, 7, 7, 7, 7], 1e-16, form=form)
    assert l == pytest.approx(7.0, rel=4e-16) and r == pytest.approx(7.0, rel=4e-16)  # weights sum to 1 only to an ulp


def test_weno_ideal_weights_closed_form(form):
    # eps -> infinity switches the nonlinear weights to the ideal ones: the result must be the
    # 5th-order linear reconstruction (2,-13,47,27,-3)/60 (and its mirror) for ANY data
    rng = np.random.default_rng(3)
    for _ in range(50):
        s = rng.normal(size=5)
        l, r = O.weno5_js(s, 1e30, form=form)
        cl = np.array([2, -13, 47, 27, -3]) / 60.0
        assert l == pytest.approx(cl @ s, rel=1e-13, abs=1e-14)
        assert r == pytest.approx(cl[::-1] @ s, rel=1e-13, abs=1e-14)


def test_weno_candidates_each_reproduce_quadratics(form):
    # cell averages of x^2 on unit cells are i^2 + 1/12; all three smoothness indicators equal 13/3, so
    # the weights are ideal and the face values are the point values (+-1/2)^2 = 1/4
    s = np.array([4, 1, 0, 1, 4]) + 1.0 / 12.0
    l, r = O.weno5_js(s, 1e-16, form=form)
    assert l == pytest.approx(0.25, abs=1e-13) and r == pytest.approx(0.25, abs=1e-13)
    # cubic: x^3 cell averages = i^3 + i/4 ; exact point value at 1/2 is 1/8 for a 5th-order linear scheme
    i = np.arange(-2, 3)
    l, _ = O.weno5_js(i ** 3 + i / 4.0, 1e30, form=form)
    assert l == pytest.approx(0.125, abs=1e-13)


def test_weno_eno_property_at_step(form):
    # the stencil that avoids the jump wins: values stay at the smooth side's level
    l, r = O.weno5_js([0, 0, 0, 1, 1], 1e-16, form=form)
    assert abs(l) < 1e-12
    l, r = O.weno5_js([0, 0, 1, 1, 1], 1e-16, form=form)
    assert abs(r - 1.0) < 1e-12
    # jump weights against brute-force evaluation of the definition with fractions-like float math
    s = np.array([1.0, 1.0, 1.0, 3.0, 3.5])
    b = [13 / 12 * (s[0] - 2 * s[1] + s[2]) ** 2 + 0.25 * (s[0] - 4 * s[1] + 3 * s[2]) ** 2,
         13 / 12 * (s[1] - 2 * s[2] + s[3]) ** 2 + 0.25 * (s[1] - s[3]) ** 2,
         13 / 12 * (s[2] - 2 * s[3] + s[4]) ** 2 + 0.25 * (3 * s[2] - 4 * s[3] + s[4]) ** 2]
    eps = 1e-6
    al = np.array([0.1, 0.6, 0.3]) / (np.array(b) + eps) ** 2
    pl = np.array([(2 * s[0] - 7 * s[1] + 11 * s[2]) / 6, (-s[1] + 5 * s[2] + 2 * s[3]) / 6, (2 * s[2] + 5 * s[3] - s[4]) / 6])
    l, _ = O.weno5_js(s, eps, form=form)
    assert l == pytest.approx((al / al.sum()) @ pl, rel=1e-14)


def test_weno_mirror_symmetry(form):
    rng = np.random.default_rng(11)
    for _ in range(100):
        s = rng.normal(size=5) * 10 ** rng.uniform(-3, 3)
        l, r = O.weno5_js(s, 1e-10, form=form)
        l2, r2 = O.weno5_js(s[::-1].copy(), 1e-10, form=form)
        assert l == pytest.approx(r2, rel=1e-12) and r == pytest.approx(l2, rel=1e-12)


def test_weno_difference_form_is_the_textbook_form_and_rounds_to_half_an_ulp():
    # Reading N2: the oracle evaluates f = c + sum_r omega_r (f^(r) - c) with the candidate
    # deviations in first differences.  (i) It is the textbook sum_r omega_r f^(r) (Jiang-Shu
    # candidates) for arbitrary data, up to the rounding of that textbook evaluation; (ii) on smooth data with an
    # offset (a velocity field u0 + small variation) its fp64 result is within 1 ulp of the 80-bit evaluation —
    # the property the parity bar needs, because the low-Mach HLLC flux amplifies velocity rounding by rho*c.
    rng = np.random.default_rng(5)
    worst_ulp = 0.0
    for k in range(300):
        if k < 150:
            s = rng.normal(size=5) * 10 ** rng.uniform(-2, 2)
            eps = 1e-6
        else:
            x0, h = rng.uniform(0, 6.28), 10 ** rng.uniform(-3, -1)
            s = 10.0 + 3.0 * np.sin(x0 + h * np.arange(-2, 3))
            eps = 1e-16
        b = [13 / 12 * (s[0] - 2 * s[1] + s[2]) ** 2 + 0.25 * (s[0] - 4 * s[1] + 3 * s[2]) ** 2,
             13 / 12 * (s[1] - 2 * s[2] + s[3]) ** 2 + 0.25 * (s[1] - s[3]) ** 2,
             13 / 12 * (s[2] - 2 * s[3] + s[4]) ** 2 + 0.25 * (3 * s[2] - 4 * s[3] + s[4]) ** 2]
        al = np.array([0.1, 0.6, 0.3]) / (np.array(b) + eps) ** 2
        ar = np.array([0.3, 0.6, 0.1]) / (np.array(b) + eps) ** 2
        pl = np.array([(2 * s[0] - 7 * s[1] + 11 * s[2]) / 6, (-s[1] + 5 * s[2] + 2 * s[3]) / 6, (2 * s[2] + 5 * s[3] - s[4]) / 6])
        pr = np.array([(-s[0] + 5 * s[1] + 2 * s[2]) / 6, (2 * s[1] + 5 * s[2] - s[3]) / 6, (11 * s[2] - 7 * s[3] + 2 * s[4]) / 6])
        l, r = O.weno5_js(s, eps)
        scale = np.abs(s).max()
        assert abs(l - (al / al.sum()) @ pl) <= 2e-14 * scale and abs(r - (ar / ar.sum()) @ pr) <= 2e-14 * scale
        # the textbook instantiation IS this transcription (same operations up to the order of a sum): a few ulp
        lt, rt = O.weno5_js(s, eps, form="textbook")
        assert abs(lt - (al / al.sum()) @ pl) <= 2e-15 * scale and abs(rt - (ar / ar.sum()) @ pr) <= 2e-15 * scale
        if k >= 150:
            l80, r80 = O.weno5_js_ld(s, eps)
            worst_ulp = max(worst_ulp, abs(l - l80) / np.spacing(abs(l80)), abs(r - r80) / np.spacing(abs(r80)))
    assert worst_ulp <= 1.0, worst_ulp


def test_weno_fifth_order_on_cell_averaged_sine(form):
    # brute-force refinement: error of the face value against the exact point value
    errs = []
    Ns = [16, 32, 64, 128]
    for N in Ns:
        h = 1.0 / N
        xe = np.arange(N + 1) * h
        avg = (np.cos(2 * np.pi * xe[:-1]) - np.cos(2 * np.pi * xe[1:])) / (2 * np.pi * h) + 2.0  # mean of 2+sin(2 pi x)
        e = 0.0
        for i in range(N):
            s = avg[[(i + k) % N for k in range(-2, 3)]]
            l, r = O.weno5_js(s, 1e-6, form=form)
            e = max(e, abs(l - (2 + np.sin(2 * np.pi * xe[i + 1]))), abs(r - (2 + np.sin(2 * np.pi * xe[i]))))
        errs.append(e)
    rates = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert rates[-1] > 4.8 and rates[-2] > 4.5, (errs, rates)


# ------------------------------------------------------------------ O4 HLLC
def _phys_flux(case, w, d):
    """F(q) of the 5-equation model written straight from PAPER.md:59 for a primitive state"""
    N, D = case.nfluids, case.ndim
    rho = w[:N].sum()
    Gam = sum(w[N + D + 1 + i] / (case.gamma[i] - 1) for i in range(N))
    Pi = sum(w[N + D + 1 + i] * case.gamma[i] * case.pi_inf[i] / (case.gamma[i] - 1) for i in range(N))
    u = w[N:N + D]
    p = w[N + D]
    E = Gam * p + Pi + 0.5 * rho * (u @ u)
    F = np.empty(case.neq)
    F[:N] = w[:N] * u[d]
    F[N:N + D] = rho * u * u[d]
    F[N + d] += p
    F[N + D] = (E + p) * u[d]
    F[N + D + 1:] = w[N + D + 1:] * u[d]
    return F


def _rand_prim(case, rng, mach=0.3):
    N, D = case.nfluids, case.ndim
    a = rng.uniform(0.05, 1, N); a /= a.sum()
    w = np.empty(case.neq)
    w[:N] = a * np.array([1.0, 1000.0, 0.138])[:N] * rng.uniform(0.8, 1.2, N)
    w[N + D] = rng.uniform(0.5e5, 2e5)
    w[N + D + 1:] = a
    w[N:N + D] = rng.uniform(-1, 1, D) * mach * 300
    return w


@pytest.mark.parametrize("ndim,nfluids", [(1, 1), (2, 2), (3, 2), (3, 3)])
def test_hllc_consistency(ndim, nfluids, form):
    case = small_case(ndim, nfluids)
    orc = O.Oracle(case, form=form)
    rng = np.random.default_rng(5)
    for d in range(ndim):
        for _ in range(20):
            w = _rand_prim(case, rng)
            F, uf, bad = orc.hllc_face(d, w, w)
            ref = _phys_flux(case, w, d)
            assert bad == 0
            assert np.allclose(F, ref, rtol=1e-12, atol=1e-9 * np.abs(ref).max())
            assert uf == pytest.approx(w[nfluids + d], rel=1e-12, abs=1e-12)


def test_hllc_supersonic_upwinding(form):
    case = small_case(3, 2, gamma=(1.4, 1.67), pi_inf=(0.0, 0.0))
    orc = O.Oracle(case, form=form)
    rng = np.random.default_rng(9)
    for d in range(3):
        wL, wR = _rand_prim(case, rng), _rand_prim(case, rng)
        for sgn, up in ((+1, "L"), (-1, "R")):
            wL2, wR2 = wL.copy(), wR.copy()
            wL2[2 + d] = sgn * 5000.0   # |u| >> c (c ~ 400)
            wR2[2 + d] = sgn * 5200.0
            F, uf, _ = orc.hllc_face(d, wL2, wR2)
            ref = _phys_flux(case, wL2 if up == "L" else wR2, d)
            assert np.array_equal(F, ref) or np.allclose(F, ref, rtol=1e-15)
            assert uf == (wL2 if up == "L" else wR2)[2 + d]


def test_hllc_stationary_contact_exact(form):
    # u = 0, equal p, jump in density AND in fluid: the contact must be resolved exactly
    case = small_case(2, 2)
    orc = O.Oracle(case, form=form)
    p = 1.0e5
    wL = np.array([1.0e-6 * 1.0, (1 - 1e-6) * 1000.0, 0.0, 0.0, p, 1.0e-6, 1 - 1e-6])
    wR = np.array([(1 - 1e-6) * 1.0, 1e-6 * 1000.0, 0.0, 0.0, p, 1 - 1e-6, 1e-6])
    for d in range(2):
        F, uf, bad = orc.hllc_face(d, wL, wR)
        exp = np.zeros(7); exp[2 + d] = p
        assert bad == 0 and uf == 0.0
        assert np.array_equal(F, exp), F


def test_hllc_mirror_symmetry(form):
    case = small_case(3, 2)
    orc = O.Oracle(case, form=form)
    rng = np.random.default_rng(21)
    N = 2
    for d in range(3):
        for _ in range(20):
            wL, wR = _rand_prim(case, rng, mach=1.5), _rand_prim(case, rng, mach=1.5)
            F, uf, _ = orc.hllc_face(d, wL, wR)
            mL, mR = wR.copy(), wL.copy()
            mL[N + d] *= -1; mR[N + d] *= -1
            Fm, ufm, _ = orc.hllc_face(d, mL, mR)
            sign = -np.ones(case.neq); sign[N + d] = 1.0
            assert np.allclose(Fm, sign * F, rtol=1e-11, atol=1e-9 * np.abs(F).max())
            assert ufm == pytest.approx(-uf, rel=1e-11, abs=1e-9)


def test_hllc_matches_textbook_form_single_ideal_gas(form):
    """For one ideal gas the flux must equal the textbook HLLC written in its OTHER standard form,
    F*_K = [S*(S_K U_K - F_K) + S_K (p_K + rho_K (S_K-u_K)(S*-u_K)) D*] / (S_K - S*),  D* = (0, n, S*)
    (ref. [31] of the paper), with the same Davis wave speeds — catches a dropped or
    mis-signed term in the star state."""
    g = 1.4
    case = small_case(3, 1, gamma=(g,), pi_inf=(0.0,))
    orc = O.Oracle(case, form=form)
    rng = np.random.default_rng(2)
    seen = set()
    for trial in range(400):
        d = trial % 3
        def rp():
            return np.array([rng.uniform(0.1, 2), *(rng.uniform(-2, 2, 3) * rng.choice([0.2, 1, 3])), rng.uniform(0.1, 2), 1.0])
        wL, wR = rp(), rp()
        F, uf, bad = orc.hllc_face(d, wL, wR)
        def U_F(w):
            rho, u, p = w[0], w[1:4], w[4]
            E = p / (g - 1) + 0.5 * rho * (u @ u)
            U = np.array([rho, *(rho * u), E])
            Fl = U * u[d]; Fl[1 + d] += p; Fl[4] += p * u[d]
            return U, Fl, rho, u[d], p, np.sqrt(g * p / rho)
        UL, FL, rL, uL, pL, cL = U_F(wL)
        UR, FR, rR, uR, pR, cR = U_F(wR)
        SL, SR = min(uL - cL, uR - cR), max(uL + cL, uR + cR)
        Ss = (pR - pL + rL * uL * (SL - uL) - rR * uR * (SR - uR)) / (rL * (SL - uL) - rR * (SR - uR))
        Dn = np.zeros(5); Dn[1 + d] = 1.0; Dn[4] = Ss
        if SL >= 0: ref = FL; seen.add("L")
        elif Ss >= 0: ref = (Ss * (SL * UL - FL) + SL * (pL + rL * (SL - uL) * (Ss - uL)) * Dn) / (SL - Ss); seen.add("*L")
        elif SR > 0: ref = (Ss * (SR * UR - FR) + SR * (pR + rR * (SR - uR) * (Ss - uR)) * Dn) / (SR - Ss); seen.add("*R")
        else: ref = FR; seen.add("R")
        assert np.allclose(F[:5], ref, rtol=1e-11, atol=1e-11 * np.abs(ref).max()), (trial, F, ref)
        # volume fraction flux and face velocity: alpha == 1 is advected like a unit scalar (A7)
        assert F[5] == pytest.approx(uf, rel=1e-13, abs=1e-13)
        # in the star region the unit-scalar flux equals the mass flux / upwind density
        if SL < 0 < SR:
            rho_up = rL if Ss >= 0 else rR
            assert uf == pytest.approx(ref[0] / rho_up, rel=1e-11, abs=1e-11)
    assert seen == {"L", "*L", "*R", "R"}


def test_hllc_textbook_and_difference_forms_agree_on_stiffened_gas_faces():
    """Random two- and three-fluid faces with water (pi_inf = 6e8) in them, all four branches: the flux typed as
    F_K + S_K (q*_K - q_K) with the star state of PAPER.md:668 formed first equals the flux of reading N3 (chi - 1 formed
    directly) up to the rounding of the subtraction q*_K - q_K, i.e. a few ulp of S_K q_K — with stiff water a dropped term
    in the star energy is ten orders of magnitude above that."""
    rng = np.random.default_rng(31)
    seen = set()
    for nfl in (2, 3):
        case = small_case(3, nfl)
        d_orc, t_orc = O.Oracle(case), O.Oracle(case, form="textbook")
        N, D = nfl, 3
        for trial in range(300):
            d = trial % 3
            wL, wR = _rand_prim(case, rng, mach=rng.choice([0.1, 1.0, 8.0])), _rand_prim(case, rng, mach=rng.choice([0.1, 1.0, 8.0]))
            if trial % 4 == 0:      # supersonic either way: the non-star branches
                s = rng.choice([-1.0, 1.0]) * 9000.0
                wL[N + d], wR[N + d] = s, 1.05 * s
            Fd, ufd, bd = d_orc.hllc_face(d, wL, wR)
            Ft, uft, bt = t_orc.hllc_face(d, wL, wR)
            assert bd == 0 and bt == 0
            # magnitudes: |S| <= |u| + c, q_K the conserved state of the two sides
            smax, qmag = 0.0, np.zeros(case.neq)
            for w in (wL, wR):
                rho = w[:N].sum()
                Gam = sum(w[N + D + 1 + i] / (case.gamma[i] - 1) for i in range(N))
                Pi = sum(w[N + D + 1 + i] * case.gamma[i] * case.pi_inf[i] / (case.gamma[i] - 1) for i in range(N))
                c = np.sqrt(((Gam + 1) * w[N + D] + Pi) / (Gam * rho))
                smax = max(smax, abs(w[N + d]) + c)
                qc = w.copy()
                qc[N:N + D] = rho * np.abs(w[N:N + D]) + rho * c
                qc[N + D] = Gam * w[N + D] + Pi + 0.5 * rho * (w[N:N + D] @ w[N:N + D])
                qmag = np.maximum(qmag, np.abs(qc))
            tol = 1e-13 * np.maximum(np.abs(Fd), smax * qmag)
            assert np.all(np.abs(Ft - Fd) <= tol), (trial, Ft - Fd, tol)
            assert abs(uft - ufd) <= 1e-13 * smax
            pure = ufd == wL[N + d] or ufd == wR[N + d]     # outside the fan the face velocity is the upwind side's own
            seen.add(("pure" if pure else "star", ufd >= 0))
    assert len(seen) == 4, seen


# ------------------------------------------------------------------ A9, A10 (definitions only: parity unpinned by the paper)
def test_cfl_dt_closed_form_uniform_state():
    case = small_case(3, 2, n=4)
    case = W.replace(case, dx=(0.1, 0.2, 0.4))
    a = np.array([0.3, 0.7]); rho0 = np.array([1.0, 1000.0]); p = 2.0e5; u = np.array([3.0, -40.0, 5.0])
    sh = case.shape[1:]
    q = W.cons_from_prim(case, [np.full(sh, a[i] * rho0[i]) for i in range(2)], [np.full(sh, x) for x in u], p, [np.full(sh, x) for x in a])
    Gam = (a / (np.array(case.gamma) - 1)).sum(); Pi = (a * np.array(case.gamma) * np.array(case.pi_inf) / (np.array(case.gamma) - 1)).sum()
    c = np.sqrt(((Gam + 1) * p + Pi) / (Gam * (a * rho0).sum()))
    expect = 0.5 / sum((abs(u[d]) + c) / case.dx[d] for d in range(3))
    assert O.Oracle(case).cfl_dt(q, 0.5) == pytest.approx(expect, rel=1e-9)


def test_sound_speed_reduces_to_eq6_for_pure_fluid():
    # (A5) with alpha=(1) : c^2 = gamma (p + pi_inf)/rho  (eq.(6)); read back through cfl_dt in 1-D with u=0
    g, pinf, rho, p = 4.4, 6.0e8, 1000.0, 1.0e5
    case = small_case(1, 1, n=4, gamma=(g,), pi_inf=(pinf,))
    sh = case.shape[1:]
    q = W.cons_from_prim(case, [np.full(sh, rho)], [np.zeros(sh)], p, [np.ones(sh)])
    dt = O.Oracle(case).cfl_dt(q, 1.0)
    assert case.dx[0] / dt == pytest.approx(np.sqrt(g * (p + pinf) / rho), rel=1e-9)


def test_clamp_definition():
    case = W.replace(small_case(1, 3, n=4), clamp=True, alpha_floor=1e-6)
    orc = O.Oracle(case)
    # inside bounds: untouched bit for bit
    q = np.array([0.5, 300.0, 0.01, 12.0, 5e8, 0.5, 0.3, 0.2])
    assert np.array_equal(orc.clamp_cell(q), q)
    # below the floor: floored, renormalised; momentum/energy untouched; negative partial density -> 0
    q2 = np.array([-1e-9, 300.0, 0.01, 12.0, 5e8, -3e-7, 0.7, 0.3 + 3e-7])
    c = orc.clamp_cell(q2)
    assert c[0] == 0.0 and c[3] == 12.0 and c[4] == 5e8 and c[1] == 300.0
    assert c[5:].sum() == pytest.approx(1.0, abs=1e-15)
    assert c[5] == pytest.approx(1e-6 / (1e-6 + 0.7 + 0.3 + 3e-7), rel=1e-14)
    assert (c[5:] >= 1e-6 / (1 + 3e-6)).all()
