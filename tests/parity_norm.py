"""The error measure of the parity bar: for each variable v the max-norm relative error
    e_v = max|gpu_v - oracle_v| / max|oracle_v|,
the bar being  max_v e_v <= tol.  Every partial density, the energy and every volume fraction is measured against its OWN
largest magnitude (air ~1 is not measured against water ~1000).  The one exception is the momentum group: a momentum
component may vanish identically by symmetry (config 3's rho*v at t = 0 away from the bubble, the transverse components of
every 1-D-like flow) and is then nothing but round-off, so the momentum components — components of one vector — are scaled
by the largest magnitude over the momentum GROUP.  `rel_err` returns that figure; `rel_err_both` also returns the looser
all-groups figure of round 1 for comparison.

Rounding noise of the reference.  The fp64 oracle is itself only one rounding of its definition: it differs from the same
text evaluated in 80-bit arithmetic (oracle_rhs_ld) by n64_v = max|o64_v - o80_v|.  Where the volume-fraction rows of the
reference are analytically zero — one fluid (alpha == 1), or uniform alpha wherever the fluid moves (configs 3 and 5 at
t = 0: the bubble / droplet is at rest ahead of the shock) — d(alpha)/dt is the round-off of two cancelling terms of size
|u|/dx, the whole reference IS rounding noise and a relative measure has no meaning.  The same holds for the partial
density of a fluid that is at rest wherever it is more than a trace (the light gas of configs 3 and 5 at t = 0: its
d(alpha rho)/dt is of trace size, 1e-6 rho_i |du|/dx at the shock, while the round-off of the resting bubble / slab
interface, where alpha_i rho_i is 10^5 times larger, is 1e-9 of that — measured, DESIGN.md §7 reading T2).  Tests that
pass `noise=` (they say why) must also name the rows that may take the allowance (`allow=`, built by `t2_rows`): the
volume fractions, and the partial density of a fluid that reading T2 names as a trace fluid at rest — nothing else.  For
those rows max|gpu - o64| <= tol*scale + 4*n64.  Every other partial density (with one fluid alpha_1 rho_1 IS the density:
real signal), momentum and energy, and every test that does not pass `noise=`, are held to the bare relative bar.
`rel_err_report` gives the figures with and without the allowance side by side for the test's failure message."""
import numpy as np


def groups(nfluids, ndim):
    N, D = nfluids, ndim
    return [list(range(0, N)), list(range(N, N + D)), [N + D], list(range(N + D + 1, 2 * N + D + 1))]


def var_names(nfluids, ndim):
    N, D = nfluids, ndim
    return ([f"arho{i + 1}" for i in range(N)] + [f"mom_{'xyz'[d]}" for d in range(D)] + ["E"] + [f"alpha{i + 1}" for i in range(N)])


def group_noise(ref, ref_ld, nfluids, ndim):
    """per-variable max|o64 - o80|: the rounding noise of the fp64 reference"""
    return [float(np.abs(ref[v] - ref_ld[v]).max()) for v in range(ref.shape[0])]


def _scales(ref, nfluids, ndim, by_group):
    sc = [0.0] * ref.shape[0]
    for gi, g in enumerate(groups(nfluids, ndim)):
        gmax = max(float(np.abs(ref[g]).max()), 1e-300)
        for v in g:
            sc[v] = gmax if (by_group or gi == 1) else max(float(np.abs(ref[v]).max()), 1e-300)
    return sc


def t2_rows(nfluids, ndim, trace_fluids=()):
    """rows that may take the noise allowance (DESIGN.md §7 reading T2): every volume fraction, and the partial density of
    each fluid in `trace_fluids` (0-based; the light gas of configs 3 and 5 at t = 0)"""
    N, D = nfluids, ndim
    for i in trace_fluids:
        assert 0 <= i < N
    return frozenset(range(N + D + 1, 2 * N + D + 1)) | frozenset(trace_fluids)


def case_t2_rows(case):
    """t2_rows of a BASELINE configuration at t = 0, by the case's name: config 3 -> fluid 1, config 5 -> fluid 2 (the light gas)"""
    trace = {"3": (1,), "5": (2,)}.get(case.name.split(":")[0], ())
    return t2_rows(case.nfluids, case.ndim, trace)


def _errs(a, ref, nfluids, ndim, noise, by_group, allow=None):
    sc = _scales(ref, nfluids, ndim, by_group)
    if noise is not None and allow is None:
        raise ValueError("a test that passes noise= must name the rows that may take the allowance (allow=t2_rows(...))")
    allowed = frozenset(allow) if noise is not None else frozenset()
    assert allowed <= t2_rows(nfluids, ndim, range(nfluids)), "only volume fractions and partial densities can be T2 rows"
    per = []
    for v in range(ref.shape[0]):
        give = 4.0 * noise[v] if v in allowed else 0.0
        per.append(max(float(np.abs(a[v] - ref[v]).max()) - give, 0.0) / sc[v])
    return per


def rel_err(a, ref, nfluids, ndim, noise=None, allow=None):
    """(worst, {variable name: e_v}) with e_v per variable (momentum components: per group); see the module text"""
    per = _errs(a, ref, nfluids, ndim, noise, False, allow)
    return max(per), dict(zip(var_names(nfluids, ndim), (float("%.3g" % e) for e in per)))


def rel_err_both(a, ref, nfluids, ndim, noise=None, allow=None):
    """(per-variable figure, all-groups figure of round 1)"""
    return (max(_errs(a, ref, nfluids, ndim, noise, False, allow)), max(_errs(a, ref, nfluids, ndim, noise, True, allow)))


def rel_err_report(a, ref, nfluids, ndim, noise, allow):
    """{variable: (e_v with the allowance, e_v without it, 4 n64_v / scale_v, allowed?)} — what a noise-passing test prints"""
    w = _errs(a, ref, nfluids, ndim, noise, False, allow)
    wo = _errs(a, ref, nfluids, ndim, None, False)
    sc = _scales(ref, nfluids, ndim, False)
    return {name: (float("%.3g" % w[v]), float("%.3g" % wo[v]), float("%.3g" % (4.0 * noise[v] / sc[v])), v in frozenset(allow))
            for v, name in enumerate(var_names(nfluids, ndim))}
