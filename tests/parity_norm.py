"""The error measure of the parity bar: max-norm relative error per variable,
each variable scaled by the largest magnitude within its GROUP (partial densities / momenta /
energy / volume fractions).  Grouping the momentum components keeps a component that vanishes by
symmetry (config 3's rho*v, every 1-D transverse direction) from being measured against round-off."""
import numpy as np


def groups(nfluids, ndim):
    N, D = nfluids, ndim
    return [list(range(0, N)), list(range(N, N + D)), [N + D], list(range(N + D + 1, 2 * N + D + 1))]


def rel_err(a, ref, nfluids, ndim):
    """max over variables of max|a-ref| / max_group|ref|; returns (worst, per-variable list)"""
    per = []
    for g in groups(nfluids, ndim):
        scale = max(float(np.abs(ref[g]).max()), 1e-300)
        for v in g:
            per.append(float(np.abs(a[v] - ref[v]).max()) / scale)
    return max(per), per
