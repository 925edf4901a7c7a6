"""Seeded synthetic inputs for the MFC hot path (DESIGN.md §4 "input recipe").

This module serves BOTH the CPU oracle and the CUDA path (tests, bench.py, smoke) and
therefore holds none of the method's arithmetic: no reconstruction, no Riemann solver, no
RHS, no time stepping.  The one physics formula here is the definition of the conservative
input state from the primitive fields an initial condition is written in (eq.(4)
and PAPER.md:117: rho e = sum_i alpha_i (p + gamma_i pi_inf_i)/(gamma_i - 1)) — that is the
inverse of the path's first step, needed to *state* an input, and neither the oracle nor the
CUDA library calls it.

The paper's workloads are full MFC cases on up to 8 B cells and the
8-PDE 3D benchmark case; none of them ships with the paper, so these inputs
take their shapes and stand in for them.  Nothing is read from disk; every field is a closed
form of the cell-centre coordinates and of a splitmix64 stream seeded by `seed`.
"""
from dataclasses import dataclass, field, replace
from typing import Tuple

import numpy as np

BC_PERIODIC, BC_EXTRAP = 0, 1
DEFAULT_SEED = 20250307


@dataclass
class Case:
    name: str
    ndim: int
    n: Tuple[int, int, int]
    dx: Tuple[float, float, float]
    nfluids: int
    gamma: Tuple[float, ...]
    pi_inf: Tuple[float, ...]
    bc_lo: Tuple[int, int, int]
    bc_hi: Tuple[int, int, int]
    weno_eps: float = 1e-16
    alpha_floor: float = 1e-6
    clamp: bool = True
    cfl: float = 0.5
    nsteps: int = 0          # number of RK3 steps of the configuration (0: run to t_end)
    t_end: float = 0.0
    seed: int = DEFAULT_SEED
    builder: str = ""        # which generator below makes q0
    model: str = "allaire"   # volume-fraction equation: "allaire" (no K div u) or "kapila" (eq. 5; two fluids)
    eta: float = 0.0         # uniform shear viscosity of PAPER.md eq.(1); 0 = inviscid (all five configurations)
    weno: str = "js"         # nonlinear weights: "js" (BASELINE.json), "m" (mapped), "z"
    shock_x: float = -1.0    # config 5 only: position of the incident shock; < 0 = the configuration's own (0.2).  Tests move it
                             # next to the droplet (surface at x = 0.30) to sample a state in which the two already interact

    @property
    def neq(self):
        return 2 * self.nfluids + self.ndim + 1

    @property
    def cells(self):
        return self.n[0] * self.n[1] * self.n[2]

    @property
    def shape(self):
        """q[v, k, j, i] — SoA, x fastest (idx = ((v*nz+k)*ny+j)*nx+i)."""
        return (self.neq, self.n[2], self.n[1], self.n[0])


# ----------------------------------------------------------------------------- RNG
class SplitMix64:
    """Counter-based 64-bit generator (public-domain splitmix64 recurrence)."""

    def __init__(self, seed):
        self.state = np.uint64(seed)

    def next_u64(self, count):
        with np.errstate(over="ignore"):
            inc = np.uint64(0x9E3779B97F4A7C15)
            z = self.state + inc * np.arange(1, count + 1, dtype=np.uint64)
            self.state = z[-1] if count else self.state
            z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
            z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
            return z ^ (z >> np.uint64(31))

    def uniform(self, count, lo=0.0, hi=1.0):
        u = (self.next_u64(count) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)
        return lo + (hi - lo) * u


# ----------------------------------------------------------------------------- state assembly
def cons_from_prim(case, arho, u, p, alpha):
    """Conservative input state from primitive fields (lists of arrays broadcastable to the grid)."""
    N, D = case.nfluids, case.ndim
    shape3 = case.shape[1:]
    q = np.empty(case.shape, dtype=np.float64)
    rho = np.zeros(shape3)
    Gam = np.zeros(shape3)
    Pi = np.zeros(shape3)
    for i in range(N):
        q[i] = arho[i]
        q[N + D + 1 + i] = alpha[i]
        rho += q[i]
        Gam += q[N + D + 1 + i] / (case.gamma[i] - 1.0)
        Pi += q[N + D + 1 + i] * case.gamma[i] * case.pi_inf[i] / (case.gamma[i] - 1.0)
    usq = np.zeros(shape3)
    for d in range(D):
        ud = np.broadcast_to(np.asarray(u[d], dtype=np.float64), shape3)
        q[N + d] = rho * ud
        usq += ud * ud
    q[N + D] = Gam * p + Pi + 0.5 * rho * usq
    return q


def centres(case):
    """cell-centre coordinates as broadcastable arrays X[1,1,nx], Y[1,ny,1], Z[nz,1,1]"""
    x = (np.arange(case.n[0]) + 0.5) * case.dx[0]
    y = (np.arange(case.n[1]) + 0.5) * case.dx[1]
    z = (np.arange(case.n[2]) + 0.5) * case.dx[2]
    return x[None, None, :], y[None, :, None], z[:, None, None]


def _clip_alpha(case, a):
    return np.clip(a, case.alpha_floor, 1.0 - (case.nfluids - 1) * case.alpha_floor)


def _normal_shock(gamma, mach, rho0, p0):
    """Rankine-Hugoniot post-shock state of an ideal gas at rest hit by a Mach-`mach` shock."""
    c0 = np.sqrt(gamma * p0 / rho0)
    pr = 1.0 + 2.0 * gamma * (mach * mach - 1.0) / (gamma + 1.0)
    rr = (gamma + 1.0) * mach * mach / ((gamma - 1.0) * mach * mach + 2.0)
    return rho0 * rr, mach * c0 * (1.0 - 1.0 / rr), p0 * pr


# ----------------------------------------------------------------------------- the five configurations
def _build_sod(case):
    X, _, _ = centres(case)
    left = np.broadcast_to(X < 0.5, case.shape[1:])
    rho = np.where(left, 1.0, 0.125)
    p = np.where(left, 1.0, 0.1)
    return cons_from_prim(case, [rho], [0.0], p, [np.ones(case.shape[1:])])


def _build_water_air_tube(case):
    X, _, _ = centres(case)
    left = np.broadcast_to(X < 0.5, case.shape[1:])
    f = case.alpha_floor
    a_w = np.where(left, 1.0 - f, f)
    a_a = 1.0 - a_w
    p = np.where(left, 1.0e9, 1.0e5)
    return cons_from_prim(case, [a_w * 1000.0, a_a * 1.0], [0.0], p, [a_w, a_a])


def _build_shock_bubble_2d(case):
    X, Y, _ = centres(case)
    r = np.sqrt((X - 0.5) ** 2 + (Y - 0.5) ** 2)
    a_l = _clip_alpha(case, 0.5 * (1.0 - np.tanh((r - 0.2) / (2.0 * case.dx[0]))))
    a_l = np.broadcast_to(a_l, case.shape[1:]).copy()
    a_a = 1.0 - a_l
    rho1, u1, p1 = _normal_shock(1.4, 1.22, 1.0, 1.0)
    post = np.broadcast_to(X < 0.25, case.shape[1:])
    rho_air = np.where(post, rho1, 1.0)
    ux = np.where(post, u1, 0.0)
    p = np.where(post, p1, 1.0)
    return cons_from_prim(case, [a_a * rho_air, a_l * 0.138], [ux, 0.0], p, [a_a, a_l])


def _build_mixing_3d(case):
    rng = SplitMix64(case.seed)
    X, Y, Z = centres(case)
    L = [case.n[d] * case.dx[d] for d in range(3)]
    nblob = 32
    cx = rng.uniform(nblob) * L[0]
    cy = rng.uniform(nblob) * L[1]
    cz = rng.uniform(nblob) * L[2]
    R = rng.uniform(nblob, 0.05, 0.12) * L[0]
    a_w = np.zeros(case.shape[1:])
    for b in range(nblob):
        ddx = np.abs(X - cx[b]); ddx = np.minimum(ddx, L[0] - ddx)
        ddy = np.abs(Y - cy[b]); ddy = np.minimum(ddy, L[1] - ddy)
        ddz = np.abs(Z - cz[b]); ddz = np.minimum(ddz, L[2] - ddz)
        r = np.sqrt(ddx ** 2 + ddy ** 2 + ddz ** 2)
        np.maximum(a_w, 0.5 * (1.0 - np.tanh((r - R[b]) / (2.0 * case.dx[0]))), out=a_w)
    a_w = _clip_alpha(case, a_w)
    a_a = 1.0 - a_w
    nmode = 16
    u = []
    for d in range(3):
        ud = np.zeros(case.shape[1:])
        kk = np.floor(rng.uniform(3 * nmode, -4.0, 5.0)).astype(np.int64).reshape(nmode, 3)
        kk = np.clip(kk, -4, 4)
        kk[np.all(kk == 0, axis=1), 0] = 1
        amp = rng.uniform(nmode, -1.0, 1.0)
        ph = rng.uniform(nmode, 0.0, 2.0 * np.pi)
        for m in range(nmode):
            ex = np.exp(2j * np.pi * kk[m, 0] * X / L[0])
            ey = np.exp(2j * np.pi * kk[m, 1] * Y / L[1])
            ez = np.exp(2j * np.pi * kk[m, 2] * Z / L[2])
            ud += amp[m] * ((ex * ey) * (ez * np.exp(1j * ph[m]))).real
        u.append(ud)
    umax = np.sqrt(u[0] ** 2 + u[1] ** 2 + u[2] ** 2).max()
    u = [ud * (10.0 / umax) for ud in u]
    # fluid 0 = air, fluid 1 = water
    return cons_from_prim(case, [a_a * 1.0, a_w * 1000.0], u, 1.0e5, [a_a, a_w])


def _build_shock_droplet_3d(case):
    X, Y, Z = centres(case)
    f = case.alpha_floor
    w = 2.0 * case.dx[0]
    r = np.sqrt((X - 0.45) ** 2 + (Y - 0.5) ** 2 + (Z - 0.5) ** 2)
    a_w = np.clip(0.5 * (1.0 - np.tanh((r - 0.15) / w)), f, 1.0 - 2.0 * f)
    slab = 0.25 * (1.0 + np.tanh((X - 0.70) / w)) * (1.0 - np.tanh((X - 0.85) / w))
    a_l = np.clip(np.minimum(np.broadcast_to(slab, case.shape[1:]), 1.0 - a_w - f), f, None)
    a_a = 1.0 - a_w - a_l
    rho1, u1, p1 = _normal_shock(1.4, 1.5, 1.0, 1.0e5)
    post = np.broadcast_to(X < (case.shock_x if case.shock_x >= 0.0 else 0.2), case.shape[1:])
    rho_air = np.where(post, rho1, 1.0)
    ux = np.where(post, u1, 0.0)
    p = np.where(post, p1, 1.0e5)
    # fluid 0 = air, 1 = water, 2 = light gas
    return cons_from_prim(case, [a_a * rho_air, a_w * 1000.0, a_l * 0.138], [ux, 0.0, 0.0], p, [a_a, a_w, a_l])


_BUILDERS = {
    "sod": _build_sod,
    "water_air_tube": _build_water_air_tube,
    "shock_bubble_2d": _build_shock_bubble_2d,
    "mixing_3d": _build_mixing_3d,
    "shock_droplet_3d": _build_shock_droplet_3d,
}

_E, _P = BC_EXTRAP, BC_PERIODIC


def config(index, n=None, seed=DEFAULT_SEED):
    """BASELINE.json configs[index-1] (index = 1..5).  `n` overrides the cells per direction
    (same domain, same shapes measured in cells) for the down-scaled parity cases."""
    if index == 1:
        nx = n or 1000
        return Case("1:sod_1d", 1, (nx, 1, 1), (1.0 / nx, 1.0, 1.0), 1, (1.4,), (0.0,), (_E,) * 3, (_E,) * 3,
                    nsteps=0, t_end=0.2, seed=seed, builder="sod")
    if index == 2:
        nx = n or 4000
        return Case("2:water_air_tube_1d", 1, (nx, 1, 1), (1.0 / nx, 1.0, 1.0), 2, (4.4, 1.4), (6.0e8, 0.0),
                    (_E,) * 3, (_E,) * 3, nsteps=500, seed=seed, builder="water_air_tube")
    if index == 3:
        nx = n or 1024
        return Case("3:shock_bubble_2d", 2, (nx, nx, 1), (1.0 / nx, 1.0 / nx, 1.0), 2, (1.4, 1.67), (0.0, 0.0),
                    (_E,) * 3, (_E,) * 3, nsteps=200, seed=seed, builder="shock_bubble_2d")
    if index == 4:
        nx = n or 256
        return Case("4:mixing_3d", 3, (nx, nx, nx), (1.0 / nx,) * 3, 2, (1.4, 4.4), (0.0, 6.0e8),
                    (_P,) * 3, (_P,) * 3, nsteps=50, seed=seed, builder="mixing_3d")
    if index == 5:
        nx = n or 512
        return Case("5:shock_droplet_3d", 3, (nx, nx, nx), (1.0 / nx,) * 3, 3, (1.4, 4.4, 1.67), (0.0, 6.0e8, 0.0),
                    (_E,) * 3, (_E,) * 3, nsteps=20, seed=seed, builder="shock_droplet_3d")
    raise ValueError("config index must be 1..5")


def taylor_green(n=64, mach=0.1, reynolds=1600.0):
    """The shape of the paper's viscous example (three-dimensional Taylor-Green vortex): single ideal gas on
    the periodic box [0, 2 pi]^3, u = V0 (sin x cos y cos z, -cos x sin y cos z, 0),
    p = p0 + rho0 V0^2/16 (cos 2x + cos 2y)(cos 2z + 2), rho = rho0; V0 = mach * sqrt(gamma p0/rho0), eta = rho0 V0 / reynolds
    (reference length 1).  Closed form, no random numbers."""
    L = 2.0 * np.pi
    gamma, rho0, p0 = 1.4, 1.0, 1.0
    v0 = mach * np.sqrt(gamma * p0 / rho0)
    return Case("taylor_green_3d", 3, (n, n, n), (L / n,) * 3, 1, (gamma,), (0.0,), (_P,) * 3, (_P,) * 3, clamp=False,
                nsteps=0, builder="taylor_green", eta=rho0 * v0 / reynolds, t_end=mach)


def _build_taylor_green(case):
    X, Y, Z = centres(case)
    gamma, rho0, p0 = case.gamma[0], 1.0, 1.0
    v0 = case.t_end * np.sqrt(gamma * p0 / rho0)  # t_end carries the Mach number of the case
    shape3 = case.shape[1:]
    u = v0 * np.sin(X) * np.cos(Y) * np.cos(Z)
    v = -v0 * np.cos(X) * np.sin(Y) * np.cos(Z)
    p = p0 + rho0 * v0 * v0 / 16.0 * (np.cos(2 * X) + np.cos(2 * Y)) * (np.cos(2 * Z) + 2.0)
    rho = np.full(shape3, rho0)
    return cons_from_prim(case, [rho], [np.broadcast_to(u, shape3), np.broadcast_to(v, shape3), 0.0],
                          np.broadcast_to(p, shape3), [np.ones(shape3)])


_BUILDERS["taylor_green"] = _build_taylor_green


def initial_state(case):
    """q0 as a C-contiguous float64 array of shape case.shape."""
    return np.ascontiguousarray(_BUILDERS[case.builder](case))


def random_admissible_state(case, seed=DEFAULT_SEED, rough=1.0, alpha_lo=0.05):
    """Seeded random admissible state (positive densities/pressure, alpha in bounds, sum alpha = 1):
    cell-wise independent values — the roughest possible input, used by unit parity tests."""
    rng = SplitMix64(seed)
    N, D = case.nfluids, case.ndim
    shape3 = case.shape[1:]
    cells = case.cells
    raw = [rng.uniform(cells, alpha_lo, 1.0).reshape(shape3) for _ in range(N)]
    s = sum(raw)
    alpha = [_clip_alpha(case, r / s) for r in raw]
    s = sum(alpha)
    alpha = [a / s for a in alpha]
    rho0 = [1.0, 1000.0, 0.138, 10.0]
    arho = [alpha[i] * rho0[i] * (1.0 + 0.2 * rough * (rng.uniform(cells).reshape(shape3) - 0.5)) for i in range(N)]
    u = [30.0 * rough * (rng.uniform(cells).reshape(shape3) - 0.5) for _ in range(D)]
    p = 1.0e5 * (1.0 + 0.5 * rough * (rng.uniform(cells).reshape(shape3) - 0.5))
    return np.ascontiguousarray(cons_from_prim(case, arho, u, p, alpha))
