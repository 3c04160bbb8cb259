"""The five BASELINE.json configs (C1..C5) as seeded synthetic problems.

`scale` shrinks the base grid by an integer factor with the same recipe (used by the CPU tests and
by parity cases the oracle finishes in seconds); scale=1 is the size BASELINE.json names.
Recipes and the readings they rest on: DESIGN.md "Synthetic inputs".
"""
import os
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field

import numpy as np

from .fields import hash_normal, lognormal_density, prim_to_cons, trilinear_sample, velocity_field
from .mesh import Tree, blockify, tree_from_criterion, uniform_tree

N = 8
SEED = 20260421
CONFIG_NAMES = ("C1", "C2", "C3", "C4", "C5")
# C5: density contrast (relative to the mean) above which a level-0 block is refined; level l uses
# RHO_C5 * 4^l (Jeans length < 8 cells with G = c_s = 1 after the amplitude normalisation of
# DESIGN.md reading R22).  Calibrated once (seed SEED+30) so that the padded tree of the full-size case
# has ~1.8e5 blocks (census 32768 / 114672 / 30928 / 3504 / 136 = 182008).  The shrunken parity cases
# use RHO_C5_SMALL: their base fields have less dynamic range, and the lower threshold keeps all four
# refinement levels populated.
RHO_C5 = 8.0
RHO_C5_SMALL = 1.30


def _pmap(fn, items):
    """fn over items on the host cores (numpy releases the GIL in the gathers and ufuncs that dominate here);
    results in order, bit-identical to the serial loop."""
    items = list(items)
    workers = min(len(items), len(os.sched_getaffinity(0)))
    if workers <= 1:
        return [fn(x) for x in items]
    with ThreadPoolExecutor(workers) as ex:
        return list(ex.map(fn, items))


@dataclass
class Problem:
    name: str
    nb0: tuple
    max_level: int
    bc: tuple              # ((lo,hi),)*3 ; 0 periodic, 1 outflow
    box_len: tuple
    gamma: float
    cfl: float
    mode: int              # 0 synchronous, 1 adaptive (level-by-level) time steps
    nsteps: int            # coarse steps
    level: np.ndarray
    ijk: np.ndarray
    U: np.ndarray          # [nb][5][8][8][8]
    notes: dict = field(default_factory=dict)

    @property
    def nblocks(self):
        return len(self.level)

    def census(self):
        return [int((self.level == l).sum()) for l in range(self.max_level + 1)]


def cell_centres(level, ijk, nb0):
    """x,y,z [nb,8,8,8] (indexed [b][k][j][i]) of cell centres in the unit box (cubic cells)."""
    n = (nb0[0] * N) * (2.0 ** level.astype(np.float64))
    c = (np.arange(N) + 0.5)
    x = (ijk[:, 0, None] * N + c[None, :]) / n[:, None]
    y = (ijk[:, 1, None] * N + c[None, :]) / n[:, None]
    z = (ijk[:, 2, None] * N + c[None, :]) / n[:, None]
    nb = len(level)
    X = np.broadcast_to(x[:, None, None, :], (nb, N, N, N))
    Y = np.broadcast_to(y[:, None, :, None], (nb, N, N, N))
    Z = np.broadcast_to(z[:, :, None, None], (nb, N, N, N))
    return X, Y, Z


def global_indices(level, ijk):
    c = np.arange(N)
    nb = len(level)
    I = np.broadcast_to((ijk[:, 0, None] * N + c)[:, None, None, :], (nb, N, N, N))
    J = np.broadcast_to((ijk[:, 1, None] * N + c)[:, None, :, None], (nb, N, N, N))
    K = np.broadcast_to((ijk[:, 2, None] * N + c)[:, :, None, None], (nb, N, N, N))
    return I, J, K


def sod(nb=4, gamma=1.4, axis=0, x0=0.5, nsteps=20, slab=False):
    """C1: Sod tube along `axis`, outflow boundaries, unit length along the tube (BASELINE.json
    configs[0]; reading R19).  slab=True keeps one block across the tube (a 1-D problem)."""
    nb0 = [1 if slab else nb] * 3
    nb0[axis] = nb
    nb0 = tuple(nb0)
    t = uniform_tree(nb0, 0, (False, False, False))
    level, ijk = t.block_list()
    X = (ijk[:, axis, None] * N + np.arange(N) + 0.5) / (nb * N)
    shape = [len(level), 1, 1, 1]
    shape[3 - axis] = N
    X = np.broadcast_to(X.reshape(shape), (len(level), N, N, N))
    left = X < x0
    rho = np.where(left, 1.0, 0.125)
    P = np.where(left, 1.0, 0.1)
    zero = np.zeros_like(rho)
    U = prim_to_cons(rho, zero, zero, zero, P, gamma)
    box = tuple(n / nb for n in nb0)
    return Problem("C1", nb0, 0, ((1, 1),) * 3, box, gamma, 0.4, 0, nsteps, level, ijk, U,
                   {"workload": "Sod tube %dx%dx%d cells, outflow, gamma=%g" % (nb0[0] * N, nb0[1] * N, nb0[2] * N, gamma)})


def turbulent_box(name, n, mach, seed, nsteps=10, gamma=5.0 / 3.0, sigma=1.0):
    """C2/C3: periodic uniform n^3, lognormal density, k^-4 velocity at rms Mach `mach`, P = 1/gamma."""
    nb = n // N
    rho, v = _pmap(lambda k: lognormal_density(n, sigma, seed) if k == 0 else velocity_field(n, mach, seed + 1), (0, 1))
    t = uniform_tree((nb, nb, nb), 0)
    level, ijk = t.block_list()
    b = [blockify(a, (nb, nb, nb)) for a in (rho, v[0], v[1], v[2])]
    del rho, v
    U = prim_to_cons(b[0], b[1], b[2], b[3], np.full_like(b[0], 1.0 / gamma), gamma)
    return Problem(name, (nb, nb, nb), 0, ((0, 0),) * 3, (1.0, 1.0, 1.0), gamma, 0.4, 0, nsteps, level, ijk, U,
                   {"workload": "periodic uniform %d^3, lognormal rho, k^-4 v, Mach %g" % (n, mach)})


def amr_sphere(nb=16, nsteps=10, seed=SEED + 20, noise=0.01, max_level=3, mode=1):
    """C4: centrally condensed sphere, rho = 1/(1+(r/0.05)^2) + 0.01, refine level l where any cell
    has rho > 4^(l-3) (reading R20), v = noise * N(0,1) (counter-based), P = 0.1, periodic."""
    gamma = 5.0 / 3.0
    nb0 = (nb, nb, nb)

    def rho_fn(x, y, z):
        r2 = (x - 0.5) ** 2 + (y - 0.5) ** 2 + (z - 0.5) ** 2
        return 1.0 / (1.0 + r2 / 0.05 ** 2) + 0.01

    def flag(l, idx):
        lev = np.full(len(idx), l, dtype=np.int32)
        out = np.zeros(len(idx), dtype=bool)

        def chunk(s):
            X, Y, Z = cell_centres(lev[s:s + 2048], idx[s:s + 2048], nb0)
            out[s:s + 2048] = (rho_fn(X, Y, Z) > 4.0 ** (l - 3)).reshape(len(X), -1).any(axis=1)
        _pmap(chunk, range(0, len(idx), 2048))
        return out

    t = tree_from_criterion(nb0, max_level, (True, True, True), flag)
    level, ijk = t.block_list()
    U = np.empty((len(level), 5, N, N, N))

    def fill(s):
        sl = slice(s, s + 2048)
        X, Y, Z = cell_centres(level[sl], ijk[sl], nb0)
        I, J, K = global_indices(level[sl], ijk[sl])
        rho = rho_fn(X, Y, Z)
        lv = level[sl][:, None, None, None]
        v = [noise * hash_normal(seed, lv, I, J, K, d) if noise else np.zeros_like(rho) for d in range(3)]
        U[sl] = prim_to_cons(rho, v[0], v[1], v[2], np.full_like(rho, 0.1), gamma)
    _pmap(fill, range(0, len(level), 2048))
    return Problem("C4", nb0, max_level, ((0, 0),) * 3, (1.0, 1.0, 1.0), gamma, 0.4, mode, nsteps, level, ijk, U,
                   {"workload": "AMR sphere base %d^3 + %d levels" % (nb * N, max_level), "census": t.census()})


def gmc(n=256, nsteps=5, seed=SEED + 30, mach=10.0, sigma=1.5, max_level=4, rho_c=RHO_C5, mode=1):
    """C5: GMC-like AMR.  Base fields on n^3 (lognormal rho-hat with mean 1, k^-4 velocity), sampled on
    finer levels by periodic trilinear interpolation; Jeans refinement (< 8 cells) = rho-hat > rho_c 4^l;
    physical density A*rho-hat with A = pi n^2 / (64 rho_c); P = rho/gamma, gamma = 1.0001 (reading R22)."""
    gamma = 1.0001
    nb = n // N
    nb0 = (nb, nb, nb)
    rho_hat, v = _pmap(lambda k: lognormal_density(n, sigma, seed) if k == 0 else velocity_field(n, mach, seed + 1), (0, 1))
    A = np.pi * n * n / (64.0 * rho_c)

    def sample(fld, lev, idx):
        X, Y, Z = cell_centres(lev, idx, nb0)
        return trilinear_sample(fld, X, Y, Z)

    def flag(l, idx):
        lev = np.full(len(idx), l, dtype=np.int32)
        out = np.zeros(len(idx), dtype=bool)

        def chunk(s):
            r = sample(rho_hat, lev[s:s + 1024], idx[s:s + 1024])
            out[s:s + 1024] = (r > rho_c * 4.0 ** l).reshape(len(r), -1).any(axis=1)
        _pmap(chunk, range(0, len(idx), 1024))
        return out

    t = tree_from_criterion(nb0, max_level, (True, True, True), flag)
    level, ijk = t.block_list()
    U = np.empty((len(level), 5, N, N, N))

    def fill(s):
        sl = slice(s, s + 1024)
        rho = A * sample(rho_hat, level[sl], ijk[sl])
        vv = [sample(c, level[sl], ijk[sl]) for c in v]
        U[sl] = prim_to_cons(rho, vv[0], vv[1], vv[2], rho / gamma, gamma)
    _pmap(fill, range(0, len(level), 1024))
    return Problem("C5", nb0, max_level, ((0, 0),) * 3, (1.0, 1.0, 1.0), gamma, 0.4, mode, nsteps, level, ijk, U,
                   {"workload": "GMC-like AMR base %d^3 + %d levels" % (n, max_level), "census": t.census(),
                    "amplitude": A, "rho_c": rho_c})


def make_config(name, scale=1):
    """Problem for BASELINE.json configs[k] (name 'C1'..'C5'); scale>1 shrinks the base grid.

    The shrunken turbulent cases (C2, C3, C5) also divide the rms Mach number by `scale`: the k^-4
    field has the same large-scale shear, so per-cell velocity jumps grow with the cell size and at
    the full Mach number a 64^3 box reaches negative pressure within a few steps (no floors, R28)."""
    if name == "C1":
        return sod(nb=max(1, 4 // scale))
    if name == "C2":
        return turbulent_box("C2", 256 // scale, 5.0 / scale, SEED)
    if name == "C3":
        return turbulent_box("C3", 512 // scale, 10.0 / scale, SEED + 10)
    if name == "C4":
        return amr_sphere(nb=16 // scale)
    if name == "C5":
        return gmc(n=256 // scale, mach=10.0 / scale, rho_c=RHO_C5 if scale == 1 else RHO_C5_SMALL)
    raise ValueError(name)
