"""Small hand-built AMR meshes and smooth seeded fields for parity cases, smoke() and the oracle pins.
No method arithmetic (pointwise initial data only)."""
import numpy as np

from .configs import Problem, cell_centres
from .fields import prim_to_cons
from .mesh import Tree


def small_amr_tree(nb=4, max_level=2, periodic=(True, True, True), offset=(0, 0, 0)):
    """nb^3 root blocks; a 2x2x2 patch of root blocks refined, and inside it a nested patch."""
    t = Tree((nb, nb, nb), max_level, periodic)
    f0 = np.zeros_like(t.exists[0])
    o = offset
    f0[1 + o[0]:3 + o[0], 1 + o[1]:3 + o[1], 1 + o[2]:3 + o[2]] = True
    t.refine(0, f0)
    if max_level >= 2:
        f1 = np.zeros_like(t.exists[1])
        f1[3 + 2 * o[0]:5 + 2 * o[0], 3 + 2 * o[1]:5 + 2 * o[1], 3 + 2 * o[2]:5 + 2 * o[2]] = True
        t.refine(1, f1)
    return t.pad_2to1()


def smooth_fields(X, Y, Z, amp=0.3, vamp=0.4):
    """Smooth periodic (unit box) positive density/pressure and a velocity field."""
    tp = 2.0 * np.pi
    rho = 1.0 + amp * np.sin(tp * X) * np.cos(tp * Y) + 0.5 * amp * np.cos(tp * (Z + 0.1)) \
        + 0.8 * np.exp(-((X - 0.47) ** 2 + (Y - 0.52) ** 2 + (Z - 0.45) ** 2) / 0.02)
    P = 1.0 + 0.5 * amp * np.cos(tp * X) * np.sin(tp * Z) + 0.3 * np.exp(-((X - 0.5) ** 2 + (Y - 0.45) ** 2 + (Z - 0.55) ** 2) / 0.03)
    vx = vamp * np.sin(tp * Y) + 0.3
    vy = vamp * np.cos(tp * Z) * np.sin(tp * X) - 0.2
    vz = vamp * np.sin(tp * (X + Y)) + 0.1
    return rho, vx, vy, vz, P


def problem_from_tree(t, gamma=5.0 / 3.0, cfl=0.4, mode=0, nsteps=1, fields=smooth_fields, bc=None, name="T"):
    level, ijk = t.block_list()
    X, Y, Z = cell_centres(level, ijk, t.nb0)
    rho, vx, vy, vz, P = fields(X, Y, Z)
    U = prim_to_cons(rho, vx, vy, vz, P, gamma)
    if bc is None:
        bc = tuple((0, 0) if per else (1, 1) for per in t.periodic)
    box = tuple(n / t.nb0[0] for n in t.nb0)
    return Problem(name, t.nb0, t.max_level, bc, box, gamma, cfl, mode, nsteps, level, ijk, U)


def add_scalars(p, s_fields):
    """The problem p with passive scalars appended: s_fields is a list of functions s(X, Y, Z) (concentration per
    unit mass, evaluated at the cell centres); the conserved densities rho*s become variables 5, 6, ... of p.U."""
    import dataclasses
    X, Y, Z = cell_centres(p.level, p.ijk, p.nb0)
    rho = p.U[:, 0]
    q = [rho * np.broadcast_to(np.asarray(f(X, Y, Z), dtype=np.float64), rho.shape) for f in s_fields]
    U = np.concatenate([p.U, np.stack(q, axis=1)], axis=1) if q else p.U
    return dataclasses.replace(p, U=np.ascontiguousarray(U), name=p.name + "+%ds" % len(q))
