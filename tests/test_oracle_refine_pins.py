"""Pins of the oracle's refinement indicators (eq. (33)-(34), PAPER.md:277-285,
and the Jeans criterion) against closed forms and invariants.  CPU only."""
import numpy as np

from helpers import oracle_for, problem_from_tree, small_amr_tree
from sfh_inputs import prim_to_cons, uniform_tree
from sfh_inputs.configs import Problem, cell_centres


def make(t, fields, gamma=1.4, bc=((1, 1),) * 3):
    level, ijk = t.block_list()
    X, Y, Z = cell_centres(level, ijk, t.nb0)
    rho, P = fields(X, Y, Z)
    z = np.zeros_like(rho)
    U = prim_to_cons(rho, z + 0.3, z - 0.2, z + 0.1, P, gamma)
    box = tuple(n / t.nb0[0] for n in t.nb0)
    p = Problem("ind", t.nb0, t.max_level, bc, box, gamma, 0.4, 0, 1, level, ijk, U)
    m = oracle_for(p)
    m.fill_ghosts(-1, 0, 0, 0.0)
    return p, m, (X, Y, Z), (rho, P)


def test_curvature_indicator_of_a_quadratic_field_is_its_closed_form():
    """q = a + b x^2 + c y^2 + d z^2: the centred second differences are exact, so
    E(q) = 2 |b + c + d| h^2 / q in every cell away from the outflow boundary."""
    t = uniform_tree((4, 4, 4), 0)
    h = 1.0 / 32
    rho_f = lambda X, Y, Z: 1.0 + 0.8 * X ** 2 + 0.5 * Y ** 2 + 0.3 * Z ** 2
    P_f = lambda X, Y, Z: 2.0 + 0.1 * X ** 2 - 0.6 * Y ** 2 + 0.2 * Z ** 2
    p, m, (X, Y, Z), (rho, P) = make(t, lambda X, Y, Z: (rho_f(X, Y, Z), P_f(X, Y, Z)))
    ind = m.refine_indicator(0)
    inner = ((p.ijk >= 1) & (p.ijk <= 2)).all(axis=1)          # blocks that do not touch the boundary
    Er = 2.0 * abs(0.8 + 0.5 + 0.3) * h * h / rho
    EP = 2.0 * abs(0.1 - 0.6 + 0.2) * h * h / P
    expect = np.maximum(Er, EP).reshape(len(rho), -1).max(axis=1)
    assert np.allclose(ind[inner], expect[inner], rtol=1e-9, atol=0)
    # at an outflow face the ghost is a copy of the edge cell: the x second difference there is q_1 - q_0
    b = np.where((p.ijk == [0, 1, 1]).all(axis=1))[0][0]
    x0, x1 = X[b, 3, 3, 0], X[b, 3, 3, 1]
    y, z = Y[b, 3, 3, 0], Z[b, 3, 3, 0]
    lap = (rho_f(x1, y, z) - rho_f(x0, y, z)) + 2 * 0.5 * h * h + 2 * 0.3 * h * h
    assert ind[b] >= abs(lap) / rho_f(x0, y, z) * (1 - 1e-9)


def test_curvature_indicator_of_a_linear_field_vanishes():
    t = uniform_tree((4, 4, 4), 0)
    p, m, _, _ = make(t, lambda X, Y, Z: (1.0 + 0.5 * X - 0.25 * Y + 0.125 * Z, 3.0 - X + 0.5 * Y + 0.25 * Z),
                      bc=((0, 0),) * 3)
    ind = m.refine_indicator(0)
    inner = ((p.ijk >= 1) & (p.ijk <= 2)).all(axis=1)
    assert ind[inner].max() < 1e-13        # blocks away from the periodic jump see a linear field
    # the periodic wrap makes the field jump at the box faces: the blocks there must see that
    assert ind[~inner].min() > 1e-2


def test_curvature_indicator_picks_the_larger_of_density_and_pressure():
    t = uniform_tree((4, 4, 4), 0)
    quad = lambda X, Y, Z: 1.0 + 0.9 * X ** 2
    flat = lambda X, Y, Z: np.full_like(X, 2.0)
    _, m1, _, _ = make(t, lambda X, Y, Z: (quad(X, Y, Z), flat(X, Y, Z)))
    _, m2, _, _ = make(t, lambda X, Y, Z: (flat(X, Y, Z), quad(X, Y, Z)))
    a, b = m1.refine_indicator(0), m2.refine_indicator(0)
    assert (a > 1e-4).all() and (b > 1e-4).all()
    p, m3, _, _ = make(t, lambda X, Y, Z: (quad(X, Y, Z), quad(X, Y, Z)))
    inner = ((p.ijk >= 1) & (p.ijk <= 2)).all(axis=1)
    assert np.allclose(m3.refine_indicator(0)[inner], a[inner], rtol=1e-9)


def test_jeans_indicator_closed_form_and_scalings():
    """Uniform state: h / lambda_J = h rho sqrt(G / (pi gamma P)) in every block; it doubles with the
    density, halves from one level to the next, and scales with sqrt(G)."""
    gamma = 1.4
    t = small_amr_tree()
    for rho0, P0, G in ((1.0, 1.0, 1.0), (2.0, 1.0, 1.0), (1.0, 0.25, 4.0)):
        p, m, _, _ = make(t, lambda X, Y, Z: (np.full_like(X, rho0), np.full_like(X, P0)), gamma=gamma,
                          bc=((0, 0),) * 3)
        J = m.refine_indicator(1, G=G)
        for l in range(p.max_level + 1):
            h = m.cell_width(l)
            expect = h * rho0 * np.sqrt(G / (np.pi * gamma * P0))
            assert np.allclose(J[p.level == l], expect, rtol=1e-13)


def test_indicators_are_invariant_under_axis_permutation():
    t = uniform_tree((2, 2, 2), 0)
    f = lambda A, B, C: (1.5 + 0.5 * np.sin(2 * np.pi * A) * np.cos(2 * np.pi * B) + 0.2 * np.cos(4 * np.pi * C),
                         1.0 + 0.3 * np.cos(2 * np.pi * (A + 2 * B)) + 0.1 * np.sin(2 * np.pi * C))
    p1, m1, _, _ = make(t, lambda X, Y, Z: f(X, Y, Z), bc=((0, 0),) * 3)
    p2, m2, _, _ = make(t, lambda X, Y, Z: f(Y, Z, X), bc=((0, 0),) * 3)
    for crit in (0, 1):
        a, b = m1.refine_indicator(crit), m2.refine_indicator(crit)
        # block (i, j, k) of the first field is block (k, i, j) of the permuted one
        key = lambda ijk: (ijk[:, 0] * 4 + ijk[:, 1]) * 4 + ijk[:, 2]
        perm = np.argsort(key(p2.ijk[:, [1, 2, 0]]))
        assert np.allclose(a[np.argsort(key(p1.ijk))], b[perm], rtol=1e-12)


def test_fine_level_of_a_fully_refined_mesh_matches_the_uniform_mesh_bitwise():
    tu = uniform_tree((4, 4, 4), 0)
    tr = uniform_tree((2, 2, 2), 1, fully_refined_to=1)
    f = lambda X, Y, Z: (1.5 + 0.5 * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y) + 0.2 * np.cos(4 * np.pi * Z),
                         1.0 + 0.3 * np.cos(2 * np.pi * (X + 2 * Y)) + 0.1 * np.sin(2 * np.pi * Z))
    pu, mu, _, _ = make(tu, f, bc=((0, 0),) * 3)
    pr, mr, _, _ = make(tr, f, bc=((0, 0),) * 3)
    key = lambda ijk: (ijk[:, 0] * 64 + ijk[:, 1]) * 64 + ijk[:, 2]
    fine = pr.level == 1
    a = mu.refine_indicator(0)[np.argsort(key(pu.ijk))]
    b = mr.refine_indicator(0)[fine][np.argsort(key(pr.ijk[fine]))]
    assert np.array_equal(a, b)
