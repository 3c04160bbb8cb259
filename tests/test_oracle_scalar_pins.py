"""Pins of the oracle's passive scalars (eq. 12-13; reading R32):
conserved densities q = rho*s carried by the Riemann solver's mass flux, F_q = F_rho * s_upwind.

What the equations fix, whatever the discretisation details:
* SC1  s uniform  =>  q = s*rho for all time (eq. 12 with R = 0 is then the continuity equation): to round-off on a
       sub-cycled AMR mesh, across prolongation, restriction and reflux.
* SC2  the hydro variables do not see the scalars: bitwise the same run with and without them.
* SC3  sum of q over the leaf cells is conserved to round-off on a periodic AMR mesh with flux correction, and is NOT
       without it (the reflux treats the scalars like the other conserved fields).
* SC4  linear advection: rho, v, P uniform and s = a + b.(x - v t) is an exact solution, and upwind fluxes with limited
       linear reconstruction, the prolongation, eq. (16) and the reflux are exact for it: to round-off away from the
       outflow boundary on the sub-cycled AMR mesh.  (A first-order scalar flux, a downwind face value or a wrong time
       fraction in the scalar ghost fill all fail it.)
* SC5  upwinding: a step in s in a uniform flow moves downstream only; cells upstream of it keep s exactly.
* SC6  maximum principle: s stays within the range of its initial values (upwind flux + minmod slopes).

Mutations of oracle/sfh_oracle.cpp these were checked to catch: downwind face value in scalar_fluxes, cell-centred
instead of reconstructed face values in the corrector, scalars left out of the reflux, of the restriction, of the
prolongation's slopes.
"""
import numpy as np
import pytest

from helpers import leaf_totals, oracle_for, problem_from_tree, small_amr_tree, smooth_fields
from sfh_inputs import add_scalars, uniform_tree
from sfh_inputs.configs import cell_centres


def wavy(X, Y, Z):
    return 1.5 + 0.5 * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * (Y + 0.2)) + 0.3 * np.cos(2 * np.pi * Z)


def blob(X, Y, Z):
    return 0.2 + np.exp(-((X - 0.5) ** 2 + (Y - 0.45) ** 2 + (Z - 0.55) ** 2) / 0.02)


def scalar_problem(mode, fields=smooth_fields, scalars=(wavy, blob), **kw):
    return add_scalars(problem_from_tree(small_amr_tree(4, 2), mode=mode, fields=fields, **kw), list(scalars))


# ------------------------------------------------------------------ SC1
@pytest.mark.parametrize("mode", [0, 1])
def test_sc1_uniform_concentration_stays_uniform(mode):
    p = scalar_problem(mode, scalars=(lambda X, Y, Z: 0.37, lambda X, Y, Z: 2.5))
    m = oracle_for(p)
    m.restrict_all(0)
    m.advance(2, mode)
    U = m.get_state()
    if mode == 1:
        assert tuple(m.nupd) == (2, 4, 8)
    assert np.abs(U[:, 5] / U[:, 0] - 0.37).max() < 2e-15
    assert np.abs(U[:, 6] / U[:, 0] - 2.5).max() < 1e-14
    assert np.abs(U[:, 0] - p.U[:, 0]).max() > 1e-3            # and the gas did move


# ------------------------------------------------------------------ SC2
@pytest.mark.parametrize("mode", [0, 1])
def test_sc2_hydro_variables_do_not_see_the_scalars(mode):
    p0 = problem_from_tree(small_amr_tree(4, 2), mode=mode)
    p2 = add_scalars(p0, [wavy, blob])
    a, b = oracle_for(p0), oracle_for(p2)
    a.restrict_all(0)
    b.restrict_all(0)
    a.advance(2, mode)
    b.advance(2, mode)
    assert np.array_equal(a.nupd, b.nupd)
    assert np.array_equal(a.get_state(), b.get_state()[:, :5])


# ------------------------------------------------------------------ SC3
def scalar_totals(m, p):
    U = m.get_state()
    leaf, h0 = m.is_leaf(), m.cell_width(0)
    out = []
    for v in range(5, U.shape[1]):
        W = np.zeros((len(U), 5) + U.shape[2:])
        W[:, 0] = U[:, v]
        out.append(leaf_totals(leaf, W, p.level, h0)[0])
    return np.array(out)


@pytest.mark.parametrize("mode", [0, 1])
def test_sc3_scalar_mass_conserved_with_reflux_and_not_without(mode):
    p = scalar_problem(mode)
    m = oracle_for(p)
    m.restrict_all(0)
    t0 = scalar_totals(m, p)
    m.advance(2, mode)
    t1 = scalar_totals(m, p)
    assert (np.abs(t1 - t0) <= 4e-15 * np.abs(t0)).all(), (t1 - t0) / t0
    m2 = oracle_for(p)
    m2.set_reflux(0)
    m2.restrict_all(0)
    m2.advance(1, mode)
    t2 = scalar_totals(m2, p)
    assert (np.abs(t2 - t0) > 1e-9 * np.abs(t0)).all()


# ------------------------------------------------------------------ SC4
A0, B, V = 1.0, np.array([0.3, -0.2, 0.25]), np.array([0.7, -0.4, 0.3])


def advection_problem(mode):
    t = small_amr_tree(6, 2, periodic=(False, False, False), offset=(1, 1, 1))
    f = lambda X, Y, Z: (np.full_like(X, 1.3), np.full_like(X, V[0]), np.full_like(X, V[1]), np.full_like(X, V[2]),
                         np.full_like(X, 0.9))
    p = problem_from_tree(t, gamma=1.4, mode=mode, fields=f)
    return add_scalars(p, [lambda X, Y, Z: A0 + B[0] * X + B[1] * Y + B[2] * Z])


def advected_s(X, Y, Z, T):
    return A0 + B[0] * (X - V[0] * T) + B[1] * (Y - V[1] * T) + B[2] * (Z - V[2] * T)


@pytest.mark.parametrize("mode", [1, 0])
def test_sc4_linear_scalar_advection_is_exact_on_a_subcycled_amr_mesh(mode):
    p = advection_problem(mode)
    m = oracle_for(p)
    m.restrict_all(0)
    X, Y, Z = cell_centres(p.level, p.ijk, p.nb0)
    d = np.minimum.reduce([X, Y, Z, 1 - X, 1 - Y, 1 - Z]) * (p.nb0[0] * 8)
    for step in (1, 2):
        m.advance(1, mode)
        if mode == 1:
            assert tuple(m.nupd) == (step, 2 * step, 4 * step)
        U = m.get_state()
        err = np.abs(U[:, 5] / U[:, 0] - advected_s(X, Y, Z, m.t.value))
        sel = d > 3 * step + 2
        assert err[sel].max() < 2e-14, (step, err[sel].max())
        assert err.max() > 1e-6                         # the outflow copy is not linear: the test has teeth
        assert np.abs(U[:, 0] - 1.3).max() < 1e-14      # the gas stays uniform


# ------------------------------------------------------------------ SC5, SC6
@pytest.mark.parametrize("vx", [0.8, -0.8])
def test_sc5_a_step_in_s_moves_downstream_only(vx):
    t = uniform_tree((4, 1, 1), 0, (False, False, False))
    f = lambda X, Y, Z: (np.full_like(X, 1.0), np.full_like(X, vx), np.zeros_like(X), np.zeros_like(X), np.full_like(X, 1.0))
    p = add_scalars(problem_from_tree(t, gamma=1.4, fields=f), [lambda X, Y, Z: np.where(X < 0.5, 1.0, 3.0)])
    m = oracle_for(p)
    m.advance(3, 0)
    U = m.get_state()
    X, _, _ = cell_centres(p.level, p.ijk, p.nb0)
    s = U[:, 5] / U[:, 0]
    h = 1.0 / 32
    if vx > 0:      # upstream of the step = left of it: untouched; the step's foot moved right
        assert (s[X < 0.5] == 1.0).all() and (np.abs(s[X > 0.5 + 8 * h] - 3.0) < 1e-15).all()
        assert s[(X > 0.5) & (X < 0.5 + h)].max() < 3.0 - 1e-3
    else:
        assert (s[X > 0.5] == 3.0).all() and (np.abs(s[X < 0.5 - 8 * h] - 1.0) < 1e-15).all()
        assert s[(X < 0.5) & (X > 0.5 - h)].min() > 1.0 + 1e-3
    assert s.min() >= 1.0 - 1e-14 and s.max() <= 3.0 + 1e-14


@pytest.mark.parametrize("mode", [0, 1])
def test_sc6_maximum_principle(mode):
    p = scalar_problem(mode)
    s0 = p.U[:, 5:] / p.U[:, :1]
    m = oracle_for(p)
    m.restrict_all(0)
    m.advance(3, mode)
    U = m.get_state()
    s = U[:, 5:] / U[:, :1]
    for q in range(2):
        assert s[:, q].min() >= s0[:, q].min() - 1e-12 and s[:, q].max() <= s0[:, q].max() + 1e-12
    assert m.status() == 0
