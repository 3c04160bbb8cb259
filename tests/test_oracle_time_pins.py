"""Pins of the oracle's TIME AXIS: which coarse copy and which time fraction tau the ghost fill uses
(`fill_ghosts_level`), the tau / tau_half schedule of the Berger-Colella recursion (`advance_adaptive`,
PAPER.md:108-120), and the CFL step (`max_speed_level` / `cfl_dt_level`).

None of them compares the oracle with itself: each is an exact solution or a closed form.

* T1  linear advection on a sub-cycled AMR mesh.  rho = a + b.(x - v t) with uniform v and P is an exact
      solution of eq. (1)-(3), and every piece of the scheme is exact for data linear in
      x and t: the HLLC flux of two states with equal u and P is the upwind contact flux (S* = u), minmod
      of two equal differences is that difference, the prolongation (reading R3) and the restriction are
      exact for linear data, eq. (16) is exact for data linear in t, and the flux
      mismatch the reflux corrects is zero.  So away from the outflow boundary (whose zero-gradient copy
      is not linear; its error travels 3 cells per step) the computed field equals the analytic one to
      round-off -- provided the fine ghosts are taken at the right time.  A wrong tau anywhere puts an
      O(dt v.b) ~ 1e-3 error into the fine ghosts.
* T2  `orc_fill_ghosts(level, which, interp, tau)` on hand-set coarse copies: for coarse data linear in
      space the prolonged value at a fine ghost centre is the coarse field evaluated there, and eq.
      (16)-(17) expands to the Bernstein form (1-tau)^2 U^n + 2 tau (1-tau) U^{n+1/2} + tau^2 U^{n+1}.
* T3  `orc_cfl_dt` on uniform states with one hot cell: dt = CFL h_l / (max_d |v_d| + sqrt(gamma P / rho))
      (reading R16).

Mutations of oracle/sfh_oracle.cpp these pins were checked to catch (each leaves the older pins green):
no temporal interpolation (coarse U^n always); tau_half = tau; sub-step fraction (s+1)/nsub; synchronous
half-state ghosts from the coarse U^n; sound speed without gamma; sum instead of max of |v_d|.
"""
import numpy as np
import pytest

from helpers import oracle_for, problem_from_tree, small_amr_tree
from sfh_inputs import prim_to_cons
from sfh_inputs.configs import cell_centres

A0, B, V, P0, GAMMA = 2.0, np.array([0.3, -0.2, 0.25]), np.array([0.7, -0.4, 0.3]), 1.0, 1.4


def advected(X, Y, Z, T):
    """The exact solution at time T as conserved variables [nb][5][8][8][8]."""
    rho = A0 + B[0] * (X - V[0] * T) + B[1] * (Y - V[1] * T) + B[2] * (Z - V[2] * T)
    one = np.ones_like(rho)
    return prim_to_cons(rho, V[0] * one, V[1] * one, V[2] * one, P0 * one, GAMMA)


def advection_problem(mode):
    """6^3 outflow root blocks, the refined 2^3-block patch (and its nested level-2 patch) in the middle:
    16 coarse cells away from every boundary."""
    t = small_amr_tree(6, 2, periodic=(False, False, False), offset=(1, 1, 1))
    f = lambda X, Y, Z: (A0 + B[0] * X + B[1] * Y + B[2] * Z, np.full_like(X, V[0]), np.full_like(X, V[1]),
                         np.full_like(X, V[2]), np.full_like(X, P0))
    return problem_from_tree(t, gamma=GAMMA, mode=mode, fields=f)


def interior_mask(p, margin):
    """Cells farther than `margin` level-0 cells from the domain boundary."""
    X, Y, Z = cell_centres(p.level, p.ijk, p.nb0)
    d = np.minimum.reduce([X, Y, Z, 1 - X, 1 - Y, 1 - Z]) * (p.nb0[0] * 8)
    return d > margin


# ------------------------------------------------------------------ T1
@pytest.mark.parametrize("mode", [1, 0])
def test_t1_linear_advection_is_exact_on_a_subcycled_amr_mesh(mode):
    p = advection_problem(mode)
    m = oracle_for(p)
    m.restrict_all(0)
    X, Y, Z = cell_centres(p.level, p.ijk, p.nb0)
    for step in (1, 2):
        m.advance(1, mode)
        if mode == 1:
            assert tuple(m.nupd) == (step, 2 * step, 4 * step)      # every finer level sub-cycles once (n = 1)
        err = np.abs(m.get_state() - advected(X, Y, Z, m.t.value))
        sel = interior_mask(p, 3 * step + 2)
        for l in range(3):
            assert (sel & (p.level == l)[:, None, None, None]).any()
        worst = err.transpose(1, 0, 2, 3, 4)[:, sel].max()
        assert worst < 2e-14, (step, worst)
        # and the test has teeth: the outflow copy's error is visible near the boundary
        assert err.max() > 1e-6


# ------------------------------------------------------------------ T2
def linear_copies(rng):
    """Three coarse 'time copies', each variable an independent linear function of (x, y, z)."""
    c = rng.normal(0.0, 1.0, (3, 5, 4))
    c[:, :, 0] += 3.0
    return c


def evaluate(c, X, Y, Z, axis=1):
    return np.stack([c[v, 0] + c[v, 1] * X + c[v, 2] * Y + c[v, 3] * Z for v in range(5)], axis=axis)


def ghost_centres(p, b):
    """Centres of the 12^3 ghosted cells of block b, [k][j][i]."""
    n = p.nb0[0] * 8 * 2.0 ** p.level[b]
    c = np.arange(-2, 10) + 0.5
    x = (p.ijk[b, 0] * 8 + c) / n
    y = (p.ijk[b, 1] * 8 + c) / n
    z = (p.ijk[b, 2] * 8 + c) / n
    return np.broadcast_to(x[None, None, :], (12, 12, 12)), np.broadcast_to(y[None, :, None], (12, 12, 12)), \
        np.broadcast_to(z[:, None, None], (12, 12, 12))


@pytest.mark.parametrize("tau", [0.0, 0.25, 0.5, 0.75, 1.0])
def test_t2_fill_ghosts_uses_eq16_at_tau_on_the_coarse_copies(tau):
    t = small_amr_tree(4, 1, periodic=(False, False, False))
    p = problem_from_tree(t, mode=1)
    m = oracle_for(p)
    rng = np.random.default_rng(21)
    coarse = linear_copies(rng)           # U^n, U^{n+1/2}, U^{n+1} of level 0
    fine = linear_copies(rng)             # the three copies of level 1 (unrelated to the coarse ones)
    X, Y, Z = cell_centres(p.level, p.ijk, p.nb0)
    is_fine = (p.level == 1)[:, None, None, None, None]
    for k in range(3):
        m.set_state(np.where(is_fine, evaluate(fine[k], X, Y, Z), evaluate(coarse[k], X, Y, Z)), k)
    w = np.array([(1 - tau) ** 2, 2 * tau * (1 - tau), tau ** 2])       # eq. (16)-(17) expanded
    lo, hi = 2 * 8, 6 * 8                                               # the level-1 patch in level-1 cells
    for which in (0, 1, 2):
        for interp in (1, 0):
            m.fill_ghosts(1, which, interp, tau)
            checked = 0
            for b in np.nonzero(p.level == 1)[0]:
                gx, gy, gz = ghost_centres(p, b)
                I = np.rint(gx * 64 - 0.5).astype(int)
                J = np.rint(gy * 64 - 0.5).astype(int)
                K = np.rint(gz * 64 - 0.5).astype(int)
                inside = (I >= lo) & (I < hi) & (J >= lo) & (J < hi) & (K >= lo) & (K < hi)
                if interp:
                    from_coarse = sum(w[k] * evaluate(coarse[k], gx, gy, gz, 0) for k in range(3))
                else:
                    from_coarse = evaluate(coarse[which], gx, gy, gz, 0)   # synchronous mode: the same copy, no interpolation
                expect = np.where(inside[None], evaluate(fine[which], gx, gy, gz, 0), from_coarse)   # [v][k][j][i]
                ghost = np.ones((12, 12, 12), bool)
                ghost[2:10, 2:10, 2:10] = False
                d = np.abs(m.U[which][b] - expect)[:, ghost]
                assert d.max() < 5e-14, (which, interp, d.max())
                checked += int((ghost & ~inside).sum())
            assert checked >= 96 * 128           # every coarse-fine face slab (and the edge/corner ghosts) was looked at


# ------------------------------------------------------------------ T3
@pytest.mark.parametrize("gamma", [1.0001, 1.4, 5.0 / 3.0])
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_t3_cfl_dt_closed_form(gamma, axis):
    t = small_amr_tree(4, 2)
    cfl = 0.37
    rho0, P0_, v0 = 1.7, 0.9, np.array([0.11, -0.13, 0.12])
    f = lambda X, Y, Z: (np.full_like(X, rho0), np.full_like(X, v0[0]), np.full_like(X, v0[1]), np.full_like(X, v0[2]),
                         np.full_like(X, P0_))
    p = problem_from_tree(t, gamma=gamma, cfl=cfl, fields=f)
    h = [1.0 / (32 * 2 ** l) for l in range(3)]
    cs0 = np.sqrt(gamma * P0_ / rho0)
    for hot_level in range(3):
        # one hot cell on one level: the largest |v_d| along `axis` (negative), denser and hotter
        U = p.U.copy()
        b = np.nonzero(p.level == hot_level)[0][5]
        vh = np.array([0.3, 0.2, -0.25])
        vh[axis] = -2.5
        rh, Ph = 0.6, 3.1
        U[b, :, 3, 4, 5] = prim_to_cons(np.array([rh]), *[np.array([x]) for x in vh], np.array([Ph]), gamma)[0]
        m = oracle_for(p, U)
        expect = [cfl * h[l] / (np.abs(v0).max() + cs0) for l in range(3)]
        expect[hot_level] = cfl * h[hot_level] / (2.5 + np.sqrt(gamma * Ph / rh))
        for l in range(3):
            assert abs(m.cfl_dt(l) - expect[l]) <= 4e-16 * expect[l], (l, m.cfl_dt(l), expect[l])
            assert abs(m.max_speed(l) - cfl * h[l] / expect[l]) <= 4e-16 * m.max_speed(l)
        assert abs(m.cfl_dt(-1) - min(expect)) <= 4e-16 * min(expect)
