"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (sfh_advance on the
whole problem, one persistent CTA per SM).

* C2 (256^3) and C4 (128^3 + 3 levels) are small enough for the oracle: every cell is compared.
* C3 (512^3): the oracle recomputes sampled outputs.  One step of the scheme reaches 3 cells (1 for the
  predictor, 2 for the corrector), so the inner 2^3 blocks of a 4^3-block sub-box cut out of the full
  initial state (outflow on the cut faces), stepped with the full problem's dt, are exactly the full
  problem's values there.
* C5 (1.8e5 blocks): properties that hold at any size -- conservation over leaf cells to round-off on
  the periodic box across refinement boundaries, and the same per-level update counts as eq. (14)-(15)
  give from the CUDA path's own CFL steps.
"""
import numpy as np
import pytest

import paper_2604_21438_b200 as sfh
from helpers import oracle_for, parity_errors
from sfh_inputs import make_config
from sfh_inputs.configs import Problem

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

TOL1, TOL10, TOLDT = 1e-12, 1e-10, 1e-14


def gpu_for(p):
    g = sfh.Mesh.from_problem(p)
    g.set_state(p.U)
    g.restrict_all(0)
    return g


def test_c2_full_size_every_cell():
    p = make_config("C2")
    o = oracle_for(p)
    g = gpu_for(p)
    o.advance(1, 0)
    g.advance(1, 0)
    assert abs(g.t.value - o.t.value) <= TOLDT * o.t.value
    err = parity_errors(g.get_state().cpu().numpy(), o.get_state(), p.gamma)
    assert (err <= TOL1).all(), err
    o.advance(9, 0)
    g.advance(9, 0)
    assert abs(g.t.value - o.t.value) <= 1e-13 * o.t.value
    assert o.status() == 0 and g.status() == 0
    err = parity_errors(g.get_state().cpu().numpy(), o.get_state(), p.gamma)
    assert (err <= TOL10).all(), err


def test_c4_full_size_adaptive_every_cell():
    p = make_config("C4")
    o = oracle_for(p)
    o.restrict_all(0)
    g = gpu_for(p)
    assert np.array_equal(g.get_state().cpu().numpy(), o.get_state())
    o.advance(1, 1)
    g.advance(1, 1)
    assert np.array_equal(o.nupd, g.nupd), (o.nupd, g.nupd)
    assert abs(g.t.value - o.t.value) <= TOLDT * o.t.value
    err = parity_errors(g.get_state().cpu().numpy(), o.get_state(), p.gamma)
    assert (err <= TOL1).all(), err
    o.advance(2, 1)
    g.advance(2, 1)
    assert np.array_equal(o.nupd, g.nupd), (o.nupd, g.nupd)
    err = parity_errors(g.get_state().cpu().numpy(), o.get_state(), p.gamma)
    assert (err <= TOL10).all(), err


def test_c3_full_size_sampled_sub_boxes():
    p = make_config("C3")
    nb = p.nb0[0]
    g = gpu_for(p)
    dt = g.cfl_dt()
    g.advance(1, 0, dt)
    Ug = g.get_state().cpu().numpy()
    where = np.full((nb, nb, nb), -1, dtype=np.int64)
    where[p.ijk[:, 0], p.ijk[:, 1], p.ijk[:, 2]] = np.arange(p.nblocks)
    rng = np.random.default_rng(3)
    S = 4
    sub_ijk = np.array([(i, j, k) for k in range(S) for j in range(S) for i in range(S)], dtype=np.int32)
    inner = ((sub_ijk >= 1) & (sub_ijk <= 2)).all(axis=1)
    compared = 0
    for _ in range(6):
        o0 = rng.integers(0, nb - S + 1, size=3)
        idx = where[o0[0] + sub_ijk[:, 0], o0[1] + sub_ijk[:, 1], o0[2] + sub_ijk[:, 2]]
        sub = Problem("C3-sub", (S, S, S), 0, ((1, 1),) * 3, (S / nb,) * 3, p.gamma, p.cfl, 0, 1,
                      np.zeros(S ** 3, dtype=np.int32), sub_ijk, np.ascontiguousarray(p.U[idx]))
        o = oracle_for(sub)
        assert o.cell_width(0) == g.cell_width(0)
        o.advance(1, 0, dt)
        Uo = o.get_state()[inner]
        Ua = Ug[idx[inner]]
        if not np.isfinite(Uo).all():      # a non-positive pressure of the Mach-10 input (R28): no parity there
            continue
        err = parity_errors(Ua, Uo, p.gamma)
        assert (err <= TOL1).all(), (o0, err)
        compared += 1
    assert compared >= 4


def leaf_mask(level, ijk):
    key = lambda l, c: (l.astype(np.int64) << 48) | (c[:, 0].astype(np.int64) << 32) | (c[:, 1].astype(np.int64) << 16) | c[:, 2]
    parents = set(key(level[level > 0] - 1, ijk[level > 0] >> 1).tolist())
    return np.array([k not in parents for k in key(level, ijk).tolist()])


def totals(U, level, leaf, max_level):
    tot = np.zeros(5, dtype=np.longdouble)
    for l in range(max_level + 1):
        sel = leaf & (level == l)
        if sel.any():
            tot += U[sel].sum(axis=(0, 2, 3, 4), dtype=np.longdouble) * np.longdouble(8.0) ** (-l)
    return tot


def test_c5_full_size_conservation_and_subcycling():
    p = make_config("C5")
    assert 1.5e5 < p.nblocks < 2.2e5, p.census()
    g = gpu_for(p)
    leaf = leaf_mask(p.level, p.ijk)
    U0 = g.get_state().cpu().numpy()
    t0 = totals(U0, p.level, leaf, p.max_level)
    del U0
    g.advance(1, 1)
    U1 = g.get_state().cpu().numpy()
    assert np.isfinite(U1).all()
    t1 = totals(U1, p.level, leaf, p.max_level)
    # momentum components nearly cancel over the box: their scale is the sum of the magnitudes
    mscale = totals(np.abs(U1), p.level, leaf, p.max_level)[1:4].max()
    assert abs(t1[0] - t0[0]) <= 1e-12 * abs(t0[0]), (t0, t1)
    assert abs(t1[4] - t0[4]) <= 1e-12 * abs(t0[4]), (t0, t1)
    assert (np.abs(t1[1:4] - t0[1:4]) <= 1e-12 * mscale).all(), (t0, t1)
    # eq. (14)-(15): each level takes 2^n sub-steps of its parent, n >= 0
    n = g.nupd
    assert n[0] == 1
    for l in range(1, p.max_level + 1):
        r = n[l] // n[l - 1]
        assert n[l] == r * n[l - 1] and r >= 1 and (r & (r - 1)) == 0, n
    assert g.status() == 0
