"""Pins of the oracle's regrid state transfer (child creation by conservative
prolongation; reading R3) against invariants.  CPU only."""
import numpy as np

from helpers import leaf_totals, oracle_for, problem_from_tree, small_amr_tree, smooth_fields
from sfh_inputs import Tree, prim_to_cons, uniform_tree
from sfh_inputs.configs import Problem, cell_centres


def refined_copy(nb=4, extra=True, drop_inner=False):
    """small_amr_tree() with one more root block refined (and optionally without its level-2 patch)."""
    t = Tree((nb, nb, nb), 2, (True, True, True))
    f0 = np.zeros_like(t.exists[0])
    f0[1:3, 1:3, 1:3] = True
    if extra:
        f0[0, 1, 1] = True
    t.refine(0, f0)
    if not drop_inner:
        f1 = np.zeros_like(t.exists[1])
        f1[3:5, 3:5, 3:5] = True
        t.refine(1, f1)
    return t.pad_2to1()


def consistent(p):
    m = oracle_for(p)
    m.restrict_all(0)
    return m


def test_transfer_to_the_same_mesh_is_the_identity():
    p = problem_from_tree(small_amr_tree(), mode=1)
    a, b = consistent(p), oracle_for(p)
    b.set_state(np.zeros_like(p.U))
    b.transfer_from(a)
    assert np.array_equal(a.get_state(), b.get_state())


def test_new_children_restrict_back_to_their_parents_and_totals_are_conserved():
    p = problem_from_tree(small_amr_tree(), mode=1)
    a = consistent(p)
    q = problem_from_tree(refined_copy(), mode=1)
    b = oracle_for(q)
    b.transfer_from(a)
    Ub = b.get_state().copy()
    # blocks present in both meshes are copies
    key = lambda lv, ijk: [(int(l), *map(int, c)) for l, c in zip(lv, ijk)]
    old = {k: n for n, k in enumerate(key(p.level, p.ijk))}
    Ua = a.get_state()
    new_blocks = 0
    for n, k in enumerate(key(q.level, q.ijk)):
        if k in old:
            assert np.array_equal(Ub[n], Ua[old[k]])
        else:
            new_blocks += 1
    assert new_blocks >= 8                               # the refined root block (+ padding)
    # conservative prolongation: restricting the new hierarchy changes nothing (to rounding) ...
    b.restrict_all(0)
    scale = np.abs(Ub).max(axis=(0, 2, 3, 4))[None, :, None, None, None]
    assert (np.abs(b.get_state() - Ub) <= 4e-16 * scale).all()
    # ... and the totals over the leaves are those of the old mesh
    ta = leaf_totals(a.is_leaf(), Ua, p.level, a.cell_width(0))
    tb = leaf_totals(b.is_leaf(), Ub, q.level, b.cell_width(0))
    assert (np.abs(ta - tb) <= 1e-14 * np.abs(ta).max()).all(), ta - tb


def test_linear_field_is_prolonged_exactly_and_uniform_state_stays_uniform():
    t0 = uniform_tree((4, 4, 4), 1)                      # level 1 declared, empty
    t1 = Tree((4, 4, 4), 1, (False, False, False))
    f0 = np.zeros_like(t1.exists[0])
    f0[1:3, 1:3, 1:3] = True
    t1.refine(0, f0)
    t1 = t1.pad_2to1()
    lin = lambda X, Y, Z: (1.0 + 0.5 * X - 0.25 * Y + 0.125 * Z, 0 * X + 0.1, 0 * X - 0.2, 0 * X + 0.3, 0 * X + 1.0)
    p = problem_from_tree(t0, fields=lin, bc=((1, 1),) * 3)
    q = problem_from_tree(t1, fields=lin, bc=((1, 1),) * 3)     # q.U: the field sampled on the new mesh
    a = oracle_for(p)
    b = oracle_for(q)
    b.set_state(np.zeros_like(q.U))
    b.transfer_from(a)
    Ub = b.get_state()
    # conserved variables of this state are linear in x, y, z (constant velocity and pressure): exact
    fine = q.level == 1
    assert fine.sum() == 64
    assert np.allclose(Ub[fine], q.U[fine], rtol=0, atol=2e-15)
    U = np.empty_like(p.U)
    U[:] = np.array([1.3, 0.4, -0.2, 0.7, 2.9])[None, :, None, None, None]
    a.set_state(U)
    b.transfer_from(a)
    assert (b.get_state() == np.array([1.3, 0.4, -0.2, 0.7, 2.9])[None, :, None, None, None]).all()


def test_coarsening_keeps_the_restricted_parents_and_two_levels_are_created_at_once():
    p = problem_from_tree(small_amr_tree(), mode=1)
    a = consistent(p)
    # coarsen: drop the level-2 patch
    q = problem_from_tree(refined_copy(extra=False, drop_inner=True), mode=1)
    b = oracle_for(q)
    b.transfer_from(a)
    key = lambda lv, ijk: [(int(l), *map(int, c)) for l, c in zip(lv, ijk)]
    old = {k: n for n, k in enumerate(key(p.level, p.ijk))}
    for n, k in enumerate(key(q.level, q.ijk)):
        assert np.array_equal(b.get_state()[n], a.get_state()[old[k]])
    # refine a uniform level-0 state by two levels in one transfer: the recursion prolongs twice
    u = problem_from_tree(uniform_tree((4, 4, 4), 2), mode=1)
    c = oracle_for(u)
    d = oracle_for(p)
    d.transfer_from(c)
    d2 = d.get_state().copy()
    d.restrict_all(0)
    scale = np.abs(d2).max(axis=(0, 2, 3, 4))[None, :, None, None, None]
    assert (np.abs(d.get_state() - d2) <= 6e-16 * scale).all()
    assert np.array_equal(d2[p.level == 0], c.get_state())
