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


# ------------------------------------------------------------------ the regrid's block list (orc_regrid)
def tree_from_flags(p, flagged, periodic):
    """The same rules with an unrelated implementation (dense boolean arrays and dilation, sfh_inputs.Tree): children
    of blocks that are flagged, or have a flagged descendant, and exist in the new tree; then the 2:1 closure."""
    t = Tree(p.nb0, p.max_level, periodic)
    f = []
    for l in range(p.max_level + 1):
        f.append(np.zeros_like(t.exists[l]))
        sel = (p.level == l) & flagged
        f[l][p.ijk[sel, 0], p.ijk[sel, 1], p.ijk[sel, 2]] = True
    for l in range(p.max_level, 0, -1):              # a flagged block flags its ancestors (reading R33)
        s = f[l].shape
        f[l - 1] |= f[l].reshape(s[0] // 2, 2, s[1] // 2, 2, s[2] // 2, 2).any(axis=(1, 3, 5))
    for l in range(p.max_level):
        t.refine(l, f[l])
    return t.pad_2to1().block_list()


def properly_nested(level, ijk, nb0, periodic, max_level):
    have = [set() for _ in range(max_level + 1)]
    for l, c in zip(level, ijk):
        have[l].add(tuple(int(x) for x in c))
    for l in range(1, max_level + 1):
        for c in have[l]:
            if (c[0] >> 1, c[1] >> 1, c[2] >> 1) not in have[l - 1]:
                return False
            if l >= 2:
                for d in np.ndindex(3, 3, 3):
                    pos, ok = [], True
                    for a in range(3):
                        x, n = c[a] + d[a] - 1, nb0[a] << l
                        if x < 0 or x >= n:
                            if not periodic[a]:
                                ok = False
                            x %= n
                        pos.append(x >> 1)
                    if ok and tuple(pos) not in have[l - 1]:
                        return False
    return True


import pytest


@pytest.mark.parametrize("periodic,offset", [((True, True, True), (0, 0, 0)), ((False, True, False), (-1, 0, 1))])
@pytest.mark.parametrize("quantile", [0.2, 0.6, 0.9])
def test_regrid_block_list_follows_the_stated_rules(periodic, offset, quantile):
    p = problem_from_tree(small_amr_tree(periodic=periodic, offset=offset), mode=1)
    m = consistent(p)
    m.advance(1, 1)
    m.fill_ghosts(-1, 0, 0, 0.0)
    ind = m.refine_indicator(0)
    thr = float(np.sort(ind)[int(quantile * len(ind))])
    new = m.regrid(0, thr)
    lev, ijk = tree_from_flags(p, ind >= thr, periodic)
    assert np.array_equal(new.level, lev) and np.array_equal(new.ijk, ijk)
    assert properly_nested(new.level, new.ijk, p.nb0, periodic, p.max_level)
    # flagged blocks that survive have their 8 children; the tree is at most one level deeper than the old one anywhere
    old = {(int(l), *map(int, c)) for l, c in zip(p.level, p.ijk)}
    newset = {(int(l), *map(int, c)) for l, c in zip(new.level, new.ijk)}
    for b in np.nonzero((ind >= thr) & (p.level < p.max_level))[0]:
        k = (int(p.level[b]), *map(int, p.ijk[b]))
        if k in newset:
            assert (k[0] + 1, 2 * k[1], 2 * k[2], 2 * k[3]) in newset
    for (l, x, y, z) in newset:
        assert l == 0 or (l, x, y, z) in old or (l - 1, x >> 1, y >> 1, z >> 1) in old
    # and the state moved with it: blocks kept are copies, the hierarchy is restriction-consistent
    U0, U1 = m.get_state(), new.get_state()
    where = {(int(l), *map(int, c)): n for n, (l, c) in enumerate(zip(p.level, p.ijk))}
    for n, (l, c) in enumerate(zip(new.level, new.ijk)):
        k = (int(l), *map(int, c))
        if k in where:
            assert np.array_equal(U1[n], U0[where[k]])
    new.restrict_all(0)
    scale = np.abs(U1).max(axis=(0, 2, 3, 4))[None, :, None, None, None]
    assert (np.abs(new.get_state() - U1) <= 6e-16 * scale).all()


def test_regrid_with_nothing_flagged_returns_the_root_grid_and_everything_flagged_deepens_by_one_level():
    p = problem_from_tree(small_amr_tree(max_level=1), mode=1)
    p.max_level = 3
    m = consistent(p)
    m.fill_ghosts(-1, 0, 0, 0.0)
    none = m.regrid(0, 1e300)
    assert (none.level == 0).all() and len(none.level) == 64
    full = m.regrid(0, -1.0)
    assert [int((full.level == l).sum()) for l in range(4)] == [64, 512, 512, 0]       # level 2 under the old level-1 patch only


@pytest.mark.parametrize("which_fine", ["all", "one"])
def test_flagged_fine_block_keeps_its_ancestors(which_fine):
    """Reading R33: a feature smaller than a coarse cell.  Level-2 blocks carry a density pattern +-delta that averages
    to zero over every 2 x 2 x 2 cells, so the restricted levels 1 and 0 are exactly uniform (indicator 0) while the
    level-2 indicator is large.  The refinement above the flagged level-2 blocks must survive the regrid although
    no block of levels 0 and 1 is flagged by its own data."""
    p = problem_from_tree(small_amr_tree(), mode=1)
    assert p.max_level == 2
    U = np.zeros_like(p.U)
    U[:, 0] = 1.0
    U[:, 4] = 1.0 / (p.gamma - 1.0)
    fine = np.flatnonzero(p.level == 2)
    marked = fine if which_fine == "all" else fine[:1]
    k, j, i = np.meshgrid(np.arange(8), np.arange(8), np.arange(8), indexing="ij")
    U[marked, 0] += 0.125 * (1.0 - 2.0 * ((i + j + k) & 1))
    m = oracle_for(p, U)
    m.restrict_all(0)
    assert (m.get_state()[p.level < 2][:, 0] == 1.0).all()           # the pattern is invisible from above
    m.fill_ghosts(-1, 0, 0, 0.0)
    ind = m.refine_indicator(0)
    thr = 1e-2                                                        # the paper's threshold
    assert (ind[p.level < 2] == 0.0).all() and (ind[marked] > 1.0).all()
    new = m.regrid(0, thr)
    old = {(int(l), *map(int, c)) for l, c in zip(p.level, p.ijk)}
    newset = {(int(l), *map(int, c)) for l, c in zip(new.level, new.ijk)}
    for b in marked:                                                  # every flagged block and its ancestors are there
        l, c = int(p.level[b]), p.ijk[b]
        while l >= 0:
            assert (l, *map(int, c)) in newset
            l, c = l - 1, c >> 1
    if which_fine == "all":
        assert newset == old                                          # nothing above the flagged patch is lost
    else:
        assert len(newset) < len(old) and (new.level == 2).sum() == 8  # the other level-2 octets go, this one stays
    lev, ijk = tree_from_flags(p, ind >= thr, (True, True, True))
    assert np.array_equal(new.level, lev) and np.array_equal(new.ijk, ijk)
    assert properly_nested(new.level, new.ijk, p.nb0, (True, True, True), p.max_level)
