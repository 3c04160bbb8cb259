"""Pins of the oracle built with blocks of 16^3 cells (oracle/build.py,
-DSFH_ORACLE_N=16).  The scheme is defined per cell and per face: how the cells are grouped into
blocks must not change a single bit of the result.  So the 16^3 oracle on a mesh of 16^3 blocks has to reproduce,
bitwise, the 8^3 oracle (pinned by tests/test_oracle_*.py) on the mesh of their octants: uniform and AMR, synchronous
and sub-cycled, with outflow boundaries, with the Roe solver, with passive scalars.  A wrong face count, register
size, ghost width or child offset in the N-dependent parts of the oracle breaks this."""
import numpy as np
import pytest

from oracle import oracle_for
from sfh_inputs import Tree, make_config, merge_state, split_state, to16, tree16_problem, uniform_tree


def amr16(periodic=(True, True, True)):
    t = Tree((4, 3, 3), 2, periodic)
    f0 = np.zeros_like(t.exists[0]); f0[1:2, 1:2, 1:2] = True
    t.refine(0, f0)
    f1 = np.zeros_like(t.exists[1]); f1[2:3, 2:4, 3:4] = True
    t.refine(1, f1)
    return t.pad_2to1()


def run_pair(p16, p8, nsteps, mode, roe=False):
    o16, o8 = oracle_for(p16), oracle_for(p8)
    assert o16.n == 16 and o8.n == 8
    for o in (o16, o8):
        if roe:
            o.set_riemann("roe")
        o.restrict_all(0)
        o.advance(nsteps, mode)
    assert o16.t.value == o8.t.value
    assert np.array_equal(o16.nupd, o8.nupd)
    assert np.array_equal(split_state(o16.get_state()), o8.get_state())
    return o16


def test_merge_and_split_are_inverse_and_keep_cell_positions():
    rng = np.random.default_rng(3)
    U8 = rng.standard_normal((16, 6, 8, 8, 8))
    U16 = merge_state(U8)
    assert U16.shape == (2, 6, 16, 16, 16)
    assert np.array_equal(split_state(U16), U8)
    # octant c = cx + 2 cy + 4 cz of block 1, variable 2, cell (k, j, i) = (3, 4, 5)
    for c in range(8):
        cx, cy, cz = c & 1, (c >> 1) & 1, c >> 2
        assert U16[1, 2, 8 * cz + 3, 8 * cy + 4, 8 * cx + 5] == U8[8 + c, 2, 3, 4, 5]


@pytest.mark.parametrize("name,scale", [("C2", 8), ("C1", 1)])
def test_uniform_mesh_bitwise(name, scale):
    p16, p8 = to16(make_config(name, scale))
    assert p16.U.shape[0] * 8 == p8.U.shape[0]
    run_pair(p16, p8, 3, 0)


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("roe", [False, True])
def test_amr_mesh_bitwise(mode, roe):
    p16, p8 = tree16_problem(amr16(), mode=mode)
    assert p16.census()[1] < 8 * p16.census()[0] and p16.census()[2] > 0      # coarse-fine faces at both interfaces
    assert p8.census() == [8 * c for c in p16.census()]
    o16 = run_pair(p16, p8, 2, mode, roe)
    if mode == 1:
        assert o16.nupd[2] > o16.nupd[0]            # the fine levels did sub-cycle


def test_amr_mesh_with_outflow_faces_and_scalars_bitwise():
    from sfh_inputs import add_scalars
    p16, p8 = tree16_problem(amr16(periodic=(False, True, False)), mode=1)
    s = [lambda X, Y, Z: 0.5 + 0.4 * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Z), lambda X, Y, Z: 0.37]
    p8s = add_scalars(p8, s)
    p16s, p8e = to16(p8s)
    assert np.array_equal(p16s.ijk, p16.ijk)
    run_pair(p16s, p8e, 2, 1)


def test_mass_conserved_on_16_blocks():
    p16, _ = tree16_problem(amr16(), mode=1)
    from helpers import leaf_totals
    o = oracle_for(p16)
    o.restrict_all(0)
    m0 = leaf_totals(o.is_leaf(), o.get_state(), p16.level, o.cell_width(0))
    o.advance(2, 1)
    m1 = leaf_totals(o.is_leaf(), o.get_state(), p16.level, o.cell_width(0))
    assert np.all(np.abs(m1 - m0) <= 1e-13 * np.maximum(np.abs(m0), 1.0))
