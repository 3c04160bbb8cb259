"""The C-ABI library loads without a GPU and exports every symbol include/sfh.h declares; the host
mesh builder (block table, neighbour map, validation) works on the CPU.  No compute calls here."""
import ctypes as C

import numpy as np
import pytest

import paper_2604_21438_b200 as sfh
from helpers import small_amr_tree
from sfh_inputs import uniform_tree


def test_library_exports_every_declared_symbol():
    L = sfh.load_library()
    names = sfh.declared_symbols()
    assert len(names) >= 20 and "sfh_create_mesh" in names and "sfh_hydro_step" in names
    for n in ("sfh_create_mesh", "sfh_fill_ghosts", "sfh_hydro_step", "sfh_flux_correct", "sfh_cfl_dt"):
        assert n in names          # the five calls BASELINE.json's north_star names
    for n in names:
        assert hasattr(L, n), n


def test_product_does_not_touch_the_oracle():
    import os
    root = os.path.dirname(os.path.abspath(sfh.__file__))
    for dirpath, _, files in os.walk(root):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "sfh_oracle" not in text, f
                assert "libsfh_oracle" not in text, f


def _mesh(t, bc=((0, 0),) * 3, **kw):
    level, ijk = t.block_list()
    return sfh.Mesh(t.nb0, t.max_level, bc, (1.0, 1.0, 1.0), 1.4, 0.4, level, ijk, bind=False, **kw), level, ijk


def test_uniform_mesh_tables():
    m, level, ijk = _mesh(uniform_tree((4, 4, 4)))
    assert m.level_range(0) == (0, 64)
    perm = m.block_order()
    assert sorted(perm.tolist()) == list(range(64))
    assert m.num_faces() == (0, 0)
    assert m.state_bytes() >= 64 * 5 * 512 * 8
    assert abs(m.cell_width(0) - 1.0 / 32) < 1e-18


def test_amr_mesh_tables_and_level_ranges():
    t = small_amr_tree()
    m, level, ijk = _mesh(t)
    census = t.census()
    first = 0
    perm = m.block_order()
    for l, c in enumerate(census):
        assert m.level_range(l) == (first, c)
        assert (level[perm[first:first + c]] == l).all()
        first += c
    nfine, ncoarse = m.num_faces()
    # the refined patch is a cube of 2x2x2 root blocks -> 4x4x4 level-1 blocks: 6 faces of 16 block faces;
    # the nested level-2 patch 2x2x2 level-1 blocks -> 4^3 level-2 blocks: again 96
    assert nfine == 96 + 96
    # coarse side: each coarse leaf face touching a covered block: 6 faces x 4 blocks, twice
    assert ncoarse == 24 + 24
    assert m.cell_width(2) == m.cell_width(0) / 4


def test_mesh_validation_rejects_bad_trees():
    t = small_amr_tree()
    level, ijk = t.block_list()
    kw = dict(bind=False)
    args = (t.nb0, t.max_level, ((0, 0),) * 3, (1.0, 1.0, 1.0), 1.4, 0.4)
    # duplicate block
    with pytest.raises(sfh.SfhError) as e:
        sfh.Mesh(*args, np.concatenate([level, level[-1:]]), np.concatenate([ijk, ijk[-1:]]), **kw)
    assert e.value.code == -2
    # missing sibling
    with pytest.raises(sfh.SfhError) as e:
        sfh.Mesh(*args, level[:-1], ijk[:-1], **kw)
    assert e.value.code == -2
    # a level-2 octet without level-1 parent
    with pytest.raises(sfh.SfhError) as e:
        lv = np.concatenate([level, np.full(8, 2, np.int32)])
        oc = np.array([[cx, cy, cz] for cz in (0, 1) for cy in (0, 1) for cx in (0, 1)], np.int32)
        sfh.Mesh(*args, lv, np.concatenate([ijk, oc]), **kw)
    assert e.value.code == -2
    # improper nesting: level-2 octet directly at the edge of the level-1 patch (its outer neighbour is level 0)
    t2 = small_amr_tree(max_level=1)
    t2.max_level = 2
    t2.exists.append(np.zeros(tuple(4 * n for n in t2.nb0), dtype=bool))
    f1 = np.zeros_like(t2.exists[1])
    f1[2, 2, 2] = True                     # corner block of the level-1 patch [2,6)^3
    t2.refine(1, f1)
    lv, ij = t2.block_list()
    with pytest.raises(sfh.SfhError) as e:
        sfh.Mesh(t2.nb0, 2, ((0, 0),) * 3, (1.0, 1.0, 1.0), 1.4, 0.4, lv, ij, **kw)
    assert e.value.code == -2 and "nesting" in str(e.value)
    # bad arguments
    with pytest.raises(sfh.SfhError) as e:
        sfh.Mesh(t.nb0, t.max_level, ((0, 1),) * 3, (1.0, 1.0, 1.0), 1.4, 0.4, level, ijk, **kw)
    assert e.value.code == -1
    # empty block list: a defined error, not a crash
    with pytest.raises(sfh.SfhError) as e:
        sfh.Mesh((1, 1, 1), 0, ((0, 0),) * 3, (1.0, 1.0, 1.0), 1.4, 0.4, np.zeros(0, np.int32),
                 np.zeros((0, 3), np.int32), **kw)
    assert e.value.code == -1


def test_compute_calls_fail_loudly_without_binding():
    m, _, _ = _mesh(uniform_tree((2, 2, 2)))
    dt = C.c_double()
    rc = m.L.sfh_cfl_dt(m.h, -1, C.byref(dt), None)
    assert rc == -5          # SFH_ESTATE: not bound; there is no CPU fallback
    rc = m.L.sfh_hydro_step(m.h, -1, 1e-3, 0, 0.0, 0.0, None)
    assert rc == -5
    import torch
    if not torch.cuda.is_available():
        with pytest.raises(sfh.SfhError):
            m.bind()


def test_regrid_block_list_host_logic_matches_the_stated_rules():
    """sfh_regrid_from_indicator (host only): the same block list as the dense-array construction of
    sfh_inputs.Tree (children of blocks that are flagged or have a flagged descendant, 2:1 closure), in the documented order."""
    from sfh_inputs import Tree
    rng = np.random.default_rng(5)
    for periodic, offset in (((True, True, True), (0, 0, 0)), ((False, True, False), (-1, 0, 1))):
        t = small_amr_tree(periodic=periodic, offset=offset)
        bc = tuple((0, 0) if per else (1, 1) for per in periodic)
        m, level, ijk = _mesh(t, bc=bc)
        for thr in (0.15, 0.5, 0.85):
            ind = rng.random(len(level))
            new = m.regrid_from_indicator(ind, thr)
            ref = Tree(t.nb0, t.max_level, periodic)
            f = []
            for l in range(t.max_level + 1):
                f.append(np.zeros_like(ref.exists[l]))
                sel = (level == l) & (ind >= thr)
                f[l][ijk[sel, 0], ijk[sel, 1], ijk[sel, 2]] = True
            for l in range(t.max_level, 0, -1):      # a flagged block flags its ancestors (reading R33)
                sh = f[l].shape
                f[l - 1] |= f[l].reshape(sh[0] // 2, 2, sh[1] // 2, 2, sh[2] // 2, 2).any(axis=(1, 3, 5))
            for l in range(t.max_level):
                ref.refine(l, f[l])
            lev, ij = ref.pad_2to1().block_list()
            assert np.array_equal(new.level, lev) and np.array_equal(new.ijk, ij)
            assert new.cfg.nscalar == m.cfg.nscalar and new.max_level == m.max_level
    with pytest.raises(sfh.SfhError):       # null indicator: a defined error
        m._chk(m.L.sfh_regrid_from_indicator(m.h, None, 0.5, C.byref(C.c_void_p())))


def test_mesh_of_16_cell_blocks_is_the_mesh_of_their_octants():
    """ncell = 16 (sfh.h): the block list counts 16^3 blocks; tables, level ranges and the block
    order refer to their 8^3 octants, entry 8 * block + octant."""
    t = small_amr_tree()
    level, ijk = t.block_list()
    m16 = sfh.Mesh(t.nb0, t.max_level, ((0, 0),) * 3, (1.0, 1.0, 1.0), 1.4, 0.4, level, ijk, bind=False, ncell=16)
    from sfh_inputs import split_blocks
    l8, ijk8 = split_blocks(level, ijk)
    m8 = sfh.Mesh(tuple(2 * n for n in t.nb0), t.max_level, ((0, 0),) * 3, (1.0, 1.0, 1.0), 1.4, 0.4, l8, ijk8, bind=False)
    assert m16.nentries() == 8 * len(level) == m8.nentries()
    assert np.array_equal(m16.block_order(), m8.block_order())
    assert m16.num_faces() == m8.num_faces() and m16.state_bytes() == m8.state_bytes()
    assert m16.cell_width(1) == m8.cell_width(1) == 1.0 / (t.nb0[0] * 16 * 2)
    for l in range(t.max_level + 1):
        assert m16.level_range(l) == m8.level_range(l)
    with pytest.raises(sfh.SfhError):
        sfh.Mesh(t.nb0, t.max_level, ((0, 0),) * 3, (1.0, 1.0, 1.0), 1.4, 0.4, level, ijk, bind=False, ncell=12)
