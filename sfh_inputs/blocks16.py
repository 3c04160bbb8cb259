"""Problems on blocks of 16^3 cells, derived from problems on 8^3 blocks: the same cells, grouped
differently.  Octant c = cx + 2 cy + 4 cz of the 16^3 block (l; I, J, K) is the 8^3 block (l; 2I + cx, 2J + cy, 2K + cz)
of a root grid twice as fine in blocks.  No method arithmetic."""
import dataclasses

import numpy as np


def split_blocks(level16, ijk16):
    """Block list of the octants, entry 8 b + c."""
    level16 = np.asarray(level16, dtype=np.int32)
    ijk16 = np.asarray(ijk16, dtype=np.int32).reshape(-1, 3)
    c = np.arange(8)
    off = np.stack([c & 1, (c >> 1) & 1, (c >> 2) & 1], axis=1).astype(np.int32)          # [8][3]
    ijk8 = (2 * ijk16[:, None, :] + off[None, :, :]).reshape(-1, 3)
    return np.repeat(level16, 8), np.ascontiguousarray(ijk8)


def merge_state(U8):
    """[8 nb][nv][8][8][8] in entry order 8 b + c  ->  [nb][nv][16][16][16]."""
    nb, nv = U8.shape[0] // 8, U8.shape[1]
    a = U8.reshape(nb, 2, 2, 2, nv, 8, 8, 8)                   # [b][cz][cy][cx][v][k][j][i]
    a = a.transpose(0, 4, 1, 5, 2, 6, 3, 7)                    # [b][v][cz][k][cy][j][cx][i]
    return np.ascontiguousarray(a).reshape(nb, nv, 16, 16, 16)


def split_state(U16):
    """Inverse of merge_state."""
    nb, nv = U16.shape[0], U16.shape[1]
    a = U16.reshape(nb, nv, 2, 8, 2, 8, 2, 8)                  # [b][v][cz][k][cy][j][cx][i]
    a = a.transpose(0, 2, 4, 6, 1, 3, 5, 7)                    # [b][cz][cy][cx][v][k][j][i]
    return np.ascontiguousarray(a).reshape(nb * 8, nv, 8, 8, 8)


def to16(p8):
    """The problem p8 (8^3 blocks, even root grid) on 16^3 blocks, and p8 reordered into the matching entry order
    8 b + c.  Every aligned 2x2x2 group of p8's blocks must be complete (true for every level > 0 of a valid octree,
    and for level 0 when the root grid is even); whether the groups form a valid octree of 16^3 blocks (refinement
    uniform over each group) is for the consumer to check."""
    assert all(n % 2 == 0 for n in p8.nb0), "root grid must be even"
    key = {}
    order16 = []
    for b in range(len(p8.level)):
        g = (int(p8.level[b]),) + tuple(int(x) >> 1 for x in p8.ijk[b])
        if g not in key:
            key[g] = len(order16)
            order16.append(g)
    nb16 = len(order16)
    assert len(p8.level) == 8 * nb16, "incomplete 2x2x2 groups"
    entry = np.empty(len(p8.level), dtype=np.int64)
    for b in range(len(p8.level)):
        g = (int(p8.level[b]),) + tuple(int(x) >> 1 for x in p8.ijk[b])
        c = (int(p8.ijk[b][0]) & 1) + 2 * (int(p8.ijk[b][1]) & 1) + 4 * (int(p8.ijk[b][2]) & 1)
        entry[8 * key[g] + c] = b
    level16 = np.array([g[0] for g in order16], dtype=np.int32)
    ijk16 = np.array([g[1:] for g in order16], dtype=np.int32).reshape(-1, 3)
    U8 = np.ascontiguousarray(p8.U[entry])
    p8e = dataclasses.replace(p8, level=np.ascontiguousarray(p8.level[entry]), ijk=np.ascontiguousarray(p8.ijk[entry]),
                              U=U8, name=p8.name + " (octant order)")
    p16 = dataclasses.replace(p8, nb0=tuple(n // 2 for n in p8.nb0), level=level16, ijk=ijk16, U=merge_state(U8),
                              name=p8.name + " (16^3 blocks)")
    return p16, p8e


def tree16_problem(t16, **kw):
    """Problem on the 16^3-block octree t16 (sfh_inputs.Tree) and the same problem on its 8^3 octants."""
    from .small import problem_from_tree
    level16, ijk16 = t16.block_list()
    level8, ijk8 = split_blocks(level16, ijk16)

    class _T:                                   # what problem_from_tree reads of a tree
        nb0 = tuple(2 * n for n in t16.nb0)
        max_level = t16.max_level
        periodic = t16.periodic

        @staticmethod
        def block_list():
            return level8, ijk8
    p8 = problem_from_tree(_T, **kw)
    return to16(p8)
