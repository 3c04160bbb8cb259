"""Octree block lists (host side, numpy).  No method arithmetic here."""
import numpy as np

N = 8


class Tree:
    """exists[l] is a dense bool array [nbx<<l, nby<<l, nbz<<l]: block (bx,by,bz) of level l exists.

    Every block of every level holds data (non-leaf blocks too, SURVEY.md section 8 conventions)."""

    def __init__(self, nb0, max_level, periodic=(True, True, True)):
        self.nb0 = tuple(int(x) for x in nb0)
        self.max_level = int(max_level)
        self.periodic = tuple(bool(p) for p in periodic)
        self.exists = [np.zeros(tuple(n << l for n in self.nb0), dtype=bool) for l in range(max_level + 1)]
        self.exists[0][...] = True

    def refine(self, l, flags):
        """Split the level-l blocks flagged (dense bool array) into 8 children."""
        assert l < self.max_level
        flags = flags & self.exists[l]
        self.exists[l + 1] |= np.repeat(np.repeat(np.repeat(flags, 2, 0), 2, 1), 2, 2)

    def _dilate(self, a):
        out = a.copy()
        for d in range(3):
            lo = np.roll(out, 1, d)
            hi = np.roll(out, -1, d)
            if not self.periodic[d]:
                sl = [slice(None)] * 3
                sl[d] = 0
                lo[tuple(sl)] = False
                sl[d] = -1
                hi[tuple(sl)] = False
            out = out | lo | hi
        return out

    @staticmethod
    def _any8(a):
        s = a.shape
        return a.reshape(s[0] // 2, 2, s[1] // 2, 2, s[2] // 2, 2).any(axis=(1, 3, 5))

    def _ensure(self, l, need):
        """Make the level-l blocks in `need` exist (creating ancestors as required)."""
        missing = need & ~self.exists[l]
        if not missing.any():
            return False
        parents = self._any8(missing)
        self._ensure(l - 1, parents)
        self.refine(l - 1, parents)
        return True

    def pad_2to1(self):
        """Proper nesting over all 26 neighbours: a level-l block's neighbours exist at level >= l-1."""
        changed = True
        while changed:
            changed = False
            for l in range(self.max_level, 1, -1):
                if not self.exists[l].any():
                    continue
                need_c = self._any8(self._dilate(self.exists[l]))      # level l-1 blocks that must exist
                changed |= self._ensure(l - 1, need_c)
        return self

    def leaf_mask(self, l):
        if l == self.max_level:
            return self.exists[l].copy()
        return self.exists[l] & ~self._any8(self.exists[l + 1])

    def block_list(self):
        """(level[nb], ijk[nb,3]) level by level, lexicographic (bx slowest) within a level."""
        lev, ijk = [], []
        for l in range(self.max_level + 1):
            idx = np.argwhere(self.exists[l]).astype(np.int32)
            ijk.append(idx)
            lev.append(np.full(len(idx), l, dtype=np.int32))
        return np.concatenate(lev), np.concatenate(ijk)

    def census(self):
        return [int(e.sum()) for e in self.exists]


def uniform_tree(nb0, max_level=0, periodic=(True, True, True), fully_refined_to=0):
    t = Tree(nb0, max_level, periodic)
    for l in range(fully_refined_to):
        t.refine(l, t.exists[l].copy())
    return t


def tree_from_criterion(nb0, max_level, periodic, flag_fn):
    """flag_fn(l, ijk[n,3]) -> bool[n]: refine these level-l blocks.  2:1 padding afterwards."""
    t = Tree(nb0, max_level, periodic)
    for l in range(max_level):
        idx = np.argwhere(t.exists[l]).astype(np.int32)
        if len(idx) == 0:
            break
        fl = np.asarray(flag_fn(l, idx), dtype=bool)
        flags = np.zeros_like(t.exists[l])
        flags[idx[fl, 0], idx[fl, 1], idx[fl, 2]] = True
        t.refine(l, flags)
    return t.pad_2to1()


def blockify(field, nb):
    """[nz,ny,nx] uniform-grid field -> [nblocks][8][8][8] in (bx slowest, bz fastest) block order,
    matching Tree.block_list() of a uniform level-0 tree with nb0 = nb."""
    nbx, nby, nbz = nb
    a = field.reshape(nbz, N, nby, N, nbx, N)            # [bz,k,by,j,bx,i]
    return np.ascontiguousarray(a.transpose(4, 2, 0, 1, 3, 5)).reshape(nbx * nby * nbz, N, N, N)


def unblockify(blocks, nb):
    nbx, nby, nbz = nb
    a = blocks.reshape(nbx, nby, nbz, N, N, N)           # [bx,by,bz,k,j,i]
    return np.ascontiguousarray(a.transpose(2, 3, 1, 4, 0, 5)).reshape(nbz * N, nby * N, nbx * N)
