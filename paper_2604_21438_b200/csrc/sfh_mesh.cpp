// sfh_mesh.cpp — host-side octree block table, neighbour map and flux-register maps of libsfh.
//
// PAPER.md:96 (self-similar octree blocks), PAPER.md:100 ("lists describing the parent-child and
// neighboring relationships are created and managed on the hosts"; blocks ordered on a
// space-filling curve).  Here: Morton order within a level (siblings contiguous, child index
// c = cx + 2cy + 4cz), levels stored one after the other so each level is one slot range.
#include <algorithm>
#include <cstdio>
#include <numeric>
#include <unordered_map>

#include "sfh_internal.h"

namespace sfh {
namespace {

inline uint64_t spread3(uint64_t v) {  // 21 bits -> every third bit
  v &= 0x1FFFFFull;
  v = (v | (v << 32)) & 0x1F00000000FFFFull;
  v = (v | (v << 16)) & 0x1F0000FF0000FFull;
  v = (v | (v << 8)) & 0x100F00F00F00F00Full;
  v = (v | (v << 4)) & 0x10C30C30C30C30C3ull;
  v = (v | (v << 2)) & 0x1249249249249249ull;
  return v;
}
inline uint64_t morton(int x, int y, int z) { return spread3(x) | (spread3(y) << 1) | (spread3(z) << 2); }
inline uint64_t hkey(int l, int x, int y, int z) {
  return (uint64_t(l) << 60) | (uint64_t(x) << 40) | (uint64_t(y) << 20) | uint64_t(z);
}

struct Lookup {
  std::unordered_map<uint64_t, int32_t> map;
  const sfh_config* cfg;
  // Same-level block at (x,y,z) of level l after applying the domain boundary rule.
  // Returns slot >= 0, NBR_COARSE (inside the domain, no block) or NBR_OUTSIDE (beyond outflow).
  int32_t at(int l, int x, int y, int z) const {
    int c[3] = {x, y, z};
    for (int d = 0; d < 3; ++d) {
      const int n = cfg->nb0[d] << l;
      if (c[d] < 0) {
        if (cfg->bc[d][0] != 0) return NBR_OUTSIDE;
        c[d] += n;
      } else if (c[d] >= n) {
        if (cfg->bc[d][1] != 0) return NBR_OUTSIDE;
        c[d] -= n;
      }
    }
    auto it = map.find(hkey(l, c[0], c[1], c[2]));
    return it == map.end() ? NBR_COARSE : it->second;
  }
};

}  // namespace

// A mesh of 16^3-cell blocks is the mesh of their 8^3 octants: block (l; I, J, K) is the eight
// blocks (l; 2I + cx, 2J + cy, 2K + cz) of a root grid twice as fine in blocks, with the same cells.  The scheme does
// not depend on how cells are grouped into blocks, so nothing else changes; only the caller's arrays are laid out in
// 16^3 blocks (caller_pos2 in sfh_kernels.cuh).
int build_host_mesh(const sfh_config& cfg_in, int64_t nblocks_in, const int32_t* level_in, const int32_t* ijk_in,
                    HostMesh& m, std::string& err) {
  char buf[256];
  if ((cfg_in.ncell != N && cfg_in.ncell != 2 * N) || cfg_in.nghost != NG) {
    err = "only ncell = 8 or 16 and nghost = 2 are supported";
    return SFH_EINVAL;
  }
  const bool bs16 = cfg_in.ncell == 2 * N;
  sfh_config cfg = cfg_in;
  int64_t nblocks = nblocks_in;
  const int32_t *level = level_in, *ijk = ijk_in;
  std::vector<int32_t> level8, ijk8;
  if (bs16) {
    if (nblocks_in <= 0 || nblocks_in > (int64_t(1) << 25) || !level_in || !ijk_in) { err = "bad block list"; return SFH_EINVAL; }
    cfg.ncell = N;
    for (int d = 0; d < 3; ++d) {
      if (cfg.nb0[d] < 1 || cfg.nb0[d] > (1 << 19)) { err = "nb0 out of range"; return SFH_EINVAL; }
      cfg.nb0[d] *= 2;
    }
    nblocks = 8 * nblocks_in;
    level8.resize(size_t(nblocks));
    ijk8.resize(size_t(3 * nblocks));
    for (int64_t b = 0; b < nblocks_in; ++b)
      for (int c = 0; c < 8; ++c) {
        level8[8 * b + c] = level_in[b];
        for (int d = 0; d < 3; ++d) ijk8[3 * (8 * b + c) + d] = 2 * ijk_in[3 * b + d] + ((c >> d) & 1);
      }
    level = level8.data();
    ijk = ijk8.data();
  }
  if (cfg.max_level < 0 || cfg.max_level >= MAX_LEVELS) { err = "max_level out of range"; return SFH_EINVAL; }
  if (nblocks <= 0 || nblocks > (int64_t(1) << 28) || !level || !ijk) { err = "bad block list"; return SFH_EINVAL; }
  for (int d = 0; d < 3; ++d) {
    if (cfg.nb0[d] < 1 || (int64_t(cfg.nb0[d]) << cfg.max_level) > (1 << 20)) { err = "nb0 out of range"; return SFH_EINVAL; }
    if (!(cfg.box_len[d] > 0.0)) { err = "box_len must be positive"; return SFH_EINVAL; }
    for (int s = 0; s < 2; ++s) if (cfg.bc[d][s] != 0 && cfg.bc[d][s] != 1) { err = "bc must be 0 or 1"; return SFH_EINVAL; }
    if ((cfg.bc[d][0] == 0) != (cfg.bc[d][1] == 0)) { err = "periodic bc must be set on both faces of an axis"; return SFH_EINVAL; }
  }
  if (!(cfg.gamma > 1.0) || !(cfg.cfl > 0.0)) { err = "gamma must be > 1 and cfl > 0"; return SFH_EINVAL; }
  if (cfg.nscalar < 0 || cfg.nscalar > SFH_MAX_SCALARS) { err = "nscalar out of range"; return SFH_EINVAL; }

  m = HostMesh();
  m.cfg = cfg;
  m.bs16 = bs16;
  m.nb = nblocks;
  m.nlev = cfg.max_level + 1;
  for (int l = 0; l < m.nlev; ++l) m.h[l] = cfg.box_len[0] / (double(cfg.nb0[0]) * N * double(1 << l));

  // ---- range checks, ordering (level-major, Morton within a level)
  std::vector<uint64_t> mkey(nblocks);
  for (int64_t b = 0; b < nblocks; ++b) {
    const int l = level[b];
    if (l < 0 || l >= m.nlev) { snprintf(buf, sizeof buf, "block %lld: level %d out of range", (long long)b, l); err = buf; return SFH_EMESH; }
    for (int d = 0; d < 3; ++d) {
      const int c = ijk[3 * b + d];
      if (c < 0 || c >= (cfg.nb0[d] << l)) { snprintf(buf, sizeof buf, "block %lld: coordinate out of range", (long long)b); err = buf; return SFH_EMESH; }
    }
    mkey[b] = morton(ijk[3 * b], ijk[3 * b + 1], ijk[3 * b + 2]);
  }
  m.perm.resize(nblocks);
  std::iota(m.perm.begin(), m.perm.end(), int64_t(0));
  std::sort(m.perm.begin(), m.perm.end(), [&](int64_t a, int64_t b) {
    if (level[a] != level[b]) return level[a] < level[b];
    if (mkey[a] != mkey[b]) return mkey[a] < mkey[b];
    return a < b;
  });
  m.lev.resize(nblocks);
  m.coord.resize(3 * nblocks);
  m.lev_first.assign(m.nlev, 0);
  m.lev_count.assign(m.nlev, 0);
  Lookup lk;
  lk.cfg = &m.cfg;
  lk.map.reserve(size_t(nblocks) * 2);
  for (int64_t s = 0; s < nblocks; ++s) {
    const int64_t b = m.perm[s];
    m.lev[s] = level[b];
    for (int d = 0; d < 3; ++d) m.coord[3 * s + d] = ijk[3 * b + d];
    m.lev_count[level[b]] += 1;
    if (!lk.map.emplace(hkey(level[b], ijk[3 * b], ijk[3 * b + 1], ijk[3 * b + 2]), int32_t(s)).second) {
      snprintf(buf, sizeof buf, "duplicate block (level %d; %d,%d,%d)", level[b], ijk[3 * b], ijk[3 * b + 1], ijk[3 * b + 2]);
      err = buf;
      return SFH_EMESH;
    }
  }
  for (int l = 1; l < m.nlev; ++l) m.lev_first[l] = m.lev_first[l - 1] + m.lev_count[l - 1];
  if (m.lev_count[0] != int64_t(cfg.nb0[0]) * cfg.nb0[1] * cfg.nb0[2]) { err = "level 0 must hold every root block"; return SFH_EMESH; }

  // ---- parent / children (complete sibling sets)
  m.parent.assign(nblocks, -1);
  m.child0.assign(nblocks, -1);
  for (int64_t s = 0; s < nblocks; ++s) {
    const int l = m.lev[s];
    const int x = m.coord[3 * s], y = m.coord[3 * s + 1], z = m.coord[3 * s + 2];
    if (l == 0) continue;
    auto it = lk.map.find(hkey(l - 1, x >> 1, y >> 1, z >> 1));
    if (it == lk.map.end()) { snprintf(buf, sizeof buf, "block (level %d; %d,%d,%d) has no parent", l, x, y, z); err = buf; return SFH_EMESH; }
    m.parent[s] = it->second;
    const int c = (x & 1) + 2 * (y & 1) + 4 * (z & 1);
    if (c == 0) {
      for (int q = 0; q < 8; ++q) {
        auto jt = lk.map.find(hkey(l, (x & ~1) + (q & 1), (y & ~1) + ((q >> 1) & 1), (z & ~1) + ((q >> 2) & 1)));
        if (jt == lk.map.end() || jt->second != int32_t(s) + q) {
          snprintf(buf, sizeof buf, "incomplete sibling set under (level %d; %d,%d,%d)", l - 1, x >> 1, y >> 1, z >> 1);
          err = buf;
          return SFH_EMESH;
        }
      }
      m.child0[it->second] = int32_t(s);
    } else if (lk.map.find(hkey(l, x & ~1, y & ~1, z & ~1)) == lk.map.end()) {
      snprintf(buf, sizeof buf, "incomplete sibling set under (level %d; %d,%d,%d)", l - 1, x >> 1, y >> 1, z >> 1);
      err = buf;
      return SFH_EMESH;
    }
  }

  // ---- 27-neighbour map + proper nesting (reading R25)
  m.nbr27.assign(size_t(nblocks) * 27, NBR_COARSE);
  for (int64_t s = 0; s < nblocks; ++s) {
    const int l = m.lev[s];
    const int x = m.coord[3 * s], y = m.coord[3 * s + 1], z = m.coord[3 * s + 2];
    for (int dz = -1; dz <= 1; ++dz) for (int dy = -1; dy <= 1; ++dy) for (int dx = -1; dx <= 1; ++dx) {
      const int32_t q = lk.at(l, x + dx, y + dy, z + dz);
      m.nbr27[s * 27 + (dz + 1) * 9 + (dy + 1) * 3 + (dx + 1)] = q;
      if (q == NBR_COARSE) {
        // floor division by two of a possibly negative coordinate, then the boundary rule of level l-1
        auto half = [](int v) { return v >= 0 ? v >> 1 : -((-v + 1) >> 1); };
        if (l == 0 || lk.at(l - 1, half(x + dx), half(y + dy), half(z + dz)) < 0) {
          snprintf(buf, sizeof buf, "improper nesting next to (level %d; %d,%d,%d)", l, x, y, z);
          err = buf;
          return SFH_EMESH;
        }
      }
    }
  }

  // ---- per-face halo sources; fine-side coarse-fine faces (ghost slab + register R)
  m.face_src.assign(size_t(nblocks) * 6, SRC_OUTFLOW);
  m.cf_first.assign(m.nlev, 0);
  m.cf_count.assign(m.nlev, 0);
  static const int fdx[6][3] = {{-1, 0, 0}, {1, 0, 0}, {0, -1, 0}, {0, 1, 0}, {0, 0, -1}, {0, 0, 1}};
  for (int64_t s = 0; s < nblocks; ++s)
    for (int f = 0; f < 6; ++f) {
      const int32_t q = m.nbr27[s * 27 + (fdx[f][2] + 1) * 9 + (fdx[f][1] + 1) * 3 + (fdx[f][0] + 1)];
      if (q >= 0) m.face_src[s * 6 + f] = q;
      else if (q == NBR_OUTSIDE) m.face_src[s * 6 + f] = SRC_OUTFLOW;
      else {
        m.face_src[s * 6 + f] = src_from_slot(int(m.cf_block.size()));
        m.cf_block.push_back(int32_t(s));
        m.cf_face.push_back(f);
        m.cf_count[m.lev[s]] += 1;
      }
    }
  for (int l = 1; l < m.nlev; ++l) m.cf_first[l] = m.cf_first[l - 1] + m.cf_count[l - 1];

  // ---- coarse-side registers: a leaf whose face neighbour is covered (has children)
  m.fslot.assign(size_t(nblocks) * 6, -1);
  m.nfh = 0;
  for (int64_t s = 0; s < nblocks; ++s) {
    if (m.child0[s] >= 0) continue;
    for (int f = 0; f < 6; ++f) {
      const int32_t q = m.face_src[s * 6 + f];
      if (q < 0 || m.child0[q] < 0) continue;
      m.fslot[s * 6 + f] = int32_t(m.nfh++);
      const int d = f >> 1, side = f & 1;
      // children of q that touch the shared face: their coordinate along d is 0 if the face is on
      // my upper side, 1 if on my lower side; their opposite face carries the fine register.
      for (int qq = 0; qq < 4; ++qq) {
        int cc[3];
        int t = 0;
        for (int dd = 0; dd < 3; ++dd) {
          if (dd == d) cc[dd] = side ? 0 : 1;
          else { cc[dd] = (qq >> t) & 1; ++t; }
        }
        const int32_t child = m.child0[q] + cc[0] + 2 * cc[1] + 4 * cc[2];
        const int32_t src = m.face_src[size_t(child) * 6 + 2 * d + (1 - side)];
        if (src > -2) { err = "internal: coarse-fine face without a fine register"; return SFH_EMESH; }
        m.fh_src.push_back(-2 - src);
      }
    }
  }

  // ---- per-level work lists
  m.restrict_first.assign(m.nlev, 0); m.restrict_count.assign(m.nlev, 0);
  m.reflux_first.assign(m.nlev, 0); m.reflux_count.assign(m.nlev, 0);
  for (int64_t s = 0; s < nblocks; ++s) {
    if (m.child0[s] >= 0) { m.restrict_list.push_back(int32_t(s)); m.restrict_count[m.lev[s]] += 1; }
    bool any = false;
    for (int f = 0; f < 6; ++f) any |= m.fslot[s * 6 + f] >= 0;
    if (any) { m.reflux_list.push_back(int32_t(s)); m.reflux_count[m.lev[s]] += 1; }
  }
  for (int l = 1; l < m.nlev; ++l) {
    m.restrict_first[l] = m.restrict_first[l - 1] + m.restrict_count[l - 1];
    m.reflux_first[l] = m.reflux_first[l - 1] + m.reflux_count[l - 1];
  }
  return SFH_OK;
}

// ---- regrid: the block list of the new tree (reading R31) ----------------
// ind[slot]: refinement indicator of every block of the old mesh (library order).  New tree: all root blocks; the
// octet under every old block of level < max_level that is still in the new tree and is flagged -- ind >= threshold
// (eq. 33 is written with >=) or a flagged descendant in the old mesh (reading R33) --; then the closure under proper nesting over the 26 neighbours (reading R25), adding whole octets
// and their ancestors.  Output: level-major, (bx, by, bz) lexicographic within a level.
int regrid_block_list(const HostMesh& old, const double* ind, double threshold, std::vector<int32_t>& level,
                      std::vector<int32_t>& ijk) {
  const sfh_config& cfg = old.cfg;
  const int nlev = old.nlev;
  std::vector<std::unordered_map<uint64_t, char>> have(nlev);     // per level: key -> present
  std::vector<std::vector<int32_t>> list(nlev);                   // per level: coordinates, 3 per block
  auto add = [&](int l, int x, int y, int z) {
    if (have[l].emplace(hkey(l, x, y, z), 1).second) { list[l].push_back(x); list[l].push_back(y); list[l].push_back(z); return true; }
    return false;
  };
  auto add_octet = [&](int l, int px, int py, int pz) {           // children of (px,py,pz) of level l-1
    bool any = false;
    for (int q = 0; q < 8; ++q) any |= add(l, 2 * px + (q & 1), 2 * py + ((q >> 1) & 1), 2 * pz + ((q >> 2) & 1));
    return any;
  };
  for (int64_t s = 0; s < old.nb && old.lev[s] == 0; ++s) add(0, old.coord[3 * s], old.coord[3 * s + 1], old.coord[3 * s + 2]);
  // flagged: own indicator >= threshold, or a flagged descendant in the old mesh (slots are level-major, so one
  // pass from the back reaches every ancestor)
  std::vector<char> flag(size_t(old.nb));
  for (int64_t s = 0; s < old.nb; ++s) flag[size_t(s)] = ind[s] >= threshold;
  for (int64_t s = old.nb - 1; s >= 0; --s)
    if (flag[size_t(s)] && old.parent[size_t(s)] >= 0) flag[size_t(old.parent[size_t(s)])] = 1;
  for (int64_t s = 0; s < old.nb; ++s) {                          // slots are level-major: parents come first
    const int l = old.lev[s];
    if (l + 1 >= nlev || !flag[size_t(s)]) continue;
    const int x = old.coord[3 * s], y = old.coord[3 * s + 1], z = old.coord[3 * s + 2];
    if (have[l].count(hkey(l, x, y, z))) add_octet(l + 1, x, y, z);
  }
  // closure: a work list of blocks whose 26 neighbour positions still have to be checked
  struct Item { int l, x, y, z; };
  std::vector<Item> work;
  for (int l = 2; l < nlev; ++l)
    for (size_t q = 0; q + 2 < list[l].size(); q += 3) work.push_back({l, list[l][q], list[l][q + 1], list[l][q + 2]});
  // make block (x,y,z) of level l exist: its octet, after the parent's; new blocks of level >= 2 join the work list
  auto ensure = [&](auto&& self, int l, int x, int y, int z) -> void {
    if (l == 0 || have[l].count(hkey(l, x, y, z))) return;
    self(self, l - 1, x >> 1, y >> 1, z >> 1);
    const size_t before = list[l].size();
    add_octet(l, x >> 1, y >> 1, z >> 1);
    if (l >= 2)
      for (size_t q = before; q + 2 < list[l].size(); q += 3) work.push_back({l, list[l][q], list[l][q + 1], list[l][q + 2]});
  };
  while (!work.empty()) {
    const Item it = work.back();
    work.pop_back();
    for (int dz = -1; dz <= 1; ++dz) for (int dy = -1; dy <= 1; ++dy) for (int dx = -1; dx <= 1; ++dx) {
      int c[3] = {it.x + dx, it.y + dy, it.z + dz};
      bool outside = false;
      for (int d = 0; d < 3; ++d) {
        const int n = cfg.nb0[d] << it.l;
        if (c[d] < 0) { if (cfg.bc[d][0] != 0) outside = true; else c[d] += n; }
        else if (c[d] >= n) { if (cfg.bc[d][1] != 0) outside = true; else c[d] -= n; }
      }
      if (!outside) ensure(ensure, it.l - 1, c[0] >> 1, c[1] >> 1, c[2] >> 1);
    }
  }
  level.clear();
  ijk.clear();
  for (int l = 0; l < nlev; ++l) {
    const size_t n = list[l].size() / 3;
    std::vector<size_t> order(n);
    std::iota(order.begin(), order.end(), size_t(0));
    const std::vector<int32_t>& c = list[l];
    std::sort(order.begin(), order.end(), [&](size_t a, size_t b) {
      if (c[3 * a] != c[3 * b]) return c[3 * a] < c[3 * b];
      if (c[3 * a + 1] != c[3 * b + 1]) return c[3 * a + 1] < c[3 * b + 1];
      return c[3 * a + 2] < c[3 * b + 2];
    });
    for (size_t q : order) { level.push_back(l); ijk.push_back(c[3 * q]); ijk.push_back(c[3 * q + 1]); ijk.push_back(c[3 * q + 2]); }
  }
  return SFH_OK;
}

}  // namespace sfh
