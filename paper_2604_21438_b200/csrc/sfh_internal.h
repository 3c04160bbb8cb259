// sfh_internal.h — shared declarations of libsfh (host mesh builder, kernels, C ABI).
// Not part of the public interface (include/sfh.h).  Shares nothing with oracle/.
#pragma once

#include <cstdint>
#include <string>
#include <vector>

#include "../../include/sfh.h"

namespace sfh {

constexpr int N = 8;            // cells per block edge
constexpr int NG = 2;           // ghost layers
constexpr int NV = 5;           // rho, rho v, rho E
constexpr int NC = N * N * N;   // interior cells per block
constexpr int BLK = NV * NC;    // doubles per block (interior-only layout) = 2560 -> 20480 B
constexpr int FACE = N * N;     // cells of one block face
constexpr int SLAB = NV * NG * FACE;  // doubles of one 2-layer ghost slab = 640 -> 5120 B
constexpr int REG = NV * FACE;        // doubles of one flux register = 320
constexpr int MAX_LEVELS = 12;

// face_src codes (per block, per face f = 2*axis + side)
constexpr int SRC_OUTFLOW = -1;                      // zero-gradient copy of the block's own layer
inline int src_from_slot(int slot) { return -2 - slot; }   // coarse-fine ghost slab `slot`
// nbr27 codes
constexpr int NBR_COARSE = -1;   // no same-level block there (inside the domain)
constexpr int NBR_OUTSIDE = -2;  // beyond an outflow boundary

struct HostMesh {
  sfh_config cfg{};                   // as the library works on it: ncell = 8 (a 16^3 mesh: nb0 doubled)
  int bs16 = 0;                       // the caller's blocks hold 16^3 cells: entry e of the block list below is
                                      // octant e & 7 of the caller's block e >> 3
  int64_t nb = 0;
  int nlev = 0;
  std::vector<int64_t> perm;          // library slot -> caller index
  std::vector<int32_t> lev;           // per slot
  std::vector<int32_t> coord;         // [nb][3]
  std::vector<int32_t> parent;        // slot of the parent or -1
  std::vector<int32_t> child0;        // slot of child 0 (children are contiguous, c = cx+2cy+4cz) or -1
  std::vector<int32_t> nbr27;         // [nb][27], index (dz+1)*9+(dy+1)*3+(dx+1)
  std::vector<int32_t> face_src;      // [nb][6]
  std::vector<int32_t> fslot;         // [nb][6] coarse-side register slot or -1
  std::vector<int64_t> lev_first, lev_count;        // [nlev]
  // coarse-fine faces, fine side (ghost slab + flux register R), sorted by block => by level
  std::vector<int32_t> cf_block, cf_face;           // [ncf]
  std::vector<int64_t> cf_first, cf_count;          // [nlev]
  // coarse-leaf faces that get a correction (register FH)
  int64_t nfh = 0;
  std::vector<int32_t> fh_src;        // [nfh][4] fine-side slots of the 4 children, q = qa + 2 qb
  // per level work lists
  std::vector<int32_t> restrict_list; // slots of non-leaf blocks, by level
  std::vector<int64_t> restrict_first, restrict_count;
  std::vector<int32_t> reflux_list;   // slots of blocks with any fslot >= 0, by level
  std::vector<int64_t> reflux_first, reflux_count;
  double h[MAX_LEVELS] = {0};
};

// Builds every table above from the caller's block list.  Returns SFH_OK / SFH_EINVAL / SFH_EMESH
// and an explanation in `err`.
int build_host_mesh(const sfh_config& cfg, int64_t nblocks, const int32_t* level, const int32_t* ijk,
                    HostMesh& out, std::string& err);

// Block list (caller order: level-major, lexicographic within a level) of the regridded tree: sfh_mesh.cpp.
int regrid_block_list(const HostMesh& old, const double* ind, double threshold, std::vector<int32_t>& level,
                      std::vector<int32_t>& ijk);

void set_error(const std::string& s);

}  // namespace sfh
