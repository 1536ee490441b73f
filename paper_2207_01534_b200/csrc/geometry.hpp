// geometry.hpp -- host-side classification and compaction of the voxel mask (product code;
// shares nothing with oracle/).  See DESIGN.md "Data layout in HBM".
//
// Voxels are classified as fluid, wall solid (solid with >= 1 fluid D3Q19 neighbour: the only
// solids Eq. (15) of PAPER.md L132 is ever evaluated on, reading R7) or buried solid.  Fluid
// nodes get compact ids [0, N_f) in x-fastest raster order, wall solids ids [N_f, N_f+N_w).
#pragma once
#include <cstdint>
#include <vector>

namespace lbmgeo {

// Direction table in the canonical order of include/lbm.h (reading R1).
constexpr int kQ = 19;
extern const int kE[kQ][3];
extern const int kOpp[kQ];

struct Geometry {
  int nx = 0, ny = 0, nz = 0, z_open = 0;
  long long nvox = 0, nf = 0, nw = 0;
  // Slab mode (multi-GPU z-slabs): the box carries `ghost` halo planes
  // at each z end.  Fluid nodes of the owned planes get ids [0, nact) in raster order, the halo
  // nodes ids [nact, nf): low halo planes first, then the high ones, each in raster order.
  // No halo: nact = nf and the ids are plain raster order.  An end of the box with halo planes is
  // a cut; an end without is the global box's end: an open plane there if z_open (open_lo /
  // open_hi), else periodic (then both ends have halo planes or neither has).
  int ghost_lo = 0, ghost_hi = 0;
  int open_lo = 0, open_hi = 0;
  long long nact = 0;
  std::vector<int32_t> vox2id;    // [nvox]  fluid id | nf + wall id | -1
  std::vector<int32_t> node_vox;  // [nf]    voxel index of fluid node n
  std::vector<int32_t> wall_vox;  // [nw]    voxel index of wall solid w
  // nbr[(i-1)*nf + n], i = 1..18: id of x+e_i: fluid id, nf + wall id, or -(m+1) where m is the
  // id of the mirror node when x+e_i lies beyond an open plane (reading R12 iv).
  std::vector<int32_t> nbr;
  // wall_nbr[(i-1)*nw + w]: fluid id of x_w+e_i (mirror across open planes), or -1 if not fluid.
  std::vector<int32_t> wall_nbr;
  // 1 / sum_i w_i (1 - phi(x_w+e_i)): the denominator of Eq. (15).
  std::vector<double> wall_inv_den;
};

// 16-bit tile-relative form of the neighbour index (halves the index traffic of the fused pass).
// For tile t (kIdxTile consecutive fluid ids) and direction i the entries of nbr are written as
//   bit 15 = 0: fluid id (or mirror node)  = meta[t][i-1]      + (e & 0x7fff)
//   bit 15 = 1: wall solid, psi index      = meta[t][18 + i-1] + (e & 0x7fff)   (already npad-based)
// "beyond an open plane" is not stored: the kernel derives it from the node's plane and e_z.
// meta[t][36] = 1 marks a "wide" tile (some offset range does not fit 15 bits, e.g. a periodic
// wrap inside the tile): the kernel then reads the tile's int32 rows instead.
constexpr int kIdxTile = 128;
constexpr int kIdxMeta = 40;  // ints per tile: 18 fluid bases, 18 wall bases, wide flag, wide-table position, 2 pad
struct Index16 {
  std::vector<uint16_t> nbr16;  // [18][stride]
  std::vector<int32_t> meta;    // [ntf][kIdxMeta]
  std::vector<int32_t> wide_rows;  // [wide_tiles][18][kIdxTile]: the int32 ids (psi indices, open-plane
                                   // sign included) of the wide tiles only; meta[t][37] = a wide
                                   // tile's position in this table
  size_t stride = 0;
  long long wide_tiles = 0;
};
// psi_wall_base = psi index of wall solid 0 (npad); stride = row stride of nbr16 (>= ntf*kIdxTile)
int build_index16(const Geometry& g, long long psi_wall_base, size_t stride, Index16& out);

// Returns 0, or -1 bad arguments, -2 no fluid voxel, -3 solid on an open plane or its interior
// neighbour plane (z in {0,1,nz-2,nz-1}), -4 out of memory.  `with_tables` = also fill nbr,
// wall_nbr, wall_inv_den.
int build(Geometry& g, const uint8_t* solid, int nx, int ny, int nz, int z_open, bool with_tables,
          int ghost_lo = 0, int ghost_hi = 0);

// Halo lists of a slab (ghost_lo, ghost_hi in {0, kSlabGhost}; z local: [0,ghost_lo) low halo,
// [ghost_lo, nz-ghost_hi) owned, [nz-ghost_hi, nz) high halo; a face without halo planes has
// empty lists).  After the fused pass the populations an
// owned boundary-plane node pushed across the cut sit in the rows of the inner halo plane's
// nodes; they are packed into one message per face and, on the neighbour slab, unpacked into the
// same rows of its owned boundary plane.  An entry exists for (direction i crossing the cut,
// node x of the destination plane) iff x - e_i is fluid (else halfway bounce-back filled the slot
// locally).  Order: direction-major in the order of kCross, raster order of x within; both slabs
// derive the same list from the same two mask planes.  Entries are pair-slot indices i*npad + id.
constexpr int kSlabGhost = 2;
struct Halo {
  std::vector<int32_t> pack[2];    // [face 0 = low, 1 = high]: source slots (inner halo plane rows)
  std::vector<int32_t> unpack[2];  // [face]: destination slots (owned boundary plane rows)
  long long psi_send[2][2];        // [face]{first id, count}: owned nodes of the 2 planes at that face
  long long psi_recv[2][2];        // [face]{first id, count}: halo nodes at that face
  long long edge_plane[2];         // fluid nodes of the outermost owned plane at that face (the only
                                   // nodes whose pushes cross the cut)
};
int build_halo(const Geometry& g, const uint8_t* solid, size_t npad, Halo& h);

}  // namespace lbmgeo
