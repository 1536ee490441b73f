// geometry.cpp -- see geometry.hpp.  Host only, O(voxels), not on the timed path.
#include "geometry.hpp"

#include <new>

namespace lbmgeo {

const int kE[kQ][3] = {{0, 0, 0},  {1, 0, 0},   {-1, 0, 0}, {0, 1, 0},  {0, -1, 0},
                       {0, 0, 1},  {0, 0, -1},  {1, 1, 0},  {-1, 1, 0}, {1, -1, 0},
                       {-1, -1, 0}, {1, 0, 1},  {-1, 0, 1}, {1, 0, -1}, {-1, 0, -1},
                       {0, 1, 1},  {0, -1, 1},  {0, 1, -1}, {0, -1, -1}};
const int kOpp[kQ] = {0, 2, 1, 4, 3, 6, 5, 10, 9, 8, 7, 14, 13, 12, 11, 18, 17, 16, 15};

namespace {

struct Box {
  int nx, ny, nz, z_open;
  // voxel index of (x,y,z)+e_i; *beyond = the true neighbour lies past an open plane and the
  // returned voxel is its mirror image across that plane.
  inline long long nb(int x, int y, int z, int i, bool* beyond) const {
    int xn = x + kE[i][0], yn = y + kE[i][1], zn = z + kE[i][2];
    if (xn < 0) xn += nx; else if (xn >= nx) xn -= nx;
    if (yn < 0) yn += ny; else if (yn >= ny) yn -= ny;
    *beyond = false;
    if (zn < 0 || zn >= nz) {
      if (z_open) { *beyond = true; zn = z - kE[i][2]; }
      else zn = zn < 0 ? zn + nz : zn - nz;
    }
    return (long long)xn + (long long)nx * ((long long)yn + (long long)ny * (long long)zn);
  }
};

}  // namespace

int build(Geometry& g, const uint8_t* solid, int nx, int ny, int nz, int z_open,
          bool with_tables) {
  if (!solid || nx < 1 || ny < 1 || nz < 1) return -1;
  const long long nvox = (long long)nx * ny * nz;
  if (nvox >= (1LL << 31)) return -1;
  if (z_open && nz < 4) return -1;
  const long long np = (long long)nx * ny;
  if (z_open) {
    const int zs[4] = {0, 1, nz - 2, nz - 1};
    for (int k = 0; k < 4; ++k)
      for (long long q = 0; q < np; ++q)
        if (solid[(long long)zs[k] * np + q]) return -3;
  }
  g.nx = nx; g.ny = ny; g.nz = nz; g.z_open = z_open ? 1 : 0; g.nvox = nvox;
  const Box box{nx, ny, nz, g.z_open};
  try {
    g.vox2id.assign(nvox, -1);
    long long nf = 0;
    for (long long v = 0; v < nvox; ++v)
      if (!solid[v]) g.vox2id[v] = (int32_t)nf++;
    if (nf == 0) return -2;
    g.nf = nf;
    g.node_vox.resize(nf);
    for (long long v = 0; v < nvox; ++v)
      if (!solid[v]) g.node_vox[g.vox2id[v]] = (int32_t)v;
    // wall solids, raster order
    long long nw = 0;
    g.wall_vox.clear();
    for (int z = 0; z < nz; ++z)
      for (int y = 0; y < ny; ++y)
        for (int x = 0; x < nx; ++x) {
          const long long v = (long long)x + nx * ((long long)y + (long long)ny * z);
          if (!solid[v]) continue;
          for (int i = 1; i < kQ; ++i) {
            bool beyond;
            if (!solid[box.nb(x, y, z, i, &beyond)]) {
              g.vox2id[v] = (int32_t)(nf + nw);
              g.wall_vox.push_back((int32_t)v);
              ++nw;
              break;
            }
          }
        }
    g.nw = nw;
    if (nf + nw >= (1LL << 31) - 64) return -1;
    if (!with_tables) return 0;
    static const double W[kQ] = {1.0 / 3,  1.0 / 18, 1.0 / 18, 1.0 / 18, 1.0 / 18, 1.0 / 18,
                                 1.0 / 18, 1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36,
                                 1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36,
                                 1.0 / 36};
    g.nbr.resize((size_t)18 * nf);
#pragma omp parallel for schedule(static)
    for (long long n = 0; n < nf; ++n) {
      const long long v = g.node_vox[n];
      const int x = (int)(v % nx), y = (int)((v / nx) % ny), z = (int)(v / np);
      for (int i = 1; i < kQ; ++i) {
        bool beyond;
        const int32_t id = g.vox2id[box.nb(x, y, z, i, &beyond)];
        g.nbr[(size_t)(i - 1) * nf + n] = beyond ? -(id + 1) : id;
      }
    }
    g.wall_nbr.resize((size_t)18 * nw);
    g.wall_inv_den.resize(nw);
#pragma omp parallel for schedule(static)
    for (long long w = 0; w < nw; ++w) {
      const long long v = g.wall_vox[w];
      const int x = (int)(v % nx), y = (int)((v / nx) % ny), z = (int)(v / np);
      double den = 0.0;
      for (int i = 1; i < kQ; ++i) {
        bool beyond;
        const int32_t id = g.vox2id[box.nb(x, y, z, i, &beyond)];
        const bool fluid = id >= 0 && id < nf;
        g.wall_nbr[(size_t)(i - 1) * nw + w] = fluid ? id : -1;
        if (fluid) den += W[i];
      }
      g.wall_inv_den[w] = 1.0 / den;
    }
  } catch (const std::bad_alloc&) {
    return -4;
  }
  return 0;
}

}  // namespace lbmgeo
