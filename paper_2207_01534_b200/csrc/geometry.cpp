// geometry.cpp -- see geometry.hpp.  Host only, O(voxels), not on the timed path.
#include "geometry.hpp"

#include <algorithm>
#include <new>
#include <utility>

namespace lbmgeo {

const int kE[kQ][3] = {{0, 0, 0},  {1, 0, 0},   {-1, 0, 0}, {0, 1, 0},  {0, -1, 0},
                       {0, 0, 1},  {0, 0, -1},  {1, 1, 0},  {-1, 1, 0}, {1, -1, 0},
                       {-1, -1, 0}, {1, 0, 1},  {-1, 0, 1}, {1, 0, -1}, {-1, 0, -1},
                       {0, 1, 1},  {0, -1, 1},  {0, 1, -1}, {0, -1, -1}};
const int kOpp[kQ] = {0, 2, 1, 4, 3, 6, 5, 10, 9, 8, 7, 14, 13, 12, 11, 18, 17, 16, 15};

namespace {

struct Box {
  int nx, ny, nz, open_lo, open_hi;
  // voxel index of (x,y,z)+e_i; *beyond = the true neighbour lies past an open plane and the
  // returned voxel is its mirror image across that plane.
  inline long long nb(int x, int y, int z, int i, bool* beyond) const {
    int xn = x + kE[i][0], yn = y + kE[i][1], zn = z + kE[i][2];
    if (xn < 0) xn += nx; else if (xn >= nx) xn -= nx;
    if (yn < 0) yn += ny; else if (yn >= ny) yn -= ny;
    *beyond = false;
    if (zn < 0 || zn >= nz) {
      if (zn < 0 ? open_lo : open_hi) { *beyond = true; zn = z - kE[i][2]; }
      else zn = zn < 0 ? zn + nz : zn - nz;  // periodic; across a halo end: never read
    }
    return (long long)xn + (long long)nx * ((long long)yn + (long long)ny * (long long)zn);
  }
};

}  // namespace

int build(Geometry& g, const uint8_t* solid, int nx, int ny, int nz, int z_open,
          bool with_tables, int ghost_lo, int ghost_hi) {
  if (!solid || nx < 1 || ny < 1 || nz < 1) return -1;
  if ((ghost_lo != 0 && ghost_lo != kSlabGhost) || (ghost_hi != 0 && ghost_hi != kSlabGhost)) return -1;
  if (!z_open && ghost_lo != ghost_hi) return -1;
  if ((ghost_lo || ghost_hi) && nz < ghost_lo + ghost_hi + 2) return -1;
  const int open_lo = z_open && !ghost_lo, open_hi = z_open && !ghost_hi;
  const long long nvox = (long long)nx * ny * nz;
  if (nvox >= (1LL << 31)) return -1;
  if (z_open && nz < 4) return -1;
  const long long np = (long long)nx * ny;
  {
    const int zs[4] = {0, 1, nz - 2, nz - 1};
    for (int k = 0; k < 4; ++k)
      if (k < 2 ? open_lo : open_hi)
        for (long long q = 0; q < np; ++q)
          if (solid[(long long)zs[k] * np + q]) return -3;
  }
  g.nx = nx; g.ny = ny; g.nz = nz; g.z_open = z_open ? 1 : 0; g.nvox = nvox;
  g.ghost_lo = ghost_lo; g.ghost_hi = ghost_hi; g.open_lo = open_lo; g.open_hi = open_hi;
  const Box box{nx, ny, nz, open_lo, open_hi};
  try {
    g.vox2id.assign(nvox, -1);
    long long nf = 0;
    // owned planes first, then the low halo planes, then the high ones (ghost = 0: plain raster)
    const long long v_lo = (long long)ghost_lo * np, v_hi = nvox - (long long)ghost_hi * np;
    for (long long v = v_lo; v < v_hi; ++v)
      if (!solid[v]) g.vox2id[v] = (int32_t)nf++;
    g.nact = nf;
    if (nf == 0) return -2;
    for (long long v = 0; v < v_lo; ++v)
      if (!solid[v]) g.vox2id[v] = (int32_t)nf++;
    for (long long v = v_hi; v < nvox; ++v)
      if (!solid[v]) g.vox2id[v] = (int32_t)nf++;
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

int build_index16(const Geometry& g, long long psi_wall_base, size_t stride, Index16& out) {
  if (g.nf <= 0 || g.nbr.empty()) return -1;
  const long long nf = g.nf;
  const int ntf = (int)((nf + kIdxTile - 1) / kIdxTile);
  if (stride < (size_t)ntf * kIdxTile) return -1;
  try {
    out.stride = stride;
    out.nbr16.assign((size_t)18 * stride, 0);
    out.meta.assign((size_t)ntf * kIdxMeta, 0);
    long long wide = 0;
#pragma omp parallel for schedule(static) reduction(+ : wide)
    for (int t = 0; t < ntf; ++t) {
      const long long n0 = (long long)t * kIdxTile, n1 = std::min<long long>(nf, n0 + kIdxTile);
      int32_t* m = &out.meta[(size_t)t * kIdxMeta];
      bool is_wide = false;
      for (int i = 0; i < 18; ++i) {
        long long fmin = -1, fmax = -1, wmin = -1, wmax = -1;
        for (long long n = n0; n < n1; ++n) {
          int32_t id = g.nbr[(size_t)i * nf + n];
          if (id < 0) id = -id - 1;
          if (id < nf) { if (fmin < 0 || id < fmin) fmin = id; if (id > fmax) fmax = id; }
          else { const long long w = id - nf; if (wmin < 0 || w < wmin) wmin = w; if (w > wmax) wmax = w; }
        }
        if (fmax - fmin > 0x7fff || wmax - wmin > 0x7fff) is_wide = true;
        m[i] = (int32_t)std::max<long long>(fmin, 0);
        m[18 + i] = (int32_t)(psi_wall_base + std::max<long long>(wmin, 0));
        for (long long n = n0; n < n1; ++n) {
          int32_t id = g.nbr[(size_t)i * nf + n];
          if (id < 0) id = -id - 1;
          uint16_t e;
          if (id < nf) e = (uint16_t)((id - std::max<long long>(fmin, 0)) & 0x7fff);
          else e = (uint16_t)(0x8000 | (((id - nf) - std::max<long long>(wmin, 0)) & 0x7fff));
          out.nbr16[(size_t)i * stride + n] = e;
        }
      }
      m[36] = is_wide ? 1 : 0;
      wide += is_wide ? 1 : 0;
    }
    out.wide_tiles = wide;
    // compact int32 table of the wide tiles (everything else is served by the 16-bit rows)
    out.wide_rows.assign((size_t)wide * 18 * kIdxTile, 0);
    long long pos = 0;
    for (int t = 0; t < ntf; ++t) {
      int32_t* m = &out.meta[(size_t)t * kIdxMeta];
      if (!m[36]) continue;
      m[37] = (int32_t)pos;
      const long long n0 = (long long)t * kIdxTile, n1 = std::min<long long>(nf, n0 + kIdxTile);
      for (int i = 0; i < 18; ++i)
        for (long long n = n0; n < n1; ++n) {
          const int32_t raw = g.nbr[(size_t)i * nf + n];
          int32_t id = raw < 0 ? -raw - 1 : raw;
          if (id >= nf) id = (int32_t)(psi_wall_base + (id - nf));
          out.wide_rows[((size_t)pos * 18 + i) * kIdxTile + (n - n0)] = raw < 0 ? -id - 1 : id;
        }
      ++pos;
    }
  } catch (const std::bad_alloc&) {
    return -4;
  }
  return 0;
}

int build_halo(const Geometry& g, const uint8_t* solid, size_t npad, Halo& h) {
  if (!solid) return -1;
  const int nx = g.nx, ny = g.ny, nz = g.nz, G = kSlabGhost;
  const int gl = g.ghost_lo, gh = g.ghost_hi;
  const long long np = (long long)nx * ny;
  // directions that cross the low cut (e_z = -1) and the high cut (e_z = +1)
  static const int kCross[2][5] = {{6, 13, 14, 17, 18}, {5, 11, 12, 15, 16}};
  try {
    for (int face = 0; face < 2; ++face) {
      h.pack[face].clear();
      h.unpack[face].clear();
      if ((face == 0 ? gl : gh) == 0) continue;            // the global box's end: nothing crosses
      // pack: what my owned boundary plane pushed into the inner halo plane of this face
      const int z_halo = face == 0 ? gl - 1 : nz - gh;     // inner halo plane
      const int z_own = face == 0 ? gl : nz - gh - 1;      // owned boundary plane
      for (int k = 0; k < 5; ++k) {
        const int i = kCross[face][k];       // travels from z_own to z_halo
        const int j = kCross[1 - face][k];   // arrives at z_own from z_halo (neighbour's push)
        for (int y = 0; y < ny; ++y)
          for (int x = 0; x < nx; ++x) {
            {  // destination x in the halo plane, source x - e_i in my owned plane
              const long long vd = x + nx * (y + (long long)ny * z_halo);
              const int xs = (x - kE[i][0] + nx) % nx, ys = (y - kE[i][1] + ny) % ny;
              const long long vs = xs + nx * (ys + (long long)ny * z_own);
              if (!solid[vd] && !solid[vs])
                h.pack[face].push_back((int32_t)((size_t)i * npad + (size_t)g.vox2id[vd]));
            }
            {  // destination x in my owned plane, source x - e_j in the halo plane
              const long long vd = x + nx * (y + (long long)ny * z_own);
              const int xs = (x - kE[j][0] + nx) % nx, ys = (y - kE[j][1] + ny) % ny;
              const long long vs = xs + nx * (ys + (long long)ny * z_halo);
              if (!solid[vd] && !solid[vs])
                h.unpack[face].push_back((int32_t)((size_t)j * npad + (size_t)g.vox2id[vd]));
            }
          }
      }
    }
    // psi: fluid ids of whole planes are contiguous (raster order inside each id block)
    auto count = [&](int z0, int z1) {
      long long c = 0;
      for (long long v = z0 * np; v < z1 * np; ++v) c += solid[v] ? 0 : 1;
      return c;
    };
    const long long n_lo = count(0, gl), n_hi = count(nz - gh, nz);
    h.psi_send[0][0] = 0;
    h.psi_send[0][1] = gl ? count(gl, gl + G) : 0;
    h.psi_send[1][1] = gh ? count(nz - gh - G, nz - gh) : 0;
    h.psi_send[1][0] = g.nact - h.psi_send[1][1];
    h.psi_recv[0][0] = g.nact;
    h.psi_recv[0][1] = n_lo;
    h.psi_recv[1][0] = g.nact + n_lo;
    h.psi_recv[1][1] = n_hi;
    h.edge_plane[0] = count(gl, gl + 1);
    h.edge_plane[1] = count(nz - gh - 1, nz - gh);
  } catch (const std::bad_alloc&) {
    return -4;
  }
  return 0;
}

}  // namespace lbmgeo
