/* lbmref.cpp -- CPU ORACLE (test infrastructure, NOT the product). See lbmref.h.
 *
 * One time step, in the order of DESIGN.md "Oracle" (reading R9), all right-hand sides at time t:
 *   1. rho_sigma = sum_i f_i            Eq. (3)  PAPER.md L69 ; j = sum_sigma sum_i e_i f_i  (Eq. 4 numerator, L71)
 *   2. rho~_sigma on wall solids        Eq. (15), chi: L141-143
 *   3. F_sigma                          Eq. (10),(11),(13) PAPER.md L98,L103,L124 ; body force L111 (R8)
 *   4. rho, tau_s, u_eq                 Eq. (5)-(8) PAPER.md L73-87 (R2, R3, R4)
 *   5. collision                        Eq. (1),(2),(9) PAPER.md L57-63, L94
 *   6. streaming + halfway bounce-back  Eq. (1) LHS; PAPER.md L191, L215 (R10)
 *   7. open planes                      PAPER.md L147-157, L107-113 (R12)
 *      NEEM variant (kinds 1-2): pinned to the textbook identity of ref. [6], its exact
 *      consequences, the frozen rule and a moving fixed point (tests/test_oracle_neem.py);
 *      Zou-He variant (kinds 3-4, R31): pinned by its defining properties and a fixed point
 *      (tests/test_oracle_zouhe.py).  The mirrored psi neighbours beyond a plane (R12 iv, the
 *      one statement PAPER.md L113 prints: psi(x+e_14) = psi(x+e_13)) are pinned by the exact
 *      cancellation of the plane-normal force they imply (tests/test_oracle_diag_open.py); that
 *      NEEM's equilibrium is taken at the COMMON velocity of Eq. (8), not a component's own, by
 *      reading the model's equilibrium off the collision step itself (tests/test_oracle_neem.py).
 *      What stays a READING -- parity unpinned -- is one detail of R12 iii: that velocity is the
 *      bare mixture velocity, without the F/2 shift of R3, also where the force at the interior
 *      neighbour is not zero; the paper prints nothing that fixes it.
 * No blocking, fusion or reordering: five plain loop nests over the dense box.
 */
#include "lbmref.h"

#include <cmath>
#include <cstring>
#include <limits>
#include <new>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

/* D3Q19 (reading R1: the velocity table is missing from PAPER.md L65-67; standard set, numbering
 * consistent with what L113 and L152-154 reveal).  w_i from PAPER.md L67. */
const int E[19][3] = {
    {0, 0, 0},  {1, 0, 0},  {-1, 0, 0}, {0, 1, 0},   {0, -1, 0}, {0, 0, 1},  {0, 0, -1},
    {1, 1, 0},  {-1, 1, 0}, {1, -1, 0}, {-1, -1, 0}, {1, 0, 1},  {-1, 0, 1}, {1, 0, -1},
    {-1, 0, -1}, {0, 1, 1}, {0, -1, 1}, {0, 1, -1},  {0, -1, -1}};
const double W[19] = {1.0 / 3.0,  1.0 / 18.0, 1.0 / 18.0, 1.0 / 18.0, 1.0 / 18.0,
                      1.0 / 18.0, 1.0 / 18.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0,
                      1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0,
                      1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0};
const int OPP[19] = {0, 2, 1, 4, 3, 6, 5, 10, 9, 8, 7, 14, 13, 12, 11, 18, 17, 16, 15};
/* directions pointing into the domain at the inlet (e_z=+1) and at the outlet (e_z=-1) */
const int INWARD[2][5] = {{5, 11, 12, 15, 16}, {6, 13, 14, 17, 18}};

}  // namespace

struct lbmref_ctx {
  int nx, ny, nz;
  long nvox, nfluid;
  lbmref_params p;
  std::vector<uint8_t> solid;     /* phi of Eq. (14): 1 solid, 0 fluid                     */
  std::vector<uint8_t> wall;      /* solid voxel with at least one fluid D3Q19 neighbour   */
  std::vector<double> f[2];       /* populations at time t  [i*nvox + idx]                 */
  std::vector<double> g[2];       /* streaming target                                      */
  std::vector<double> Psi[2];     /* rho_sigma on fluid, rho~_sigma on wall solids (Eq.14) */
  std::vector<double> frozen[2][2]; /* [plane][comp][k*nx*ny + x + nx*y], k over INWARD     */
};

namespace {

inline long vidx(const lbmref_ctx* c, int x, int y, int z) {
  return (long)x + (long)c->nx * ((long)y + (long)c->ny * (long)z);
}
inline int wrap(int a, int n) { return a < 0 ? a + n : (a >= n ? a - n : a); }

/* Index of the voxel x+e_i. Periodic wrap in x, y (and z unless z_open). Across an open plane
 * the neighbour is replaced by its mirror image (R12 iv) and *beyond is set. */
inline long neighbour(const lbmref_ctx* c, int x, int y, int z, int i, bool* beyond) {
  int xn = wrap(x + E[i][0], c->nx);
  int yn = wrap(y + E[i][1], c->ny);
  int zn = z + E[i][2];
  *beyond = false;
  if (zn < 0 || zn >= c->nz) {
    if (c->p.z_open) {
      *beyond = true;
      zn = z - E[i][2];
    } else {
      zn = wrap(zn, c->nz);
    }
  }
  return vidx(c, xn, yn, zn);
}

inline double feq(int i, double rho, const double u[3]) {
  /* Eq. (2) PAPER.md L63 with c_s^2 = 1/3 (L65, R18) */
  double eu = E[i][0] * u[0] + E[i][1] * u[1] + E[i][2] * u[2];
  double uu = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
  return W[i] * rho * (1.0 + 3.0 * eu + 4.5 * eu * eu - 1.5 * uu);
}

/* steps 1 and 2: Psi on fluid and wall-solid voxels */
void compute_Psi(lbmref_ctx* c) {
  const long nv = c->nvox;
#pragma omp parallel for schedule(static)
  for (long v = 0; v < nv; ++v) {
    for (int s = 0; s < 2; ++s) {
      double r = 0.0;
      if (!c->solid[v])
        for (int i = 0; i < 19; ++i) r += c->f[s][i * nv + v];
      c->Psi[s][v] = r;
    }
  }
  const double chi[2] = {1.0 + c->p.xi, 1.0 - c->p.xi};
#pragma omp parallel for collapse(2) schedule(static)
  for (int z = 0; z < c->nz; ++z)
    for (int y = 0; y < c->ny; ++y)
      for (int x = 0; x < c->nx; ++x) {
        long v = vidx(c, x, y, z);
        if (!c->wall[v]) continue;
        double num[2] = {0.0, 0.0}, den = 0.0;
        for (int i = 1; i < 19; ++i) {
          bool beyond;
          long n = neighbour(c, x, y, z, i, &beyond);
          if (c->solid[n]) continue; /* factor (1 - phi) of Eq. (15) */
          num[0] += W[i] * c->Psi[0][n];
          num[1] += W[i] * c->Psi[1][n];
          den += W[i];
        }
        c->Psi[0][v] = chi[0] * num[0] / den; /* Eq. (15) */
        c->Psi[1][v] = chi[1] * num[1] / den;
      }
}

/* step 3 at one fluid node: F_sigma = -G rho_sigma sum_i w_i Psi_sigmabar(x+e_i) e_i + rho_sigma g */
inline void node_force(const lbmref_ctx* c, int x, int y, int z, double F[2][3]) {
  long v = vidx(c, x, y, z);
  double S[2][3] = {{0, 0, 0}, {0, 0, 0}};
  for (int i = 1; i < 19; ++i) {
    bool beyond;
    long n = neighbour(c, x, y, z, i, &beyond);
    for (int s = 0; s < 2; ++s)
      for (int a = 0; a < 3; ++a) S[s][a] += W[i] * c->Psi[s][n] * E[i][a];
  }
  for (int s = 0; s < 2; ++s)
    for (int a = 0; a < 3; ++a)
      F[s][a] = -c->p.G * c->Psi[s][v] * S[1 - s][a] + c->Psi[s][v] * c->p.accel[a];
}

/* steps 1 (momentum part) and 4 at one fluid node */
inline void node_velocity(const lbmref_ctx* c, long v, const double F[2][3], double u[3],
                          double* rho_tot) {
  const long nv = c->nvox;
  double j[3] = {0, 0, 0};
  for (int s = 0; s < 2; ++s)
    for (int i = 0; i < 19; ++i)
      for (int a = 0; a < 3; ++a) j[a] += E[i][a] * c->f[s][i * nv + v];
  double rho = c->Psi[0][v] + c->Psi[1][v]; /* Eq. (5) */
  double hf = c->p.half_force ? 0.5 : 0.0;
  for (int a = 0; a < 3; ++a) u[a] = (j[a] + hf * (F[0][a] + F[1][a])) / rho; /* Eq. (8), R3, R4 */
  *rho_tot = rho;
}

void record_frozen(lbmref_ctx* c, int comp) {
  if (!c->p.z_open) return;
  const long nv = c->nvox, np = (long)c->nx * c->ny;
  for (int plane = 0; plane < 2; ++plane) {
    int z = plane == 0 ? 0 : c->nz - 1;
    c->frozen[plane][comp].assign(5 * np, 0.0);
    for (int k = 0; k < 5; ++k)
      for (long q = 0; q < np; ++q)
        c->frozen[plane][comp][k * np + q] = c->f[comp][INWARD[plane][k] * nv + (long)z * np + q];
  }
}

}  // namespace

extern "C" {

void lbmref_lattice(double* w, int* e, int* opp) {
  for (int i = 0; i < 19; ++i) {
    w[i] = W[i];
    opp[i] = OPP[i];
    for (int a = 0; a < 3; ++a) e[3 * i + a] = E[i][a];
  }
}

int lbmref_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

int lbmref_create(lbmref_ctx** out, const uint8_t* solid, int nx, int ny, int nz,
                  const lbmref_params* p) {
  if (!out || !solid || !p || nx < 1 || ny < 1 || nz < 1) return -1;
  if (!(p->tau[0] > 0.5) || !(p->tau[1] > 0.5)) return -1;
  if (p->z_open) {
    if (nz < 4) return -1;
    if (p->inlet_kind < 1 || p->inlet_kind > 4) return -1;
    if (p->outlet_kind != 1 && p->outlet_kind != 3) return -1;
    if (p->inlet_comp < 0 || p->inlet_comp > 1 || p->outlet_comp < 0 || p->outlet_comp > 1)
      return -1;
  }
  lbmref_ctx* c = new (std::nothrow) lbmref_ctx;
  if (!c) return -4;
  c->nx = nx; c->ny = ny; c->nz = nz;
  c->nvox = (long)nx * ny * nz;
  c->p = *p;
  try {
    c->solid.assign(solid, solid + c->nvox);
    for (long v = 0; v < c->nvox; ++v) c->solid[v] = c->solid[v] ? 1 : 0;
    c->wall.assign(c->nvox, 0);
    for (int s = 0; s < 2; ++s) {
      c->f[s].assign(19 * c->nvox, 0.0);
      c->g[s].assign(19 * c->nvox, 0.0);
      c->Psi[s].assign(c->nvox, 0.0);
    }
  } catch (...) {
    delete c;
    return -4;
  }
  c->nfluid = 0;
  for (long v = 0; v < c->nvox; ++v) c->nfluid += !c->solid[v];
  if (c->nfluid == 0) { delete c; return -2; }
  if (p->z_open) {
    /* both open planes and their interior neighbours are pure reservoir (R12) */
    const int zs[4] = {0, 1, nz - 2, nz - 1};
    for (int k = 0; k < 4; ++k)
      for (long q = 0; q < (long)nx * ny; ++q)
        if (c->solid[(long)zs[k] * nx * ny + q]) { delete c; return -3; }
  }
  for (int z = 0; z < nz; ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        long v = vidx(c, x, y, z);
        if (!c->solid[v]) continue;
        for (int i = 1; i < 19; ++i) {
          bool beyond;
          long n = neighbour(c, x, y, z, i, &beyond);
          if (!c->solid[n]) { c->wall[v] = 1; break; }
        }
      }
  *out = c;
  return 0;
}

void lbmref_destroy(lbmref_ctx* c) { delete c; }

long long lbmref_num_fluid(lbmref_ctx* c) { return c ? c->nfluid : -1; }

int lbmref_set_boundary(lbmref_ctx* c, double inlet_value, double outlet_rho) {
  if (!c || !c->p.z_open || !std::isfinite(inlet_value) || !std::isfinite(outlet_rho)) return -1;
  if (c->p.inlet_kind == 1 || c->p.inlet_kind == 3) c->p.inlet_rho = inlet_value;
  else c->p.inlet_uz = inlet_value;
  c->p.outlet_rho = outlet_rho;
  return 0;
}

int lbmref_set_density(lbmref_ctx* c, const double* rhoA, const double* rhoB) {
  if (!c || !rhoA || !rhoB) return -1;
  const double* r[2] = {rhoA, rhoB};
  const long nv = c->nvox;
  for (int s = 0; s < 2; ++s) {
    for (int i = 0; i < 19; ++i)
      for (long v = 0; v < nv; ++v)
        c->f[s][i * nv + v] = c->solid[v] ? 0.0 : W[i] * r[s][v]; /* R11 */
    record_frozen(c, s);
  }
  return 0;
}

int lbmref_set_populations(lbmref_ctx* c, int comp, const double* f) {
  if (!c || !f || comp < 0 || comp > 1) return -1;
  const long nv = c->nvox;
  for (int i = 0; i < 19; ++i)
    for (long v = 0; v < nv; ++v) c->f[comp][i * nv + v] = c->solid[v] ? 0.0 : f[i * nv + v];
  record_frozen(c, comp); /* R27 */
  return 0;
}

int lbmref_get_populations(lbmref_ctx* c, int comp, double* f) {
  if (!c || !f || comp < 0 || comp > 1) return -1;
  std::memcpy(f, c->f[comp].data(), sizeof(double) * 19 * c->nvox);
  return 0;
}

/* Zou-He condition ("Apply Zou-He (ZH) method [34] or ... NEEM"; ref. [34] is the
 * D3Q19 form of Hecht & Harting) on the Dirichlet component's own populations at one node of an
 * open plane, after streaming (reading R31).  sgn = +1 at the inlet (the 5 unknowns have
 * e_z = +1), -1 at the outlet.  With K0 = sum of the populations with e_z = 0 and Km = sum of
 * the known ones leaving the domain (e_z = -sgn), mass and z-momentum give
 *     rho (1 - sgn u_z) = K0 + 2 Km ,
 * which fixes u_z from the imposed rho (kind 3) or rho from the imposed u_z (kind 4); u_x = u_y
 * = 0 are imposed.  The unknowns are the bounce-back of the non-equilibrium part,
 *     f_i = f_opp(i) + 6 w_i rho (e_i . u)  -/+  the transverse corrections N_x, N_y
 * chosen so that the x- and y-momentum of the node vanish:
 *     N_a = 1/2 * sum over the in-plane populations of e_ia f_i      (a = x, y). */
static void zou_he_plane_node(lbmref_ctx* c, int s, long v, int plane, int kind, double rho_given) {
  const long nv = c->nvox;
  const int sgn = plane == 0 ? 1 : -1;
  double K0 = 0.0, Km = 0.0, Nx = 0.0, Ny = 0.0;
  for (int i = 0; i < 19; ++i) {
    const double fi = c->g[s][i * nv + v];
    if (E[i][2] == 0) {
      K0 += fi;
      Nx += 0.5 * E[i][0] * fi;
      Ny += 0.5 * E[i][1] * fi;
    } else if (E[i][2] == -sgn) {
      Km += fi;
    }
  }
  double rho, uz;
  if (kind == 3) {
    rho = rho_given;
    uz = sgn * (1.0 - (K0 + 2.0 * Km) / rho);
  } else {
    uz = c->p.inlet_uz;
    rho = (K0 + 2.0 * Km) / (1.0 - sgn * uz);
  }
  for (int i = 0; i < 19; ++i) {
    if (E[i][2] != sgn) continue;
    c->g[s][i * nv + v] = c->g[s][OPP[i] * nv + v] + 6.0 * W[i] * rho * (E[i][2] * uz) -
                          E[i][0] * Nx - E[i][1] * Ny;
  }
}

int lbmref_step(lbmref_ctx* c, int nsteps) {
  if (!c || nsteps < 0) return -1;
  const long nv = c->nvox;
  const long np = (long)c->nx * c->ny;
  const double qnan = std::numeric_limits<double>::quiet_NaN();
  for (int it = 0; it < nsteps; ++it) {
    /* steps 1-2 */
    compute_Psi(c);
    /* steps 3-5: collide in place, f <- f* (the collision is local) */
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < c->nz; ++z)
      for (int y = 0; y < c->ny; ++y)
        for (int x = 0; x < c->nx; ++x) {
          long v = vidx(c, x, y, z);
          if (c->solid[v]) continue;
          double F[2][3], u[3], rho;
          node_force(c, x, y, z, F);
          node_velocity(c, v, F, u, &rho);
          double tau_s = (c->Psi[0][v] * c->p.tau[0] + c->Psi[1][v] * c->p.tau[1]) / rho; /* Eq. 6-7, R2 */
          for (int s = 0; s < 2; ++s)
            for (int i = 0; i < 19; ++i) {
              double eu = E[i][0] * u[0] + E[i][1] * u[1] + E[i][2] * u[2];
              double eF = E[i][0] * F[s][0] + E[i][1] * F[s][1] + E[i][2] * F[s][2];
              double emuF = (E[i][0] - u[0]) * F[s][0] + (E[i][1] - u[1]) * F[s][1] +
                            (E[i][2] - u[2]) * F[s][2];
              double S = W[i] * (3.0 * emuF + 9.0 * eu * eF); /* Eq. (9) */
              double fi = c->f[s][i * nv + v];
              c->f[s][i * nv + v] = fi - (fi - feq(i, c->Psi[s][v], u)) / tau_s +
                                    (1.0 - 1.0 / (2.0 * tau_s)) * S; /* Eq. (1) */
            }
        }
    /* step 6: f_i(x, t+1) = f*_i(x - e_i); bounce back where x - e_i is solid */
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < c->nz; ++z)
      for (int y = 0; y < c->ny; ++y)
        for (int x = 0; x < c->nx; ++x) {
          long v = vidx(c, x, y, z);
          for (int s = 0; s < 2; ++s)
            for (int i = 0; i < 19; ++i) {
              double val = 0.0;
              if (!c->solid[v]) {
                bool beyond;
                long src = neighbour(c, x, y, z, OPP[i], &beyond); /* x - e_i */
                if (beyond) val = qnan;                  /* filled by step 7 */
                else if (c->solid[src]) val = c->f[s][OPP[i] * nv + v];
                else val = c->f[s][i * nv + src];
              }
              c->g[s][i * nv + v] = val;
            }
        }
    /* step 7: open planes (R12) on the new buffer */
    if (c->p.z_open) {
      for (int plane = 0; plane < 2; ++plane) {
        const int zb = plane == 0 ? 0 : c->nz - 1;
        const int zf = plane == 0 ? 1 : c->nz - 2;
        const int dc = plane == 0 ? c->p.inlet_comp : c->p.outlet_comp; /* Dirichlet component */
        const int kind = plane == 0 ? c->p.inlet_kind : c->p.outlet_kind;
        const double rho_given = plane == 0 ? c->p.inlet_rho : c->p.outlet_rho;
        for (long q = 0; q < np; ++q) {
          long vb = (long)zb * np + q, vf = (long)zf * np + q;
          double rf[2] = {0, 0}, j[3] = {0, 0, 0};
          for (int s = 0; s < 2; ++s)
            for (int i = 0; i < 19; ++i) {
              double fi = c->g[s][i * nv + vf];
              rf[s] += fi;
              for (int a = 0; a < 3; ++a) j[a] += E[i][a] * fi;
            }
          double uf[3], ub[3], rho_b;
          for (int a = 0; a < 3; ++a) uf[a] = j[a] / (rf[0] + rf[1]); /* R12 iii */
          if (kind == 1) {
            rho_b = rho_given;
            for (int a = 0; a < 3; ++a) ub[a] = uf[a];
          } else {
            rho_b = rf[dc];
            ub[0] = 0.0; ub[1] = 0.0; ub[2] = c->p.inlet_uz;
          }
          if (kind <= 2) {
            for (int i = 0; i < 19; ++i) /* NEEM */
              c->g[dc][i * nv + vb] =
                  feq(i, rho_b, ub) + (c->g[dc][i * nv + vf] - feq(i, rf[dc], uf));
          } else {
            zou_he_plane_node(c, dc, vb, plane, kind, rho_given);
          }
          const int oc = 1 - dc; /* inward populations keep their initial values */
          for (int k = 0; k < 5; ++k)
            c->g[oc][INWARD[plane][k] * nv + vb] = c->frozen[plane][oc][k * np + q];
        }
      }
    }
    for (int s = 0; s < 2; ++s) c->f[s].swap(c->g[s]);
  }
  return 0;
}

int lbmref_get_macroscopic(lbmref_ctx* c, double* rhoA, double* rhoB, double* ux, double* uy,
                           double* uz, double* P) {
  if (!c) return -1;
  compute_Psi(c);
  for (int z = 0; z < c->nz; ++z)
    for (int y = 0; y < c->ny; ++y)
      for (int x = 0; x < c->nx; ++x) {
        long v = vidx(c, x, y, z);
        double r0 = 0, r1 = 0, u[3] = {0, 0, 0}, pr = 0;
        if (!c->solid[v]) {
          double F[2][3], rho;
          node_force(c, x, y, z, F);
          node_velocity(c, v, F, u, &rho);
          r0 = c->Psi[0][v];
          r1 = c->Psi[1][v];
          pr = (r0 + r1) / 3.0 + (c->p.G / 3.0) * r0 * r1; /* Eq. (12), R13 */
        }
        if (rhoA) rhoA[v] = r0;
        if (rhoB) rhoB[v] = r1;
        if (ux) ux[v] = u[0];
        if (uy) uy[v] = u[1];
        if (uz) uz[v] = u[2];
        if (P) P[v] = pr;
      }
  return 0;
}

int lbmref_diagnostics(lbmref_ctx* c, double mass[2], double momentum[3]) {
  if (!c || !mass || !momentum) return -1;
  const long nv = c->nvox;
  long double m[2] = {0, 0}, mo[3] = {0, 0, 0}; /* extended accumulators: the sums are pins */
  for (int s = 0; s < 2; ++s)
    for (int i = 0; i < 19; ++i)
      for (long v = 0; v < nv; ++v) {
        if (c->solid[v]) continue;
        double fi = c->f[s][i * nv + v];
        m[s] += fi;
        for (int a = 0; a < 3; ++a) mo[a] += E[i][a] * fi;
      }
  mass[0] = (double)m[0]; mass[1] = (double)m[1];
  for (int a = 0; a < 3; ++a) momentum[a] = (double)mo[a];
  return 0;
}

/* R14: a fluid node belongs to component c iff rho_c > rho_other (tie -> component 1) */
static inline int owner(const lbmref_ctx* c, long v) { return c->Psi[0][v] > c->Psi[1][v] ? 0 : 1; }

int lbmref_saturation(lbmref_ctx* c, int comp, int z0, int z1, double* S) {
  if (!c || !S || comp < 0 || comp > 1 || z0 < 0 || z1 > c->nz || z0 >= z1) return -1;
  compute_Psi(c);
  const long np = (long)c->nx * c->ny;
  long cnt = 0, tot = 0;
  for (long v = z0 * np; v < z1 * np; ++v) {
    if (c->solid[v]) continue;
    ++tot;
    cnt += owner(c, v) == comp;
  }
  if (tot == 0) return -2;
  *S = (double)cnt / (double)tot;
  return 0;
}

/* R15: nodes of phase `comp` in [z0,z1) whose 6-connected same-phase cluster (periodic in x,y,
 * never across z) reaches neither plane z=0 nor plane z=nz-1. */
int lbmref_trapped_volume(lbmref_ctx* c, int comp, int z0, int z1, long long* nodes, double* mass) {
  if (!c || !nodes || !mass || comp < 0 || comp > 1 || z0 < 0 || z1 > c->nz || z0 >= z1) return -1;
  compute_Psi(c);
  const long nv = c->nvox, np = (long)c->nx * c->ny;
  std::vector<uint8_t> state(nv, 0); /* 1 = phase node, 2 = reached from an end plane */
  for (long v = 0; v < nv; ++v) state[v] = (!c->solid[v] && owner(c, v) == comp) ? 1 : 0;
  std::vector<long> stack;
  for (int plane = 0; plane < 2; ++plane) {
    long base = plane == 0 ? 0 : (long)(c->nz - 1) * np;
    for (long q = 0; q < np; ++q)
      if (state[base + q] == 1) { state[base + q] = 2; stack.push_back(base + q); }
  }
  const int d6[6][3] = {{1, 0, 0}, {-1, 0, 0}, {0, 1, 0}, {0, -1, 0}, {0, 0, 1}, {0, 0, -1}};
  while (!stack.empty()) {
    long v = stack.back();
    stack.pop_back();
    int x = (int)(v % c->nx), y = (int)((v / c->nx) % c->ny), z = (int)(v / np);
    for (int k = 0; k < 6; ++k) {
      int zn = z + d6[k][2];
      if (zn < 0 || zn >= c->nz) continue;
      long n = vidx(c, wrap(x + d6[k][0], c->nx), wrap(y + d6[k][1], c->ny), zn);
      if (state[n] == 1) { state[n] = 2; stack.push_back(n); }
    }
  }
  long long cnt = 0;
  double m = 0.0;
  for (long v = z0 * np; v < z1 * np; ++v)
    if (state[v] == 1) { ++cnt; m += c->Psi[comp][v]; }
  *nodes = cnt;
  *mass = m;
  return 0;
}

}  /* extern "C" */
