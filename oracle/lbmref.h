/* lbmref.h -- CPU ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, dense fp64 restatement of the two-component pseudopotential D3Q19 lattice
 * Boltzmann step of arXiv 2207.01534 (Eq. 1-15), written from the paper and from
 * the readings R1-R27 listed in DESIGN.md.  It shares no code, header, table or helper with
 * the CUDA path under paper_2207_01534_b200/.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.
 *
 * Parity pins (tests/test_oracle_*.py): lattice identities, stationarity, exact mass and
 * momentum conservation, lattice symmetries, G=0 shear-wave decay, discrete Poiseuille
 * closed form, flat-interface coexistence 0.027, Laplace gamma=0.071
 * (PAPER.md L181), contact-angle fit, brute-force flood fill.
 * Open planes (lbmref_step with z_open=1): the NEEM formula, the frozen rule, the Zou-He
 * variant and the psi mirror across the planes are pinned by identities,
 * fixed points and an exact force cancellation (tests/test_oracle_neem.py, _zouhe.py,
 * _diag_open.py), and so is the choice of the common velocity of Eq. (8) for NEEM's
 * equilibrium.  PARITY UNPINNED: one detail the garbled passage PAPER.md L147-157 leaves open
 * -- that velocity carries no F/2 shift where the force is not zero (reading R12 iii).
 *
 * Layout: dense arrays are indexed idx = x + nx*(y + ny*z); populations are
 * f[i*nvox + idx] per component with the direction order returned by lbmref_lattice.
 */
#ifndef LBMREF_H
#define LBMREF_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct lbmref_ctx lbmref_ctx;

typedef struct {
  double G;          /* G_coh of Eq. (11)/(13); positive = repulsion   */
  double tau[2];     /* tau^(sigma), Eq. (7) PAPER.md L81 (reading R2: nu=(tau-1/2)/3)    */
  double xi;         /* chi1 = 1+xi, chi2 = 1-xi                       */
  double accel[3];   /* g; F^b_sigma = rho_sigma g (reading R8)            */
  int z_open;        /* 0 periodic in z; 1 inlet plane z=0, outlet plane z=nz-1           */
  int inlet_kind;    /* 1 density (NEEM), 2 velocity (NEEM), 3 density (Zou-He), 4 velocity
                        (Zou-He)                                     */
  int inlet_comp;    /* component (0/1) that gets the Dirichlet condition at the inlet    */
  double inlet_rho;
  double inlet_uz;
  int outlet_kind;   /* 1 density (NEEM), 3 density (Zou-He)                              */
  int outlet_comp;
  double outlet_rho;
  int storage_bits;  /* ignored by the oracle (always fp64)                               */
  int half_force;    /* 1: u_eq carries F/2 (reading R3); 0: literal Eq. (4), neg. control */
} lbmref_params;

/* all functions return 0 on success, a negative code otherwise */
int lbmref_create(lbmref_ctx** out, const uint8_t* solid, int nx, int ny, int nz,
                  const lbmref_params* p);
void lbmref_destroy(lbmref_ctx* c);
int lbmref_set_density(lbmref_ctx* c, const double* rhoA, const double* rhoB);
int lbmref_set_populations(lbmref_ctx* c, int comp, const double* f);
int lbmref_get_populations(lbmref_ctx* c, int comp, double* f);
int lbmref_step(lbmref_ctx* c, int n);
int lbmref_get_macroscopic(lbmref_ctx* c, double* rhoA, double* rhoB, double* ux, double* uy,
                           double* uz, double* P);
int lbmref_diagnostics(lbmref_ctx* c, double mass[2], double momentum[3]);
int lbmref_saturation(lbmref_ctx* c, int comp, int z0, int z1, double* S);
int lbmref_trapped_volume(lbmref_ctx* c, int comp, int z0, int z1, long long* nodes,
                          double* mass);
long long lbmref_num_fluid(lbmref_ctx* c);
/* Change the imposed inlet value (rho for inlet_kind 1, u_z for inlet_kind 2) and the outlet
 * density between steps: the pressure ramp of the drainage protocol, PAPER.md L223 ("the inlet
 * density was gradually increased while the outlet density was kept constant").  A setter only. */
int lbmref_set_boundary(lbmref_ctx* c, double inlet_value, double outlet_rho);
/* the oracle's own lattice: w[19], e[19*3] (x,y,z), opp[19] */
void lbmref_lattice(double* w, int* e, int* opp);
int lbmref_threads(void);

#ifdef __cplusplus
}
#endif
#endif
