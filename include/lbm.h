/* lbm.h -- C ABI of the B200-native two-component pseudopotential D3Q19 lattice Boltzmann step
 * of arXiv 2207.01534 (Eq. 1-15, boundary treatment PAPER.md L107-113 / L147-157).
 *
 * One lbm_ctx is one simulation on one GPU (the current CUDA device at lbm_create time).
 * Every step of the hot path runs in hand-written sm_100a kernels;
 * PyTorch is used only for device memory (its CUDA caching allocator) and for the stream
 * (torch's current CUDA stream).  There is NO CPU fallback: without a CUDA device lbm_create
 * fails with LBM_ECUDA.
 *
 * Conventions
 *  - All pointers are HOST pointers unless a parameter says "device".  The caller owns every
 *    host buffer; the library copies during the call and never retains a caller pointer.  The
 *    library owns all device memory and releases it in lbm_destroy.
 *  - Dense arrays are indexed idx = x + nx*(y + ny*z) (x fastest).  Values at solid voxels are
 *    written as 0 on output and ignored on input.
 *  - Populations use the canonical D3Q19 order (reading R1 of PAPER.md
 *    L65-67, whose velocity table is missing):
 *      0:(0,0,0) 1:(+,0,0) 2:(-,0,0) 3:(0,+,0) 4:(0,-,0) 5:(0,0,+) 6:(0,0,-) 7:(+,+,0) 8:(-,+,0)
 *      9:(+,-,0) 10:(-,-,0) 11:(+,0,+) 12:(-,0,+) 13:(+,0,-) 14:(-,0,-) 15:(0,+,+) 16:(0,-,+)
 *      17:(0,+,-) 18:(0,-,-);  w = 1/3, 1/18 (1-6), 1/36 (7-18)
 *  - Every function returns LBM_OK (0) or a negative LBM_E* code; no C++ exception crosses the
 *    ABI; lbm_last_error() returns a thread-local message for the last failure.
 *  - x and y are always periodic; z is periodic (z_open=0) or carries an inlet plane z=0 and an
 *    outlet plane z=nz-1 (z_open=1).  Walls are solid voxels of the mask.
 *  - lbm_step is asynchronous (enqueued on torch's current CUDA stream); every getter and
 *    diagnostic synchronises that stream before returning.
 */
#ifndef LBM_B200_H
#define LBM_B200_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum {
  LBM_OK = 0,
  LBM_EINVAL = -1,   /* NULL pointer, bad size, tau <= 1/2, bad enum value, bad z-range           */
  LBM_ENOFLUID = -2, /* the mask has no fluid voxel (or the z-range of a query has none)          */
  LBM_ESOLIDOPEN = -3, /* z_open=1 and a solid voxel lies on z in {0,1,nz-2,nz-1} (reading R12)   */
  LBM_ENOMEM = -4,   /* host or device allocation failed                                          */
  LBM_ECUDA = -5,    /* CUDA runtime error, or no CUDA device                                     */
  LBM_ENONFINITE = -6 /* a diagnostic found a non-finite state                                    */
};

typedef struct lbm_ctx lbm_ctx; /* opaque */

/* Parameters (plain data, copied by lbm_create). */
typedef struct {
  double G;          /* G_coh of Eq. (11)/(13); positive = inter-component
                        repulsion; the same value couples fluid-fluid and fluid-solid (L124)     */
  double tau[2];     /* tau^(sigma) of Eq. (7), each > 1/2 (reading R2)            */
  double xi;         /* wettability: chi_1 = 1+xi, chi_2 = 1-xi               */
  double accel[3];   /* g; body force F^b_sigma = rho_sigma g (reading R8)        */
  int z_open;        /* 0: periodic in z.  1: inlet plane z=0, outlet plane z=nz-1               */
  int inlet_kind;    /* 1: density (NEEM), 2: velocity (NEEM), 3: density (Zou-He), 4: velocity
                        (Zou-He); PAPER.md L149 ("Zou-He (ZH) method [34] or ... NEEM"), L223   */
  int inlet_comp;    /* component (0 or 1) that receives the Dirichlet condition at the inlet;
                        the other keeps its inward populations frozen        */
  double inlet_rho;  /* density imposed when inlet_kind is 1 or 3                                */
  double inlet_uz;   /* velocity imposed when inlet_kind is 2 or 4                               */
  int outlet_kind;   /* 1: density (NEEM), 3: density (Zou-He)                                   */
  int outlet_comp;
  double outlet_rho;
  int storage_bits;  /* 64: fp64 storage and arithmetic (validation build);
                        32: fp32 storage and arithmetic (production build)                       */
  int half_force;    /* 1: u_eq carries F/2 (reading R3); 0: literal Eq. (4) (negative control)  */
} lbm_params;

/* Execution options (plain data, copied by lbm_create_opt; every combination computes the same
 * numbers bit for bit -- tests/test_gpu_parity.py -- they select how the step is scheduled).
 * lbm_options_default fills in the defaults; lbm_create uses them. */
typedef struct {
  int graph;        /* -1 (default) replay a captured CUDA graph of 16 steps on boxes of
                       <= 600 000 fluid nodes, 0 never, 1 always                                    */
  int pdl;          /* 1 (default) programmatic dependent launch of the three passes    */
  int reverse;      /* 1 (default) the fused pass walks the tiles backwards (L2 reuse
                       across the two passes)                                                       */
  int keep_psi_mb;  /* L2 budget in MB for psi stored with evict_last priority
                       (default 48; 0: plain stores)                                                */
} lbm_options;
void lbm_options_default(lbm_options* o);

/* Build a simulation from a geometry mask (binary rock image).
 *  solid: nx*ny*nz bytes, nonzero = solid.  Classifies voxels, compacts the fluid nodes,
 *  builds the neighbour index, allocates and uploads.  Populations start at zero: call
 *  lbm_set_density or lbm_set_populations next.  *out is written only on success. */
int lbm_create(lbm_ctx** out, const uint8_t* solid, int nx, int ny, int nz, const lbm_params* p);
/* The same with explicit execution options (opt == NULL: the defaults).  LBM_EINVAL on a value
 * outside the documented ones. */
int lbm_create_opt(lbm_ctx** out, const uint8_t* solid, int nx, int ny, int nz,
                   const lbm_params* p, const lbm_options* opt);
/* Synchronises the device (kernels of the context may be in flight on any stream it was used
 * from), then releases everything.  NULL is allowed. */
void lbm_destroy(lbm_ctx* c);
/* What lbm_create chose: info[1] 1 if lbm_step replays CUDA graphs, [2] pdl, [3] reverse,
 * [4] share of the psi lines stored with evict_last priority, in 1/1000, [5] tiles that read
 * int32 ids from the compact wide-tile table instead of the 16-bit rows; [0], [6], [7] reserved
 * (0). */
int lbm_step_info(lbm_ctx* c, int info[8]);

/* f_i^sigma = w_i * rho_sigma (reading R11); dense double arrays of nx*ny*nz.  Also records the
 * frozen inlet/outlet populations (reading R27). */
int lbm_set_density(lbm_ctx* c, const double* rhoA, const double* rhoB);
/* Checkpoint interface: dense [19][nz][ny][nx] doubles of one component, canonical order. */
int lbm_set_populations(lbm_ctx* c, int comp, const double* f);
int lbm_get_populations(lbm_ctx* c, int comp, double* f);
/* Change the imposed inlet value (density or velocity, by inlet_kind) and the outlet density
 * between steps (pressure ramps of PAPER.md L223). */
int lbm_set_boundary(lbm_ctx* c, double inlet_value, double outlet_rho);

/* Advance n time steps (SURVEY.md §8c steps 1-7 per step): density pass (Eq. 3), virtual solid
 * density (Eq. 14-15), forces (Eq. 10, 11, 13), tau_s and u_eq (Eq. 5-8), collision (Eq. 1, 2,
 * 9), streaming with halfway bounce-back, open-plane fix (L147-157).
 * Asynchronous on torch's current stream; n >= 0.  A context may be used from different streams
 * in turn: a call on another stream than the previous call's first waits for the work enqueued
 * there.  The open-plane fix of the last step is deferred: it is applied by the
 * next lbm_step (inside its density pass) or by the next getter, whichever comes first, with the
 * boundary values that were in force when the step ran; callers always observe a complete state. */
int lbm_step(lbm_ctx* c, int n);
int lbm_sync(lbm_ctx* c);

/* rho_sigma (Eq. 3), u = u_eq (Eq. 8) and P (Eq. 12, reading R13) of the current
 * state; any output pointer may be NULL. */
int lbm_get_macroscopic(lbm_ctx* c, double* rhoA, double* rhoB, double* ux, double* uy,
                        double* uz, double* P);
/* mass[sigma] = sum_x rho_sigma; momentum = sum_x sum_sigma sum_i e_i f_i (bare). fp64 sums in
 * a fixed order (deterministic). */
int lbm_diagnostics(lbm_ctx* c, double mass[2], double momentum[3]);
/* Saturation of component comp in z in [z0,z1): fraction of fluid nodes with rho_comp greater
 * than the other density (tie -> component 1) (reading R14). */
int lbm_saturation(lbm_ctx* c, int comp, int z0, int z1, double* S);
/* Trapped volume (reading R15): phase-comp nodes in [z0,z1) whose 6-connected
 * same-phase cluster (periodic in x,y; not across z) touches neither z=0 nor z=nz-1; *nodes is
 * their number, *mass the sum of rho_comp over them.  The phase of a node is decided as in
 * lbm_saturation.  Runs on the GPU (lock-free union-find over the compact ids, 8 B per fluid
 * node of temporary device memory); an empty z-range gives 0.  Synchronises. */
int lbm_trapped_volume(lbm_ctx* c, int comp, int z0, int z1, long long* nodes, double* mass);
/* lbm_trapped_volume without any allocation: same query, same kernels, same result (node count
 * and mass bit-identical), but the scratch of the connected-component labelling (8 B per fluid
 * node + 19 KB of partial sums) lives in a file-scope device array of the library instead of a
 * temporary buffer from the caching allocator.  The call performs no cudaMalloc / cudaFree and
 * calls no allocating routine; it is for callers that cannot allocate (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc).  Limits and caveats:
 *  - boxes of at most LBM_STATIC_MAX_NODES fluid nodes; more -> LBM_EINVAL with a message naming
 *    the limit (use lbm_trapped_volume);
 *  - every GPU that loads the library holds the array (8 MiB + 19 KB) until the process exits;
 *  - ALL contexts on a device share the one array and it keeps the last call's contents (the call
 *    rewrites every word it reads, nothing needs clearing): two calls that overlap on the GPU --
 *    from different streams or host threads -- race.  One call at a time per device;
 *  - not available on slab contexts.  Synchronises like lbm_trapped_volume. */
#define LBM_STATIC_MAX_NODES 1048576
int lbm_trapped_volume_static(lbm_ctx* c, int comp, int z0, int z1, long long* nodes, double* mass);
/* Mean over the fluid nodes with z in [z0,z1) of the pressure of Eq. (12) (reading R13):
 * P = (rho_A+rho_B)/3 + (G/3) rho_A rho_B.  The capillary pressure of the drainage protocol
 * is P_c = mean over the inlet layer - mean over the outlet layer.  Computed on
 * the GPU in the storage precision per node, accumulated in fp64 in a fixed order.
 * LBM_ENOFLUID if the range holds no fluid node.  Synchronises. */
int lbm_mean_pressure(lbm_ctx* c, int z0, int z1, double* P);

long long lbm_num_fluid(lbm_ctx* c);       /* N_f, or -1 */
long long lbm_num_wall_solid(lbm_ctx* c);  /* N_w: solid voxels with >= 1 fluid D3Q19 neighbour */
/* Device bytes the context holds, split as [0] populations, [1] psi, [2] index tables, [3] other. */
int lbm_memory_bytes(lbm_ctx* c, long long bytes[4]);
/* Device time (ms) of the kernels of the last lbm_step call, by kind, measured with CUDA events
 * on the launching stream when profiling is enabled with lbm_set_profiling(c, 1):
 * ms[0] density pass (in the default path it carries the open-plane fix of the previous step),
 * [1] virtual-solid pass, [2] collide+stream,
 * [3] open-plane fix when it is launched on its own; launches = number of kernel launches of that
 * call.  Synchronises. */
int lbm_set_profiling(lbm_ctx* c, int on);
int lbm_last_step_profile(lbm_ctx* c, double ms[4], long long* launches);
const char* lbm_last_error(void);

/* Host-only helper (no GPU needed): builds the compact index exactly as lbm_create does and
 * returns it for inspection.  vox2id (nx*ny*nz int32, caller-allocated): fluid id in [0,N_f),
 * N_f + wall id for wall solids, -1 for buried solids.  nbr (18*N_f int32, caller-allocated,
 * may be NULL; pass capacity in nbr_cap as a count of int32): nbr[(i-1)*N_f + n] for direction
 * i = 1..18: id of x+e_i (fluid id, or N_f + wall id), or -(m+1) with m the mirror node when
 * x+e_i lies beyond an open plane.  Returns N_f through *nf and N_w through *nw. */
int lbm_build_index(const uint8_t* solid, int nx, int ny, int nz, int z_open, int32_t* vox2id,
                    int32_t* nbr, long long nbr_cap, long long* nf, long long* nw);

/* ---- z-slab sharding across GPUs --------
 * The step has two grid-wide dependencies (Eq. 11/13: every node's force needs its
 * neighbours' rho(t); Eq. 15: every wall solid's rho~(t) needs its fluid neighbours' rho(t)) and
 * one transport across a cut (Eq. 1 LHS: 5 populations per component cross a z-plane).  The box
 * is cut into contiguous z-slabs, one lbm_ctx per slab (one per GPU).  An end of a slab is either a
 * CUT (halo_lo / halo_hi = 1: the mask carries LBM_SLAB_GHOST = 2 halo planes there, copies of the
 * neighbour slab's planes) or the global box's own end (0: no halo planes; allowed only when
 * z_open = 1, and the slab then owns the inlet plane z = 0 / the outlet plane z = nz-1 with the
 * open-plane treatment of PAPER.md L147-157).  A z-periodic box has cuts at both ends of every
 * slab (the halo planes wrap around).  nz_local = owned + 2*(halo_lo + halo_hi), owned >= 2.
 * One time step of a slab is, in this order (anything else returns LBM_EINVAL),
 *     lbm_slab_density(c, 0)     a1 on the two owned planes at each face (the psi the neighbours need)
 *     psi exchange START         buffers 0,1 (send) -> the neighbours' 2,3 (receive)
 *     lbm_slab_density(c, 1)     a1 on the interior: overlaps the exchange
 *     psi exchange COMPLETE
 *     lbm_slab_collide(c, 0)     a2 on all wall solids of the local box; a3-a6 on the tiles of the
 *                                outermost owned plane of each face; pack of what crossed a cut
 *     population exchange START  buffers 4,5 (send) -> the neighbours' 6,7 (receive)
 *     lbm_slab_collide(c, 1)     a3-a6 on the interior tiles: overlaps the exchange
 *     population exchange COMPLETE
 *     lbm_slab_unpack(c)         received populations -> rows of the owned boundary planes
 * (a getter may follow lbm_slab_density(c, 1) + the completed psi exchange; the next step then
 * starts again with lbm_slab_density(c, 0)),
 * and the result on the owned nodes is bit-identical to the unsharded lbm_step (same kernels, same
 * summation order).  The exchanges move DEVICE buffers and are the caller's (NCCL send/recv
 * through torch.distributed in paper_2207_01534_b200/slab.py; device copies when several slabs
 * live on one GPU).  All calls are asynchronous on torch's current stream.
 * lbm_set_density / lbm_set_populations / lbm_get_* take dense arrays of the LOCAL box
 * (nx*ny*nz_local); halo voxels are ignored on input and written as 0 by lbm_get_macroscopic,
 * which in slab mode requires both lbm_slab_density parts + the psi exchange to have been done on
 * the current state; so do lbm_saturation and lbm_mean_pressure, whose z-range is in LOCAL planes
 * and which cover the owned nodes only (halo planes are empty ranges).  lbm_diagnostics sums over
 * the owned nodes.  lbm_step and lbm_trapped_volume return LBM_EINVAL on a slab context (the
 * trapped volume of a cut box is the lbm_slab_ccl_* sequence below). */
#define LBM_SLAB_GHOST 2
int lbm_create_slab(lbm_ctx** out, const uint8_t* solid_local, int nx, int ny, int nz_local,
                    const lbm_params* p, int halo_lo, int halo_hi);
int lbm_create_slab_opt(lbm_ctx** out, const uint8_t* solid_local, int nx, int ny, int nz_local,
                        const lbm_params* p, const lbm_options* opt, int halo_lo, int halo_hi);
int lbm_slab_density(lbm_ctx* c, int part);
int lbm_slab_collide(lbm_ctx* c, int part);
int lbm_slab_unpack(lbm_ctx* c);
/* Exchange buffers (DEVICE pointers into the context's memory, valid until lbm_destroy; psi
 * buffers are (rho_A, rho_B) pairs of the storage type, population buffers (f_A, f_B) pairs).
 * which = 2*kind + face, face 0 = low z, 1 = high z:
 *   kind 0: psi of my two owned planes at that face (send)   kind 1: psi of my two halo planes (receive)
 *   kind 2: packed populations that left through that face   kind 3: populations arriving through it
 *   kind 4 (which 8, 9): cluster flags of my boundary planes  kind 5 (which 10, 11): the neighbours' (ints)
 * A slab's send buffer of face 1 has the byte count of its upper neighbour's receive buffer of
 * face 0, and vice versa (both are derived from the same mask planes). */
int lbm_slab_buffer(lbm_ctx* c, int which, void** dev, long long* bytes);
long long lbm_num_owned(lbm_ctx* c);   /* fluid nodes of the owned planes, or -1 */
/* The sharded step inside the library, one rank (process) per GPU, slab r of N on rank r: the
 * exchanges are grouped ncclSend / ncclRecv to the two ring neighbours on a side stream, ordered
 * against the launches by events, so that the psi exchange runs beside the interior density pass
 * and the population exchange beside the interior fused pass -- no host work between the
 * launches of a step beyond enqueuing them.  lbm_comm_unique_id (on ONE rank) makes the
 * rendezvous token, which the caller distributes to all ranks by whatever means it has
 * (torch.distributed broadcast in paper_2207_01534_b200/slab.py); lbm_slab_comm_init is
 * collective over the N ranks (it creates the NCCL communicator; N = 1 is allowed: the single
 * slab of a z-periodic box exchanges with itself); lbm_slab_step(c, n) then advances n time
 * steps, asynchronously on torch's current stream, each in the order listed above including
 * lbm_slab_unpack; lbm_slab_exchange(c, kind) is one exchange on its own (kind 0 psi, 1
 * populations, 2 the cluster-flag planes of the trapped-volume query), in line on the current
 * stream.  The result is bit-identical to the unsharded lbm_step and to the call-by-call
 * sequence with caller-side exchanges.  LBM_ECUDA on an NCCL error. */
#define LBM_COMM_ID_BYTES 128
int lbm_comm_unique_id(char id[LBM_COMM_ID_BYTES]);
int lbm_slab_comm_init(lbm_ctx* c, const char id[LBM_COMM_ID_BYTES], int rank, int world);
int lbm_slab_step(lbm_ctx* c, int n);
int lbm_slab_exchange(lbm_ctx* c, int kind);
/* Trapped volume (reading R15) of a box cut into slabs.  Every slab labels the connected
 * components of the phase-comp nodes it owns (lbm_slab_ccl_begin; needs psi of the current state
 * like the other slab queries; mark_lo / mark_hi = this slab owns the global plane z = 0 /
 * z = nz-1, whose clusters are "connected to an end").  Then, until no slab reports a change:
 * lbm_slab_ccl_export fills buffers 8 (low face) and 9 (high face) of lbm_slab_buffer with one
 * int per (x,y) of the outermost owned plane -- the end-connected flag of the phase cluster
 * there, -1 where there is none --, the caller moves them into the neighbours' buffers 11 and 10,
 * and lbm_slab_ccl_import raises the flags of the clusters of its own boundary-plane nodes whose
 * neighbour across the cut is end-connected (use_lo / use_hi = 0 ignores a face: the box's own
 * end, or the periodic wrap, across which R15 does not connect); *changed = clusters newly
 * flagged.  lbm_slab_ccl_finish counts the nodes, and adds rho_comp, of the unflagged clusters in
 * the LOCAL planes [z0,z1) and ends the session.  import and finish synchronise. */
int lbm_slab_ccl_begin(lbm_ctx* c, int comp, int mark_lo, int mark_hi);
int lbm_slab_ccl_export(lbm_ctx* c);
int lbm_slab_ccl_import(lbm_ctx* c, int use_lo, int use_hi, int* changed);
int lbm_slab_ccl_finish(lbm_ctx* c, int z0, int z1, long long* nodes, double* mass);
/* Host-only helper (no GPU needed): the halo lists lbm_create_slab builds, decoded for inspection.
 * pack_dir_vox / unpack_dir_vox: caller-allocated, 2*cap int32 each; entry k is (direction i,
 * local voxel index of the node whose row slot is read / written), low face first then high face;
 * n_pack / n_unpack: entries per face; psi_send / psi_recv: fluid nodes per face of the psi
 * exchange; *n_owned: fluid nodes of the owned planes. */
int lbm_build_slab_halo(const uint8_t* solid_local, int nx, int ny, int nz_local, int z_open,
                        int halo_lo, int halo_hi, int32_t* pack_dir_vox, int32_t* unpack_dir_vox, long long cap,
                        long long n_pack[2], long long n_unpack[2], long long psi_send[2],
                        long long psi_recv[2], long long* n_owned);

#ifdef __cplusplus
}
#endif
#endif
