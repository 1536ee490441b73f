// lbm.cu -- the C ABI of include/lbm.h: host orchestration of the sm_100a kernels.
// Product code; no CPU fallback; shares nothing with oracle/.
#include "../../include/lbm.h"

#include <cuda_runtime.h>
#include <nccl.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <utility>
#include <vector>

#include "geometry.hpp"
#include "kernels.cuh"

extern "C" void* lbm_shim_alloc(size_t bytes);
extern "C" void lbm_shim_free(void* p);
extern "C" void* lbm_shim_stream(void);

namespace {

thread_local std::string g_err;

int fail(int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_err = buf;
  return code;
}

#define CU(call)                                                                         \
  do {                                                                                   \
    cudaError_t e_ = (call);                                                             \
    if (e_ != cudaSuccess)                                                               \
      return fail(LBM_ECUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_),     \
                  __FILE__, __LINE__);                                                   \
  } while (0)

inline unsigned blocks(long long n, int b) { return (unsigned)((n + b - 1) / b); }
inline size_t pad64(long long n) { return (size_t)((n + 63) / 64 * 64); }
// population / neighbour rows are padded to whole 256-node tiles so that every bulk copy of the
// fused pass is a full, 1 KB-aligned segment
inline size_t pad256(long long n) { return (size_t)((n + 255) / 256 * 256); }

struct ProfEvent {
  int kind;
  cudaEvent_t a, b;
};

// RAII for temporary device buffers from torch's caching allocator
struct DevBuf {
  void* p = nullptr;
  explicit DevBuf(size_t bytes) { p = lbm_shim_alloc(bytes ? bytes : 1); }
  ~DevBuf() { lbm_shim_free(p); }
  DevBuf(const DevBuf&) = delete;
  DevBuf& operator=(const DevBuf&) = delete;
};

}  // namespace

struct lbm_ctx {
  lbm_params p{};
  int nx = 0, ny = 0, nz = 0, np = 0, bits = 32, device = 0;
  long long nvox = 0;
  int nf = 0, nw = 0;
  int nact = 0;             // ids [0,nact) are updated by this context; = nf unless slab mode
  int slab = 0;             // 1: z-slab of a larger box (halo planes at the ends that are cuts)
  int open_end[2] = {0, 0}; // this box's low / high z end is an open plane (inlet / outlet)
  int* halo_slots = nullptr;         // [pack low | pack high | unpack low | unpack high] pair slots
  void* halo_send = nullptr;         // [pack low | pack high] (A,B) pairs
  void* halo_recv = nullptr;         // [unpack low | unpack high] (A,B) pairs
  int n_pack[2] = {0, 0}, n_unpack[2] = {0, 0};
  long long psi_send[2][2] = {{0, 0}, {0, 0}}, psi_recv[2][2] = {{0, 0}, {0, 0}};
  int edge_plane[2] = {0, 0};        // fluid nodes of the outermost owned plane at each end
  int* ccl = nullptr;                // slab trapped volume: parent[nact] | flag[nact] | 4 planes of
                                     // np ints (send low, send high, receive low, receive high) | counter
  int ccl_comp = -1;                 // component of the running ccl session, -1: none
  int slab_phase = 0;       // next slab call: 0 density(0), 1 density(1), 2 collide(0), 3 collide(1),
                            // 4 unpack
  // slab mode: id ranges [0, bnd_lo1) and [bnd_hi0, nact) hold the two owned planes at each face
  // (rounded to 256 ids), tiles [0, tile_lo1) and [tile_hi0, tiles) the outermost owned plane
  int bnd_lo1 = 0, bnd_hi0 = 0, tile_lo1 = 0, tile_hi0 = 0;
  size_t npad = 0, nwpad = 0, esz = 4;
  std::vector<int32_t> zstart;  // [nz+1] first fluid id of every z-plane (host copy, used by queries)
  void* f[2] = {nullptr, nullptr};                // two buffers of [19][npad][2 comps] T
  void* psi = nullptr;                            // [nf+nw] Vec2<T>
  int* nbr_wide = nullptr;                        // [wide tiles][18][128] int32 ids of the wide tiles
  int* wall_nbr = nullptr;                        // [18][nwpad]
  void* wall_inv_den = nullptr;                   // [nw] T
  int* node_vox_d = nullptr;                      // [nf]
  void* frozen = nullptr;                         // [2 planes][2 comps][5][np] T
  double* partial = nullptr;                      // [diag blocks][6]
  double* diag_out = nullptr;                     // [6] + count
  int diag_blocks = 0;
  int cur = 0;
  bool open_pending = false;  // the open-plane fix of the last step has not been applied yet (it
                              // is folded into the next density pass, or applied by a getter)
  int num_sms = 148;
  uint16_t* nbr16 = nullptr;         // [18][npad]
  int* nbr16_meta = nullptr;         // [tiles][kIdxMeta]
  long long wide_tiles = 0;
  int reverse = 1;          // the fused pass walks the tiles backwards (L2 reuse across the passes)
  float keep_psi = 0.f;     // share of the psi lines stored with L2 evict_last priority, from
  int keep_psi_mb = 48;     // this budget: min(1, MB / psi bytes) (0: off)
  int pdl = 1;              // programmatic dependent launch of the three passes
  // Launch-bound boxes (a step of config 1 or 2 is three kernels of 3-8 us each): lbm_step replays
  // a captured CUDA graph of kGraphSteps steps (programmatic-dependent-launch edges included)
  // instead of launching every kernel from the host.  One graph per starting buffer parity;
  // dropped when a kernel argument changes (lbm_set_boundary).  lbm_options.graph (default:
  // on for boxes of up to kGraphAutoNodes fluid nodes, where the host launch rate is the limit).
  int graph_mode = -1;      // -1 auto, 0 off, 1 on
  cudaGraphExec_t graph_exec[2] = {nullptr, nullptr};
  cudaStream_t cap_stream = nullptr;   // capture happens here (torch's current stream may be the
                                       // legacy default stream, which cannot be captured); the
                                       // graphs are launched on the caller's stream
  long long graph_launches = 0;   // kernel launches inside one graph
  long long steps_done = 0;
  // Streams: work is enqueued on torch's current stream at each call.  The context remembers the
  // last stream it used; a call on a different stream first waits (event) for the work enqueued on
  // the previous one, and lbm_destroy synchronises the device before the buffers go back to the
  // caching allocator.
  // Native slab ring (lbm_slab_comm_init / lbm_slab_step): NCCL communicator over the slabs, one
  // rank per GPU; the exchanges run on comm_stream beside the interior launches of the same pass.
  ncclComm_t comm = nullptr;
  int comm_rank = 0, comm_world = 0;
  cudaStream_t comm_stream = nullptr;
  cudaEvent_t comm_ev[4] = {nullptr, nullptr, nullptr, nullptr};
  cudaStream_t last_stream = nullptr;
  bool has_stream = false;
  cudaEvent_t order_ev = nullptr;
  long long bytes[4] = {0, 0, 0, 0};
  bool prof = false;
  std::vector<ProfEvent> prof_events;
  double prof_ms[4] = {0, 0, 0, 0};
  long long prof_launches = 0;

  void drop_graphs() {
    for (auto& g : graph_exec) { if (g) cudaGraphExecDestroy(g); g = nullptr; }
  }
  ~lbm_ctx() {
    drop_graphs();
    if (cap_stream) cudaStreamDestroy(cap_stream);
    if (order_ev) cudaEventDestroy(order_ev);
    if (comm) ncclCommDestroy(comm);
    if (comm_stream) cudaStreamDestroy(comm_stream);
    for (auto& e : comm_ev) if (e) cudaEventDestroy(e);
    for (auto& e : prof_events) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
    lbm_shim_free(f[0]); lbm_shim_free(f[1]); lbm_shim_free(psi);
    lbm_shim_free(nbr_wide);
    lbm_shim_free(wall_nbr); lbm_shim_free(wall_inv_den); lbm_shim_free(node_vox_d);
    lbm_shim_free(frozen); lbm_shim_free(partial); lbm_shim_free(diag_out);
    lbm_shim_free(nbr16);
    lbm_shim_free(nbr16_meta);
    lbm_shim_free(halo_slots); lbm_shim_free(halo_send); lbm_shim_free(halo_recv);
    lbm_shim_free(ccl);
  }
};

namespace {

using namespace lbmk;

template <typename T>
Consts<T> make_consts(const lbm_params& p) {
  Consts<T> c;
  c.G = (T)p.G; c.tauA = (T)p.tau[0]; c.tauB = (T)p.tau[1];
  c.gx = (T)p.accel[0]; c.gy = (T)p.accel[1]; c.gz = (T)p.accel[2];
  c.hf = p.half_force ? (T)0.5 : (T)0;
  c.chiA = (T)(1.0 + p.xi); c.chiB = (T)(1.0 - p.xi);
  return c;
}

constexpr int kGraphSteps = 16;            // even: the buffer parity returns to its start
constexpr int kGraphAutoNodes = 600000;    // above this a step is long enough to hide the launches
template <typename T>
OpenPlane<T> make_open(const lbm_params& p, const int (&open_end)[2]) {
  OpenPlane<T> o;
  o.dc[0] = p.inlet_comp; o.dc[1] = p.outlet_comp;
  o.kind[0] = open_end[0] ? p.inlet_kind : 0; o.kind[1] = open_end[1] ? p.outlet_kind : 0;
  o.rho[0] = (T)p.inlet_rho; o.rho[1] = (T)p.outlet_rho;
  o.uz[0] = (T)p.inlet_uz; o.uz[1] = (T)0;
  return o;
}

NbrView make_view(const lbm_ctx* c) {
  NbrView v;
  v.nbr16 = (const uint16_t*)c->nbr16;
  v.meta = c->nbr16_meta;
  v.wide = c->nbr_wide;
  v.np_lo = c->open_end[0] ? c->np : 0;
  v.np_hi = c->open_end[1] ? c->np : 0;
  v.nact = c->nact;
  return v;
}

cudaStream_t cur_stream() { return (cudaStream_t)lbm_shim_stream(); }

// torch's current stream, ordered after whatever this context enqueued on another stream before
cudaStream_t use_stream(lbm_ctx* c) {
  cudaStream_t st = cur_stream();
  if (c->has_stream && st != c->last_stream) {
    if (!c->order_ev) cudaEventCreateWithFlags(&c->order_ev, cudaEventDisableTiming);
    if (c->order_ev) {
      cudaEventRecord(c->order_ev, c->last_stream);
      cudaStreamWaitEvent(st, c->order_ev, 0);
    } else {
      cudaStreamSynchronize(c->last_stream);
    }
  }
  c->last_stream = st;
  c->has_stream = true;
  return st;
}

struct ProfOff {  // queries run their density / wall passes unprofiled; restored on every exit path
  lbm_ctx* c; bool was;
  explicit ProfOff(lbm_ctx* c_) : c(c_), was(c_->prof) { c->prof = false; }
  ~ProfOff() { c->prof = was; }
};

struct Timed {  // brackets one launch with events when profiling is on
  lbm_ctx* c; cudaStream_t st; int kind; ProfEvent ev{};
  Timed(lbm_ctx* c_, cudaStream_t st_, int kind_) : c(c_), st(st_), kind(kind_) {
    if (c->prof) {
      ev.kind = kind;
      cudaEventCreate(&ev.a); cudaEventCreate(&ev.b);
      cudaEventRecord(ev.a, st);
    }
  }
  ~Timed() {
    if (c->prof) { cudaEventRecord(ev.b, st); c->prof_events.push_back(ev); }
    ++c->prof_launches;
  }
};

// Launch with the programmatic-stream-serialization attribute: the kernel's blocks may become
// resident while the previous kernel of the stream drains, and run up to their pdl_wait().
template <typename... KArgs, typename... Args>
void launch_k(bool pdl, void (*kern)(KArgs...), unsigned grid, unsigned block, size_t smem,
              cudaStream_t st, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(block);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = pdl ? 1 : 0;
  cudaLaunchKernelEx(&cfg, kern, std::forward<Args>(args)...);
}

// a1 (+ the deferred a0 of the previous step) on the current buffer, ids [0, nact).
// part: -1 whole range; slab mode: 0 = the boundary id ranges of both faces, 1 = the interior.
template <typename T>
void launch_density(lbm_ctx* c, cudaStream_t st, int part = -1) {
  T* fin = (T*)c->f[c->cur];
  const bool pdl = c->pdl && !c->prof;  // events between the launches would serialise them anyway
  Timed t(c, st, 0);
  NodeRange r{0, (int)blocks(c->nact, 256), 0, c->nact};
  unsigned grid = blocks(c->nact, 256);
  if (c->open_pending && part != 1) {  // a0 of the previous step rides along (k_density_open);
    // in slab mode with the boundary launch: the open planes lie inside the boundary id ranges
    const unsigned nbp = blocks(2LL * c->np, 256);
    if (part == 0) {
      r.split = c->bnd_lo1 / 256;
      r.a1 = c->bnd_hi0;
      grid = (unsigned)r.split + blocks(c->nact - c->bnd_hi0, 256);
    }
    launch_k(pdl, k_density_open<T>, nbp + grid, 256, 0, st, fin,
             (Vec2<T>*)c->psi, (const T*)c->frozen, c->nact, c->np, c->npad, (int)nbp,
             make_open<T>(c->p, c->open_end), c->keep_psi, r);
    c->open_pending = false;
  } else {
    if (part == 0) {
      r.split = c->bnd_lo1 / 256;
      r.a1 = c->bnd_hi0;
      grid = (unsigned)r.split + blocks(c->nact - c->bnd_hi0, 256);
    } else if (part == 1) {
      r.a0 = c->bnd_lo1;
      r.nend = c->bnd_hi0;
      grid = (unsigned)((c->bnd_hi0 - c->bnd_lo1) / 256);
      r.split = (int)grid;
    }
    if (grid > 0)
      launch_k(pdl, k_density<T>, grid, 256, 0, st, (const T*)fin, (Vec2<T>*)c->psi, r, c->npad,
               c->keep_psi);
  }
}

// a2 on every wall solid of the box
template <typename T>
void launch_wall(lbm_ctx* c, cudaStream_t st) {
  if (c->nw <= 0) return;
  const bool pdl = c->pdl && !c->prof;
  Timed t(c, st, 1);
  launch_k(pdl, k_wallpsi<T>, blocks(c->nw, 256), 256, 0, st, (Vec2<T>*)c->psi,
           (const int*)c->wall_nbr, (const T*)c->wall_inv_den, c->npad, c->nw, c->nwpad,
           (T)(1.0 + c->p.xi), (T)(1.0 - c->p.xi), c->keep_psi);
}

// a1 + a2.  Slab mode: the density pass (lbm_slab_density) and the psi halo exchange are the
// caller's; only the wall pass runs here.
template <typename T>
void launch_psi(lbm_ctx* c, cudaStream_t st) {
  if (!c->slab) launch_density<T>(c, st);
  launch_wall<T>(c, st);
}

// Apply a deferred open-plane fix now (getters that read the populations directly).
template <typename T>
void apply_pending_T(lbm_ctx* c, cudaStream_t st) {
  if (!c->open_pending) return;
  k_open_planes<T><<<blocks(2LL * c->np, 128), 128, 0, st>>>((T*)c->f[c->cur], (const T*)c->frozen,
                                                             c->nact, c->np, c->npad,
                                                             make_open<T>(c->p, c->open_end));
  c->open_pending = false;
}
void apply_pending(lbm_ctx* c, cudaStream_t st) {
  if (c->bits == 64) apply_pending_T<double>(c, st); else apply_pending_T<float>(c, st);
}

// a3-a6: the fused pass of the split step (bulk-async staged tiles).
template <typename T, int TN, int MINB, int IDX>
void launch_bulk(lbm_ctx* c, const T* fin, T* fout, const Consts<T>& k, cudaStream_t st, int part) {
  constexpr bool kRemainder = sizeof(T) == 4;
  constexpr size_t smem = IDX == 1 ? collide16_smem_bytes<T, TN, (MINB >= 7)>()
                                   : collide_smem_bytes<T, TN>();
  static bool configured[64] = {};  // function attributes are per device
  if (!configured[c->device & 63]) {
    if (cudaFuncSetAttribute(k_collide_stream_bulk<T, TN, MINB, kRemainder, IDX>,
                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) == cudaSuccess)
      configured[c->device & 63] = true;
  }
  Idx16 ix;
  ix.nbr16 = c->nbr16;
  ix.meta = c->nbr16_meta;
  ix.np_lo = c->open_end[0] ? c->np : 0;
  ix.np_hi = c->open_end[1] ? c->np : 0;
  ix.reverse = c->reverse;
  ix.nact = c->nact;
  static_assert(TN == 128 || TN == 256, "tile ranges below are in units of 128 ids");
  const int per = TN / 128;                      // slab tile ranges are kept in 128-id tiles
  unsigned grid = blocks(c->nact, TN);
  ix.tile0 = 0; ix.split = (int)grid; ix.tile1 = 0;
  if (part == 0) {                               // boundary tiles of both faces
    const int lo1 = (c->tile_lo1 + per - 1) / per, hi0 = std::max(lo1, c->tile_hi0 / per);
    ix.split = lo1; ix.tile1 = hi0;
    grid = (unsigned)lo1 + (blocks(c->nact, TN) - (unsigned)hi0);
  } else if (part == 1) {                        // interior tiles
    const int lo1 = (c->tile_lo1 + per - 1) / per, hi0 = std::max(lo1, c->tile_hi0 / per);
    ix.tile0 = lo1;
    grid = (unsigned)(hi0 - lo1);
    ix.split = (int)grid;
  }
  if (grid == 0) return;
  // Overlap only behind the wall pass: its blocks trigger after their own wait, i.e. once the
  // density pass (which may have rewritten the open planes of fin) is complete and visible.
  launch_k(c->pdl && !c->prof && c->nw > 0, k_collide_stream_bulk<T, TN, MINB, kRemainder, IDX>,
           grid, TN, smem, st, fin, fout, (const Vec2<T>*)c->psi,
           (const int*)c->nbr_wide, c->nf, c->npad, k, ix);
}

template <typename T>
void launch_collide(lbm_ctx* c, const T* fin, T* fout, const Consts<T>& k, cudaStream_t st,
                    int part = -1) {
  // fp32: 128-node tiles, 7 CTAs per SM at 72 registers (6 and 8 CTAs, 64- and 256-node tiles were
  // measured slower); fp64 validation build: 2 CTAs per SM
  if constexpr (sizeof(T) == 4) {
    launch_bulk<T, 128, 7, 1>(c, fin, fout, k, st, part);
  } else {
    launch_bulk<T, 128, 2, 1>(c, fin, fout, k, st, part);
  }
}

template <typename T>
int step_T(lbm_ctx* c, int n, cudaStream_t st) {
  const Consts<T> k = make_consts<T>(c->p);
  for (int it = 0; it < n; ++it) {
    const T* fin = (const T*)c->f[c->cur];
    T* fout = (T*)c->f[c->cur ^ 1];
    launch_psi<T>(c, st);
    {
      Timed t(c, st, 2);
      launch_collide<T>(c, fin, fout, k, st);
    }
    c->cur ^= 1;
    if (c->p.z_open) c->open_pending = true;  // a0 is folded into the next density pass
  }
  CU(cudaPeekAtLastError());
  return LBM_OK;
}

// n steps, through graph replays where that pays (see lbm_ctx::graph_mode)
template <typename T>
int step_graphed_T(lbm_ctx* c, int n, cudaStream_t st) {
  const bool want = c->graph_mode == 1 || (c->graph_mode < 0 && c->nf <= kGraphAutoNodes);
  const bool open = c->open_end[0] || c->open_end[1];
  // the first steps run directly: they configure the kernels' attributes and bring the deferred
  // open-plane fix into its steady state (pending at the start of every step)
  if (!want || c->prof || c->slab) {
    c->steps_done += n;
    return step_T<T>(c, n, st);
  }
  if (c->steps_done == 0 || (open && !c->open_pending)) {
    if (n == 0) return LBM_OK;
    if (int rc = step_T<T>(c, 1, st)) return rc;
    ++c->steps_done;
    --n;
  }
  while (n >= kGraphSteps) {
    cudaGraphExec_t& exec = c->graph_exec[c->cur];
    if (!exec) {
      const long long before = c->prof_launches;
      cudaGraph_t graph = nullptr;
      if (!c->cap_stream) CU(cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking));
      CU(cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal));
      const int rc = step_T<T>(c, kGraphSteps, c->cap_stream);   // captured, not executed
      const cudaError_t e = cudaStreamEndCapture(c->cap_stream, &graph);
      c->graph_launches = c->prof_launches - before;
      c->prof_launches = before;
      if (rc || e != cudaSuccess || !graph) {
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        c->graph_mode = 0;   // capture is not available here: plain launches from now on
        return rc ? rc : step_T<T>(c, n, st);
      }
      const cudaError_t ei = cudaGraphInstantiate(&exec, graph, 0);
      cudaGraphDestroy(graph);
      if (ei != cudaSuccess) {
        exec = nullptr;
        cudaGetLastError();
        c->graph_mode = 0;
        return step_T<T>(c, n, st);
      }
    }
    CU(cudaGraphLaunch(exec, st));
    c->prof_launches += c->graph_launches;
    c->steps_done += kGraphSteps;
    n -= kGraphSteps;
  }
  c->steps_done += n;
  return step_T<T>(c, n, st);
}

template <typename T>
int record_frozen_T(lbm_ctx* c, int comp, cudaStream_t st) {
  if (!c->open_end[0] && !c->open_end[1]) return LBM_OK;
  k_record_frozen<T><<<blocks(2LL * c->np, 128), 128, 0, st>>>(
      (const T*)c->f[c->cur], (T*)c->frozen, comp, c->nact, c->np, c->npad,
      c->open_end[0] | (c->open_end[1] << 1));
  CU(cudaPeekAtLastError());
  return LBM_OK;
}

int check_ctx(lbm_ctx* c) {
  if (!c) return fail(LBM_EINVAL, "NULL context");
  cudaError_t e = cudaSetDevice(c->device);
  if (e != cudaSuccess) return fail(LBM_ECUDA, "cudaSetDevice: %s", cudaGetErrorString(e));
  return LBM_OK;
}

int validate_params(const lbm_params* p, int nz) {
  if (!(p->tau[0] > 0.5) || !(p->tau[1] > 0.5) || !std::isfinite(p->tau[0]) ||
      !std::isfinite(p->tau[1]))
    return fail(LBM_EINVAL, "relaxation times must be finite and > 1/2");
  if (!std::isfinite(p->G) || !std::isfinite(p->xi))
    return fail(LBM_EINVAL, "G and xi must be finite");
  if (p->storage_bits != 32 && p->storage_bits != 64)
    return fail(LBM_EINVAL, "storage_bits must be 32 or 64");
  if (p->z_open) {
    if (nz < 4) return fail(LBM_EINVAL, "z_open needs nz >= 4");
    if (p->inlet_kind < 1 || p->inlet_kind > 4)
      return fail(LBM_EINVAL, "inlet_kind must be 1, 2 (NEEM density, velocity) or 3, 4 (Zou-He)");
    if (p->outlet_kind != 1 && p->outlet_kind != 3)
      return fail(LBM_EINVAL, "outlet_kind must be 1 (NEEM density) or 3 (Zou-He density)");
    if (p->inlet_comp < 0 || p->inlet_comp > 1 || p->outlet_comp < 0 || p->outlet_comp > 1)
      return fail(LBM_EINVAL, "inlet_comp / outlet_comp must be 0 or 1");
  }
  return LBM_OK;
}

}  // namespace

extern "C" {

const char* lbm_last_error(void) { return g_err.c_str(); }

int lbm_build_index(const uint8_t* solid, int nx, int ny, int nz, int z_open, int32_t* vox2id,
                    int32_t* nbr, long long nbr_cap, long long* nf, long long* nw) {
  if (!solid || !vox2id || !nf || !nw) return fail(LBM_EINVAL, "NULL argument");
  lbmgeo::Geometry g;
  const int rc = lbmgeo::build(g, solid, nx, ny, nz, z_open, nbr != nullptr);
  if (rc) return fail(rc, "geometry build failed (%d)", rc);
  std::memcpy(vox2id, g.vox2id.data(), sizeof(int32_t) * g.nvox);
  *nf = g.nf;
  *nw = g.nw;
  if (nbr) {
    if (nbr_cap < 18 * g.nf) return fail(LBM_EINVAL, "nbr capacity too small");
    std::memcpy(nbr, g.nbr.data(), sizeof(int32_t) * 18 * g.nf);
  }
  return LBM_OK;
}

void lbm_options_default(lbm_options* o) {
  if (!o) return;
  o->graph = -1;
  o->pdl = 1;
  o->reverse = 1;
  o->keep_psi_mb = 48;
}

static int validate_options(const lbm_options* o) {
  if (o->graph < -1 || o->graph > 1) return fail(LBM_EINVAL, "options.graph must be -1, 0 or 1");
  if ((o->pdl != 0 && o->pdl != 1) || (o->reverse != 0 && o->reverse != 1))
    return fail(LBM_EINVAL, "options.pdl and options.reverse must be 0 or 1");
  if (o->keep_psi_mb < 0) return fail(LBM_EINVAL, "options.keep_psi_mb must be >= 0");
  return LBM_OK;
}

static int create_impl(lbm_ctx** out, const uint8_t* solid, int nx, int ny, int nz,
                       const lbm_params* p, const lbm_options* opt, bool slab, int halo_lo,
                       int halo_hi) {
  if (!out || !solid || !p) return fail(LBM_EINVAL, "NULL argument");
  lbm_options o;
  lbm_options_default(&o);
  if (opt) o = *opt;
  if (int rc = validate_options(&o)) return rc;
  if (nx < 1 || ny < 1 || nz < 1) return fail(LBM_EINVAL, "box dimensions must be positive");
  if (int rc = validate_params(p, nz)) return rc;
  if (slab && ((halo_lo != 0 && halo_lo != 1) || (halo_hi != 0 && halo_hi != 1)))
    return fail(LBM_EINVAL, "halo_lo / halo_hi must be 0 or 1");
  if (slab && !p->z_open && !(halo_lo && halo_hi))
    return fail(LBM_EINVAL, "a slab of a z-periodic box is a cut at both ends (halo_lo = halo_hi = 1)");
  const int ghost_lo = slab && halo_lo ? lbmgeo::kSlabGhost : 0;
  const int ghost_hi = slab && halo_hi ? lbmgeo::kSlabGhost : 0;
  if (slab && nz < ghost_lo + ghost_hi + 2)
    return fail(LBM_EINVAL, "a slab needs >= 2 owned planes plus %d halo planes per cut end",
                lbmgeo::kSlabGhost);
  lbmgeo::Geometry g;
  {
    const int rc = lbmgeo::build(g, solid, nx, ny, nz, p->z_open, true, ghost_lo, ghost_hi);
    if (rc == -2) return fail(LBM_ENOFLUID, "the mask has no fluid voxel");
    if (rc == -3) return fail(LBM_ESOLIDOPEN, "solid voxel on an open plane or its neighbour plane");
    if (rc == -4) return fail(LBM_ENOMEM, "host allocation failed");
    if (rc) return fail(LBM_EINVAL, "bad geometry arguments");
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
    cudaGetLastError();
    return fail(LBM_ECUDA, "no CUDA device: this library has no CPU fallback");
  }
  int device = 0;
  CU(cudaGetDevice(&device));
  lbm_ctx* c = new (std::nothrow) lbm_ctx;
  if (!c) return fail(LBM_ENOMEM, "host allocation failed");
  c->device = device;
  cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, c->device);
  c->p = *p;
  c->nx = nx; c->ny = ny; c->nz = nz; c->np = nx * ny; c->nvox = g.nvox;
  c->nf = (int)g.nf; c->nw = (int)g.nw;
  c->nact = (int)g.nact; c->slab = slab ? 1 : 0;
  c->open_end[0] = g.open_lo; c->open_end[1] = g.open_hi;
  c->bits = p->storage_bits; c->esz = p->storage_bits / 8;
  c->reverse = o.reverse;
  c->pdl = o.pdl;
  c->graph_mode = o.graph;
  c->keep_psi_mb = o.keep_psi_mb;
  c->npad = pad256(g.nf); c->nwpad = pad64(g.nw);
  // pair-slot indices i * npad + k and psi indices npad + w are 32-bit
  if ((size_t)19 * c->npad >= ((size_t)1 << 31) || c->npad + c->nwpad >= ((size_t)1 << 31)) {
    delete c;
    return fail(LBM_EINVAL, "too many fluid nodes for 32-bit slot indices");
  }
  c->zstart.assign(nz + 1, 0);
  for (long long n = 0; n < g.nact; ++n) ++c->zstart[g.node_vox[n] / c->np + 1];
  for (int z = 0; z < nz; ++z) c->zstart[z + 1] += c->zstart[z];
  cudaStream_t st = use_stream(c);
  const size_t fbytes = (size_t)2 * 19 * c->npad * c->esz;
  const size_t psibytes = (c->npad + c->nwpad) * 2 * c->esz;  // wall part starts at npad
  const size_t wnbrbytes = (size_t)18 * c->nwpad * sizeof(int);
  const size_t frozenbytes = p->z_open ? (size_t)2 * 2 * 5 * c->np * c->esz : 0;
  c->diag_blocks = 148 * 8;
  c->f[0] = lbm_shim_alloc(fbytes);
  c->f[1] = lbm_shim_alloc(fbytes);
  c->psi = lbm_shim_alloc(psibytes);
  c->wall_nbr = (int*)lbm_shim_alloc(wnbrbytes ? wnbrbytes : 4);
  c->wall_inv_den = lbm_shim_alloc(g.nw ? g.nw * c->esz : 4);
  c->node_vox_d = (int*)lbm_shim_alloc(g.nf * sizeof(int));
  c->frozen = lbm_shim_alloc(frozenbytes ? frozenbytes : 4);
  c->partial = (double*)lbm_shim_alloc((size_t)c->diag_blocks * kDiagVals * sizeof(double));
  c->diag_out = (double*)lbm_shim_alloc(8 * sizeof(double));
  if (!c->f[0] || !c->f[1] || !c->psi || !c->wall_nbr || !c->wall_inv_den ||
      !c->node_vox_d || !c->frozen || !c->partial || !c->diag_out) {
    delete c;
    return fail(LBM_ENOMEM, "device allocation failed (populations need %zu bytes per buffer)",
                fbytes);
  }
  c->bytes[0] = 2 * (long long)fbytes;
  c->bytes[1] = (long long)psibytes;
  c->keep_psi = c->keep_psi_mb > 0
                    ? (float)std::min(1.0, (double)c->keep_psi_mb * 1048576.0 / (double)psibytes)
                    : 0.f;
  c->bytes[2] = (long long)(wnbrbytes + g.nw * c->esz + g.nf * sizeof(int));
  c->bytes[3] = (long long)(frozenbytes + c->diag_blocks * kDiagVals * 8 + 64);
  cudaError_t e = cudaSuccess;
  auto up = [&](void* dst, const void* src, size_t bytes) {
    if (e == cudaSuccess && bytes) e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, st);
  };
  e = cudaMemsetAsync(c->f[0], 0, fbytes, st);
  if (e == cudaSuccess) e = cudaMemsetAsync(c->f[1], 0, fbytes, st);
  if (e == cudaSuccess) e = cudaMemsetAsync(c->psi, 0, psibytes, st);
  if (e == cudaSuccess && frozenbytes) e = cudaMemsetAsync(c->frozen, 0, frozenbytes, st);
  // (wall ids are stored as psi indices npad + w: the wall part of psi starts on a tile boundary)
  lbmgeo::Index16 i16;
  {
    if (lbmgeo::build_index16(g, (long long)c->npad, c->npad, i16) != 0) {
      delete c;
      return fail(LBM_ENOMEM, "index16 build failed");
    }
    c->wide_tiles = i16.wide_tiles;
  }
  for (int i = 0; i < 18; ++i) {
    up(c->wall_nbr + (size_t)i * c->nwpad, g.wall_nbr.data() + (size_t)i * g.nw,
         g.nw * sizeof(int));
  }
  up(c->node_vox_d, g.node_vox.data(), g.nf * sizeof(int));
  std::vector<float> invf;
  if (c->bits == 32) {
    invf.assign(g.wall_inv_den.begin(), g.wall_inv_den.end());
    up(c->wall_inv_den, invf.data(), g.nw * sizeof(float));
  } else {
    up(c->wall_inv_den, g.wall_inv_den.data(), g.nw * sizeof(double));
  }
  {
    c->nbr16 = (uint16_t*)lbm_shim_alloc(i16.nbr16.size() * sizeof(uint16_t));
    c->nbr16_meta = (int*)lbm_shim_alloc(i16.meta.size() * sizeof(int32_t) + 16);
    if (!c->nbr16 || !c->nbr16_meta) {
      delete c;
      return fail(LBM_ENOMEM, "device allocation failed (index16)");
    }
    up(c->nbr16, i16.nbr16.data(), i16.nbr16.size() * sizeof(uint16_t));
    up(c->nbr16_meta, i16.meta.data(), i16.meta.size() * sizeof(int32_t));
    c->bytes[2] += (long long)(i16.nbr16.size() * 2 + i16.meta.size() * 4);
    c->nbr_wide = (int*)lbm_shim_alloc(i16.wide_rows.size() * sizeof(int32_t) + 16);
    if (!c->nbr_wide) {
      delete c;
      return fail(LBM_ENOMEM, "device allocation failed (wide-tile table)");
    }
    up(c->nbr_wide, i16.wide_rows.data(), i16.wide_rows.size() * sizeof(int32_t));
    c->bytes[2] += (long long)(i16.wide_rows.size() * 4);
  }
  lbmgeo::Halo halo;  // declared here: its lists are upload sources until the sync below
  if (c->slab) {
    if (lbmgeo::build_halo(g, solid, c->npad, halo) != 0) {
      delete c;
      return fail(LBM_ENOMEM, "halo list build failed");
    }
    size_t nslots = 0;
    for (int fc = 0; fc < 2; ++fc) {
      c->n_pack[fc] = (int)halo.pack[fc].size();
      c->n_unpack[fc] = (int)halo.unpack[fc].size();
      nslots += halo.pack[fc].size() + halo.unpack[fc].size();
      for (int k = 0; k < 2; ++k) {
        c->psi_send[fc][k] = halo.psi_send[fc][k];
        c->psi_recv[fc][k] = halo.psi_recv[fc][k];
      }
    }
    {  // boundary-first launch ranges (ids in units of 256, tiles of 128)
      const long long na = g.nact;
      // an open end's plane rides in the boundary launch too (its deferred fix needs it there)
      const long long n_hi = g.open_hi ? c->np : halo.psi_send[1][1];
      const long long n_lo = g.open_lo ? c->np : halo.psi_send[0][1];
      long long hi0 = std::max(0LL, na - n_hi) / 256 * 256;
      long long lo1 = std::min((long long)pad256(n_lo), hi0);
      c->bnd_lo1 = (int)lo1; c->bnd_hi0 = (int)hi0;
      c->edge_plane[0] = (int)halo.edge_plane[0]; c->edge_plane[1] = (int)halo.edge_plane[1];
      c->tile_lo1 = (int)((halo.edge_plane[0] + 127) / 128);
      c->tile_hi0 = (int)(std::max(0LL, na - halo.edge_plane[1]) / 128);
    }
    const size_t sendb = (size_t)(c->n_pack[0] + c->n_pack[1]) * 2 * c->esz;
    const size_t recvb = (size_t)(c->n_unpack[0] + c->n_unpack[1]) * 2 * c->esz;
    c->halo_slots = (int*)lbm_shim_alloc(nslots * sizeof(int) + 16);
    c->halo_send = lbm_shim_alloc(sendb + 16);
    c->halo_recv = lbm_shim_alloc(recvb + 16);
    if (!c->halo_slots || !c->halo_send || !c->halo_recv) {
      delete c;
      return fail(LBM_ENOMEM, "device allocation failed (halo)");
    }
    int* d = c->halo_slots;
    for (int fc = 0; fc < 2; ++fc) { up(d, halo.pack[fc].data(), halo.pack[fc].size() * 4); d += halo.pack[fc].size(); }
    for (int fc = 0; fc < 2; ++fc) { up(d, halo.unpack[fc].data(), halo.unpack[fc].size() * 4); d += halo.unpack[fc].size(); }
    c->bytes[2] += (long long)(nslots * sizeof(int));
    c->bytes[3] += (long long)(sendb + recvb);
    const size_t cclb = ((size_t)2 * c->nact + (size_t)4 * c->np + 4) * sizeof(int);
    c->ccl = (int*)lbm_shim_alloc(cclb);
    if (!c->ccl) {
      delete c;
      return fail(LBM_ENOMEM, "device allocation failed (slab ccl)");
    }
    c->bytes[3] += (long long)cclb;
  }
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);  // host sources die with this scope
  if (e != cudaSuccess) {
    delete c;
    return fail(LBM_ECUDA, "upload failed: %s", cudaGetErrorString(e));
  }
  *out = c;
  return LBM_OK;
}

int lbm_build_slab_halo(const uint8_t* solid_local, int nx, int ny, int nz_local, int z_open,
                        int halo_lo, int halo_hi, int32_t* pack_dir_vox, int32_t* unpack_dir_vox, long long cap,
                        long long n_pack[2], long long n_unpack[2], long long psi_send[2],
                        long long psi_recv[2], long long* n_owned) {
  if (!solid_local || !pack_dir_vox || !unpack_dir_vox || !n_pack || !n_unpack || !psi_send ||
      !psi_recv || !n_owned)
    return fail(LBM_EINVAL, "NULL argument");
  lbmgeo::Geometry g;
  const int rc = lbmgeo::build(g, solid_local, nx, ny, nz_local, z_open, false,
                               halo_lo ? lbmgeo::kSlabGhost : 0, halo_hi ? lbmgeo::kSlabGhost : 0);
  if (rc) return fail(rc == -2 ? LBM_ENOFLUID : LBM_EINVAL, "geometry build failed (%d)", rc);
  const size_t npad = pad256(g.nf);
  lbmgeo::Halo h;
  if (lbmgeo::build_halo(g, solid_local, npad, h) != 0) return fail(LBM_ENOMEM, "halo build failed");
  if ((long long)(h.pack[0].size() + h.pack[1].size()) > cap ||
      (long long)(h.unpack[0].size() + h.unpack[1].size()) > cap)
    return fail(LBM_EINVAL, "list capacity too small");
  for (int pass = 0; pass < 2; ++pass) {
    int32_t* o = pass ? unpack_dir_vox : pack_dir_vox;
    for (int fc = 0; fc < 2; ++fc) {
      const std::vector<int32_t>& l = pass ? h.unpack[fc] : h.pack[fc];
      for (int32_t slot : l) {
        *o++ = (int32_t)((size_t)slot / npad);
        *o++ = g.node_vox[(size_t)slot % npad];
      }
      (pass ? n_unpack : n_pack)[fc] = (long long)l.size();
    }
  }
  for (int fc = 0; fc < 2; ++fc) { psi_send[fc] = h.psi_send[fc][1]; psi_recv[fc] = h.psi_recv[fc][1]; }
  *n_owned = g.nact;
  return LBM_OK;
}

int lbm_create(lbm_ctx** out, const uint8_t* solid, int nx, int ny, int nz, const lbm_params* p) {
  return create_impl(out, solid, nx, ny, nz, p, nullptr, false, 0, 0);
}

int lbm_create_opt(lbm_ctx** out, const uint8_t* solid, int nx, int ny, int nz,
                   const lbm_params* p, const lbm_options* opt) {
  return create_impl(out, solid, nx, ny, nz, p, opt, false, 0, 0);
}

int lbm_create_slab(lbm_ctx** out, const uint8_t* solid_local, int nx, int ny, int nz_local,
                    const lbm_params* p, int halo_lo, int halo_hi) {
  return create_impl(out, solid_local, nx, ny, nz_local, p, nullptr, true, halo_lo, halo_hi);
}

int lbm_create_slab_opt(lbm_ctx** out, const uint8_t* solid_local, int nx, int ny, int nz_local,
                        const lbm_params* p, const lbm_options* opt, int halo_lo, int halo_hi) {
  return create_impl(out, solid_local, nx, ny, nz_local, p, opt, true, halo_lo, halo_hi);
}

int lbm_step_info(lbm_ctx* c, int info[8]) {
  if (!c || !info) return fail(LBM_EINVAL, "NULL argument");
  const bool graph = c->graph_mode == 1 || (c->graph_mode < 0 && c->nf <= kGraphAutoNodes);
  info[0] = 0;
  info[1] = graph && !c->slab ? 1 : 0;
  info[2] = c->pdl; info[3] = c->reverse;
  info[4] = (int)(c->keep_psi * 1000.f + 0.5f);
  info[5] = (int)std::min<long long>(c->wide_tiles, 2147483647LL);
  info[6] = 0; info[7] = 0;
  return LBM_OK;
}

long long lbm_num_owned(lbm_ctx* c) { return c ? c->nact : -1; }

int lbm_slab_density(lbm_ctx* c, int part) {
  if (int rc = check_ctx(c)) return rc;
  if (!c->slab) return fail(LBM_EINVAL, "not a slab context");
  if (part != 0 && part != 1) return fail(LBM_EINVAL, "part must be 0 or 1");
  // part 0 may restart a step that stopped after its density pass (getters do that)
  if (part == 0 ? c->slab_phase > 2 : c->slab_phase != 1)
    return fail(LBM_EINVAL, "slab calls out of order (expected phase %d)", c->slab_phase);
  cudaStream_t st = use_stream(c);
  if (c->bits == 64) launch_density<double>(c, st, part); else launch_density<float>(c, st, part);
  CU(cudaPeekAtLastError());
  c->slab_phase = part + 1;
  return LBM_OK;
}

extern "C++" {
template <typename T>
static int slab_collide_T(lbm_ctx* c, int part, cudaStream_t st) {
  const T* fin = (const T*)c->f[c->cur];
  T* fout = (T*)c->f[c->cur ^ 1];
  if (part == 0) launch_wall<T>(c, st);
  {
    Timed t(c, st, 2);
    launch_collide<T>(c, fin, fout, make_consts<T>(c->p), st, part);
  }
  const int np = c->n_pack[0] + c->n_pack[1];
  if (part == 0 && np) {  // the boundary tiles are the only ones that push across a cut
    Timed t(c, st, 3);
    k_halo_pack<T><<<blocks(np, 256), 256, 0, st>>>((const T*)fout, c->halo_slots,
                                                    (T*)c->halo_send, np);
  }
  if (part == 1) {
    c->cur ^= 1;
    if (c->open_end[0] || c->open_end[1]) c->open_pending = true;  // a0 rides in the next density(0)
  }
  CU(cudaPeekAtLastError());
  return LBM_OK;
}
}  // extern "C++"

int lbm_slab_collide(lbm_ctx* c, int part) {
  if (int rc = check_ctx(c)) return rc;
  if (!c->slab) return fail(LBM_EINVAL, "not a slab context");
  if (part != 0 && part != 1) return fail(LBM_EINVAL, "part must be 0 or 1");
  if (c->slab_phase != 2 + part)
    return fail(LBM_EINVAL, "slab calls out of order (expected phase %d)", c->slab_phase);
  cudaStream_t st = use_stream(c);
  if (int rc = c->bits == 64 ? slab_collide_T<double>(c, part, st) : slab_collide_T<float>(c, part, st))
    return rc;
  c->slab_phase = 3 + part;
  return LBM_OK;
}

int lbm_slab_unpack(lbm_ctx* c) {
  if (int rc = check_ctx(c)) return rc;
  if (!c->slab) return fail(LBM_EINVAL, "not a slab context");
  if (c->slab_phase != 4)
    return fail(LBM_EINVAL, "slab calls out of order (expected phase %d)", c->slab_phase);
  cudaStream_t st = use_stream(c);
  const int nu = c->n_unpack[0] + c->n_unpack[1];
  const int* slots = c->halo_slots + c->n_pack[0] + c->n_pack[1];
  if (nu) {
    Timed t(c, st, 3);
    if (c->bits == 64)
      k_halo_unpack<double><<<blocks(nu, 256), 256, 0, st>>>((double*)c->f[c->cur], slots,
                                                             (const double*)c->halo_recv, nu);
    else
      k_halo_unpack<float><<<blocks(nu, 256), 256, 0, st>>>((float*)c->f[c->cur], slots,
                                                            (const float*)c->halo_recv, nu);
  }
  CU(cudaPeekAtLastError());
  c->slab_phase = 0;
  return LBM_OK;
}

int lbm_slab_ccl_begin(lbm_ctx* c, int comp, int mark_lo, int mark_hi) {
  if (int rc = check_ctx(c)) return rc;
  if (!c->slab) return fail(LBM_EINVAL, "not a slab context");
  if (comp < 0 || comp > 1) return fail(LBM_EINVAL, "bad argument");
  if (c->slab_phase != 2)
    return fail(LBM_EINVAL, "slab context: lbm_slab_ccl_begin needs both lbm_slab_density parts and "
                            "the psi exchange on the current state");
  cudaStream_t st = use_stream(c);
  const int na = c->nact;
  int* parent = c->ccl;
  int* flag = parent + na;
  const int g = blocks(na, 256);
  if (c->bits == 64)
    k_ccl_init<double><<<g, 256, 0, st>>>((const Vec2<double>*)c->psi, na, comp, parent, flag);
  else
    k_ccl_init<float><<<g, 256, 0, st>>>((const Vec2<float>*)c->psi, na, comp, parent, flag);
  k_ccl_unite<<<g, 256, 0, st>>>(make_view(c), na, c->npad, parent);   // ids >= na (halo) are skipped
  k_ccl_flatten<<<g, 256, 0, st>>>(na, parent);
  const int a1 = mark_lo ? c->edge_plane[0] : 0, b0 = mark_hi ? na - c->edge_plane[1] : na;
  if (a1 + (na - b0) > 0)
    k_ccl_mark<<<blocks(a1 + (na - b0), 256), 256, 0, st>>>(parent, 0, a1, b0, na, flag);
  CU(cudaPeekAtLastError());
  c->ccl_comp = comp;
  return LBM_OK;
}

int lbm_slab_ccl_export(lbm_ctx* c) {
  if (int rc = check_ctx(c)) return rc;
  if (!c->slab || c->ccl_comp < 0) return fail(LBM_EINVAL, "no lbm_slab_ccl_begin on this context");
  cudaStream_t st = use_stream(c);
  const int na = c->nact;
  int* parent = c->ccl;
  int* flag = parent + na;
  int* planes = parent + (size_t)2 * na;
  CU(cudaMemsetAsync(planes, 0xff, (size_t)2 * c->np * sizeof(int), st));  // -1: nothing there
  if (c->edge_plane[0] > 0)
    k_ccl_export<<<blocks(c->edge_plane[0], 256), 256, 0, st>>>(parent, flag, c->node_vox_d, 0,
                                                                c->edge_plane[0], c->np, planes);
  if (c->edge_plane[1] > 0)
    k_ccl_export<<<blocks(c->edge_plane[1], 256), 256, 0, st>>>(
        parent, flag, c->node_vox_d, na - c->edge_plane[1], na, c->np, planes + c->np);
  CU(cudaPeekAtLastError());
  return LBM_OK;
}

int lbm_slab_ccl_import(lbm_ctx* c, int use_lo, int use_hi, int* changed) {
  if (int rc = check_ctx(c)) return rc;
  if (!changed) return fail(LBM_EINVAL, "NULL argument");
  if (!c->slab || c->ccl_comp < 0) return fail(LBM_EINVAL, "no lbm_slab_ccl_begin on this context");
  cudaStream_t st = use_stream(c);
  const int na = c->nact;
  int* parent = c->ccl;
  int* flag = parent + na;
  int* planes = parent + (size_t)2 * na;
  int* counter = planes + (size_t)4 * c->np;
  CU(cudaMemsetAsync(counter, 0, sizeof(int), st));
  if (use_lo && c->edge_plane[0] > 0)
    k_ccl_import<<<blocks(c->edge_plane[0], 256), 256, 0, st>>>(
        parent, flag, c->node_vox_d, 0, c->edge_plane[0], c->np, planes + (size_t)2 * c->np, counter);
  if (use_hi && c->edge_plane[1] > 0)
    k_ccl_import<<<blocks(c->edge_plane[1], 256), 256, 0, st>>>(
        parent, flag, c->node_vox_d, na - c->edge_plane[1], na, c->np, planes + (size_t)3 * c->np,
        counter);
  CU(cudaPeekAtLastError());
  int h = 0;
  CU(cudaMemcpyAsync(&h, counter, sizeof h, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  *changed = h;
  return LBM_OK;
}

int lbm_slab_ccl_finish(lbm_ctx* c, int z0, int z1, long long* nodes, double* mass) {
  if (int rc = check_ctx(c)) return rc;
  if (!nodes || !mass || z0 < 0 || z1 > c->nz || z0 > z1) return fail(LBM_EINVAL, "bad argument");
  if (!c->slab || c->ccl_comp < 0) return fail(LBM_EINVAL, "no lbm_slab_ccl_begin on this context");
  cudaStream_t st = use_stream(c);
  const int na = c->nact, comp = c->ccl_comp;
  int* parent = c->ccl;
  int* flag = parent + na;
  const int n0 = c->zstart[z0], n1 = c->zstart[z1];
  const int chunk = std::max(kCclBlock, (int)(((long long)(n1 - n0) + 1183) / 1184));
  const int nb = n1 > n0 ? blocks(n1 - n0, chunk) : 0;
  DevBuf tmp(((size_t)2 * nb + 2) * sizeof(double));
  if (!tmp.p) return fail(LBM_ENOMEM, "device allocation failed");
  double* partial = (double*)tmp.p;
  double* out = partial + (size_t)2 * nb;
  if (nb > 0) {
    if (c->bits == 64)
      k_ccl_count<double><<<nb, kCclBlock, 0, st>>>((const Vec2<double>*)c->psi, parent, flag, n0,
                                                    n1, comp, chunk, partial);
    else
      k_ccl_count<float><<<nb, kCclBlock, 0, st>>>((const Vec2<float>*)c->psi, parent, flag, n0, n1,
                                                   comp, chunk, partial);
  }
  k_sum_pairs<<<1, 32, 0, st>>>(partial, nb, out);
  CU(cudaPeekAtLastError());
  double h[2] = {0.0, 0.0};
  CU(cudaMemcpyAsync(h, out, sizeof h, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  *mass = h[0];
  *nodes = (long long)h[1];
  c->ccl_comp = -1;
  return LBM_OK;
}

extern "C++" {
// exchange buffer `which` of a slab context (include/lbm.h lbm_slab_buffer)
static void slab_buffer_of(lbm_ctx* c, int which, void** dev, long long* bytes) {
  if (which >= 8) {  // cluster-flag planes of the trapped-volume query: send low/high, receive low/high
    *dev = c->ccl + (size_t)2 * c->nact + (size_t)(which - 8) * c->np;
    *bytes = (long long)c->np * (long long)sizeof(int);
    return;
  }
  const size_t pair = 2 * c->esz;
  const int face = which & 1;
  switch (which >> 1) {
    case 0:  // psi of my two owned planes at that face
      *dev = (char*)c->psi + (size_t)c->psi_send[face][0] * pair;
      *bytes = c->psi_send[face][1] * (long long)pair;
      break;
    case 1:  // psi of my halo planes at that face
      *dev = (char*)c->psi + (size_t)c->psi_recv[face][0] * pair;
      *bytes = c->psi_recv[face][1] * (long long)pair;
      break;
    case 2:  // packed populations leaving through that face
      *dev = (char*)c->halo_send + (face ? (size_t)c->n_pack[0] * pair : 0);
      *bytes = c->n_pack[face] * (long long)pair;
      break;
    default:  // populations arriving through that face
      *dev = (char*)c->halo_recv + (face ? (size_t)c->n_unpack[0] * pair : 0);
      *bytes = c->n_unpack[face] * (long long)pair;
      break;
  }
}

#define NC(call)                                                                          \
  do {                                                                                    \
    ncclResult_t r_ = (call);                                                             \
    if (r_ != ncclSuccess)                                                                \
      return fail(LBM_ECUDA, "%s failed: %s (%s:%d)", #call, ncclGetErrorString(r_),      \
                  __FILE__, __LINE__);                                                    \
  } while (0)

// One neighbour exchange on the slab ring, enqueued on `cs`: kind 0 = psi planes (buffers 0,1 ->
// the neighbours' 2,3), kind 1 = populations that crossed a cut (4,5 -> 6,7).  My high-face
// message goes to rank+1 and lands in its low halo, my low-face message to rank-1 and lands in
// its high halo.  Posting order (send up, send down, receive from below, receive from above)
// keeps the two messages between the same pair of ranks matched at world sizes 1 and 2.  Empty
// messages (the ends of a z-open box) are skipped on both sides: the sizes derive from the same
// mask planes.
static int slab_exchange(lbm_ctx* c, int kind, cudaStream_t cs) {
  void* b[4];
  long long n[4];
  for (int k = 0; k < 4; ++k) slab_buffer_of(c, 4 * kind + k, &b[k], &n[k]);
  const int up = (c->comm_rank + 1) % c->comm_world;
  const int down = (c->comm_rank + c->comm_world - 1) % c->comm_world;
  if (n[0] + n[1] + n[2] + n[3] == 0) return LBM_OK;
  NC(ncclGroupStart());
  if (n[1]) NC(ncclSend(b[1], (size_t)n[1], ncclChar, up, c->comm, cs));
  if (n[0]) NC(ncclSend(b[0], (size_t)n[0], ncclChar, down, c->comm, cs));
  if (n[2]) NC(ncclRecv(b[2], (size_t)n[2], ncclChar, down, c->comm, cs));
  if (n[3]) NC(ncclRecv(b[3], (size_t)n[3], ncclChar, up, c->comm, cs));
  NC(ncclGroupEnd());
  return LBM_OK;
}

// One sharded time step with both exchanges beside the interior launches (the order of
// include/lbm.h "z-slab sharding"): st = compute stream, c->comm_stream = exchanges.
template <typename T>
static int slab_step_once(lbm_ctx* c, cudaStream_t st) {
  cudaStream_t cs = c->comm_stream;
  launch_density<T>(c, st, 0);
  CU(cudaEventRecord(c->comm_ev[0], st));
  CU(cudaStreamWaitEvent(cs, c->comm_ev[0], 0));
  if (int rc = slab_exchange(c, 0, cs)) return rc;
  CU(cudaEventRecord(c->comm_ev[1], cs));
  launch_density<T>(c, st, 1);
  CU(cudaStreamWaitEvent(st, c->comm_ev[1], 0));
  c->slab_phase = 2;
  if (int rc = slab_collide_T<T>(c, 0, st)) return rc;
  CU(cudaEventRecord(c->comm_ev[2], st));
  CU(cudaStreamWaitEvent(cs, c->comm_ev[2], 0));
  if (int rc = slab_exchange(c, 1, cs)) return rc;
  CU(cudaEventRecord(c->comm_ev[3], cs));
  if (int rc = slab_collide_T<T>(c, 1, st)) return rc;
  CU(cudaStreamWaitEvent(st, c->comm_ev[3], 0));
  c->slab_phase = 4;
  return LBM_OK;
}
}  // extern "C++"

int lbm_comm_unique_id(char id[LBM_COMM_ID_BYTES]) {
  if (!id) return fail(LBM_EINVAL, "NULL argument");
  static_assert(sizeof(ncclUniqueId) == LBM_COMM_ID_BYTES, "ncclUniqueId size");
  ncclUniqueId u;
  NC(ncclGetUniqueId(&u));
  std::memcpy(id, &u, sizeof u);
  return LBM_OK;
}

int lbm_slab_comm_init(lbm_ctx* c, const char id[LBM_COMM_ID_BYTES], int rank, int world) {
  if (int rc = check_ctx(c)) return rc;
  if (!c->slab) return fail(LBM_EINVAL, "not a slab context");
  if (!id || world < 1 || rank < 0 || rank >= world) return fail(LBM_EINVAL, "bad argument");
  if (c->comm) return fail(LBM_EINVAL, "the context already has a communicator");
  ncclUniqueId u;
  std::memcpy(&u, id, sizeof u);
  NC(ncclCommInitRank(&c->comm, world, u, rank));
  c->comm_rank = rank;
  c->comm_world = world;
  CU(cudaStreamCreateWithFlags(&c->comm_stream, cudaStreamNonBlocking));
  for (auto& e : c->comm_ev) CU(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  return LBM_OK;
}

int lbm_slab_step(lbm_ctx* c, int n) {
  if (int rc = check_ctx(c)) return rc;
  if (!c->slab) return fail(LBM_EINVAL, "not a slab context");
  if (!c->comm) return fail(LBM_EINVAL, "lbm_slab_step needs lbm_slab_comm_init");
  if (n < 0) return fail(LBM_EINVAL, "n must be >= 0");
  if (c->slab_phase > 2)
    return fail(LBM_EINVAL, "slab calls out of order (expected phase %d)", c->slab_phase);
  cudaStream_t st = use_stream(c);
  for (int it = 0; it < n; ++it) {
    if (int rc = c->bits == 64 ? slab_step_once<double>(c, st) : slab_step_once<float>(c, st))
      return rc;
    if (int rc = lbm_slab_unpack(c)) return rc;
  }
  return LBM_OK;
}

int lbm_slab_exchange(lbm_ctx* c, int kind) {
  if (int rc = check_ctx(c)) return rc;
  if (!c->slab) return fail(LBM_EINVAL, "not a slab context");
  if (!c->comm) return fail(LBM_EINVAL, "lbm_slab_exchange needs lbm_slab_comm_init");
  if (kind < 0 || kind > 2) return fail(LBM_EINVAL, "kind must be 0 (psi), 1 (populations) or 2 (cluster flags)");
  return slab_exchange(c, kind, use_stream(c));   // in line on the caller's stream
}

int lbm_slab_buffer(lbm_ctx* c, int which, void** dev, long long* bytes) {
  if (!c || !dev || !bytes) return fail(LBM_EINVAL, "NULL argument");
  if (!c->slab) return fail(LBM_EINVAL, "not a slab context");
  if (which < 0 || which > 11) return fail(LBM_EINVAL, "which must be 0..11");
  slab_buffer_of(c, which, dev, bytes);
  return LBM_OK;
}

void lbm_destroy(lbm_ctx* c) {
  if (!c) return;
  cudaSetDevice(c->device);
  // kernels of this context may be in flight on any stream it was used from: the buffers go back to
  // torch's caching allocator, which would hand them out again at once
  cudaDeviceSynchronize();
  delete c;
}

long long lbm_num_fluid(lbm_ctx* c) { return c ? c->nf : -1; }
long long lbm_num_wall_solid(lbm_ctx* c) { return c ? c->nw : -1; }

int lbm_memory_bytes(lbm_ctx* c, long long bytes[4]) {
  if (!c || !bytes) return fail(LBM_EINVAL, "NULL argument");
  for (int k = 0; k < 4; ++k) bytes[k] = c->bytes[k];
  return LBM_OK;
}

int lbm_set_boundary(lbm_ctx* c, double inlet_value, double outlet_rho) {
  if (!c) return fail(LBM_EINVAL, "NULL context");
  if (!c->p.z_open) return fail(LBM_EINVAL, "z is periodic: no boundary values to set");
  if (c->slab && c->slab_phase > 2)
    return fail(LBM_EINVAL, "slab context: lbm_set_boundary is not allowed inside a step");
  if (!std::isfinite(inlet_value) || !std::isfinite(outlet_rho))
    return fail(LBM_EINVAL, "boundary values must be finite");
  if (int rc = check_ctx(c)) return rc;
  apply_pending(c, use_stream(c));  // the last step's fix uses the values it was run with
  c->drop_graphs();                // the boundary values are kernel arguments
  if (c->p.inlet_kind == 1 || c->p.inlet_kind == 3) c->p.inlet_rho = inlet_value;
  else c->p.inlet_uz = inlet_value;
  c->p.outlet_rho = outlet_rho;
  return LBM_OK;
}

int lbm_sync(lbm_ctx* c) {
  if (int rc = check_ctx(c)) return rc;
  CU(cudaStreamSynchronize(use_stream(c)));
  return LBM_OK;
}

int lbm_step(lbm_ctx* c, int n) {
  if (int rc = check_ctx(c)) return rc;
  if (n < 0) return fail(LBM_EINVAL, "n must be >= 0");
  if (c->slab)
    return fail(LBM_EINVAL, "slab context: a step is lbm_slab_density, psi exchange, "
                            "lbm_slab_collide, population exchange, lbm_slab_unpack");
  cudaStream_t st = use_stream(c);
  if (c->prof) {
    for (auto& e : c->prof_events) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
    c->prof_events.clear();
  }
  c->prof_launches = 0;
  return c->bits == 64 ? step_graphed_T<double>(c, n, st) : step_graphed_T<float>(c, n, st);
}

int lbm_set_profiling(lbm_ctx* c, int on) {
  if (!c) return fail(LBM_EINVAL, "NULL context");
  c->prof = on != 0;
  for (auto& e : c->prof_events) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
  c->prof_events.clear();  // slab phases accumulate from here on; lbm_step restarts per call
  c->prof_launches = 0;
  return LBM_OK;
}

int lbm_last_step_profile(lbm_ctx* c, double ms[4], long long* launches) {
  if (int rc = check_ctx(c)) return rc;
  if (!ms || !launches) return fail(LBM_EINVAL, "NULL argument");
  CU(cudaStreamSynchronize(use_stream(c)));
  for (int k = 0; k < 4; ++k) ms[k] = 0.0;
  for (auto& e : c->prof_events) {
    float t = 0.f;
    CU(cudaEventElapsedTime(&t, e.a, e.b));
    ms[e.kind] += t;
  }
  *launches = c->prof_launches;
  return LBM_OK;
}

int lbm_set_density(lbm_ctx* c, const double* rhoA, const double* rhoB) {
  if (int rc = check_ctx(c)) return rc;
  if (!rhoA || !rhoB) return fail(LBM_EINVAL, "NULL argument");
  cudaStream_t st = use_stream(c);
  c->open_pending = false;  // the whole state is replaced
  const size_t bytes = (size_t)c->nvox * sizeof(double);
  DevBuf a(bytes), b(bytes);
  if (!a.p || !b.p) return fail(LBM_ENOMEM, "device staging allocation failed");
  CU(cudaMemcpyAsync(a.p, rhoA, bytes, cudaMemcpyHostToDevice, st));
  CU(cudaMemcpyAsync(b.p, rhoB, bytes, cudaMemcpyHostToDevice, st));
  if (c->bits == 64)
    k_init_density<double><<<blocks(c->nf, 256), 256, 0, st>>>(
        (const double*)a.p, (const double*)b.p, c->node_vox_d, (double*)c->f[c->cur], c->nf, c->npad);
  else
    k_init_density<float><<<blocks(c->nf, 256), 256, 0, st>>>(
        (const double*)a.p, (const double*)b.p, c->node_vox_d, (float*)c->f[c->cur], c->nf, c->npad);
  CU(cudaPeekAtLastError());
  for (int s = 0; s < 2; ++s)
    if (int rc = c->bits == 64 ? record_frozen_T<double>(c, s, st) : record_frozen_T<float>(c, s, st))
      return rc;
  CU(cudaStreamSynchronize(st));
  return LBM_OK;
}

int lbm_set_populations(lbm_ctx* c, int comp, const double* f) {
  if (int rc = check_ctx(c)) return rc;
  if (!f || comp < 0 || comp > 1) return fail(LBM_EINVAL, "bad argument");
  cudaStream_t st = use_stream(c);
  apply_pending(c, st);  // the other component keeps its (completed) state
  const size_t bytes = (size_t)c->nvox * sizeof(double);
  DevBuf d(bytes);
  if (!d.p) return fail(LBM_ENOMEM, "device staging allocation failed");
  for (int i = 0; i < Q; ++i) {
    CU(cudaMemcpyAsync(d.p, f + (size_t)i * c->nvox, bytes, cudaMemcpyHostToDevice, st));
    const size_t row = pidx(comp, i, 0, c->npad);  // element stride 2: components are interleaved
    if (c->bits == 64)
      k_dense_to_compact<double><<<blocks(c->nf, 256), 256, 0, st>>>(
          (const double*)d.p, c->node_vox_d, (double*)c->f[c->cur] + row, c->nf, 2);
    else
      k_dense_to_compact<float><<<blocks(c->nf, 256), 256, 0, st>>>(
          (const double*)d.p, c->node_vox_d, (float*)c->f[c->cur] + row, c->nf, 2);
    CU(cudaStreamSynchronize(st));  // pageable source: keep the staging buffer reuse ordered
  }
  CU(cudaPeekAtLastError());
  if (int rc = c->bits == 64 ? record_frozen_T<double>(c, comp, st)
                             : record_frozen_T<float>(c, comp, st))
    return rc;
  CU(cudaStreamSynchronize(st));
  return LBM_OK;
}

int lbm_get_populations(lbm_ctx* c, int comp, double* f) {
  if (int rc = check_ctx(c)) return rc;
  if (!f || comp < 0 || comp > 1) return fail(LBM_EINVAL, "bad argument");
  cudaStream_t st = use_stream(c);
  apply_pending(c, st);
  const size_t bytes = (size_t)c->nvox * sizeof(double);
  DevBuf d(bytes);
  if (!d.p) return fail(LBM_ENOMEM, "device staging allocation failed");
  for (int i = 0; i < Q; ++i) {
    CU(cudaMemsetAsync(d.p, 0, bytes, st));
    const size_t row = pidx(comp, i, 0, c->npad);  // element stride 2: components are interleaved
    if (c->bits == 64)
      k_compact_to_dense<double><<<blocks(c->nf, 256), 256, 0, st>>>(
          (const double*)c->f[c->cur] + row, c->node_vox_d, (double*)d.p, c->nf, 2);
    else
      k_compact_to_dense<float><<<blocks(c->nf, 256), 256, 0, st>>>(
          (const float*)c->f[c->cur] + row, c->node_vox_d, (double*)d.p, c->nf, 2);
    CU(cudaMemcpyAsync(f + (size_t)i * c->nvox, d.p, bytes, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
  }
  return LBM_OK;
}

int lbm_get_macroscopic(lbm_ctx* c, double* rhoA, double* rhoB, double* ux, double* uy,
                        double* uz, double* P) {
  if (int rc = check_ctx(c)) return rc;
  if (c->slab && c->slab_phase != 2)
    return fail(LBM_EINVAL, "slab context: lbm_get_macroscopic needs both lbm_slab_density parts "
                            "and the psi exchange on the current state");
  cudaStream_t st = use_stream(c);
  const int na = c->nact;  // owned nodes (all fluid nodes unless slab mode)
  DevBuf m((size_t)6 * na * sizeof(double));
  const size_t bytes = (size_t)c->nvox * sizeof(double);
  DevBuf d(bytes);
  if (!m.p || !d.p) return fail(LBM_ENOMEM, "device staging allocation failed");
  {
  ProfOff guard(c);
  if (c->bits == 64) {
    launch_psi<double>(c, st);
    k_macroscopic<double><<<blocks(na, 256), 256, 0, st>>>(
        (const double*)c->f[c->cur], (const Vec2<double>*)c->psi, make_view(c), (double*)m.p, na,
        c->npad, make_consts<double>(c->p));
  } else {
    launch_psi<float>(c, st);
    k_macroscopic<float><<<blocks(na, 256), 256, 0, st>>>(
        (const float*)c->f[c->cur], (const Vec2<float>*)c->psi, make_view(c), (double*)m.p, na,
        c->npad, make_consts<float>(c->p));
  }
  }
  CU(cudaPeekAtLastError());
  double* outs[6] = {rhoA, rhoB, ux, uy, uz, P};
  for (int q = 0; q < 6; ++q) {
    if (!outs[q]) continue;
    CU(cudaMemsetAsync(d.p, 0, bytes, st));
    k_compact_to_dense<double><<<blocks(na, 256), 256, 0, st>>>(
        (const double*)m.p + (size_t)q * na, c->node_vox_d, (double*)d.p, na, 1);
    CU(cudaMemcpyAsync(outs[q], d.p, bytes, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
  }
  CU(cudaStreamSynchronize(st));
  return LBM_OK;
}

int lbm_diagnostics(lbm_ctx* c, double mass[2], double momentum[3]) {
  if (int rc = check_ctx(c)) return rc;
  if (!mass || !momentum) return fail(LBM_EINVAL, "NULL argument");
  cudaStream_t st = use_stream(c);
  apply_pending(c, st);
  const int nb = c->diag_blocks;
  if (c->bits == 64)
    k_diag_partial<double><<<nb, kDiagBlock, 0, st>>>((const double*)c->f[c->cur], c->partial,
                                                      c->nact, c->npad);
  else
    k_diag_partial<float><<<nb, kDiagBlock, 0, st>>>((const float*)c->f[c->cur], c->partial, c->nact,
                                                     c->npad);
  k_diag_final<<<1, 32, 0, st>>>(c->partial, c->diag_out, nb);
  CU(cudaPeekAtLastError());
  double h[kDiagVals];
  CU(cudaMemcpyAsync(h, c->diag_out, sizeof h, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  mass[0] = h[0]; mass[1] = h[1];
  momentum[0] = h[2]; momentum[1] = h[3]; momentum[2] = h[4];
  if (h[5] != 0.0 || !std::isfinite(h[0]) || !std::isfinite(h[1]))
    return fail(LBM_ENONFINITE, "non-finite populations detected");
  return LBM_OK;
}

int lbm_saturation(lbm_ctx* c, int comp, int z0, int z1, double* S) {
  if (int rc = check_ctx(c)) return rc;
  if (c->slab && c->slab_phase != 2)
    return fail(LBM_EINVAL, "slab context: lbm_saturation needs both lbm_slab_density parts and the psi "
                            "exchange on the current state");
  if (!S || comp < 0 || comp > 1 || z0 < 0 || z1 > c->nz || z0 >= z1)
    return fail(LBM_EINVAL, "bad argument");
  const int n0 = c->zstart[z0], n1 = c->zstart[z1];
  if (n1 <= n0) return fail(LBM_ENOFLUID, "no fluid node in the z-range");
  cudaStream_t st = use_stream(c);
  ProfOff guard(c);
  unsigned long long* cnt = (unsigned long long*)(c->diag_out + 7);
  CU(cudaMemsetAsync(cnt, 0, sizeof(unsigned long long), st));
  if (c->bits == 64) {
    launch_psi<double>(c, st);
    k_count_phase<double><<<blocks(n1 - n0, 256), 256, 0, st>>>((const Vec2<double>*)c->psi, n0,
                                                                n1, comp, cnt);
  } else {
    launch_psi<float>(c, st);
    k_count_phase<float><<<blocks(n1 - n0, 256), 256, 0, st>>>((const Vec2<float>*)c->psi, n0, n1,
                                                               comp, cnt);
  }
  CU(cudaPeekAtLastError());
  unsigned long long h = 0;
  CU(cudaMemcpyAsync(&h, cnt, sizeof h, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  *S = (double)h / (double)(n1 - n0);
  return LBM_OK;
}

int lbm_trapped_volume(lbm_ctx* c, int comp, int z0, int z1, long long* nodes, double* mass) {
  if (int rc = check_ctx(c)) return rc;
  if (c->slab) return fail(LBM_EINVAL, "lbm_trapped_volume is not available on a slab context");
  if (!nodes || !mass || comp < 0 || comp > 1 || z0 < 0 || z1 > c->nz || z0 >= z1)
    return fail(LBM_EINVAL, "bad argument");
  cudaStream_t st = use_stream(c);
  {
    ProfOff guard(c);
    if (c->bits == 64) launch_psi<double>(c, st); else launch_psi<float>(c, st);
  }
  CU(cudaPeekAtLastError());
  const int nf = c->nf, nz = c->nz;
  const int n0 = c->zstart[z0], n1 = c->zstart[z1];
  // scratch: parent[nf], flag[nf] (int32), per-block partials and the two results (double)
  const int chunk = std::max(kCclBlock, (int)(((long long)(n1 - n0) + 1183) / 1184));
  const int nb = n1 > n0 ? blocks(n1 - n0, chunk) : 0;
  const size_t ints = ((size_t)2 * nf + 1) & ~(size_t)1;
  DevBuf tmp(ints * sizeof(int) + ((size_t)2 * nb + 2) * sizeof(double));
  if (!tmp.p) return fail(LBM_ENOMEM, "device allocation failed");
  int* parent = (int*)tmp.p;
  int* flag = parent + nf;
  double* partial = (double*)(parent + ints);
  double* out = partial + (size_t)2 * nb;
  const int g = blocks(nf, 256);
  if (c->bits == 64)
    k_ccl_init<double><<<g, 256, 0, st>>>((const Vec2<double>*)c->psi, nf, comp, parent, flag);
  else
    k_ccl_init<float><<<g, 256, 0, st>>>((const Vec2<float>*)c->psi, nf, comp, parent, flag);
  k_ccl_unite<<<g, 256, 0, st>>>(make_view(c), nf, c->npad, parent);
  k_ccl_flatten<<<g, 256, 0, st>>>(nf, parent);
  const int a0 = c->zstart[0], a1 = c->zstart[1], b0 = c->zstart[nz - 1], b1 = c->zstart[nz];
  if ((a1 - a0) + (b1 - b0) > 0)
    k_ccl_mark<<<blocks((a1 - a0) + (b1 - b0), 256), 256, 0, st>>>(parent, a0, a1, b0, b1, flag);
  if (nb > 0) {
    if (c->bits == 64)
      k_ccl_count<double><<<nb, kCclBlock, 0, st>>>((const Vec2<double>*)c->psi, parent, flag, n0,
                                                    n1, comp, chunk, partial);
    else
      k_ccl_count<float><<<nb, kCclBlock, 0, st>>>((const Vec2<float>*)c->psi, parent, flag, n0, n1,
                                                   comp, chunk, partial);
  }
  k_sum_pairs<<<1, 32, 0, st>>>(partial, nb, out);
  CU(cudaPeekAtLastError());
  double h[2] = {0.0, 0.0};
  CU(cudaMemcpyAsync(h, out, sizeof h, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  *mass = h[0];
  *nodes = (long long)h[1];
  return LBM_OK;
}

// ---- lbm_trapped_volume_static: the trapped-volume query without any allocation ---------------
// Scratch of the union-find kernels (parent[nf] | flag[nf] int32, then 2 * blocks + 2 doubles of
// partial sums) in a file-scope device array instead of a buffer from the caching allocator, for
// callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid
// cudaMalloc).  Every GPU that loads the library holds the array (8 MiB + 19 KB) until exit.
// In HOST code the array's name is a host-side stand-in, not a device address: the kernels get
// the address cudaGetSymbolAddress returns, looked up once per device with that device current.
constexpr long long kStaticMaxNodes = LBM_STATIC_MAX_NODES;
constexpr int kStaticMaxBlocks = 1184;   // blocks of k_ccl_count: 8 per SM x 148
constexpr size_t kStaticScratchBytes =
    (size_t)kStaticMaxNodes * 2 * sizeof(int) + ((size_t)2 * kStaticMaxBlocks + 2) * sizeof(double);
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

int lbm_trapped_volume_static(lbm_ctx* c, int comp, int z0, int z1, long long* nodes,
                              double* mass) {
  if (int rc = check_ctx(c)) return rc;   // makes the context's device current
  if (c->slab) return fail(LBM_EINVAL, "lbm_trapped_volume_static is not available on a slab context");
  if (!nodes || !mass || comp < 0 || comp > 1 || z0 < 0 || z1 > c->nz || z0 >= z1)
    return fail(LBM_EINVAL, "bad argument");
  if ((long long)c->nf > kStaticMaxNodes)
    return fail(LBM_EINVAL,
                "lbm_trapped_volume_static: the box has %d fluid nodes, the static scratch serves at "
                "most LBM_STATIC_MAX_NODES = %lld; use lbm_trapped_volume",
                c->nf, kStaticMaxNodes);
  // device address of g_static_scratch: looked up once per device, with that device current
  static void* scratch_of_device[64] = {};
  void* scratch = c->device < 64 ? scratch_of_device[c->device] : nullptr;
  if (!scratch) {
    CU(cudaGetSymbolAddress(&scratch, g_static_scratch));
    if (!scratch) return fail(LBM_ECUDA, "cudaGetSymbolAddress returned a null address");
    if (c->device < 64) scratch_of_device[c->device] = scratch;
  }
  cudaStream_t st = use_stream(c);
  {
    ProfOff guard(c);
    if (c->bits == 64) launch_psi<double>(c, st); else launch_psi<float>(c, st);
  }
  CU(cudaPeekAtLastError());
  const int nf = c->nf, nz = c->nz;
  const int n0 = c->zstart[z0], n1 = c->zstart[z1];
  const int chunk = std::max(kCclBlock, (int)(((long long)(n1 - n0) + kStaticMaxBlocks - 1) / kStaticMaxBlocks));
  const int nb = n1 > n0 ? blocks(n1 - n0, chunk) : 0;   // <= kStaticMaxBlocks
  const size_t ints = ((size_t)2 * nf + 1) & ~(size_t)1;
  // The array keeps the previous call's contents.  Nothing has to be cleared: k_ccl_init writes
  // parent[n] and flag[n] of every node before anything reads them, k_ccl_count every partial it
  // is summed from, k_sum_pairs both results.
  int* parent = (int*)scratch;
  int* flag = parent + nf;
  double* partial = (double*)(parent + ints);
  double* out = partial + (size_t)2 * nb;
  const int g = blocks(nf, 256);
  if (c->bits == 64)
    k_ccl_init<double><<<g, 256, 0, st>>>((const Vec2<double>*)c->psi, nf, comp, parent, flag);
  else
    k_ccl_init<float><<<g, 256, 0, st>>>((const Vec2<float>*)c->psi, nf, comp, parent, flag);
  k_ccl_unite<<<g, 256, 0, st>>>(make_view(c), nf, c->npad, parent);
  k_ccl_flatten<<<g, 256, 0, st>>>(nf, parent);
  const int a0 = c->zstart[0], a1 = c->zstart[1], b0 = c->zstart[nz - 1], b1 = c->zstart[nz];
  if ((a1 - a0) + (b1 - b0) > 0)
    k_ccl_mark<<<blocks((a1 - a0) + (b1 - b0), 256), 256, 0, st>>>(parent, a0, a1, b0, b1, flag);
  if (nb > 0) {
    if (c->bits == 64)
      k_ccl_count<double><<<nb, kCclBlock, 0, st>>>((const Vec2<double>*)c->psi, parent, flag, n0,
                                                    n1, comp, chunk, partial);
    else
      k_ccl_count<float><<<nb, kCclBlock, 0, st>>>((const Vec2<float>*)c->psi, parent, flag, n0, n1,
                                                   comp, chunk, partial);
  }
  k_sum_pairs<<<1, 32, 0, st>>>(partial, nb, out);
  CU(cudaPeekAtLastError());
  double h[2] = {0.0, 0.0};
  CU(cudaMemcpyAsync(h, out, sizeof h, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  *mass = h[0];
  *nodes = (long long)h[1];
  return LBM_OK;
}

int lbm_mean_pressure(lbm_ctx* c, int z0, int z1, double* P) {
  if (int rc = check_ctx(c)) return rc;
  if (c->slab && c->slab_phase != 2)
    return fail(LBM_EINVAL, "slab context: lbm_mean_pressure needs both lbm_slab_density parts and the psi "
                            "exchange on the current state");
  if (!P || z0 < 0 || z1 > c->nz || z0 >= z1) return fail(LBM_EINVAL, "bad argument");
  const int n0 = c->zstart[z0], n1 = c->zstart[z1];
  if (n1 <= n0) return fail(LBM_ENOFLUID, "no fluid node in the z-range");
  cudaStream_t st = use_stream(c);
  {
    ProfOff guard(c);
    if (c->bits == 64) launch_psi<double>(c, st); else launch_psi<float>(c, st);
  }
  CU(cudaPeekAtLastError());
  const int chunk = std::max(kCclBlock, (int)(((long long)(n1 - n0) + 1183) / 1184));
  const int nb = blocks(n1 - n0, chunk);
  DevBuf tmp(((size_t)2 * nb + 2) * sizeof(double));
  if (!tmp.p) return fail(LBM_ENOMEM, "device allocation failed");
  double* partial = (double*)tmp.p;
  double* out = partial + (size_t)2 * nb;
  if (c->bits == 64)
    k_pressure_sum<double><<<nb, kCclBlock, 0, st>>>((const Vec2<double>*)c->psi, n0, n1, c->p.G,
                                                     chunk, partial);
  else
    k_pressure_sum<float><<<nb, kCclBlock, 0, st>>>((const Vec2<float>*)c->psi, n0, n1,
                                                    (float)c->p.G, chunk, partial);
  k_sum_pairs<<<1, 32, 0, st>>>(partial, nb, out);
  CU(cudaPeekAtLastError());
  double h[2] = {0.0, 0.0};
  CU(cudaMemcpyAsync(h, out, sizeof h, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  *P = h[0] / h[1];
  return LBM_OK;
}

}  // extern "C"
