// kernels.cuh -- sm_100a kernels of the two-component D3Q19 pseudopotential LBM step.
// Product code: written from PAPER.md (arXiv 2207.01534) Eq. (1)-(15); shares nothing with
// oracle/.  Layout and byte counts: DESIGN.md "Data layout in HBM" and "Kernels".
//
// Storage (T = float or double):
//   f   [19 dirs][npad][2 comps]   populations at time t (post-streaming): the two components of a
//                                  population are adjacent (one 8-byte pair in fp32), node id next
//   psi [npad + nwpad] of Vec2<T>  (rho_A, rho_B) at fluid id n; (rho~_A, rho~_B) of wall solid w at
//                                  npad + w (both parts start on a tile boundary)
//   nbr [18][npad] int32           psi index of x+e_i: < nf fluid id; >= npad wall solid;
//                                  -(m+1) beyond an open plane, m = mirror node (see geometry.hpp)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace lbmk {

constexpr int Q = 19;

// D3Q19 in the canonical order of include/lbm.h (reading R1 of PAPER.md L65-67).
__host__ __device__ constexpr int ex(int i) {
  constexpr int t[Q] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
  return t[i];
}
__host__ __device__ constexpr int ey(int i) {
  constexpr int t[Q] = {0, 0, 0, 1, -1, 0, 0, 1, 1, -1, -1, 0, 0, 0, 0, 1, -1, 1, -1};
  return t[i];
}
__host__ __device__ constexpr int ez(int i) {
  constexpr int t[Q] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, 1, -1, -1, 1, 1, -1, -1};
  return t[i];
}
__host__ __device__ constexpr int opp(int i) {
  constexpr int t[Q] = {0, 2, 1, 4, 3, 6, 5, 10, 9, 8, 7, 14, 13, 12, 11, 18, 17, 16, 15};
  return t[i];
}
// w_i
template <typename T>
__host__ __device__ constexpr T wgt(int i) {
  return i == 0 ? T(1.0 / 3.0) : (i < 7 ? T(1.0 / 18.0) : T(1.0 / 36.0));
}
// the 5 directions with e_z = +1 (inward at the inlet) and with e_z = -1 (inward at the outlet)
__host__ __device__ constexpr int inward(int plane, int k) {
  constexpr int t[2][5] = {{5, 11, 12, 15, 16}, {6, 13, 14, 17, 18}};
  return t[plane][k];
}

// index of population (component s, direction i, node n) in f
__host__ __device__ __forceinline__ size_t pidx(int s, int i, size_t n, size_t npad) {
  return ((size_t)i * npad + n) * 2 + (size_t)s;
}

// Programmatic dependent launch: a kernel launched with the stream-serialization attribute may
// begin while the previous kernel of the stream drains; everything that reads what that kernel
// (or, transitively, an earlier one) wrote must come after this wait.  A no-op otherwise.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
// Lets the next kernel's blocks become resident (and run up to their pdl_wait) already now.
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;"); }

// L2 eviction priority of a store: lines written with evict_last outlive the streaming traffic
// around them.  psi (8 B per node, written by the density and wall passes, gathered 19 times by
// the fused pass, rewritten every step) then never leaves L2 when it fits; `frac` is the share of
// the lines that gets the priority (chosen by address, the same lines every step), 0 = plain store.
__device__ __forceinline__ uint64_t l2_keep_policy(float frac) {
  uint64_t pol = 0;
  if (frac > 0.f)
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, %1;" : "=l"(pol) : "f"(frac));
  return pol;
}

template <typename T> struct Vec2;
template <> struct __align__(8) Vec2<float> { float a, b; };
template <> struct __align__(16) Vec2<double> { double a, b; };
// pol == 0: plain store
__device__ __forceinline__ void store_vec2(Vec2<float>* p, Vec2<float> v, uint64_t pol) {
  if (pol == 0) { *p = v; return; }
  asm volatile("st.global.L2::cache_hint.v2.f32 [%0], {%1, %2}, %3;" ::"l"(p), "f"(v.a), "f"(v.b),
               "l"(pol)
               : "memory");
}
__device__ __forceinline__ void store_vec2(Vec2<double>* p, Vec2<double> v, uint64_t pol) {
  if (pol == 0) { *p = v; return; }
  asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(p), "d"(v.a), "d"(v.b),
               "l"(pol)
               : "memory");
}

// Explicitly rounded scalar operations.  The same device function is inlined into several kernels
// (the open-plane fix runs in k_open_planes and k_density_open; the tile function in the fp32 and
// fp64 fused passes of every index form); left to the compiler, whether a*b+c becomes one FMA or a
// multiply and an add depends on the surrounding code, and the kernels would differ in the last
// bit.  Every product-sum of such shared code is therefore spelled out.
__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ float add_rn(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ double add_rn(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ float fma_rn(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ double fma_rn(double a, double b, double c) { return __fma_rn(a, b, c); }

template <typename T>
struct Consts {
  T G;            // G_coh, Eq. (11)/(13)
  T tauA, tauB;   // Eq. (7)
  T gx, gy, gz;   // body acceleration (R8)
  T hf;           // 0.5 (reading R3) or 0 (literal Eq. 4)
  T chiA, chiB;   // 1+xi, 1-xi
};

// ---------------------------------------------------------------------------------------------
// a1  density / psi pass: rho_sigma = sum_i f_i^sigma (Eq. 3); psi = rho (L105).
// One thread per fluid node; every load is a fully coalesced row read.
// Node range of a launch: blocks [0, split) take ids from a0 on, the remaining blocks from a1 on
// (whole pass: a0 = 0, split = grid; slab mode launches the two boundary id ranges first and the
// interior separately, so that the psi halo exchange overlaps the interior; a0, a1 are multiples
// of the block size, which keeps every warp's loads line-aligned).
struct NodeRange {
  int a0, split, a1;
  int nend;   // ids >= nend are not processed
};
template <typename T>
__global__ void __launch_bounds__(256) k_density(const T* __restrict__ f, Vec2<T>* __restrict__ psi,
                                                 NodeRange r, size_t npad, float keep_psi) {
  const int b = (int)blockIdx.x;
  const int n = (b < r.split ? r.a0 + b * (int)blockDim.x : r.a1 + (b - r.split) * (int)blockDim.x) +
                (int)threadIdx.x;
  pdl_wait();  // f was written by the previous step's fused pass
  if (n >= r.nend) return;
  const Vec2<T>* f2 = reinterpret_cast<const Vec2<T>*>(f);
  Vec2<T> v[Q];
#pragma unroll
  for (int i = 0; i < Q; ++i) v[i] = f2[(size_t)i * npad + n];
  T ra = v[0].a, rb = v[0].b;
#pragma unroll
  for (int i = 1; i < Q; ++i) { ra += v[i].a; rb += v[i].b; }
  Vec2<T> o; o.a = ra; o.b = rb;
  store_vec2(psi + n, o, l2_keep_policy(keep_psi));
}

// ---------------------------------------------------------------------------------------------
// a2  virtual solid density on wall solids (improved virtual solid density scheme):
//   rho~_sigma(x) = chi_sigma * sum_i w_i rho_sigma(x+e_i)(1-phi(x+e_i)) / sum_i w_i (1-phi)
// Eq. (14)-(15) PAPER.md L128-133; chi: L141-143.  wall_nbr < 0 means "not fluid".
template <typename T>
__global__ void __launch_bounds__(256) k_wallpsi(Vec2<T>* __restrict__ psi,
                                                 const int* __restrict__ wall_nbr,
                                                 const T* __restrict__ inv_den,
                                                 size_t wall_base, int nw, size_t nwpad, T chiA,
                                                 T chiB, float keep_psi) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  const bool live = w < nw;
  int id[Q];
#pragma unroll
  for (int i = 1; i < Q; ++i) id[i] = live ? wall_nbr[(size_t)(i - 1) * nwpad + w] : -1;
  const T s = live ? inv_den[w] : T(0);
  pdl_wait();  // the index is static; psi comes from the density pass
  // From here on the density pass is complete and visible, so the fused pass may move in beside
  // this latency-bound kernel and stage its first tiles (populations, index) before its own wait
  // (measured: 0.3861 -> 0.3845 ms per step on config 4; the same trigger in the density pass is
  // neutral, in the fused pass it costs 8 %: early density blocks take its registers).
  pdl_trigger();
  if (!live) return;
  T na = T(0), nb = T(0);
#pragma unroll
  for (int i = 1; i < Q; ++i) {
    if (id[i] >= 0) {
      const Vec2<T> p = psi[id[i]];
      na = fma_rn(wgt<T>(i), p.a, na);
      nb = fma_rn(wgt<T>(i), p.b, nb);
    }
  }
  Vec2<T> o; o.a = mul_rn(mul_rn(chiA, na), s); o.b = mul_rn(mul_rn(chiB, nb), s);
  // wall ids are stored at wall_base = npad (tile-aligned)
  store_vec2(psi + wall_base + w, o, l2_keep_policy(keep_psi));
}

// ---------------------------------------------------------------------------------------------
// Per-node mixture quantities shared by the collide kernel and the macroscopic getter.
// a3: F_sigma = -G rho_sigma sum_i w_i Psi_sigmabar(x+e_i) e_i + rho_sigma g
//     (Eq. 10, 11, 13; one combined 18-term sum, reading R6)
// a4: rho = rho_A + rho_B; tau_s = (rho_A tau_A + rho_B tau_B)/rho (Eq. 5-7, R2);
//     u_eq = (sum_sigma sum_i e_i f_i + hf * sum_sigma F_sigma)/rho (Eq. 8, R3, R4)
template <typename T>
struct NodeState {
  T rhoA, rhoB;
  T FA[3], FB[3];
  T u[3];
  T om;  // 1/tau_s
};

template <typename T>
__device__ __forceinline__ void gather_force_sums(const Vec2<T>* __restrict__ psi,
                                                  const int (&id)[Q], T (&SA)[3], T (&SB)[3]) {
  // axis neighbours (w = 1/18) and diagonal neighbours (w = 1/36) summed separately
  T a1[3] = {T(0), T(0), T(0)}, b1[3] = {T(0), T(0), T(0)};
  T a2[3] = {T(0), T(0), T(0)}, b2[3] = {T(0), T(0), T(0)};
#pragma unroll
  for (int i = 1; i < Q; ++i) {
    const int k = id[i] >= 0 ? id[i] : -id[i] - 1;  // mirror node beyond an open plane (R12 iv)
    const Vec2<T> p = psi[k];
    if (i < 7) {
      if (ex(i)) { a1[0] += T(ex(i)) * p.a; b1[0] += T(ex(i)) * p.b; }
      if (ey(i)) { a1[1] += T(ey(i)) * p.a; b1[1] += T(ey(i)) * p.b; }
      if (ez(i)) { a1[2] += T(ez(i)) * p.a; b1[2] += T(ez(i)) * p.b; }
    } else {
      if (ex(i)) { a2[0] += T(ex(i)) * p.a; b2[0] += T(ex(i)) * p.b; }
      if (ey(i)) { a2[1] += T(ey(i)) * p.a; b2[1] += T(ey(i)) * p.b; }
      if (ez(i)) { a2[2] += T(ez(i)) * p.a; b2[2] += T(ez(i)) * p.b; }
    }
  }
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    SA[d] = wgt<T>(1) * a1[d] + wgt<T>(7) * a2[d];
    SB[d] = wgt<T>(1) * b1[d] + wgt<T>(7) * b2[d];
  }
}

template <typename T>
__device__ __forceinline__ void node_state(const T (&fa)[Q], const T (&fb)[Q],
                                           const Vec2<T>* __restrict__ psi, const int (&id)[Q],
                                           const Consts<T>& c, NodeState<T>& s) {
  T ra = fa[0], rb = fb[0];
  T j[3] = {T(0), T(0), T(0)};
#pragma unroll
  for (int i = 1; i < Q; ++i) {
    ra += fa[i];
    rb += fb[i];
    const T t = fa[i] + fb[i];
    if (ex(i)) j[0] += T(ex(i)) * t;
    if (ey(i)) j[1] += T(ey(i)) * t;
    if (ez(i)) j[2] += T(ez(i)) * t;
  }
  T SA[3], SB[3];
  gather_force_sums<T>(psi, id, SA, SB);
  const T g[3] = {c.gx, c.gy, c.gz};
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    s.FA[d] = -c.G * ra * SB[d] + ra * g[d];
    s.FB[d] = -c.G * rb * SA[d] + rb * g[d];
  }
  const T inv = T(1) / (ra + rb);
#pragma unroll
  for (int d = 0; d < 3; ++d) s.u[d] = (j[d] + c.hf * (s.FA[d] + s.FB[d])) * inv;
  s.om = (ra + rb) / (ra * c.tauA + rb * c.tauB);
  s.rhoA = ra;
  s.rhoB = rb;
}

// ---------------------------------------------------------------------------------------------
// a3-a6 fused: forces, tau_s/u_eq, collision, push-streaming with halfway bounce-back.
//   f*_i = f_i - (f_i - feq_i)/tau_s + (1 - 1/(2 tau_s)) S_i                     Eq. (1)
//   feq_i = w_i rho_sigma [1 + 3 e.u + 4.5 (e.u)^2 - 1.5 u.u]                     Eq. (2)
//   S_i  = w_i [3 (e_i - u).F_sigma + 9 (e_i.u)(e_i.F_sigma)]                     Eq. (9)
//   f_i(x+e_i, t+1) = f*_i(x,t);  x+e_i solid -> f_opp(i)(x, t+1) = f*_i(x,t)     L191, L215 (R10)
// REMAINDER (fp32 build): the rest population is written as rho_sigma - sum_{i>=1} f*_i, which
// equals Eq. (1) for i=0 exactly in exact arithmetic (sum_i feq = rho, sum_i S_i = 0) and removes
// the 1.5e-8-per-step mass drift that the fp32-rounded weights (sum = 1 + 1.49e-8) would inject
// (DESIGN.md "fp32 build").
// (the formulas above are implemented by collide_tile_thread below)

// ---------------------------------------------------------------------------------------------
// Bulk-async (TMA engine) staging for the fused pass.  One CTA owns a tile of TN consecutive
// node ids; its 38 population rows and 18 neighbour-index rows are TN-element contiguous,
// 16-byte-aligned segments of the SoA arrays, so the whole tile arrives in shared memory through
// 56 cp.async.bulk copies (SASS UBLKCP) that complete on one mbarrier.  Registers then hold only
// the working set, so several CTAs per SM keep >100 KB of loads in flight per SM with no
// register cost -- what the one-node-per-thread register version (167 registers, 12 % occupancy,
// 34 % of HBM peak; profiles/r1_v1_collide.md) could not do.
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
               "r"(bytes)
               : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
// Warp-uniform wait: lane 0 polls, the result is broadcast with a shuffle, so the spin loop's
// exit condition is a warp-uniform value.  (A spin whose exit depends on a per-thread asm result
// makes ptxas treat everything after it as divergent: it then re-materialises the global-memory
// descriptor with an R2UR pair in front of every load/store -- ~100 extra XU-pipe instructions per
// thread, measured in profiles/r1_v2_collide.md.)  Must be called by all 32 lanes of a warp.
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  const bool leader = (threadIdx.x & 31) == 0;
  while (true) {
    uint32_t ok = 0;
    if (leader) ok = mbar_try_wait(bar, parity) ? 1u : 0u;
    if (__shfl_sync(0xffffffffu, ok, 0)) break;
  }
}
// One lane of a converged warp, chosen by hardware (elect.sync): the compiler keeps the guarded
// code on the uniform datapath, so cp.async.bulk is issued as a single UBLKCP per copy.  (Issuing
// one copy per lane instead compiles to a VOTEU/R2UR.BROADCAST loop that serialises the 56 copies
// of a tile at ~50 cycles each: profiles/r1_v2_collide.md.)
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile(
      "{\n"
      ".reg .pred P;\n"
      "elect.sync _|P, 0xffffffff;\n"
      "selp.u32 %0, 1, 0, P;\n"
      "}\n"
      : "=r"(pred));
  return pred != 0;
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes,
                                         uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
          "r"(smem_u32(dst)),
      "l"(src), "r"(bytes), "r"(smem_u32(bar))
      : "memory");
}

// e_i . (x,y,z) without a zero-initialised accumulator (0 + x cannot be folded under IEEE rules)
template <typename T>
__device__ __forceinline__ T edot(int i, T x, T y, T z) {
  T r = T(0);
  bool init = false;
  if (ex(i)) { r = T(ex(i)) * x; init = true; }
  if (ey(i)) { r = init ? r + T(ey(i)) * y : T(ey(i)) * y; init = true; }
  if (ez(i)) { r = init ? r + T(ez(i)) * z : T(ez(i)) * z; init = true; }
  return r;
}

template <typename T, int TN>
constexpr size_t collide_smem_bytes() {
  return (size_t)2 * Q * TN * sizeof(T) + (size_t)18 * TN * sizeof(int);
}

// ---------------------------------------------------------------------------------------------
// Component pairs.  The two fluid components go through identical arithmetic with different
// (rho, F) and the same u, so the fused pass carries every per-component quantity as a pair
// (A, B).  For fp32 the pair operations are Blackwell's packed FP32x2 instructions (PTX
// add/sub/mul/fma .f32x2 -> SASS FADD2/FMUL2/FFMA2, two FP32 results per issue slot; a scalar
// broadcast operand and the half-swap are free operand modifiers); for fp64 they are two plain
// operations.  This halves the floating-point issue slots of an issue-bound kernel.
template <typename T> struct alignas(2 * sizeof(T)) Pr { T a, b; };

__device__ __forceinline__ Pr<double> padd(Pr<double> x, Pr<double> y) { return {x.a + y.a, x.b + y.b}; }
__device__ __forceinline__ Pr<double> psub(Pr<double> x, Pr<double> y) { return {x.a - y.a, x.b - y.b}; }
__device__ __forceinline__ Pr<double> pmul(Pr<double> x, Pr<double> y) {
  return {__dmul_rn(x.a, y.a), __dmul_rn(x.b, y.b)};
}
__device__ __forceinline__ Pr<double> pfma(Pr<double> x, Pr<double> y, Pr<double> z) {
  return {__fma_rn(x.a, y.a, z.a), __fma_rn(x.b, y.b, z.b)};
}
__device__ __forceinline__ Pr<float> padd(Pr<float> x, Pr<float> y) {
  Pr<float> d;
  asm("{.reg .b64 ra,rb,rd; mov.b64 ra,{%2,%3}; mov.b64 rb,{%4,%5}; add.rn.f32x2 rd,ra,rb; "
      "mov.b64 {%0,%1},rd;}"
      : "=f"(d.a), "=f"(d.b) : "f"(x.a), "f"(x.b), "f"(y.a), "f"(y.b));
  return d;
}
__device__ __forceinline__ Pr<float> psub(Pr<float> x, Pr<float> y) {
  Pr<float> d;
  asm("{.reg .b64 ra,rb,rd; mov.b64 ra,{%2,%3}; mov.b64 rb,{%4,%5}; sub.rn.f32x2 rd,ra,rb; "
      "mov.b64 {%0,%1},rd;}"
      : "=f"(d.a), "=f"(d.b) : "f"(x.a), "f"(x.b), "f"(y.a), "f"(y.b));
  return d;
}
__device__ __forceinline__ Pr<float> pmul(Pr<float> x, Pr<float> y) {
  Pr<float> d;
  asm("{.reg .b64 ra,rb,rd; mov.b64 ra,{%2,%3}; mov.b64 rb,{%4,%5}; mul.rn.f32x2 rd,ra,rb; "
      "mov.b64 {%0,%1},rd;}"
      : "=f"(d.a), "=f"(d.b) : "f"(x.a), "f"(x.b), "f"(y.a), "f"(y.b));
  return d;
}
__device__ __forceinline__ Pr<float> pfma(Pr<float> x, Pr<float> y, Pr<float> z) {
  Pr<float> d;
  asm("{.reg .b64 ra,rb,rc,rd; mov.b64 ra,{%2,%3}; mov.b64 rb,{%4,%5}; mov.b64 rc,{%6,%7}; "
      "fma.rn.f32x2 rd,ra,rb,rc; mov.b64 {%0,%1},rd;}"
      : "=f"(d.a), "=f"(d.b)
      : "f"(x.a), "f"(x.b), "f"(y.a), "f"(y.b), "f"(z.a), "f"(z.b));
  return d;
}
template <typename T> __device__ __forceinline__ Pr<T> pbc(T s) { return {s, s}; }       // broadcast
template <typename T> __device__ __forceinline__ Pr<T> pswap(Pr<T> x) { return {x.b, x.a}; }

// e_i . (X, Y, Z) on pairs, no zero-initialised accumulator
template <typename T>
__device__ __forceinline__ Pr<T> edot2(int i, Pr<T> x, Pr<T> y, Pr<T> z) {
  Pr<T> r = {T(0), T(0)};
  bool init = false;
  if (ex(i)) { r = ex(i) > 0 ? x : psub(r, x); init = true; }
  if (ey(i)) { r = !init ? (ey(i) > 0 ? y : psub(r, y)) : (ey(i) > 0 ? padd(r, y) : psub(r, y)); init = true; }
  if (ez(i)) { r = !init ? (ez(i) > 0 ? z : psub(r, z)) : (ez(i) > 0 ? padd(r, z) : psub(r, z)); init = true; }
  return r;
}

// Per-thread work of the fused pass on a staged tile: sf = [38][TN] populations, sid = [18][TN]
// neighbour ids in shared memory; tid = column of this thread in the tile; n = its node id.
// Threads of the ragged last tile (valid = false) compute on the zero padding and only their
// stores are predicated off, so control flow stays warp-uniform.
template <typename T, int TN, bool REMAINDER>
__device__ __forceinline__ void collide_tile_thread(const T* __restrict__ sf,
                                                    const int* __restrict__ sid, const int tid,
                                                    const int n, const bool valid,
                                                    T* __restrict__ fout,
                                                    const Vec2<T>* __restrict__ psi, const int nf,
                                                    const size_t npad, const Consts<T>& c) {
  using P = Pr<T>;
  // staged populations: [19][TN] pairs (A, B); column tid
  const P* sfp = reinterpret_cast<const P*>(sf) + tid;
  const int* sidc = sid + tid;

  // a3 inputs: Psi gathers through the staged neighbour ids.  S[d] = sum_i w_i e_id Psi(x+e_i) as
  // a pair (A, B); axis (w=1/18) and diagonal (w=1/36) neighbours are summed separately.
  P S[3];
  {
    P a1[3] = {{T(0), T(0)}, {T(0), T(0)}, {T(0), T(0)}};
    P a2[3] = {{T(0), T(0)}, {T(0), T(0)}, {T(0), T(0)}};
#pragma unroll
    for (int i = 1; i < Q; ++i) {
      const int k0 = sidc[(i - 1) * TN];
      const int k = k0 >= 0 ? k0 : -k0 - 1;  // mirror node beyond an open plane (R12 iv)
      const Vec2<T> v = psi[k];
      const P p = {v.a, v.b};
      P* acc = i < 7 ? a1 : a2;
      if (ex(i)) acc[0] = ex(i) > 0 ? padd(acc[0], p) : psub(acc[0], p);
      if (ey(i)) acc[1] = ey(i) > 0 ? padd(acc[1], p) : psub(acc[1], p);
      if (ez(i)) acc[2] = ez(i) > 0 ? padd(acc[2], p) : psub(acc[2], p);
    }
#pragma unroll
    for (int d = 0; d < 3; ++d)
      S[d] = pfma(pbc(wgt<T>(1)), a1[d], pmul(pbc(wgt<T>(7)), a2[d]));
  }
  // a1 (recomputed locally): R = (rho_A, rho_B); J[d] = per-component bare momentum
  P R = sfp[0];
  P J[3] = {{T(0), T(0)}, {T(0), T(0)}, {T(0), T(0)}};
#pragma unroll
  for (int i = 1; i < Q; ++i) {
    const P f = sfp[i * TN];
    R = padd(R, f);
    if (ex(i)) J[0] = ex(i) > 0 ? padd(J[0], f) : psub(J[0], f);
    if (ey(i)) J[1] = ey(i) > 0 ? padd(J[1], f) : psub(J[1], f);
    if (ez(i)) J[2] = ez(i) > 0 ? padd(J[2], f) : psub(J[2], f);
  }
  // a3: F_sigma = rho_sigma (-G S_sigmabar + g)   (Eq. 10, 11, 13; body force R8)
  const T g[3] = {c.gx, c.gy, c.gz};
  P F[3];
  T u[3];
  const T rho = R.a + R.b;
  const T inv = T(1) / rho;
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    F[d] = pmul(R, pfma(pbc(-c.G), pswap(S[d]), pbc(g[d])));
    // a4: u_eq = (sum_sigma j_sigma + hf * sum_sigma F_sigma) / rho   (Eq. 8, R3)
    u[d] = mul_rn(fma_rn(c.hf, add_rn(F[d].a, F[d].b), add_rn(J[d].a, J[d].b)), inv);
  }
  const T om = rho / fma_rn(R.a, c.tauA, mul_rn(R.b, c.tauB));  // 1/tau_s, Eq. (6)-(7)
  // a5 in opposite-direction pairs (i, opp(i)): with A = 1 + 4.5 (e.u)^2 - 1.5 u.u and
  // B = 9 (e.u)(e.F) - 3 u.F, Eq. (1),(2),(9) give
  //   f*_i      = (1-om) f_i      + [om w rho A + cS w B] + 3 [om w rho (e.u) + cS w (e.F)]
  //   f*_opp(i) = (1-om) f_opp(i) + [om w rho A + cS w B] - 3 [om w rho (e.u) + cS w (e.F)]
  // with cS = 1 - om/2; both components at once as pairs.
  const T k0 = fma_rn(T(-1.5), fma_rn(u[2], u[2], fma_rn(u[1], u[1], mul_rn(u[0], u[0]))), T(1));
  const T c1 = T(1) - om, cS = fma_rn(T(-0.5), om, T(1));
  const P M3UF = pmul(pbc(T(-3)), pfma(pbc(u[0]), F[0], pfma(pbc(u[1]), F[1], pmul(pbc(u[2]), F[2]))));
  const P KA1 = pmul(pbc(mul_rn(om, wgt<T>(1))), R), KA2 = pmul(pbc(mul_rn(om, wgt<T>(7))), R);
  const T kB1 = mul_rn(cS, wgt<T>(1)), kB2 = mul_rn(cS, wgt<T>(7));
  const unsigned np32 = (unsigned)npad;  // 19 * npad < 2^31: 32-bit pair-slot indices
  P* fo = reinterpret_cast<P*>(fout);  // pair (A, B) of population i at node k: fo[i * npad + k]
  P acc = {T(0), T(0)};
#pragma unroll
  for (int i = 1; i < Q; i += 2) {  // canonical order: the opposite of an odd i is its partner
    static_assert(opp(1) == 2 && opp(7) == 10 && opp(9) == 8, "pairing below relies on the table");
    const int ip = i, im = opp(i);
    const P KA = ip < 7 ? KA1 : KA2;
    const T kB = ip < 7 ? kB1 : kB2;
    const T eu = edot<T>(ip, u[0], u[1], u[2]);
    const P EF = edot2<T>(ip, F[0], F[1], F[2]);
    const T A = fma_rn(mul_rn(T(4.5), eu), eu, k0);
    const P B = pfma(pbc(mul_rn(T(9), eu)), EF, M3UF);
    const P X = pfma(KA, pbc(A), pmul(pbc(kB), B));
    const P Y = pfma(KA, pbc(eu), pmul(pbc(kB), EF));
    const P fp = sfp[ip * TN];
    const P fm = sfp[im * TN];
    const P vp = pfma(pbc(c1), fp, pfma(Y, pbc(T(3)), X));
    const P vm = pfma(pbc(c1), fm, pfma(Y, pbc(T(-3)), X));
    acc = padd(acc, padd(vp, vm));
    // a6: push-streaming with halfway bounce-back, branch-free: the slot is computed once per
    // direction; one predicated 8-byte store carries both components of a population
    // (k < 0: the population leaves through an open plane and is dropped).
    {
      const int k = sidc[(ip - 1) * TN];
      const unsigned slot = (unsigned)k < (unsigned)nf ? (unsigned)ip * np32 + (unsigned)k
                                                       : (unsigned)im * np32 + (unsigned)n;
      if (valid && k >= 0) fo[slot] = vp;
    }
    {
      const int k = sidc[(im - 1) * TN];
      const unsigned slot = (unsigned)k < (unsigned)nf ? (unsigned)im * np32 + (unsigned)k
                                                       : (unsigned)ip * np32 + (unsigned)n;
      if (valid && k >= 0) fo[slot] = vm;
    }
  }
  // rest population: Eq. (1) with e_0 = 0, or the remainder rho - sum_{i>=1} f*_i (fp32 build)
  P v0;
  if (REMAINDER) {
    v0 = psub(R, acc);
  } else {
    const T w0 = wgt<T>(0);
    const P f0 = sfp[0];
    v0 = pfma(pbc(c1), f0, pfma(pbc(mul_rn(mul_rn(om, w0), k0)), R, pmul(pbc(mul_rn(cS, w0)), M3UF)));
  }
  if (valid) fo[n] = v0;
}

// 16-bit tile-relative neighbour index (geometry.hpp Index16): per tile 18 rows of TN uint16 plus
// a 160 B record of bases.  Halves the index bytes of the fused pass (72 -> 37 B per node).
constexpr int kIdxMeta = 40;
struct Idx16 {
  const uint16_t* nbr16;  // [18][npad]
  const int* meta;        // [tiles][kIdxMeta]
  int np_lo, np_hi;       // nodes per open plane (nx*ny) at the low / high z end, 0 if that end is
                          // not an open plane (periodic, or a slab cut)
  int reverse;            // 1: CTA b takes tile gridDim-1-b
  int nact;               // nodes this pass updates: ids [0,nact).  = nf, except in slab mode, where
                          // the halo nodes [nact,nf) only receive pushes
  int tile0, split, tile1;  // tiles of this launch: position b < split -> tile0 + b, else
                            // tile1 + (b - split)  (whole pass: 0, grid, 0; slab mode: the boundary
                            // tiles of both faces in one launch, the interior in another)
};

// ALIAS: the 16-bit rows are staged into the upper half of the int32 id array they are decoded
// into (every thread first takes its 18 entries into registers, one CTA barrier, then writes the
// decoded ids): 4.6 KB less shared memory per CTA, which lets a 7th CTA onto the SM.
template <typename T, int TN, bool ALIAS = false>
constexpr size_t collide16_smem_bytes() {
  return collide_smem_bytes<T, TN>() + (ALIAS ? 0 : (size_t)18 * TN * sizeof(uint16_t)) +
         kIdxMeta * sizeof(int);
}

// Shared-memory carve-up of one staged tile (16-bit index form)
template <typename T, int TN, bool ALIAS>
struct TileSmem {
  T* sf;           // [38][TN] populations
  int* sid;        // [18][TN] decoded neighbour ids
  uint16_t* s16;   // [18][TN] staged 16-bit rows (inside the upper half of sid when ALIAS)
  int* smeta;      // [kIdxMeta]
  __device__ __forceinline__ explicit TileSmem(unsigned char* raw) {
    sf = reinterpret_cast<T*>(raw);
    sid = reinterpret_cast<int*>(raw + (size_t)2 * Q * TN * sizeof(T));
    s16 = reinterpret_cast<uint16_t*>(raw + collide_smem_bytes<T, TN>() -
                                      (ALIAS ? (size_t)18 * TN * sizeof(uint16_t) : 0));
    smeta = reinterpret_cast<int*>(raw + collide16_smem_bytes<T, TN, ALIAS>() -
                                   kIdxMeta * sizeof(int));
  }
};

// Stage one tile: 19 population rows of TN (A, B) pairs, 18 rows of 16-bit index, the tile's
// record of bases -> shared memory, completion on `bar`.  Call from one converged warp.
template <typename T, int TN, bool ALIAS>
__device__ __forceinline__ void stage_tile16(const TileSmem<T, TN, ALIAS> sm,
                                             const T* __restrict__ fin, const Idx16& ix,
                                             size_t npad, unsigned tile, uint64_t* bar) {
  const size_t t0 = (size_t)tile * TN;
  if (elect_one()) {
    mbar_expect_tx(bar, (uint32_t)((size_t)2 * Q * TN * sizeof(T) +
                                   (size_t)18 * TN * sizeof(uint16_t) + kIdxMeta * sizeof(int)));
#pragma unroll
    for (int r = 0; r < Q; ++r)  // one row of TN (A, B) pairs per direction
      bulk_g2s(sm.sf + (size_t)r * TN * 2, fin + ((size_t)r * npad + t0) * 2,
               2 * TN * sizeof(T), bar);
#pragma unroll
    for (int r = 0; r < 18; ++r)
      bulk_g2s(sm.s16 + (size_t)r * TN, ix.nbr16 + (size_t)r * npad + t0, TN * sizeof(uint16_t),
               bar);
    bulk_g2s(sm.smeta, ix.meta + (size_t)tile * kIdxMeta, kIdxMeta * sizeof(int), bar);
  }
  __syncwarp();
}

// After the staged tile has arrived: decode this thread's column of the 16-bit rows into the
// int32 form the tile function reads.  A neighbour beyond an open plane (reading R12 iv) is
// recognised from the node's plane and e_z.  Rare "wide" tiles (an offset range does not fit 15
// bits) take int32 ids from the compact wide-tile table with a second round of bulk copies (one
// more phase of `bar`).
// Called by every thread of the CTA.
template <typename T, int TN, bool ALIAS>
__device__ __forceinline__ void decode_tile16(const TileSmem<T, TN, ALIAS> sm,
                                              const int* __restrict__ nbr, const Idx16& ix,
                                              size_t npad, size_t t0, int n, int tid, int warp,
                                              uint64_t* bar, uint32_t& phase) {
  const int wide = __shfl_sync(0xffffffffu, sm.smeta[36], 0);
  if (wide) {
    if (warp == 0) {
      if (elect_one()) {
        mbar_expect_tx(bar, (uint32_t)((size_t)18 * TN * sizeof(int)));
#pragma unroll
        for (int r = 0; r < 18; ++r)   // nbr = the compact table of the wide tiles, [pos][18][TN]
          bulk_g2s(sm.sid + (size_t)r * TN, nbr + ((size_t)sm.smeta[37] * 18 + r) * TN,
                   TN * sizeof(int), bar);
      }
      __syncwarp();
    }
    mbar_wait(bar, phase);
    phase ^= 1u;
  } else {
    const bool lo_plane = n < ix.np_lo, hi_plane = n >= ix.nact - ix.np_hi;
    int ev[Q];
    if constexpr (ALIAS) {
#pragma unroll
      for (int i = 1; i < Q; ++i) ev[i] = sm.s16[(i - 1) * TN + tid];
      __syncthreads();  // every column is in registers before the ids overwrite the rows
    }
#pragma unroll
    for (int i = 1; i < Q; ++i) {
      const int e = ALIAS ? ev[i] : (int)sm.s16[(i - 1) * TN + tid];
      int k = sm.smeta[(e >> 15) * 18 + (i - 1)] + (e & 0x7fff);
      if (ez(i) < 0) k = lo_plane ? -k - 1 : k;
      if (ez(i) > 0) k = hi_plane ? -k - 1 : k;
      sm.sid[(i - 1) * TN + tid] = k;
    }
  }
}

// The fused pass (a3-a6): one CTA per tile.
// IDX: index form; 1 = 16-bit tile-relative rows (the only one left: the geometric index, 2, and
// 8-bit rows were measured slower and removed)
template <typename T, int TN, int MINB, bool REMAINDER, int IDX>
__global__ void __launch_bounds__(TN, MINB)
    k_collide_stream_bulk(const T* __restrict__ fin, T* __restrict__ fout,
                          const Vec2<T>* __restrict__ psi, const int* __restrict__ nbr, int nf,
                          size_t npad, Consts<T> c, Idx16 ix) {
  static_assert(IDX == 1, "index form");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr bool kAlias = MINB >= 7;
  const TileSmem<T, TN, kAlias> sm(smem_raw);
  __shared__ uint64_t bar;
  const int tid = threadIdx.x;
  // Tiles are taken from the END of the id range first: the density pass that ran just before
  // walked the range forwards, so the last ~100 MB of populations it read are still in L2, and
  // this kernel's last writes (the head of the range) are what the next density pass reads first.
  const int pos = ix.reverse ? (int)(gridDim.x - 1u - blockIdx.x) : (int)blockIdx.x;
  const unsigned tile = (unsigned)(pos < ix.split ? ix.tile0 + pos : ix.tile1 + (pos - ix.split));
  const size_t t0 = (size_t)tile * TN;
  if (tid == 0) mbar_init(&bar, 1);
  __syncthreads();
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);  // compiler-visible warp-uniform value
  const int n = (int)t0 + tid;
  uint32_t phase = 0;
  if (warp == 0) stage_tile16<T, TN, kAlias>(sm, fin, ix, npad, tile, &bar);
  // the bulk copies above read the populations (complete since the previous step; the density
  // pass that fixed the open planes finished before the wall pass began) and the static index;
  // psi and the wall psi are this step's
  pdl_wait();
  mbar_wait(&bar, phase);
  phase ^= 1u;
  decode_tile16<T, TN, kAlias>(sm, nbr, ix, npad, t0, n, tid, warp, &bar, phase);
  collide_tile_thread<T, TN, REMAINDER>(sm.sf, sm.sid, tid, n, n < ix.nact, fout, psi, nf, npad, c);
}

// ---------------------------------------------------------------------------------------------
// a0  open-plane fix on the new buffer (reading R12 of PAPER.md L147-157, L223): planes z=0 and
// z=nz-1 are all fluid, so their ids are q, nf-np+q and their interior neighbours np+q,
// nf-2np+q.  Dirichlet component: all 19 populations <- feq(rho_b,u_b) + [f(x_f) - feq(rho(x_f),
// u_f)] (non-equilibrium extrapolation), or only its 5 inward populations by the Zou-He rule
// (kinds 3, 4); other component: its 5 inward populations <- frozen.
template <typename T>
struct OpenPlane {
  int dc[2];       // Dirichlet component at inlet / outlet
  int kind[2];     // 1 density (NEEM), 2 velocity (NEEM), 3 density (Zou-He), 4 velocity (Zou-He);
                   // 0: that end of this box is not an open plane (a slab cut)
  T rho[2];        // imposed density (kinds 1, 3)
  T uz[2];         // imposed velocity (kinds 2, 4)
};

template <typename T>
__device__ __forceinline__ T feq_of(int i, T rho, const T (&u)[3]) {
  T eu = T(0);
  if (ex(i)) eu += T(ex(i)) * u[0];
  if (ey(i)) eu += T(ey(i)) * u[1];
  if (ez(i)) eu += T(ez(i)) * u[2];
  const T uu = fma_rn(u[2], u[2], fma_rn(u[1], u[1], mul_rn(u[0], u[0])));
  T t = fma_rn(T(3), eu, T(1));
  t = fma_rn(mul_rn(T(4.5), eu), eu, t);
  t = fma_rn(T(-1.5), uu, t);
  return mul_rn(mul_rn(wgt<T>(i), rho), t);
}

// One node of an open plane: applies the fix in place and returns the node's new densities,
// summed in direction order like the density pass does.
template <typename T>
__device__ __forceinline__ Vec2<T> open_plane_node(T* __restrict__ f, const T* __restrict__ frozen,
                                                   int nf, int np, size_t npad,
                                                   const OpenPlane<T>& op, int plane, int q) {
  const int vb = plane == 0 ? q : nf - np + q;
  const int vf = plane == 0 ? np + q : nf - 2 * np + q;
  const int dc = op.dc[plane];
  T rd = T(0);  // new density of the Dirichlet component
  if (op.kind[plane] <= 2) {
    T ff[2][Q];
    T rf[2] = {T(0), T(0)}, j[3] = {T(0), T(0), T(0)};
#pragma unroll
    for (int s = 0; s < 2; ++s)
#pragma unroll
      for (int i = 0; i < Q; ++i) {
        const T v = f[pidx(s, i, vf, npad)];
        ff[s][i] = v;
        rf[s] += v;
        if (ex(i)) j[0] += T(ex(i)) * v;
        if (ey(i)) j[1] += T(ey(i)) * v;
        if (ez(i)) j[2] += T(ez(i)) * v;
      }
    const T inv = T(1) / (rf[0] + rf[1]);
    const T uf[3] = {mul_rn(j[0], inv), mul_rn(j[1], inv), mul_rn(j[2], inv)};  // R12 iii: bare mixture velocity
    const T rfd = dc == 0 ? rf[0] : rf[1];
    T rho_b, ub[3];
    if (op.kind[plane] == 1) {
      rho_b = op.rho[plane];
      ub[0] = uf[0]; ub[1] = uf[1]; ub[2] = uf[2];
    } else {
      rho_b = rfd;
      ub[0] = T(0); ub[1] = T(0); ub[2] = op.uz[plane];
    }
#pragma unroll
    for (int i = 0; i < Q; ++i) {
      const T fi = dc == 0 ? ff[0][i] : ff[1][i];
      const T v = add_rn(feq_of<T>(i, rho_b, ub), add_rn(fi, -feq_of<T>(i, rfd, uf)));
      f[pidx(dc, i, vb, npad)] = v;
      rd = i == 0 ? v : rd + v;
    }
  } else {
    // Zou-He variant (ref. [34]; reading R31), kinds 3 (density) and 4 (velocity):
    // purely local.  The 14 populations streaming delivered stay; the 5 that would come from
    // beyond the plane are the bounce-back of the non-equilibrium part, with the transverse
    // corrections N_x, N_y that make the node's x- and y-momentum vanish.  From mass and
    // z-momentum, rho (1 - sgn u_z) = K0 + 2 Km (K0: in-plane sum, Km: outgoing sum).
    const int sgn = plane == 0 ? 1 : -1;
    T fb[Q];
    T K0 = T(0), Km = T(0), Nx = T(0), Ny = T(0);
#pragma unroll
    for (int i = 0; i < Q; ++i) {
      if (ez(i) == 0) {
        const T v = f[pidx(dc, i, vb, npad)];
        fb[i] = v;
        K0 += v;
        if (ex(i)) Nx = fma_rn(T(0.5) * T(ex(i)), v, Nx);
        if (ey(i)) Ny = fma_rn(T(0.5) * T(ey(i)), v, Ny);
      } else if (ez(i) == -sgn) {
        const T v = f[pidx(dc, i, vb, npad)];
        fb[i] = v;
        Km += v;
      } else {
        fb[i] = T(0);  // unknown: whatever the slot holds is stale
      }
    }
    T rho, uz;
    if (op.kind[plane] == 3) {
      rho = op.rho[plane];
      uz = mul_rn(T(sgn), add_rn(T(1), -(fma_rn(T(2), Km, K0) / rho)));
    } else {
      uz = op.uz[plane];
      rho = fma_rn(T(2), Km, K0) / add_rn(T(1), -mul_rn(T(sgn), uz));
    }
#pragma unroll
    for (int i = 1; i < Q; ++i) {
      if (ez(i) == 0 || ez(i) != sgn) continue;
      T v = add_rn(fb[opp(i)], mul_rn(mul_rn(T(6) * wgt<T>(i), rho), mul_rn(T(ez(i)), uz)));
      if (ex(i)) v = add_rn(v, -mul_rn(T(ex(i)), Nx));
      if (ey(i)) v = add_rn(v, -mul_rn(T(ey(i)), Ny));
      fb[i] = v;
      f[pidx(dc, i, vb, npad)] = v;
    }
#pragma unroll
    for (int i = 0; i < Q; ++i) rd = i == 0 ? fb[i] : rd + fb[i];
  }
  const int oc = 1 - dc;
  T ro = T(0);  // new density of the other component: 14 streamed + 5 frozen populations
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    T v;
    if (plane == 0 ? ez(i) > 0 : ez(i) < 0) {
      int k = 0;
#pragma unroll
      for (int kk = 0; kk < 5; ++kk)
        if (inward(0, kk) == i || inward(1, kk) == i) k = kk;
      v = frozen[((size_t)(plane * 2 + oc) * 5 + k) * np + q];
      f[pidx(oc, i, vb, npad)] = v;
    } else {
      v = f[pidx(oc, i, vb, npad)];
    }
    ro = i == 0 ? v : ro + v;
  }
  Vec2<T> o;
  o.a = dc == 0 ? rd : ro;
  o.b = dc == 0 ? ro : rd;
  return o;
}

template <typename T>
__global__ void __launch_bounds__(128) k_open_planes(T* __restrict__ f,
                                                     const T* __restrict__ frozen, int nf, int np,
                                                     size_t npad, OpenPlane<T> op) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= 2 * np) return;
  const int plane = t / np;
  if (op.kind[plane] == 0) return;
  open_plane_node<T>(f, frozen, nf, np, npad, op, plane, t - plane * np);
}

// a0 + a1 in one launch: the first `nb_planes` blocks fix the two open planes (they only read the
// interior neighbour planes) and write those nodes' psi themselves; the remaining blocks are the
// density pass on every node that is not on an open plane.  Launched alone the plane fix is a
// short latency-bound kernel of 2*nx*ny threads that adds ~12 us to every step; scheduled first
// inside the density pass its dependent chain overlaps the streaming blocks.
template <typename T>
__global__ void __launch_bounds__(256, 4)
    k_density_open(T* __restrict__ f, Vec2<T>* __restrict__ psi, const T* __restrict__ frozen,
                   int nf, int np, size_t npad, int nb_planes, OpenPlane<T> op, float keep_psi,
                   NodeRange r) {
  // nf = number of nodes this context updates (all fluid nodes; the owned ones in slab mode)
  pdl_wait();  // f was written by the previous step's fused pass
  const uint64_t pol = l2_keep_policy(keep_psi);
  if ((int)blockIdx.x >= nb_planes) {
    const int b = (int)blockIdx.x - nb_planes;
    const int n = (b < r.split ? r.a0 + b * (int)blockDim.x : r.a1 + (b - r.split) * (int)blockDim.x) +
                  (int)threadIdx.x;
    if (n >= r.nend || (op.kind[0] && n < np) || (op.kind[1] && n >= nf - np)) return;
    const Vec2<T>* f2 = reinterpret_cast<const Vec2<T>*>(f);
    Vec2<T> v[Q];
#pragma unroll
    for (int i = 0; i < Q; ++i) v[i] = f2[(size_t)i * npad + n];
    T ra = v[0].a, rb = v[0].b;
#pragma unroll
    for (int i = 1; i < Q; ++i) { ra += v[i].a; rb += v[i].b; }
    Vec2<T> o; o.a = ra; o.b = rb;
    store_vec2(psi + n, o, pol);
  } else {  // the plane blocks come first so that their dependent chain overlaps the streaming
    const int t = (int)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= 2 * np) return;
    const int plane = t / np, q = t - plane * np;
    if (op.kind[plane] == 0) return;
    store_vec2(psi + (plane == 0 ? q : nf - np + q),
               open_plane_node<T>(f, frozen, nf, np, npad, op, plane, q), pol);
  }
}

// ---------------------------------------------------------------------------------------------
// Slab halo (multi-GPU z-slabs): the 5 populations per component that crossed a
// cut sit, after the fused pass, in the rows of the inner halo plane's nodes.  k_halo_pack gathers
// them (both faces in one launch) into the send buffer through a precomputed slot list;
// k_halo_unpack scatters what the neighbour slabs sent into the rows of the owned boundary
// planes.  One (A, B) pair per entry; geometry.hpp Halo.
template <typename T>
__global__ void __launch_bounds__(256) k_halo_pack(const T* __restrict__ f,
                                                   const int* __restrict__ slots,
                                                   T* __restrict__ buf, int n) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  reinterpret_cast<Vec2<T>*>(buf)[k] = reinterpret_cast<const Vec2<T>*>(f)[slots[k]];
}
template <typename T>
__global__ void __launch_bounds__(256) k_halo_unpack(T* __restrict__ f,
                                                     const int* __restrict__ slots,
                                                     const T* __restrict__ buf, int n) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  reinterpret_cast<Vec2<T>*>(f)[slots[k]] = reinterpret_cast<const Vec2<T>*>(buf)[k];
}

// frozen[plane][comp][k][q] <- f[comp][inward(plane,k)][plane node q]   (reading R27)
template <typename T>
__global__ void k_record_frozen(const T* __restrict__ f, T* __restrict__ frozen, int comp, int nf,
                                int np, size_t npad, int planes /* bit p: plane p is open */) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= 2 * np) return;
  const int plane = t / np, q = t - plane * np;
  if (!((planes >> plane) & 1)) return;
  const int vb = plane == 0 ? q : nf - np + q;
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    const int i = plane == 0 ? inward(0, k) : inward(1, k);
    frozen[((size_t)(plane * 2 + comp) * 5 + k) * np + q] = f[pidx(comp, i, vb, npad)];
  }
}

// ---------------------------------------------------------------------------------------------
// Initialisation and I/O between dense host-ordered double arrays (device copies) and the
// compact store.  node_vox[n] = dense voxel index of fluid node n.
template <typename T>
__global__ void k_init_density(const double* __restrict__ rhoA, const double* __restrict__ rhoB,
                               const int* __restrict__ node_vox, T* __restrict__ f, int nf,
                               size_t npad) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= nf) return;
  const int v = node_vox[n];
  const double ra = rhoA[v], rb = rhoB[v];
#pragma unroll
  for (int i = 0; i < Q; ++i) {  // f_i = w_i rho (reading R11)
    f[pidx(0, i, n, npad)] = (T)(wgt<double>(i) * ra);
    f[pidx(1, i, n, npad)] = (T)(wgt<double>(i) * rb);
  }
}

template <typename T>
__global__ void k_dense_to_compact(const double* __restrict__ dense,
                                   const int* __restrict__ node_vox, T* __restrict__ row, int nf,
                                   int stride) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n < nf) row[(size_t)n * stride] = (T)dense[node_vox[n]];
}

template <typename T>
__global__ void k_compact_to_dense(const T* __restrict__ row, const int* __restrict__ node_vox,
                                   double* __restrict__ dense, int nf, int stride) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n < nf) dense[node_vox[n]] = (double)row[(size_t)n * stride];
}

// Neighbour ids for the kernels outside the time step (macroscopic getter, connected components):
// decoded from the 16-bit rows exactly as the fused pass does, wide tiles from the compact table.
struct NbrView {
  const uint16_t* nbr16;    // [18][npad]
  const int* meta;          // [tiles][kIdxMeta]
  const int* wide;          // [wide tiles][18][128]
  int np_lo, np_hi, nact;   // open planes, as in Idx16
};
// psi index of x+e_i for node n, i = 1..18 (negative: -(mirror id + 1) beyond an open plane)
__device__ __forceinline__ int nbr_id(const NbrView& v, size_t npad, int n, int i) {
  const int* m = v.meta + (size_t)(n >> 7) * kIdxMeta;
  if (m[36]) return v.wide[((size_t)m[37] * 18 + (i - 1)) * 128 + (n & 127)];
  const int e = v.nbr16[(size_t)(i - 1) * npad + n];
  int k = m[(e >> 15) * 18 + (i - 1)] + (e & 0x7fff);
  if (ez(i) < 0 && n < v.np_lo) k = -k - 1;
  if (ez(i) > 0 && n >= v.nact - v.np_hi) k = -k - 1;
  return k;
}

// rho_sigma, u = u_eq, P = (rho_A+rho_B)/3 + (G/3) rho_A rho_B (Eq. 12, R13) into
// compact double rows out[q][nf], q = rhoA, rhoB, ux, uy, uz, P.  Needs psi of the current state.
template <typename T>
__global__ void __launch_bounds__(256) k_macroscopic(const T* __restrict__ fin,
                                                     const Vec2<T>* __restrict__ psi,
                                                     NbrView nv,
                                                     double* __restrict__ out, int nf, size_t npad,
                                                     Consts<T> c) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= nf) return;
  int id[Q];
  id[0] = n;
#pragma unroll
  for (int i = 1; i < Q; ++i) id[i] = nbr_id(nv, npad, n, i);
  T fa[Q], fb[Q];
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    fa[i] = fin[pidx(0, i, n, npad)];
    fb[i] = fin[pidx(1, i, n, npad)];
  }
  NodeState<T> s;
  node_state<T>(fa, fb, psi, id, c, s);
  out[n] = (double)s.rhoA;
  out[(size_t)nf + n] = (double)s.rhoB;
  out[(size_t)2 * nf + n] = (double)s.u[0];
  out[(size_t)3 * nf + n] = (double)s.u[1];
  out[(size_t)4 * nf + n] = (double)s.u[2];
  out[(size_t)5 * nf + n] =
      (double)((s.rhoA + s.rhoB) / T(3) + (c.G / T(3)) * s.rhoA * s.rhoB);
}

// ---------------------------------------------------------------------------------------------
// a7  diagnostics: warp-shuffle block reductions into one fp64 partial per block, then a
// single-block fixed-order second stage: the sums are deterministic.
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  return v;
}

constexpr int kDiagVals = 6;  // mass A, mass B, momentum x,y,z, non-finite count
constexpr int kDiagBlock = 256;

template <typename T>
__global__ void __launch_bounds__(kDiagBlock) k_diag_partial(const T* __restrict__ f,
                                                             double* __restrict__ partial, int nf,
                                                             size_t npad) {
  double acc[kDiagVals] = {0, 0, 0, 0, 0, 0};
  for (int n = blockIdx.x * blockDim.x + threadIdx.x; n < nf; n += gridDim.x * blockDim.x) {
#pragma unroll
    for (int s = 0; s < 2; ++s)
#pragma unroll
      for (int i = 0; i < Q; ++i) {
        const double v = (double)f[pidx(s, i, n, npad)];
        acc[s] += v;
        if (ex(i)) acc[2] += ex(i) * v;
        if (ey(i)) acc[3] += ey(i) * v;
        if (ez(i)) acc[4] += ez(i) * v;
        if (!isfinite(v)) acc[5] += 1.0;
      }
  }
  __shared__ double sm[kDiagVals][kDiagBlock / 32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < kDiagVals; ++k) {
    const double v = warp_sum(acc[k]);
    if (lane == 0) sm[k][wid] = v;
  }
  __syncthreads();
  if (threadIdx.x < kDiagVals) {
    double t = 0.0;
    for (int w = 0; w < kDiagBlock / 32; ++w) t += sm[threadIdx.x][w];
    partial[(size_t)blockIdx.x * kDiagVals + threadIdx.x] = t;
  }
}

__global__ void k_diag_final(const double* __restrict__ partial, double* __restrict__ out,
                             int nblocks) {
  const int k = threadIdx.x;
  if (k >= kDiagVals) return;
  double t = 0.0;
  for (int b = 0; b < nblocks; ++b) t += partial[(size_t)b * kDiagVals + k];
  out[k] = t;
}

// Saturation (reading R14): count nodes in the id range [n0,n1) whose
// rho_comp exceeds the other density (tie -> component 1).  Integer atomics: deterministic.
template <typename T>
__global__ void k_count_phase(const Vec2<T>* __restrict__ psi, int n0, int n1, int comp,
                              unsigned long long* __restrict__ count) {
  const int n = n0 + blockIdx.x * blockDim.x + threadIdx.x;
  int mine = 0;
  if (n < n1) {
    const Vec2<T> p = psi[n];
    const int owner = p.a > p.b ? 0 : 1;
    mine = owner == comp;
  }
  const unsigned b = __ballot_sync(0xffffffffu, mine);
  if ((threadIdx.x & 31) == 0 && b) atomicAdd(count, (unsigned long long)__popc(b));
}

// ---------------------------------------------------------------------------------------------
// a7  trapped volume (reading R15): connected components of the phase-comp
// fluid nodes over the 6-neighbour graph (periodic in x,y; no edge across the z ends), by
// lock-free union-find on the compact ids.  parent[n] = -1 for nodes of the other phase; a
// larger root is always hooked under a smaller one, so the root of a cluster is its smallest id
// and the result does not depend on the interleaving.  Every access to parent[] goes to L2
// (ld.cg / st.cg / atomics): a stale L1 line could make the hook loop spin.
template <typename T>
__global__ void __launch_bounds__(256) k_ccl_init(const Vec2<T>* __restrict__ psi, int nf, int comp,
                                                  int* __restrict__ parent, int* __restrict__ flag) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= nf) return;
  const Vec2<T> p = psi[n];
  const int owner = p.a > p.b ? 0 : 1;  // tie -> component 1, as k_count_phase
  parent[n] = owner == comp ? n : -1;
  flag[n] = 0;
}

__device__ __forceinline__ int ccl_find(int* parent, int x) {
  int p = __ldcg(parent + x);
  while (p != x) {  // path halving: x is not a root and never becomes one again
    const int g = __ldcg(parent + p);
    if (g != p) __stcg(parent + x, g);
    x = p;
    p = g;
  }
  return x;
}

__device__ __forceinline__ void ccl_unite(int* parent, int a, int b) {
  for (;;) {
    a = ccl_find(parent, a);
    b = ccl_find(parent, b);
    if (a == b) return;
    if (a < b) { const int t = a; a = b; b = t; }
    if (atomicCAS(parent + a, a, b) == a) return;  // else a was hooked meanwhile: look again
  }
}

// one thread per fluid node: joins it to its +x, +y, +z neighbour of the same phase (each edge of
// the graph is the forward edge of exactly one of its ends; the periodic wrap in z is the one
// forward neighbour with a smaller id, and a neighbour beyond an open plane is negative)
__global__ void __launch_bounds__(256) k_ccl_unite(NbrView nv, int nf, size_t npad, int* parent) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= nf || __ldcg(parent + n) < 0) return;
#pragma unroll
  for (int i = 1; i <= 5; i += 2) {
    static_assert(ex(1) == 1 && ey(3) == 1 && ez(5) == 1, "forward axis directions");
    const int m = nbr_id(nv, npad, n, i);
    if (m < 0 || m >= nf || (i == 5 && m <= n)) continue;
    if (__ldcg(parent + m) < 0) continue;
    ccl_unite(parent, n, m);
  }
}

// after the last union: parent[n] <- root.  The walk only reads (a path-halving store by another
// thread could land after this thread's final store and leave a non-root behind); whatever it
// meets on the way is either an old ancestor or already the root.
__global__ void __launch_bounds__(256) k_ccl_flatten(int nf, int* parent) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= nf) return;
  int x = __ldcg(parent + n);
  if (x < 0) return;
  for (int p = __ldcg(parent + x); p != x; p = __ldcg(parent + x)) x = p;
  __stcg(parent + n, x);
}

// clusters with a node on z = 0 or z = nz-1 are connected to an end plane; [a0,a1) and [b0,b1)
// are the id ranges of those two planes
__global__ void __launch_bounds__(256) k_ccl_mark(const int* __restrict__ parent, int a0, int a1,
                                                  int b0, int b1, int* __restrict__ flag) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  const int na = a1 - a0;
  if (k >= na + (b1 - b0)) return;
  const int n = k < na ? a0 + k : b0 + (k - na);
  const int r = parent[n];
  if (r >= 0) flag[r] = 1;
}

// Trapped volume across slab cuts.  Each slab labels its owned nodes on its own (the kernels
// above; edges into halo nodes are skipped because their ids are >= the owned count), marks the
// clusters that touch a global end plane it owns, and then the "connected to an end plane" flag is
// propagated across the cuts until nothing changes: k_ccl_export writes, for every (x,y) of an
// owned boundary plane, the flag of the phase cluster there (-1: solid or other phase) into a
// dense nx*ny plane; the neighbour slab's k_ccl_import reads the plane at the (x,y) of its own
// boundary-plane nodes (the 6-neighbour across the cut) and raises the flag of their clusters.
__global__ void __launch_bounds__(256) k_ccl_export(const int* __restrict__ parent,
                                                    const int* __restrict__ flag,
                                                    const int* __restrict__ node_vox, int n0, int n1,
                                                    int np, int* __restrict__ out) {
  const int n = n0 + blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= n1) return;
  const int r = parent[n];
  out[node_vox[n] % np] = r >= 0 ? flag[r] : -1;
}
__global__ void __launch_bounds__(256) k_ccl_import(const int* __restrict__ parent, int* flag,
                                                    const int* __restrict__ node_vox, int n0, int n1,
                                                    int np, const int* __restrict__ in,
                                                    int* __restrict__ changed) {
  const int n = n0 + blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= n1) return;
  const int r = parent[n];
  if (r < 0 || in[node_vox[n] % np] != 1) return;
  if (atomicExch(flag + r, 1) == 0) atomicAdd(changed, 1);
}

// nodes and mass of the unmarked clusters in the id range [n0,n1); block b takes one contiguous
// chunk and k_sum_pairs adds the per-block results in block order (deterministic)
constexpr int kCclBlock = 256;
template <typename T>
__global__ void __launch_bounds__(kCclBlock) k_ccl_count(const Vec2<T>* __restrict__ psi,
                                                         const int* __restrict__ parent,
                                                         const int* __restrict__ flag, int n0, int n1,
                                                         int comp, int chunk,
                                                         double* __restrict__ partial) {
  __shared__ double smass[kCclBlock / 32];
  __shared__ long long scnt[kCclBlock / 32];
  const int lo = n0 + blockIdx.x * chunk;
  const int hi = min(n1, lo + chunk);
  double mass = 0.0;
  long long cnt = 0;
  for (int n = lo + threadIdx.x; n < hi; n += kCclBlock) {
    const int r = parent[n];
    if (r >= 0 && flag[r] == 0) {
      const Vec2<T> p = psi[n];
      mass += (double)(comp == 0 ? p.a : p.b);
      ++cnt;
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    mass += __shfl_down_sync(0xffffffffu, mass, o);
    cnt += __shfl_down_sync(0xffffffffu, cnt, o);
  }
  if ((threadIdx.x & 31) == 0) { smass[threadIdx.x >> 5] = mass; scnt[threadIdx.x >> 5] = cnt; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < kCclBlock / 32; ++w) { mass += smass[w]; cnt += scnt[w]; }
    partial[2 * blockIdx.x] = mass;
    partial[2 * blockIdx.x + 1] = (double)cnt;  // exact: < 2^53
  }
}

__global__ void k_sum_pairs(const double* __restrict__ partial, int nblocks, double* __restrict__ out) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  double mass = 0.0, cnt = 0.0;
  for (int b = 0; b < nblocks; ++b) { mass += partial[2 * b]; cnt += partial[2 * b + 1]; }
  out[0] = mass;
  out[1] = cnt;
}


// Mean pressure over an id range (capillary pressure P_c = P_in - P_out of PAPER.md L223 is the
// difference of two such plane means): per-block sums of P = (rho_A+rho_B)/3 + (G/3) rho_A rho_B
// (Eq. 12, reading R13), evaluated in T exactly as k_macroscopic does, accumulated in fp64;
// k_sum_pairs adds the blocks in order.
template <typename T>
__global__ void __launch_bounds__(kCclBlock) k_pressure_sum(const Vec2<T>* __restrict__ psi, int n0,
                                                            int n1, T G, int chunk,
                                                            double* __restrict__ partial) {
  __shared__ double ssum[kCclBlock / 32];
  const int lo = n0 + blockIdx.x * chunk;
  const int hi = min(n1, lo + chunk);
  double sum = 0.0;
  for (int n = lo + threadIdx.x; n < hi; n += kCclBlock) {
    const Vec2<T> p = psi[n];
    sum += (double)((p.a + p.b) / T(3) + (G / T(3)) * p.a * p.b);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) sum += __shfl_down_sync(0xffffffffu, sum, o);
  if ((threadIdx.x & 31) == 0) ssum[threadIdx.x >> 5] = sum;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < kCclBlock / 32; ++w) sum += ssum[w];
    partial[2 * blockIdx.x] = sum;
    partial[2 * blockIdx.x + 1] = (double)(hi - lo);
  }
}

}  // namespace lbmk
