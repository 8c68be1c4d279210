// bssn_tma.cuh -- device side of the fused BSSN kernel: persistent CTAs, one grid point per thread, the
// (tile + 3-cell halo) box of ONE variable at a time staged into shared memory by TMA (cp.async.bulk.tensor)
// through a 5-slot mbarrier ring, so that every stencil read is an LDS with a compile-time offset.
// The variables are consumed in an order chosen to keep the live register set small (H2 in SURVEY.md):
//   beta^i -> gt_ij -> [Christoffels, quadratic part of R~_ij] -> Gt^i -> chi -> alpha -> K -> At_ij -> B^i -> A
// Each variable's derivatives are contracted / folded into the few values the pointwise expression needs as
// soon as they are produced, and each right-hand side leaves through the fused RK4 stage update the moment
// it is complete.  Mathematics: readings S2-S6, S10 of DESIGN.md (same system as bssn_point.cuh; that file
// serves the split variant).
#pragma once
#ifndef CHM_EMULATE
#include <cuda.h>
#endif

#include "bssn_point.cuh"

namespace chm {

// ---- TMA / mbarrier: host emulation (tests/native/cta_emu.hpp; the kernel source is compiled unchanged) ------------
#ifdef CHM_EMULATE
#define CHM_DYNAMIC_SMEM(name) unsigned char* name = chm_emu::t_cta->smem
inline uint32_t smem_u32(const void* p) { return chm_emu::smem_offset(p); }
inline void mbar_init(uint64_t* bar, int count) { chm_emu::mbar_init(bar, count); }
inline void mbar_expect_tx(uint64_t* bar, uint32_t bytes) { chm_emu::mbar_expect_tx(bar, bytes); }
inline bool mbar_try(uint32_t bar, uint32_t parity) { return chm_emu::mbar_try_wait(chm_emu::smem_at(bar), parity); }
constexpr long long kWaitBudget = 120000000000LL;   // nanoseconds here: 256 OS threads on a few cores are slow
inline void mbar_wait(uint64_t* bar, uint32_t parity, unsigned* err, unsigned code) {
  const uint32_t b = smem_u32(bar);
  const long long t0 = clock64();
  for (unsigned it = 1;; ++it) {
    if (mbar_try(b, parity)) return;
    if (*reinterpret_cast<volatile unsigned*>(err) != 0u) return;
    if (clock64() - t0 > kWaitBudget) { atomicCAS(err, 0u, code); return; }
  }
}
inline void tma_load_4d(void* dst, const CUtensorMap* tm, uint64_t* bar, int x, int y, int z, int v) {
  chm_emu::tma_load_4d(dst, tm, bar, x, y, z, v);
}
inline uint64_t l2_policy_evict_first() { return 0; }
inline void tma_load_4d_hint(void* dst, const CUtensorMap* tm, uint64_t* bar, int x, int y, int z, int v, uint64_t) {
  chm_emu::tma_load_4d(dst, tm, bar, x, y, z, v);
}
inline bool mbar_arrive_is_last(uint64_t* bar) { return chm_emu::mbar_arrive(bar) == 1; }
inline void fence_mbar_init() {}
template <int COUNT> inline void named_barrier(int id) { chm_emu::sync_named(id, COUNT); }
#else
#define CHM_DYNAMIC_SMEM(name) extern __shared__ __align__(128) unsigned char name[]
// ---- TMA / mbarrier PTX wrappers ----------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  return ok != 0;
}
// Bounded wait.  A wrong expect_tx byte count, a TMA load that never lands or a refill that is never issued must
// end as an error code, not as a hung device: after kWaitBudget clock cycles (seconds; a whole launch takes
// milliseconds) the waiter records `code` in the handle's device error word and carries on WITHOUT the data --
// every address these kernels form depends on the tile index only, never on loaded values, so running on is
// memory-safe; the results are garbage and chemora_synchronize reports CHEMORA_ECUDA.  Once the word is set,
// every later wait of the launch gives up after its first 256 polls.
constexpr long long kWaitBudget = 4000000000LL;
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity, unsigned* err, unsigned code) {
  const uint32_t b = smem_u32(bar);
  if (mbar_try(b, parity)) return;
  const long long t0 = clock64();
#pragma unroll 1
  for (unsigned it = 1;; ++it) {
    if (mbar_try(b, parity)) return;
    if ((it & 255u) == 0u) {
      if (*reinterpret_cast<volatile unsigned*>(err) != 0u) return;
      if (clock64() - t0 > kWaitBudget) { atomicCAS(err, 0u, code); return; }
    }
  }
}
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* tm, uint64_t* bar, int x, int y, int z,
                                            int v) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(smem_u32(dst)), "l"(tm), "r"(smem_u32(bar)), "r"(x), "r"(y), "r"(z), "r"(v) : "memory");
}

__device__ __forceinline__ uint64_t l2_policy_evict_first() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ void tma_load_4d_hint(void* dst, const CUtensorMap* tm, uint64_t* bar, int x, int y, int z,
                                                 int v, uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
      " [%0], [%1, {%3, %4, %5, %6}], [%2], %7;"
      ::"r"(smem_u32(dst)), "l"(tm), "r"(smem_u32(bar)), "r"(x), "r"(y), "r"(z), "r"(v), "l"(policy) : "memory");
}
// One arrival on a "buffer released" mbarrier (expected count = number of warps); true if it was the last one of the
// phase (the state returned by arrive is the one before this arrival: one arrival pending = ours).  Release semantics
// order the warp's earlier reads of the buffer before the arrival; no MEMBAR is generated (SYNCS.ARRIVE).
__device__ __forceinline__ bool mbar_arrive_is_last(uint64_t* bar) {
  uint64_t state;
  uint32_t pending;
  asm volatile("mbarrier.arrive.shared::cta.b64 %0, [%1];" : "=l"(state) : "r"(smem_u32(bar)) : "memory");
  asm volatile("mbarrier.pending_count.b64 %0, %1;" : "=r"(pending) : "l"(state));
  return pending == 1;
}
// shared-memory counter increment, relaxed: no MEMBAR (an acq_rel atomic compiles to MEMBAR.ALL.CTA, which also
// waits for the warp's outstanding global stores).  The ordering needed -- this warp's LDS reads of a buffer
// before the increment -- comes from the SM executing one warp's shared-memory instructions in program order
// (the property the usual "LDS ... then mbarrier.arrive" consumer release relies on); the refill is an async
// TMA write issued after the last increment was observed.
__device__ __forceinline__ unsigned smem_add_relaxed(unsigned* p, unsigned v) {
  unsigned old;
  asm volatile("atom.relaxed.cta.shared::cta.add.u32 %0, [%1], %2;" : "=r"(old) : "r"(smem_u32(p)), "r"(v) : "memory");
  return old;
}

// mbarrier initialisation made visible to the async proxy (TMA) before the first load is issued
__device__ __forceinline__ void fence_mbar_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
// named barrier `id` (1..15) over COUNT threads
template <int COUNT>
__device__ __forceinline__ void named_barrier(int id) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(COUNT) : "memory");
}
#endif   // CHM_EMULATE

// ---- stencil reads from the staged box -------------------------------------------------------------------------
// `c` points at this thread's own grid point inside the current slot; BX, BY are the box row / plane extents.
template <int BX, int BY>
struct BoxPoint {
  const double* c;
  __device__ __forceinline__ double at(int di, int dj, int dk) const { return c[(dk * BY + dj) * BX + di]; }
  __device__ __forceinline__ double ax(int a, int m) const {
    return a == 0 ? at(m, 0, 0) : (a == 1 ? at(0, m, 0) : at(0, 0, m));
  }
  __device__ __forceinline__ double ax2(int a, int m, int b, int n) const {
    int d[3] = {0, 0, 0};
    d[a] = m; d[b] = n;
    return at(d[0], d[1], d[2]);
  }
};

// Star-shaped staging (sections that need only the three axis stencils: first derivatives, advection, dissipation):
// three slab boxes instead of the cuboid -- the tile + x-halo, the tile + y-halo, the tile + z-halo -- each a pointer
// to this thread's own point in it; SY, SZ are the y- and z-strides of the y- and z-slab (rows of TX + 2).
template <int SY, int SZ>
struct StarPoint {
  const double *cx, *cy, *cz;
  __device__ __forceinline__ double at(int, int, int) const { return cx[0]; }   // only ever the point itself
  __device__ __forceinline__ double ax(int a, int m) const { return a == 0 ? cx[m] : (a == 1 ? cy[m * SY] : cz[m * SZ]); }
};

// Per-point upwind/dissipation weights: beta^a d^up_a u + KO(u) = sum_a  wq[a] * q_a(u) + ws[a] * sp_a(u)
//   q_a  = s3 - 6 s2 + 15 s1   (s_k = (u[+k]-u0) + (u[-k]-u0))      symmetric 7-point (the KO stencil)
//   sp_a = 21 e1 - 6 e2 + e3   (e_k = u[+k] - u[-k])                 antisymmetric 7-point
// because the one-point-off-centre upwind stencils of reading S2 satisfy  up(+-) = (sp +- q) / 24h, so
//   wq[a] = |beta^a| / 24h + eps/64h ,   ws[a] = beta^a / 24h .
struct AdvW { double wq[3], ws[3]; };

// one axis of one variable: centred d1, d2 and the advection+dissipation contribution, all from 6 reads
template <class P>
__device__ __forceinline__ void axis_full(const P& p, double f0, int a, const Coef& C, const AdvW& w, double& d1,
                                          double& d2, double& ad) {
  const double p1 = p.ax(a, 1), m1 = p.ax(a, -1), p2 = p.ax(a, 2), m2 = p.ax(a, -2), p3 = p.ax(a, 3), m3 = p.ax(a, -3);
  const double e1 = p1 - m1, e2 = p2 - m2, e3 = p3 - m3;
  const double s1 = (p1 - f0) + (m1 - f0), s2 = (p2 - f0) + (m2 - f0), s3 = (p3 - f0) + (m3 - f0);
  d1 = (8.0 * e1 - e2) * (C.inv_h * (1.0 / 12.0));
  d2 = (16.0 * s1 - s2) * (C.inv_h2 * (1.0 / 12.0));
  const double q = (s3 - 6.0 * s2) + 15.0 * s1;
  const double sp = (21.0 * e1 - 6.0 * e2) + e3;
  const double c = w.wq[a] * q + w.ws[a] * sp;
  ad = a == 0 ? c : ad + c;   // axis 0 starts the sum (no 0.0 + c instruction)
}
template <class P>
__device__ __forceinline__ void axis_d1_ad(const P& p, double f0, int a, const Coef& C, const AdvW& w, double& d1,
                                           double& ad) {
  const double p1 = p.ax(a, 1), m1 = p.ax(a, -1), p2 = p.ax(a, 2), m2 = p.ax(a, -2), p3 = p.ax(a, 3), m3 = p.ax(a, -3);
  const double e1 = p1 - m1, e2 = p2 - m2, e3 = p3 - m3;
  const double s1 = (p1 - f0) + (m1 - f0), s2 = (p2 - f0) + (m2 - f0), s3 = (p3 - f0) + (m3 - f0);
  d1 = (8.0 * e1 - e2) * (C.inv_h * (1.0 / 12.0));
  const double q = (s3 - 6.0 * s2) + 15.0 * s1;
  const double sp = (21.0 * e1 - 6.0 * e2) + e3;
  const double c = w.wq[a] * q + w.ws[a] * sp;
  ad = a == 0 ? c : ad + c;   // axis 0 starts the sum (no 0.0 + c instruction)
}
template <class P>
__device__ __forceinline__ void axis_ad(const P& p, double f0, int a, const AdvW& w, double& ad) {
  const double p1 = p.ax(a, 1), m1 = p.ax(a, -1), p2 = p.ax(a, 2), m2 = p.ax(a, -2), p3 = p.ax(a, 3), m3 = p.ax(a, -3);
  const double e1 = p1 - m1, e2 = p2 - m2, e3 = p3 - m3;
  const double s1 = (p1 - f0) + (m1 - f0), s2 = (p2 - f0) + (m2 - f0), s3 = (p3 - f0) + (m3 - f0);
  const double q = (s3 - 6.0 * s2) + 15.0 * s1;
  const double sp = (21.0 * e1 - 6.0 * e2) + e3;
  const double c = w.wq[a] * q + w.ws[a] * sp;
  ad = a == 0 ? c : ad + c;   // axis 0 starts the sum (no 0.0 + c instruction)
}
// dissipation only (slot A): ko * q
template <class P>
__device__ __forceinline__ double axis_q(const P& p, double f0, int a) {
  const double s1 = (p.ax(a, 1) - f0) + (p.ax(a, -1) - f0), s2 = (p.ax(a, 2) - f0) + (p.ax(a, -2) - f0),
               s3 = (p.ax(a, 3) - f0) + (p.ax(a, -3) - f0);
  return (s3 - 6.0 * s2) + 15.0 * s1;
}
// mixed derivative d_a d_b (a != b), 16 reads
template <class P>
__device__ __forceinline__ double mixed(const P& p, int a, int b, const Coef& C) {
  double r[4];
  const int off[4] = {1, -1, 2, -2};
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    const int m = off[t];
    const double e1 = p.ax2(a, m, b, 1) - p.ax2(a, m, b, -1);
    const double e2 = p.ax2(a, m, b, 2) - p.ax2(a, m, b, -2);
    r[t] = 8.0 * e1 - e2;
  }
  return (8.0 * (r[0] - r[1]) - (r[2] - r[3])) * (C.inv_h2 * (1.0 / 144.0));
}

// all of one "full" variable (beta^i, gt_ij, chi, alpha): d1[3], packed d2[6], ad
template <class P>
__device__ __forceinline__ void var_full(const P& p, const Coef& C, const AdvW& w, double* d1, double* d2, double& ad) {
  const double f0 = p.at(0, 0, 0);
  axis_full(p, f0, 0, C, w, d1[0], d2[0], ad);
  axis_full(p, f0, 1, C, w, d1[1], d2[3], ad);
  axis_full(p, f0, 2, C, w, d1[2], d2[5], ad);
  d2[1] = mixed(p, 0, 1, C);
  d2[2] = mixed(p, 0, 2, C);
  d2[4] = mixed(p, 1, 2, C);
}
template <class P>
__device__ __forceinline__ void var_d1_ad(const P& p, const Coef& C, const AdvW& w, double* d1, double& ad) {
  const double f0 = p.at(0, 0, 0);
  axis_d1_ad(p, f0, 0, C, w, d1[0], ad);
  axis_d1_ad(p, f0, 1, C, w, d1[1], ad);
  axis_d1_ad(p, f0, 2, C, w, d1[2], ad);
}
template <class P>
__device__ __forceinline__ double var_ad(const P& p, const AdvW& w) {
  const double f0 = p.at(0, 0, 0);
  double ad;
  axis_ad(p, f0, 0, w, ad);
  axis_ad(p, f0, 1, w, ad);
  axis_ad(p, f0, 2, w, ad);
  return ad;
}

// ---- 8th order (the paper's configuration: 5 ghost zones) -------------------------------------
// Centred: d1 (3,-32,168,-672,0,672,-168,32,-3)/840h, d2 (-9,128,-1008,8064,-14350,...)/5040h^2.  The two one-sided
// upwind stencils over offsets -3..+5 (-5,60,-420,-378,1050,-420,140,-30,3)/840h split into an antisymmetric part
//   A = 735 e1 - 240 e2 + 72.5 e3 - 15 e4 + 1.5 e5   and a symmetric part   S = 315 s1 - 180 s2 + 67.5 s3 - 15 s4 + 1.5 s5
// (e_k = u[+k] - u[-k], s_k = (u[+k]-u0) + (u[-k]-u0)):  up(+-) = (A +- S)/840h, so
//   beta d^up u + KO(u) = ws A + wq S + sum_k kq_k s_k,   ws = beta/840h, wq = |beta|/840h,
// kq = the dissipation weights of Coef (order 5: ko (15, -6, 1, 0, 0); order 9, reading S6b: all five).
template <class P, bool D1, bool D2>
__device__ __forceinline__ void axis8(const P& p, double f0, int a, const Coef& C, const AdvW& w, double& d1, double& d2,
                                      double& ad) {
  double e[6], s[6];
#pragma unroll
  for (int k = 1; k <= 5; ++k) {
    const double pk = p.ax(a, k), mk = p.ax(a, -k);
    e[k] = pk - mk;
    s[k] = (pk - f0) + (mk - f0);
  }
  if (D1) d1 = ((672.0 * e[1] - 168.0 * e[2]) + (32.0 * e[3] - 3.0 * e[4])) * (C.inv_h * (1.0 / 840.0));
  if (D2) d2 = ((8064.0 * s[1] - 1008.0 * s[2]) + (128.0 * s[3] - 9.0 * s[4])) * (C.inv_h2 * (1.0 / 5040.0));
  const double A = ((735.0 * e[1] - 240.0 * e[2]) + (72.5 * e[3] - 15.0 * e[4])) + 1.5 * e[5];
  const double S = ((315.0 * s[1] - 180.0 * s[2]) + (67.5 * s[3] - 15.0 * s[4])) + 1.5 * s[5];
  const double q = ((C.kq[4] * s[5] + C.kq[3] * s[4]) + (C.kq[2] * s[3] + C.kq[1] * s[2])) + C.kq[0] * s[1];
  const double c = (w.ws[a] * A + w.wq[a] * S) + q;
  ad = a == 0 ? c : ad + c;
}
// dissipation alone along one axis (the inert slot A)
template <class P>
__device__ __forceinline__ double axis_ko8(const P& p, double f0, int a, const Coef& C) {
  double s[6];
#pragma unroll
  for (int k = 1; k <= 5; ++k) s[k] = (p.ax(a, k) - f0) + (p.ax(a, -k) - f0);
  return ((C.kq[4] * s[5] + C.kq[3] * s[4]) + (C.kq[2] * s[3] + C.kq[1] * s[2])) + C.kq[0] * s[1];
}
// mixed derivative d_a d_b (a != b) at 8th order, 64 reads
template <class P>
__device__ __forceinline__ double mixed8(const P& p, int a, int b, const Coef& C) {
  double r[8];
  const int off[8] = {1, -1, 2, -2, 3, -3, 4, -4};
#pragma unroll
  for (int t = 0; t < 8; ++t) {
    const int m = off[t];
    const double e1 = p.ax2(a, m, b, 1) - p.ax2(a, m, b, -1), e2 = p.ax2(a, m, b, 2) - p.ax2(a, m, b, -2);
    const double e3 = p.ax2(a, m, b, 3) - p.ax2(a, m, b, -3), e4 = p.ax2(a, m, b, 4) - p.ax2(a, m, b, -4);
    r[t] = (672.0 * e1 - 168.0 * e2) + (32.0 * e3 - 3.0 * e4);
  }
  return ((672.0 * (r[0] - r[1]) - 168.0 * (r[2] - r[3])) + (32.0 * (r[4] - r[5]) - 3.0 * (r[6] - r[7]))) *
         (C.inv_h2 * (1.0 / (840.0 * 840.0)));
}
template <class P>
__device__ __forceinline__ void var_full8(const P& p, const Coef& C, const AdvW& w, double* d1, double* d2, double& ad) {
  const double f0 = p.at(0, 0, 0);
  axis8<P, true, true>(p, f0, 0, C, w, d1[0], d2[0], ad);
  axis8<P, true, true>(p, f0, 1, C, w, d1[1], d2[3], ad);
  axis8<P, true, true>(p, f0, 2, C, w, d1[2], d2[5], ad);
  d2[1] = mixed8(p, 0, 1, C);
  d2[2] = mixed8(p, 0, 2, C);
  d2[4] = mixed8(p, 1, 2, C);
}
template <class P>
__device__ __forceinline__ void var_d1_ad8(const P& p, const Coef& C, const AdvW& w, double* d1, double& ad) {
  const double f0 = p.at(0, 0, 0);
  double dummy;
  axis8<P, true, false>(p, f0, 0, C, w, d1[0], dummy, ad);
  axis8<P, true, false>(p, f0, 1, C, w, d1[1], dummy, ad);
  axis8<P, true, false>(p, f0, 2, C, w, d1[2], dummy, ad);
}
template <class P>
__device__ __forceinline__ double var_ad8(const P& p, const Coef& C, const AdvW& w) {
  const double f0 = p.at(0, 0, 0);
  double ad, dummy;
  axis8<P, false, false>(p, f0, 0, C, w, dummy, dummy, ad);
  axis8<P, false, false>(p, f0, 1, C, w, dummy, dummy, ad);
  axis8<P, false, false>(p, f0, 2, C, w, dummy, dummy, ad);
  return ad;
}

// consumption order of the 25 variables (slot of order index o is o % 5)
__host__ __device__ __forceinline__ constexpr int order_var(int o) {
  return o < 3 ? V_BETA + o : o < 9 ? V_GT + (o - 3) : o < 12 ? V_GAM + (o - 9) : o == 12 ? V_CHI : o == 13 ? V_ALPHA
         : o == 14 ? V_K : o < 21 ? V_AT + (o - 15) : o < 24 ? V_B + (o - 21) : V_A;
}

}  // namespace chm
