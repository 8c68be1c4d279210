// kernels_bssn_ws.cu -- warp-specialised form of the fused BSSN kernel (derivatives + RHS + RK4 stage), sm_100a.
//
// Same mathematics, tile traversal and TMA box ring as kernels_bssn_tma.cu, but the CTA has 12 warps in two roles:
//   * 8 "point" warps (one grid point per thread, 216 registers after setmaxnreg.inc) evaluate the stencils of the
//     11 variables whose second derivatives are needed (beta^i, gt_ij, chi, alpha) and the whole pointwise
//     expression, and emit every right-hand side through the fused RK4 stage update;
//   * 4 "stencil" warps (two grid points per thread, 72 registers after setmaxnreg.dec) evaluate the stencils of
//     the other 14 variables (Gt^i, K: first derivatives + advection/dissipation; At_ij, B^i, A: advection/
//     dissipation only) and hand the 29 resulting values per point to the point warps through shared memory.
// The fused kernel is bound by the latency of its own LDS -> FP64 chains at 8 warps per SM (254 registers); the
// stencil warps add a third warp to every scheduler without costing the point warps their registers, and take
// 20 % of the instruction stream off them.  PAPER.md:268-270 ("fat kernels") is the problem this addresses.
#include "bssn_tma.cuh"

namespace chm {

namespace ws {

constexpr int kSlots = 6;     // 3 box slots per role
constexpr int kCenVars = 21;
__device__ __forceinline__ constexpr int cen_index(int v) { return v < 14 ? v : v - 3; }
constexpr int kLines = 29;    // result lines (one double per point each) handed from stencil to point warps
constexpr int kRes = 14;      // variables produced by the stencil warps
// is section o evaluated by the stencil warps?
__device__ __forceinline__ constexpr bool produced(int o) { return (o >= 9 && o <= 11) || o >= 14; }
__device__ __forceinline__ constexpr int ridx(int o) { return o <= 11 ? o - 9 : o - 11; }
__device__ __forceinline__ constexpr int line0(int o) {
  return o <= 11 ? 4 * (o - 9) : o == 14 ? 12 : o <= 20 ? 16 + (o - 15) : o <= 23 ? 22 + 2 * (o - 21) : 28;
}

// Two independent box rings of kRing slots each, one per role, so the stencil warps run decoupled from the point
// warps (up to a tile ahead, bounded by the result lines).  Ring position c = 0..10 of the point warps' 11 boxes
// and p = 0..13 of the stencil warps' 14 boxes; slot = position % kRing, so a slot is used ring_uses(n, slot)
// times per tile and the mbarrier parity of a use follows from the tile count and the position.
constexpr int kRing = 3, kNumP = 11, kNumS = 14;
__device__ __forceinline__ constexpr int point_o(int c) { return c < 9 ? c : 12 + (c - 9); }
__device__ __forceinline__ constexpr int point_c(int o) { return o < 9 ? o : 9 + (o - 12); }
__device__ __forceinline__ constexpr int stencil_o(int p) { return p < 3 ? 9 + p : 14 + (p - 3); }
__device__ __forceinline__ constexpr int ring_uses(int n, int slot) { return (n - slot + kRing - 1) / kRing; }

template <int TX, int TY, int TZ>
struct Cfg {
  static_assert(TX * TY * TZ == 256, "8 point warps, one grid point per thread");
  static_assert(TX % 2 == 0 && ((TX + 2) * TY * TZ) % 16 == 0, "tile boxes must stay 128-byte aligned in smem");
  static constexpr int BX = TX + 6, BY = TY + 6, BZ = TZ + 6;
  static constexpr int SLOT = (BX * BY * BZ + 15) / 16 * 16;
  static constexpr uint32_t BOX_BYTES = (uint32_t)BX * BY * BZ * 8u;
  static constexpr int NPT = 256, NPROD = 128, THREADS = NPT + NPROD;
  static constexpr int TILE = (TX + 2) * TY * TZ;
  static constexpr uint32_t TILE_BYTES = (uint32_t)TILE * 8u;
  static constexpr int CEN = kCenVars * TILE;
  static constexpr int RES = kLines * NPT;
  static constexpr int NBAR = kSlots + 1 + 2 * kRes;          // fullP[3], fullS[3], cfull, rfull[14], rempty[14]
  static constexpr int NCNT = kSlots + 1;                     // point-warp / stencil-warp slot counters, cen
  static constexpr size_t SMEM = (size_t)(kSlots * SLOT + CEN + RES) * 8 + NBAR * 8 + NCNT * 4 + 128;
};

__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

}  // namespace ws

template <int TX, int TY, int TZ>
__global__ void __launch_bounds__(384, 1)
bssn_ws_kernel(const __grid_constant__ CUtensorMap tm, const __grid_constant__ CUtensorMap tmCen, Layout L, Coef C,
               Stage st, int ntx, int nty, int ntz, int cy) {
  using namespace ws;
  using K = Cfg<TX, TY, TZ>;
  constexpr int BX = K::BX, BY = K::BY, SLOT = K::SLOT, TILE = K::TILE, NPT = K::NPT;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double* sm = reinterpret_cast<double*>(smem_raw);
  double* cbuf = sm + kSlots * SLOT;                                   // [kCenVars][TILE] point values
  double* res = cbuf + K::CEN;                                         // [kLines][NPT]
  uint64_t* fullP = reinterpret_cast<uint64_t*>(res + K::RES);         // [kRing] box for the point warps arrived
  uint64_t* fullS = fullP + kRing;                                     // [kRing] box for the stencil warps arrived
  uint64_t* cfull = fullS + kRing;
  uint64_t* rfull = cfull + 1;                                         // [kRes] results written
  uint64_t* rempty = rfull + kRes;                                     // [kRes] results read
  unsigned* cntP = reinterpret_cast<unsigned*>(rempty + kRes);         // [kRing] point warps that left a slot
  unsigned* cntS = cntP + kRing;                                       // [kRing] stencil warps that left a slot
  unsigned* cntC = cntS + kRing;                                      // warps (all 12) that left the point values
  const int ntiles = ntx * nty * ntz;
  const int tid = threadIdx.x, lane = tid & 31;
  const bool point_role = tid < NPT;
  const int goffx = L.xo - 3, goff = L.g - 3;

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < kSlots + 1; ++s) mbar_init(&fullP[s], 1);
#pragma unroll
    for (int s = 0; s < kRes; ++s) { mbar_init(&rfull[s], 4); mbar_init(&rempty[s], 8); }
#pragma unroll
    for (int s = 0; s < K::NCNT; ++s) cntP[s] = 0u;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();

  // tile order: columns of cy tile rows (full x extent), z-layers inside a column, then y, then x
  auto decode = [&](int idx, int& bx, int& by, int& bz) {
    const int per_col = ntx * cy * ntz;
    const int c = idx / per_col;
    int r = idx - c * per_col;
    const int cyt = min(cy, nty - c * cy), layer = ntx * cyt;
    bz = r / layer; r -= bz * layer;
    const int ry = r / ntx;
    by = c * cy + ry; bx = r - ry * ntx;
  };
  // box of section o into ring slot `slot` of the point (slots 0..2) or stencil (slots 3..5) ring
  auto issue_point = [&](int c, int x0, int y0, int z0) {
    const int slot = c % kRing;
    mbar_expect_tx(&fullP[slot], K::BOX_BYTES);
    tma_load_4d(sm + slot * SLOT, &tm, &fullP[slot], x0, y0, z0, order_var(point_o(c)));
  };
  auto issue_stencil = [&](int p, int x0, int y0, int z0) {
    const int slot = p % kRing;
    mbar_expect_tx(&fullS[slot], K::BOX_BYTES);
    tma_load_4d(sm + (kRing + slot) * SLOT, &tm, &fullS[slot], x0, y0, z0, order_var(stencil_o(p)));
  };
  auto issue_cen = [&](int x0, int y0, int z0) {
    mbar_expect_tx(cfull, (uint32_t)kCenVars * K::TILE_BYTES);
    tma_load_4d(cbuf, &tmCen, cfull, x0 + 2, y0 + 3, z0 + 3, 0);
    tma_load_4d(cbuf + 7 * TILE, &tmCen, cfull, x0 + 2, y0 + 3, z0 + 3, 7);
    tma_load_4d(cbuf + 14 * TILE, &tmCen, cfull, x0 + 2, y0 + 3, z0 + 3, 17);
  };
  // one warp leaves a buffer; true for lane 0 of the last of `nw` warps (see smem_add_relaxed)
  auto leave = [&](unsigned* counter, unsigned nw) {
    __syncwarp();
    bool last = false;
    if (lane == 0) last = (smem_add_relaxed(counter, 1u) + 1u) % nw == 0u;
    return last;
  };
  if (tid == 0 && (int)blockIdx.x < ntiles) {
    int bx, by, bz;
    decode(blockIdx.x, bx, by, bz);
    const int x0 = bx * TX + goffx, y0 = by * TY + goff, z0 = bz * TZ + goff;
    issue_cen(x0, y0, z0);
#pragma unroll
    for (int c = 0; c < kRing; ++c) { issue_point(c, x0, y0, z0); issue_stencil(c, x0, y0, z0); }
  }
  __syncthreads();   // every warp converged before the role split (setmaxnreg is .sync.aligned)

  if (!point_role) {
    // =============================== stencil warps: two grid points per thread ===============================
    asm volatile("setmaxnreg.dec.sync.aligned.u32 72;");
    const int ptid = tid - NPT;
    int coffS[2], toffS[2];
#pragma unroll
    for (int n = 0; n < 2; ++n) {
      const int pid = ptid + n * K::NPROD;
      const int lx = pid % TX, ly = (pid / TX) % TY, lz = pid / (TX * TY);
      coffS[n] = ((lz + 3) * BY + (ly + 3)) * BX + lx + 3;
      toffS[n] = (lz * TY + ly) * (TX + 2) + lx + 1;
    }
    int t = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++t) {
      int bx, by, bz;
      decode(tile, bx, by, bz);
      const bool has_next = tile + (int)gridDim.x < ntiles;
      int nx0 = 0, ny0 = 0, nz0 = 0;
      if (has_next) {
        int b0, b1, b2;
        decode(tile + gridDim.x, b0, b1, b2);
        nx0 = b0 * TX + goffx; ny0 = b1 * TY + goff; nz0 = b2 * TZ + goff;
      }
      mbar_wait(cfull, (uint32_t)(t & 1));
      AdvW w[2];
#pragma unroll
      for (int n = 0; n < 2; ++n)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
          const double b = cbuf[cen_index(V_BETA + a) * TILE + toffS[n]];
          w[n].ws[a] = b * (C.inv_h * (1.0 / 24.0));
          w[n].wq[a] = fabs(b) * (C.inv_h * (1.0 / 24.0)) + C.ko;
        }
      if (leave(cntC, 12u) && has_next) issue_cen(nx0, ny0, nz0);

#pragma unroll
      for (int ps = 0; ps < kNumS; ++ps) {
        const int o = stencil_o(ps);
        const int slot = ps % kRing;
        mbar_wait(&fullS[slot], (uint32_t)((t * ring_uses(kNumS, slot) + ps / kRing) & 1));
        if (t > 0) mbar_wait(&rempty[ridx(o)], (uint32_t)((t - 1) & 1));
#pragma unroll
        for (int n = 0; n < 2; ++n) {
          const BoxPoint<BX, BY> p{sm + (kRing + slot) * SLOT + coffS[n]};
          double* r = res + line0(o) * NPT + ptid + n * K::NPROD;
          if (o <= 14) {                       // Gt^k, K: centred first derivatives + advection/dissipation
            double d1[3], ad;
            var_d1_ad(p, C, w[n], d1, ad);
            r[0] = d1[0]; r[NPT] = d1[1]; r[2 * NPT] = d1[2]; r[3 * NPT] = ad;
          } else if (o <= 20) {                // At_ij
            r[0] = var_ad(p, w[n]);
          } else if (o <= 23) {                // B^i: advection/dissipation and the point value
            r[0] = var_ad(p, w[n]);
            r[NPT] = p.at(0, 0, 0);
          } else {                             // A: dissipation only
            const double f0 = p.at(0, 0, 0);
            r[0] = C.ko * ((axis_q(p, f0, 0) + axis_q(p, f0, 1)) + axis_q(p, f0, 2));
          }
        }
        if (leave(&cntS[slot], 4u)) {   // the last stencil warp out refills the slot, 3 boxes ahead
          if (ps + kRing < kNumS) issue_stencil(ps + kRing, bx * TX + goffx, by * TY + goff, bz * TZ + goff);
          else if (has_next) issue_stencil(ps % kRing, nx0, ny0, nz0);
        }
        if (lane == 0) mbar_arrive(&rfull[ridx(o)]);   // after the __syncwarp in leave(): the warp's results are written
      }
    }
    return;
  }

  // ================================= point warps: one grid point per thread =================================
  asm volatile("setmaxnreg.inc.sync.aligned.u32 216;");
  const int lx = tid % TX, ly = (tid / TX) % TY, lz = tid / (TX * TY);
  const int coff = ((lz + 3) * BY + (ly + 3)) * BX + lx + 3;
  const int toff = (lz * TY + ly) * (TX + 2) + lx + 1;   // this thread's point inside a tile box
  const double* cb = cbuf + toff;
  const double* rs = res + tid;                          // this thread's column of the result lines
  int t = 0;
  for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++t) {
    int bx, by, bz;
    decode(tile, bx, by, bz);
    const int i = bx * TX + lx, j = by * TY + ly, k = bz * TZ + lz;
    const bool valid = i < L.nx && j < L.ny && k < L.nz;
    const long q = (long)((valid ? k : 0) + L.g) * L.plane + (long)((valid ? j : 0) + L.g) * L.pitch +
                   ((valid ? i : 0) + L.xo);
    auto cen = [&](int v) { return cb[cen_index(v) * TILE]; };
    // RK4 stage operands (U, S) of variable v at this point: global loads issued at the top of the section that
    // emits v, consumed at its end
    auto pre = [&](int v) {
      StagePre pr{0.0, 0.0};
      const long qq = q + v * L.vstride;
      if (st.mode == MODE_FIRST) pr.u = __ldg(st.in + qq);
      else if (st.mode == MODE_SSP) { pr.u = __ldcs(st.U + qq); pr.s = __ldg(st.in + qq); }
      else if (st.mode != MODE_RHS) { pr.u = __ldcs(st.U + qq); pr.s = __ldcs(st.S + qq); }
      return pr;
    };
    auto emit = [&](int v, double kk, const StagePre& pr) { if (valid) stage_emit(st, q + v * L.vstride, kk, pr); };
    auto box = [&](int o) {
      const int c = point_c(o), slot = c % kRing;
      mbar_wait(&fullP[slot], (uint32_t)((t * ring_uses(kNumP, slot) + c / kRing) & 1));
      return BoxPoint<BX, BY>{sm + slot * SLOT + coff};
    };
    const bool has_next = tile + (int)gridDim.x < ntiles;
    int nx0 = 0, ny0 = 0, nz0 = 0;           // origin of this CTA's next tile
    if (has_next) {
      int b0, b1, b2;
      decode(tile + gridDim.x, b0, b1, b2);
      nx0 = b0 * TX + goffx; ny0 = b1 * TY + goff; nz0 = b2 * TZ + goff;
    }
    // this warp leaves the box of section o; the last point warp refills the slot 5 loads ahead
    auto done = [&](int o) {
      const int c = point_c(o);
      if (leave(&cntP[c % kRing], 8u)) {
        if (c + kRing < kNumP) issue_point(c + kRing, bx * TX + goffx, by * TY + goff, bz * TZ + goff);
        else if (has_next) issue_point(c % kRing, nx0, ny0, nz0);
      }
    };
    // results of a section evaluated by the stencil warps: wait for them / hand the lines back
    auto results = [&](int o) { mbar_wait(&rfull[ridx(o)], (uint32_t)(t & 1)); return rs + line0(o) * NPT; };
    auto results_done = [&](int o) {
      __syncwarp();
      if (lane == 0) mbar_arrive(&rempty[ridx(o)]);
    };

    const double third = 1.0 / 3.0, two_thirds = 2.0 / 3.0;
    mbar_wait(cfull, (uint32_t)(t & 1));
    // ---- point values needed before their own boxes arrive: metric, shift ----------------------------------
    double g[6], gu[6];
#pragma unroll
    for (int s = 0; s < 6; ++s) g[s] = cen(V_GT + s);
    {
      const double c00 = g[3] * g[5] - g[4] * g[4], c01 = g[2] * g[4] - g[1] * g[5], c02 = g[1] * g[4] - g[2] * g[3];
      const double idet = 1.0 / (g[0] * c00 + g[1] * c01 + g[2] * c02);
      gu[0] = c00 * idet; gu[1] = c01 * idet; gu[2] = c02 * idet;
      gu[3] = (g[0] * g[5] - g[2] * g[2]) * idet;
      gu[4] = (g[1] * g[2] - g[0] * g[4]) * idet;
      gu[5] = (g[0] * g[3] - g[1] * g[1]) * idet;
    }
    AdvW w;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const double b = cen(V_BETA + a);
      w.ws[a] = b * (C.inv_h * (1.0 / 24.0));
      w.wq[a] = fabs(b) * (C.inv_h * (1.0 / 24.0)) + C.ko;
    }
    const double alpha = cen(V_ALPHA), trK = cen(V_K), chi = cen(V_CHI);

    // ---- o = 0..2: beta^i : d_j beta^i, gtu^{jk} d_j d_k beta^i, d_j (d_k beta^k) ----------------------------
    double db[3][3], lapb[3], gdiv[3];   // db[j][i] = d_j beta^i ; gdiv[j] = d_j d_k beta^k
#pragma unroll
    for (int i2 = 0; i2 < 3; ++i2) {
      const double Bc = cen(V_B + i2);
      const StagePre pr = pre(V_BETA + i2);
      auto p = box(i2);
      double d1[3], d2[6], ad;
      var_full(p, C, w, d1, d2, ad);
      done(i2);
#pragma unroll
      for (int a = 0; a < 3; ++a) { db[a][i2] = d1[a]; gdiv[a] = i2 == 0 ? d2[sym(a, i2)] : gdiv[a] + d2[sym(a, i2)]; }
      lapb[i2] = sdot(gu, d2);
      emit(V_BETA + i2, C.sgc * Bc + ad, pr);
    }
    const double divb = (db[0][0] + db[1][1]) + db[2][2];

    // ---- o = 3..8: gt_ij : d_k gt_ij kept for the Christoffels, gtu^{lm} d_l d_m gt_ij folded into R~_ij ---
    double At[6], Rt[6], dg[3][6];
#pragma unroll
    for (int s = 0; s < 6; ++s) At[s] = cen(V_AT + s);
    if (leave(cntC, 12u) && has_next) issue_cen(nx0, ny0, nz0);   // last read of the point values
#pragma unroll
    for (int i2 = 0; i2 < 3; ++i2)
#pragma unroll
      for (int j2 = i2; j2 < 3; ++j2) {
        const int s = sym(i2, j2);
        const StagePre pr = pre(V_GT + s);
        auto p = box(3 + s);
        double d1[3], d2[6], ad;
        var_full(p, C, w, d1, d2, ad);
        done(3 + s);
        dg[0][s] = d1[0]; dg[1][s] = d1[1]; dg[2][s] = d1[2];
        Rt[s] = -0.5 * sdot(gu, d2);
        double lie;
#pragma unroll
        for (int k2 = 0; k2 < 3; ++k2) {
          const double c = g[sym(i2, k2)] * db[j2][k2] + g[sym(j2, k2)] * db[i2][k2];
          lie = k2 == 0 ? c : lie + c;
        }
        emit(V_GT + s, (lie - two_thirds * g[s] * divb) - 2.0 * alpha * At[s] + ad, pr);
      }

    // ---- Christoffels: Cl[k][s(i,j)] = Gamma~_kij, Cu[k][s] = Gamma~^k_ij, Gn[k] = gtu^{ij} Gamma~^k_ij ----
    double Cu[3][6], Gn[3];
    {
      double Cl[3][6];
#pragma unroll
      for (int k2 = 0; k2 < 3; ++k2)
#pragma unroll
        for (int i2 = 0; i2 < 3; ++i2)
#pragma unroll
          for (int j2 = i2; j2 < 3; ++j2)
            Cl[k2][sym(i2, j2)] = 0.5 * ((dg[i2][sym(k2, j2)] + dg[j2][sym(k2, i2)]) - dg[k2][sym(i2, j2)]);
#pragma unroll
      for (int k2 = 0; k2 < 3; ++k2) {
#pragma unroll
        for (int s = 0; s < 6; ++s)
          Cu[k2][s] = gu[sym(k2, 0)] * Cl[0][s] + gu[sym(k2, 1)] * Cl[1][s] + gu[sym(k2, 2)] * Cl[2][s];
        Gn[k2] = sdot(gu, Cu[k2]);
      }
      // R~_ij += 1/2 Gamma~^k_n (Gamma~_ijk + Gamma~_jik)
      //        + gtu^{lm} (Gamma~^k_li Gamma~_jkm + Gamma~^k_lj Gamma~_ikm + Gamma~^k_im Gamma~_klj)
      // with the inverse metric contracted once: W[i][m] = gtu^{lm} Gamma~^k_li (per k), so the three products are
      //   sum_m W[i][m] Gamma~_jkm + W[j][m] Gamma~_ikm   and   sum_l W[i][l] Gamma~_klj
#pragma unroll
      for (int i2 = 0; i2 < 3; ++i2)
#pragma unroll
        for (int j2 = i2; j2 < 3; ++j2) {
          const double c = (Gn[0] * (Cl[i2][sym(j2, 0)] + Cl[j2][sym(i2, 0)]) +
                            Gn[1] * (Cl[i2][sym(j2, 1)] + Cl[j2][sym(i2, 1)])) +
                           Gn[2] * (Cl[i2][sym(j2, 2)] + Cl[j2][sym(i2, 2)]);
          Rt[sym(i2, j2)] += 0.5 * c;
        }
#pragma unroll
      for (int k2 = 0; k2 < 3; ++k2) {
        double W[3][3];
#pragma unroll
        for (int i2 = 0; i2 < 3; ++i2)
#pragma unroll
          for (int m = 0; m < 3; ++m)
            W[i2][m] = gu[sym(0, m)] * Cu[k2][sym(0, i2)] + gu[sym(1, m)] * Cu[k2][sym(1, i2)] +
                       gu[sym(2, m)] * Cu[k2][sym(2, i2)];
#pragma unroll
        for (int i2 = 0; i2 < 3; ++i2)
#pragma unroll
          for (int j2 = i2; j2 < 3; ++j2) {
            double acc = W[i2][0] * Cl[k2][sym(0, j2)] + W[i2][1] * Cl[k2][sym(1, j2)] + W[i2][2] * Cl[k2][sym(2, j2)];
            const double t1 = W[i2][0] * Cl[j2][sym(k2, 0)] + W[i2][1] * Cl[j2][sym(k2, 1)] + W[i2][2] * Cl[j2][sym(k2, 2)];
            if (i2 == j2) acc += 2.0 * t1;
            else acc += t1 + (W[j2][0] * Cl[i2][sym(k2, 0)] + W[j2][1] * Cl[i2][sym(k2, 1)] + W[j2][2] * Cl[i2][sym(k2, 2)]);
            Rt[sym(i2, j2)] += acc;
          }
      }
    }

    // ---- o = 9..11: Gt^k (stencil warps): R~_ij += 1/2 (gt_ki d_j Gt^k + gt_kj d_i Gt^k) ---------------------
    // (the advection of Gt^k is read at the end, where it is used)
#pragma unroll
    for (int k2 = 0; k2 < 3; ++k2) {
      const double* r = results(9 + k2);
      const double d1[3] = {r[0], r[NPT], r[2 * NPT]};
#pragma unroll
      for (int i2 = 0; i2 < 3; ++i2)
#pragma unroll
        for (int j2 = i2; j2 < 3; ++j2)
          Rt[sym(i2, j2)] += 0.5 * (g[sym(k2, i2)] * d1[j2] + g[sym(k2, j2)] * d1[i2]);
    }

    // ---- o = 12: chi : R_ij = R~_ij + R^chi_ij --------------------------------------------------------------
    const double ichi = 1.0 / chi;
    double dchi[3];
    {
      const StagePre pr = pre(V_CHI);
      auto p = box(12);
      double d2[6], ad;
      var_full(p, C, w, dchi, d2, ad);
      done(12);
      emit(V_CHI, two_thirds * chi * (alpha * trK - divb) + ad, pr);
      double cd[6], cc[6];   // D~_i D~_j chi ; d_i chi d_j chi
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = a; b < 3; ++b) {
          const int s = sym(a, b);
          cd[s] = d2[s] - (Cu[0][s] * dchi[0] + Cu[1][s] * dchi[1] + Cu[2][s] * dchi[2]);
          cc[s] = dchi[a] * dchi[b];
        }
      const double trcd = sdot(gu, cd), trcc = sdot(gu, cc);
      const double h2 = 0.5 * ichi, h4 = 0.25 * ichi * ichi;
#pragma unroll
      for (int s = 0; s < 6; ++s) Rt[s] += h2 * (cd[s] + g[s] * trcd) - h4 * (cc[s] + 3.0 * g[s] * trcc);
    }

    // ---- o = 13: alpha : X_ij = alpha R_ij - D_i D_j alpha ; D^2 alpha -----------------------------------------
    double dal[3], lap_alpha;
    {
      const StagePre pr = pre(V_ALPHA);
      auto p = box(13);
      double d2[6], ad;
      var_full(p, C, w, dal, d2, ad);
      done(13);
      emit(V_ALPHA, -2.0 * alpha * trK + ad, pr);
      double cd[6], ca[6];   // d_i d_j alpha - Gamma~^k_ij d_k alpha ; d_i chi d_j alpha + d_j chi d_i alpha
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = a; b < 3; ++b) {
          const int s = sym(a, b);
          cd[s] = d2[s] - (Cu[0][s] * dal[0] + Cu[1][s] * dal[1] + Cu[2][s] * dal[2]);
          ca[s] = dchi[a] * dal[b] + dchi[b] * dal[a];
        }
      const double trcd = sdot(gu, cd), trca = 0.5 * sdot(gu, ca);   // trca = gtu^{kl} d_k chi d_l alpha
      lap_alpha = chi * trcd - 0.5 * trca;
      const double h2 = 0.5 * ichi;
#pragma unroll
      for (int s = 0; s < 6; ++s) Rt[s] = alpha * Rt[s] - (cd[s] + h2 * (ca[s] - g[s] * trca));   // Rt now holds X_ij
    }

    // ---- extrinsic curvature with raised indices -------------------------------------------------------------
    double Am[3][3], Au[6];   // At^i_j ; At^{ij}
#pragma unroll
    for (int i2 = 0; i2 < 3; ++i2)
#pragma unroll
      for (int j2 = 0; j2 < 3; ++j2)
        Am[i2][j2] = gu[sym(i2, 0)] * At[sym(0, j2)] + gu[sym(i2, 1)] * At[sym(1, j2)] + gu[sym(i2, 2)] * At[sym(2, j2)];
#pragma unroll
    for (int i2 = 0; i2 < 3; ++i2)
#pragma unroll
      for (int j2 = i2; j2 < 3; ++j2)
        Au[sym(i2, j2)] = Am[i2][0] * gu[sym(0, j2)] + Am[i2][1] * gu[sym(1, j2)] + Am[i2][2] * gu[sym(2, j2)];

    // ---- o = 14: K (stencil warps; its first derivatives are read at the end, where they are used) -----------
    {
      const StagePre pr = pre(V_K);
      const double ad = results(14)[3 * NPT];
      emit(V_K, (alpha * (sdot(Au, At) + third * trK * trK) - lap_alpha) + ad, pr);
    }

    // ---- o = 15..20: At_ij (stencil warps) ------------------------------------------------------------------------
    {
      const double trX = sdot(gu, Rt);
#pragma unroll
      for (int i2 = 0; i2 < 3; ++i2)
#pragma unroll
        for (int j2 = i2; j2 < 3; ++j2) {
          const int s = sym(i2, j2);
          const StagePre pr = pre(V_AT + s);
          double AA, lie;
#pragma unroll
          for (int k2 = 0; k2 < 3; ++k2) {
            const double c = At[sym(i2, k2)] * db[j2][k2] + At[sym(j2, k2)] * db[i2][k2];
            AA = k2 == 0 ? At[sym(i2, k2)] * Am[k2][j2] : AA + At[sym(i2, k2)] * Am[k2][j2];
            lie = k2 == 0 ? c : lie + c;
          }
          const double ad = results(15 + s)[0];
          results_done(15 + s);
          emit(V_AT + s, chi * (Rt[s] - third * g[s] * trX) + alpha * (trK * At[s] - 2.0 * AA) +
                             (lie - two_thirds * At[s] * divb) + ad, pr);
        }
    }

    // ---- o = 21..23: B^i, together with Gt^i (stencil warps) -----------------------------------------------------
    double dK[3];
    {
      const double* r = results(14);
      dK[0] = r[0]; dK[1] = r[NPT]; dK[2] = r[2 * NPT];
      results_done(14);
    }
#pragma unroll
    for (int i2 = 0; i2 < 3; ++i2) {
      const StagePre prG = pre(V_GAM + i2), prB = pre(V_B + i2);
      double rr = lapb[i2];
      double t2 = sdot(Cu[i2], Au);   // Gamma~^i_jk At^{jk}
#pragma unroll
      for (int j2 = 0; j2 < 3; ++j2) {
        rr += third * gu[sym(i2, j2)] * gdiv[j2];
        t2 -= two_thirds * gu[sym(i2, j2)] * dK[j2] + 1.5 * ichi * Au[sym(i2, j2)] * dchi[j2];
        rr -= 2.0 * Au[sym(i2, j2)] * dal[j2] + Gn[j2] * db[j2][i2];
      }
      rr += 2.0 * alpha * t2 + two_thirds * Gn[i2] * divb;
      const double adG = results(9 + i2)[3 * NPT];
      results_done(9 + i2);
      const double* rb = results(21 + i2);
      const double adB = rb[0], Bi = rb[NPT];
      results_done(21 + i2);
      emit(V_GAM + i2, rr + adG, prG);
      emit(V_B + i2, (rr - C.eta * Bi) + adB, prB);
    }

    // ---- o = 24: A (inert slot, dissipation only; stencil warps) -------------------------------------------------
    {
      const StagePre pr = pre(V_A);
      const double kA = results(24)[0];
      results_done(24);
      emit(V_A, kA, pr);
    }
  }
}

// ---- host side: tensor maps + launch ---------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn ws_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  }
  return fn;
}

template <int TX, int TY, int TZ>
static cudaError_t ws_go(const Layout& L, const Coef& C, const Stage* st, cudaStream_t s, cudaFuncAttributes* a) {
  using K = ws::Cfg<TX, TY, TZ>;
  auto kern = bssn_ws_kernel<TX, TY, TZ>;
  if (a) return cudaFuncGetAttributes(a, kern);
  EncodeTiledFn enc = ws_encode_fn();
  if (!enc) return cudaErrorNotSupported;
  CUtensorMap tm, tmCen;
  cuuint64_t dims[4] = {(cuuint64_t)L.pitch, (cuuint64_t)L.tot_y, (cuuint64_t)L.tot_z, (cuuint64_t)L.nvars};
  cuuint64_t strides[3] = {(cuuint64_t)L.pitch * 8, (cuuint64_t)L.plane * 8, (cuuint64_t)L.vstride * 8};
  cuuint32_t estr[4] = {1, 1, 1, 1};
  cuuint32_t box[4] = {(cuuint32_t)K::BX, (cuuint32_t)K::BY, (cuuint32_t)K::BZ, 1};
  cuuint32_t cbox[4] = {(cuuint32_t)(TX + 2), (cuuint32_t)TY, (cuuint32_t)TZ, 7};
  if (enc(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<double*>(st->in), dims, strides, box, estr,
          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS ||
      enc(&tmCen, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<double*>(st->in), dims, strides, cbox, estr,
          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)K::SMEM);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int ntx = (L.nx + TX - 1) / TX, nty = (L.ny + TY - 1) / TY, ntz = (L.nz + TZ - 1) / TZ;
  const int ntiles = ntx * nty * ntz;
  const int grid = ntiles < sms ? ntiles : sms;              // persistent: one CTA per SM
  const int cy = L.col_rows / TY > 0 ? L.col_rows / TY : 1;   // tile rows per traversal column
  kern<<<grid, K::THREADS, K::SMEM, s>>>(tm, tmCen, L, C, *st, ntx, nty, ntz, cy);
  return cudaGetLastError();
}

static cudaError_t ws_dispatch(int which, const Layout& L, const Coef& C, const Stage* st, cudaStream_t s,
                               cudaFuncAttributes* a) {
  switch (which) {
    case 0: return ws_go<16, 4, 4>(L, C, st, s, a);
    case 1: return ws_go<16, 8, 2>(L, C, st, s, a);
    case 2: return ws_go<16, 2, 8>(L, C, st, s, a);
  }
  return cudaErrorInvalidValue;
}

cudaError_t launch_bssn_ws(const Layout& L, const Coef& C, int which, const Stage& st, cudaStream_t s) {
  return ws_dispatch(which, L, C, &st, s, nullptr);
}
cudaError_t kernel_info_bssn_ws(int which, cudaFuncAttributes* a) {
  Layout L{}; Coef C{};
  return ws_dispatch(which, L, C, nullptr, 0, a);
}

}  // namespace chm

