// kernels_bssn_tma.cu -- the fused BSSN kernel (derivatives + RHS + RK4 stage update), sm_100a:
// persistent CTAs, TMA-staged per-variable boxes in a 5-slot mbarrier ring, compile-time stencil offsets.
// No block-wide barrier in the tile loop: a slot is released warp by warp through a shared-memory counter and
// the last warp to leave it issues the slot's next TMA load, so warps drift apart (up to 5 variables) and the
// shared-memory-read phase of one warp overlaps the FP64 phase of another.  Tiles are visited column by column
// (full x extent, Layout::col_rows rows of y, all z) so that the z-halo of a box is still in L2 when the tile
// above it is processed; the read-once RK4 operands carry an L2 evict-first policy and stores are streaming.
// See bssn_tma.cuh for the design; DESIGN.md "Kernels" for the roofline that bounds it.
#include <type_traits>

#include <cstdio>

#include "bssn_tma.cuh"
#include "tma_check.cuh"

namespace chm {

// box ring: 5 slots for the 4th-order tiles (25 variables % 5 == 0: the slot of a variable is the same in every
// tile), 3 for the 8th-order one (shared memory), where slot and parity follow from the load number 25 t + o
// point ("centre") values staged per tile: variables 0..13 (chi, gt, K, At) and 17..23 (alpha, beta, B)
constexpr int kCenVars = 21;
__device__ __forceinline__ constexpr int cen_index(int v) { return v < 14 ? v : v - 3; }
// variables whose right-hand side leaves in section o (first, second; -1 = none)
__host__ __device__ __forceinline__ constexpr int emit_var(int o, int n) {
  return o < 9 ? (n == 0 ? order_var(o) : -1) : o < 12 ? -1 : o < 21 ? (n == 0 ? order_var(o) : -1)
         : o < 24 ? (n == 0 ? V_GAM + (o - 21) : V_B + (o - 21)) : (n == 0 ? V_A : -1);
}

// ---- interleaved section layout (IL) -----------------------------------------------------
// The plain layout ends every tile with ten cheap sections (At_ij x6, B^i x3, A: 18 reads and ~57 FP64 each) that
// consume a 17.6 KB box every ~500 cycles and outrun the TMA fill (profiles/r01_l: 14 % of all warp-stall samples
// wait for those boxes).  IL evaluates the advection + dissipation stencil of At_ij and B^i EARLY, between the
// expensive beta^i / gt_ij sections, parks the one double per point it yields in a per-thread table in shared
// memory, and ends the tile with three box-less EMIT sections that only fetch Runge-Kutta operand tiles (eight per
// section, requested five sections ahead, i.e. under the expensive chi / alpha / K sections) plus two empty ones:
//   o:  0 b1 | 1 At11* | 2 b2 | 3 At12* | 4 b3 | 5 At13* | 6 gt11 | 7 At22* | 8 gt12 | 9 At23* | 10 gt13 | 11 At33* |
//       12 gt22 | 13 B1* | 14 gt23 | 15 B2* | 16 gt33 | 17 B3* | 18 Gt1 | 19 A | 20 Gt2 | 21 Gt3 | 22 chi | 23 alpha |
//       24 K | 25 emit At11..At22 | 26 emit At23, At33, Gt1, Gt2 | 27 emit Gt3, B1..B3 | 28, 29 empty
// 30 = 6 x 5 sections: slot = o mod 5 and parity = (o / 5) & 1 are compile-time constants of a section.
struct SecIL {
  static constexpr int N = 30;
  __host__ __device__ static constexpr int beta(int i) { return 2 * i; }
  __host__ __device__ static constexpr int at(int s) { return s < 3 ? 1 + 2 * s : 7 + 2 * (s - 3); }
  __host__ __device__ static constexpr int gt(int s) { return 6 + 2 * s; }
  __host__ __device__ static constexpr int b(int i) { return 13 + 2 * i; }
  __host__ __device__ static constexpr int gam(int k) { return k == 0 ? 18 : 19 + k; }
  static constexpr int a = 19, chi = 22, alpha = 23, k = 24, emit0 = 25;
  // variable whose box section o stages (-1: none)
  __host__ __device__ static constexpr int var(int o) {
    return o < 6 ? ((o & 1) ? V_AT + o / 2 : V_BETA + o / 2)
           : o < 12 ? ((o & 1) ? V_AT + 3 + (o - 7) / 2 : V_GT + (o - 6) / 2)
           : o < 18 ? ((o & 1) ? V_B + (o - 13) / 2 : V_GT + (o - 6) / 2)
           : o == 18 ? V_GAM : o == 19 ? V_A : o < 22 ? V_GAM + (o - 19) : o == 22 ? V_CHI : o == 23 ? V_ALPHA
           : o == 24 ? V_K : -1;
  }
  // variable whose right-hand side leaves in box section o, with its operand tiles next to the box (-1: none)
  __host__ __device__ static constexpr int emit(int o) {
    return o < 18 ? ((o & 1) ? -1 : var(o)) : (o == 19 || o == 22 || o == 23 || o == 24) ? var(o) : -1;
  }
};
struct SecPlain {
  static constexpr int N = 25;
  __host__ __device__ static constexpr int beta(int i) { return i; }
  __host__ __device__ static constexpr int gt(int s) { return 3 + s; }
  __host__ __device__ static constexpr int gam(int k) { return 9 + k; }
  __host__ __device__ static constexpr int at(int s) { return 15 + s; }
  __host__ __device__ static constexpr int b(int i) { return 21 + i; }
  static constexpr int chi = 12, alpha = 13, k = 14, a = 24;
};

// DEEP (interleaved layout only): six ring slots instead of five in the same shared memory -- a box section of the
// interleaved layout emits at most one variable, so a slot needs two operand tiles instead of four, and 30 sections
// divide by six as well as by five (the slot stays a compile-time constant of a section)
template <int TX, int TY, int TZ, int ORDER = 4, bool IL = false, bool DEEP = false>
struct TmaCfg {
  static_assert(!DEEP || IL, "the six-slot ring belongs to the interleaved layout");
  static_assert(!IL || (ORDER == 4 && TX * TY * TZ == 256), "the interleaved layout is built for 4th order, 256-point tiles");
  static constexpr int H = ORDER == 8 ? 5 : 3;    // halo: upwinded stencils reach order/2 + 1 cells
  static_assert(TX % 2 == 0 && ((TX + 2) * TY * TZ) % 16 == 0, "tile boxes must stay 128-byte aligned in smem");
  static constexpr int BX = TX + 2 * H, BY = TY + 2 * H, BZ = TZ + 2 * H;
  static constexpr int SLOT = (BX * BY * BZ + 15) / 16 * 16;          // doubles, 128-byte multiple
  static constexpr uint32_t BOX_BYTES = (uint32_t)BX * BY * BZ * 8u;
  static constexpr int THREADS = TX * TY * TZ;
  static_assert(THREADS <= 256, "one point per thread at 252-255 registers: at most eight warps");
  // ring slots (a 6-slot ring fits the 16x4x4 tile but its run-time slot index costs more than the depth gains:
  // 8.2 ms vs 6.3 ms)
  static constexpr int NS = DEEP ? 6 : ORDER == 8 ? 3 : 5;   // 8th order: 41 KB boxes, three fit
  static constexpr int TILE = (TX + 2) * TY * TZ;                      // doubles in one (TX+2,TY,TZ) tile box
  static constexpr uint32_t TILE_BYTES = (uint32_t)TILE * 8u;
  static constexpr int SLOTX = SLOT + (DEEP ? 2 : 4) * TILE;   // box + RK4 operands (U,S) of up to two emitted variables
  static constexpr int CEN = kCenVars * TILE;     // point values needed ahead of their own boxes
  // first derivatives shared between threads for the mixed second derivatives (two buffers, alternating):
  // D_y f on the tile + 2 columns of x-halo, D_z f on the tile + 2 columns of x-halo + 2 rows of y-halo
  static constexpr int DYX = TX + ORDER;             // x-halo = reach of the centred first derivative (order/2) on each side
  static constexpr int DY_N = DYX * TY * TZ, DZ_N = DYX * (TY + ORDER) * TZ;
  // (planes of 128 threads: measured no gain over the one-pass form)
  static constexpr bool TWOPASS = TX * TY == 64 || TX * TY == 32;
  static constexpr int DB = TWOPASS ? (DY_N + DZ_N + 15) / 16 * 16 : 0;
  // IL: per-thread table of parked values: the advection + dissipation results of At_ij (6) and B^i (3), and B^i (3)
  static constexpr int TAB = IL ? 12 * THREADS : 0;
  static_assert(!IL || 8 * TILE <= SLOTX, "the eight operand tiles of an emit section must fit one ring slot");
  static constexpr size_t SMEM = (size_t)(NS * SLOTX + CEN + 2 * DB + TAB) * 8 + (NS + 1) * 8 + (NS + 1) * 8 + 64 + 16 + 64 + 128;
  static constexpr int NWARPS = THREADS / 32;
  // shared-memory map in doubles from the dynamic base (the kernel and the host-side validator both use these)
  __host__ __device__ static constexpr int box_off(int slot) { return slot * SLOTX; }
  __host__ __device__ static constexpr int op_off(int slot, int n) { return slot * SLOTX + SLOT + n * TILE; }   // n: U0, S0, U1, S1
  __host__ __device__ static constexpr int cen_off(int group) { return NS * SLOTX + 7 * group * TILE; }        // three 7-variable groups
  __host__ __device__ static constexpr int dbuf_off() { return NS * SLOTX + CEN; }
  __host__ __device__ static constexpr int tab_off() { return NS * SLOTX + CEN + 2 * DB; }
  __host__ __device__ static constexpr int eop_off(int slot, int n) { return slot * SLOTX + n * TILE; }   // IL emit sections: U0..U3, S0..S3
  __host__ __device__ static constexpr int bar_off() { return NS * SLOTX + CEN + 2 * DB + TAB; }                      // full[NS], cfull, empty[NS + 1]
};
// the kernel body; tmU4 / tmS4 / tmU3 / tmS3: operand maps with 4 and 3 consecutive variables per box (IL emit sections)
// EARLY: a full variable's own right-hand side (which needs none of its mixed derivatives) leaves BEFORE the plane
// barrier of the two-pass mixed derivatives instead of after it, so the time a warp would spend waiting for its
// plane partner is spent on the operand reads, the stage update and the stores (capture L: 4 % of stall samples)
// FILL: fill-only mode, see the branch at the top of the tile loop and chemora_measure_box_fill
template <int TX, int TY, int TZ, int MODE, int ORDER, bool IL, bool EARLY = false, bool DEEP = false, bool FILL = false>
__device__ __forceinline__ void bssn_tma_body(const CUtensorMap& tm, const CUtensorMap& tmCen, const CUtensorMap& tmU,
                                              const CUtensorMap& tmS, const CUtensorMap& tmU4, const CUtensorMap& tmS4,
                                              const CUtensorMap& tmU3, const CUtensorMap& tmS3, const Layout& L,
                                              const Coef& C, const Stage& st, int ntx, int nty, int ntz, int cy) {
  using Cfg = TmaCfg<TX, TY, TZ, ORDER, IL, DEEP>;
  constexpr int H = Cfg::H;
  constexpr int BX = Cfg::BX, BY = Cfg::BY, SLOT = Cfg::SLOT, SLOTX = Cfg::SLOTX, TILE = Cfg::TILE;
  constexpr unsigned NW = Cfg::NWARPS;
  constexpr int kSlots = Cfg::NS;
  using Sec = std::conditional_t<IL, SecIL, SecPlain>;
  constexpr int NSEC = Sec::N;   // sections per tile: the ring position of section o of tile t is NSEC t + o
  CHM_DYNAMIC_SMEM(smem_raw);
  double* sm = reinterpret_cast<double*>(smem_raw);   // dynamic smem base: 128-byte aligned (no static smem)
  double* cbuf = sm + Cfg::cen_off(0);                                 // [kCenVars][TILE]
  double* dbuf = sm + Cfg::dbuf_off();                                 // [2][DB] shared first derivatives
  double* tabp = sm + Cfg::tab_off() + threadIdx.x;                    // IL: this thread's parked values, entry e at e * THREADS
  uint64_t* full = reinterpret_cast<uint64_t*>(sm + Cfg::bar_off());   // [kSlots] boxes, then [1] point values
  uint64_t* cfull = full + kSlots;
  uint64_t* empty = cfull + 1;                                         // [kSlots] + [1]: warps that left a buffer
  constexpr int nops = MODE == MODE_RHS ? 0 : (MODE == MODE_FIRST ? 1 : 2);   // RK4 operands per emitted var
  const int ntiles = ntx * nty * ntz;

  const int tid = threadIdx.x, lane = tid & 31;
  const int lx = tid % TX, ly = (tid / TX) % TY, lz = tid / (TX * TY);
  const int coff = ((lz + H) * BY + (ly + H)) * BX + lx + H;
  // halo-box origin relative to the tile origin in padded coordinates.  TMA needs every row of a box to start
  // on a 16-byte boundary: the layout makes L.xo - 3 even, and the (TX,TY,TZ) tile boxes (point values, RK4
  // operands) are loaded two columns wider, from x0 + 2, and read at column + 1.
  const int goffx = L.xo - H, goff = L.g - H;
  const uint64_t pol_stream = l2_policy_evict_first();   // U, S: read once per launch

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < kSlots + 1; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NW); }
    fence_mbar_init();
  }
  uint32_t* after_bars = reinterpret_cast<uint32_t*>(empty + kSlots + 1);   // one word kept free, then the origins
  int* org = reinterpret_cast<int*>((reinterpret_cast<uintptr_t>(after_bars + 1) + 15) & ~uintptr_t(15));   // [4][4]
  __syncthreads();

  // tile order (see the file header): idx -> (bx, by, bz)
  auto decode = [&](int idx, int& bx, int& by, int& bz) {
    const int per_col = ntx * cy * ntz;
    const int c = idx / per_col;
    int r = idx - c * per_col;
    const int cyt = min(cy, nty - c * cy), layer = ntx * cyt;
    bz = r / layer; r -= bz * layer;
    const int ry = r / ntx;
    by = c * cy + ry; bx = r - ry * ntx;
  };
  // Origins (padded coordinates minus halo) of this CTA's tiles t and t+1 live in a 4-entry shared-memory ring
  // (entry t & 3: x0, y0, z0, valid), written one tile ahead by lane 0 of every warp (identical values), so the
  // refill path needs no registers for them.  Warps drift less than one tile apart, so entries t, t+1 are stable.
  auto put_origin = [&](int e, int tl, bool one_writer = false) {
    int b0 = 0, b1 = 0, b2 = 0;
    const bool ok = tl < ntiles;
    if (ok) decode(tl, b0, b1, b2);
    if (one_writer ? tid == 0 : lane == 0) {
      int4 v = make_int4(b0 * TX + goffx, b1 * TY + goff, b2 * TZ + goff, ok ? 1 : 0);
      *reinterpret_cast<int4*>(org + 4 * (e & 3)) = v;
    }
  };
  // box of variable order o of the tile whose origin (padded, minus halo) is (x0,y0,z0); issued by one thread
  auto issue = [&](int o, int slot, int x0, int y0, int z0) {
    if constexpr (IL) {
      const int tx0 = x0 + H - 1, ty0 = y0 + H, tz0 = z0 + H;   // tile-box origin
      if (o >= SecIL::emit0) {
        // emit sections: eight operand tiles (U of four variables, then S of the same four) and no box; the two
        // empty sections, and the emit sections of a plain right-hand-side evaluation (no operands), complete
        // their phase with the issuer's arrival alone
        if (o >= SecIL::emit0 + 3 || nops == 0) { mbar_arrive_is_last(&full[slot]); return; }
        mbar_expect_tx(&full[slot], (uint32_t)(4 * nops) * Cfg::TILE_BYTES);
        const int e = o - SecIL::emit0;
        double* base = sm + Cfg::eop_off(slot, 0);
        if (e < 2) {        // At11..At22 (variables 8..11) / At23, At33, Gt1, Gt2 (variables 12..15): one box each
          tma_load_4d_hint(base, &tmU4, &full[slot], tx0, ty0, tz0, V_AT + 4 * e, pol_stream);
          if (nops == 2) tma_load_4d_hint(base + 4 * TILE, &tmS4, &full[slot], tx0, ty0, tz0, V_AT + 4 * e, pol_stream);
        } else {            // Gt3 (variable 16), then B1..B3 (variables 21..23)
          tma_load_4d_hint(base, &tmU, &full[slot], tx0, ty0, tz0, V_GAM + 2, pol_stream);
          tma_load_4d_hint(base + TILE, &tmU3, &full[slot], tx0, ty0, tz0, V_B, pol_stream);
          if (nops == 2) {
            tma_load_4d_hint(base + 4 * TILE, &tmS, &full[slot], tx0, ty0, tz0, V_GAM + 2, pol_stream);
            tma_load_4d_hint(base + 5 * TILE, &tmS3, &full[slot], tx0, ty0, tz0, V_B, pol_stream);
          }
        }
        return;
      }
      const int ve = SecIL::emit(o);
      mbar_expect_tx(&full[slot], Cfg::BOX_BYTES + (uint32_t)(ve >= 0 ? nops : 0) * Cfg::TILE_BYTES);
      tma_load_4d(sm + Cfg::box_off(slot), &tm, &full[slot], x0, y0, z0, SecIL::var(o));
      if (ve >= 0 && nops >= 1) tma_load_4d_hint(sm + Cfg::op_off(slot, 0), &tmU, &full[slot], tx0, ty0, tz0, ve, pol_stream);
      if (ve >= 0 && nops == 2) tma_load_4d_hint(sm + Cfg::op_off(slot, 1), &tmS, &full[slot], tx0, ty0, tz0, ve, pol_stream);
      return;
    }
    const int v0 = emit_var(o, 0), v1 = emit_var(o, 1);
    const int nem = (v0 >= 0) + (v1 >= 0);
    mbar_expect_tx(&full[slot], Cfg::BOX_BYTES + (uint32_t)(nops * nem) * Cfg::TILE_BYTES);
    tma_load_4d(sm + Cfg::box_off(slot), &tm, &full[slot], x0, y0, z0, order_var(o));
    if (v0 >= 0 && nops >= 1) tma_load_4d_hint(sm + Cfg::op_off(slot, 0), &tmU, &full[slot], x0 + H - 1, y0 + H, z0 + H, v0, pol_stream);
    if (v0 >= 0 && nops == 2) tma_load_4d_hint(sm + Cfg::op_off(slot, 1), &tmS, &full[slot], x0 + H - 1, y0 + H, z0 + H, v0, pol_stream);
    if (v1 >= 0 && nops >= 1) tma_load_4d_hint(sm + Cfg::op_off(slot, 2), &tmU, &full[slot], x0 + H - 1, y0 + H, z0 + H, v1, pol_stream);
    if (v1 >= 0 && nops == 2) tma_load_4d_hint(sm + Cfg::op_off(slot, 3), &tmS, &full[slot], x0 + H - 1, y0 + H, z0 + H, v1, pol_stream);
  };
  // point values of a tile (three 7-variable boxes: vars 0..6, 7..13, 17..23)
  auto issue_cen = [&](int x0, int y0, int z0) {
    mbar_expect_tx(cfull, (uint32_t)kCenVars * Cfg::TILE_BYTES);
    tma_load_4d(sm + Cfg::cen_off(0), &tmCen, cfull, x0 + H - 1, y0 + H, z0 + H, 0);
    tma_load_4d(sm + Cfg::cen_off(1), &tmCen, cfull, x0 + H - 1, y0 + H, z0 + H, 7);
    tma_load_4d(sm + Cfg::cen_off(2), &tmCen, cfull, x0 + H - 1, y0 + H, z0 + H, 17);
  };
  // one warp leaves buffer b (all its reads of it are done); true for lane 0 of the last of the NW warps
  auto leave = [&](int b) {
    __syncwarp();
    bool last = false;
    if (lane == 0) {
      last = mbar_arrive_is_last(&empty[b]);
    }
    return last;
  };
  put_origin(0, blockIdx.x, true);   // one writer: the block barrier below publishes it
  __syncthreads();
  if (tid == 0 && (int)blockIdx.x < ntiles) {
    const int x0 = org[0], y0 = org[1], z0 = org[2];
    issue_cen(x0, y0, z0);
#pragma unroll
    for (int o = 0; o < kSlots; ++o) issue(o, o, x0, y0, z0);
  }

  int t = 0;
  for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++t) {
    // this tile's and the next tile's origin are kept in registers (measured faster than re-reading the ring)
    int4 own, nxt = make_int4(0, 0, 0, 0);
    int b0, b1, b2;
    decode(tile, b0, b1, b2);
    own = make_int4(b0 * TX + goffx, b1 * TY + goff, b2 * TZ + goff, 1);
    if (tile + (int)gridDim.x < ntiles) {
      decode(tile + gridDim.x, b0, b1, b2);
      nxt = make_int4(b0 * TX + goffx, b1 * TY + goff, b2 * TZ + goff, 1);
    }
    const int i = own.x - goffx + lx, j = own.y - goff + ly, k = own.z - goff + lz;
    const bool valid = i < L.nx && j < L.ny && k < L.nz;
    const long q = (long)((valid ? k : 0) + L.g) * L.plane + (long)((valid ? j : 0) + L.g) * L.pitch +
                   ((valid ? i : 0) + L.xo);
    const int toff = (lz * TY + ly) * (TX + 2) + lx + 1;   // this thread's point inside a tile box
    const double* cb = cbuf + toff;
    auto cen = [&](int v) { return cb[cen_index(v) * TILE]; };
    // RK4 stage operands (U, S) of the n-th variable emitted by section o: staged by TMA next to the box;
    // read after box(o) and before done(o)
    // ring slot and mbarrier parity of section o of this CTA's t-th tile (load number 25 t + o)
    auto slot_of = [&](int o) { return (kSlots == 5 || IL) ? o % kSlots : (25 * t + o) % kSlots; };
    auto parity_of = [&](int o) {
      // 30 sections: 6 phases of a slot per tile with five slots (no dependence on t), 5 with six slots
      if constexpr (IL) return (uint32_t)((NSEC / kSlots) * t + o / kSlots) & 1u;
      else return (uint32_t)(kSlots == 5 ? (t + o / 5) & 1 : ((25 * t + o) / kSlots) & 1);
    };
    // IL emit sections: operands (U, S) of the n-th variable of the section (U tiles 0..3, S tiles 4..7 of the slot)
    auto pre_e = [&](int o, int n) {
      const double* op = sm + Cfg::eop_off(slot_of(o), n) + toff;
      return StagePre{op[0], op[4 * TILE]};
    };
    auto pre = [&](int o, int n) {
      const double* op = sm + slot_of(o) * SLOTX + SLOT + 2 * n * TILE + toff;
      return StagePre{op[0], op[TILE]};
    };
    auto emit = [&](int v, double k, const StagePre& pr) { stage_emit_t<MODE>(st, q + v * L.vstride, k, pr, valid); };

    // section o: wait for its box, hand out the accessor; done(o): this warp leaves the slot; the last warp to
    // leave refills it with the box 5 loads ahead (of this tile, or of this CTA's next tile)
    auto box = [&](int o) {
      mbar_wait(&full[slot_of(o)], parity_of(o), L.err, 0x10000u + (unsigned)o + 1u);
      return BoxPoint<BX, BY>{sm + slot_of(o) * SLOTX + coff};
    };
    auto done = [&](int o) {
      if (leave(slot_of(o))) {   // the refill is load number 25 t + o + kSlots: same slot
        const int4 a = o + kSlots < NSEC ? own : nxt;
        if (o + kSlots < NSEC) issue(o + kSlots, slot_of(o), a.x, a.y, a.z);
        else if (a.w) issue(o + kSlots - NSEC, slot_of(o), a.x, a.y, a.z);
      }
    };
    // the point values are last read just before section 3 (At)
    auto done_cen = [&]() {
      if (leave(kSlots)) {
        const int4 a = nxt;
        if (a.w) issue_cen(a.x, a.y, a.z);
      }
    };

    // all derivatives of a "full" variable (section o, n-th full variable of the tile), then done(o).
    // Two-pass mixed derivatives: every thread publishes D_y f and D_z f of its own point (it has them already),
    // the block adds them on the 2-cell x-halo (and D_z f on the 2-cell y-halo), and after one block barrier
    // d_xy = D_x(D_y f), d_xz = D_x(D_z f), d_yz = D_y(D_z f) cost 4 reads each instead of 16.
    auto full_var = [&](const BoxPoint<BX, BY>& p, const AdvW& w, int o, int n, double* d1, double* d2, double& ad,
                        auto&& early) {
      if constexpr (Cfg::TWOPASS) {
      constexpr int DYX = Cfg::DYX, ZS = BX * BY, HM = ORDER / 2;   // HM: reach of the centred first derivative
      const double f0 = p.at(0, 0, 0);
      if (ORDER == 4) {
        axis_full(p, f0, 0, C, w, d1[0], d2[0], ad);
        axis_full(p, f0, 1, C, w, d1[1], d2[3], ad);
        axis_full(p, f0, 2, C, w, d1[2], d2[5], ad);
      } else {
        axis8<BoxPoint<BX, BY>, true, true>(p, f0, 0, C, w, d1[0], d2[0], ad);
        axis8<BoxPoint<BX, BY>, true, true>(p, f0, 1, C, w, d1[1], d2[3], ad);
        axis8<BoxPoint<BX, BY>, true, true>(p, f0, 2, C, w, d1[2], d2[5], ad);
      }
      double* Dy = dbuf + ((t + n) & 1) * Cfg::DB;
      double* Dz = Dy + Cfg::DY_N;
      const double cD = C.inv_h * (ORDER == 4 ? 1.0 / 12.0 : 1.0 / 840.0);
      // centred first derivative along the direction with element stride s, from a pointer to the point
      auto D1 = [&](const double* c, int s) {
        if (ORDER == 4) return (8.0 * (c[s] - c[-s]) - (c[2 * s] - c[-2 * s])) * cD;
        return ((672.0 * (c[s] - c[-s]) - 168.0 * (c[2 * s] - c[-2 * s])) + (32.0 * (c[3 * s] - c[-3 * s]) - 3.0 * (c[4 * s] - c[-4 * s]))) * cD;
      };
      Dy[(lz * TY + ly) * DYX + lx + HM] = d1[1];
      Dz[(lz * (TY + 2 * HM) + ly + HM) * DYX + lx + HM] = d1[2];
      const double* sb = p.c - coff;   // slot base
      if constexpr (TX * TY == 64) {
        // One z-plane of the tile = PLANE threads = two warps, and every first derivative a thread reads
        // below comes from its own plane: the plane's warps fill the plane's halo entries and meet at a
        // PLANE-thread named barrier instead of a block barrier.
        constexpr int PLANE = TX * TY;
        const int u0 = tid % PLANE;
        for (int u = u0; u < TX * 2 * HM; u += PLANE) {                       // D_z f on the y-halo rows -2,-1,TY,TY+1
          const int hx = u % TX, hyi = u / TX;
          const int yy = hyi < HM ? hyi - HM : TY + hyi - HM;
          const double* c = sb + ((lz + H) * BY + (yy + H)) * BX + hx + H;
          Dz[(lz * (TY + 2 * HM) + yy + HM) * DYX + hx + HM] = D1(c, ZS);
        }
        // D_y f, D_z f on the 4 x-halo columns: 8 * TY evaluations per plane, started at a warp of the plane
        // chosen so that every scheduler (warp w runs on scheduler w % 4) gets the same share
        const int start = ((lz + 1) >> 1) & 1;
        for (int l = (u0 - 32 * start + PLANE) % PLANE; l < 4 * HM * TY; l += PLANE) {
          const int kind = l / (2 * HM * TY), hh = l % (2 * HM * TY);
          const int hxi = hh % (2 * HM), hy = hh / (2 * HM);
          const int xx = hxi < HM ? hxi - HM : TX + hxi - HM;
          const double* c = sb + ((lz + H) * BY + (hy + H)) * BX + xx + H;
          const int st1 = kind == 0 ? BX : ZS;
          const double v = D1(c, st1);
          if (kind == 0) Dy[(lz * TY + hy) * DYX + xx + HM] = v;
          else Dz[(lz * (TY + 2 * HM) + hy + HM) * DYX + xx + HM] = v;
        }
        done(o);
        early();
        named_barrier<PLANE>(1 + lz);
      } else if constexpr (TX * TY == 32) {
        // One z-plane of the tile = one warp: the warp fills its own plane's halo entries; no barrier at all.
#pragma unroll
        for (int e = 0; e < (TX * 2 * HM) / 32; ++e) {                         // D_z f on the y-halo rows
          const int u = lane + 32 * e, hx = u % TX, hyi = u / TX;
          const int yy = hyi < HM ? hyi - HM : TY + hyi - HM;
          const double* c = sb + ((lz + H) * BY + (yy + H)) * BX + hx + H;
          Dz[(lz * (TY + 2 * HM) + yy + HM) * DYX + hx + HM] = D1(c, ZS);
        }
        if (lane < 8 * TY) {                                              // D_y f, D_z f on the 4 x-halo columns
          const int kind = lane / (4 * TY), hh = lane % (4 * TY);
          const int hxi = hh % (2 * HM), hy = hh / (2 * HM);
          const int xx = hxi < HM ? hxi - HM : TX + hxi - HM;
          const double* c = sb + ((lz + H) * BY + (hy + H)) * BX + xx + H;
          const int st1 = kind == 0 ? BX : ZS;
          const double v = D1(c, st1);
          if (kind == 0) Dy[(lz * TY + hy) * DYX + xx + HM] = v;
          else Dz[(lz * (TY + 2 * HM) + hy + HM) * DYX + xx + HM] = v;
        }
        done(o);
        early();
        __syncwarp();
      } else {
        static_assert(TX * TY == 64 || TX * TY == 32, "two-pass mixed derivatives: a z-plane of one or two warps");
      }
      const double* y = Dy + (lz * TY + ly) * DYX + lx + HM;
      const double* z = Dz + (lz * (TY + 2 * HM) + ly + HM) * DYX + lx + HM;
      d2[1] = D1(y, 1);
      d2[2] = D1(z, 1);
      d2[4] = D1(z, DYX);
      } else {
        if (ORDER == 4) var_full(p, C, w, d1, d2, ad); else var_full8(p, C, w, d1, d2, ad);
        done(o);
        early();
      }
    };
    auto nothing = [] {};

    // IL: the advection + dissipation stencil of the variable staged by section o, parked in table entry e
    // (a thread reads back only what it wrote itself: no synchronisation, no hazard across tiles)
    auto park_ad = [&](int o, int e, const AdvW& w) {
      auto p = box(o);
      const double ad = var_ad(p, w);
      done(o);
      tabp[e * Cfg::THREADS] = ad;
    };
    // IL: wait for a box-less section (operand tiles only, or nothing)
    auto wait_sec = [&](int o) { mbar_wait(&full[slot_of(o)], parity_of(o), L.err, 0x10000u + (unsigned)o + 1u); };

    const double third = 1.0 / 3.0, two_thirds = 2.0 / 3.0;
    mbar_wait(cfull, (uint32_t)(t & 1), L.err, 0x10080u);
    if constexpr (FILL) {
      // Fill-only mode (chemora_measure_box_fill): the whole TMA protocol of a launch -- every box, operand tile and
      // point-value tile requested, awaited, released and refilled by the code the full kernel uses -- and no
      // arithmetic: a thread reads its own point of every box.  What remains is the cost of moving the data into
      // shared memory, the "third floor" of DESIGN.md section 6.5, measured through the validated launch path.
      double acc = cen(V_CHI);
      done_cen();
#pragma unroll
      for (int o = 0; o < NSEC; ++o) {
        if (IL && o >= SecIL::emit0) {
          wait_sec(o);
          if (nops != 0 && o < SecIL::emit0 + 3) acc += pre_e(o, 0).u;
        } else {
          const auto p = box(o);
          acc += p.at(0, 0, 0);
        }
        done(o);
      }
      if (acc == 1.2345678e300 && valid) st.S[q] = acc;   // never true: keeps the reads alive
      continue;
    }
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
      if (ORDER == 4) {
        w.ws[a] = b * (C.inv_h * (1.0 / 24.0));
        w.wq[a] = fabs(b) * (C.inv_h * (1.0 / 24.0)) + C.ko;
      } else {   // 8th order: KO is added separately (its stencil is not the symmetric part of the upwind one)
        w.ws[a] = b * (C.inv_h * (1.0 / 840.0));
        w.wq[a] = fabs(b) * (C.inv_h * (1.0 / 840.0));
      }
    }
    const double alpha = cen(V_ALPHA), trK = cen(V_K), chi = cen(V_CHI);

    // ---- o = 0..2: beta^i : d_j beta^i, gtu^{jk} d_j d_k beta^i, d_j (d_k beta^k) ----------------------------
    double db[3][3], lapb[3], gdiv[3];   // db[j][i] = d_j beta^i ; gdiv[j] = d_j d_k beta^k
#pragma unroll
    for (int i2 = 0; i2 < 3; ++i2) {
      const double Bc = cen(V_B + i2);
      auto p = box(Sec::beta(i2));
      const StagePre pr = pre(Sec::beta(i2), 0);
      double d1[3], d2[6], ad;
      auto em = [&] { emit(V_BETA + i2, C.sgc * Bc + ad, pr); };
      if constexpr (EARLY) full_var(p, w, Sec::beta(i2), i2, d1, d2, ad, em);
      else full_var(p, w, Sec::beta(i2), i2, d1, d2, ad, nothing);
#pragma unroll
      for (int a = 0; a < 3; ++a) { db[a][i2] = d1[a]; gdiv[a] = i2 == 0 ? d2[sym(a, i2)] : gdiv[a] + d2[sym(a, i2)]; }
      lapb[i2] = sdot(gu, d2);
      if constexpr (!EARLY) em();
      if constexpr (IL) park_ad(SecIL::at(i2), i2, w);   // At11, At12, At13
    }
    double divb = (db[0][0] + db[1][1]) + db[2][2];

    // ---- o = 3..8: gt_ij : d_k gt_ij kept for the Christoffels, gtu^{lm} d_l d_m gt_ij folded into R~_ij ---
    double At[6], Rt[6], dg[3][6];
#pragma unroll
    for (int s = 0; s < 6; ++s) At[s] = cen(V_AT + s);
    done_cen();
#pragma unroll
    for (int i2 = 0; i2 < 3; ++i2)
#pragma unroll
      for (int j2 = i2; j2 < 3; ++j2) {
        const int s = sym(i2, j2);
        auto p = box(Sec::gt(s));
        const StagePre pr = pre(Sec::gt(s), 0);
        double d1[3], d2[6], ad;
        auto em = [&] {
          double lie;
#pragma unroll
          for (int k2 = 0; k2 < 3; ++k2) {
            const double c = g[sym(i2, k2)] * db[j2][k2] + g[sym(j2, k2)] * db[i2][k2];
            lie = k2 == 0 ? c : lie + c;
          }
          emit(V_GT + s, (lie - two_thirds * g[s] * divb) - 2.0 * alpha * At[s] + ad, pr);
        };
        if constexpr (EARLY) full_var(p, w, Sec::gt(s), 3 + s, d1, d2, ad, em);
        else full_var(p, w, Sec::gt(s), 3 + s, d1, d2, ad, nothing);
        dg[0][s] = d1[0]; dg[1][s] = d1[1]; dg[2][s] = d1[2];
        Rt[s] = -0.5 * sdot(gu, d2);
        if constexpr (!EARLY) em();
        if constexpr (IL) {
          if (s < 3) park_ad(SecIL::at(3 + s), 3 + s, w);   // At22, At23, At33
          else {                                             // B1, B2, B3: the stencil result and the point value
            auto pb = box(SecIL::b(s - 3));
            const double Bi = pb.at(0, 0, 0), adB = var_ad(pb, w);
            done(SecIL::b(s - 3));
            tabp[(6 + s - 3) * Cfg::THREADS] = adB;
            tabp[(9 + s - 3) * Cfg::THREADS] = Bi;
          }
        }
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
      // R~_ij += 1/2 Gamma~^k_n (Gamma~_ijk + Gamma~_jik)
      //        + gtu^{lm} (Gamma~^k_li Gamma~_jkm + Gamma~^k_lj Gamma~_ikm + Gamma~^k_im Gamma~_klj)
      // with the inverse metric contracted once: W[i][m] = gtu^{lm} Gamma~^k_li (per k), so the three products are
      //   sum_m W[i][m] Gamma~_jkm + W[j][m] Gamma~_ikm   and   sum_l W[i][l] Gamma~_klj.
      // One k at a time, so that only Gamma~^k_ij of that k is live next to Gamma~_kij.
#pragma unroll
      for (int k2 = 0; k2 < 3; ++k2) {
        double Ck[6];
#pragma unroll
        for (int s = 0; s < 6; ++s)
          Ck[s] = gu[sym(k2, 0)] * Cl[0][s] + gu[sym(k2, 1)] * Cl[1][s] + gu[sym(k2, 2)] * Cl[2][s];
        Gn[k2] = sdot(gu, Ck);
        double W[3][3];
#pragma unroll
        for (int i2 = 0; i2 < 3; ++i2)
#pragma unroll
          for (int m = 0; m < 3; ++m)
            W[i2][m] = gu[sym(0, m)] * Ck[sym(0, i2)] + gu[sym(1, m)] * Ck[sym(1, i2)] + gu[sym(2, m)] * Ck[sym(2, i2)];
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
#pragma unroll
        for (int s = 0; s < 6; ++s) Cu[k2][s] = Ck[s];
      }
#pragma unroll
      for (int i2 = 0; i2 < 3; ++i2)
#pragma unroll
        for (int j2 = i2; j2 < 3; ++j2) {
          const double c = (Gn[0] * (Cl[i2][sym(j2, 0)] + Cl[j2][sym(i2, 0)]) +
                            Gn[1] * (Cl[i2][sym(j2, 1)] + Cl[j2][sym(i2, 1)])) +
                           Gn[2] * (Cl[i2][sym(j2, 2)] + Cl[j2][sym(i2, 2)]);
          Rt[sym(i2, j2)] += 0.5 * c;
        }
    }

    // A (inert slot, dissipation only): the last section of the plain layout, between Gt1 and Gt2 in the interleaved one
    auto section_A = [&]() {
      auto p = box(Sec::a);
      const StagePre pr = pre(Sec::a, 0);
      const double f0 = p.at(0, 0, 0);
      double rA;
      if (ORDER == 4) rA = C.ko * ((axis_q(p, f0, 0) + axis_q(p, f0, 1)) + axis_q(p, f0, 2));
      else rA = (axis_ko8(p, f0, 0, C) + axis_ko8(p, f0, 1, C)) + axis_ko8(p, f0, 2, C);
      done(Sec::a);
      emit(V_A, rA, pr);
    };

    // ---- o = 9..11: Gt^k : R~_ij += 1/2 (gt_ki d_j Gt^k + gt_kj d_i Gt^k); advection kept for the end ------
    double adG[3];
#pragma unroll
    for (int k2 = 0; k2 < 3; ++k2) {
      auto p = box(Sec::gam(k2));
      double d1[3];
      if (ORDER == 4) var_d1_ad(p, C, w, d1, adG[k2]); else var_d1_ad8(p, C, w, d1, adG[k2]);
      done(Sec::gam(k2));
      if constexpr (IL) { if (k2 == 0) section_A(); }
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
      auto p = box(Sec::chi);
      const StagePre pr = pre(Sec::chi, 0);
      double d2[6], ad;
      auto em = [&] { emit(V_CHI, two_thirds * chi * (alpha * trK - divb) + ad, pr); };
      if constexpr (EARLY) full_var(p, w, Sec::chi, 9, dchi, d2, ad, em);
      else { full_var(p, w, Sec::chi, 9, dchi, d2, ad, nothing); em(); }
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
      auto p = box(Sec::alpha);
      const StagePre pr = pre(Sec::alpha, 0);
      double d2[6], ad;
      auto em = [&] { emit(V_ALPHA, -2.0 * alpha * trK + ad, pr); };
      if constexpr (EARLY) full_var(p, w, Sec::alpha, 10, dal, d2, ad, em);
      else { full_var(p, w, Sec::alpha, 10, dal, d2, ad, nothing); em(); }
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

    // ---- o = 14: K -------------------------------------------------------------------------------------------
    double dK[3];
    {
      auto p = box(Sec::k);
      const StagePre pr = pre(Sec::k, 0);
      double ad;
      if (ORDER == 4) var_d1_ad(p, C, w, dK, ad); else var_d1_ad8(p, C, w, dK, ad);
      done(Sec::k);
      emit(V_K, (alpha * (sdot(Au, At) + third * trK * trK) - lap_alpha) + ad, pr);
    }

    // ---- o = 15..20: At_ij -------------------------------------------------------------------------------------
    if constexpr (IL) {
      // Interleaved layout: the stencil results of At_ij and B^i were parked early; what is left is pointwise.  All
      // twelve right-hand sides are formed here, then leave through the three emit sections (operand tiles only).
      double kAt[6], kG[3], kB[3];
      const double trX = sdot(gu, Rt);
#pragma unroll
      for (int i2 = 0; i2 < 3; ++i2)
#pragma unroll
        for (int j2 = i2; j2 < 3; ++j2) {
          const int s = sym(i2, j2);
          double AA, lie;
#pragma unroll
          for (int k2 = 0; k2 < 3; ++k2) {
            const double c = At[sym(i2, k2)] * db[j2][k2] + At[sym(j2, k2)] * db[i2][k2];
            AA = k2 == 0 ? At[sym(i2, k2)] * Am[k2][j2] : AA + At[sym(i2, k2)] * Am[k2][j2];
            lie = k2 == 0 ? c : lie + c;
          }
          const double rest = chi * (Rt[s] - third * g[s] * trX) + alpha * (trK * At[s] - 2.0 * AA) +
                              (lie - two_thirds * At[s] * divb);
          kAt[s] = rest + tabp[s * Cfg::THREADS];
        }
#pragma unroll
      for (int i2 = 0; i2 < 3; ++i2) {
        double r = lapb[i2];
        double t2 = sdot(Cu[i2], Au);   // Gamma~^i_jk At^{jk}
#pragma unroll
        for (int j2 = 0; j2 < 3; ++j2) {
          r += third * gu[sym(i2, j2)] * gdiv[j2];
          t2 -= two_thirds * gu[sym(i2, j2)] * dK[j2] + 1.5 * ichi * Au[sym(i2, j2)] * dchi[j2];
          r -= 2.0 * Au[sym(i2, j2)] * dal[j2] + Gn[j2] * db[j2][i2];
        }
        r += 2.0 * alpha * t2 + two_thirds * Gn[i2] * divb;
        kG[i2] = r + adG[i2];
        kB[i2] = (r - C.eta * tabp[(9 + i2) * Cfg::THREADS]) + tabp[(6 + i2) * Cfg::THREADS];
      }
      constexpr int E = SecIL::emit0;
      wait_sec(E);          // At11, At12, At13, At22 (variables 8..11)
      { const StagePre p0 = pre_e(E, 0), p1 = pre_e(E, 1), p2 = pre_e(E, 2), p3 = pre_e(E, 3);
        done(E);
        emit(V_AT + 0, kAt[0], p0); emit(V_AT + 1, kAt[1], p1); emit(V_AT + 2, kAt[2], p2); emit(V_AT + 3, kAt[3], p3); }
      wait_sec(E + 1);      // At23, At33, Gt1, Gt2 (variables 12..15)
      { const StagePre p0 = pre_e(E + 1, 0), p1 = pre_e(E + 1, 1), p2 = pre_e(E + 1, 2), p3 = pre_e(E + 1, 3);
        done(E + 1);
        emit(V_AT + 4, kAt[4], p0); emit(V_AT + 5, kAt[5], p1); emit(V_GAM + 0, kG[0], p2); emit(V_GAM + 1, kG[1], p3); }
      wait_sec(E + 2);      // Gt3 (variable 16), B1, B2, B3 (variables 21..23)
      { const StagePre p0 = pre_e(E + 2, 0), p1 = pre_e(E + 2, 1), p2 = pre_e(E + 2, 2), p3 = pre_e(E + 2, 3);
        done(E + 2);
        emit(V_GAM + 2, kG[2], p0); emit(V_B + 0, kB[0], p1); emit(V_B + 1, kB[1], p2); emit(V_B + 2, kB[2], p3); }
      wait_sec(E + 3); done(E + 3);   // the two empty sections keep slot = o mod 5: their release refills the slots
      wait_sec(E + 4); done(E + 4);   // with the next tile's sections 3 and 4
      continue;
    }
    if constexpr (Cfg::TWOPASS && TX * TY == 64) {
      // The kernel is bound by instruction fetch at 8th order (150 KB of code), so the six advection stencils are
      // ONE loop body.  The box-independent part of each right-hand side goes through a per-thread table laid
      // over this thread's OWN z-plane of the shared first-derivative buffers (components 0..2 in the buffer of
      // chi, n = 9; components 3..5 in the buffer of alpha, n = 10): a plane's entries are touched by the
      // plane's two warps only, and the plane barrier below orders the partner's last reads before these
      // writes; the next tile's first full variables write the buffers only after every warp has left
      // section 20 (the table is read before a section's slot is released).
      constexpr int PLANE = TX * TY, HM = ORDER / 2, NY = TY * Cfg::DYX, NZ = (TY + 2 * HM) * Cfg::DYX;
      static_assert(3 * PLANE <= NY + NZ, "table does not fit the plane's share of a buffer");
      const int u0 = tid % PLANE;
      auto tab = [&](int s) {
        double* b = dbuf + ((t + (s < 3 ? 1 : 0)) & 1) * Cfg::DB;
        const int e = (s < 3 ? s : s - 3) * PLANE + u0;
        return e < NY ? b + lz * NY + e : b + Cfg::DY_N + lz * NZ + (e - NY);
      };
      named_barrier<PLANE>(1 + lz);
      const double trX = sdot(gu, Rt);
#pragma unroll
      for (int i2 = 0; i2 < 3; ++i2)
#pragma unroll
        for (int j2 = i2; j2 < 3; ++j2) {
          const int s = sym(i2, j2);
          double AA, lie;
#pragma unroll
          for (int k2 = 0; k2 < 3; ++k2) {
            const double c = At[sym(i2, k2)] * db[j2][k2] + At[sym(j2, k2)] * db[i2][k2];
            AA = k2 == 0 ? At[sym(i2, k2)] * Am[k2][j2] : AA + At[sym(i2, k2)] * Am[k2][j2];
            lie = k2 == 0 ? c : lie + c;
          }
          *tab(s) = chi * (Rt[s] - third * g[s] * trX) + alpha * (trK * At[s] - 2.0 * AA) +
                    (lie - two_thirds * At[s] * divb);
        }
#pragma unroll 1
      for (int s = 0; s < 6; ++s) {
        auto p = box(SecPlain::at(s));
        const StagePre pr = pre(SecPlain::at(s), 0);
        const double ad = ORDER == 4 ? var_ad(p, w) : var_ad8(p, C, w);
        const double rest = *tab(s);
        done(SecPlain::at(s));
        emit(V_AT + s, rest + ad, pr);
      }
    } else {
      const double trX = sdot(gu, Rt);
#pragma unroll
      for (int i2 = 0; i2 < 3; ++i2)
#pragma unroll
        for (int j2 = i2; j2 < 3; ++j2) {
          const int s = sym(i2, j2);
          auto p = box(SecPlain::at(s));
          const StagePre pr = pre(SecPlain::at(s), 0);
          const double ad = ORDER == 4 ? var_ad(p, w) : var_ad8(p, C, w);
          done(SecPlain::at(s));
          double AA, lie;
#pragma unroll
          for (int k2 = 0; k2 < 3; ++k2) {
            const double c = At[sym(i2, k2)] * db[j2][k2] + At[sym(j2, k2)] * db[i2][k2];
            AA = k2 == 0 ? At[sym(i2, k2)] * Am[k2][j2] : AA + At[sym(i2, k2)] * Am[k2][j2];
            lie = k2 == 0 ? c : lie + c;
          }
          emit(V_AT + s, chi * (Rt[s] - third * g[s] * trX) + alpha * (trK * At[s] - 2.0 * AA) +
                             (lie - two_thirds * At[s] * divb) + ad, pr);
        }
    }

    // ---- o = 21..23: B^i, together with Gt^i ---------------------------------------------------------------------
#pragma unroll
    for (int i2 = 0; i2 < 3; ++i2) {
      auto p = box(SecPlain::b(i2));
      const StagePre prG = pre(SecPlain::b(i2), 0), prB = pre(SecPlain::b(i2), 1);
      const double Bi = p.at(0, 0, 0);
      const double adB = ORDER == 4 ? var_ad(p, w) : var_ad8(p, C, w);
      done(SecPlain::b(i2));
      double r = lapb[i2];
      double t2 = sdot(Cu[i2], Au);   // Gamma~^i_jk At^{jk}
#pragma unroll
      for (int j2 = 0; j2 < 3; ++j2) {
        r += third * gu[sym(i2, j2)] * gdiv[j2];
        t2 -= two_thirds * gu[sym(i2, j2)] * dK[j2] + 1.5 * ichi * Au[sym(i2, j2)] * dchi[j2];
        r -= 2.0 * Au[sym(i2, j2)] * dal[j2] + Gn[j2] * db[j2][i2];
      }
      r += 2.0 * alpha * t2 + two_thirds * Gn[i2] * divb;
      emit(V_GAM + i2, r + adG[i2], prG);
      emit(V_B + i2, (r - C.eta * Bi) + adB, prB);
    }

    // ---- o = 24: A (inert slot, dissipation only) -----------------------------------------------------------------
    section_A();
  }
}

// plain section layout: fused tile ids 0..4 (and the 8th-order instance)
template <int TX, int TY, int TZ, int MODE, int ORDER>
__global__ void __launch_bounds__(TX* TY* TZ, 1)
bssn_tma_kernel(const __grid_constant__ CUtensorMap tm, const __grid_constant__ CUtensorMap tmCen,
                const __grid_constant__ CUtensorMap tmU, const __grid_constant__ CUtensorMap tmS, Layout L, Coef C, Stage st, int ntx, int nty, int ntz, int cy) {
  bssn_tma_body<TX, TY, TZ, MODE, ORDER, false>(tm, tmCen, tmU, tmS, tmU, tmS, tmU, tmS, L, C, st, ntx, nty, ntz, cy);
}
// interleaved section layout (4th order, 256-point tiles)
template <int TX, int TY, int TZ, int MODE, bool EARLY = false, bool DEEP = false>
__global__ void __launch_bounds__(TX* TY* TZ, 1)
bssn_tma_il_kernel(const __grid_constant__ CUtensorMap tm, const __grid_constant__ CUtensorMap tmCen,
                   const __grid_constant__ CUtensorMap tmU, const __grid_constant__ CUtensorMap tmS,
                   const __grid_constant__ CUtensorMap tmU4, const __grid_constant__ CUtensorMap tmS4,
                   const __grid_constant__ CUtensorMap tmU3, const __grid_constant__ CUtensorMap tmS3, Layout L, Coef C,
                   Stage st, int ntx, int nty, int ntz, int cy) {
  bssn_tma_body<TX, TY, TZ, MODE, 4, true, EARLY, DEEP>(tm, tmCen, tmU, tmS, tmU4, tmS4, tmU3, tmS3, L, C, st, ntx, nty, ntz, cy);
}

// fill-only mode of either layout (chemora_measure_box_fill): same arguments, same launch plan, no arithmetic
template <int TX, int TY, int TZ, int MODE, bool IL, bool DEEP>
__global__ void __launch_bounds__(TX* TY* TZ, 1)
bssn_fill_kernel(const __grid_constant__ CUtensorMap tm, const __grid_constant__ CUtensorMap tmCen,
                 const __grid_constant__ CUtensorMap tmU, const __grid_constant__ CUtensorMap tmS,
                 const __grid_constant__ CUtensorMap tmU4, const __grid_constant__ CUtensorMap tmS4,
                 const __grid_constant__ CUtensorMap tmU3, const __grid_constant__ CUtensorMap tmS3, Layout L, Coef C,
                 Stage st, int ntx, int nty, int ntz, int cy) {
  bssn_tma_body<TX, TY, TZ, MODE, 4, IL, false, DEEP, true>(tm, tmCen, tmU, tmS, tmU4, tmS4, tmU3, tmS3, L, C, st, ntx, nty, ntz, cy);
}

// ---- launch plans (pure host code: also compiled when the kernel source is built for the CTA emulator) ------------
// What one launch of bssn_tma_kernel<TX,TY,TZ,MODE,ORDER> issues, for the validator: every section's box and
// operand loads with the mbarrier byte count the kernel announces for it (one "barrier" entry per section, one for
// the point-value tiles).  xo: Layout::xo (decides the parity of the x coordinates).
template <int TX, int TY, int TZ, int ORDER, bool IL = false, bool DEEP = false>
static TmaPlan bssn_plan(int mode, int xo) {
  using Cfg = TmaCfg<TX, TY, TZ, ORDER, IL, DEEP>;
  char name[64];
  snprintf(name, sizeof name, "bssn_tma%s_kernel<%d,%d,%d,order %d%s>", IL ? "_il" : "", TX, TY, TZ, ORDER, DEEP ? ",6 slots" : "");
  TmaPlan p;
  p.kernel = name;
  p.smem_bytes = Cfg::SMEM;
  p.threads = Cfg::THREADS;
  p.barrier_off = (size_t)Cfg::bar_off() * 8;
  p.n_barriers = 2 * (Cfg::NS + 1);
  const int nops = mode == MODE_RHS ? 0 : (mode == MODE_FIRST ? 1 : 2);
  const int par_box = (xo - Cfg::H) & 1, par_tile = (xo - 1) & 1;
  const auto tile_load = [&](const char* what, int off, int nv, int bar) {
    p.loads.push_back({what, (size_t)off * 8, {(uint32_t)(TX + 2), (uint32_t)TY, (uint32_t)TZ, (uint32_t)nv}, bar, par_tile});
  };
  for (int o = 0; IL && o < SecIL::N; ++o) {   // interleaved layout: 25 box sections, 3 emit sections, 2 empty ones
    const int slot = o % Cfg::NS;
    if (o >= SecIL::emit0) {
      const int e = o - SecIL::emit0;
      p.expect.push_back(e < 3 ? (uint32_t)(4 * nops) * Cfg::TILE_BYTES : 0u);
      if (e < 2 && nops >= 1) tile_load("operand tiles U x4", Cfg::eop_off(slot, 0), 4, o);
      if (e < 2 && nops == 2) tile_load("operand tiles S x4", Cfg::eop_off(slot, 4), 4, o);
      if (e == 2 && nops >= 1) { tile_load("operand tile U", Cfg::eop_off(slot, 0), 1, o); tile_load("operand tiles U x3", Cfg::eop_off(slot, 1), 3, o); }
      if (e == 2 && nops == 2) { tile_load("operand tile S", Cfg::eop_off(slot, 4), 1, o); tile_load("operand tiles S x3", Cfg::eop_off(slot, 5), 3, o); }
      continue;
    }
    const bool em = SecIL::emit(o) >= 0;
    p.expect.push_back(Cfg::BOX_BYTES + (uint32_t)(em ? nops : 0) * Cfg::TILE_BYTES);
    p.loads.push_back({"halo box", (size_t)Cfg::box_off(slot) * 8, {(uint32_t)Cfg::BX, (uint32_t)Cfg::BY, (uint32_t)Cfg::BZ, 1}, o, par_box});
    if (em && nops >= 1) tile_load("RK operand tile", Cfg::op_off(slot, 0), 1, o);
    if (em && nops == 2) tile_load("RK operand tile", Cfg::op_off(slot, 1), 1, o);
  }
  for (int o = 0; !IL && o < 25; ++o) {
    const int slot = o % Cfg::NS, v0 = emit_var(o, 0), v1 = emit_var(o, 1), nem = (v0 >= 0) + (v1 >= 0);
    p.expect.push_back(Cfg::BOX_BYTES + (uint32_t)(nops * nem) * Cfg::TILE_BYTES);
    p.loads.push_back({"halo box", (size_t)Cfg::box_off(slot) * 8, {(uint32_t)Cfg::BX, (uint32_t)Cfg::BY, (uint32_t)Cfg::BZ, 1}, o, par_box});
    for (int n = 0; n < 4; ++n) {
      const bool has = (n < 2 ? v0 >= 0 : v1 >= 0) && ((n & 1) ? nops == 2 : nops >= 1);
      if (has) p.loads.push_back({"RK operand tile", (size_t)Cfg::op_off(slot, n) * 8, {(uint32_t)(TX + 2), (uint32_t)TY, (uint32_t)TZ, 1}, o, par_tile});
    }
  }
  p.expect.push_back((uint32_t)kCenVars * Cfg::TILE_BYTES);
  for (int grp = 0; grp < 3; ++grp) tile_load("point-value tiles", Cfg::cen_off(grp), 7, (int)p.expect.size() - 1);
  return p;
}

void plans_bssn_fused(std::vector<TmaPlan>& out) {
  for (int mode = MODE_RHS; mode <= MODE_SSP; ++mode)
    for (int g = 3; g <= 6; ++g) {   // every ghost width the layout rule gives a different xo for
      const int xo = ((g - 3) & 1) ? g + 1 : g;
      out.push_back(bssn_plan<16, 4, 4, 4>(mode, xo));
      out.push_back(bssn_plan<16, 8, 2, 4>(mode, xo));
      out.push_back(bssn_plan<8, 4, 8, 4>(mode, xo));
      out.push_back(bssn_plan<16, 2, 8, 4>(mode, xo));
      out.push_back(bssn_plan<16, 4, 2, 4>(mode, xo));
      out.push_back(bssn_plan<16, 4, 4, 4, true>(mode, xo));   // ids 5 and 6 issue the same loads
      out.push_back(bssn_plan<16, 4, 4, 4, true, true>(mode, xo));
      if (g >= 5) out.push_back(bssn_plan<16, 4, 4, 8>(mode, xo));
    }
}

// the plan of fused tile id `tile` at FD order `order` (the dispatch of tma_dispatch below); false: no such variant
inline bool bssn_plan_for(int order, int tile, int mode, int xo, TmaPlan* out) {
  if (order == 8) { if (tile != 0) return false; *out = bssn_plan<16, 4, 4, 8>(mode, xo); return true; }
  switch (tile) {
    case 0: *out = bssn_plan<16, 4, 4, 4>(mode, xo); return true;
    case 1: *out = bssn_plan<16, 8, 2, 4>(mode, xo); return true;
    case 2: *out = bssn_plan<8, 4, 8, 4>(mode, xo); return true;
    case 3: *out = bssn_plan<16, 2, 8, 4>(mode, xo); return true;
    case 4: *out = bssn_plan<16, 4, 2, 4>(mode, xo); return true;
    case 5: case 6: *out = bssn_plan<16, 4, 4, 4, true>(mode, xo); return true;
    case 7: *out = bssn_plan<16, 4, 4, 4, true, true>(mode, xo); return true;
  }
  return false;
}

#ifndef CHM_EMULATE
// ---- host side: tensor map + launch -----------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
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

template <int TX, int TY, int TZ, int MODE, int ORDER, bool IL = false, bool EARLY = false, bool DEEP = false, bool FILL = false>
static cudaError_t tma_go_mode(const Layout& L, const Coef& C, const Stage* st, cudaStream_t s, cudaFuncAttributes* a) {
  using Cfg = TmaCfg<TX, TY, TZ, ORDER, IL, DEEP>;
  const void* kern;
  if constexpr (FILL) kern = (const void*)bssn_fill_kernel<TX, TY, TZ, MODE, IL, DEEP>;
  else if constexpr (IL) kern = (const void*)bssn_tma_il_kernel<TX, TY, TZ, MODE, EARLY, DEEP>;
  else kern = (const void*)bssn_tma_kernel<TX, TY, TZ, MODE, ORDER>;
  if (a) return cudaFuncGetAttributes(a, kern);
  // nothing is launched unless the validator accepts what this instance will issue on this layout
  if (!launch_allowed(bssn_plan<TX, TY, TZ, ORDER, IL, DEEP>(MODE, L.xo), L, st->in, L.xo - Cfg::H, Cfg::H)) return cudaErrorInvalidValue;
  EncodeTiledFn enc = encode_fn();
  if (!enc) return cudaErrorNotSupported;
  CUtensorMap tm, tmCen, tmU, tmS, tmU4, tmS4, tmU3, tmS3;
  cuuint64_t dims[4] = {(cuuint64_t)L.pitch, (cuuint64_t)L.tot_y, (cuuint64_t)L.tot_z, (cuuint64_t)L.nvars};
  cuuint64_t strides[3] = {(cuuint64_t)L.pitch * 8, (cuuint64_t)L.plane * 8, (cuuint64_t)L.vstride * 8};
  cuuint32_t box[4] = {(cuuint32_t)Cfg::BX, (cuuint32_t)Cfg::BY, (cuuint32_t)Cfg::BZ, 1};
  cuuint32_t estr[4] = {1, 1, 1, 1};
  CUresult r = enc(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<double*>(st->in), dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
  auto tile_map = [&](CUtensorMap* m, const double* base, int nv) {
    cuuint32_t b[4] = {(cuuint32_t)(TX + 2), (cuuint32_t)TY, (cuuint32_t)TZ, (cuuint32_t)nv};
    return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<double*>(base), dims, strides, b, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  };
  // RK4 operands: MODE_FIRST reads U == in; MODE_MID / MODE_LAST read U and S; MODE_RHS none (maps unused)
  // MODE_SSP reads U and the evaluated state itself
  const double* ubase = st->mode == MODE_FIRST || st->mode == MODE_RHS ? st->in : st->U;
  const double* sbase = st->mode == MODE_MID || st->mode == MODE_LAST ? st->S : st->in;
  if (!ubase || !sbase || (reinterpret_cast<uintptr_t>(ubase) | reinterpret_cast<uintptr_t>(sbase)) % 128) return cudaErrorInvalidValue;
  if (tile_map(&tmCen, st->in, 7) != CUDA_SUCCESS || tile_map(&tmU, ubase, 1) != CUDA_SUCCESS ||
      tile_map(&tmS, sbase, 1) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  if ((IL || FILL) && (tile_map(&tmU4, ubase, 4) != CUDA_SUCCESS || tile_map(&tmS4, sbase, 4) != CUDA_SUCCESS ||
             tile_map(&tmU3, ubase, 3) != CUDA_SUCCESS || tile_map(&tmS3, sbase, 3) != CUDA_SUCCESS))
    return cudaErrorInvalidValue;
  // per launch: function attributes are per device, and the call is cheap
  cudaError_t ea = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
  if (ea != cudaSuccess) return ea;
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int ntx = (L.nx + TX - 1) / TX, nty = (L.ny + TY - 1) / TY, ntz = (L.nz + TZ - 1) / TZ;
  const int ntiles = ntx * nty * ntz;
  int blocks_per_sm = 1;
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks_per_sm, kern, Cfg::THREADS, Cfg::SMEM);
  if (blocks_per_sm < 1) blocks_per_sm = 1;
  const int grid = ntiles < sms * blocks_per_sm ? ntiles : sms * blocks_per_sm;
  const int cy = L.col_rows / TY > 0 ? L.col_rows / TY : 1;   // tile rows per traversal column
  if constexpr (FILL)
    bssn_fill_kernel<TX, TY, TZ, MODE, IL, DEEP><<<grid, Cfg::THREADS, Cfg::SMEM, s>>>(tm, tmCen, tmU, tmS, tmU4, tmS4, tmU3, tmS3, L, C,
                                                                                 *st, ntx, nty, ntz, cy);
  else if constexpr (IL)
    bssn_tma_il_kernel<TX, TY, TZ, MODE, EARLY, DEEP><<<grid, Cfg::THREADS, Cfg::SMEM, s>>>(tm, tmCen, tmU, tmS, tmU4, tmS4, tmU3, tmS3, L, C,
                                                                                *st, ntx, nty, ntz, cy);
  else
    bssn_tma_kernel<TX, TY, TZ, MODE, ORDER><<<grid, Cfg::THREADS, Cfg::SMEM, s>>>(tm, tmCen, tmU, tmS, L, C, *st, ntx, nty, ntz, cy);
  return cudaGetLastError();
}

template <int TX, int TY, int TZ, int ORDER = 4, bool IL = false, bool EARLY = false, bool DEEP = false>
static cudaError_t tma_go(const Layout& L, const Coef& C, const Stage* st, cudaStream_t s, cudaFuncAttributes* a) {
  switch (st ? st->mode : MODE_MID) {   // kernel_info reports the common (middle-stage) instance
    case MODE_RHS: return tma_go_mode<TX, TY, TZ, MODE_RHS, ORDER, IL, EARLY, DEEP>(L, C, st, s, a);
    case MODE_FIRST: return tma_go_mode<TX, TY, TZ, MODE_FIRST, ORDER, IL, EARLY, DEEP>(L, C, st, s, a);
    case MODE_MID: return tma_go_mode<TX, TY, TZ, MODE_MID, ORDER, IL, EARLY, DEEP>(L, C, st, s, a);
    case MODE_LAST: return tma_go_mode<TX, TY, TZ, MODE_LAST, ORDER, IL, EARLY, DEEP>(L, C, st, s, a);
    case MODE_SSP: return tma_go_mode<TX, TY, TZ, MODE_SSP, ORDER, IL, EARLY, DEEP>(L, C, st, s, a);
  }
  return cudaErrorInvalidValue;
}

static cudaError_t tma_dispatch(int order, int tile, const Layout& L, const Coef& C, const Stage* st, cudaStream_t s,
                                cudaFuncAttributes* a) {
  if (order == 8) return tile == 0 ? tma_go<16, 4, 4, 8>(L, C, st, s, a) : cudaErrorInvalidValue;   // one 8th-order tile
  switch (tile) {
    case 0: return tma_go<16, 4, 4>(L, C, st, s, a);
    case 1: return tma_go<16, 8, 2>(L, C, st, s, a);
    case 2: return tma_go<8, 4, 8>(L, C, st, s, a);
    case 3: return tma_go<16, 2, 8>(L, C, st, s, a);
    case 4: return tma_go<16, 4, 2>(L, C, st, s, a);
    case 5: return tma_go<16, 4, 4, 4, true>(L, C, st, s, a);   // interleaved section layout
    case 6: return tma_go<16, 4, 4, 4, true, true>(L, C, st, s, a);   // the same, right-hand sides emitted before the plane barrier
    case 7: return tma_go<16, 4, 4, 4, true, true, true>(L, C, st, s, a);   // the same with a six-slot ring
  }
  return cudaErrorInvalidValue;
}

cudaError_t launch_bssn_fused(const Layout& L, const Coef& C, int order, int tile, const Stage& st, cudaStream_t s) {
  return tma_dispatch(order, tile, L, C, &st, s, nullptr);
}
// fill-only mode of a middle Runge-Kutta stage, 4th order (id 6 moves what id 5 moves)
cudaError_t launch_bssn_fill(const Layout& L, const Coef& C, int tile, const Stage& st, cudaStream_t s) {
  if (st.mode != MODE_MID) return cudaErrorInvalidValue;
  switch (tile) {
    case 0: return tma_go_mode<16, 4, 4, MODE_MID, 4, false, false, false, true>(L, C, &st, s, nullptr);
    case 1: return tma_go_mode<16, 8, 2, MODE_MID, 4, false, false, false, true>(L, C, &st, s, nullptr);
    case 2: return tma_go_mode<8, 4, 8, MODE_MID, 4, false, false, false, true>(L, C, &st, s, nullptr);
    case 3: return tma_go_mode<16, 2, 8, MODE_MID, 4, false, false, false, true>(L, C, &st, s, nullptr);
    case 4: return tma_go_mode<16, 4, 2, MODE_MID, 4, false, false, false, true>(L, C, &st, s, nullptr);
    case 5: case 6: return tma_go_mode<16, 4, 4, MODE_MID, 4, true, false, false, true>(L, C, &st, s, nullptr);
    case 7: return tma_go_mode<16, 4, 4, MODE_MID, 4, true, false, true, true>(L, C, &st, s, nullptr);
  }
  return cudaErrorInvalidValue;
}
cudaError_t kernel_info_bssn_fused(int order, int tile, cudaFuncAttributes* a) {
  Layout L{}; Coef C{};
  return tma_dispatch(order, tile, L, C, nullptr, 0, a);
}

#endif   // CHM_EMULATE

}  // namespace chm
