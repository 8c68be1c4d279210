// libchemora_emu.cpp -- the library's own host code (csrc/chemora.cu: the C ABI of include/chemora.h) compiled with g++
// on top of the emulated kernels: every kernel source of csrc/ built for the host (-DCHM_EMULATE, cta_emu.hpp), the CUDA
// runtime calls chemora.cu makes stubbed on host memory (cuda_rt_stub.hpp), and the launchers of common.cuh implemented
// here with the same dispatch tables and the same launch validator as the real ones, running the kernels under the CTA
// emulator.  Built by tests/test_abi_emulated.py as a shared library of its own; the package never loads it (there is
// no CPU fallback in the product: paper_1307_6488_b200/binding.py loads libchemora.so or fails).
// What it is for: the host logic written without GPU access -- stage plans, chemora_autotune with its agreement guard
// and col_rows sweep, the timing event pool, the ghosted state copies, the radiative step order, the device error word
// -- runs here behind the same Python binding and the same test functions that run on the GPU.
#include "cta_emu.hpp"
#include "cuda_rt_stub.hpp"

#include "../../paper_1307_6488_b200/csrc/kernels_basic.cu"
#include "../../paper_1307_6488_b200/csrc/kernels_boundary.cu"
#include "../../paper_1307_6488_b200/csrc/kernels_bssn.cu"
#include "../../paper_1307_6488_b200/csrc/kernels_bssn_tma.cu"
#include "../../paper_1307_6488_b200/csrc/kernels_wave_tma.cu"

namespace chm {

constexpr int kEmuSMs = 4;   // persistent grids: at most this many CTAs (run one after the other)

static cudaFuncAttributes fake_attr() { return cudaFuncAttributes{128, 0, 0}; }

// ---- kernels_basic.cu ---------------------------------------------------------------------------------------------
cudaError_t launch_fill_ghosts(const Layout& L, double* state, cudaStream_t, const FillLink* link) {
  const int g = L.g;
  if (g == 0) return cudaSuccess;
  const long rowsA = 2L * g * L.tot_y, rowsAB = rowsA + 2L * g * L.nz, rowsC = (long)L.nz * L.ny;
  int lpr_shift = 0;
  while ((1 << lpr_shift) < 2 * g && lpr_shift < 5) ++lpr_shift;
  const long tasks = rowsAB + (rowsC + (32 >> lpr_shift) - 1) / (32 >> lpr_shift);
  const FillLink self{state, L.vstride, L.nz, state, L.vstride};
  const FillLink use = link ? *link : self;
  chm_emu::run_grid_serial((int)((tasks + 7) / 8), L.nvars, 1, 256, 1,
                           [&] { fill_ghosts_kernel(L, state, (int)rowsA, (int)rowsAB, lpr_shift, use); });
  return cudaSuccess;
}
cudaError_t launch_pack(const Layout& L, const double* packed, double* state, bool to_state, cudaStream_t) {
  if (to_state) chm_emu::run_grid_serial((L.nx + 255) / 256, L.ny, L.nz * L.nvars, 256, 1, [&] { pack_kernel(L, packed, state, true); });
  else chm_emu::run_grid_serial((L.nx + 255) / 256, L.ny, L.nz * L.nvars, 256, 1,
                                [&] { pack_kernel(L, state, const_cast<double*>(packed), false); });
  return cudaSuccess;
}
cudaError_t launch_enforce(const Layout& L, double* state, cudaStream_t) {
  chm_emu::run_grid_serial((L.nx + 255) / 256, L.ny, L.nz, 256, 1, [&] { enforce_kernel(L, state); });
  return cudaSuccess;
}
cudaError_t launch_energy(const Layout& L, const double* state, double* eps_out, double* sum, cudaStream_t) {
  chm_emu::run_grid((L.nx + 255) / 256, 256, 1, 0, [&] { energy_kernel(L, state, eps_out, sum); }, L.ny, L.nz);
  return cudaSuccess;
}
cudaError_t launch_dfma_peak(int, int, int, double*, cudaStream_t) { return cudaSuccess; }   // nothing to measure here

// ---- kernels_boundary.cu ------------------------------------------------------------------------------------------
cudaError_t launch_radiative(const Layout& L, const Stage& st, double h, unsigned uinf_mask, cudaStream_t) {
  if (L.g < 2) return cudaErrorInvalidValue;
  const RadGeom G = rad_geom(L);
  chm_emu::run_grid_serial((int)((G.tasks + 7) / 8), L.nvars, 1, 256, 1,
                           [&] { radiative_kernel(L, st, h, uinf_mask, (int)G.rowsA, (int)G.rowsAB, G.lpr_shift); });
  return cudaSuccess;
}
cudaError_t launch_maxdiff(const double* a, const double* b, long vstride, int nvars, unsigned long long* out, cudaStream_t) {
  long blocks = (vstride + 256L * 8 - 1) / (256L * 8);
  if (blocks > 1024) blocks = 1024;
  if (blocks < 1) blocks = 1;
  chm_emu::run_grid((int)blocks, 256, 1, 0, [&] { maxdiff_kernel(a, b, vstride, out); }, nvars);
  return cudaSuccess;
}

}  // namespace chm

namespace chm {

// ---- L1-path wave kernels (kernels_basic.cu): tile ids 0..5 = kTilesMarch ----------------------------------------------
template <class K>
static cudaError_t emu_march(const Layout& L, int tx, int ty, int tz, K&& kern) {
  chm_emu::run_grid_serial((L.nx + tx - 1) / tx, (L.ny + ty - 1) / ty, (L.nz + tz - 1) / tz, tx, ty, kern);
  return cudaSuccess;
}
#define CHM_EMU_TILES(CALL)                                                                                        \
  switch (tile) {                                                                                                  \
    case 0: return CALL(32, 4, 8);  case 1: return CALL(32, 8, 8);  case 2: return CALL(64, 2, 8);                 \
    case 3: return CALL(64, 4, 8);  case 4: return CALL(128, 2, 8); case 5: return CALL(16, 16, 8);                \
  }                                                                                                                \
  return cudaErrorInvalidValue;

template <int ORDER, bool KO>
static cudaError_t emu_wave(int tile, const Layout& L, const Coef& C, const Stage& st) {
#define W(TX, TY, TZ) emu_march(L, TX, TY, TZ, [&] { wave_kernel<ORDER, KO, TX, TY, TZ>(L, C, st); })
  CHM_EMU_TILES(W)
#undef W
}
template <int ORDER, bool KO>
static cudaError_t emu_wave1(int tile, const Layout& L, const Coef& C, const Stage& st) {
#define W(TX, TY, TZ) emu_march(L, TX, TY, TZ, [&] { wave1_kernel<ORDER, KO, TX, TY, TZ>(L, C, st); })
  CHM_EMU_TILES(W)
#undef W
}
cudaError_t launch_wave(const Layout& L, const Coef& C, int order, int tile, const Stage& st, cudaStream_t) {
  const bool ko = C.ko != 0.0;
  if (order == 4) return ko ? emu_wave<4, true>(tile, L, C, st) : emu_wave<4, false>(tile, L, C, st);
  if (order == 8) return ko ? emu_wave<8, true>(tile, L, C, st) : emu_wave<8, false>(tile, L, C, st);
  return cudaErrorInvalidValue;
}
cudaError_t launch_wave1(const Layout& L, const Coef& C, int order, int tile, const Stage& st, cudaStream_t) {
  const bool ko = C.ko != 0.0;
  if (order == 4) return ko ? emu_wave1<4, true>(tile, L, C, st) : emu_wave1<4, false>(tile, L, C, st);
  if (order == 8) return ko ? emu_wave1<8, true>(tile, L, C, st) : emu_wave1<8, false>(tile, L, C, st);
  return cudaErrorInvalidValue;
}
cudaError_t kernel_info_wave(int, int tile, cudaFuncAttributes* a) { *a = fake_attr(); return tile >= 0 && tile < 6 ? cudaSuccess : cudaErrorInvalidValue; }
cudaError_t kernel_info_wave1(int, int tile, cudaFuncAttributes* a) { *a = fake_attr(); return tile >= 0 && tile < 6 ? cudaSuccess : cudaErrorInvalidValue; }

// ---- derivative-split BSSN variant (kernels_bssn.cu) -----------------------------------------------------------------
cudaError_t launch_bssn_derivs(const Layout& L, const Coef& C, int order, int tile, const double* in, double* derivs, cudaStream_t) {
#define D4(TX, TY, TZ) emu_march(L, TX, TY, TZ, [&] { bssn_derivs_kernel<TX, TY, TZ, 4>(L, C, in, derivs); })
#define D8(TX, TY, TZ) emu_march(L, TX, TY, TZ, [&] { bssn_derivs_kernel<TX, TY, TZ, 8>(L, C, in, derivs); })
  if (order == 4) { CHM_EMU_TILES(D4) }
  if (order == 8) { CHM_EMU_TILES(D8) }
#undef D4
#undef D8
  return cudaErrorInvalidValue;
}
cudaError_t launch_bssn_from_derivs(const Layout& L, const Coef& C, int tile, const double* derivs, const Stage& st, cudaStream_t) {
#define F(TX, TY, TZ) emu_march(L, TX, TY, TZ, [&] { bssn_from_derivs_kernel<TX, TY, TZ>(L, C, derivs, st); })
  CHM_EMU_TILES(F)
#undef F
}
cudaError_t kernel_info_bssn_split(int, int tile, cudaFuncAttributes* a) { *a = fake_attr(); return tile >= 0 && tile < 6 ? cudaSuccess : cudaErrorInvalidValue; }

static CUtensorMap emu_map(const Layout& L, const double* base, uint32_t bx, uint32_t by, uint32_t bz, uint32_t bv) {
  CUtensorMap m;
  m.base = base;
  m.dims[0] = L.pitch; m.dims[1] = L.tot_y; m.dims[2] = L.tot_z; m.dims[3] = L.nvars;
  m.strides[0] = L.pitch * 8; m.strides[1] = L.plane * 8; m.strides[2] = L.vstride * 8;
  m.box[0] = bx; m.box[1] = by; m.box[2] = bz; m.box[3] = bv;
  return m;
}

// ---- fused BSSN kernel (kernels_bssn_tma.cu): as tma_go_mode, the launch replaced by the CTA emulator -----------------
template <int TX, int TY, int TZ, int MODE, int ORDER, bool IL, bool EARLY, bool DEEP>
static cudaError_t emu_fused(const Layout& L, const Coef& C, const Stage& st) {
  using Cfg = TmaCfg<TX, TY, TZ, ORDER, IL, DEEP>;
  if (!launch_allowed(bssn_plan<TX, TY, TZ, ORDER, IL, DEEP>(MODE, L.xo), L, st.in, L.xo - Cfg::H, Cfg::H)) return cudaErrorInvalidValue;
  const double* ubase = st.mode == MODE_FIRST || st.mode == MODE_RHS ? st.in : st.U;
  const double* sbase = st.mode == MODE_MID || st.mode == MODE_LAST ? st.S : st.in;
  if (!ubase || !sbase || (reinterpret_cast<uintptr_t>(ubase) | reinterpret_cast<uintptr_t>(sbase)) % 128) return cudaErrorInvalidValue;
  const CUtensorMap tm = emu_map(L, st.in, Cfg::BX, Cfg::BY, Cfg::BZ, 1), tmCen = emu_map(L, st.in, TX + 2, TY, TZ, 7),
                    tmU = emu_map(L, ubase, TX + 2, TY, TZ, 1), tmS = emu_map(L, sbase, TX + 2, TY, TZ, 1),
                    tmU4 = emu_map(L, ubase, TX + 2, TY, TZ, 4), tmS4 = emu_map(L, sbase, TX + 2, TY, TZ, 4),
                    tmU3 = emu_map(L, ubase, TX + 2, TY, TZ, 3), tmS3 = emu_map(L, sbase, TX + 2, TY, TZ, 3);
  const int ntx = (L.nx + TX - 1) / TX, nty = (L.ny + TY - 1) / TY, ntz = (L.nz + TZ - 1) / TZ;
  const int ntiles = ntx * nty * ntz, grid = ntiles < kEmuSMs ? ntiles : kEmuSMs;
  const int cy = L.col_rows / TY > 0 ? L.col_rows / TY : 1;
  chm_emu::run_grid(grid, Cfg::THREADS, 1, Cfg::SMEM, [&] {
    if constexpr (IL) bssn_tma_il_kernel<TX, TY, TZ, MODE, EARLY, DEEP>(tm, tmCen, tmU, tmS, tmU4, tmS4, tmU3, tmS3, L, C, st, ntx, nty, ntz, cy);
    else bssn_tma_kernel<TX, TY, TZ, MODE, ORDER>(tm, tmCen, tmU, tmS, L, C, st, ntx, nty, ntz, cy);
  });
  return cudaSuccess;
}
template <int TX, int TY, int TZ, int ORDER = 4, bool IL = false, bool EARLY = false, bool DEEP = false>
static cudaError_t emu_fused_mode(const Layout& L, const Coef& C, const Stage& st) {
  switch (st.mode) {
    case MODE_RHS: return emu_fused<TX, TY, TZ, MODE_RHS, ORDER, IL, EARLY, DEEP>(L, C, st);
    case MODE_FIRST: return emu_fused<TX, TY, TZ, MODE_FIRST, ORDER, IL, EARLY, DEEP>(L, C, st);
    case MODE_MID: return emu_fused<TX, TY, TZ, MODE_MID, ORDER, IL, EARLY, DEEP>(L, C, st);
    case MODE_LAST: return emu_fused<TX, TY, TZ, MODE_LAST, ORDER, IL, EARLY, DEEP>(L, C, st);
    case MODE_SSP: return emu_fused<TX, TY, TZ, MODE_SSP, ORDER, IL, EARLY, DEEP>(L, C, st);
  }
  return cudaErrorInvalidValue;
}
// Fault injection for the tests of the runtime sweep's guard and of the error-word plumbing (environment variables, read
// at every launch): CHM_EMU_BREAK_TILE=<id>: that fused id computes with a doubled eta, i.e. a different right-hand side;
// CHM_EMU_TIMEOUT_TILE=<id>: after that id's launch the device error word holds the code a timed-out wait for the box
// of section 12 would leave.
static cudaError_t launch_bssn_fused_real(const Layout& L, const Coef& C, int order, int tile, const Stage& st);
cudaError_t launch_bssn_fused(const Layout& L, const Coef& C, int order, int tile, const Stage& st, cudaStream_t) {
  const char* brk = getenv("CHM_EMU_BREAK_TILE");
  const char* tmo = getenv("CHM_EMU_TIMEOUT_TILE");
  Coef C2 = C;
  if (brk && atoi(brk) == tile) C2.eta *= 2.0;
  const cudaError_t e = launch_bssn_fused_real(L, C2, order, tile, st);
  if (e == cudaSuccess && tmo && atoi(tmo) == tile && L.err) *L.err = 0x10000u + 13u;
  return e;
}
static cudaError_t launch_bssn_fused_real(const Layout& L, const Coef& C, int order, int tile, const Stage& st) {   // = tma_dispatch
  if (order == 8) return tile == 0 ? emu_fused_mode<16, 4, 4, 8>(L, C, st) : cudaErrorInvalidValue;
  switch (tile) {
    case 0: return emu_fused_mode<16, 4, 4>(L, C, st);
    case 1: return emu_fused_mode<16, 8, 2>(L, C, st);
    case 2: return emu_fused_mode<8, 4, 8>(L, C, st);
    case 3: return emu_fused_mode<16, 2, 8>(L, C, st);
    case 4: return emu_fused_mode<16, 4, 2>(L, C, st);
    case 5: return emu_fused_mode<16, 4, 4, 4, true>(L, C, st);
    case 6: return emu_fused_mode<16, 4, 4, 4, true, true>(L, C, st);
    case 7: return emu_fused_mode<16, 4, 4, 4, true, true, true>(L, C, st);
  }
  return cudaErrorInvalidValue;
}
// fill-only mode (launch_bssn_fill): as emu_fused with the fill kernel
template <int TX, int TY, int TZ, bool IL, bool DEEP>
static cudaError_t emu_fill(const Layout& L, const Coef& C, const Stage& st) {
  using Cfg = TmaCfg<TX, TY, TZ, 4, IL, DEEP>;
  if (!launch_allowed(bssn_plan<TX, TY, TZ, 4, IL, DEEP>(MODE_MID, L.xo), L, st.in, L.xo - Cfg::H, Cfg::H)) return cudaErrorInvalidValue;
  const CUtensorMap tm = emu_map(L, st.in, Cfg::BX, Cfg::BY, Cfg::BZ, 1), tmCen = emu_map(L, st.in, TX + 2, TY, TZ, 7),
                    tmU = emu_map(L, st.U, TX + 2, TY, TZ, 1), tmS = emu_map(L, st.S, TX + 2, TY, TZ, 1),
                    tmU4 = emu_map(L, st.U, TX + 2, TY, TZ, 4), tmS4 = emu_map(L, st.S, TX + 2, TY, TZ, 4),
                    tmU3 = emu_map(L, st.U, TX + 2, TY, TZ, 3), tmS3 = emu_map(L, st.S, TX + 2, TY, TZ, 3);
  const int ntx = (L.nx + TX - 1) / TX, nty = (L.ny + TY - 1) / TY, ntz = (L.nz + TZ - 1) / TZ;
  const int ntiles = ntx * nty * ntz, grid = ntiles < kEmuSMs ? ntiles : kEmuSMs;
  const int cy = L.col_rows / TY > 0 ? L.col_rows / TY : 1;
  chm_emu::run_grid(grid, Cfg::THREADS, 1, Cfg::SMEM, [&] {
    bssn_fill_kernel<TX, TY, TZ, MODE_MID, IL, DEEP>(tm, tmCen, tmU, tmS, tmU4, tmS4, tmU3, tmS3, L, C, st, ntx, nty, ntz, cy);
  });
  return cudaSuccess;
}
cudaError_t launch_bssn_fill(const Layout& L, const Coef& C, int tile, const Stage& st, cudaStream_t) {
  if (st.mode != MODE_MID) return cudaErrorInvalidValue;
  switch (tile) {
    case 0: return emu_fill<16, 4, 4, false, false>(L, C, st);
    case 1: return emu_fill<16, 8, 2, false, false>(L, C, st);
    case 2: return emu_fill<8, 4, 8, false, false>(L, C, st);
    case 3: return emu_fill<16, 2, 8, false, false>(L, C, st);
    case 4: return emu_fill<16, 4, 2, false, false>(L, C, st);
    case 5: case 6: return emu_fill<16, 4, 4, true, false>(L, C, st);
    case 7: return emu_fill<16, 4, 4, true, true>(L, C, st);
  }
  return cudaErrorInvalidValue;
}
cudaError_t kernel_info_bssn_fused(int order, int tile, cudaFuncAttributes* a) {
  *a = fake_attr();
  return (order == 8 ? tile == 0 : (tile >= 0 && tile < kNumFused)) ? cudaSuccess : cudaErrorInvalidValue;
}

// ---- plane-ring kernels (kernels_wave_tma.cu): as wv_go ----------------------------------------------------------------
template <int ORDER, bool KO, int TX, int TY, int ZC, int NV>
static cudaError_t emu_ring(const Layout& L, const Coef& C, const Stage& st) {
  using K = wv::Cfg<ORDER, KO, TX, TY, NV>;
  if constexpr (!K::FITS) return cudaErrorInvalidValue;
  else {
    if (L.nvars != NV || !launch_allowed(wv_plan<ORDER, KO, TX, TY, NV>(L.xo), L, st.in, L.xo - K::R, K::R)) return cudaErrorInvalidValue;
    const CUtensorMap tm = emu_map(L, st.in, K::ROW, K::COLS, 1, NV);
    const int ntx = (L.nx + TX - 1) / TX, nty = (L.ny + TY - 1) / TY, ntz = (L.nz + ZC - 1) / ZC;
    const int nitems = ntx * nty * ntz, grid = nitems < kEmuSMs ? nitems : kEmuSMs;
    chm_emu::run_grid(grid, TX, TY, K::SMEM, [&] { wave_tma_kernel<ORDER, KO, TX, TY, ZC, NV>(tm, L, C, st, ntx, nty, ntz); });
    return cudaSuccess;
  }
}
template <int ORDER, bool KO>
static cudaError_t emu_ring_pick(int nv, int which, const Layout& L, const Coef& C, const Stage& st) {
  if (nv == 2) switch (which) {
    case 0: return emu_ring<ORDER, KO, 32, 16, 32, 2>(L, C, st);
    case 1: return emu_ring<ORDER, KO, 32, 16, 64, 2>(L, C, st);
    case 2: return emu_ring<ORDER, KO, 64, 8, 32, 2>(L, C, st);
  }
  if (nv == 5) switch (which) {
    case 0: return emu_ring<ORDER, KO, 16, 8, 64, 5>(L, C, st);
    case 1: return emu_ring<ORDER, KO, 16, 16, 64, 5>(L, C, st);
    case 2: return emu_ring<ORDER, KO, 32, 8, 64, 5>(L, C, st);
  }
  return cudaErrorInvalidValue;
}
static cudaError_t emu_ring_dispatch(int nv, int order, bool ko, int which, const Layout& L, const Coef& C, const Stage& st) {
  if (order == 4) return ko ? emu_ring_pick<4, true>(nv, which, L, C, st) : emu_ring_pick<4, false>(nv, which, L, C, st);
  if (order == 8) return ko ? emu_ring_pick<8, true>(nv, which, L, C, st) : emu_ring_pick<8, false>(nv, which, L, C, st);
  return cudaErrorInvalidValue;
}
cudaError_t launch_wave_tma(const Layout& L, const Coef& C, int order, int which, const Stage& st, cudaStream_t) {
  return emu_ring_dispatch(2, order, C.ko != 0.0, which, L, C, st);
}
cudaError_t launch_wave1_tma(const Layout& L, const Coef& C, int order, int which, const Stage& st, cudaStream_t) {
  return emu_ring_dispatch(5, order, C.ko != 0.0, which, L, C, st);
}
template <int ORDER, bool KO>
static bool ring5_fits(int which) {
  return which == 0 ? wv::Cfg<ORDER, KO, 16, 8, 5>::FITS : which == 1 ? wv::Cfg<ORDER, KO, 16, 16, 5>::FITS
         : which == 2 ? wv::Cfg<ORDER, KO, 32, 8, 5>::FITS : false;
}
bool wave1_tma_ok(const Layout& L, int order, bool ko, int which) {   // as the real one: layout suits TMA and the ring fits
  if (!wave_tma_ok(L, order, ko)) return false;
  if (order == 4) return ko ? ring5_fits<4, true>(which) : ring5_fits<4, false>(which);
  if (order == 8) return ko ? ring5_fits<8, true>(which) : ring5_fits<8, false>(which);
  return false;
}
cudaError_t kernel_info_wave_tma(int, int which, cudaFuncAttributes* a) { *a = fake_attr(); return which >= 0 && which < 3 ? cudaSuccess : cudaErrorInvalidValue; }
cudaError_t kernel_info_wave1_tma(int, int which, cudaFuncAttributes* a) { *a = fake_attr(); return which >= 0 && which < 3 ? cudaSuccess : cudaErrorInvalidValue; }

}  // namespace chm

// ---- the library's host code, unchanged ---------------------------------------------------------------------------------
#include "../../paper_1307_6488_b200/csrc/chemora.cu"
