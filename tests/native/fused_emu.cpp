// fused_emu.cpp -- runs the fused BSSN kernel's SOURCE (csrc/kernels_bssn_tma.cu, compiled for the host with
// -DCHM_EMULATE on top of cta_emu.hpp) over a small block: persistent CTAs, the mbarrier ring, the TMA boxes, the
// warp-wise slot release and refill, the two-pass mixed derivatives with their plane barriers, the Runge-Kutta
// epilogues -- everything but the hardware.  Test infrastructure only (tests/test_fused_kernel_emulated.py).
//
//   (mode 12 = the fill-only kernel of a middle stage)
//   fused_emu <order> <tile> <mode> <nx> <ny> <nz> <g> <h> <eps> <eta> <sgc> <ko_order> <a> <ca> <cb> <grid>
//             <in.bin> <U.bin> <S.bin> <out.bin>
// in/U/S.bin: ghosted arrays [25][nz+2g][ny+2g][nx+2g] (ghosts of `in` filled); out.bin: three such arrays in a row:
// the buffer Stage::out points to, then S, then U, as the launch left them.  Prints "err <word> loads <n> bytes <n>".
#include "cta_emu.hpp"

#include "../../paper_1307_6488_b200/csrc/kernels_bssn_tma.cu"

using namespace chm;

static Layout make_layout(int nx, int ny, int nz, int g) {   // the rule of chemora_create (csrc/chemora.cu)
  Layout L{};
  L.nx = nx; L.ny = ny; L.nz = nz; L.g = g; L.nvars = 25;
  L.xo = ((g - 3) & 1) ? g + 1 : g;
  L.pitch = ((long)L.xo + nx + g + 15) / 16 * 16;
  L.tot_y = ny + 2 * g; L.tot_z = nz + 2 * g;
  L.plane = L.pitch * L.tot_y;
  L.vstride = L.plane * L.tot_z;
  L.col_rows = getenv("CHM_COL_ROWS") ? atoi(getenv("CHM_COL_ROWS")) : 32;   // tile traversal: any value, same result
  return L;
}

static std::vector<double> to_padded(const Layout& L, const std::vector<double>& ghosted) {
  std::vector<double> p((size_t)L.nvars * L.vstride, 0.0);
  const long tx = L.nx + 2 * L.g;
  for (int v = 0; v < L.nvars; ++v)
    for (int k = 0; k < L.tot_z; ++k)
      for (int j = 0; j < L.tot_y; ++j)
        memcpy(&p[(size_t)v * L.vstride + (size_t)k * L.plane + (size_t)j * L.pitch + (L.xo - L.g)],
               &ghosted[(((size_t)v * L.tot_z + k) * L.tot_y + j) * tx], tx * 8);
  return p;
}
static void from_padded(const Layout& L, const double* p, std::vector<double>& ghosted) {
  const long tx = L.nx + 2 * L.g;
  for (int v = 0; v < L.nvars; ++v)
    for (int k = 0; k < L.tot_z; ++k)
      for (int j = 0; j < L.tot_y; ++j)
        memcpy(&ghosted[(((size_t)v * L.tot_z + k) * L.tot_y + j) * tx],
               &p[(size_t)v * L.vstride + (size_t)k * L.plane + (size_t)j * L.pitch + (L.xo - L.g)], tx * 8);
}

// IL: 0 plain layout, 1 interleaved, 2 + early emission, 3 + six-slot ring; FILL: the fill-only kernel
template <int TX, int TY, int TZ, int MODE, int ORDER, int IL = 0, bool FILL = false>
static chm_emu::Stats run(const Layout& L, const Coef& C, const Stage& st, int grid_req) {
  using Cfg = TmaCfg<TX, TY, TZ, ORDER, IL != 0, IL == 3>;
  auto map = [&](const double* base, uint32_t bx, uint32_t by, uint32_t bz, uint32_t bv) {
    CUtensorMap m;
    m.base = base;
    m.dims[0] = L.pitch; m.dims[1] = L.tot_y; m.dims[2] = L.tot_z; m.dims[3] = L.nvars;
    m.strides[0] = L.pitch * 8; m.strides[1] = L.plane * 8; m.strides[2] = L.vstride * 8;
    m.box[0] = bx; m.box[1] = by; m.box[2] = bz; m.box[3] = bv;
    return m;
  };
  // as tma_go_mode: operand maps by mode
  const double* ubase = st.mode == MODE_FIRST || st.mode == MODE_RHS ? st.in : st.U;
  const double* sbase = st.mode == MODE_MID || st.mode == MODE_LAST ? st.S : st.in;
  const CUtensorMap tm = map(st.in, Cfg::BX, Cfg::BY, Cfg::BZ, 1), tmCen = map(st.in, TX + 2, TY, TZ, 7),
                    tmU = map(ubase, TX + 2, TY, TZ, 1), tmS = map(sbase, TX + 2, TY, TZ, 1);
  const int ntx = (L.nx + TX - 1) / TX, nty = (L.ny + TY - 1) / TY, ntz = (L.nz + TZ - 1) / TZ;
  const int ntiles = ntx * nty * ntz, grid = ntiles < grid_req ? ntiles : grid_req;
  const int cy = L.col_rows / TY > 0 ? L.col_rows / TY : 1;
  if constexpr (FILL && ORDER == 4) {
    const CUtensorMap tmU4 = map(ubase, TX + 2, TY, TZ, 4), tmS4 = map(sbase, TX + 2, TY, TZ, 4),
                      tmU3 = map(ubase, TX + 2, TY, TZ, 3), tmS3 = map(sbase, TX + 2, TY, TZ, 3);
    return chm_emu::run_grid(grid, Cfg::THREADS, 1, Cfg::SMEM, [&] {
      bssn_fill_kernel<TX, TY, TZ, MODE, IL != 0, IL == 3>(tm, tmCen, tmU, tmS, tmU4, tmS4, tmU3, tmS3, L, C, st, ntx, nty, ntz, cy);
    });
  } else if constexpr (IL != 0) {   // the interleaved layout's operand maps: 4 and 3 consecutive variables a box
    const CUtensorMap tmU4 = map(ubase, TX + 2, TY, TZ, 4), tmS4 = map(sbase, TX + 2, TY, TZ, 4),
                      tmU3 = map(ubase, TX + 2, TY, TZ, 3), tmS3 = map(sbase, TX + 2, TY, TZ, 3);
    return chm_emu::run_grid(grid, Cfg::THREADS, 1, Cfg::SMEM, [&] {
      bssn_tma_il_kernel<TX, TY, TZ, MODE, IL >= 2, IL == 3>(tm, tmCen, tmU, tmS, tmU4, tmS4, tmU3, tmS3, L, C, st, ntx, nty, ntz, cy);
    });
  } else {
    return chm_emu::run_grid(grid, Cfg::THREADS, 1, Cfg::SMEM, [&] {
      bssn_tma_kernel<TX, TY, TZ, MODE, ORDER>(tm, tmCen, tmU, tmS, L, C, st, ntx, nty, ntz, cy);
    });
  }
}

template <int TX, int TY, int TZ, int ORDER, int IL = 0>
static chm_emu::Stats run_mode(int mode, const Layout& L, const Coef& C, const Stage& st, int grid) {
  if (mode == 10 + MODE_MID) return run<TX, TY, TZ, MODE_MID, ORDER, IL, true>(L, C, st, grid);   // fill-only
  switch (mode) {
    case MODE_RHS: return run<TX, TY, TZ, MODE_RHS, ORDER, IL>(L, C, st, grid);
    case MODE_FIRST: return run<TX, TY, TZ, MODE_FIRST, ORDER, IL>(L, C, st, grid);
    case MODE_MID: return run<TX, TY, TZ, MODE_MID, ORDER, IL>(L, C, st, grid);
    case MODE_LAST: return run<TX, TY, TZ, MODE_LAST, ORDER, IL>(L, C, st, grid);
    case MODE_SSP: return run<TX, TY, TZ, MODE_SSP, ORDER, IL>(L, C, st, grid);
  }
  abort();
}

int main(int argc, char** argv) {
  if (argc != 21) return 2;
  const int order = atoi(argv[1]), tile = atoi(argv[2]), mode = atoi(argv[3]), nx = atoi(argv[4]), ny = atoi(argv[5]),
            nz = atoi(argv[6]), g = atoi(argv[7]), ko_order = atoi(argv[12]), grid = atoi(argv[16]);
  const double h = atof(argv[8]), eps = atof(argv[9]), eta = atof(argv[10]), sgc = atof(argv[11]), a = atof(argv[13]),
               ca = atof(argv[14]), cb = atof(argv[15]);
  Layout L = make_layout(nx, ny, nz, g);
  unsigned err = 0;
  L.err = &err;
  const size_t ng = (size_t)25 * L.tot_z * L.tot_y * (nx + 2 * g);
  auto load = [&](const char* path) {
    std::vector<double> v(ng);
    FILE* f = fopen(path, "rb");
    if (!f || fread(v.data(), 8, ng, f) != ng) { fprintf(stderr, "cannot read %s\n", path); exit(3); }
    fclose(f);
    return to_padded(L, v);
  };
  std::vector<double> in = load(argv[17]), U = load(argv[18]), S = load(argv[19]);
  std::vector<double> out((size_t)25 * L.vstride, 0.0);
  auto al = [](std::vector<double>& v) { return v.data(); };   // vectors of doubles are 16-byte aligned: enough here
  Coef C;   // as chemora.cu's make_coef
  C.inv_h = 1.0 / h; C.inv_h2 = 1.0 / (h * h); C.ko = eps / (64.0 * h); C.eta = eta; C.sgc = sgc;
  const double w5[5] = {15.0, -6.0, 1.0, 0.0, 0.0}, w9[5] = {210.0, -120.0, 45.0, -10.0, 1.0};
  for (int k = 0; k < 5; ++k) C.kq[k] = ko_order == 9 ? eps / (1024.0 * h) * w9[k] : C.ko * w5[k];
  Stage st{al(in), al(U), al(S), al(out), a, mode >= 10 ? mode - 10 : mode, ca, cb};
  if (mode == MODE_FIRST) st.U = al(in);   // stage 1 reads U == in
  chm_emu::Stats s;
  if (order == 8 && tile == 0) s = run_mode<16, 4, 4, 8>(mode, L, C, st, grid);
  else if (order == 4 && tile == 0) s = run_mode<16, 4, 4, 4>(mode, L, C, st, grid);
  else if (order == 4 && tile == 1) s = run_mode<16, 8, 2, 4>(mode, L, C, st, grid);
  else if (order == 4 && tile == 3) s = run_mode<16, 2, 8, 4>(mode, L, C, st, grid);
  else if (order == 4 && tile == 5) s = run_mode<16, 4, 4, 4, 1>(mode, L, C, st, grid);
  else if (order == 4 && tile == 6) s = run_mode<16, 4, 4, 4, 2>(mode, L, C, st, grid);
  else if (order == 4 && tile == 7) s = run_mode<16, 4, 4, 4, 3>(mode, L, C, st, grid);
  else { fprintf(stderr, "instance not built into the emulator\n"); return 5; }
  std::vector<double> o(ng), so(ng), uo(ng);
  from_padded(L, out.data(), o); from_padded(L, S.data(), so); from_padded(L, (mode == MODE_FIRST ? in : U).data(), uo);
  FILE* f = fopen(argv[20], "wb");
  if (!f) return 4;
  fwrite(o.data(), 8, ng, f); fwrite(so.data(), 8, ng, f); fwrite(uo.data(), 8, ng, f);
  fclose(f);
  printf("err %u loads %ld bytes %ld\n", err, s.tma_loads, s.tma_bytes);
  return 0;
}
