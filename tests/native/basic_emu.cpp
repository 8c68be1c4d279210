// basic_emu.cpp -- runs the remaining kernels' SOURCE on the host (cta_emu.hpp): csrc/kernels_basic.cu (periodic ghost
// fill, pack/unpack, constraint enforcement, the L1-path kernels of both wave systems, the Energy calculation) and
// csrc/kernels_bssn.cu (the derivative-split BSSN variant: derivative kernel, then right-hand side from the arrays),
// each on the grid its launcher gives it (geometry restated here: the launchers themselves are host CUDA code).
// Test infrastructure only.
//   basic_emu <op> <system> <order> <nx> <ny> <nz> <g> <h> <eps> <tile> <mode> <a> <ko_order> <in.bin> <out.bin>
//   op: fill | roundtrip | enforce | wave | split | energy        (system 0 wave, 1 BSSN, 2 Sample-1)
// in.bin: ghosted [V][nz+2g][ny+2g][nx+2g]; out.bin: the ghosted result (wave/split: Stage::out of a plain RHS launch
// or, mode 2, of a middle RK4 stage with U = S = in; energy: packed field [nz][ny][nx] followed by the grid sum).
#include "cta_emu.hpp"

#include "../../paper_1307_6488_b200/csrc/kernels_basic.cu"
#include "../../paper_1307_6488_b200/csrc/kernels_bssn.cu"

using namespace chm;

int main(int argc, char** argv) {
  if (argc != 16) return 2;
  const std::string op = argv[1];
  const int system = atoi(argv[2]), order = atoi(argv[3]), nx = atoi(argv[4]), ny = atoi(argv[5]), nz = atoi(argv[6]),
            g = atoi(argv[7]), tile = atoi(argv[10]), mode = atoi(argv[11]), ko_order = atoi(argv[13]);
  const double h = atof(argv[8]), eps = atof(argv[9]), a = atof(argv[12]);
  const int V = system == 0 ? 2 : system == 1 ? 25 : 5;
  Layout L{};   // the rule of chemora_create
  L.nx = nx; L.ny = ny; L.nz = nz; L.g = g; L.nvars = V;
  L.xo = (system == 1 && ((g - 3) & 1)) ? g + 1 : g;
  L.pitch = ((long)L.xo + nx + g + 15) / 16 * 16;
  L.tot_y = ny + 2 * g; L.tot_z = nz + 2 * g;
  L.plane = L.pitch * L.tot_y; L.vstride = L.plane * L.tot_z;
  const long tx = nx + 2 * g;
  const size_t rows = (size_t)V * L.tot_z * L.tot_y, ng = rows * tx;
  std::vector<double> ghosted(ng), in((size_t)V * L.vstride, 0.0), out((size_t)V * L.vstride, 0.0);
  FILE* f = fopen(argv[14], "rb");
  if (!f || fread(ghosted.data(), 8, ng, f) != ng) return 3;
  fclose(f);
  for (size_t r = 0; r < rows; ++r) memcpy(&in[r * L.pitch + (L.xo - g)], &ghosted[r * tx], tx * 8);
  Coef C{};   // as chemora.cu's make_coef
  C.inv_h = 1.0 / h; C.inv_h2 = 1.0 / (h * h); C.ko = eps / (64.0 * h); C.eta = 1.0; C.sgc = 0.75;
  const double w5[5] = {15.0, -6.0, 1.0, 0.0, 0.0}, w9[5] = {210.0, -120.0, 45.0, -10.0, 1.0};
  for (int k = 0; k < 5; ++k) C.kq[k] = ko_order == 9 ? eps / (1024.0 * h) * w9[k] : C.ko * w5[k];
  std::vector<double> S(in), U(in);
  Stage st{in.data(), U.data(), S.data(), out.data(), a, mode, 0.0, 0.0};
  const double* result = out.data();
  std::vector<double> extra;
  const TileShape T = kTilesMarch[tile % 6];
  const int gx = (nx + T.tx - 1) / T.tx, gy = (ny + T.ty - 1) / T.ty, gz = (nz + T.tz - 1) / T.tz;

  if (op == "fill") {            // launch_fill_ghosts
    const long rowsA = 2L * g * L.tot_y, rowsAB = rowsA + 2L * g * L.nz, rowsC = (long)L.nz * L.ny;
    int lpr_shift = 0;
    while ((1 << lpr_shift) < 2 * g && lpr_shift < 5) ++lpr_shift;
    const long tasks = rowsAB + (rowsC + (32 >> lpr_shift) - 1) / (32 >> lpr_shift);
    const FillLink self{in.data(), L.vstride, L.nz, in.data(), L.vstride};
    chm_emu::run_grid_serial((int)((tasks + 7) / 8), V, 1, 256, 1,
                             [&] { fill_ghosts_kernel(L, in.data(), (int)rowsA, (int)rowsAB, lpr_shift, self); });
    result = in.data();
  } else if (op == "roundtrip") {   // launch_pack both ways: padded interior -> packed -> a fresh padded state
    std::vector<double> packed((size_t)V * nx * ny * nz);
    chm_emu::run_grid_serial((nx + 255) / 256, ny, nz * V, 256, 1, [&] { pack_kernel(L, in.data(), packed.data(), false); });
    chm_emu::run_grid_serial((nx + 255) / 256, ny, nz * V, 256, 1, [&] { pack_kernel(L, packed.data(), out.data(), true); });
  } else if (op == "enforce") {     // launch_enforce
    chm_emu::run_grid_serial((nx + 255) / 256, ny, nz, 256, 1, [&] { enforce_kernel(L, in.data()); });
    result = in.data();
  } else if (op == "wave") {        // wave_go / wave1_go: tile ids 0, 1, 5 built here
    auto go = [&](auto kern) { chm_emu::run_grid_serial(gx, gy, gz, T.tx, T.ty, [&] { kern(L, C, st); }); };
    const bool ko = eps != 0.0;
#define WV(K, O, KOF) \
    (tile == 0 ? go(K<O, KOF, 32, 4, 8>) : tile == 1 ? go(K<O, KOF, 32, 8, 8>) : go(K<O, KOF, 16, 16, 8>))
    if (tile != 0 && tile != 1 && tile != 5) return 5;
    if (system == 0) { if (order == 4) { if (ko) WV(wave_kernel, 4, true); else WV(wave_kernel, 4, false); }
                       else { if (ko) WV(wave_kernel, 8, true); else WV(wave_kernel, 8, false); } }
    else { if (order == 4) { if (ko) WV(wave1_kernel, 4, true); else WV(wave1_kernel, 4, false); }
           else { if (ko) WV(wave1_kernel, 8, true); else WV(wave1_kernel, 8, false); } }
  } else if (op == "split") {       // bssn_go: derivatives into 136 arrays, then the right-hand side from them
    const long n = packed_stride(L);
    std::vector<double> derivs((size_t)kNumDerivArrays * n, 0.0);
    if (tile != 0 && tile != 5) return 5;
    auto run2 = [&](auto dk, auto fk) {
      chm_emu::run_grid_serial(gx, gy, gz, T.tx, T.ty, [&] { dk(L, C, in.data(), derivs.data()); });
      chm_emu::run_grid_serial(gx, gy, gz, T.tx, T.ty, [&] { fk(L, C, derivs.data(), st); });
    };
    if (tile == 0) { if (order == 4) run2(bssn_derivs_kernel<32, 4, 8, 4>, bssn_from_derivs_kernel<32, 4, 8>);
                     else run2(bssn_derivs_kernel<32, 4, 8, 8>, bssn_from_derivs_kernel<32, 4, 8>); }
    else { if (order == 4) run2(bssn_derivs_kernel<16, 16, 8, 4>, bssn_from_derivs_kernel<16, 16, 8>);
           else run2(bssn_derivs_kernel<16, 16, 8, 8>, bssn_from_derivs_kernel<16, 16, 8>); }
  } else if (op == "energy") {      // launch_energy: field + grid sum (warp shuffles, a block barrier, one atomic per block)
    extra.assign((size_t)nx * ny * nz + 1, 0.0);
    chm_emu::run_grid((nx + 255) / 256, 256, 1, 0, [&] { energy_kernel(L, in.data(), extra.data(), &extra[(size_t)nx * ny * nz]); }, ny, nz);
    f = fopen(argv[15], "wb");
    fwrite(extra.data(), 8, extra.size(), f);
    fclose(f);
    return 0;
  } else return 2;
  for (size_t r = 0; r < rows; ++r) memcpy(&ghosted[r * tx], &result[r * L.pitch + (L.xo - g)], tx * 8);
  f = fopen(argv[15], "wb");
  if (!f) return 4;
  fwrite(ghosted.data(), 8, ng, f);
  if (mode == MODE_MID) {   // S too
    for (size_t r = 0; r < rows; ++r) memcpy(&ghosted[r * tx], &S[r * L.pitch + (L.xo - g)], tx * 8);
    fwrite(ghosted.data(), 8, ng, f);
  }
  fclose(f);
  return 0;
}
