// wave_emu.cpp -- runs the plane-ring kernel's SOURCE (csrc/kernels_wave_tma.cu: the (phi, pi) system and, with five
// variables a plane, the paper's Sample-1 system) on the host, on top of cta_emu.hpp.  Test infrastructure only.
//
//   wave_emu <nvars 2|5> <order> <ko 0|1> <which> <mode> <nx> <ny> <nz> <g> <h> <eps> <a> <ca> <cb> <grid>
//            <in.bin> <U.bin> <S.bin> <out.bin>
// in/U/S.bin: ghosted arrays [V][nz+2g][ny+2g][nx+2g]; out.bin: Stage::out, S, U as the launch left them.
#include "cta_emu.hpp"

#include "../../paper_1307_6488_b200/csrc/kernels_wave_tma.cu"

using namespace chm;

static Layout make_layout(int nx, int ny, int nz, int g, int V) {   // the rule of chemora_create for the wave systems
  Layout L{};
  L.nx = nx; L.ny = ny; L.nz = nz; L.g = g; L.nvars = V;
  L.xo = g;
  L.pitch = ((long)L.xo + nx + g + 15) / 16 * 16;
  L.tot_y = ny + 2 * g; L.tot_z = nz + 2 * g;
  L.plane = L.pitch * L.tot_y;
  L.vstride = L.plane * L.tot_z;
  L.col_rows = 32;
  return L;
}

template <int ORDER, bool KO, int TX, int TY, int ZC, int NV>
static chm_emu::Stats run(const Layout& L, const Coef& C, const Stage& st, int grid_req) {
  using K = wv::Cfg<ORDER, KO, TX, TY, NV>;
  if constexpr (!K::FITS) { fprintf(stderr, "ring does not fit\n"); exit(6); }
  else {
    CUtensorMap tm;
    tm.base = st.in;
    tm.dims[0] = L.pitch; tm.dims[1] = L.tot_y; tm.dims[2] = L.tot_z; tm.dims[3] = L.nvars;
    tm.strides[0] = L.pitch * 8; tm.strides[1] = L.plane * 8; tm.strides[2] = L.vstride * 8;
    tm.box[0] = K::ROW; tm.box[1] = K::COLS; tm.box[2] = 1; tm.box[3] = NV;
    const int ntx = (L.nx + TX - 1) / TX, nty = (L.ny + TY - 1) / TY, ntz = (L.nz + ZC - 1) / ZC;
    const int nitems = ntx * nty * ntz, grid = nitems < grid_req ? nitems : grid_req;
    return chm_emu::run_grid(grid, TX, TY, K::SMEM, [&] { wave_tma_kernel<ORDER, KO, TX, TY, ZC, NV>(tm, L, C, st, ntx, nty, ntz); });
  }
}

template <int ORDER, bool KO>
static chm_emu::Stats pick(int V, int which, const Layout& L, const Coef& C, const Stage& st, int grid) {
  if (V == 2 && which == 0) return run<ORDER, KO, 32, 16, 32, 2>(L, C, st, grid);
  if (V == 2 && which == 2) return run<ORDER, KO, 64, 8, 32, 2>(L, C, st, grid);
  if (V == 5 && which == 0) return run<ORDER, KO, 16, 8, 64, 5>(L, C, st, grid);
  if (V == 5 && which == 1) return run<ORDER, KO, 16, 16, 64, 5>(L, C, st, grid);
  fprintf(stderr, "instance not built into the emulator\n");
  exit(5);
}

int main(int argc, char** argv) {
  if (argc != 20) return 2;
  const int V = atoi(argv[1]), order = atoi(argv[2]), ko = atoi(argv[3]), which = atoi(argv[4]), mode = atoi(argv[5]),
            nx = atoi(argv[6]), ny = atoi(argv[7]), nz = atoi(argv[8]), g = atoi(argv[9]), grid = atoi(argv[15]);
  const double h = atof(argv[10]), eps = atof(argv[11]), a = atof(argv[12]), ca = atof(argv[13]), cb = atof(argv[14]);
  Layout L = make_layout(nx, ny, nz, g, V);
  unsigned err = 0;
  L.err = &err;
  const long tx = nx + 2 * g;
  const size_t ng = (size_t)V * L.tot_z * L.tot_y * tx;
  auto load = [&](const char* path) {
    std::vector<double> v(ng), p((size_t)V * L.vstride, 0.0);
    FILE* f = fopen(path, "rb");
    if (!f || fread(v.data(), 8, ng, f) != ng) { fprintf(stderr, "cannot read %s\n", path); exit(3); }
    fclose(f);
    for (size_t r = 0; r < (size_t)V * L.tot_z * L.tot_y; ++r) memcpy(&p[r * L.pitch + (L.xo - g)], &v[r * tx], tx * 8);
    return p;
  };
  std::vector<double> in = load(argv[16]), U = load(argv[17]), S = load(argv[18]), out((size_t)V * L.vstride, 0.0);
  Coef C{};
  C.inv_h = 1.0 / h; C.inv_h2 = 1.0 / (h * h); C.ko = ko ? eps / (64.0 * h) : 0.0;
  Stage st{in.data(), mode == MODE_FIRST ? in.data() : U.data(), S.data(), out.data(), a, mode, ca, cb};
  chm_emu::Stats s;
  if (order == 4) s = ko ? pick<4, true>(V, which, L, C, st, grid) : pick<4, false>(V, which, L, C, st, grid);
  else s = ko ? pick<8, true>(V, which, L, C, st, grid) : pick<8, false>(V, which, L, C, st, grid);
  FILE* f = fopen(argv[19], "wb");
  if (!f) return 4;
  for (const std::vector<double>* b : {&out, &S, mode == MODE_FIRST ? &in : &U}) {
    std::vector<double> v(ng);
    for (size_t r = 0; r < (size_t)V * L.tot_z * L.tot_y; ++r) memcpy(&v[r * tx], &(*b)[r * L.pitch + (L.xo - g)], tx * 8);
    fwrite(v.data(), 8, ng, f);
  }
  fclose(f);
  printf("err %u loads %ld bytes %ld\n", err, s.tma_loads, s.tma_bytes);
  return 0;
}
