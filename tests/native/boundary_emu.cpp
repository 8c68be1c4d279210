// boundary_emu.cpp -- runs csrc/kernels_boundary.cu's kernels (the radiative face kernel, the sweep guard's agreement
// norm) on the host on top of cta_emu.hpp, with the launch geometry of their launchers.  Test infrastructure only.
//   boundary_emu rad <system 0|1|2> <nx> <ny> <nz> <g> <h> <mode> <a> <ca> <cb> <in.bin> <U.bin> <S.bin> <out.bin>
//   boundary_emu maxdiff <nvars> <n per variable> <a.bin> <b.bin>        -> prints 2 x nvars doubles
#include "cta_emu.hpp"

#include "../../paper_1307_6488_b200/csrc/kernels_boundary.cu"

using namespace chm;

int main(int argc, char** argv) {
  if (argc >= 2 && !strcmp(argv[1], "maxdiff")) {
    const int V = atoi(argv[2]);
    const long n = atol(argv[3]);
    std::vector<double> a((size_t)V * n), b((size_t)V * n);
    FILE* f = fopen(argv[4], "rb"); if (!f || fread(a.data(), 8, a.size(), f) != a.size()) return 3; fclose(f);
    f = fopen(argv[5], "rb"); if (!f || fread(b.data(), 8, b.size(), f) != b.size()) return 3; fclose(f);
    std::vector<unsigned long long> out(2 * V, 0);
    long blocks = (n + 256L * 8 - 1) / (256L * 8);   // as launch_maxdiff
    if (blocks > 1024) blocks = 1024;
    if (blocks < 1) blocks = 1;
    chm_emu::run_grid((int)blocks, 256, 1, 0, [&] { maxdiff_kernel(a.data(), b.data(), n, out.data()); }, V);
    for (int i = 0; i < 2 * V; ++i) { double d; memcpy(&d, &out[i], 8); printf("%.17g\n", d); }
    return 0;
  }
  if (argc != 16 || strcmp(argv[1], "rad")) return 2;
  const int system = atoi(argv[2]), nx = atoi(argv[3]), ny = atoi(argv[4]), nz = atoi(argv[5]), g = atoi(argv[6]),
            mode = atoi(argv[8]);
  const double h = atof(argv[7]), a = atof(argv[9]), ca = atof(argv[10]), cb = atof(argv[11]);
  const int V = system == 0 ? 2 : system == 1 ? 25 : 5;
  Layout L{};   // the rule of chemora_create
  L.nx = nx; L.ny = ny; L.nz = nz; L.g = g; L.nvars = V;
  L.xo = (system == 1 && ((g - 3) & 1)) ? g + 1 : g;
  L.pitch = ((long)L.xo + nx + g + 15) / 16 * 16;
  L.tot_y = ny + 2 * g; L.tot_z = nz + 2 * g;
  L.plane = L.pitch * L.tot_y; L.vstride = L.plane * L.tot_z;
  const long tx = nx + 2 * g;
  const size_t ng = (size_t)V * L.tot_z * L.tot_y * tx, rows = (size_t)V * L.tot_z * L.tot_y;
  auto load = [&](const char* path) {
    std::vector<double> v(ng), p((size_t)V * L.vstride, 0.0);
    FILE* f = fopen(path, "rb");
    if (!f || fread(v.data(), 8, ng, f) != ng) { fprintf(stderr, "cannot read %s\n", path); exit(3); }
    fclose(f);
    for (size_t r = 0; r < rows; ++r) memcpy(&p[r * L.pitch + (L.xo - g)], &v[r * tx], tx * 8);
    return p;
  };
  std::vector<double> in = load(argv[12]), U = load(argv[13]), S = load(argv[14]), out((size_t)V * L.vstride, 7.0);
  Stage st{in.data(), mode == MODE_FIRST ? in.data() : U.data(), S.data(), out.data(), a, mode, ca, cb};
  const unsigned mask = system == 1 ? (1u << 0) | (1u << 1) | (1u << 4) | (1u << 6) | (1u << 17) : 0u;   // as chemora.cu
  const RadGeom G = rad_geom(L);
  chm_emu::run_grid_serial((int)((G.tasks + 7) / 8), V, 1, 256, 1,   // no barrier, no shuffle: thread after thread
                           [&] { radiative_kernel(L, st, h, mask, (int)G.rowsA, (int)G.rowsAB, G.lpr_shift); });
  FILE* f = fopen(argv[15], "wb");
  if (!f) return 4;
  for (const std::vector<double>* b : {&out, &S, mode == MODE_FIRST ? &in : &U}) {
    std::vector<double> v(ng);
    for (size_t r = 0; r < rows; ++r) memcpy(&v[r * tx], &(*b)[r * L.pitch + (L.xo - g)], tx * 8);
    fwrite(v.data(), 8, ng, f);
  }
  fclose(f);
  return 0;
}
